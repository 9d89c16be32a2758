// mvd_reduce_sum_static: the fp64 sum of a device float array (the numerator of psi^0, the mean of all views,
// PAPER.md L304 / L421) for callers that have no device memory to spare and no way to get any.
//
// Who that is.  mvd_reduce_sum (mvd.cu) wants a scratch buffer from its caller, and the Python binding gets one from
// torch's allocator on every call.  Three kinds of callers of this library cannot do that:
//   * a deconvolution that has already handed the whole GPU to its workspace (config 5 whole: ~150 of 180 GB), or a
//     process whose memory pool has taken all of HBM up front: a cudaMalloc there fails, and a request to the pool
//     may trigger a defragmenting free/malloc round that stalls every stream;
//   * the acquisition side of a time-lapse, which sums each new time-point while other streams upload the next one:
//     cudaMalloc and cudaFree synchronise the whole device, so one allocation per time-point serialises the copies
//     the stream schedule was built to overlap;
//   * a plug-in inside a host application (an image-processing suite driving the C ABI) that is given device
//     pointers to views but is not allowed to allocate on the application's device.
// For them the partial sums live in a fixed array in the library's own device image (g_scratch below, ~128 KB per GPU
// that loads libmvd.so, held until the process exits).  The entry point calls no cudaMalloc, cudaFree or any library
// routine that allocates; the caller passes only the input and the host address of the result.
//
// This file is self-contained: it shares no kernel with mvd.cu and changes none of its paths.
#include "../../include/mvd.h"

#include <cuda_runtime.h>

#include <cstdio>
#include <mutex>

namespace {

constexpr int kThreads = 256;
constexpr long long kChunk = 65536;            // floats summed by one block into one partial (256 KB of input)
constexpr int kMaxChunks = 16384;              // partials the array holds
constexpr long long kMaxN = kChunk * kMaxChunks;   // 2^30 floats = 4 GiB of input (config 5: 2^29 voxels per view)
constexpr int kResultSlot = kMaxChunks;        // g_scratch[kResultSlot]     : the total
constexpr int kTicketSlot = kMaxChunks + 1;    // g_scratch[kTicketSlot] (as unsigned): blocks that have finished
constexpr int kMaxDevices = 64;

// The scratch.  Every call on a device uses this one array and finds in it whatever the last call left.
// In HOST code the name g_scratch is only a handle for cudaGetSymbolAddress: it is not a device address and must never
// be passed to a kernel as one (scratch_of below is the only place host code mentions it).
static __device__ __align__(256) double g_scratch[kMaxChunks + 32];

__device__ __forceinline__ double block_sum(double v, double* red) {
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_down_sync(0xffffffffu, v, o);
  __syncthreads();
  if (lane == 0) red[warp] = v;
  __syncthreads();
  v = (threadIdx.x < kThreads / 32) ? red[threadIdx.x] : 0.0;
  if (warp == 0) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_down_sync(0xffffffffu, v, o);
  }
  return v;   // valid in thread 0
}

// Block b sums a[b*kChunk, min(n, (b+1)*kChunk)) into scratch[b]; the block that finishes last adds the partials in
// index order (so the result does not depend on which block that is, nor on the SM count of the device), stores the
// total in scratch[kResultSlot] and puts the ticket back to zero for the next call.
__global__ void __launch_bounds__(kThreads) sum_chunks_kernel(const float* __restrict__ a, long long n,
                                                              double* __restrict__ scratch) {
  __shared__ double red[32];
  __shared__ bool is_last;
  const long long lo = (long long)blockIdx.x * kChunk;
  const long long m = (n - lo < kChunk) ? (n - lo) : kChunk;   // may be <= 0 only when n == 0
  const float* p = a + lo;
  double s = 0.0;
  const long long m4 = ((reinterpret_cast<size_t>(p) & 15) == 0 && m > 0) ? m / 4 : 0;
  const float4* p4 = reinterpret_cast<const float4*>(p);
  for (long long j = threadIdx.x; j < m4; j += kThreads) {
    const float4 v = __ldg(p4 + j);
    s += (double)v.x + (double)v.y + (double)v.z + (double)v.w;
  }
  for (long long j = m4 * 4 + threadIdx.x; j < m; j += kThreads) s += (double)__ldg(p + j);
  s = block_sum(s, red);
  unsigned int* ticket = reinterpret_cast<unsigned int*>(scratch + kTicketSlot);
  if (threadIdx.x == 0) {
    scratch[blockIdx.x] = s;
    __threadfence();
    is_last = atomicAdd(ticket, 1u) == gridDim.x - 1;
  }
  __syncthreads();
  if (!is_last) return;
  __threadfence();
  double t = 0.0;
  for (int i = threadIdx.x; i < (int)gridDim.x; i += kThreads) t += __ldcg(scratch + i);
  t = block_sum(t, red);
  if (threadIdx.x == 0) {
    scratch[kResultSlot] = t;
    *ticket = 0u;
  }
}

thread_local char t_err[256] = "";

mvd_status fail(mvd_status s, const char* fmt, long long a = 0, long long b = 0) {
  snprintf(t_err, sizeof t_err, fmt, a, b);
  return s;
}

mvd_status fail_cuda(cudaError_t e, const char* what) {
  snprintf(t_err, sizeof t_err, "mvd_reduce_sum_static: %s: %s", what, cudaGetErrorString(e));
  return MVD_ERR_CUDA;
}

// Device address of g_scratch on the CURRENT device, looked up once per device (the first call on a device does it:
// cudaGetSymbolAddress may load the module there, so that call belongs before any stream capture).
cudaError_t scratch_of(int dev, double** out) {
  static std::mutex mu;
  static double* addr[kMaxDevices] = {};
  std::lock_guard<std::mutex> lock(mu);
  if (!addr[dev]) {
    double* p = nullptr;
    const cudaError_t e = cudaGetSymbolAddress(reinterpret_cast<void**>(&p), g_scratch);
    if (e != cudaSuccess) return e;
    addr[dev] = p;
  }
  *out = addr[dev];
  return cudaSuccess;
}

}  // namespace

extern "C" {

long long mvd_reduce_sum_static_max(void) { return kMaxN; }

const char* mvd_reduce_sum_static_error(void) { return t_err; }

mvd_status mvd_reduce_sum_static(const float* src, long long n, void* stream, double* host_out) {
  t_err[0] = 0;
  if (!src || !host_out) return fail(MVD_ERR_INVALID_ARG, "mvd_reduce_sum_static: src and host_out must not be NULL");
  if (n < 0) return fail(MVD_ERR_INVALID_ARG, "mvd_reduce_sum_static: n = %lld is negative", n);
  if (n > kMaxN)
    return fail(MVD_ERR_UNSUPPORTED,
                "mvd_reduce_sum_static: n = %lld exceeds the %lld floats the built-in scratch array covers; "
                "split the input or use mvd_reduce_sum with your own scratch", n, kMaxN);
  int dev = -1;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return fail_cuda(e, "cudaGetDevice");
  if (dev < 0 || dev >= kMaxDevices)
    return fail(MVD_ERR_UNSUPPORTED, "mvd_reduce_sum_static: device ordinal %lld beyond the %lld this build tracks", dev,
                kMaxDevices);
  double* scratch = nullptr;
  e = scratch_of(dev, &scratch);
  if (e != cudaSuccess) return fail_cuda(e, "cudaGetSymbolAddress of the scratch array");
  cudaStream_t st = reinterpret_cast<cudaStream_t>(stream);
  // the ticket has to start at zero.  A call that ran to its end leaves it there, one that died half-way does not.
  e = cudaMemsetAsync(scratch + kTicketSlot, 0, sizeof(double), st);
  if (e != cudaSuccess) return fail_cuda(e, "clearing the ticket");
  const int nchunks = n == 0 ? 1 : (int)((n + kChunk - 1) / kChunk);
  sum_chunks_kernel<<<nchunks, kThreads, 0, st>>>(src, n, scratch);
  e = cudaGetLastError();
  if (e != cudaSuccess) return fail_cuda(e, "kernel launch");
  e = cudaMemcpyAsync(host_out, scratch + kResultSlot, sizeof(double), cudaMemcpyDeviceToHost, st);
  if (e == cudaSuccess) e = cudaStreamSynchronize(st);
  if (e != cudaSuccess) return fail_cuda(e, "reading the result back");
  return MVD_OK;
}

}  // extern "C"
