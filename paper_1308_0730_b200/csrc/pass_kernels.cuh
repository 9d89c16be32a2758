// Pencil-pass kernels of the multi-view Richardson-Lucy iteration, templated on the split
// M = A*B of the pencil length (sm_100a; fp32; no tensor cores: the path is HBM-bound FFT and
// pointwise work, "two convolutions computed in Fourier space and several
// per-pixel operations").
//
// One length-M DFT is two register-resident transforms (fft_reg.cuh) with ONE shared-memory
// transposition between them:
//   form F:  in  n = n1*B + n2 (a thread owns n2, holds all n1)  -> A-point FFT over n1 -> twiddle
//            W_M^{n2 k1} -> smem -> a thread owns k1, holds all n2 -> B-point FFT over n2
//            -> out k = k1 + A*k2.
//   form G:  the mirror image (in k = k1 + A*k2 owned by k1; out n = n1*B + n2 owned by n2).
// F followed by G (or G followed by F) chains through registers, which is what lets the fused
// kernels below keep a pencil on chip between the forward and the inverse transform:
//   zconv_kernel : z-forward (F) . kernel spectrum . z-inverse (G)       (S1/S3 of DESIGN.md)
//   xrow_kernel  : x-inverse (G) -> crop + quotient/update -> zero-pad + x-forward (F)   (S2/S4)
//   strided_fft_kernel : plain F along y (or z), pruned input / cropped output.
// Global memory is touched exactly once per element per pass, always with the unit-stride axis
// across the lanes of a warp.
#pragma once

#include <cstdlib>

#include "fft_ops.h"
#include "fft_reg.cuh"

namespace mvd {

template <int A, int B>
struct PassCfg {
  static constexpr int M = A * B;
  static constexpr int AB_MAX = A > B ? A : B;
  // 512 threads cap the kernel at 128 registers/thread: enough up to 27-point transforms
  static constexpr int MAX_THREADS = AB_MAX > 27 ? 256 : 512;
  static constexpr int AP = A | 1;   // odd strides: conflict-free 64-bit shared-memory columns
  static constexpr int BP = B | 1;
  static constexpr int ROW_F2 = (A * BP > B * AP) ? A * BP : B * AP;   // float2 per row (xrow)
};

MVD_DEV float2 ld_tw(const float2* tw, int idx) { return __ldg(tw + idx); }

// Tikhonov-regularised value of an update u (mvd.h, R14): positive root of (lam/2) psi^2 + psi - u = 0
// in the cancellation-free form 2u / (1 + sqrt(1 + 2 lam u)).  Hardware reciprocal square root and reciprocal
// (a few ulp: far inside the 1e-5 budget) keep the regularised path at six instructions per voxel, so the
// unregularised path (lam = 0, a uniform branch) keeps its code size and issue slots.
MVD_DEV float tikhonov_value(float u, float lam) {
  const float t = fmaf(2.f * lam, u, 1.f);          // >= 1: no denormal or zero handling needed
  float r, q;
  asm("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(t));
  asm("div.approx.ftz.f32 %0, %1, %2;" : "=f"(q) : "f"(2.f * u), "f"(fmaf(t, r, 1.f)));
  return q;
}
MVD_DEV float tikhonov_update(float u, float lam) { return lam > 0.f ? tikhonov_value(u, lam) : u; }

// =========================================================================================
// strided pencil FFT, form F, direction DIR (-1 forward, +1 inverse; unnormalised)
// =========================================================================================
template <int A, int B, int DIR>
__global__ void __launch_bounds__(PassCfg<A, B>::MAX_THREADS)
strided_fft_kernel(const StridedArgs p) {
  extern __shared__ float2 sm[];
  const int T = p.T;
  const long long blk = blockIdx.x;
  const int tile = int(blk % p.tiles_per_line);
  const long long outer = blk / p.tiles_per_line;
  const long long x0 = (long long)tile * T;
  const int xvalid = int(min((long long)T, p.line_len - x0));
  const float2* in = p.in + outer * p.in_outer_stride + x0;
  float2* out = p.out + outer * p.out_outer_stride + x0;

  for (int i = threadIdx.x; i < T * B; i += blockDim.x) {
    const int n2 = i / T;
    const int x = i - n2 * T;
    const bool xv = x < xvalid;
    float2 v[A];
    static_for<0, A>([&](auto n1_) {
      constexpr int n1 = decltype(n1_)::value;
      const int n = n1 * B + n2;
      v[n1] = (xv && n < p.n_in) ? in[(long long)n * p.in_pstride + x] : make_float2(0.f, 0.f);
    });
    FftReg<A, DIR>::run(v);
    static_for<0, A>([&](auto k1_) {
      constexpr int k1 = decltype(k1_)::value;
      if constexpr (k1 > 0) {
        const float2 w = ld_tw(p.tw, n2 * k1);
        v[k1] = DIR < 0 ? cmul(v[k1], w) : cmul_conj(v[k1], w);
      }
      sm[k1 * B * T + i] = v[k1];
    });
  }
  __syncthreads();
  for (int j = threadIdx.x; j < T * A; j += blockDim.x) {
    const int k1 = j / T;
    const int x = j - k1 * T;
    float2 u[B];
    static_for<0, B>([&](auto n2_) {
      constexpr int n2 = decltype(n2_)::value;
      u[n2] = sm[(k1 * B + n2) * T + x];
    });
    FftReg<B, DIR>::run(u);
    if (x < xvalid) {
      static_for<0, B>([&](auto k2_) {
        constexpr int k2 = decltype(k2_)::value;
        const int k = k1 + A * k2;
        if (k < p.n_out) out[(long long)k * p.out_pstride + x] = u[k2];
      });
    }
  }
}

// =========================================================================================
// fused z pass: crop(IFFT_z( FFT_z(zero-padded pencil) * spectrum ))
// One round per CTA: T*max(A,B) <= blockDim.x.
// =========================================================================================
template <int A, int B>
__global__ void __launch_bounds__(PassCfg<A, B>::MAX_THREADS)
zconv_kernel(const ZconvArgs p) {
  extern __shared__ float2 sm[];
  const int T = p.T;
  const long long x0 = (long long)blockIdx.x * T;
  const int xvalid = int(min((long long)T, p.plane - x0));
  const float2* in = p.in + x0;
  float2* out = p.out + x0;
  const float2* spec = p.spec + x0;
  const int tid = threadIdx.x;

  // F1: thread (x, n2)
  const int n2 = tid / T;
  const int xa = tid - n2 * T;
  const bool act1 = tid < T * B;
  if (act1) {
    const bool xv = xa < xvalid;
    float2 v[A];
    static_for<0, A>([&](auto n1_) {
      constexpr int n1 = decltype(n1_)::value;
      const int n = n1 * B + n2;
      v[n1] = (xv && n < p.nz) ? in[(long long)n * p.plane + xa] : make_float2(0.f, 0.f);
    });
    FftReg<A, -1>::run(v);
    static_for<0, A>([&](auto k1_) {
      constexpr int k1 = decltype(k1_)::value;
      if constexpr (k1 > 0) v[k1] = cmul(v[k1], ld_tw(p.tw, n2 * k1));
      sm[k1 * B * T + tid] = v[k1];
    });
  }
  __syncthreads();

  // F2 . spectrum . G1: thread (x, k1)
  const int k1 = tid / T;            // same split as n2 (both are tid / T)
  const bool act2 = tid < T * A;
  float2 u[B];
  if (act2) {
    static_for<0, B>([&](auto n2_) {
      constexpr int m = decltype(n2_)::value;
      u[m] = sm[(k1 * B + m) * T + xa];
    });
    FftReg<B, -1>::run(u);
    const bool xv = xa < xvalid;
    static_for<0, B>([&](auto k2_) {
      constexpr int k2 = decltype(k2_)::value;
      const float2 h = xv ? spec[(long long)(k1 + A * k2) * p.plane + xa] : make_float2(0.f, 0.f);
      u[k2] = cmul(u[k2], h);
    });
    FftReg<B, 1>::run(u);            // inverse over k2 -> index n2
    static_for<1, B>([&](auto n2_) {
      constexpr int m = decltype(n2_)::value;
      u[m] = cmul_conj(u[m], ld_tw(p.tw, m * k1));
    });
  }
  __syncthreads();                   // every thread has read its F-exchange column
  if (act2) {
    static_for<0, B>([&](auto n2_) {
      constexpr int m = decltype(n2_)::value;
      sm[(k1 * B + m) * T + xa] = u[m];
    });
  }
  __syncthreads();

  // G2: thread (x, n2)
  if (act1 && xa < xvalid) {
    float2 v[A];
    static_for<0, A>([&](auto k1_) {
      constexpr int kk = decltype(k1_)::value;
      v[kk] = sm[kk * B * T + tid];
    });
    FftReg<A, 1>::run(v);            // inverse over k1 -> index n1
    static_for<0, A>([&](auto n1_) {
      constexpr int n1 = decltype(n1_)::value;
      const int n = n1 * B + n2;
      if (n < p.nz) out[(long long)n * p.plane + xa] = v[n1];
    });
  }
}

// =========================================================================================
// fused row pass along x.
//
// Half-row packing: the real row psi[0..Nx) is split at hx = ceil(Nx/2) and
// carried as ONE complex row c[n] = psi[n] + i*psi[n+hx], n < hx, zero-padded to M >= hx + 2*rx.
// The kernels are real, so a complex convolution convolves the two halves independently; the
// full linear convolution of each half (support [-rx, hx+rx)) is recovered without aliasing and
// the two are overlap-added:  out[x] = Re c[x]   (+ Im c[M + x - hx]  for x >= hx - rx)   x <  hx
//                             out[x] = Im c[x-hx] (+ Re c[x]           for x <  hx + rx)   x >= hx
// =========================================================================================
template <int A, int B, int MODE>
__global__ void __launch_bounds__(PassCfg<A, B>::MAX_THREADS)
xrow_kernel(const XArgs p) {
  using Cfg = PassCfg<A, B>;
  constexpr int M = Cfg::M, AP = Cfg::AP, BP = Cfg::BP, RS = Cfg::ROW_F2;
  extern __shared__ float2 sm[];
  const int R = p.rows_per_cta;
  float* halo_re = reinterpret_cast<float*>(sm + (size_t)R * RS);
  float* halo_im = halo_re + R * p.rx;
  const int tid = threadIdx.x;
  const long long row0 = (long long)blockIdx.x * R;

  // thread roles
  const int rowA = tid / A, k1 = tid - rowA * A;      // owns k1 (G1, F2)
  const int rowB = tid / B, n2 = tid - rowB * B;      // owns n2 (G2, pointwise, F1)
  const long long growA = row0 + rowA, growB = row0 + rowB;
  const bool actA = tid < R * A && growA < p.nrows;
  const bool actB = tid < R * B && growB < p.nrows;
  const long long offA = actA ? ((growA / p.ny_rows) * p.plane_pitch + (growA % p.ny_rows) * (long long)M) : 0;

  float2 c[A];   // the row segment owned by (rowB, n2): c[n1] <-> n = n1*B + n2

  if constexpr (MODE != X_LOAD) {
    // ---- G1: inverse B-point transforms over k2 --------------------------------------------
    if (actA) {
      float2 u[B];
      const float2* src = p.in + offA + k1;
      static_for<0, B>([&](auto k2_) {
        constexpr int k2 = decltype(k2_)::value;
        u[k2] = src[A * k2];
      });
      FftReg<B, 1>::run(u);
      static_for<0, B>([&](auto n2_) {
        constexpr int m = decltype(n2_)::value;
        if constexpr (m > 0) u[m] = cmul_conj(u[m], ld_tw(p.tw, m * k1));   // conj(W)^{n2 k1}
        sm[rowA * RS + m * AP + k1] = u[m];
      });
    }
    __syncthreads();
    // ---- G2: inverse A-point transforms over k1 -> c[n1] -------------------------------------
    if (actB) {
      static_for<0, A>([&](auto k1_) {
        constexpr int kk = decltype(k1_)::value;
        c[kk] = sm[rowB * RS + n2 * AP + kk];
      });
      FftReg<A, 1>::run(c);
      // publish the overlap regions: Re c[hx .. hx+rx) and Im c[M-rx .. M)
      static_for<0, A>([&](auto n1_) {
        constexpr int n1 = decltype(n1_)::value;
        const int n = n1 * B + n2;
        if (n >= p.hx && n < p.hx + p.rx) halo_re[rowB * p.rx + (n - p.hx)] = c[n1].x;
        if (n >= M - p.rx) halo_im[rowB * p.rx + (n - (M - p.rx))] = c[n1].y;
      });
    }
    __syncthreads();
  }

  // ---- pointwise stage on the real row -------------------------------------------------------
  float flux = 0.f, l1 = 0.f;
  bool do_forward = true;
  if constexpr (MODE == X_ACCUM) do_forward = (p.acc_mode == ACC_LAST || p.acc_mode == ACC_ONLY);
  if (actB) {
    const long long rbase = growB * (long long)p.nx;
    if constexpr (MODE == X_LOAD) {
      if (p.complex_in) {
        const long long off = (growB / p.ny_rows) * p.plane_pitch + (growB % p.ny_rows) * (long long)M;
        static_for<0, A>([&](auto n1_) {
          constexpr int n1 = decltype(n1_)::value;
          c[n1] = p.in[off + n1 * B + n2];
        });
      } else {
        static_for<0, A>([&](auto n1_) {
          constexpr int n1 = decltype(n1_)::value;
          const int n = n1 * B + n2;
          float2 z = make_float2(0.f, 0.f);
          if (n < p.hx) {
            z.x = p.phi[rbase + n];
            if (n + p.hx < p.nx) z.y = p.phi[rbase + n + p.hx];
          }
          c[n1] = z;
        });
      }
    } else {
      static_for<0, A>([&](auto n1_) {
        constexpr int n1 = decltype(n1_)::value;
        const int n = n1 * B + n2;
        float2 z = make_float2(0.f, 0.f);
        if (n < p.hx) {
          float vt = c[n1].x;                     // result at x = n
          float vb = c[n1].y;                     // result at x = n + hx
          if (n >= p.hx - p.rx) vt += halo_im[rowB * p.rx + (n - (p.hx - p.rx))];
          if (n < p.rx) vb += halo_re[rowB * p.rx + n];
          const bool has_b = n + p.hx < p.nx;
          const long long it = rbase + n, ib = rbase + n + p.hx;
          if constexpr (MODE == X_QUOT) {
            z.x = p.phi[it] / fmaxf(vt, p.eps);
            if (has_b) z.y = p.phi[ib] / fmaxf(vb, p.eps);
          } else if constexpr (MODE == X_UPDATE) {
            const float o = p.psi[it];
            const float nw = fmaxf(tikhonov_update(o * vt, p.tikhonov), p.psi_floor);
            p.psi[it] = nw;
            flux += nw;
            l1 += fabsf(nw - o);
            z.x = nw;
            if (has_b) {
              const float o2 = p.psi[ib];
              const float nw2 = fmaxf(tikhonov_update(o2 * vb, p.tikhonov), p.psi_floor);
              p.psi[ib] = nw2;
              flux += nw2;
              l1 += fabsf(nw2 - o2);
              z.y = nw2;
            }
          } else {   // X_ACCUM
            if (p.acc_mode == ACC_STORE) {
              p.acc[it] = vt;
              if (has_b) p.acc[ib] = vb;
            } else {
              float ft = p.literal_product ? vt : fmaxf(vt, 0.f);
              float fb = p.literal_product ? vb : fmaxf(vb, 0.f);
              if (p.root_each) {
                ft = __powf(ft, p.inv_nviews);
                fb = __powf(fb, p.inv_nviews);
              }
              if (p.acc_mode == ACC_MID || p.acc_mode == ACC_LAST) {
                ft *= p.acc[it];
                if (has_b) fb *= p.acc[ib];
              }
              if (p.acc_mode == ACC_FIRST || p.acc_mode == ACC_MID) {
                p.acc[it] = ft;
                if (has_b) p.acc[ib] = fb;
              } else {
                if (!p.literal_product && !p.root_each && p.inv_nviews != 1.f) {
                  ft = __powf(ft, p.inv_nviews);
                  fb = __powf(fb, p.inv_nviews);
                }
                const float o = p.psi[it];
                const float nw = fmaxf(tikhonov_update(o * ft, p.tikhonov), p.psi_floor);
                p.psi[it] = nw;
                flux += nw;
                l1 += fabsf(nw - o);
                z.x = nw;
                if (has_b) {
                  const float o2 = p.psi[ib];
                  const float nw2 = fmaxf(tikhonov_update(o2 * fb, p.tikhonov), p.psi_floor);
                  p.psi[ib] = nw2;
                  flux += nw2;
                  l1 += fabsf(nw2 - o2);
                  z.y = nw2;
                }
              }
            }
          }
        }
        c[n1] = z;
      });
    }
  }

  // ---- per-CTA statistics of the update: {sum psi_new, sum |psi_new - psi_old|} ----------------
  if constexpr (MODE == X_UPDATE || MODE == X_ACCUM) {
    if (MODE == X_UPDATE || do_forward) {
      double df = flux, dl = l1;
#pragma unroll
      for (int o = 16; o > 0; o >>= 1) {
        df += __shfl_down_sync(0xffffffffu, df, o);
        dl += __shfl_down_sync(0xffffffffu, dl, o);
      }
      __shared__ double red[2][32];
      const int warp = tid >> 5, lane = tid & 31;
      if (lane == 0) { red[0][warp] = df; red[1][warp] = dl; }
      __syncthreads();
      if (warp == 0) {
        const int nw = (blockDim.x + 31) >> 5;
        df = lane < nw ? red[0][lane] : 0.0;
        dl = lane < nw ? red[1][lane] : 0.0;
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) {
          df += __shfl_down_sync(0xffffffffu, df, o);
          dl += __shfl_down_sync(0xffffffffu, dl, o);
        }
        if (lane == 0) {
          p.partials[2 * (size_t)blockIdx.x] = df;
          p.partials[2 * (size_t)blockIdx.x + 1] = dl;
        }
      }
    }
  }
  if (!do_forward) return;

  // ---- F1: forward A-point transforms over n1 ----------------------------------------------------
  if (actB) {
    FftReg<A, -1>::run(c);
    static_for<0, A>([&](auto k1_) {
      constexpr int kk = decltype(k1_)::value;
      if constexpr (kk > 0) c[kk] = cmul(c[kk], ld_tw(p.tw, n2 * kk));   // W^{n2 k1}
      sm[rowB * RS + kk * BP + n2] = c[kk];
    });
  }
  __syncthreads();
  // ---- F2: forward B-point transforms over n2, store k = k1 + A*k2 -------------------------------
  if (actA) {
    float2 u[B];
    static_for<0, B>([&](auto n2_) {
      constexpr int m = decltype(n2_)::value;
      u[m] = sm[rowA * RS + k1 * BP + m];
    });
    FftReg<B, -1>::run(u);
    float2* dst = p.out + offA + k1;
    static_for<0, B>([&](auto k2_) {
      constexpr int k2 = decltype(k2_)::value;
      dst[A * k2] = u[k2];
    });
  }
}

// =========================================================================================
// host-side launchers (one set per length, referenced by the LengthOps table)
// =========================================================================================
template <int A, int B>
struct Launch {
  using Cfg = PassCfg<A, B>;

  static size_t strided_smem(int T) { return (size_t)T * Cfg::M * sizeof(float2); }
  static size_t xrow_smem(int rows, int rx) {
    return (size_t)rows * Cfg::ROW_F2 * sizeof(float2) + (size_t)2 * rows * rx * sizeof(float);
  }

  static cudaError_t init() {
    const int big = 200 * 1024;
    cudaError_t e;
#define MVD_SET(k) \
  e = cudaFuncSetAttribute(k, cudaFuncAttributeMaxDynamicSharedMemorySize, big); \
  if (e != cudaSuccess) return e;
    MVD_SET((strided_fft_kernel<A, B, -1>));
    MVD_SET((strided_fft_kernel<A, B, 1>));
    MVD_SET((zconv_kernel<A, B>));
    MVD_SET((xrow_kernel<A, B, X_LOAD>));
    MVD_SET((xrow_kernel<A, B, X_QUOT>));
    MVD_SET((xrow_kernel<A, B, X_UPDATE>));
    MVD_SET((xrow_kernel<A, B, X_ACCUM>));
#undef MVD_SET
    return cudaSuccess;
  }

  static cudaError_t strided(const StridedArgs& a, int dir, cudaStream_t s) {
    const long long grid = a.n_outer * a.tiles_per_line;
    if (grid <= 0) return cudaSuccess;
    const size_t smem = strided_smem(a.T);
    if (dir < 0) strided_fft_kernel<A, B, -1><<<(unsigned)grid, a.nthreads, smem, s>>>(a);
    else strided_fft_kernel<A, B, 1><<<(unsigned)grid, a.nthreads, smem, s>>>(a);
    return cudaGetLastError();
  }

  static cudaError_t zconv(const ZconvArgs& a, cudaStream_t s) {
    const long long grid = (a.plane + a.T - 1) / a.T;
    if (grid <= 0) return cudaSuccess;
    zconv_kernel<A, B><<<(unsigned)grid, a.nthreads, strided_smem(a.T), s>>>(a);
    return cudaGetLastError();
  }

  static cudaError_t xrow(const XArgs& a, int mode, cudaStream_t s) {
    const long long grid = (a.nrows + a.rows_per_cta - 1) / a.rows_per_cta;
    if (grid <= 0) return cudaSuccess;
    const size_t smem = xrow_smem(a.rows_per_cta, a.rx);
    switch (mode) {
      case X_LOAD: xrow_kernel<A, B, X_LOAD><<<(unsigned)grid, a.nthreads, smem, s>>>(a); break;
      case X_QUOT: xrow_kernel<A, B, X_QUOT><<<(unsigned)grid, a.nthreads, smem, s>>>(a); break;
      case X_UPDATE: xrow_kernel<A, B, X_UPDATE><<<(unsigned)grid, a.nthreads, smem, s>>>(a); break;
      case X_ACCUM: xrow_kernel<A, B, X_ACCUM><<<(unsigned)grid, a.nthreads, smem, s>>>(a); break;
      default: return cudaErrorInvalidValue;
    }
    return cudaGetLastError();
  }

};

}  // namespace mvd
