// TMA-staged pencil passes (sm_100a): the same transforms as pass_kernels.cuh, with every HBM
// read staged through shared memory by the copy engine (async_copy.cuh), persistent CTAs and
// double-buffered tiles, so the next tile is in flight while the current one is transformed and
// no load ever sits in registers or L1.
//
//   xrow_tma_kernel   : x-inverse -> crop + quotient / OSEM update -> zero-pad + x-forward
//                       (S2 / S4 of DESIGN.md; eq. 13, eq. 109-112)
//   strided_tma_kernel: y pass, form F, pruned input (TMA zero fill) / cropped output
//   zconv_tma_kernel  : z-forward . spectrum . z-inverse, input tile and spectrum tile by TMA
#pragma once

#include <cstdio>

#include "async_copy.cuh"
#include "pass_kernels.cuh"

namespace mvd {

// shared-memory row strides of the x pass that keep the column accesses conflict-free
//   complex rows: stride == A or A+1 (mod 16) float2 and even (16-byte rows for the bulk copy)
//   real rows   : stride a multiple of 4 floats, as close to B (mod 32) as that allows
__host__ __device__ constexpr int xrow_cstride(int M, int A) {
  int s = M;
  while ((s & 1) || !((s % 16) == (A % 16) || (s % 16) == ((A + 1) % 16))) ++s;
  return s;
}
__host__ __device__ constexpr int xrow_rstride(int nx, int B) {
  int s = (nx + 3 + 3) / 4 * 4;   // + 3: a row whose global address is not 16-byte aligned is staged from the aligned
                                  // address below it and sits up to 3 floats into its shared-memory row
  const int want = (B % 32) / 4 * 4;
  while ((s % 32) != want) s += 4;
  return s;
}

// tile width (contiguous complex elements) of the TMA-staged y and z passes: compile-time, so every
// shared-memory offset of the in-place transforms is an immediate
constexpr int kTmaTile = kTmaTileHost;
// thread cap of the TMA-staged x pass, and the resident CTAs per SM its register budget is sized for:
// 4 (<= 102 registers) while the larger transform has <= 21 points, fewer for larger radices (no spills)
constexpr int kXrowTmaThreads = 160;
constexpr int xrow_min_blocks(int ab_max) { return ab_max <= 21 ? 4 : (ab_max <= 28 ? 3 : 2); }

// FLAGS (compile-time, so the common kernels carry no code for the rare paths): XF_TIK = Tikhonov-regularised
// update (mvd.h, R14); XF_LAST = the last view of a combined iteration (root, psi update, forward transform)
enum XFlags { XF_TIK = 1, XF_LAST = 2 };

template <int A, int B, int MODE, int FLAGS>
__global__ void __launch_bounds__(kXrowTmaThreads, xrow_min_blocks(PassCfg<A, B>::AB_MAX)) xrow_tma_kernel(const XArgs p) {
  using Cfg = PassCfg<A, B>;
  constexpr int M = Cfg::M, AP = Cfg::AP, BP = Cfg::BP;
  constexpr int CS = xrow_cstride(M, A);
  static_assert(MODE == X_QUOT || MODE == X_UPDATE || MODE == X_UPDATE_W || MODE == X_ACCUM, "TMA-staged x pass: no X_LOAD");
  // X_ACCUM (combined variants): running product of the f_v in acc; the last view takes the root,
  // updates psi and transforms the new estimate.  acc is the staged real row (read for MID / LAST).
  static_assert(MODE == X_ACCUM || !(FLAGS & XF_LAST), "XF_LAST belongs to X_ACCUM");
  static_assert(MODE != X_QUOT && (MODE != X_ACCUM || (FLAGS & XF_LAST)) || !(FLAGS & XF_TIK), "XF_TIK belongs to the psi updates");
  constexpr bool tik = (FLAGS & XF_TIK) != 0;
  const bool acc_read = MODE == X_ACCUM && (p.acc_mode == ACC_MID || p.acc_mode == ACC_LAST);
  constexpr bool acc_last = MODE == X_ACCUM && (FLAGS & XF_LAST) != 0;   // acc_mode is ACC_LAST or ACC_ONLY
  constexpr bool do_forward = MODE != X_ACCUM || acc_last;
  const bool need_real = MODE != X_ACCUM || acc_read;          // real rows staged at all
  const bool real_bulk = need_real && p.bulk_real, real_plain = need_real && !p.bulk_real;
  // bulk_real == 2: rows of the real arrays start at addresses that are not multiples of 16 bytes (Nx not a multiple of
  // 4, or a misaligned base).  A row is then staged from the aligned address below it (the copy also brings the last
  // floats of the previous row and the first of the next) and read at an offset of `shift` floats; only the first
  // and the last row of the array, whose aligned windows could leave it, are loaded with plain loads.
  const bool shifted = real_bulk && p.bulk_real == 2;
  extern __shared__ __align__(128) unsigned char smem_raw[];
  const int R = p.rows_per_cta;
  const int RSTR = p.real_stride;
  const int RS = p.exch_stride, RSG = p.exch_stride_g, RSF = p.exch_stride_f;
  // layout: [R][CS] float2 complex rows | [R][RSTR] float real rows | exch [R][RS] float2 |
  //         tw2 [M] float2 | halos | barriers.  One stage: each staging buffer is refilled for the
  //         next tile as soon as its last reader of this tile has passed a barrier.
  float2* wst = reinterpret_cast<float2*>(smem_raw);
  float* rst = reinterpret_cast<float*>(wst + (size_t)R * CS);
  constexpr bool has_w = MODE == X_UPDATE_W;                      // section 12 weights
  float* wrst = rst + (size_t)R * RSTR;                           // [R][RSTR] weight rows (only with weights)
  float2* sm = reinterpret_cast<float2*>(rst + (size_t)(has_w ? 2 : 1) * R * RSTR);
  float2* tw2 = sm + (size_t)R * RS;                              // tw2[n2*AP + k1] = W_M^(n2 k1)
  float* halo_re = reinterpret_cast<float*>(tw2 + B * AP);
  float* halo_im = halo_re + R * p.rx;
  uint64_t* bars = reinterpret_cast<uint64_t*>(
      (reinterpret_cast<uintptr_t>(halo_im + R * p.rx) + 7) & ~uintptr_t(7));
  const int tid = threadIdx.x;
  const float* real_src = MODE == X_QUOT ? p.phi : (MODE == X_ACCUM ? p.acc : p.psi);
  const int ntiles = (int)((p.nrows + R - 1) / R);
  const int nrows_i = (int)p.nrows;
  const unsigned mis_r = shifted ? (unsigned)((reinterpret_cast<uintptr_t>(real_src) >> 2) & 3u) : 0u;
  const unsigned mis_w = (shifted && has_w) ? (unsigned)((reinterpret_cast<uintptr_t>(p.wts) >> 2) & 3u) : 0u;
  auto row_shift = [&](unsigned mis, int g) { return (int)((mis + (unsigned)g * (unsigned)p.nx) & 3u); };
  // a row is staged by a bulk copy only if its whole 16-byte-aligned window [g*nx - a, g*nx - a + roundup4(a + nx))
  // lies inside the array (for nx >= 3 that excludes at most the first and the last row; shorter rows: a few more)
  auto row_staged = [&](int a, int g) {
    const long long lo = (long long)g * p.nx - a, hi = lo + ((a + p.nx + 3) & ~3);
    return lo >= 0 && hi <= (long long)nrows_i * p.nx;
  };

  if (tid == 0) {
    mbar_init(&bars[0], 1);   // complex rows landed
    mbar_init(&bars[1], 1);   // real rows landed
    mbar_fence_init();
  }
  for (int j = tid; j < M; j += blockDim.x) tw2[(j / A) * AP + (j % A)] = __ldg(p.tw + (j / A) * (j % A));
  __syncthreads();

  // warp 0 issues the copies of a tile: lane l stages rows l, l+32, ...
  auto issue_w = [&](int t) {
    const int tile = p.reverse ? ntiles - 1 - t : t;
    const int row0 = tile * R;
    const int rv = min(R, nrows_i - row0);
    if (tid == 0) mbar_expect_tx(&bars[0], (uint32_t)rv * (uint32_t)(M * sizeof(float2)));
    __syncwarp();
    for (int r = tid; r < rv; r += 32) {
      const unsigned g = (unsigned)(row0 + r);
      const unsigned zq = g / (unsigned)p.ny_rows, yr = g - zq * (unsigned)p.ny_rows;
      bulk_g2s(wst + (size_t)r * CS, p.in + (long long)zq * p.plane_pitch + (long long)yr * M, M * sizeof(float2), &bars[0]);
    }
  };
  auto issue_r = [&](int t) {
    const int tile = p.reverse ? ntiles - 1 - t : t;
    const int row0 = tile * R;
    const int rv = min(R, nrows_i - row0);
    if (!shifted) {
      if (tid == 0) mbar_expect_tx(&bars[1], (uint32_t)rv * (uint32_t)(p.nx * sizeof(float)) * (has_w ? 2u : 1u));
      __syncwarp();
      for (int r = tid; r < rv; r += 32) {
        bulk_g2s(rst + (size_t)r * RSTR, real_src + (long long)(row0 + r) * p.nx, p.nx * sizeof(float), &bars[1]);
        if (has_w) bulk_g2s(wrst + (size_t)r * RSTR, p.wts + (long long)(row0 + r) * p.nx, p.nx * sizeof(float), &bars[1]);
      }
      return;
    }
    uint32_t bytes = 0;
    for (int r = tid; r < rv; r += 32) {
      const int g = row0 + r, a = row_shift(mis_r, g);
      if (row_staged(a, g)) bytes += (uint32_t)(((a + p.nx) * 4 + 15) & ~15);
      if (has_w) {
        const int aw = row_shift(mis_w, g);
        if (row_staged(aw, g)) bytes += (uint32_t)(((aw + p.nx) * 4 + 15) & ~15);
      }
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) bytes += __shfl_xor_sync(0xffffffffu, bytes, o);
    if (tid == 0) mbar_expect_tx(&bars[1], bytes);
    __syncwarp();
    for (int r = tid; r < rv; r += 32) {
      const int g = row0 + r, a = row_shift(mis_r, g);
      if (row_staged(a, g))
        bulk_g2s(rst + (size_t)r * RSTR, real_src + (long long)g * p.nx - a, (uint32_t)(((a + p.nx) * 4 + 15) & ~15), &bars[1]);
      if (has_w) {
        const int aw = row_shift(mis_w, g);
        if (row_staged(aw, g))
          bulk_g2s(wrst + (size_t)r * RSTR, p.wts + (long long)g * p.nx - aw, (uint32_t)(((aw + p.nx) * 4 + 15) & ~15), &bars[1]);
      }
    }
  };

  const int rowA = tid / A, k1 = tid - rowA * A;
  const int rowB = tid / B, n2 = tid - rowB * B;
  double dflux = 0.0, dl1 = 0.0;

  if (tid < 32 && (int)blockIdx.x < ntiles) {
    issue_w((int)blockIdx.x);
    if (real_bulk) issue_r((int)blockIdx.x);
  }

  int it = 0;
  for (int tile = blockIdx.x; tile < ntiles; tile += gridDim.x, ++it) {
    const int row0 = (p.reverse ? ntiles - 1 - tile : tile) * R;
    const int growA = row0 + rowA, growB = row0 + rowB;
    const bool actA = tid < R * A && growA < nrows_i;
    const bool actB = tid < R * B && growB < nrows_i;
    const bool more = tile + (int)gridDim.x < ntiles;
    if (shifted) {      // the first / last row of the array: plain loads into the same shifted position
      const int rv = min(R, nrows_i - row0);
      for (int r = 0; r < rv; ++r) {
        const int g = row0 + r, a = row_shift(mis_r, g);
        if (!row_staged(a, g))
          for (int x = tid; x < p.nx; x += blockDim.x) rst[(size_t)r * RSTR + a + x] = real_src[(long long)g * p.nx + x];
        if (has_w) {
          const int aw = row_shift(mis_w, g);
          if (!row_staged(aw, g))
            for (int x = tid; x < p.nx; x += blockDim.x) wrst[(size_t)r * RSTR + aw + x] = p.wts[(long long)g * p.nx + x];
        }
      }
    }
    if (real_plain) {   // staging by bulk copies switched off (MVD_XBULK=0): plain loads of this tile's real rows
      const int rv = min(R, nrows_i - row0);
      for (int i = tid; i < rv * p.nx; i += blockDim.x) {
        const int r = i / p.nx, x = i - r * p.nx;
        rst[(size_t)r * RSTR + x] = real_src[(long long)(row0 + r) * p.nx + x];
        if (has_w) wrst[(size_t)r * RSTR + x] = p.wts[(long long)(row0 + r) * p.nx + x];
      }
    }
    mbar_wait(&bars[0], it & 1);

    float2 c[A];
    float flux = 0.f, l1 = 0.f;
    // ---- G1: inverse B-point transforms over k2 ------------------------------------------------
    if (actA) {
      float2 u[B];
      const float2* src = wst + (size_t)rowA * CS + k1;
      static_for<0, B>([&](auto k2_) {
        constexpr int k2 = decltype(k2_)::value;
        u[k2] = src[A * k2];
      });
      FftReg<B, 1>::run(u);
      static_for<0, B>([&](auto n2_) {
        constexpr int m = decltype(n2_)::value;
        if constexpr (m > 0) u[m] = cmul_conj(u[m], tw2[m * AP + k1]);
        sm[rowA * RSG + m * AP + k1] = u[m];
      });
    }
    __syncthreads();
    // every G1 read of the complex rows is done: stage the next tile's
    if (tid < 32 && more) issue_w(tile + (int)gridDim.x);
    // ---- G2: inverse A-point transforms over k1 -> c[n1], n = n1*B + n2 ------------------------
    if (actB) {
      static_for<0, A>([&](auto k1_) {
        constexpr int kk = decltype(k1_)::value;
        c[kk] = sm[rowB * RSG + n2 * AP + kk];
      });
      FftReg<A, 1>::run(c);
      static_for<0, A>([&](auto n1_) {
        constexpr int n1 = decltype(n1_)::value;
        // warp-uniform: does [n1*B, n1*B + B) touch an overlap region at all?
        if (n1 * B + B > p.hx && (n1 * B < p.hx + p.rx || n1 * B + B > M - p.rx)) {
          const int n = n1 * B + n2;
          if (n >= p.hx && n < p.hx + p.rx) halo_re[rowB * p.rx + (n - p.hx)] = c[n1].x;
          if (n >= M - p.rx) halo_im[rowB * p.rx + (n - (M - p.rx))] = c[n1].y;
        }
      });
    }
    __syncthreads();
    if (real_bulk) mbar_wait(&bars[1], it & 1);
    // ---- pointwise stage on the real row -------------------------------------------------------
    if (actB) {
      const long long rbase = (long long)growB * p.nx;
      const float* rrow = rst + (size_t)rowB * RSTR + (shifted ? row_shift(mis_r, growB) : 0);
      const float* wrow = wrst + (size_t)rowB * RSTR + (shifted ? row_shift(mis_w, growB) : 0);
      float* prow = p.psi + rbase;
      float* arow = p.acc + rbase;
      const int lo_int = p.rx, hi_int = min(p.hx - p.rx, p.nx - p.hx);   // interior: no overlap, both halves live
      // one voxel: x = row position, v = convolution result there; returns the value carried into
      // the forward transform (quotient / new estimate / nothing)
      auto voxel = [&](int x, float v) -> float {
        if constexpr (MODE == X_QUOT) {
          return __fdividef(rrow[x], fmaxf(v, p.eps));                    // S2, R4
        } else if constexpr (MODE == X_UPDATE || MODE == X_UPDATE_W) {
          const float o = rrow[x];
          if (has_w) v = fmaf(wrow[x], v - 1.f, 1.f);                     // section 12: fraction w of the RL step
          float u = o * v;
          if constexpr (tik) u = tikhonov_value(u, p.tikhonov);           // R14
          const float nw = fmaxf(u, p.psi_floor);                         // eq. 109-112, R4
          prow[x] = nw;
          flux += nw;
          l1 += fabsf(nw - o);
          return nw;
        } else {                                                          // X_ACCUM (eq. 70 / 104, R1)
          float f = p.literal_product ? v : fmaxf(v, 0.f);
          if (p.root_each) f = __powf(f, p.inv_nviews);                   // many views: root first, product after
          if (acc_read) f *= rrow[x];
          if constexpr (!acc_last) {
            arow[x] = f;
            return 0.f;
          }
          // eq. 44: the |V|-th root as exp2(log2(f) / V) on the special-function unit (f is a product of V
          // ratios near 1: the hardware log2 / exp2 keep the relative error at a few 1e-7)
          if (!p.literal_product && !p.root_each && p.inv_nviews != 1.f) f = __powf(f, p.inv_nviews);
          const float o = prow[x];
          float u = o * f;
          if constexpr (tik) u = tikhonov_value(u, p.tikhonov);           // R14
          const float nw = fmaxf(u, p.psi_floor);
          prow[x] = nw;
          flux += nw;
          l1 += fabsf(nw - o);
          return nw;
        }
      };
      static_for<0, A>([&](auto n1_) {
        constexpr int n1 = decltype(n1_)::value;
        const int n = n1 * B + n2;
        float2 z = make_float2(0.f, 0.f);
        if (n1 * B >= lo_int && n1 * B + B <= hi_int) {     // warp-uniform fast path
          z.x = voxel(n, c[n1].x);
          z.y = voxel(n + p.hx, c[n1].y);
        } else if (n < p.hx) {
          float vt = c[n1].x, vb = c[n1].y;
          if (n >= p.hx - p.rx) vt += halo_im[rowB * p.rx + (n - (p.hx - p.rx))];
          if (n < p.rx) vb += halo_re[rowB * p.rx + n];
          z.x = voxel(n, vt);
          if (n + p.hx < p.nx) z.y = voxel(n + p.hx, vb);
        }
        c[n1] = z;
      });
      // ---- F1: forward A-point transforms over n1 ----------------------------------------------
      if (do_forward) {
        FftReg<A, -1>::run(c);
        static_for<0, A>([&](auto k1_) {
          constexpr int kk = decltype(k1_)::value;
          if constexpr (kk > 0) c[kk] = cmul(c[kk], tw2[n2 * AP + kk]);
          sm[rowB * RSF + kk * BP + n2] = c[kk];
        });
      }
    }
    // rows that could not be staged were written into rst / wrst by ordinary stores; the copy engine (async proxy)
    // refills those slots next
    if (shifted) fence_proxy_async();
    __syncthreads();
    // every read of the real rows is done: stage the next tile's
    if (tid < 32 && more && real_bulk) issue_r(tile + (int)gridDim.x);
    // ---- F2: forward B-point transforms over n2, store k = k1 + A*k2 ---------------------------
    if (actA && do_forward) {
      float2 u[B];
      static_for<0, B>([&](auto n2_) {
        constexpr int m = decltype(n2_)::value;
        u[m] = sm[rowA * RSF + k1 * BP + m];
      });
      FftReg<B, -1>::run(u);
      const unsigned zq = (unsigned)growA / (unsigned)p.ny_rows, yr = (unsigned)growA - zq * (unsigned)p.ny_rows;
      float2* dst = p.out + (long long)zq * p.plane_pitch + (long long)yr * M + k1;
      static_for<0, B>([&](auto k2_) {
        constexpr int k2 = decltype(k2_)::value;
        dst[A * k2] = u[k2];
      });
    }
    dflux += (double)flux;
    dl1 += (double)l1;
    __syncthreads();   // the exchange buffer is rewritten by the next tile's G1
  }

  // ---- per-CTA statistics of the update: {sum psi_new, sum |psi_new - psi_old|} ----------------
  if (MODE == X_UPDATE || MODE == X_UPDATE_W || acc_last) {
    double df = dflux, dl = dl1;
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

// =========================================================================================
// strided pencil FFT (form F), TMA-staged.  Tile = T contiguous complex elements x the whole
// pencil, laid out [n][T] in shared memory by the tensor copy (rows >= n_in arrive as zeros:
// the zero padding is never stored in HBM).  Both register transforms run in place on the tile:
//   stage 1: item (n2, x) owns rows n1*B + n2 -> A-point FFT, twiddle -> rows k1*B + n2
//   stage 2: item (k1, x) owns rows k1*B + n2 -> B-point FFT -> global rows k1 + A*k2 (< n_out)
// =========================================================================================
// PAIR: a thread transforms two adjacent columns at once, so every shared-memory and global access is 128 bits wide
// (half the load / store / address instructions, half the threads, twice the independent work per thread).
template <int A, int B>
constexpr int strided_tma_pair_threads() {
  constexpr int items = strided_tma_tile(A * B) / 2 * PassCfg<A, B>::AB_MAX;
  constexpr int t = (items + 31) / 32 * 32;
  return t < 512 ? t : 512;
}
template <int A, int B, int DIR, bool PAIR>
__global__ void __launch_bounds__(PAIR ? strided_tma_pair_threads<A, B>() : PassCfg<A, B>::MAX_THREADS)
strided_tma_kernel(const __grid_constant__ StridedTmaArgs p) {
  constexpr int M = A * B;
  extern __shared__ __align__(128) unsigned char smem_raw[];
  constexpr int T = strided_tma_tile(M);
  const int NR = p.boxr * p.nbox;
  const int nst = p.nst;                                          // tile stages: 1 or 2
  float2* buf = reinterpret_cast<float2*>(smem_raw);            // [nst][NR][T]
  constexpr int AP = PassCfg<A, B>::AP;
  float2* tws = buf + (size_t)nst * NR * T;                        // [B][AP]
  uint64_t* bars = reinterpret_cast<uint64_t*>(tws + B * AP);
  const int tid = threadIdx.x;
  const int ntiles = p.n_xt * p.n_outer;

  if (tid == 0) {
    mbar_init(&bars[0], 1);
    mbar_init(&bars[1], 1);
    mbar_fence_init();
  }
  for (int j = tid; j < M; j += blockDim.x) tws[(j / A) * AP + (j % A)] = __ldg(p.tw + (j / A) * (j % A));   // tws[n2*AP + k1] = W^(n2 k1)
  __syncthreads();

  auto issue = [&](int t, int s) {
    const int tile = p.reverse ? ntiles - 1 - t : t;
    const int outer = tile / p.n_xt;
    const int x0 = (p.xt0 + (tile - outer * p.n_xt)) * T;
    mbar_expect_tx(&bars[s], (uint32_t)(NR * T * sizeof(float2)));
    for (int b = 0; b < p.nbox; ++b)
      tma_load_3d(buf + ((size_t)s * NR + b * p.boxr) * T, &p.in_map, x0, b * p.boxr, outer, &bars[s]);
  };

  if (tid == 0 && (int)blockIdx.x < ntiles) issue((int)blockIdx.x, 0);

  int it = 0;
  for (int tile = blockIdx.x; tile < ntiles; tile += gridDim.x, ++it) {
    const int s = nst == 2 ? (it & 1) : 0;
    float2* sm = buf + (size_t)s * NR * T;
    const bool more = tile + (int)gridDim.x < ntiles;
    // two stages: the other stage was last read before the final barrier of the previous tile
    if (tid == 0 && more && nst == 2) issue(tile + (int)gridDim.x, s ^ 1);
    const int rtile = p.reverse ? ntiles - 1 - tile : tile;
    const int outer = rtile / p.n_xt;
    const int x0 = (p.xt0 + (rtile - outer * p.n_xt)) * T;
    const int xvalid = min(T, p.line_len - x0);
    mbar_wait(&bars[s], nst == 2 ? ((it >> 1) & 1) : (it & 1));

    if constexpr (PAIR) {
      constexpr int H = T / 2;                     // float4 (two complex) per tile row
      float4* sm4 = reinterpret_cast<float4*>(sm);
      for (int i = tid; i < H * B; i += blockDim.x) {
        const int n2 = i / H;
        float2 v0[A], v1[A];
        static_for<0, A>([&](auto n1_) {
          constexpr int n1 = decltype(n1_)::value;
          const float4 q = sm4[n1 * B * H + i];
          v0[n1] = make_float2(q.x, q.y);
          v1[n1] = make_float2(q.z, q.w);
        });
        FftReg<A, DIR>::run(v0);
        FftReg<A, DIR>::run(v1);
        static_for<0, A>([&](auto k1_) {
          constexpr int k1 = decltype(k1_)::value;
          if constexpr (k1 > 0) {
            const float2 w = tws[n2 * AP + k1];
            v0[k1] = DIR < 0 ? cmul(v0[k1], w) : cmul_conj(v0[k1], w);
            v1[k1] = DIR < 0 ? cmul(v1[k1], w) : cmul_conj(v1[k1], w);
          }
          sm4[k1 * B * H + i] = make_float4(v0[k1].x, v0[k1].y, v1[k1].x, v1[k1].y);
        });
      }
    } else {
    for (int i = tid; i < T * B; i += blockDim.x) {
        const int n2 = i / T;
        float2 v[A];
        static_for<0, A>([&](auto n1_) {
          constexpr int n1 = decltype(n1_)::value;
          v[n1] = sm[n1 * B * T + i];
        });
        FftReg<A, DIR>::run(v);
        static_for<0, A>([&](auto k1_) {
          constexpr int k1 = decltype(k1_)::value;
          if constexpr (k1 > 0) {
            const float2 w = tws[n2 * AP + k1];
            v[k1] = DIR < 0 ? cmul(v[k1], w) : cmul_conj(v[k1], w);
          }
          sm[k1 * B * T + i] = v[k1];
        });
      }
    }
    __syncthreads();
    if constexpr (PAIR) {
      constexpr int H = T / 2;
      const float4* sm4 = reinterpret_cast<const float4*>(sm);
      float2* out = p.out + (long long)outer * p.out_outer_stride + x0;
      for (int j = tid; j < H * A; j += blockDim.x) {
        const int k1 = j / H;
        const int xp = j - k1 * H;
        float2 u0[B], u1[B];
        static_for<0, B>([&](auto n2_) {
          constexpr int n2 = decltype(n2_)::value;
          const float4 q = sm4[(k1 * B + n2) * H + xp];
          u0[n2] = make_float2(q.x, q.y);
          u1[n2] = make_float2(q.z, q.w);
        });
        FftReg<B, DIR>::run(u0);
        FftReg<B, DIR>::run(u1);
        if (2 * xp < xvalid) {                     // line_len and T are even: a pair is valid or not as a whole
          float4* o = reinterpret_cast<float4*>(out + (long long)k1 * p.out_pstride + 2 * xp);
          static_for<0, B>([&](auto k2_) {
            constexpr int k2 = decltype(k2_)::value;
            if (k1 + A * k2 < p.n_out)
              *reinterpret_cast<float4*>(reinterpret_cast<float2*>(o) + (long long)(A * k2) * p.out_pstride) =
                  make_float4(u0[k2].x, u0[k2].y, u1[k2].x, u1[k2].y);
          });
        }
      }
      fence_proxy_async();
      __syncthreads();
      if (tid == 0 && more && nst == 1) issue(tile + (int)gridDim.x, 0);
    } else {
      float2* out = p.out + (long long)outer * p.out_outer_stride + x0;
      for (int j = tid; j < T * A; j += blockDim.x) {
        const int k1 = j / T;
        const int x = j - k1 * T;
        float2 u[B];
        static_for<0, B>([&](auto n2_) {
          constexpr int n2 = decltype(n2_)::value;
          u[n2] = sm[(k1 * B + n2) * T + x];
        });
        FftReg<B, DIR>::run(u);
        if (x < xvalid) {
          float2* o = out + (long long)k1 * p.out_pstride + x;
          static_for<0, B>([&](auto k2_) {
            constexpr int k2 = decltype(k2_)::value;
            if (k1 + A * k2 < p.n_out) o[(long long)(A * k2) * p.out_pstride] = u[k2];
          });
        }
      }
      // the tile was transformed in place by ordinary stores; the copy engine (async proxy) refills it
      fence_proxy_async();
      __syncthreads();   // every read of this tile is done
      if (tid == 0 && more && nst == 1) issue(tile + (int)gridDim.x, 0);   // one stage: refill it now
    }
  }
}

// =========================================================================================
// fused z pass, TMA-staged: crop(IFFT_z( FFT_z(zero-padded pencil) * spectrum )).
// Tile = T contiguous x of one row y, all z: the input tile [z][T] (planes >= nz arrive as zeros)
// and the spectrum tile [k][T] are both staged by tensor copies; the four register transforms
// run in place on the input tile.
// =========================================================================================
template <int A, int B, int TX>
__global__ void __launch_bounds__(PassCfg<A, B>::MAX_THREADS)
zconv_tma_kernel(const __grid_constant__ ZconvTmaArgs p) {
  constexpr int M = A * B;
  extern __shared__ __align__(128) unsigned char smem_raw[];
  // 16 columns per tile: TX = 8 contiguous x of two consecutive rows y, or TX = 16 x of one row (128-byte pieces:
  // better for long pencils, where one CTA per SM is all that fits)
  constexpr int T = 2 * kTmaTile, TY = T / TX;
  static_assert(TX == 8 || TX == 16, "z tile: 8 x 2 or 16 x 1");
  const int NR = p.boxr * p.nbox;
  const int nst = p.nst_in;                                       // input stages: 1 or 2
  float2* buf = reinterpret_cast<float2*>(smem_raw);            // [nst][NR][T] input tiles
  float2* sbuf = buf + (size_t)nst * NR * T;                     // [NR][T] spectrum tile (one stage)
  constexpr int AP = PassCfg<A, B>::AP;
  float2* tws = sbuf + (size_t)NR * T;                           // [B][AP]
  uint64_t* bars = reinterpret_cast<uint64_t*>(tws + B * AP);   // [0..1] input stages, [2] spectrum
  const int tid = threadIdx.x;
  const int ny2 = (p.my + TY - 1) / TY;                           // row groups
  const int ntiles = p.n_xt * ny2;

  if (tid == 0) {
    mbar_init(&bars[0], 1);
    mbar_init(&bars[1], 1);
    mbar_init(&bars[2], 1);
    mbar_fence_init();
  }
  for (int j = tid; j < M; j += blockDim.x) tws[(j / A) * AP + (j % A)] = __ldg(p.tw + (j / A) * (j % A));   // tws[n2*AP + k1] = W^(n2 k1)
  __syncthreads();

  auto issue_in = [&](int tile, int s) {
    const int yp = tile / p.n_xt;
    const int y = TY * yp;
    const int x0 = (p.xt0 + (tile - yp * p.n_xt)) * TX;
    mbar_expect_tx(&bars[s], (uint32_t)(NR * T * sizeof(float2)));
    for (int b = 0; b < p.nbox; ++b)
      tma_load_3d(buf + ((size_t)s * NR + b * p.boxr) * T, &p.in_map, x0, y, b * p.boxr, &bars[s]);
  };
  auto issue_spec = [&](int tile) {
    const int yp = tile / p.n_xt;
    const int y = TY * yp;
    const int x0 = (p.xt0 + (tile - yp * p.n_xt)) * TX;
    mbar_expect_tx(&bars[2], (uint32_t)(NR * T * sizeof(float2)));
    for (int b = 0; b < p.nbox; ++b)
      tma_load_3d(sbuf + (size_t)(b * p.boxr) * T, &p.spec_map, x0, y, b * p.boxr, &bars[2]);
  };

  if (tid == 0 && (int)blockIdx.x < ntiles) {
    issue_in((int)blockIdx.x, 0);
    issue_spec((int)blockIdx.x);
  }

  int it = 0;
  for (int tile = blockIdx.x; tile < ntiles; tile += gridDim.x, ++it) {
    const int s = nst == 2 ? (it & 1) : 0;
    float2* sm = buf + (size_t)s * NR * T;
    const float2* sp = sbuf;
    const bool more = tile + (int)gridDim.x < ntiles;
    // two input stages: the other stage was last read before the final barrier of the previous tile
    if (tid == 0 && more && nst == 2) issue_in(tile + (int)gridDim.x, s ^ 1);
    const int yp = tile / p.n_xt;
    const int y = TY * yp;
    const int x0 = (p.xt0 + (tile - yp * p.n_xt)) * TX;
    const int xvalid = min(TX, p.mx - x0);
    const int yvalid = min(TY, p.my - y);
    mbar_wait(&bars[s], nst == 2 ? ((it >> 1) & 1) : (it & 1));

    // F1: item (n2, x), forward A-point transforms over n1
    for (int i = tid; i < T * B; i += blockDim.x) {
      const int n2 = i / T;
      float2 v[A];
      static_for<0, A>([&](auto n1_) {
        constexpr int n1 = decltype(n1_)::value;
        v[n1] = sm[n1 * B * T + i];
      });
      FftReg<A, -1>::run(v);
      static_for<0, A>([&](auto k1_) {
        constexpr int k1 = decltype(k1_)::value;
        if constexpr (k1 > 0) v[k1] = cmul(v[k1], tws[n2 * AP + k1]);
        sm[k1 * B * T + i] = v[k1];
      });
    }
    __syncthreads();
    mbar_wait(&bars[2], it & 1);
    // F2 . spectrum . G1: item (k1, x)
    for (int j = tid; j < T * A; j += blockDim.x) {
      const int k1 = j / T;
      const int x = j - k1 * T;
      float2 u[B];
      static_for<0, B>([&](auto n2_) {
        constexpr int m = decltype(n2_)::value;
        u[m] = sm[(k1 * B + m) * T + x];
      });
      FftReg<B, -1>::run(u);
      static_for<0, B>([&](auto k2_) {
        constexpr int k2 = decltype(k2_)::value;
        u[k2] = cmul(u[k2], sp[(k1 + A * k2) * T + x]);
      });
      FftReg<B, 1>::run(u);
      static_for<0, B>([&](auto n2_) {
        constexpr int m = decltype(n2_)::value;
        if constexpr (m > 0) u[m] = cmul_conj(u[m], tws[m * AP + k1]);
        sm[(k1 * B + m) * T + x] = u[m];
      });
    }
    __syncthreads();
    // every read of the spectrum tile is done: stage the next tile's
    if (tid == 0 && more) issue_spec(tile + (int)gridDim.x);
    // G2: item (n2, x), inverse A-point transforms over k1, store planes n1*B + n2 < nz
    float2* out = p.out + (long long)y * p.mx + x0;
    for (int i = tid; i < T * B; i += blockDim.x) {
      const int n2 = i / T;
      const int col = i - n2 * T;
      const int yy = col / TX, x = col - yy * TX;
      float2 v[A];
      static_for<0, A>([&](auto k1_) {
        constexpr int kk = decltype(k1_)::value;
        v[kk] = sm[kk * B * T + i];
      });
      FftReg<A, 1>::run(v);
      if (x < xvalid && yy < yvalid) {
        float2* o = out + (long long)n2 * p.plane + yy * p.mx + x;
        static_for<0, A>([&](auto n1_) {
          constexpr int n1 = decltype(n1_)::value;
          if (n1 * B + n2 < p.nz) o[(long long)(n1 * B) * p.plane] = v[n1];
        });
      }
    }
    fence_proxy_async();   // in-place stores to the tile before the copy engine refills it
    __syncthreads();
    if (tid == 0 && more && nst == 1) issue_in(tile + (int)gridDim.x, 0);   // one input stage: refill now
  }
}

// host-side launchers of the TMA-staged passes
template <int A, int B>
struct LaunchTma {
  using Cfg = PassCfg<A, B>;

  // exchange rows are at most ROW_F2 + 16 float2 (the planner searches the conflict-free stride there)
  static size_t xrow_smem(int rows, int rx, int nx, int weighted) {
    return (size_t)rows * xrow_cstride(Cfg::M, A) * sizeof(float2) +
           (size_t)(weighted ? 2 : 1) * rows * xrow_rstride(nx, B) * sizeof(float) + (size_t)rows * (Cfg::ROW_F2 + 16) * sizeof(float2) +
           (size_t)B * Cfg::AP * sizeof(float2) + (size_t)2 * rows * rx * sizeof(float) + 32;
  }

  static cudaError_t init() {
    cudaError_t e;
#define MVD_SET(k) \
  e = cudaFuncSetAttribute(k, cudaFuncAttributeMaxDynamicSharedMemorySize, 220 * 1024); \
  if (e != cudaSuccess) { fprintf(stderr, "smem attr failed %d x %d: %s\n", A, B, #k); return e; } \
  e = cudaFuncSetAttribute(k, cudaFuncAttributePreferredSharedMemoryCarveout, cudaSharedmemCarveoutMaxShared); \
  if (e != cudaSuccess) { fprintf(stderr, "carveout attr failed %d x %d: %s\n", A, B, #k); return e; }
    MVD_SET((xrow_tma_kernel<A, B, X_QUOT, 0>));
    MVD_SET((xrow_tma_kernel<A, B, X_UPDATE, 0>));
    MVD_SET((xrow_tma_kernel<A, B, X_UPDATE, XF_TIK>));
    MVD_SET((xrow_tma_kernel<A, B, X_UPDATE_W, 0>));
    MVD_SET((xrow_tma_kernel<A, B, X_UPDATE_W, XF_TIK>));
    MVD_SET((xrow_tma_kernel<A, B, X_ACCUM, 0>));
    MVD_SET((xrow_tma_kernel<A, B, X_ACCUM, XF_LAST>));
    MVD_SET((xrow_tma_kernel<A, B, X_ACCUM, XF_LAST | XF_TIK>));
    MVD_SET((strided_tma_kernel<A, B, -1, false>));
    MVD_SET((strided_tma_kernel<A, B, 1, false>));
    MVD_SET((strided_tma_kernel<A, B, -1, true>));
    MVD_SET((strided_tma_kernel<A, B, 1, true>));
    MVD_SET((zconv_tma_kernel<A, B, 8>));
    MVD_SET((zconv_tma_kernel<A, B, 16>));
#undef MVD_SET
    return cudaSuccess;
  }

  // the kernel of (mode, flags); flags: XF_TIK for a regularised update, XF_LAST for the last view of X_ACCUM
  using XKernel = void (*)(const XArgs);
  static XKernel xrow_kernel_of(int mode, int flags) {
    const bool t = (flags & XF_TIK) != 0;
    switch (mode) {
      case X_QUOT: return xrow_tma_kernel<A, B, X_QUOT, 0>;
      case X_UPDATE: return t ? xrow_tma_kernel<A, B, X_UPDATE, XF_TIK> : xrow_tma_kernel<A, B, X_UPDATE, 0>;
      case X_UPDATE_W: return t ? xrow_tma_kernel<A, B, X_UPDATE_W, XF_TIK> : xrow_tma_kernel<A, B, X_UPDATE_W, 0>;
      case X_ACCUM:
        if (!(flags & XF_LAST)) return xrow_tma_kernel<A, B, X_ACCUM, 0>;
        return t ? xrow_tma_kernel<A, B, X_ACCUM, XF_LAST | XF_TIK> : xrow_tma_kernel<A, B, X_ACCUM, XF_LAST>;
      default: return nullptr;
    }
  }
  static int xrow_flags(const XArgs& a, int mode) {
    const bool last = mode == X_ACCUM && (a.acc_mode == ACC_LAST || a.acc_mode == ACC_ONLY);
    const bool upd = mode == X_UPDATE || mode == X_UPDATE_W || last;
    return (last ? XF_LAST : 0) | ((upd && a.tikhonov > 0.f) ? XF_TIK : 0);
  }

  static int xrow_blocks_per_sm(int mode, int flags, int nthreads, size_t smem) {
    int n = 0;
    XKernel k = xrow_kernel_of(mode, flags);
    if (!k) return 0;
    return cudaOccupancyMaxActiveBlocksPerMultiprocessor(&n, k, nthreads, smem) == cudaSuccess ? n : 0;
  }

  static size_t strided_smem(int T, int boxr, int nbox, int nst) {
    return (size_t)nst * boxr * nbox * T * sizeof(float2) + (size_t)B * Cfg::AP * sizeof(float2) + 16;
  }
  static size_t zconv_smem(int T, int boxr, int nbox, int nst_in) {   // T = 8 x 2 rows = 16 columns
    return (size_t)(nst_in + 1) * boxr * nbox * 2 * T * sizeof(float2) + (size_t)B * Cfg::AP * sizeof(float2) + 32;
  }
  // the kernel a launch with these arguments selects, and its block size: the occupancy query and the launch agree
  using SKernel = void (*)(const StridedTmaArgs);
  static bool strided_pair(const StridedTmaArgs& a) { return a.pair && (a.line_len % 2 == 0) && (a.T % 2 == 0); }
  static SKernel strided_kernel_of(int dir, bool pair) {
    return dir < 0 ? (pair ? (SKernel)strided_tma_kernel<A, B, -1, true> : (SKernel)strided_tma_kernel<A, B, -1, false>)
                   : (pair ? (SKernel)strided_tma_kernel<A, B, 1, true> : (SKernel)strided_tma_kernel<A, B, 1, false>);
  }
  static int strided_threads(const StridedTmaArgs& a) { return strided_pair(a) ? strided_tma_pair_threads<A, B>() : a.nthreads; }
  static int strided_blocks_per_sm(const StridedTmaArgs& a, int dir) {
    int n = 0;
    const cudaError_t e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(
        &n, strided_kernel_of(dir, strided_pair(a)), strided_threads(a), strided_smem(a.T, a.boxr, a.nbox, a.nst));
    return e == cudaSuccess ? n : 0;
  }
  static int zconv_blocks_per_sm(const ZconvTmaArgs& a) {
    int n = 0;
    const size_t smem = zconv_smem(a.T, a.boxr, a.nbox, a.nst_in);
    const cudaError_t e = a.tx == 16 ? cudaOccupancyMaxActiveBlocksPerMultiprocessor(&n, zconv_tma_kernel<A, B, 16>, a.nthreads, smem)
                                     : cudaOccupancyMaxActiveBlocksPerMultiprocessor(&n, zconv_tma_kernel<A, B, 8>, a.nthreads, smem);
    return e == cudaSuccess ? n : 0;
  }
  static cudaError_t strided(const StridedTmaArgs& a, int dir, cudaStream_t s) {
    if (a.grid <= 0) return cudaSuccess;
    const size_t smem = strided_smem(a.T, a.boxr, a.nbox, a.nst);
    strided_kernel_of(dir, strided_pair(a))<<<a.grid, strided_threads(a), smem, s>>>(a);
    return cudaGetLastError();
  }
  static cudaError_t zconv(const ZconvTmaArgs& a, cudaStream_t s) {
    if (a.grid <= 0) return cudaSuccess;
    const size_t smem = zconv_smem(a.T, a.boxr, a.nbox, a.nst_in);
    if (a.tx == 16) zconv_tma_kernel<A, B, 16><<<a.grid, a.nthreads, smem, s>>>(a);
    else zconv_tma_kernel<A, B, 8><<<a.grid, a.nthreads, smem, s>>>(a);
    return cudaGetLastError();
  }

  static cudaError_t xrow(const XArgs& a, int mode, cudaStream_t s) {
    if (a.grid <= 0) return cudaSuccess;
    const size_t smem = xrow_smem(a.rows_per_cta, a.rx, a.nx, mode == X_UPDATE_W);
    XKernel k = xrow_kernel_of(mode, xrow_flags(a, mode));
    if (!k) return cudaErrorInvalidValue;
    k<<<a.grid, a.nthreads, smem, s>>>(a);
    return cudaGetLastError();
  }
  static int xrow_flags_of(const XArgs& a, int mode) { return xrow_flags(a, mode); }
};

}  // namespace mvd
