// Host-visible description of the per-length transform kernels (one LengthOps per supported
// pencil length M = A*B).  The kernels themselves are templates in pass_kernels.cuh and are
// instantiated once per length in inst.cu; mvd.cu only sees this table.
#pragma once

#include <cuda.h>
#include <cuda_runtime.h>

namespace mvd {

#ifndef MVD_TMA_TILE
#define MVD_TMA_TILE 8
#endif
constexpr int kTmaTileHost = MVD_TMA_TILE;   // == kTmaTile of pass_tma.cuh
// tile width of the TMA-staged y pass for pencil length M: 8 for short pencils (three CTAs per SM with two
// stages), 12 for 501-1140 points (measured: config 4 115 -> 111 us, config 5 1227 -> 1003 us), 8 beyond
// (two 12-wide stages no longer fit)
__host__ __device__ constexpr int strided_tma_tile(int M) { return (M > 500 && M <= 1140) ? 12 : kTmaTileHost; }

// ---- TMA-staged strided pass (pass_tma.cuh): persistent CTAs, tiles of T contiguous complex
//      elements x the whole pencil, loaded by tensor copies with zero fill beyond n_in ----------
struct StridedTmaArgs {
  CUtensorMap in_map;      // dims (x: line_len, pencil: n_in, outer: n_outer); box (T, boxr, 1)
  int pair;                // 1: two adjacent columns per thread, 128-bit accesses (needs even line_len and T)
  float2* out;
  const float2* tw;        // tw[j] = exp(-2*pi*i*j/M)
  int T, nthreads, grid;
  int boxr, nbox;          // the pencil is staged as nbox boxes of boxr rows (boxr*nbox >= M)
  int xt0, n_xt;           // x tiles [xt0, xt0 + n_xt) of every line are processed
  int line_len;            // contiguous extent (complex elements)
  int n_outer;
  long long out_outer_stride, out_pstride;
  int n_out;               // pencil outputs >= n_out are not stored
  int reverse;             // walk the tiles last to first (reads what the previous pass wrote last: L2 hits)
  int nst;                 // shared-memory stages of the tile: 1 or 2
};

// ---- TMA-staged fused z pass: input tile and spectrum tile by tensor copies --------------------
struct ZconvTmaArgs {
  CUtensorMap in_map;      // dims (x: Mx, y: My, z: nz);  box (T, 1, boxr)
  CUtensorMap spec_map;    // dims (x: Mx, y: My, z: Mz);  box (T, 1, boxr)
  float2* out;
  const float2* tw;
  int T, nthreads, grid;
  int boxr, nbox;
  int xt0, n_xt;           // x tiles [xt0, xt0 + n_xt) of every row
  int tx;                  // contiguous x per tile: 8 (two rows y per tile) or 16 (one row)
  int mx, my;              // row length and rows per plane
  long long plane;         // elements between z planes of `out`
  int nz;                  // planes written
  int nst_in;              // shared-memory stages of the input tile: 1 or 2
};

// ---- strided pencil FFT (y pass, plain z pass): pencils along a strided axis, tiles of T
//      contiguous complex elements across the unit-stride axis --------------------------------
struct StridedArgs {
  const float2* in;
  float2* out;
  const float2* tw;        // tw[j] = exp(-2*pi*i*j/M), j < M
  int T;                   // tile width (contiguous complex elements)
  int nthreads;
  int tiles_per_line;
  long long line_len;      // contiguous extent
  long long n_outer;       // number of lines
  long long in_outer_stride, out_outer_stride;
  long long in_pstride, out_pstride;   // element stride along the pencil
  int n_in;                // pencil inputs >= n_in are zero (never read)
  int n_out;               // pencil outputs >= n_out are not stored
  int reverse;             // walk the tiles last to first (reads what the previous pass wrote last: L2 hits)
  int nst;                 // shared-memory stages of the tile: 1 or 2
};

// ---- fused z pass: forward FFT along z, multiply by a kernel spectrum, inverse FFT ----------
struct ZconvArgs {
  const float2* in;
  float2* out;
  const float2* spec;      // [Mz][plane] complex, already scaled by 1/(Mx*My*Mz)
  const float2* tw;
  int T;
  int nthreads;
  long long plane;         // My*Mx2: element stride along z, and the contiguous extent
  int nz;                  // planes read and written (zero padding beyond is implicit)
};

// ---- fused row pass along x (see pass_kernels.cuh for the half-row packing) -------------------
enum XMode {
  X_LOAD = 0,              // (psi | complex rows) -> forward FFT
  X_QUOT = 1,              // inverse FFT -> q = phi / max(b, eps) -> forward FFT
  X_UPDATE = 2,            // inverse FFT -> psi <- max(psi*f, floor) -> forward FFT   (OSEM)
  X_ACCUM = 3,             // inverse FFT -> raw store | product accumulation | final combined update
  X_UPDATE_W = 4           // X_UPDATE with a per-view weight image (section 12): psi <- psi*(1 + w (f - 1))
};
enum AccMode { ACC_STORE = 0, ACC_FIRST = 1, ACC_MID = 2, ACC_LAST = 3, ACC_ONLY = 4 };

struct XArgs {
  const float2* in;        // work buffer rows (inverse input)
  float2* out;             // work buffer rows (forward output)
  const float2* tw;
  int rows_per_cta;
  int nthreads;
  long long nrows;         // rows processed = ny_rows * nz
  int ny_rows;             // rows used per plane
  long long plane_pitch;   // elements between planes of the work buffer (My*Mx2)
  int nx;                  // real row length Nx
  int hx;                  // (Nx+1)/2: element n of the half row carries x=n (re) and x=n+hx (im)
  int rx;                  // PSF half-size along x of this view
  const float* phi;        // X_QUOT: view; X_LOAD: psi (real input)
  const float* wts;        // X_UPDATE: weight image of this view (section 12) or NULL
  float* psi;              // X_UPDATE / ACC_LAST: estimate, updated in place
  float* acc;              // X_ACCUM: product accumulator / raw destination
  double* partials;        // per-CTA {flux, l1} (X_UPDATE, ACC_LAST)
  float eps, psi_floor, inv_nviews;
  float tikhonov;          // lambda of the Tikhonov-regularised update (0 = off), see mvd.h
  int acc_mode;            // AccMode
  int literal_product;
  int root_each;           // X_ACCUM: every factor takes the |V|-th root before entering the product (many views)
  int complex_in;          // X_LOAD: rows of `in` are complex and transformed in full
  // TMA-staged variant (pass_tma.cuh)
  int real_stride;         // floats between real rows in shared memory
  int bulk_real;           // real rows staged by bulk copies: 1 = rows 16-byte aligned, 2 = from the aligned address below each row; 0 = plain loads
  int grid;                // persistent CTAs
  int reverse;             // walk the tiles last to first
  int exch_stride;         // float2 per row of the exchange buffer (allocation)
  int exch_stride_g;       // row stride of the inverse-side exchange layout [n2*AP + k1]
  int exch_stride_f;       // row stride of the forward-side exchange layout [k1*BP + n2]
};

struct LengthOps {
  int M, A, B;
  int max_threads;         // launch bound of the kernels of this length
  cudaError_t (*init)();   // opt in to > 48 KB dynamic shared memory
  cudaError_t (*strided)(const StridedArgs&, int dir, cudaStream_t);
  cudaError_t (*zconv)(const ZconvArgs&, cudaStream_t);
  cudaError_t (*xrow)(const XArgs&, int mode, cudaStream_t);
  size_t (*strided_smem)(int T);
  size_t (*xrow_smem)(int rows, int rx);
  // TMA-staged passes (pass_tma.cuh)
  cudaError_t (*xrow_tma)(const XArgs&, int mode, cudaStream_t);
  size_t (*xrow_tma_smem)(int rows, int rx, int nx, int weighted);
  int (*xrow_tma_blocks_per_sm)(int mode, int flags, int nthreads, size_t smem);
  int (*xrow_tma_flags)(const XArgs&, int mode);   // compile-time variant of the kernel this launch selects
  cudaError_t (*strided_tma)(const StridedTmaArgs&, int dir, cudaStream_t);
  size_t (*strided_tma_smem)(int T, int boxr, int nbox, int nst);
  int (*strided_tma_blocks_per_sm)(const StridedTmaArgs&, int dir);   // resident CTAs per SM of the kernel this launch selects
  cudaError_t (*zconv_tma)(const ZconvTmaArgs&, cudaStream_t);
  size_t (*zconv_tma_smem)(int T, int boxr, int nbox, int nst_in);
  int (*zconv_tma_blocks_per_sm)(const ZconvTmaArgs&);
};

// table of all compiled lengths, ascending in M
const LengthOps* const* length_table(int* count);

}  // namespace mvd
