/* mvd.h -- C ABI of the B200 multi-view Richardson-Lucy deconvolution library (libmvd.so).
 *
 * What the library computes (citations are PAPER.md lines of arXiv 1308.0730, "Efficient
 * Bayesian-based Multi-View Deconvolution"; "R<n>" are the readings listed in DESIGN.md):
 *
 *   For every view v of V registered views phi_v with point spread function P_v
 *       b_v   = psi (*) P_v                               expected image     (eq. 1, eq. 13)
 *       q_v   = phi_v / max(b_v, eps)                     quotient           (L306; clamp R4)
 *       f_v   = q_v (*) K_v                               back-projection    (eq. 70, eq. 104)
 *   with (*) the linear convolution, zero extension outside the volume, output cropped to the
 *   volume (R3), and K_v the back-projector:
 *       PLAIN     K_v = P_v*  (mirrored PSF, L312)                            eq. 70
 *       COMPOUND  K_v = P_v* . prod_{w!=v} crop(P_v* (*) P_w (*) P_w*)        eq. 105
 *       OPT1      K_v = P_v* . prod_{w!=v} crop(P_v* (*) P_w)                 eq. 107
 *       OPT2      K_v = (P_v*)^V                                              eq. 108 L751-758 (R9)
 *   (pointwise products on the box of P_v, centre aligned, renormalised to sum 1: R5, R6).
 *   The estimate is then updated
 *       MVD_OSEM         psi <- max(psi * f_v, psi_floor) after every view, v = 0..V-1   (eq. 109-112)
 *       MVD_INDEPENDENT  psi <- max(psi * (prod_v max(f_v,0))^(1/V), psi_floor), K = PLAIN     (eq. 70; root: eq. 44, R1)
 *       MVD_EFFICIENT    same combination, K = COMPOUND                                        (eq. 104)
 *   One iteration = every view has contributed once (footnote L817).
 *   Options: per-view weights (section 12), Tikhonov regularisation (L64, L869): see mvd_options.
 *
 * Memory conventions
 *   - Volumes are fp32, x fastest: element (x,y,z) at [(z*Ny + y)*Nx + x].  dims = {Nx,Ny,Nz}.
 *   - `views` are DEVICE pointers; they are BORROWED (read-only, never copied) and must stay valid
 *     until mvd_destroy, and unchanged while a call that reads them may be in flight (mvd_restart is
 *     the call that accepts new contents).
 *   - `psfs` are HOST pointers, x fastest, dims psf_dims[v] = {Kx,Ky,Kz}, all odd (K may exceed N),
 *     values >= 0 with a positive sum (eq. 4).  They are copied during mvd_create.
 *   - ALL device memory the library uses is the caller's `workspace` (device pointer, at least
 *     mvd_workspace_size bytes, 256-byte aligned).  It must outlive the context.  The estimate psi
 *     lives inside it.  The library itself allocates no device memory.
 *   - `stream` is a cudaStream_t (as void*); NULL = the legacy default stream.  Every call enqueues
 *     its work on that stream; mvd_iterate is asynchronous.  Calls that return data to the HOST
 *     synchronise the stream.
 * Errors: every call returns an mvd_status, never throws or aborts.  On failure mvd_create sets
 *   *out = NULL.  A CUDA error is sticky: later calls on the context return MVD_ERR_STATE.
 * Threading: one context per stream; calls on one context are not re-entrant.
 */
#ifndef MVD_H_
#define MVD_H_

#include <stddef.h>

#if defined(__GNUC__)
#define MVD_API __attribute__((visibility("default")))
#else
#define MVD_API
#endif

#ifdef __cplusplus
extern "C" {
#endif

typedef struct mvd_ctx mvd_ctx;   /* opaque; created by mvd_create, freed by mvd_destroy */

typedef enum {
  MVD_OK = 0,
  MVD_ERR_INVALID_ARG = 1,   /* NULL pointer, bad dims, even PSF size, bad enum */
  MVD_ERR_UNSUPPORTED = 2,   /* no FFT length available for this size */
  MVD_ERR_WORKSPACE = 3,     /* workspace NULL, misaligned or too small */
  MVD_ERR_CUDA = 4,          /* a CUDA call failed (see mvd_last_error) */
  MVD_ERR_STATE = 5          /* call not valid in this state: context broken by an earlier CUDA error, or a
                              * view-parallel context driven through the wrong calls (see mvd_last_error) */
} mvd_status;

typedef enum {
  MVD_INDEPENDENT = 0,       /* eq. 70:  combined update, back-projector P_v*              */
  MVD_EFFICIENT = 1,         /* eq. 104: combined update, back-projector P_v^compound      */
  MVD_OSEM = 2               /* eq. 109-112: sequential updates, back-projector per kernel_mode */
} mvd_variant;

typedef enum {
  MVD_KERNEL_AUTO = 0,       /* INDEPENDENT -> PLAIN; EFFICIENT, OSEM -> COMPOUND (R2)     */
  MVD_KERNEL_PLAIN = 1,      /* with MVD_OSEM: classical OS-EM, eq. 114-117       */
  MVD_KERNEL_COMPOUND = 2,
  MVD_KERNEL_OPT1 = 3,
  MVD_KERNEL_OPT2 = 4
} mvd_kernel_mode;

typedef struct {
  size_t struct_size;        /* = sizeof(mvd_options); lets the struct grow compatibly      */
  int kernel_mode;           /* mvd_kernel_mode                                             */
  int literal_product;       /* combined variants: 0 = |V|-th root (eq. 44, default), 1 = bare product of eq. 2/38/104 */
  float eps;                 /* denominator clamp, <= 0 -> default 1e-6 (R4)                */
  float psi_floor;           /* estimate floor,    <  0 -> default 1e-6 (R4); 0 allowed     */
  const float* psi0;         /* optional DEVICE pointer to an initial estimate (N voxels); NULL -> mean of all views (L304, L421) */
  int fft_dims[3];           /* {Mx2, My, Mz}; 0 -> the library picks.  Mx2 is the length of the half-row transform */
  void* workspace;           /* DEVICE pointer, caller owned                                */
  size_t workspace_bytes;
  void* stream;              /* cudaStream_t                                                */
  int use_graph;             /* 1: mvd_iterate replays one captured CUDA graph per iteration (needs a non-default stream: MVD_ERR_UNSUPPORTED otherwise) */
  const float* const* weights; /* optional: n_views DEVICE pointers to per-view weight images (N voxels each, values in
                                * [0,1], borrowed like the views), section 12: a sequential update
                                * applies the fraction w_v of the change an RL step suggests,
                                * psi <- max(psi * (1 + w_v (f_v - 1)), floor).  MVD_OSEM only (else
                                * MVD_ERR_UNSUPPORTED).  NULL -> no weights.  How the weights are built (cosine
                                * blending, sum over views <= c) is the caller's business. */
  const int* local_views;    /* view-parallel combined variants: indices (ascending, unique) of the views THIS context owns;
                              * NULL -> all.  All n_views PSFs are still given (the compound kernels need them), views[v]
                              * may be NULL for views not listed.  Such a context is driven by mvd_partial_product /
                              * mvd_apply_product, not mvd_iterate; psi0 or psi0_value must be given. */
  int n_local;               /* length of local_views */
  float psi0_value;          /* > 0: constant initial estimate (a multi-rank caller passes the mean over ALL views) */
  void* views_ready;         /* optional cudaEvent_t: mvd_create makes its stream wait for it before the first read of
                              * the views (the initial estimate), so the caller's host-to-device copy of the views
                              * (on another stream) overlaps the PSF precompute.  NULL -> the views are ready. */
  float tikhonov_lambda;     /* >= 0; 0 = off.  Tikhonov regularisation of every psi update (ref. 20; the
                              * paper prints no formula: reading R14 of DESIGN.md).  With u the unregularised new value
                              * (psi*f_v, or psi*(prod f_v)^(1/V)), the update stores the positive root of
                              * (lambda/2) psi^2 + psi - u = 0, psi = 2u / (1 + sqrt(1 + 2 lambda u)), then applies the floor:
                              * the EM M-step for the Poisson likelihood with the penalty (lambda/4) sum psi^2.           */
  int block_rank;            /* mvd_deconvolve_blocked only: with block_world > 1 this call processes the blocks whose  */
  int block_world;           /* index (x fastest, then y, then z) is congruent to block_rank modulo block_world and     */
                             /* leaves the rest of dst untouched: blocks dealt over GPUs.  0 -> all.    */
} mvd_options;

/* Fills *opt with the defaults (struct_size set, everything else 0/NULL/defaults). */
MVD_API void mvd_options_init(mvd_options* opt);

/* Bytes of workspace mvd_create needs for this problem; 0 if the arguments are invalid or
 * unsupported.  `opt` may be NULL (defaults); only kernel_mode and fft_dims are read. */
MVD_API size_t mvd_workspace_size(int n_views, const int dims[3], const int (*psf_dims)[3],
                          mvd_variant variant, const mvd_options* opt);

/* The FFT lengths {Mx2, My, Mz} the library would use (for reporting algorithmic bytes). */
MVD_API mvd_status mvd_plan_dims(int n_views, const int dims[3], const int (*psf_dims)[3],
                         const mvd_options* opt, int fft_dims_out[3]);

/* Quality of the current estimate against a caller-supplied reference volume (DEVICE pointer, N voxels): the two
 * measures the paper reports, the average absolute difference and the cross-correlation
 * (Pearson coefficient, L48).  fp64 accumulation in warp-shuffle reductions; synchronises the stream.
 * Either output pointer may be NULL. */
MVD_API mvd_status mvd_compare(mvd_ctx* ctx, const float* ref_device, double* average_difference,
                               double* cross_correlation);

/* View-parallel form of the combined variants ("all view contributions can be computed at the same
 * time"; eq. 70 / 104 with the root of eq. 44).  Each rank owns some views and the same psi:
 *   mvd_partial_product : acc <- prod over the context's own views of max(f_v, 0) (f_v itself if literal_product),
 *                         every f_v computed from the current psi; psi is not changed.  Asynchronous.
 *   mvd_get_product     : DEVICE pointer to acc (N voxels, fp32, inside the workspace): the caller multiplies the
 *                         ranks' partial products element-wise in place (one all-reduce with the PRODUCT operator).
 *   mvd_apply_product   : psi <- max(psi * acc^(1/total_views), floor) (no root if literal_product), statistics;
 *                         counts as one iteration.  Every rank applies the same product, so psi stays replicated.
 * MVD_INDEPENDENT / MVD_EFFICIENT only (MVD_ERR_UNSUPPORTED for MVD_OSEM: sequential updates do not split).
 * mvd_reduce_sum: sum of n device floats in fp64 -> *host_out (for the global mean of the views); scratch = DEVICE
 * memory of at least mvd_reduce_scratch_bytes() on the device of src (a constant of the build: it does not depend on
 * which device is current when it is asked for). */
MVD_API mvd_status mvd_partial_product(mvd_ctx* ctx);
MVD_API mvd_status mvd_get_product(mvd_ctx* ctx, float** acc_device);
MVD_API mvd_status mvd_apply_product(mvd_ctx* ctx, int total_views);
MVD_API size_t mvd_reduce_scratch_bytes(void);
MVD_API mvd_status mvd_reduce_sum(const float* src_device, long long n, void* scratch_device, void* stream,
                                  double* host_out);

/* mvd_reduce_sum for callers that cannot supply scratch memory (same quantity: the sum of n device floats in fp64,
 * the numerator of the initial estimate psi^0 = mean of the views, PAPER.md L304 / L421).
 *
 * Every other call of this library works in memory the caller hands over, and mvd_reduce_sum is no exception: it
 * needs a scratch buffer.  Some callers have none to give and cannot allocate one: a job whose workspace already
 * fills the GPU (config 5 whole takes ~150 of 180 GB) or whose memory pool took all of HBM at start-up, so that
 * cudaMalloc fails; a time-lapse loop that sums every new time-point while other streams upload the next, where one
 * cudaMalloc/cudaFree pair per time-point would synchronise the device and undo the overlap; a plug-in of a host
 * application that receives device pointers but may not allocate on that application's GPU.  This call keeps its
 * partial sums in a fixed array compiled into the library's device image instead: about 128 KB on every GPU that
 * loads libmvd.so, held until the process exits.  It calls no cudaMalloc, cudaFree or allocating routine.
 *
 *   src_device  n floats on the CURRENT device (borrowed, read-only; any alignment); stream must belong to it.
 *   n           0 <= n <= mvd_reduce_sum_static_max() = 2^30 floats (one partial per 65536 floats, 16384 partials).
 *               Larger n: MVD_ERR_UNSUPPORTED, nothing is launched; split the input and add the pieces, or use
 *               mvd_reduce_sum.  n < 0 or a NULL pointer: MVD_ERR_INVALID_ARG.  CUDA failure: MVD_ERR_CUDA.
 *   host_out    HOST address of the result; the stream is synchronised before the call returns.
 *   mvd_reduce_sum_static_error(): the reason for the calling thread's last failure, "" after a success.
 * The result is the same for every launch and every GPU (fixed chunks, partials added in index order); it equals
 * mvd_reduce_sum's up to the rounding order of the fp64 additions (relative difference ~1e-15).
 * Set-up: the first call on each device looks up the array's device address (with that device current) and keeps it;
 * make that first call before any stream capture begins on that device.
 * Sharing: all calls on a device use the one array, which still holds the previous call's partials; the call clears
 * the one word that has to start at zero by itself.  Two calls whose GPU work overlaps (two streams, two host
 * threads) race on the array and return garbage: issue them one after the other (each call synchronises its stream
 * before it returns, so back-to-back calls from one thread are safe). */
MVD_API long long mvd_reduce_sum_static_max(void);
MVD_API const char* mvd_reduce_sum_static_error(void);
MVD_API mvd_status mvd_reduce_sum_static(const float* src_device, long long n, void* stream, double* host_out);

/* Builds a context: normalises the PSFs, computes the back-projectors K_v on the device (eq. 105 /
 * 107 / 108), their spectra and those of P_v, and the initial estimate.  Synchronises the stream
 * before returning.  See the header comment for pointer kinds and ownership. */
MVD_API mvd_status mvd_create(mvd_ctx** out, int n_views,
                      const float* const* views,      /* n_views DEVICE pointers   */
                      const int dims[3],
                      const float* const* psfs,       /* n_views HOST pointers     */
                      const int (*psf_dims)[3],
                      mvd_variant variant, const mvd_options* opt /* workspace required */);

/* Advances n >= 0 iterations (asynchronous on the stream). */
MVD_API mvd_status mvd_iterate(mvd_ctx* ctx, int n);

/* Copies the current estimate (Nx*Ny*Nz floats) to dst: a device pointer if dst_is_device != 0
 * (asynchronous on the stream), else a host pointer (the stream is synchronised). */
MVD_API mvd_status mvd_get_estimate(mvd_ctx* ctx, float* dst, int dst_is_device);

/* Replaces the estimate (device pointer, N voxels); resume / fixed-point tests. */
MVD_API mvd_status mvd_set_estimate(mvd_ctx* ctx, const float* src_device);

/* Starts over on NEW CONTENTS of the same view buffers: the next time-point of a time-lapse acquired with the same
 * PSFs (series of hundreds of time-points), so that the PSF precompute and the spectra of
 * mvd_create are paid once per series.  The caller overwrites the borrowed view buffers (same pointers) after every
 * earlier call on this context has completed, then calls mvd_restart: the stream waits for `views_ready` (optional
 * cudaEvent_t recorded after the caller's copy, NULL = already there), the estimate is re-initialised exactly as
 * mvd_create does (psi0 / psi0_value of the options, else the mean of the views), the iteration count and the
 * statistics are reset.  Asynchronous on the stream. */
MVD_API mvd_status mvd_restart(mvd_ctx* ctx, void* views_ready);

/* Statistics of the LAST psi update: flux = sum psi_new, l1_change = sum |psi_new - psi_old|
 * (the reductions the paper's quality curves use, L127).  Synchronises.  Any pointer may be NULL. */
MVD_API mvd_status mvd_get_stats(mvd_ctx* ctx, double* flux, double* l1_change, int* iterations_done);

/* Copies back-projector K_v (psf_dims[v] floats... as doubles, x fastest) to a HOST buffer.
 * Lets tests compare the device precompute (eq. 105) with the oracle directly.  Synchronises. */
MVD_API mvd_status mvd_get_back_projector(mvd_ctx* ctx, int view, double* dst_host);

/* One zero-extended "same" convolution of a device volume with view v's PSF (which = 0) or
 * back-projector (which = 1) through the library's FFT path: dst = crop(src (*) kernel).
 * src and dst are DEVICE pointers to N voxels (may alias).  Uses the context's work buffers: the
 * next mvd_iterate re-derives its transform state.  For per-stage parity tests.  In a view-parallel
 * context only the views it owns have spectra: MVD_ERR_INVALID_ARG for the others. */
MVD_API mvd_status mvd_convolve(mvd_ctx* ctx, int view, int which, const float* src, float* dst);

/* Number of kernel launches the library has issued on this context since creation. */
MVD_API long long mvd_launch_count(const mvd_ctx* ctx);

/* Per-kernel-class device timing, for the roofline report.  While
 * enabled, every pass kernel of mvd_iterate is bracketed by a pair of CUDA events on the context's
 * stream (not available with use_graph: MVD_ERR_STATE).  mvd_profile_read synchronises the stream,
 * writes the summed device time (milliseconds) and the launch count of each class into two HOST
 * arrays of MVD_K_COUNT entries, and clears the record. */
typedef enum {
  MVD_K_Y_FWD = 0,           /* y forward pencil pass (pruned input)                         */
  MVD_K_Y_INV = 1,           /* y inverse pencil pass (cropped output)                       */
  MVD_K_Z_CONV = 2,          /* z forward . spectrum . z inverse                             */
  MVD_K_X_QUOT = 3,          /* x inverse -> quotient -> x forward                           */
  MVD_K_X_UPDATE = 4,        /* x inverse -> psi update -> x forward (OSEM)                  */
  MVD_K_X_ACCUM = 5,         /* x inverse -> product accumulation / combined update          */
  MVD_K_X_LOAD = 6,          /* x forward of psi (first iteration, after mvd_set_estimate)   */
  MVD_K_COUNT = 7
} mvd_kernel_class;
MVD_API mvd_status mvd_profile(mvd_ctx* ctx, int enable);
MVD_API mvd_status mvd_profile_read(mvd_ctx* ctx, double* total_ms_host, long long* launches_host);
MVD_API const char* mvd_kernel_class_name(int kernel_class);

/* Block-wise processing (L64, L943; R13): tiles the volume into blocks of block_dims, extends
 * every block by `halo` voxels of neighbouring data per side (clipped at the volume faces; halo
 * = NULL -> PSF half-size), runs `iterations` iterations on each extended block with
 * psi0 = mean over the whole volume, and pastes the central block into dst (DEVICE, N voxels).
 * All device memory comes from opt->workspace (size: mvd_blocked_workspace_size).  The whole-volume
 * options weights, views_ready, local_views, psi0 and psi0_value are refused (MVD_ERR_UNSUPPORTED). */
MVD_API size_t mvd_blocked_workspace_size(int n_views, const int dims[3], const int (*psf_dims)[3],
                                  mvd_variant variant, const mvd_options* opt,
                                  const int block_dims[3], const int halo[3]);
MVD_API mvd_status mvd_deconvolve_blocked(int n_views, const float* const* views, const int dims[3],
                                  const float* const* psfs, const int (*psf_dims)[3],
                                  mvd_variant variant, const mvd_options* opt,
                                  const int block_dims[3], const int halo[3], int iterations,
                                  float* dst_device, long long* launches_out);

MVD_API void mvd_destroy(mvd_ctx* ctx);                    /* NULL-safe */
MVD_API const char* mvd_status_string(mvd_status s);
MVD_API const char* mvd_last_error(const mvd_ctx* ctx);    /* "" if none; valid until the next call */

#ifdef __cplusplus
}
#endif
#endif /* MVD_H_ */
