// libmvd.so: context, planner and launch sequences behind the C ABI of include/mvd.h.
//
// Path per view-update (eq. 1, eq. 13, eq. 104,
// eq. 109-112), all on the device, one stream:
//   y-forward -> [z-forward . P_v spectrum . z-inverse] -> y-inverse
//     -> [x-inverse -> quotient phi_v/max(b,eps) -> x-forward]
//   y-forward -> [z-forward . K_v spectrum . z-inverse] -> y-inverse
//     -> [x-inverse -> psi update (or product accumulation) -> x-forward of the new psi]
// The oracle (oracle/) is never used here; without a CUDA device every call fails with
// MVD_ERR_CUDA.
#include "../../include/mvd.h"

#include <algorithm>
#include <cmath>
#include <cstdarg>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <mutex>
#include <new>
#include <array>
#include <vector>

#include "fft_ops.h"
#include "misc_kernels.cuh"

namespace mvd {

// ---------------------------------------------------------------------------------------
// table of compiled lengths (one object file per line of lengths.def)
// ---------------------------------------------------------------------------------------
#define MVD_LEN(A, B) extern const LengthOps ops_##A##_##B;
#include "lengths.def"
#undef MVD_LEN

static const LengthOps* const g_lengths_unsorted[] = {
#define MVD_LEN(A, B) &ops_##A##_##B,
#include "lengths.def"
#undef MVD_LEN
};

const LengthOps* const* length_table(int* count) {
  static std::vector<const LengthOps*> sorted = [] {
    std::vector<const LengthOps*> v(std::begin(g_lengths_unsorted), std::end(g_lengths_unsorted));
    std::sort(v.begin(), v.end(), [](const LengthOps* a, const LengthOps* b) { return a->M < b->M; });
    return v;
  }();
  *count = (int)sorted.size();
  return sorted.data();
}

// smallest compiled length >= min_len (or exactly `exact`); need_even: the x length, whose rows are
// staged by 16-byte bulk copies and whose pitch is a TMA stride
static const LengthOps* find_length(int min_len, int exact, bool need_even) {
  int n;
  const LengthOps* const* t = length_table(&n);
  for (int i = 0; i < n; ++i) {
    if (need_even && (t[i]->M & 1)) continue;
    if (exact > 0) {
      if (t[i]->M == exact) return t[i]->M >= min_len ? t[i] : nullptr;
    } else if (t[i]->M >= min_len) {
      return t[i];
    }
  }
  return nullptr;
}

// ---------------------------------------------------------------------------------------
// plan: sizes, FFT lengths, tiles, workspace layout
// ---------------------------------------------------------------------------------------
static inline size_t align_up(size_t x, size_t a) { return (x + a - 1) / a * a; }
static inline int round_up32(int x) { return (x + 31) / 32 * 32; }

struct Plan {
  int V = 0;
  int N[3] = {0, 0, 0};
  std::vector<Dims3> K;          // per view
  int r[3] = {0, 0, 0};          // max half-size per axis
  int hx = 0;
  const LengthOps *lx = nullptr, *ly = nullptr, *lz = nullptr;
  int Mx = 0, My = 0, Mz = 0;
  long long nvox = 0, plane = 0, wsize = 0, ssize = 0;   // elements
  bool combined = false;
  int weighted = 0;              // per-view weight images given (section 12): the x update stages them too
  int kmode = MVD_KERNEL_PLAIN;
  // tiles
  int Ty = 0, nty = 0, Tz = 0, ntz = 0, Tzs = 0, ntzs = 0, Tys = 0, ntys = 0, Rx = 0, ntx = 0;
  int nctax = 0;
  // TMA-staged x pass
  int xtma = 0, Rxt = 0, ntxt = 0, xt_rstride = 0, xt_exch = 0, xt_exch_g = 0, xt_exch_f = 0;
  // TMA-staged y and z passes: tile width, threads, pencil boxes (boxr rows x nbox >= M)
  int ytma = 0, Tyt = 0, ntyt = 0, ybox = 0, ynbox = 0, ynst = 2;
  int ztma = 0, Tzt = 0, ntzt = 0, zbox = 0, znbox = 0, znst = 2;
  // workspace offsets (bytes)
  size_t off_twx = 0, off_twy = 0, off_twz = 0, off_psi = 0, off_acc = 0, off_w = 0, off_w0 = 0,
         off_spec = 0, off_psf = 0, off_kern = 0, off_auto = 0, off_partials = 0,
         off_scalars = 0, off_cmp = 0, total = 0;
  size_t psf_stride = 0, auto_stride = 0;   // elements (doubles) per view
  int sum_blocks = 0;
};

// Shared-memory wavefronts of the x pass's exchange buffer for one row stride: 64-bit accesses are
// served per half-warp, one wavefront per distinct bank pair multiplicity.  g_layout: rows written by
// (row, k1) lanes at [m*AP + k1] and read by (row, n2) lanes at [n2*AP + kk]; else the forward layout
// [k1*BP + m] / [kk*BP + n2].
static long long exch_wavefronts(int A, int B, int R, int nthreads, int RS, bool g_layout) {
  const int AP = A | 1, BP = B | 1;
  long long total = 0;
  for (int hw = 0; hw < nthreads / 16; ++hw) {
    for (int pass = 0; pass < 2; ++pass) {
      const int role = pass == 0 ? A : B;          // lanes per row
      const int reps = pass == 0 ? B : A;          // unrolled accesses per thread
      for (int m = 0; m < reps; ++m) {
        int cnt[16] = {0};
        int worst = 0;
        for (int l = 0; l < 16; ++l) {
          const int t = hw * 16 + l;
          if (t >= R * role) continue;
          const int row = t / role, q = t % role;
          int addr;
          if (g_layout) addr = pass == 0 ? row * RS + m * AP + q : row * RS + q * AP + m;
          else addr = pass == 0 ? row * RS + q * BP + m : row * RS + m * BP + q;
          worst = std::max(worst, ++cnt[addr & 15]);
        }
        total += worst;
      }
    }
  }
  return total;
}

static int best_exch_stride(int A, int B, int R, int nthreads, int min_stride, bool g_layout) {
  int best = min_stride;
  long long best_cost = -1;
  for (int rs = min_stride; rs < min_stride + 16; ++rs) {
    const long long cst = exch_wavefronts(A, B, R, nthreads, rs, g_layout);
    if (best_cost < 0 || cst < best_cost) { best_cost = cst; best = rs; }
  }
  return best;
}

// SMs of the current device (148 on B200); 148 when there is no device (host-only planning calls)
static int sm_count() {
  int dev = 0, n = 0;
  if (cudaGetDevice(&dev) != cudaSuccess || cudaDeviceGetAttribute(&n, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess || n <= 0) {
    cudaGetLastError();
    n = 148;
  }
  return n;
}
// grid of the grid-stride reduction / fill kernels: 8 CTAs of 256 threads per SM
static int reduce_blocks() { return 8 * sm_count(); }

// combined variants: the running product of the f_v is kept in fp32; beyond this many views every factor takes the
// |V|-th root before it enters the product (same value, no overflow or underflow for any V the ABI accepts)
constexpr int kRootEachViews = 16;

// Tuning / comparison knobs: ONE environment variable, read once per plan and once per context,
//   MVD_TUNE="key=value,key=value,..."   (integer values; unknown keys are ignored)
// Every knob selects another kernel or tile shape, never another result (tests/test_gpu_parity.py runs them against
// the oracle).  Keys: xtma ytma ztma (0: register-staged fallback kernels of pass_kernels.cuh), rxt xt_smem_kb
// (rows / shared-memory cap of an x tile), ynst znst (tile stages of the y / z pass), ztx (8: z tile of 8 x by 2 rows),
// ypair (0/1: column pairs in the y pass; default on from 1000-point pencils), xbulk (0: real rows by plain loads),
// flip (0: no alternating tile order), corr_tiled (0: untiled precompute correlation), and for the fallback
// kernels ty tz rx xthreads.
struct Tune {
  static constexpr int kMax = 24;
  char key[kMax][16];
  int val[kMax];
  int n = 0;
  Tune() {
    const char* s = getenv("MVD_TUNE");
    while (s && *s && n < kMax) {
      const char* eq = strchr(s, '=');
      const char* end = strchr(s, ',');
      if (!end) end = s + strlen(s);
      if (eq && eq < end && eq - s > 0 && eq - s < 16) {
        memcpy(key[n], s, (size_t)(eq - s));
        key[n][eq - s] = 0;
        val[n] = atoi(eq + 1);
        ++n;
      }
      s = *end ? end + 1 : end;
    }
  }
  int get(const char* k, int dflt) const {
    for (int i = 0; i < n; ++i)
      if (strcmp(key[i], k) == 0) return val[i];
    return dflt;
  }
};

// tile width for a strided pass over a contiguous extent L; single_round: T*max(A,B) <= max_threads
static void choose_tile(const LengthOps* l, long long L, bool single_round, int force, int* T_out,
                        int* nthreads_out) {
  const int ab = std::max(l->A, l->B);
  const size_t smem_cap = 100 * 1024;
  int best = 0;
  double best_score = -1.0;
  const int cand[] = {16, 20, 24, 32, 28, 12, 8, 4};
  for (int T : cand) {
    if (l->strided_smem(T) > smem_cap && T > 4) continue;
    if (single_round && T * ab > l->max_threads) continue;
    const double eff = double(L) / double(((L + T - 1) / T) * T);
    const double seg = T >= 16 ? 1.0 : (T >= 8 ? 0.85 : 0.6);   // short segments waste DRAM bursts
    const double score = eff * seg;
    if (score > best_score + 1e-9) { best_score = score; best = T; }
  }
  if (best == 0) best = std::max(1, std::min(4, l->max_threads / ab));
  if (force > 0 && (!single_round || force * ab <= l->max_threads)) best = force;
  const int items = best * ab;
  const int rounds = (items + l->max_threads - 1) / l->max_threads;
  *T_out = best;
  *nthreads_out = std::min(l->max_threads, round_up32((items + rounds - 1) / rounds));
}

static mvd_status make_plan(Plan& P, int n_views, const int dims[3], const int (*psf_dims)[3],
                            mvd_variant variant, const mvd_options* opt) {
  if (n_views < 1 || n_views > 4096 || !dims || !psf_dims) return MVD_ERR_INVALID_ARG;
  if ((int)variant < 0 || (int)variant > 2) return MVD_ERR_INVALID_ARG;
  int kmode = opt ? opt->kernel_mode : MVD_KERNEL_AUTO;
  if (kmode < 0 || kmode > 4) return MVD_ERR_INVALID_ARG;
  if (kmode == MVD_KERNEL_AUTO) kmode = (variant == MVD_INDEPENDENT) ? MVD_KERNEL_PLAIN : MVD_KERNEL_COMPOUND;
  P.kmode = kmode;
  P.V = n_views;
  P.combined = variant != MVD_OSEM;
  P.weighted = (opt && opt->weights) ? 1 : 0;
  if (P.weighted && P.combined) return MVD_ERR_UNSUPPORTED;   // weights belong to the sequential updates (L897)
  for (int a = 0; a < 3; ++a) {
    if (dims[a] < 1 || dims[a] > (1 << 20)) return MVD_ERR_INVALID_ARG;
    P.N[a] = dims[a];
    P.r[a] = 0;
  }
  P.K.resize(n_views);
  for (int v = 0; v < n_views; ++v) {
    for (int a = 0; a < 3; ++a) {
      const int k = psf_dims[v][a];
      if (k < 1 || (k & 1) == 0 || k > (1 << 12)) return MVD_ERR_INVALID_ARG;
      P.r[a] = std::max(P.r[a], (k - 1) / 2);
    }
    P.K[v] = Dims3{psf_dims[v][0], psf_dims[v][1], psf_dims[v][2]};
  }
  P.hx = (P.N[0] + 1) / 2;
  // alias-free 'same' output needs M >= N + r; the wrapped kernel taps need M >= K = 2r + 1
  const int need[3] = {P.hx + 2 * P.r[0], std::max(P.N[1] + P.r[1], 2 * P.r[1] + 1),
                       std::max(P.N[2] + P.r[2], 2 * P.r[2] + 1)};
  const LengthOps* l[3];
  for (int a = 0; a < 3; ++a) {
    const int want = opt ? opt->fft_dims[a] : 0;
    if (want < 0) return MVD_ERR_INVALID_ARG;
    l[a] = find_length(need[a], want, a == 0);
    if (!l[a]) return want > 0 ? MVD_ERR_INVALID_ARG : MVD_ERR_UNSUPPORTED;
  }
  P.lx = l[0]; P.ly = l[1]; P.lz = l[2];
  P.Mx = l[0]->M; P.My = l[1]->M; P.Mz = l[2]->M;
  P.nvox = (long long)P.N[0] * P.N[1] * P.N[2];
  P.plane = (long long)P.My * P.Mx;
  P.wsize = P.plane * P.N[2];
  P.ssize = P.plane * P.Mz;

  const Tune tune;
  choose_tile(P.ly, P.Mx, false, tune.get("ty", 0), &P.Ty, &P.nty);
  choose_tile(P.lz, P.plane, true, tune.get("tz", 0), &P.Tz, &P.ntz);
  choose_tile(P.lz, P.plane, false, 0, &P.Tzs, &P.ntzs);
  choose_tile(P.ly, P.Mx, false, 0, &P.Tys, &P.ntys);
  {
    const int ab = std::max(P.lx->A, P.lx->B);
    int R = std::max(1, tune.get("xthreads", 256) / ab);
    const int force = tune.get("rx", 0);
    if (force > 0) R = force;
    R = std::min(R, std::max(1, P.lx->max_threads / ab));
    while (R > 1 && P.lx->xrow_smem(R, P.r[0]) > 160 * 1024) --R;
    P.Rx = R;
    P.ntx = round_up32(R * ab);
    // spectrum construction runs the same kernel over My*Mz rows
    const long long rows_max = std::max((long long)P.N[1] * P.N[2], (long long)P.My * P.Mz);
    P.nctax = (int)((rows_max + R - 1) / R);
  }

  {
    // TMA-staged y and z passes: tile widths are multiples of 4 (16-byte rows, 128-byte boxes)
    auto plan_tma = [&](const LengthOps* l, bool zconv, int* T_out, int* nt_out, int* box_out, int* nbox_out) {
      const int ab = std::max(l->A, l->B);
      const int nbox = (l->M + 255) / 256;
      const int boxr = ((l->M + nbox - 1) / nbox + 3) / 4 * 4;
      const int T = zconv ? kTmaTileHost : strided_tma_tile(l->M);   // the kernels are compiled for one tile width
      const int items = T * ab * (zconv ? 2 : 1);   // the z tile is 16 columns
      const int rounds = (items + l->max_threads - 1) / l->max_threads;
      *T_out = T;
      *nt_out = std::min(l->max_threads, round_up32((items + rounds - 1) / rounds));
      *box_out = boxr;
      *nbox_out = nbox;
      const size_t smem = zconv ? l->zconv_tma_smem(T, boxr, nbox, P.znst) : l->strided_tma_smem(T, boxr, nbox, P.ynst);
      return smem <= 220 * 1024;
    };
    P.znst = tune.get("znst", 2) == 1 ? 1 : 2;
    {
      // two tile stages whenever they fit (one stage with more CTAs per SM measured slower on config 5)
      const int nbox = (P.ly->M + 255) / 256;
      const int boxr = ((P.ly->M + nbox - 1) / nbox + 3) / 4 * 4;
      P.ynst = P.ly->strided_tma_smem(strided_tma_tile(P.ly->M), boxr, nbox, 2) <= 218 * 1024 ? 2 : 1;
      const int force = tune.get("ynst", 0);
      if (force == 1 || force == 2) P.ynst = force;
      const int nbz = (P.lz->M + 255) / 256;
      const int bxz = ((P.lz->M + nbz - 1) / nbz + 3) / 4 * 4;
      if (tune.get("znst", 0) == 0) P.znst = P.lz->zconv_tma_smem(kTmaTileHost, bxz, nbz, 2) <= 218 * 1024 ? 2 : 1;
    }
    P.ytma = tune.get("ytma", 1);
    P.ztma = tune.get("ztma", 1);
    if (!plan_tma(P.ly, false, &P.Tyt, &P.ntyt, &P.ybox, &P.ynbox)) P.ytma = 0;
    if (!plan_tma(P.lz, true, &P.Tzt, &P.ntzt, &P.zbox, &P.znbox)) P.ztma = 0;
  }
  {
    // TMA-staged x pass (quotient / OSEM update): rows per tile sized for >= 3 resident CTAs per SM
    const int ab = std::max(P.lx->A, P.lx->B);
    P.xtma = tune.get("xtma", 1);
    int R = std::max(1, 160 / ab);   // kXrowTmaThreads of pass_tma.cuh
    const int force = tune.get("rxt", 0);
    // 45 KB: five CTAs per SM; larger radices hold fewer CTAs (registers), so they get larger tiles
    const size_t cap = (size_t)tune.get("xt_smem_kb", ab <= 21 ? 45 : (ab <= 28 ? 72 : 100)) * 1024;
    while (R > 1 && P.lx->xrow_tma_smem(R, P.r[0], P.N[0], P.weighted) > cap) --R;
    if (force > 0 && force * ab <= 160 && P.lx->xrow_tma_smem(force, P.r[0], P.N[0], P.weighted) <= 220 * 1024) R = force;
    if (P.lx->xrow_tma_smem(R, P.r[0], P.N[0], P.weighted) > 220 * 1024) P.xtma = 0;
    P.Rxt = R;
    P.ntxt = round_up32(R * ab);
    int s = (P.N[0] + 3 + 3) / 4 * 4;   // == xrow_rstride of pass_tma.cuh
    const int want = (P.lx->B % 32) / 4 * 4;
    while ((s % 32) != want) s += 4;
    P.xt_rstride = s;
    const int A = P.lx->A, B = P.lx->B;
    const int row_min = std::max(A * (B | 1), B * (A | 1));
    P.xt_exch = row_min + 16;
    P.xt_exch_g = best_exch_stride(A, B, R, P.ntxt, B * (A | 1), true);
    P.xt_exch_f = best_exch_stride(A, B, R, P.ntxt, A * (B | 1), false);
  }

  // workspace layout
  size_t o = 0;
  auto take = [&](size_t bytes) { size_t at = o; o = align_up(o + bytes, 256); return at; };
  P.off_twx = take((size_t)P.Mx * sizeof(float2));
  P.off_twy = take((size_t)P.My * sizeof(float2));
  P.off_twz = take((size_t)P.Mz * sizeof(float2));
  P.off_psi = take((size_t)P.nvox * sizeof(float));
  P.off_acc = take((size_t)P.nvox * sizeof(float));
  P.off_w = take((size_t)P.wsize * sizeof(float2));
  P.off_w0 = P.combined ? take((size_t)P.wsize * sizeof(float2)) : 0;
  P.off_spec = take((size_t)P.ssize * sizeof(float2) * 2 * P.V);
  size_t kmax = 0, amax = 0;
  for (int v = 0; v < P.V; ++v) {
    const Dims3 k = P.K[v];
    kmax = std::max(kmax, (size_t)k.x * k.y * k.z);
    amax = std::max(amax, (size_t)(2 * k.x - 1) * (2 * k.y - 1) * (2 * k.z - 1));
  }
  P.psf_stride = align_up(kmax, 32);
  P.auto_stride = align_up(amax, 32);
  P.off_psf = take(P.psf_stride * sizeof(double) * P.V);
  P.off_kern = take(P.psf_stride * sizeof(double) * P.V);
  P.off_auto = take(kmode == MVD_KERNEL_COMPOUND ? P.auto_stride * sizeof(double) * P.V : 256);
  P.sum_blocks = reduce_blocks();
  P.off_partials = take(sizeof(double) * 2 * (size_t)std::max(P.nctax, P.sum_blocks));
  P.off_scalars = take(sizeof(double) * (size_t)(P.V + 8));
  P.off_cmp = take(sizeof(double) * (6 * 192 + 8));   // mvd_compare partials
  P.total = o;
  return MVD_OK;
}

}  // namespace mvd

using namespace mvd;

// ---------------------------------------------------------------------------------------
// context
// ---------------------------------------------------------------------------------------
struct mvd_ctx {
  Plan P;
  mvd_variant variant = MVD_OSEM;
  int literal = 0;
  float eps = 1e-6f, psi_floor = 1e-6f, tikhonov = 0.f;
  cudaStream_t stream = nullptr;
  char* ws = nullptr;
  char* psf_staging = nullptr;   // pinned, device-mapped host copy of the PSF taps (process-wide buffer, held under its lock)
  cudaEvent_t staged_read = nullptr;   // recorded behind the last kernel that reads psf_staging
  std::vector<const float*> views;
  std::vector<const float*> weights;   // empty or one per view (borrowed)
  std::vector<char> is_local;          // view-parallel contexts: which views this context owns (all by default)
  bool partial = false;
  float psi0_value = 0.f;
  const float* psi0_ptr = nullptr;     // options.psi0 (borrowed), for mvd_restart
  bool w_valid = false;        // the work buffer holds the x-forward transform of the current psi
  int y_pair = 0;              // y pass: two columns per thread, 128-bit shared-memory and global accesses
                               // (MVD_YPAIR=0/1; default: on for pencils of 1000 points or more)
  int corr_tiled = 1;          // 0: the untiled fp64 correlation kernel of the precompute (MVD_CORR_TILED=0)
  int xbulk = 1;               // 0: real rows of the x pass by plain loads (MVD_XBULK=0, for comparison)
  int ztx = 16;                // z pass tile: 16 x of one row (default), or 8 x of two rows y
  bool broken = false;
  bool stats_valid = false;
  int stats_ncta = 0;
  int iters = 0;
  long long launches = 0;
  int use_graph = 0;
  cudaGraphExec_t graph_exec = nullptr;
  long long graph_launches = 0;
  int graph_stats_ncta = 0;          // CTAs of the update kernel that write the statistics partials (as captured)
  char err[512] = {0};
  int num_sms = 148;
  int xt_blocks[5][4] = {};          // resident CTAs per SM of the TMA-staged x pass, per (mode, compile-time flags)
  int flip = 0;                      // tile direction of the next x / y launch (alternates: L2 reuse)
  int use_flip = 1;
  int yt_blocks[2][2] = {};          // ... of the TMA-staged y pass, per (direction, column-pair variant)
  int zt_blocks[2] = {0, 0};         // ... of the TMA-staged z pass, per tile shape (8 x 2, 16 x 1)
  // per-kernel-class event timing (mvd_profile)
  bool profiling = false;
  std::vector<cudaEvent_t> ev_pool;
  size_t ev_used = 0;
  struct Rec { int cls; cudaEvent_t a, b; };
  std::vector<Rec> recs;
  cudaEvent_t next_event() {
    if (ev_used == ev_pool.size()) {
      cudaEvent_t e = nullptr;
      if (cudaEventCreate(&e) != cudaSuccess) return nullptr;
      ev_pool.push_back(e);
    }
    return ev_pool[ev_used++];
  }

  float2* twx() { return reinterpret_cast<float2*>(ws + P.off_twx); }
  float2* twy() { return reinterpret_cast<float2*>(ws + P.off_twy); }
  float2* twz() { return reinterpret_cast<float2*>(ws + P.off_twz); }
  float* psi() { return reinterpret_cast<float*>(ws + P.off_psi); }
  float* acc() { return reinterpret_cast<float*>(ws + P.off_acc); }
  float2* W() { return reinterpret_cast<float2*>(ws + P.off_w); }
  float2* W0() { return reinterpret_cast<float2*>(ws + P.off_w0); }
  float2* specH(int v) { return reinterpret_cast<float2*>(ws + P.off_spec) + (size_t)(2 * v) * P.ssize; }
  float2* specK(int v) { return reinterpret_cast<float2*>(ws + P.off_spec) + (size_t)(2 * v + 1) * P.ssize; }
  double* psf(int v) { return reinterpret_cast<double*>(ws + P.off_psf) + (size_t)v * P.psf_stride; }
  double* kern(int v) { return reinterpret_cast<double*>(ws + P.off_kern) + (size_t)v * P.psf_stride; }
  double* autoc(int v) { return reinterpret_cast<double*>(ws + P.off_auto) + (size_t)v * P.auto_stride; }
  double* partials() { return reinterpret_cast<double*>(ws + P.off_partials); }
  double* scalars() { return reinterpret_cast<double*>(ws + P.off_scalars); }   // [0..V) view sums, [V],[V+1] stats

  bool fail(cudaError_t e, const char* what) {
    if (e == cudaSuccess) return false;
    snprintf(err, sizeof(err), "%s: %s", what, cudaGetErrorString(e));
    broken = true;
    return true;
  }
};

#define MVD_CK(call, what) \
  do { if (c->fail((call), what)) return MVD_ERR_CUDA; } while (0)

namespace {

// brackets one launch with events while profiling is on
struct ProfScope {
  mvd_ctx* c;
  cudaEvent_t a = nullptr, b = nullptr;
  int cls;
  ProfScope(mvd_ctx* c_, int cls_) : c(c_), cls(cls_) {
    if (!c->profiling) return;
    a = c->next_event();
    b = c->next_event();
    if (a && b) cudaEventRecord(a, c->stream);
  }
  ~ProfScope() {
    if (!c->profiling || !a || !b) return;
    cudaEventRecord(b, c->stream);
    c->recs.push_back(mvd_ctx::Rec{cls, a, b});
  }
};

// ---- tensor maps (driver entry point resolved through the runtime: no link against libcuda) --
typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*,
                                  const cuuint64_t*, const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave,
                                  CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

EncodeTiledFn encode_tiled_fn() {
  static EncodeTiledFn fn = [] {
    void* p = nullptr;
    cudaDriverEntryPointQueryResult q;
    if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &q) != cudaSuccess ||
        q != cudaDriverEntryPointSuccess)
      p = nullptr;
    return reinterpret_cast<EncodeTiledFn>(p);
  }();
  return fn;
}

// 3-D map over complex64 elements (carried as 8-byte words): dims d0 (contiguous), d1, d2 with
// element strides s1, s2; box b0 x b1 x b2; elements outside the dims are delivered as zeros
bool make_map3(CUtensorMap* m, const void* base, long long d0, long long d1, long long d2, long long s1,
               long long s2, int b0, int b1, int b2) {
  EncodeTiledFn fn = encode_tiled_fn();
  if (!fn) return false;
  const cuuint64_t gdim[3] = {(cuuint64_t)d0, (cuuint64_t)d1, (cuuint64_t)d2};
  const cuuint64_t gstr[2] = {(cuuint64_t)s1 * 8, (cuuint64_t)s2 * 8};
  const cuuint32_t box[3] = {(cuuint32_t)b0, (cuuint32_t)b1, (cuuint32_t)b2};
  const cuuint32_t est[3] = {1, 1, 1};
  return fn(m, CU_TENSOR_MAP_DATA_TYPE_UINT64, 3, const_cast<void*>(base), gdim, gstr, box, est,
            CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_128B,
            CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
}

mvd_status y_pass_tma(mvd_ctx* c, float2* buf, int dir, int nz_planes, int xt0, int n_xt) {
  const Plan& P = c->P;
  StridedTmaArgs a{};
  const int n_in = dir < 0 ? P.N[1] : P.My;
  if (!make_map3(&a.in_map, buf, P.Mx, n_in, nz_planes, P.Mx, P.plane, P.Tyt, P.ybox, 1)) {
    snprintf(c->err, sizeof(c->err), "y pass: cuTensorMapEncodeTiled failed");
    c->broken = true;
    return MVD_ERR_CUDA;
  }
  a.out = buf; a.tw = c->twy();
  a.pair = c->y_pair;
  a.T = P.Tyt; a.nthreads = P.ntyt; a.boxr = P.ybox; a.nbox = P.ynbox;
  a.xt0 = xt0; a.n_xt = n_xt; a.nst = P.ynst;
  a.line_len = P.Mx; a.n_outer = nz_planes;
  a.out_outer_stride = P.plane; a.out_pstride = P.Mx;
  a.n_out = dir < 0 ? P.My : P.N[1];
  a.reverse = c->use_flip ? (c->flip ^= 1) : 0;
  int& bl = c->yt_blocks[dir < 0 ? 0 : 1][a.pair ? 1 : 0];
  if (bl == 0) bl = P.ly->strided_tma_blocks_per_sm(a, dir);
  if (bl <= 0) { snprintf(c->err, sizeof(c->err), "y pass: kernel does not fit on an SM"); c->broken = true; return MVD_ERR_CUDA; }
  a.grid = (int)std::min<long long>((long long)n_xt * nz_planes, (long long)c->num_sms * bl);
  {
    ProfScope ps(c, dir < 0 ? MVD_K_Y_FWD : MVD_K_Y_INV);
    MVD_CK(P.ly->strided_tma(a, dir, c->stream), "y pass (TMA)");
  }
  ++c->launches;
  return MVD_OK;
}

mvd_status z_conv_tma(mvd_ctx* c, const float2* in, float2* out, const float2* spec, int xt0, int n_xt) {
  const Plan& P = c->P;
  ZconvTmaArgs a{};
  const int tx = c->ztx, ty = 2 * P.Tzt / tx;
  n_xt = (P.Mx + tx - 1) / tx;
  if (!make_map3(&a.in_map, in, P.Mx, P.My, P.N[2], P.Mx, P.plane, tx, ty, P.zbox) ||
      !make_map3(&a.spec_map, spec, P.Mx, P.My, P.Mz, P.Mx, P.plane, tx, ty, P.zbox)) {
    snprintf(c->err, sizeof(c->err), "z pass: cuTensorMapEncodeTiled failed");
    c->broken = true;
    return MVD_ERR_CUDA;
  }
  a.out = out; a.tw = c->twz();
  a.T = P.Tzt; a.nthreads = P.ntzt; a.boxr = P.zbox; a.nbox = P.znbox;
  a.xt0 = xt0; a.n_xt = n_xt; a.tx = tx;
  a.mx = P.Mx; a.my = P.My; a.plane = P.plane; a.nz = P.N[2]; a.nst_in = P.znst;
  int& bl = c->zt_blocks[tx == 16 ? 1 : 0];
  if (bl == 0) bl = P.lz->zconv_tma_blocks_per_sm(a);
  if (bl <= 0) { snprintf(c->err, sizeof(c->err), "z pass: kernel does not fit on an SM"); c->broken = true; return MVD_ERR_CUDA; }
  a.grid = (int)std::min<long long>((long long)n_xt * ((P.My + ty - 1) / ty), (long long)c->num_sms * bl);
  {
    ProfScope ps(c, MVD_K_Z_CONV);
    MVD_CK(P.lz->zconv_tma(a, c->stream), "z convolution pass (TMA)");
  }
  ++c->launches;
  return MVD_OK;
}

// ---- pass launchers -------------------------------------------------------------------------
mvd_status y_pass(mvd_ctx* c, float2* buf, int dir, int nz_planes, bool full) {
  const Plan& P = c->P;
  if (P.ytma && !full) return y_pass_tma(c, buf, dir, nz_planes, 0, (P.Mx + P.Tyt - 1) / P.Tyt);
  StridedArgs a{};
  a.in = buf; a.out = buf; a.tw = c->twy();
  a.T = full ? P.Tys : P.Ty;
  a.nthreads = full ? P.ntys : P.nty;
  a.line_len = P.Mx;
  a.tiles_per_line = (P.Mx + a.T - 1) / a.T;
  a.n_outer = nz_planes;
  a.in_outer_stride = a.out_outer_stride = P.plane;
  a.in_pstride = a.out_pstride = P.Mx;
  if (full) { a.n_in = P.My; a.n_out = P.My; }
  else if (dir < 0) { a.n_in = P.N[1]; a.n_out = P.My; }
  else { a.n_in = P.My; a.n_out = P.N[1]; }
  {
    ProfScope ps(c, dir < 0 ? MVD_K_Y_FWD : MVD_K_Y_INV);
    MVD_CK(P.ly->strided(a, dir, c->stream), "y pass");
  }
  ++c->launches;
  return MVD_OK;
}

mvd_status z_plain_fwd(mvd_ctx* c, float2* buf) {
  const Plan& P = c->P;
  StridedArgs a{};
  a.in = buf; a.out = buf; a.tw = c->twz();
  a.T = P.Tzs; a.nthreads = P.ntzs;
  a.line_len = P.plane;
  a.tiles_per_line = (int)((P.plane + a.T - 1) / a.T);
  a.n_outer = 1;
  a.in_outer_stride = a.out_outer_stride = 0;
  a.in_pstride = a.out_pstride = P.plane;
  a.n_in = P.Mz; a.n_out = P.Mz;
  MVD_CK(P.lz->strided(a, -1, c->stream), "z pass");
  ++c->launches;
  return MVD_OK;
}

mvd_status z_conv(mvd_ctx* c, const float2* in, float2* out, const float2* spec) {
  const Plan& P = c->P;
  if (P.ztma) return z_conv_tma(c, in, out, spec, 0, (P.Mx + P.Tzt - 1) / P.Tzt);
  ZconvArgs a{};
  a.in = in; a.out = out; a.spec = spec; a.tw = c->twz();
  a.T = P.Tz; a.nthreads = P.ntz; a.plane = P.plane; a.nz = P.N[2];
  {
    ProfScope ps(c, MVD_K_Z_CONV);
    MVD_CK(P.lz->zconv(a, c->stream), "z convolution pass");
  }
  ++c->launches;
  return MVD_OK;
}

XArgs x_args(mvd_ctx* c, const float2* in, float2* out, int rx) {
  const Plan& P = c->P;
  XArgs a{};
  a.in = in; a.out = out; a.tw = c->twx();
  a.rows_per_cta = P.Rx; a.nthreads = P.ntx;
  a.nrows = (long long)P.N[1] * P.N[2];
  a.ny_rows = P.N[1];
  a.plane_pitch = P.plane;
  a.nx = P.N[0]; a.hx = P.hx; a.rx = rx;
  a.psi = c->psi(); a.acc = c->acc(); a.partials = c->partials();
  a.eps = c->eps; a.psi_floor = c->psi_floor; a.inv_nviews = 1.0f / (float)P.V;
  a.tikhonov = c->tikhonov;
  a.root_each = (!c->literal && P.V > kRootEachViews) ? 1 : 0;
  a.literal_product = c->literal;
  return a;
}

mvd_status x_pass(mvd_ctx* c, const XArgs& a_in, int mode) {
  static const int cls[5] = {MVD_K_X_LOAD, MVD_K_X_QUOT, MVD_K_X_UPDATE, MVD_K_X_ACCUM, MVD_K_X_UPDATE};
  const Plan& P = c->P;
  XArgs a = a_in;
  const bool tma = P.xtma && (mode == X_QUOT || mode == X_UPDATE || mode == X_UPDATE_W || (mode == X_ACCUM && a_in.acc_mode != ACC_STORE));
  if (tma) {
    // persistent CTAs, tiles of Rxt rows staged by bulk copies (pass_tma.cuh)
    a.rows_per_cta = P.Rxt;
    a.nthreads = P.ntxt;
    a.real_stride = P.xt_rstride;
    a.reverse = c->use_flip ? (c->flip ^= 1) : 0;
    a.exch_stride = P.xt_exch; a.exch_stride_g = P.xt_exch_g; a.exch_stride_f = P.xt_exch_f;
    const float* real_src = mode == X_QUOT ? a.phi : (mode == X_ACCUM ? a.acc : a.psi);
    // 1: every row of the real arrays is 16-byte aligned; 2: rows staged from the aligned address below them
    a.bulk_real = ((P.N[0] % 4 == 0) && ((reinterpret_cast<size_t>(real_src) & 15) == 0) &&
                   ((reinterpret_cast<size_t>(a.wts) & 15) == 0)) ? 1 : 2;
    if (!c->xbulk) a.bulk_real = 0;
    const int flags = P.lx->xrow_tma_flags(a, mode) & 3;
    int& bl = c->xt_blocks[mode][flags];
    if (bl == 0) {
      bl = P.lx->xrow_tma_blocks_per_sm(mode, flags, a.nthreads, P.lx->xrow_tma_smem(a.rows_per_cta, P.r[0], P.N[0], mode == X_UPDATE_W));
      if (bl <= 0) { snprintf(c->err, sizeof(c->err), "x pass: kernel does not fit on an SM"); c->broken = true; return MVD_ERR_CUDA; }
    }
    const long long ntiles = (a.nrows + a.rows_per_cta - 1) / a.rows_per_cta;
    a.grid = (int)std::min<long long>(std::min<long long>(ntiles, (long long)c->num_sms * bl), P.sum_blocks);
    {
      ProfScope ps(c, cls[mode]);
      MVD_CK(P.lx->xrow_tma(a, mode, c->stream), "x pass (TMA)");
    }
  } else {
    ProfScope ps(c, cls[mode]);
    MVD_CK(P.lx->xrow(a, mode, c->stream), "x pass");
  }
  ++c->launches;
  if (mode == X_UPDATE || mode == X_UPDATE_W || (mode == X_ACCUM && (a.acc_mode == ACC_LAST || a.acc_mode == ACC_ONLY))) {
    c->stats_valid = true;
    c->stats_ncta = tma ? a.grid : (int)((a.nrows + a.rows_per_cta - 1) / a.rows_per_cta);
  }
  return MVD_OK;
}

mvd_status x_load(mvd_ctx* c, const float* src, float2* out) {
  XArgs a = x_args(c, nullptr, out, 0);
  a.phi = src;
  return x_pass(c, a, X_LOAD);
}

#define MVD_TRY(expr) do { mvd_status s_ = (expr); if (s_ != MVD_OK) return s_; } while (0)

// crop(src (*) kernel) with the forward transform of src already in `buf` rows: y, z, y passes
mvd_status conv_core(mvd_ctx* c, const float2* in, float2* buf, const float2* spec, bool skip_yfwd) {
  if (!skip_yfwd) MVD_TRY(y_pass(c, buf, -1, c->P.N[2], false));
  MVD_TRY(z_conv(c, in ? in : buf, buf, spec));
  MVD_TRY(y_pass(c, buf, +1, c->P.N[2], false));
  return MVD_OK;
}

// one iteration (every view contributes once, L817); requires w_valid
mvd_status iteration_body(mvd_ctx* c) {
  const Plan& P = c->P;
  if (!P.combined) {
    // eq. 109-112: psi updated after every view, index order (R11)
    for (int v = 0; v < P.V; ++v) {
      const int rx = (P.K[v].x - 1) / 2;
      MVD_TRY(conv_core(c, nullptr, c->W(), c->specH(v), false));
      XArgs q = x_args(c, c->W(), c->W(), rx);
      q.phi = c->views[v];
      MVD_TRY(x_pass(c, q, X_QUOT));
      MVD_TRY(conv_core(c, nullptr, c->W(), c->specK(v), false));
      XArgs u = x_args(c, c->W(), c->W(), rx);
      u.wts = c->weights.empty() ? nullptr : c->weights[v];
      MVD_TRY(x_pass(c, u, u.wts ? X_UPDATE_W : X_UPDATE));
    }
  } else {
    // eq. 70 / 104: every f_v from the same psi; the x and y forward passes of psi are shared
    MVD_TRY(y_pass(c, c->W0(), -1, P.N[2], false));
    for (int v = 0; v < P.V; ++v) {
      const int rx = (P.K[v].x - 1) / 2;
      MVD_TRY(conv_core(c, c->W0(), c->W(), c->specH(v), true));
      XArgs q = x_args(c, c->W(), c->W(), rx);
      q.phi = c->views[v];
      MVD_TRY(x_pass(c, q, X_QUOT));
      MVD_TRY(conv_core(c, nullptr, c->W(), c->specK(v), false));
      XArgs u = x_args(c, c->W(), c->W0(), rx);
      u.acc_mode = P.V == 1 ? ACC_ONLY : (v == 0 ? ACC_FIRST : (v == P.V - 1 ? ACC_LAST : ACC_MID));
      MVD_TRY(x_pass(c, u, X_ACCUM));
    }
  }
  return MVD_OK;
}

mvd_status ensure_w(mvd_ctx* c) {
  if (c->w_valid) return MVD_OK;
  MVD_TRY(x_load(c, c->psi(), c->P.combined ? c->W0() : c->W()));
  c->w_valid = true;
  return MVD_OK;
}

// ---- pinned staging buffer of the PSF taps (process-wide, grow-only) -----------------------------
std::mutex g_staging_mutex;
char* g_staging = nullptr;
size_t g_staging_bytes = 0;

char* staging_acquire(size_t bytes) {
  g_staging_mutex.lock();
  if (bytes > g_staging_bytes) {
    if (g_staging) cudaFreeHost(g_staging);
    g_staging = nullptr;
    g_staging_bytes = 0;
    const size_t want = std::max(bytes, (size_t)1 << 20);
    if (cudaHostAlloc(reinterpret_cast<void**>(&g_staging), want, cudaHostAllocMapped | cudaHostAllocPortable) != cudaSuccess) {
      cudaGetLastError();
      g_staging = nullptr;
      g_staging_mutex.unlock();
      return nullptr;
    }
    g_staging_bytes = want;
  }
  return g_staging;
}
void staging_release() { g_staging_mutex.unlock(); }

// ---- precompute (S0) ---------------------------------------------------------------------------
mvd_status build_spectrum(mvd_ctx* c, const double* kern, Dims3 K, float2* spec) {
  const Plan& P = c->P;
  MVD_CK(cudaMemsetAsync(spec, 0, (size_t)P.ssize * sizeof(float2), c->stream), "memset spectrum");
  const long long tot = (long long)K.x * K.y * K.z;
  const double scale = 1.0 / ((double)P.Mx * (double)P.My * (double)P.Mz);
  scatter_kernel<<<(unsigned)((tot + 255) / 256), 256, 0, c->stream>>>(kern, K, spec,
                                                                        Dims3{P.Mx, P.My, P.Mz}, scale);
  MVD_CK(cudaGetLastError(), "scatter_kernel");
  ++c->launches;
  // The taps sit (wrapped) in the planes z in [0, cz] and [Mz-cz, Mz) and, there, in the rows y in [0, cy] and
  // [My-cy, My): the x pass only visits those rows, the y pass only those planes; the z pass sees the whole buffer.
  const int cz = (K.z - 1) / 2, cy = (K.y - 1) / 2;
  int zr[2][2] = {{0, std::min(cz + 1, P.Mz)}, {std::max(P.Mz - cz, cz + 1), P.Mz}};   // [z0, z1)
  int yr[2][2] = {{0, std::min(cy + 1, P.My)}, {std::max(P.My - cy, cy + 1), P.My}};
  for (int iz = 0; iz < 2; ++iz) {
    const int z0 = zr[iz][0], nz = zr[iz][1] - z0;
    if (nz <= 0) continue;
    float2* zbase = spec + (long long)z0 * P.plane;
    // x: complex rows, in place
    for (int iy = 0; iy < 2; ++iy) {
      const int y0 = yr[iy][0], ny = yr[iy][1] - y0;
      if (ny <= 0) continue;
      XArgs a = x_args(c, zbase + (long long)y0 * P.Mx, zbase + (long long)y0 * P.Mx, 0);
      a.nrows = (long long)ny * nz;
      a.ny_rows = ny;
      a.complex_in = 1;
      MVD_TRY(x_pass(c, a, X_LOAD));
    }
    // y: full pencils of these planes
    StridedArgs s{};
    s.in = zbase; s.out = zbase; s.tw = c->twy();
    s.T = P.Tys; s.nthreads = P.ntys;
    s.line_len = P.Mx; s.tiles_per_line = (P.Mx + s.T - 1) / s.T;
    s.n_outer = nz;
    s.in_outer_stride = s.out_outer_stride = P.plane;
    s.in_pstride = s.out_pstride = P.Mx;
    s.n_in = P.My; s.n_out = P.My;
    MVD_CK(P.ly->strided(s, -1, c->stream), "y pass (spectrum)");
    ++c->launches;
  }
  MVD_TRY(z_plain_fwd(c, spec));
  return MVD_OK;
}

// shared_kern: the back-projectors K_v of an earlier context of the same problem (blocked mode: one
// context per block shape, same PSFs), V * psf_stride doubles on the device; NULL -> compute them
mvd_status precompute(mvd_ctx* c, const float* const* psfs_host, const double* shared_kern) {
  const Plan& P = c->P;
  // twiddle tables, generated on the device in double.  mvd_create issues NO host-to-device copy: a copy would
  // queue on the copy engine behind the caller's (possibly still running) upload of the views and serialise the
  // whole precompute with it (measured: 34 ms of H2D + 31 ms of precompute instead of max of the two)
  {
    const int M[3] = {P.Mx, P.My, P.Mz};
    float2* dst[3] = {c->twx(), c->twy(), c->twz()};
    for (int a = 0; a < 3; ++a) {
      twiddle_kernel<<<(M[a] + 255) / 256, 256, 0, c->stream>>>(dst[a], M[a]);
      MVD_CK(cudaGetLastError(), "twiddle_kernel");
      ++c->launches;
    }
  }
  // normalised PSFs in fp64 (eq. 4): the taps are staged in pinned host memory that the device reads in place
  {
    size_t total = 0;
    for (int v = 0; v < P.V; ++v) total += align_up((size_t)P.K[v].x * P.K[v].y * P.K[v].z * sizeof(float), 256);
    // one grow-only pinned buffer per process, handed from one mvd_create to the next (allocating and freeing
    // mapped pinned memory per context cost tens of milliseconds now and then: the block-wise mode creates a context
    // per block shape); held under a lock until the last normalise kernel has read it (event below), so that
    // concurrent mvd_create calls of per-GPU threads serialise on this short section only
    c->psf_staging = staging_acquire(total);
    if (!c->psf_staging) { snprintf(c->err, sizeof(c->err), "pinned PSF staging: allocation failed"); return MVD_ERR_CUDA; }
    char* dev_base = nullptr;
    MVD_CK(cudaHostGetDevicePointer(reinterpret_cast<void**>(&dev_base), c->psf_staging, 0), "pinned PSF staging");
    size_t off = 0;
    for (int v = 0; v < P.V; ++v) {
      const Dims3 K = P.K[v];
      const int n = K.x * K.y * K.z;
      double hsum = 0.0;
      for (int i = 0; i < n; ++i) {
        const float t = psfs_host[v][i];
        if (!(t >= 0.f) || !std::isfinite(t)) { snprintf(c->err, sizeof(c->err), "PSF %d has a negative or non-finite tap", v); return MVD_ERR_INVALID_ARG; }
        hsum += t;
      }
      if (!(hsum > 0.0)) { snprintf(c->err, sizeof(c->err), "PSF %d sums to zero", v); return MVD_ERR_INVALID_ARG; }
      memcpy(c->psf_staging + off, psfs_host[v], sizeof(float) * n);
      normalise_kernel<float><<<1, 1024, 0, c->stream>>>(reinterpret_cast<const float*>(dev_base + off), n, c->psf(v));
      MVD_CK(cudaGetLastError(), "normalise_kernel");
      ++c->launches;
      off += align_up(sizeof(float) * n, 256);
    }
    MVD_CK(cudaEventCreateWithFlags(&c->staged_read, cudaEventDisableTiming), "staging event");
    MVD_CK(cudaEventRecord(c->staged_read, c->stream), "staging event");
  }
  // back-projectors K_v (O3)
  if (shared_kern) {
    MVD_CK(cudaMemcpyAsync(c->kern(0), shared_kern, sizeof(double) * P.psf_stride * P.V, cudaMemcpyDeviceToDevice, c->stream),
           "back-projector copy");
  }
  if (!shared_kern && P.kmode == MVD_KERNEL_COMPOUND) {
    for (int w = 0; w < P.V; ++w) {
      const Dims3 K = P.K[w];
      const long long tot = (long long)(2 * K.x - 1) * (2 * K.y - 1) * (2 * K.z - 1);
      if (2 * K.x - 1 <= 128 && c->corr_tiled)   // P_w (*) P_w* = sum_u P[K-1-u] P[m - u] read backwards (symmetric)
        corr_crop_mul_tiled_kernel<<<(unsigned)((2 * K.y - 1) * (2 * K.z - 1)), 128, 0, c->stream>>>(
            c->psf(w), K, c->psf(w), K, c->autoc(w), Dims3{2 * K.x - 1, 2 * K.y - 1, 2 * K.z - 1}, Dims3{0, 0, 0}, 1);
      else
        autocorr_kernel<<<(unsigned)((tot + 127) / 128), 128, 0, c->stream>>>(c->psf(w), K, c->autoc(w));
      MVD_CK(cudaGetLastError(), "autocorr_kernel");
      ++c->launches;
    }
  }
  for (int v = 0; v < P.V; ++v) {
    if (!c->is_local[v] || shared_kern) continue;
    const Dims3 K = P.K[v];
    const long long tot = (long long)K.x * K.y * K.z;
    const unsigned g256 = (unsigned)((tot + 255) / 256), g128 = (unsigned)((tot + 31) / 32);   // corr: one block of 256 threads per 32 taps
    flip_pow_kernel<<<g256, 256, 0, c->stream>>>(c->psf(v), K, P.kmode == MVD_KERNEL_OPT2 ? P.V : 1, c->kern(v));
    MVD_CK(cudaGetLastError(), "flip_pow_kernel");
    ++c->launches;
    if (P.kmode == MVD_KERNEL_COMPOUND || P.kmode == MVD_KERNEL_OPT1) {
      for (int w = 0; w < P.V; ++w) {
        if (w == v) continue;
        const Dims3 Kw = P.K[w];
        const double* gsrc = P.kmode == MVD_KERNEL_COMPOUND ? c->autoc(w) : c->psf(w);
        const Dims3 gd = P.kmode == MVD_KERNEL_COMPOUND ? Dims3{2 * Kw.x - 1, 2 * Kw.y - 1, 2 * Kw.z - 1} : Kw;
        if (K.x <= 128 && c->corr_tiled)
          corr_crop_mul_tiled_kernel<<<(unsigned)(K.y * K.z), 128, 0, c->stream>>>(
              c->psf(v), K, gsrc, gd, c->kern(v), K, Dims3{(gd.x - 1) / 2, (gd.y - 1) / 2, (gd.z - 1) / 2}, 0);
        else
          corr_crop_mul_kernel<<<g128, 256, 0, c->stream>>>(c->psf(v), K, gsrc, gd, c->kern(v));
        MVD_CK(cudaGetLastError(), "corr_crop_mul_kernel");
        ++c->launches;
      }
    }
    if (P.kmode != MVD_KERNEL_PLAIN) {
      normalise_kernel<double><<<1, 1024, 0, c->stream>>>(c->kern(v), (int)tot, c->kern(v));   // R5
      MVD_CK(cudaGetLastError(), "normalise_kernel");
      ++c->launches;
    }
  }
  // spectra of P_v and K_v
  for (int v = 0; v < P.V; ++v) {
    if (!c->is_local[v]) continue;
    MVD_TRY(build_spectrum(c, c->psf(v), P.K[v], c->specH(v)));
    MVD_TRY(build_spectrum(c, c->kern(v), P.K[v], c->specK(v)));
  }
  return MVD_OK;
}

mvd_status init_estimate(mvd_ctx* c, const float* psi0) {
  const Plan& P = c->P;
  if (psi0) {
    MVD_CK(cudaMemcpyAsync(c->psi(), psi0, sizeof(float) * P.nvox, cudaMemcpyDeviceToDevice, c->stream), "psi0 copy");
  } else if (c->psi0_value > 0.f) {
    fill_value_kernel<<<P.sum_blocks, 256, 0, c->stream>>>(c->psi(), P.nvox, c->psi0_value);
    MVD_CK(cudaGetLastError(), "fill_value_kernel");
    ++c->launches;
  } else if (c->partial) {
    snprintf(c->err, sizeof(c->err), "a view-parallel context needs psi0 or psi0_value");
    return MVD_ERR_INVALID_ARG;
  } else {
    // psi^0 = average intensity over all views (L304, L421)
    for (int v = 0; v < P.V; ++v) {
      sum_f32_kernel<<<P.sum_blocks, 256, 0, c->stream>>>(c->views[v], P.nvox, c->partials());
      MVD_CK(cudaGetLastError(), "sum_f32_kernel");
      final_sum_kernel<<<1, 256, 0, c->stream>>>(c->partials(), P.sum_blocks, 1, c->scalars() + v);
      MVD_CK(cudaGetLastError(), "final_sum_kernel");
      c->launches += 2;
    }
    fill_mean_kernel<<<P.sum_blocks, 256, 0, c->stream>>>(c->psi(), P.nvox, c->scalars(), P.V, (double)P.nvox * P.V);
    MVD_CK(cudaGetLastError(), "fill_mean_kernel");
    ++c->launches;
  }
  c->w_valid = false;
  c->stats_valid = false;
  return MVD_OK;
}

const mvd_options* defaults(const mvd_options* opt, mvd_options* tmp) {
  mvd_options_init(tmp);
  if (opt) {
    const size_t n = std::min(opt->struct_size, sizeof(mvd_options));
    if (n >= sizeof(size_t)) memcpy(tmp, opt, n);
    tmp->struct_size = sizeof(mvd_options);
  }
  return tmp;
}

}  // namespace

// ---------------------------------------------------------------------------------------
// C ABI
// ---------------------------------------------------------------------------------------
extern "C" {

void mvd_options_init(mvd_options* opt) {
  if (!opt) return;
  memset(opt, 0, sizeof(*opt));
  opt->struct_size = sizeof(*opt);
  opt->eps = 1e-6f;
  opt->psi_floor = 1e-6f;
}

size_t mvd_workspace_size(int n_views, const int dims[3], const int (*psf_dims)[3],
                          mvd_variant variant, const mvd_options* opt) {
  mvd_options tmp;
  Plan P;
  if (make_plan(P, n_views, dims, psf_dims, variant, defaults(opt, &tmp)) != MVD_OK) return 0;
  return P.total;
}

mvd_status mvd_plan_dims(int n_views, const int dims[3], const int (*psf_dims)[3],
                         const mvd_options* opt, int fft_dims_out[3]) {
  if (!fft_dims_out) return MVD_ERR_INVALID_ARG;
  mvd_options tmp;
  Plan P;
  mvd_status s = make_plan(P, n_views, dims, psf_dims, MVD_OSEM, defaults(opt, &tmp));
  if (s != MVD_OK) return s;
  fft_dims_out[0] = P.Mx; fft_dims_out[1] = P.My; fft_dims_out[2] = P.Mz;
  return MVD_OK;
}

static mvd_status create_impl(mvd_ctx** out, int n_views, const float* const* views, const int dims[3],
                              const float* const* psfs, const int (*psf_dims)[3], mvd_variant variant,
                              const mvd_options* opt_in, const double* shared_kern);

mvd_status mvd_create(mvd_ctx** out, int n_views, const float* const* views, const int dims[3],
                      const float* const* psfs, const int (*psf_dims)[3], mvd_variant variant,
                      const mvd_options* opt_in) {
  return create_impl(out, n_views, views, dims, psfs, psf_dims, variant, opt_in, nullptr);
}

static mvd_status create_impl(mvd_ctx** out, int n_views, const float* const* views, const int dims[3],
                              const float* const* psfs, const int (*psf_dims)[3], mvd_variant variant,
                              const mvd_options* opt_in, const double* shared_kern) {
  if (!out) return MVD_ERR_INVALID_ARG;
  *out = nullptr;
  if (!views || !psfs || !dims || !psf_dims || !opt_in) return MVD_ERR_INVALID_ARG;
  mvd_options tmp;
  const mvd_options* opt = defaults(opt_in, &tmp);
  if (n_views < 1) return MVD_ERR_INVALID_ARG;
  std::vector<char> is_local((size_t)n_views, opt->local_views ? 0 : 1);
  if (opt->local_views) {
    if (variant == MVD_OSEM) return MVD_ERR_UNSUPPORTED;      // sequential updates do not split over ranks
    if (opt->n_local < 1 || opt->weights) return MVD_ERR_INVALID_ARG;
    for (int i = 0; i < opt->n_local; ++i) {
      const int v = opt->local_views[i];
      if (v < 0 || v >= n_views || is_local[v] || (i > 0 && v <= opt->local_views[i - 1])) return MVD_ERR_INVALID_ARG;
      is_local[v] = 1;
    }
  }
  for (int v = 0; v < n_views; ++v)
    if ((is_local[v] && !views[v]) || !psfs[v]) return MVD_ERR_INVALID_ARG;
  mvd_ctx* c = new (std::nothrow) mvd_ctx();
  if (!c) return MVD_ERR_INVALID_ARG;
  c->is_local = is_local;
  c->partial = opt->local_views != nullptr;
  c->psi0_value = opt->psi0_value;
  mvd_status s = make_plan(c->P, n_views, dims, psf_dims, variant, opt);
  if (s != MVD_OK) { delete c; return s; }
  if (!opt->workspace || (reinterpret_cast<size_t>(opt->workspace) & 255) || opt->workspace_bytes < c->P.total) {
    delete c;
    return MVD_ERR_WORKSPACE;
  }
  c->variant = variant;
  c->literal = opt->literal_product ? 1 : 0;
  c->eps = opt->eps > 0.f ? opt->eps : 1e-6f;
  c->psi_floor = opt->psi_floor >= 0.f ? opt->psi_floor : 1e-6f;
  if (!(opt->tikhonov_lambda >= 0.f) || !std::isfinite(opt->tikhonov_lambda)) { delete c; return MVD_ERR_INVALID_ARG; }
  c->tikhonov = opt->tikhonov_lambda;
  c->stream = reinterpret_cast<cudaStream_t>(opt->stream);
  c->ws = reinterpret_cast<char*>(opt->workspace);
  c->use_graph = opt->use_graph;
  const Tune tune;
  c->use_flip = tune.get("flip", 1);
  {   // measured: 1050-point pencils (one CTA per SM) 937 -> 887 us per launch; 525-point pencils 110 -> 112 us
    const int yp = tune.get("ypair", -1);
    c->y_pair = yp < 0 ? (c->P.My >= 1000 ? 1 : 0) : (yp ? 1 : 0);
  }
  c->corr_tiled = tune.get("corr_tiled", 1);
  c->xbulk = tune.get("xbulk", 1);
  c->ztx = tune.get("ztx", 16) == 8 ? 8 : 16;   // 16 x 1 measured faster than 8 x 2 on configs 2-5
  if (c->use_graph && !c->stream) {   // the legacy default stream cannot be captured
    fprintf(stderr, "mvd_create: use_graph needs a non-default stream\n");
    delete c;
    return MVD_ERR_UNSUPPORTED;
  }
  c->views.assign(views, views + n_views);
  if (opt->weights && !c->P.xtma) {   // only the TMA-staged update applies weights
    delete c;
    return MVD_ERR_UNSUPPORTED;
  }
  if (opt->weights) {
    for (int v = 0; v < n_views; ++v)
      if (!opt->weights[v]) { delete c; return MVD_ERR_INVALID_ARG; }
    c->weights.assign(opt->weights, opt->weights + n_views);
  }

  cudaError_t e = cudaSuccess;
  {
    int dev = 0;
    if (cudaGetDevice(&dev) == cudaSuccess) cudaDeviceGetAttribute(&c->num_sms, cudaDevAttrMultiProcessorCount, dev);
  }
  const LengthOps* ls[3] = {c->P.lx, c->P.ly, c->P.lz};
  for (int a = 0; a < 3 && e == cudaSuccess; ++a) e = ls[a]->init();
  if (e == cudaSuccess) e = cudaStreamSynchronize(c->stream);
  if (e != cudaSuccess) {
    fprintf(stderr, "mvd_create: kernel attribute setup failed: %s\n", cudaGetErrorString(e));
    delete c;
    return MVD_ERR_CUDA;
  }

  s = precompute(c, psfs, shared_kern);
  if (c->psf_staging) {
    // the kernels that read the staged taps are the first of the precompute: normally long done by now.
    // No event (an early failure) -> wait for the whole stream
    if (!c->staged_read || cudaEventSynchronize(c->staged_read) != cudaSuccess) cudaStreamSynchronize(c->stream);
    staging_release();
    c->psf_staging = nullptr;
  }
  if (c->staged_read) { cudaEventDestroy(c->staged_read); c->staged_read = nullptr; }
  if (s == MVD_OK && opt->views_ready &&
      c->fail(cudaStreamWaitEvent(c->stream, reinterpret_cast<cudaEvent_t>(opt->views_ready), 0), "views_ready"))
    s = MVD_ERR_CUDA;
  c->psi0_ptr = opt->psi0;
  if (s == MVD_OK) s = init_estimate(c, opt->psi0);
  if (s == MVD_OK && c->fail(cudaStreamSynchronize(c->stream), "mvd_create")) s = MVD_ERR_CUDA;
  if (s != MVD_OK) {
    if (c->err[0]) fprintf(stderr, "mvd_create: %s\n", c->err);
    delete c;
    return s;
  }
  *out = c;
  return MVD_OK;
}

mvd_status mvd_iterate(mvd_ctx* c, int n) {
  if (!c || n < 0) return MVD_ERR_INVALID_ARG;
  if (c->broken) return MVD_ERR_STATE;
  if (c->partial) {   // view-parallel contexts advance through mvd_partial_product / mvd_apply_product
    snprintf(c->err, sizeof(c->err), "view-parallel context: use mvd_partial_product / mvd_apply_product");
    return MVD_ERR_STATE;
  }
  if (n == 0) return MVD_OK;
  MVD_TRY(ensure_w(c));
  if (c->use_graph) {
    if (!c->graph_exec) {
      cudaGraph_t g = nullptr;
      const long long before = c->launches;
      MVD_CK(cudaStreamBeginCapture(c->stream, cudaStreamCaptureModeThreadLocal), "graph capture begin");
      mvd_status s = iteration_body(c);
      cudaError_t e = cudaStreamEndCapture(c->stream, &g);
      if (s != MVD_OK || e != cudaSuccess) {
        if (g) cudaGraphDestroy(g);
        if (s != MVD_OK) return s;
      }
      MVD_CK(e, "graph capture end");
      c->graph_launches = c->launches - before;
      c->launches = before;
      c->graph_stats_ncta = c->stats_ncta;
      e = cudaGraphInstantiate(&c->graph_exec, g, 0);
      cudaGraphDestroy(g);
      MVD_CK(e, "graph instantiate");
    }
    for (int i = 0; i < n; ++i) {
      MVD_CK(cudaGraphLaunch(c->graph_exec, c->stream), "graph launch");
      c->launches += c->graph_launches;
      ++c->iters;
    }
    // the replayed update kernel wrote its partials: same statistics as the plain launches
    c->stats_valid = true;
    c->stats_ncta = c->graph_stats_ncta;
    return MVD_OK;
  }
  for (int i = 0; i < n; ++i) {
    MVD_TRY(iteration_body(c));
    ++c->iters;
  }
  return MVD_OK;
}

mvd_status mvd_compare(mvd_ctx* c, const float* ref, double* avg_diff, double* xcorr) {
  if (!c || !ref) return MVD_ERR_INVALID_ARG;
  if (c->broken) return MVD_ERR_STATE;
  const Plan& P = c->P;
  const int nb = 192;
  double* part = reinterpret_cast<double*>(c->ws + P.off_cmp);
  compare_kernel<<<nb, 256, 0, c->stream>>>(c->psi(), ref, P.nvox, part);
  MVD_CK(cudaGetLastError(), "compare_kernel");
  final_sum_kernel<<<1, 256, 0, c->stream>>>(part, nb, 6, part + 6 * nb);
  MVD_CK(cudaGetLastError(), "final_sum_kernel");
  c->launches += 2;
  double h[6];
  MVD_CK(cudaMemcpyAsync(h, part + 6 * nb, sizeof(h), cudaMemcpyDeviceToHost, c->stream), "compare copy");
  MVD_CK(cudaStreamSynchronize(c->stream), "compare copy");
  const double n = (double)P.nvox;
  if (avg_diff) *avg_diff = h[0] / n;
  if (xcorr) {
    const double cov = h[5] - h[1] * h[2] / n, va = h[3] - h[1] * h[1] / n, vr = h[4] - h[2] * h[2] / n;
    *xcorr = (va > 0.0 && vr > 0.0) ? cov / sqrt(va * vr) : 0.0;
  }
  return MVD_OK;
}

mvd_status mvd_partial_product(mvd_ctx* c) {
  if (!c) return MVD_ERR_INVALID_ARG;
  if (c->broken) return MVD_ERR_STATE;
  const Plan& P = c->P;
  if (!P.combined) return MVD_ERR_UNSUPPORTED;
  MVD_TRY(ensure_w(c));
  // eq. 70 / 104: every f_v of this context's views from the same psi; the x and y forward passes of psi are shared
  MVD_TRY(y_pass(c, c->W0(), -1, P.N[2], false));
  bool first = true;
  for (int v = 0; v < P.V; ++v) {
    if (!c->is_local[v]) continue;
    const int rx = (P.K[v].x - 1) / 2;
    MVD_TRY(conv_core(c, c->W0(), c->W(), c->specH(v), true));
    XArgs q = x_args(c, c->W(), c->W(), rx);
    q.phi = c->views[v];
    MVD_TRY(x_pass(c, q, X_QUOT));
    MVD_TRY(conv_core(c, nullptr, c->W(), c->specK(v), false));
    XArgs u = x_args(c, c->W(), c->W0(), rx);
    u.acc_mode = first ? ACC_FIRST : ACC_MID;
    first = false;
    MVD_TRY(x_pass(c, u, X_ACCUM));
  }
  c->w_valid = false;            // the y pass ran in place on W0: it no longer holds the x transform of psi
  return MVD_OK;
}

mvd_status mvd_get_product(mvd_ctx* c, float** acc_device) {
  if (!c || !acc_device) return MVD_ERR_INVALID_ARG;
  *acc_device = c->acc();
  return MVD_OK;
}

mvd_status mvd_apply_product(mvd_ctx* c, int total_views) {
  if (!c || total_views < 1) return MVD_ERR_INVALID_ARG;
  if (c->broken) return MVD_ERR_STATE;
  const Plan& P = c->P;
  if (!P.combined) return MVD_ERR_UNSUPPORTED;
  // with more than kRootEachViews views the factors were rooted one by one (x pass): no root left to take here
  const int no_root = c->literal || (!c->literal && P.V > kRootEachViews);
  apply_product_kernel<<<P.sum_blocks, 256, 0, c->stream>>>(c->psi(), c->acc(), P.nvox, 1.0f / (float)total_views,
                                                          no_root, c->psi_floor, c->tikhonov, c->partials());
  MVD_CK(cudaGetLastError(), "apply_product_kernel");
  ++c->launches;
  c->w_valid = false;
  c->stats_valid = true;
  c->stats_ncta = P.sum_blocks;
  ++c->iters;
  return MVD_OK;
}

// the scratch layout does not depend on the device that happens to be current: kMaxReduceBlocks partials + the total
static constexpr int kMaxReduceBlocks = 2048;
size_t mvd_reduce_scratch_bytes(void) { return sizeof(double) * (size_t)(kMaxReduceBlocks + 8); }

mvd_status mvd_reduce_sum(const float* src, long long n, void* scratch, void* stream, double* host_out) {
  if (!src || n < 0 || !scratch || !host_out) return MVD_ERR_INVALID_ARG;
  cudaStream_t st = reinterpret_cast<cudaStream_t>(stream);
  double* part = reinterpret_cast<double*>(scratch);
  const int nb = std::min(mvd::reduce_blocks(), kMaxReduceBlocks);
  sum_f32_kernel<<<nb, 256, 0, st>>>(src, n, part);
  if (cudaGetLastError() != cudaSuccess) return MVD_ERR_CUDA;
  final_sum_kernel<<<1, 256, 0, st>>>(part, nb, 1, part + nb);
  if (cudaGetLastError() != cudaSuccess) return MVD_ERR_CUDA;
  if (cudaMemcpyAsync(host_out, part + nb, sizeof(double), cudaMemcpyDeviceToHost, st) != cudaSuccess ||
      cudaStreamSynchronize(st) != cudaSuccess)
    return MVD_ERR_CUDA;
  return MVD_OK;
}

mvd_status mvd_get_estimate(mvd_ctx* c, float* dst, int dst_is_device) {
  if (!c || !dst) return MVD_ERR_INVALID_ARG;
  if (c->broken) return MVD_ERR_STATE;
  const size_t bytes = sizeof(float) * (size_t)c->P.nvox;
  if (dst_is_device) {
    MVD_CK(cudaMemcpyAsync(dst, c->psi(), bytes, cudaMemcpyDeviceToDevice, c->stream), "estimate copy");
  } else {
    MVD_CK(cudaMemcpyAsync(dst, c->psi(), bytes, cudaMemcpyDeviceToHost, c->stream), "estimate copy");
    MVD_CK(cudaStreamSynchronize(c->stream), "estimate copy");
  }
  return MVD_OK;
}

mvd_status mvd_set_estimate(mvd_ctx* c, const float* src_device) {
  if (!c || !src_device) return MVD_ERR_INVALID_ARG;
  if (c->broken) return MVD_ERR_STATE;
  MVD_CK(cudaMemcpyAsync(c->psi(), src_device, sizeof(float) * (size_t)c->P.nvox, cudaMemcpyDeviceToDevice, c->stream), "estimate copy");
  c->w_valid = false;
  c->stats_valid = false;
  return MVD_OK;
}

mvd_status mvd_restart(mvd_ctx* c, void* views_ready) {
  if (!c) return MVD_ERR_INVALID_ARG;
  if (c->broken) return MVD_ERR_STATE;
  if (views_ready) MVD_CK(cudaStreamWaitEvent(c->stream, reinterpret_cast<cudaEvent_t>(views_ready), 0), "views_ready");
  MVD_TRY(init_estimate(c, c->psi0_ptr));
  c->iters = 0;
  return MVD_OK;
}

mvd_status mvd_get_stats(mvd_ctx* c, double* flux, double* l1_change, int* iterations_done) {
  if (!c) return MVD_ERR_INVALID_ARG;
  if (c->broken) return MVD_ERR_STATE;
  double h[2] = {0.0, 0.0};
  double* d = c->scalars() + c->P.V;
  if (c->stats_valid) {
    final_sum_kernel<<<1, 256, 0, c->stream>>>(c->partials(), c->stats_ncta, 2, d);
    MVD_CK(cudaGetLastError(), "final_sum_kernel");
    ++c->launches;
  } else {
    // no update yet: flux of the current estimate, no change
    sum_f32_kernel<<<c->P.sum_blocks, 256, 0, c->stream>>>(c->psi(), c->P.nvox, c->partials());
    MVD_CK(cudaGetLastError(), "sum_f32_kernel");
    final_sum_kernel<<<1, 256, 0, c->stream>>>(c->partials(), c->P.sum_blocks, 1, d);
    MVD_CK(cudaGetLastError(), "final_sum_kernel");
    MVD_CK(cudaMemsetAsync(d + 1, 0, sizeof(double), c->stream), "memset");
    c->launches += 2;
  }
  MVD_CK(cudaMemcpyAsync(h, d, sizeof(h), cudaMemcpyDeviceToHost, c->stream), "stats copy");
  MVD_CK(cudaStreamSynchronize(c->stream), "stats copy");
  if (flux) *flux = h[0];
  if (l1_change) *l1_change = h[1];
  if (iterations_done) *iterations_done = c->iters;
  return MVD_OK;
}

mvd_status mvd_get_back_projector(mvd_ctx* c, int view, double* dst_host) {
  if (!c || !dst_host || view < 0 || view >= c->P.V) return MVD_ERR_INVALID_ARG;
  if (c->broken) return MVD_ERR_STATE;
  const Dims3 K = c->P.K[view];
  MVD_CK(cudaMemcpyAsync(dst_host, c->kern(view), sizeof(double) * (size_t)K.x * K.y * K.z, cudaMemcpyDeviceToHost, c->stream), "kernel copy");
  MVD_CK(cudaStreamSynchronize(c->stream), "kernel copy");
  return MVD_OK;
}

mvd_status mvd_convolve(mvd_ctx* c, int view, int which, const float* src, float* dst) {
  if (!c || !src || !dst || view < 0 || view >= c->P.V || which < 0 || which > 1) return MVD_ERR_INVALID_ARG;
  if (c->broken) return MVD_ERR_STATE;
  if (!c->is_local[view]) {   // view-parallel context: no spectra were built for views of other ranks
    snprintf(c->err, sizeof(c->err), "view %d belongs to another rank of this view-parallel context", view);
    return MVD_ERR_INVALID_ARG;
  }
  c->w_valid = false;
  MVD_TRY(x_load(c, src, c->W()));
  MVD_TRY(conv_core(c, nullptr, c->W(), which ? c->specK(view) : c->specH(view), false));
  XArgs a = x_args(c, c->W(), c->W(), (c->P.K[view].x - 1) / 2);
  a.acc = dst;
  a.acc_mode = ACC_STORE;
  return x_pass(c, a, X_ACCUM);
}

long long mvd_launch_count(const mvd_ctx* c) { return c ? c->launches : 0; }

mvd_status mvd_profile(mvd_ctx* c, int enable) {
  if (!c) return MVD_ERR_INVALID_ARG;
  if (c->broken || (enable && c->use_graph)) return MVD_ERR_STATE;
  c->profiling = enable != 0;
  return MVD_OK;
}

mvd_status mvd_profile_read(mvd_ctx* c, double* total_ms, long long* launches) {
  if (!c || !total_ms || !launches) return MVD_ERR_INVALID_ARG;
  if (c->broken) return MVD_ERR_STATE;
  MVD_CK(cudaStreamSynchronize(c->stream), "profile read");
  for (int k = 0; k < MVD_K_COUNT; ++k) { total_ms[k] = 0.0; launches[k] = 0; }
  for (const mvd_ctx::Rec& r : c->recs) {
    float ms = 0.f;
    MVD_CK(cudaEventElapsedTime(&ms, r.a, r.b), "profile read");
    total_ms[r.cls] += ms;
    ++launches[r.cls];
  }
  c->recs.clear();
  c->ev_used = 0;
  return MVD_OK;
}

const char* mvd_kernel_class_name(int k) {
  static const char* const names[MVD_K_COUNT] = {"y_fwd", "y_inv", "z_conv", "x_quot", "x_update", "x_accum", "x_load"};
  return (k >= 0 && k < MVD_K_COUNT) ? names[k] : "";
}

void mvd_destroy(mvd_ctx* c) {
  if (!c) return;
  if (c->graph_exec) cudaGraphExecDestroy(c->graph_exec);
  for (cudaEvent_t e : c->ev_pool) cudaEventDestroy(e);
  delete c;
}

const char* mvd_status_string(mvd_status s) {
  switch (s) {
    case MVD_OK: return "ok";
    case MVD_ERR_INVALID_ARG: return "invalid argument";
    case MVD_ERR_UNSUPPORTED: return "unsupported size (no FFT length available)";
    case MVD_ERR_WORKSPACE: return "workspace missing, misaligned or too small";
    case MVD_ERR_CUDA: return "CUDA error";
    case MVD_ERR_STATE: return "call not valid in this state of the context (see mvd_last_error)";
  }
  return "unknown status";
}

const char* mvd_last_error(const mvd_ctx* c) { return c ? c->err : ""; }

}  // extern "C"

// ---- block-wise processing (S6; L64, L943; R13) ----------------------------------------------------
namespace {

struct Seg { int c0, c1, e0, e1; };   // central [c0,c1), extended [e0,e1)

std::vector<Seg> segments(int n, int block, int halo) {
  std::vector<Seg> out;
  for (int s = 0; s < n; s += block) {
    const int e = std::min(s + block, n);
    out.push_back(Seg{s, e, std::max(s - halo, 0), std::min(e + halo, n)});
  }
  return out;
}

struct BlockedLayout {
  int halo[3];
  std::vector<Seg> seg[3];
  size_t max_ext = 0;          // voxels of the largest extended block
  size_t ctx_bytes = 0;        // largest context workspace over the distinct extended shapes
  std::vector<std::array<int, 3>> shapes;
  size_t off_scal = 0, off_views = 0, off_psi0 = 0, off_est = 0, off_kern = 0, off_ctx = 0, total = 0;
  size_t kern_bytes = 0;       // back-projectors shared by the contexts of all block shapes
};

mvd_status blocked_layout(BlockedLayout& L, int n_views, const int dims[3], const int (*psf_dims)[3],
                          mvd_variant variant, const mvd_options* opt, const int block_dims[3],
                          const int halo[3]) {
  if (n_views < 1 || !dims || !psf_dims || !block_dims) return MVD_ERR_INVALID_ARG;
  for (int a = 0; a < 3; ++a) {
    if (dims[a] < 1 || block_dims[a] < 1) return MVD_ERR_INVALID_ARG;
    int h = 0;
    for (int v = 0; v < n_views; ++v) h = std::max(h, (psf_dims[v][a] - 1) / 2);
    L.halo[a] = halo ? halo[a] : h;
    if (L.halo[a] < 0) return MVD_ERR_INVALID_ARG;
    L.seg[a] = segments(dims[a], block_dims[a], L.halo[a]);
  }
  for (const Seg& sz : L.seg[2])
    for (const Seg& sy : L.seg[1])
      for (const Seg& sx : L.seg[0]) {
        std::array<int, 3> e = {sx.e1 - sx.e0, sy.e1 - sy.e0, sz.e1 - sz.e0};
        if (std::find(L.shapes.begin(), L.shapes.end(), e) == L.shapes.end()) L.shapes.push_back(e);
      }
  mvd_options o = *opt;
  o.fft_dims[0] = o.fft_dims[1] = o.fft_dims[2] = 0;
  for (const auto& e : L.shapes) {
    const int d[3] = {e[0], e[1], e[2]};
    const size_t b = mvd_workspace_size(n_views, d, psf_dims, variant, &o);
    if (b == 0) return MVD_ERR_UNSUPPORTED;
    L.ctx_bytes = std::max(L.ctx_bytes, b);
    L.max_ext = std::max(L.max_ext, (size_t)e[0] * e[1] * e[2]);
  }
  size_t off = 0;
  auto take = [&](size_t bytes) { size_t at = off; off = align_up(off + bytes, 256); return at; };
  L.off_scal = take(sizeof(double) * (size_t)(reduce_blocks() + n_views + 8));
  L.off_views = take(align_up(L.max_ext * sizeof(float), 256) * n_views);
  L.off_psi0 = take(L.max_ext * sizeof(float));
  L.off_est = take(L.max_ext * sizeof(float));
  {
    size_t kmax = 0;
    for (int v = 0; v < n_views; ++v)
      kmax = std::max(kmax, (size_t)psf_dims[v][0] * psf_dims[v][1] * psf_dims[v][2]);
    L.kern_bytes = align_up(kmax, 32) * sizeof(double) * n_views;   // = psf_stride * V of every context
  }
  L.off_kern = take(L.kern_bytes);
  L.off_ctx = take(L.ctx_bytes);
  L.total = off;
  return MVD_OK;
}

}  // namespace

extern "C" size_t mvd_blocked_workspace_size(int n_views, const int dims[3], const int (*psf_dims)[3],
                                             mvd_variant variant, const mvd_options* opt_in,
                                             const int block_dims[3], const int halo[3]) {
  mvd_options tmp;
  BlockedLayout L;
  if (blocked_layout(L, n_views, dims, psf_dims, variant, defaults(opt_in, &tmp), block_dims, halo) != MVD_OK) return 0;
  return L.total;
}

extern "C" mvd_status mvd_deconvolve_blocked(int n_views, const float* const* views, const int dims[3],
                                             const float* const* psfs, const int (*psf_dims)[3],
                                             mvd_variant variant, const mvd_options* opt_in,
                                             const int block_dims[3], const int halo[3], int iterations,
                                             float* dst, long long* launches_out) {
  if (!views || !psfs || !dst || !opt_in || iterations < 0) return MVD_ERR_INVALID_ARG;
  mvd_options tmp;
  const mvd_options* opt = defaults(opt_in, &tmp);
  if (opt->weights || opt->views_ready || opt->local_views || opt->psi0 || opt->psi0_value != 0.f)
    return MVD_ERR_UNSUPPORTED;   // whole-volume options
  const int bworld = opt->block_world > 1 ? opt->block_world : 1;
  if (opt->block_rank < 0 || opt->block_rank >= bworld) return MVD_ERR_INVALID_ARG;
  BlockedLayout L;
  mvd_status s = blocked_layout(L, n_views, dims, psf_dims, variant, opt, block_dims, halo);
  if (s != MVD_OK) return s;
  if (!opt->workspace || (reinterpret_cast<size_t>(opt->workspace) & 255) || opt->workspace_bytes < L.total)
    return MVD_ERR_WORKSPACE;
  char* ws = reinterpret_cast<char*>(opt->workspace);
  cudaStream_t st = reinterpret_cast<cudaStream_t>(opt->stream);
  double* partial = reinterpret_cast<double*>(ws + L.off_scal);
  const int nb = reduce_blocks();
  double* sums = partial + nb;
  const size_t vstride = align_up(L.max_ext * sizeof(float), 256);
  std::vector<const float*> bviews(n_views);
  for (int v = 0; v < n_views; ++v) bviews[v] = reinterpret_cast<const float*>(ws + L.off_views + v * vstride);
  float* psi0 = reinterpret_cast<float*>(ws + L.off_psi0);
  float* est = reinterpret_cast<float*>(ws + L.off_est);
  long long launches = 0;
  const Dims3 N{dims[0], dims[1], dims[2]};
  const long long nvox = (long long)dims[0] * dims[1] * dims[2];

  // psi^0 = mean over the WHOLE volume and all views (R13), kept on the device
  for (int v = 0; v < n_views; ++v) {
    if (!views[v]) return MVD_ERR_INVALID_ARG;
    sum_f32_kernel<<<nb, 256, 0, st>>>(views[v], nvox, partial);
    final_sum_kernel<<<1, 256, 0, st>>>(partial, nb, 1, sums + v);
    launches += 2;
  }
  fill_mean_kernel<<<nb, 256, 0, st>>>(psi0, (long long)L.max_ext, sums, n_views, (double)nvox * n_views);
  ++launches;
  if (cudaGetLastError() != cudaSuccess) return MVD_ERR_CUDA;

  double* shared_kern = reinterpret_cast<double*>(ws + L.off_kern);
  bool have_kern = false;
  for (const auto& shape : L.shapes) {
    const int d[3] = {shape[0], shape[1], shape[2]};
    // blocks of this shape that belong to this rank (blocks dealt round-robin by index, L225)
    bool mine = false;
    {
      long long idx = 0;
      for (const Seg& sz : L.seg[2])
        for (const Seg& sy : L.seg[1])
          for (const Seg& sx : L.seg[0]) {
            if (sx.e1 - sx.e0 == d[0] && sy.e1 - sy.e0 == d[1] && sz.e1 - sz.e0 == d[2] && idx % bworld == opt->block_rank) mine = true;
            ++idx;
          }
    }
    if (!mine) continue;
    mvd_options o = *opt;
    o.fft_dims[0] = o.fft_dims[1] = o.fft_dims[2] = 0;
    o.block_rank = o.block_world = 0;
    o.psi0 = psi0;
    o.workspace = ws + L.off_ctx;
    o.workspace_bytes = L.ctx_bytes;
    mvd_ctx* c = nullptr;
    s = create_impl(&c, n_views, bviews.data(), d, psfs, psf_dims, variant, &o, have_kern ? shared_kern : nullptr);
    if (s != MVD_OK) return s;
    if (!have_kern) {   // the back-projectors depend on the PSFs only: computed once, reused by the other shapes
      if (sizeof(double) * c->P.psf_stride * c->P.V != L.kern_bytes ||
          cudaMemcpyAsync(shared_kern, c->kern(0), L.kern_bytes, cudaMemcpyDeviceToDevice, st) != cudaSuccess) {
        mvd_destroy(c);
        return MVD_ERR_CUDA;
      }
      have_kern = true;
    }
    const Dims3 E{d[0], d[1], d[2]};
    const long long ext = (long long)d[0] * d[1] * d[2];
    const unsigned grid = (unsigned)std::min<long long>((ext + 255) / 256, (long long)nb * 8);
    long long bidx = -1;
    for (const Seg& sz : L.seg[2])
      for (const Seg& sy : L.seg[1])
        for (const Seg& sx : L.seg[0]) {
          ++bidx;
          if (sx.e1 - sx.e0 != d[0] || sy.e1 - sy.e0 != d[1] || sz.e1 - sz.e0 != d[2]) continue;
          if (bidx % bworld != opt->block_rank) continue;
          for (int v = 0; v < n_views; ++v) {
            gather_block_kernel<<<grid, 256, 0, st>>>(views[v], N, Dims3{sx.e0, sy.e0, sz.e0}, E,
                                                      const_cast<float*>(bviews[v]));
            ++launches;
          }
          s = mvd_set_estimate(c, psi0);
          if (s == MVD_OK) s = mvd_iterate(c, iterations);
          if (s == MVD_OK) s = mvd_get_estimate(c, est, 1);
          if (s != MVD_OK) { mvd_destroy(c); return s; }
          paste_block_kernel<<<grid, 256, 0, st>>>(est, E, Dims3{sx.c0 - sx.e0, sy.c0 - sy.e0, sz.c0 - sz.e0},
                                                   Dims3{sx.c1 - sx.c0, sy.c1 - sy.c0, sz.c1 - sz.c0}, dst, N,
                                                   Dims3{sx.c0, sy.c0, sz.c0});
          ++launches;
        }
    if (cudaStreamSynchronize(st) != cudaSuccess || cudaGetLastError() != cudaSuccess) { mvd_destroy(c); return MVD_ERR_CUDA; }
    launches += mvd_launch_count(c);
    mvd_destroy(c);
  }
  if (launches_out) *launches_out = launches;
  return MVD_OK;
}
