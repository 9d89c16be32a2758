"""fp64 CPU oracle for the multi-view Richardson-Lucy iteration of arXiv 1308.0730.

TEST INFRASTRUCTURE ONLY.  This is the slow, plain reference the CUDA path is checked
against.  Only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s cpu_baseline /
``--impl reference`` legs may import it.  It shares no code with
``paper_1308_0730_b200`` (no kernels, headers, tables, helpers) and imports nothing from it.

What it computes (PAPER.md line numbers; "R<n>" = reading listed in DESIGN.md):

* eq. 3 (L258) / section 6 (L560-562): every integral is a convolution with a spatially
  constant PSF, all views in one frame.  ``same(a, k)`` below is that convolution with zero
  extension outside the volume and the output cropped to the volume (R3).
* section 2.1.1 (L312), L574: the second convolution uses the mirrored kernel P*.
* eq. 13 (L302-306): one RL update = blur, quotient, back-project, multiply.
* eq. 70 (L562): combined update with P_v* ("independent").
* eq. 104-105 (L724-734): combined update with the compound kernel ("efficient").
* eq. 107 / 108 (L748, L755): optimisation I / II back-projectors.
* eq. 109-112 (L769-776), eq. 114-117 (L786-793): sequential (OSEM) schedule.
* eq. 44 (L455) + L464: the combined update takes the |V|-th root (R1).
* L64, L869 + ref. 20: optional Tikhonov regularisation of every update (R14; the paper prints no
  formula, see ``tikhonov`` below: parity unpinned by the paper).

Arrays are numpy, shape (Nz, Ny, Nx), x fastest.  All arithmetic is float64.

Pins (tests/test_oracle_pins.py): P1 brute force == FFT, P2 V=1 == classical RL, P3 flux
identity (eq. 52-55), P4 fixed point (L306), P5 identical views (L847), P6 delta PSF (L851),
P7 Gaussian closed form of eq. 105, P8 monotone likelihood (eq. 39-43), P9 ordering (L807-809),
hand-computed worked example (tests/golden/rl_1d_worked_example.txt); deconvolve_blocked: exact
equality with the whole-volume result when the halo covers the dependence radius (2r per
view-update), delta PSF with halo 0, and a negative control with halo r.
Parity unpinned by the paper (shared definitions only, R2/R4/R13): eps / psi_floor clamps,
psi0 = mean over all views, the OSEM=compound default, the halo WIDTH r of the block mode
(the block mechanics themselves are pinned as above).
"""
from __future__ import annotations

import os

import numpy as np
import scipy.fft as sfft

EPS_DEFAULT = 1e-6        # R4: q = phi / max(b, eps)
FLOOR_DEFAULT = 1e-6      # R4: psi <- max(psi * f, psi_floor)

VARIANTS = ("independent", "efficient", "osem")
KERNEL_MODES = ("auto", "plain", "compound", "opt1", "opt2")


def _workers():
    return len(os.sched_getaffinity(0))


# --------------------------------------------------------------------------------------
# O1. definitions
# --------------------------------------------------------------------------------------
def normalise(p):
    """eq. 4 (L262): every distribution integrates to 1."""
    p = np.asarray(p, dtype=np.float64)
    return p / p.sum()


def flip(k):
    """P*(x) = P(-x) (L312, L574): mirror every axis."""
    return np.asarray(k)[::-1, ::-1, ::-1]


def conv_full_direct(a, b):
    """Full linear convolution (a * b)[n] = sum_m a[m] b[n-m], brute force over the taps of b."""
    a = np.asarray(a, dtype=np.float64)
    b = np.asarray(b, dtype=np.float64)
    az, ay, ax = a.shape
    out = np.zeros((az + b.shape[0] - 1, ay + b.shape[1] - 1, ax + b.shape[2] - 1))
    for uz in range(b.shape[0]):
        for uy in range(b.shape[1]):
            for ux in range(b.shape[2]):
                out[uz:uz + az, uy:uy + ay, ux:ux + ax] += b[uz, uy, ux] * a
    return out


def conv_full_fft(a, b):
    """Same result as conv_full_direct through scipy.fft at size Na+Nb-1 or larger."""
    a = np.asarray(a, dtype=np.float64)
    b = np.asarray(b, dtype=np.float64)
    full = [na + nb - 1 for na, nb in zip(a.shape, b.shape)]
    shape = [sfft.next_fast_len(n, real=True) for n in full]
    w = _workers()
    out = sfft.irfftn(sfft.rfftn(a, shape, workers=w) * sfft.rfftn(b, shape, workers=w), shape, workers=w)
    return out[:full[0], :full[1], :full[2]]


def _centre(k):
    return tuple((n - 1) // 2 for n in k.shape)


def same_direct(a, k):
    """same(a,k)[xi] = sum_u k[u] a[xi - (u - c)], a = 0 outside the volume, c = (K-1)/2."""
    k = np.asarray(k, dtype=np.float64)
    a = np.asarray(a, dtype=np.float64)
    cz, cy, cx = _centre(k)
    full = conv_full_direct(a, k)
    nz, ny, nx = a.shape
    return full[cz:cz + nz, cy:cy + ny, cx:cx + nx]


def same_fft(a, k):
    k = np.asarray(k, dtype=np.float64)
    a = np.asarray(a, dtype=np.float64)
    cz, cy, cx = _centre(k)
    full = conv_full_fft(a, k)
    nz, ny, nx = a.shape
    return full[cz:cz + nz, cy:cy + ny, cx:cx + nx]


def _same(backend):
    return {"fft": same_fft, "direct": same_direct}[backend]


def _full(backend):
    return {"fft": conv_full_fft, "direct": conv_full_direct}[backend]


def _crop_centre(t, box):
    """Central crop of t (odd sizes) to the odd-sized ``box`` (R6: centre-aligned)."""
    sl = []
    for n, b in zip(t.shape, box):
        c = (n - 1) // 2
        h = (b - 1) // 2
        if h > c:
            raise ValueError("crop box larger than array")
        sl.append(slice(c - h, c + h + 1))
    return t[tuple(sl)]


# --------------------------------------------------------------------------------------
# O3. back-projectors
# --------------------------------------------------------------------------------------
def resolve_kernel_mode(variant, kernel_mode):
    """R2: independent -> plain (eq. 70); efficient, osem -> compound (eq. 104, 109-112)."""
    if kernel_mode == "auto":
        return "plain" if variant == "independent" else "compound"
    return kernel_mode


def back_projector(psfs, v, mode, backend="fft"):
    """K_v for view v.  ``psfs`` are the normalised P_w, shape (Kz,Ky,Kx) each, odd sizes.

    plain    : P_v*                                                  (eq. 70)
    compound : P_v* . prod_{w != v} crop(P_v* * P_w * P_w*)          (eq. 105)
    opt1     : P_v* . prod_{w != v} crop(P_v* * P_w)                 (eq. 107)
    opt2     : (P_v*)^|V|  (one factor for v, one per w in W_v; R9)  (eq. 108)
    The product is pointwise ("scalar multiplication", L734) on the box of P_v, factors
    centre-aligned (R6); the result is renormalised to sum 1 (R5, eq. 4).
    """
    full = _full(backend)
    pv_star = flip(psfs[v]).astype(np.float64)
    if mode == "plain":
        return pv_star.copy()
    if mode == "opt2":
        return normalise(pv_star ** len(psfs))
    if mode not in ("compound", "opt1"):
        raise ValueError(mode)
    k = pv_star.copy()
    for w, pw in enumerate(psfs):
        if w == v:
            continue
        t = full(pv_star, pw)                       # P_v* * P_w
        if mode == "compound":
            t = full(t, flip(pw))                   # ... * P_w*
        k = k * _crop_centre(t, pv_star.shape)
    return normalise(k)


# --------------------------------------------------------------------------------------
# O2/O4/O5. the iteration
# --------------------------------------------------------------------------------------
def initial_estimate(views):
    """psi^0: constant = average intensity of the measured data (L304; all views, R: mean over V)."""
    tot = 0.0
    cnt = 0
    for phi in views:
        phi = np.asarray(phi, dtype=np.float64)
        tot += phi.sum()
        cnt += phi.size
    return np.full(np.asarray(views[0]).shape, tot / cnt)


def tikhonov(u, lam):
    """Tikhonov-regularised value of an update (L64 "option for Tikhonov regularization", L869, ref. 20).

    PAPER.md gives no formula (reading R14).  Used here: the EM M-step for the Poisson likelihood with the
    quadratic (Tikhonov) penalty (lam/4) * sum psi^2.  With u = psi^r * f the unpenalised update, the new
    estimate maximises  u log(psi) - psi - (lam/4) psi^2  per voxel:  u/psi - 1 - (lam/2) psi = 0, i.e. it is
    the positive root of  (lam/2) psi^2 + psi - u = 0:
        psi = (sqrt(1 + 2 lam u) - 1) / lam  =  2 u / (1 + sqrt(1 + 2 lam u))     (second form: no cancellation)
    lam = 0 leaves u unchanged; psi < u for lam > 0 ("slows down convergence", L869)."""
    if lam == 0.0:
        return u
    return 2.0 * u / (1.0 + np.sqrt(1.0 + 2.0 * lam * u))


def rl_factor(psi, phi, p, k, eps=EPS_DEFAULT, backend="fft"):
    """f_v = (phi_v / (psi * P_v)) * K_v (eq. 1, eq. 13, EM description L306)."""
    same = _same(backend)
    b = same(psi, p)                                # expected value phi^r = psi^r * P_v
    q = np.asarray(phi, dtype=np.float64) / np.maximum(b, eps)
    return same(q, k)                               # q is zero outside the volume (R3)


class Oracle:
    """Holds normalised PSFs, back-projectors and psi; ``iterate(n)`` advances n iterations.

    One iteration = every view contributed once (footnote L817).
    """

    def __init__(self, views, psfs, variant="osem", kernel_mode="auto", literal_product=False,
                 eps=EPS_DEFAULT, psi_floor=FLOOR_DEFAULT, psi0=None, backend="fft", weights=None,
                 tikhonov_lambda=0.0):
        if variant not in VARIANTS:
            raise ValueError(variant)
        if weights is not None and variant != "osem":
            raise ValueError("per-view weights belong to the sequential updates (section 12, L897)")
        if kernel_mode not in KERNEL_MODES:
            raise ValueError(kernel_mode)
        self.views = [np.asarray(v, dtype=np.float64) for v in views]
        self.psfs = [normalise(p) for p in psfs]
        for p in self.psfs:
            if any(n % 2 == 0 for n in p.shape):
                raise ValueError("PSF dims must be odd")
        self.variant = variant
        self.kernel_mode = resolve_kernel_mode(variant, kernel_mode)
        self.literal_product = bool(literal_product)
        self.eps = float(eps)
        self.psi_floor = float(psi_floor)
        self.backend = backend
        self.tikhonov_lambda = float(tikhonov_lambda)
        if self.tikhonov_lambda < 0.0:
            raise ValueError("tikhonov_lambda must be >= 0")
        self.kernels = [back_projector(self.psfs, v, self.kernel_mode, backend)
                        for v in range(len(self.psfs))]
        self.weights = None if weights is None else [np.asarray(w, dtype=np.float64) for w in weights]
        self.psi = initial_estimate(self.views) if psi0 is None else np.array(psi0, dtype=np.float64)
        self.iterations_done = 0
        self.flux = float(self.psi.sum())
        self.l1_change = 0.0

    # -- one psi update, bookkeeping of the two statistics the library reports (S5) --
    def _commit(self, new):
        self.l1_change = float(np.abs(new - self.psi).sum())
        self.flux = float(new.sum())
        self.psi = new

    def factor(self, v):
        return rl_factor(self.psi, self.views[v], self.psfs[v], self.kernels[v], self.eps, self.backend)

    def view_update(self, v):
        """One sequential update with view v (one line of eq. 109-112): psi <- max(psi f_v, floor)."""
        if self.variant != "osem":
            raise ValueError("view_update is the sequential (OSEM) step")
        f = self.factor(v)
        if self.weights is not None:
            # section 12 (L897): the weight 0..1 of a pixel is "the fraction of change
            # suggested by a Lucy-Richardson update step that will be applied":
            # psi*f = psi + (psi*f - psi)  ->  psi + w*(psi*f - psi) = psi*(1 + w*(f - 1))
            f = 1.0 + self.weights[v] * (f - 1.0)
        self._commit(np.maximum(tikhonov(self.psi * f, self.tikhonov_lambda), self.psi_floor))
        return self.psi

    def iterate(self, n=1):
        nv = len(self.views)
        for _ in range(n):
            if self.variant == "osem":
                # eq. 109-112 / 114-117: psi is updated after every view, index order (R11)
                for v in range(nv):
                    self.view_update(v)
            else:
                # eq. 70 / 104: every f_v from the same psi^r, multiplicative combination
                prod = np.ones_like(self.psi)
                for v in range(nv):
                    f = self.factor(v)
                    prod *= f if self.literal_product else np.maximum(f, 0.0)
                if not self.literal_product:
                    prod = prod ** (1.0 / nv)       # eq. 44: geometric mean (R1)
                self._commit(np.maximum(tikhonov(self.psi * prod, self.tikhonov_lambda), self.psi_floor))
            self.iterations_done += 1
        return self.psi


def deconvolve(views, psfs, variant="osem", iterations=1, **kw):
    o = Oracle(views, psfs, variant, **kw)
    o.iterate(iterations)
    return o.psi


# --------------------------------------------------------------------------------------
# section 12 (L891-903): weight images for partially overlapping views
# --------------------------------------------------------------------------------------
def blending_weights(shape_zyx, lo_zyx, hi_zyx, border):
    """Weight image of one view whose data covers the box [lo, hi) of the common frame: 1 in the
    central part, falling to 0 at the faces of the box "following a cosine function" over
    `border` voxels (L891), 0 outside the box.  Per axis the ramp at distance d (in voxels, the
    face voxel has d = 0.5) is 0.5*(1 - cos(pi*d/border)); the three axes multiply.  [reading R16:
    the paper gives neither the ramp width nor how axes combine]"""
    w = np.ones(shape_zyx, dtype=np.float64)
    for ax in range(3):
        idx = np.arange(shape_zyx[ax], dtype=np.float64)
        d = np.minimum(idx - lo_zyx[ax] + 0.5, hi_zyx[ax] - idx - 0.5)     # distance to the nearer face
        r = np.where(d <= 0, 0.0, np.where(d >= border, 1.0, 0.5 * (1.0 - np.cos(np.pi * d / border))))
        sh = [1, 1, 1]
        sh[ax] = -1
        w = w * r.reshape(sh)
    return w


def normalise_weights(weights, max_sum=1.0):
    """Scale the weights of every pixel so that their sum over the views is <= max_sum (default 1:
    "normalized to <= 1", L897; max_sum = number of overlapping views the user allows, L903).
    Weights are only ever scaled down: "individual weights are never increased above 1" (L895)."""
    ws = [np.asarray(w, dtype=np.float64) for w in weights]
    tot = np.sum(ws, axis=0)
    scale = np.where(tot > max_sum, max_sum / np.maximum(tot, 1e-300), 1.0)
    return [w * scale for w in ws]


# --------------------------------------------------------------------------------------
# quality metrics the paper uses (L127 average difference, L48 cross-correlation)
# --------------------------------------------------------------------------------------
def average_difference(psi, ref):
    return float(np.abs(np.asarray(psi, np.float64) - np.asarray(ref, np.float64)).mean())


def cross_correlation(psi, ref):
    a = np.asarray(psi, np.float64).ravel()
    b = np.asarray(ref, np.float64).ravel()
    a = a - a.mean()
    b = b - b.mean()
    return float((a @ b) / np.sqrt((a @ a) * (b @ b)))


# --------------------------------------------------------------------------------------
# O6. block-wise processing (L64, L943; R13)
# --------------------------------------------------------------------------------------
def block_grid(dims_zyx, block_zyx):
    """Start/stop of the central blocks tiling the volume (last block per axis may be short)."""
    out = []
    for z0 in range(0, dims_zyx[0], block_zyx[0]):
        for y0 in range(0, dims_zyx[1], block_zyx[1]):
            for x0 in range(0, dims_zyx[2], block_zyx[2]):
                out.append(((z0, min(z0 + block_zyx[0], dims_zyx[0])),
                            (y0, min(y0 + block_zyx[1], dims_zyx[1])),
                            (x0, min(x0 + block_zyx[2], dims_zyx[2]))))
    return out


def deconvolve_blocked(views, psfs, block_zyx, variant="osem", iterations=1, halo_zyx=None, **kw):
    """Each block is extended by a halo of real neighbouring data (clipped at the volume faces,
    so zero extension applies only beyond the volume), deconvolved on its own for all
    iterations with psi^0 = the WHOLE-volume mean, and its central part pasted (R13).
    halo defaults to the PSF half-size r = (K-1)/2 per axis."""
    views = [np.asarray(v, dtype=np.float64) for v in views]
    shape = views[0].shape
    if halo_zyx is None:
        halo_zyx = tuple(max((p.shape[a] - 1) // 2 for p in psfs) for a in range(3))
    psi0 = float(initial_estimate(views).flat[0])
    out = np.empty(shape)
    for (z0, z1), (y0, y1), (x0, x1) in block_grid(shape, block_zyx):
        ez0, ez1 = max(z0 - halo_zyx[0], 0), min(z1 + halo_zyx[0], shape[0])
        ey0, ey1 = max(y0 - halo_zyx[1], 0), min(y1 + halo_zyx[1], shape[1])
        ex0, ex1 = max(x0 - halo_zyx[2], 0), min(x1 + halo_zyx[2], shape[2])
        sub = [v[ez0:ez1, ey0:ey1, ex0:ex1] for v in views]
        o = Oracle(sub, psfs, variant, psi0=np.full(sub[0].shape, psi0), **kw)
        o.iterate(iterations)
        out[z0:z1, y0:y1, x0:x1] = o.psi[z0 - ez0:z1 - ez0, y0 - ey0:y1 - ey0, x0 - ex0:x1 - ex0]
    return out
