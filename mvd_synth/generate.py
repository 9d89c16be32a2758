"""Seeded generators for the five BASELINE.json configs plus a tiny asymmetric case.

Conventions
-----------
* ``dims`` / ``psf_dims`` are (x, y, z) triples, x fastest in memory; numpy arrays have
  shape (Nz, Ny, Nx), C order, i.e. ``a[z, y, x]``.
* PSFs are sampled Gaussians exp(-u^T S^-1 u / 2) at integer offsets u in the stated
  box, S = R_y(theta) diag(sxy^2, sxy^2, sz^2) R_y(theta)^T (rotation about the y axis,
  the paper's rotation axis), truncated to the box and normalised to sum 1.
* views: phi_v = Poisson(s * same(GT, P_v)) drawn in float64, stored float32.  The blur
  is a plain zero-extended "same" convolution done with scipy.fft at a size >= N+K-1;
  it is the data recipe, not the method under test.
* Every random draw comes from numpy.random.default_rng([13080730, k, stream]).
  stream 0 = objects, stream 100+v = Poisson noise of view v (so views can be drawn
  in parallel and independently of V).
"""
from __future__ import annotations

import math
import os
from concurrent.futures import ThreadPoolExecutor
from dataclasses import dataclass, field

import numpy as np
import scipy.fft as sfft

SEED = 13080730


@dataclass
class Problem:
    """One synthetic multi-view acquisition."""

    k: int
    dims: tuple            # (Nx, Ny, Nz)
    psf_dims: tuple        # (Kx, Ky, Kz), same box for every view
    gt: np.ndarray         # (Nz, Ny, Nx) float32, scaled ground truth (same units as views)
    psfs: list             # V arrays (Kz, Ky, Kx) float32, each sums to ~1
    views: list            # V arrays (Nz, Ny, Nx) float32, >= 0
    iterations: int
    variants: tuple        # variant names BASELINE asks for on this config
    meta: dict = field(default_factory=dict)

    @property
    def n_views(self) -> int:
        return len(self.views)


# k -> recipe.  Items BASELINE.json leaves open are readings, listed in DESIGN.md.
CONFIGS = {
    1: dict(dims=(64, 64, 64), psf=(15, 15, 31), sxy=1.2, sz=4.0,
            angles=(0.0, 90.0, 180.0, 270.0), beads=40, nuclei=0, shell=False,
            peak=None, iterations=10, variants=("osem",)),
    2: dict(dims=(128, 128, 128), psf=(17, 17, 35), sxy=1.3, sz=4.55,
            angles=(0.0, 120.0, 240.0), beads=0, nuclei=500, shell=False,
            peak=None, iterations=20, variants=("independent", "efficient", "osem")),
    3: dict(dims=(256, 256, 128), psf=(19, 19, 41), sxy=1.5, sz=5.5,
            angles=tuple(60.0 * i for i in range(6)), beads=100, nuclei=3000, shell=True,
            peak=300.0, iterations=15, variants=("osem",)),
    4: dict(dims=(512, 512, 256), psf=(21, 21, 45), sxy=1.6, sz=6.4,
            angles=tuple(360.0 * i / 7 for i in range(7)), beads=100, nuclei=20000, shell=True,
            peak=500.0, iterations=10, variants=("osem",)),
    5: dict(dims=(1024, 1024, 512), psf=(25, 25, 51), sxy=1.8, sz=7.2,
            angles=tuple(60.0 * i for i in range(6)), beads=100, nuclei=80000, shell=True,
            peak=500.0, iterations=5, variants=("osem",)),
}

BACKGROUND = 5.0


def gaussian_psf(psf_dims, sxy, sz, angle_deg):
    """Anisotropic Gaussian rotated by ``angle_deg`` about y, sampled in the box, sum 1."""
    kx, ky, kz = psf_dims
    t = math.radians(angle_deg)
    c, s = math.cos(t), math.sin(t)
    # columns/rows ordered (x, y, z); rotation about y mixes x and z
    rot = np.array([[c, 0.0, s], [0.0, 1.0, 0.0], [-s, 0.0, c]])
    cov = rot @ np.diag([sxy ** 2, sxy ** 2, sz ** 2]) @ rot.T
    prec = np.linalg.inv(cov)
    uz, uy, ux = np.meshgrid(np.arange(kz) - (kz - 1) // 2,
                             np.arange(ky) - (ky - 1) // 2,
                             np.arange(kx) - (kx - 1) // 2, indexing="ij")
    u = np.stack([ux, uy, uz], axis=-1).astype(np.float64)
    q = np.einsum("...i,ij,...j->...", u, prec, u)
    p = np.exp(-0.5 * q)
    p /= p.sum()
    return p.astype(np.float32)


def random_psf(rng, psf_dims):
    """Non-negative, deliberately asymmetric kernel (random taps + an off-centre peak)."""
    kx, ky, kz = psf_dims
    p = rng.random((kz, ky, kx))
    p[rng.integers(kz), rng.integers(ky), rng.integers(kx)] += 4.0
    p /= p.sum()
    return p.astype(np.float32)


def _blur_same(a, psf, dtype):
    """Zero-extended 'same' convolution with a centred odd kernel via scipy.fft."""
    kz, ky, kx = psf.shape
    shape = [sfft.next_fast_len(n + k - 1, real=True) for n, k in zip(a.shape, psf.shape)]
    workers = len(os.sched_getaffinity(0))
    fa = sfft.rfftn(a.astype(dtype, copy=False), shape, workers=workers)
    fa *= sfft.rfftn(psf.astype(dtype), shape, workers=workers)
    full = sfft.irfftn(fa, shape, workers=workers)
    del fa
    cz, cy, cx = (kz - 1) // 2, (ky - 1) // 2, (kx - 1) // 2
    nz, ny, nx = a.shape
    return full[cz:cz + nz, cy:cy + ny, cx:cx + nx]


def _paint_ellipsoids(gt, rng, n, shell):
    nz, ny, nx = gt.shape
    dims = np.array([nx, ny, nz], dtype=np.float64)
    if shell:
        # centres in an ellipsoidal shell: semi-axes 0.42*N, thickness 0.10*N
        d = rng.normal(size=(n, 3))
        d /= np.linalg.norm(d, axis=1, keepdims=True)
        rad = rng.uniform(0.37, 0.47, size=(n, 1))
        centres = dims / 2.0 + d * rad * dims
    else:
        margin = np.minimum(6.0, dims / 4.0)
        centres = rng.uniform(margin, dims - margin, size=(n, 3))
    radii = rng.uniform(3.0, 6.0, size=(n, 3))
    inten = rng.uniform(200.0, 800.0, size=n)
    for (cx, cy, cz), (rx, ry, rz), val in zip(centres, radii, inten):
        x0, x1 = max(int(cx - rx), 0), min(int(cx + rx) + 2, nx)
        y0, y1 = max(int(cy - ry), 0), min(int(cy + ry) + 2, ny)
        z0, z1 = max(int(cz - rz), 0), min(int(cz + rz) + 2, nz)
        if x0 >= x1 or y0 >= y1 or z0 >= z1:
            continue
        zz = ((np.arange(z0, z1) - cz) / rz) ** 2
        yy = ((np.arange(y0, y1) - cy) / ry) ** 2
        xx = ((np.arange(x0, x1) - cx) / rx) ** 2
        inside = (zz[:, None, None] + yy[None, :, None] + xx[None, None, :]) <= 1.0
        sub = gt[z0:z1, y0:y1, x0:x1]
        np.maximum(sub, np.where(inside, val, 0.0), out=sub)


def _add_beads(gt, rng, n):
    nz, ny, nx = gt.shape
    dims = np.array([nx, ny, nz], dtype=np.float64)
    margin = np.minimum(4.0, dims / 4.0)
    centres = rng.uniform(margin, dims - margin, size=(n, 3))
    sig = rng.uniform(1.0, 2.0, size=n)
    amp = rng.uniform(100.0, 1000.0, size=n)
    for (cx, cy, cz), s, a in zip(centres, sig, amp):
        h = int(math.ceil(4 * s))
        x0, x1 = max(int(cx) - h, 0), min(int(cx) + h + 1, nx)
        y0, y1 = max(int(cy) - h, 0), min(int(cy) + h + 1, ny)
        z0, z1 = max(int(cz) - h, 0), min(int(cz) + h + 1, nz)
        gz = np.exp(-0.5 * ((np.arange(z0, z1) - cz) / s) ** 2)
        gy = np.exp(-0.5 * ((np.arange(y0, y1) - cy) / s) ** 2)
        gx = np.exp(-0.5 * ((np.arange(x0, x1) - cx) / s) ** 2)
        gt[z0:z1, y0:y1, x0:x1] += a * gz[:, None, None] * gy[None, :, None] * gx[None, None, :]


def _poisson_f32(lam, rng, chunk=16):
    """Poisson draw slab by slab (bounds float64 temporaries); result float32."""
    out = np.empty(lam.shape, dtype=np.float32)
    for z0 in range(0, lam.shape[0], chunk):
        l = np.maximum(lam[z0:z0 + chunk].astype(np.float64), 0.0)
        out[z0:z0 + chunk] = rng.poisson(l)
    return out


def make_problem(k, n_views=None, noise=True, dims=None, psf_dims=None):
    """Build config ``k`` (1..5).  ``dims`` / ``psf_dims`` / ``n_views`` shrink it (same recipe,
    same seeds) for tests that want the config's structure at a size the oracle finishes fast."""
    rec = CONFIGS[k]
    dims = tuple(dims or rec["dims"])
    psf_dims = tuple(psf_dims or rec["psf"])
    angles = rec["angles"] if n_views is None else rec["angles"][:n_views]
    nx, ny, nz = dims
    big = nx * ny * nz > (1 << 25)
    work = np.float32 if big else np.float64

    rng = np.random.default_rng([SEED, k, 0])
    gt = np.zeros((nz, ny, nx), dtype=np.float64 if not big else np.float32)
    scale = (nx * ny * nz) / float(np.prod(rec["dims"]))      # shrunk copies keep the density
    if rec["nuclei"]:
        _paint_ellipsoids(gt, rng, max(1, int(round(rec["nuclei"] * scale))), rec["shell"])
    if rec["beads"]:
        _add_beads(gt, rng, max(1, int(round(rec["beads"] * scale))))
    gt += BACKGROUND

    psfs = [gaussian_psf(psf_dims, rec["sxy"], rec["sz"], a) for a in angles]
    blurred = [_blur_same(gt, p, work) for p in psfs]
    s = 1.0
    if rec["peak"] is not None:
        s = rec["peak"] / max(float(b.max()) for b in blurred)

    def _draw(v):
        lam = blurred[v] * s
        if not noise:
            return np.maximum(lam, 0.0).astype(np.float32)
        return _poisson_f32(lam, np.random.default_rng([SEED, k, 100 + v]))

    with ThreadPoolExecutor(max_workers=min(len(psfs), len(os.sched_getaffinity(0)))) as ex:
        views = list(ex.map(_draw, range(len(psfs))))
    return Problem(k=k, dims=dims, psf_dims=psf_dims, gt=(gt * s).astype(np.float32), psfs=psfs,
                   views=views, iterations=rec["iterations"], variants=rec["variants"],
                   meta=dict(scale=s, angles=tuple(angles), noise=noise))


def make_tiny_asymmetric(dims=(24, 20, 18), psf_dims=(5, 7, 9), n_views=3, noise=True, seed_stream=0):
    """k=0: tiny volume with random NON-symmetric PSFs.  Every BASELINE config uses centred
    Gaussians (point-symmetric, flip(P)=P); this case is the one that fails if a mirror,
    centring or crop offset is wrong."""
    nx, ny, nz = dims
    rng = np.random.default_rng([SEED, 0, seed_stream])
    gt = np.full((nz, ny, nx), BACKGROUND)
    _add_beads(gt, rng, 6)
    gt += 40.0 * rng.random(gt.shape)
    psfs = [random_psf(rng, psf_dims) for _ in range(n_views)]
    views = []
    for v, p in enumerate(psfs):
        lam = np.maximum(_blur_same(gt, p, np.float64), 0.0)
        if noise:
            views.append(np.random.default_rng([SEED, 0, 100 + v + 1000 * seed_stream]).poisson(lam).astype(np.float32))
        else:
            views.append(lam.astype(np.float32))
    return Problem(k=0, dims=tuple(dims), psf_dims=tuple(psf_dims), gt=gt.astype(np.float32), psfs=psfs,
                   views=views, iterations=5, variants=("independent", "efficient", "osem"),
                   meta=dict(scale=1.0, noise=noise))
