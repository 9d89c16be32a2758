"""Pins of the fp64 oracle against what the paper and the mathematics fix (no GPU).

Each test names the PAPER.md passage it rests on.  The pins are chosen so that a dropped
mirror, a wrong centre/crop offset, a missing root, a transposed axis or a wrong compound
product fails at least one of them.
"""
import os
from fractions import Fraction

import numpy as np
import pytest
import scipy.ndimage as ndi
import scipy.signal as sps

import mvd_synth
from oracle import mvd_oracle as O

HERE = os.path.dirname(os.path.abspath(__file__))


@pytest.fixture(scope="module")
def tiny():
    return mvd_synth.make_tiny_asymmetric(dims=(11, 9, 7), psf_dims=(5, 3, 7), n_views=3)


# ---- worked example (tests/golden/rl_1d_worked_example.txt; eq. 13) -----------------
def test_worked_example_eq13():
    rows = [l.split() for l in open(os.path.join(HERE, "golden", "rl_1d_worked_example.txt"))
            if l.strip() and not l.startswith("#")]
    col = lambda i: np.array([float(Fraction(r[i])) for r in rows])
    phi, p, b, q, f, psi1 = (col(i) for i in range(6))
    vol = lambda a: a.reshape(1, 1, -1)
    psi0 = O.initial_estimate([vol(phi)])
    assert np.allclose(psi0, 8.0)
    for same in (O.same_direct, O.same_fft):
        assert np.allclose(same(psi0, vol(p)).ravel(), b, rtol=1e-14)
        assert np.allclose(same(vol(q), O.flip(vol(p))).ravel(), f, rtol=1e-14)
    for variant in O.VARIANTS:
        out = O.deconvolve([vol(phi)], [vol(p)], variant, 1, eps=0.0, psi_floor=0.0)
        assert np.allclose(out.ravel(), psi1, rtol=1e-13)


# ---- P1: brute force == FFT (definition, eq. 3) -----------------------------------
def test_p1_direct_equals_fft(tiny):
    rng = np.random.default_rng(1)
    a = rng.random((7, 9, 11))
    for p in tiny.psfs:
        assert np.abs(O.same_direct(a, p) - O.same_fft(a, p)).max() < 1e-13
        assert np.abs(O.conv_full_direct(a, p) - O.conv_full_fft(a, p)).max() < 1e-13


def test_p1_same_matches_library_conventions(tiny):
    """same() against two library routines that define centring/flip themselves:
    scipy.signal.convolve(mode='same') and scipy.ndimage.correlate(mode='constant')."""
    rng = np.random.default_rng(2)
    a = rng.random((7, 9, 11))
    p = tiny.psfs[0].astype(np.float64)
    ref = sps.convolve(a, p, mode="same", method="direct")
    assert np.abs(O.same_direct(a, p) - ref).max() < 1e-13
    # convolution with the mirrored kernel is correlation with the kernel (L312)
    ref2 = ndi.correlate(a, p, mode="constant", cval=0.0)
    assert np.abs(O.same_direct(a, O.flip(p)) - ref2).max() < 1e-13


@pytest.mark.parametrize("variant,mode", [("independent", "auto"), ("efficient", "auto"),
                                          ("osem", "auto"), ("osem", "plain"), ("efficient", "opt1"),
                                          ("osem", "opt2")])
def test_p1_full_iteration_backends_agree(tiny, variant, mode):
    a = O.deconvolve(tiny.views, tiny.psfs, variant, 2, kernel_mode=mode, backend="direct")
    b = O.deconvolve(tiny.views, tiny.psfs, variant, 2, kernel_mode=mode, backend="fft")
    assert np.abs(a - b).max() / np.abs(a).max() < 1e-12


# ---- P2: one view == classical RL (L421, L628 W = empty set, L780) ------------------------
def test_p2_single_view_is_classical_rl(tiny):
    phi, p = tiny.views[0].astype(np.float64), tiny.psfs[0].astype(np.float64)
    p = p / p.sum()
    # classical RL written with library routines only (scipy.ndimage): blur = convolve,
    # back-projection = correlate with the same kernel (integration over x, L312).
    psi = np.full(phi.shape, phi.mean())
    for _ in range(3):
        b = ndi.convolve(psi, p, mode="constant", cval=0.0)
        psi = psi * ndi.correlate(phi / b, p, mode="constant", cval=0.0)
    outs = [O.deconvolve([phi], [p], v, 3, kernel_mode=m)
            for v in O.VARIANTS for m in ("auto", "plain", "compound", "opt1", "opt2")]
    for o in outs:
        assert np.abs(o - psi).max() / psi.max() < 1e-12
    k = O.back_projector([p], 0, "compound")
    assert np.abs(k - O.flip(p)).max() < 1e-15


# ---- P3: flux identity (eq. 52-55) ----------------------------------------------
def test_p3_flux_identity_pins_mirror_and_centre(tiny):
    psi = np.random.default_rng(3).random(tiny.views[0].shape) + 0.5
    for phi, p in zip(tiny.views, tiny.psfs):
        p = O.normalise(p)
        f = O.rl_factor(psi, phi, p, O.flip(p), eps=0.0)
        assert abs((psi * f).sum() / phi.astype(np.float64).sum() - 1.0) < 1e-12
        # the un-mirrored kernel must NOT conserve flux on an asymmetric PSF
        f_bad = O.rl_factor(psi, phi, p, p, eps=0.0)
        assert abs((psi * f_bad).sum() / phi.astype(np.float64).sum() - 1.0) > 1e-5


def test_p3_combined_root_flux_bound(tiny):
    """eq. 56-62 (AM >= GM): sum psi_new <= mean_v sum phi_v for the rooted combined update."""
    o = O.Oracle(tiny.views, tiny.psfs, "independent")
    bound = np.mean([v.astype(np.float64).sum() for v in tiny.views])
    for _ in range(4):
        o.iterate(1)
        assert o.psi.sum() <= bound * (1 + 1e-12)
    assert o.flux == pytest.approx(o.psi.sum(), rel=1e-15)


# ---- P4: fixed point (L306) ---------------------------------------------------------------
def test_p4_fixed_point(tiny):
    rng = np.random.default_rng(4)
    shape = (15, 13, 17)
    star = rng.random(shape) + 1.0
    psfs = [O.normalise(p) for p in tiny.psfs]
    views = [O.same_fft(star, p) for p in psfs]
    rz, ry, rx = 3, 1, 2            # PSF half sizes for box (Kx,Ky,Kz) = (5,3,7)
    for mode in ("plain", "compound", "opt1", "opt2"):
        for v in range(3):
            k = O.back_projector(psfs, v, mode)
            f = O.rl_factor(star, views[v], psfs[v], k, eps=0.0)
            inner = f[rz:-rz, ry:-ry, rx:-rx]
            assert np.abs(inner - 1.0).max() < 1e-12          # interior: f == 1
            assert np.abs(f - O.same_direct(np.ones(shape), k)).max() < 1e-12   # closed form
            assert f.min() < 0.9                               # faces are darkened (R3 ii)


# ---- P5: identical views (L847) -----------------------------------------------------------
def test_p5_identical_views(tiny):
    phi, p = tiny.views[1], tiny.psfs[1]
    one = O.deconvolve([phi], [p], "independent", 3)
    four = O.deconvolve([phi] * 4, [p] * 4, "independent", 3)
    assert np.abs(one - four).max() / one.max() < 1e-12
    # OSEM with plain kernels and V copies = V single-view iterations per iteration
    osem = O.deconvolve([phi] * 4, [p] * 4, "osem", 1, kernel_mode="plain")
    rl4 = O.deconvolve([phi], [p], "osem", 4, kernel_mode="plain")
    assert np.abs(osem - rl4).max() / rl4.max() < 1e-12
    # and the literal product (eq. 38 as printed) is NOT one view: it takes V unit steps at once
    lit = O.deconvolve([phi] * 4, [p] * 4, "independent", 1, literal_product=True)
    assert np.abs(lit - O.deconvolve([phi], [p], "independent", 1)).max() / one.max() > 1e-3


# ---- P6: delta PSF (L851) -----------------------------------------------------------------
def test_p6_delta_psf(tiny):
    delta = np.zeros((7, 3, 5))
    delta[3, 1, 2] = 1.0
    views = [v.astype(np.float64) + 1.0 for v in tiny.views]
    for mode in ("plain", "compound", "opt1", "opt2"):
        k = O.back_projector([delta] * 3, 0, mode)
        assert np.abs(k - delta).max() < 1e-15
    assert np.allclose(O.deconvolve(views[:1], [delta], "osem", 1), views[0], rtol=1e-14)
    assert np.allclose(O.deconvolve(views, [delta] * 3, "osem", 1), views[-1], rtol=1e-14)
    gm = (views[0] * views[1] * views[2]) ** (1.0 / 3.0)
    assert np.allclose(O.deconvolve(views, [delta] * 3, "efficient", 1), gm, rtol=1e-13)


# ---- P7: compound kernel of Gaussians, closed form (eq. 105 + Gaussian algebra) --------------
def _cov(sxy, sz, deg):
    t = np.radians(deg)
    c, s = np.cos(t), np.sin(t)
    r = np.array([[c, 0, s], [0, 1, 0], [-s, 0, c]])
    return r @ np.diag([sxy ** 2, sxy ** 2, sz ** 2]) @ r.T


def _gauss_box(cov, box):
    kx, ky, kz = box
    uz, uy, ux = np.meshgrid(np.arange(kz) - kz // 2, np.arange(ky) - ky // 2, np.arange(kx) - kx // 2,
                             indexing="ij")
    u = np.stack([ux, uy, uz], -1).astype(float)
    g = np.exp(-0.5 * np.einsum("...i,ij,...j->...", u, np.linalg.inv(cov), u))
    return g / g.sum()


@pytest.mark.parametrize("mode", ["compound", "opt1"])
def test_p7_compound_gaussian_closed_form(mode):
    box = (27, 27, 27)
    angles = (0.0, 50.0, 100.0, 150.0)
    covs = [_cov(1.6, 2.6, a) for a in angles]
    psfs = [_gauss_box(c, box) for c in covs]
    for v in range(len(covs)):
        k = O.back_projector(psfs, v, mode)
        lam = np.linalg.inv(covs[v])
        for w in range(len(covs)):
            if w != v:
                # Gaussian * Gaussian adds covariances; pointwise product adds precisions
                lam = lam + np.linalg.inv(covs[v] + (2 if mode == "compound" else 1) * covs[w])
        ref = _gauss_box(np.linalg.inv(lam), box)
        assert np.linalg.norm(k - ref) / np.linalg.norm(ref) < 2e-6
    # a mistake such as leaving out P_w* or the P_v* factor is visible at this tolerance
    wrong = O.back_projector(psfs, 0, "opt1" if mode == "compound" else "compound")
    lam = np.linalg.inv(covs[0]) + sum(np.linalg.inv(covs[0] + (2 if mode == "compound" else 1) * covs[w])
                                       for w in (1, 2, 3))
    assert np.linalg.norm(wrong - _gauss_box(np.linalg.inv(lam), box)) > 1e-3 * np.linalg.norm(wrong)


def test_opt2_is_power_of_mirrored_psf(tiny):
    psfs = [O.normalise(p) for p in tiny.psfs]
    k = O.back_projector(psfs, 2, "opt2")
    ref = O.flip(psfs[2]) ** 3
    assert np.abs(k - ref / ref.sum()).max() < 1e-16


def test_compound_is_asymmetric_product_on_psf_box(tiny):
    """eq. 105 on non-symmetric PSFs, written out tap by tap (triple sum over offsets measured
    from each kernel's centre) for two output taps; k is normalised, so compare their ratio."""
    psfs = [O.normalise(p) for p in tiny.psfs]
    k = O.back_projector(psfs, 0, "compound", backend="direct")
    pvs = O.flip(psfs[0])
    c = tuple(n // 2 for n in pvs.shape)

    def t_vw(pw, u):                                    # (P_v* * P_w * P_w*)(u - c)
        pws = O.flip(pw)
        tot = 0.0
        for a in np.ndindex(pvs.shape):
            for b in np.ndindex(pw.shape):
                idx = tuple((u[i] - c[i]) - (a[i] - c[i]) - (b[i] - c[i]) + c[i] for i in range(3))
                if all(0 <= idx[i] < pws.shape[i] for i in range(3)):
                    tot += pvs[a] * pw[b] * pws[idx]
        return tot

    def tap(u):
        return pvs[u] * t_vw(psfs[1], u) * t_vw(psfs[2], u)

    u1, u2 = (1, 2, 0), c
    assert k[u1] / k[u2] == pytest.approx(tap(u1) / tap(u2), rel=1e-12)


# ---- P8: monotone likelihood (eq. 39-43) --------------------------------------------
def test_p8_likelihood_monotone(tiny):
    """The proof needs sum_x P(x|xi) = 1 wherever psi* > 0 (Jensen, eq. 46-47) and equal view
    integrals (eq. 62): psi* supported >= r away from the faces, noise-free views."""
    rng = np.random.default_rng(8)
    shape = (19, 11, 15)
    star = np.zeros(shape)
    star[3:-3, 1:-1, 2:-2] = rng.random((13, 9, 11)) ** 3 * 50 + 0.1
    psfs = [O.normalise(p) for p in tiny.psfs]
    views = [O.same_fft(star, p) for p in psfs]
    for v in views:
        assert v.sum() == pytest.approx(star.sum(), rel=1e-13)
    mask = star > 0
    for kernel_mode in ("plain",):
        o = O.Oracle(views, psfs, "independent", kernel_mode=kernel_mode, eps=0.0, psi_floor=0.0)
        last = -np.inf
        for _ in range(15):
            o.iterate(1)
            l = float(-(star[mask] * np.log(star[mask] / o.psi[mask])).sum())     # eq. 39
            assert l >= last - 1e-9
            assert o.psi.sum() <= star.sum() * (1 + 1e-12)                         # eq. 56
            last = l
    # without the root the printed product of eq. 38 does not keep eq. 56
    lit = O.Oracle(views, psfs, "independent", literal_product=True, eps=0.0, psi_floor=0.0)
    lit.iterate(3)
    assert lit.psi.sum() > star.sum() * 1.01 or not np.isfinite(lit.psi).all()


# ---- P9: ordering of the variants (L807-809) -------------------------------------------------
def test_p9_variant_ordering():
    prob = mvd_synth.make_problem(2, dims=(40, 36, 32), psf_dims=(9, 9, 17), noise=False)
    gt = prob.gt.astype(np.float64)
    inner = (slice(8, -8), slice(4, -4), slice(4, -4))
    err = {}
    for variant in O.VARIANTS:
        o = O.Oracle(prob.views, prob.psfs, variant)
        e = []
        for _ in range(6):
            o.iterate(1)
            e.append(O.average_difference(o.psi[inner], gt[inner]))
        assert all(b < a for a, b in zip(e, e[1:])), variant      # every variant improves
        err[variant] = e[-1]
    assert err["osem"] < err["efficient"] < err["independent"]


# ---- blocks (L64, L943; R13) -----------------------------------------------------------------
def test_blocked_equals_whole_when_one_block(tiny):
    whole = O.deconvolve(tiny.views, tiny.psfs, "osem", 2)
    blk = O.deconvolve_blocked(tiny.views, tiny.psfs, tiny.views[0].shape, "osem", 2)
    assert np.abs(whole - blk).max() / whole.max() < 1e-13


def test_blocked_is_close_to_whole_in_block_interiors():
    prob = mvd_synth.make_problem(1, dims=(32, 32, 32), psf_dims=(5, 5, 9), n_views=2)
    whole = O.deconvolve(prob.views, prob.psfs, "osem", 1)
    blk = O.deconvolve_blocked(prob.views, prob.psfs, (16, 16, 16), "osem", 1, halo_zyx=(8, 4, 4))
    # halo = 2r: after ONE osem iteration of 2 views the dependence radius is 2 views x 2 convs x r,
    # so only block centres agree closely; the blocked mode is an approximation (L943)
    rel = np.abs(whole - blk) / np.maximum(whole, 1e-6)
    assert np.median(rel) < 1e-2
    assert blk.shape == whole.shape and np.isfinite(blk).all()


def _dependence_exact_case(n_views, seed):
    """Asymmetric PSFs of different half-size per axis, a volume that the blocks tile raggedly."""
    rng = np.random.default_rng([13080730, 600 + seed])
    shape = (23, 19, 26)                                        # (Nz, Ny, Nx)
    box = (5, 3, 7)                                             # (Kx, Ky, Kz): r = (2, 1, 3)
    psfs = [mvd_synth.random_psf(rng, box) for _ in range(n_views)]
    views = [rng.random(shape) * 40 + 5 for _ in range(n_views)]
    return views, psfs, (3, 1, 2)                               # r in (z, y, x) order


@pytest.mark.parametrize("block_zyx", [(8, 7, 9), (23, 6, 26), (5, 19, 4), (12, 10, 13)])
def test_blocked_equals_whole_exactly_when_halo_covers_the_dependence_radius(block_zyx):
    """R13 / L943.  One view-update reads psi within 2r of a voxel (b = psi*P needs r, f = q*K another
    r) and psi^0 is the same constant on both sides, so with V = 1, one iteration and halo = 2r the
    block-wise result IS the whole-volume result at every voxel (clipping the halo at a volume face
    is the same zero extension).  A +-1 error in the halo clip or the paste offset fails this."""
    views, psfs, r = _dependence_exact_case(1, 0)
    whole = O.deconvolve(views, psfs, "osem", 1)
    blk = O.deconvolve_blocked(views, psfs, block_zyx, "osem", 1, halo_zyx=tuple(2 * x for x in r))
    assert np.abs(blk - whole).max() / whole.max() < 1e-12
    # all three schedules coincide for one view (P2), blocked too
    blk2 = O.deconvolve_blocked(views, psfs, block_zyx, "efficient", 1, halo_zyx=tuple(2 * x for x in r))
    assert np.abs(blk2 - whole).max() / whole.max() < 1e-12


def test_blocked_exact_for_several_views_and_iterations_with_the_full_radius():
    """Sequential updates chain: V views x n iterations read psi within 2r*V*n; halo of that size is exact."""
    views, psfs, r = _dependence_exact_case(2, 1)
    whole = O.deconvolve(views, psfs, "osem", 1, kernel_mode="plain")
    halo = tuple(2 * x * 2 for x in r)
    blk = O.deconvolve_blocked(views, psfs, (8, 7, 9), "osem", 1, halo_zyx=halo, kernel_mode="plain")
    assert np.abs(blk - whole).max() / whole.max() < 1e-12


def test_blocked_with_too_small_a_halo_differs_at_block_borders_only():
    """Negative control: halo = r (the BASELINE rule) is NOT exact: voxels within r of an inner block
    border see b computed from a zero-extended psi.  Voxels >= 2r - halo = r inside their block are exact."""
    views, psfs, r = _dependence_exact_case(1, 2)
    whole = O.deconvolve(views, psfs, "osem", 1)
    block = (12, 10, 13)
    blk = O.deconvolve_blocked(views, psfs, block, "osem", 1, halo_zyx=r)
    rel = np.abs(blk - whole) / whole.max()
    assert rel.max() > 1e-4                                      # the borders do differ
    exact = np.zeros(whole.shape, bool)                          # distance >= r from every inner block border
    for (z0, z1), (y0, y1), (x0, x1) in O.block_grid(whole.shape, block):
        lo = [z0 + (r[0] if z0 > 0 else 0), y0 + (r[1] if y0 > 0 else 0), x0 + (r[2] if x0 > 0 else 0)]
        hi = [z1 - (r[0] if z1 < whole.shape[0] else 0), y1 - (r[1] if y1 < whole.shape[1] else 0),
              x1 - (r[2] if x1 < whole.shape[2] else 0)]
        exact[lo[0]:hi[0], lo[1]:hi[1], lo[2]:hi[2]] = True
    assert exact.any() and (~exact).any()
    assert rel[exact].max() < 1e-12
    assert rel[~exact].max() == rel.max()


def test_blocked_delta_psf_needs_no_halo():
    """L851: with delta PSFs nothing is read from a neighbour: halo 0, any block shape == whole."""
    views, _, _ = _dependence_exact_case(3, 3)
    delta = np.zeros((3, 3, 3))
    delta[1, 1, 1] = 1.0
    for variant in ("osem", "efficient"):
        whole = O.deconvolve(views, [delta] * 3, variant, 2)
        blk = O.deconvolve_blocked(views, [delta] * 3, (7, 5, 11), variant, 2, halo_zyx=(0, 0, 0))
        assert np.abs(blk - whole).max() / whole.max() < 1e-13      # FFT sizes differ per block: rounding only


def test_view_update_is_the_osem_step():
    """Oracle.view_update(v) (what bench.py times) is exactly one line of eq. 109-112: V of them = iterate(1)."""
    views, psfs, _ = _dependence_exact_case(3, 4)
    a = O.Oracle(views, psfs, "osem")
    b = O.Oracle(views, psfs, "osem")
    a.iterate(1)
    for v in range(3):
        b.view_update(v)
    assert np.array_equal(a.psi, b.psi) and a.flux == b.flux and a.l1_change == b.l1_change
    with pytest.raises(ValueError):
        O.Oracle(views, psfs, "efficient").view_update(0)


# --------------------------------------------------------------------------------------
# Tikhonov regularisation (L64, L869, ref. 20; reading R14: no formula in PAPER.md -> parity unpinned by the
# paper; what is pinned here is that the oracle computes the penalised M-step it documents)
# --------------------------------------------------------------------------------------
def test_tikhonov_update_solves_the_penalised_m_step(tiny):
    """With u the unregularised update, the regularised one is the positive root of (lam/2) psi^2 + psi - u = 0,
    i.e. the stationary point of u log(psi) - psi - (lam/4) psi^2 per voxel; checked from the UNREGULARISED oracle's
    update (so a wrong factor, sign or a regularisation applied to f instead of psi*f fails)."""
    rng = np.random.default_rng(11)
    psi0 = rng.random(tiny.views[0].shape) * 80 + 1
    for variant in ("osem", "efficient"):
        plain = O.Oracle(tiny.views[:1] if variant == "osem" else tiny.views, tiny.psfs[:1] if variant == "osem" else tiny.psfs,
                         variant, psi0=psi0)
        plain.iterate(1)
        u = plain.psi                                              # psi0 * f (osem, V = 1) / psi0 * (prod f)^(1/V)
        for lam in (0.0006, 0.006, 0.06, 2.0):                     # the paper's values (L145, L151) and a large one
            reg = O.Oracle(plain.views, [p.copy() for p in plain.psfs], variant, psi0=psi0, tikhonov_lambda=lam)
            reg.iterate(1)
            r = reg.psi
            assert np.allclose(0.5 * lam * r * r + r, u, rtol=1e-12, atol=0)          # the quadratic
            assert np.allclose(u / r - 1.0 - 0.5 * lam * r, 0.0, atol=1e-10)         # the stationarity condition
            assert np.all(r > 0) and np.all(r < u)                                    # damped, positive
            assert np.allclose(r, (np.sqrt(1 + 2 * lam * u) - 1) / lam, rtol=1e-9)    # the textbook root formula
    # closed values: u = 4, lam = 1/2 -> psi^2/4 + psi - 4 = 0 -> psi = 2(sqrt(5) - 1)
    assert O.tikhonov(np.array([4.0]), 0.5)[0] == pytest.approx(2 * (np.sqrt(5.0) - 1), rel=1e-15)
    assert O.tikhonov(np.array([1.5]), 1.0)[0] == pytest.approx(1.0, rel=1e-15)        # psi^2/2 + psi - 3/2 = 0 -> psi = 1


def test_tikhonov_zero_lambda_is_the_plain_update_and_lambda_orders_the_flux(tiny):
    a = O.deconvolve(tiny.views, tiny.psfs, "osem", 3)
    b = O.deconvolve(tiny.views, tiny.psfs, "osem", 3, tikhonov_lambda=0.0)
    assert np.array_equal(a, b)
    c = O.deconvolve(tiny.views, tiny.psfs, "osem", 3, tikhonov_lambda=1e-12)
    assert np.allclose(a, c, rtol=1e-7)                           # lam*u/2 ~ 1e-10 per update, amplified by the iteration
    # first order in lambda: psi = u - lam u^2 / 2 + O(lam^2)
    u = np.array([0.5, 3.0, 40.0])
    lam = 1e-6
    assert np.allclose(O.tikhonov(u, lam), u - 0.5 * lam * u * u, rtol=1e-9)
    flux = []
    for lam in (0.0, 0.0006, 0.006, 0.06):
        o = O.Oracle(tiny.views, tiny.psfs, "osem", tikhonov_lambda=lam)
        o.iterate(2)
        flux.append(o.flux)
    assert all(y < x for x, y in zip(flux, flux[1:]))              # more regularisation, less flux
    with pytest.raises(ValueError):
        O.Oracle(tiny.views, tiny.psfs, "osem", tikhonov_lambda=-1.0)


# --------------------------------------------------------------------------------------
# section 12 (L891-903): weights of partially overlapping views
# --------------------------------------------------------------------------------------
def test_weights_interpolate_between_old_estimate_and_rl_step(tiny):
    """L897: the weight is "the fraction of change suggested by a Lucy-Richardson update step":
    per voxel psi_w = (1-w) psi + w psi_RL.  Checked against the (pinned) unweighted update, so a
    wrong sign or a dropped '1 +' fails; w = 1 is the plain update, w = 0 leaves psi untouched."""
    rng = np.random.default_rng(3)
    views, psfs = tiny.views[:1], tiny.psfs[:1]
    psi0 = rng.random(views[0].shape) * 50 + 1
    plain = O.Oracle(views, psfs, "osem", kernel_mode="plain", psi0=psi0)
    plain.iterate(1)
    w = rng.random(views[0].shape)
    w[:2] = 0.0
    w[-2:] = 1.0
    ow = O.Oracle(views, psfs, "osem", kernel_mode="plain", psi0=psi0, weights=[w])
    ow.iterate(1)
    assert np.allclose(ow.psi, (1 - w) * psi0 + w * plain.psi, rtol=1e-13, atol=0)
    assert np.array_equal(ow.psi[:2], psi0[:2])
    assert np.allclose(ow.psi[-2:], plain.psi[-2:], rtol=1e-14)


def test_unit_weights_change_nothing_and_zero_view_is_skipped(tiny):
    ones = [np.ones(tiny.views[0].shape)] * 3
    a = O.deconvolve(tiny.views, tiny.psfs, "osem", 2)
    b = O.deconvolve(tiny.views, tiny.psfs, "osem", 2, weights=ones)
    assert np.allclose(a, b, rtol=1e-14)
    # a view with weight 0 everywhere contributes nothing: same as running without that view's update
    w = [np.ones(tiny.views[0].shape), np.zeros(tiny.views[0].shape), np.ones(tiny.views[0].shape)]
    c = O.Oracle(tiny.views, tiny.psfs, "osem", kernel_mode="plain", weights=w)
    c.iterate(1)
    d = O.Oracle([tiny.views[0], tiny.views[2]], [tiny.psfs[0], tiny.psfs[2]], "osem", kernel_mode="plain",
                 psi0=O.initial_estimate(tiny.views))
    d.iterate(1)
    assert np.allclose(c.psi, d.psi, rtol=1e-13)
    with pytest.raises(ValueError):
        O.Oracle(tiny.views, tiny.psfs, "efficient", weights=ones)


def test_blending_weights_closed_form():
    """L891: 1 in the central part, cosine ramp to 0 at the faces of the view's box, 0 outside."""
    shape, lo, hi, border = (9, 30, 40), (0, 4, 10), (9, 26, 34), 6
    w = O.blending_weights(shape, lo, hi, border)
    assert w.min() >= 0 and w.max() <= 1
    assert np.all(w[:, :4] == 0) and np.all(w[:, 26:] == 0) and np.all(w[:, :, :10] == 0) and np.all(w[:, :, 34:] == 0)
    # along x through the centre of y (z spans 9 voxels with border 6: the z ramp is a constant factor)
    line = w[4, 15, :]
    zf, yf = 0.5 * (1 - np.cos(np.pi * 4.5 / 6)), 1.0
    for x, d in ((10, 0.5), (12, 2.5), (13, 3.5), (33, 0.5), (31, 2.5)):
        assert line[x] == pytest.approx(zf * yf * 0.5 * (1 - np.cos(np.pi * d / border)), rel=1e-12)
    assert np.allclose(line[16:28], zf)                           # plateau
    assert np.allclose(line[10:34], line[10:34][::-1])            # symmetric
    assert np.all(np.diff(line[10:17]) > 0)                       # monotone ramp
    # half-way up the ramp the weight is one half (cos(pi/2) = 0)
    assert 0.5 * (1 - np.cos(np.pi * 3.0 / 6)) == pytest.approx(0.5)


def test_normalise_weights_never_increases_and_caps_the_sum():
    rng = np.random.default_rng(9)
    ws = [rng.random((4, 5, 6)) for _ in range(4)]
    for cap in (1.0, 2.0):
        out = O.normalise_weights(ws, cap)
        tot = np.sum(out, axis=0)
        assert np.all(tot <= cap + 1e-12)
        for a, b in zip(ws, out):
            assert np.all(b <= a + 1e-15)                          # "never increased above 1" (L895)
        untouched = np.sum(ws, axis=0) <= cap
        for a, b in zip(ws, out):
            assert np.array_equal(a[untouched], b[untouched])
        capped = ~untouched
        assert np.allclose(tot[capped], cap)


def test_quality_metrics_are_the_library_definitions():
    """L48 cross-correlation = Pearson coefficient (numpy.corrcoef); L127 average difference = mean |a-b|."""
    rng = np.random.default_rng(4)
    a, b = rng.random((5, 6, 7)), rng.random((5, 6, 7))
    assert O.cross_correlation(a, b) == pytest.approx(np.corrcoef(a.ravel(), b.ravel())[0, 1], rel=1e-12)
    assert O.cross_correlation(a, 3 * a + 2) == pytest.approx(1.0, rel=1e-12)
    assert O.cross_correlation(a, -a) == pytest.approx(-1.0, rel=1e-12)
    assert O.average_difference(a, a + 0.25) == pytest.approx(0.25, rel=1e-12)
    assert O.average_difference(a, b) == pytest.approx(np.mean(np.abs(a - b)), rel=1e-14)
