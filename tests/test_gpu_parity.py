"""Parity of the CUDA path (through the C ABI, via the thin binding) with the fp64 oracle.

Every test runs on the same seeded inputs on both sides (mvd_synth) and compares element by
element.  Tolerances are the ones BASELINE.json:north_star states:
    relative L2 <= 1e-5 after 1 iteration, <= 1e-4 after >= 10 iterations,
    max per-voxel relative error <= 1e-3 with the denominator max(|oracle|, psi_floor)  (R12).
The oracle side never sees a value produced by the CUDA path.
"""
import numpy as np
import pytest

import mvd_synth
from oracle import mvd_oracle as O

pytestmark = pytest.mark.gpu

FLOOR = 1e-6
TOL_L2_1 = 1e-5
TOL_L2_10 = 1e-4
TOL_MAX = 1e-3


def errors(g, o, floor=FLOOR):
    g = np.asarray(g, dtype=np.float64)
    o = np.asarray(o, dtype=np.float64)
    rel_l2 = np.linalg.norm((g - o).ravel()) / np.linalg.norm(o.ravel())
    rel_max = float((np.abs(g - o) / np.maximum(np.abs(o), floor)).max())
    return float(rel_l2), rel_max


def check(g, o, iters, what=""):
    assert np.isfinite(g).all(), what
    l2, mx = errors(g, o)
    tol = TOL_L2_1 if iters <= 1 else TOL_L2_10
    assert l2 <= tol, "%s: rel-L2 %.3g > %.1g after %d iterations" % (what, l2, tol, iters)
    assert mx <= TOL_MAX, "%s: max per-voxel rel %.3g after %d iterations" % (what, mx, iters)
    return l2, mx


@pytest.fixture(scope="module")
def mvd():
    import torch
    import paper_1308_0730_b200 as m
    assert torch.cuda.is_available()
    m.load_library()          # fails loudly if libmvd.so is missing: there is no fallback
    return m


def to_dev(arrs):
    import torch
    return [torch.from_numpy(np.ascontiguousarray(a)).cuda() for a in arrs]


def gpu_checkpoints(mvd, prob, variant, mode, checkpoints, **kw):
    views = to_dev(prob.views)
    if kw.get("use_graph"):
        import torch
        torch.cuda.synchronize()
        kw["stream"] = torch.cuda.Stream()       # the legacy default stream cannot be captured
    d = mvd.Deconvolver(views, prob.psfs, variant=variant, kernel_mode=mode, **kw)
    out, done = {}, 0
    for c in checkpoints:
        d.iterate(c - done)
        done = c
        out[c] = d.get_estimate_host()
    stats = d.get_stats()
    d.close()
    return out, stats


def oracle_checkpoints(prob, variant, mode, checkpoints, **kw):
    o = O.Oracle(prob.views, prob.psfs, variant, kernel_mode=mode, **kw)
    out, done = {}, 0
    for c in checkpoints:
        o.iterate(c - done)
        done = c
        out[c] = o.psi.copy()
    return out, o


# ------------------------------------------------------------------------------------------
# k = 0: tiny volume, random NON-symmetric PSFs (the case a missing mirror / centre offset fails)
# ------------------------------------------------------------------------------------------
@pytest.fixture(scope="module")
def tiny():
    return mvd_synth.make_tiny_asymmetric()


ALL_MODES = [("independent", "auto"), ("efficient", "auto"), ("osem", "auto"), ("osem", "plain"),
             ("efficient", "opt1"), ("osem", "opt1"), ("osem", "opt2"), ("independent", "compound")]


@pytest.mark.parametrize("variant,mode", ALL_MODES)
def test_tiny_asymmetric_all_variants(mvd, tiny, variant, mode):
    g, st = gpu_checkpoints(mvd, tiny, variant, mode, (1, 3, 10))
    o, orc = oracle_checkpoints(tiny, variant, mode, (1, 3, 10))
    for c in (1, 3, 10):
        check(g[c], o[c], c, "%s/%s" % (variant, mode))
    assert st["iterations_done"] == 10
    assert st["flux"] == pytest.approx(orc.flux, rel=1e-5)
    assert st["l1_change"] == pytest.approx(orc.l1_change, rel=2e-3, abs=1e-3 * orc.flux * 1e-3)


def test_tiny_direct_sum_oracle_backend(mvd, tiny):
    """The brute-force (direct-sum) oracle, not only its FFT back-end, agrees with the GPU."""
    small = mvd_synth.make_tiny_asymmetric(dims=(12, 10, 9), psf_dims=(5, 3, 7), n_views=2)
    g, _ = gpu_checkpoints(mvd, small, "osem", "auto", (2,))
    o = O.deconvolve(small.views, small.psfs, "osem", 2, backend="direct")
    check(g[2], o, 2, "direct-sum")


def test_tiny_literal_product(mvd, tiny):
    """literal_product=1: the bare product of eq. 2/38/104 (R1), parity for one iteration."""
    g, _ = gpu_checkpoints(mvd, tiny, "efficient", "auto", (1,), literal_product=True)
    o, _ = oracle_checkpoints(tiny, "efficient", "auto", (1,), literal_product=True)
    check(g[1], o[1], 1, "literal product")


@pytest.mark.parametrize("mode", ["plain", "compound", "opt1", "opt2"])
def test_back_projectors_match_oracle(mvd, tiny, mode):
    """Device precompute of eq. 105 / 107 / 108 (fp64) against the oracle's construction."""
    d = mvd.Deconvolver(to_dev(tiny.views), tiny.psfs, variant="osem", kernel_mode=mode)
    psfs = [O.normalise(p) for p in tiny.psfs]
    for v in range(tiny.n_views):
        k = d.get_back_projector(v)
        ref = O.back_projector(psfs, v, mode, backend="direct")
        assert np.abs(k - ref).max() <= 1e-12 * ref.max(), (mode, v)
    d.close()


def test_back_projector_mixed_psf_sizes(mvd):
    """R6: views may have PSF boxes of different sizes; factors are centre-aligned and cropped."""
    rng = np.random.default_rng([mvd_synth.generate.SEED, 77])
    boxes = [(5, 7, 9), (7, 5, 5), (3, 9, 7)]
    psfs = [mvd_synth.random_psf(rng, b) for b in boxes]
    views = [(50 * rng.random((20, 22, 26)) + 5).astype(np.float32) for _ in boxes]
    d = mvd.Deconvolver(to_dev(views), psfs, variant="osem")
    npsfs = [O.normalise(p) for p in psfs]
    for v in range(3):
        ref = O.back_projector(npsfs, v, "compound", backend="direct")
        assert np.abs(d.get_back_projector(v) - ref).max() <= 1e-12 * ref.max()
    d.iterate(2)
    g = d.get_estimate_host()
    d.close()
    check(g, O.deconvolve(views, psfs, "osem", 2), 2, "mixed PSF boxes")


@pytest.mark.parametrize("dims,box", [((24, 20, 18), (5, 7, 9)), ((33, 17, 9), (3, 5, 7)),
                                      ((7, 40, 5), (7, 3, 5)), ((95, 31, 22), (9, 9, 15)),
                                      ((6, 12, 4), (9, 5, 7))])   # last: PSF box larger than the volume
def test_single_convolution_matches_direct_definition(mvd, dims, box):
    """One zero-extended 'same' convolution through the pencil-FFT path (S1/S3) against the
    oracle, for PSF and back-projector, odd and even Nx, ragged tiles."""
    p = mvd_synth.make_tiny_asymmetric(dims=dims, psf_dims=box, n_views=2)
    d = mvd.Deconvolver(to_dev(p.views), p.psfs, variant="osem", kernel_mode="plain")
    rng = np.random.default_rng(5)
    src = rng.random(p.views[0].shape).astype(np.float32) * 10
    import torch
    for v in range(2):
        pn = O.normalise(p.psfs[v])
        for which, k in ((0, pn), (1, O.flip(pn))):
            got = d.convolve(v, which, torch.from_numpy(src).cuda()).cpu().numpy()
            ref = O.same_fft(src, k)
            l2, mx = errors(got, ref)
            assert l2 < 2e-6 and mx < 1e-4, (dims, box, v, which, l2, mx)
    d.close()


# ------------------------------------------------------------------------------------------
# invariants on the GPU output itself (T4): flux identity, fixed point, identical views, delta
# ------------------------------------------------------------------------------------------
def test_gpu_flux_identity(mvd, tiny):
    """P3 (eq. 52-55): plain kernel, one view-update => sum psi_new = sum phi_v."""
    d = mvd.Deconvolver(to_dev(tiny.views[:1]), tiny.psfs[:1], variant="osem", kernel_mode="plain")
    d.iterate(1)
    st = d.get_stats()
    d.close()
    assert st["flux"] == pytest.approx(float(tiny.views[0].astype(np.float64).sum()), rel=2e-6)


def test_gpu_fixed_point(mvd):
    """P4 (L306): noise-free data from psi*, psi = psi* => f = same(1, K): 1 in the interior."""
    import torch
    p = mvd_synth.make_tiny_asymmetric(dims=(30, 28, 26), psf_dims=(5, 5, 7), n_views=2, noise=False)
    pn = [O.normalise(q) for q in p.psfs]
    views = [O.same_fft(p.gt, q).astype(np.float32) for q in pn]
    d = mvd.Deconvolver(to_dev(views), p.psfs, variant="osem", kernel_mode="plain",
                        psi0=torch.from_numpy(p.gt).cuda())
    d.iterate(1)
    g = d.get_estimate_host()
    d.close()
    # view 0 darkens the faces (R3 ii); view 1 then sees b != phi within 2r of a face and spreads
    # that by another r: the exact fixed point survives at distance >= 3r = (9,6,6) from the faces
    ratio = g / p.gt
    inner = ratio[9:-9, 6:-6, 6:-6]
    assert np.abs(inner - 1).max() < 5e-6
    # one view alone: f = same(1, K) is 1 at distance >= r and < 1 on the faces
    d = mvd.Deconvolver(to_dev(views[:1]), p.psfs[:1], variant="osem", kernel_mode="plain",
                        psi0=torch.from_numpy(p.gt).cuda())
    d.iterate(1)
    ratio = d.get_estimate_host() / p.gt
    d.close()
    assert np.abs(ratio[3:-3, 2:-2, 2:-2] - 1).max() < 5e-6
    assert ratio.min() > 0.05 and ratio.max() < 1 + 5e-6 and ratio[0, 0, 0] < 0.6


def test_gpu_identical_views_equal_single_view(mvd, tiny):
    """P5 (L847): V copies of one (phi, P), combined + root == one view."""
    one, _ = gpu_checkpoints(mvd, _sub(tiny, [0]), "independent", "auto", (3,))
    four, _ = gpu_checkpoints(mvd, _sub(tiny, [0, 0, 0, 0]), "independent", "auto", (3,))
    l2, mx = errors(four[3], one[3])
    assert l2 < 3e-6 and mx < 1e-4


def test_many_views_product_neither_overflows_nor_underflows(mvd, tiny):
    """Combined variants keep a running fp32 product of the f_v.  With 40 views and an estimate far below (above) the
    data every factor is ~30 (~1/30) and the bare product leaves the fp32 range; beyond 16 views the library roots
    every factor before it enters the product.  Result: that of the oracle (P5: identical views == one view)."""
    import torch
    V = 40
    p = _sub(tiny, [0] * V)
    mean = float(np.mean(tiny.views[0], dtype=np.float64))
    for scale in (1.0 / 30.0, 30.0):
        psi0 = np.full(tiny.views[0].shape, mean * scale, np.float32)
        for variant in ("independent", "efficient"):
            d = mvd.Deconvolver(to_dev(p.views), p.psfs, variant=variant, psi0=torch.from_numpy(psi0).cuda())
            d.iterate(1)
            g1 = d.get_estimate_host()
            d.iterate(2)
            g3 = d.get_estimate_host()
            d.close()
            o = O.Oracle(p.views, p.psfs, variant, psi0=psi0)
            o.iterate(1)
            check(g1, o.psi, 1, "40 views %s x%g" % (variant, scale))
            o.iterate(2)
            check(g3, o.psi, 3, "40 views %s x%g" % (variant, scale))
    # the view-parallel calls take the same guard (partial products of rooted factors, no root in apply_product)
    views = to_dev(p.views)
    psi0 = np.full(tiny.views[0].shape, mean / 30.0, np.float32)
    ranks = [mvd.Deconvolver([views[v] for v in mvd.split_views(V, 2, r)], p.psfs, variant="independent",
                             local_views=mvd.split_views(V, 2, r), psi0=torch.from_numpy(psi0).cuda()) for r in range(2)]
    for d in ranks:
        d.partial_product()
    torch.cuda.synchronize()
    prod = ranks[0].product_tensor() * ranks[1].product_tensor()
    for d in ranks:
        d.product_tensor().copy_(prod)
        d.apply_product(V)
    o = O.Oracle(p.views, p.psfs, "independent", psi0=psi0)
    o.iterate(1)
    check(ranks[0].get_estimate_host(), o.psi, 1, "40 views, view-parallel")
    for d in ranks:
        d.close()


def test_gpu_delta_psf(mvd, tiny):
    """P6 (L851): delta PSFs: OSEM ends on the last view, combined on the geometric mean."""
    delta = np.zeros((3, 3, 3), np.float32)
    delta[1, 1, 1] = 1
    views = [v + 1 for v in tiny.views]
    prob = mvd_synth.Problem(0, tiny.dims, (3, 3, 3), tiny.gt, [delta] * 3, views, 1, ())
    g, _ = gpu_checkpoints(mvd, prob, "osem", "auto", (1,))
    check(g[1], views[-1], 1, "delta OSEM")
    g, _ = gpu_checkpoints(mvd, prob, "efficient", "auto", (1,))
    gm = np.exp(np.mean([np.log(v.astype(np.float64)) for v in views], axis=0))
    check(g[1], gm, 1, "delta combined")


def _sub(prob, idx):
    return mvd_synth.Problem(prob.k, prob.dims, prob.psf_dims, prob.gt, [prob.psfs[i] for i in idx],
                             [prob.views[i] for i in idx], prob.iterations, prob.variants)


def test_set_estimate_resume_and_graph_replay(mvd, tiny):
    """mvd_set_estimate / psi0 resume reproduce an uninterrupted run; CUDA-graph replay of the
    iteration gives bit-identical results to plain launches."""
    a, _ = gpu_checkpoints(mvd, tiny, "osem", "auto", (2, 4))
    import torch
    d = mvd.Deconvolver(to_dev(tiny.views), tiny.psfs, variant="osem", psi0=torch.from_numpy(a[2]).cuda())
    d.iterate(2)
    assert np.array_equal(d.get_estimate_host(), a[4])
    d.set_estimate(torch.from_numpy(a[2]).cuda())
    d.iterate(2)
    assert np.array_equal(d.get_estimate_host(), a[4])
    d.close()
    for variant in ("osem", "efficient"):
        p, _ = gpu_checkpoints(mvd, tiny, variant, "auto", (3,))
        g, _ = gpu_checkpoints(mvd, tiny, variant, "auto", (3,), use_graph=True)
        assert np.array_equal(p[3], g[3])
    with pytest.raises(mvd.MvdError):                # default stream + graph: refused at create
        mvd.Deconvolver(to_dev(tiny.views), tiny.psfs, use_graph=True, stream=torch.cuda.default_stream())


@pytest.mark.parametrize("variant", ["osem", "efficient"])
def test_stats_after_set_estimate_graph_equals_plain_and_oracle(mvd, tiny, variant):
    """mvd_get_stats after mvd_set_estimate + mvd_iterate: the replayed graph's update kernel wrote its
    partials, so graph and plain-launch contexts report the same flux and l1_change, those of the oracle."""
    import torch
    start = (tiny.gt * 0.5 + 7.0).astype(np.float32)
    o = O.Oracle(tiny.views, tiny.psfs, variant, psi0=start)
    o.iterate(2)
    got = {}
    for use_graph in (False, True):
        torch.cuda.synchronize()
        kw = {"use_graph": True, "stream": torch.cuda.Stream()} if use_graph else {}
        d = mvd.Deconvolver(to_dev(tiny.views), tiny.psfs, variant=variant, **kw)
        d.iterate(1)                                     # the graph is captured on some other estimate
        d.set_estimate(torch.from_numpy(start).cuda())
        st0 = d.get_stats()                              # no update since set_estimate: flux of psi, no change
        assert st0["l1_change"] == 0.0 and st0["flux"] == pytest.approx(float(start.astype(np.float64).sum()), rel=1e-6)
        d.iterate(2)
        got[use_graph] = (d.get_stats(), d.get_estimate_host())
        d.close()
    assert got[True][0]["flux"] == got[False][0]["flux"] and got[True][0]["l1_change"] == got[False][0]["l1_change"]
    assert np.array_equal(got[True][1], got[False][1])
    assert got[True][0]["l1_change"] > 0
    assert got[True][0]["flux"] == pytest.approx(o.flux, rel=1e-5)
    assert got[True][0]["l1_change"] == pytest.approx(o.l1_change, rel=2e-3)


def test_restart_on_new_view_contents_equals_a_fresh_context(mvd, tiny):
    """mvd_restart (time-lapse, L64 / L242): new contents in the same view buffers, same PSFs: bit-identical to a
    context created on those contents, with plain launches and under graph replay; the oracle agrees."""
    import torch
    second = mvd_synth.make_tiny_asymmetric(seed_stream=3)        # another "time-point": other data ...
    second_views = [v.copy() for v in second.views]
    for use_graph in (False, True):
        torch.cuda.synchronize()
        kw = {"use_graph": True, "stream": torch.cuda.Stream()} if use_graph else {}
        bufs = to_dev(tiny.views)
        d = mvd.Deconvolver(bufs, tiny.psfs, variant="osem", **kw)
        d.iterate(3)
        first = d.get_estimate_host()
        copy_stream = torch.cuda.Stream()
        with torch.cuda.stream(copy_stream):
            for b, v in zip(bufs, second_views):
                b.copy_(torch.from_numpy(v), non_blocking=True)
            ready = torch.cuda.Event()
            ready.record(copy_stream)
        d.restart(ready)
        assert d.get_stats()["iterations_done"] == 0
        d.iterate(3)
        again = d.get_estimate_host()
        st = d.get_stats()
        d.close()
        fresh, fst = gpu_checkpoints(mvd, mvd_synth.Problem(0, tiny.dims, tiny.psf_dims, tiny.gt, tiny.psfs, second_views, 3, ()),
                                     "osem", "auto", (3,), **({"use_graph": True} if use_graph else {}))
        assert np.array_equal(again, fresh[3]) and not np.array_equal(again, first)
        assert st == fst
    o = O.Oracle(second_views, tiny.psfs, "osem")                  # ... with the first time-point's PSFs
    o.iterate(3)
    check(again, o.psi, 3, "restart")


def test_eps_and_floor_clamps(mvd, tiny):
    """R4: zero-valued data drive psi to the floor on both sides identically."""
    views = [v.copy() for v in tiny.views]
    for v in views:
        v[:6] = 0
    prob = mvd_synth.Problem(0, tiny.dims, tiny.psf_dims, tiny.gt, tiny.psfs, views, 1, ())
    g, _ = gpu_checkpoints(mvd, prob, "osem", "auto", (12,), eps=1e-3, psi_floor=1e-2)
    o, _ = oracle_checkpoints(prob, "osem", "auto", (12,), eps=1e-3, psi_floor=1e-2)
    assert (o[12] == 1e-2).any()
    assert np.isfinite(g[12]).all()
    l2, _ = errors(g[12], o[12], 1e-2)
    mx = float((np.abs(g[12] - o[12]) / np.maximum(np.abs(o[12]), 1e-2)).max())
    assert l2 <= TOL_L2_10 and mx <= TOL_MAX


# ------------------------------------------------------------------------------------------
# BASELINE configs 1-3 at full size, every iteration count BASELINE names
# ------------------------------------------------------------------------------------------
def test_config1_efficient_osem_10_iterations(mvd):
    p = mvd_synth.make_problem(1)
    g, st = gpu_checkpoints(mvd, p, "osem", "auto", (1, 10))
    o, orc = oracle_checkpoints(p, "osem", "auto", (1, 10))
    check(g[1], o[1], 1, "config 1")
    check(g[10], o[10], 10, "config 1")
    assert st["flux"] == pytest.approx(orc.flux, rel=1e-5)


@pytest.fixture(scope="module")
def config2():
    return mvd_synth.make_problem(2)


@pytest.mark.parametrize("variant,mode", [("independent", "auto"), ("efficient", "auto"),
                                          ("osem", "auto"), ("osem", "plain")])
def test_config2_all_variants_20_iterations(mvd, config2, variant, mode):
    g, _ = gpu_checkpoints(mvd, config2, variant, mode, (1, 10, 20))
    o, _ = oracle_checkpoints(config2, variant, mode, (1, 10, 20))
    for c in (1, 10, 20):
        check(g[c], o[c], c, "config 2 %s/%s" % (variant, mode))


def test_config3_efficient_osem_15_iterations(mvd):
    p = mvd_synth.make_problem(3)
    g, _ = gpu_checkpoints(mvd, p, "osem", "auto", (1, 15))
    o, _ = oracle_checkpoints(p, "osem", "auto", (1, 15))
    check(g[1], o[1], 1, "config 3")
    check(g[15], o[15], 15, "config 3")


# ------------------------------------------------------------------------------------------
# block-wise mode (S6, R13)
# ------------------------------------------------------------------------------------------
def test_blocked_matches_blocked_oracle(mvd):
    p = mvd_synth.make_problem(1, dims=(48, 40, 36), psf_dims=(7, 7, 11))
    block = (20, 24, 16)                                   # (x,y,z): ragged last blocks
    got, launches = mvd.deconvolve_blocked(to_dev(p.views), p.psfs, block, 3, variant="osem")
    ref = O.deconvolve_blocked(p.views, p.psfs, block[::-1], "osem", 3)
    check(got.cpu().numpy(), ref, 3, "blocked")
    assert launches > 0


def test_blocked_blocks_dealt_over_two_ranks(mvd):
    """PAPER.md L225 (blocks on two GPUs): block_world = 2 deals the blocks round-robin; the two ranks' calls write
    disjoint blocks of one result, together bit-identical to the single call; each leaves the other's blocks alone."""
    import torch
    p = mvd_synth.make_problem(1, dims=(48, 40, 36), psf_dims=(7, 7, 11))
    block = (20, 24, 16)
    views = to_dev(p.views)
    whole, _ = mvd.deconvolve_blocked(views, p.psfs, block, 2, variant="osem")
    out = torch.full_like(whole, -1.0)
    r0, l0 = mvd.deconvolve_blocked(views, p.psfs, block, 2, variant="osem", block_rank=0, block_world=2, out=out)
    assert r0 is out
    part = out.cpu().numpy()
    assert (part == -1.0).any() and (part != -1.0).any()                 # rank 0 wrote its blocks only
    nb = [-(-n // b) for n, b in zip((48, 40, 36), block)]               # blocks per axis (x, y, z)
    for iz in range(nb[2]):
        for iy in range(nb[1]):
            for ix in range(nb[0]):
                idx = (iz * nb[1] + iy) * nb[0] + ix
                blk = part[iz * block[2]:(iz + 1) * block[2], iy * block[1]:(iy + 1) * block[1], ix * block[0]:(ix + 1) * block[0]]
                assert ((blk == -1.0).all() if idx % 2 else (blk != -1.0).all()), (ix, iy, iz)
    _, l1 = mvd.deconvolve_blocked(views, p.psfs, block, 2, variant="osem", block_rank=1, block_world=2, out=out)
    assert torch.equal(out, whole) and l0 > 0 and l1 > 0
    with pytest.raises(mvd.MvdError):
        mvd.deconvolve_blocked(views, p.psfs, block, 2, variant="osem", block_rank=2, block_world=2)


def test_blocked_single_block_equals_whole(mvd, tiny):
    got, _ = mvd.deconvolve_blocked(to_dev(tiny.views), tiny.psfs, (64, 64, 64), 2, variant="efficient")
    whole, _ = gpu_checkpoints(mvd, tiny, "efficient", "auto", (2,))
    assert np.array_equal(got.cpu().numpy(), whole[2])


# ------------------------------------------------------------------------------------------
# BASELINE config 4 at full size, in the launch configuration bench.py times (CUDA graph replay)
# ------------------------------------------------------------------------------------------
@pytest.fixture(scope="module")
def config4():
    return mvd_synth.make_problem(4)


def test_config4_bench_configuration(mvd, config4):
    """512x512x256, 7 views, efficient-OSEM, one CUDA graph per iteration: every voxel against the
    oracle after 1, 2 and 10 iterations (north_star: rel-L2 <= 1e-5 after 1 iteration, <= 1e-4 after 10,
    max per-voxel rel <= 1e-3).  70 view-updates; the oracle needs ~13 s per iteration on 16 cores."""
    p = config4
    g, st = gpu_checkpoints(mvd, p, "osem", "auto", (1, 2, 10), use_graph=True)
    o, orc = oracle_checkpoints(p, "osem", "auto", (1, 2, 10))
    check(g[1], o[1], 1, "config 4")
    l2, mx = errors(g[2], o[2])
    assert l2 <= 2e-5 and mx <= TOL_MAX, (l2, mx)      # 2 iterations: well inside the 10-iteration bound
    check(g[10], o[10], 10, "config 4")
    assert st["iterations_done"] == 10
    assert st["flux"] == pytest.approx(orc.flux, rel=1e-5)
    assert st["l1_change"] == pytest.approx(orc.l1_change, rel=2e-3)


def _combined_variants_plain_and_graph(mvd, p, what):
    """independent (eq. 70) and efficient (eq. 104) with the root of eq. 44: the shared forward pass
    (W0), the product accumulation and the powf root of the X_ACCUM kernels, as plain launches and
    under CUDA-graph replay, against the oracle after 1 and 3 iterations."""
    for variant in ("independent", "efficient"):
        o, orc = oracle_checkpoints(p, variant, "auto", (1, 3))
        plain, st = gpu_checkpoints(mvd, p, variant, "auto", (1, 3))
        graph, stg = gpu_checkpoints(mvd, p, variant, "auto", (1, 3), use_graph=True)
        for c in (1, 3):
            check(plain[c], o[c], c, "%s %s" % (what, variant))
            assert np.array_equal(plain[c], graph[c]), (what, variant, c)
        assert st["flux"] == pytest.approx(orc.flux, rel=1e-5)
        assert stg == st                                 # graph replay reports the same statistics


def test_config3_combined_variants(mvd):
    _combined_variants_plain_and_graph(mvd, mvd_synth.make_problem(3), "config 3")


def test_config4_combined_variants(mvd, config4):
    _combined_variants_plain_and_graph(mvd, config4, "config 4")


def test_config1_combined_variants(mvd):
    _combined_variants_plain_and_graph(mvd, mvd_synth.make_problem(1), "config 1")


# ------------------------------------------------------------------------------------------
# BASELINE config 5 size (1024x1024x512, PSF 25x25x51): the oracle cannot run the whole volume in
# seconds, so (i) one 'same' convolution is checked at sampled voxels against the direct-sum
# definition (O1) and (ii) the flux identity P3, which holds at any size, is checked after one update
# ------------------------------------------------------------------------------------------
def test_config5_size_sampled_voxels_and_flux(mvd):
    import torch
    dims, box = (1024, 1024, 512), (25, 25, 51)
    nx, ny, nz = dims
    rng = np.random.default_rng([13080730, 5, 77])
    psf = mvd_synth.generate.random_psf(rng, box)               # asymmetric: a missing mirror fails
    view = (rng.random((nz, ny, nx), dtype=np.float32) * 100.0 + 5.0)
    dview = torch.from_numpy(view).cuda()
    d = mvd.Deconvolver([dview], [psf], variant="osem", kernel_mode="plain")
    mx, my, mz = d.fft_dims
    assert mx >= 512 + 24 and my >= 1024 + 12 and mz >= 512 + 25     # M >= N + r (hx + 2 rx along x)
    pn = O.normalise(psf)
    cz, cy, cx = [(k - 1) // 2 for k in pn.shape]
    # sampled voxels: corners, faces, interior
    pts = [(0, 0, 0), (nz - 1, ny - 1, nx - 1), (0, ny - 1, 5), (nz - 1, 0, nx // 2), (nz // 2, ny // 2, nx // 2 - 1),
           (nz // 2, ny // 2, nx // 2), (3, 511, 512), (300, 1023, 0)]
    pts += [tuple(int(rng.integers(n)) for n in (nz, ny, nx)) for _ in range(40)]
    for which, k in ((0, pn), (1, O.flip(pn))):
        got = d.convolve(0, which, dview)
        for (z, y, x) in pts:
            acc = 0.0                                            # same(a,k)[xi] = sum_u k[u] a[xi - (u - c)]
            for uz in range(k.shape[0]):
                zz = z - (uz - cz)
                if zz < 0 or zz >= nz:
                    continue
                y0, y1 = max(0, y + cy - (ny - 1)), min(k.shape[1] - 1, y + cy)
                x0, x1 = max(0, x + cx - (nx - 1)), min(k.shape[2] - 1, x + cx)
                kk = k[uz, y0:y1 + 1, x0:x1 + 1].astype(np.float64)
                aa = view[zz, y + cy - y1:y + cy - y0 + 1, x + cx - x1:x + cx - x0 + 1].astype(np.float64)[::-1, ::-1]
                acc += float((kk * aa).sum())
            gv = float(got[z, y, x])
            assert abs(gv - acc) <= 2e-5 * abs(acc), (which, (z, y, x), gv, acc)
        del got
    d.iterate(1)
    st = d.get_stats()
    d.close()
    assert st["flux"] == pytest.approx(float(view.astype(np.float64).sum()), rel=2e-6)


def test_repeated_runs_are_bit_identical(mvd, config2):
    """The staged pipelines (mbarrier phases, refilled tiles) must not race: the same problem run
    several times in fresh contexts, with plain launches and under graph replay, gives the same bits."""
    ref = None
    for rep in range(4):
        g, _ = gpu_checkpoints(mvd, config2, "osem", "auto", (3,), use_graph=bool(rep & 1))
        if ref is None:
            ref = g[3]
        assert np.array_equal(g[3], ref), "run %d differs" % rep
    g, _ = gpu_checkpoints(mvd, config2, "efficient", "auto", (2,))
    h, _ = gpu_checkpoints(mvd, config2, "efficient", "auto", (2,))
    assert np.array_equal(g[2], h[2])


# ------------------------------------------------------------------------------------------
# section 12 (L891-903): per-view weights of partially overlapping views, sequential updates
# ------------------------------------------------------------------------------------------
def _partial_overlap_weights(shape, n_views):
    """View v covers a box shifted along x (and y for odd v): cosine-blended, sum over views <= 1."""
    nz, ny, nx = shape
    ws = []
    for v in range(n_views):
        lo = (0, (ny // 6) * (v & 1), (nx // 8) * v)
        hi = (nz, ny - (ny // 7) * ((v + 1) & 1), nx - (nx // 8) * (n_views - 1 - v))
        ws.append(O.blending_weights(shape, lo, hi, border=5))
    return O.normalise_weights(ws, 1.0)


@pytest.mark.parametrize("dims,box", [((24, 20, 18), (5, 7, 9)), ((33, 17, 9), (3, 5, 7))])   # aligned rows / odd Nx
def test_weighted_osem_matches_oracle(mvd, dims, box):
    import torch
    p = mvd_synth.make_tiny_asymmetric(dims=dims, psf_dims=box, n_views=3)
    ws = _partial_overlap_weights(p.views[0].shape, 3)
    wdev = [torch.from_numpy(w.astype(np.float32)).cuda() for w in ws]
    w32 = [w.astype(np.float32).astype(np.float64) for w in ws]       # both sides see the same fp32 weights
    for mode in ("auto", "plain"):
        d = mvd.Deconvolver(to_dev(p.views), p.psfs, variant="osem", kernel_mode=mode, weights=wdev)
        o = O.Oracle(p.views, p.psfs, "osem", kernel_mode=mode, weights=w32)
        d.iterate(1)
        o.iterate(1)
        check(d.get_estimate_host(), o.psi, 1, "weighted %s" % mode)
        d.iterate(4)
        o.iterate(4)
        check(d.get_estimate_host(), o.psi, 5, "weighted %s" % mode)
        d.close()


def test_weights_one_equal_no_weights_and_combined_variants_refuse(mvd, tiny):
    import torch
    ones = [torch.ones(tiny.views[0].shape, device="cuda") for _ in tiny.views]
    a, _ = gpu_checkpoints(mvd, tiny, "osem", "auto", (3,))
    b, _ = gpu_checkpoints(mvd, tiny, "osem", "auto", (3,), weights=ones)
    l2, mx = errors(b[3], a[3])
    assert l2 < 1e-6 and mx < 1e-5                                    # 1 + 1*(f-1) rounds once more than f
    with pytest.raises(mvd.MvdError):
        mvd.Deconvolver(to_dev(tiny.views), tiny.psfs, variant="efficient", weights=ones)


def test_weighted_config2_size(mvd, config2):
    """Weights at a size that spans many tiles: 128^3, 3 views, 5 iterations."""
    import torch
    ws = _partial_overlap_weights(config2.views[0].shape, 3)
    wdev = [torch.from_numpy(w.astype(np.float32)).cuda() for w in ws]
    w32 = [w.astype(np.float32).astype(np.float64) for w in ws]
    g, _ = gpu_checkpoints(mvd, config2, "osem", "auto", (1, 5), weights=wdev, use_graph=True)
    o, _ = oracle_checkpoints(config2, "osem", "auto", (1, 5), weights=w32)
    check(g[1], o[1], 1, "weighted config 2")
    check(g[5], o[5], 5, "weighted config 2")


# ------------------------------------------------------------------------------------------
# Tikhonov regularisation (L64, L869; R14): fused into the update kernels, zero extra bytes
# ------------------------------------------------------------------------------------------
@pytest.mark.parametrize("variant", ["osem", "efficient", "independent"])
def test_tikhonov_matches_oracle(mvd, tiny, variant):
    for lam in (0.006, 0.06):                                       # values of the paper's sweep (L145)
        g, st = gpu_checkpoints(mvd, tiny, variant, "auto", (1, 5), tikhonov_lambda=lam)
        o, orc = oracle_checkpoints(tiny, variant, "auto", (1, 5), tikhonov_lambda=lam)
        check(g[1], o[1], 1, "tikhonov %s %g" % (variant, lam))
        check(g[5], o[5], 5, "tikhonov %s %g" % (variant, lam))
        assert st["flux"] == pytest.approx(orc.flux, rel=1e-5)
    plain, _ = gpu_checkpoints(mvd, tiny, variant, "auto", (2,))
    zero, _ = gpu_checkpoints(mvd, tiny, variant, "auto", (2,), tikhonov_lambda=0.0)
    assert np.array_equal(plain[2], zero[2])                        # lambda = 0: the unregularised path, bit for bit
    reg, _ = gpu_checkpoints(mvd, tiny, variant, "auto", (2,), tikhonov_lambda=0.06)
    assert reg[2].sum(dtype=np.float64) < plain[2].sum(dtype=np.float64)
    with pytest.raises(mvd.MvdError):
        gpu_checkpoints(mvd, tiny, variant, "auto", (1,), tikhonov_lambda=-0.5)


def test_tikhonov_config2_size_with_weights_blocks_and_view_parallel(mvd, config2, tiny):
    """lambda = 0.006 (the paper's real-data value, Suppl. Table 1) at 128^3 under graph replay; with section-12
    weights; in block-wise mode; and through the view-parallel calls (apply_product_kernel)."""
    import torch
    lam = 0.006
    g, _ = gpu_checkpoints(mvd, config2, "osem", "auto", (1, 10), tikhonov_lambda=lam, use_graph=True)
    o, _ = oracle_checkpoints(config2, "osem", "auto", (1, 10), tikhonov_lambda=lam)
    check(g[1], o[1], 1, "tikhonov config 2")
    check(g[10], o[10], 10, "tikhonov config 2")
    ws = _partial_overlap_weights(tiny.views[0].shape, 3)
    wdev = [torch.from_numpy(w.astype(np.float32)).cuda() for w in ws]
    w32 = [w.astype(np.float32).astype(np.float64) for w in ws]
    g, _ = gpu_checkpoints(mvd, tiny, "osem", "auto", (3,), tikhonov_lambda=lam, weights=wdev)
    o, _ = oracle_checkpoints(tiny, "osem", "auto", (3,), tikhonov_lambda=lam, weights=w32)
    check(g[3], o[3], 3, "tikhonov + weights")
    p = mvd_synth.make_problem(1, dims=(48, 40, 36), psf_dims=(7, 7, 11))
    got, _ = mvd.deconvolve_blocked(to_dev(p.views), p.psfs, (20, 24, 16), 3, variant="osem", tikhonov_lambda=lam)
    ref = O.deconvolve_blocked(p.views, p.psfs, (16, 24, 20), "osem", 3, tikhonov_lambda=lam)
    check(got.cpu().numpy(), ref, 3, "tikhonov blocked")
    d = mvd.ViewParallelDeconvolver(to_dev(tiny.views), tiny.psfs, variant="efficient", tikhonov_lambda=lam)
    d.iterate(2)
    orc = O.Oracle(tiny.views, tiny.psfs, "efficient", tikhonov_lambda=lam)
    orc.iterate(2)
    check(d.get_estimate_host(), orc.psi, 2, "tikhonov view-parallel")
    d.close()


# ------------------------------------------------------------------------------------------
# view-parallel combined variants (L815): two "ranks" emulated on one GPU as two
# contexts that own different views; their partial products are multiplied as the all-reduce would
# ------------------------------------------------------------------------------------------
@pytest.mark.parametrize("variant", ["independent", "efficient"])
def test_view_parallel_two_emulated_ranks(mvd, tiny, variant):
    import torch
    V = len(tiny.views)
    views = to_dev(tiny.views)
    mean = sum(mvd.reduce_sum(v) for v in views) / sum(v.numel() for v in views)
    assert mean == pytest.approx(float(np.mean([v.astype(np.float64).mean() for v in tiny.views])), rel=1e-12)
    ranks = []
    for r in range(2):
        loc = mvd.split_views(V, 2, r)
        ranks.append(mvd.Deconvolver([views[v] for v in loc], tiny.psfs, variant=variant, local_views=loc,
                                     psi0_value=mean))
    o = O.Oracle(tiny.views, tiny.psfs, variant)
    for it in range(3):
        for d in ranks:
            d.partial_product()
        torch.cuda.synchronize()
        prod = ranks[0].product_tensor() * ranks[1].product_tensor()      # = all-reduce(PRODUCT)
        for d in ranks:
            d.product_tensor().copy_(prod)
            d.apply_product(V)
        o.iterate(1)
        a, b = ranks[0].get_estimate_host(), ranks[1].get_estimate_host()
        assert np.array_equal(a, b)                                          # psi stays replicated
        check(a, o.psi, it + 1, "view-parallel %s" % variant)
    st = ranks[0].get_stats()
    assert st["flux"] == pytest.approx(o.flux, rel=1e-5) and st["iterations_done"] == 3
    with pytest.raises(mvd.MvdError):
        ranks[0].iterate(1)                                                  # split contexts do not iterate alone
    for d in ranks:
        d.close()
    with pytest.raises(mvd.MvdError):
        mvd.Deconvolver([views[0]], tiny.psfs, variant="osem", local_views=[0], psi0_value=mean)


def test_view_parallel_driver_world_1_equals_oracle(mvd, tiny):
    d = mvd.ViewParallelDeconvolver(to_dev(tiny.views), tiny.psfs, variant="efficient")
    d.iterate(2)
    o = O.Oracle(tiny.views, tiny.psfs, "efficient")
    o.iterate(2)
    check(d.get_estimate_host(), o.psi, 2, "view-parallel driver")
    d.close()


# ------------------------------------------------------------------------------------------
# every compiled pencil length (csrc/lengths.def), on every axis: one 'same' convolution with the
# FFT length of that axis forced, against the oracle.  Covers every register transform (radices
# 2,3,4,5,7 in all their mixes), the TMA-staged y/z passes and the x pass for every (A, B).
# ------------------------------------------------------------------------------------------
def _compiled_lengths():
    import os
    import re
    path = os.path.join(os.path.dirname(os.path.dirname(os.path.abspath(__file__))), "paper_1308_0730_b200", "csrc",
                        "lengths.def")
    out = []
    for line in open(path):
        m = re.match(r"\s*MVD_LEN\((\d+),\s*(\d+)\)", line)
        if m:
            out.append(int(m.group(1)) * int(m.group(2)))
    return sorted(out)


@pytest.mark.parametrize("axis", [0, 1, 2])
def test_every_compiled_length_on_every_axis(mvd, axis):
    import torch
    rng = np.random.default_rng([7, axis])
    box = (5, 5, 5)                                   # (Kx,Ky,Kz), r = 2
    psf = mvd_synth.generate.random_psf(rng, box)
    pn = O.normalise(psf)
    tested = 0
    for M in _compiled_lengths():
        if M < 8 or (axis == 0 and M % 2):            # x lengths are even (16-byte rows)
            continue
        dims = [6, 7, 5]
        dims[axis] = 2 * (M - 4) if axis == 0 else M - 2          # the largest volume this length serves
        if dims[axis] < 3:
            continue
        fft = [0, 0, 0]
        fft[axis] = M
        view = (rng.random((dims[2], dims[1], dims[0]), dtype=np.float32) * 10 + 1)
        d = mvd.Deconvolver([torch.from_numpy(view).cuda()], [psf], variant="osem", kernel_mode="plain",
                            fft_dims=tuple(fft))
        assert d.fft_dims[axis] == M
        for which, k in ((0, pn), (1, O.flip(pn))):
            got = d.convolve(0, which, torch.from_numpy(view).cuda()).cpu().numpy()
            l2, mx = errors(got, O.same_fft(view, k))
            assert l2 < 3e-6 and mx < 1e-4, (axis, M, which, l2, mx)
        # and the fused x kernels (quotient, update) of this length: one OSEM iteration against the oracle
        d.iterate(1)
        o = O.Oracle([view], [psf], "osem", kernel_mode="plain")
        o.iterate(1)
        check(d.get_estimate_host(), o.psi, 1, "length %d axis %d" % (M, axis))
        d.close()
        tested += 1
    assert tested >= 50


def test_register_staged_fallback_kernels_match_too(mvd, tiny, monkeypatch):
    """The register-staged passes (pass_kernels.cuh) stay as the fallback when a pencil does not fit
    the TMA-staged tiles; MVD_TUNE="xtma=0,ytma=0,ztma=0" selects them.  Same parity bar."""
    monkeypatch.setenv("MVD_TUNE", "xtma=0,ytma=0,ztma=0")
    for variant in ("osem", "efficient"):
        g, _ = gpu_checkpoints(mvd, tiny, variant, "auto", (1, 3))
        o, _ = oracle_checkpoints(tiny, variant, "auto", (1, 3))
        check(g[1], o[1], 1, "fallback %s" % variant)
        check(g[3], o[3], 3, "fallback %s" % variant)


def test_tuning_knobs_keep_parity(mvd, tiny, monkeypatch):
    """The keys of MVD_TUNE (csrc/mvd.cu) select other kernels or tile shapes, never other results: plain loads of the
    real rows, the 8 x 2 z tile, column pairs in the y pass, one tile stage, no alternating tile order, and several at
    once.  Same parity bar, and bit-identical to the default: every variant does the same arithmetic per element."""
    ref, _ = gpu_checkpoints(mvd, tiny, "osem", "auto", (3,))
    o, _ = oracle_checkpoints(tiny, "osem", "auto", (3,))
    for knobs in ("xbulk=0", "ztx=8", "ypair=1", "ynst=1,znst=1", "flip=0", "ypair=1,ztx=8,xbulk=0,rxt=2", "nosuchkey=3"):
        monkeypatch.setenv("MVD_TUNE", knobs)
        g, _ = gpu_checkpoints(mvd, tiny, "osem", "auto", (3,), use_graph=True)
        check(g[3], o[3], 3, knobs)
        assert np.array_equal(g[3], ref[3]), knobs
    monkeypatch.delenv("MVD_TUNE")


def test_views_not_16_byte_aligned(mvd):
    """Borrowed views (and weights) only need float alignment: rows that cannot be staged by 16-byte
    bulk copies take the plain-load path inside the same kernel."""
    import torch
    p = mvd_synth.make_tiny_asymmetric(dims=(24, 20, 18), psf_dims=(5, 7, 9), n_views=2)
    n = p.views[0].size
    views, wts = [], []
    ws = _partial_overlap_weights(p.views[0].shape, 2)
    for v, w in zip(p.views, ws):
        big = torch.zeros(n + 3, dtype=torch.float32, device="cuda")
        big[1:1 + n] = torch.from_numpy(v.ravel()).cuda()
        views.append(big[1:1 + n].view(p.views[0].shape))
        bw = torch.zeros(n + 3, dtype=torch.float32, device="cuda")
        bw[3:3 + n] = torch.from_numpy(w.astype(np.float32).ravel()).cuda()
        wts.append(bw[3:3 + n].view(p.views[0].shape))
        assert views[-1].data_ptr() % 16 == 4 and wts[-1].data_ptr() % 16 == 12
    w32 = [w.astype(np.float32).astype(np.float64) for w in ws]
    for kw, okw in (({}, {}), ({"weights": wts}, {"weights": w32})):
        d = mvd.Deconvolver(views, p.psfs, variant="osem", **kw)
        d.iterate(3)
        o = O.Oracle(p.views, p.psfs, "osem", **okw)
        o.iterate(3)
        check(d.get_estimate_host(), o.psi, 3, "misaligned views %s" % list(kw))
        d.close()


def test_quality_metrics_against_a_reference(mvd):
    """mvd_compare: average difference (L127) and cross-correlation (L48) of psi against the ground
    truth, against the same measures computed by the oracle module on the same estimate."""
    import torch
    p = mvd_synth.make_problem(1, dims=(40, 36, 32), psf_dims=(7, 7, 15))
    d = mvd.Deconvolver(to_dev(p.views), p.psfs, variant="osem")
    d.iterate(3)
    st0 = d.get_stats()
    psi = d.get_estimate_host().astype(np.float64)
    ad, cc = d.compare(torch.from_numpy(p.gt.astype(np.float32)).cuda())
    gt32 = p.gt.astype(np.float32).astype(np.float64)
    assert ad == pytest.approx(O.average_difference(psi, gt32), rel=1e-9)
    assert cc == pytest.approx(O.cross_correlation(psi, gt32), rel=1e-9)
    assert 0.0 < cc <= 1.0
    assert d.get_stats() == st0                       # the update statistics survive a comparison
    d.close()


def test_blocked_config2_size_shares_back_projectors(mvd, config2):
    """128^3, PSF 17x17x35, 64^3 blocks + halo: 8 blocks of several extended shapes (one context per
    shape, the compound kernels computed once and shared) against the blocked oracle."""
    block = (64, 64, 64)
    got, launches = mvd.deconvolve_blocked(to_dev(config2.views), config2.psfs, block, 3, variant="osem")
    ref = O.deconvolve_blocked(config2.views, config2.psfs, block[::-1], "osem", 3)
    check(got.cpu().numpy(), ref, 3, "blocked config 2")
    assert launches > 8 * 3 * 3 * 8


# ------------------------------------------------------------------------------------------
# seeded random small problems: odd / even / prime extents (rows that are not 16-byte aligned, ragged tiles, PSF
# boxes larger than the volume), every variant and kernel mode, with and without weights, Tikhonov, graph replay
# ------------------------------------------------------------------------------------------
@pytest.mark.parametrize("case", range(16))
def test_random_small_problems(mvd, case):
    import torch
    rng = np.random.default_rng([13080730, 900, case])
    dims = tuple(int(rng.integers(5, 72)) for _ in range(3))                     # (Nx, Ny, Nz)
    box = tuple(int(2 * rng.integers(1, 6) + 1) for _ in range(3))               # odd 3..11
    V = int(rng.integers(1, 5))
    variant = ("osem", "efficient", "independent")[int(rng.integers(3))]
    mode = ("auto", "plain", "compound", "opt1", "opt2")[int(rng.integers(5))]
    lam = float(rng.choice([0.0, 0.0, 0.006, 0.06]))
    use_w = variant == "osem" and bool(rng.integers(2))
    use_graph = bool(rng.integers(2))
    iters = int(rng.integers(1, 4))
    p = mvd_synth.make_tiny_asymmetric(dims=dims, psf_dims=box, n_views=V, seed_stream=50 + case)
    kw, okw = {}, {}
    if lam:
        kw["tikhonov_lambda"] = okw["tikhonov_lambda"] = lam
    if use_w:
        ws = [rng.random(p.views[0].shape).astype(np.float32) for _ in range(V)]
        kw["weights"] = [torch.from_numpy(w).cuda() for w in ws]
        okw["weights"] = [w.astype(np.float64) for w in ws]
    if use_graph:
        kw["use_graph"] = True
    g, st = gpu_checkpoints(mvd, p, variant, mode, (1, iters) if iters > 1 else (1,), **kw)
    o, orc = oracle_checkpoints(p, variant, mode, (1, iters) if iters > 1 else (1,), **okw)
    what = "case %d: dims %s box %s V=%d %s/%s lam=%g w=%s graph=%s" % (case, dims, box, V, variant, mode, lam, use_w, use_graph)
    check(g[1], o[1], 1, what)
    check(g[iters], o[iters], iters, what)
    assert st["flux"] == pytest.approx(orc.flux, rel=1e-5), what
