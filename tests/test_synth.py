"""The seeded input generators: determinism, shapes, value ranges (no GPU)."""
import numpy as np

import mvd_synth


def test_config1_shapes_and_determinism():
    a = mvd_synth.make_problem(1, dims=(32, 24, 20), psf_dims=(7, 7, 15))
    b = mvd_synth.make_problem(1, dims=(32, 24, 20), psf_dims=(7, 7, 15))
    assert a.n_views == 4 and a.dims == (32, 24, 20)
    for va, vb, p in zip(a.views, b.views, a.psfs):
        assert va.shape == (20, 24, 32) and va.dtype == np.float32
        assert np.array_equal(va, vb)
        assert (va >= 0).all()
        assert p.shape == (15, 7, 7) and abs(p.sum() - 1) < 1e-6 and (p >= 0).all()
    # 0 and 180 degrees give the same (point-symmetric) Gaussian: the blind spot DESIGN.md names
    assert np.allclose(a.psfs[0], a.psfs[2], atol=1e-7)
    assert np.allclose(a.psfs[0], a.psfs[0][::-1, ::-1, ::-1], atol=1e-7)
    # views carry roughly the same flux (R10)
    sums = [float(v.sum()) for v in a.views]
    assert max(sums) / min(sums) < 1.10


def test_rotated_psf_is_elongated_along_x_at_90_degrees():
    p0 = mvd_synth.gaussian_psf((15, 15, 31), 1.2, 4.0, 0.0)
    p90 = mvd_synth.gaussian_psf((15, 15, 31), 1.2, 4.0, 90.0)
    prof = lambda p, ax: p.sum(axis=tuple(i for i in range(3) if i != ax))
    width = lambda q: float((q * (np.arange(q.size) - q.size // 2) ** 2).sum() / q.sum()) ** 0.5
    assert width(prof(p0, 0)) > 2.5 * width(prof(p0, 2))      # z-long at 0 degrees (axis 0 = z)
    assert width(prof(p90, 2)) > 2.5 * width(prof(p90, 0))    # x-long at 90 degrees


def test_tiny_asymmetric_is_asymmetric():
    t = mvd_synth.make_tiny_asymmetric()
    assert t.dims == (24, 20, 18) and t.n_views == 3
    for p in t.psfs:
        assert p.shape == (9, 7, 5)
        assert np.abs(p - p[::-1, ::-1, ::-1]).max() > 1e-3


def test_peak_scaling_config3_shrunk():
    p = mvd_synth.make_problem(3, dims=(48, 48, 24), psf_dims=(9, 9, 21), n_views=3, noise=False)
    assert max(float(v.max()) for v in p.views) == np.float32(300.0)
