"""Seeded synthetic SPIM-shaped inputs (ground truth, PSFs, views).

This module serves BOTH the oracle-side tests and the CUDA-side tests/bench, so it
holds none of the deconvolution method's arithmetic: it only draws phantoms, samples
Gaussian PSFs, blurs the phantom with a library FFT (scipy.fft) and draws Poisson
noise.  It imports neither ``oracle`` nor ``paper_1308_0730_b200``.

Recipe: DESIGN.md "Synthetic inputs"; shapes follow BASELINE.json ``configs`` and the
paper's workloads (6-12 views, anisotropic Gaussian-like PSFs rotated about one axis,
Poisson noise, bead/nuclei content in an embryo-like shell: PAPER.md L913, L857-859,
Suppl. Table 1).
"""
from .generate import (  # noqa: F401
    CONFIGS,
    Problem,
    gaussian_psf,
    make_problem,
    make_tiny_asymmetric,
    random_psf,
)
