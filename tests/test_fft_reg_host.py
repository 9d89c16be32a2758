"""T1: the register-resident mixed-radix transforms of csrc/fft_reg.cuh against a plain DFT.

fft_reg.cuh compiles as plain C++ with MVD_HOST_TEST; tests/host/fft_reg_host.cpp instantiates FftReg<N, +-1> for every
factor length the pencil lengths of csrc/lengths.def use (A, B <= 36) and this test compares them with numpy.fft on
random complex input: forward = sum x[n] exp(-2 pi i n k / N), inverse = the conjugate kernel, both unnormalised, natural
order in and out.  A wrong twiddle, radix order or sign in any butterfly fails here without a GPU."""
import os
import re
import subprocess

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _factor_lengths():
    out = set()
    for line in open(os.path.join(ROOT, "paper_1308_0730_b200", "csrc", "lengths.def")):
        m = re.match(r"\s*MVD_LEN\((\d+),\s*(\d+)\)", line)
        if m:
            out.update((int(m.group(1)), int(m.group(2))))
    return sorted(out)


@pytest.fixture(scope="module")
def harness(tmp_path_factory):
    exe = str(tmp_path_factory.mktemp("fftreg") / "fft_reg_host")
    src = os.path.join(ROOT, "tests", "host", "fft_reg_host.cpp")
    r = subprocess.run(["g++", "-std=c++17", "-O1", "-ffp-contract=off", src, "-o", exe], capture_output=True, text=True)
    assert r.returncode == 0, r.stderr[-3000:]
    return exe


def test_every_factor_length_matches_numpy_fft(harness):
    rng = np.random.default_rng(1308)
    lengths = _factor_lengths()
    assert lengths[0] == 2 and lengths[-1] == 36 and len(lengths) >= 20
    lines, cases = [], []
    for n in lengths:
        for d in (-1, 1):
            x = (rng.standard_normal(n) + 1j * rng.standard_normal(n)).astype(np.complex64)
            cases.append((n, d, x))
            lines.append("%d %d " % (n, d) + " ".join("%.9g %.9g" % (z.real, z.imag) for z in x))
    r = subprocess.run([harness], input="\n".join(lines) + "\n", capture_output=True, text=True)
    assert r.returncode == 0, (r.returncode, r.stderr[-1000:])
    rows = r.stdout.strip().splitlines()
    assert len(rows) == len(cases)
    for (n, d, x), row in zip(cases, rows):
        got = np.array(row.split(), dtype=np.float64)
        got = got[0::2] + 1j * got[1::2]
        ref = np.fft.fft(x.astype(np.complex128)) if d < 0 else np.fft.ifft(x.astype(np.complex128)) * n
        err = np.abs(got - ref).max() / np.abs(ref).max()
        assert err < 3e-6, (n, d, err)


def test_impulse_and_constant(harness):
    """delta -> all ones; constant -> N at k = 0 and 0 elsewhere (exact in fp32 up to rounding of the sums)."""
    lines = []
    for n in (7, 20, 25, 36):
        delta = ["1 0"] + ["0 0"] * (n - 1)
        const = ["1 0"] * n
        lines.append("%d -1 %s" % (n, " ".join(delta)))
        lines.append("%d -1 %s" % (n, " ".join(const)))
    r = subprocess.run([harness], input="\n".join(lines) + "\n", capture_output=True, text=True)
    rows = [np.array(t.split(), dtype=np.float64) for t in r.stdout.strip().splitlines()]
    for i, n in enumerate((7, 20, 25, 36)):
        d, c = rows[2 * i], rows[2 * i + 1]
        assert np.allclose(d[0::2], 1.0, atol=1e-6) and np.allclose(d[1::2], 0.0, atol=1e-6)
        assert c[0] == pytest.approx(n, rel=1e-6) and np.abs(c[2:]).max() < 1e-5 * n
