"""mvd_reduce_sum_static against mvd_reduce_sum: the no-allocation entry point gives the same sum.

Why the entry point exists: every device byte this library touches is the caller's, and mvd_reduce_sum follows that
rule by asking for a scratch buffer.  A caller whose workspace already fills the GPU, a time-lapse loop that must not
pay cudaMalloc's device-wide synchronisation between time-points, or a plug-in that may not allocate on its host
application's device has no buffer to give.  For them the partial sums live in one fixed array inside the library's
device image, which every call on the device shares and which keeps the previous call's contents.  That sharing is what
this file checks: two calls in a row, the second on a shorter and different input, must each agree with the
scratch-buffer path, so nothing left behind by the first call may leak into the second.

The file sorts last on purpose (pytest -x stops at the first failure; a failure here should not hide the parity tests).
It passes alone in a fresh process (first call = the per-device address look-up) and after the rest of the suite.
"""
import pytest

import paper_1308_0730_b200 as mvd

pytestmark = pytest.mark.gpu

# both paths add the same fp32 values in fp64 and differ only in the order of the additions: a few ulp of the sum.
# The parity tests compare flux at rel 1e-6; this is the sharper bound the arithmetic gives.
REL = 1e-12


def _views(n, seed, offset):
    import torch
    g = torch.Generator(device="cuda").manual_seed(seed)
    # SPIM-like intensities: background 5 plus a positive signal (mvd_synth's value range), so the sum is far from 0
    full = 5.0 + 100.0 * torch.rand(n + offset, generator=g, device="cuda", dtype=torch.float32)
    return full[offset:]          # a view: offset = 1 gives a pointer that is only 4-byte aligned


def test_two_calls_in_a_row_match_the_scratch_buffer_path():
    import torch
    torch.cuda.set_device(0)
    # first: 5 chunks and a ragged tail; second: fewer chunks, other values, and a pointer that is not 16-byte
    # aligned (the scalar branch).  Stale partials of the first call sit beyond the second call's range.
    a = _views(5 * 65536 + 1234, seed=11, offset=0)
    b = _views(2 * 65536 - 77, seed=12, offset=1)
    assert b.data_ptr() % 16 != 0
    want_a, want_b = mvd.reduce_sum(a), mvd.reduce_sum(b)          # existing path, scratch from torch
    got_a = mvd.reduce_sum_static(a)
    got_b = mvd.reduce_sum_static(b)
    assert abs(got_a - want_a) <= REL * abs(want_a)
    assert abs(got_b - want_b) <= REL * abs(want_b)
    # and against the definition, so that both paths being wrong together would show
    assert abs(got_a - a.double().sum().item()) <= REL * abs(want_a)
    assert abs(got_b - b.double().sum().item()) <= REL * abs(want_b)
    # a third call repeats the first bit for bit: fixed chunks, partials added in index order
    assert mvd.reduce_sum_static(a) == got_a


def test_small_and_empty_inputs():
    import torch
    torch.cuda.set_device(0)
    one = torch.full((1,), 3.5, device="cuda")
    assert mvd.reduce_sum_static(one) == 3.5
    few = _views(1000, seed=13, offset=0)
    assert abs(mvd.reduce_sum_static(few) - mvd.reduce_sum(few)) <= REL * mvd.reduce_sum(few)
    lib = mvd.load_library()
    import ctypes as C
    out = C.c_double(-1.0)
    assert lib.mvd_reduce_sum_static(one.data_ptr(), 0, None, C.byref(out)) == 0 and out.value == 0.0


def test_sizes_beyond_the_array_are_refused_without_touching_the_gpu():
    import ctypes as C
    import torch
    torch.cuda.set_device(0)
    lib = mvd.load_library()
    limit = int(lib.mvd_reduce_sum_static_max())
    assert limit == 2 ** 30
    x = torch.ones(16, device="cuda")
    out = C.c_double(-1.0)
    st = lib.mvd_reduce_sum_static(x.data_ptr(), limit + 1, None, C.byref(out))   # only n is wrong: nothing is read
    assert st == 2 and out.value == -1.0                                           # MVD_ERR_UNSUPPORTED
    msg = lib.mvd_reduce_sum_static_error().decode()
    assert str(limit) in msg and str(limit + 1) in msg
    assert lib.mvd_reduce_sum_static(x.data_ptr(), -1, None, C.byref(out)) == 1    # MVD_ERR_INVALID_ARG
    assert lib.mvd_reduce_sum_static(None, 4, None, C.byref(out)) == 1
    with pytest.raises(mvd.MvdError):
        mvd.reduce_sum_static(torch.ones(8, 8, device="cuda")[:, ::2])             # would need a copy: refused
    # the array is still usable after the refusals
    assert mvd.reduce_sum_static(x) == 16.0
    assert lib.mvd_reduce_sum_static_error().decode() == ""


def test_the_call_leaves_device_memory_as_it_found_it():
    import torch
    torch.cuda.set_device(0)
    x = _views(3 * 65536 + 5, seed=14, offset=0)
    mvd.reduce_sum_static(x)                       # set-up call (module load, address look-up) outside the comparison
    torch.cuda.synchronize()
    torch_before = torch.cuda.memory_allocated()
    free_before, _ = torch.cuda.mem_get_info()
    for _ in range(3):
        mvd.reduce_sum_static(x)
    torch.cuda.synchronize()
    assert torch.cuda.memory_allocated() == torch_before
    assert torch.cuda.mem_get_info()[0] >= free_before      # the driver handed out nothing either
