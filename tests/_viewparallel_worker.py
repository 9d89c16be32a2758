"""Worker of tests/test_multirank_host.py::test_view_parallel_exchange_two_gloo_ranks: the exchange
step of the view-parallel combined variants (one all-reduce(SUM) for psi^0, one all-reduce(PRODUCT)
of the partial products per iteration) on 2 gloo ranks, with each rank's factors computed by the
fp64 oracle on CPU; the result must equal the single-process combined iteration (eq. 70 / 104 + eq. 44)."""
import os
import sys

import numpy as np
import torch
import torch.distributed as dist

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)
import mvd_synth  # noqa: E402
from oracle import mvd_oracle as O  # noqa: E402
from paper_1308_0730_b200.binding import split_views  # noqa: E402  (pure host logic, no GPU)


def main():
    dist.init_process_group("gloo")
    rank, world = dist.get_rank(), dist.get_world_size()
    p = mvd_synth.make_tiny_asymmetric()
    V = len(p.views)
    mine = split_views(V, world, rank)
    assert sorted(sum((split_views(V, world, r) for r in range(world)), [])) == list(range(V))
    # psi^0: mean over all views from local sums
    tot = torch.tensor([sum(float(p.views[v].astype(np.float64).sum()) for v in mine),
                        float(sum(p.views[v].size for v in mine))], dtype=torch.float64)
    dist.all_reduce(tot, op=dist.ReduceOp.SUM)
    psi = np.full(p.views[0].shape, float(tot[0] / tot[1]))
    ref = O.Oracle(p.views, p.psfs, "efficient")
    assert np.allclose(psi, ref.psi, rtol=1e-14)
    kernels = ref.kernels                                   # compound kernels need all PSFs on every rank
    for _ in range(2):
        part = np.ones_like(psi)
        for v in mine:
            part *= np.maximum(O.rl_factor(psi, p.views[v], ref.psfs[v], kernels[v]), 0.0)
        t = torch.from_numpy(part)
        dist.all_reduce(t, op=dist.ReduceOp.PRODUCT)
        psi = np.maximum(psi * t.numpy() ** (1.0 / V), O.FLOOR_DEFAULT)
        ref.iterate(1)
        assert np.allclose(psi, ref.psi, rtol=1e-12), float(np.abs(psi / ref.psi - 1).max())
    dist.barrier()
    dist.destroy_process_group()
    print("rank %d ok" % rank)


if __name__ == "__main__":
    main()
