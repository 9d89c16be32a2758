"""Worker of tests/test_multirank_host.py: one of WORLD_SIZE gloo ranks on CPU.  Exercises the host
logic bench.py uses when --gpus N > 1 (replicas only): rank 0 draws the
problem and hands it to the others, times are reduced with MAX over ranks, the value is the
whole-job aggregate."""
import os
import sys

import numpy as np
import torch.distributed as dist

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)
import bench  # noqa: E402
import mvd_synth  # noqa: E402


def main():
    dist.init_process_group("gloo")
    rank, world = dist.get_rank(), dist.get_world_size()
    prob = bench.load_problem(1, rank, world, dist)
    ref = mvd_synth.make_problem(1)                       # every rank can redraw: seeds are fixed
    assert len(prob.views) == len(ref.views) == 4
    for a, b in zip(prob.views, ref.views):
        assert np.array_equal(a, b)
    for a, b in zip(prob.psfs, ref.psfs):
        assert np.array_equal(a, b)
    # slowest replica sets the time; value counts the units of all replicas
    mine = [10.0 + rank, 5.0 - rank]
    got = bench.max_over_ranks(mine, world, dist, "cpu")
    assert got == [10.0 + world - 1, 5.0], got
    v = bench.replica_throughput(world, 1e6, 4, got[0])
    assert abs(v - world * 1e6 * 4 / (got[0] * 1e-3) / 1e9) < 1e-12
    dist.barrier()
    dist.destroy_process_group()
    print("rank %d ok" % rank)


if __name__ == "__main__":
    main()
