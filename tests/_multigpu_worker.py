"""Worker of tests/test_multigpu.py: one of WORLD_SIZE NCCL ranks, one GPU each.

(a) view-parallel combined variants: views dealt round-robin, one
    all-reduce(PRODUCT) per iteration on the library's stream; psi must stay bit-identical on every rank and
    match the fp64 oracle within the north_star tolerances.
(b) blocks dealt over the ranks (L225): every rank deconvolves its share of the blocks, the shares are disjoint,
    their sum is the single-GPU blocked result and matches the blocked oracle."""
import os
import sys

import numpy as np
import torch
import torch.distributed as dist

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)
import mvd_synth  # noqa: E402
import paper_1308_0730_b200 as mvd  # noqa: E402
from oracle import mvd_oracle as O  # noqa: E402


def errors(g, o):
    g, o = np.asarray(g, np.float64), np.asarray(o, np.float64)
    return (float(np.linalg.norm(g - o) / np.linalg.norm(o)), float((np.abs(g - o) / np.maximum(np.abs(o), 1e-6)).max()))


def main():
    local = int(os.environ["LOCAL_RANK"])
    torch.cuda.set_device(local)
    dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    rank, world = dist.get_rank(), dist.get_world_size()
    p = mvd_synth.make_tiny_asymmetric(dims=(40, 36, 30), psf_dims=(5, 7, 9), n_views=4)
    V = len(p.views)
    for variant in ("efficient", "independent"):
        mine = mvd.split_views(V, world, rank)
        d = mvd.ViewParallelDeconvolver([torch.from_numpy(p.views[v]).cuda() for v in mine], p.psfs, variant=variant,
                                        rank=rank, world=world, stream=torch.cuda.Stream())
        o = O.Oracle(p.views, p.psfs, variant)
        for it in range(3):
            d.iterate(1)
            o.iterate(1)
            g = d.get_estimate_host()
            l2, mx = errors(g, o.psi)
            assert l2 <= (1e-5 if it == 0 else 1e-4) and mx <= 1e-3, (variant, it, l2, mx)
            t = torch.from_numpy(g).cuda()
            parts = [torch.empty_like(t) for _ in range(world)]
            dist.all_gather(parts, t)
            for q in parts:
                assert torch.equal(q, parts[0]), "psi differs between ranks"
        st = d.get_stats()
        assert abs(st["flux"] - o.flux) <= 1e-5 * o.flux and st["iterations_done"] == 3
        d.close()
    # (b) blocks dealt over the ranks
    q = mvd_synth.make_problem(1, dims=(48, 40, 36), psf_dims=(7, 7, 11))
    views = [torch.from_numpy(v).cuda() for v in q.views]
    block = (20, 24, 16)
    part, _ = mvd.deconvolve_blocked(views, q.psfs, block, 2, variant="osem", block_rank=rank, block_world=world)
    owned = (part != 0).to(torch.float32)
    total, cover = part.clone(), owned.clone()
    dist.all_reduce(total)
    dist.all_reduce(cover)
    assert bool((cover == 1).all()), "blocks of the ranks overlap or leave gaps"
    ref = O.deconvolve_blocked(q.views, q.psfs, block[::-1], "osem", 2)
    l2, mx = errors(total.cpu().numpy(), ref)
    assert l2 <= 1e-4 and mx <= 1e-3, (l2, mx)
    dist.barrier()
    dist.destroy_process_group()
    print("rank %d ok" % rank)


if __name__ == "__main__":
    main()
