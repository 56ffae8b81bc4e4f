"""The N > 1 path on CPU: two processes over gloo ("replicas only").

The path has no data-path collective (BASELINE.json north_star); what N > 1 adds is the split of
the orbit's frames over the ranks and the reduction of timing / counters, both host logic."""
import os
import socket
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, n_steps, out):
    import torch
    import torch.distributed as dist
    from paper_1012_2909_b200 import replicas
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        mine = replicas.frames_of_rank(n_steps, rank, world)
        gathered = [None] * world
        dist.all_gather_object(gathered, mine)
        # per-rank figures: rank r took (10 + r) ms and counted (100 + r, 7) units
        ms, sums = replicas.reduce_run(dist, "cpu", 10.0 + rank, [100 + rank, 7])
        dist.barrier()
        if rank == 0:
            out.put((gathered, ms, sums))
    finally:
        dist.destroy_process_group()


@pytest.mark.parametrize("n_steps", [4, 24, 180])
def test_two_replicas_split_the_orbit_and_reduce(n_steps):
    import torch.multiprocessing as mp
    ctx = mp.get_context("spawn")
    out = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, n_steps, out)) for r in range(2)]
    for p in procs:
        p.start()
    gathered, ms, sums = out.get(timeout=120)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    a, b = gathered
    assert len(a) == len(b) == n_steps
    assert not set(a) & set(b), "two replicas rendered the same frame"
    allf = sorted(a + b)
    assert len(set(allf)) == 2 * n_steps
    # evenly spread over the 360-frame orbit, interleaved over the ranks
    gaps = [y - x for x, y in zip(allf, allf[1:])]
    assert max(gaps) - min(gaps) <= 1
    assert ms == 11.0                      # the slowest rank
    assert sums == [201, 14]               # counters add up


def test_single_process_is_the_identity():
    from paper_1012_2909_b200 import replicas
    assert replicas.reduce_run(None, "cpu", 3.5, [1, 2]) == (3.5, [1, 2])
    assert replicas.frames_of_rank(4, 0, 1) == [0, 90, 180, 270]
    assert replicas.orbit_frame(359, 360) == 359


# ---- NEXT-1 plumbing (paper_1012_2909_b200/sortlast.py): slab partition and the strip exchange
def test_slab_groups_cover_the_grid():
    from paper_1012_2909_b200 import sortlast as sl
    for grid, world in [((8, 8, 16), 8), ((3, 3, 5), 2), ((3, 3, 5), 3), ((2, 2, 1), 4), ((16, 16, 8), 8)]:
        first = sl.slab_groups(grid, world)
        assert len(first) == world + 1 and first[0] == 0 and first[-1] == grid[0] * grid[1] * grid[2]
        sizes = [b - a for a, b in zip(first, first[1:])]
        assert all(s >= 0 and s % (grid[0] * grid[1]) == 0 for s in sizes)
        assert max(sizes) - min(sizes) <= grid[0] * grid[1]


def test_balanced_groups_minimise_the_heaviest_slab():
    """Linear partition of z-layers by weight (paper_1012_2909_b200/sortlast.py): brute force over all cuts."""
    import itertools
    import numpy as np
    from paper_1012_2909_b200 import sortlast as sl
    rng = np.random.default_rng(5)
    for n, world in ((6, 3), (8, 4), (5, 2), (4, 4), (3, 5)):
        wts = rng.uniform(0.5, 4.0, n)
        first = sl.balanced_groups(wts, 7, world)
        assert first[0] == 0 and first[-1] == 7 * n and all(b >= a for a, b in zip(first, first[1:])) and all(f % 7 == 0 for f in first)
        cuts = [f // 7 for f in first]
        got = max(wts[a:b].sum() for a, b in zip(cuts, cuts[1:]) if b > a)
        k = min(world, n)
        best = min(max(wts[a:b].sum() for a, b in zip((0,) + c, c + (n,))) for c in itertools.combinations(range(1, n), k - 1))
        assert abs(got - best) < 1e-12


def _exchange_worker(rank, world, port, out):
    import torch
    import torch.distributed as dist
    from paper_1012_2909_b200 import sortlast as sl
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        H, W, ch = 7, 5, 4                                   # 7 rows over 2 ranks: a padded last strip
        partial = (torch.arange(H * W * ch, dtype=torch.float32).view(H, W, ch) + 1000.0 * rank)
        versions = sl.exchange_strips(dist, partial, world)  # [sender, rows, W, ch]
        rows = sl.strip_rows(H, world)
        ok = versions.shape == (world, rows, W, ch)
        for sender in range(world):
            want = torch.zeros((rows, W, ch))
            src = torch.arange(H * W * ch, dtype=torch.float32).view(H, W, ch) + 1000.0 * sender
            h = max(0, min(rows, H - rank * rows))
            want[:h] = src[rank * rows:rank * rows + h]
            ok = ok and torch.equal(versions[sender], want)
        # "fold" stand-in (the real one is a CUDA kernel): keep the local rank's version
        frame = sl.gather_strips(dist, versions[rank].clone(), world, H)
        gathered = [None] * world
        dist.all_gather_object(gathered, (ok, frame.shape, float(frame.sum())))
        if rank == 0:
            out.put(gathered)
    finally:
        dist.destroy_process_group()


def test_strip_exchange_over_gloo():
    import torch.multiprocessing as mp
    ctx = mp.get_context("spawn")
    out = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_exchange_worker, args=(r, 2, port, out)) for r in range(2)]
    for p in procs:
        p.start()
    res = out.get(timeout=120)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    assert all(r[0] for r in res)
    assert all(tuple(r[1]) == (7, 5, 4) for r in res)
    assert res[0][2] == res[1][2]                            # every rank ends with the same frame
