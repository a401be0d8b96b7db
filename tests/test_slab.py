"""Host side of the x-slab decomposition (paper_1310_1905_b200/slab.py): who sends which list to whom
and by how much x is shifted, exercised with gloo ranks on CPU tensors (world sizes 2 and 3).  The pack / unpack kernels
themselves are covered on the GPU by tests/test_parity_gpu.py::test_three_slabs_on_one_gpu_match_the_oracle_on_the_whole_domain."""
import os
import socket

import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_1310_1905_b200 import slab


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _fake_list(rank, side, count):
    """A list of `count` SDs whose every attribute encodes (sender, side, index), so that a mix-up shows."""
    base = 1000 * rank + 100 * side
    i = torch.arange(count, dtype=torch.float64)
    d = {k: base + i + 0.1 * j for j, k in enumerate(("rw2", "rd3", "kappa", "x", "y", "z"))}
    d["n"] = (base + torch.arange(count)).to(torch.int64)
    d["id"] = (base + torch.arange(count)).to(torch.int32)
    return d


def _worker(rank, world, port, out):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        # rank r sends r + 1 SDs leftwards and 2 r SDs rightwards (rank 0: an empty right list)
        left, right = _fake_list(rank, 0, rank + 1), _fake_list(rank, 1, 2 * rank)
        from_left, from_right = slab.exchange_lists(left, right)
        out.put((rank, {k: v.tolist() for k, v in from_left.items()}, {k: v.tolist() for k, v in from_right.items()}))
        dist.barrier()
    finally:
        dist.destroy_process_group()


def _run(world):
    ctx = mp.get_context("spawn")
    out = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, world, port, out)) for r in range(world)]
    for p in procs:
        p.start()
    res = sorted((out.get(timeout=120) for _ in procs), key=lambda t: t[0])
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    for rank, from_left, from_right in res:
        ln, rn = (rank - 1) % world, (rank + 1) % world
        want_l, want_r = _fake_list(ln, 1, 2 * ln), _fake_list(rn, 0, rn + 1)   # left neighbour's RIGHT list, right neighbour's LEFT list
        for k in slab.KEYS:
            assert from_left[k] == want_l[k].tolist(), (rank, k)
            assert from_right[k] == want_r[k].tolist(), (rank, k)


def test_exchange_lists_two_gloo_ranks_where_both_neighbours_are_the_same_rank():
    _run(2)


def test_exchange_lists_three_gloo_ranks_ring():
    _run(3)


def test_columns_neighbours_and_shifts():
    assert slab.split_columns(16, 2) == [(0, 8), (8, 8)]
    assert slab.split_columns(75, 4) == [(0, 19), (19, 19), (38, 19), (57, 18)]
    assert sum(n for _, n in slab.split_columns(128, 8)) == 128
    assert slab.neighbours(0, 4) == (3, 1) and slab.neighbours(3, 4) == (2, 0)
    widths = [380.0, 380.0, 380.0, 360.0]
    # from the left neighbour an SD arrives with x >= that neighbour's width; from the right one with x < 0
    assert slab.arrival_shifts(0, widths) == (-360.0, 380.0)      # rank 0's left neighbour is rank 3 (periodic)
    assert slab.arrival_shifts(3, widths) == (-380.0, 360.0)
    # a single rank wraps around: what left through the right face comes back from the left
    l, r = _fake_list(0, 0, 2), _fake_list(0, 1, 3)
    fl, fr = slab.exchange_lists(l, r, rank=0, world=1)
    assert fl is r and fr is l
