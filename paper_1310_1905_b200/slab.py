"""Domain decomposition along x (PAPER.md :843): host-side exchange of the super-droplets that
crossed a slab's faces.  Plumbing only: which list goes to which neighbour, by how much its x is shifted, and the
``torch.distributed`` send/recv (``nccl`` on GPUs, ``gloo`` in the CPU tests).  The lists themselves come from, and go
back into, the library's kernels (``Particles.pack_leavers`` / ``unpack_arrivals``); nothing here touches an attribute
other than to move it.

Slabs: rank r of P owns the columns [i0_r, i0_r + nx_r) of the global grid, periodic in x, in a context created with
``open_x=True`` on ``nx_r`` columns whose x coordinate is relative to the slab.  An SD that leaves rank r through its
right face (x >= X_r) arrives at rank (r+1) mod P with x - X_r; through its left face (x < 0) at rank (r-1) mod P with
x + X_{r-1}.
"""
import torch
import torch.distributed as dist

KEYS = ("n", "rw2", "rd3", "kappa", "x", "y", "z", "id")


def split_columns(nx, world):
    """(first column, number of columns) of every rank: nx columns dealt as evenly as possible, in order."""
    base, extra = divmod(nx, world)
    out, i0 = [], 0
    for r in range(world):
        n = base + (1 if r < extra else 0)
        out.append((i0, n))
        i0 += n
    return out


def neighbours(rank, world):
    return (rank - 1) % world, (rank + 1) % world


def arrival_shifts(rank, widths):
    """x shifts for what arrives from the left neighbour (its right list) and from the right neighbour (its left list)."""
    left, _ = neighbours(rank, len(widths))
    return -widths[left], widths[rank]


def exchange_lists(left, right, rank=None, world=None, group=None):
    """Sends this rank's `left` / `right` lists (dicts of 1-D tensors keyed by KEYS, equal length within a list) to its left /
    right neighbour and returns (from_left, from_right): what the left neighbour sent rightwards and what the right
    neighbour sent leftwards.  Works on CPU tensors with gloo and on CUDA tensors with nccl; world == 1 wraps around."""
    rank = dist.get_rank(group) if rank is None else rank
    world = dist.get_world_size(group) if world is None else world
    if world == 1:
        return right, left
    ln, rn = neighbours(rank, world)
    dev = left["n"].device
    # counts first (the lists have data-dependent lengths)
    mine = torch.tensor([left["n"].numel(), right["n"].numel()], dtype=torch.int64, device=dev)
    counts = [torch.zeros(2, dtype=torch.int64, device=dev) for _ in range(world)]
    dist.all_gather(counts, mine, group=group)
    n_from_left, n_from_right = int(counts[ln][1]), int(counts[rn][0])
    from_left = {k: torch.empty(n_from_left, dtype=left[k].dtype, device=dev) for k in KEYS}
    from_right = {k: torch.empty(n_from_right, dtype=left[k].dtype, device=dev) for k in KEYS}
    ops = []
    for t, k in enumerate(KEYS):   # tags keep the two directions apart when both neighbours are the same rank (world == 2)
        if left[k].numel():
            ops.append(dist.P2POp(dist.isend, left[k].contiguous(), ln, group, tag=2 * t))
        if right[k].numel():
            ops.append(dist.P2POp(dist.isend, right[k].contiguous(), rn, group, tag=2 * t + 1))
        # receives in the order the peer sends (its left list, then its right list): nccl matches messages between two
        # ranks in posting order and ignores tags
        if n_from_right:
            ops.append(dist.P2POp(dist.irecv, from_right[k], rn, group, tag=2 * t))
        if n_from_left:
            ops.append(dist.P2POp(dist.irecv, from_left[k], ln, group, tag=2 * t + 1))
    if ops:
        for req in dist.batch_isend_irecv(ops):
            req.wait()
    return from_left, from_right


def exchange(p, widths, cap, rank=None, world=None, group=None):
    """One exchange step of a rank's ``Particles`` p (open_x) after step_async: pack, send/recv, unpack.  widths: slab
    widths [m] of all ranks; cap: SDs a list may hold.  Returns the numbers (sent left, sent right, got from left, got from right)."""
    rank = dist.get_rank(group) if rank is None else rank
    left, right = p.pack_leavers(cap)
    from_left, from_right = exchange_lists(left, right, rank, len(widths), group)
    s_left, s_right = arrival_shifts(rank, widths)
    p.unpack_arrivals(from_left, s_left)
    p.unpack_arrivals(from_right, s_right)
    return left["n"].numel(), right["n"].numel(), from_left["n"].numel(), from_right["n"].numel()


def exchange_local(parts, widths, cap):
    """The same exchange between contexts living in ONE process (one GPU holding every slab): parts[r] is rank r's
    Particles.  Used by the single-GPU parity test of the pack / unpack kernels; no communication library involved."""
    world = len(parts)
    lists = [p.pack_leavers(cap) for p in parts]
    for r, p in enumerate(parts):
        ln, rn = neighbours(r, world)
        s_left, s_right = arrival_shifts(r, widths)
        p.unpack_arrivals(lists[ln][1], s_left)
        p.unpack_arrivals(lists[rn][0], s_right)
    return [(l["n"].numel(), r["n"].numel()) for l, r in lists]
