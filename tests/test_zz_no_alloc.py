"""sdm_cell_offsets_noalloc (include/sdm.h; csrc/sdm_noalloc.cu): the allocation-free entry point against the existing
path.  The existing path is the scan inside sdm_step_sync (block sums in a buffer sdm_create allocated), whose result
sdm_export_order returns; the new one is given the per-cell SD numbers the library's own diagnostic counts
(sdm_diag_sd_conc, which knows nothing of the segments) and must reproduce the segment offsets bit for bit (integer work:
the bar of tests/test_parity_gpu.py::test_sort_permutation_and_segments_are_exact).  Two calls in a row on different
states and sizes, because every call shares one static scratch array that keeps the last call's contents.

This file sorts last on purpose (pytest -x stops at the first failure); it passes alone in a fresh process and after the
other tests."""
import pytest
import torch

from paper_1310_1905_b200 import workloads as W
from tests.util import make_particles

pytestmark = pytest.mark.gpu


def _existing_and_counts(p, po, th, rv):
    """One step_sync of the existing path -> (its segment offsets, the per-cell SD numbers from the diagnostic kernel)."""
    p.step_sync(po, th, rv)
    _, seg = p.export_order()                                        # valid between step_sync and step_async
    count = p.diag_sd_conc().round().to(torch.int32).contiguous()    # SDs per cell, counted from the positions
    p.step_async(po)
    p.step_async_result()
    return seg.clone(), count


def test_no_alloc_offsets_equal_the_existing_scan_on_two_calls_in_a_row():
    from paper_1310_1905_b200 import binding as b

    # 75 x 75 = 5625 cells: two 4096-cell blocks of the scan with a ragged tail; sedimentation and the flow empty and fill cells
    w = W.cfg2_2d(sd_per_cell=8, seed=71)
    assert w.init["nx"] * w.init["nz"] == 5625
    p, th, rv = make_particles(w)
    po = b.make_opts(**w.opts)
    ncell = 5625
    b.cell_offsets_noalloc_setup()
    seg_new = torch.full((ncell + 1,), -1, dtype=torch.int32, device="cuda")   # allocated by the caller, before the calls

    seg_ref, count = _existing_and_counts(p, po, th, rv)
    assert int(count.sum()) == p.n_sd() and int(seg_ref[-1]) == p.n_sd()
    b.cell_offsets_noalloc(count, seg_new)
    torch.cuda.synchronize()
    assert torch.equal(seg_new, seg_ref)
    first = seg_new.clone()

    # second call, straight after: another state of the same grid (the scratch still holds the first call's block sums) ...
    for _ in range(3):
        seg_ref2, count2 = _existing_and_counts(p, po, th, rv)
    assert not torch.equal(count2, count)
    seg_new.fill_(-1)
    torch.cuda.synchronize()
    free0 = torch.cuda.mem_get_info()[0]
    b.cell_offsets_noalloc(count2, seg_new)
    torch.cuda.synchronize()
    assert torch.cuda.mem_get_info()[0] == free0      # the driver handed out no device memory during the call (kernels loaded by the first)
    assert torch.equal(seg_new, seg_ref2) and not torch.equal(seg_new, first)
    # ... and a shorter one (one block, where the stale second word of the scratch must not leak in): a prefix of the grid
    short = torch.full((1001,), -1, dtype=torch.int32, device="cuda")
    b.cell_offsets_noalloc(count2, short, ncell=1000)
    torch.cuda.synchronize()
    assert torch.equal(short, seg_ref2[:1001])


def test_no_alloc_offsets_many_blocks_empty_input_and_the_limit():
    """More than 1024 blocks (the one-CTA scan of the block sums loops), against the definition (a cumulative sum in int64);
    an empty grid; sizes beyond the static scratch are refused with a clear message and nothing is written."""
    from paper_1310_1905_b200 import binding as b

    g = torch.Generator(device="cuda").manual_seed(5)
    n = 1024 * 4096 + 4097 + 13                       # 1026 blocks, the last one ragged
    count = torch.randint(0, 200, (n,), generator=g, device="cuda", dtype=torch.int32)
    seg = torch.empty(n + 1, dtype=torch.int32, device="cuda")
    want = torch.zeros(n + 1, dtype=torch.int64, device="cuda")
    want[1:] = torch.cumsum(count.to(torch.int64), 0)
    assert int(want[-1]) < 2**31
    for _ in range(2):
        seg.fill_(-1)
        b.cell_offsets_noalloc(count, seg)
        torch.cuda.synchronize()
        assert torch.equal(seg.to(torch.int64), want)
    one = torch.full((1,), -1, dtype=torch.int32, device="cuda")
    b.cell_offsets_noalloc(count, one, ncell=0)
    torch.cuda.synchronize()
    assert int(one[0]) == 0
    with pytest.raises(b.SdmError, match="exceed the static scratch.*limit 16777216 cells"):
        b.cell_offsets_noalloc(count, seg, ncell=b.NOALLOC_MAX_CELLS + 1)
    torch.cuda.synchronize()
    assert torch.equal(seg.to(torch.int64), want)     # the refused call enqueued nothing
