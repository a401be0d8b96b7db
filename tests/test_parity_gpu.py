"""Parity of the CUDA path (through the C ABI) against the oracle, element by element, on the same
seeded inputs.  Bars (BASELINE.json north_star): multiplicities, ids, order and pairings bit-exact;
radii, positions, th, rv within 1e-9 relative (fp64); near-tie collision decisions counted."""
import numpy as np
import pytest
import torch

import oracle
from paper_1310_1905_b200 import workloads as W
from tests.util import make_oracle, make_particles, np_, sorted_by_id

pytestmark = pytest.mark.gpu

RTOL = 1e-9


def binding():
    from paper_1310_1905_b200 import binding as b

    return b


def rain_mix(w, seed=5, frac=0.25):
    """Give a fraction of the SDs cloud/drizzle/rain sizes so that coalescence and sedimentation act within a
    few steps (the t = 0 population is all haze), and put some large drops just above the ground."""
    N = w.n_sd
    idx = torch.arange(N, dtype=torch.int64)
    u = W.hash_uniform(seed, 101, idx)
    v = W.hash_uniform(seed, 102, idx)
    big = u < frac
    r = torch.exp(np.log(3e-6) + v * (np.log(400e-6) - np.log(3e-6)))
    rw2 = torch.where(big, r * r, w.state["rw2"])
    w.state["rw2"] = torch.maximum(rw2, (w.state["rd3"] ** (1.0 / 3.0)) ** 2 * 1.0001)
    # rain-sized SDs carry far fewer real drops
    w.state["n"] = torch.where(big, torch.clamp(w.state["n"] // 1000, min=1), w.state["n"])
    if w.state["z"] is not None:
        low = W.hash_uniform(seed, 103, idx) < 0.02
        w.state["z"] = torch.where(low & big, w.state["z"] * 0.002, w.state["z"])
    return w


def compare_states(p, o, positions=True, rtol=RTOL, drift=None):
    """drift = (fraction, rtol_loose), for free-running trajectories of hundreds of steps only: the wet radii of all but
    `fraction` of the SDs within rtol, every one within rtol_loose ("trajectory bar": a droplet that
    evaporates towards its dry size multiplies a relative difference in r^2 by r^2_before / r^2_now, so a difference at
    the rounding level surfaces, for the few steps that takes, above 1e-9 on a few SDs in 10^5, and decays again); positions
    within rtol_loose metres (a falling drop integrates the fall speed of its drifted radius over hundreds of steps)."""
    g = sorted_by_id(p.export_state())
    r = sorted_by_id(o.get_state())
    assert len(g["id"]) == len(r["id"])
    np.testing.assert_array_equal(g["id"].astype(np.uint32), r["id"])
    np.testing.assert_array_equal(g["n"].astype(np.uint64), r["n"])      # multiplicities: bit-exact
    live = r["n"] > 0
    if drift is None:
        np.testing.assert_allclose(np.sqrt(g["rw2"]), np.sqrt(r["rw2"]), rtol=rtol)
    else:
        rel = np.abs(np.sqrt(g["rw2"]) - np.sqrt(r["rw2"])) / np.sqrt(r["rw2"])
        assert np.count_nonzero(rel > rtol) <= drift[0] * rel.size, (np.count_nonzero(rel > rtol), rel.size)
        assert rel.max() <= drift[1], rel.max()
    np.testing.assert_allclose(np.cbrt(g["rd3"]), np.cbrt(r["rd3"]), rtol=rtol)
    np.testing.assert_allclose(g["kappa"], r["kappa"], rtol=rtol)
    if positions:
        for k, present in zip("xyz", p.dims):
            if present:   # (free-running: a position integrates the fall speed of a radius that drifted, see the docstring)
                np.testing.assert_allclose(g[k][live], r[k][live], rtol=rtol, atol=1e-9 if drift is None else drift[1])
    return g, r


def compare_fields(th, rv, o, rtol=RTOL):
    oth, orv = o.get_fields()
    np.testing.assert_allclose(np_(th).ravel(), oth, rtol=rtol)
    np.testing.assert_allclose(np_(rv).ravel(), orv, rtol=rtol)


def run_both(w, steps, group=0, opts=None, check_every=1, recycle=False, threads=4, **override):
    b = binding()
    kw = dict(w.opts)
    kw.update(opts or {})
    o = make_oracle(w, threads=threads, **override)
    p, th, rv = make_particles(w, **override)
    if recycle:
        o.set_recycle(True)
        p.set_recycle(True)
    if group:
        p.set_group_size(group)
    oo, po = oracle.make_opts(**kw), b.make_opts(**kw)
    for s in range(steps):
        fo = o.step(oo)
        p.step_sync(po, th, rv)
        p.step_async(po)
        fp = p.step_async_result()
        # rain flux = sum of N (4/3) pi rho_w r_w^3 over SDs whose radii match within RTOL -> 3 RTOL
        np.testing.assert_allclose(fp, fo, rtol=3 * RTOL, atol=1e-300)
        if (s + 1) % check_every == 0 or s == steps - 1:
            compare_states(p, o, positions=True)
            compare_fields(th, rv, o)
    return p, o, th, rv


# ----------------------------------------------------------------------------------------------- sort
@pytest.mark.parametrize("group", [0, 4, 8, 16, 32, 256])
def test_sort_permutation_and_segments_are_exact(group):
    """a0-a2: compaction + (cell, Philox key, id) order identical to std::sort on the tuple."""
    b = binding()
    w = W.cfg2_2d(sd_per_cell=20, nx=23, nz=17, seed=3)
    n = w.state["n"].clone()
    n[::13] = 0   # dead SDs must be compacted away
    w.state["n"] = n
    w.state["id"] = torch.flip(w.state["id"], [0]).contiguous()   # ids unrelated to storage order
    o = make_oracle(w)
    p, th, rv = make_particles(w)
    if group:
        p.set_group_size(group)
    for step in (0, 5):
        o.set_step(step)
        p.set_step(step)
        o.stage("sort")
        po = b.make_opts(adve=False, sedi=False, cond=False, coal=False)
        p.step_sync(po, th, rv)
        ids, seg = p.export_order()
        oids, oseg = o.get_order()
        np.testing.assert_array_equal(np_(seg).astype(np.int64), oseg)
        np.testing.assert_array_equal(np_(ids).astype(np.uint32), oids)
        assert p.n_sd() == o.n_sd() == int((n != 0).sum())
        p.step_async(po)
        o.step_async(oracle.make_opts(adve=False, sedi=False, cond=False, coal=False))
    assert p.stats()["max_cell_count"] == np.diff(oseg).max()


# ----------------------------------------------------------------------------------------------- box
def test_box_golovin_trajectory_bit_exact_multiplicities():
    """configs[0]: 2^13 SDs in one cell, Golovin kernel, coalescence only."""
    w = W.box_golovin(seed=42)
    p, o, _, _ = run_both(w, 400, check_every=100)
    sp, so = p.stats(), o.counters()
    assert sp["pairs"] == so["pairs"] and sp["collisions"] == so["collisions"] and so["collisions"] > 1000
    assert sp["near_ties"] == so["near_ties"] and so["near_ties"] <= 1e-6 * so["pairs"] + 1
    assert p.n_sd() == o.n_sd() < w.n_sd


# ----------------------------------------------------------------------------------------------- full step
@pytest.mark.parametrize("group", [0, 8, 32, 256])
def test_full_step_2d_single_and_few_steps(group):
    w = rain_mix(W.cfg2_2d(sd_per_cell=32, nx=20, nz=24, seed=11))
    p, o, th, rv = run_both(w, 4, group=group)
    sp, so = p.stats(), o.counters()
    assert sp["pairs"] == so["pairs"] and sp["collisions"] == so["collisions"] and so["collisions"] > 50
    assert sp["ill_posed"] == so["ill_posed"]
    assert sp["sd_substeps"] == so["sd_substeps"]
    assert o.rain_flux_total() > 0 and p.n_sd() < w.n_sd   # sedimentation removed SDs, compaction followed


def test_trajectory_2d_30_steps():
    w = rain_mix(W.cfg2_2d(sd_per_cell=16, nx=16, nz=16, seed=2))
    p, o, th, rv = run_both(w, 30, check_every=10)
    sp, so = p.stats(), o.counters()
    assert sp["collisions"] == so["collisions"] and sp["ill_posed"] == so["ill_posed"]
    assert so["near_ties"] <= 1e-6 * so["pairs"] + 1


def test_full_step_3d():
    w = rain_mix(W.cfg4_3d(sd_per_cell=64, nx=6, ny=5, nz=16, seed=4))
    p, o, th, rv = run_both(w, 3)
    assert p.stats()["collisions"] == o.counters()["collisions"] > 0


def test_sparse_cells_many_cells_per_tile():
    """4 SDs per cell on 800 x 670 cells: tiles of several dozen cells (the sparse instantiation of k_coal_move_tile, its
    offset scan beyond 32 cells per tile, the flat staging loops), all-pairs rank counting; and a small box without any
    spatial dimension through the tile kernel."""
    import os
    w = rain_mix(W.cfg2_2d(sd_per_cell=4, nx=800, nz=670, seed=15), frac=0.4)   # 2.14 M SDs: beyond the few-wave tile sizing
    p, o, th, rv = run_both(w, 3, threads=os.cpu_count() or 4)
    sp, so = p.stats(), o.counters()
    assert sp["coal_tile_cells"] >= 8 and sp["cond_tile_cells"] >= 8
    assert sp["pairs"] == so["pairs"] and sp["collisions"] == so["collisions"] > 0
    wb = W.box_golovin(seed=45, n_sd=256)
    p, o, _, _ = run_both(wb, 20, check_every=5, dx=12.0, dy=12.0, dz=12.0)
    assert p.stats()["coal_tile_cells"] == 1 and p.stats()["collisions"] == o.counters()["collisions"] > 50


def test_hydro_tab_kernel_and_paper_variant_without_multiple_coalescence():
    w = rain_mix(W.cfg3_2d_drizzle(sd_per_cell=48, nx=10, nz=12, seed=6))
    run_both(w, 3)
    run_both(w, 2, multi_coal=False)


def test_coalescence_substeps_reshuffle():
    """sstp_coal > 1: new keys and a new sort inside the cell every substep, dead SDs dropped (:624)."""
    w = rain_mix(W.cfg2_2d(sd_per_cell=40, nx=8, nz=8, seed=9), frac=0.6)
    for group in (0, 256):
        p, o, _, _ = run_both(w, 3, group=group, opts=dict(sstp_coal=4, cond=False))
        assert p.stats()["collisions"] == o.counters()["collisions"] > 100


def test_process_toggles():
    w = rain_mix(W.cfg2_2d(sd_per_cell=16, nx=8, nz=8, seed=10))
    for opts in (dict(adve=True, sedi=False, cond=False, coal=False), dict(adve=False, sedi=True, cond=False, coal=False),
                 dict(adve=False, sedi=False, cond=True, coal=False), dict(adve=False, sedi=False, cond=False, coal=True),
                 dict(adve=False, sedi=False, cond=False, coal=False)):
        run_both(w, 2, opts=opts)


def test_crowded_cells_fall_back_to_global_memory_paths():
    """One cell with far more SDs than shared memory can stage: condensation and coalescence run in place."""
    w = rain_mix(W.cfg2_2d(sd_per_cell=1500, nx=2, nz=3, seed=12), frac=0.3)
    w.state["x"] = w.state["x"] * 0.4   # crowd everything into the first column: 3 cells with ~3000 SDs
    p, o, _, _ = run_both(w, 2, group=32, opts=dict(sstp_cond=2))
    assert p.stats()["max_cell_count"] > 2500


def test_cells_of_a_thousand_sds():
    """~1000 SDs per cell (top of the configs[4] sweep): the 1280-slot condensation tile kernel, bitonic ranks by a
    CTA per cell, the per-cell coalescence kernel."""
    w = rain_mix(W.cfg2_2d(sd_per_cell=1000, nx=3, nz=4, seed=14), frac=0.3)
    p, o, _, _ = run_both(w, 2, opts=dict(sstp_cond=3))
    assert 800 < p.stats()["max_cell_count"] <= 1280
    assert p.stats()["collisions"] == o.counters()["collisions"] > 0


# ----------------------------------------------------------------------------------------------- API
def test_strided_fields_and_optional_arguments():
    """arrinfo_t strides (:730-745): halo-padded, non-contiguous th/rv/rhod give the same result."""
    b = binding()
    w = rain_mix(W.cfg2_2d(sd_per_cell=16, nx=9, nz=7, seed=13))
    p1, th1, rv1 = make_particles(w)
    p2, _, _ = make_particles(w)
    pad_th = torch.full((9 + 4, 7 + 6), -1.0, dtype=torch.float64, device="cuda")
    pad_rv = torch.full((7 + 2, 9 + 2), -1.0, dtype=torch.float64, device="cuda")   # transposed storage
    th2 = pad_th[2:-2, 3:-3]
    rv2 = pad_rv[1:-1, 1:-1].t()
    th2.copy_(w.th.cuda())
    rv2.copy_(w.rv.cuda())
    rhod_pad = torch.zeros((9, 2 * 7), dtype=torch.float64, device="cuda")
    rhod2 = rhod_pad[:, ::2]
    rhod2.copy_(w.rhod.cuda())
    po = b.make_opts(**w.opts)
    for _ in range(2):
        p1.step_sync(po, th1, rv1)
        p1.step_async(po)
        p2.step_sync(po, th2, rv2, rhod=rhod2)
        p2.step_async(po)
    assert torch.equal(th1, th2) and torch.equal(rv1, rv2)
    assert pad_th[0, 0] == -1 and pad_th[-1, -1] == -1 and pad_rv[0, 0] == -1   # halo untouched
    a, c = sorted_by_id(p1.export_state()), sorted_by_id(p2.export_state())
    for k in a:
        np.testing.assert_array_equal(a[k], c[k])


def test_new_courant_fields_and_rhod_handed_to_step_sync_mid_run():
    """step_sync with new Courant fields and a new rho_d in the middle of a run (:751, :816: "may be omitted when unchanged"):
    k_coal_move_tile takes its eq. 16 coefficients from a per-cell table (k_cell_move_consts) that must be rebuilt exactly
    then; the oracle is handed the same fields before the same step."""
    from tests.util import courant_xyz

    b = binding()
    w = rain_mix(W.cfg2_2d(sd_per_cell=24, nx=12, nz=16, seed=61))
    o = make_oracle(w)
    p, th, rv = make_particles(w)
    oo, po = oracle.make_opts(**w.opts), b.make_opts(**w.opts)
    c = courant_xyz(w)
    for s in range(6):
        kw = {}
        if s == 2:     # the flow reversed and halved from here on (rho_d C stays non-divergent)
            cx2, cz2 = (-0.5 * c["x"]).contiguous(), (-0.5 * c["z"]).contiguous()
            o.set_fields(cx=np_(cx2).ravel(), cz=np_(cz2).ravel())
            kw = dict(courant_1=cx2.cuda(), courant_2=cz2.cuda())
        if s == 4:     # a new rho_d alone (the table divides the Courant fields by it)
            rhod2 = (1.002 * w.rhod).contiguous()
            o.set_fields(rhod=np_(rhod2).ravel())
            kw = dict(rhod=rhod2.cuda())
        fo = o.step(oo)
        p.step_sync(po, th, rv, **kw)
        p.step_async(po)
        np.testing.assert_allclose(p.step_async_result(), fo, rtol=3 * RTOL, atol=1e-300)
        compare_states(p, o, positions=True)
        compare_fields(th, rv, o)
    assert p.stats()["coal_tile_cells"] > 0     # the tile kernel (and its table) did run


def test_step_host_matches_device_path():
    b = binding()
    w = rain_mix(W.cfg2_2d(sd_per_cell=16, nx=9, nz=7, seed=14))
    p1, th1, rv1 = make_particles(w)
    p2, _, _ = make_particles(w)
    th_h, rv_h = w.th.clone().pin_memory(), w.rv.clone().pin_memory()
    po = b.make_opts(**w.opts)
    for _ in range(3):
        p1.step_sync(po, th1, rv1)
        p1.step_async(po)
        f1 = p1.step_async_result()
        f2 = p2.step_host(po, th_h, rv_h)
        assert f1 == f2
    assert torch.equal(th1.cpu(), th_h) and torch.equal(rv1.cpu(), rv_h)


def test_diagnostics_match_oracle():
    """Moments are sums of N r^k over radii that match the oracle's within RTOL (Newton root against the
    bisected one), so M^k matches within k * RTOL (plus summation order, ~1e-15); counts are exact."""
    w = rain_mix(W.cfg2_2d(sd_per_cell=24, nx=11, nz=9, seed=15))
    p, o, th, rv = run_both(w, 2)
    np.testing.assert_array_equal(np_(p.diag_sd_conc()).ravel(), o.diag_sd_conc())
    for lo, hi in ((0.5e-6, 25e-6), (25e-6, 1.0), (0.0, 1.0)):   # thresholds of PAPER.md :862
        p.diag_wet_rng(lo, hi)
        for k in (0, 3):
            np.testing.assert_allclose(np_(p.diag_wet_mom(k)).ravel(), o.diag_mom(1, lo, hi, k), rtol=max(k, 1) * RTOL)
    p.diag_dry_rng(10e-9, 1e-6)
    np.testing.assert_allclose(np_(p.diag_dry_mom(1)).ravel(), o.diag_mom(0, 10e-9, 1e-6, 1), rtol=RTOL)


def test_edge_cases_empty_single_and_errors():
    b = binding()
    w = W.cfg2_2d(sd_per_cell=4, nx=4, nz=4, seed=16)
    po = b.make_opts(**w.opts)
    # empty population
    e = W.cfg2_2d(sd_per_cell=4, nx=4, nz=4, seed=16)
    e.state = {k: (None if v is None else v[:0]) for k, v in e.state.items()}
    p, th, rv = make_particles(e, max_sd=8)
    for _ in range(2):
        p.step_sync(po, th, rv)
        p.step_async(po)
    assert p.step_async_result() == 0.0 and p.n_sd() == 0 and torch.equal(th.cpu(), w.th)
    assert np_(p.diag_sd_conc()).sum() == 0
    # a single SD
    s = W.cfg2_2d(sd_per_cell=4, nx=4, nz=4, seed=16)
    s.state = {k: (None if v is None else v[:1].clone()) for k, v in s.state.items()}
    run_both(s, 2)
    # errors, not UB
    p, th, rv = make_particles(w)
    with pytest.raises(b.SdmError, match="step_sync of this step"):
        p.step_async(po)
    p.step_sync(po, th, rv)
    with pytest.raises(b.SdmError, match="called twice"):
        p.step_sync(po, th, rv)
    with pytest.raises(b.SdmError, match="exceeds max_sd"):
        make_particles(w, max_sd=w.n_sd - 1)
    with pytest.raises(b.SdmError, match="real_bytes|max_sd"):
        b.Particles(nx=2, nz=2, max_sd=0)


@pytest.mark.parametrize("mode", ["fp64", "fp32_sweep_recycle", "3d_larger"])
def test_runs_are_reproducible_bit_for_bit(mode):
    """Storage order inside a cell and the order of list appends depend on atomics, results must not (this is also the
    race detector of the tile kernels: compute-sanitizer is not available on the GPU pool)."""
    b = binding()
    if mode == "3d_larger":
        w = rain_mix(W.cfg4_3d(sd_per_cell=64, nx=16, ny=16, nz=64, seed=18))
    else:
        w = rain_mix(W.cfg2_2d(sd_per_cell=32, nx=12, nz=12, seed=17))
    outs = []
    for _ in range(3 if mode != "3d_larger" else 2):
        if mode == "fp32_sweep_recycle":
            st32 = {k: (v if v is None or k in ("n", "id") else v.to(torch.float32).cuda()) for k, v in w.state.items()}
            p = b.Particles(max_sd=w.n_sd, sd_conc_mean=w.meta["sd_per_cell"], real_bytes=4, **w.init)
            cs = [c.cuda() for c in w.courants] + [None] * (3 - len(w.courants))
            p.init_from_arrays(w.rhod.cuda(), w.state["n"].cuda(), st32["rw2"], st32["rd3"], st32["kappa"], st32["x"], st32["y"], st32["z"],
                               w.state["id"].cuda(), courant_1=cs[0], courant_2=cs[1], courant_3=cs[2])
            th, rv = w.th.cuda().clone(), w.rv.cuda().clone()
            p.set_cond_arith(4)
            p.set_recycle(True)
        else:
            p, th, rv = make_particles(w)
        po = b.make_opts(**w.opts)
        for _ in range(4):
            p.step_sync(po, th, rv)
            p.step_async(po)
        outs.append((sorted_by_id(p.export_state()), th.clone(), rv.clone()))
    for o in outs[1:]:
        for k in outs[0][0]:
            np.testing.assert_array_equal(outs[0][0][k], o[0][k])
        assert torch.equal(outs[0][1], o[1]) and torch.equal(outs[0][2], o[2])


# ------------------------------------------------------------------------------------ full size (bench.py's launch)
def test_full_size_3d_sampled_columns_match_oracle():
    """configs[3] at full size (128 x 128 x 64 cells, 67 108 864 SDs), in the launch configuration bench.py times.
    Every stage but the reorder is local to a column of cells, so the oracle can compute a sampled block of
    columns on its own: after 3 steps of the whole domain on the GPU, the SDs of a 16 x 16 x 64 block (1.05 M SDs)
    and of a 2 x 1 x 64 block whose cells touch both periodic borders are handed to the oracle (same ids, same step
    counter, fields and Courant numbers sliced), both advance, and the blocks' SDs are compared one by one.
    Horizontal positions are compared modulo the block width (an SD that leaves the block wraps in the oracle's small
    periodic domain).  The large block is compared over TWO steps: after the first, its border columns have exchanged
    SDs with the rest of the domain (in the oracle: with the opposite border), so the second step is compared on the
    SDs and cells of its interior 14 x 14 columns, which no SD from outside can have reached (Courant numbers < 1)."""
    import os
    b = binding()
    torch.cuda.empty_cache()
    w = W.cfg4_3d(device="cuda")
    nx, ny, nz, dx = w.init["nx"], w.init["ny"], w.init["nz"], w.init["dx"]
    n_total = w.n_sd
    assert n_total == 67108864
    p = b.Particles(max_sd=n_total, sd_conc_mean=64, **w.init)
    s = w.state
    p.init_from_arrays(w.rhod, s["n"], s["rw2"], s["rd3"], s["kappa"], s["x"], s["y"], s["z"], s["id"],
                       courant_1=w.courants[0], courant_2=w.courants[1], courant_3=w.courants[2])
    th, rv = w.th.clone(), w.rv.clone()
    w.state = None
    del s
    torch.cuda.empty_cache()
    po, oo = b.make_opts(**w.opts), oracle.make_opts(**w.opts)
    for _ in range(3):
        p.step_sync(po, th, rv)
        p.step_async(po)
    st = p.export_state()                      # storage order, dead SDs of the last step still present
    N0 = st["id"].numel()
    blocks = [(37, 90, 16, 16), (0, 127, 2, 1)]  # (i0, j0, bx, by); the second touches both periodic borders' cells
    ci = torch.clamp((st["x"] / dx).floor().long(), 0, nx - 1)
    cj = torch.clamp((st["y"] / dx).floor().long(), 0, ny - 1)
    oracles, picks = [], []
    for (i0, j0, bx, by) in blocks:
        m = (ci >= i0) & (ci < i0 + bx) & (cj >= j0) & (cj < j0 + by) & (st["n"] > 0)
        sel = torch.nonzero(m).flatten()
        o = oracle.Oracle(**dict(w.init, nx=bx, ny=by))
        o.set_threads(os.cpu_count() or 4)
        sl = (slice(i0, i0 + bx), slice(j0, j0 + by))
        c1, c2, c3 = w.courants
        o.set_fields(th=np_(th[sl]).ravel(), rv=np_(rv[sl]).ravel(), rhod=np_(w.rhod[sl]).ravel(),
                     cx=np_(c1[i0:i0 + bx + 1, j0:j0 + by]).ravel(), cy=np_(c2[i0:i0 + bx, j0:j0 + by + 1]).ravel(),
                     cz=np_(c3[sl]).ravel())
        o.set_state(np_(st["n"][sel]).astype(np.uint64), np_(st["rw2"][sel]), np_(st["rd3"][sel]), np_(st["kappa"][sel]),
                    x=np_(st["x"][sel] - i0 * dx), y=np_(st["y"][sel] - j0 * dx), z=np_(st["z"][sel]),
                    id=np_(st["id"][sel]).astype(np.uint32))
        o.set_step(3)
        oracles.append(o)
        picks.append(st["id"][sel].long())
        assert sel.numel() > 0.8 * 64 * bx * by * nz
    assert picks[0].numel() > 1000000
    del st, ci, cj, m, sel

    def compare(g, r, keep, i0, j0, bx, by):
        """r: oracle state sorted by id; keep: mask over it; g: exported device state (dict of CUDA tensors)."""
        where = torch.full((n_total,), -1, dtype=torch.int64, device="cuda")
        where[g["id"].long()] = torch.arange(g["id"].numel(), device="cuda")
        ids = torch.from_numpy(r["id"][keep].astype(np.int64)).cuda()
        pos = where[ids]
        assert bool((pos >= 0).all())
        gg = {k: np_(v[pos]) for k, v in g.items()}
        rr = {k: v[keep] for k, v in r.items()}
        np.testing.assert_array_equal(gg["n"].astype(np.uint64), rr["n"])          # multiplicities: bit-exact
        np.testing.assert_allclose(np.sqrt(gg["rw2"]), np.sqrt(rr["rw2"]), rtol=RTOL)
        np.testing.assert_allclose(np.cbrt(gg["rd3"]), np.cbrt(rr["rd3"]), rtol=RTOL)
        np.testing.assert_allclose(gg["kappa"], rr["kappa"], rtol=RTOL)
        live = rr["n"] > 0
        np.testing.assert_allclose(gg["z"][live], rr["z"][live], rtol=RTOL, atol=1e-9)
        for k, o0, L, big in (("x", i0 * dx, bx * dx, nx * dx), ("y", j0 * dx, by * dx, ny * dx)):
            d = np.mod(gg[k][live] - o0, big)            # the block may sit across the periodic border of the domain
            d = np.mod(d - rr[k][live] + 0.5 * L, L) - 0.5 * L
            assert np.max(np.abs(d)) < 1e-8
        return int(keep.sum())

    th_before = th.clone()
    p.step_sync(po, th, rv)
    p.step_async(po)
    g = p.export_state()
    ncoll = 0
    interior = None
    for (i0, j0, bx, by), o in zip(blocks, oracles):
        o.step(oo)
        r = sorted_by_id(o.get_state())
        n_cmp = compare(g, r, np.ones(r["id"].shape, dtype=bool), i0, j0, bx, by)
        assert n_cmp > 0.8 * 64 * bx * by * nz
        oth, orv = o.get_fields()
        sl = (slice(i0, i0 + bx), slice(j0, j0 + by))
        np.testing.assert_allclose(np_(th[sl]).ravel(), oth, rtol=RTOL)
        np.testing.assert_allclose(np_(rv[sl]).ravel(), orv, rtol=RTOL)
        assert not np.array_equal(np_(th_before[sl]).ravel(), oth)                 # condensation did act
        ncoll += o.counters()["collisions"]
        if bx >= 4:   # SDs that start the second step in an interior column of the block
            oi = np.clip(np.floor(r["x"] / dx).astype(np.int64), 0, bx - 1)
            oj = np.clip(np.floor(r["y"] / dx).astype(np.int64), 0, by - 1)
            interior = (r["n"] > 0) & (oi >= 1) & (oi <= bx - 2) & (oj >= 1) & (oj <= by - 2)
            interior_ids = r["id"][interior]
    assert g["id"].numel() <= N0
    del g
    # second compared step: the interior of the large block
    (i0, j0, bx, by), o = blocks[0], oracles[0]
    p.step_sync(po, th, rv)
    p.step_async(po)
    g = p.export_state()
    o.step(oo)
    r = sorted_by_id(o.get_state())
    keep = np.isin(r["id"], interior_ids)
    assert keep.sum() == interior_ids.size > 0.7 * 64 * bx * by * nz
    compare(g, r, keep, i0, j0, bx, by)
    oth, orv = o.get_fields()
    sl = (slice(i0 + 1, i0 + bx - 1), slice(j0 + 1, j0 + by - 1))
    np.testing.assert_allclose(np_(th[sl]), oth.reshape(bx, by, nz)[1:-1, 1:-1], rtol=RTOL)
    np.testing.assert_allclose(np_(rv[sl]), orv.reshape(bx, by, nz)[1:-1, 1:-1], rtol=RTOL)


# ------------------------------------------------------------------------------------ init() (section 5.1.6)
VOCALS = [(0.61, 60e6, 0.02e-6, 1.4), (0.61, 40e6, 0.075e-6, 1.6)]


@pytest.mark.parametrize("case", ["2d", "3d_subdomain", "mixture"])
def test_device_init_matches_oracle_init(case):
    """sdm_init vs the oracle's init on the same fields, seed and modes: ids, positions (hence cells) bit-equal,
    dry and wet radii within 1e-9, the range of :657 equal.  Multiplicities are floor(x + 1/2) of a product that
    contains exp() of the two maths libraries (1 ulp apart at worst): they must agree exactly for all but a
    1e-4 fraction of the SDs, and there differ by 1."""
    b = binding()
    if case == "2d":
        w, modes, ext = W.cfg2_2d(sd_per_cell=32, nx=12, nz=75, seed=21), VOCALS, {}
    elif case == "3d_subdomain":
        w, modes = W.cfg4_3d(sd_per_cell=16, nx=6, ny=5, nz=64, seed=22), VOCALS
        ext = dict(x0=20.0, x1=100.0, y0=0.0, y1=60.0, z0=200.0, z1=1280.0)
    else:
        w, modes, ext = W.cfg2_2d(sd_per_cell=64, nx=8, nz=75, seed=23), [(0.61, 60e6, 0.02e-6, 1.4), (1.28, 40e6, 0.075e-6, 1.6)], {}
    sd = w.meta["sd_per_cell"]
    o = make_oracle(w)
    N, ranges = o.init(modes, float(sd), **ext)
    p = b.Particles(max_sd=N + 7, sd_conc_mean=float(sd), modes=modes, **dict(w.init, **ext))
    cs = [c.cuda() for c in w.courants] + [None] * (3 - len(w.courants))
    th, rv = w.th.cuda(), w.rv.cuda()
    p.init(th, rv, w.rhod.cuda(), *cs)
    assert p.n_sd() == N
    for g, (lo, hi) in enumerate(ranges):
        np.testing.assert_allclose(p.init_range(g), (lo, hi), rtol=0, atol=1e-12)
    gs, rs = sorted_by_id(p.export_state()), sorted_by_id(o.get_state())
    np.testing.assert_array_equal(gs["id"].astype(np.uint32), rs["id"])
    for k, present in zip("xyz", p.dims):
        if present:
            np.testing.assert_array_equal(gs[k], rs[k])
    np.testing.assert_array_equal(gs["kappa"], rs["kappa"])
    np.testing.assert_allclose(np.cbrt(gs["rd3"]), np.cbrt(rs["rd3"]), rtol=RTOL)
    np.testing.assert_allclose(np.sqrt(gs["rw2"]), np.sqrt(rs["rw2"]), rtol=RTOL)
    dn = gs["n"].astype(np.int64) - rs["n"].astype(np.int64)
    assert np.abs(dn).max() <= 1 and np.count_nonzero(dn) <= 1e-4 * N + 1
    # th, rv untouched (:663); the initialised population steps like a loaded one
    np.testing.assert_array_equal(np_(th), np_(w.th))
    agree = dn == 0
    if agree.all():
        po, oo = b.make_opts(**w.opts), oracle.make_opts(**w.opts)
        o.step(oo)
        p.step_sync(po, th, rv)
        p.step_async(po)
        compare_states(p, o)
        compare_fields(th, rv, o)


def test_device_init_errors():
    b = binding()
    w = W.cfg2_2d(sd_per_cell=8, nx=4, nz=4, seed=1)
    p = b.Particles(max_sd=1000, sd_conc_mean=8.0, **w.init)                      # no modes
    with pytest.raises(b.SdmError, match="without dry-aerosol modes"):
        p.init(w.th.cuda(), w.rv.cuda(), w.rhod.cuda())
    p = b.Particles(max_sd=100, sd_conc_mean=8.0, modes=VOCALS, **w.init)        # 128 SDs do not fit
    with pytest.raises(b.SdmError, match="exceeds max_sd"):
        p.init(w.th.cuda(), w.rv.cuda(), w.rhod.cuda())
    with pytest.raises(b.SdmError, match="too dilute"):
        b.Particles(max_sd=100, sd_conc_mean=8.0, modes=[(0.61, 1e-3, 0.02e-6, 1.4)], **w.init)
    with pytest.raises(b.SdmError, match="inside the grid"):
        b.Particles(max_sd=100, sd_conc_mean=8.0, modes=VOCALS, **dict(w.init, x1=1e6))


# ------------------------------------------------------------------------------------ which root of eq. 17
def test_first_step_in_supersaturated_air_takes_the_bisection_root():
    """The initial haze (equilibrium at RH <= 0.95) under RH_max = 1.05 is far from equilibrium: eq. 17 then has
    several roots inside the bracket of eq. 18-19, or two (the ill-posed case of :579).  The paper's bisection
    defines which one is meant; the Newton path must certify a single root or defer to that procedure."""
    w = W.cfg2_2d(sd_per_cell=24, nx=6, nz=75, seed=21)     # full height: cells from RH 0.66 to the 1.05 cap
    p, o, th, rv = run_both(w, 2)
    sp, so = p.stats(), o.counters()
    assert sp["ill_posed"] == so["ill_posed"] > 100


def test_root_selection_scan_of_independent_sds():
    """Sizes from barely wet to 3000 r_d, r_d from 1 nm to 2 um, kappa 0.05-1.55, RH 0.3-1.05, multiplicity 1 (no
    feedback: every SD-substep is an independent instance of eq. 17-19): radii and ill-posed counts must match."""
    seed, nx, nz, sd = 7, 24, 24, 64
    w = W.cfg2_2d(sd_per_cell=sd, nx=nx, nz=nz, seed=seed)
    idx = torch.arange(w.n_sd, dtype=torch.int64)
    u1, u2, u3 = (W.hash_uniform(seed, 200 + k, idx) for k in range(3))
    rd = torch.exp(np.log(1e-9) + u1 * (np.log(2e-6) - np.log(1e-9)))
    w.state["rd3"] = rd ** 3
    w.state["rw2"] = (rd * torch.exp(1e-4 + u2 * u2 * np.log(3e3))) ** 2
    w.state["kappa"] = torch.where(u3 < 0.5, torch.full_like(u3, 0.61), 0.05 + 1.5 * u3)
    w.state["n"] = torch.ones_like(w.state["n"])
    ci = torch.arange(nx, dtype=torch.float64)[:, None].expand(nx, nz)
    w.rv = w.rv * (0.35 + 0.95 * ci / (nx - 1))
    p, o, th, rv = run_both(w, 2, opts=dict(coal=False, adve=False, sedi=False))
    sp, so = p.stats(), o.counters()
    assert sp["ill_posed"] == so["ill_posed"] > 50
    assert sp["cond_slow"] > 0.02 * sp["sd_substeps"]       # the literal-bisection path was exercised


# ------------------------------------------------------------------------------------ fp32 particle state
def _fp32_case(w, steps=1, recycle=False, arith=8, **opts):
    """Single-step parity with real_bytes = 4 (north_star: 1e-4 on radii in fp32): the state is rounded to fp32
    first, the oracle starts from exactly those values in fp64, and before every further step the oracle is
    re-loaded with the device's (fp32) state, so that each step is compared on its own."""
    b = binding()
    st32 = {k: (v if v is None or k in ("n", "id") else v.to(torch.float32)) for k, v in w.state.items()}
    w.state = {k: (v if v is None or k in ("n", "id") else v.to(torch.float64)) for k, v in st32.items()}
    o = make_oracle(w, threads=4)
    p = b.Particles(max_sd=w.n_sd, sd_conc_mean=w.meta["sd_per_cell"], real_bytes=4, **w.init)
    cs = [c.cuda() for c in w.courants] + [None] * (3 - len(w.courants))
    g = {k: (None if v is None else v.cuda()) for k, v in st32.items()}
    p.init_from_arrays(w.rhod.cuda(), g["n"], g["rw2"], g["rd3"], g["kappa"], g["x"], g["y"], g["z"], g["id"],
                       courant_1=cs[0], courant_2=cs[1], courant_3=cs[2])
    th, rv = w.th.cuda().clone(), w.rv.cuda().clone()
    if recycle:
        o.set_recycle(True)
        p.set_recycle(True)
    p.set_cond_arith(arith)
    kw = dict(w.opts)
    kw.update(opts)
    po, oo = b.make_opts(**kw), oracle.make_opts(**kw)
    for s in range(steps):
        fo = o.step(oo)
        p.step_sync(po, th, rv)
        p.step_async(po)
        fp = p.step_async_result()
        ex = p.export_state()
        assert ex["rw2"].dtype == torch.float32 and ex["x"].dtype == torch.float32
        gs, rs = sorted_by_id(ex), sorted_by_id(o.get_state())
        np.testing.assert_array_equal(gs["id"].astype(np.uint32), rs["id"])
        np.testing.assert_array_equal(gs["n"].astype(np.uint64), rs["n"])             # multiplicities: bit-exact
        np.testing.assert_allclose(np.sqrt(gs["rw2"].astype(np.float64)), np.sqrt(rs["rw2"]), rtol=1e-4)
        np.testing.assert_allclose(np.cbrt(gs["rd3"].astype(np.float64)), np.cbrt(rs["rd3"]), rtol=1e-4)
        np.testing.assert_allclose(gs["kappa"], rs["kappa"], rtol=1e-4)
        live = rs["n"] > 0
        for k, present in zip("xyz", p.dims):
            if present:   # fp32 positions: half an ulp of the domain size
                np.testing.assert_allclose(gs[k][live], rs[k][live], rtol=1e-6, atol=1e-6 * 3000.0)
        oth, orv = o.get_fields()
        np.testing.assert_allclose(np_(th).ravel(), oth, rtol=1e-6)
        np.testing.assert_allclose(np_(rv).ravel(), orv, rtol=1e-6)
        np.testing.assert_allclose(fp, fo, rtol=3e-4, atol=1e-300)
        assert p.stats()["collisions"] == o.counters()["collisions"]
        # next step from the device's rounded state
        o.set_state(gs["n"].astype(np.uint64), gs["rw2"].astype(np.float64), gs["rd3"].astype(np.float64),
                    gs["kappa"].astype(np.float64), x=gs["x"].astype(np.float64), y=gs["y"].astype(np.float64),
                    z=gs["z"].astype(np.float64), id=gs["id"].astype(np.uint32))
        o.set_fields(th=np_(th).ravel(), rv=np_(rv).ravel())
    return p, o


def test_fp32_state_2d_and_3d():
    p, o = _fp32_case(rain_mix(W.cfg2_2d(sd_per_cell=32, nx=10, nz=40, seed=31)), steps=3)
    assert o.counters()["collisions"] > 0
    _fp32_case(rain_mix(W.cfg4_3d(sd_per_cell=64, nx=4, ny=3, nz=32, seed=32)), steps=2)


def test_fp32_state_fallback_kernels():
    """fp32 storage through the per-cell kernels: coalescence substeps (k_coal_move<G>), ~1000 SDs per cell (medium
    condensation tile, bucket ranks) and one crowded cell (in-place condensation and coalescence)."""
    _fp32_case(rain_mix(W.cfg2_2d(sd_per_cell=40, nx=6, nz=8, seed=33), frac=0.5), steps=2, sstp_coal=3)
    _fp32_case(rain_mix(W.cfg2_2d(sd_per_cell=1000, nx=2, nz=3, seed=34), frac=0.3), steps=1, sstp_cond=3)
    w = rain_mix(W.cfg2_2d(sd_per_cell=1500, nx=2, nz=3, seed=35), frac=0.3)
    w.state["x"] = w.state["x"] * 0.4
    _fp32_case(w, steps=1, sstp_cond=2)


def test_fp32_init_and_diagnostics():
    b = binding()
    w = W.cfg2_2d(sd_per_cell=32, nx=8, nz=30, seed=36)
    p = b.Particles(max_sd=w.n_sd + 8, sd_conc_mean=32.0, modes=VOCALS, real_bytes=4, **w.init)
    p64 = b.Particles(max_sd=w.n_sd + 8, sd_conc_mean=32.0, modes=VOCALS, **w.init)
    cs = [c.cuda() for c in w.courants]
    for q in (p, p64):
        q.init(w.th.cuda(), w.rv.cuda(), w.rhod.cuda(), *cs)
    a, r = sorted_by_id(p.export_state()), sorted_by_id(p64.export_state())
    np.testing.assert_array_equal(a["n"], r["n"])
    for k in ("rw2", "rd3", "x", "z"):
        np.testing.assert_allclose(a[k], r[k], rtol=2e-7)
    p.diag_wet_rng(0.0, 1.0)
    p64.diag_wet_rng(0.0, 1.0)
    np.testing.assert_allclose(np_(p.diag_wet_mom(3)), np_(p64.diag_wet_mom(3)), rtol=1e-5)
    with pytest.raises(b.SdmError, match="float32"):
        p.init_from_arrays(w.rhod.cuda(), w.state["n"].cuda(), w.state["rw2"].cuda(), w.state["rd3"].cuda(), w.state["kappa"].cuda(),
                           w.state["x"].cuda(), None, w.state["z"].cuda())


# ----------------------------------------------------------------------------------------------- recycling
def test_recycling_box_golovin_keeps_every_sd_and_matches_the_oracle():
    """PAPER.md :641: SDs left with zero multiplicity by equal-multiplicity collisions are recycled at the beginning of
    the next step.  configs[0] starts with equal multiplicities everywhere, so ties (order by id) and halving of odd
    multiplicities are exercised from the first steps on."""
    w = W.box_golovin(seed=43)
    p, o, _, _ = run_both(w, 500, check_every=50, recycle=True)
    assert p.n_sd() == o.n_sd() == w.n_sd
    assert p.stats()["recycled"] == o.recycled > 500
    sp, so = p.stats(), o.counters()
    assert sp["pairs"] == so["pairs"] and sp["collisions"] == so["collisions"]


def test_recycling_of_sds_that_left_the_domain():
    """PAPER.md :651: SDs that sedimented out of the domain 'undergo the same recycling procedure'."""
    w = rain_mix(W.cfg2_2d(nx=12, nz=12, sd_per_cell=40, seed=9), seed=9, frac=0.3)
    p, o, _, _ = run_both(w, 12, recycle=True)
    assert p.stats()["recycled"] == o.recycled > 20
    assert p.n_sd() == o.n_sd() == w.n_sd
    # fp32 state: the same, each step compared on its own from the device's rounded state
    w = rain_mix(W.cfg2_2d(nx=12, nz=12, sd_per_cell=40, seed=10), seed=10, frac=0.3)
    p, o = _fp32_case(w, steps=8, recycle=True)
    assert p.stats()["recycled"] == o.recycled > 10


@pytest.mark.parametrize("spc,n_dead,distinct", [(34, 9000, 1), (34, 200, 7), (6, 4000, 3), (78, 1, 1000000), (1, 600, 2)])
def test_recycling_selection_with_ties_across_sort_tiles(spc, n_dead, distinct):
    """The donors are exactly the oracle's: many equal multiplicities (order by id decides), candidate lists longer than
    one shared-memory sort tile (global bitonic steps), fewer donors than dead SDs, multiplicity 1 never halved."""
    w = W.cfg2_2d(nx=30, nz=30, sd_per_cell=spc, seed=7)
    n_sd = w.n_sd
    idx = torch.arange(n_sd, dtype=torch.int64)
    u = W.hash_uniform(3, 11, idx)
    n = (1 if distinct > 1 else 6) + (W.hash_uniform(3, 12, idx) * distinct).to(torch.int64)   # ties; N = 1 cannot give
    w.state["n"] = torch.where(u < n_dead / n_sd, torch.zeros_like(n), n)
    w.state["id"] = torch.randperm(n_sd, generator=torch.Generator().manual_seed(1)).to(torch.int32)
    p, o, _, _ = run_both(w, 1, opts=dict(coal=False, cond=False, adve=False, sedi=False), recycle=True)
    assert p.stats()["recycled"] == o.recycled > 0
    assert p.n_sd() == o.n_sd()


@pytest.mark.parametrize("recycle", [False, True])
def test_box_golovin_full_length_16_seeds_against_the_closed_form(recycle):
    """configs[0] at full length on the CUDA path: 16 seeds x 3600 steps; the zeroth moment follows
    M0 = n0 exp(-b n0 v0 t) (Golovin 1963) within the sampling error of the pooled seeds, the first moment is
    constant.  With compaction only ~40 SDs are left at 3600 s; with the paper's recycling all 2^13 stay and the
    late-time tolerance is that of the oracle's pin (tests/test_oracle_pins.py)."""
    b = binding()
    times = (1200, 2400, 3600)
    M0 = {t: [] for t in times}
    for seed in range(42, 58):
        w = W.box_golovin(seed=seed)
        p, th, rv = make_particles(w)
        if recycle:
            p.set_recycle(True)
        po = b.make_opts(**w.opts)
        m_ini = float((w.state["n"].double() * w.state["rw2"] ** 1.5).sum())
        for t in range(1, 3601):
            p.step_sync(po, th, rv)
            p.step_async(po)
            if t in times:
                st = p.export_state()
                nn, r3 = st["n"].double(), st["rw2"].double() ** 1.5
                np.testing.assert_allclose(float((nn * r3).sum()), m_ini, rtol=1e-12)
                M0[t].append(float(nn.sum()) / w.meta["V"])
        assert (p.n_sd() == w.n_sd) if recycle else (p.n_sd() < 200)
    n0, v0, bb = w.meta["n0"], w.meta["v0"], w.meta["b"]
    tol = {1200: 0.05, 2400: 0.08, 3600: 0.12} if recycle else {1200: 0.06, 2400: 0.12, 3600: 0.35}
    for t in times:
        ratio = np.mean(M0[t]) / (n0 * np.exp(-bb * n0 * v0 * t))
        assert abs(ratio - 1) < tol[t], (t, ratio)


# ----------------------------------------------------------------------------------------------- fp32 arithmetic
def test_fp32_arithmetic_condensation_2d_3d_and_first_step():
    """sdm_set_cond_arith(4): the condensation sweep in single precision (real_t = float, PAPER.md :747).  north_star:
    radii within 1e-4 of the fp64 oracle started from the same fp32 state, multiplicities and collisions bit-exact."""
    p, o = _fp32_case(rain_mix(W.cfg2_2d(sd_per_cell=32, nx=10, nz=75, seed=41)), steps=4, arith=4)
    assert o.counters()["collisions"] > 0
    _fp32_case(rain_mix(W.cfg4_3d(sd_per_cell=64, nx=4, ny=3, nz=64, seed=42)), steps=3, arith=4)
    # haze only, from the initial condition at full height: the first step under RH_max = 1.05 (multi-root brackets)
    _fp32_case(W.cfg2_2d(sd_per_cell=64, nx=4, nz=75, seed=43), steps=3, arith=4)
    # sparse cells (8 SDs per cell: many cells per tile, the flat staging loop) and cells of ~1000 SDs (medium tile)
    _fp32_case(rain_mix(W.cfg2_2d(sd_per_cell=8, nx=16, nz=40, seed=45)), steps=3, arith=4)
    _fp32_case(rain_mix(W.cfg2_2d(sd_per_cell=1000, nx=2, nz=3, seed=44), frac=0.3), steps=2, sstp_cond=3, arith=4)
    # one crowded cell (beyond every tile kernel): solved in fp64 in place
    w = rain_mix(W.cfg2_2d(sd_per_cell=1500, nx=2, nz=3, seed=46), frac=0.3)
    w.state["x"] = w.state["x"] * 0.4
    _fp32_case(w, steps=1, sstp_cond=2, arith=4)
    with pytest.raises(Exception):
        make_particles(W.cfg2_2d(sd_per_cell=8, nx=2, nz=2, seed=1))[0].set_cond_arith(4)   # fp64 state: refused


def test_measured_fp64_peak_and_n_live():
    """sdm_measure_fp64_peak (the denominator of the condensation roofline): a B200 retires 64 fp64 FMAs per clock
    per SM; the measurement must land within a few per cent of that and of 148 x 64 x 2 x clock.  sdm_n_live = sdm_n_sd."""
    b = binding()
    tflops, per_clk = b.measure_fp64_peak()
    assert 58.0 < per_clk <= 64.5, per_clk
    assert 15.0 < tflops < 40.0, tflops   # 36.6 at 1965 MHz; a power-capped clock lowers it
    p, th, rv = make_particles(W.cfg2_2d(sd_per_cell=8, nx=4, nz=4, seed=3))
    assert p.n_live() == p.n_sd() == 128


# ----------------------------------------------------------------------------------------------- adaptive substeps
def test_adaptive_condensation_substeps_match_the_oracle():
    """sdm_opts.cond_adapt_tol > 0 (reading R-adapt; PAPER.md :566 "planned"): every cell takes the number of
    substeps the oracle's rule gives it - the totals of SD-substeps are equal, far below the fixed count - and ends where
    the oracle ends it, to the usual bars.  Full-height 2D column set (haze below, cloud base, supersaturated top), a 3D
    case, the fp32 state with fp64 arithmetic, cells of ~1000 SDs (medium tile) and one crowded cell (in-place kernel)."""
    b = binding()
    w = rain_mix(W.cfg2_2d(sd_per_cell=32, nx=10, nz=75, seed=71))
    for tol in (0.5, 0.05):
        p, o, th, rv = run_both(w, 6, opts=dict(cond_adapt_tol=tol))
        sp, so = p.stats(), o.counters()
        assert sp["sd_substeps"] == so["sd_substeps"] and sp["ill_posed"] == so["ill_posed"]
        assert sp["collisions"] == so["collisions"]
        assert so["sd_substeps"] < 0.8 * 10 * 6 * w.n_sd
    fixed = 10 * 6 * w.n_sd
    assert so["sd_substeps"] > 0.15 * fixed        # the cloudy cells keep (most of) their substeps at the tighter tolerance
    p, o, _, _ = run_both(rain_mix(W.cfg4_3d(sd_per_cell=64, nx=5, ny=4, nz=64, seed=72)), 3, opts=dict(cond_adapt_tol=0.2))
    assert p.stats()["sd_substeps"] == o.counters()["sd_substeps"]
    p, o, _, _ = run_both(rain_mix(W.cfg2_2d(sd_per_cell=1000, nx=2, nz=3, seed=73), frac=0.3), 2, opts=dict(sstp_cond=6, cond_adapt_tol=0.2))
    assert p.stats()["sd_substeps"] == o.counters()["sd_substeps"] and p.stats()["cond_variant"] == 2
    wc = rain_mix(W.cfg2_2d(sd_per_cell=1500, nx=2, nz=3, seed=74), frac=0.3)
    wc.state["x"] = wc.state["x"] * 0.4
    p, o, _, _ = run_both(wc, 2, group=32, opts=dict(sstp_cond=4, cond_adapt_tol=0.2))
    assert p.stats()["sd_substeps"] == o.counters()["sd_substeps"] and p.stats()["cond_variant"] == 3
    wc = rain_mix(W.cfg2_2d(sd_per_cell=1500, nx=2, nz=2, seed=76), frac=0.3)
    wc.state["x"] = wc.state["x"] * 0.499
    wc.state["z"] = wc.state["z"] * 0.499          # ~6000 SDs in one cell: beyond every tile kernel
    p, o, _, _ = run_both(wc, 2, opts=dict(sstp_cond=4, cond_adapt_tol=0.2))
    assert p.stats()["sd_substeps"] == o.counters()["sd_substeps"] and p.stats()["cond_variant"] == 0
    p, o = _fp32_case(rain_mix(W.cfg2_2d(sd_per_cell=32, nx=6, nz=75, seed=75)), steps=2, cond_adapt_tol=0.3)
    assert p.stats()["sd_substeps"] == o.counters()["sd_substeps"]
    w4 = W.cfg2_2d(sd_per_cell=8, nx=2, nz=2, seed=1)
    w4.state = {k: (v if v is None or k in ("n", "id") else v.to(torch.float32)) for k, v in w4.state.items()}
    q, th, rv = make_particles(w4, real_bytes=4)
    q.set_cond_arith(4)
    with pytest.raises(b.SdmError, match="cond_adapt_tol"):
        q.step_sync(b.make_opts(cond_adapt_tol=0.1, RH_max=1.05), th, rv)


def test_adaptive_coalescence_substeps_match_the_oracle():
    """sdm_opts.coal_adapt_max > 1 (reading R-adapt-coal; PAPER.md :645 "planned"): cells whose first grouping has
    a pair with P > 1 take more substeps, each with new random pairs.  The Golovin box of configs[0] (P reaches 25 there), with
    and without multiple coalescence, and a 2D rain case in a small volume; pairs examined, collisions and multiplicities as the
    oracle's, and more pairs examined than the fixed step examines."""
    w = W.box_golovin(seed=44)
    for multi in (True, False):
        # the box shrunk to 40^3 m^3: 15.6 times the collision probabilities of configs[0], P above 1 from the start
        p, o, _, _ = run_both(w, 60, check_every=20, opts=dict(coal_adapt_max=8), multi_coal=multi, dx=40.0, dy=40.0, dz=40.0)
        sp, so = p.stats(), o.counters()
        assert sp["pairs"] == so["pairs"] and sp["collisions"] == so["collisions"] and sp["near_ties"] == so["near_ties"]
        assert so["pairs"] > 1.5 * 60 * (p.n_sd() // 2)           # several groupings per step
        assert p.n_sd() == o.n_sd()
    w2 = rain_mix(W.cfg2_2d(sd_per_cell=40, nx=6, nz=8, seed=93), frac=0.6)
    w2.state["n"] = w2.state["n"] * 2000                           # crowded with real drops: P of the rain pairs exceeds 1
    for group in (0, 256):
        p, o, _, _ = run_both(w2, 3, group=group, opts=dict(coal_adapt_max=4, sstp_coal=2, cond=False))
        sp, so = p.stats(), o.counters()
        assert sp["pairs"] == so["pairs"] and sp["collisions"] == so["collisions"] > 100
        assert so["pairs"] > 3 * 2 * (w2.n_sd // 2) * 0.9 * 1.05  # some cells took more than sstp_coal groupings
    assert p.stats()["coal_tile_cells"] == 0                       # the per-cell kernel ran


# ----------------------------------------------------------------------------------------------- sync / async
def test_upstream_advect_matches_the_oracle_bit_for_bit():
    """sdm_upstream_advect, the prototype transport solver of PAPER.md Figure 7 (:831-852; upstream scheme :219-235): the same
    IEEE operations in the same order as the oracle's restatement, so the fields are equal to the bit - 2D and 3D, dense
    and halo-padded (strided) fields, five steps in a row."""
    for w in (W.cfg2_2d(sd_per_cell=4, nx=23, nz=17, seed=81), W.cfg4_3d(sd_per_cell=2, nx=9, ny=7, nz=11, seed=82)):
        o = make_oracle(w)
        p, th, rv = make_particles(w)
        shape = tuple(th.shape)
        pad = torch.zeros(tuple(n + 4 for n in shape), dtype=torch.float64, device="cuda")
        view = pad[tuple(slice(2, 2 + n) for n in shape)]
        view.copy_(th + 0.01 * torch.rand(shape, dtype=torch.float64, device="cuda"))
        dense = view.clone()
        ref = np_(dense).ravel()
        for _ in range(5):
            p.upstream_advect(dense)
            p.upstream_advect(view)       # non-contiguous: strides of the padded array
            ref = o.upstream_advect(ref)
        np.testing.assert_array_equal(np_(dense).ravel(), ref)
        np.testing.assert_array_equal(np_(view.contiguous()).ravel(), ref)
        assert float(pad.sum()) == pytest.approx(float(view.sum()))   # the halo was not touched
        assert np.abs(ref - np_(th).ravel()).max() > 1e-4


def test_step_async_overlaps_an_eulerian_solver_on_another_stream():
    """PAPER.md :816 and Figure 7 (:833-848): step_sync returns th, rv for the host model, step_async (coalescence +
    movement, which touch neither) runs while the Eulerian solver advances th, rv.  The solver is the library's upstream
    step (sdm_upstream_advect, Fig. 7's "prototype transport equation solver") on a second stream, ordered after
    step_sync by an event.  Checked: step_async returns to the host before its device work is done, the overlapped run
    equals the serialised one bit for bit, and it matches the oracle driven through the same calling sequence."""
    b = binding()
    w = W.cfg4_3d(sd_per_cell=64, nx=48, ny=48, nz=64, seed=61, device="cuda")

    def run(overlap):
        p, th, rv = make_particles(w)
        po = b.make_opts(**w.opts)
        s1, s2 = torch.cuda.Stream(), torch.cuda.Stream()
        returned_early = 0
        torch.cuda.synchronize()
        for _ in range(3):
            with torch.cuda.stream(s1):
                p.step_sync(po, th, rv)
                ready = torch.cuda.Event()
                ready.record(s1)
                p.step_async(po)
                done = torch.cuda.Event()
                done.record(s1)
                returned_early += int(not done.query())
            if not overlap:
                s1.synchronize()
            with torch.cuda.stream(s2):
                s2.wait_event(ready)
                p.upstream_advect(th)
                p.upstream_advect(rv)
            s1.wait_stream(s2)   # the next step_sync reads the solver's th, rv
            with torch.cuda.stream(s1):
                p.step_async_result()
        torch.cuda.synchronize()
        return sorted_by_id(p.export_state()), th.clone(), rv.clone(), returned_early

    a, th_a, rv_a, early = run(overlap=True)
    s, th_s, rv_s, _ = run(overlap=False)
    assert early >= 2   # the host got control back while coalescence + movement were still running
    for k in a:
        np.testing.assert_array_equal(a[k], s[k])
    assert torch.equal(th_a, th_s) and torch.equal(rv_a, rv_s)
    # the oracle driven in the same order, on a sub-domain it finishes in seconds
    wo = W.cfg4_3d(sd_per_cell=64, nx=4, ny=4, nz=64, seed=62)
    o = make_oracle(wo, threads=4)
    p, th, rv = make_particles(wo)
    po, oo = b.make_opts(**wo.opts), oracle.make_opts(**wo.opts)
    for _ in range(3):
        p.step_sync(po, th, rv)
        o.step_sync(oo)
        p.step_async(po)
        o.step_async(oo)
        p.upstream_advect(th)
        p.upstream_advect(rv)
        oth, orv = o.get_fields()
        o.set_fields(th=o.upstream_advect(oth), rv=o.upstream_advect(orv))
    compare_states(p, o)
    compare_fields(th, rv, o)


# ----------------------------------------------------------------------------------------------- slabs along x
@pytest.mark.parametrize("dims", ["2d", "3d"])
def test_three_slabs_on_one_gpu_match_the_oracle_on_the_whole_domain(dims):
    """the domain split into slabs of columns, one open_x context each (here all on one GPU, the
    periodic neighbour of the last being the first), SDs that crossed a face handed over after every step
    (sdm_pack_leavers / sdm_unpack_arrivals, slab.exchange_local).  Every other stage is local to a cell and the Philox
    streams are keyed by the SD id, which travels with the SD: the union of the slabs must follow the oracle's
    run on the whole periodic domain - multiplicities bit-exact, radii and fields to 1e-9, positions (in global
    coordinates) to 1e-9 of the domain.  Unequal slab widths, rain mix, 8 steps; SDs do change slabs in both directions."""
    from paper_1310_1905_b200 import slab

    b = binding()
    if dims == "2d":
        w = rain_mix(W.cfg2_2d(sd_per_cell=24, nx=13, nz=20, seed=91))
        w.courants = [c * 6.0 for c in w.courants]          # a brisk flow: Courant numbers up to ~0.4, many crossings
    else:
        w = rain_mix(W.cfg4_3d(sd_per_cell=16, nx=7, ny=4, nz=16, seed=92))
        w.courants = [c * 4.0 for c in w.courants]
    nx, dx = w.init["nx"], w.init["dx"]
    cols = slab.split_columns(nx, 3)
    widths = [n * dx for _, n in cols]
    o = make_oracle(w, threads=4)
    xs = w.state["x"]
    parts, fields, n_moved = [], [], 0
    for (i0, n) in cols:
        m = (xs >= i0 * dx) & (xs < (i0 + n) * dx)
        st = {k: (None if v is None else v[m].cuda()) for k, v in w.state.items()}
        st["x"] = st["x"] - i0 * dx
        p = b.Particles(max_sd=w.n_sd, sd_conc_mean=w.meta["sd_per_cell"], open_x=True, **dict(w.init, nx=n))
        c = [cc.cuda() for cc in w.courants]
        c[0] = c[0][i0:i0 + n + 1].contiguous()
        c[1:] = [cc[i0:i0 + n].contiguous() for cc in c[1:]]
        c += [None] * (3 - len(c))
        p.init_from_arrays(w.rhod[i0:i0 + n].contiguous().cuda(), st["n"], st["rw2"], st["rd3"], st["kappa"], st["x"], st["y"], st["z"], st["id"],
                           courant_1=c[0], courant_2=c[1], courant_3=c[2])
        parts.append(p)
        fields.append((w.th[i0:i0 + n].contiguous().cuda().clone(), w.rv[i0:i0 + n].contiguous().cuda().clone()))
    po, oo = b.make_opts(**w.opts), oracle.make_opts(**w.opts)
    for step in range(8):
        fo = o.step(oo)
        flux = 0.0
        for p, (th, rv) in zip(parts, fields):
            p.step_sync(po, th, rv)
            p.step_async(po)
            flux += p.step_async_result()
        n_moved += sum(l + r for l, r in slab.exchange_local(parts, widths, cap=4096))
        np.testing.assert_allclose(flux, fo, rtol=1e-8, atol=1e-300)
        # the union of the slabs in global coordinates against the oracle
        g = {k: [] for k in ("n", "rw2", "rd3", "kappa", "x", "y", "z", "id")}
        for (i0, n), p in zip(cols, parts):
            ex = p.export_state()
            ex["x"] = ex["x"] + i0 * dx
            for k in g:
                g[k].append(ex[k])
        g = sorted_by_id({k: torch.cat(v) for k, v in g.items()})
        r = sorted_by_id(o.get_state())
        keep = g["n"] != 0                         # a handed-over SD leaves a dead slot behind until the next compaction
        g = {k: v[keep] for k, v in g.items()}
        rk = r["n"] != 0
        np.testing.assert_array_equal(g["id"].astype(np.uint32), r["id"][rk])
        np.testing.assert_array_equal(g["n"].astype(np.uint64), r["n"][rk])
        np.testing.assert_allclose(np.sqrt(g["rw2"]), np.sqrt(r["rw2"][rk]), rtol=RTOL)
        np.testing.assert_allclose(np.cbrt(g["rd3"]), np.cbrt(r["rd3"][rk]), rtol=RTOL)
        X = nx * dx
        d = np.mod(g["x"] - r["x"][rk] + 0.5 * X, X) - 0.5 * X
        assert np.abs(d).max() < 1e-9 * X
        np.testing.assert_allclose(g["z"], r["z"][rk], rtol=RTOL, atol=1e-9)
        if dims == "3d":
            np.testing.assert_allclose(g["y"], r["y"][rk], rtol=RTOL, atol=1e-9)
        oth, orv = o.get_fields()
        th_all = torch.cat([f[0] for f in fields], 0)
        rv_all = torch.cat([f[1] for f in fields], 0)
        np.testing.assert_allclose(np_(th_all).ravel(), oth, rtol=RTOL)
        np.testing.assert_allclose(np_(rv_all).ravel(), orv, rtol=RTOL)
    assert n_moved > 100
    assert sum(p.stats()["collisions"] for p in parts) == o.counters()["collisions"] > 0
    # misuse is refused
    q, th, rv = make_particles(W.cfg2_2d(sd_per_cell=4, nx=3, nz=3, seed=1))
    with pytest.raises(b.SdmError, match="open_x"):
        q.pack_leavers(16)


def test_fp32_arithmetic_root_selection_scan_of_independent_sds():
    """The scan of test_root_selection_scan_of_independent_sds with the fp32 sweep: r_d from 1 nm to 2 um, sizes from
    barely wet to 3000 r_d, kappa 0.05-1.55, RH 0.3-1.05, multiplicity 1 (no feedback).  Whatever the fp32 certificate
    lets through must land on the root the paper's bisection defines, to 1e-4; the rest goes to the fp64 list."""
    seed, nx, nz, sd = 8, 24, 24, 64
    w = W.cfg2_2d(sd_per_cell=sd, nx=nx, nz=nz, seed=seed)
    idx = torch.arange(w.n_sd, dtype=torch.int64)
    u1, u2, u3 = (W.hash_uniform(seed, 200 + k, idx) for k in range(3))
    rd = torch.exp(np.log(1e-9) + u1 * (np.log(2e-6) - np.log(1e-9)))
    w.state["rd3"] = rd ** 3
    w.state["rw2"] = (rd * torch.exp(1e-4 + u2 * u2 * np.log(3e3))) ** 2
    w.state["kappa"] = torch.where(u3 < 0.5, torch.full_like(u3, 0.61), 0.05 + 1.5 * u3)
    w.state["n"] = torch.ones_like(w.state["n"])
    ci = torch.arange(nx, dtype=torch.float64)[:, None].expand(nx, nz)
    w.rv = w.rv * (0.35 + 0.95 * ci / (nx - 1))
    p, o = _fp32_case(w, steps=2, arith=4, coal=False, adve=False, sedi=False)
    sp = p.stats()
    assert sp["cond_slow"] > 0.02 * sp["sd_substeps"]       # the fp64 list was exercised
    assert sp["cond_slow"] < 0.5 * sp["sd_substeps"]        # ... and the fp32 sweep solved most
