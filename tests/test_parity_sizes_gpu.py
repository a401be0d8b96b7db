"""Parity at the sizes and lengths BASELINE.json's configs name ("next round" item 2): configs[1] and
configs[2] on their 75 x 75 grid over a few hundred steps against the OpenMP oracle, the corners of the launch sizing
(one cell of more than 16384 SDs, the spin-up combination of processes, the sstp_cond > 500 fallback of the fp32 sweep).
Same bars as tests/test_parity_gpu.py: multiplicities bit-exact, radii / positions / th / rv within 1e-9, collision,
near-tie and ill-posed counters equal."""
import os

import numpy as np
import pytest
import torch

import oracle
from paper_1310_1905_b200 import workloads as W
from tests.test_parity_gpu import _fp32_case, compare_fields, compare_states, rain_mix, run_both
from tests.util import courant_xyz, make_oracle, make_particles, np_, sorted_by_id

pytestmark = pytest.mark.gpu

THREADS = os.cpu_count() or 4


def _counters_equal(p, o):
    sp, so = p.stats(), o.counters()
    for k in ("pairs", "collisions", "near_ties", "ill_posed", "sd_substeps"):
        assert sp[k] == so[k], (k, sp[k], so[k])
    assert so["near_ties"] <= 1e-6 * so["pairs"] + 1
    return sp, so


DRIFT = (5e-3, 1e-6)   # free-running trajectories: all but 0.5 % of the SDs within 1e-9, every one within 1e-6 (see compare_states)


def _trajectory(w, steps, every):
    """Free-running GPU and oracle trajectories from the same initial state, compared every `every` steps with the
    trajectory bar (multiplicities bit-exact, fields 1e-9, radii per DRIFT), the rain flux every step.  In addition, at
    every checkpoint a SECOND oracle is loaded with the device's state and fields (teacher forcing) and the next step
    is compared with the strict single-step bar, 1e-9 on every SD: parity of the developed states the run passes through."""
    from paper_1310_1905_b200 import binding as b

    o = make_oracle(w, threads=THREADS)
    p, th, rv = make_particles(w)
    oo, po = oracle.make_opts(**w.opts), b.make_opts(**w.opts)
    forced = None
    for s in range(steps):
        if s > 0 and s % every == 0:
            g = sorted_by_id(p.export_state())
            forced = oracle.Oracle(**w.init)
            forced.set_threads(THREADS)
            c = courant_xyz(w)
            forced.set_fields(th=np_(th).ravel(), rv=np_(rv).ravel(), rhod=np_(w.rhod).ravel(),
                              cx=None if c["x"] is None else np_(c["x"]).ravel(), cy=None if c["y"] is None else np_(c["y"]).ravel(),
                              cz=None if c["z"] is None else np_(c["z"]).ravel())
            forced.set_state(g["n"].astype(np.uint64), g["rw2"], g["rd3"], g["kappa"], x=g["x"], y=g["y"] if w.init["ny"] > 0 else None, z=g["z"],
                             id=g["id"].astype(np.uint32))
            forced.set_step(s)
        fo = o.step(oo)
        p.step_sync(po, th, rv)
        p.step_async(po)
        fp = p.step_async_result()
        np.testing.assert_allclose(fp, fo, rtol=1e-7, atol=1e-300)
        if forced is not None:
            ff = forced.step(oo)
            np.testing.assert_allclose(fp, ff, rtol=3e-9, atol=1e-300)
            compare_states(p, forced)
            compare_fields(th, rv, forced)
            forced = None
        if (s + 1) % every == 0:
            compare_states(p, o, drift=DRIFT)
            compare_fields(th, rv, o)
    return p, o, th, rv


def test_config1_75x75_32_per_cell_600_step_prefix():
    """configs[1] as BASELINE.json states it (PAPER.md :101-138, :858-860): 75 x 75 cells of 20 m, 32 SDs per cell
    (180 000 SDs), geometric kernel, 10 condensation substeps, from the haze-only initial condition: the first 600 of
    its 3600 steps.  The cloud forms above ~800 m during this prefix, so activation, the slow list of the first steps,
    evaporation in the downdraught and the first collisions are all in it."""
    w = W.cfg2_2d()
    assert w.n_sd == 180000 and w.init["nx"] == 75 and w.init["nz"] == 75
    p, o, th, rv = _trajectory(w, 600, 100)
    sp, so = _counters_equal(p, o)
    assert sp["sd_substeps"] > 0.95 * 180000 * 10 * 600
    assert float(rv.min()) < 7.4e-3   # vapour was taken up by the cloud: condensation did act on the fields


def test_config2_75x75_128_per_cell_hydro_tab_200_steps():
    """configs[2]: the same grid with 128 SDs per cell (720 000 SDs), r_v = 8.5 g/kg, the tabulated-efficiency kernel
    (stand-in table, DESIGN.md R-efftab) and the terminal-velocity formula; a quarter of the SDs are given cloud to rain
    sizes so that the table is exercised from the first step on (the run proper needs ~1000 steps to form drizzle)."""
    w = rain_mix(W.cfg3_2d_drizzle(), seed=21, frac=0.25)
    assert w.n_sd == 720000 and w.init["kernel"] == "hydro_tab"
    p, o, th, rv = _trajectory(w, 200, 50)
    sp, so = _counters_equal(p, o)
    assert so["collisions"] > 10000 and o.rain_flux_total() > 0
    assert p.n_sd() == o.n_sd() < w.n_sd


LONG = pytest.mark.skipif(os.environ.get("SDM_LONG_TESTS", "") != "1", reason="full-length runs (10 and 35 minutes of oracle time): set SDM_LONG_TESTS=1")


@LONG
def test_config1_full_length_3600_steps():
    """configs[1] over its full 3600 steps (PAPER.md :858-860: the paper's own run), compared every 300 steps: free-running
    trajectory bar + the strict single-step bar from the device's state at every checkpoint."""
    p, o, th, rv = _trajectory(W.cfg2_2d(), 3600, 300)
    _counters_equal(p, o)
    assert o.rain_flux_total() > 0


@LONG
def test_config2_full_length_3600_steps():
    """configs[2] (720 000 SDs, r_v = 8.5 g/kg, tabulated efficiencies) over its full 3600 steps from the haze-only initial
    condition: the drizzle-forming run."""
    p, o, th, rv = _trajectory(W.cfg3_2d_drizzle(), 3600, 300)
    sp, so = _counters_equal(p, o)
    assert so["collisions"] > 1000


def test_one_cell_at_the_capacity_of_a_cta():
    """One cell with ~12 000 SDs (P = 16384, the most a CTA sorts in shared memory): the CTA-wide bitonic ranks
    (k_rank<256>), the in-place condensation kernel (k_cond<false>) and the in-place per-cell coalescence kernel
    (k_coal_move<256>) at the largest size the library accepts; a cell beyond 16384 SDs is refused with
    SDM_ERR_CAPACITY (include/sdm.h), not mis-sorted."""
    from paper_1310_1905_b200 import binding as b

    w = rain_mix(W.cfg2_2d(sd_per_cell=3000, nx=2, nz=2, seed=51), frac=0.3)
    w.state["x"] = w.state["x"] * 0.499     # everything into cell (0, 0)
    w.state["z"] = w.state["z"] * 0.499
    p, o, _, _ = run_both(w, 2, opts=dict(sstp_cond=2), threads=THREADS)
    assert 8192 < p.stats()["max_cell_count"] <= 16384
    assert p.stats()["cond_variant"] == 0 and p.stats()["coal_tile_cells"] == 0
    assert p.stats()["collisions"] == o.counters()["collisions"] > 100
    w = W.cfg2_2d(sd_per_cell=4200, nx=2, nz=2, seed=52)
    w.state["x"] = w.state["x"] * 0.499
    w.state["z"] = w.state["z"] * 0.499
    q, th, rv = make_particles(w)
    with pytest.raises(b.SdmError, match="more super-droplets than one CTA"):
        q.step_sync(b.make_opts(**w.opts), th, rv)


def test_spin_up_combination_cond_and_adve_only_under_rh_max():
    """The 2-hour spin-up of PAPER.md :132-134: condensation and advection only (coal = sedi = 0), growth limited by
    RH_max = 1.05 in the supersaturated upper third of the domain."""
    w = W.cfg2_2d(sd_per_cell=32, nx=12, nz=75, seed=53)
    p, o, th, rv = run_both(w, 20, check_every=5, opts=dict(coal=False, sedi=False, RH_max=1.05), threads=THREADS)
    sp, so = p.stats(), o.counters()
    assert sp["pairs"] == so["pairs"] == 0 and sp["ill_posed"] == so["ill_posed"]
    assert p.n_sd() == o.n_sd() == w.n_sd   # nothing sediments out, nothing coalesces


def test_fp32_sweep_falls_back_to_fp64_arithmetic_beyond_500_substeps():
    """sdm_set_cond_arith(4) with sstp_cond = 600: the packed per-lane counters of k_cond4f hold 500 substeps, so the
    library runs the fp64-arithmetic kernel on the fp32 state (sdm_api.cu); radii within the fp32 bar all the same."""
    w = rain_mix(W.cfg2_2d(sd_per_cell=16, nx=4, nz=20, seed=54))
    p, o = _fp32_case(w, steps=1, arith=4, sstp_cond=600)
    assert p.stats()["sd_substeps"] == o.counters()["sd_substeps"] == 600 * w.n_sd
