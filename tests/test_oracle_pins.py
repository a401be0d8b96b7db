"""Pins for the oracle (run with -m "not gpu").

Each test checks ``oracle/`` against something other than itself: values printed by the paper or the
literature (tests/golden), closed forms, invariants, brute force on tiny inputs.  Citations are
PAPER.md line numbers (``:NNN``).
"""
import itertools
import os

import numpy as np
import pytest
from scipy import integrate, optimize, special

import oracle

L = oracle.lib()

RHO_W, SIGMA_W, R_V, R_D, C_PD, P1000 = 1000.0, 0.072, 461.5, 287.0, 1005.0, 1e5


# ----------------------------------------------------------------------------- Philox
def test_philox_known_answers(golden_dir):
    rows = [l.split() for l in open(os.path.join(golden_dir, "philox_kat.txt")) if l.strip() and l[0] != "#"]
    assert len(rows) == 3
    for r in rows:
        v = [int(t, 16) for t in r if t != "->"]
        out = oracle.philox(v[0:4], v[4:6])
        assert [int(t) for t in out] == v[6:10]


def test_philox_counter_sensitivity():
    # a dropped counter word or key word would leave the output unchanged under that word's change
    base = oracle.philox([1, 2, 3, 4], [5, 6])
    for w in range(4):
        c = [1, 2, 3, 4]
        c[w] += 1
        assert (oracle.philox(c, [5, 6]) != base).all()
    assert (oracle.philox([1, 2, 3, 4], [6, 6]) != base).all()
    assert (oracle.philox([1, 2, 3, 4], [5, 7]) != base).all()


# ----------------------------------------------------------------------------- sort / pairing
def _grid_oracle(nx=4, nz=3, **kw):
    return oracle.Oracle(nx=nx, ny=0, nz=nz, dx=10.0, dy=1.0, dz=20.0, dt=1.0, **kw)


def test_sort_is_lexicographic_definition():
    """:624 + BASELINE north_star: order = sort on (cell, Philox key, id); key = Philox(id, step, 0, 0).w0."""
    rng = np.random.default_rng(3)
    N = 500
    o = _grid_oracle(seed=0x1234567855AA)
    x, z = rng.uniform(0, 40, N), rng.uniform(0, 60, N)
    ids = rng.permutation(10 * N)[:N].astype(np.uint32)
    n = rng.integers(1, 100, N).astype(np.uint64)
    n[::17] = 0  # dead SDs never reach the sort
    o.set_state(n, np.full(N, 1e-12), np.full(N, 1e-24), np.full(N, 0.5), x=x, z=z, id=ids)
    o.set_step(7)
    o.stage("sort")
    got_ids, seg = o.get_order()
    live = n > 0
    cell = (np.floor(x / 10.0).astype(int) * 1 + 0) * 3 + np.floor(z / 20.0).astype(int)
    key = [int(oracle.philox([int(i), 7, 0, 0], [0x567855AA, 0x1234])[0]) for i in ids]
    tup = sorted((int(cell[s]), key[s], int(ids[s])) for s in range(N) if live[s])
    assert [t[2] for t in tup] == [int(i) for i in got_ids]
    counts = np.bincount([t[0] for t in tup], minlength=12)
    assert (np.diff(seg) == counts).all()
    assert o.n_sd() == live.sum()  # compaction happened


def test_pairings_of_four_are_uniform():
    """:624 "randomly grouped into non-overlapping pairs": each of the 3 pairings of 4 SDs has frequency 1/3."""
    o = oracle.Oracle(dx=1, dy=1, dz=1, seed=99)
    ones = np.ones(4)
    counts = {}
    T = 30000
    for t in range(T):
        o.set_state(np.full(4, 5, np.uint64), ones, ones, ones)
        o.set_step(t)
        o.stage("sort")
        ids, _ = o.get_order()
        p = frozenset([frozenset(ids[:2].tolist()), frozenset(ids[2:].tolist())])
        counts[p] = counts.get(p, 0) + 1
    assert len(counts) == 3
    for c in counts.values():
        assert abs(c / T - 1 / 3) < 4.5 * np.sqrt(2 / 9 / T)


@pytest.mark.parametrize("nsd", [3, 4, 5, 6])
def test_pair_probability_bruteforce(nsd):
    """:626-631 eq. 27: thanks to the factor n(n-1)/2 / floor(n/2), the expected number of collision
    events of every unordered pair (i,j) per step equals the unscaled max(N_i,N_j) K dt/dV."""
    rng = np.random.default_rng(nsd)
    n = (np.array([7, 11, 13, 17, 19, 23][:nsd]) * 1000).astype(np.uint64)
    r = rng.uniform(10e-6, 30e-6, nsd)
    v = 4 / 3 * np.pi * r**3
    b, dV, dt = 1500.0, 1e-3, 1.0
    o = oracle.Oracle(dx=0.1, dy=0.1, dz=0.1, dt=dt, kernel="golovin", golovin_b=b, seed=4242)
    op = oracle.make_opts(adve=False, sedi=False, cond=False, coal=True)
    pairs = list(itertools.combinations(range(nsd), 2))
    expect = {pr: max(n[pr[0]], n[pr[1]]) * b * (v[pr[0]] + v[pr[1]]) * dt / dV for pr in pairs}
    scale = (nsd * (nsd - 1) / 2) / (nsd // 2)
    assert max(expect.values()) * scale < 1.0  # stay in the single-collision regime
    T = 60000
    hits = dict.fromkeys(pairs, 0)
    rw2, rd3, kap = r**2, np.full(nsd, 1e-27), np.full(nsd, 0.5)
    for t in range(T):
        o.set_state(n, rw2, rd3, kap)
        o.set_step(t)
        o.stage("sort")
        o.stage("coal", op)
        st = o.get_state()
        grown = np.nonzero(st["rw2"] != rw2)[0]
        shrunk = np.nonzero(st["n"] != n)[0]
        assert len(grown) == len(shrunk)
        for k in grown:  # the partner is the SD whose multiplicity dropped by n_k
            j = [j for j in shrunk if n[j] - st["n"][j] == n[k]]
            assert len(j) == 1
            hits[tuple(sorted((int(k), int(j[0]))))] += 1
    for pr in pairs:
        p = expect[pr]
        sd = np.sqrt(T * p * scale)  # event count ~ Binomial with variance <= T p scale / scale... use generous bound
        assert abs(hits[pr] - T * p) < 4.5 * max(sd / np.sqrt(scale), 3.0), (pr, hits[pr], T * p)


def test_adaptive_coalescence_substeps_from_pij():
    """DESIGN.md reading R-adapt-coal (PAPER.md :645 "use the values of P_ij to control an adaptive timestep logic"): a cell
    takes sstp_coal * m substeps, m = min(coal_adapt_max, ceil(max P_ij over its first grouping)).  Pinned by (i) the
    paper's variant without multiple coalescence on a pair with P = 3.7: one substep yields exactly one event per step (the
    undersampling :645 describes), m = 2 exactly two, and m = 4 substeps of P' = 0.925 a Binomial(4, 0.925) number whose mean
    is the 3.7 collisions the probability stands for; (ii) the rule restated on a 9-SD Golovin cell from the grouping the
    oracle reports: the candidate pairs examined are m * floor(n/2); (iii) coal_adapt_max <= 1 is the fixed step bit for bit."""
    b, dV, dt = 1500.0, 1.0, 1.0
    rj, rk, nj = 1e-6, 30e-6, 10**9            # many small droplets (j) against one big drop (k): k hardly changes when hit
    K = b * 4 / 3 * np.pi * (rj**3 + rk**3)
    dV = nj * K * dt / 3.7                     # P = N_j K dt / dV = 3.7 (two SDs: the factor of eq. 27 is 1)
    side = dV ** (1 / 3)
    T = 3000

    def mean_drop(**kw):
        o = oracle.Oracle(dx=side, dy=side, dz=side, dt=dt, kernel="golovin", golovin_b=b, multi_coal=False, seed=11)
        op = oracle.make_opts(adve=False, sedi=False, cond=False, coal=True, **kw)
        drops = []
        for t in range(T):
            o.set_state(np.array([nj, 1], np.uint64), np.array([rj**2, rk**2]), np.full(2, 1e-27), np.full(2, 0.5))
            o.set_step(t)
            o.stage("sort")
            o.stage("coal", op)
            drops.append(nj - int(o.get_state()["n"][0]))
        return np.array(drops)

    assert set(mean_drop()) == {1}                                   # fixed: u < 1 < P every step, one event, 2.7 lost
    assert set(mean_drop(coal_adapt_max=2)) == {2}                   # capped at m = 2: P' = 1.85 still above 1
    d = mean_drop(coal_adapt_max=8)                                  # m = ceil(3.7) = 4, P' = 0.925
    assert d.max() == 4 and d.min() >= 1
    assert abs(d.mean() - 3.7) < 4.5 * np.sqrt(4 * 0.925 * 0.075 / T)
    assert set(mean_drop(coal_adapt_max=8, sstp_coal=2)) <= {1, 2, 3, 4}   # P(dt/2) = 1.85 -> m = 2: again 4 substeps
    # (ii) the rule on a cell of 9 SDs
    rng = np.random.default_rng(12)
    nsd = 9
    n = (np.array([7, 11, 13, 17, 19, 23, 29, 31, 37]) * 10**6).astype(np.uint64)
    r = rng.uniform(10e-6, 30e-6, nsd)
    v = 4 / 3 * np.pi * r**3
    scale = (nsd * (nsd - 1) / 2) / (nsd // 2)
    for want_m, cap in ((1, 8), (3, 8), (6, 8), (5, 5)):
        o = oracle.Oracle(dx=1.0, dy=1.0, dz=1.0, dt=dt, kernel="golovin", golovin_b=b, seed=77)
        o.set_state(n, r**2, np.full(nsd, 1e-27), np.full(nsd, 0.5))
        o.stage("sort")
        ids, _ = o.get_order()
        P1 = max(float(max(n[i], n[j])) * b * (v[i] + v[j]) * dt * scale for i, j in zip(ids[0:-1:2], ids[1::2]))   # at dV = 1
        target = {1: 0.8, 3: 2.5, 6: 5.5, 5: 7.3}[want_m]            # the P_max this case is built to have
        side = (P1 / target) ** (1 / 3)
        o = oracle.Oracle(dx=side, dy=side, dz=side, dt=dt, kernel="golovin", golovin_b=b, seed=77)
        o.set_state(n, r**2, np.full(nsd, 1e-27), np.full(nsd, 0.5))
        o.stage("sort")
        ids2, _ = o.get_order()
        np.testing.assert_array_equal(ids, ids2)                    # the grouping does not depend on the cell volume
        o.stage("coal", oracle.make_opts(adve=False, sedi=False, cond=False, coal=True, coal_adapt_max=cap))
        assert o.counters()["pairs"] == want_m * (nsd // 2), (want_m, o.counters()["pairs"])
    # (iii) off means off
    for mx in (0, 1):
        a = oracle.Oracle(dx=0.01, dy=0.01, dz=0.01, dt=dt, kernel="golovin", golovin_b=b, seed=5)
        f = oracle.Oracle(dx=0.01, dy=0.01, dz=0.01, dt=dt, kernel="golovin", golovin_b=b, seed=5)
        for o, kw in ((a, dict(coal_adapt_max=mx)), (f, {})):
            o.set_state(n, r**2, np.full(nsd, 1e-27), np.full(nsd, 0.5))
            for _ in range(5):
                o.step(oracle.make_opts(adve=False, sedi=False, cond=False, coal=True, **kw))
        for k in ("n", "rw2", "rd3"):
            np.testing.assert_array_equal(a.get_state()[k], f.get_state()[k])


def _stokes(r, eta, rho_a):
    """Stokes fall speed 2 r^2 g (rho_w - rho_a) / (9 eta): the r -> 0 limit of the terminal-velocity formula (:649),
    within 3e-3 of it up to 1 um (test_terminal_velocity_stokes_limit_and_textbook)."""
    return 2.0 * r * r * 9.81 * (RHO_W - rho_a) / (9.0 * eta)


def _two_sd_collisions(kernel, rj, rk, nj, dV, dt=1.0, sstp_coal=1, **kw):
    """One coalescence stage on a cell holding exactly two SDs (N_j = nj >> N_k = 1, so n_c(n_c-1)/2 / floor(n_c/2) = 1
    and the cap floor(N_j/N_k) is far away).  With multiple coalescence gamma = floor(p) + [u < frac p] (north_star), so
    the drop of N_j equals p = N_j K dt/dV to within one event per substep: K is read off deterministically."""
    side = dV ** (1 / 3)
    o = oracle.Oracle(dx=side, dy=side, dz=side, dt=dt, kernel=kernel, seed=7, **kw)
    op = oracle.make_opts(adve=False, sedi=False, cond=False, coal=True, sstp_coal=sstp_coal)
    o.set_state(np.array([nj, 1], np.uint64), np.array([rj**2, rk**2]), np.full(2, 1e-27), np.full(2, 0.5))
    o.stage("sort")
    o.stage("coal", op)
    st = o.get_state()
    assert st["n"][1] == 1
    return nj - int(st["n"][0]), st


@pytest.mark.parametrize("rj,rk", [(0.4e-6, 1.0e-6), (1.0e-6, 0.3e-6), (0.7e-6, 0.9e-6)])
def test_geometric_kernel_is_eq28(rj, rk):
    """:633-637 eq. 28: K = E pi (r_j + r_k)^2 |v_j - v_k| (E = 1 for `geometric`).  Sub-micron drops fall at the
    Stokes speed (closed form), so the expected number of events of the pair is known without the oracle:
    N_j pi (r_j + r_k)^2 |v_j - v_k| dt / dV.  A dropped square, a missing pi, volumes in place of radii, a sum in
    place of the difference of the fall speeds or a swapped operand each change it by far more than the 1 % bar."""
    ct = oracle.cell_thermo(300.0, 0.0, 1.0)      # the default fields of a fresh oracle (th = 300 K, r_v = 0, rho_d = 1)
    vj, vk = _stokes(rj, ct["eta"], ct["rho_a"]), _stokes(rk, ct["eta"], ct["rho_a"])
    K = np.pi * (rj + rk) ** 2 * abs(vj - vk)
    dV, dt = 1e-9, 1.0
    nj = int(2000.5 * dV / (K * dt))              # p = 2000.5
    got, _ = _two_sd_collisions("geometric", rj, rk, nj, dV, dt)
    assert abs(got - nj * K * dt / dV) <= 1 + 0.01 * 2000.5, (got, nj * K * dt / dV)
    # and the time step enters linearly
    got2, _ = _two_sd_collisions("geometric", rj, rk, nj, dV, 0.5 * dt)
    assert abs(got2 - 0.5 * nj * K * dt / dV) <= 1 + 0.01 * 1000.0


def test_hydro_tab_kernel_is_eq28_times_the_tabulated_efficiency():
    """:633-637 eq. 28 with E(collector radius, small/large ratio) from a 2 x 2 table: the bilinear value is computed
    by hand here (collector = the LARGER drop whichever of the two SDs carries the larger multiplicity)."""
    R, q = np.array([0.5e-6, 1.5e-6]), np.array([0.2, 0.8])
    tab = np.array([[0.1, 0.3], [0.6, 1.0]])
    ct = oracle.cell_thermo(300.0, 0.0, 1.0)
    for rj, rk in ((0.4e-6, 1.0e-6), (1.0e-6, 0.4e-6), (1.2e-6, 0.9e-6)):
        rl, rs = max(rj, rk), min(rj, rk)
        t, u = (rl - R[0]) / (R[1] - R[0]), (rs / rl - q[0]) / (q[1] - q[0])
        E = (1 - t) * (1 - u) * tab[0, 0] + (1 - t) * u * tab[0, 1] + t * (1 - u) * tab[1, 0] + t * u * tab[1, 1]
        K = E * np.pi * (rj + rk) ** 2 * abs(_stokes(rj, ct["eta"], ct["rho_a"]) - _stokes(rk, ct["eta"], ct["rho_a"]))
        dV = 1e-9
        nj = int(3000.5 * dV / K)
        got, _ = _two_sd_collisions("hydro_tab", rj, rk, nj, dV, eff_R=R, eff_q=q, eff_tab=tab)
        assert abs(got - nj * K / dV) <= 1 + 0.01 * 3000.5, (rj, rk, got, nj * K / dV)


def test_coalescence_substeps_use_dt_over_sstp_coal():
    """:624 / DESIGN.md reading R-sstp-coal: each of the sstp_coal substeps applies eq. 27 with dt'' = dt / sstp_coal.
    Two-SD cell, Golovin kernel with v_j << v_k so that K hardly changes when k grows: the events of one step add up
    to N_j K dt / dV whatever the number of substeps (a full dt per substep would give sstp_coal times as many)."""
    rj, rk, b, dV = 1e-6, 100e-6, 1500.0, 1e-3
    K = b * 4 / 3 * np.pi * (rj**3 + rk**3)
    nj = int(1000.5 * dV / K)
    for sstp in (1, 4, 5):
        got, st = _two_sd_collisions("golovin", rj, rk, nj, dV, sstp_coal=sstp, golovin_b=b)
        growth = 1 + got * rj**3 / rk**3           # v_k grew by the collected volume: K rose by less than this
        assert 1000.5 - sstp <= got <= 1000.5 * growth + sstp, (sstp, got)
        np.testing.assert_allclose(st["rw2"][1] ** 1.5, rk**3 + got * rj**3, rtol=1e-13)


@pytest.mark.parametrize("kernel,nsd,sstp", [("geometric", 4, 1), ("geometric", 5, 1), ("geometric", 4, 4)])
def test_pair_probability_bruteforce_geometric(kernel, nsd, sstp):
    """eq. 27 with eq. 28 on 4-5-SD cells of distinct radii (and once with sstp_coal = 4): the expected events of every
    unordered pair per step are max(N_i, N_j) pi (r_i + r_j)^2 |v_i - v_j| dt/dV with Stokes fall speeds."""
    n = (np.array([7, 11, 13, 17, 19][:nsd]) * 10**9).astype(np.uint64)
    r = np.array([0.35, 0.95, 0.6, 0.8, 0.45][:nsd]) * 1e-6
    ct = oracle.cell_thermo(300.0, 0.0, 1.0)
    v = _stokes(r, ct["eta"], ct["rho_a"])
    pairs = list(itertools.combinations(range(nsd), 2))
    scale = (nsd * (nsd - 1) / 2) / (nsd // 2)
    K = {pr: np.pi * (r[pr[0]] + r[pr[1]]) ** 2 * abs(v[pr[0]] - v[pr[1]]) for pr in pairs}
    dV = max(float(max(n[a], n[b])) * K[(a, b)] for a, b in pairs) * scale / (0.5 if sstp == 1 else 0.12)
    expect = {pr: float(max(n[pr[0]], n[pr[1]])) * K[pr] / dV for pr in pairs}
    side = dV ** (1 / 3)
    o = oracle.Oracle(dx=side, dy=side, dz=side, dt=1.0, kernel=kernel, seed=99)
    op = oracle.make_opts(adve=False, sedi=False, cond=False, coal=True, sstp_coal=sstp)
    T = 40000
    hits, ambiguous = dict.fromkeys(pairs, 0), 0
    rw2, rd3, kap = r**2, np.full(nsd, 1e-27), np.full(nsd, 0.5)
    for t in range(T):
        o.set_state(n, rw2, rd3, kap)
        o.set_step(t)
        o.stage("sort")
        o.stage("coal", op)
        st = o.get_state()
        grown, shrunk = np.nonzero(st["rw2"] != rw2)[0], np.nonzero(st["n"] != n)[0]
        found = []
        for k in grown:   # the partner is the SD whose multiplicity dropped by n_k
            j = [j for j in shrunk if n[j] - st["n"][j] == n[k]]
            if len(j) == 1:
                found.append(tuple(sorted((int(k), int(j[0])))))
        if len(found) != len(grown) or len(grown) != len(shrunk):
            ambiguous += 1      # two events touching one SD within the substeps of a step: not attributable
            continue
        for pr in found:
            hits[pr] += 1
    assert ambiguous <= (0 if sstp == 1 else 0.01 * T)
    for pr in pairs:
        p = expect[pr]
        tol = 4.5 * np.sqrt(T * p) + (0.0 if sstp == 1 else 0.12 * T * p)   # substeps: second-order depletion of the sample
        assert abs(hits[pr] - T * p) < max(tol, 8.0), (pr, hits[pr], T * p)
    assert sum(hits.values()) > 3000


def test_collision_update_worked_example():
    """:639-643 with DESIGN.md reading R-collision (Shima 2009 rule): hand-computed two-SD cell."""
    b, dV, dt = 1.0, 1.0, 1.0
    rj, rk = 2.0e-1, 1.0e-1
    vj, vk = 4 / 3 * np.pi * rj**3, 4 / 3 * np.pi * rk**3
    nj, nk = 8, 2
    p = nj * b * (vj + vk) * dt / dV  # n_c = 2 -> scale factor 1
    assert 0.3 < p < 0.31
    # choose b so that p = 10.3 > floor(n_j/n_k) = 4  -> g = 4, SD j dies
    o = oracle.Oracle(dx=1, dy=1, dz=1, dt=dt, kernel="golovin", golovin_b=10.3 / p, seed=1)
    op = oracle.make_opts(adve=False, sedi=False, cond=False, coal=True)
    o.set_state(np.array([nj, nk], np.uint64), np.array([rj**2, rk**2]), np.array([3e-24, 1e-24]), np.array([0.2, 0.8]))
    o.stage("sort")
    o.stage("coal", op)
    st = o.get_state()
    j, k = (0, 1)
    assert st["n"].tolist() == [0, 2]
    assert st["rw2"][j] == rj**2 and st["rd3"][j] == 3e-24 and st["kappa"][j] == 0.2  # j keeps its radii
    np.testing.assert_allclose(st["rw2"][k] ** 1.5, rk**3 + 4 * rj**3, rtol=1e-14)
    np.testing.assert_allclose(st["rd3"][k], 1e-24 + 4 * 3e-24, rtol=1e-15)
    np.testing.assert_allclose(st["kappa"][k], (4 * 3e-24 * 0.2 + 1e-24 * 0.8) / (13e-24), rtol=1e-15)
    # p = 2.5 -> gamma in {2, 3} (multi_coal) but exactly {0 or 1} in the paper's variant (:645)
    for multi, allowed in ((True, {2, 3}), (False, {1})):
        seen = set()
        o = oracle.Oracle(dx=1, dy=1, dz=1, dt=dt, kernel="golovin", golovin_b=2.5 / p, seed=1, multi_coal=multi)
        for t in range(40):
            o.set_state(np.array([nj, nk], np.uint64), np.array([rj**2, rk**2]), np.array([3e-24, 1e-24]), np.array([0.2, 0.8]))
            o.set_step(t)
            o.stage("sort")
            o.stage("coal", op)
            seen.add((nj - int(o.get_state()["n"][0])) // nk)
        assert seen == allowed


def test_equal_multiplicity_tie_break_first_in_order_is_j():
    """DESIGN.md reading R-tie: on N_i = N_j the first SD in sorted order loses its multiplicity (:641)."""
    o = oracle.Oracle(dx=1, dy=1, dz=1, dt=1.0, kernel="golovin", golovin_b=1e18, seed=5)
    op = oracle.make_opts(adve=False, sedi=False, cond=False, coal=True)
    for t in range(20):
        o.set_state(np.array([5, 5], np.uint64), np.array([1e-10, 4e-10]), np.full(2, 1e-27), np.full(2, 0.5))
        o.set_step(t)
        o.stage("sort")
        first = int(o.get_order()[0][0])
        o.stage("coal", op)
        n = o.get_state()["n"]
        assert n[first] == 0 and n[1 - first] == 5


def test_coalescence_conserves_mass_and_sum_n_is_monotone():
    """:643 extensive attributes are summed: sum N r_w^3 and sum N r_d^3 are conserved (this is what decides
    reading R-collision, the printed wording of :639 does not conserve mass); sum N never grows."""
    rng = np.random.default_rng(11)
    N = 4000
    o = _grid_oracle(kernel="geometric", seed=77)
    o.set_fields(th=np.full(12, 289.0), rv=np.full(12, 7.5e-3), rhod=np.full(12, 1.1))
    n = rng.integers(1, 10**6, N).astype(np.uint64) * 1000
    r = np.exp(rng.uniform(np.log(1e-6), np.log(300e-6), N))
    rd3 = np.exp(rng.uniform(np.log(1e-24), np.log(1e-20), N))
    kap = rng.choice([0.3, 0.61, 1.2], N)
    o.set_state(n, r**2, rd3, kap, x=rng.uniform(0, 40, N), z=rng.uniform(0, 60, N))
    op = oracle.make_opts(adve=False, sedi=False, cond=False, coal=True, sstp_coal=3)
    f = np.float64
    m_w0, m_d0, s0 = (n.astype(f) * r**3).sum(), (n.astype(f) * rd3).sum(), int(n.sum())
    kd0 = (n.astype(f) * rd3 * kap).sum()
    for _ in range(20):
        o.step(op)
        st = o.get_state()
        nn = st["n"].astype(f)
        assert abs((nn * st["rw2"] ** 1.5).sum() / m_w0 - 1) < 1e-13
        assert abs((nn * st["rd3"]).sum() / m_d0 - 1) < 1e-13
        assert abs((nn * st["rd3"] * st["kappa"]).sum() / kd0 - 1) < 1e-13  # dry-volume-weighted kappa
        s1 = int(st["n"].sum())
        assert s1 <= s0
        s0 = s1
    c = o.counters()
    assert c["collisions"] > 1000 and s0 < int(n.sum())  # the test did exercise collisions (incl. gamma > 1)


# ----------------------------------------------------------------------------- Golovin box
def golovin_n(v, t, n0, v0, b):
    """Golovin (1963) solution for K = b(u+v), n(v,0) = n0/v0 exp(-v/v0)."""
    T = b * n0 * v0 * t
    tau = 1 - np.exp(-T)
    x = v / v0
    return n0 / v0 * (1 - tau) / (x * np.sqrt(tau)) * special.ive(1, 2 * x * np.sqrt(tau)) * np.exp(-x * (1 - np.sqrt(tau)) ** 2)


def test_golovin_closed_form_moments():
    n0, v0, b, t = 2.0**23, 4 / 3 * np.pi * 30.531e-6**3, 1500.0, 1200.0
    T = b * n0 * v0 * t
    lx = np.linspace(-30, 9, 400001)  # trapezoid in ln(v/v0); integrand is smooth and decays at both ends
    M = [np.trapezoid(golovin_n(np.exp(lx) * v0, t, n0, v0, b) * (np.exp(lx) * v0) ** (k + 1), lx) for k in range(3)]
    np.testing.assert_allclose(M[0], n0 * np.exp(-T), rtol=1e-6)
    np.testing.assert_allclose(M[1], n0 * v0, rtol=1e-6)
    np.testing.assert_allclose(M[2], 2 * n0 * v0**2 * np.exp(2 * T), rtol=1e-6)


def test_box_golovin_against_analytic_solution():
    """BASELINE.json configs[0]: V=1e6 m^3, 2^13 SDs, n0=2^23 m^-3, v0=(4/3)pi(30.531um)^3, b=1500/s, dt=1 s.
    Pooled over 16 seeds, the zeroth moment and the binned mass spectrum follow the Golovin solution."""
    N, n0, V, b = 2**13, 2.0**23, 1e6, 1500.0
    v0 = 4 / 3 * np.pi * 30.531e-6**3
    op = oracle.make_opts(adve=False, sedi=False, cond=False, coal=True)
    edges = np.exp(np.linspace(np.log(5e-6), np.log(2e-3), 25))
    times = (1200, 2400, 3600)
    M0 = {t: [] for t in times}
    hist = {t: np.zeros(len(edges) - 1) for t in times}
    mass = []
    for seed in range(42, 58):
        rng = np.random.default_rng(seed)
        v = rng.exponential(v0, N)
        o = oracle.Oracle(dx=100, dy=100, dz=100, dt=1.0, kernel="golovin", golovin_b=b, seed=seed)
        n = np.full(N, int(n0 * V / N), np.uint64)
        o.set_state(n, (v / (4 / 3 * np.pi)) ** (2 / 3), np.full(N, 1e-27), np.full(N, 0.5))
        m_ini = (n * v).sum()
        for t in range(1, 3601):
            o.step(op)
            if t in times:
                st = o.get_state()
                live = st["n"] > 0
                r = np.sqrt(st["rw2"][live])
                nn = st["n"][live].astype(float)
                M0[t].append(nn.sum() / V)
                hist[t] += np.histogram(r, edges, weights=nn * 4 / 3 * np.pi * r**3)[0] / V
                mass.append((nn * 4 / 3 * np.pi * r**3).sum() / m_ini)
    np.testing.assert_allclose(mass, 1.0, rtol=1e-12)  # first moment constant
    tol_M0 = {1200: 0.06, 2400: 0.12, 3600: 0.35}  # sampling error grows as the SD count decays
    for t in times:
        T = b * n0 * v0 * t
        ratio = np.mean(M0[t]) / (n0 * np.exp(-T))
        assert abs(ratio - 1) < tol_M0[t], (t, ratio)
    # mass density per bin at 1200 s against the integral of the closed form
    t = 1200
    ana = np.array([integrate.quad(lambda lr: golovin_n(4 / 3 * np.pi * np.exp(3 * lr), t, n0, v0, b)
                                   * (4 / 3 * np.pi * np.exp(3 * lr)) ** 2 * 3, np.log(a), np.log(c))[0]
                    for a, c in zip(edges[:-1], edges[1:])])
    sim = hist[t] / 16
    assert abs(ana.sum() / (n0 * v0) - 1) < 1e-3
    big = ana > 0.02 * ana.sum()
    assert big.sum() >= 5
    assert np.abs(sim[big] / ana[big] - 1).max() < 0.2, (sim[big] / ana[big])
    assert np.abs(sim - ana).sum() / ana.sum() < 0.1
    # the mode of the mass spectrum moves to larger radii as in the closed form
    assert np.argmax(hist[3600]) > np.argmax(hist[1200])


# ----------------------------------------------------------------------------- recycling (PAPER.md :641, :651)
def _recycle_case(n):
    N = len(n)
    rng = np.random.default_rng(3)
    ids = rng.permutation(N).astype(np.uint32)   # storage order is not id order
    o = oracle.Oracle(dx=100, dy=100, dz=100, kernel="golovin")
    rw2 = rng.uniform(1e-12, 1e-10, N)
    o.set_state(n, rw2, rw2**1.5 * 1e-3, rng.uniform(0.1, 1.0, N), rng.uniform(0, 100, N), rng.uniform(0, 100, N),
                rng.uniform(0, 100, N), id=ids)
    before = o.get_state()
    o.stage_recycle()
    return before, o.get_state(), o


def test_recycling_takes_the_highest_multiplicities_and_halves_them():
    """PAPER.md :641: 'first looks for computational particles with highest multiplicites and then assignes their
    properties to the recycled particles halving the multiplicity'.  Checked as properties of the result, not by
    re-sorting: what changed, who gave, who received, and that no SD that kept its multiplicity outranks a donor."""
    rng = np.random.default_rng(11)
    n = rng.integers(1, 50, 400).astype(np.uint64)   # many ties
    n[rng.choice(400, 37, replace=False)] = 0
    b, a, o = _recycle_case(n)
    dead = b["n"] == 0
    assert o.recycled == 37 and (a["n"] > 0).all()
    assert int(a["n"].sum()) == int(b["n"].sum())                                   # real particles conserved exactly
    for k in ("rw2", "rd3"):                                                        # extensive totals conserved
        np.testing.assert_allclose((a["n"] * a[k] ** (1.5 if k == "rw2" else 1)).sum(),
                                   (b["n"] * b[k] ** (1.5 if k == "rw2" else 1)).sum(), rtol=1e-14)
    np.testing.assert_array_equal(a["id"], b["id"])                                 # ids are persistent
    donors = np.flatnonzero(~dead & (a["n"] != b["n"]))
    assert len(donors) == 37
    # every donor kept the larger half, and exactly one recycled SD holds the other half with the donor's attributes
    taken = set()
    for s in donors:
        half = int(b["n"][s]) // 2
        assert int(a["n"][s]) == int(b["n"][s]) - half
        m = np.flatnonzero(dead & (a["n"] == half) & (a["rw2"] == b["rw2"][s]) & (a["x"] == b["x"][s]) & (a["kappa"] == b["kappa"][s])
                           & (a["rd3"] == b["rd3"][s]) & (a["y"] == b["y"][s]) & (a["z"] == b["z"][s]))
        assert len(m) == 1 and m[0] not in taken
        taken.add(int(m[0]))
    # the donors are the top of the order (multiplicity descending, id ascending): nobody left out outranks one
    rest = np.flatnonzero(~dead & (a["n"] == b["n"]))
    worst = min((int(b["n"][s]), -int(b["id"][s])) for s in donors)
    assert all((int(b["n"][s]), -int(b["id"][s])) < worst for s in rest)
    # donors in rank order serve the dead SDs in id order
    rank = sorted(donors, key=lambda s: (-int(b["n"][s]), int(b["id"][s])))
    dead_by_id = sorted(np.flatnonzero(dead), key=lambda s: int(b["id"][s]))
    for s, d in zip(rank, dead_by_id):
        assert a["rw2"][d] == b["rw2"][s] and int(a["n"][d]) == int(b["n"][s]) // 2


def test_recycling_without_enough_donors_and_without_dead():
    n = np.array([1, 0, 1, 0, 3, 0, 1, 2], np.uint64)       # two SDs can be halved, three are dead
    b, a, o = _recycle_case(n)
    assert o.recycled == 2 and int(a["n"].sum()) == int(b["n"].sum())
    dead_ids = sorted(int(i) for i in b["id"][b["n"] == 0])
    still_dead = [int(i) for i in a["id"][a["n"] == 0]]
    assert still_dead == [dead_ids[-1]]                      # the dead SD of highest id is not served
    assert sorted(a["n"].tolist()) == [0, 1, 1, 1, 1, 1, 1, 2]
    n = np.array([4, 7, 1], np.uint64)
    b, a, o = _recycle_case(n)
    assert o.recycled == 0 and all((a[k] == b[k]).all() for k in a)


def test_box_golovin_with_recycling_keeps_the_sample_and_the_late_spectrum():
    """configs[0] with the paper's recycling instead of compaction: the SD count stays at 2^13, so the zeroth moment
    still follows the Golovin solution at 3600 s (compaction alone is left with ~40 SDs there) and the second
    moment, carried by the few largest drops, is not lost."""
    N, n0, V, b = 2**13, 2.0**23, 1e6, 1500.0
    v0 = 4 / 3 * np.pi * 30.531e-6**3
    op = oracle.make_opts(adve=False, sedi=False, cond=False, coal=True)
    times = (1200, 2400, 3600)
    M0 = {t: [] for t in times}
    M2 = {t: [] for t in times}
    for seed in range(42, 46):
        v = np.random.default_rng(seed).exponential(v0, N)
        o = oracle.Oracle(dx=100, dy=100, dz=100, dt=1.0, kernel="golovin", golovin_b=b, seed=seed)
        o.set_recycle(True)
        n = np.full(N, int(n0 * V / N), np.uint64)
        o.set_state(n, (v / (4 / 3 * np.pi)) ** (2 / 3), np.full(N, 1e-27), np.full(N, 0.5))
        m_ini = (n * v).sum()
        for t in range(1, 3601):
            o.step(op)
            if t in times:
                st = o.get_state()
                assert (st["n"] > 0).sum() >= 0.995 * N
                vv = 4 / 3 * np.pi * st["rw2"] ** 1.5
                nn = st["n"].astype(float)
                np.testing.assert_allclose((nn * vv).sum(), m_ini, rtol=1e-12)
                M0[t].append(nn.sum() / V)
                M2[t].append((nn * vv * vv).sum() / V)
    for t, tol in zip(times, (0.05, 0.08, 0.12)):
        T = b * n0 * v0 * t
        assert abs(np.mean(M0[t]) / (n0 * np.exp(-T)) - 1) < tol, (t, np.mean(M0[t]) / (n0 * np.exp(-T)))
    T = b * n0 * v0 * 2400
    assert 0.6 < np.mean(M2[2400]) / (2 * n0 * v0**2 * np.exp(2 * T)) < 1.4


# ----------------------------------------------------------------------------- thermodynamics
def test_T_p_inversion_of_eq41():
    """:1016-1018 eq. 41 theta = T (p_1000/p_d)^(R_d/c_pd), p_d = rho_d R_d T  <=>  eq. 43 (:1044)."""
    for th, rhod in ((289.0, 1.2), (300.0, 0.9), (275.0, 1.05)):
        T = L.orc_T(th, rhod)
        pd = rhod * R_D * T
        np.testing.assert_allclose(T * (P1000 / pd) ** (R_D / C_PD), th, rtol=1e-14)
        np.testing.assert_allclose(L.orc_p(rhod, 0.01, T), rhod * (R_D + 0.01 * R_V) * T, rtol=1e-15)  # eq. 44


def test_pvs_textbook_and_clausius_clapeyron(golden_dir):
    for l in open(os.path.join(golden_dir, "textbook_values.txt")):
        w = l.split()
        if w and w[0] == "pvs":
            np.testing.assert_allclose(L.orc_pvs(float(w[1])), float(w[2]), rtol=float(w[3]))
    # d ln p_vs/dT = l_v/(R_v T^2) with l_v of Table 2 (:1087)
    for T in (265.0, 280.0, 300.0):
        h = 1e-3
        d = (np.log(L.orc_pvs(T + h)) - np.log(L.orc_pvs(T - h))) / (2 * h)
        lv = 2.5e6 + (1850.0 - 4218.0) * (T - 273.16)
        np.testing.assert_allclose(L.orc_lv(T), lv, rtol=1e-15)
        np.testing.assert_allclose(d, lv / (R_V * T * T), rtol=1e-7)


def test_terminal_velocity_stokes_limit_and_textbook(golden_dir):
    T, rhod = 293.15, 1.2
    eta = L.orc_eta(T)
    assert abs(eta / 1.81e-5 - 1) < 0.01  # air at 20 C
    for r in (1e-8, 1e-7, 1e-6):
        stokes = 2 * r * r * 9.81 * (RHO_W - rhod) / (9 * eta)
        assert abs(L.orc_vterm(r, T, rhod, 0.0) / stokes - 1) < 3e-3
    for l in open(os.path.join(golden_dir, "textbook_values.txt")):
        w = l.split()
        if w and w[0] == "vt":
            np.testing.assert_allclose(L.orc_vterm(float(w[1]), T, rhod, 0.0), float(w[2]), rtol=float(w[3]))
    v = [L.orc_vterm(r, T, rhod, 0.0) for r in np.geomspace(1e-9, 3e-3, 200)]
    assert (np.diff(v) > 0).all()


# ----------------------------------------------------------------------------- growth law
TH, RHOD = 289.0, 1.1


def _rv_for_RH(RH):
    ct = oracle.cell_thermo(TH, 0.0, RHOD)
    return RH * ct["rho_vs"] / RHOD


def _S_eq(r, rd3, kappa):
    """kappa-Koehler equilibrium saturation (eq. 22 with Table 2 :1056, :1074), written independently."""
    T = L.orc_T(TH, RHOD)
    A = 2 * SIGMA_W / (R_V * T * RHO_W)
    return (r**3 - rd3) / (r**3 - rd3 * (1 - kappa)) * np.exp(A / r)


def test_growth_rate_sign_changes_at_koehler_equilibrium():
    rd3, kappa = (50e-9) ** 3, 0.61
    for r in (60e-9, 0.2e-6, 1e-6, 10e-6):
        S = _S_eq(r, rd3, kappa)
        fp = L.orc_growth_f(r * r, rd3, kappa, TH, _rv_for_RH(S * (1 + 1e-6)), RHOD, 44.0, r * r)
        fm = L.orc_growth_f(r * r, rd3, kappa, TH, _rv_for_RH(S * (1 - 1e-6)), RHOD, 44.0, r * r)
        assert fp > 0 > fm


def test_koehler_critical_point_closed_forms():
    """r_c = sqrt(3 kappa r_d^3 / A), ln S_c = sqrt(4 A^3 / (27 kappa r_d^3)) (dilute limit)."""
    T = L.orc_T(TH, RHOD)
    A = 2 * SIGMA_W / (R_V * T * RHO_W)
    for rd, kappa in ((30e-9, 0.61), (80e-9, 0.61), (50e-9, 1.2)):
        rd3 = rd**3

        def S_of_r(r):  # saturation at which the oracle's growth rate vanishes (f is linear in RH)
            y = r * r
            f1 = L.orc_growth_f(y, rd3, kappa, TH, _rv_for_RH(1.0), RHOD, 44.0, y)
            f2 = L.orc_growth_f(y, rd3, kappa, TH, _rv_for_RH(1.01), RHOD, 44.0, y)
            return 1.0 - f1 * 0.01 / (f2 - f1)

        res = optimize.minimize_scalar(lambda lr: -S_of_r(np.exp(lr)), bounds=(np.log(1.5 * rd), np.log(100 * rd)), method="bounded",
                                       options=dict(xatol=1e-10))
        rc, Sc = np.exp(res.x), -res.fun
        np.testing.assert_allclose(rc, np.sqrt(3 * kappa * rd3 / A), rtol=0.02)
        np.testing.assert_allclose(np.log(Sc), np.sqrt(4 * A**3 / (27 * kappa * rd3)), rtol=0.02)


def test_subsaturated_relaxation_reaches_koehler_root():
    """at fixed RH < 1 without feedback the implicit scheme converges to RH = a_w exp(A/r)."""
    for rd, RH in ((20e-9, 0.7), (60e-9, 0.9), (0.15e-6, 0.98)):
        rd3, kappa = rd**3, 0.61
        rv = _rv_for_RH(RH)
        y = (3 * rd) ** 2
        for _ in range(400):
            y, _ill = oracle.cond_substep(y, rd3, kappa, TH, rv, RHOD, 44.0, 0.1)
        np.testing.assert_allclose(_S_eq(np.sqrt(y), rd3, kappa), RH, rtol=1e-12)


def test_large_drop_limit_is_linear_in_r2():
    """for a big dilute drop a_w -> 1, exp(A/r) -> 1, beta -> 1: d r^2/dt constant, so the
    implicit step (eq. 17) equals the explicit one."""
    rd3, kappa, rv = (10e-9) ** 3, 0.61, _rv_for_RH(1.01)
    y0 = (20e-6) ** 2
    f0 = L.orc_growth_f(y0, rd3, kappa, TH, rv, RHOD, 44.0, y0)
    y1, ill = oracle.cond_substep(y0, rd3, kappa, TH, rv, RHOD, 44.0, 0.1)
    assert not ill and f0 > 0
    assert abs((y1 - y0) / (0.1 * f0) - 1) < 2e-3
    # Maxwell-Mason magnitude: r dr/dt = D_eff/rho_w * rho_vs * (S - 1), D_eff ~ O(1e-5) m^2/s
    ct = oracle.cell_thermo(TH, rv, RHOD)
    Deff = f0 * RHO_W / (2 * ct["rho_vs"] * (1.01 - _S_eq(20e-6, rd3, kappa)))
    assert 0.5e-5 < Deff < 2.5e-5


def test_implicit_equation_residual_and_bracket_rules():
    """:568-579 eq. 17-19: the returned value solves y - y0 - dt' f(y) = 0 inside [a, b]; an ill-posed bracket
    returns (a+b)/2 which is the explicit Euler step (:579)."""
    rng = np.random.default_rng(5)
    n_ill = n_ok = 0
    for _ in range(3000):
        rd = np.exp(rng.uniform(np.log(8e-9), np.log(0.5e-6)))
        rd3, kappa = rd**3, 0.61
        r0 = rd * np.exp(rng.uniform(np.log(1.02), np.log(40.0)))
        RH = rng.choice([0.6, 0.95, 1.002, 1.05])
        rv, dtp, y0 = _rv_for_RH(RH), 0.1, r0 * r0
        f0 = L.orc_growth_f(y0, rd3, kappa, TH, rv, RHOD, 44.0, y0)
        y1, ill = oracle.cond_substep(y0, rd3, kappa, TH, rv, RHOD, 44.0, dtp)
        a = max(rd3 ** (2 / 3), y0 + min(2 * dtp * f0, 0))
        b = y0 + max(2 * dtp * f0, 0)
        assert a * (1 - 1e-15) <= y1 <= b * (1 + 1e-15)
        if ill:
            n_ill += 1
            np.testing.assert_allclose(y1, 0.5 * (a + b), rtol=1e-15)
            if a > rd3 ** (2 / 3) * (1 + 1e-12):
                np.testing.assert_allclose(y1, y0 + dtp * f0, rtol=1e-14)  # Euler
        else:
            n_ok += 1
            # g(y) = y - y0 - dt' f(y) changes sign within 2e-12 (relative) of the returned value; closer than
            # that the rounding noise of RH - a_w exp(A/r) in f exceeds |g| (measured ~1e-13 y)
            g = [y - y0 - dtp * L.orc_growth_f(y, rd3, kappa, TH, rv, RHOD, 44.0, y0) for y in (y1 * (1 - 2e-12), y1 * (1 + 2e-12))]
            assert g[0] * g[1] <= 0.0
    assert n_ok > 2000 and n_ill > 0


def test_condensation_conserves_total_water_and_heats():
    """:608-618 eq. 25-26: r_v + (4 pi rho_w/3) sum N r_w^3/(rho_d dV) is constant per cell to rounding."""
    rng = np.random.default_rng(8)
    nx, nz, N = 3, 4, 1500
    o = oracle.Oracle(nx=nx, ny=0, nz=nz, dx=20.0, dy=1.0, dz=20.0, dt=1.0, seed=3)
    ncell = nx * nz
    th0 = np.full(ncell, 289.0)
    rhod = np.linspace(1.15, 1.05, ncell)
    rv0 = np.array([_rv_for_RH(s) for s in np.linspace(0.9, 1.04, ncell)]) * 1.1 / rhod
    o.set_fields(th=th0, rv=rv0, rhod=rhod)
    rd = np.exp(rng.uniform(np.log(10e-9), np.log(0.3e-6), N))
    n = rng.integers(10**6, 10**9, N).astype(np.uint64)
    x, z = rng.uniform(0, 60, N), rng.uniform(0, 80, N)
    o.set_state(n, (2 * rd) ** 2, rd**3, np.full(N, 0.61), x=x, z=z)
    cell = np.floor(x / 20).astype(int) * nz + np.floor(z / 20).astype(int)
    dV = 20.0 * 1.0 * 20.0

    def water(rv, st):
        liq = np.bincount(cell, weights=st["n"].astype(float) * st["rw2"] ** 1.5, minlength=ncell)
        return rv + 4 * np.pi * RHO_W / 3 * liq / (rhod * dV)

    w0 = water(rv0, o.get_state())
    op = oracle.make_opts(adve=False, sedi=False, cond=True, coal=False, RH_max=1.05, sstp_cond=10)
    for _ in range(5):
        o.step(op)
    th1, rv1 = o.get_fields()
    w1 = water(rv1, o.get_state())
    np.testing.assert_allclose(w1, w0, rtol=2e-14)
    assert np.abs(rv1 - rv0).max() > 1e-6  # something did condense / evaporate
    # eq. 26: d theta = -theta l_v/(c_pd T) d r_v
    T = np.array([L.orc_T(t, r) for t, r in zip(th0, rhod)])
    lv = np.array([L.orc_lv(t) for t in T])
    np.testing.assert_allclose((th1 - th0) / (rv1 - rv0), -th0 * lv / (C_PD * T), rtol=2e-3)
    assert o.counters()["sd_substeps"] == 5 * 10 * N


def test_adaptive_condensation_substeps_rule_limits_and_water_budget():
    """DESIGN.md reading R-adapt (PAPER.md :566 "An adaptive timestep choice mechanism is planned"): a cell takes the
    smallest divisor d of sstp_cond with d >= sstp_cond eps / tol, eps = |d r_v| / (r_v max(|RH - 1|, 1e-3)) with d r_v the
    vapour one explicit step of the cell's growth rates would take up (eq. 25, d(r_w^3) = (3/2) r_w dt f).  Pinned by
    (i) the limits: tol -> 0 is the fixed-substep step bit for bit, tol -> infinity is one substep per cell; (ii) the
    rule restated here on the growth rates (themselves pinned above) predicts every cell's substep count, and the
    counts span 1, 2, 5, 10; (iii) condensation is cell-local, so each cell must end exactly where the fixed-substep
    oracle with sstp_cond = d ends it; (iv) the water budget of eq. 25 holds whatever the counts are."""
    from tests import pin_helpers as _ph

    rng = np.random.default_rng(18)
    nx, nz, N, sstp, dt = 4, 6, 2400, 10, 1.0
    ncell = nx * nz
    th0 = np.full(ncell, 289.0)
    rhod = np.linspace(1.15, 1.05, ncell)
    # from dry air to a 4 % supersaturation: haze in equilibrium below, activating droplets above
    rv0 = np.array([_rv_for_RH(s) for s in np.linspace(0.80, 1.04, ncell)]) * 1.1 / rhod
    rd = np.exp(rng.uniform(np.log(10e-9), np.log(0.3e-6), N))
    x, z = rng.uniform(0, 20.0 * nx, N), rng.uniform(0, 20.0 * nz, N)
    cell = np.floor(x / 20).astype(int) * nz + np.floor(z / 20).astype(int)
    # fewer real particles per SD in the lower of the moist cells: their uptake, and with it eps, then spans two decades
    n = (rng.integers(10**6, 10**9, N) * 10.0 ** np.clip(-1.5 + 0.15 * (cell - 12), -1.5, 0.0)).astype(np.uint64)
    ct = [oracle.cell_thermo(th0[q], rv0[q], rhod[q]) for q in range(ncell)]
    rw = np.array([_ph.equilibrium_rw_brentq(rd[i] ** 3, 0.61, min(0.95, ct[cell[i]]["RH"]), ct[cell[i]]["T"]) for i in range(N)])
    # off equilibrium by 1e-7 (lowest cell) to 1e-2 (highest), so that eps spans decades
    rw = rw * np.exp(rng.normal(0.0, 1.0, N) * 10.0 ** (-7.0 + 5.0 * cell / (ncell - 1)))

    def run(steps=1, **kw):
        o = oracle.Oracle(nx=nx, ny=0, nz=nz, dx=20.0, dy=1.0, dz=20.0, dt=dt, seed=3)
        o.set_fields(th=th0, rv=rv0, rhod=rhod)
        o.set_state(n, rw**2, rd**3, np.full(N, 0.61), x=x, z=z)
        op = oracle.make_opts(adve=False, sedi=False, cond=True, coal=False, RH_max=1.05, **kw)
        for _ in range(steps):
            o.step(op)
        st = o.get_state()
        order = np.argsort(st["id"])
        return {k: v[order] for k, v in st.items()}, o.get_fields(), o.counters()

    fixed = {d: run(sstp_cond=d) for d in (1, 2, 5, 10)}
    # (i) limits
    for tol, d in ((1e-300, 10), (1e300, 1)):
        st, (th, rv), cnt = run(sstp_cond=sstp, cond_adapt_tol=tol)
        np.testing.assert_array_equal(st["rw2"], fixed[d][0]["rw2"])
        np.testing.assert_array_equal(rv, fixed[d][1][1])
        assert cnt["sd_substeps"] == d * N
    # (ii) the rule, restated: eps per cell from the growth rates at the start of the step
    tol = 0.006
    f0 = np.array([L.orc_growth_f(rw[i] ** 2, rd[i] ** 3, 0.61, th0[cell[i]], rv0[cell[i]], rhod[cell[i]], 1.05, rw[i] ** 2) for i in range(N)])
    est = np.bincount(cell, weights=n.astype(float) * 1.5 * rw * dt * f0, minlength=ncell)
    RH = np.array([min(c["RH"], 1.05) for c in ct])
    eps = 4 * np.pi * RHO_W / 3 / (rhod * 20.0 * 1.0 * 20.0) * np.abs(est) / (rv0 * np.maximum(np.abs(RH - 1.0), 1e-3))
    want = sstp * eps / tol
    n_c = np.array([next((d for d in (1, 2, 5) if d >= w), 10) for w in want])
    assert set(n_c) == {1, 2, 5, 10}, (np.bincount(n_c), want)   # the case exercises every count
    assert min(np.abs(want - d).min() for d in (1, 2, 5)) > 1e-6   # no cell sits on a threshold
    st, (th, rv), cnt = run(sstp_cond=sstp, cond_adapt_tol=tol)
    assert cnt["sd_substeps"] == int(np.sum(n_c[cell]))
    # (iii) every cell ends where the fixed-substep oracle with its own count ends it
    for d in (1, 2, 5, 10):
        m = n_c[cell] == d
        np.testing.assert_array_equal(st["rw2"][m], fixed[d][0]["rw2"][m])
        np.testing.assert_array_equal(rv[n_c == d], fixed[d][1][1][n_c == d])
        np.testing.assert_array_equal(th[n_c == d], fixed[d][1][0][n_c == d])
    # (iv) eq. 25 over five adaptive steps
    dV = 20.0 * 1.0 * 20.0
    st5, (th5, rv5), _ = run(steps=5, sstp_cond=sstp, cond_adapt_tol=tol)
    liq0 = np.bincount(cell, weights=n.astype(float) * rw**3, minlength=ncell)
    liq5 = np.bincount(cell, weights=st5["n"].astype(float) * st5["rw2"] ** 1.5, minlength=ncell)
    np.testing.assert_allclose(rv5 + 4 * np.pi * RHO_W / 3 * liq5 / (rhod * dV), rv0 + 4 * np.pi * RHO_W / 3 * liq0 / (rhod * dV), rtol=2e-14)
    assert np.abs(rv5 - rv0).max() > 1e-6


# ----------------------------------------------------------------------------- Eulerian transport (Fig. 7 prototype solver)
def test_upstream_step_is_the_textbook_donor_cell_scheme():
    """PAPER.md :219-235 (upstream scheme), Figure 7 (:831-852): the Eulerian step the host model takes between step_sync
    and the next one.  Pinned by what the donor-cell scheme is known to do: a Courant number of +1 / -1 shifts the field
    by exactly one cell down / up the axis, 1/2 averages a cell with its upwind neighbour, the flux form conserves
    sum(rho_d psi) on the periodic domain, and a constant field is a fixed point of a discretely non-divergent flow."""
    rng = np.random.default_rng(23)
    # 1D along x: rho_d = 1, so the array holds plain Courant numbers
    nx = 17
    psi = rng.uniform(1.0, 2.0, nx)
    for C, expect in ((1.0, np.roll(psi, 1)), (-1.0, np.roll(psi, -1)), (0.5, 0.5 * psi + 0.5 * np.roll(psi, 1)),
                      (-0.25, 0.75 * psi + 0.25 * np.roll(psi, -1))):
        o = oracle.Oracle(nx=nx, ny=0, nz=0, dx=1.0, dy=1.0, dz=1.0, dt=1.0)
        o.set_fields(th=np.ones(nx), rv=np.ones(nx), rhod=np.ones(nx), cx=np.full(nx + 1, C))
        np.testing.assert_allclose(o.upstream_advect(psi), expect, rtol=1e-15)
    # 3D: a non-divergent flow from two stream functions differenced on the C-grid, rho_d varying with height
    nx, ny, nz = 6, 5, 7
    psi1, psi2 = rng.normal(size=(nx + 1, nz + 1)), rng.normal(size=(ny + 1, nz + 1))
    psi1[-1], psi2[-1] = psi1[0], psi2[0]                         # periodic in x and y
    psi1[:, 0] = psi1[:, -1] = psi2[:, 0] = psi2[:, -1] = 0.0     # no flow through bottom and top
    cx = np.broadcast_to((-0.2 * (psi1[:, 1:] - psi1[:, :-1]))[:, None, :], (nx + 1, ny, nz))
    cy = np.broadcast_to((-0.2 * (psi2[:, 1:] - psi2[:, :-1]))[None, :, :], (nx, ny + 1, nz))
    cz = 0.2 * ((psi1[1:, :] - psi1[:-1, :])[:, None, :] + (psi2[1:, :] - psi2[:-1, :])[None, :, :])
    rhod = np.broadcast_to(np.linspace(1.2, 1.0, nz), (nx, ny, nz)).ravel().copy()
    o = oracle.Oracle(nx=nx, ny=ny, nz=nz, dx=1.0, dy=1.0, dz=1.0, dt=1.0)
    o.set_fields(th=np.ones(nx * ny * nz), rv=np.ones(nx * ny * nz), rhod=rhod, cx=cx.ravel(), cy=cy.ravel(), cz=cz.ravel())
    f = rng.uniform(280.0, 300.0, nx * ny * nz)
    g = o.upstream_advect(f)
    assert np.abs(g - f).max() > 1e-3                             # the field did move
    np.testing.assert_allclose(np.sum(rhod * g), np.sum(rhod * f), rtol=1e-14)
    const = np.full(nx * ny * nz, 289.0)
    np.testing.assert_allclose(o.upstream_advect(const), const, rtol=1e-14)
    # a y-only and a z-only shift, to pin the index arithmetic of every dimension
    for dim, shift_axis in (("y", 1), ("z", 2)):
        kw = dict(cx=np.zeros((nx + 1) * ny * nz), cy=np.zeros(nx * (ny + 1) * nz), cz=np.zeros(nx * ny * (nz + 1)))
        kw["c" + dim] = np.ones_like(kw["c" + dim])
        o.set_fields(th=const, rv=const, rhod=np.ones(nx * ny * nz), **kw)
        h = o.upstream_advect(f).reshape(nx, ny, nz)
        f3 = f.reshape(nx, ny, nz)
        if dim == "y":
            np.testing.assert_allclose(h, np.roll(f3, 1, axis=1), rtol=1e-15)
        else:   # not periodic in z: the boundary value enters at the bottom
            np.testing.assert_allclose(h[:, :, 1:], f3[:, :, :-1], rtol=1e-15)
            np.testing.assert_allclose(h[:, :, 0], f3[:, :, 0], rtol=1e-15)


# ----------------------------------------------------------------------------- advection / sedimentation
def test_advection_closed_form_solves_backward_euler():
    """:536-556: eq. 16 is the solution of eq. 13-15."""
    rng = np.random.default_rng(2)
    for _ in range(200):
        dx = rng.uniform(5, 50)
        i = rng.integers(0, 70)
        x = (i + rng.uniform(0, 1)) * dx
        Clo, Chi = rng.uniform(-0.3, 0.3, 2)
        xn = L.orc_adve_1d(x, dx, Clo, Chi)
        omega = xn / dx - np.floor(x / dx)  # eq. 15
        C = (1 - omega) * Clo + omega * Chi  # eq. 14
        assert abs(xn - (x + dx * C)) < 1e-12 * dx * 70  # eq. 13
        np.testing.assert_allclose(L.orc_adve_1d(x, dx, Clo, Clo), x + dx * Clo, rtol=1e-15)  # dC = 0
    # a wall with C = 0 is never crossed
    for x in (0.01, 5.0, 9.99):
        assert L.orc_adve_1d(x, 10.0, 0.0, -0.5) >= 0.0
        assert L.orc_adve_1d(x, 10.0, 0.5, 0.0) <= 10.0


def test_move_stage_matches_eq16_per_dimension_and_sediments():
    rng = np.random.default_rng(4)
    nx, nz, N = 5, 4, 300
    dx, dz, dt = 10.0, 20.0, 1.0
    o = oracle.Oracle(nx=nx, ny=0, nz=nz, dx=dx, dy=1.0, dz=dz, dt=dt, seed=1)
    rhod = rng.uniform(1.0, 1.2, nx * nz)
    cx = rng.uniform(-0.2, 0.2, (nx + 1, nz))
    cx[-1] = cx[0]
    cz = rng.uniform(-0.1, 0.1, (nx, nz + 1))
    cz[:, 0] = cz[:, -1] = 0
    o.set_fields(th=np.full(nx * nz, 289.0), rv=np.full(nx * nz, 7e-3), rhod=rhod, cx=cx.ravel(), cz=cz.ravel())
    x, z = rng.uniform(0, nx * dx, N), rng.uniform(0, nz * dz, N)
    r = np.exp(rng.uniform(np.log(1e-6), np.log(1e-3), N))
    z[:40] = rng.uniform(0, 3.0, 40)
    r[:40] = 1e-3  # big drops near the ground will fall out
    n = rng.integers(1, 10**6, N).astype(np.uint64)
    o.set_state(n, r * r, np.full(N, 1e-24), np.full(N, 0.61), x=x, z=z)
    op = oracle.make_opts(adve=True, sedi=True, cond=False, coal=False)
    flux = o.step(op)
    st = o.get_state()
    i, k = np.floor(x / dx).astype(int), np.floor(z / dz).astype(int)
    rd_ = rhod.reshape(nx, nz)[i, k]
    xe = np.array([L.orc_adve_1d(a, dx, lo / q, hi / q) for a, lo, hi, q in zip(x, cx[i, k], cx[i + 1, k], rd_)])
    ze = np.array([L.orc_adve_1d(a, dz, lo / q, hi / q) for a, lo, hi, q in zip(z, cz[i, k], cz[i, k + 1], rd_)])
    T = L.orc_T(289.0, 1.0)
    vt = np.array([L.orc_vterm(rr, L.orc_T(289.0, q), q, 7e-3) for rr, q in zip(r, rd_)])
    ze = ze - vt * dt
    xe = np.where(xe < 0, xe + nx * dx, xe)
    xe = np.where(xe >= nx * dx, xe - nx * dx, xe)
    np.testing.assert_allclose(st["x"], xe, rtol=1e-14)
    np.testing.assert_allclose(st["z"], ze, rtol=1e-13, atol=1e-13)
    out = ze < 0
    assert out.sum() >= 30 and (st["n"][out] == 0).all() and (st["n"][~out] == n[~out]).all()
    np.testing.assert_allclose(flux, (n[out] * 4 / 3 * np.pi * RHO_W * r[out] ** 3).sum(), rtol=1e-13)
    # next step compacts the dead ones away, stably
    o.step(oracle.make_opts(adve=False, sedi=False, cond=False, coal=False))
    assert o.get_state()["id"].tolist() == np.nonzero(~out)[0].tolist()


def test_move_stage_3d_indexes_every_courant_component():
    """:534-556 eq. 16 in three dimensions with the C-grid shapes of :751 ((nx+1) x ny x nz, nx x (ny+1) x nz,
    nx x ny x (nz+1)), all different sizes so that a transposed or mis-strided index picks a different number;
    every component random in all three directions; periodic in x and y (:558)."""
    rng = np.random.default_rng(14)
    nx, ny, nz, N = 5, 3, 4, 600
    dx, dy, dz, dt = 10.0, 7.0, 20.0, 1.0
    o = oracle.Oracle(nx=nx, ny=ny, nz=nz, dx=dx, dy=dy, dz=dz, dt=dt, seed=1)
    rhod = rng.uniform(1.0, 1.2, (nx, ny, nz))
    cx = rng.uniform(-0.3, 0.3, (nx + 1, ny, nz))
    cy = rng.uniform(-0.3, 0.3, (nx, ny + 1, nz))
    cz = rng.uniform(-0.1, 0.1, (nx, ny, nz + 1))
    cz[:, :, 0] = cz[:, :, -1] = 0
    o.set_fields(th=np.full(rhod.size, 289.0), rv=np.full(rhod.size, 7e-3), rhod=rhod.ravel(), cx=cx.ravel(), cy=cy.ravel(),
                 cz=cz.ravel())
    x, y, z = rng.uniform(0, nx * dx, N), rng.uniform(0, ny * dy, N), rng.uniform(0, nz * dz, N)
    n = rng.integers(1, 10**6, N).astype(np.uint64)
    o.set_state(n, np.full(N, (5e-6) ** 2), np.full(N, 1e-24), np.full(N, 0.61), x=x, y=y, z=z)
    o.step(oracle.make_opts(adve=True, sedi=False, cond=False, coal=False))
    st = o.get_state()
    i, j, k = np.floor(x / dx).astype(int), np.floor(y / dy).astype(int), np.floor(z / dz).astype(int)
    q = rhod[i, j, k]

    def eq16(a, d, idx, lo, hi):      # backward Euler with the Courant number interpolated to the NEW position
        dC = hi - lo
        return (a + d * (lo - idx * dC)) / (1 - dC)

    xe = eq16(x, dx, i, cx[i, j, k] / q, cx[i + 1, j, k] / q)
    ye = eq16(y, dy, j, cy[i, j, k] / q, cy[i, j + 1, k] / q)
    ze = eq16(z, dz, k, cz[i, j, k] / q, cz[i, j, k + 1] / q)
    om = xe / dx - i                                               # eq. 13-15 hold at the new position
    np.testing.assert_allclose(xe, x + dx * ((1 - om) * cx[i, j, k] + om * cx[i + 1, j, k]) / q, rtol=1e-13)
    om = ye / dy - j
    np.testing.assert_allclose(ye, y + dy * ((1 - om) * cy[i, j, k] + om * cy[i, j + 1, k]) / q, rtol=1e-13)
    om = ze / dz - k
    np.testing.assert_allclose(ze, z + dz * ((1 - om) * cz[i, j, k] + om * cz[i, j, k + 1]) / q, rtol=1e-13, atol=1e-12)
    xe = np.where(xe < 0, xe + nx * dx, np.where(xe >= nx * dx, xe - nx * dx, xe))
    ye = np.where(ye < 0, ye + ny * dy, np.where(ye >= ny * dy, ye - ny * dy, ye))
    assert (np.abs(xe - x) > 1.0).sum() > N // 2 and ((xe < x - 20) | (xe > x + 20)).sum() > 0    # wraps happened
    np.testing.assert_allclose(st["x"], xe, rtol=1e-14)
    np.testing.assert_allclose(st["y"], ye, rtol=1e-14)
    np.testing.assert_allclose(st["z"], ze, rtol=1e-14, atol=1e-13)
    assert (st["n"] == n).all()


# ----------------------------------------------------------------------------- diagnostics / table / threads
def test_moments_bruteforce():
    """:818-823 eq. 29."""
    rng = np.random.default_rng(6)
    nx, ny, nz, N = 3, 2, 4, 2000
    o = oracle.Oracle(nx=nx, ny=ny, nz=nz, dx=10.0, dy=5.0, dz=20.0, dt=1.0)
    rhod = rng.uniform(1.0, 1.2, nx * ny * nz)
    o.set_fields(rhod=rhod)
    x, y, z = rng.uniform(0, 30, N), rng.uniform(0, 10, N), rng.uniform(0, 80, N)
    rw, rd = np.exp(rng.uniform(np.log(1e-7), np.log(1e-4), N)), np.exp(rng.uniform(np.log(1e-9), np.log(1e-6), N))
    n = rng.integers(0, 1000, N).astype(np.uint64)
    o.set_state(n, rw**2, rd**3, np.full(N, 0.61), x=x, y=y, z=z)
    cell = (np.floor(x / 10).astype(int) * ny + np.floor(y / 5).astype(int)) * nz + np.floor(z / 20).astype(int)
    dV = 10.0 * 5.0 * 20.0
    for wet, r in ((1, rw), (0, rd)):
        for k in (0, 1, 3):
            lo, hi = np.quantile(r, [0.2, 0.7])
            m = (r >= lo) & (r < hi)
            ref = np.zeros(nx * ny * nz)
            for s in np.nonzero(m)[0]:
                ref[cell[s]] += float(n[s]) * r[s] ** k
            np.testing.assert_allclose(o.diag_mom(wet, lo, hi, k), ref / (rhod * dV), rtol=1e-13)
    np.testing.assert_array_equal(o.diag_sd_conc(), np.bincount(cell[n > 0], minlength=nx * ny * nz))


def test_efficiency_table_bilinear_and_clamped():
    R = np.array([10e-6, 20e-6, 40e-6])
    q = np.array([0.0, 0.5, 1.0])
    tab = np.array([[0.0, 0.1, 0.2], [0.3, 0.5, 0.7], [1.0, 1.0, 0.9]])
    o = oracle.Oracle(dx=1, dy=1, dz=1, kernel="hydro_tab", eff_R=R, eff_q=q, eff_tab=tab)
    for a in range(3):
        for c in range(3):
            assert abs(o.eff(R[a], q[c]) - tab[a, c]) < 1e-15
    np.testing.assert_allclose(o.eff(15e-6, 0.25), tab[:2, :2].mean(), rtol=1e-14)
    np.testing.assert_allclose(o.eff(30e-6, 0.5), 0.75, rtol=1e-14)
    assert o.eff(1e-6, 0.5) == o.eff(10e-6, 0.5) and o.eff(1e-3, 2.0) == tab[2, 2]


def test_openmp_over_cells_is_bitwise_identical_to_serial():
    rng = np.random.default_rng(21)
    nx, nz, N = 6, 6, 3000
    res = []
    for threads in (1, 4):
        o = oracle.Oracle(nx=nx, ny=0, nz=nz, dx=20.0, dy=1.0, dz=20.0, dt=1.0, seed=9)
        o.set_threads(threads)
        rr = np.random.default_rng(21)
        rd = np.exp(rr.uniform(np.log(10e-9), np.log(0.3e-6), N))
        o.set_fields(th=np.full(36, 289.0), rv=np.full(36, 9e-3), rhod=np.full(36, 1.1))
        o.set_state(rr.integers(10**6, 10**9, N).astype(np.uint64), (30 * rd) ** 2, rd**3, np.full(N, 0.61),
                    x=rr.uniform(0, 120, N), z=rr.uniform(0, 120, N))
        op = oracle.make_opts(RH_max=1.05)
        for _ in range(3):
            o.step(op)
        res.append((o.get_state(), o.get_fields()))
    for k in res[0][0]:
        np.testing.assert_array_equal(res[0][0][k], res[1][0][k])
    np.testing.assert_array_equal(res[0][1][0], res[1][1][0])


# ------------------------------------------------------------------------------ initialisation (section 5.1.6)
# These pins import nothing from the product package: the environment and the second statement of each rule come
# from tests/pin_helpers.py (numpy + scipy).
from tests import pin_helpers as H   # noqa: E402

VOCALS = H.VOCALS   # PAPER.md :117-130 (mode diameters 0.04, 0.15 um)


def _init_case(sd=64, nx=6, nz=75, seed=5, modes=VOCALS):
    """A 2D column set-up (cells of 20 m x 1 m x 20 m, theta = 289 K, r_v = 7.5 g/kg, hydrostatic rho_d, :115)
    initialised by the oracle's init().  Returns (rho_d(z), oracle, N, ranges, state)."""
    o = oracle.Oracle(nx=nx, ny=0, nz=nz, dx=20.0, dy=1.0, dz=20.0, dt=1.0, seed=seed)
    th, rv, rhod, rz = H.column_fields(nx, nz)
    o.set_fields(th=th, rv=rv, rhod=rhod)
    N, ranges = o.init(modes, float(sd))
    return rz, o, N, ranges, o.get_state()


def test_init_range_rule_and_agreement_with_root_finding():
    """:657: the multiplicity at both ends of the r_d range is >= 1 and just outside it is < 1; the limits equal
    the outermost roots of n(ln r)(hi - lo)/sd_conc dV = 1 found by brentq on the continuous density, to the
    oracle's grid step."""
    rz, o, N, ranges, s = _init_case()
    lo, hi = ranges[0]
    assert N == 64 * 6 * 75 and len(ranges) == 1
    step = (np.log(1e-4) - np.log(1e-10)) / 200000
    rlo, rhi = H.rd_range_by_root_finding(VOCALS, 64.0, 20.0 * 1.0 * 20.0)
    assert rlo - 1e-9 <= lo <= rlo + 2 * step and rhi - 2 * step <= hi <= rhi + 1e-9
    assert 1e-9 < np.exp(lo) < 5e-9 and 1e-6 < np.exp(hi) < 3e-6      # about 2 nm .. 1.7 um

    def mult(lnr):   # eq. 3 written out again, at STP density
        dens = sum(n / (np.sqrt(2 * np.pi) * np.log(sg)) * np.exp(-(lnr - np.log(rm)) ** 2 / (2 * np.log(sg) ** 2))
                   for _, n, rm, sg in VOCALS)
        return dens * (hi - lo) / 64.0 * (20.0 * 1.0 * 20.0)

    assert mult(lo) >= 1.0 and mult(hi) >= 1.0 and mult(lo - step) < 1.0 and mult(hi + step) < 1.0


def test_init_positions_sizes_and_total_concentration():
    """:655 uniform positions, :657 log-uniform dry radii inside the range, :659 the SDs of a cell add up to the
    spectrum's total concentration scaled by rho_d / rho_STP (Monte-Carlo: within 5 standard errors)."""
    rhod, o, N, ranges, s = _init_case(sd=128, nx=8)
    lo, hi = ranges[0]
    X, Z = 8 * 20.0, 75 * 20.0
    assert s["x"].min() >= 0 and s["x"].max() < X and s["z"].min() >= 0 and s["z"].max() < Z
    assert abs(s["x"].mean() / X - 0.5) < 5 / np.sqrt(12 * N) and abs(s["z"].mean() / Z - 0.5) < 5 / np.sqrt(12 * N)
    lnr = np.log(s["rd3"]) / 3
    assert lnr.min() >= lo - 1e-12 and lnr.max() <= hi + 1e-12
    assert abs((lnr.mean() - lo) / (hi - lo) - 0.5) < 5 / np.sqrt(12 * N)
    np.testing.assert_array_equal(s["id"], np.arange(N, dtype=np.uint32))
    assert np.all(s["kappa"] == 0.61) and s["n"].min() >= 1
    # total concentration: integral of eq. 3 over the range (erf closed form) x <rho_d>/rho_STP
    from math import erf, log, sqrt
    tot = sum(n * 0.5 * (erf((hi - log(rm)) / (sqrt(2) * log(sg))) - erf((lo - log(rm)) / (sqrt(2) * log(sg))))
              for _, n, rm, sg in VOCALS)
    rho_stp = 101325.0 / (287.0 * 293.15)
    k = np.clip((s["z"] / 20.0).astype(int), 0, 74)
    expect = tot * rhod.mean() / rho_stp
    got = s["n"].sum() / (X * 1.0 * Z)
    # per-SD weights n_i have a wide distribution: standard error from the sample itself
    se = np.sqrt(N * np.var(s["n"].astype(np.float64))) / (X * Z)
    assert abs(got - expect) < 5 * se and se < 0.05 * expect
    # multiplicity of one SD follows the formula of :659 with its own cell's density
    i = int(np.argmax(s["n"]))
    dens = sum(n / (np.sqrt(2 * np.pi) * np.log(sg)) * np.exp(-(lnr[i] - np.log(rm)) ** 2 / (2 * np.log(sg) ** 2)) for _, n, rm, sg in VOCALS)
    assert s["n"][i] == np.floor(dens * (hi - lo) / 128.0 * 400.0 * rhod[k[i]] / rho_stp + 0.5)


def test_init_wet_radius_is_the_koehler_equilibrium_at_min_rh_095():
    """:661-665: zero growth rate (RH = a_w exp(A/r)) at the cell's RH, capped at 0.95; the root lies on the stable
    branch below the critical radius; agrees with scipy's brentq on the Koehler curve (tests/pin_helpers.py)."""
    rhod, o, N, ranges, s = _init_case(sd=32, nx=4)
    k = np.clip((s["z"] / 20.0).astype(int), 0, 74)
    T = np.array([oracle.cell_thermo(289.0, 7.5e-3, float(r))["T"] for r in rhod])
    RH = np.array([oracle.cell_thermo(289.0, 7.5e-3, float(r))["RH"] for r in rhod])
    A = 2 * 0.072 / (461.5 * T * 1000.0)
    r = np.sqrt(s["rw2"])
    r3 = r ** 3
    S = (r3 - s["rd3"]) / (r3 - s["rd3"] * (1 - 0.61)) * np.exp(A[k] / r)
    np.testing.assert_allclose(S, np.minimum(RH[k], 0.95), rtol=1e-11)
    assert np.all(r > np.cbrt(s["rd3"])) and np.all(r < np.sqrt(3 * 0.61 * s["rd3"] / A[k]))
    assert RH.max() > 1.0 and RH.min() < 0.7          # the profile spans clear and (super)saturated air
    pick = np.random.default_rng(0).choice(N, 1500, replace=False)
    ref = np.array([H.equilibrium_rw_brentq(float(s["rd3"][i]), 0.61, float(min(RH[k[i]], 0.95)), float(T[k[i]])) for i in pick])
    np.testing.assert_allclose(r[pick], ref, rtol=1e-9)


def test_init_external_mixture_shares_the_sds_between_kappas():
    """:659 "externally mixed aerosol ... multiple spectra, each characterised by different kappa": SD i belongs to
    spectrum i mod G, each spectrum has its own range and its SDs reproduce its own concentration."""
    modes = [(0.61, 60e6, 0.02e-6, 1.4), (1.28, 40e6, 0.075e-6, 1.6)]
    rhod, o, N, ranges, s = _init_case(sd=128, nx=8, modes=modes)
    assert len(ranges) == 2 and ranges[0] != ranges[1]
    assert np.all(s["kappa"][0::2] == 0.61) and np.all(s["kappa"][1::2] == 1.28)
    from math import erf, log, sqrt
    rho_ratio = rhod.mean() / (101325.0 / (287.0 * 293.15))
    for g, (kap, n, rm, sg) in enumerate(modes):
        lo, hi = ranges[g]
        tot = n * 0.5 * (erf((hi - log(rm)) / (sqrt(2) * log(sg))) - erf((lo - log(rm)) / (sqrt(2) * log(sg))))
        ng = s["n"][g::2].astype(np.float64)
        got = ng.sum() / (160.0 * 1500.0)
        se = np.sqrt(len(ng) * np.var(ng)) / (160.0 * 1500.0)
        assert abs(got - tot * rho_ratio) < 5 * se
