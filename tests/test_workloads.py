"""CPU checks of the seeded input generators."""
import math

import torch

from paper_1310_1905_b200 import workloads as W


def test_hydrostatic_profile_values():
    # SURVEY.md 8d [S]: z = 10 m: T 289.14, rhod 1.2071, RH 0.665; z = 810 m: RH 1.009; z = 1490 m: T 274.76, rhod 1.0625, RH 1.47
    p = W.hydrostatic_profile(torch.tensor([10.0, 810.0, 1490.0], dtype=torch.float64))
    assert torch.allclose(p["T"][[0, 2]], torch.tensor([289.14, 274.76], dtype=torch.float64), atol=0.01)
    assert torch.allclose(p["rhod"][[0, 2]], torch.tensor([1.2071, 1.0625], dtype=torch.float64), atol=1e-4)
    assert torch.allclose(p["RH"], torch.tensor([0.665, 1.009, 1.47], dtype=torch.float64), atol=2e-3)
    # hydrostatic balance of the total pressure: dp/dz = -g rho_d (1 + rv)
    z = torch.linspace(0, 1500, 3001, dtype=torch.float64)
    q = W.hydrostatic_profile(z)
    pres = q["rhod"] * (W.R_D + 7.5e-3 * W.R_V) * q["T"]
    dpdz = (pres[2:] - pres[:-2]) / (z[2:] - z[:-2])
    assert torch.allclose(dpdz, -W.G_ACC * q["rhod"][1:-1] * (1 + 7.5e-3), rtol=1e-5)
    assert abs(float(pres[0]) - 101500.0) < 1e-6


def test_2d_setup_is_nondivergent_and_periodic():
    w = W.cfg2_2d(sd_per_cell=32)
    c1, c2 = w.courants
    assert c1.shape == (76, 75) and c2.shape == (75, 76)   # PAPER.md :751
    div = (c1[1:] - c1[:-1]) + (c2[:, 1:] - c2[:, :-1])
    assert div.abs().max() < 1e-16
    assert (c1[0] - c1[-1]).abs().max() == 0 and c2[:, 0].abs().max() < 1e-16 and c2[:, -1].abs().max() < 1e-16
    assert 0.029 < c1.abs().max() < 0.031 and 0.059 < c2.abs().max() < 0.061   # SURVEY.md 8d [S]
    lo, hi = w.meta["rd_range"]
    assert 1e-9 < lo < 3e-9 and 1e-6 < hi < 2.5e-6
    s = w.state
    assert s["n"].min() >= 1 and 4e9 < s["n"].max() < 8e9
    # total concentration ~ (60 + 40) cm^-3 scaled by rhod/rho_STP
    conc = s["n"].sum().item() / (1500.0 * 1500.0 * 1.0)
    assert 0.85e8 < conc < 1.0e8
    assert ((s["rw2"].sqrt() ** 3) > s["rd3"]).all()
    assert (s["x"] >= 0).all() and (s["x"] < 1500).all() and (s["z"] >= 0).all() and (s["z"] < 1500).all()


def test_3d_setup_is_nondivergent():
    w = W.cfg4_3d(sd_per_cell=2, nx=8, ny=6, nz=16)
    c1, c2, c3 = w.courants
    assert c1.shape == (9, 6, 16) and c2.shape == (8, 7, 16) and c3.shape == (8, 6, 17)
    div = (c1[1:] - c1[:-1]) + (c2[:, 1:] - c2[:, :-1]) + (c3[:, :, 1:] - c3[:, :, :-1])
    assert div.abs().max() < 1e-16
    assert c3[:, :, 0].abs().max() < 1e-16 and c3[:, :, -1].abs().max() < 1e-16


def test_generators_are_deterministic_and_hash_is_uniform():
    a, b = W.cfg2_2d(sd_per_cell=2, seed=7), W.cfg2_2d(sd_per_cell=2, seed=7)
    for k in ("n", "rw2", "rd3", "x", "z"):
        assert torch.equal(a.state[k], b.state[k])
    c = W.cfg2_2d(sd_per_cell=2, seed=8)
    assert not torch.equal(a.state["x"], c.state["x"])
    u = W.hash_uniform(3, 5, torch.arange(400000))
    assert abs(u.mean().item() - 0.5) < 3e-3 and abs(u.var().item() * 12 - 1) < 1e-2 and 0 < u.min() and u.max() < 1
    # chunked generation gives the same numbers
    assert torch.equal(u[1000:2000], W.hash_uniform(3, 5, torch.arange(1000, 2000)))


def test_box_and_table():
    w = W.box_golovin(seed=42)
    v = 4 / 3 * math.pi * w.state["rw2"] ** 1.5
    assert abs(v.mean().item() / w.meta["v0"] - 1) < 0.04
    assert w.state["n"][0].item() == 2**23 * 10**6 // 2**13
    R, q, E = W.efficiency_table_standin()
    assert E.shape == (15, 21) and E.min() >= 0 and E.max() <= 1 and (E[-1] == 1).all() and (E[:, 0] == 0)[:5].all()
