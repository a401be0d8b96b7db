"""Seeded synthetic inputs for the configurations of BASELINE.json (recipe: DESIGN.md "Input recipe").

This module serves both the oracle-side tests and the CUDA path with the SAME arrays.  It holds none
of the time-step arithmetic of the method (no Philox, no growth/coalescence/advection code): it only
builds initial conditions -- thermodynamic profiles, Courant fields, aerosol populations in
equilibrium with their environment (PAPER.md :101-138, :653-665) -- and imports neither ``oracle``
nor the binding.  All randomness comes from a counter-based hash of (seed, stream, index), so the
numbers do not depend on the device, the chunking or the order of generation.

Everything is torch; pass ``device="cuda"`` to generate large populations on the GPU.
"""
import math
from dataclasses import dataclass, field

import torch

F64 = torch.float64

# physical constants used ONLY to set up initial conditions (same literature values as DESIGN.md lists)
R_D, R_V, C_PD, C_PV, C_L = 287.0, 461.5, 1005.0, 1850.0, 4218.0
L_V0, T_0, P_VS0, P_1000, G_ACC = 2.5e6, 273.16, 611.73, 1.0e5, 9.81
RHO_W, SIGMA_W = 1000.0, 0.072
RHO_STP = 101325.0 / (R_D * 293.15)   # PAPER.md :130 "standard conditions (T=20C and p=1013.25 hPa)"


def _i64(v):
    v &= (1 << 64) - 1
    return v - (1 << 64) if v >= (1 << 63) else v


_C1, _C2, _C3 = _i64(0x9E3779B97F4A7C15), _i64(0xBF58476D1CE4E5B9), _i64(0x94D049BB133111EB)


def _lsr(z, k):
    return (z >> k) & ((1 << (64 - k)) - 1)


def hash_uniform(seed, stream, idx):
    """Uniform (0,1) doubles from a splitmix64-style hash of (seed, stream, idx); idx: int64 tensor."""
    z = idx * _C1 + _i64((seed * 0xD1342543DE82EF95 + stream * 0xA24BAED4963EE407 + 0x632BE59BD9B4E019))
    z = (z ^ _lsr(z, 30)) * _C2
    z = (z ^ _lsr(z, 27)) * _C3
    z = z ^ _lsr(z, 31)
    return (_lsr(z, 11).to(F64) + 0.5) * (1.0 / 9007199254740992.0)


def p_vs(T):
    a = (L_V0 + (C_L - C_PV) * T_0) / R_V
    b = (C_L - C_PV) / R_V
    return P_VS0 * torch.exp(a * (1.0 / T_0 - 1.0 / T) - b * torch.log(T / T_0))


def hydrostatic_profile(z, th0=289.0, rv0=7.5e-3, p0=101500.0):
    """theta = th0, r_v = rv0 constant with height, hydrostatic rho_d(z) from p0 at z = 0 (PAPER.md :115).
    Closed form: with eps = R_d/R_v, Exner pi(z) = pi_0 - g (1+rv) z / ((1+rv/eps) c_pd theta)."""
    eps = R_D / R_V
    pd0 = p0 / (1.0 + rv0 / eps)
    pi0 = (pd0 / P_1000) ** (R_D / C_PD)
    pi = pi0 - G_ACC * (1.0 + rv0) * z / ((1.0 + rv0 / eps) * C_PD * th0)
    T = th0 * pi
    pd = P_1000 * pi ** (C_PD / R_D)
    rhod = pd / (R_D * T)
    RH = rv0 * rhod * R_V * T / p_vs(T)
    return dict(T=T, rhod=rhod, RH=RH)


@dataclass
class Mode:
    n_stp: float   # [m^-3] at STP
    r_mean: float  # [m] mode radius
    sigma_g: float


# PAPER.md :117-130: the paper prints mode DIAMETERS d = 0.04 / 0.15 um, so r_m = 0.02 / 0.075 um
VOCALS_MODES = (Mode(60e6, 0.02e-6, 1.4), Mode(40e6, 0.075e-6, 1.6))
KAPPA_AMMONIUM_SULPHATE = 0.61


def n_lnr(lnr, modes):
    """eq. 3 (:119) as a density in ln r_d [m^-3 per unit ln r] at STP."""
    out = torch.zeros_like(lnr)
    for m in modes:
        ls = math.log(m.sigma_g)
        out = out + m.n_stp / (math.sqrt(2 * math.pi) * ls) * torch.exp(-((lnr - math.log(m.r_mean)) ** 2) / (2 * ls * ls))
    return out


def auto_rd_range(modes, sd_conc_mean, dV):
    """:657: smallest/largest r_d such that the multiplicity of an SD there is >= 1; the criterion depends on
    the width of the range itself, so iterate to the fixed point."""
    lo, hi = math.log(1e-9), math.log(1e-5)
    grid = torch.linspace(math.log(1e-10), math.log(1e-4), 200001, dtype=F64)
    dens = n_lnr(grid, modes)
    for _ in range(50):
        mult = dens * (hi - lo) / sd_conc_mean * dV
        ok = torch.nonzero(mult >= 1.0).flatten()
        nlo, nhi = float(grid[ok[0]]), float(grid[ok[-1]])
        if abs(nlo - lo) + abs(nhi - hi) < 1e-9:
            break
        lo, hi = nlo, nhi
    return lo, hi


def equilibrium_rw(rd3, kappa, RH, T):
    """Wet radius with RH = a_w exp(A/r) on the stable branch (PAPER.md :661-665), by bisection in ln r."""
    A = 2 * SIGMA_W / (R_V * T * RHO_W)
    rd = rd3 ** (1.0 / 3.0)
    lo = torch.log(rd)
    hi = lo + math.log(1e3)
    for _ in range(70):
        mid = 0.5 * (lo + hi)
        r = torch.exp(mid)
        r3 = r * r * r
        S = (r3 - rd3) / (r3 - rd3 * (1 - kappa)) * torch.exp(A / r)
        up = S < RH
        lo = torch.where(up, mid, lo)
        hi = torch.where(up, hi, mid)
    return torch.exp(0.5 * (lo + hi))


def efficiency_table_standin(n_R=15, n_q=21):
    """STAND-IN collision-efficiency table (the real Hall/Davis-type values are not in the container and are
    not written from memory): a smooth Long-(1974)-type analytic shape on a 15 x 21 grid,
    E = min(1, 4.5e4 R_cm^2 (1 - 3e-4 / r_cm)) for R <= 50 um and 1 above, r = q R."""
    R = torch.exp(torch.linspace(math.log(10e-6), math.log(300e-6), n_R, dtype=F64))
    q = torch.linspace(0.0, 1.0, n_q, dtype=F64)
    Rc = (R * 100.0)[:, None]
    rc = torch.clamp(Rc * q[None, :], min=1e-12)
    E = torch.clamp(4.5e4 * Rc * Rc * (1.0 - 3e-4 / rc), 0.0, 1.0)
    E = torch.where(Rc > 50e-4, torch.ones_like(E), E)
    return R, q, E.contiguous()


@dataclass
class Workload:
    name: str
    init: dict                 # keyword arguments common to oracle.Oracle(...) and binding.Particles(...)
    opts: dict                 # keyword arguments of make_opts
    th: torch.Tensor           # fields, shape = present dimensions
    rv: torch.Tensor
    rhod: torch.Tensor
    courants: list             # rho_d * Courant per present dimension (Arakawa-C shapes)
    state: dict                # n (int64), rw2, rd3, kappa, x, y, z (None if absent), id (int32)
    meta: dict = field(default_factory=dict)

    @property
    def n_sd(self):
        return self.state["n"].numel()


def box_golovin(seed=42, n_sd=2**13, device="cpu"):
    """configs[0]: one cell V = 1e6 m^3, n0 = 2^23 m^-3, exponential volume distribution with
    v0 = (4/3) pi (30.531 um)^3, equal multiplicities, Golovin b = 1500/s, dt = 1 s."""
    V, n0 = 1e6, 2.0**23
    v0 = 4.0 / 3.0 * math.pi * 30.531e-6**3
    idx = torch.arange(n_sd, dtype=torch.int64, device=device)
    u = hash_uniform(seed, 1, idx)
    v = -v0 * torch.log(u)
    rw2 = (v / (4.0 / 3.0 * math.pi)) ** (2.0 / 3.0)
    one = torch.ones(1, dtype=F64, device=device)
    st = dict(n=torch.full((n_sd,), int(n0 * V / n_sd), dtype=torch.int64, device=device), rw2=rw2,
              rd3=torch.full((n_sd,), 1e-27, dtype=F64, device=device), kappa=torch.full((n_sd,), 0.5, dtype=F64, device=device),
              x=None, y=None, z=None, id=idx.to(torch.int32))
    return Workload("box_golovin", dict(nx=0, ny=0, nz=0, dx=100.0, dy=100.0, dz=100.0, dt=1.0, kernel="golovin", golovin_b=1500.0, seed=seed),
                    dict(adve=False, sedi=False, cond=False, coal=True, sstp_coal=1), 300.0 * one, 0.0 * one, 1.0 * one, [], st,
                    dict(V=V, n0=n0, v0=v0, b=1500.0))


def _psi2d(x, z, X, Z, w_max):
    """eq. 2 (:111), kept exactly as printed (reading R-psi)."""
    return -w_max * (X / math.pi) * torch.sin(math.pi * z / Z) * torch.cos(2 * math.pi * x / X)


def kinematic(nx, ny, nz, dx, sd_per_cell, rv0=7.5e-3, th0=289.0, w_max=0.6, kernel="geometric", seed=42, dt=1.0,
              device="cpu", sstp_cond=10, sstp_coal=1, RH_max=1.05, modes=VOCALS_MODES, kappa=KAPPA_AMMONIUM_SULPHATE, name=None):
    """2D (ny = 0) or 3D prescribed-flow set-up (PAPER.md :89-138; 3D flow: DESIGN.md reading R-flow3d).
    Grid cells are cubes of size dx (2D: depth dy = 1 m)."""
    three = ny > 0
    dy = dx if three else 1.0
    dz = dx
    X, Y, Z = nx * dx, (ny * dy if three else 1.0), nz * dz
    dev = device
    zc = (torch.arange(nz, dtype=F64, device=dev) + 0.5) * dz
    prof = hydrostatic_profile(zc, th0, rv0)
    shape = (nx, ny, nz) if three else (nx, nz)
    rhod = prof["rhod"].expand(shape).contiguous()
    th = torch.full(shape, th0, dtype=F64, device=dev)
    rv = torch.full(shape, rv0, dtype=F64, device=dev)
    # rho_d * Courant from the stream function differenced on the Arakawa-C grid (:113)
    xe = torch.arange(nx + 1, dtype=F64, device=dev) * dx
    ze = torch.arange(nz + 1, dtype=F64, device=dev) * dz
    if not three:
        psi = _psi2d(xe[:, None], ze[None, :], X, Z, w_max)                # corners (nx+1, nz+1)
        c1 = -(psi[:, 1:] - psi[:, :-1]) / dz * dt / dx                    # rho_d u dt/dx at x-edges (nx+1, nz)
        c2 = (psi[1:, :] - psi[:-1, :]) / dx * dt / dz                     # rho_d w dt/dz at z-edges (nx, nz+1)
        courants = [c1.contiguous(), c2.contiguous()]
    else:
        ye = torch.arange(ny + 1, dtype=F64, device=dev) * dy
        psi1 = 0.5 * _psi2d(xe[:, None], ze[None, :], X, Z, w_max)         # (nx+1, nz+1), in the x-z plane
        psi2 = 0.5 * _psi2d(ye[:, None], ze[None, :], Y, Z, w_max)         # (ny+1, nz+1), in the y-z plane
        u = -(psi1[:, 1:] - psi1[:, :-1]) / dz                             # (nx+1, nz)
        v = -(psi2[:, 1:] - psi2[:, :-1]) / dz                             # (ny+1, nz)
        w = (psi1[1:, :] - psi1[:-1, :])[:, None, :] / dx + (psi2[1:, :] - psi2[:-1, :])[None, :, :] / dy   # (nx, ny, nz+1)
        c1 = (u * dt / dx)[:, None, :].expand(nx + 1, ny, nz).contiguous()
        c2 = (v * dt / dy)[None, :, :].expand(nx, ny + 1, nz).contiguous()
        c3 = (w * dt / dz).contiguous()
        courants = [c1, c2, c3]
    # aerosol population (:653-665)
    ncell = nx * max(ny, 1) * nz
    N = int(round(sd_per_cell * ncell))
    dV = dx * dy * dz
    lo, hi = auto_rd_range(modes, sd_per_cell, dV)
    idx = torch.arange(N, dtype=torch.int64, device=dev)
    x = hash_uniform(seed, 11, idx) * X
    z = hash_uniform(seed, 13, idx) * Z
    y = hash_uniform(seed, 12, idx) * Y if three else None
    lnr = lo + (hi - lo) * hash_uniform(seed, 14, idx)
    k = torch.clamp((z / dz).floor().to(torch.int64), 0, nz - 1)
    rhod_sd = prof["rhod"][k]
    mult = n_lnr(lnr, modes) * (hi - lo) / sd_per_cell * dV * (rhod_sd / RHO_STP)
    n = torch.clamp(torch.floor(mult + 0.5), min=1.0).to(torch.int64)
    rd3 = torch.exp(3.0 * lnr)
    kap = torch.full((N,), kappa, dtype=F64, device=dev)
    rw = equilibrium_rw(rd3, kap, torch.clamp(prof["RH"][k], max=0.95), prof["T"][k])
    st = dict(n=n, rw2=rw * rw, rd3=rd3, kappa=kap, x=x, y=y, z=z, id=idx.to(torch.int32))
    init = dict(nx=nx, ny=ny, nz=nz, dx=dx, dy=dy, dz=dz, dt=dt, kernel=kernel, seed=seed)
    if kernel == "hydro_tab":
        R, q, E = efficiency_table_standin()
        init.update(eff_R=R.numpy(), eff_q=q.numpy(), eff_tab=E.numpy())
    opts = dict(adve=True, sedi=True, cond=True, coal=True, RH_max=RH_max, sstp_cond=sstp_cond, sstp_coal=sstp_coal)
    return Workload(name or ("kinematic_3d" if three else "kinematic_2d"), init, opts, th, rv, rhod, courants, st,
                    dict(rd_range=(math.exp(lo), math.exp(hi)), sd_per_cell=sd_per_cell, X=X, Y=Y, Z=Z))


def cfg2_2d(sd_per_cell=32, nx=75, nz=75, **kw):
    """configs[1]: 75 x 75 cells of 20 m, 32 SD/cell, geometric kernel (the paper's own run, :858-860)."""
    return kinematic(nx, 0, nz, 20.0, sd_per_cell, name="2d_75x75", **kw)


def cfg3_2d_drizzle(sd_per_cell=128, nx=75, nz=75, **kw):
    """configs[2]: same grid, 128 SD/cell, tabulated-efficiency kernel, r_v = 8.5 g/kg."""
    return kinematic(nx, 0, nz, 20.0, sd_per_cell, rv0=8.5e-3, kernel="hydro_tab", name="2d_75x75_drizzle", **kw)


def cfg4_3d(sd_per_cell=64, nx=128, ny=128, nz=64, **kw):
    """configs[3]: 128 x 128 x 64 cells of 20 m, 64 SD/cell (67M SDs), w_max = 1 m/s."""
    return kinematic(nx, ny, nz, 20.0, sd_per_cell, w_max=1.0, name=f"3d_{nx}x{ny}x{nz}", **kw)


def cfg5_sweep(sd_per_cell, n=256, **kw):
    """configs[4]: 2D 256 x 256 cells over the same 1.5 km x 1.5 km domain."""
    return kinematic(n, 0, n, 1500.0 / n, sd_per_cell, name=f"2d_{n}x{n}_sd{sd_per_cell}", **kw)
