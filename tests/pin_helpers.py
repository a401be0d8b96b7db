"""Test-side restatements used ONLY by the oracle pins (tests/test_oracle_pins.py, -m "not gpu").

Nothing here is imported by ``oracle/`` or by the product package, and nothing here imports them: the
pins of the oracle's section-5.1.6 initialisation need (i) an environment to initialise into and (ii) a
second, independently written statement of the rules the oracle is checked against.  numpy + scipy only.
Citations are PAPER.md line numbers.
"""
import math

import numpy as np
from scipy import optimize

R_D, R_V, C_PD = 287.0, 461.5, 1005.0
P_1000, G_ACC = 1.0e5, 9.81
RHO_W, SIGMA_W = 1000.0, 0.072
RHO_STP = 101325.0 / (R_D * 293.15)      # :130 "T = 20 C and p = 1013.25 hPa"
# :117-130 (the paper prints mode diameters 0.04 / 0.15 um): (kappa, N at STP [m^-3], r_m [m], sigma_g)
VOCALS = [(0.61, 60e6, 0.02e-6, 1.4), (0.61, 40e6, 0.075e-6, 1.6)]


def hydrostatic_rhod(z, th0=289.0, rv0=7.5e-3, p0=101500.0):
    """Dry-air density of a column with constant theta and r_v in hydrostatic balance from p0 at z = 0 (:115):
    with eps = R_d/R_v the Exner function is linear in z, pi(z) = pi_0 - g (1 + rv) z / ((1 + rv/eps) c_pd theta)."""
    eps = R_D / R_V
    pd0 = p0 / (1.0 + rv0 / eps)
    pi0 = (pd0 / P_1000) ** (R_D / C_PD)
    pi = pi0 - G_ACC * (1.0 + rv0) * np.asarray(z, dtype=np.float64) / ((1.0 + rv0 / eps) * C_PD * th0)
    T = th0 * pi
    return P_1000 * pi ** (C_PD / R_D) / (R_D * T)


def column_fields(nx, nz, dz=20.0, th0=289.0, rv0=7.5e-3):
    """Dense C-order (i, k) fields of a 2D set-up with the profile above: th, rv, rhod (each nx*nz) and rhod(z)."""
    rz = hydrostatic_rhod((np.arange(nz) + 0.5) * dz, th0, rv0)
    return np.full(nx * nz, th0), np.full(nx * nz, rv0), np.tile(rz, nx), rz


def spectrum_density(lnr, modes=VOCALS):
    """eq. 3 (:119) as a density in ln r_d at STP [m^-3]."""
    lnr = np.asarray(lnr, dtype=np.float64)
    out = np.zeros_like(lnr)
    for _, n, rm, sg in modes:
        ls = math.log(sg)
        out = out + n / (math.sqrt(2 * math.pi) * ls) * np.exp(-((lnr - math.log(rm)) ** 2) / (2 * ls * ls))
    return out


def rd_range_by_root_finding(modes, sd_conc, dV):
    """:657 "multiplicity for both the minimal and the maximal radii be greater or equal one": the limits are the
    two outermost solutions of n(ln r) (hi - lo) / sd_conc dV = 1, a fixed point in (lo, hi).  Solved here with
    brentq on the continuous density (the oracle scans a grid): agreement to the grid step is the pin."""
    peak = optimize.minimize_scalar(lambda q: -float(spectrum_density(q, modes)), bounds=(math.log(1e-9), math.log(1e-5)),
                                    method="bounded").x
    lo, hi = math.log(1e-9), math.log(1e-5)
    for _ in range(200):
        f = lambda q: float(spectrum_density(q, modes)) * (hi - lo) / sd_conc * dV - 1.0   # noqa: E731
        nlo = optimize.brentq(f, math.log(1e-10), peak, xtol=1e-14)
        nhi = optimize.brentq(f, peak, math.log(1e-4), xtol=1e-14)
        done = abs(nlo - lo) + abs(nhi - hi) < 1e-12
        lo, hi = nlo, nhi
        if done:
            break
    return lo, hi


def koehler_saturation(r, rd3, kappa, T):
    """a_w exp(A / r) of eq. 22 with Table 2 (:1056, :1074)."""
    A = 2 * SIGMA_W / (R_V * T * RHO_W)
    r3 = r ** 3
    return (r3 - rd3) / (r3 - rd3 * (1 - kappa)) * np.exp(A / r)


def equilibrium_rw_brentq(rd3, kappa, RH, T):
    """Root of a_w exp(A/r) = RH on the stable branch r_d < r < sqrt(3 kappa r_d^3 / A) (:661-665), one SD at a time."""
    A = 2 * SIGMA_W / (R_V * T * RHO_W)
    lo, hi = rd3 ** (1 / 3) * (1 + 1e-12), math.sqrt(3 * kappa * rd3 / A)
    return optimize.brentq(lambda r: koehler_saturation(r, rd3, kappa, T) - RH, lo, hi, xtol=1e-22, rtol=1e-14)
