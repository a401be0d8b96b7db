"""ORACLE (test infrastructure, not the product).

ctypes wrapper over ``oracle/sdm_oracle.cpp``: a plain, slow fp64 CPU
implementation of the super-droplet step of arxiv 1310.1905 (§5.1).
Only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s
``cpu_baseline`` / ``--impl reference`` legs may import this package.  It
imports nothing from ``paper_1310_1905_b200`` and shares no code with the
CUDA path.
"""
import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = [os.path.join(_HERE, f) for f in ("sdm_oracle.cpp", "formulae.h")]
# ORACLE_SANITIZE=1 (environment): the same source built with -fsanitize=address,undefined into liboracle_san.so;
# the process must then run with LD_PRELOAD=$(gcc -print-file-name=libasan.so) (tests/test_oracle_sanitize.py does).
_SANITIZE = os.environ.get("ORACLE_SANITIZE", "") == "1"
_SO = os.path.join(_HERE, "liboracle_san.so" if _SANITIZE else "liboracle.so")


def build(force=False):
    """Compile the oracle with gcc (-O2, no FMA contraction, OpenMP over cells)."""
    if not force and os.path.exists(_SO) and all(os.path.getmtime(_SO) >= os.path.getmtime(s) for s in _SRC):
        return _SO
    cmd = ["g++", "-O2", "-ffp-contract=off", "-fopenmp", "-shared", "-fPIC", _SRC[0], "-o", _SO]
    if _SANITIZE:
        cmd[1:2] = ["-O1", "-g", "-fsanitize=address,undefined", "-fno-sanitize-recover=undefined", "-fno-omit-frame-pointer"]
    subprocess.check_call(cmd)
    return _SO


class _Init(C.Structure):
    _fields_ = [("nx", C.c_int), ("ny", C.c_int), ("nz", C.c_int),
                ("dx", C.c_double), ("dy", C.c_double), ("dz", C.c_double), ("dt", C.c_double),
                ("kernel", C.c_int), ("golovin_b", C.c_double), ("multi_coal", C.c_int),
                ("seed", C.c_uint64), ("n_eff_R", C.c_int), ("n_eff_q", C.c_int),
                ("eff_R", C.c_void_p), ("eff_q", C.c_void_p), ("eff_tab", C.c_void_p)]


class _Opts(C.Structure):
    _fields_ = [("adve", C.c_int), ("sedi", C.c_int), ("cond", C.c_int), ("coal", C.c_int),
                ("RH_max", C.c_double), ("sstp_cond", C.c_int), ("sstp_coal", C.c_int), ("cond_adapt_tol", C.c_double), ("coal_adapt_max", C.c_int)]


class _Counters(C.Structure):
    _fields_ = [(k, C.c_longlong) for k in
                ("pairs", "collisions", "near_ties", "ill_posed", "f_evals", "sd_substeps")]


_lib = None


def lib():
    global _lib
    if _lib is None:
        build()
        L = C.CDLL(_SO)
        L.orc_create.restype = C.c_void_p
        L.orc_create.argtypes = [C.POINTER(_Init)]
        for name in ("orc_destroy", "orc_stage_sort"):
            getattr(L, name).argtypes = [C.c_void_p]
            getattr(L, name).restype = None
        for name in ("orc_stage_cond", "orc_stage_thermo", "orc_stage_coal", "orc_stage_move", "orc_step_sync"):
            getattr(L, name).argtypes = [C.c_void_p, C.POINTER(_Opts)]
            getattr(L, name).restype = None
        for name in ("orc_step_async", "orc_step"):
            getattr(L, name).argtypes = [C.c_void_p, C.POINTER(_Opts)]
            getattr(L, name).restype = C.c_double
        L.orc_set_threads.argtypes = [C.c_void_p, C.c_int]
        L.orc_max_threads.restype = C.c_int
        L.orc_set_state.argtypes = [C.c_void_p, C.c_long] + [C.c_void_p] * 8
        L.orc_set_fields.argtypes = [C.c_void_p] + [C.c_void_p] * 6
        L.orc_set_step.argtypes = [C.c_void_p, C.c_uint32]
        L.orc_set_recycle.argtypes = [C.c_void_p, C.c_int]
        L.orc_recycled.argtypes = [C.c_void_p]
        L.orc_recycled.restype = C.c_longlong
        L.orc_stage_recycle.argtypes = [C.c_void_p]
        L.orc_stage_recycle.restype = None
        L.orc_init.argtypes = [C.c_void_p, C.c_int, C.c_void_p, C.c_double] + [C.c_double] * 6 + [C.c_void_p]
        L.orc_init.restype = C.c_long
        L.orc_get_step.argtypes = [C.c_void_p]
        L.orc_get_step.restype = C.c_uint32
        L.orc_n_sd.argtypes = [C.c_void_p]
        L.orc_n_sd.restype = C.c_long
        L.orc_n_live.argtypes = [C.c_void_p]
        L.orc_n_live.restype = C.c_long
        L.orc_get_state.argtypes = [C.c_void_p] + [C.c_void_p] * 8
        L.orc_get_fields.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p]
        L.orc_get_order.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p]
        L.orc_get_counters.argtypes = [C.c_void_p, C.POINTER(_Counters)]
        L.orc_upstream_advect.argtypes = [C.c_void_p, C.c_void_p]
        L.orc_rain_flux_total.argtypes = [C.c_void_p]
        L.orc_rain_flux_total.restype = C.c_double
        L.orc_diag_mom.argtypes = [C.c_void_p, C.c_int, C.c_double, C.c_double, C.c_int, C.c_void_p]
        L.orc_diag_sd_conc.argtypes = [C.c_void_p, C.c_void_p]
        L.orc_philox.argtypes = [C.c_void_p] * 3
        for name, nargs in (("orc_T", 2), ("orc_p", 3), ("orc_pvs", 1), ("orc_lv", 1), ("orc_eta", 1),
                            ("orc_vterm", 4), ("orc_growth_f", 8), ("orc_adve_1d", 4)):
            getattr(L, name).argtypes = [C.c_double] * nargs
            getattr(L, name).restype = C.c_double
        L.orc_cell_thermo.argtypes = [C.c_double] * 4 + [C.c_void_p]
        L.orc_cond_substep.argtypes = [C.c_double] * 8 + [C.POINTER(C.c_int)]
        L.orc_cond_substep.restype = C.c_double
        L.orc_eff.argtypes = [C.c_void_p, C.c_double, C.c_double]
        L.orc_eff.restype = C.c_double
        _lib = L
    return _lib


def _ptr(a):
    return None if a is None else a.ctypes.data_as(C.c_void_p)


def _f64(a):
    return None if a is None else np.ascontiguousarray(a, dtype=np.float64)


KERNELS = {"geometric": 0, "golovin": 1, "hydro_tab": 2}


def make_opts(adve=True, sedi=True, cond=True, coal=True, RH_max=44.0, sstp_cond=10, sstp_coal=1, cond_adapt_tol=0.0, coal_adapt_max=0):
    return _Opts(int(adve), int(sedi), int(cond), int(coal), float(RH_max), int(sstp_cond), int(sstp_coal), float(cond_adapt_tol),
                 int(coal_adapt_max))


class Oracle:
    """One oracle instance = one particles_t of PAPER.md Listing 5.5 (:755-790)."""

    def __init__(self, nx=0, ny=0, nz=0, dx=1.0, dy=1.0, dz=1.0, dt=1.0, kernel="geometric",
                 golovin_b=1500.0, multi_coal=True, seed=42, eff_R=None, eff_q=None, eff_tab=None):
        self.L = lib()
        self._keep = [_f64(eff_R), _f64(eff_q), _f64(eff_tab)]
        ini = _Init(nx, ny, nz, dx, dy, dz, dt, KERNELS[kernel], golovin_b, int(multi_coal), seed,
                    0 if eff_R is None else len(eff_R), 0 if eff_q is None else len(eff_q),
                    _ptr(self._keep[0]), _ptr(self._keep[1]), _ptr(self._keep[2]))
        self.h = self.L.orc_create(C.byref(ini))
        self.NX, self.NY, self.NZ = max(nx, 1), max(ny, 1), max(nz, 1)
        self.o_dx, self.o_dy, self.o_dz = dx, dy, dz
        self.ncell = self.NX * self.NY * self.NZ

    def __del__(self):
        try:
            self.L.orc_destroy(self.h)
        except Exception:
            pass

    def set_threads(self, n):
        self.L.orc_set_threads(self.h, n)

    def set_state(self, n, rw2, rd3, kappa, x=None, y=None, z=None, id=None):
        N = len(n)
        n = np.ascontiguousarray(n, dtype=np.uint64)
        id = np.arange(N, dtype=np.uint32) if id is None else np.ascontiguousarray(id, dtype=np.uint32)
        arrs = [_f64(a) for a in (rw2, rd3, kappa, x, y, z)]
        self.L.orc_set_state(self.h, N, _ptr(n), *[_ptr(a) for a in arrs], _ptr(id))

    def set_fields(self, th=None, rv=None, rhod=None, cx=None, cy=None, cz=None):
        arrs = [_f64(a) for a in (th, rv, rhod, cx, cy, cz)]
        self.L.orc_set_fields(self.h, *[_ptr(a) for a in arrs])

    def init(self, modes, sd_conc_mean, x0=0.0, y0=0.0, z0=0.0, x1=None, y1=None, z1=None):
        """PAPER.md section 5.1.6: modes = [(kappa, N_stp, r_mean, sigma_g), ...]; uses the fields set before.
        Returns (number of SDs, [(ln r_lo, ln r_hi) per spectrum])."""
        m = np.ascontiguousarray(np.asarray(modes, dtype=np.float64).reshape(-1, 4))
        x1 = self.o_dx * self.NX if x1 is None else x1
        y1 = self.o_dy * self.NY if y1 is None else y1
        z1 = self.o_dz * self.NZ if z1 is None else z1
        ranges = np.zeros(2 * len(m), dtype=np.float64)
        N = self.L.orc_init(self.h, len(m), _ptr(m), float(sd_conc_mean), x0, y0, z0, x1, y1, z1, _ptr(ranges))
        G = len(dict.fromkeys(m[:, 0].tolist()))
        return N, [(ranges[2 * g], ranges[2 * g + 1]) for g in range(G)]

    def set_step(self, step):
        self.L.orc_set_step(self.h, step)

    def set_recycle(self, on):
        """PAPER.md :641, :651: recycle zero-multiplicity SDs at the beginning of each step (default: compaction only)."""
        self.L.orc_set_recycle(self.h, int(bool(on)))

    def stage_recycle(self):
        self.L.orc_stage_recycle(self.h)

    @property
    def recycled(self):
        return int(self.L.orc_recycled(self.h))

    @property
    def step_count(self):
        return self.L.orc_get_step(self.h)

    def stage(self, name, opts=None):
        if name == "sort":
            self.L.orc_stage_sort(self.h)
        else:
            getattr(self.L, "orc_stage_" + name)(self.h, C.byref(opts))

    def step_sync(self, opts):
        self.L.orc_step_sync(self.h, C.byref(opts))

    def step_async(self, opts):
        return self.L.orc_step_async(self.h, C.byref(opts))

    def step(self, opts):
        return self.L.orc_step(self.h, C.byref(opts))

    def n_sd(self):
        return self.L.orc_n_sd(self.h)

    def n_live(self):
        return self.L.orc_n_live(self.h)

    def get_state(self):
        N = self.n_sd()
        out = dict(n=np.empty(N, np.uint64), rw2=np.empty(N), rd3=np.empty(N), kappa=np.empty(N),
                   x=np.empty(N), y=np.empty(N), z=np.empty(N), id=np.empty(N, np.uint32))
        self.L.orc_get_state(self.h, *[_ptr(out[k]) for k in ("n", "rw2", "rd3", "kappa", "x", "y", "z", "id")])
        return out

    def get_fields(self):
        th, rv = np.empty(self.ncell), np.empty(self.ncell)
        self.L.orc_get_fields(self.h, _ptr(th), _ptr(rv))
        return th, rv

    def get_order(self):
        N = self.n_sd()
        ids, seg = np.empty(N, np.uint32), np.empty(self.ncell + 1, np.int64)
        self.L.orc_get_order(self.h, _ptr(ids), _ptr(seg))
        return ids, seg

    def upstream_advect(self, psi):
        """One first-order upstream step (PAPER.md :219-235; the transport solver of Fig. 7) of the dense C-order field psi
        with the rho_d x Courant arrays set by set_fields; returns the new field."""
        out = np.ascontiguousarray(psi, dtype=np.float64).copy()
        self.L.orc_upstream_advect(self.h, _ptr(out))
        return out

    def counters(self):
        c = _Counters()
        self.L.orc_get_counters(self.h, C.byref(c))
        return {k: getattr(c, k) for k, _ in _Counters._fields_}

    def rain_flux_total(self):
        return self.L.orc_rain_flux_total(self.h)

    def diag_mom(self, wet, r_mi, r_mx, k):
        out = np.empty(self.ncell)
        self.L.orc_diag_mom(self.h, int(wet), r_mi, r_mx, k, _ptr(out))
        return out

    def diag_sd_conc(self):
        out = np.empty(self.ncell)
        self.L.orc_diag_sd_conc(self.h, _ptr(out))
        return out

    def eff(self, R, q):
        return self.L.orc_eff(self.h, R, q)


def philox(ctr, key):
    c = np.asarray(ctr, dtype=np.uint32)
    k = np.asarray(key, dtype=np.uint32)
    o = np.empty(4, np.uint32)
    lib().orc_philox(_ptr(c), _ptr(k), _ptr(o))
    return o


def cell_thermo(th, rv, rhod, RH_max=44.0):
    o = np.empty(8)
    lib().orc_cell_thermo(th, rv, rhod, RH_max, _ptr(o))
    return dict(zip(("T", "p", "lv", "rho_vs", "RH", "A", "eta", "rho_a"), o))


def cond_substep(y0, rd3, kappa, th, rv, rhod, RH_max, dtp):
    ip = C.c_int(0)
    y = lib().orc_cond_substep(y0, rd3, kappa, th, rv, rhod, RH_max, dtp, C.byref(ip))
    return y, ip.value
