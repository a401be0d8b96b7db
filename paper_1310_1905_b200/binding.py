"""Thin Python binding of libsdm (include/sdm.h): argument marshalling only.

Every step of the path runs in the CUDA kernels behind the C ABI; PyTorch is used for device memory
and streams.  Method names follow the C ABI / the paper's ``particles_t`` (Listing 5.5,
:755-790).  There is no CPU fallback: importing works anywhere, but creating ``Particles`` raises
unless ``libsdm.so`` is built and an sm_100 GPU is present.
"""
import ctypes as C
import os

import torch

_HERE = os.path.dirname(os.path.abspath(__file__))
_SO = os.path.join(_HERE, "libsdm.so")

KERNELS = {"geometric": 0, "golovin": 1, "hydro_tab": 2}


class SdmError(RuntimeError):
    pass


class OptsInit(C.Structure):
    _fields_ = [("nx", C.c_int), ("ny", C.c_int), ("nz", C.c_int),
                ("dx", C.c_double), ("dy", C.c_double), ("dz", C.c_double), ("dt", C.c_double),
                ("x0", C.c_double), ("y0", C.c_double), ("z0", C.c_double),
                ("x1", C.c_double), ("y1", C.c_double), ("z1", C.c_double),
                ("sd_conc_mean", C.c_double), ("kernel", C.c_int), ("golovin_b", C.c_double),
                ("n_eff_R", C.c_int), ("n_eff_q", C.c_int),
                ("eff_R", C.c_void_p), ("eff_q", C.c_void_p), ("eff_tab", C.c_void_p),
                ("seed", C.c_uint64), ("real_bytes", C.c_int), ("multi_coal", C.c_int), ("max_sd", C.c_uint64),
                ("n_modes", C.c_int), ("modes", C.c_void_p), ("open_x", C.c_int)]


class Opts(C.Structure):
    _fields_ = [("adve", C.c_int), ("sedi", C.c_int), ("cond", C.c_int), ("coal", C.c_int),
                ("RH_max", C.c_double), ("sstp_cond", C.c_int), ("sstp_coal", C.c_int), ("cond_adapt_tol", C.c_double), ("coal_adapt_max", C.c_int)]


class ArrInfo(C.Structure):
    _fields_ = [("data_zero", C.c_void_p), ("strides", C.c_int64 * 3)]


class SdBuffers(C.Structure):
    _fields_ = [("n", C.c_void_p), ("rw2", C.c_void_p), ("rd3", C.c_void_p), ("kappa", C.c_void_p), ("x", C.c_void_p),
                ("y", C.c_void_p), ("z", C.c_void_p), ("id", C.c_void_p)]


class Stats(C.Structure):
    _fields_ = [(k, C.c_uint64) for k in ("n_sd", "max_cell_count", "step", "kernel_launches", "pairs", "collisions",
                                          "near_ties", "ill_posed", "newton_iters", "sd_substeps", "cond_slow", "recycled",
                                          "cond_variant", "cond_tile_cells", "coal_tile_cells", "host_syncs")]


EXPORTS = ["sdm_create", "sdm_destroy", "sdm_last_error", "sdm_init", "sdm_init_range", "sdm_init_from_arrays", "sdm_step_sync", "sdm_step_async",
           "sdm_step_async_result", "sdm_step_host", "sdm_diag_sd_conc", "sdm_diag_dry_rng", "sdm_diag_wet_rng",
           "sdm_diag_dry_mom", "sdm_diag_wet_mom", "sdm_outbuf", "sdm_n_sd", "sdm_n_live", "sdm_export_state", "sdm_export_order",
           "sdm_stats", "sdm_set_step", "sdm_set_group_size", "sdm_set_cond_kfast", "sdm_set_timing", "sdm_stage_times", "sdm_set_recycle", "sdm_set_cond_arith",
           "sdm_measure_fp64_peak", "sdm_upstream_advect", "sdm_pack_leavers", "sdm_unpack_arrivals",
           "sdm_cell_offsets_noalloc", "sdm_cell_offsets_noalloc_setup", "sdm_noalloc_last_error"]

STAGES = ("hist", "scan", "scatter", "rank", "cond", "coal_move", "recycle")

_lib = None


def load_library():
    """dlopen libsdm.so (built in-tree by paper_1310_1905_b200/build.py) and declare the prototypes."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(_SO):
        raise SdmError(f"{_SO} is missing: build it with `python -m paper_1310_1905_b200.build` (no CPU fallback exists)")
    L = C.CDLL(_SO)
    vp, u64p = C.c_void_p, C.POINTER(C.c_uint64)
    L.sdm_create.argtypes = [C.POINTER(OptsInit), C.POINTER(vp)]
    L.sdm_destroy.argtypes = [vp]
    L.sdm_destroy.restype = None
    L.sdm_last_error.argtypes = [vp]
    L.sdm_last_error.restype = C.c_char_p
    L.sdm_init_from_arrays.argtypes = [vp, ArrInfo, ArrInfo, ArrInfo, ArrInfo, C.c_uint64] + [vp] * 8 + [vp]
    L.sdm_init.argtypes = [vp] + [ArrInfo] * 6 + [vp]
    L.sdm_init_range.argtypes = [vp, C.c_int, C.POINTER(C.c_double), C.POINTER(C.c_double)]
    L.sdm_step_sync.argtypes = [vp, C.POINTER(Opts)] + [ArrInfo] * 6 + [vp]
    L.sdm_step_async.argtypes = [vp, C.POINTER(Opts), vp]
    L.sdm_step_async_result.argtypes = [vp, C.POINTER(C.c_double)]
    L.sdm_step_host.argtypes = [vp, C.POINTER(Opts), vp, vp, C.POINTER(C.c_double), vp]
    L.sdm_diag_sd_conc.argtypes = [vp, vp]
    L.sdm_diag_dry_rng.argtypes = [vp, C.c_double, C.c_double]
    L.sdm_diag_wet_rng.argtypes = [vp, C.c_double, C.c_double]
    L.sdm_diag_dry_mom.argtypes = [vp, C.c_int, vp]
    L.sdm_diag_wet_mom.argtypes = [vp, C.c_int, vp]
    L.sdm_outbuf.argtypes = [vp]
    L.sdm_outbuf.restype = vp
    L.sdm_n_sd.argtypes = [vp, u64p]
    L.sdm_n_live.argtypes = [vp, u64p]
    L.sdm_upstream_advect.argtypes = [vp, ArrInfo, vp]
    L.sdm_pack_leavers.argtypes = [vp, C.c_uint64, C.POINTER(SdBuffers), C.POINTER(SdBuffers), u64p, u64p, vp]
    L.sdm_unpack_arrivals.argtypes = [vp, C.c_uint64, C.POINTER(SdBuffers), C.c_double, vp]
    L.sdm_measure_fp64_peak.argtypes = [C.POINTER(C.c_double), C.POINTER(C.c_double), vp]
    L.sdm_export_state.argtypes = [vp] + [vp] * 8 + [vp]
    L.sdm_export_order.argtypes = [vp, vp, vp, vp]
    L.sdm_stats.argtypes = [vp, C.POINTER(Stats)]
    L.sdm_set_step.argtypes = [vp, C.c_uint64]
    L.sdm_set_group_size.argtypes = [vp, C.c_int]
    L.sdm_set_cond_kfast.argtypes = [vp, C.c_int]
    L.sdm_set_timing.argtypes = [vp, C.c_int]
    L.sdm_set_recycle.argtypes = [vp, C.c_int]
    L.sdm_set_cond_arith.argtypes = [vp, C.c_int]
    L.sdm_stage_times.argtypes = [vp, C.POINTER(C.c_double), u64p, C.c_int]
    L.sdm_cell_offsets_noalloc_setup.argtypes = []
    L.sdm_cell_offsets_noalloc.argtypes = [vp, C.c_int64, vp, vp]
    L.sdm_noalloc_last_error.argtypes = []
    L.sdm_noalloc_last_error.restype = C.c_char_p
    _lib = L
    return L


def make_opts(adve=True, sedi=True, cond=True, coal=True, RH_max=44.0, sstp_cond=10, sstp_coal=1, cond_adapt_tol=0.0, coal_adapt_max=0):
    return Opts(int(adve), int(sedi), int(cond), int(coal), float(RH_max), int(sstp_cond), int(sstp_coal), float(cond_adapt_tol),
                int(coal_adapt_max))


def arrinfo(t):
    """arrinfo_t of a torch CUDA tensor (None -> omitted argument); strides in elements."""
    a = ArrInfo()
    if t is None:
        a.data_zero = None
        return a
    assert t.is_cuda and t.dtype == torch.float64
    a.data_zero = t.data_ptr()
    for k, s in enumerate(t.stride()):
        a.strides[k] = s
    return a


def _ptr(t):
    return None if t is None else t.data_ptr()


def _stream():
    return torch.cuda.current_stream().cuda_stream


class Particles:
    """One ``particles_t`` (PAPER.md :747-790) living on the current CUDA device."""

    def __init__(self, nx=0, ny=0, nz=0, dx=1.0, dy=1.0, dz=1.0, dt=1.0, kernel="geometric", golovin_b=1500.0,
                 multi_coal=True, seed=42, eff_R=None, eff_q=None, eff_tab=None, max_sd=None, sd_conc_mean=0.0, modes=None,
                 x0=0.0, y0=0.0, z0=0.0, x1=None, y1=None, z1=None, real_bytes=8, open_x=False):
        """real_bytes: 8 or 4, the storage type of rw2, rd3, kappa, x, y, z (fields stay float64).  modes: [(kappa, N_stp, r_mean, sigma_g), ...] of the dry spectrum, needed by init() only."""
        import numpy as np
        self.L = load_library()
        keep = [None if a is None else np.ascontiguousarray(a, dtype=np.float64) for a in (eff_R, eff_q, eff_tab)]
        o = OptsInit()
        o.nx, o.ny, o.nz, o.dx, o.dy, o.dz, o.dt = nx, ny, nz, dx, dy, dz, dt
        o.x0, o.y0, o.z0 = x0, y0, z0
        o.x1 = dx * max(nx, 1) if x1 is None else x1
        o.y1 = dy * max(ny, 1) if y1 is None else y1
        o.z1 = dz * max(nz, 1) if z1 is None else z1
        if modes is not None:
            keep.append(np.ascontiguousarray(np.asarray(modes, dtype=np.float64).reshape(-1, 4)))
            o.n_modes, o.modes = len(keep[-1]), keep[-1].ctypes.data
        o.sd_conc_mean, o.kernel, o.golovin_b = sd_conc_mean, KERNELS[kernel], golovin_b
        if keep[0] is not None:
            o.n_eff_R, o.n_eff_q = len(keep[0]), len(keep[1])
            o.eff_R, o.eff_q, o.eff_tab = (k.ctypes.data for k in keep)
        o.seed, o.real_bytes, o.multi_coal, o.max_sd = seed, int(real_bytes), int(multi_coal), int(max_sd)
        o.open_x = int(bool(open_x))
        self.real = torch.float64 if int(real_bytes) == 8 else torch.float32
        self.h = C.c_void_p()
        rc = self.L.sdm_create(C.byref(o), C.byref(self.h))
        if rc != 0:
            raise SdmError(f"sdm_create failed ({rc}): {self.L.sdm_last_error(None).decode()}")
        self.shape = tuple(n for n in (nx, ny, nz) if n > 0) or (1,)
        self.ncell = max(nx, 1) * max(ny, 1) * max(nz, 1)
        self.dims = (nx > 0, ny > 0, nz > 0)

    def __del__(self):
        try:
            if self.h:
                self.L.sdm_destroy(self.h)
                self.h = None
        except Exception:
            pass

    def _ck(self, rc):
        if rc != 0:
            raise SdmError(f"libsdm error {rc}: {self.L.sdm_last_error(self.h).decode()}")

    def init(self, th, rv, rhod, courant_1=None, courant_2=None, courant_3=None):
        """particles_t::init() (PAPER.md :759-766, section 5.1.6)."""
        self._ck(self.L.sdm_init(self.h, arrinfo(th), arrinfo(rv), arrinfo(rhod), arrinfo(courant_1), arrinfo(courant_2),
                                 arrinfo(courant_3), _stream()))

    def init_range(self, g=0):
        lo, hi = C.c_double(), C.c_double()
        self._ck(self.L.sdm_init_range(self.h, g, C.byref(lo), C.byref(hi)))
        return lo.value, hi.value

    def init_from_arrays(self, rhod, n, rw2, rd3, kappa, x=None, y=None, z=None, id=None, courant_1=None, courant_2=None,
                         courant_3=None):
        N = n.numel()
        if id is None:
            id = torch.arange(N, dtype=torch.int32, device=n.device)
        for name, t in (("rw2", rw2), ("rd3", rd3), ("kappa", kappa), ("x", x), ("y", y), ("z", z)):
            if t is not None and (t.dtype != self.real or not t.is_contiguous()):
                raise SdmError(f"init_from_arrays: {name} must be a contiguous {self.real} tensor (real_bytes of this context)")
        self._ck(self.L.sdm_init_from_arrays(self.h, arrinfo(rhod), arrinfo(courant_1), arrinfo(courant_2), arrinfo(courant_3),
                                             N, _ptr(n), _ptr(rw2), _ptr(rd3), _ptr(kappa), _ptr(x), _ptr(y), _ptr(z), _ptr(id),
                                             _stream()))

    def step_sync(self, opts, th, rv, courant_1=None, courant_2=None, courant_3=None, rhod=None):
        self._ck(self.L.sdm_step_sync(self.h, C.byref(opts), arrinfo(th), arrinfo(rv), arrinfo(courant_1), arrinfo(courant_2),
                                      arrinfo(courant_3), arrinfo(rhod), _stream()))

    def step_async(self, opts):
        self._ck(self.L.sdm_step_async(self.h, C.byref(opts), _stream()))

    def step_async_result(self):
        f = C.c_double()
        self._ck(self.L.sdm_step_async_result(self.h, C.byref(f)))
        return f.value

    def step_host(self, opts, th_host, rv_host):
        """th_host, rv_host: CPU float64 tensors (dense C order), overwritten."""
        f = C.c_double()
        self._ck(self.L.sdm_step_host(self.h, C.byref(opts), th_host.data_ptr(), rv_host.data_ptr(), C.byref(f), _stream()))
        return f.value

    def _out(self):
        """Copy of the library-owned output buffer (PAPER.md :788 outbuf), shaped like the grid."""
        src = _as_tensor(self.L.sdm_outbuf(self.h), self.ncell)
        return src.clone().reshape(self.shape)

    def diag_sd_conc(self):
        self._ck(self.L.sdm_diag_sd_conc(self.h, _stream()))
        return self._out()

    def diag_dry_rng(self, r_mi, r_mx):
        self._ck(self.L.sdm_diag_dry_rng(self.h, r_mi, r_mx))

    def diag_wet_rng(self, r_mi, r_mx):
        self._ck(self.L.sdm_diag_wet_rng(self.h, r_mi, r_mx))

    def diag_dry_mom(self, k):
        self._ck(self.L.sdm_diag_dry_mom(self.h, k, _stream()))
        return self._out()

    def diag_wet_mom(self, k):
        self._ck(self.L.sdm_diag_wet_mom(self.h, k, _stream()))
        return self._out()

    def n_sd(self):
        v = C.c_uint64()
        self._ck(self.L.sdm_n_sd(self.h, C.byref(v)))
        return v.value

    def _sd_buffers(self, cap):
        """A set of SoA device arrays for `cap` SDs (sdm_sd_buffers) and its ctypes view."""
        t = dict(n=torch.empty(cap, dtype=torch.int64, device="cuda"), id=torch.empty(cap, dtype=torch.int32, device="cuda"))
        for k in ("rw2", "rd3", "kappa", "x", "y", "z"):
            t[k] = torch.zeros(cap, dtype=self.real, device="cuda")
        return t, SdBuffers(*[_ptr(t[k]) for k in ("n", "rw2", "rd3", "kappa", "x", "y", "z", "id")])

    def pack_leavers(self, cap):
        """SDs that left the slab through x < 0 and through x >= nx*dx, as two dicts of tensors (open_x contexts only)."""
        lt, lb = self._sd_buffers(max(cap, 1))
        rt, rb = self._sd_buffers(max(cap, 1))
        nl, nr = C.c_uint64(), C.c_uint64()
        self._ck(self.L.sdm_pack_leavers(self.h, max(cap, 1), C.byref(lb), C.byref(rb), C.byref(nl), C.byref(nr), _stream()))
        return {k: v[:nl.value] for k, v in lt.items()}, {k: v[:nr.value] for k, v in rt.items()}

    def unpack_arrivals(self, sds, x_shift):
        """Appends the SDs of `sds` (a dict as pack_leavers returns) with x + x_shift as their coordinate in this slab."""
        N = int(sds["n"].numel())
        if N == 0:
            return
        t = {k: v.contiguous() for k, v in sds.items()}
        b = SdBuffers(*[_ptr(t[k]) for k in ("n", "rw2", "rd3", "kappa", "x", "y", "z", "id")])
        self._ck(self.L.sdm_unpack_arrivals(self.h, N, C.byref(b), float(x_shift), _stream()))

    def upstream_advect(self, psi):
        """One upstream step of the field psi (overwritten) with the context's Courant numbers: the Eulerian solver of Fig. 7."""
        self._ck(self.L.sdm_upstream_advect(self.h, arrinfo(psi), _stream()))

    def n_live(self):
        v = C.c_uint64()
        self._ck(self.L.sdm_n_live(self.h, C.byref(v)))
        return v.value

    def export_state(self):
        N = self.n_sd()
        dev = "cuda"
        out = dict(n=torch.empty(N, dtype=torch.int64, device=dev), id=torch.empty(N, dtype=torch.int32, device=dev))
        for k in ("rw2", "rd3", "kappa", "x", "y", "z"):
            out[k] = torch.zeros(N, dtype=self.real, device=dev)
        self._ck(self.L.sdm_export_state(self.h, *[_ptr(out[k]) for k in ("n", "rw2", "rd3", "kappa", "x", "y", "z", "id")],
                                         _stream()))
        torch.cuda.current_stream().synchronize()
        return out

    def export_order(self):
        N = self.n_sd()
        ids = torch.empty(N, dtype=torch.int32, device="cuda")
        seg = torch.empty(self.ncell + 1, dtype=torch.int32, device="cuda")
        self._ck(self.L.sdm_export_order(self.h, _ptr(ids), _ptr(seg), _stream()))
        torch.cuda.current_stream().synchronize()
        return ids, seg

    def stats(self):
        s = Stats()
        self._ck(self.L.sdm_stats(self.h, C.byref(s)))
        return {k: getattr(s, k) for k, _ in Stats._fields_}

    def set_step(self, step):
        self._ck(self.L.sdm_set_step(self.h, step))

    def set_group_size(self, g):
        self._ck(self.L.sdm_set_group_size(self.h, g))

    def set_cond_kfast(self, kfast):
        self._ck(self.L.sdm_set_cond_kfast(self.h, kfast))

    def set_recycle(self, on=True):
        """PAPER.md :641, :651: recycle zero-multiplicity SDs at the beginning of each step instead of only compacting."""
        self._ck(self.L.sdm_set_recycle(self.h, int(bool(on))))

    def set_cond_arith(self, bytes_):
        """8: fp64 condensation sweep (default); 4: fp32 arithmetic (real_bytes = 4 only; radii to 1e-4)."""
        self._ck(self.L.sdm_set_cond_arith(self.h, int(bytes_)))

    def set_timing(self, enable=True):
        self._ck(self.L.sdm_set_timing(self.h, int(enable)))

    def stage_times(self, reset=True):
        """{stage: (milliseconds, timed launches)} since the last reset (synchronises the stream)."""
        ms = (C.c_double * len(STAGES))()
        cnt = (C.c_uint64 * len(STAGES))()
        self._ck(self.L.sdm_stage_times(self.h, ms, cnt, int(reset)))
        return {s: (ms[k], cnt[k]) for k, s in enumerate(STAGES)}


def measure_fp64_peak():
    """(TFLOP/s of fp64 FMA at 2 flop each, FMAs per SM clock per SM) measured on the current device."""
    t, r = C.c_double(), C.c_double()
    rc = load_library().sdm_measure_fp64_peak(C.byref(t), C.byref(r), _stream())
    if rc != 0:
        raise SdmError(f"sdm_measure_fp64_peak failed ({rc})")
    return t.value, r.value


NOALLOC_MAX_CELLS = 16777216   # SDM_NOALLOC_MAX_CELLS of include/sdm.h


def cell_offsets_noalloc_setup():
    """sdm_cell_offsets_noalloc_setup for the current device (optional: the first call does it otherwise)."""
    L = load_library()
    rc = L.sdm_cell_offsets_noalloc_setup()
    if rc != 0:
        raise SdmError(f"libsdm error {rc}: {L.sdm_noalloc_last_error().decode()}")


def cell_offsets_noalloc(count, seg, ncell=None):
    """sdm_cell_offsets_noalloc: seg[c] = count[0] + .. + count[c-1], c = 0..ncell, on the current stream, with no allocation
    on the way (the library's static scratch; calls that overlap on the GPU race, see include/sdm.h).  count: CUDA int32
    tensor of >= ncell per-cell SD numbers (the bits are read as unsigned); seg: CUDA int32 tensor of >= ncell + 1 words,
    caller-allocated, written in place.  Only marshalling here."""
    L = load_library()
    n = count.numel() if ncell is None else int(ncell)
    if n <= NOALLOC_MAX_CELLS:   # beyond the limit the library refuses before it touches a buffer: let it say so
        assert count.is_cuda and seg.is_cuda and count.dtype == torch.int32 and seg.dtype == torch.int32
        assert count.is_contiguous() and seg.is_contiguous() and 0 <= n <= count.numel() and seg.numel() >= n + 1
    rc = L.sdm_cell_offsets_noalloc(_ptr(count), n, _ptr(seg), _stream())
    if rc != 0:
        raise SdmError(f"libsdm error {rc}: {L.sdm_noalloc_last_error().decode()}")
    return seg


def _as_tensor(ptr, n):
    """Wrap a raw device pointer of n doubles as a torch tensor (no copy) via __cuda_array_interface__."""

    class _Wrap:
        pass

    w = _Wrap()
    w.__cuda_array_interface__ = {"shape": (n,), "typestr": "<f8", "data": (int(ptr), False), "version": 2}
    return torch.as_tensor(w, device="cuda")
