"""Thin ctypes binding of libchan.so (include/chan.h): argument marshalling only.

PyTorch is used for device memory and the CUDA stream; every step of the path runs in the library's
kernels.  There is no fallback: if the shared library is missing, :func:`load` raises.
"""
import ctypes as C
import os

import numpy as np
import torch

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libchan.so")
_lib = None

OK, EINVAL, ENOSPACE, ESTATE, ECUDA, ELIMIT = 0, -1, -2, -3, -4, -5
STATS_ACCUMULATE, STATS_READ, STATS_RESET = 1, 2, 4
F_V, F_PHI, F_OMY, F_U, F_W, F_OMX, F_OMZ, F_H1, F_H2, F_H3, F_HV_PREV, F_HG_PREV = range(12)
STAGE_DERIVE, STAGE_NONLINEAR, STAGE_YSOLVE = range(3)

EXPORTS = [
    "chan_create", "chan_destroy", "chan_workspace_bytes", "chan_bind", "chan_set_state", "chan_get_state",
    "chan_set_state_host", "chan_get_state_host", "chan_substep", "chan_step", "chan_filter_store",
    "chan_filter_store_host", "chan_step_filter", "chan_stats", "chan_get_scalars", "chan_set_pgrad", "chan_strerror",
    "chan_debug_get_field", "chan_debug_set_field", "chan_debug_run_stage", "chan_debug_set_substep_index",
    "chan_debug_get_band_tables", "chan_debug_launch_count", "chan_debug_transpose",
    "chan_debug_profile", "chan_debug_profile_read", "chan_debug_set_tuning", "chan_debug_get_tuning", "chan_debug_describe", "chan_debug_fma_peak", "chan_set_filter_precision", "chan_run",
    "chan_post_scratch_bytes", "chan_post_pressure", "chan_post_strain_norm", "chan_post_sgs",
    "chan_mesh_helmholtz_error", "chan_mesh_optimize", "chan_spectra",
    "chan_post_strain_norm_static", "chan_post_strain_norm_static_limit",
]
KERNEL_CLASSES = ["d1_forward", "derive_down", "derive_up", "zfft_inv", "xfft_prod", "zfft_fwd", "mean", "y1", "y2", "y3",
                  "y4", "y5", "transpose", "filter_copy", "xfft_prod_filter", "zfft_fwd_filter", "stats", "planes_merged", "post"]


class Grid(C.Structure):
    _fields_ = [("nx", C.c_int), ("ny", C.c_int), ("nz", C.c_int)]


class Box(C.Structure):
    _fields_ = [("lx", C.c_double), ("lz", C.c_double), ("y", C.POINTER(C.c_double))]


class Opts(C.Structure):
    _fields_ = [("lhs_halfwidth", C.c_int), ("rhs_halfwidth", C.c_int), ("forcing", C.c_int)]


class Tuning(C.Structure):
    """chan_tuning_t of include/chan.h (0 = the plan's own choice)."""
    _fields_ = [("xfuse", C.c_int), ("maxradix_z", C.c_int), ("maxradix_x", C.c_int), ("tz", C.c_int), ("zthreads", C.c_int),
                ("xthreads", C.c_int), ("chunk_mb", C.c_int), ("planes_per_chunk", C.c_int), ("plane_overlap", C.c_int),
                ("z_cluster", C.c_int), ("reserved", C.c_int * 6)]


class Run(C.Structure):
    """chan_run_t of include/chan.h."""
    _fields_ = [("nsteps", C.c_int), ("filter_every", C.c_int), ("stats_every", C.c_int), ("kx_cut", C.c_int), ("kz_cut", C.c_int),
                ("dev_ring", C.c_void_p), ("slot_bytes", C.c_size_t), ("ring_slots", C.c_int)]


class ChanError(RuntimeError):
    def __init__(self, status, where):
        self.status = status
        msg = load().chan_strerror(status).decode()
        super().__init__(f"{where}: {msg} ({status})")


def load():
    """dlopen libchan.so built in-tree by ``__graft_entry__.build()``; raises if it is not there."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise RuntimeError(f"{LIB_PATH} is missing: run `python -c 'import __graft_entry__ as g; g.build()'` "
                           "(there is no CPU fallback)")
    lib = C.CDLL(LIB_PATH)
    vp, i, d, sz = C.c_void_p, C.c_int, C.c_double, C.c_size_t
    sig = {
        "chan_create": (i, [C.POINTER(vp), C.POINTER(Grid), C.POINTER(Box), d, d, C.POINTER(Opts)]),
        "chan_destroy": (i, [vp]),
        "chan_workspace_bytes": (sz, [vp]),
        "chan_bind": (i, [vp, vp, sz, vp]),
        "chan_set_state": (i, [vp] * 6),
        "chan_get_state": (i, [vp] * 6),
        "chan_set_state_host": (i, [vp] * 6),
        "chan_get_state_host": (i, [vp] * 6),
        "chan_substep": (i, [vp]),
        "chan_step": (i, [vp]),
        "chan_filter_store": (i, [vp, i, i, vp, sz]),
        "chan_filter_store_host": (i, [vp, i, i, vp, sz]),
        "chan_step_filter": (i, [vp, i, i, vp, sz]),
        "chan_stats": (i, [vp, i, vp, C.POINTER(C.c_longlong)]),
        "chan_get_scalars": (i, [vp, vp]),
        "chan_set_pgrad": (i, [vp, d]),
        "chan_strerror": (C.c_char_p, [i]),
        "chan_debug_get_field": (i, [vp, i, vp]),
        "chan_debug_set_field": (i, [vp, i, vp]),
        "chan_debug_run_stage": (i, [vp, i]),
        "chan_debug_set_substep_index": (i, [vp, i]),
        "chan_debug_get_band_tables": (i, [vp, vp]),
        "chan_debug_launch_count": (C.c_longlong, [vp]),
        "chan_debug_transpose": (i, [vp, i, vp, vp]),
        "chan_debug_profile": (i, [vp, i]),
        "chan_debug_profile_read": (i, [vp, vp, vp]),
        "chan_debug_set_tuning": (i, [vp, C.POINTER(Tuning)]),
        "chan_debug_get_tuning": (i, [vp, C.POINTER(Tuning)]),
        "chan_debug_describe": (i, [vp, C.c_char_p, sz]),
        "chan_debug_fma_peak": (i, [vp, C.POINTER(C.c_double)]),
        "chan_set_filter_precision": (i, [vp, i]),
        "chan_run": (i, [vp, C.POINTER(Run), C.POINTER(C.c_longlong)]),
        "chan_mesh_helmholtz_error": (i, [i, vp, d, i, vp]),
        "chan_mesh_optimize": (i, [i, vp, i, d, d, i, vp, vp]),
        "chan_spectra": (i, [vp, vp, sz, vp, sz]),
        "chan_post_scratch_bytes": (sz, [vp, i, i]),
        "chan_post_pressure": (i, [vp, i, i, vp, vp, vp, sz]),
        "chan_post_strain_norm": (i, [vp, i, i, vp, vp, vp, sz]),
        "chan_post_sgs": (i, [vp, i, i, vp, vp, vp, sz]),
        "chan_post_strain_norm_static": (i, [vp, i, i, vp, vp]),
        "chan_post_strain_norm_static_limit": (sz, []),
    }
    for name, (res, args) in sig.items():
        fn = getattr(lib, name)
        fn.restype, fn.argtypes = res, args
    _lib = lib
    return lib


def _chk(status, where):
    if status != OK:
        raise ChanError(status, where)


def mesh_helmholtz_error(y, lam, nfirst):
    """chan_mesh_helmholtz_error: (error at y = -1, error at y = +1)."""
    y = np.ascontiguousarray(y, dtype=np.float64)
    out = np.zeros(2)
    _chk(load().chan_mesh_helmholtz_error(y.size, y.ctypes.data, float(lam), int(nfirst), out.ctypes.data), "chan_mesh_helmholtz_error")
    return out


def mesh_optimize(y, npoints, lam, max_shift=0.25, sweeps=8):
    """chan_mesh_optimize: (new mesh, errors before [2], errors after [2])."""
    y = np.array(y, dtype=np.float64, copy=True)
    eb, ea = np.zeros(2), np.zeros(2)
    _chk(load().chan_mesh_optimize(y.size, y.ctypes.data, int(npoints), float(lam), float(max_shift), int(sweeps), eb.ctypes.data,
                                   ea.ctypes.data), "chan_mesh_optimize")
    return y, eb, ea


class Channel:
    """Owner of one ``chan_t`` handle plus its torch-allocated workspace (names follow include/chan.h)."""

    def __init__(self, nx, ny, nz, lx, lz, y, re_tau, dt, forcing=0, half_lhs=3, half_rhs=3, tuning=None):
        self.lib = load()
        self.nx, self.ny, self.nz = nx, ny, nz
        y = np.ascontiguousarray(y, dtype=np.float64)
        self._y = y
        self.h = C.c_void_p()
        grid = Grid(nx, ny, nz)
        box = Box(lx, lz, y.ctypes.data_as(C.POINTER(C.c_double)))
        opts = Opts(half_lhs, half_rhs, forcing)
        _chk(self.lib.chan_create(C.byref(self.h), C.byref(grid), C.byref(box), re_tau, dt, C.byref(opts)), "chan_create")
        self.ws = None
        self.shape = (nz, nx // 2, ny)
        if tuning:
            self.debug_set_tuning(**tuning)

    def debug_set_tuning(self, **kw):
        """chan_debug_set_tuning (before bind): keyword = field of chan_tuning_t."""
        t = Tuning()
        for k, v in kw.items():
            if k not in dict(Tuning._fields_) or k in ("reserved", "planes_per_chunk"):
                raise KeyError(k)
            setattr(t, k, int(v))
        _chk(self.lib.chan_debug_set_tuning(self.h, C.byref(t)), "chan_debug_set_tuning")

    def debug_get_tuning(self):
        t = Tuning()
        _chk(self.lib.chan_debug_get_tuning(self.h, C.byref(t)), "chan_debug_get_tuning")
        return {k: getattr(t, k) for k, _ in Tuning._fields_ if k != "reserved"}

    def debug_describe(self):
        buf = C.create_string_buffer(512)
        _chk(self.lib.chan_debug_describe(self.h, buf, 512), "chan_debug_describe")
        return buf.value.decode()

    def workspace_bytes(self):
        return int(self.lib.chan_workspace_bytes(self.h))

    def bind(self, device="cuda:0", stream=None):
        if not torch.cuda.is_available():
            raise RuntimeError("chan_bind needs a CUDA device (there is no CPU fallback)")
        self.device = torch.device(device)
        n = self.workspace_bytes()
        self.ws = torch.empty(n + 256, dtype=torch.uint8, device=self.device)
        ptr = (self.ws.data_ptr() + 255) // 256 * 256
        self.stream = stream if stream is not None else torch.cuda.current_stream(self.device)
        _chk(self.lib.chan_bind(self.h, ptr, n, self.stream.cuda_stream), "chan_bind")
        return self

    # ---- state -------------------------------------------------------------------------------------
    def _dev(self, a, dtype):
        t = torch.as_tensor(a, dtype=dtype).to(self.device).contiguous()
        return t

    def set_state(self, v, phi, omy, U, W):
        ts = [self._dev(a, torch.complex128) for a in (v, phi, omy)] + [self._dev(a, torch.float64) for a in (U, W)]
        for t in ts[:3]:
            assert tuple(t.shape) == self.shape
        _chk(self.lib.chan_set_state(self.h, *[t.data_ptr() for t in ts]), "chan_set_state")
        self._keep = ts

    def get_state(self):
        v, phi, omy = (torch.empty(self.shape, dtype=torch.complex128, device=self.device) for _ in range(3))
        U, W = (torch.empty(self.ny, dtype=torch.float64, device=self.device) for _ in range(2))
        _chk(self.lib.chan_get_state(self.h, v.data_ptr(), phi.data_ptr(), omy.data_ptr(), U.data_ptr(), W.data_ptr()),
             "chan_get_state")
        return v, phi, omy, U, W

    def set_state_host(self, v, phi, omy, U, W):
        """Host tensors/arrays (pinned or pageable, C-contiguous complex128 / float64)."""
        ptrs = [_host_ptr(a) for a in (v, phi, omy, U, W)]
        _chk(self.lib.chan_set_state_host(self.h, *ptrs), "chan_set_state_host")

    def get_state_host(self, v, phi, omy, U, W):
        ptrs = [_host_ptr(a) for a in (v, phi, omy, U, W)]
        _chk(self.lib.chan_get_state_host(self.h, *ptrs), "chan_get_state_host")

    # ---- time stepping -----------------------------------------------------------------------------
    def substep(self):
        _chk(self.lib.chan_substep(self.h), "chan_substep")

    def step(self):
        _chk(self.lib.chan_step(self.h), "chan_step")

    # ---- filter and statistics ---------------------------------------------------------------------
    def set_filter_precision(self, bytes_per_real):
        """8: complex128 database (default); 4: complex64 (rounded once from the fp64 result)."""
        _chk(self.lib.chan_set_filter_precision(self.h, int(bytes_per_real)), "chan_set_filter_precision")
        self._fdtype = torch.complex64 if bytes_per_real == 4 else torch.complex128

    def _fout(self, kx_cut, kz_cut, out, lead=()):
        dt = getattr(self, "_fdtype", torch.complex128)
        if out is None:
            out = torch.empty(tuple(lead) + (10, self.ny, 2 * kz_cut + 1, kx_cut + 1), dtype=dt, device=self.device)
        assert out.dtype == dt and out.is_contiguous()
        return out

    def filter_store(self, kx_cut, kz_cut, out=None):
        out = self._fout(kx_cut, kz_cut, out)
        _chk(self.lib.chan_filter_store(self.h, kx_cut, kz_cut, out.data_ptr(), out.numel() * out.element_size()), "chan_filter_store")
        return out

    def step_filter(self, kx_cut, kz_cut, out=None):
        """filter_store of the current state fused into the step that follows."""
        out = self._fout(kx_cut, kz_cut, out)
        _chk(self.lib.chan_step_filter(self.h, kx_cut, kz_cut, out.data_ptr(), out.numel() * out.element_size()), "chan_step_filter")
        return out

    def filter_store_host(self, kx_cut, kz_cut, out):
        _chk(self.lib.chan_filter_store_host(self.h, kx_cut, kz_cut, _host_ptr(out), out.numel() * out.element_size()),
             "chan_filter_store_host")
        return out

    def run(self, nsteps, filter_every, stats_every, kx_cut, kz_cut, ring=None, ring_slots=None):
        """chan_run: nsteps full steps with the snapshot cadence; returns (ring tensor [slots][10][ny][..][..], emitted)."""
        if filter_every > 0:
            if ring is None:
                slots = ring_slots or (nsteps + filter_every - 1) // filter_every
                ring = self._fout(kx_cut, kz_cut, None, lead=(max(slots, 1),))
            slots = ring.shape[0]
            r = Run(nsteps, filter_every, stats_every, kx_cut, kz_cut, ring.data_ptr(), ring[0].numel() * ring.element_size(), slots)
        else:
            r = Run(nsteps, 0, stats_every, kx_cut, kz_cut, None, 0, 0)
        n = C.c_longlong(0)
        _chk(self.lib.chan_run(self.h, C.byref(r), C.byref(n)), "chan_run")
        return ring, int(n.value)

    # ---- post-processing of a stored database (NEXT-2) ----------------------------------------------
    def _post(self, fn, name, kx_cut, kz_cut, db, lead=()):
        assert db.dtype == torch.complex128 and db.is_contiguous() and tuple(db.shape) == (10, self.ny, 2 * kz_cut + 1, kx_cut + 1)
        out = torch.empty(tuple(lead) + (self.ny, 2 * kz_cut + 1, kx_cut + 1), dtype=torch.complex128, device=self.device)
        n = int(self.lib.chan_post_scratch_bytes(self.h, kx_cut, kz_cut))
        scratch = torch.empty(max(n, 16), dtype=torch.uint8, device=self.device)
        _chk(fn(self.h, kx_cut, kz_cut, db.data_ptr(), out.data_ptr(), scratch.data_ptr(), n), name)
        self._post_keep = scratch
        return out

    def post_pressure(self, kx_cut, kz_cut, db):
        return self._post(self.lib.chan_post_pressure, "chan_post_pressure", kx_cut, kz_cut, db)

    def post_strain_norm(self, kx_cut, kz_cut, db):
        return self._post(self.lib.chan_post_strain_norm, "chan_post_strain_norm", kx_cut, kz_cut, db)

    def post_strain_norm_static(self, kx_cut, kz_cut, db, out):
        """chan_post_strain_norm_static: caller-owned ``out``; the scratch is the library's static device array."""
        assert db.dtype == torch.complex128 and db.is_contiguous() and out.dtype == torch.complex128 and out.is_contiguous()
        assert tuple(out.shape) == (self.ny, 2 * kz_cut + 1, kx_cut + 1)
        _chk(self.lib.chan_post_strain_norm_static(self.h, kx_cut, kz_cut, db.data_ptr(), out.data_ptr()), "chan_post_strain_norm_static")
        return out

    def post_sgs(self, kx_cut, kz_cut, db):
        return self._post(self.lib.chan_post_sgs, "chan_post_sgs", kx_cut, kz_cut, db, lead=(6,))

    def stats(self, flags):
        out = np.zeros((10, self.ny))
        n = C.c_longlong(0)
        _chk(self.lib.chan_stats(self.h, flags, out.ctypes.data, C.byref(n)), "chan_stats")
        return out, int(n.value)

    def spectra(self):
        """chan_spectra: (ex [7][ny][nx/2], ez [7][ny][nz]) float64 device tensors."""
        ex = torch.empty((7, self.ny, self.nx // 2), dtype=torch.float64, device=self.device)
        ez = torch.empty((7, self.ny, self.nz), dtype=torch.float64, device=self.device)
        _chk(self.lib.chan_spectra(self.h, ex.data_ptr(), ex.numel() * 8, ez.data_ptr(), ez.numel() * 8), "chan_spectra")
        return ex, ez

    def scalars(self):
        out = np.zeros(4)
        _chk(self.lib.chan_get_scalars(self.h, out.ctypes.data), "chan_get_scalars")
        return out

    def set_pgrad(self, g):
        _chk(self.lib.chan_set_pgrad(self.h, float(g)), "chan_set_pgrad")

    # ---- debug hooks -------------------------------------------------------------------------------
    def debug_get_field(self, field):
        out = torch.empty(self.shape, dtype=torch.complex128, device=self.device)
        _chk(self.lib.chan_debug_get_field(self.h, field, out.data_ptr()), "chan_debug_get_field")
        return out

    def debug_set_field(self, field, a):
        t = self._dev(a, torch.complex128)
        assert tuple(t.shape) == self.shape
        _chk(self.lib.chan_debug_set_field(self.h, field, t.data_ptr()), "chan_debug_set_field")
        torch.cuda.synchronize(self.device)

    def debug_run_stage(self, stage):
        _chk(self.lib.chan_debug_run_stage(self.h, stage), "chan_debug_run_stage")

    def debug_set_substep_index(self, i):
        _chk(self.lib.chan_debug_set_substep_index(self.h, i), "chan_debug_set_substep_index")

    def debug_band_tables(self):
        out = np.zeros((4, self.ny, 7))
        _chk(self.lib.chan_debug_get_band_tables(self.h, out.ctypes.data), "chan_debug_get_band_tables")
        return out

    def debug_fma_peak(self):
        """Measured fp64 FMA throughput of the device in TFLOP/s (register-only micro-kernel)."""
        out = C.c_double(0.0)
        _chk(self.lib.chan_debug_fma_peak(self.h, C.byref(out)), "chan_debug_fma_peak")
        return float(out.value)

    def debug_launch_count(self):
        return int(self.lib.chan_debug_launch_count(self.h))

    def debug_transpose(self, direction, src, dst):
        _chk(self.lib.chan_debug_transpose(self.h, direction, src.data_ptr(), dst.data_ptr()), "chan_debug_transpose")

    def debug_profile(self, enable):
        _chk(self.lib.chan_debug_profile(self.h, int(enable)), "chan_debug_profile")

    def debug_profile_read(self):
        """{kernel class: (summed milliseconds, launches)} since debug_profile(True)."""
        n = len(KERNEL_CLASSES)
        ms = np.zeros(n)
        cnt = np.zeros(n, dtype=np.int64)
        _chk(self.lib.chan_debug_profile_read(self.h, ms.ctypes.data, cnt.ctypes.data), "chan_debug_profile_read")
        return {k: (float(ms[j]), int(cnt[j])) for j, k in enumerate(KERNEL_CLASSES)}

    def close(self):
        if self.h:
            if self.ws is not None:
                torch.cuda.synchronize(self.device)
            self.lib.chan_destroy(self.h)
            self.h = C.c_void_p()
            self.ws = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


def _host_ptr(a):
    if isinstance(a, torch.Tensor):
        assert a.device.type == "cpu" and a.is_contiguous()
        return a.data_ptr()
    a = np.asarray(a)
    assert a.flags["C_CONTIGUOUS"]
    return a.ctypes.data
