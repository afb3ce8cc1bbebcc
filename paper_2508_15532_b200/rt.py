"""Thin Python binding of librt_b200.so (include/rt.h): argument marshalling only.

Every step of the path runs in the library's CUDA kernels.  torch is used for device memory and streams only.
There is no CPU fallback: if the shared library is missing, importing this module raises.
"""
import ctypes
import os

import numpy as np
import torch

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "librt_b200.so")

BC = {"periodic": 0, "outflow": 1, "zero": 2, "fixed": 3, "reflect": 4}
METRIC = {"minkowski": 0, "mink_cyl": 1, "ks_mks": 2, "snake": 3, "bl_mks": 4, "user": 5}
GEOM = dict(g_c=0, e_c=1, einv_c=2, sqrtg_c=3, omega_c=4, n0_c=5, angcoef=6)
SYMBOLS = ["rt_init", "rt_free", "rt_ndir", "rt_ndir_padded", "rt_get_directions", "rt_get_geometry", "rt_cfl_dt",
           "rt_set_boundary", "rt_set_fluid", "rt_transport", "rt_transport_static", "rt_angular_flux", "rt_source_implicit", "rt_moments",
           "rt_step", "rt_step_host", "rt_step_slab", "rt_profile_enable", "rt_profile_read", "rt_transport_info", "rt_launch_count", "rt_last_cuda_error", "rt_strerror"]


class RtGrid(ctypes.Structure):
    _fields_ = [("n", ctypes.c_int * 3), ("x0", ctypes.c_double * 3), ("dx", ctypes.c_double * 3),
                ("bc_lo", ctypes.c_int * 3), ("bc_hi", ctypes.c_int * 3),
                ("zero_lo", ctypes.c_int * 3), ("zero_hi", ctypes.c_int * 3)]


# RT_USER host callbacks: void fn(const double x[3], double out[4][4], void *user)
METRIC_FN = ctypes.CFUNCTYPE(None, ctypes.POINTER(ctypes.c_double), ctypes.POINTER(ctypes.c_double), ctypes.c_void_p)


class RtMetric(ctypes.Structure):
    _fields_ = [("kind", ctypes.c_int), ("a", ctypes.c_double), ("hslope", ctypes.c_double), ("x3_symmetric", ctypes.c_int),
                ("snake_A", ctypes.c_double), ("snake_k", ctypes.c_double),
                ("g_fn", METRIC_FN), ("e_fn", METRIC_FN), ("user", ctypes.c_void_p)]


def _metric_callback(fn):
    """Python callable x[3] -> array [4,4]  ->  C callback of rt_metric (argument marshalling only)."""
    def cb(x, out, _user):
        a = np.asarray(fn(np.array([x[0], x[1], x[2]])), dtype=np.float64).reshape(16)
        for q in range(16):
            out[q] = a[q]
    return METRIC_FN(cb)


class RtOptions(ctypes.Structure):
    _fields_ = [("limiter", ctypes.c_int), ("angular_recon", ctypes.c_int), ("source_method", ctypes.c_int),
                ("n0_floor", ctypes.c_double), ("rho_floor", ctypes.c_double), ("kappa_a0", ctypes.c_double),
                ("kappa_s", ctypes.c_double), ("a_rad", ctypes.c_double), ("Y_over_rho", ctypes.c_double),
                ("abar", ctypes.c_double), ("transport_variant", ctypes.c_int), ("transport_tile", ctypes.c_int * 3),
                ("grid_axis", ctypes.c_double * 3), ("grid_boost", ctypes.c_double * 3), ("angflux_split", ctypes.c_int), ("source_literal", ctypes.c_int)]


def load_library(path=LIB_PATH):
    """dlopen the C-ABI library and declare its signatures.  Raises if it is missing (no fallback)."""
    if not os.path.exists(path):
        raise ImportError("librt_b200.so not built: run `python -m paper_2508_15532_b200.build` (needs nvcc); "
                          "there is no CPU fallback")
    lib = ctypes.CDLL(path)
    vp, dbl, ci = ctypes.c_void_p, ctypes.c_double, ctypes.c_int
    lib.rt_init.argtypes = [ctypes.POINTER(RtGrid), ctypes.POINTER(RtMetric), ci, ctypes.POINTER(RtOptions), ctypes.POINTER(vp)]
    lib.rt_free.argtypes = [vp]
    lib.rt_ndir.argtypes = [vp]
    lib.rt_ndir_padded.argtypes = [vp]
    lib.rt_get_directions.argtypes = [vp, vp, vp, vp, vp]
    lib.rt_get_geometry.argtypes = [vp, ci, vp]
    lib.rt_cfl_dt.argtypes = [vp, vp]
    lib.rt_set_boundary.argtypes = [vp, ci, ci, vp]
    lib.rt_set_fluid.argtypes = [vp, vp, vp, vp, vp]
    lib.rt_transport.argtypes = [vp, vp, vp, vp, dbl, vp]
    lib.rt_transport_static.argtypes = [vp, vp, vp, vp, dbl, vp]
    lib.rt_angular_flux.argtypes = [vp, vp, vp, dbl, vp]
    lib.rt_source_implicit.argtypes = [vp, vp, vp, dbl, vp, vp]
    lib.rt_moments.argtypes = [vp, vp, vp, vp]
    lib.rt_step.argtypes = [vp, vp, vp, vp, vp, dbl, vp, vp]
    lib.rt_step_host.argtypes = [vp, vp, vp, vp, vp, dbl, vp, vp]
    lib.rt_step_slab.argtypes = [vp, vp, vp, vp, vp, dbl, vp, vp, vp, vp, vp, vp, vp]
    lib.rt_profile_enable.argtypes = [vp, ci]
    lib.rt_profile_read.argtypes = [vp, vp, vp]
    lib.rt_transport_info.argtypes = [vp, vp]
    lib.rt_launch_count.argtypes = [vp]
    lib.rt_launch_count.restype = ctypes.c_longlong
    lib.rt_strerror.argtypes = [ci]
    lib.rt_strerror.restype = ctypes.c_char_p
    return lib


_lib = None


def lib():
    global _lib
    if _lib is None:
        _lib = load_library()
    return _lib


class RtError(RuntimeError):
    pass


def _check(rc):
    if rc != 0:
        raise RtError("%s (code %d, cuda %d)" % (lib().rt_strerror(rc).decode(), rc, lib().rt_last_cuda_error()))


def _ptr(t):
    if t is None:
        return None
    assert t.is_cuda and t.dtype in (torch.float64, torch.int32), "device fp64 tensor expected"
    assert t.is_contiguous()
    return ctypes.c_void_p(t.data_ptr())


def _stream():
    return ctypes.c_void_p(torch.cuda.current_stream().cuda_stream)


DEFAULT_OPTIONS = dict(limiter=0, angular_recon=0, source_method=2, n0_floor=0.1, rho_floor=5e-4, kappa_a0=0.0,
                       kappa_s=0.0, a_rad=1.0, Y_over_rho=1.5, abar=1.0, transport_variant=0,
                       transport_tile=(0, 0, 0))


class RtContext:
    """rt_init .. rt_free.  Intensity tensors are [N3, N2, N1, pitch] fp64 on the device (pad entries zero)."""

    def __init__(self, grid, metric_kind, metric_params, level, options=None, device="cuda:0"):
        if not torch.cuda.is_available():
            raise RtError("no CUDA device: librt_b200 has no CPU path")
        self.device = torch.device(device)
        torch.cuda.set_device(self.device)
        g = RtGrid()
        g.n[:] = grid["n"]; g.x0[:] = grid["x0"]; g.dx[:] = grid["dx"]
        g.bc_lo[:] = [BC[b] for b in grid["bc_lo"]]; g.bc_hi[:] = [BC[b] for b in grid["bc_hi"]]
        g.zero_lo[:] = grid.get("zero_lo", (0, 0, 0)); g.zero_hi[:] = grid.get("zero_hi", (0, 0, 0))
        mp = dict(metric_params or {})
        m = RtMetric(METRIC[metric_kind], mp.get("a", 0.0), mp.get("hslope", 0.3), 1, mp.get("A", 0.0), mp.get("k", 0.0))
        if metric_kind == "user":   # params: g = callable x[3] -> g[4,4]; e = callable x[3] -> e[mu, a] or None (library tetrad)
            self._cb = (_metric_callback(mp["g"]), _metric_callback(mp["e"]) if mp.get("e") is not None else METRIC_FN())
            m.g_fn, m.e_fn = self._cb
        od = dict(DEFAULT_OPTIONS)
        for k, v in (options or {}).items():
            od[{"method": "source_method", "ang_recon": "angular_recon"}.get(k, k)] = v
        for k in ("grid_axis", "grid_boost", "transport_tile"):   # vectors: tuples -> ctypes arrays
            if k in od and not isinstance(od[k], ctypes.Array):
                od[k] = ((ctypes.c_int if k == "transport_tile" else ctypes.c_double) * 3)(*od[k])
        o = RtOptions(**od)
        self._h = ctypes.c_void_p()
        _check(lib().rt_init(ctypes.byref(g), ctypes.byref(m), int(level), ctypes.byref(o), ctypes.byref(self._h)))
        self.n = tuple(int(x) for x in grid["n"])
        self.shape = self.n[::-1]
        self.nd = lib().rt_ndir(self._h)
        self.pitch = lib().rt_ndir_padded(self._h)
        self.ncell = self.n[0] * self.n[1] * self.n[2]
        self._keep = {}
        self._nfail = torch.zeros(1, dtype=torch.int32, device=self.device)

    def close(self):
        if self._h:
            lib().rt_free(self._h)
            self._h = ctypes.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    # ---- tables -------------------------------------------------------------------------------------------
    def directions(self):
        nhat, w = np.empty((self.nd, 3)), np.empty(self.nd)
        nnb, nb = np.empty(self.nd, np.int32), np.empty((self.nd, 6), np.int32)
        _check(lib().rt_get_directions(self._h, nhat.ctypes.data, w.ctypes.data, nnb.ctypes.data, nb.ctypes.data))
        return dict(nhat=nhat, w=w, nnb=nnb, nb=nb)

    def geometry(self, which):
        ncol = self.n[0] * self.n[1]
        shp = {"g_c": (4, 4), "e_c": (4, 4), "einv_c": (4, 4), "sqrtg_c": (), "omega_c": (4, 4, 4), "n0_c": (self.nd,),
               "angcoef": (6, self.nd)}[which]
        out = np.empty((1, self.n[1], self.n[0]) + shp)
        assert out.size == ncol * int(np.prod(shp, dtype=np.int64))
        _check(lib().rt_get_geometry(self._h, GEOM[which], out.ctypes.data))
        return out

    def cfl_dt(self):
        out = np.zeros(2)
        _check(lib().rt_cfl_dt(self._h, out.ctypes.data))
        return float(out[0]), float(out[1])

    # ---- helpers for the padded layout ----------------------------------------------------------------------
    def to_device(self, I_host):
        """numpy [N3,N2,N1,nd] -> device tensor [N3,N2,N1,pitch] (pad = 0)."""
        I = torch.zeros(self.shape + (self.pitch,), dtype=torch.float64, device=self.device)
        I[..., :self.nd] = torch.as_tensor(np.ascontiguousarray(I_host).reshape(self.shape + (self.nd,)), device=self.device)
        return I

    def to_host(self, I_dev):
        return I_dev[..., :self.nd].cpu().numpy()

    # ---- the rt_* calls -------------------------------------------------------------------------------------
    def set_boundary(self, dim, side, ghost_dev):
        self._keep[("ghost", dim, side)] = ghost_dev
        _check(lib().rt_set_boundary(self._h, dim, side, _ptr(ghost_dev)))

    def set_fluid(self, rho, T, u4=None):
        _check(lib().rt_set_fluid(self._h, _ptr(rho), _ptr(T), _ptr(u4), _stream()))

    def transport(self, I_in, I_base, I_out, dt):
        _check(lib().rt_transport(self._h, _ptr(I_in), _ptr(I_base), _ptr(I_out), float(dt), _stream()))

    def transport_static(self, I_in, I_base, I_out, dt):
        """rt_transport_static: rt_transport without any allocation (scratch in a static device array; RT_ETOOBIG beyond it)."""
        _check(lib().rt_transport_static(self._h, _ptr(I_in), _ptr(I_base), _ptr(I_out), float(dt), _stream()))

    def angular_flux(self, I_in, I_inout, dt):
        _check(lib().rt_angular_flux(self._h, _ptr(I_in), _ptr(I_inout), float(dt), _stream()))

    def source_implicit(self, I, T, dt):
        _check(lib().rt_source_implicit(self._h, _ptr(I), _ptr(T), float(dt), _ptr(self._nfail), _stream()))

    def moments(self, I, R):
        _check(lib().rt_moments(self._h, _ptr(I), _ptr(R), _stream()))

    def step(self, I, T, dt, R=None, G=None):
        _check(lib().rt_step(self._h, _ptr(I), _ptr(T), _ptr(R), _ptr(G), float(dt), _ptr(self._nfail), _stream()))

    def step_slab(self, I, T, dt, R, G, send_lo, send_hi, halo_stream):
        """rt_step_slab: send_lo / send_hi = (I planes [4, N2, N1, pitch], T planes [4, N2, N1]) device tensors or None; the boundary
        work runs on `halo_stream` (a torch.cuda.Stream), the whole-slab step on the current stream."""
        sl = (None, None) if send_lo is None else send_lo
        sh = (None, None) if send_hi is None else send_hi
        _check(lib().rt_step_slab(self._h, _ptr(I), _ptr(T), _ptr(R), _ptr(G), float(dt), _ptr(self._nfail), _ptr(sl[0]), _ptr(sl[1]),
                                  _ptr(sh[0]), _ptr(sh[1]), _stream(), ctypes.c_void_p(halo_stream.cuda_stream)))

    def step_host(self, I_host, T_host, dt, R_host=None, G_host=None):
        """rt_step_host: HOST tensors (pinned fp64, padded layout); returns the failed-cell count of this call."""
        nf = ctypes.c_int(0)
        hp = lambda t: None if t is None else ctypes.c_void_p(t.data_ptr())
        for t in (I_host, T_host, R_host, G_host):
            assert t is None or (not t.is_cuda and t.dtype == torch.float64 and t.is_contiguous())
        _check(lib().rt_step_host(self._h, hp(I_host), hp(T_host), hp(R_host), hp(G_host), float(dt), ctypes.byref(nf), _stream()))
        return nf.value

    def n_fail(self):
        return int(self._nfail.item())

    def profile_enable(self, on=True):
        _check(lib().rt_profile_enable(self._h, int(on)))

    def profile_read(self):
        """dict kernel class -> (milliseconds, launches) since the last read."""
        ms, cnt = np.zeros(5), np.zeros(5, np.int64)
        _check(lib().rt_profile_read(self._h, ms.ctypes.data, cnt.ctypes.data))
        names = ("facecoef", "transport", "angular", "source", "moments")
        return {n: (float(ms[i]), int(cnt[i])) for i, n in enumerate(names)}

    def transport_info(self):
        """(variant actually used, (TX, TY, DCH) of the tile kernel)."""
        out = np.zeros(4, np.int32)
        _check(lib().rt_transport_info(self._h, out.ctypes.data))
        return int(out[0]), tuple(int(v) for v in out[1:])

    def launch_count(self):
        return int(lib().rt_launch_count(self._h))
