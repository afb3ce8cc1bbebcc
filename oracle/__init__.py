"""ORACLE package -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.

A plain, slow CPU implementation of the radiation hot path of PAPER.md (arxiv 2508.15532), written
from the paper and pinned by tests/test_oracle_*.py against closed forms, invariants and the values the
paper prints.  Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs
may import this package.  It imports nothing from the CUDA package and shares no code with it.

  geodesic.py   O1  angular grid (numpy)
  geometry.py   O2  metric / tetrad / Ricci rotation coefficients (numpy)
  rt_oracle.c   O3-O8 stepping (plain C, sequential sums), built on demand with gcc

Parity status: every function is pinned.  MAPR angular reconstruction (ang_recon=1) is a reading of a method the paper only
names: its stated properties (second order, linear exactness, conservation, arg-min and tie rules) are pinned; its
identity with the cited Christov & Popov method (not in the container) cannot be checked.
"""
import ctypes
import os
import subprocess

import numpy as np

from . import geodesic, geometry

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "rt_oracle.c")
_LIB = os.path.join(_HERE, "_build", "librt_oracle.so")

BC = {"periodic": 0, "outflow": 1, "zero": 2, "fixed": 3, "reflect": 4}
_dp = ctypes.POINTER(ctypes.c_double)
_ip = ctypes.POINTER(ctypes.c_int)


class _Problem(ctypes.Structure):
    _fields_ = [
        ("n", ctypes.c_int * 3), ("n3g", ctypes.c_int), ("dx", ctypes.c_double * 3),
        ("bc_lo", ctypes.c_int * 3), ("bc_hi", ctypes.c_int * 3),
        ("zero_lo", ctypes.c_int * 3), ("zero_hi", ctypes.c_int * 3),
        ("nd", ctypes.c_int), ("nhat", _dp), ("w", _dp), ("nnb", _ip), ("nb", _ip),
        ("dlam", _dp), ("emid", _dp), ("eun", _dp),
        ("g_c", _dp), ("e_c", _dp), ("einv_c", _dp), ("sqrtg_c", _dp), ("omega_c", _dp),
        ("g_f", _dp * 3), ("e_f", _dp * 3), ("sqrtg_f", _dp * 3),
        ("limiter", ctypes.c_int), ("ang_recon", ctypes.c_int), ("method", ctypes.c_int),
        ("n0_floor", ctypes.c_double), ("rho_floor", ctypes.c_double), ("kappa_a0", ctypes.c_double),
        ("kappa_s", ctypes.c_double), ("a_rad", ctypes.c_double), ("Y_over_rho", ctypes.c_double),
        ("abar", ctypes.c_double),
        ("rho", _dp), ("u4", _dp), ("ghost", (_dp * 2) * 3), ("mirror", _ip * 3),
        ("angflux_split", ctypes.c_int), ("source_literal", ctypes.c_int),
    ]


def build_lib(force=False):
    """Compile rt_oracle.c (building the checker is not using it)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        os.makedirs(os.path.dirname(_LIB), exist_ok=True)
        subprocess.check_call(["gcc", "-O2", "-ffp-contract=off", "-fopenmp", "-shared", "-fPIC",
                               "-o", _LIB, _SRC, "-lm"])
    return _LIB


_lib = None


def _load():
    global _lib
    if _lib is None:
        _lib = ctypes.CDLL(build_lib())
        pp = ctypes.POINTER(_Problem)
        _lib.orc_transport.argtypes = [pp, _dp, _dp, _dp, _dp, ctypes.c_double]
        _lib.orc_angular.argtypes = [pp, _dp, _dp, ctypes.c_double]
        _lib.orc_source.argtypes = [pp, _dp, _dp, ctypes.c_double]
        _lib.orc_source.restype = ctypes.c_int
        _lib.orc_moments.argtypes = [pp, _dp, _dp]
        _lib.orc_step.argtypes = [pp, _dp, _dp, _dp, _dp, ctypes.c_double, _dp, _dp, _dp]
        _lib.orc_step.restype = ctypes.c_int
        _lib.orc_cfl.argtypes = [pp, _dp]
        _lib.orc_mapr_gradient.argtypes = [pp, _dp, ctypes.c_int, _dp]
    return _lib


def _c(a, dtype=np.float64):
    return np.ascontiguousarray(a, dtype=dtype)


def _ptr(a):
    return a.ctypes.data_as(_ip if a.dtype == np.int32 else _dp)


def mirror_map(nhat, a):
    """Permutation m with nhat[m[s]] = nhat[s] with component a negated, or None if the grid lacks that symmetry."""
    nhat = np.asarray(nhat)
    flipped = nhat.copy()
    flipped[:, a] *= -1.0
    d = np.abs(flipped[:, None, :] - nhat[None, :, :]).max(-1)       # [s, t]
    m = d.argmin(1)
    if d[np.arange(len(nhat)), m].max() > 1e-9 or len(set(m.tolist())) != len(nhat):
        return None
    return m.astype(np.int32)


DEFAULT_OPTIONS = dict(limiter=0, ang_recon=0, method=2, n0_floor=0.1, rho_floor=5e-4, kappa_a0=0.0,
                       kappa_s=0.0, a_rad=1.0, Y_over_rho=1.5, abar=1.0, angflux_split=0, source_literal=0)


class Oracle:
    """One radiation problem: grid + metric + angular level + options (+ fluid, set later).

    grid: dict(n=(N1,N2,N3), x0=(..), dx=(..), bc_lo=(..), bc_hi=(..) names from BC,
               zero_lo=(..), zero_hi=(..) optional, x3_symmetric=bool)
    Intensity arrays are numpy [N3, N2, N1, nd] (s fastest, no padding).
    """

    def __init__(self, grid, metric_kind, metric_params, level, options=None):
        self.grid = dict(grid)
        self.kind, self.params = metric_kind, dict(metric_params or {})
        self.opt = dict(DEFAULT_OPTIONS)
        self.opt.update(options or {})
        # (angular-grid options stay on the Python side: the C core only sees the tables)
        self.ang = geodesic.build(level, boost=self.opt.pop("grid_boost", None), axis=self.opt.pop("grid_axis", None))
        self.nd = self.ang["nd"]
        self.tab = geometry.build_tables(self.grid, self.kind, self.params)
        n = self.grid["n"]
        self.n = tuple(int(x) for x in n)
        self.Nc = n[0] * n[1] * n[2]
        self._keep = []
        P = _Problem()
        P.n[:] = n
        P.n3g = 1 if self.grid.get("x3_symmetric", False) else n[2]
        P.dx[:] = self.grid["dx"]
        P.bc_lo[:] = [BC[b] for b in self.grid["bc_lo"]]
        P.bc_hi[:] = [BC[b] for b in self.grid["bc_hi"]]
        P.zero_lo[:] = self.grid.get("zero_lo", (0, 0, 0))
        P.zero_hi[:] = self.grid.get("zero_hi", (0, 0, 0))
        P.nd = self.nd
        for name in ("nhat", "w", "dlam", "emid", "eun"):
            a = _c(self.ang[name]); self._keep.append(a); setattr(P, name, _ptr(a))
        for name in ("nnb", "nb"):
            a = _c(self.ang[name], np.int32); self._keep.append(a); setattr(P, name, _ptr(a))
        for name in ("g_c", "e_c", "einv_c", "sqrtg_c", "omega_c"):
            a = _c(self.tab[name]); self._keep.append(a); setattr(P, name, _ptr(a))
        for a_ in range(3):
            for name in ("g_f", "e_f", "sqrtg_f"):
                a = _c(self.tab["%s%d" % (name, a_)]); self._keep.append(a)
                getattr(P, name)[a_] = _ptr(a)
        for k, v in self.opt.items():
            setattr(P, k, v)
        # reflecting ("symmetric", L709, S23) boundaries: the direction with the normal tetrad component flipped.  Only
        # a dim whose flip maps the geodesic grid onto itself can reflect (with the pole along 3-hat and a vertex at
        # azimuth 0 that is dim 2-hat = x2: the x-z plane is a mirror plane of the icosahedron, the others are not)
        self.mirror = [mirror_map(self.ang["nhat"], a_) for a_ in range(3)]
        for a_ in range(3):
            if "reflect" in (self.grid["bc_lo"][a_], self.grid["bc_hi"][a_]):
                if self.mirror[a_] is None:
                    raise ValueError("the angular grid has no mirror symmetry across dim %d" % a_)
                m = _c(self.mirror[a_], np.int32); self._keep.append(m); P.mirror[a_] = _ptr(m)
        self.P = P
        self.set_fluid(np.zeros(self.n[::-1]), np.ones(self.n[::-1]), None)

    # ---- inputs -------------------------------------------------------------------------------
    def set_fluid(self, rho, T, u4):
        """rho[N3,N2,N1], T (kept as the transport-stage temperature), u4[4,N3,N2,N1] coordinate u^mu
        (None = the tetrad's own rest frame e_0-hat)."""
        self.rho = _c(rho).reshape(self.n[::-1])
        self.T = _c(T).reshape(self.n[::-1]).copy()
        if u4 is None:
            e0 = self.tab["e_c"][..., :, 0]                                  # [E3, N2, N1, 4]
            u4 = np.moveaxis(np.broadcast_to(e0, self.n[::-1] + (4,)), -1, 0)
        self.u4 = _c(u4).reshape((4,) + self.n[::-1])
        self.P.rho, self.P.u4 = _ptr(self.rho), _ptr(self.u4)

    def set_boundary(self, dim, side, ghost):
        """BC 'fixed': ghost[2, face cells, nd], layer 0 next to the interior."""
        g = _c(ghost)
        self._keep.append(g)
        self.P.ghost[dim][side] = _ptr(g)

    def _I(self, I):
        I = _c(I)
        assert I.size == self.Nc * self.nd
        return I

    # ---- the rt_* calls ------------------------------------------------------------------------
    def transport(self, I_in, I_base, dt, T=None):
        I_in, I_base = self._I(I_in), self._I(I_base)
        out = np.empty_like(I_in)
        T = self.T if T is None else _c(T)
        _load().orc_transport(ctypes.byref(self.P), _ptr(I_in), _ptr(T), _ptr(I_base), _ptr(out), dt)
        return out

    def angular_flux(self, I_in, I_inout, dt):
        I_in = self._I(I_in)
        out = self._I(I_inout).copy()
        _load().orc_angular(ctypes.byref(self.P), _ptr(I_in), _ptr(out), dt)
        return out

    def source_implicit(self, I, T, dt):
        I, T = self._I(I).copy(), _c(T).copy()
        nf = _load().orc_source(ctypes.byref(self.P), _ptr(I), _ptr(T), dt)
        return I, T, nf

    def moments(self, I):
        I = self._I(I)
        R = np.empty((16,) + self.n[::-1])
        _load().orc_moments(ctypes.byref(self.P), _ptr(I), _ptr(R))
        return R

    def step(self, I, T, dt):
        """One predictor-corrector step O8.  returns (I, T, R[16,..], G[4,..], n_fail)."""
        I, T = self._I(I).copy(), _c(T).copy()
        R = np.empty((16,) + self.n[::-1]); G = np.empty((4,) + self.n[::-1])
        Ih = np.empty_like(I); Th = np.empty_like(T); Rb = np.empty_like(R)
        nf = _load().orc_step(ctypes.byref(self.P), _ptr(I), _ptr(T), _ptr(R), _ptr(G), dt,
                              _ptr(Ih), _ptr(Th), _ptr(Rb))
        return I, T, R, G, nf

    def mapr_gradient(self, Ic, s):
        """O4' gradient (3-vector tangent at nhat_s) of direction s for one cell's intensities Ic[nd]."""
        Ic, g = _c(Ic), np.zeros(3)
        _load().orc_mapr_gradient(ctypes.byref(self.P), _ptr(Ic), int(s), _ptr(g))
        return g

    def cfl(self):
        """(spatial bound L464, angular bound S14)."""
        out = np.zeros(2)
        _load().orc_cfl(ctypes.byref(self.P), _ptr(out))
        return float(out[0]), float(out[1])
