"""RT_USER: metric (and optionally tetrad) from the caller's host functions (rt_metric.g_fn / e_fn, called inside rt_init only).

(1) callbacks that return the Kerr-Schild metric / the paper's A3-A4 tetrad give the tables of the built-in RT_KS_MKS kind;
(2) a metric the library has never seen -- conformally flat with a lapse and a shift, x3-independent -- runs whole steps with
    opacities and a moving fluid against the oracle, with the library's own tetrad and with a caller-supplied one.
"""
import numpy as np
import pytest

import rt_workloads as W
from oracle import geometry as G
from parity_util import TOL, make_pair, rel_err, run_steps

pytestmark = pytest.mark.gpu


@pytest.mark.parametrize("with_tetrad", [False, True])
def test_user_callbacks_returning_kerr_schild_give_the_builtin_tables(with_tetrad):
    from paper_2508_15532_b200 import rt
    cfg = W.config(4, n=(10, 8, 2))
    kind, params = cfg["metric"]
    ref = rt.RtContext(cfg["grid"], kind, params, 2, cfg["options"])
    user = dict(g=lambda x: G.metric(kind, params, x), e=(lambda x: G.tetrad(kind, params, x)[0]) if with_tetrad else None)
    ctx = rt.RtContext(cfg["grid"], "user", user, 2, cfg["options"])
    for which, tol in (("g_c", 1e-13), ("e_c", 1e-12), ("einv_c", 1e-11), ("sqrtg_c", 1e-12), ("omega_c", 1e-9), ("angcoef", 1e-9)):
        a, b = ctx.geometry(which), ref.geometry(which)
        assert np.isfinite(a).all() and np.abs(a - b).max() <= tol * max(1.0, np.abs(b).max()), which
    assert ctx.cfl_dt() == pytest.approx(ref.cfl_dt(), rel=1e-9)
    ctx.close(); ref.close()


def _toy_metric(x):
    """g = -N^2 dt^2 + psi^4 delta_ij (dx^i + b^i dt)(dx^j + b^j dt), N, psi, b functions of (x1, x2)."""
    c1, s2 = np.cos(2 * np.pi * x[0]), np.sin(2 * np.pi * x[1])
    N = 1.0 - 0.2 * c1 * s2
    p4 = (1.0 + 0.1 * np.sin(2 * np.pi * x[0]) * np.cos(2 * np.pi * x[1])) ** 4
    b = np.array([0.15 * s2, -0.1 * c1, 0.05 * c1 * s2])
    g = np.zeros((4, 4))
    g[1:, 1:] = p4 * np.eye(3)
    g[0, 1:] = g[1:, 0] = p4 * b
    g[0, 0] = -N * N + p4 * (b @ b)
    return g


def _toy_tetrad(x):
    """A different orthonormal frame of the same metric: e_0 as Eq 4 demands, the space-like legs turned about e_3 by an angle that
    varies over the mesh (any such frame is admissible, L57-79; its Ricci rotation coefficients differ from the default frame's)."""
    g = _toy_metric(x)
    e, _ = G._tetrad_from_metric(g[None])
    e = e[0]
    al = 0.3 * np.sin(2 * np.pi * x[0])
    out = e.copy()
    out[:, 1] = np.cos(al) * e[:, 1] + np.sin(al) * e[:, 2]
    out[:, 2] = -np.sin(al) * e[:, 1] + np.cos(al) * e[:, 2]
    return out


@pytest.mark.parametrize("efun", [None, _toy_tetrad])
def test_steps_in_a_user_metric_match_the_oracle(efun):
    cfg = W.config(2, n=(10, 8, 4))
    cfg["grid"] = dict(cfg["grid"], x3_symmetric=True)
    cfg["metric"] = ("user", dict(g=_toy_metric, e=efun))
    cfg["options"] = dict(cfg["options"], kappa_s=3.0, n0_floor=0.1)
    cfg["dt"] = None
    orc, ctx, f, dt = make_pair(cfg)
    assert np.abs(orc.tab["omega_c"]).max() > 0.05          # the angular flux is at work
    assert np.abs(ctx.geometry("omega_c")[0] - orc.tab["omega_c"][0]).max() < 1e-9
    rng = np.random.default_rng(2)
    f["I0"] = f["I0"] + rng.uniform(0.05, 0.1, size=f["I0"].shape)
    out = run_steps(orc, ctx, f, 0.5 * dt, 3)
    for k in ("I", "T", "R"):
        assert rel_err(*out[k]) <= TOL, k
    assert float(np.abs(out["G"][0] - out["G"][1]).max() * out["dt"] / np.abs(out["R"][1]).max()) <= TOL
    ctx.close()


def test_user_metric_needs_its_function_and_x3_symmetry():
    import ctypes
    from paper_2508_15532_b200 import rt
    lib = rt.lib()
    g = rt.RtGrid(); g.n[:] = (4, 4, 2); g.x0[:] = (0, 0, 0); g.dx[:] = (0.1, 0.1, 0.1)
    g.bc_lo[:] = (0, 0, 0); g.bc_hi[:] = (0, 0, 0)
    o = rt.RtOptions(**rt.DEFAULT_OPTIONS)
    h = ctypes.c_void_p()
    m = rt.RtMetric(rt.METRIC["user"], 0.0, 0.3, 1, 0.0, 0.0)              # no g_fn
    assert lib.rt_init(ctypes.byref(g), ctypes.byref(m), 2, ctypes.byref(o), ctypes.byref(h)) == -1
    cb = rt._metric_callback(_toy_metric)
    m = rt.RtMetric(rt.METRIC["user"], 0.0, 0.3, 0, 0.0, 0.0); m.g_fn = cb  # x3_symmetric = 0
    assert lib.rt_init(ctypes.byref(g), ctypes.byref(m), 2, ctypes.byref(o), ctypes.byref(h)) == -1
