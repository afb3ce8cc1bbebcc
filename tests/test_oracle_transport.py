"""Pins for O3-O5 (oracle/rt_oracle.c transport + angular update): exact facts, closed forms.  CPU only."""
import numpy as np
import pytest

from oracle import Oracle

PER = ("periodic",) * 3


def _flat(n, level=2, **opt):
    grid = dict(n=n, x0=(0.0, 0.0, 0.0), dx=tuple(1.0 / max(n) for _ in range(3)), bc_lo=PER, bc_hi=PER)
    o = dict(method=0)
    o.update(opt)
    return Oracle(grid, "minkowski", {}, level, o)


def test_uniform_field_is_invariant():
    o = _flat((6, 5, 4))
    I = np.full((4, 5, 6, o.nd), 0.37)
    assert np.abs(o.transport(I, I, 0.05) - I).max() < 1e-15
    assert np.abs(o.angular_flux(I, I, 0.05) - I).max() == 0.0        # omega = 0 in Cartesian flat space


def test_donor_cell_exact_shift_along_pole():
    """First-order upwind at dt = dx along the polar direction (an exact grid direction, nhat = +-z)
    shifts the field by exactly one cell."""
    o = _flat((3, 3, 8), limiter=3)
    rng = np.random.default_rng(0)
    I = rng.uniform(size=(8, 3, 3, o.nd))
    out = o.transport(I, I, 1.0 / 8).reshape(I.shape)
    assert np.abs(out[..., 0] - np.roll(I[..., 0], 1, axis=0)).max() < 1e-14      # s = 0: +z
    assert np.abs(out[..., -1] - np.roll(I[..., -1], -1, axis=0)).max() < 1e-14    # s = nd-1: -z


def test_conservation_periodic_vacuum_and_opaque():
    """sum_l sqrt(-g) sum_s w_s n^0 n_0 I is conserved to round-off by the flux-difference form (Eq 18)."""
    rng = np.random.default_rng(1)
    for opt in (dict(), dict(kappa_s=40.0)):
        o = _flat((6, 5, 4), **opt)
        rho = np.ones((4, 5, 6)) * (rng.uniform(size=(4, 5, 6)) > 0.3)           # mixed vacuum / opaque faces
        u4 = np.zeros((4, 4, 5, 6))
        v = 0.3 * rng.uniform(-1, 1, size=(3, 4, 5, 6))
        u4[0] = 1 / np.sqrt(1 - (v ** 2).sum(0))
        u4[1:] = u4[0] * v
        o.set_fluid(rho, np.ones((4, 5, 6)), u4)
        I = rng.uniform(size=(4, 5, 6, o.nd))
        out = o.transport(I, I, 0.02).reshape(I.shape)
        assert np.abs(out - I).max() > 1e-3
        tot0, tot1 = (I * o.ang["w"]).sum(), (out * o.ang["w"]).sum()
        assert abs(tot1 - tot0) < 1e-12 * abs(tot0)


def _muscl_1d(u, c, nu):
    """Textbook MUSCL (MC limiter, forward Euler) for u_t + c u_x = 0, periodic; independent 10-line check."""
    dm, dp = u - np.roll(u, 1), np.roll(u, -1) - u
    s = np.where(dm * dp > 0, np.sign(dm) * np.minimum(np.minimum(2 * np.abs(dm), 2 * np.abs(dp)), 0.5 * np.abs(dm + dp)), 0.0)
    uL, uR = u + 0.5 * s, np.roll(u - 0.5 * s, -1)          # states at face i+1/2
    F = c * np.where(c > 0, uL, uR)
    return u - nu * (F - np.roll(F, 1))


def test_pli_mc_equals_textbook_muscl():
    o = _flat((32, 1, 1))
    rng = np.random.default_rng(2)
    I = rng.uniform(size=(1, 1, 32, o.nd))
    dt = 0.4 / 32
    out = o.transport(I, I, dt).reshape(I.shape)
    for s in (0, 5, 17, 30, 41):
        ref = _muscl_1d(I[0, 0, :, s], o.ang["nhat"][s, 0], dt * 32)
        assert np.abs(out[0, 0, :, s] - ref).max() < 1e-14


def test_beam_stays_on_its_ray_and_moves_at_c():
    """Config-1-like beam (L490-496, L478): injected at x = 0 along a grid direction in the z = 0 plane."""
    N = 32
    grid = dict(n=(N, N, 1), x0=(0, 0, 0), dx=(1 / N,) * 3, bc_lo=("fixed", "outflow", "periodic"),
                bc_hi=("outflow", "outflow", "periodic"))
    o = Oracle(grid, "minkowski", {}, 2, dict(method=0))
    nh = o.ang["nhat"]
    s = int(np.argmax(nh @ (np.array([1, 1, 0]) / np.sqrt(2))))
    ghost = np.zeros((2, N, o.nd))
    ghost[:, 4:8, s] = 1.0
    o.set_boundary(0, 0, ghost)
    I = np.zeros((1, N, N, o.nd))
    dt, nst = 0.4 / N, 40
    for _ in range(nst):
        Ih = o.transport(I, I, dt / 2)
        I = o.transport(Ih, I, dt).reshape(I.shape)
    assert np.abs(np.delete(I, s, axis=-1)).max() == 0.0             # directions do not mix in flat space
    b = I[0, :, :, s]
    assert b.min() > -1e-12 and b.max() < 1 + 1e-12                  # limited scheme: no new extrema
    x = (np.arange(N) + 0.5) / N
    t = nst * dt
    # front position along x: the x-integrated profile of the beam ends at x = nhat_x * t (speed of light = 1)
    prof = b.sum(0) / b.sum(0).max()
    front = x[np.argmin(np.abs(prof - 0.5))]
    assert abs(front - nh[s, 0] * t) < 2.0 / N
    # centroid in y at a given x follows the straight ray y = y0 + x * ny/nx
    i = N // 5
    yc = (b[:, i] * x).sum() / b[:, i].sum()
    assert abs(yc - (6.0 / N + x[i] * nh[s, 1] / nh[s, 0])) < 1.0 / N


def test_opaque_flux_reduces_to_eq_B9():
    """tau >> 1: Eq 23 -> 1/2 mu (I_i + I_{i+1}) e^-tau - |mu|/(2 tau) (I_{i+1} - I_i)  (Eq B9): with
    e^-tau negligible only the diffusive term survives, with coefficient |mu| f(tau)/2 -> |mu|/(2 tau)."""
    N = 16
    o = _flat((N, 1, 1), kappa_s=1.0e4 * N)
    o.set_fluid(np.ones((1, 1, N)), np.ones((1, 1, N)), None)
    rng = np.random.default_rng(3)
    I = rng.uniform(size=(1, 1, N, o.nd))
    dt = 0.5 / N
    tau = 1.0e4 * N * dt
    out = o.transport(I, I, dt).reshape(I.shape)
    mu = np.abs(o.ang["nhat"][:, 0])
    lap = np.roll(I, -1, axis=2) - 2 * I + np.roll(I, 1, axis=2)
    ref = I + dt * N * mu / (2 * tau) * lap
    assert np.abs(out - ref).max() < 1e-12


def test_angular_update_conserves_per_cell_and_masks():
    """KS: sum_s w_s delta(n^0 n_0 I)_s = 0 per cell when nothing is masked (r >= 3), and masked
    directions (n_0 > -0.1) are zeroed near the horizon."""
    for lo, hi, expect_mask in ((np.log(4.0), np.log(8.0), False), (np.log(1.3), np.log(1.9), True)):
        grid = dict(n=(4, 4, 1), x0=(lo, 0.2, 0.0), dx=((hi - lo) / 4, 0.15, 0.1), bc_lo=("outflow", "outflow", "periodic"),
                    bc_hi=("outflow", "outflow", "periodic"), x3_symmetric=True)
        o = Oracle(grid, "ks_mks", dict(a=0.9, hslope=0.3), 4, dict(method=0))
        rng = np.random.default_rng(4)
        I = rng.uniform(0.5, 1.0, size=(1, 4, 4, o.nd))
        dt = 1e-3
        out = o.angular_flux(I, I, dt).reshape(I.shape)
        e, g = o.tab["e_c"], o.tab["g_c"]
        n = e[..., :, 0][..., None, :] + np.einsum("...mi,si->...sm", e[..., :, 1:], o.ang["nhat"])
        n0 = np.einsum("...m,...sm->...s", g[..., 0, :], n)
        masked = n0 > -0.1
        assert masked.any() == expect_mask
        assert np.all(out[masked] == 0.0)
        if not expect_mask:
            d = ((out - I) * n[..., 0] * n0 * o.ang["w"]).sum(-1)
            assert np.abs(d).max() < 1e-15 * 50
            assert np.abs(out - I).max() > 1e-6


def test_second_order_convergence_smooth_profile():
    """O8 stepping in vacuum: L1 error of a smooth advected 1-D profile drops ~4x per grid doubling."""
    errs = []
    for N in (32, 64):
        grid = dict(n=(N, 1, 1), x0=(0, 0, 0), dx=(1 / N,) * 3, bc_lo=PER, bc_hi=PER)
        o = Oracle(grid, "minkowski", {}, 1, dict(method=0, limiter=2))
        x = (np.arange(N) + 0.5) / N
        I0 = np.tile((1 + 0.5 * np.sin(2 * np.pi * x))[None, None, :, None], (1, 1, 1, o.nd))
        I, T = I0.copy(), np.ones((1, 1, N))
        dt, nst = 0.4 / N, N // 2
        for _ in range(nst):
            I, T, R, Gf, nf = o.step(I, T, dt)
        I = I.reshape(I0.shape)
        s = 1                                                     # nhat_x = 0.5257...
        ex = 1 + 0.5 * np.sin(2 * np.pi * (x - o.ang["nhat"][s, 0] * dt * nst))
        errs.append(np.abs(I[0, 0, :, s] - ex).mean())
    assert errs[0] / errs[1] > 3.0


def test_mapr_linear_exactness_constant_reduction_and_conservation():
    """O4' (MAPR, reading S6; PARITY UNPINNED beyond these facts): exact for fields linear in the tangent plane,
    reduces to donor cell for a constant field, and stays conservative per cell."""
    o = Oracle(dict(n=(1, 1, 1), x0=(0, 0, 0), dx=(1, 1, 1), bc_lo=PER, bc_hi=PER), "minkowski", {}, 4, dict(method=0, ang_recon=1))
    nh, nb, nnb = o.ang["nhat"], o.ang["nb"], o.ang["nnb"]
    rng = np.random.default_rng(11)
    for s in (0, 7, 50, 161):
        c0 = nh[s]
        g = rng.normal(size=3)
        g -= (g @ c0) * c0                                    # a gradient in the tangent plane at n_s
        I = np.zeros(o.nd)
        I[s] = 0.3
        for t in nb[s, :nnb[s]]:
            dot = c0 @ nh[t]
            p = nh[t] - dot * c0
            I[t] = 0.3 + g @ (np.arctan2(np.linalg.norm(p), dot) * p / np.linalg.norm(p))   # independent log map
        assert np.abs(o.mapr_gradient(I, s) - g).max() < 1e-12
    # constant field: gradient zero, MAPR == donor cell; and per-cell conservation in a curved metric
    grid = dict(n=(3, 3, 1), x0=(np.log(4.0), 0.3, 0.0), dx=(0.2, 0.1, 0.1), bc_lo=("outflow", "outflow", "periodic"),
                bc_hi=("outflow", "outflow", "periodic"), x3_symmetric=True)
    om = Oracle(grid, "ks_mks", dict(a=0.9, hslope=0.3), 4, dict(method=0, ang_recon=1))
    od = Oracle(grid, "ks_mks", dict(a=0.9, hslope=0.3), 4, dict(method=0, ang_recon=0))
    Ic = np.tile(rng.uniform(0.5, 1.0, size=(1, 3, 3, 1)), (1, 1, 1, om.nd))
    assert np.abs(om.angular_flux(Ic, Ic, 1e-3) - od.angular_flux(Ic, Ic, 1e-3)).max() < 1e-15
    I = rng.uniform(0.5, 1.0, size=(1, 3, 3, om.nd))
    out = om.angular_flux(I, I, 1e-3).reshape(I.shape)
    e, g = om.tab["e_c"], om.tab["g_c"]
    n = e[..., :, 0][..., None, :] + np.einsum("...mi,si->...sm", e[..., :, 1:], om.ang["nhat"])
    n0 = np.einsum("...m,...sm->...s", g[..., 0, :], n)
    assert np.abs(((out - I) * n[..., 0] * n0 * om.ang["w"]).sum(-1)).max() < 1e-16 * 50
    assert np.abs(out - od.angular_flux(I, I, 1e-3).reshape(I.shape)).max() > 1e-7        # and it is not donor cell


def test_snake_coordinates_beam_is_straight_in_cartesian():
    """PAPER.md 4.6 (L559, Fig 7; A = 0.1, k = 2): a beam in snake coordinates bends in (w, y) but is a straight line
    once mapped back to x = w + A sin(k pi y).  The intensity centroid of every mesh column must sit on the central
    ray within 1.5 cells, while the straight line in (w, y) is several cells away (so a wrong sign or a missing
    delta in n^w fails)."""
    import math
    import rt_workloads as W
    N = 48
    cfg = W.config(6, n=(N, N, 1), level=2)
    kind, params = cfg["metric"]
    orc = Oracle(cfg["grid"], kind, params, cfg["level"], cfg["options"])
    f = W.fields(cfg, orc.ang["nhat"], orc.tab["e_c"])
    orc.set_fluid(f["rho"], f["T"], f["u4"])
    for (d, s), g in f["ghosts"].items():
        orc.set_boundary(d, s, g)
    dt = cfg["dt"]
    I, T = f["I0"].copy(), f["T"].copy()
    for _ in range(int(0.9 / dt)):
        out = orc.step(I, T, dt)
        I, T = out[0], out[1]
    s = f["beam_dir"]
    n = orc.ang["nhat"][s]
    Ib = I.reshape(N, N, -1)[:, :, s]          # [j, i]
    A, k = params["A"], params["k"]
    y = (np.arange(N) + 0.5) / N
    y0 = 0.5 * (N // 8 + N // 4) / N             # centre of the illuminated rows
    ts = np.linspace(0.0, 1.5, 30001)            # the central ray, straight in Cartesian coordinates
    xr, yr = A * math.sin(k * math.pi * y0) + n[0] * ts, y0 + n[1] * ts
    wr = xr - A * np.sin(k * np.pi * yr)
    worst, bent = 0.0, 0.0
    for i in range(4, 22, 2):
        col = Ib[:, i]
        assert col.sum() > 1.0
        yb = (col * y).sum() / col.sum()
        wi = (i + 0.5) / N
        worst = max(worst, abs(yb - yr[np.argmax(wr >= wi)]) * N)
        bent = max(bent, abs(yb - (y0 + n[1] / n[0] * wi)) * N)
    assert worst < 1.5, worst
    assert bent > 4.0, bent


@pytest.mark.parametrize("v", [0.05, -0.05])
def test_dynamic_diffusion_pulse_is_advected_with_the_flow(v):
    """PAPER.md 4.9 (L656-664): in a scattering-dominated medium moving uniformly with v^x = 0.05 "the radiation should
    be advected with the flow": after t = 2 the pulse has moved by v t (here to 0.5 %; either sign).  This is the pin of
    Eq 23's advective term (readings S10/S11: n^0 v^a I, upwinded on v): without it the pulse does not move, with the
    downwind choice it is unstable, with a wrong sign it moves the other way."""
    import math
    N = 64
    grid = dict(n=(N, 1, 1), x0=(0.0, 0.0, 0.0), dx=(1.0 / N,) * 3, bc_lo=("periodic",) * 3, bc_hi=("periodic",) * 3)
    o = Oracle(grid, "minkowski", {}, 2, dict(method=1, kappa_a0=0.0, kappa_s=10.0 * N, a_rad=1.0, Y_over_rho=1.5))
    nd, w = o.nd, o.ang["w"]
    x = (np.arange(N) + 0.5) / N
    gam = 1.0 / math.sqrt(1.0 - v * v)
    u4 = np.zeros((4, 1, 1, N)); u4[0] = gam; u4[1] = gam * v
    o.set_fluid(np.ones((1, 1, N)), np.ones((1, 1, N)), u4)
    I = np.repeat(np.exp(-(x - 0.5) ** 2 / (2 * 0.08 ** 2))[:, None] / (4 * np.pi), nd, axis=1).reshape(1, 1, N, nd).copy()
    T = np.ones((1, 1, N))

    def centroid(I):   # periodic centroid of the lab-frame energy density
        E = (I.reshape(N, nd) * w).sum(1)
        return (np.angle((E * np.exp(2j * np.pi * x)).sum()) / (2 * np.pi)) % 1.0

    c0, dt, t = centroid(I), 0.5 / N, 0.0
    for _ in range(256):
        out = o.step(I, T, dt)
        I, T = out[0], out[1]
        t += dt
    assert abs((centroid(I) - c0) - v * t) < 0.005 * abs(v * t)


@pytest.mark.parametrize("matter", [False, True])
def test_reflecting_boundary_is_the_mirror_image_problem(matter):
    """'Symmetric boundaries for the polar angle' (L709; reading S23: mirror cell, direction with the normal tetrad
    component flipped, normal fluid velocity reversed).  A reflecting wall at x2 = 0 must give exactly what the doubled
    domain with mirror-symmetric data gives in its upper half -- intensities, temperature and moments."""
    import math
    from oracle import mirror_map
    n1, n2, n3 = 5, 6, 3
    opt = dict(method=2, kappa_a0=8.0, kappa_s=4.0, a_rad=1.0, Y_over_rho=1.5) if matter else dict(method=0)
    dx = (0.1, 0.1, 0.1)
    half = dict(n=(n1, n2, n3), x0=(0.0, 0.0, 0.0), dx=dx, bc_lo=("periodic", "reflect", "periodic"),
                bc_hi=("periodic", "outflow", "periodic"))
    full = dict(n=(n1, 2 * n2, n3), x0=(0.0, -n2 * dx[1], 0.0), dx=dx, bc_lo=("periodic", "outflow", "periodic"),
                bc_hi=("periodic", "outflow", "periodic"))
    oh, of = Oracle(half, "minkowski", {}, 2, opt), Oracle(full, "minkowski", {}, 2, opt)
    nd = oh.nd
    m = mirror_map(oh.ang["nhat"], 1)
    assert m is not None and (m[m] == np.arange(nd)).all() and (m != np.arange(nd)).any()
    assert mirror_map(oh.ang["nhat"], 0) is None and mirror_map(oh.ang["nhat"], 2) is None   # no such symmetry (S2)
    with pytest.raises(ValueError):
        Oracle(dict(half, bc_lo=("reflect", "outflow", "periodic"), bc_hi=("outflow", "outflow", "periodic")), "minkowski", {}, 2, opt)
    rng = np.random.default_rng(12)
    I = rng.uniform(0.2, 1.0, (n3, n2, n1, nd))
    rho, T = rng.uniform(0.5, 1.5, (n3, n2, n1)), rng.uniform(0.8, 1.2, (n3, n2, n1))
    v = 0.3 * rng.uniform(-1, 1, (3, n3, n2, n1))
    gam = 1.0 / np.sqrt(1.0 - (v ** 2).sum(0))
    u4 = np.concatenate([gam[None], gam[None] * v])
    flip = lambda a: a[:, ::-1]                                         # mirror in x2 (arrays are [k, j, i, ...])
    If = np.concatenate([flip(I)[..., m], I], axis=1)
    rhof, Tf = np.concatenate([flip(rho), rho], 1), np.concatenate([flip(T), T], 1)
    u4m = u4[:, :, ::-1].copy(); u4m[2] *= -1.0                          # u^y reversed in the image
    u4f = np.concatenate([u4m, u4], axis=2)
    if matter:
        oh.set_fluid(rho, T, u4); of.set_fluid(rhof, Tf, u4f)
    dt = 0.03
    Th, Tfull = T.copy(), Tf.copy()
    for _ in range(4):
        I, Th, Rh, Gh, _ = oh.step(I, Th, dt)
        If, Tfull, Rf, Gf, _ = of.step(If, Tfull, dt)
    I, If = I.reshape(n3, n2, n1, nd), If.reshape(n3, 2 * n2, n1, nd)
    tol = 1e-13      # (the grid's mirror pairs agree to 3e-16 only, so not bit for bit)
    assert np.abs(If[:, n2:] - I).max() < tol
    assert np.abs(If[:, :n2] - I[:, ::-1][..., m]).max() < tol          # and the image stays the image
    assert np.abs(Tfull.reshape(n3, 2 * n2, n1)[:, n2:] - Th.reshape(n3, n2, n1)).max() < tol
    assert np.abs(Rf.reshape(16, n3, 2 * n2, n1)[:, :, n2:] - Rh.reshape(16, n3, n2, n1)).max() < tol
    # and it is not what an open boundary gives
    oo = Oracle(dict(half, bc_lo=("periodic", "outflow", "periodic")), "minkowski", {}, 2, opt)
    if matter:
        oo.set_fluid(rho, T, u4)
    Io = oo.step(I.copy(), Th.copy(), dt)[0].reshape(I.shape)
    Ir = oh.step(I.copy(), Th.copy(), dt)[0].reshape(I.shape)
    assert np.abs(Io - Ir)[:, 0].max() > 1e-4
