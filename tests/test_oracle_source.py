"""Pins for O6-O8 (implicit source step, moments, step driver).  CPU only."""
import os

import numpy as np
import pytest

from oracle import Oracle

PER = ("periodic",) * 3
FOURPI = 4 * np.pi
GOLD = dict((l.split()[0], float(l.split()[1])) for l in open(os.path.join(os.path.dirname(__file__), "golden", "paper_values.txt"))
            if l.strip() and not l.startswith("#"))


def _cell(level=4, kind="minkowski", params=None, grid=None, **opt):
    grid = grid or dict(n=(1, 1, 1), x0=(0, 0, 0), dx=(1, 1, 1), bc_lo=PER, bc_hi=PER)
    return Oracle(grid, kind, params or {}, level, opt)


def _boosted_u(v):
    v = np.asarray(v, float)
    g = 1 / np.sqrt(1 - v @ v)
    return np.concatenate([[g], g * v]).reshape(4, 1, 1, 1)


@pytest.mark.parametrize("method", [1, 2, 3])
def test_equilibration_paper_4_10(method):
    """L672-693: Gamma = 5/3, T_gas = 2, T_rad = 1, rho = 1, a_rad = k_B/(mu m_p) = 1: relaxes to T_eq with
    T_rad^4 + 1.5 T_gas = 4 conserved every step (Fig 12 bottom panel)."""
    o = _cell(method=method, kappa_a0=1.0, kappa_s=0.3)
    o.set_fluid(np.ones((1, 1, 1)), np.full((1, 1, 1), 2.0), None)
    I, T = np.full(o.nd, 1 / FOURPI), np.array([2.0])
    w = o.ang["w"]
    for _ in range(300):
        I, T, nf = o.source_implicit(I, T, 0.2)
        assert nf == 0
        assert abs((I * w).sum() + 1.5 * T[0] - 4.0) < 1e-11
    assert abs(T[0] - GOLD["T_eq"]) < 1e-9
    assert abs(((I * w).sum()) ** 0.25 - GOLD["T_eq"]) < 1e-9
    assert np.abs(I - I.mean()).max() < 1e-15                       # stays isotropic


def test_equilibrium_is_a_fixed_point_also_for_moving_fluid_energy_balance():
    for method in (1, 2, 3):
        o = _cell(method=method, kappa_a0=2.0, kappa_s=0.5)
        o.set_fluid(np.ones((1, 1, 1)), np.full((1, 1, 1), 1.3), None)
        I0, T0 = np.full(o.nd, 1.3 ** 4 / FOURPI), np.array([1.3])
        I, T, nf = o.source_implicit(I0, T0, 0.7)
        assert nf == 0 and abs(T[0] - 1.3) < 1e-13 and np.abs(I - I0).max() < 1e-14


@pytest.mark.parametrize("method", [1, 2, 3])
def test_energy_equation_eq39_and_eq40_moving_fluid(method):
    """Eq 39: Y (T+ - T-) = -(E+ - E-) with E = sum Ibar dOmegabar (fluid frame, S17), for a moving fluid and
    an anisotropic field; and sum Ibar+ dOmegabar = E+ of Eq 39 (S19b, conservative reading)."""
    o = _cell(method=method, kappa_a0=1.5, kappa_s=0.8)
    u4 = _boosted_u([0.3, -0.2, 0.4])
    o.set_fluid(np.full((1, 1, 1), 1.2), np.full((1, 1, 1), 0.9), u4)
    rng = np.random.default_rng(5)
    I0, T0 = rng.uniform(0.1, 1.0, o.nd), np.array([0.9])
    I, T, nf = o.source_implicit(I0, T0, 0.35)
    assert nf == 0
    nbar = u4[0, 0, 0, 0] - o.ang["nhat"] @ u4[1:, 0, 0, 0]
    Em, Ep = (nbar ** 2 * I0 * o.ang["w"]).sum(), (nbar ** 2 * I * o.ang["w"]).sum()
    Y = 1.5 * 1.2
    tol = 1e-12 if method != 3 else 1e-10
    assert abs(Y * (T[0] - T0[0]) + (Ep - Em)) < tol * Em


def test_frozen_temperature_backward_euler_closed_form():
    """Y -> infinity freezes T: per direction I_k = B - (B - I_0) (1 + alpha dt)^-k, B = a T^4 / 4 pi (static fluid)."""
    o = _cell(method=1, kappa_a0=2.0, kappa_s=0.0, Y_over_rho=1e30)
    Tg = 1.1
    o.set_fluid(np.ones((1, 1, 1)), np.full((1, 1, 1), Tg), None)
    alpha, B, dt = 2.0 * Tg ** -3.5, Tg ** 4 / FOURPI, 0.3
    rng = np.random.default_rng(6)
    I0 = rng.uniform(0, 1, o.nd)
    I, T = I0.copy(), np.array([Tg])
    for k in range(1, 6):
        I, T, nf = o.source_implicit(I, T, dt)
        assert np.abs(I - (B - (B - I0) * (1 + alpha * dt) ** -k)).max() < 1e-13
    assert abs(T[0] - Tg) < 1e-13


def test_pure_scattering_static_isotropises():
    """kappa_a = 0, static fluid: E unchanged, T unchanged, anisotropy x 1/(1 + alpha_s dt) per step."""
    o = _cell(method=1, kappa_a0=0.0, kappa_s=3.0)
    o.set_fluid(np.ones((1, 1, 1)), np.ones((1, 1, 1)), None)
    rng = np.random.default_rng(7)
    I0 = rng.uniform(0, 1, o.nd)
    w = o.ang["w"]
    E0 = (I0 * w).sum()
    I, T, nf = o.source_implicit(I0, np.ones(1), 0.25)
    assert abs((I * w).sum() - E0) < 1e-14 * E0 and abs(T[0] - 1) < 1e-13
    assert np.abs((I - E0 / FOURPI) - (I0 - E0 / FOURPI) / (1 + 3.0 * 0.25)).max() < 1e-14


def _sums(o, I0, T0, rho, dt, u4):
    nbar = u4[0].ravel()[0] - o.ang["nhat"] @ u4[1:].reshape(3)
    alpha = o.opt["kappa_a0"] * rho ** 2 * T0 ** -3.5 + o.opt["kappa_s"] * rho
    d = u4[0].ravel()[0] * 0 + 1.0 + nbar * alpha * dt            # n^0 = 1 in flat space
    w = o.ang["w"]
    E = (nbar ** 2 * I0 * w).sum()
    A1 = (1.0 / d * nbar ** 2 * I0 * w).sum()
    A2 = dt / FOURPI * (w / (nbar * d)).sum()
    return E, A1, A2, alpha


def test_temperature_roots_against_numpy_roots():
    """Method 1: quartic Eq 42; Method 2: quadratic in sqrt(T) Eq 43 (closed form); Method 3: Eq 46 as a degree-9
    polynomial in sqrt(T) (S19).  The oracle's T+ must be the physical root given by numpy.roots."""
    rho, T0, dt = 1.2, 0.9, 0.35
    u4 = _boosted_u([0.3, -0.2, 0.4])
    rng = np.random.default_rng(5)
    for method in (1, 2, 3):
        o = _cell(method=method, kappa_a0=1.5, kappa_s=0.8)
        o.set_fluid(np.full((1, 1, 1), rho), np.full((1, 1, 1), T0), u4)
        I0 = np.random.default_rng(5).uniform(0.1, 1.0, o.nd)
        _, T, nf = o.source_implicit(I0, np.array([T0]), dt)
        E, A1, A2, alpha = _sums(o, I0, T0, rho, dt, u4)
        Y, als, N = 1.5 * rho, 0.8 * rho, 1.5 * rho ** 2
        W = E + Y * T0
        b, c = Y * (1 - A2 * als), A1 - Y * (1 - A2 * als) * T0 - (1 - A2 * als) * E
        if method == 1:
            roots = np.roots([A2 * N * T0 ** -3.5, 0, 0, b, c])
        elif method == 2:
            a = A2 * N
            x = (-a + np.sqrt(a * a - 4 * b * c)) / (2 * b)
            roots = np.array([x * x])
        else:
            A1p, A2p = alpha * dt * A1, alpha * dt * A2
            p = np.zeros(10)                                       # coefficients of x^9 ... x^0, x = sqrt(T)
            p[0] = Y * als * (A2p - dt)
            p[1] = -A2p * N
            p[2] = -(A2p * als * W + A1p - W * als * dt)
            p[7] = -Y * N * dt
            p[9] = W * N * dt
            roots = np.roots(p)
            roots = roots[(np.abs(roots.imag) < 1e-9) & (roots.real > 0)].real ** 2
        roots = np.asarray(roots)
        roots = roots[np.isreal(roots)].real
        roots = roots[(roots > 0) & (roots <= W / Y * (1 + 1e-12))]
        assert len(roots) == 1 and nf == 0
        assert abs(T[0] - roots[0]) < 1e-11 * roots[0]


def test_safeguarded_newton_brackets_root_for_stiff_data():
    """L355/L401: a raw Newton iteration on Eq 42 can leave T > 0 for stiff data; the root itself always lies in
    (0, W/Y] because f(0) = c0 < 0 <= f(W/Y) (DESIGN reading S20), so no cell may fail here."""
    o = _cell(method=1, kappa_a0=5e3, kappa_s=0.0, Y_over_rho=1e-3)
    o.set_fluid(np.ones((1, 1, 1)), np.full((1, 1, 1), 3.0), None)
    I, T, nf = o.source_implicit(np.zeros(o.nd), np.array([3.0]), 10.0)
    assert nf == 0 and 0 < T[0] < 3.0
    E = (I * o.ang["w"]).sum()
    assert abs(E + 1e-3 * T[0] - 1e-3 * 3.0) < 1e-12


def test_density_floor_skips_interaction():
    o = _cell(method=2, kappa_a0=5.0, kappa_s=5.0)
    o.set_fluid(np.full((1, 1, 1), 4e-4), np.ones((1, 1, 1)), None)          # below 5e-4 (L468)
    I0 = np.random.default_rng(8).uniform(size=o.nd)
    I, T, nf = o.source_implicit(I0, np.ones(1), 1.0)
    assert np.all(I == I0) and T[0] == 1.0 and nf == 0


def test_moments_isotropic_single_direction_and_trace():
    o = _cell()
    E = 2.5
    R = o.moments(np.full(o.nd, E / FOURPI)).reshape(4, 4)
    assert np.abs(R - np.diag([-E, E / 3, E / 3, E / 3])).max() < 1e-14        # S24: R^mu_nu
    I = np.zeros(o.nd)
    I[7] = 1.7
    n = np.concatenate([[1.0], o.ang["nhat"][7]])
    R = o.moments(I).reshape(4, 4)
    assert np.abs(R - o.ang["w"][7] * 1.7 * np.outer(n, n * [-1, 1, 1, 1])).max() < 1e-15
    # curved space: n is null => R^mu_mu = 0 to round-off, for any intensity
    grid = dict(n=(3, 3, 1), x0=(np.log(3.0), 0.3, 0.0), dx=(0.2, 0.1, 0.1), bc_lo=PER, bc_hi=PER, x3_symmetric=True)
    ok = _cell(kind="ks_mks", params=dict(a=0.9, hslope=0.3), grid=grid)
    I = np.random.default_rng(9).uniform(size=(1, 3, 3, ok.nd))
    R = ok.moments(I)
    tr = R[0] + R[5] + R[10] + R[15]
    assert np.abs(tr).max() < 1e-13 * np.abs(R).max()


def test_step_on_homogeneous_static_problem_is_one_source_step():
    """O8: with no gradients the predictor only feeds (zero) fluxes, so rt_step(dt) = one O6 with dt;
    G_nu = -(R^0_nu after - before)/dt (Eq 36/48) and energy lost by radiation heats the gas."""
    grid = dict(n=(3, 2, 2), x0=(0, 0, 0), dx=(0.1,) * 3, bc_lo=PER, bc_hi=PER)
    o = Oracle(grid, "minkowski", {}, 2, dict(method=2, kappa_a0=3.0, kappa_s=1.0))
    rho, T0 = np.ones((2, 2, 3)), np.full((2, 2, 3), 1.4)
    o.set_fluid(rho, T0, None)
    I0 = np.tile(np.random.default_rng(10).uniform(0.1, 0.3, o.nd), (2, 2, 3, 1))
    I, T, R, G, nf = o.step(I0, T0, 0.05)
    I1, T1, nf1 = o.source_implicit(I0, T0, 0.05)
    assert np.abs(I - I1).max() < 1e-15 and np.abs(T - T1).max() < 1e-15
    Rb = o.moments(I0)
    assert np.abs(G.reshape(4, -1) + (R.reshape(16, -1)[:4] - Rb.reshape(16, -1)[:4]) / 0.05).max() < 1e-13
    # R^0_0 = -E: G_0 dt = E+ - E- = -Y (T+ - T-)
    assert np.abs(G[0] * 0.05 + 1.5 * (T.reshape(T0.shape) - T0)).max() < 1e-13
