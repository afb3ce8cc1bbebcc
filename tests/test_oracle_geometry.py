"""Pins for O2 (oracle/geometry.py) and the sign conventions of O4: exact facts only.  CPU only."""
import os

import numpy as np
import pytest

from oracle import Oracle, geodesic
from oracle import geometry as G


def _ks_points(a, n=200, lo=0.15, hi=0.85, seed=0):
    rng = np.random.default_rng(seed)
    rh = 1 + np.sqrt(1 - a * a)
    return np.stack([np.log(rng.uniform(0.9 * rh, 50, n)), rng.uniform(lo, hi, n), rng.uniform(0, 6.28, n)], -1)


@pytest.mark.parametrize("a", [0.0, 0.9, 0.9375])
def test_ks_tetrad_eq1_eq4_inverse(a):
    X = _ks_points(a, lo=0.02, hi=0.98)
    P = dict(a=a, hslope=0.3)
    g = G.metric("ks_mks", P, X)
    e, ei = G.tetrad("ks_mks", P, X)
    eta = np.einsum("...ma,...nb,...mn->...ab", e, e, g)
    assert np.abs(eta - G.ETA).max() < 5e-14                                           # Eq 1
    assert np.abs(np.einsum("...am,...mb->...ab", ei, e) - np.eye(4)).max() < 5e-14     # L67
    gi = np.linalg.inv(g)
    e0 = -gi[..., 0, :] / np.sqrt(-gi[..., 0, 0])[..., None]
    assert np.abs(e0 - e[..., :, 0]).max() < 5e-14                                      # Eq 4
    assert np.all(e[..., 0, 1:] == 0)           # spatial legs have no time component => n^0 = 1/lapse for all s
    # sqrt(-g) of Kerr-Schild is Sigma sin(theta), times the Jacobian of the logical map
    r, th, drdx, dthdx = G._ks_map(P, X)
    sg = (r * r + a * a * np.cos(th) ** 2) * np.sin(th) * drdx * dthdx
    assert np.allclose(G.sqrt_neg_g("ks_mks", P, X), sg, rtol=1e-11)


def test_ks_metric_is_vacuum_solution_inverse_component():
    # g^{tt} of Kerr-Schild is -(1 + 2r/Sigma) exactly (lapse^-2), g^{t phi} = 0: independent textbook facts
    a = 0.9
    X = _ks_points(a)
    P = dict(a=a, hslope=0.3)
    r, th, _, _ = G._ks_map(P, X)
    gi = np.linalg.inv(G.metric("ks_mks", P, X))
    H = 2 * r / (r * r + a * a * np.cos(th) ** 2)
    assert np.allclose(gi[..., 0, 0], -(1 + H), rtol=1e-11)
    assert np.abs(gi[..., 0, 3]).max() < 1e-11


def test_omega_antisymmetry_and_flat_values():
    a = 0.9
    X = _ks_points(a)
    om = G.ricci_rotation("ks_mks", dict(a=a, hslope=0.3), X)
    oml = np.einsum("ab,...bcd->...acd", G.ETA, om)
    assert np.abs(oml + np.swapaxes(oml, -3, -1)).max() < 1e-10       # omega_{acd} = -omega_{dca} (6th-order FD, h = 5e-4: S15)
    assert np.abs(G.ricci_rotation("minkowski", {}, X)).max() == 0.0
    # cylindrical tetrad in flat space: only omega^R_{phi phi} = -1/R and omega^phi_{phi R} = +1/R
    X = np.array([[1.3, 0.7, 0.4]])
    om = G.ricci_rotation("mink_cyl", {}, X)[0]
    R = np.hypot(1.3, 0.7)
    ref = np.zeros((4, 4, 4))
    ref[1, 2, 2], ref[2, 2, 1] = -1 / R, 1 / R
    assert np.abs(om - ref).max() < 1e-10


def test_angular_acceleration_is_rate_of_change_of_tetrad_components():
    """a^i(n) = -(omega^i_cd - n^i omega^0_cd) n^c n^d must equal d/dlambda of the tetrad components of a FIXED
    Cartesian direction along its own straight ray (flat space, rotating tetrad): fixes the sign of Eq 7/8."""
    x0 = np.array([1.3, 0.7, 0.4])
    rng = np.random.default_rng(1)
    for _ in range(5):
        d = rng.normal(size=3)
        d /= np.linalg.norm(d)                      # Cartesian direction of the ray

        def comps(lam):
            e, ei = G.tetrad("mink_cyl", {}, (x0 + lam * d)[None])
            return ei[0, 1:, 1:] @ d                 # nhat^i = e^i_mu d^mu

        h = 1e-4
        exact = (-comps(2 * h) + 8 * comps(h) - 8 * comps(-h) + comps(-2 * h)) / (12 * h)
        nh = comps(0.0)
        om = G.ricci_rotation("mink_cyl", {}, x0[None])[0]
        n4 = np.concatenate([[1.0], nh])
        acc = -np.einsum("icd,c,d->i", om[1:], n4, n4) + nh * np.einsum("cd,c,d->", om[0], n4, n4)
        assert np.abs(acc - exact).max() < 1e-9


@pytest.mark.parametrize("level,tol", [(2, 3.0e-2), (4, 1.5e-2), (8, 0.8e-2)])
def test_discrete_liouville(level, tol):
    """For I = 1 in flat space with a rotating tetrad the spatial divergence d_a n^a_s and the angular
    divergence D_Omega(s) of the oracle must cancel up to the (first-order) angular truncation error.
    This fixes the relative sign of the spatial and angular terms, of u_e and of a.  SURVEY probe values:
    1.7e-2 / 8.2e-3 / 4.0e-3 at 42 / 162 / 642 directions, with max|d_a n^a| = 0.68."""
    x0 = np.array([1.3, 0.7, 0.4])
    h = 1e-3
    grid = dict(n=(1, 1, 1), x0=tuple(x0 - h / 2), dx=(h, h, h), bc_lo=("outflow",) * 3, bc_hi=("outflow",) * 3)
    o = Oracle(grid, "mink_cyl", {}, level, dict(method=0, limiter=3))
    I = np.ones((1, 1, 1, o.nd))
    dt = 1e-3
    # transport of a uniform field: I_out - 1 = -dt * div_x / (n^0 n_0) with n^0 n_0 = -1
    divx = -(o.transport(I, I, dt) - I).reshape(-1) / dt * (-1.0)
    divo = -(o.angular_flux(I, I, dt) - I).reshape(-1) / dt * (-1.0)
    assert np.abs(divx).max() > 0.5                     # the terms are individually O(1) ...
    assert np.abs(divx + divo).max() < tol              # ... and cancel
    # and the angular update is conservative per cell: sum_s w_s delta(n^0 n_0 I)_s = 0
    assert abs((o.ang["w"] * divo).sum()) < 1e-11      # (1e-16 / dt round-off)


def test_photon_orbit_radii_eq53():
    # Eq 53 (L569) as an exact formula; paper prints r1 ~ 2.34, r2 ~ 3.53 for a = 0.5 (L648)
    a = 0.5
    r1 = 2 * (1 + np.cos(2 / 3 * np.arccos(-a)))
    r2 = 2 * (1 + np.cos(2 / 3 * np.arccos(+a)))
    assert abs(r1 - 2.34) < 0.01 and abs(r2 - 3.53) < 0.01
    # cross-check with the oracle's metric (equatorial plane, x2 = 0.5 <=> theta = pi/2):
    # Omega of a circular photon orbit solves g_tt + 2 g_tphi Om + g_phiphi Om^2 = 0 and its r-derivative = 0
    def disc(x1):
        gg = G.metric("ks_mks", dict(a=a, hslope=0.3), np.array([[x1, 0.5, 0.0]]))[0]
        return gg[0, 0], gg[0, 3], gg[3, 3]
    gtt, gtp, gpp = disc(np.log(r1))
    Om = (-gtp + np.sqrt(gtp ** 2 - gtt * gpp)) / gpp          # prograde null angular velocity
    h = 1e-5
    f = lambda x1: (lambda t: t[0] + 2 * t[1] * Om + t[2] * Om * Om)(disc(x1))
    assert abs((f(np.log(r1) + h) - f(np.log(r1) - h)) / (2 * h)) < 1e-6


def test_snake_metric_tetrad_and_zero_connection():
    """App A.1 (L802-806): snake coordinates w = x - A sin(k pi y).  The metric must be the pull-back of the flat metric
    through the coordinate map (Jacobian by finite differences of the MAP, independent of the oracle's A1 formula);
    the tetrad (A2 under reading S27) must satisfy Eq 1, be the Cartesian frame, and therefore have omega = 0."""
    P = dict(A=0.1, k=2.0)
    rng = np.random.default_rng(5)
    X = rng.uniform(0.0, 1.0, (40, 3))

    def cart(Xw):   # (w, y, z) -> (x, y, z)
        return np.stack([Xw[..., 0] + P["A"] * np.sin(P["k"] * np.pi * Xw[..., 1]), Xw[..., 1], Xw[..., 2]], -1)

    h = 1e-5
    J = np.zeros((40, 3, 3))   # J[p, a, i] = d x^a / d X^i
    for i in range(3):
        d = np.zeros(3); d[i] = h
        J[:, :, i] = (cart(X + d) - cart(X - d)) / (2 * h)
    g = G.metric("snake", P, X)
    assert np.abs(g[:, 1:, 1:] - np.einsum("pai,paj->pij", J, J)).max() < 1e-9
    assert np.abs(g[:, 0, 0] + 1).max() == 0 and np.abs(g[:, 0, 1:]).max() == 0
    assert np.abs(G.sqrt_neg_g("snake", P, X) - 1.0).max() < 1e-14           # det J = 1
    e, einv = G.tetrad("snake", P, X)
    assert np.abs(np.einsum("pma,pmn,pnb->pab", e, g, e) - G.ETA).max() < 1e-14      # Eq 1
    assert np.abs(np.einsum("pam,pmb->pab", einv, e) - np.eye(4)).max() < 1e-14
    # Cartesian frame: pushing e_a forward with J gives the unit vectors
    assert np.abs(np.einsum("pai,pib->pab", J, e[:, 1:, 1:]) - np.eye(3)).max() < 1e-9
    # a parallel frame in flat space: all Ricci rotation coefficients vanish (to the FD truncation error)
    assert np.abs(G.ricci_rotation("snake", P, X)).max() < 1e-8
    # n^w = n^x - delta n^y: a ray along y-hat moves backwards in w where delta > 0
    delta = P["A"] * P["k"] * np.pi * np.cos(P["k"] * np.pi * X[:, 1])
    assert np.abs(e[:, 1, 2] + delta).max() < 1e-14


def _radial_acceleration_of_phi_hat(a, r, sign):
    """a^r-hat of the direction n-hat = +-phi-hat from the oracle's Ricci rotation coefficients in Boyer-Lindquist
    coordinates on the equator: a^i = -(omega^i_cd - n^i omega^0_cd) n^c n^d  (Eq 7-8 in the 3-vector form, S4)."""
    P = dict(a=a, hslope=0.3)
    om = G.ricci_rotation("bl_mks", P, np.array([[np.log(r), 0.5, 0.0]]))[0]
    n = np.array([1.0, 0.0, 0.0, sign])
    acc = -(np.einsum("icd,c,d->i", om, n, n) - n * np.einsum("cd,c,d->", om[0], n, n))
    assert abs(acc[2]) < 1e-12 and abs(acc[3]) < 1e-12        # stays in the equatorial plane, stays unit
    return acc[1]


@pytest.mark.parametrize("a", [0.5, -0.5, 0.7, -0.7, 0.95, -0.95])
def test_bl_tetrad_and_circular_photon_orbits_eq53(a):
    """Section 4.7 (L563-592).  In the frame of the zero-angular-momentum observers (e_0 normal to t = const, Eq 4) a photon
    on a circular orbit moves along +-phi-hat for ever, i.e. the angular acceleration that drives the angular fluxes
    (Eq 7-8 -> Eq 19) vanishes for n-hat = +-phi-hat exactly at the radii of Eq 53 (L569), r = 2 [1 + cos(2/3 arccos(-+a))]
    -- the paper's spins are +-0.5, +-0.7, +-0.95 (L586) -- and changes sign there: inside the direction turns inwards,
    outside outwards ("we expect to switch from escaping to infalling radiation as we cross the circular orbit radius").
    This pins the oracle's omega in a curved space-time against a number the paper prints (r1 ~ 2.34, r2 ~ 3.53, L648)."""
    P = dict(a=a, hslope=0.3)
    rh = 1 + np.sqrt(1 - a * a)
    X = np.stack([np.log(np.linspace(rh + 0.2, 8.0, 7)), np.linspace(0.2, 0.8, 7), np.zeros(7)], -1)
    g = G.metric("bl_mks", P, X)
    e, einv = G.tetrad("bl_mks", P, X)
    assert np.abs(np.einsum("...ma,...mn,...nb->...ab", e, g, e) - G.ETA).max() < 1e-13        # Eq 1
    gi = np.linalg.inv(g)
    assert np.abs(e[..., :, 0] + gi[..., 0, :] / np.sqrt(-gi[..., 0, 0])[..., None]).max() < 1e-13   # Eq 4
    assert np.abs(np.einsum("...am,...mb->...ab", einv, e) - np.eye(4)).max() < 1e-13
    for sign, r_eq53 in ((+1.0, 2 * (1 + np.cos(2 / 3 * np.arccos(-a)))), (-1.0, 2 * (1 + np.cos(2 / 3 * np.arccos(+a))))):
        lo, hi = max(rh + 0.05, r_eq53 - 0.5), r_eq53 + 0.5
        flo, fhi = _radial_acceleration_of_phi_hat(a, lo, sign), _radial_acceleration_of_phi_hat(a, hi, sign)
        assert flo < 0 < fhi                                                        # infalling inside, escaping outside
        for _ in range(60):
            mid = 0.5 * (lo + hi)
            if _radial_acceleration_of_phi_hat(a, mid, sign) < 0:
                lo = mid
            else:
                hi = mid
        assert abs(0.5 * (lo + hi) - r_eq53) < 1e-8
    if a == 0.5:                                                                    # the values the paper prints (L648)
        gold = dict((l.split()[0], float(l.split()[1])) for l in open(os.path.join(os.path.dirname(__file__), "golden", "paper_values.txt"))
                    if l.strip() and not l.startswith("#"))
        assert abs(2 * (1 + np.cos(2 / 3 * np.arccos(-a))) - gold["photon_r1_a0.5"]) < 0.01
        assert abs(2 * (1 + np.cos(2 / 3 * np.arccos(+a))) - gold["photon_r2_a0.5"]) < 0.01


def test_generic_tetrad_of_a_user_metric_reproduces_the_papers_closed_forms():
    """The tetrad the 'user' metric kind builds when the caller gives none (e_0 from Eq 4, Gram-Schmidt of d_3, d_2, d_1) is, for
    the Kerr-Schild metric, the closed form A3-A4 of the paper (L814-850) and, for Boyer-Lindquist, the zero-angular-momentum
    frame; for any metric it is orthonormal, g_{mu nu} e^mu_a e^nu_b = eta_ab, with e_0 normal to t = const."""
    rng = np.random.default_rng(11)
    X = np.stack([rng.uniform(0.9, 3.0, 40), rng.uniform(0.05, 0.95, 40), rng.uniform(0, 6, 40)], -1)
    for kind in ("ks_mks", "bl_mks"):
        params = dict(a=0.7, hslope=0.3)
        g = G.metric(kind, params, X)
        e_ref, einv_ref = G.tetrad(kind, params, X)
        e, einv = G._tetrad_from_metric(g)
        assert np.abs(e - e_ref).max() < 1e-12 and np.abs(einv - einv_ref).max() < 1e-11
    # an arbitrary stationary metric with lapse, shift and a non-diagonal 3-metric
    A = rng.normal(size=(6, 3, 3)) * 0.2 + np.eye(3)
    gam = np.einsum("nij,nkj->nik", A, A)
    beta = rng.normal(size=(6, 3)) * 0.2
    lapse = rng.uniform(0.5, 1.5, 6)
    g = np.zeros((6, 4, 4))
    g[:, 1:, 1:] = gam
    g[:, 0, 1:] = g[:, 1:, 0] = np.einsum("nij,nj->ni", gam, beta)
    g[:, 0, 0] = -lapse ** 2 + np.einsum("ni,nij,nj->n", beta, gam, beta)
    e, einv = G._tetrad_from_metric(g)
    eta = np.diag([-1.0, 1, 1, 1])
    assert np.abs(np.einsum("nma,nmk,nkb->nab", e, g, e) - eta).max() < 1e-13
    assert np.abs(np.einsum("nam,nmb->nab", einv, e) - np.eye(4)).max() < 1e-13
    # Eq 4: e_0 = (1, -beta^i) / lapse; the space-like legs have no time component, d_3 keeps its direction
    assert np.abs(e[:, 0, 0] - 1 / lapse).max() < 1e-13 and np.abs(e[:, 1:, 0] + beta / lapse[:, None]).max() < 1e-13
    assert np.abs(e[:, 0, 1:]).max() == 0.0 and np.abs(e[:, 1:3, 3]).max() == 0.0
    # through the 'user' kind: the same numbers
    prm = dict(g=lambda x: g[int(round(x[0]))], e=None)
    Xi = np.stack([np.arange(6.0), np.zeros(6), np.zeros(6)], -1)
    e2, einv2 = G.tetrad("user", prm, Xi)
    assert np.array_equal(e2, e) and np.array_equal(einv2, einv)
