"""Pins for the oriented / Lorentz-deformed geodesic grid ("the grid can be deformed in advance by performing a
Lorentz transformation of its directions.  It can also be easily oriented along a pre-defined direction").  CPU only.

What fixes the construction other than itself: the Doppler identity of an aberration and its inverse, the Voronoi / Delaunay
definitions checked by brute force over all cell centres, the closed-form Jacobian of the aberration map for the cell areas
(second-order convergence in the cell size), and rotation invariance.
"""
import numpy as np
import pytest

from oracle import geodesic

BETA = np.array([0.3, -0.2, 0.45])


def _gamma(b):
    return 1.0 / np.sqrt(1.0 - b @ b)


def test_aberration_obeys_the_doppler_identity_and_inverts():
    g0 = geodesic.build(4)
    g = geodesic.build(4, boost=BETA)
    n, n1 = g0["nhat"], g["nhat"]
    gam = _gamma(BETA)
    assert np.abs(np.linalg.norm(n1, axis=1) - 1.0).max() < 1e-15
    # photon energy ratio there and back: gamma (1 + beta.n) * gamma (1 - beta.n') = 1
    assert np.abs(gam * (1 + n @ BETA) * gam * (1 - n1 @ BETA) - 1.0).max() < 1e-14
    # the component perpendicular to beta shrinks by the Doppler factor: n'_perp = n_perp / (gamma (1 + beta.n))
    bh = BETA / np.linalg.norm(BETA)
    perp = lambda v: v - np.outer(v @ bh, bh)
    assert np.abs(perp(n1) - perp(n) / (gam * (1 + n @ BETA))[:, None]).max() < 1e-14
    # the inverse boost restores the regular centres
    back = geodesic._aberrate(n1, -BETA)
    assert np.abs(back - n).max() < 1e-14
    # directions crowd around +beta: more than half of them in the forward hemisphere
    assert (n1 @ bh > 0).sum() > 0.7 * len(n1) and abs((n @ bh > 0).sum() - 0.5 * len(n)) <= 0.06 * len(n)


@pytest.mark.parametrize("kw", [dict(boost=BETA), dict(axis=(1.0, 2.0, -0.5)), dict(boost=(0.0, 0.0, 0.6), axis=(0.0, 1.0, 0.0))])
def test_deformed_cells_are_the_voronoi_cells_of_the_deformed_centres(kw):
    """Numbering and neighbour lists are those of the regular grid; every edge centre is equidistant from the two cells it
    separates and no third centre is closer (the definition of a Voronoi edge, L213), every corner of a cell is equidistant
    from three centres with no centre inside that circle (Delaunay), areas add up to the sphere."""
    g0 = geodesic.build(4)
    g = geodesic.build(4, **kw)
    n = g["nhat"]
    assert (g["nb"] == g0["nb"]).all() and (g["nnb"] == g0["nnb"]).all()
    assert abs(g["w"].sum() - 4 * np.pi) < 1e-13 and g["w"].min() > 0
    for s in range(g["nd"]):
        k = g["nnb"][s]
        for e in range(k):
            t = g["nb"][s, e]
            m = g["emid"][s, e]
            d = n @ m
            assert abs(d[s] - d[t]) < 1e-13
            assert np.sort(d)[-3] < d[s] - 1e-9                  # s and t are the two nearest centres, strictly
            # outward normal: tangent at the edge centre, pointing from s to t
            u = g["eun"][s, e]
            assert abs(u @ m) < 1e-13 and abs(u @ u - 1) < 1e-13 and u @ (n[t] - n[s]) > 0
            # the corner between this edge and the next: equidistant from s, t, t2, nobody nearer
            t2 = g["nb"][s, (e + 1) % k]
            c = np.cross(n[t] - n[s], n[t2] - n[s])
            c /= np.linalg.norm(c)
            if c @ n[s] < 0:
                c = -c
            dc = n @ c
            assert max(abs(dc[s] - dc[t]), abs(dc[s] - dc[t2])) < 1e-13
            assert (dc > dc[s] + 1e-12).sum() == 0
    # the same edge seen from both sides
    for s in range(g["nd"]):
        for e in range(g["nnb"][s]):
            t = g["nb"][s, e]
            q = list(g["nb"][t, :g["nnb"][t]]).index(s)
            assert abs(g["dlam"][s, e] - g["dlam"][t, q]) < 1e-14
            assert np.abs(g["emid"][s, e] - g["emid"][t, q]).max() < 1e-14
            assert np.abs(g["eun"][s, e] + g["eun"][t, q]).max() < 1e-13


def test_cell_areas_follow_the_jacobian_of_the_aberration_to_second_order():
    """d Omega' = d Omega / (gamma (1 + beta.n))^2 (the solid-angle transformation of special relativity); a Voronoi cell of
    finite size obeys it up to terms of second order in its diameter: the worst deviation drops about 4x per generation."""
    gam = _gamma(BETA)
    errs = []
    for level in (2, 4, 8):
        g0, g = geodesic.build(level), geodesic.build(level, boost=BETA)
        ratio = g["w"] / g0["w"] * (gam * (1 + g0["nhat"] @ BETA)) ** 2
        errs.append(np.abs(ratio - 1.0).max())
    assert errs[0] < 0.25 and errs[1] < 0.35 * errs[0] and errs[2] < 0.35 * errs[1]


def test_orientation_is_a_rigid_rotation():
    g0 = geodesic.build(4)
    axis = np.array([1.0, 2.0, -0.5])
    g = geodesic.build(4, axis=axis)
    assert np.abs(g["nhat"][0] - axis / np.linalg.norm(axis)).max() < 1e-15           # the pole cell
    assert np.abs(g["nhat"] @ g["nhat"].T - g0["nhat"] @ g0["nhat"].T).max() < 1e-14     # all mutual angles kept
    assert np.abs(g["w"] - g0["w"]).max() < 1e-14 and np.abs(g["dlam"] - g0["dlam"]).max() < 1e-14
    # handedness kept (a reflection would keep the angles too)
    tri = lambda gg: np.linalg.det(gg["nhat"][[0, 1, 2]])
    assert tri(g) * tri(g0) > 0
    # the opposite pole
    gm = geodesic.build(4, axis=(0, 0, -2.0))
    assert np.abs(gm["nhat"][0] - [0, 0, -1]).max() < 1e-15 and np.abs(gm["w"] - g0["w"]).max() < 1e-14


def test_quadrature_of_the_deformed_grid_converges_to_the_boosted_isotropic_energy():
    """A field that is isotropic in the frame of the regular grid, I' = 1, is I = D^4 in the frame it moves in (I / nu^4
    invariant), D = 1 / (gamma (1 - beta.n)).  Its energy density there is the closed form 4 pi gamma^2 (1 + beta^2 / 3); the
    deformed grid's cell areas times the centre values converge to it at second order (error / 4 per generation)."""
    b = np.array([0.0, 0.0, 0.8])
    gam = _gamma(b)
    exact = 4 * np.pi * gam ** 2 * (1 + b @ b / 3)
    err = []
    for level in (2, 4, 8):
        g = geodesic.build(level, boost=b)
        D = 1.0 / (gam * (1 - g["nhat"] @ b))
        err.append(abs((g["w"] * D ** 4).sum() / exact - 1.0))
    assert err[0] < 0.15 and err[1] < 0.3 * err[0] and err[2] < 0.3 * err[1]
