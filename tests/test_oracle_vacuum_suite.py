"""Oracle pins from the paper's vacuum test suite that need no new geometry: the spherical flash of section 4.1
(the front is at d = t, c = 1) and the steady point source of section 4.2 (L486-488: 1/d^2 decay).  CPU
only, small meshes; tests/test_gpu_vacuum_suite.py repeats both on the GPU at the paper's 64^3 x 642 directions.

The steady source is imposed by the CALLER: after every rt_step it writes the source intensity back into the central cells
(the library owns no source term other than the fluid's; the caller owns I).
"""
import numpy as np

from oracle import Oracle

OUT = ("outflow",) * 3


def _box(N, level):
    grid = dict(n=(N, N, N), x0=(-1.0, -1.0, -1.0), dx=(2.0 / N,) * 3, bc_lo=OUT, bc_hi=OUT)
    o = Oracle(grid, "minkowski", {}, level, dict(method=0))
    x = -1.0 + (np.arange(N) + 0.5) * 2.0 / N
    Z, Y, X = np.meshgrid(x, x, x, indexing="ij")
    return o, np.stack([X, Y, Z], -1), 2.0 / N


def test_flash_front_moves_at_c_direction_by_direction():
    """A 3^3-cell isotropic flash: the packet of direction s has its centroid at t n-hat_s (within a third of a cell), so the
    energy-weighted mean distance is t and nothing runs ahead of the front by more than the flash size plus numerical
    diffusion (L478: "the radiation front is expected to have moved by a distance d = 1 ... c = 1"); energy is conserved
    until the front reaches the boundary."""
    N = 21
    o, X, dx = _box(N, 2)
    c = N // 2
    I = np.zeros((N, N, N, o.nd))
    I[c - 1:c + 2, c - 1:c + 2, c - 1:c + 2, :] = 1.0
    T = np.ones((N, N, N))
    w = o.ang["w"]
    E0 = (I * w).sum()
    dt, nst = 0.4 * dx, 12
    for _ in range(nst):
        I, T, R, G, nf = o.step(I, T, dt)
    I = I.reshape(N, N, N, o.nd)
    t = dt * nst
    assert abs((I * w).sum() - E0) < 1e-12 * E0
    for s in (0, 7, 20, 33, 41):
        m = I[..., s]
        cen = (m[..., None] * X).sum((0, 1, 2)) / m.sum()
        assert np.abs(cen - t * o.ang["nhat"][s]).max() < dx / 3
    E = (I * w).sum(-1)
    d = np.linalg.norm(X, axis=-1)
    assert abs((E * d).sum() / E.sum() - t) < 0.6 * dx
    assert E[d > t + 1.5 * dx * np.sqrt(3) + 2.5 * dx].sum() < 2e-3 * E.sum()


def test_steady_point_source_decays_as_inverse_square():
    """Steady central source: once the front has passed, what leaves the source per unit time crosses every sphere, so the
    energy inside radius r grows linearly with r: E ~ 1/d^2 on the angular average (L488)."""
    N = 21
    o, X, dx = _box(N, 2)
    c = N // 2
    src = (slice(c - 1, c + 2),) * 3
    I = np.zeros((N, N, N, o.nd))
    I[src] = 1.0
    T = np.ones((N, N, N))
    w = o.ang["w"]
    dt = 0.4 * dx
    for _ in range(30):                                   # t = 1.14: the front has left the box along the axes
        I, T, R, G, nf = o.step(I, T, dt)
        I = I.reshape(N, N, N, o.nd)
        I[src] = 1.0                                      # the caller re-imposes the source
    E = (I * w).sum(-1)
    d = np.linalg.norm(X, axis=-1)
    # energy inside radius r grows linearly in r (an exact 1/d^2 field sampled on this mesh is linear to 2 %; 1/d or 1/d^3
    # deviate by 10 % and 13 %)
    rs = np.arange(3.0, 9.6, 0.5) * dx
    C = np.array([E[d < r].sum() for r in rs])
    res = C - np.polyval(np.polyfit(rs, C, 1), rs)
    assert np.abs(res).max() < 0.05 * (C[-1] - C[0])
    # the same statement as a power law of the shell-averaged energy density (two-cell shells)
    edges = np.array([3.0, 5.0, 7.0, 9.0]) * dx
    mean_E = np.array([E[(d >= a) & (d < b)].mean() for a, b in zip(edges[:-1], edges[1:])])
    slope = np.polyfit(np.log(0.5 * (edges[:-1] + edges[1:])), np.log(mean_E), 1)[0]
    assert abs(slope + 2.0) < 0.3
