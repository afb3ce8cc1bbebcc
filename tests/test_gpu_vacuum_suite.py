"""The paper's spherical flash (section 4.1) and steady point source (section 4.2) on the GPU: parity with the
oracle on a small mesh (the steady source re-imposed by the caller between steps on both sides), then the paper's own set-up
-- [-2, 2]^3, 64^3 cells, G3 = 642 directions -- checked against what the paper states: the front is at d = t (c = 1), the
steady source decays as 1/d^2."""
import numpy as np
import pytest

from oracle import Oracle
from parity_util import TOL, rel_err

pytestmark = pytest.mark.gpu
OUT = ("outflow",) * 3


def _grid(N, half):
    return dict(n=(N, N, N), x0=(-half,) * 3, dx=(2.0 * half / N,) * 3, bc_lo=OUT, bc_hi=OUT)


def _ctx(grid, level):
    import torch
    from paper_2508_15532_b200 import rt
    ctx = rt.RtContext(grid, "minkowski", {}, level, dict(method=0))
    one = torch.ones(ctx.shape, dtype=torch.float64, device=ctx.device)
    ctx.set_fluid(torch.zeros_like(one), one, None)
    return ctx


def test_flash_and_steady_source_match_the_oracle():
    import torch
    N, level = 13, 2
    grid = _grid(N, 1.0)
    orc = Oracle(grid, "minkowski", {}, level, dict(method=0))
    ctx = _ctx(grid, level)
    c = N // 2
    src = (slice(c - 1, c + 2),) * 3
    I_o = np.zeros((N, N, N, orc.nd)); I_o[src] = 1.0
    T_o = np.ones((N, N, N))
    I_g = ctx.to_device(I_o); T_g = torch.ones(ctx.shape, dtype=torch.float64, device=ctx.device)
    dt = 0.4 * grid["dx"][0]
    for k in range(10):
        I_o, T_o, R_o, G_o, nf = orc.step(I_o, T_o, dt)
        ctx.step(I_g, T_g, dt, None, None)
        if k >= 4:                                            # first a flash, then a steady source: the caller re-imposes it
            I_o = I_o.reshape(N, N, N, orc.nd); I_o[src] = 1.0
            I_g[c - 1:c + 2, c - 1:c + 2, c - 1:c + 2, :ctx.nd] = 1.0
    torch.cuda.synchronize()
    assert rel_err(ctx.to_host(I_g), np.asarray(I_o).reshape(N, N, N, orc.nd)) <= TOL
    ctx.close()


def _coords(ctx, grid):
    import torch
    N = grid["n"][0]
    x = grid["x0"][0] + (torch.arange(N, dtype=torch.float64, device=ctx.device) + 0.5) * grid["dx"][0]
    Z, Y, X = torch.meshgrid(x, x, x, indexing="ij")
    return torch.stack([X, Y, Z], -1)


def test_flash_front_at_d_equals_t_paper_setup():
    import torch
    N, level = 64, 8                                          # G3: 642 directions (L213)
    grid = _grid(N, 2.0)
    ctx = _ctx(grid, level)
    assert ctx.nd == 642
    dx = grid["dx"][0]
    c = N // 2
    I = torch.zeros(ctx.shape + (ctx.pitch,), dtype=torch.float64, device=ctx.device)
    I[c - 1:c + 2, c - 1:c + 2, c - 1:c + 2, :ctx.nd] = 1.0  # (even N: the 3^3 source sits half a cell off the origin)
    T = torch.ones(ctx.shape, dtype=torch.float64, device=ctx.device)
    w = torch.as_tensor(ctx.directions()["w"], device=ctx.device)
    X = _coords(ctx, grid)
    x0 = (I[..., :ctx.nd] * w).sum(-1)
    E0 = float(x0.sum())
    cen0 = (x0[..., None] * X).sum((0, 1, 2)) / E0
    dt, nst = 0.4 * dx, 40                                    # t = 1.0
    for _ in range(nst):
        ctx.step(I, T, dt, None, None)
    torch.cuda.synchronize()
    t = dt * nst
    E = (I[..., :ctx.nd] * w).sum(-1)
    assert abs(float(E.sum()) - E0) <= 1e-12 * E0             # nothing has reached the boundary: conserved to round-off
    d = (X - cen0).norm(dim=-1)
    assert abs(float((E * d).sum() / E.sum()) - t) < 0.6 * dx         # the front is at d = t  (Fig 2)
    assert float(E[d > t + 1.5 * dx * 3 ** 0.5 + 2.5 * dx].sum()) < 2e-3 * E0   # nothing ahead of it beyond flash size + diffusion
    assert float(E[d < t - 1.5 * dx * 3 ** 0.5 - 4.0 * dx].sum()) < 2e-2 * E0   # and it is a shell: the inside has emptied
    nh = torch.as_tensor(ctx.directions()["nhat"], device=ctx.device)
    for s in (0, 100, 321, 500, 641):                         # each direction's packet sits at t n-hat_s
        m = I[..., s]
        cen = (m[..., None] * X).sum((0, 1, 2)) / m.sum() - cen0
        assert float((cen - t * nh[s]).abs().max()) < dx / 3
    ctx.close()


def test_steady_source_inverse_square_paper_setup():
    import torch
    N, level = 64, 8
    grid = _grid(N, 2.0)
    ctx = _ctx(grid, level)
    dx = grid["dx"][0]
    c = N // 2
    I = torch.zeros(ctx.shape + (ctx.pitch,), dtype=torch.float64, device=ctx.device)
    T = torch.ones(ctx.shape, dtype=torch.float64, device=ctx.device)
    w = torch.as_tensor(ctx.directions()["w"], device=ctx.device)
    dt = 0.4 * dx
    for _ in range(150):                                      # t = 3.75 > 2 sqrt 3: the front has left through the corners
        I[c - 1:c + 2, c - 1:c + 2, c - 1:c + 2, :ctx.nd] = 1.0       # the caller's steady source
        ctx.step(I, T, dt, None, None)
    torch.cuda.synchronize()
    E = (I[..., :ctx.nd] * w).sum(-1)
    X = _coords(ctx, grid)
    d = (X - X[c - 1:c + 2, c - 1:c + 2, c - 1:c + 2].mean((0, 1, 2))).norm(dim=-1)
    # what leaves the source crosses every sphere: the energy inside radius r grows linearly with r
    rs = torch.arange(4.0, 28.1, 1.0, dtype=torch.float64, device=ctx.device) * dx
    C = torch.stack([E[d < r].sum() for r in rs])
    A = torch.stack([rs, torch.ones_like(rs)], 1)
    coef = torch.linalg.lstsq(A, C[:, None]).solution[:, 0]
    res = C - A @ coef
    assert float(res.abs().max()) < 0.02 * float(C[-1] - C[0])
    # ... i.e. the shell-averaged energy density falls as 1/d^2 (Fig 3, right)
    edges = torch.arange(4.0, 28.1, 3.0, dtype=torch.float64, device=ctx.device) * dx
    mean_E = torch.stack([E[(d >= a) & (d < b)].mean() for a, b in zip(edges[:-1], edges[1:])])
    mid = 0.5 * (edges[:-1] + edges[1:])
    B = torch.stack([mid.log(), torch.ones_like(mid)], 1)
    slope = float(torch.linalg.lstsq(B, mean_E.log()[:, None]).solution[0, 0])
    assert abs(slope + 2.0) < 0.08, slope
    ctx.close()
