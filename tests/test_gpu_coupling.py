"""Moving-fluid terms and the coupling to a fluid solver, end to end on the GPU (Eq 48).

(1) boosted equilibrium: radiation that is isotropic and thermal in the frame of a MOVING fluid is a fixed point of rt_step up
    to the quadrature mismatch of reading S18 (literal 4 pi against sum dOmega-bar), and its moments are those of a perfect
    radiation fluid R^mu_nu = (4/3) E u^mu u_nu + (E/3) delta^mu_nu;
(2) the caller-side loop of the paper's scheme (L448-456): the 4-force G_nu that rt_step hands back drives a toy gas-energy
    update on the caller's side, the new gas temperature goes back in through rt_set_fluid, several steps in a row; gas +
    radiation energy is conserved to round-off and the loop agrees with the same loop run on the oracle.
"""
import numpy as np
import pytest

import rt_workloads as W
from oracle import Oracle
from parity_util import TOL, rel_err

pytestmark = pytest.mark.gpu
PER = ("periodic",) * 3
FOURPI = 4 * np.pi


def _pair(grid, opt, level=4):
    from paper_2508_15532_b200 import rt
    return Oracle(grid, "minkowski", {}, level, opt), rt.RtContext(grid, "minkowski", {}, level, opt)


@pytest.mark.parametrize("v", [(0.0, 0.0, 0.0), (0.3, -0.2, 0.1)])
def test_boosted_equilibrium_is_a_fixed_point_up_to_the_quadrature(v):
    import torch
    n = (6, 5, 4)
    grid = dict(n=n, x0=(0, 0, 0), dx=(0.1,) * 3, bc_lo=PER, bc_hi=PER)
    opt = dict(method=2, kappa_a0=2.0, kappa_s=0.5)
    orc, ctx = _pair(grid, opt)
    v = np.asarray(v)
    gam = 1 / np.sqrt(1 - v @ v)
    u = np.concatenate([[gam], gam * v])
    shp = n[::-1]
    u4 = np.broadcast_to(u[:, None, None, None], (4,) + shp).copy()
    T0, rho = 1.3, 1.0
    nh, w = orc.ang["nhat"], orc.ang["w"]
    nbar = u[0] - nh @ u[1:]                                   # Eq 5: nu-bar / nu-hat
    I0 = np.broadcast_to((T0 ** 4 / FOURPI) / nbar ** 4, shp + (orc.nd,)).copy()     # I / nu^4 invariant (S17)
    delta = (w / nbar ** 2).sum() / FOURPI - 1.0               # S18: sum dOmega-bar against the literal 4 pi
    assert abs(delta) < (1e-14 if not v.any() else 2e-2)
    rhoa, Ta = np.full(shp, rho), np.full(shp, T0)
    orc.set_fluid(rhoa, Ta, u4)
    dev = ctx.device
    ctx.set_fluid(torch.as_tensor(rhoa, device=dev), torch.as_tensor(Ta, device=dev), torch.as_tensor(u4, device=dev))
    dt = 0.04
    Io, To, Ro, Go, nf = orc.step(I0, Ta, dt)
    I = ctx.to_device(I0); T = torch.as_tensor(Ta, device=dev).clone()
    R = torch.zeros((16,) + shp, dtype=torch.float64, device=dev); G = torch.zeros((4,) + shp, dtype=torch.float64, device=dev)
    ctx.step(I, T, dt, R, G)
    torch.cuda.synchronize()
    assert nf == 0 and ctx.n_fail() == 0
    Ig, Tg, Rg, Gg = ctx.to_host(I), T.cpu().numpy(), R.cpu().numpy(), G.cpu().numpy()
    # GPU == oracle
    assert rel_err(Ig, Io.reshape(Ig.shape)) <= TOL and rel_err(Tg, To.reshape(shp)) <= TOL and rel_err(Rg, Ro) <= TOL
    assert np.abs(Gg - Go).max() * dt <= TOL * np.abs(Ro).max()
    # fixed point: exact for a static fluid, within the quadrature mismatch for a moving one
    tol = 1e-13 if not v.any() else 3.0 * abs(delta)
    assert np.abs(Tg - T0).max() <= tol * T0 and np.abs(Ig - I0).max() <= tol * np.abs(I0).max()
    assert np.abs(Gg).max() * dt <= max(tol, 1e-13) * T0 ** 4
    # moments of a perfect radiation fluid (flat space: u_nu = eta u^nu)
    E = T0 ** 4
    ul = u * np.array([-1.0, 1, 1, 1])
    Rex = (4.0 / 3.0) * E * np.outer(u, ul) + (E / 3.0) * np.eye(4)
    # (static: exact by the grid's symmetry; moving: the 162-direction quadrature of the boosted field, which varies as
    # nbar^-4 over the sphere, is good to ~1e-4 of E)
    assert np.abs(Rg.reshape(4, 4, -1) - Rex[..., None]).max() <= (1e-12 if not v.any() else 2e-4) * E
    ctx.close()


def test_caller_side_energy_update_from_G_closes_the_loop():
    """The GRMHD side of L448-456 as a toy: gas energy density e = Y T per cell, updated by the caller from the returned
    4-force, de = -G_0 dt (Eq 48 with R^0_0 = -E: G_0 = dE/dt), new T handed back through rt_set_fluid and as T_inout."""
    import torch
    cfg = W.config(2, n=(8, 6, 5))
    kind, params = cfg["metric"]
    from paper_2508_15532_b200 import rt
    orc = Oracle(cfg["grid"], kind, params, cfg["level"], cfg["options"])
    ctx = rt.RtContext(cfg["grid"], kind, params, cfg["level"], cfg["options"])
    f = W.fields(cfg, orc.ang["nhat"], orc.tab["e_c"])
    dev = ctx.device
    rho_d = torch.as_tensor(f["rho"], device=dev).contiguous()
    Y = cfg["options"].get("Y_over_rho", 1.5) * f["rho"]
    Y_d = torch.as_tensor(Y, device=dev)
    dt = cfg["dt"]
    I_o, T_o = f["I0"].copy(), f["T"].copy()
    I_g = ctx.to_device(f["I0"]); T_g = torch.as_tensor(f["T"], device=dev).contiguous().clone()
    R_g = torch.zeros((16,) + ctx.shape, dtype=torch.float64, device=dev); G_g = torch.zeros((4,) + ctx.shape, dtype=torch.float64, device=dev)
    w = torch.as_tensor(orc.ang["w"], device=dev)
    tot0 = float((Y_d * T_g).sum() + (I_g[..., :ctx.nd] * w).sum())
    for step in range(6):
        # oracle side of the same loop
        orc.set_fluid(f["rho"], T_o, None)
        I_o, T_lib_o, R_o, G_o, nf = orc.step(I_o, T_o, dt)
        T_o = T_o + (-G_o[0] * dt / Y).reshape(T_o.shape)
        # GPU side
        ctx.set_fluid(rho_d, T_g, None)
        T_lib = T_g.clone()
        ctx.step(I_g, T_lib, dt, R_g, G_g)
        T_g = T_g - G_g[0] * dt / Y_d                          # the caller's update, on the device
        torch.cuda.synchronize()
        assert nf == 0 and ctx.n_fail() == 0
        # the 4-force carries exactly the energy the library's own T took (Eq 39): the two temperatures agree
        assert float((T_g - T_lib).abs().max()) <= 1e-12 * float(T_g.abs().max())
        # gas + radiation energy (R^0_0 = -E, flat space, periodic): conserved to round-off
        tot = float((Y_d * T_g).sum() - R_g[0].sum())
        assert abs(tot - tot0) <= 1e-12 * abs(tot0)
        assert rel_err(T_g.cpu().numpy(), T_o.reshape(ctx.shape)) <= TOL
        assert rel_err(ctx.to_host(I_g), I_o.reshape(ctx.shape + (ctx.nd,))) <= TOL
    assert float((T_g - torch.as_tensor(f["T"], device=dev)).abs().max()) > 1e-3      # the gas did cool
    ctx.close()
