"""Shared harness of the GPU parity tests: the SAME seeded arrays go to the oracle and to the CUDA library."""
import numpy as np

import rt_workloads as W
from oracle import Oracle

TOL = 1e-10   # BASELINE.json north_star: max|gpu - oracle| / max|oracle| per field, fp64


def rel_err(a, b):
    a, b = np.asarray(a, float), np.asarray(b, float)
    den = np.abs(b).max()
    return float(np.abs(a - b).max() / den) if den > 0 else float(np.abs(a).max())


def make_pair(cfg, gpu_options=None):
    """Build (oracle, RtContext, fields, dt) for a workload config; inputs are generated once from the oracle's
    tables and handed to both sides."""
    import torch
    from paper_2508_15532_b200 import rt

    kind, params = cfg["metric"]
    orc = Oracle(cfg["grid"], kind, params, cfg["level"], cfg["options"])
    ctx = rt.RtContext(cfg["grid"], kind, params, cfg["level"], dict(cfg["options"], **(gpu_options or {})))   # gpu_options: kernel-variant switches the oracle does not have
    f = W.fields(cfg, orc.ang["nhat"], orc.tab["e_c"])
    orc.set_fluid(f["rho"], f["T"], f["u4"])
    dev = ctx.device
    rho = torch.as_tensor(f["rho"], device=dev).contiguous()
    T = torch.as_tensor(f["T"], device=dev).contiguous()
    u4 = None if f["u4"] is None else torch.as_tensor(f["u4"], device=dev).contiguous()
    ctx.set_fluid(rho, T, u4)
    for (dim, side), g in f["ghosts"].items():
        orc.set_boundary(dim, side, g)
        gd = torch.zeros(g.shape[:2] + (ctx.pitch,), dtype=torch.float64, device=dev)
        gd[..., :ctx.nd] = torch.as_tensor(g, device=dev)
        ctx.set_boundary(dim, side, gd)
    dt = cfg["dt"]
    if dt is None:
        dt = min(orc.cfl())
    return orc, ctx, f, dt


def run_steps(orc, ctx, f, dt, nsteps, want_moments=True):
    """Run nsteps of rt_step on both sides; returns dict of (gpu, oracle) pairs."""
    import torch

    dev = ctx.device
    I_o, T_o = f["I0"].copy(), f["T"].copy()
    I_g = ctx.to_device(f["I0"])
    T_g = torch.as_tensor(f["T"], device=dev).contiguous().clone()
    R_g = torch.zeros((16,) + ctx.shape, dtype=torch.float64, device=dev)
    G_g = torch.zeros((4,) + ctx.shape, dtype=torch.float64, device=dev)
    nf_o = 0
    for _ in range(nsteps):
        I_o, T_o, R_o, G_o, nf = orc.step(I_o, T_o, dt)
        nf_o += nf
        ctx.step(I_g, T_g, dt, R_g if want_moments else None, G_g if want_moments else None)
    torch.cuda.synchronize()
    shp = ctx.shape
    out = dict(I=(ctx.to_host(I_g), I_o.reshape(shp + (ctx.nd,))), T=(T_g.cpu().numpy(), T_o.reshape(shp)))
    if want_moments:
        out["R"] = (R_g.cpu().numpy(), R_o)
        out["G"] = (G_g.cpu().numpy(), G_o)
    out["nfail"] = (ctx.n_fail(), nf_o)
    out["dt"] = dt
    assert float(I_g[..., ctx.nd:].abs().max()) == 0.0 if ctx.pitch > ctx.nd else True
    return out
