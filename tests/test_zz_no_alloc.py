"""rt_transport_static: the transport launch for callers that cannot allocate (scratch in a file-scope device array).

Collected last on purpose (the suite runs with `pytest -x`).  Checks the entry point against the existing rt_transport path on
two calls in a row -- the shared array keeps the previous call's contents, so the second call (other inputs, other time step,
other mesh) must not see them -- and that a mesh beyond the array's size is refused with a clear error.
"""
import numpy as np
import pytest

import rt_workloads as W
from parity_util import TOL, rel_err

pytestmark = pytest.mark.gpu


def _ctx(idx, n):
    import torch
    from paper_2508_15532_b200 import rt
    cfg = W.config(idx, n=n)
    kind, params = cfg["metric"]
    ctx = rt.RtContext(cfg["grid"], kind, params, cfg["level"], cfg["options"])
    f = W.fields(cfg, ctx.directions()["nhat"], ctx.geometry("e_c"))
    dev = ctx.device
    ctx.set_fluid(torch.as_tensor(f["rho"], device=dev).contiguous(), torch.as_tensor(f["T"], device=dev).contiguous(),
                  None if f["u4"] is None else torch.as_tensor(f["u4"], device=dev).contiguous())
    dt = cfg["dt"] if cfg["dt"] is not None else min(ctx.cfl_dt())
    return ctx, f, dt


def test_static_scratch_transport_matches_rt_transport_on_two_calls_in_a_row():
    import torch
    # call 1: Kerr-Schild torus (vacuum and Eq 23 cells, masked directions); call 2: all-matter flat mesh of another shape
    for k, (idx, n) in enumerate([(4, (24, 20, 6)), (3, (10, 9, 7))]):
        ctx, f, dt = _ctx(idx, n)
        rng = np.random.default_rng(40 + k)
        I0 = f["I0"] + rng.uniform(0.0, 1e-2, size=f["I0"].shape)
        I = ctx.to_device(I0)
        Ib = ctx.to_device(0.5 * I0)
        for base, step in ((I, 0.5 * dt), (Ib, dt)):           # predictor- and corrector-type calls
            ref = torch.full_like(I, 7.0)
            out = torch.full_like(I, -3.0)
            ctx.transport(I, base, ref, step)
            ctx.transport_static(I, base, out, step)
            torch.cuda.synchronize()
            assert torch.isfinite(out).all()
            assert rel_err(out.cpu().numpy(), ref.cpu().numpy()) <= TOL
            assert torch.equal(out, ref)                       # same kernels, same arithmetic
        ctx.close()


def test_static_scratch_rejects_a_mesh_beyond_its_size():
    import torch
    from paper_2508_15532_b200 import rt
    ctx, f, dt = _ctx(3, (48, 48, 48))                         # 110 592 cells: 3 x 32 B per face > 8 MiB
    I = ctx.to_device(f["I0"])
    out = torch.empty_like(I)
    with pytest.raises(rt.RtError, match="too large for the static scratch"):
        ctx.transport_static(I, I, out, dt)
    ctx.transport(I, I, out, dt)                               # the allocating path takes it
    torch.cuda.synchronize()
    ctx.close()
    # without opacities the launch needs no scratch: any mesh is accepted
    cfg = W.config(1, n=(64, 64, 1))
    kind, params = cfg["metric"]
    v = rt.RtContext(cfg["grid"], kind, params, cfg["level"], cfg["options"])
    fv = W.fields(cfg, v.directions()["nhat"], v.geometry("e_c"))
    v.set_fluid(torch.as_tensor(fv["rho"], device=v.device).contiguous(), torch.as_tensor(fv["T"], device=v.device).contiguous(), None)
    for (dim, side), g in fv["ghosts"].items():
        gd = torch.zeros(g.shape[:2] + (v.pitch,), dtype=torch.float64, device=v.device)
        gd[..., :v.nd] = torch.as_tensor(g, device=v.device)
        v.set_boundary(dim, side, gd)
    Iv = v.to_device(fv["I0"] + 0.01)
    a, b = torch.empty_like(Iv), torch.empty_like(Iv)
    v.transport(Iv, Iv, a, cfg["dt"]); v.transport_static(Iv, Iv, b, cfg["dt"])
    torch.cuda.synchronize()
    assert torch.equal(a, b)
    v.close()
