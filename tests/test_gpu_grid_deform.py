"""The oriented / Lorentz-deformed geodesic grid (rt_options.grid_axis, grid_boost) on the GPU: the library's
tables against the oracle's, and whole steps on such a grid against the oracle (every kernel only sees the tables: cell
centres, areas, neighbour lists, edge data -> angular coefficients)."""
import numpy as np
import pytest

import rt_workloads as W
from oracle import Oracle
from parity_util import TOL, make_pair, rel_err, run_steps

pytestmark = pytest.mark.gpu


@pytest.mark.parametrize("kw", [dict(grid_boost=(0.3, 0.0, 0.4), grid_axis=(1.0, 0.0, 1.0)), dict(grid_boost=(0.2, -0.3, 0.1)),
                                dict(grid_axis=(0.0, 0.0, -1.0))])
@pytest.mark.parametrize("level", [2, 4, 6])
def test_tables_of_the_deformed_grid_match_the_oracle(kw, level):
    from paper_2508_15532_b200 import rt
    cfg = W.config(3, n=(4, 4, 4))
    kind, params = cfg["metric"]
    orc = Oracle(cfg["grid"], kind, params, level, dict(cfg["options"], **kw))
    ctx = rt.RtContext(cfg["grid"], kind, params, level, dict(cfg["options"], **kw))
    d = ctx.directions()
    assert np.abs(d["nhat"] - orc.ang["nhat"]).max() < 1e-14
    assert np.abs(d["w"] - orc.ang["w"]).max() < 1e-14 and abs(d["w"].sum() - 4 * np.pi) < 1e-13
    assert (d["nb"] == orc.ang["nb"]).all() and (d["nnb"] == orc.ang["nnb"]).all()
    ctx.close()


@pytest.mark.parametrize("idx,n,steps,kw", [
    (4, (16, 12, 6), 3, dict(grid_boost=(0.3, 0.0, 0.4), grid_axis=(1.0, 0.0, 1.0))),        # Kerr-Schild: angular flux on the deformed cells
    (4, (12, 10, 4), 2, dict(grid_boost=(0.0, 0.0, -0.5), ang_recon=1)),                       # MAPR on the deformed grid
    (3, (9, 8, 7), 2, dict(grid_boost=(0.2, -0.3, 0.1))),                                      # no mirror symmetry left (periodic mesh)
    (5, (8, 6, 4), 2, dict(grid_boost=(0.25, 0.0, 0.25)))])                                    # 362 directions, moving fluid
def test_steps_on_a_deformed_grid_match_the_oracle(idx, n, steps, kw):
    cfg = W.config(idx, n=n)
    cfg["options"] = dict(cfg["options"], **kw)
    orc, ctx, f, dt = make_pair(cfg)
    out = run_steps(orc, ctx, f, dt, steps)
    for k in ("I", "T", "R"):
        assert rel_err(*out[k]) <= TOL, k
    assert float(np.abs(out["G"][0] - out["G"][1]).max() * out["dt"] / np.abs(out["R"][1]).max()) <= TOL
    assert out["nfail"][0] == out["nfail"][1]
    ctx.close()


def test_a_grid_without_the_mirror_plane_cannot_reflect():
    from paper_2508_15532_b200 import rt
    cfg = W.config(3, n=(4, 4, 4))
    g = cfg["grid"]
    grid = dict(g, bc_lo=(g["bc_lo"][0], "reflect", g["bc_lo"][2]), bc_hi=(g["bc_hi"][0], "reflect", g["bc_hi"][2]))
    kind, params = cfg["metric"]
    rt.RtContext(grid, kind, params, 2, dict(cfg["options"], grid_boost=(0.3, 0.0, 0.2))).close()        # x-z plane still a mirror plane
    with pytest.raises(rt.RtError):
        rt.RtContext(grid, kind, params, 2, dict(cfg["options"], grid_boost=(0.0, 0.3, 0.0)))
    with pytest.raises(ValueError):
        Oracle(grid, kind, params, 2, dict(cfg["options"], grid_boost=(0.0, 0.3, 0.0)))
    with pytest.raises(rt.RtError):
        rt.RtContext(cfg["grid"], kind, params, 2, dict(cfg["options"], grid_boost=(0.0, 0.8, 0.7)))     # |beta| >= 1


# ---- Eq 19 term by term (rt_options.angflux_split, L239 as printed) ----------------------------------------------------------
@pytest.mark.parametrize("idx,n,steps,kw", [(4, (16, 12, 6), 3, dict(angflux_split=1)),
                                            (5, (8, 6, 4), 2, dict(angflux_split=1, grid_boost=(0.2, 0.0, 0.3)))])
def test_steps_with_the_split_angular_flux_match_the_oracle(idx, n, steps, kw):
    cfg = W.config(idx, n=n)
    cfg["options"] = dict(cfg["options"], **kw)
    orc, ctx, f, dt = make_pair(cfg)
    assert abs(min(ctx.cfl_dt()) - min(orc.cfl())) <= 1e-9 * min(orc.cfl())       # the outflow-rate bound follows the option
    out = run_steps(orc, ctx, f, dt, steps)
    for k in ("I", "T", "R"):
        assert rel_err(*out[k]) <= TOL, k
    assert out["nfail"][0] == out["nfail"][1]
    ctx.close()
    # and it is not the default flux in disguise
    cfg0 = W.config(idx, n=n)
    cfg0["options"] = dict(cfg0["options"], **{k: v for k, v in kw.items() if k != "angflux_split"})
    orc0, ctx0, f0, dt0 = make_pair(cfg0)
    out0 = run_steps(orc0, ctx0, f0, dt, steps)
    assert rel_err(out0["I"][0], out["I"][0]) > 1e-6
    ctx0.close()


def test_split_angular_flux_is_donor_cell_only():
    from paper_2508_15532_b200 import rt
    cfg = W.config(4, n=(8, 6, 2))
    kind, params = cfg["metric"]
    with pytest.raises(rt.RtError):
        rt.RtContext(cfg["grid"], kind, params, 2, dict(cfg["options"], angflux_split=1, ang_recon=1))
