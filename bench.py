#!/usr/bin/env python
"""bench.py -- throughput of the radiation hot path (one rt_step = predictor + corrector: transport, angular flux,
implicit source, moments) on a synthetic workload shaped like BASELINE.json's configs.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config 1..5] [--impl reference]

Prints ONE JSON line.  metric = cell-direction updates/s (fp64): N_cells * N_dirs * steps / time of rt_step, with
inputs resident in HBM.  `e2e` = the same through the C ABI with pinned HOST buffers (H2D of I, T and D2H of I, T,
R, G inside the timed region).  `roofline` = dominant kernel, algorithmic bytes / CUDA-event time / measured HBM peak.
`cpu_baseline` = the oracle timed on a bounded sample on this box's cores (a baseline, not the target).
N > 1: the mesh grows with N along x3 and is cut into slabs, one per rank, with a 4-plane halo
exchanged point to point once per step (inside the timed region); value = owned cell-directions of all ranks * steps /
max-over-ranks time ("weak").  --multi slab-strong: the config's own mesh cut into N slabs ("strong"; every rank still carries
its 8 halo planes, so thin slabs pay for them).  --multi box [--pgrid P2xP3]: the config's own mesh in x2 x x3 boxes.  --multi
replicas: N independent copies instead.
"""
import argparse
import json
import os
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

METRIC = "cell-direction updates/s (fp64)"
UNIT = "cell-direction updates/s"


def parse():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=None, help="timed steps (default: 200 for the CUDA arm = about a second of timed region on config 4; 3 for --impl reference)")
    ap.add_argument("--warmup", type=int, default=None, help="untimed warm-up steps (default 5; 1 for --impl reference)")
    ap.add_argument("--config", type=int, default=4, help="BASELINE.json config index 1..5 (4 = Kerr-Schild, the roofline config); 6 = snake-coordinates beam (PAPER 4.6)")
    ap.add_argument("--impl", default="b200", choices=["b200", "reference"])
    ap.add_argument("--pgrid", default=None, help="--multi box: process grid P2xP3 along x2 and x3 (default: the most square factorisation of N)")
    ap.add_argument("--multi", default="slab", choices=["slab", "slab-strong", "box", "replicas"],
                    help="N > 1: slab decomposition along x3 with halo exchange -- the mesh grows with N (slab, weak scaling, default) or "
                         "stays the config's (slab-strong: strong scaling, 8 halo planes per rank on fewer owned ones; box: the config's mesh cut "
                         "along x2 and x3, dist.BoxDomain) -- or independent replicas")
    ap.add_argument("--overlap", action="store_true", help="N > 1, slab modes: boundary planes first, their transfer overlapped with the whole-slab step (dist.SlabDomain.step_overlapped)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--size", default=None, help="override grid, e.g. 64x48x32 (debug)")
    ap.add_argument("--transport-tile", type=str, default="0,0,0", help="rt_options.transport_tile: TX,TY,DCH of the TMA tile kernel (0,0,0 = chosen by rt_init)")
    ap.add_argument("--transport-variant", type=int, default=0, choices=[0, 1],
                    help="rt_options.transport_variant: 0 = x2 stencil from L1/L2 (default), 1 = staged in shared memory")
    return ap.parse_args()


# ---- clocks ---------------------------------------------------------------------------------------------------------
class ClockSampler:
    """nvidia-smi sampled DURING the timed region (B200_PROFILING.md clocks line)."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index=0):
        self.rows, self.proc, self.index = [], None, index

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), "--query-gpu=" + self.Q,
                                          "--format=csv,noheader,nounits", "-lms", "100"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.th = threading.Thread(target=self._read, daemon=True)
            self.th.start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append([x.strip() for x in line.split(",")])

    def stop(self):
        if not self.proc:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        try:
            self.proc.wait(timeout=2)
        except Exception:
            pass
        sm = sorted(float(r[0]) for r in self.rows if r and r[0].replace(".", "").isdigit())
        mx = [float(r[1]) for r in self.rows if len(r) > 1 and r[1].replace(".", "").isdigit()]
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        reasons = [n for i, n in enumerate(names) if any(len(r) > 3 + i and r[3 + i].lower().startswith("active") for r in self.rows)]
        pw = [float(r[2]) for r in self.rows if len(r) > 2 and r[2].replace(".", "").isdigit()]
        return {"sm_mhz": sm[len(sm) // 2] if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "power_w_max": max(pw) if pw else None, "samples": len(sm), "reasons": reasons}


def max_over_ranks(x, world, device=None):
    """Multi-GPU timing rule: the slowest rank defines the time.  all_reduce(MAX) over the default process group."""
    if world <= 1:
        return float(x)
    import torch
    import torch.distributed as dist
    t = torch.tensor([float(x)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def aggregate_value(units_per_rank_step, steps, world, ms):
    """Whole-job throughput: every rank processes the same units (replicas / weak scaling); time = max over ranks."""
    return units_per_rank_step * steps * world / (ms * 1e-3)


def measured_peak():
    """(GB/s, which) -- MEASURED_PEAKS.json (driver-written), else the profiling guide's fallback."""
    try:
        with open(os.path.join(ROOT, "MEASURED_PEAKS.json")) as f:
            return float(json.load(f)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    except Exception:
        return 6650.0, "fallback (B200_PROFILING.md 6.65 TB/s)"


# ---- workload -------------------------------------------------------------------------------------------------------
# Algorithmic bytes per cell-direction per LAUNCH of each kernel class:
# what the method must move at this kernel boundary, fp64 = 8 B.  transport: read I_in, (read I_base when it is a
# different array: corrector only), write I_out; angular: read I_in, read+write I_inout; source: read+write I.
ALGO_BYTES = {"transport_pred": 16.0, "transport_corr": 24.0, "angular": 24.0, "source": 16.0}
ISSUE_PEAK = 148 * 4 * 1.965e9          # warp instructions / s: 148 SMs x 4 schedulers x 1 issue per clock at 1965 MHz
# Fixed byte counts of SURVEY.md 8(d) per cell-direction per rt_step: 32 B if each stage read and wrote the intensity once
# (the fully fused ideal), 74 B for two kernels per stage.  The step's fraction of the roofline is quoted against both.
STEP_BYTES_IDEAL, STEP_BYTES_TWO_KERNEL = 32.0, 74.0


def ncu_metrics(cfg_index):
    """ncu-derived per-class figures (DRAM bytes, warp instructions, L2 -> L1 bytes of one rt_step) from the newest
    profiles/*_metrics_c<config>.json whose recorded source hash equals the hash of the library sources that are running.
    None when no capture of THIS build is committed: nothing measured on another build is ever attached to a live time."""
    import glob
    from paper_2508_15532_b200.ncu_metrics import source_hash
    cur = source_hash()
    for path in sorted(glob.glob(os.path.join(ROOT, "profiles", "*_metrics_c%d.json" % cfg_index)), reverse=True):
        try:
            with open(path) as f:
                doc = json.load(f)
        except Exception:
            continue
        if doc.get("source_hash") == cur and doc.get("config") == cfg_index:
            return doc["classes"], os.path.relpath(path, ROOT)
    return None, None


TRANSPORT_VARIANT = 0    # set from --transport-variant
TRANSPORT_TILE = (0, 0, 0)


def make_config(args):
    import rt_workloads as W
    n = tuple(int(x) for x in args.size.split("x")) if args.size else None
    return W.config(args.config, n=n)


def workload_name(cfg):
    n = cfg["grid"]["n"]
    return "%s %dx%dx%d x %d dirs" % (cfg["name"], n[0], n[1], n[2], 10 * cfg["level"] ** 2 + 2)


def setup_gpu(cfg, device):
    """Context + device-resident seeded inputs.  Tables needed by the generator come from the LIBRARY (no oracle)."""
    import numpy as np
    import torch
    import rt_workloads as W
    from paper_2508_15532_b200 import rt

    kind, params = cfg["metric"]
    ctx = rt.RtContext(cfg["grid"], kind, params, cfg["level"], dict(cfg["options"], transport_variant=TRANSPORT_VARIANT, transport_tile=TRANSPORT_TILE), device=device)
    f = W.fields(cfg, ctx.directions()["nhat"], ctx.geometry("e_c"))
    dev = ctx.device
    rho = torch.as_tensor(f["rho"], device=dev).contiguous()
    T = torch.as_tensor(f["T"], device=dev).contiguous()
    u4 = None if f["u4"] is None else torch.as_tensor(f["u4"], device=dev).contiguous()
    ctx.set_fluid(rho, T, u4)
    for (dim, side), g in f["ghosts"].items():
        gd = torch.zeros(g.shape[:2] + (ctx.pitch,), dtype=torch.float64, device=dev)
        gd[..., :ctx.nd] = torch.as_tensor(g, device=dev)
        ctx.set_boundary(dim, side, gd)
    dt = cfg["dt"] if cfg["dt"] is not None else min(ctx.cfl_dt())
    I = ctx.to_device(f["I0"])
    return ctx, f, I, T.clone(), dt


def setup_slab(args, cfg, rank, world, device):
    """N > 1: the mesh grows with N along x3 (weak scaling: every rank owns the config's n3 planes) and is cut into
    slabs; each rank generates the seeded fields of its own extended slab and one halo exchange makes the margins
    consistent.  returns (SlabDomain, global cfg, dt)."""
    import torch
    import torch.distributed as dist
    import rt_workloads as W
    from paper_2508_15532_b200.dist import SlabDomain

    n = cfg["grid"]["n"]
    gcfg = W.config(args.config, n=(n[0], n[1], n[2] * (1 if args.multi == "slab-strong" else world)))
    slab = SlabDomain(gcfg, rank, world, device=device)
    gen = dict(gcfg, grid=dict(slab.grid), seed=gcfg["seed"] + rank)
    f = W.fields(gen, slab.ctx.directions()["nhat"], slab.ctx.geometry("e_c"))
    slab.set_fields(f, local=True)
    slab.exchange_halo()
    dt = gcfg["dt"] if gcfg["dt"] is not None else min(slab.ctx.cfl_dt())
    t = torch.tensor([dt], dtype=torch.float64, device=slab.device)
    dist.all_reduce(t, op=dist.ReduceOp.MIN)       # one global time step (not on the data path)
    return slab, gcfg, float(t.item())


def setup_box(args, cfg, rank, world, device):
    """N > 1, --multi box: the config's own mesh cut into P2 x P3 boxes along x2 and x3 (strong scaling), 4-cell halos on both axes,
    exchanged axis by axis once per step.  Every rank generates the global seeded fields and keeps its box.  returns (BoxDomain, dt)."""
    import torch
    import torch.distributed as dist
    import rt_workloads as W
    from paper_2508_15532_b200.dist import BoxDomain
    if args.pgrid:
        p2, p3 = (int(x) for x in args.pgrid.lower().split("x"))
    else:
        p2 = max(d for d in range(1, int(world ** 0.5) + 1) if world % d == 0)
        p3 = world // p2
    if p2 * p3 != world:
        raise ValueError("--pgrid %dx%d does not match %d ranks" % (p2, p3, world))
    box = BoxDomain(cfg, rank, p2, p3, device=device)
    kind, params = cfg["metric"]
    f = W.fields(cfg, box.ctx.directions()["nhat"], _global_e_c(cfg, kind, params))
    box.set_fields(f)
    dt = cfg["dt"] if cfg["dt"] is not None else min(box.ctx.cfl_dt())
    t = torch.tensor([dt], dtype=torch.float64, device=box.device)
    dist.all_reduce(t, op=dist.ReduceOp.MIN)
    return box, float(t.item())


def _global_e_c(cfg, kind, params):
    """tetrad at the cell centres of the GLOBAL mesh (input of the field generator; the oracle's geometry module is a table builder
    the generators already rely on in the tests -- here a throw-away one-plane context of the library gives the same table)"""
    from paper_2508_15532_b200 import rt
    g = dict(cfg["grid"])
    n = g["n"]
    g["n"] = (n[0], n[1], min(n[2], 8))
    probe = rt.RtContext(g, kind, params, cfg["level"], cfg["options"])
    e = probe.geometry("e_c")
    probe.close()
    return e


def run_gpu(args, rank, world):
    import numpy as np
    import torch
    import torch.distributed as dist

    local = int(os.environ.get("LOCAL_RANK", 0)) % max(torch.cuda.device_count(), 1)
    device = "cuda:%d" % local
    torch.cuda.set_device(local)
    cfg = make_config(args)
    slab, multi = None, "single GPU"
    if world > 1 and args.multi in ("slab", "slab-strong"):
        try:
            slab, cfg, dt = setup_slab(args, cfg, rank, world, device)
            multi = ("slab decomposition along x3 (%s: %d planes per rank), deep halo: 4 planes of I and T per neighbour "
                     "per step over %s send/recv, %d planes computed per rank" % ("strong, the config's mesh" if args.multi == "slab-strong" else "weak",
                                                                                 slab.layout.k1 - slab.layout.k0, dist.get_backend(), slab.layout.n3_local))
        except Exception as e:   # e.g. slabs thinner than the halo: fall back to independent replicas, and say so
            slab, multi = None, "replicas only (slab decomposition unavailable: %s)" % str(e)[:120]
    elif world > 1 and args.multi == "box":
        try:
            slab, dt = setup_box(args, cfg, rank, world, device)
            L = slab.layout
            multi = ("box decomposition %d x %d along x2, x3 (strong, the config's mesh: %d rows x %d planes owned, %d x %d computed per rank), "
                     "4-cell halos exchanged axis by axis once per step over %s send/recv"
                     % (L.p2, L.p3, L.L2.k1 - L.L2.k0, L.L3.k1 - L.L3.k0, L.L2.n3_local, L.L3.n3_local, dist.get_backend()))
        except Exception as e:
            slab, multi = None, "replicas only (box decomposition unavailable: %s)" % str(e)[:120]
    elif world > 1:
        multi = "replicas only (--multi replicas)"
    if slab is not None:
        ctx, I, T, R, G = slab.ctx, slab.I, slab.T, slab.R, slab.G
        dev = ctx.device
        units = slab.owned_units                     # cells this rank OWNS x directions (halo planes are not counted)
        ov = bool(args.overlap and hasattr(slab, "enable_overlap") and slab.enable_overlap())
        if args.overlap:
            multi += "; boundary first, transfer overlapped with the whole-slab step" if ov else "; --overlap not applicable here (plain exchange)"
        step = (lambda: slab.step(dt, overlap=True)) if ov else (lambda: slab.step(dt))
    else:
        ctx, f, I, T, dt = setup_gpu(cfg, device)
        dev = ctx.device
        R = torch.zeros((16,) + ctx.shape, dtype=torch.float64, device=dev)
        G = torch.zeros((4,) + ctx.shape, dtype=torch.float64, device=dev)
        units = ctx.ncell * ctx.nd                   # cell-direction updates per step
        step = lambda: ctx.step(I, T, dt, R, G)
    kernel_units = ctx.ncell * ctx.nd                # what one launch processes (incl. halo planes)
    units_total = units * world
    if slab is not None:                             # slabs may own different numbers of planes
        ut = torch.tensor([float(units)], dtype=torch.float64, device=dev)
        dist.all_reduce(ut)
        units_total = int(ut.item())
    I0, T0 = I.clone(), T.clone()

    def barrier():
        torch.cuda.synchronize()
        if world > 1:
            dist.barrier()

    for _ in range(max(args.warmup, 3)):
        step()
    barrier()
    I.copy_(I0); T.copy_(T0)
    ctx._nfail.zero_()                               # failed temperature solves are counted over the timed region only
    ctx.profile_enable(True)
    ctx.profile_read()
    l0 = ctx.launch_count()
    clocks = ClockSampler(local)
    clocks.start()
    barrier()
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    ev0.record()
    for _ in range(args.steps):
        step()
    ev1.record()
    barrier()
    ms = ev0.elapsed_time(ev1)
    clk = clocks.stop()
    prof = ctx.profile_read()
    ctx.profile_enable(False)
    launches = ctx.launch_count() - l0
    finite = bool(torch.isfinite(I).all().item())
    n_fail = ctx.n_fail()
    ms = max_over_ranks(ms, world, dev)
    # entries that carry work: not a masked direction (n_0 > -n0_floor, L284), not in a zero band (L709)
    n0 = ctx.geometry("n0_c")                        # [E3, N2, N1, nd]
    g = cfg["grid"] if slab is None else slab.grid
    live = (n0 <= -float(cfg["options"].get("n0_floor", 0.1)))
    zl, zh = g.get("zero_lo", (0, 0, 0)), g.get("zero_hi", (0, 0, 0))
    n1_, n2_, n3_ = g["n"]
    live[:, :zl[1]] = False; live[:, n2_ - zh[1]:] = False; live[:, :, :zl[0]] = False; live[:, :, n1_ - zh[0]:] = False
    live_fraction = float(live.mean()) * (n3_ - zl[2] - zh[2]) / n3_

    # ---- end to end through the C ABI with pinned HOST buffers (H2D + D2H inside the timed region) ----
    e2e = None
    if not args.no_e2e:
        hI = torch.empty(I.shape, dtype=torch.float64, pin_memory=True); hI.copy_(I0)
        hT = torch.empty(T.shape, dtype=torch.float64, pin_memory=True); hT.copy_(T0)
        hR = torch.empty(R.shape, dtype=torch.float64, pin_memory=True)
        hG = torch.empty(G.shape, dtype=torch.float64, pin_memory=True)
        ksteps = min(args.steps, 5)
        def one():   # the user-facing C-ABI call with HOST buffers: H2D, rt_step, D2H inside rt_step_host; the state
            if slab is None:
                ctx.step_host(hI, hT, dt, hR, hG)   # lives in pinned host memory and evolves from step to step
            else:                                   # sharded: the halo exchange sits between the step and the D2H
                I.copy_(hI, non_blocking=True); T.copy_(hT, non_blocking=True)
                slab.step(dt)
                hI.copy_(I, non_blocking=True); hT.copy_(T, non_blocking=True)
                hR.copy_(R, non_blocking=True); hG.copy_(G, non_blocking=True)
        one()
        barrier()
        t0 = time.perf_counter()
        ev0.record()
        for _ in range(ksteps):
            one()
        ev1.record()
        barrier()
        ems = ev0.elapsed_time(ev1)
        ems = max_over_ranks(ems, world, dev)
        h2d = (hI.numel() + hT.numel()) * 8
        d2h = (hI.numel() + hT.numel() + hR.numel() + hG.numel()) * 8
        e2e = {"value": units_total * ksteps / (ems * 1e-3), "unit": UNIT, "h2d_bytes_per_step": h2d,
               "d2h_bytes_per_step": d2h, "steps": ksteps, "ms_per_step": ems / ksteps,
               "path": "rt_step_host: one C-ABI call on pinned host buffers; inside it x3 slabs with a 4-plane halo, H2D / rt_step / D2H overlapped on three streams" if slab is None else
                       "H2D -> SlabDomain.step (rt_step + halo exchange) -> D2H"}
        # Coupled mode, the way the paper drives the module (L448-456): the radiation state stays on the GPU; every step the
        # fluid state (rho, T, u^mu: what the GRMHD sector owns) comes from pinned host buffers, and the moments R, the
        # 4-force G and the new T go back.  Extra figure beside the strict one above (which moves the intensity both ways).
        if slab is None and world == 1:
            try:
                pin = lambda a: torch.empty(tuple(a.shape), dtype=torch.float64, pin_memory=True).copy_(torch.as_tensor(a))
                hrho, hTc = pin(f["rho"]), pin(T0.cpu())
                hu4 = None if f["u4"] is None else pin(f["u4"])
                drho = torch.empty_like(T)
                du4 = None if hu4 is None else torch.empty(tuple(hu4.shape), dtype=torch.float64, device=dev)
                I.copy_(I0)
                # R (16 components, the bulk of what goes back) is not what the fluid update waits for: it leaves on a second
                # stream while the next step runs, double-buffered on both sides; G and T are waited for every step
                copy_stream = torch.cuda.Stream(device=dev)
                Rb, hRb, done = [R, torch.empty_like(R)], [hR, torch.empty_like(hR).pin_memory()], [None, None]
                def three(k):
                    b = k & 1
                    main = torch.cuda.current_stream(dev)
                    drho.copy_(hrho, non_blocking=True); T.copy_(hTc, non_blocking=True)
                    if du4 is not None:
                        du4.copy_(hu4, non_blocking=True)
                    ctx.set_fluid(drho, T, du4)
                    if done[b] is not None:
                        main.wait_event(done[b])      # the copy of two steps ago has left this R buffer
                    ctx.step(I, T, dt, Rb[b], G)
                    stepped = torch.cuda.Event(); stepped.record(main)
                    copy_stream.wait_event(stepped)
                    with torch.cuda.stream(copy_stream):
                        hRb[b].copy_(Rb[b], non_blocking=True)
                        done[b] = torch.cuda.Event(); done[b].record(copy_stream)
                    hG.copy_(G, non_blocking=True); hTc.copy_(T, non_blocking=True)
                    main.synchronize()                # the host consumes G, T before it produces the next fluid state
                three(0); three(1)
                barrier()
                ev0.record()
                for k in range(ksteps):
                    three(k)
                ev1.record()
                copy_stream.synchronize()
                barrier()
                cms = ev0.elapsed_time(ev1)
                hR = hRb[(ksteps - 1) & 1]
                if bool(torch.isfinite(hR).all().item()):
                    e2e["coupled"] = {"value": units * ksteps / (cms * 1e-3), "ms_per_step": cms / ksteps,
                                      "h2d_bytes_per_step": (hrho.numel() + hTc.numel() + (0 if hu4 is None else hu4.numel())) * 8,
                                      "d2h_bytes_per_step": (hR.numel() + hG.numel() + hTc.numel()) * 8,
                                      "path": "intensity resident on the GPU; per step H2D of rho, T, u4 -> rt_set_fluid -> rt_step -> "
                                              "D2H of G, T (host synchronised on them every step) and of R on a second stream, "
                                              "overlapping the next step (two buffers)"}
            except Exception as ex:
                e2e["coupled_error"] = str(ex)[:160]
    return dict(cfg=cfg, ctx=ctx, ms=ms, units=units, units_total=units_total, slab=slab is not None, kernel_units=kernel_units, prof=prof, launches=launches, clk=clk, e2e=e2e,
                finite=finite, dt=dt, multi=multi, n_fail=n_fail, live_fraction=live_fraction)


# ---- oracle legs (the only places bench.py may execute oracle/) ----------------------------------------------------
ORACLE_SAMPLE = {1: (64, 64, 1), 2: (24, 24, 24), 3: (24, 24, 24), 4: (64, 48, 16), 5: (32, 24, 8), 6: (64, 64, 1)}


def run_oracle(cfg_index, steps, warmup=0, threads=None):
    """The oracle as it stands on this box's host cores, on a bounded sample of the workload: the same config
    (metric, tetrad, opacities, seeded fields, CFL rule) on a coarser grid.  threads: OpenMP threads of the oracle's cell
    loop (None = all cores).  returns (updates/s, cores, sample, ms per step, cfg)."""
    import ctypes
    import numpy as np
    import rt_workloads as W
    from oracle import Oracle

    ncores = int(os.environ.get("OMP_NUM_THREADS", os.cpu_count() or 1))
    try:   # the thread count of the OpenMP runtime the oracle's library uses (the oracle itself is not touched)
        ctypes.CDLL("libgomp.so.1").omp_set_num_threads(int(threads or ncores))
    except OSError:
        threads = None

    n = ORACLE_SAMPLE[cfg_index]
    cfg = W.config(cfg_index, n=n)
    kind, params = cfg["metric"]
    orc = Oracle(cfg["grid"], kind, params, cfg["level"], cfg["options"])
    f = W.fields(cfg, orc.ang["nhat"], orc.tab["e_c"])
    orc.set_fluid(f["rho"], f["T"], f["u4"])
    for (dim, side), g in f["ghosts"].items():
        orc.set_boundary(dim, side, g)
    dt = cfg["dt"] if cfg["dt"] is not None else min(orc.cfl())
    I, T = f["I0"], f["T"]
    for _ in range(warmup):
        I, T, R, G, nf = orc.step(I, T, dt)
    t0 = time.perf_counter()
    for _ in range(steps):
        I, T, R, G, nf = orc.step(I, T, dt)
    el = time.perf_counter() - t0
    units = n[0] * n[1] * n[2] * orc.nd
    cores = int(threads or ncores)
    sample = "oracle rt_step x%d on %s at %dx%dx%d x %d dirs (same config, coarser grid), OpenMP over cells, %d thread%s" % (
        steps, cfg["name"], n[0], n[1], n[2], orc.nd, cores, "" if cores == 1 else "s")
    return units * steps / el, cores, sample, el / steps * 1e3, cfg


def main_reference(args):
    rank = int(os.environ.get("RANK", 0))
    if rank != 0:
        return
    # exactly K timed steps after W warm-up steps, each step = one oracle rt_step on the bounded sample (0.1-1 s per step)
    val, cores, sample, ms, cfg = run_oracle(args.config, max(1, args.steps), warmup=max(0, args.warmup))
    import rt_workloads as W
    full = W.config(args.config)
    line = {"impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": ms, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": workload_name(full), "timed_sample": sample},
            "cpu_baseline": {"value": val, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
            "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line))


def main():
    args = parse()
    if args.steps is None:
        args.steps = 3 if args.impl == "reference" else 200
    if args.warmup is None:
        args.warmup = 1 if args.impl == "reference" else 5
    global TRANSPORT_VARIANT, TRANSPORT_TILE
    TRANSPORT_VARIANT = args.transport_variant
    TRANSPORT_TILE = (tuple(int(v) for v in args.transport_tile.split(",")) + (0,) * 3)[:3]
    if args.impl == "reference":
        return main_reference(args)
    import torch
    import torch.distributed as dist
    world = int(os.environ.get("WORLD_SIZE", 1))
    rank = int(os.environ.get("RANK", 0))
    if world > 1:
        # RT_BENCH_BACKEND=gloo: functional check of the N > 1 path on a box with fewer GPUs than ranks (halo staged
        # through the host; never a measurement)
        backend = os.environ.get("RT_BENCH_BACKEND", "nccl")
        import datetime
        tmo = datetime.timedelta(minutes=5)      # a stuck exchange aborts instead of hanging the job
        if backend == "nccl":
            dist.init_process_group("nccl", device_id=torch.device("cuda:%d" % int(os.environ.get("LOCAL_RANK", 0))), timeout=tmo)
        else:
            dist.init_process_group(backend, timeout=tmo)
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device and no CPU fallback (use --impl reference for the oracle)")
    r = run_gpu(args, rank, world)
    if rank == 0:
        ms, K = r["ms"], args.steps
        value = r["units_total"] * K / (ms * 1e-3)   # whole job: the units all ranks own, over the max-over-ranks time
        units = r["kernel_units"]                 # per-launch units of the roofline figures
        peak, which = measured_peak()
        prof = r["prof"]
        dom = max(("transport", "angular", "source"), key=lambda k: prof[k][0])
        dms, dcnt = prof[dom]
        per_unit = {"transport": 0.5 * (ALGO_BYTES["transport_pred"] + ALGO_BYTES["transport_corr"]),
                    "angular": ALGO_BYTES["angular"], "source": ALGO_BYTES["source"]}
        achieved = per_unit[dom] * units / (dms / max(dcnt, 1) * 1e-3) / 1e9 if dcnt else 0.0
        single = args.size is None and world == 1
        ncu, ncu_path = ncu_metrics(args.config) if single else (None, None)
        per_step = lambda key: (ncu[dom][key] if ncu and dom in ncu and key in ncu[dom] else None)
        launches_per_step = max(dcnt, 1) / K
        dom_s_per_step = dms / K * 1e-3
        traffic = per_step("dram_bytes")
        winstr = per_step("warp_instr")
        l2b = per_step("l2_to_l1_bytes")
        step_s = ms / K * 1e-3
        roof = {"bound": "hbm", "kernel": dom, "achieved": achieved, "peak": peak, "unit": "GB/s",
                "frac": achieved / peak,
                # ncu figures of THIS build only (hash-matched, see ncu_metrics()); per launch of the class like `achieved`
                "traffic": traffic / launches_per_step if traffic else None,
                "traffic_source": ncu_path, "peak_source": which,
                "algorithmic_bytes_per_launch": per_unit[dom] * units,
                "algorithmic_bytes_per_cell_dir_per_launch": per_unit[dom],
                "kernel_ms_per_step": {k: prof[k][0] / K for k in prof},
                "kernel_launches_per_step": {k: prof[k][1] / K for k in prof},
                "issue": ({"warp_instr_per_step": winstr, "achieved": winstr / dom_s_per_step, "peak": ISSUE_PEAK, "unit": "warp-instr/s",
                           "frac": winstr / dom_s_per_step / ISSUE_PEAK, "source": "instruction count from %s, time live" % ncu_path}
                          if winstr and dcnt else None),
                "l2": ({"l2_to_l1_bytes_per_launch": l2b / launches_per_step, "times_algorithmic": l2b / launches_per_step / (per_unit[dom] * units),
                        "source": ncu_path} if l2b else None),
                # the whole step against the two fixed byte counts of SURVEY.md 8(d) (a design with more kernel boundaries cannot
                # raise its own numerator)
                "step_frac_of_peak_32B": STEP_BYTES_IDEAL * r["units"] / step_s / 1e9 / peak,
                "step_frac_of_peak_74B": STEP_BYTES_TWO_KERNEL * r["units"] / step_s / 1e9 / peak}
        line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": K, "warmup": max(args.warmup, 3),
                "ms_per_step": ms / K, "higher_is_better": True, "scaling": "strong" if (world > 1 and args.multi in ("slab-strong", "box") and r["slab"]) else "weak",
                "vs_baseline": None, "dtype": "f64",
                "data": "synthetic",
                "config": {"workload": workload_name(r["cfg"]), "dt": r["dt"], "l2": "inputs larger than L2 (one I copy >= 1 GB vs 126 MB)"
                           if units * 8 > 2.0e8 else "inputs FIT in L2 (latency-bound config; HBM fraction not meaningful)",
                           "multi_gpu": r["multi"], "transport_variant": TRANSPORT_VARIANT, "transport_path": list(r["ctx"].transport_info()),
                           "finite": r["finite"], "n_fail": r["n_fail"],
                           # share of the (cell, direction) entries that carry work (not masked, not in a zero band); the
                           # others only ever hold 0.0 -- `value` counts every entry
                           "live_fraction": r["live_fraction"]},
                "clocks": r["clk"], "e2e": r["e2e"], "gpu_launches": r["launches"], "roofline": roof}
        if r["n_fail"]:
            raise SystemExit("bench.py: %d temperature solves failed inside the timed region" % r["n_fail"])
        if not args.no_cpu_baseline and world == 1:
            val, cores, sample, oms, _ = run_oracle(args.config, 2)
            val1, _, sample1, _, _ = run_oracle(args.config, 1, threads=1)
            line["cpu_baseline"] = {"value": val, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample,
                                    "single_thread": {"value": val1, "cores": 1, "sample": sample1}}
        print(json.dumps(line))
    if world > 1:
        dist.barrier()
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
