"""rt_step on HOST-resident state with the PCIe copies overlapped with the compute: the mesh is cut into x3 slabs (the
deep-halo decomposition of dist.py, all slabs on ONE GPU), the planes of I^n stream to the device once, each slab
starts its rt_step as soon as its planes (and 4 halo planes each side) have arrived, and its owned planes stream back
while later slabs are still arriving or computing.  H2D, compute and D2H run on three streams; PCIe is full duplex, so
the step costs about one direction's transfer time instead of the sum of both plus the compute (`rt_step_host`, the
single C-ABI call, does H2D -> step -> D2H back to back).

Results are those of rt_step on the whole mesh, bit for bit (tests/test_gpu_dist.py): every slab runs the same kernels
on the same values (see dist.py for the domain-of-dependence argument).

The new state goes to a SECOND set of host buffers (later slabs still read halo planes of the old state).
"""
import numpy as np
import torch

from .dist import SlabDomain, SlabLayout


def _runs(planes):
    """Maximal runs of consecutive global plane indices in `planes` as (local_start, global_start, length)."""
    out, s = [], 0
    for q in range(1, len(planes) + 1):
        if q == len(planes) or planes[q] != planes[q - 1] + 1:
            out.append((s, int(planes[s]), q - s))
            s = q
    return out


class HostPipeline:
    def __init__(self, cfg, nslab, device="cuda:0"):
        self.cfg, self.nslab = cfg, nslab
        noop = lambda layout, tensors, group: None          # halos come from the full input copy, not from neighbours
        self.doms = [SlabDomain(cfg, r, nslab, device=device, exchange_fn=noop) for r in range(nslab)]
        d0 = self.doms[0]
        self.device, self.pitch, self.nd = d0.device, d0.ctx.pitch, d0.ctx.nd
        n1, n2, n3 = cfg["grid"]["n"]
        self.shape = (n3, n2, n1)
        self.units = n1 * n2 * n3 * self.nd
        # the whole input state on the device (each plane crosses PCIe once); slabs copy their range out of it
        self.I_in = torch.empty(self.shape + (self.pitch,), dtype=torch.float64, device=self.device)
        self.T_in = torch.empty(self.shape, dtype=torch.float64, device=self.device)
        for d in self.doms:
            d.I = torch.empty(d.ctx.shape + (self.pitch,), dtype=torch.float64, device=self.device)
            d.T = torch.empty(d.ctx.shape, dtype=torch.float64, device=self.device)
        self.s_in, self.s_cmp, self.s_out = (torch.cuda.Stream(device=self.device) for _ in range(3))
        # upload order: the planes slab 0 needs first (its lower halo wraps to the top of a periodic mesh), then upwards
        first = [int(p) for p in self.doms[0].layout.planes if p >= self.doms[0].layout.k1 + self.doms[0].layout.ext_hi]
        self.order = _runs(np.array(first + [p for p in range(n3) if p not in set(first)]))

    def set_fields(self, f):
        """GLOBAL fluid arrays and boundary ghosts (rt_workloads.fields layout); the intensity comes per step."""
        for d in self.doms:
            d.set_fields(f, state=False)

    def step_host(self, hI, hT, hI_out, hT_out, hR, hG, dt):
        """hI [N3,N2,N1,pitch], hT [N3,N2,N1]: pinned fp64 input state; hI_out, hT_out, hR [16,...], hG [4,...]: pinned
        outputs (hR / hG may be None).  Returns after everything has landed on the host."""
        cur = torch.cuda.current_stream(self.device)
        for s in (self.s_in, self.s_cmp, self.s_out):
            s.wait_stream(cur)
        n3 = self.shape[0]
        arrived = np.zeros(n3, dtype=bool)
        ev_in = []                                            # (event, planes arrived so far)
        with torch.cuda.stream(self.s_in):
            for _, g0, ln in self.order:
                # chunks of at most a slab's worth of planes, so the first slab can start early
                step = max(1, n3 // self.nslab)
                for a in range(g0, g0 + ln, step):
                    b = min(g0 + ln, a + step)
                    self.I_in[a:b].copy_(hI[a:b], non_blocking=True)
                    self.T_in[a:b].copy_(hT[a:b], non_blocking=True)
                    arrived[a:b] = True
                    e = torch.cuda.Event()
                    e.record(self.s_in)
                    ev_in.append((e, arrived.copy()))
        for d in self.doms:
            L = d.layout
            e = next(ev for ev, have in ev_in if have[L.planes].all())
            with torch.cuda.stream(self.s_cmp):
                self.s_cmp.wait_event(e)
                for l0, g0, ln in _runs(L.planes):           # device-to-device: the slab's planes incl. halo
                    d.I[l0:l0 + ln].copy_(self.I_in[g0:g0 + ln], non_blocking=True)
                    d.T[l0:l0 + ln].copy_(self.T_in[g0:g0 + ln], non_blocking=True)
                d.ctx.step(d.I, d.T, dt, d.R if hR is not None else None, d.G if hG is not None else None)
                done = torch.cuda.Event()
                done.record(self.s_cmp)
            with torch.cuda.stream(self.s_out):
                self.s_out.wait_event(done)
                o = L.owned
                hI_out[L.k0:L.k1].copy_(d.I[o], non_blocking=True)
                hT_out[L.k0:L.k1].copy_(d.T[o], non_blocking=True)
                if hR is not None:
                    for c in range(16):
                        hR[c, L.k0:L.k1].copy_(d.R[c, o], non_blocking=True)
                if hG is not None:
                    for c in range(4):
                        hG[c, L.k0:L.k1].copy_(d.G[c, o], non_blocking=True)
        cur.wait_stream(self.s_out)
        cur.wait_stream(self.s_cmp)
        cur.wait_stream(self.s_in)

    def launch_count(self):
        return sum(d.ctx.launch_count() for d in self.doms)
