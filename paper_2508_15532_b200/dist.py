"""Multi-GPU: slab decomposition of the mesh along x3 with a deep (communication-avoiding) halo.

SURVEY.md 8(e): the path shards by spatial domain decomposition, all directions of a cell kept together; the paper
lists it as missing.  One rt_step (predictor + corrector, each a 2-cell stencil) has a domain of
dependence of +-4 cells, so a rank that carries MARGIN = 4 extra x3-planes on every cut side can run the plain
single-GPU rt_step on its extended slab and still produce the exact single-domain result on the planes it OWNS; the
planes in the margin are then overwritten with the neighbours' owned values.  That is ONE exchange per step (4 planes
of I and T per neighbour and direction: contiguous memory, sent in place, no packing) instead of one per stage, at the
price of 8 / n3_local redundant planes of compute.  The cut faces get an OUTFLOW boundary, whose influence stays
inside the margin.  Periodic x3 wraps the neighbour relation.

Layout logic (`SlabLayout`) and the exchange (`exchange`) work on any torch tensors, so they are covered by gloo tests
on CPU; `SlabDomain` adds the library context and is the thing a user steps.  One process per GPU.
"""
import numpy as np

MARGIN = 4   # domain of dependence of one predictor-corrector step, in cells


class SlabLayout:
    """Index arithmetic of rank `rank` of `world` for a mesh with n3 planes."""

    def __init__(self, n3, periodic, rank, world, margin=MARGIN):
        if world < 1 or not (0 <= rank < world):
            raise ValueError("bad rank/world")
        base, rem = divmod(n3, world)
        sizes = [base + (1 if r < rem else 0) for r in range(world)]
        if world > 1 and min(sizes) < margin:
            raise ValueError("slab thinner than the halo: n3 = %d over %d ranks" % (n3, world))
        starts = np.concatenate([[0], np.cumsum(sizes)])
        self.n3, self.periodic, self.rank, self.world, self.margin = n3, bool(periodic), rank, world, margin
        self.k0, self.k1 = int(starts[rank]), int(starts[rank + 1])           # owned global planes [k0, k1)
        self.lo_cut = world > 1 and (self.periodic or rank > 0)
        self.hi_cut = world > 1 and (self.periodic or rank < world - 1)
        self.ext_lo = margin if self.lo_cut else 0
        self.ext_hi = margin if self.hi_cut else 0
        self.left = (rank - 1) % world if self.lo_cut else None
        self.right = (rank + 1) % world if self.hi_cut else None
        self.n3_local = self.k1 - self.k0 + self.ext_lo + self.ext_hi
        # global plane index of every local plane (wrapped for periodic x3)
        self.planes = np.arange(self.k0 - self.ext_lo, self.k1 + self.ext_hi) % n3
        self.owned = slice(self.ext_lo, self.ext_lo + self.k1 - self.k0)       # local planes this rank owns

    # local plane ranges of the four halo pieces
    def send_lo(self):   # my lowest owned planes -> left neighbour's upper margin
        return slice(self.ext_lo, self.ext_lo + self.margin)

    def send_hi(self):   # my highest owned planes -> right neighbour's lower margin
        return slice(self.owned.stop - self.margin, self.owned.stop)

    def recv_lo(self):
        return slice(0, self.ext_lo)

    def recv_hi(self):
        return slice(self.owned.stop, self.owned.stop + self.ext_hi)


def exchange(layout, tensors, group=None):
    """Overwrite the margins of every tensor in `tensors` (x3 is their leading axis) with the neighbours' owned planes.

    Point-to-point only (no collective): per tensor at most two sends and two receives, posted in an order that also
    matches when the left and the right neighbour are the same rank (world = 2, periodic): sends (to left, to right),
    receives (from right, from left)."""
    import torch
    import torch.distributed as dist
    if layout.world == 1:
        return
    # NCCL moves device memory directly (NVLink / NVSwitch peer copies); gloo has no point-to-point path for CUDA
    # tensors, so there the halo planes are staged through host memory (functional fallback, used by the tests)
    stage = dist.get_backend(group) == "gloo" and any(t.is_cuda for t in tensors)
    ops, landed = [], []

    def send(t, sl, peer):
        ops.append(dist.P2POp(dist.isend, t[sl].cpu() if stage else t[sl], peer, group))

    def recv(t, sl, peer):
        buf = torch.empty(t[sl].shape, dtype=t.dtype) if stage else t[sl]
        if stage:
            landed.append((t, sl, buf))
        ops.append(dist.P2POp(dist.irecv, buf, peer, group))

    for t in tensors:
        if layout.lo_cut:
            send(t, layout.send_lo(), layout.left)
        if layout.hi_cut:
            send(t, layout.send_hi(), layout.right)
        if layout.hi_cut:
            recv(t, layout.recv_hi(), layout.right)
        if layout.lo_cut:
            recv(t, layout.recv_lo(), layout.left)
    for req in dist.batch_isend_irecv(ops):
        req.wait()
    for t, sl, buf in landed:
        t[sl].copy_(buf)


def local_grid(grid, layout):
    """The extended slab of `layout` as a grid description for rt_init: x3 extent and origin of the local planes,
    OUTFLOW on cut faces, the physical boundary (and its zero band) only where the slab touches it."""
    g = dict(grid)
    n1, n2, _ = grid["n"]
    g["n"] = (n1, n2, layout.n3_local)
    x0, dx = list(grid["x0"]), grid["dx"]
    x0[2] = x0[2] + (layout.k0 - layout.ext_lo) * dx[2]
    g["x0"] = tuple(x0)
    bl, bh = list(grid["bc_lo"]), list(grid["bc_hi"])
    if layout.world > 1:
        bl[2] = "outflow" if layout.lo_cut else grid["bc_lo"][2]
        bh[2] = "outflow" if layout.hi_cut else grid["bc_hi"][2]
        if layout.periodic:   # a periodic dimension cut into slabs is no longer periodic locally
            bl[2] = bh[2] = "outflow"
    g["bc_lo"], g["bc_hi"] = tuple(bl), tuple(bh)
    zl, zh = list(grid.get("zero_lo", (0, 0, 0))), list(grid.get("zero_hi", (0, 0, 0)))
    if layout.lo_cut:
        zl[2] = 0
    if layout.hi_cut:
        zh[2] = 0
    g["zero_lo"], g["zero_hi"] = tuple(zl), tuple(zh)
    return g


class SlabDomain:
    """One rank's share of a mesh: library context on the extended slab + the per-step halo exchange.

    fields: dict with GLOBAL arrays I0[N3,N2,N1,nd], rho, T, u4 (or None) and ghosts {(dim, side): [2][faces][nd]} as
    rt_workloads.fields() returns them, or LOCAL arrays already cut to `layout.planes` when local=True (then the
    margins may hold anything: call exchange_halo() once before the first step)."""

    def __init__(self, cfg, rank, world, device="cuda:0", group=None, exchange_fn=None):
        import torch
        from . import rt
        grid = cfg["grid"]
        self.layout = SlabLayout(grid["n"][2], grid["bc_lo"][2] == "periodic", rank, world)
        self.group, self._exchange = group, exchange_fn or exchange
        kind, params = cfg["metric"]
        self.cfg, self.grid = cfg, local_grid(grid, self.layout)
        self.ctx = rt.RtContext(self.grid, kind, params, cfg["level"], cfg["options"], device=device)
        self.device = self.ctx.device
        self.I = self.T = None
        self.R = torch.zeros((16,) + self.ctx.shape, dtype=torch.float64, device=self.device)
        self.G = torch.zeros((4,) + self.ctx.shape, dtype=torch.float64, device=self.device)
        self.owned_units = (self.layout.k1 - self.layout.k0) * grid["n"][0] * grid["n"][1] * self.ctx.nd

    def set_fields(self, f, local=False, state=True):
        import torch
        L, dev = self.layout, self.device
        cut = (lambda a: a) if local else (lambda a: a[L.planes])
        cut4 = (lambda a: a) if local else (lambda a: a[:, L.planes])
        rho, T = np.ascontiguousarray(cut(f["rho"])), np.ascontiguousarray(cut(f["T"]))
        u4 = None if f.get("u4") is None else torch.as_tensor(np.ascontiguousarray(cut4(f["u4"])), device=dev)
        rho_d, T_d = torch.as_tensor(rho, device=dev), torch.as_tensor(T, device=dev)
        if local and L.world > 1:
            # locally generated fields: the margins of the FLUID arrays must hold the neighbours' owned planes as well (they
            # enter the face opacities and the source step of the margin cells, whose influence reaches owned planes)
            comps = [] if u4 is None else [u4[m] for m in range(4)]
            self._exchange(L, [rho_d, T_d] + comps, self.group)
            T = T_d.cpu().numpy()
        self.ctx.set_fluid(rho_d, T_d, u4)
        if state:   # (state=False: fluid and boundary data only; the caller owns I and T)
            self.I = self.ctx.to_device(np.ascontiguousarray(cut(f["I0"])))
            self.T = torch.as_tensor(T, device=dev).clone()
        n1, n2, _ = self.cfg["grid"]["n"]
        for (dim, side), g in f.get("ghosts", {}).items():
            g = np.asarray(g)
            if dim == 2:   # an x3 ghost belongs to the rank at that physical end
                if (side == 0 and L.lo_cut) or (side == 1 and L.hi_cut):
                    continue
            elif not local:   # x1 / x2 ghosts are [layer][k * N + other][s]: keep this slab's planes
                per = n2 if dim == 0 else n1
                g = g.reshape(2, -1, per, g.shape[-1])[:, L.planes].reshape(2, -1, g.shape[-1])
            gd = torch.zeros(g.shape[:2] + (self.ctx.pitch,), dtype=torch.float64, device=dev)
            gd[..., :self.ctx.nd] = torch.as_tensor(np.ascontiguousarray(g), device=dev)
            self.ctx.set_boundary(dim, side, gd)

    def exchange_halo(self):
        self._exchange(self.layout, [self.I, self.T], self.group)

    def step(self, dt, moments=True):
        """One rt_step on the slab, then the halo exchange.  R, G are exact on the owned planes."""
        self.ctx.step(self.I, self.T, dt, self.R if moments else None, self.G if moments else None)
        self.exchange_halo()

    def owned(self, t, lead=0):
        """View of the owned planes of a slab tensor whose x3 axis is `lead`."""
        idx = [slice(None)] * t.dim()
        idx[lead] = self.layout.owned
        return t[tuple(idx)]


def exchange_local(domains):
    """The same halo update for slabs that live in ONE process (all ranks of a decomposition held in a list, e.g. several
    slabs time-sliced on one GPU): margins are copied straight from the neighbours' owned planes.  Call it after every
    slab has taken its step (use ctx.step directly, not SlabDomain.step)."""
    import torch
    new = []
    for d in domains:   # read everything first: a margin must receive the neighbour's PRE-exchange owned planes
        L, got = d.layout, {}
        for name in ("I", "T"):
            t = getattr(d, name)
            if L.lo_cut:
                src = domains[L.left]
                got[(name, "lo")] = getattr(src, name)[src.layout.send_hi()].to(t.device, copy=True)
            if L.hi_cut:
                src = domains[L.right]
                got[(name, "hi")] = getattr(src, name)[src.layout.send_lo()].to(t.device, copy=True)
        new.append(got)
    for d, got in zip(domains, new):
        L = d.layout
        for (name, side), v in got.items():
            getattr(d, name)[L.recv_lo() if side == "lo" else L.recv_hi()].copy_(v)
    if torch.cuda.is_available():
        torch.cuda.synchronize()
