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
        self._sub, self._side, self._rho_d, self._T0_d, self._u4_d, self._has_ghosts = {}, None, None, None, None, False

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
        self._rho_d, self._T0_d, self._u4_d = rho_d, T_d, u4          # kept for enable_overlap()
        self._has_ghosts = bool(f.get("ghosts"))
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

    def step(self, dt, moments=True, overlap=False):
        """One rt_step on the slab, then the halo exchange.  R, G are exact on the owned planes.  overlap=True: boundary first
        (enable_overlap() must have been called), see step_overlapped()."""
        if overlap and self._sub:
            return self.step_overlapped(dt, moments)
        self.ctx.step(self.I, self.T, dt, self.R if moments else None, self.G if moments else None)
        self.exchange_halo()

    # ---- boundary first: "treating the boundaries first and overlapping the transfer with the interior" -----------
    # The planes a neighbour needs are final only after the corrector, so they can leave early only if they are stepped first.  The
    # library does that below the ABI (rt_step_slab, include/rt.h): on each cut side a sub-slab of 3 MARGIN planes is stepped by a
    # context of its own on a side stream, its middle planes land in send buffers, and the transfer runs while the main stream steps
    # the whole slab; what is received lands in buffers and is copied into the margins at the end.  The price is 2 x 3 MARGIN extra
    # planes of compute per step for a transfer that takes 1-2 % of a step on NVLink: an option for slow
    # interconnects, not the default.  Same kernels, same values: the planes sent are bit-identical to the whole-slab step's.
    def enable_overlap(self):
        """Allocate the send buffers.  Returns False (the plain path stays) where the scheme does not apply: a single rank, fewer
        than 2 MARGIN owned planes, caller-supplied ghost data (FIXED boundaries)."""
        import torch
        L = self.layout
        fixed = "fixed" in tuple(self.grid["bc_lo"]) + tuple(self.grid["bc_hi"])
        if L.world == 1 or (L.k1 - L.k0) < 2 * L.margin or fixed or self.I is None:
            return False
        mk = lambda t: torch.empty((L.margin,) + tuple(t.shape[1:]), dtype=t.dtype, device=t.device)
        self._sub = {"lo": (mk(self.I), mk(self.T)) if L.lo_cut else None, "hi": (mk(self.I), mk(self.T)) if L.hi_cut else None}
        return True

    def boundary_first(self, dt, moments=True):
        """rt_step_slab on the current stream and a side stream; returns the send buffers {side: (I planes, T planes)} (the MARGIN owned
        planes next to each cut after this step).  The whole-slab step has been issued on the current stream when this returns."""
        import torch
        if self._side is None:
            self._side = torch.cuda.Stream(device=self.device)
        self.ctx.step_slab(self.I, self.T, dt, self.R if moments else None, self.G if moments else None, self._sub["lo"], self._sub["hi"], self._side)
        return {k: v for k, v in self._sub.items() if v is not None}

    def step_overlapped(self, dt, moments=True):
        import torch
        import torch.distributed as dist
        L = self.layout
        main = torch.cuda.current_stream(self.device)
        bufs = self.boundary_first(dt, moments)      # boundary sub-slabs on the side stream, the whole slab on the main stream
        landed = []
        with torch.cuda.stream(self._side):          # the transfer: ordered after the boundary work, concurrent with the main stream
            stage = dist.get_backend(self.group) == "gloo"
            ops = []
            def send(t, peer):
                ops.append(dist.P2POp(dist.isend, t.cpu() if stage else t, peer, self.group))
            def recv(tensor, dst_sl, peer):
                like = tensor[dst_sl]
                buf = torch.empty(like.shape, dtype=like.dtype, device="cpu" if stage else like.device)
                landed.append((tensor, dst_sl, buf))
                ops.append(dist.P2POp(dist.irecv, buf, peer, self.group))
            for which in (0, 1):                     # I, then T: the order of exchange()
                tensor = self.I if which == 0 else self.T
                if L.lo_cut:
                    send(bufs["lo"][which], L.left)
                if L.hi_cut:
                    send(bufs["hi"][which], L.right)
                if L.hi_cut:
                    recv(tensor, L.recv_hi(), L.right)
                if L.lo_cut:
                    recv(tensor, L.recv_lo(), L.left)
            reqs = dist.batch_isend_irecv(ops)
        for r in reqs:
            r.wait()
        main.wait_stream(self._side)
        for tensor, sl, buf in landed:               # (on the main stream: after the whole-slab step)
            tensor[sl].copy_(buf)

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


# ---- two-dimensional decomposition: x2 x x3 boxes ------------------------------------------------------------------------------------
# The same deep-halo scheme along two axes: a rank owns a box of rows (x2) and planes (x3) and carries MARGIN of each on every cut side.
# Thin x3 slabs pay 8 / n3_local redundant planes; cutting x2 as well keeps both factors small on many ranks (8 ranks on a 96 x 64
# (x2, x3) mesh: 2 x 4 boxes compute (48 + 4..8) x (16 + 8) instead of 96 x (8 + 8): 1.6x the owned cells instead of 2x).  The halo is
# exchanged axis by axis -- x3 first (contiguous planes, all local rows), then x2 (rows of all local planes, margins included, packed
# by `.contiguous()`) -- so the corner blocks arrive through the second phase.  rank = r3 * p2 + r2.
class BoxLayout:
    def __init__(self, n2, n3, periodic2, periodic3, rank, p2, p3, margin=MARGIN):
        if p2 < 1 or p3 < 1 or not (0 <= rank < p2 * p3):
            raise ValueError("bad rank / process grid")
        self.p2, self.p3, self.rank, self.world = p2, p3, rank, p2 * p3
        self.r2, self.r3 = rank % p2, rank // p2
        self.L2 = SlabLayout(n2, periodic2, self.r2, p2, margin)
        self.L3 = SlabLayout(n3, periodic3, self.r3, p3, margin)

    def peer(self, axis, r):
        """global rank of the box at position r along `axis` (2 or 3) in my row / column of the process grid"""
        return self.r3 * self.p2 + r if axis == 2 else r * self.p2 + self.r2


def _axis_slice(t, axis, sl):
    idx = [slice(None)] * t.dim()
    idx[axis] = sl
    return t[tuple(idx)]


def exchange_axis(layout, tensors, axes, left, right, group=None):
    """`exchange` along an arbitrary tensor axis: tensors[i]'s decomposed axis is axes[i]; left / right are the neighbours' global
    ranks.  Non-leading axes give strided pieces: sent from a packed copy, received into a buffer and copied in."""
    import torch
    import torch.distributed as dist
    if layout.world == 1:
        return
    stage = dist.get_backend(group) == "gloo" and any(t.is_cuda for t in tensors)
    ops, landed = [], []
    for t, ax in zip(tensors, axes):
        def send(sl, peer):
            piece = _axis_slice(t, ax, sl).contiguous()
            ops.append(dist.P2POp(dist.isend, piece.cpu() if stage else piece, peer, group))

        def recv(sl, peer):
            view = _axis_slice(t, ax, sl)
            buf = torch.empty(view.shape, dtype=t.dtype, device="cpu" if stage else t.device)
            landed.append((view, buf))
            ops.append(dist.P2POp(dist.irecv, buf, peer, group))

        if layout.lo_cut:
            send(layout.send_lo(), left)
        if layout.hi_cut:
            send(layout.send_hi(), right)
        if layout.hi_cut:
            recv(layout.recv_hi(), right)
        if layout.lo_cut:
            recv(layout.recv_lo(), left)
    for req in dist.batch_isend_irecv(ops):
        req.wait()
    for view, buf in landed:
        view.copy_(buf)


def exchange_box(layout, tensors, axes3, axes2, group=None):
    """Halo update of a BoxLayout: x3 first, then x2 (whose pieces span the x3 margins: corners)."""
    L = layout
    if L.p3 > 1:
        exchange_axis(L.L3, tensors, axes3, None if L.L3.left is None else L.peer(3, L.L3.left),
                      None if L.L3.right is None else L.peer(3, L.L3.right), group)
    if L.p2 > 1:
        exchange_axis(L.L2, tensors, axes2, None if L.L2.left is None else L.peer(2, L.L2.left),
                      None if L.L2.right is None else L.peer(2, L.L2.right), group)


def _cut_grid(g, grid, layout, dim):
    """the part of local_grid() that concerns one dim, for a 1-D layout along it"""
    n = list(g["n"]); n[dim] = layout.n3_local; g["n"] = tuple(n)
    x0 = list(g["x0"]); x0[dim] = grid["x0"][dim] + (layout.k0 - layout.ext_lo) * grid["dx"][dim]; g["x0"] = tuple(x0)
    bl, bh = list(g["bc_lo"]), list(g["bc_hi"])
    if layout.world > 1:
        bl[dim] = "outflow" if layout.lo_cut else grid["bc_lo"][dim]
        bh[dim] = "outflow" if layout.hi_cut else grid["bc_hi"][dim]
        if layout.periodic:
            bl[dim] = bh[dim] = "outflow"
    g["bc_lo"], g["bc_hi"] = tuple(bl), tuple(bh)
    zl, zh = list(g.get("zero_lo", (0, 0, 0))), list(g.get("zero_hi", (0, 0, 0)))
    if layout.lo_cut:
        zl[dim] = 0
    if layout.hi_cut:
        zh[dim] = 0
    g["zero_lo"], g["zero_hi"] = tuple(zl), tuple(zh)
    return g


def local_grid_box(grid, layout):
    g = dict(grid)
    g.setdefault("zero_lo", (0, 0, 0)); g.setdefault("zero_hi", (0, 0, 0))
    g = _cut_grid(g, grid, layout.L3, 2)
    return _cut_grid(g, grid, layout.L2, 1)


class BoxDomain:
    """One rank's box of a mesh decomposed along x2 and x3 (see BoxLayout): library context on the extended box + the halo exchange.
    Same interface as SlabDomain (global fields are cut here)."""

    def __init__(self, cfg, rank, p2, p3, device="cuda:0", group=None):
        import torch
        from . import rt
        grid = cfg["grid"]
        self.layout = BoxLayout(grid["n"][1], grid["n"][2], grid["bc_lo"][1] == "periodic", grid["bc_lo"][2] == "periodic", rank, p2, p3)
        self.group = group
        kind, params = cfg["metric"]
        self.cfg, self.grid = cfg, local_grid_box(grid, self.layout)
        self.ctx = rt.RtContext(self.grid, kind, params, cfg["level"], cfg["options"], device=device)
        self.device = self.ctx.device
        self.I = self.T = None
        self.R = torch.zeros((16,) + self.ctx.shape, dtype=torch.float64, device=self.device)
        self.G = torch.zeros((4,) + self.ctx.shape, dtype=torch.float64, device=self.device)
        L2, L3 = self.layout.L2, self.layout.L3
        self.owned_units = (L3.k1 - L3.k0) * (L2.k1 - L2.k0) * grid["n"][0] * self.ctx.nd

    def _cut(self, a, lead=0):
        """global [.., N3, N2, ...] -> this box's planes and rows (x3 at axis `lead`)"""
        L2, L3 = self.layout.L2, self.layout.L3
        a = np.take(a, L3.planes, axis=lead)
        return np.ascontiguousarray(np.take(a, L2.planes, axis=lead + 1))

    def set_fields(self, f):
        import torch
        dev, L2, L3 = self.device, self.layout.L2, self.layout.L3
        rho, T = self._cut(f["rho"]), self._cut(f["T"])
        u4 = None if f.get("u4") is None else torch.as_tensor(self._cut(f["u4"], 1), device=dev)
        self.ctx.set_fluid(torch.as_tensor(rho, device=dev), torch.as_tensor(T, device=dev), u4)
        self.I = self.ctx.to_device(self._cut(f["I0"]))
        self.T = torch.as_tensor(T, device=dev).clone()
        n1, n2, n3 = self.cfg["grid"]["n"]
        for (dim, side), g in f.get("ghosts", {}).items():
            g = np.asarray(g)
            nd = g.shape[-1]
            if dim == 0:      # [layer][k * N2 + j]
                g = g.reshape(2, n3, n2, nd)[:, L3.planes][:, :, L2.planes].reshape(2, -1, nd)
            elif dim == 1:    # [layer][k * N1 + i]: belongs to the boxes at that physical end of x2
                if (side == 0 and L2.lo_cut) or (side == 1 and L2.hi_cut):
                    continue
                g = g.reshape(2, n3, n1, nd)[:, L3.planes].reshape(2, -1, nd)
            else:             # [layer][j * N1 + i]
                if (side == 0 and L3.lo_cut) or (side == 1 and L3.hi_cut):
                    continue
                g = g.reshape(2, n2, n1, nd)[:, L2.planes].reshape(2, -1, nd)
            gd = torch.zeros(g.shape[:2] + (self.ctx.pitch,), dtype=torch.float64, device=dev)
            gd[..., :self.ctx.nd] = torch.as_tensor(np.ascontiguousarray(g), device=dev)
            self.ctx.set_boundary(dim, side, gd)

    def exchange_halo(self):
        exchange_box(self.layout, [self.I, self.T], [0, 0], [1, 1], self.group)

    def step(self, dt, moments=True):
        self.ctx.step(self.I, self.T, dt, self.R if moments else None, self.G if moments else None)
        self.exchange_halo()

    def owned(self, t, lead=0):
        """View of the owned planes and rows of a box tensor whose x3 axis is `lead` (x2 follows it)."""
        idx = [slice(None)] * t.dim()
        idx[lead], idx[lead + 1] = self.layout.L3.owned, self.layout.L2.owned
        return t[tuple(idx)]


def exchange_local_box(domains):
    """exchange_box for boxes that live in ONE process (list index = rank): x3 phase, then x2 phase, each reading everything before
    it writes anything."""
    import torch
    for axis, attr, tax in ((3, "L3", 0), (2, "L2", 1)):
        new = []
        for d in domains:
            L, got = getattr(d.layout, attr), {}
            for name in ("I", "T"):
                t = getattr(d, name)
                if L.lo_cut:
                    src = domains[d.layout.peer(axis, L.left)]
                    got[(name, "lo")] = _axis_slice(getattr(src, name), tax, getattr(src.layout, attr).send_hi()).to(t.device, copy=True)
                if L.hi_cut:
                    src = domains[d.layout.peer(axis, L.right)]
                    got[(name, "hi")] = _axis_slice(getattr(src, name), tax, getattr(src.layout, attr).send_lo()).to(t.device, copy=True)
            new.append(got)
        for d, got in zip(domains, new):
            L = getattr(d.layout, attr)
            for (name, side), v in got.items():
                _axis_slice(getattr(d, name), tax, L.recv_lo() if side == "lo" else L.recv_hi()).copy_(v)
    if torch.cuda.is_available():
        torch.cuda.synchronize()
