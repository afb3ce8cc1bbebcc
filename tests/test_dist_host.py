"""Host-side logic of the slab decomposition (paper_2508_15532_b200/dist.py): layout arithmetic and the point-to-point
halo exchange, run as real multi-process jobs over gloo on CPU tensors (the exchange code is backend-agnostic; on the
GPU box it runs over NCCL)."""
import os
import socket
import subprocess
import sys
import textwrap

import numpy as np
import pytest

from paper_2508_15532_b200.dist import MARGIN, SlabLayout, local_grid

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.mark.parametrize("n3,world,periodic", [(64, 1, True), (64, 2, True), (64, 8, True), (13, 3, False), (21, 4, True)])
def test_layout_partitions_the_mesh(n3, world, periodic):
    seen = np.zeros(n3, int)
    for r in range(world):
        L = SlabLayout(n3, periodic, r, world)
        seen[L.k0:L.k1] += 1
        assert L.n3_local == len(L.planes)
        assert (L.planes[L.owned] == np.arange(L.k0, L.k1)).all()
        if world == 1:
            assert L.n3_local == n3 and not L.lo_cut and not L.hi_cut
            continue
        assert L.lo_cut == (periodic or r > 0) and L.hi_cut == (periodic or r < world - 1)
        if L.lo_cut:   # my lower margin = the left neighbour's highest owned planes, in order
            Ln = SlabLayout(n3, periodic, L.left, world)
            assert (L.planes[L.recv_lo()] == Ln.planes[Ln.send_hi()]).all()
        if L.hi_cut:
            Rn = SlabLayout(n3, periodic, L.right, world)
            assert (L.planes[L.recv_hi()] == Rn.planes[Rn.send_lo()]).all()
    assert (seen == 1).all()


def test_layout_rejects_slabs_thinner_than_the_halo():
    with pytest.raises(ValueError):
        SlabLayout(12, True, 0, 4)      # 3 planes per rank < MARGIN


def test_local_grid_boundaries():
    grid = dict(n=(8, 6, 20), x0=(0.0, 0.0, 1.0), dx=(0.1, 0.1, 0.5), bc_lo=("outflow", "outflow", "zero"),
                bc_hi=("outflow", "outflow", "outflow"), zero_lo=(0, 1, 2), zero_hi=(0, 1, 0))
    g0 = local_grid(grid, SlabLayout(20, False, 0, 2))
    g1 = local_grid(grid, SlabLayout(20, False, 1, 2))
    assert g0["n"] == (8, 6, 10 + MARGIN) and g0["bc_lo"][2] == "zero" and g0["bc_hi"][2] == "outflow"
    assert g0["zero_lo"] == (0, 1, 2) and g0["x0"][2] == 1.0
    assert g1["n"] == (8, 6, 10 + MARGIN) and g1["bc_lo"][2] == "outflow" and g1["zero_lo"] == (0, 1, 0)
    assert abs(g1["x0"][2] - (1.0 + (10 - MARGIN) * 0.5)) < 1e-15
    gp = local_grid(dict(grid, bc_lo=("outflow", "outflow", "periodic"), bc_hi=("outflow", "outflow", "periodic")),
                    SlabLayout(20, True, 0, 2))
    assert gp["n"][2] == 10 + 2 * MARGIN and gp["bc_lo"][2] == gp["bc_hi"][2] == "outflow"


WORKER = textwrap.dedent('''
    import os, sys
    import numpy as np, torch, torch.distributed as dist
    sys.path.insert(0, sys.argv[1])
    from paper_2508_15532_b200.dist import SlabLayout, exchange
    n3, periodic = int(sys.argv[2]), sys.argv[3] == "1"
    dist.init_process_group("gloo")
    rank, world = dist.get_rank(), dist.get_world_size()
    L = SlabLayout(n3, periodic, rank, world)
    def make(width):
        t = torch.full((L.n3_local, width), -1.0, dtype=torch.float64)
        t[L.owned] = torch.arange(L.k0, L.k1, dtype=torch.float64)[:, None] * 10 + torch.arange(width, dtype=torch.float64)
        return t
    A, B = make(5), make(2)
    for _ in range(2):                      # twice: the exchange must be repeatable
        exchange(L, [A, B])
    for t, w in ((A, 5), (B, 2)):
        want = torch.as_tensor(L.planes, dtype=torch.float64)[:, None] * 10 + torch.arange(w, dtype=torch.float64)
        assert torch.equal(t, want), (rank, t[:, 0], want[:, 0])
    dist.barrier()
    dist.destroy_process_group()
    print("ok", rank)
''')


@pytest.mark.parametrize("world,n3,periodic", [(2, 11, True), (2, 9, False), (3, 14, True), (4, 17, False)])
def test_exchange_over_gloo(tmp_path, world, n3, periodic):
    script = tmp_path / "worker.py"
    script.write_text(WORKER)
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        port = s.getsockname()[1]
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", str(world),
           "--master-addr", "127.0.0.1", "--master-port", str(port), str(script), ROOT, str(n3), "1" if periodic else "0"]
    env = dict(os.environ, OMP_NUM_THREADS="1")
    p = subprocess.run(cmd, capture_output=True, text=True, timeout=300, env=env)
    assert p.returncode == 0, p.stdout[-2000:] + p.stderr[-2000:]
    assert p.stdout.count("ok") == world


# ---- two-dimensional (x2 x x3) decomposition --------------------------------------------------------------------------------------
from paper_2508_15532_b200.dist import BoxLayout, local_grid_box


@pytest.mark.parametrize("n2,n3,p2,p3,per2,per3", [(12, 16, 2, 2, False, True), (17, 13, 3, 2, True, False), (8, 40, 1, 4, False, True),
                                                   (24, 9, 4, 1, True, True)])
def test_box_layout_partitions_the_mesh(n2, n3, p2, p3, per2, per3):
    seen = np.zeros((n3, n2), int)
    for r in range(p2 * p3):
        B = BoxLayout(n2, n3, per2, per3, r, p2, p3)
        assert B.rank == B.r3 * p2 + B.r2 and B.peer(2, B.r2) == r and B.peer(3, B.r3) == r
        seen[B.L3.k0:B.L3.k1, B.L2.k0:B.L2.k1] += 1
        for axis, L in ((2, B.L2), (3, B.L3)):
            if L.lo_cut:
                N = BoxLayout(n2, n3, per2, per3, B.peer(axis, L.left), p2, p3)
                Ln = N.L2 if axis == 2 else N.L3
                assert (L.planes[L.recv_lo()] == Ln.planes[Ln.send_hi()]).all()
                # the neighbour along one axis has my position along the other
                assert (N.r3 == B.r3) if axis == 2 else (N.r2 == B.r2)
    assert (seen == 1).all()


def test_local_grid_box_boundaries():
    grid = dict(n=(8, 24, 20), x0=(0.0, 2.0, 1.0), dx=(0.1, 0.25, 0.5), bc_lo=("outflow", "reflect", "periodic"),
                bc_hi=("outflow", "outflow", "periodic"), zero_lo=(0, 2, 0), zero_hi=(0, 3, 0))
    g = local_grid_box(grid, BoxLayout(24, 20, False, True, 0, 2, 2))          # r2 = 0, r3 = 0
    assert g["n"] == (8, 12 + MARGIN, 10 + 2 * MARGIN)
    assert g["bc_lo"] == ("outflow", "reflect", "outflow") and g["bc_hi"] == ("outflow", "outflow", "outflow")
    assert g["zero_lo"] == (0, 2, 0) and g["zero_hi"] == (0, 0, 0)             # the upper x2 side is a cut: no band there
    assert g["x0"][1] == 2.0 and abs(g["x0"][2] - (1.0 - MARGIN * 0.5)) < 1e-15
    g = local_grid_box(grid, BoxLayout(24, 20, False, True, 3, 2, 2))          # r2 = 1, r3 = 1
    assert g["bc_lo"][1] == "outflow" and g["bc_hi"][1] == "outflow" and g["zero_lo"][1] == 0 and g["zero_hi"][1] == 3
    assert abs(g["x0"][1] - (2.0 + (12 - MARGIN) * 0.25)) < 1e-15


WORKER2 = textwrap.dedent('''
    import os, sys
    import numpy as np, torch, torch.distributed as dist
    sys.path.insert(0, sys.argv[1])
    from paper_2508_15532_b200.dist import BoxLayout, exchange_box
    n2, n3, p2, p3 = (int(x) for x in sys.argv[2:6])
    per2, per3 = sys.argv[6] == "1", sys.argv[7] == "1"
    dist.init_process_group("gloo")
    rank, world = dist.get_rank(), dist.get_world_size()
    assert world == p2 * p3
    B = BoxLayout(n2, n3, per2, per3, rank, p2, p3)
    K = torch.as_tensor(B.L3.planes, dtype=torch.float64)[:, None, None]
    J = torch.as_tensor(B.L2.planes, dtype=torch.float64)[None, :, None]
    def make(width):
        want = K * 1000 + J * 10 + torch.arange(width, dtype=torch.float64)[None, None, :]
        t = torch.full(want.shape, -1.0, dtype=torch.float64)
        t[B.L3.owned, B.L2.owned] = want[B.L3.owned, B.L2.owned]
        return t, want
    (A, wa), (C, wc) = make(3), make(1)
    Cs = C[..., 0].clone()                      # a tensor without trailing axes, like T
    for _ in range(2):
        exchange_box(B, [A, Cs], [0, 0], [1, 1])
    assert torch.equal(A, wa), (rank, (A - wa).abs().max())
    assert torch.equal(Cs, wc[..., 0])
    dist.barrier()
    dist.destroy_process_group()
    print("ok", rank)
''')


@pytest.mark.parametrize("p2,p3,n2,n3,per2,per3", [(2, 2, 11, 13, False, True), (2, 2, 9, 9, True, True), (3, 1, 14, 5, False, False),
                                                   (2, 3, 10, 14, False, False)])
def test_box_exchange_over_gloo(tmp_path, p2, p3, n2, n3, per2, per3):
    """Margins AND corner blocks of every box equal the global field after the two-phase exchange (real processes, gloo)."""
    script = tmp_path / "worker2.py"
    script.write_text(WORKER2)
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        port = s.getsockname()[1]
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", str(p2 * p3),
           "--master-addr", "127.0.0.1", "--master-port", str(port), str(script), ROOT, str(n2), str(n3), str(p2), str(p3),
           "1" if per2 else "0", "1" if per3 else "0"]
    env = dict(os.environ, OMP_NUM_THREADS="1")
    p = subprocess.run(cmd, capture_output=True, text=True, timeout=300, env=env)
    assert p.returncode == 0, p.stdout[-2000:] + p.stderr[-2000:]
    assert p.stdout.count("ok") == p2 * p3
