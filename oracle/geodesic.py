"""ORACLE (test infrastructure, not product code) -- O1: geodesic angular grid.

Plain numpy, fp64, written from PAPER.md section 3.3 (L207-217): icosahedron on the unit sphere,
Delaunay edges bisected and projected, Voronoi diagram of the triangulation as the angular cells.
Shares no code with the CUDA path (paper_2508_15532_b200/csrc/rt_geodesic.cpp is an independent
implementation; the two must agree to round-off).

Readings (restated in DESIGN.md):
  S1  BASELINE "level n" has N_d = 10 n^2 + 2.  n = 2^a * m (m odd): `a` bisect-and-project
      generations (the paper's rule, L211-213), then one frequency-m barycentric subdivision of every
      triangle, projected.  n = 2, 4 are the paper's G1, G2; n = 6 = bisect then trisect.
  S2  pole of the grid along tetrad axis 3; canonical order = z descending, then azimuth ascending.
  S3  weights w_s = exact spherical area of the Voronoi cell (sum = 4 pi).
Edge quantities: corners c1, c2 of the shared Voronoi edge, length
dlam = angle(c1, c2), centre m = normalize(c1 + c2), outward unit normal u (tangent at m,
perpendicular to the edge, pointing from s to its neighbour t).
"""
import numpy as np

_TOL = 1e-9


def _unit(v):
    return v / np.linalg.norm(v, axis=-1, keepdims=True)


def _icosahedron():
    """12 vertices: poles at +-z, upper ring at latitude atan(1/2), azimuth 2 pi k/5, lower ring offset pi/5."""
    lat = np.arctan(0.5)
    v = [(0.0, 0.0, 1.0)]
    for k in range(5):
        az = 2 * np.pi * k / 5
        v.append((np.cos(lat) * np.cos(az), np.cos(lat) * np.sin(az), np.sin(lat)))
    for k in range(5):
        az = 2 * np.pi * k / 5 + np.pi / 5
        v.append((np.cos(lat) * np.cos(az), np.cos(lat) * np.sin(az), -np.sin(lat)))
    v.append((0.0, 0.0, -1.0))
    v = np.array(v)
    # faces = all triples of mutually nearest vertices (edge length of the unit icosahedron)
    d = np.linalg.norm(v[:, None, :] - v[None, :, :], axis=-1)
    edge = np.sort(d[0])[1]
    adj = np.abs(d - edge) < 1e-6
    tris = []
    for a in range(12):
        for b in range(a + 1, 12):
            for c in range(b + 1, 12):
                if adj[a, b] and adj[b, c] and adj[a, c]:
                    tris.append((a, b, c))
    assert len(tris) == 20
    return v, tris


def _subdivide(verts, tris, m):
    """Frequency-m subdivision of every triangle (m=2: the paper's edge bisection), projected to the sphere."""
    verts = [np.array(x) for x in verts]
    edge_pts = {}

    def edge_point(a, b, q):  # point q/m of the way from a to b (q = 1..m-1)
        lo, hi = (a, b) if a < b else (b, a)
        qq = q if a < b else m - q
        key = (lo, hi, qq)
        if key not in edge_pts:
            p = ((m - qq) * verts[lo] + qq * verts[hi]) / m
            verts.append(p / np.linalg.norm(p))
            edge_pts[key] = len(verts) - 1
        return edge_pts[key]

    new_tris = []
    for (a, b, c) in tris:
        # lattice point (i, j): i steps toward b, j steps toward c, from a
        idx = {}
        for i in range(m + 1):
            for j in range(m + 1 - i):
                k = m - i - j
                if i == 0 and j == 0:
                    idx[(i, j)] = a
                elif i == m:
                    idx[(i, j)] = b
                elif j == m:
                    idx[(i, j)] = c
                elif j == 0:
                    idx[(i, j)] = edge_point(a, b, i)
                elif i == 0:
                    idx[(i, j)] = edge_point(a, c, j)
                elif k == 0:
                    idx[(i, j)] = edge_point(b, c, j)
                else:
                    p = (k * verts[a] + i * verts[b] + j * verts[c]) / m
                    verts.append(p / np.linalg.norm(p))
                    idx[(i, j)] = len(verts) - 1
        for i in range(m):
            for j in range(m - i):
                new_tris.append((idx[(i, j)], idx[(i + 1, j)], idx[(i, j + 1)]))
                if i + j < m - 1:
                    new_tris.append((idx[(i + 1, j)], idx[(i + 1, j + 1)], idx[(i, j + 1)]))
    return np.array(verts), new_tris


def _canonical_order(v):
    """S2: z descending (ties within 1e-9), then azimuth in [0, 2pi) ascending."""
    az = np.arctan2(v[:, 1], v[:, 0])
    az = np.where(az < -_TOL, az + 2 * np.pi, az)
    az = np.where(np.abs(az) <= _TOL, 0.0, az)
    order = sorted(range(len(v)), key=lambda i: (-round(v[i, 2] / (10 * _TOL)), az[i]))
    # guard the rounding: neighbours in the sorted list with |dz| < tol must be in one group
    zs = v[order, 2]
    groups = np.concatenate([[0], np.cumsum(np.abs(np.diff(zs)) > _TOL)])
    order = [order[i] for i in sorted(range(len(order)), key=lambda i: (groups[i], az[order[i]]))]
    return np.array(order)


def _tri_solid_angle(a, b, c):
    """Van Oosterom-Strackee: tan(Omega/2) = |a.(b x c)| / (1 + a.b + b.c + c.a) for unit vectors."""
    num = abs(np.dot(a, np.cross(b, c)))
    den = 1.0 + np.dot(a, b) + np.dot(b, c) + np.dot(c, a)
    return 2.0 * np.arctan2(num, den)


def _orient(n, axis):
    """Rotation that takes the grid's pole (0,0,1) to the unit vector along `axis` about the axis perpendicular to both (L215:
    "It can also be easily oriented along a pre-defined direction"); the opposite pole is reached by a half turn about x."""
    a = np.asarray(axis, dtype=float)
    a = a / np.linalg.norm(a)
    z = np.array([0.0, 0.0, 1.0])
    k = np.cross(z, a)
    sn, cs = np.linalg.norm(k), float(np.dot(z, a))
    if sn < 1e-15:
        return n.copy() if cs > 0 else n * np.array([1.0, -1.0, -1.0])
    k = k / sn
    # Rodrigues: v cos + (k x v) sin + k (k.v)(1 - cos)
    return n * cs + np.cross(k, n) * sn + np.outer(n @ k, k) * (1.0 - cs)


def _aberrate(n, beta):
    """Directions n of a frame that moves with velocity beta (c = 1) seen from the frame it moves in: the Lorentz
    transformation of the null vector (1, n) (L215: "the grid can be deformed in advance by performing a Lorentz
    transformation of its directions").  k'^0 = gamma (1 + beta.n), k' = n + [gamma + (gamma - 1) (beta.n) / beta^2] beta ... written
    with gamma^2 / (gamma + 1) = (gamma - 1) / beta^2 so that beta -> 0 is regular."""
    b = np.asarray(beta, dtype=float)
    b2 = float(b @ b)
    assert b2 < 1.0
    gam = 1.0 / np.sqrt(1.0 - b2)
    bn = n @ b
    k0 = gam * (1.0 + bn)
    ks = n + np.outer(gam + gam * gam / (gam + 1.0) * bn, b)
    return ks / k0[:, None]


def build(level, boost=None, axis=None):
    """Return the tables of the geodesic grid with N_d = 10 level^2 + 2 cells.

    axis: direction the grid's pole is turned to (None = tetrad axis 3, S2); boost: velocity of the frame in which the grid is
    the regular one (None = no deformation).  Both act on the cell centres of the regular grid IN ITS CANONICAL ORDER (the
    numbering and the neighbour lists do not change: a Lorentz transformation maps circles on the sphere to circles, so the
    Delaunay triangulation of the deformed centres is the same set of triangles); the Voronoi cells, their areas and edges
    are then those of the deformed centres.

    dict: nd, nhat[nd,3], w[nd], nnb[nd], nb[nd,6] (-1 padded, counter-clockwise seen from outside,
    starting at the lowest neighbour index), dlam[nd,6], emid[nd,6,3], eun[nd,6,3].
    """
    n = int(level)
    assert n >= 1
    a, m = 0, n
    while m % 2 == 0:
        m //= 2
        a += 1
    verts, tris = _icosahedron()
    for _ in range(a):
        verts, tris = _subdivide(verts, tris, 2)
    if m > 1:
        verts, tris = _subdivide(verts, tris, m)
    nd = len(verts)
    assert nd == 10 * n * n + 2, (nd, n)
    order = _canonical_order(verts)
    rank = np.empty(nd, dtype=int)
    rank[order] = np.arange(nd)
    nhat = _unit(verts[order])
    if axis is not None and np.any(np.asarray(axis) != 0):
        nhat = _unit(_orient(nhat, axis))
    if boost is not None and np.any(np.asarray(boost) != 0):
        nhat = _unit(_aberrate(nhat, boost))
    tris = [tuple(rank[list(t)]) for t in tris]

    # circumcentre of each Delaunay triangle = a Voronoi corner
    cc = []
    for (p, q, r) in tris:
        c = np.cross(nhat[q] - nhat[p], nhat[r] - nhat[p])
        c /= np.linalg.norm(c)
        if np.dot(c, nhat[p]) < 0:
            c = -c
        cc.append(c)
    cc = np.array(cc)

    tri_of = [[] for _ in range(nd)]
    for ti, t in enumerate(tris):
        for p in t:
            tri_of[p].append(ti)

    nnb = np.zeros(nd, dtype=np.int32)
    nb = -np.ones((nd, 6), dtype=np.int32)
    w = np.zeros(nd)
    dlam = np.zeros((nd, 6))
    emid = np.zeros((nd, 6, 3))
    eun = np.zeros((nd, 6, 3))
    for s in range(nd):
        c0 = nhat[s]
        # local tangent frame to order neighbours counter-clockwise (seen from outside the sphere)
        ref = np.array([1.0, 0, 0]) if abs(c0[0]) < 0.9 else np.array([0, 1.0, 0])
        e1 = ref - np.dot(ref, c0) * c0
        e1 /= np.linalg.norm(e1)
        e2 = np.cross(c0, e1)
        neigh = sorted({p for ti in tri_of[s] for p in tris[ti] if p != s})
        ang = {t: np.arctan2(np.dot(nhat[t], e2), np.dot(nhat[t], e1)) for t in neigh}
        ccw = sorted(neigh, key=lambda t: ang[t])
        k0 = ccw.index(min(ccw))
        ccw = ccw[k0:] + ccw[:k0]
        nnb[s] = len(ccw)
        assert nnb[s] in (5, 6)
        area = 0.0
        for e, t in enumerate(ccw):
            shared = [ti for ti in tri_of[s] if t in tris[ti]]
            assert len(shared) == 2
            c1, c2 = cc[shared[0]], cc[shared[1]]
            nb[s, e] = t
            dlam[s, e] = np.arctan2(np.linalg.norm(np.cross(c1, c2)), np.dot(c1, c2))
            mid = c1 + c2
            mid /= np.linalg.norm(mid)
            emid[s, e] = mid
            tt = nhat[t] - np.dot(nhat[t], mid) * mid
            ss = c0 - np.dot(c0, mid) * mid
            u = tt - ss
            eun[s, e] = u / np.linalg.norm(u)
            area += _tri_solid_angle(c0, c1, c2)
        w[s] = area
    return dict(nd=nd, nhat=nhat, w=w, nnb=nnb, nb=nb, dlam=dlam, emid=emid, eun=eun)
