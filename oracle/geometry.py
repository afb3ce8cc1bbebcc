"""ORACLE (test infrastructure, not product code) -- O2: metric, tetrad, Ricci rotation coefficients.

Plain numpy, fp64, written from PAPER.md 2.1 (Eq 1-4), Eq 8 (L107-109), Appendix A (L798-850).
Shares no code with the CUDA path (which builds its tetrad by a generic Gram-Schmidt in C++).

Index conventions: coordinates x^mu = (x^0, x^1, x^2, x^3) are the LOGICAL mesh coordinates (L201);
e[..., mu, a] = e^mu_{a-hat};  einv[..., a, mu] = e^{a-hat}_mu;  g[..., mu, nu] covariant metric;
omega[..., a, c, d] = omega^{a-hat}_{c-hat d-hat} = e^a_beta e^mu_c nabla_mu e^beta_d   (Eq 8).

Metric kinds
  'minkowski'  Cartesian, identity tetrad (L79).
  'mink_cyl'   Cartesian coordinates, flat metric, ROTATING (cylindrical) tetrad e_1=R-hat, e_2=phi-hat,
               e_3=z-hat ("any orthonormal set is valid", L79; the paper's Eq 51 is garbled, S26).  Used to pin
               the angular-flux sign conventions and to exercise omega != 0 cheaply.
  'ks_mks'     Kerr-Schild (t, r, theta, phi), mass 1, spin a, in logical coordinates r = exp(x1),
               theta = pi x2 + (1-h)/2 sin(2 pi x2), phi = x3 (S26).  Tetrad = A3-A4 with reading S25:
               alpha is the LAPSE (1+2r/Sigma)^(-1/2) (A5b prints its inverse; A4a and Eq 4 need the lapse),
               gamma^{ij} is the INVERSE of the 3-metric gamma_ij = g_ij (A5d as printed gives a non-unit e_r).
  'bl_mks'     Boyer-Lindquist (t, r, theta, phi), mass 1, spin a, same logical map as 'ks_mks'; the coordinates of the
               photon-orbit test (section 4.7: "non-horizon-penetrating coordinates ..., namely Boyer-Lindquist"; App A,
               L816, names Kerr-Schild for the same test -- the body text is followed: only in the frame of the
               zero-angular-momentum observers, the tetrad whose e_0 is normal to t = const (Eq 4), does a circular photon
               orbit point exactly along phi-hat, the grid's pole, L590).  Tetrad in closed form: e_t = (1/alpha)(d_t + w d_phi),
               e_r = sqrt(Delta/Sigma) d_r, e_theta = d_theta / sqrt(Sigma), e_phi = d_phi / sqrt(g_phiphi), with
               alpha^2 = Sigma Delta / A, w = 2 a r / A, A = (r^2+a^2)^2 - a^2 Delta sin^2 theta.  Outside the horizon only.
  'snake'      flat space in snake coordinates (t, w, y, z), w = x - A sin(k pi y) (App A.1): metric A1
               with delta = A k pi cos(k pi y); tetrad A2 under reading S27: the printed matrix is the CO-frame
               e^{a-hat}_mu = [[1,0,0,0],[0,1,delta,0],[0,0,1,0],[0,0,0,1]] (rows dt, dx = dw + delta dy, dy, dz) with
               its second row's two entries transposed in print -- as printed neither the matrix nor its transpose is
               orthonormal in A1 (Eq 1 fails), the co-frame reading is.  It is the Cartesian frame, so omega = 0.
Finite differences (S15): 6th-order central, h = 5e-4 in logical coordinates.
"""
import numpy as np

FD_H = 5e-4
ETA = np.diag([-1.0, 1.0, 1.0, 1.0])


def _ks_map(params, X):
    h = params.get("hslope", 0.3)
    r = np.exp(X[..., 0])
    th = np.pi * X[..., 1] + 0.5 * (1.0 - h) * np.sin(2 * np.pi * X[..., 1])
    drdx = r
    dthdx = np.pi + np.pi * (1.0 - h) * np.cos(2 * np.pi * X[..., 1])
    return r, th, drdx, dthdx


def _ks_metric_phys(a, r, th):
    """Kerr-Schild covariant metric in (t, r, theta, phi), M = 1."""
    s2 = np.sin(th) ** 2
    Sig = r * r + a * a * np.cos(th) ** 2
    H = 2.0 * r / Sig
    g = np.zeros(r.shape + (4, 4))
    g[..., 0, 0] = -1.0 + H
    g[..., 0, 1] = g[..., 1, 0] = H
    g[..., 0, 3] = g[..., 3, 0] = -a * H * s2
    g[..., 1, 1] = 1.0 + H
    g[..., 1, 3] = g[..., 3, 1] = -a * s2 * (1.0 + H)
    g[..., 2, 2] = Sig
    g[..., 3, 3] = s2 * (Sig + a * a * s2 * (1.0 + H))
    return g, Sig, H


def _bl_metric_phys(a, r, th):
    """Boyer-Lindquist covariant metric in (t, r, theta, phi), M = 1; also Sigma, Delta, A."""
    s2 = np.sin(th) ** 2
    Sig = r * r + a * a * np.cos(th) ** 2
    Del = r * r - 2.0 * r + a * a
    A = (r * r + a * a) ** 2 - a * a * Del * s2
    g = np.zeros(r.shape + (4, 4))
    g[..., 0, 0] = -(1.0 - 2.0 * r / Sig)
    g[..., 0, 3] = g[..., 3, 0] = -2.0 * a * r * s2 / Sig
    g[..., 1, 1] = Sig / Del
    g[..., 2, 2] = Sig
    g[..., 3, 3] = A * s2 / Sig
    return g, Sig, Del, A


def _snake_delta(params, X):
    """delta = A k pi cos(k pi y) (below Eq A1); y is the second logical coordinate."""
    A, k = params["A"], params["k"]
    return A * k * np.pi * np.cos(k * np.pi * X[..., 1])


def metric(kind, params, X):
    """Covariant metric g_{mu nu} at logical points X[..., 3]."""
    X = np.asarray(X, dtype=np.float64)
    if kind in ("minkowski", "mink_cyl"):
        return np.broadcast_to(ETA, X.shape[:-1] + (4, 4)).copy()
    if kind == "snake":
        d = _snake_delta(params, X)
        g = np.broadcast_to(ETA, X.shape[:-1] + (4, 4)).copy()   # Eq A1
        g[..., 1, 2] = d
        g[..., 2, 1] = d
        g[..., 2, 2] = 1.0 + d * d
        return g
    if kind in ("ks_mks", "bl_mks"):
        r, th, drdx, dthdx = _ks_map(params, X)
        g = _ks_metric_phys(params["a"], r, th)[0] if kind == "ks_mks" else _bl_metric_phys(params["a"], r, th)[0]
        J = np.ones(r.shape + (4,))
        J[..., 1] = drdx
        J[..., 2] = dthdx
        return g * J[..., :, None] * J[..., None, :]
    if kind == "user":   # the caller's metric: params["g"](x[3]) -> g[4, 4], point by point
        flat = X.reshape(-1, 3)
        return np.array([np.asarray(params["g"](x), dtype=np.float64) for x in flat]).reshape(X.shape[:-1] + (4, 4))
    raise ValueError(kind)


def _tetrad_from_metric(g):
    """Tetrad of a stationary metric g[..., 4, 4] when the caller gives none (L57-79): e_0 is the unit normal of the t = const
    slices (Eq 4: e^mu_0 = -g^{0 mu} / sqrt(-g^{00})); the three space-like legs are the coordinate vectors d_3, d_2, d_1 made
    orthonormal in that order (d_3 keeps its direction: with x3 = phi this is the locally non-rotating frame of A3-A4).
    einv[a][mu] = eta_ab g_{mu nu} e^nu_b."""
    gi = np.linalg.inv(g)
    e = np.zeros(g.shape)
    e[..., :, 0] = -gi[..., 0, :] / np.sqrt(-gi[..., 0, 0])[..., None]
    legs = {}
    for a in (3, 2, 1):
        v = np.zeros(g.shape[:-1])
        v[..., a] = 1.0
        for b in range(3, a, -1):
            pr = np.einsum("...i,...ij,...j->...", v[..., 1:], g[..., 1:, 1:], legs[b][..., 1:])
            v = v - pr[..., None] * legs[b]
        nrm = np.sqrt(np.einsum("...i,...ij,...j->...", v[..., 1:], g[..., 1:, 1:], v[..., 1:]))
        legs[a] = v / nrm[..., None]
        e[..., :, a] = legs[a]
    einv = np.einsum("ab,...mn,...nb->...am", ETA, g, e)
    return e, einv


def tetrad(kind, params, X):
    """(e[..., mu, a], einv[..., a, mu]) at logical points X[..., 3]."""
    X = np.asarray(X, dtype=np.float64)
    shp = X.shape[:-1]
    if kind == "user":
        g = metric(kind, params, X)
        if params.get("e") is None:
            return _tetrad_from_metric(g)
        flat = X.reshape(-1, 3)
        e = np.array([np.asarray(params["e"](x), dtype=np.float64) for x in flat]).reshape(shp + (4, 4))
        return e, np.einsum("ab,...mn,...nb->...am", ETA, g, e)
    if kind == "minkowski":
        e = np.broadcast_to(np.eye(4), shp + (4, 4)).copy()
        return e, e.copy()
    if kind == "mink_cyl":
        x, y = X[..., 0], X[..., 1]
        R = np.sqrt(x * x + y * y)
        e = np.zeros(shp + (4, 4))
        e[..., 0, 0] = 1.0
        e[..., 1, 1] = x / R   # e_1 = R-hat
        e[..., 2, 1] = y / R
        e[..., 1, 2] = -y / R  # e_2 = phi-hat
        e[..., 2, 2] = x / R
        e[..., 3, 3] = 1.0
        einv = np.swapaxes(e, -1, -2).copy()  # orthogonal matrix in flat space
        return e, einv
    if kind == "snake":
        d = _snake_delta(params, X)
        einv = np.broadcast_to(np.eye(4), shp + (4, 4)).copy()   # Eq A2 read as the co-frame (S27)
        einv[..., 1, 2] = d
        return np.linalg.inv(einv), einv
    if kind == "bl_mks":
        r, th, drdx, dthdx = _ks_map(params, X)
        a = params["a"]
        g, Sig, Del, A = _bl_metric_phys(a, r, th)
        alpha = np.sqrt(Sig * Del / A)          # lapse of the t = const slices
        w = 2.0 * a * r / A                     # frame dragging: the ZAMO's d phi / d t
        e = np.zeros(shp + (4, 4))
        einv = np.zeros(shp + (4, 4))
        with np.errstate(divide="ignore", invalid="ignore"):
            gpp = np.sqrt(g[..., 3, 3])
            e[..., 0, 0] = 1.0 / alpha
            e[..., 3, 0] = w / alpha
            e[..., 1, 1] = np.sqrt(Del / Sig) / drdx
            e[..., 2, 2] = 1.0 / np.sqrt(Sig) / dthdx
            e[..., 3, 3] = 1.0 / gpp
            einv[..., 0, 0] = alpha
            einv[..., 1, 1] = np.sqrt(Sig / Del) * drdx
            einv[..., 2, 2] = np.sqrt(Sig) * dthdx
            einv[..., 3, 0] = -w * gpp
            einv[..., 3, 3] = gpp
        return e, einv
    if kind == "ks_mks":
        r, th, drdx, dthdx = _ks_map(params, X)
        g, Sig, H = _ks_metric_phys(params["a"], r, th)
        alpha = 1.0 / np.sqrt(1.0 + H)          # lapse (S25)
        betar = H / (1.0 + H)                   # A5c
        gam = g[..., 1:, 1:]                    # A5e
        # on the polar axis gamma_phiphi = 0: the 3-metric is singular and the tetrad undefined there
        # (a zero-area face); substitute the identity so inv() runs, the caller discards those points
        bad = ~(gam[..., 2, 2] > 0)
        gam_safe = gam.copy()
        gam_safe[bad] = np.eye(3)
        gami = np.linalg.inv(gam_safe)                # reading S25
        e = np.zeros(shp + (4, 4))
        einv = np.zeros(shp + (4, 4))
        grr_u, grp_u = gami[..., 0, 0], gami[..., 0, 2]
        g_thth, g_pp, g_rp = gam[..., 1, 1], gam[..., 2, 2], gam[..., 0, 2]
        # A4: e^delta_{a-hat}, in (t, r, theta, phi)
        e[..., 0, 0] = 1.0 / alpha
        e[..., 1, 0] = -betar / alpha
        e[..., 1, 1] = np.sqrt(grr_u)
        e[..., 3, 1] = grp_u / np.sqrt(grr_u)
        e[..., 2, 2] = 1.0 / np.sqrt(g_thth)
        with np.errstate(divide="ignore", invalid="ignore"):
            e[..., 3, 3] = 1.0 / np.sqrt(g_pp)
            # A3: e^{a-hat}_delta
            einv[..., 0, 0] = alpha
            einv[..., 1, 0] = betar / np.sqrt(grr_u)
            einv[..., 1, 1] = 1.0 / np.sqrt(grr_u)
            einv[..., 2, 2] = np.sqrt(g_thth)
            einv[..., 3, 0] = betar * g_rp / np.sqrt(g_pp)
            einv[..., 3, 1] = g_rp / np.sqrt(g_pp)
            einv[..., 3, 3] = np.sqrt(g_pp)
        # to logical coordinates: e'^mu = (dx'^mu/dx^nu) e^nu ; e'_mu = e_nu dx^nu/dx'^mu
        e[..., 1, :] /= drdx[..., None]
        e[..., 2, :] /= dthdx[..., None]
        einv[..., :, 1] *= drdx[..., None]
        einv[..., :, 2] *= dthdx[..., None]
        return e, einv
    raise ValueError(kind)


def sqrt_neg_g(kind, params, X):
    g = metric(kind, params, X)
    return np.sqrt(np.maximum(-np.linalg.det(g), 0.0))


def _fd(fun, X):
    """d fun / d x^i (i = 1..3), 6th-order central differences with step FD_H (reading S15 of DESIGN.md: the paper says only
    "finite difference", L109); returns [..., 3, (fun shape)].  Truncation h^6 f^(7) / 140, round-off ~ 1.5 eps |f| / h."""
    out = []
    for i in range(3):
        d = np.zeros(3)
        d[i] = FD_H
        f = (45.0 * (fun(X + d) - fun(X - d)) - 9.0 * (fun(X + 2 * d) - fun(X - 2 * d)) + (fun(X + 3 * d) - fun(X - 3 * d))) / (60.0 * FD_H)
        out.append(f)
    return np.stack(out, axis=len(X.shape) - 1)


def ricci_rotation(kind, params, X):
    """omega^a_{cd} (Eq 8) at logical points X[..., 3]; stationary metric => d/dx^0 = 0 (L79)."""
    X = np.asarray(X, dtype=np.float64)
    if kind == "minkowski":
        return np.zeros(X.shape[:-1] + (4, 4, 4))
    g = metric(kind, params, X)
    ginv = np.linalg.inv(g)
    e, einv = tetrad(kind, params, X)
    dg3 = _fd(lambda Y: metric(kind, params, Y), X)          # [..., i, s, l]
    de3 = _fd(lambda Y: tetrad(kind, params, Y)[0], X)       # [..., i, beta, d]
    shp = X.shape[:-1]
    dg = np.zeros(shp + (4, 4, 4))                           # dg[mu, s, l] = d_mu g_{s l}
    de = np.zeros(shp + (4, 4, 4))                           # de[mu, beta, d] = d_mu e^beta_d
    dg[..., 1:, :, :] = dg3
    de[..., 1:, :, :] = de3
    # Gamma^b_{m l} = 1/2 g^{b s} (d_m g_{s l} + d_l g_{s m} - d_s g_{m l})
    t = dg + np.swapaxes(dg, -3, -1)                         # [m, s, l]: d_m g_{sl} + d_l g_{sm}
    t = t - np.moveaxis(dg, -3, -2)                          # minus d_s g_{ml}, laid out as [m, s, l]
    Gam = 0.5 * np.einsum("...bs,...msl->...bml", ginv, t)
    nab = de + np.einsum("...bml,...ld->...mbd", Gam, e)     # nabla_mu e^beta_d  [mu, beta, d]
    return np.einsum("...ab,...mc,...mbd->...acd", einv, e, nab)


def cell_coords(grid, dim=None):
    """Logical coordinates of cell centres (dim None) or of the LOWER faces along `dim` (0, 1, 2), extents
    N + 1 along that dim.  grid: dict n=(N1,N2,N3), x0=(..), dx=(..), x3_symmetric.  Returned shape
    [E3, E2, E1, 3] with E3 = 1 if x3_symmetric (geometry evaluated at the first x3 centre)."""
    n, x0, dx = grid["n"], grid["x0"], grid["dx"]
    ax = []
    for a in range(3):
        if a == dim:
            ax.append(x0[a] + dx[a] * np.arange(n[a] + 1))
        else:
            ax.append(x0[a] + dx[a] * (np.arange(n[a]) + 0.5))
    if grid.get("x3_symmetric", False):
        ax[2] = ax[2][:1] if dim != 2 else ax[2][:1]
    X3, X2, X1 = np.meshgrid(ax[2], ax[1], ax[0], indexing="ij")
    return np.stack([X1, X2, X3], axis=-1)


def build_tables(grid, kind, params):
    """All geometry tables the stepping oracle (rt_oracle.c) reads.  See cell_coords for shapes."""
    T = {}
    Xc = cell_coords(grid)
    T["g_c"] = metric(kind, params, Xc)
    T["e_c"], T["einv_c"] = tetrad(kind, params, Xc)
    T["sqrtg_c"] = sqrt_neg_g(kind, params, Xc)
    T["omega_c"] = ricci_rotation(kind, params, Xc)
    for a in range(3):
        Xf = cell_coords(grid, a)
        gf = metric(kind, params, Xf)
        ef, _ = tetrad(kind, params, Xf)
        sg = sqrt_neg_g(kind, params, Xf)
        # zero-area faces (polar axis): the tetrad is undefined there and no flux can cross (S23 / DESIGN)
        dead = ~(sg > 1e-300) | ~np.isfinite(ef).all(axis=(-1, -2))
        ef = np.where(dead[..., None, None], 0.0, ef)
        sg = np.where(dead, 0.0, sg)
        T["g_f%d" % a], T["e_f%d" % a], T["sqrtg_f%d" % a] = gf, ef, sg
    return T
