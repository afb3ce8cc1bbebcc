"""Seeded synthetic workloads shaped like BASELINE.json's five configs,
plus config 6 = the snake-coordinates beam of PAPER.md 4.6 (L557-559).

This module serves BOTH the oracle and the CUDA path and therefore holds NONE of the method's arithmetic:
it only fills arrays (random fields, profiles) from `numpy.random.default_rng(seed)`, seed = 1000 + config
index.  Anything that needs the method's tables (direction vectors, tetrads) takes them as arguments from
whichever side is calling.  No dataset exists for this paper: these inputs stand in for its tests
(colliding beams L490-496, equilibration, static diffusion L619-644, radiating disk L594-617 and
the accretion torus L705-725; the Fishbone-Moncrief formulas are not in PAPER.md, a smooth torus with the
same radii stands in).

Array layout everywhere: [N3, N2, N1(, nd)], direction index fastest, no padding.
"""
import math

import numpy as np

FULL_SIZES = {1: (64, 64, 1), 2: (64, 64, 64), 3: (128, 128, 128), 4: (128, 96, 64), 5: (192, 128, 96), 6: (128, 128, 1),
              7: (512, 1, 256)}
LEVELS = {1: 2, 2: 4, 3: 4, 4: 4, 5: 6, 6: 4, 7: 8}
NSTEPS = {1: 100, 2: 200, 3: 500, 4: 50, 5: 20, 6: 400, 7: 1000}
NAMES = {1: "flat_beam_2d", 2: "flat_thermal_relaxation", 3: "scattering_diffusion",
         4: "kerr_schild_torus", 5: "coupled_accretion_step", 6: "snake_beam", 7: "bl_photon_orbit"}


def config(idx, n=None, level=None):
    """Static description of config `idx` (1-5); `n` overrides the grid size (scaled-down parity cases)."""
    n = tuple(n or FULL_SIZES[idx])
    level = level or LEVELS[idx]
    c = dict(index=idx, name=NAMES[idx], level=level, nsteps=NSTEPS[idx], seed=1000 + idx)
    per = ("periodic",) * 3
    if idx == 1:
        N = n[0]
        c["grid"] = dict(n=n, x0=(0.0, 0.0, 0.0), dx=(1.0 / N, 1.0 / N, 1.0 / N),
                         bc_lo=("fixed", "outflow", "periodic"), bc_hi=("outflow", "outflow", "periodic"),
                         x3_symmetric=False)
        c["metric"] = ("minkowski", {})
        c["options"] = dict(method=0, kappa_a0=0.0, kappa_s=0.0)
        c["dt"] = 0.4 / N
    elif idx == 2:
        N = n[0]
        c["grid"] = dict(n=n, x0=(0.0, 0.0, 0.0), dx=(1.0 / N,) * 3, bc_lo=per, bc_hi=per, x3_symmetric=False)
        c["metric"] = ("minkowski", {})
        # kappa_a = kappa_a0 rho T^-3.5 with optical depth 1 per cell at rho = T = 1
        c["options"] = dict(method=2, kappa_a0=float(N), kappa_s=0.0, a_rad=1.0, Y_over_rho=1.5)
        c["dt"] = 0.5 / N
    elif idx == 3:
        N = n[0]
        c["grid"] = dict(n=n, x0=(-0.5,) * 3, dx=(1.0 / N,) * 3, bc_lo=per, bc_hi=per, x3_symmetric=False)
        c["metric"] = ("minkowski", {})
        c["options"] = dict(method=1, kappa_a0=0.0, kappa_s=10.0 * N, a_rad=1.0, Y_over_rho=1.5)
        c["dt"] = 0.5 / N
    elif idx in (4, 5):
        a = 0.9 if idx == 4 else 0.9375
        rh = 1.0 + math.sqrt(1.0 - a * a)
        x1lo, x1hi = math.log(0.9 * rh), math.log(50.0)
        band = max(2, n[1] // 24) if n[1] >= 8 else 0          # "zero the four cells closest to the poles" (L709)
        c["grid"] = dict(n=n, x0=(x1lo, 0.0, 0.0),
                         dx=((x1hi - x1lo) / n[0], 1.0 / n[1], 2.0 * math.pi / n[2]),
                         bc_lo=("outflow", "outflow", "periodic"), bc_hi=("outflow", "outflow", "periodic"),
                         zero_lo=(0, band, 0), zero_hi=(0, band, 0), x3_symmetric=True)
        c["metric"] = ("ks_mks", dict(a=a, hslope=0.3))
        c["options"] = dict(method=2, kappa_a0=10.0, kappa_s=20.0, a_rad=1.0, Y_over_rho=1.5)
        c["dt"] = None      # from the CFL bounds of whichever side runs it (L464 + angular bound, S14)
    elif idx == 6:
        # PAPER.md 4.6 (L559): A = 0.1, k = 2.0, 128 x 128, G2 angular grid; [0,1]^2 in (w, y); a beam enters through
        # the w-low boundary and must be straight once mapped back to x = w + A sin(k pi y)
        N = n[0]
        c["grid"] = dict(n=n, x0=(0.0, 0.0, 0.0), dx=(1.0 / N, 1.0 / n[1], 1.0 / N),
                         bc_lo=("fixed", "outflow", "periodic"), bc_hi=("outflow", "outflow", "periodic"),
                         x3_symmetric=True)
        c["metric"] = ("snake", dict(A=0.1, k=2.0))
        c["options"] = dict(method=0, kappa_a0=0.0, kappa_s=0.0)
        c["dt"] = 0.2 / N      # |n^w| <= 1 + A k pi = 1.63
    elif idx == 7:
        # PAPER.md 4.7 (L563-592): beams on the two circular photon orbits of a Kerr hole, a = +0.5, equatorial (r, phi) mesh of
        # 512 x 256, G3 = 642 directions with the pole along phi-hat, Boyer-Lindquist coordinates.  One x2 cell centred on the
        # equator (theta = pi/2 at x2 = 1/2) with OUTFLOW on both sides stands for the paper's 2-D mesh; r in [2, 5] is
        # log-spaced (outside the horizon, r_h = 1.87; the orbits sit at 2.347 and 3.532, Eq 53)
        a = 0.5
        x1lo, x1hi = math.log(2.0), math.log(5.0)
        c["grid"] = dict(n=n, x0=(x1lo, 0.5 - 0.01 * n[1], 0.0), dx=((x1hi - x1lo) / n[0], 0.02, 2.0 * math.pi / n[2]),
                         bc_lo=("outflow", "outflow", "periodic"), bc_hi=("outflow", "outflow", "periodic"), x3_symmetric=True)
        c["metric"] = ("bl_mks", dict(a=a, hslope=0.3))
        c["options"] = dict(method=0, kappa_a0=0.0, kappa_s=0.0)
        c["dt"] = None
        c["orbits"] = tuple(2.0 * (1.0 + math.cos(2.0 / 3.0 * math.acos(sg * a))) for sg in (-1.0, 1.0))   # Eq 53: co-, counter-rotating
    else:
        raise ValueError(idx)
    return c


def beam_direction(nhat):
    """Config 1: index of the grid direction nearest (1,1,0)/sqrt2 (lowest index on ties)."""
    d = np.asarray(nhat) @ (np.array([1.0, 1.0, 0.0]) / math.sqrt(2.0))
    return int(np.argmax(d))


def _smooth_field(rng, X, nmodes=8, kmax=3):
    """Sum of a few random low-wavenumber Fourier modes on the logical coordinates, values in about [-1, 1]."""
    f = np.zeros(X.shape[:-1])
    span = X.reshape(-1, 3).max(0) - X.reshape(-1, 3).min(0) + 1e-300
    for _ in range(nmodes):
        kv = rng.integers(-kmax, kmax + 1, size=3) * 2.0 * math.pi / span
        f += rng.uniform(0.3, 1.0) * np.sin(X @ kv + rng.uniform(0, 2 * math.pi))
    return f / math.sqrt(nmodes)


def fields(cfg, nhat, e_c=None):
    """Seeded initial data for `cfg`: dict(I0[N3,N2,N1,nd], rho, T, u4[4,N3,N2,N1] or None, ghosts={(dim,side): arr}).

    nhat[nd,3]: the caller's direction table.  e_c[E3,N2,N1,4,4] = e^mu_a at cell centres (E3 = 1 when the
    geometry is x3-symmetric), needed by configs 4-5 only to turn tetrad-frame velocities into u^mu.
    """
    idx = cfg["index"]
    n1, n2, n3 = cfg["grid"]["n"]
    nd = len(nhat)
    rng = np.random.default_rng(cfg["seed"])
    x0, dx = cfg["grid"]["x0"], cfg["grid"]["dx"]
    ax = [x0[a] + dx[a] * (np.arange(cfg["grid"]["n"][a]) + 0.5) for a in range(3)]
    X3, X2, X1 = np.meshgrid(ax[2], ax[1], ax[0], indexing="ij")
    shp = (n3, n2, n1)
    out = dict(u4=None, ghosts={})
    if idx in (1, 6):
        s_star = beam_direction(nhat)
        out["I0"] = np.zeros(shp + (nd,))
        out["rho"] = np.zeros(shp)
        out["T"] = np.ones(shp)
        g = np.zeros((2, n3 * n2, nd))                  # x-low ghosts: [layer][k*N2 + j][s]
        j0, j1 = n2 // 8, n2 // 4                       # rows [8, 16) at N = 64
        for k in range(n3):
            g[:, k * n2 + j0:k * n2 + j1, s_star] = 1.0
        out["ghosts"][(0, 0)] = g
        out["beam_dir"] = s_star
    elif idx == 7:
        # "initializing a small strip of cells along these radii, namely in the three cells closest to the circular orbit
        # radius" (L573): the co-rotating beam in the grid's pole direction +phi-hat (the first direction), the counter-
        # rotating one in -phi-hat (the last), each over an arc of phi an eighth of the circle long
        out["I0"] = np.zeros(shp + (nd,))
        out["rho"] = np.zeros(shp)
        out["T"] = np.ones(shp)
        r = np.exp(ax[0])
        arc = max(1, n3 // 8)
        out["strips"] = []
        for rph, s_dir, k0 in ((cfg["orbits"][0], 0, n3 // 16), (cfg["orbits"][1], nd - 1, n3 // 2)):
            ic = int(np.argmin(np.abs(r - rph)))
            i0, i1 = max(0, ic - 1), min(n1, ic + 2)
            out["I0"][k0:k0 + arc, :, i0:i1, s_dir] = 1.0
            out["strips"].append(dict(r=rph, s=s_dir, i=(i0, i1), k=(k0, k0 + arc)))
    elif idx == 2:
        out["I0"] = np.zeros(shp + (nd,))
        out["rho"] = np.ones(shp)
        out["T"] = rng.uniform(0.9, 1.1, size=shp)
    elif idx == 3:
        r2 = X1 ** 2 + X2 ** 2 + X3 ** 2
        E = np.exp(-r2 / (2 * 0.05 ** 2))
        xi = rng.uniform(-1.0, 1.0, size=shp + (nd,))
        out["I0"] = (E / (4 * math.pi))[..., None] * (1.0 + 1e-3 * xi)
        out["rho"] = np.ones(shp)
        out["T"] = np.ones(shp)
    else:
        h = cfg["metric"][1]["hslope"]
        r = np.exp(X1)
        th = math.pi * X2 + 0.5 * (1 - h) * np.sin(2 * math.pi * X2)
        R, z = r * np.sin(th), r * np.cos(th)
        d2 = (R - 12.0) ** 2 + z ** 2                    # torus: pressure maximum at 12, inner edge at 6
        rho = np.maximum(0.0, 1.0 - d2 / 36.0) ** 1.5
        rho *= 1.0 + 0.01 * rng.uniform(-1, 1, size=shp)
        T = (0.2 + 0.8 * np.sqrt(np.maximum(0.0, 1.0 - d2 / 36.0))) * (1.0 + 0.01 * rng.uniform(-1, 1, size=shp))
        X = np.stack([X1, X2, X3], -1)
        beta = np.zeros(shp + (3,))
        beta[..., 2] = 0.5 * np.minimum(1.0, np.sqrt(6.0 / r))        # Keplerian-like rotation in the tetrad frame
        if idx == 5:
            rho *= 1.0 + 0.3 * _smooth_field(rng, X)
            for i in range(3):
                beta[..., i] += 0.1 * _smooth_field(rng, X)
        b2 = np.minimum((beta ** 2).sum(-1), 0.64)
        gam = 1.0 / np.sqrt(1.0 - b2)
        uh = np.concatenate([gam[..., None], gam[..., None] * beta], -1)           # u^a-hat
        e = np.broadcast_to(np.asarray(e_c), shp + (4, 4))
        out["u4"] = np.ascontiguousarray(np.moveaxis(np.einsum("...ma,...a->...m", e, uh), -1, 0))
        thermal = (T ** 4 / (4 * math.pi)) * (rho >= 5e-4)
        out["I0"] = (thermal[..., None] * (1.0 + 0.01 * rng.uniform(-1, 1, size=shp + (nd,)))
                     + 1e-3 * (1.0 + 0.5 * rng.uniform(-1, 1, size=shp + (nd,))))
        out["rho"], out["T"] = rho, T
        if idx == 5:
            out["B"] = 1e-2 * np.stack([_smooth_field(rng, X) for _ in range(3)])   # generated, unused (GRMHD sector)
    return out


def novikov_thorne_T(r, a, alpha=0.05):
    """PAPER.md Eq 54-55 (L598-608) in code units: the Novikov-Thorne disk temperature up to the constant (4e7 K) (M / 3 Msun)^-1/4,
    T ~ alpha^-1/4 r^-3/8 A^-1/2 B^1/2 E^1/4, with A, B, E as printed (Eq 55a-c).  Input data of the radiating-disk workload."""
    r = np.asarray(r, dtype=np.float64)
    A = 1.0 + a * a / r ** 2 + 2.0 * a * a / r ** 3
    B = 1.0 + np.sqrt(a * a / r ** 3)
    E = 1.0 + 4.0 * a * a / r ** 2 - 4.0 * a * a / r ** 3 + 3.0 * a ** 4 / r ** 4
    return alpha ** -0.25 * r ** -0.375 * A ** -0.5 * B ** 0.5 * E ** 0.25


def radiating_disk(cfg, a_rad=1.0, r_in=6.0, r_out=10.0):
    """PAPER.md 4.8 (L594-617): "a strip of cells along the equator" between r = 6 and 10 that radiates isotropically in the
    tetrad frame with I = a_rad T^4 / (4 pi) (Eq 56), T from Eq 54.  For a Kerr-Schild config of this module (logical x1 = ln r,
    x2 = theta map) returns (j0, j1, i0, i1, I_disk[i1 - i0]): the rows next to the equator, the radial cells of the strip and
    the intensity each of them is held at (the caller re-imposes it after every step)."""
    g = cfg["grid"]
    n1, n2 = g["n"][0], g["n"][1]
    r = np.exp(g["x0"][0] + (np.arange(n1) + 0.5) * g["dx"][0])
    sel = np.where((r >= r_in) & (r <= r_out))[0]
    i0, i1 = int(sel[0]), int(sel[-1]) + 1
    j0, j1 = (n2 // 2 - 1, n2 // 2 + 1) if n2 % 2 == 0 else (n2 // 2, n2 // 2 + 1)
    T = novikov_thorne_T(r[i0:i1], cfg["metric"][1]["a"])
    return j0, j1, i0, i1, a_rad * T ** 4 / (4.0 * math.pi)
