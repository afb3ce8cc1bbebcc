/* ORACLE -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.
 *
 * Plain, slow, sequential-sum fp64 implementation of the per-step radiation update of PAPER.md
 * (arxiv 2508.15532, cuHARM radiation module), written from the paper step by step:
 *   O3  spatial transport      Eq 18 (L193), PLI L225, Eq 20 (L245), Eq 21-23 (L252-278), n_0 gate L280
 *   O4  angular flux           Eq 19 (L239-241), Eq 7-8 (L99-109)  [donor cell, or MAPR (L227)]
 *   O5  conserved update+mask  Eq 18
 *   O6  implicit source step   Eq 5 (L85), Eq 33, 35, 39-46 (L340-430), floor L468
 *   O7  moments / 4-force      Eq 13 (L141), Eq 36/48 (L361, L442)
 *   O8  predictor-corrector    L448-456
 * Readings of silent / garbled passages are those of SURVEY.md 8(c) (S4-S24), restated in DESIGN.md.
 *
 * Shares NO code with the CUDA path.  Geometry and angular tables come from oracle/geometry.py and
 * oracle/geodesic.py.  Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference
 * legs may call this.  Compile: gcc -O2 -ffp-contract=off -fopenmp -shared -fPIC.
 *
 * Layout: intensity I[cell][s], cell = (k*N2 + j)*N1 + i, s fastest, pitch = nd (no padding).
 * Geometry tables: index gc = (kg*N2 + j)*N1 + i with kg = (n3g == 1 ? 0 : k)  (x3-symmetric storage).
 * Parity status: every function is pinned (tests/test_oracle_*.py).  MAPR (ang_recon = 1) is a READING of a method the paper
 * only names (L227, S6): its stated properties -- second-order convergence, linear exactness, reduction to donor cell,
 * per-cell conservation, the arg-min and tie rules -- are pinned (tests/test_oracle_pins2.py, test_oracle_transport.py);
 * that its candidate planes are those of the cited Christov & Popov paper (not in the container) cannot be checked.
 */
#include <math.h>
#include <stdlib.h>
#include <string.h>

#define BC_PERIODIC 0
#define BC_OUTFLOW 1
#define BC_ZERO 2
#define BC_FIXED 3
#define BC_REFLECT 4  /* "symmetric" boundary (L709, S23): mirror cell, direction with the normal tetrad component flipped */

typedef struct {
    int n[3];
    int n3g;
    double dx[3];
    int bc_lo[3], bc_hi[3];
    int zero_lo[3], zero_hi[3]; /* bands of interior cells next to a boundary whose I is reset to 0 (L709) */
    int nd;
    const double *nhat, *w;
    const int *nnb, *nb;
    const double *dlam, *emid, *eun;
    const double *g_c, *e_c, *einv_c, *sqrtg_c, *omega_c;
    const double *g_f[3], *e_f[3], *sqrtg_f[3];
    int limiter;   /* 0 MC, 1 minmod, 2 van Leer (S7), 3 none (donor cell) */
    int ang_recon; /* 0 donor cell, 1 MAPR (S6) */
    int method;    /* 0 no source step; 1, 2, 3 = Methods 1-3 (L359-430) */
    double n0_floor, rho_floor, kappa_a0, kappa_s, a_rad, Y_over_rho, abar;
    const double *rho, *u4;     /* rho[Nc]; u4[4][Nc] coordinate-frame u^mu */
    const double *ghost[3][2];  /* BC_FIXED: [2 layers][face cells][nd], layer 0 next to the interior */
    const int *mirror[3];       /* BC_REFLECT: mirror[a][s] = the direction with n-hat^a flipped (a permutation) */
    int angflux_split;          /* 0: Eq 19 upwinded on the total normal velocity (S5); 1: term by term as printed (L239) */
    int source_literal;         /* 0: Eq 35 with the coefficients the temperature equation was built from (S19b, conservative);
                                   1: "the opacities must be updated and are therefore recalculated for the new value of T_+" (L432)
                                   taken literally for Methods 2 and 3: every opacity of Eq 35 at T_+ */
} orc_problem;

static const double FOURPI = 12.566370614359172953850573533118;

static long ncells(const orc_problem *P) { return (long)P->n[0] * P->n[1] * P->n[2]; }
static long cidx(const orc_problem *P, int i, int j, int k) { return ((long)k * P->n[1] + j) * P->n[0] + i; }
static long gidx(const orc_problem *P, int i, int j, int k) {
    return ((long)(P->n3g == 1 ? 0 : k) * P->n[1] + j) * P->n[0] + i;
}
/* lower face of cell (i,j,k) along dim a; face arrays have extent N_a + 1 along a */
static long fidx(const orc_problem *P, int a, int i, int j, int k) {
    int e0 = P->n[0] + (a == 0), e1 = P->n[1] + (a == 1);
    int kk = (P->n3g == 1) ? 0 : k;
    return ((long)kk * e1 + j) * e0 + i;
}

/* n^mu = e^mu_a nhat^a with nhat^a = (1, nhat)   (Eq 6) */
static void dir_coord(const double *e /*[4][4] e[mu][a]*/, const double *nh, double n[4]) {
    for (int mu = 0; mu < 4; ++mu)
        n[mu] = e[mu * 4 + 0] + e[mu * 4 + 1] * nh[0] + e[mu * 4 + 2] * nh[1] + e[mu * 4 + 3] * nh[2];
}
static double lower0(const double *g /*[4][4]*/, const double n[4]) {
    return g[0] * n[0] + g[1] * n[1] + g[2] * n[2] + g[3] * n[3];
}
/* centre n^0 and n_0 of (cell, s) */
static void centre_n0(const orc_problem *P, int i, int j, int k, int s, double *nup0, double *ndn0) {
    long g = gidx(P, i, j, k);
    double n[4];
    dir_coord(P->e_c + 16 * g, P->nhat + 3 * s, n);
    *nup0 = n[0];
    *ndn0 = lower0(P->g_c + 16 * g, n);
}

static double sgn(double x) { return (x > 0) - (x < 0); }
static double minmod3(double a, double b, double c) {
    if (a > 0 && b > 0 && c > 0) return fmin(a, fmin(b, c));
    if (a < 0 && b < 0 && c < 0) return fmax(a, fmax(b, c));
    return 0.0;
}
/* limited slope from the backward and forward differences (S7) */
static double slope(int limiter, double dm, double dp) {
    if (limiter == 0) return minmod3(2.0 * dm, 0.5 * (dm + dp), 2.0 * dp);
    if (limiter == 1) return (dm * dp > 0) ? (fabs(dm) < fabs(dp) ? dm : dp) : 0.0;
    if (limiter == 3) return 0.0;                                   /* donor cell (first order) */
    return (dm * dp > 0) ? 2.0 * dm * dp / (dm + dp) : 0.0;
}

/* resolve a possibly out-of-range index along dim a.  returns 1 and the interior index in *c if the
 * value lives in the interior array; 0 if it is zero; 2 if it is a fixed ghost (*c = layer); 3 if it is the
 * mirror image of interior cell *c (reflecting boundary: read it in the mirrored direction). */
static int resolve(const orc_problem *P, int a, int c, int *cout) {
    int N = P->n[a];
    if (c >= 0 && c < N) { *cout = c; return 1; }
    int bc = (c < 0) ? P->bc_lo[a] : P->bc_hi[a];
    if (bc == BC_PERIODIC) { *cout = ((c % N) + N) % N; return 1; }
    if (bc == BC_OUTFLOW) { *cout = (c < 0) ? 0 : N - 1; return 1; }
    if (bc == BC_ZERO) return 0;
    if (bc == BC_REFLECT) { *cout = (c < 0) ? (-1 - c) : (2 * N - 1 - c); return 3; }   /* mirror image cell */
    *cout = (c < 0) ? (-1 - c) : (c - N); /* ghost layer 0 or 1 */
    return 2;
}
/* intensity at (i,j,k,s) where exactly one of the indices may lie in the 2-deep ghost zone of dim a */
static double getI(const orc_problem *P, const double *I, int a, int idx[3], int s) {
    int c, r = resolve(P, a, idx[a], &c);
    if (r == 0) return 0.0;
    if (r == 1 || r == 3) {
        int q[3] = {idx[0], idx[1], idx[2]};
        q[a] = c;
        return I[cidx(P, q[0], q[1], q[2]) * P->nd + (r == 3 ? P->mirror[a][s] : s)];
    }
    /* fixed ghost: face-cell index runs over the two other dims, lower dim fastest */
    int b1 = (a == 0) ? 1 : 0, b2 = (a == 2) ? 1 : 2;
    long fc = (long)idx[b2] * P->n[b1] + idx[b1];
    long nface = (long)P->n[b1] * P->n[b2];
    int side = idx[a] < 0 ? 0 : 1;
    return P->ghost[a][side][((long)c * nface + fc) * P->nd + s];
}
/* fluid quantities in ghost zones: periodic wraps, reflecting mirrors, everything else copies the nearest interior cell */
static long fluid_cell(const orc_problem *P, int a, int idx[3]) {
    int q[3] = {idx[0], idx[1], idx[2]};
    int N = P->n[a], c = q[a];
    if (c < 0 || c >= N) {
        int bc = (c < 0) ? P->bc_lo[a] : P->bc_hi[a];
        if (bc == BC_REFLECT) q[a] = (c < 0) ? (-1 - c) : (2 * N - 1 - c);
        else q[a] = (bc == BC_PERIODIC) ? ((c % N) + N) % N : (c < 0 ? 0 : N - 1);
    }
    return cidx(P, q[0], q[1], q[2]);
}
/* +1, or -1 for a mirror-image cell behind a reflecting boundary of dim a (its normal velocity is reversed) */
static double mirror_sign(const orc_problem *P, int a, const int idx[3]) {
    int c = idx[a];
    if (c < 0) return P->bc_lo[a] == BC_REFLECT ? -1.0 : 1.0;
    if (c >= P->n[a]) return P->bc_hi[a] == BC_REFLECT ? -1.0 : 1.0;
    return 1.0;
}
/* fluid-frame total opacity alpha = rho (kappa_a + kappa_s), kappa_a = kappa_a0 rho T^-3.5 (S13, S21);
 * zero below the density floor (L468 (i)) */
static void opacities(const orc_problem *P, double rho, double T, double *alpha_a, double *alpha_s) {
    if (rho < P->rho_floor) { *alpha_a = 0; *alpha_s = 0; return; }
    *alpha_a = (P->kappa_a0 != 0.0) ? P->kappa_a0 * rho * rho * pow(T, -3.5) : 0.0;
    *alpha_s = P->kappa_s * rho;
}
static double alpha_tot(const orc_problem *P, const double *T, long c) {
    double aa, as;
    opacities(P, P->rho[c], T[c], &aa, &as);
    return aa + as;
}
static double vel(const orc_problem *P, long c, int a) { /* v^a = u^a / u^0 (S11) */
    long Nc = ncells(P);
    return P->u4[(1 + a) * Nc + c] / P->u4[c];
}
static int zero_banded(const orc_problem *P, int i, int j, int k) {
    int q[3] = {i, j, k};
    for (int a = 0; a < 3; ++a)
        if (q[a] < P->zero_lo[a] || q[a] >= P->n[a] - P->zero_hi[a]) return 1;
    return 0;
}

/* numerical flux through the UPPER face along dim a of cell idx (may be -1: the domain's lower boundary
 * face), direction s, NOT yet multiplied by sqrt(-g_f).  O3. */
static double face_flux(const orc_problem *P, const double *I, const double *T, int a, int idx[3], int s, double dt) {
    int L[3] = {idx[0], idx[1], idx[2]}, R[3] = {idx[0], idx[1], idx[2]};
    R[a] += 1;
    int q[3];
    double Im1, I0, I1, I2;
    memcpy(q, L, sizeof q); q[a] -= 1; Im1 = getI(P, I, a, q, s);
    I0 = getI(P, I, a, L, s);
    I1 = getI(P, I, a, R, s);
    memcpy(q, R, sizeof q); q[a] += 1; I2 = getI(P, I, a, q, s);
    double sL = slope(P->limiter, I0 - Im1, I1 - I0);
    double sR = slope(P->limiter, I1 - I0, I2 - I1);
    double IL = I0 + 0.5 * sL, IR = I1 - 0.5 * sR;       /* PLI states at the face (L225) */

    long f = fidx(P, a, R[0], R[1], R[2]);                /* lower face of the right cell */
    if (!(P->sqrtg_f[a][f] > 0.0)) return 0.0;            /* zero-area (polar-axis) face */
    double n[4];
    dir_coord(P->e_f[a] + 16 * f, P->nhat + 3 * s, n);
    double n0f = lower0(P->g_f[a] + 16 * f, n);
    double na = n[1 + a];

    /* no flux between cells where the sign of n_0 changes (L280); only between two cells of the mesh */
    int cl, cr, rl = resolve(P, a, L[a], &cl), rr = resolve(P, a, R[a], &cr);
    if (rl == 1 && rr == 1) {   /* an OUTFLOW ghost is a copy of its own neighbour: same cell, same sign */
        int ql[3] = {L[0], L[1], L[2]}, qr[3] = {R[0], R[1], R[2]};
        ql[a] = cl; qr[a] = cr;
        double u, d0l, d0r;
        centre_n0(P, ql[0], ql[1], ql[2], s, &u, &d0l);
        centre_n0(P, qr[0], qr[1], qr[2], s, &u, &d0r);
        if (sgn(d0l) != sgn(d0r)) return 0.0;
    }

    long fl = fluid_cell(P, a, L), fr = fluid_cell(P, a, R);
    double tau = P->abar * 0.5 * (alpha_tot(P, T, fl) + alpha_tot(P, T, fr)) * dt;   /* L262, S13 */
    if (tau == 0.0)                                                                  /* S12: vacuum face */
        return n0f * na * (na > 0 ? IL : IR);                                        /* Eq 20 */

    double ftau = sqrt(-expm1(-tau * tau) / (tau * tau));   /* Eq 21-22 with exp(-tau^2) in all branches (S8) */
    double etau = exp(-tau);
    /* PLI-reconstructed fluid 3-velocity at the face (L276) */
    int qq[3];
    memcpy(qq, L, sizeof qq); qq[a] -= 1; long fm = fluid_cell(P, a, qq); double sm = mirror_sign(P, a, qq);
    memcpy(qq, R, sizeof qq); qq[a] += 1; long fp = fluid_cell(P, a, qq); double sp = mirror_sign(P, a, qq);
    double vm = sm * vel(P, fm, a), v0 = mirror_sign(P, a, L) * vel(P, fl, a), v1 = mirror_sign(P, a, R) * vel(P, fr, a),
           v2 = sp * vel(P, fp, a);
    double vL = v0 + 0.5 * slope(P->limiter, v0 - vm, v1 - v0);
    double vR = v1 - 0.5 * slope(P->limiter, v1 - v0, v2 - v1);
    double adv;
    if (vL > 0 && vR > 0) adv = vL * IL;                   /* upwind (S11) */
    else if (vL < 0 && vR < 0) adv = vR * IR;
    else adv = vL * IL + vR * IR;                          /* one-sided speeds (L276) */
    /* Eq 23 with S8-S10: S+/(S+ - S-) = 1/2, S+S-/(S+ - S-) = -|n^a| f(tau)/2, all times n_0,
     * advected quantity n^0 v^a I */
    return n0f * (0.5 * na * (IL + IR) * etau - 0.5 * fabs(na) * ftau * (I1 - I0) + (1.0 - etau) * n[0] * adv);
}

/* D_x of O3 for one (cell, s) */
static double div_x(const orc_problem *P, const double *I, const double *T, int i, int j, int k, int s, double dt) {
    double D = 0.0;
    long gc = gidx(P, i, j, k);
    for (int a = 0; a < 3; ++a) {
        int up[3] = {i, j, k}, lo[3] = {i, j, k};
        lo[a] -= 1;
        double Fp = face_flux(P, I, T, a, up, s, dt), Fm = face_flux(P, I, T, a, lo, s, dt);
        up[a] += 1;
        long fp = fidx(P, a, up[0], up[1], up[2]), fm = fidx(P, a, i, j, k);
        D += (P->sqrtg_f[a][fp] * Fp - P->sqrtg_f[a][fm] * Fm) / (P->sqrtg_c[gc] * P->dx[a]);
    }
    return D;
}

/* normal angular velocity V_e = a(m_e).u_e = -u_i omega^i_{cd} m^c m^d, m^c = (1, m_e) (O4, S4) and
 * n_0 at the edge centre, for edge e of direction s in the cell with geometry index gc */
static void edge_coeff2(const orc_problem *P, long gc, int s, int e, double *V, double *n0e, double Vsplit[2]);
static void edge_coeff(const orc_problem *P, long gc, int s, int e, double *V, double *n0e) {
    double Vs[2];
    edge_coeff2(P, gc, s, e, V, n0e, Vs);
}
/* the same, and the two terms of Eq 19 as printed (L239): the normal velocity split along the unit vectors of the tetrad-frame
 * angles, V_zeta = (a.e_zeta)(u.e_zeta), V_psi = (a.e_psi)(u.e_psi), n-hat = (sin zeta cos psi, sin zeta sin psi, cos zeta);
 * V = V_zeta + V_psi since u is tangent to the sphere at the edge centre */
static void edge_coeff2(const orc_problem *P, long gc, int s, int e, double *V, double *n0e, double Vsplit[2]) {
    const double *m3 = P->emid + 3 * (6 * s + e), *u3 = P->eun + 3 * (6 * s + e);
    double m[4] = {1.0, m3[0], m3[1], m3[2]};
    const double *om = P->omega_c + 64 * gc;
    double v = 0.0, a3[3];
    for (int ii = 1; ii < 4; ++ii) {
        double q = 0.0;
        for (int c = 0; c < 4; ++c)
            for (int d = 0; d < 4; ++d) q += om[(ii * 4 + c) * 4 + d] * m[c] * m[d];
        a3[ii - 1] = -q;              /* a^i up to its component along m, which no tangent vector sees */
        v -= u3[ii - 1] * q;
    }
    {
        double sz = sqrt(m3[0] * m3[0] + m3[1] * m3[1]);
        double cp = sz > 0 ? m3[0] / sz : 1.0, sp = sz > 0 ? m3[1] / sz : 0.0;
        double ez[3] = {m3[2] * cp, m3[2] * sp, -sz}, ep[3] = {-sp, cp, 0.0};
        Vsplit[0] = (a3[0] * ez[0] + a3[1] * ez[1] + a3[2] * ez[2]) * (u3[0] * ez[0] + u3[1] * ez[1] + u3[2] * ez[2]);
        Vsplit[1] = (a3[0] * ep[0] + a3[1] * ep[1] + a3[2] * ep[2]) * (u3[0] * ep[0] + u3[1] * ep[1] + u3[2] * ep[2]);
    }
    *V = v;
    double n[4];
    dir_coord(P->e_c + 16 * gc, m3, n);
    *n0e = lower0(P->g_c + 16 * gc, n);
}

/* MAPR gradient of cell s in its tangent plane (O4', S6); returns gradient as a 3-vector tangent at nhat_s */
static void mapr_gradient(const orc_problem *P, const double *Ic /*[nd] one cell*/, int s, double grad[3]) {
    const double *c0 = P->nhat + 3 * s;
    int nn = P->nnb[s];
    double xi[6][3], dI[6];
    for (int e = 0; e < nn; ++e) {
        int t = P->nb[6 * s + e];
        const double *ct = P->nhat + 3 * t;
        double dot = c0[0] * ct[0] + c0[1] * ct[1] + c0[2] * ct[2];
        double p[3] = {ct[0] - dot * c0[0], ct[1] - dot * c0[1], ct[2] - dot * c0[2]};
        double pn = sqrt(p[0] * p[0] + p[1] * p[1] + p[2] * p[2]);
        double ang = atan2(pn, dot);
        for (int x = 0; x < 3; ++x) xi[e][x] = ang * p[x] / pn;     /* log map */
        dI[e] = Ic[t] - Ic[s];
    }
    double best = INFINITY;
    grad[0] = grad[1] = grad[2] = 0.0;
    for (int e = 0; e < nn; ++e) {
        int e2 = (e + 1) % nn;
        /* plane through (0,0), (xi_e, dI_e), (xi_e2, dI_e2): gradient G in span(xi_e, xi_e2) with G.xi = dI */
        double a11 = 0, a12 = 0, a22 = 0;
        for (int x = 0; x < 3; ++x) { a11 += xi[e][x] * xi[e][x]; a12 += xi[e][x] * xi[e2][x]; a22 += xi[e2][x] * xi[e2][x]; }
        double det = a11 * a22 - a12 * a12;
        double c1 = (dI[e] * a22 - dI[e2] * a12) / det, c2 = (dI[e2] * a11 - dI[e] * a12) / det;
        double G[3], nrm = 0;
        for (int x = 0; x < 3; ++x) { G[x] = c1 * xi[e][x] + c2 * xi[e2][x]; nrm += G[x] * G[x]; }
        /* ties -> lowest e, where a tie is agreement to round-off: equal (e.g. masked, zero) neighbours make
         * consecutive candidates tie structurally, and the winner must not depend on the last bit (S6) */
        if (nrm < best * (1.0 - 1e-12)) { best = nrm; grad[0] = G[0]; grad[1] = G[1]; grad[2] = G[2]; }
    }
}
/* test hook: the MAPR gradient of cell s for one cell's intensities */
void orc_mapr_gradient(const orc_problem *P, const double *Ic, int s, double grad[3]) { mapr_gradient(P, Ic, s, grad); }

static double mapr_edge_value(const orc_problem *P, const double *Ic, int s, int e, const double grad[3]) {
    const double *c0 = P->nhat + 3 * s, *m = P->emid + 3 * (6 * s + e);
    double dot = c0[0] * m[0] + c0[1] * m[1] + c0[2] * m[2];
    double p[3] = {m[0] - dot * c0[0], m[1] - dot * c0[1], m[2] - dot * c0[2]};
    double pn = sqrt(p[0] * p[0] + p[1] * p[1] + p[2] * p[2]);
    double ang = atan2(pn, dot);
    return Ic[s] + ang * (grad[0] * p[0] + grad[1] * p[1] + grad[2] * p[2]) / pn;
}

/* D_Omega of O4 for one (cell, s).  Ic = the cell's nd intensities. */
static double div_omega(const orc_problem *P, const double *Ic, int i, int j, int k, int s) {
    long gc = gidx(P, i, j, k);
    double sum = 0.0, up0, n0s;
    centre_n0(P, i, j, k, s, &up0, &n0s);
    double gs[3];
    if (P->ang_recon == 1) mapr_gradient(P, Ic, s, gs);
    for (int e = 0; e < P->nnb[s]; ++e) {
        int t = P->nb[6 * s + e];
        double V, n0e, n0t, Vs[2];
        edge_coeff2(P, gc, s, e, &V, &n0e, Vs);
        centre_n0(P, i, j, k, t, &up0, &n0t);
        if (sgn(n0s) != sgn(n0t)) continue;               /* L280 applied to angular neighbours */
        double IL = Ic[s], IR = Ic[t];                    /* donor cell (L227) */
        if (P->ang_recon == 1) {
            double gt[3];
            int et = -1;
            for (int q = 0; q < P->nnb[t]; ++q) if (P->nb[6 * t + q] == s) et = q;
            mapr_gradient(P, Ic, t, gt);
            IL = mapr_edge_value(P, Ic, s, e, gs);
            IR = mapr_edge_value(P, Ic, t, et, gt);
        }
        double F = n0e * V * (V > 0 ? IL : IR);           /* Eq 19 upwinded on the total normal velocity (S5) */
        if (P->angflux_split)                             /* ... or each of its two terms on its own (L239, as printed) */
            F = n0e * (Vs[0] * (Vs[0] > 0 ? IL : IR) + Vs[1] * (Vs[1] > 0 ? IL : IR));
        sum += P->dlam[6 * s + e] * F;
    }
    return sum / P->w[s];
}

static int masked(const orc_problem *P, double n0) { return n0 > -P->n0_floor; }   /* S14 (ii) */

/* rt_transport: I_out = (n^0 n_0 I_base - dt D_x[I_in]) / (n^0 n_0), then mask + zero band.  O3 + O5. */
void orc_transport(const orc_problem *P, const double *I_in, const double *T, const double *I_base, double *I_out, double dt) {
    int nd = P->nd;
#pragma omp parallel for collapse(2) schedule(static)
    for (int k = 0; k < P->n[2]; ++k)
        for (int j = 0; j < P->n[1]; ++j)
            for (int i = 0; i < P->n[0]; ++i) {
                long c = cidx(P, i, j, k);
                int zb = zero_banded(P, i, j, k);
                for (int s = 0; s < nd; ++s) {
                    double nu0, nd0;
                    centre_n0(P, i, j, k, s, &nu0, &nd0);
                    if (zb || masked(P, nd0)) { I_out[c * nd + s] = 0.0; continue; }
                    double D = div_x(P, I_in, T, i, j, k, s, dt);
                    double U = nu0 * nd0 * I_base[c * nd + s] - dt * D;
                    I_out[c * nd + s] = U / (nu0 * nd0);
                }
            }
}

/* rt_angular_flux: I_inout -= dt D_Omega[I_in] / (n^0 n_0), then mask + zero band.  O4 + O5. */
void orc_angular(const orc_problem *P, const double *I_in, double *I_inout, double dt) {
    int nd = P->nd;
#pragma omp parallel for collapse(2) schedule(static)
    for (int k = 0; k < P->n[2]; ++k)
        for (int j = 0; j < P->n[1]; ++j)
            for (int i = 0; i < P->n[0]; ++i) {
                long c = cidx(P, i, j, k);
                int zb = zero_banded(P, i, j, k);
                for (int s = 0; s < nd; ++s) {
                    double nu0, nd0;
                    centre_n0(P, i, j, k, s, &nu0, &nd0);
                    if (zb || masked(P, nd0)) { I_inout[c * nd + s] = 0.0; continue; }
                    double D = div_omega(P, I_in + c * nd, i, j, k, s);
                    I_inout[c * nd + s] -= dt * D / (nu0 * nd0);
                }
            }
}

/* residual of the temperature equation, oriented so that f(0+) < 0 < f(W/Y), and its derivative.
 * Method 1: Eq 42; Method 2: Eq 43; Method 3: minus Eq 46 (S19: A' = alpha_- dt A). */
typedef struct { int method; double a4, b1, c0;            /* methods 1, 2: a4*g(T) + b1*T + c0 */
                 double k45, k4, k35, k1, k0; } teq;       /* method 3: coefficients of Eq 46 */
static void teq_eval(const teq *q, double T, double *f, double *df) {
    if (q->method == 1) { *f = q->a4 * T * T * T * T + q->b1 * T + q->c0; *df = 4.0 * q->a4 * T * T * T + q->b1; }
    else if (q->method == 2) { double r = sqrt(T); *f = q->a4 * r + q->b1 * T + q->c0; *df = 0.5 * q->a4 / r + q->b1; }
    else {
        double r = sqrt(T), T3 = T * T * T, T35 = T3 * r, T4 = T3 * T, T45 = T4 * r;
        double F = q->k45 * T45 + q->k4 * T4 + q->k35 * T35 + q->k1 * T + q->k0;
        double dF = 4.5 * q->k45 * T35 + 4.0 * q->k4 * T3 + 3.5 * q->k35 * T3 / r + q->k1;
        *f = -F; *df = -dF;
    }
}
/* Newton-Raphson (L399) from the guess T_-, safeguarded by the bracket (0, W/Y] (S20): an iterate outside the
 * CLOSED current bracket [lo, hi] (or not positive) is replaced by the midpoint.  Closed, because for pure scattering
 * the root is T_- itself, i.e. the first iterate lands on a bracket end; an open test would reject it and bisect ~45
 * times towards the same number.  returns 0 on success, 1 if there is no positive root (T left unchanged). */
static int solve_T(const teq *q, double Tminus, double Thi, double *Tplus) {
    double lo = 0.0, hi = Thi, f, df;
    if (!(Thi > 0.0)) return 1;
    teq_eval(q, hi, &f, &df);
    if (!(f >= 0.0)) return 1;
    if (q->method != 3 && !(q->c0 < 0.0)) return 1;       /* f(0) >= 0: no positive root (L401) */
    double T = (Tminus > lo && Tminus < hi) ? Tminus : 0.5 * (lo + hi);
    for (int it = 0; it < 100; ++it) {
        teq_eval(q, T, &f, &df);
        if (f < 0) lo = T; else hi = T;
        double Tn = T - f / df;
        if (!(Tn > 0.0 && Tn >= lo && Tn <= hi)) Tn = 0.5 * (lo + hi);   /* closed bracket: a root AT an end (T+ = T-) is kept */
        double d = Tn - T;
        T = Tn;
        if (fabs(d) <= 1e-14 * T) break;
    }
    *Tplus = T;
    return 0;
}

/* rt_source_implicit: O6, in place on (I, T).  returns the number of cells whose solve failed. */
int orc_source(const orc_problem *P, double *I, double *T, double dt) {
    int nd = P->nd, nfail = 0;
    long Nc = ncells(P);
    if (P->method == 0) return 0;
#pragma omp parallel for collapse(2) schedule(static) reduction(+ : nfail)
    for (int k = 0; k < P->n[2]; ++k)
        for (int j = 0; j < P->n[1]; ++j)
            for (int i = 0; i < P->n[0]; ++i) {
                long c = cidx(P, i, j, k), gc = gidx(P, i, j, k);
                double rho = P->rho[c], Tm = T[c], aa, as;
                opacities(P, rho, Tm, &aa, &as);
                double alpha = aa + as;
                if (alpha == 0.0) continue;                                     /* L468 (i) / nothing to do */
                /* u^a-hat = e^a_mu u^mu (L87) */
                double uh[4];
                for (int a = 0; a < 4; ++a) {
                    uh[a] = 0.0;
                    for (int mu = 0; mu < 4; ++mu) uh[a] += P->einv_c[16 * gc + 4 * a + mu] * P->u4[mu * Nc + c];
                }
                double E = 0, A1 = 0, A2 = 0;
                double *Ic = I + c * nd;
                for (int s = 0; s < nd; ++s) {
                    double nu0, nd0;
                    centre_n0(P, i, j, k, s, &nu0, &nd0);
                    if (masked(P, nd0)) continue;
                    const double *nh = P->nhat + 3 * s;
                    double nbar = uh[0] - (uh[1] * nh[0] + uh[2] * nh[1] + uh[3] * nh[2]);   /* Eq 5, first row */
                    double Ibar = nbar * nbar * nbar * nbar * Ic[s];                          /* S17 */
                    double dOm = P->w[s] / (nbar * nbar);
                    double d = nu0 + nbar * alpha * dt;
                    E += Ibar * dOm;                                                          /* Eq 33 */
                    A1 += nu0 / d * Ibar * dOm;                                               /* Eq 41a */
                    A2 += nbar / d * dOm;                                                     /* Eq 41b */
                }
                A2 *= dt / FOURPI;
                double Y = P->Y_over_rho * rho, W = E + Y * Tm;
                double Nbar = P->kappa_a0 * rho * rho;      /* alpha^a = Nbar T^-3.5 (L403, L430) */
                teq q;
                q.method = P->method;
                if (P->method == 1) { q.a4 = A2 * aa * P->a_rad; }
                else if (P->method == 2) { q.a4 = A2 * Nbar * P->a_rad; }
                q.b1 = Y * (1.0 - A2 * as);
                q.c0 = A1 - Y * (1.0 - A2 * as) * Tm - (1.0 - A2 * as) * E;
                if (P->method == 3) {
                    double A1p = alpha * dt * A1, A2p = alpha * dt * A2;                     /* S19 */
                    q.k45 = Y * as * (A2p - dt);
                    q.k4 = -A2p * Nbar * P->a_rad;
                    q.k35 = -(A2p * as * W + A1p - W * as * dt);
                    q.k1 = -Y * Nbar * dt;
                    q.k0 = W * Nbar * dt;
                }
                double Tp;
                if (solve_T(&q, Tm, W / Y, &Tp)) { nfail += 1; continue; }
                double Ep = W - Y * Tp;                                                       /* Eq 39 */
                double emis, scale = 1.0;
                if (P->method == 1) emis = aa * P->a_rad * Tp * Tp * Tp * Tp;
                else emis = Nbar * P->a_rad * sqrt(Tp);                                      /* alpha_P(T+) a T+^4 */
                if (P->method == 3) scale = alpha / (as + Nbar * pow(Tp, -3.5));             /* alpha_- / alpha_+ */
                double S = emis + as * Ep;
                double alpha_upd = alpha;                                                     /* the opacity inside d_s of Eq 35 */
                if (P->source_literal && P->method != 1) {                                   /* L432, literal (S19b) */
                    alpha_upd = as + Nbar * pow(Tp, -3.5);
                    scale = 1.0;
                }
                for (int s = 0; s < nd; ++s) {
                    double nu0, nd0;
                    centre_n0(P, i, j, k, s, &nu0, &nd0);
                    if (masked(P, nd0)) continue;
                    const double *nh = P->nhat + 3 * s;
                    double nbar = uh[0] - (uh[1] * nh[0] + uh[2] * nh[1] + uh[3] * nh[2]);
                    double n4 = nbar * nbar * nbar * nbar;
                    double d = nu0 + nbar * alpha_upd * dt;
                    double Ibar = n4 * Ic[s];
                    double Ip = scale * (nu0 / d * Ibar + nbar * dt / (FOURPI * d) * S);     /* Eq 35 */
                    Ic[s] = Ip / n4;                                                          /* L432 */
                }
                T[c] = Tp;
            }
    return nfail;
}

/* rt_moments: R^mu_nu = sum_s w_s I_s n^mu n_nu, R[16][Nc], c = 4 mu + nu.  O7 (Eq 13, S24). */
void orc_moments(const orc_problem *P, const double *I, double *R) {
    int nd = P->nd;
    long Nc = ncells(P);
#pragma omp parallel for collapse(2) schedule(static)
    for (int k = 0; k < P->n[2]; ++k)
        for (int j = 0; j < P->n[1]; ++j)
            for (int i = 0; i < P->n[0]; ++i) {
                long c = cidx(P, i, j, k), gc = gidx(P, i, j, k);
                double acc[16] = {0};
                for (int s = 0; s < nd; ++s) {
                    double n[4], nl[4];
                    dir_coord(P->e_c + 16 * gc, P->nhat + 3 * s, n);
                    for (int nu = 0; nu < 4; ++nu) {
                        nl[nu] = 0.0;
                        for (int l = 0; l < 4; ++l) nl[nu] += P->g_c[16 * gc + 4 * nu + l] * n[l];
                    }
                    double wI = P->w[s] * I[c * nd + s];
                    for (int mu = 0; mu < 4; ++mu)
                        for (int nu = 0; nu < 4; ++nu) acc[4 * mu + nu] += wI * n[mu] * nl[nu];
                }
                for (int q = 0; q < 16; ++q) R[q * Nc + c] = acc[q];
            }
}

/* one stage of O8: I* = O5(I_base; fluxes of I_flux with opacities at T_flux; delta), written to I_out
 * (I_out may alias I_base); T_out starts as a copy of T_base; then optional moments of I*, then O6. */
static int stage(const orc_problem *P, const double *I_flux, const double *T_flux, const double *I_base,
                 const double *T_base, double *I_out, double *T_out, double delta, double *R_before) {
    long Nc = ncells(P);
    orc_transport(P, I_flux, T_flux, I_base, I_out, delta);
    orc_angular(P, I_flux, I_out, delta);
    if (T_out != T_base) memcpy(T_out, T_base, sizeof(double) * Nc);
    if (R_before) orc_moments(P, I_out, R_before);
    return orc_source(P, I_out, T_out, delta);
}

/* rt_step: O8 (L448-456, S22).  I, T in place; R_out[16][Nc]; G_out[4][Nc] (may be NULL);
 * Ih, Th, Rb = caller-provided scratch (nd*Nc, Nc, 16*Nc).  returns failed-cell count (both stages). */
int orc_step(const orc_problem *P, double *I, double *T, double *R_out, double *G_out, double dt,
             double *Ih, double *Th, double *Rb) {
    long Nc = ncells(P);
    int nf = stage(P, I, T, I, T, Ih, Th, 0.5 * dt, NULL);            /* predictor: dt/2 */
    nf += stage(P, Ih, Th, I, T, I, T, dt, Rb);                       /* corrector: fluxes from the half step */
    orc_moments(P, I, R_out);
    if (G_out)
        for (int nu = 0; nu < 4; ++nu)
            for (long c = 0; c < Nc; ++c) G_out[nu * Nc + c] = -(R_out[nu * Nc + c] - Rb[nu * Nc + c]) / dt;   /* Eq 36/48 */
    return nf;
}

/* time-step bound: half the light-crossing time of the smallest cell (L464) and the angular outflow-rate
 * bound of S14.  out[0] = spatial bound, out[1] = angular bound (INFINITY when omega = 0). */
void orc_cfl(const orc_problem *P, double out[2]) {
    double dts = INFINITY, dta = INFINITY;
    int kmax = (P->n3g == 1) ? 1 : P->n[2];
    for (int k = 0; k < kmax; ++k)
        for (int j = 0; j < P->n[1]; ++j)
            for (int i = 0; i < P->n[0]; ++i) {
                if (zero_banded(P, i, j, P->n3g == 1 ? P->zero_lo[2] : k)) continue;
                long gc = gidx(P, i, j, k);
                for (int s = 0; s < P->nd; ++s) {
                    double n[4];
                    dir_coord(P->e_c + 16 * gc, P->nhat + 3 * s, n);
                    double n0 = lower0(P->g_c + 16 * gc, n);
                    if (masked(P, n0)) continue;
                    for (int a = 0; a < 3; ++a)
                        if (n[1 + a] != 0.0) dts = fmin(dts, 0.5 * P->dx[a] * n[0] / fabs(n[1 + a]));
                    double rate = 0.0;
                    for (int e = 0; e < P->nnb[s]; ++e) {
                        double V, n0e, Vs[2];
                        edge_coeff2(P, gc, s, e, &V, &n0e, Vs);
                        if (P->angflux_split) V = fmax(Vs[0], 0.0) + fmax(Vs[1], 0.0);   /* what leaves through this edge */
                        if (V > 0) rate += V * fabs(n0e) * P->dlam[6 * s + e] / P->w[s];
                    }
                    if (rate > 0) dta = fmin(dta, 0.5 * fabs(n[0] * n0) / rate);
                }
            }
    out[0] = dts;
    out[1] = dta;
}
