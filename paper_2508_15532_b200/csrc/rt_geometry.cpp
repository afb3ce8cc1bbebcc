// Metric, tetrad and Ricci rotation coefficients for librt_b200 (host, init-time only).
//
// PAPER.md 2.1.1 (Eq 1-4): orthonormal tetrad with e_0 normal to x^0 = const (Eq 4); Eq 8 (L107-109):
// omega^a_{cd} = e^a_beta e^mu_c nabla_mu e^beta_d by finite differences plus the connection; Appendix A.2
// (L814-850): Kerr-Schild tetrad of Takahashi (2008).  The KS tetrad is built here by Gram-Schmidt of the
// coordinate basis in the order d_3, d_2, d_1 with the 3-metric gamma_ij = g_ij (the locally non-rotating frame:
// e_phi along d_phi, e_theta along d_theta, e_r the remaining orthogonal direction), which is what A3-A4 are with
// reading S25 of DESIGN.md (alpha = lapse, gamma^{ij} = inverse 3-metric).
#include <cmath>
#include <cstring>

#include "rt_internal.h"

namespace rt {
namespace {

const double PI = 3.14159265358979323846;
const double FD_H = 5e-4;

void zero44(double m[4][4]) { std::memset(m, 0, sizeof(double) * 16); }

bool invert44(const double a[4][4], double inv[4][4], double *det_out) {
    double m[4][8];
    for (int i = 0; i < 4; ++i)
        for (int j = 0; j < 4; ++j) { m[i][j] = a[i][j]; m[i][4 + j] = (i == j); }
    double det = 1.0;
    for (int c = 0; c < 4; ++c) {
        int p = c;
        for (int r = c + 1; r < 4; ++r)
            if (std::fabs(m[r][c]) > std::fabs(m[p][c])) p = r;
        if (m[p][c] == 0.0) { if (det_out) *det_out = 0.0; return false; }
        if (p != c) { for (int j = 0; j < 8; ++j) std::swap(m[p][j], m[c][j]); det = -det; }
        det *= m[c][c];
        double piv = 1.0 / m[c][c];
        for (int j = 0; j < 8; ++j) m[c][j] *= piv;
        for (int r = 0; r < 4; ++r)
            if (r != c) {
                double f = m[r][c];
                if (f != 0.0) for (int j = 0; j < 8; ++j) m[r][j] -= f * m[c][j];
            }
    }
    for (int i = 0; i < 4; ++i) for (int j = 0; j < 4; ++j) inv[i][j] = m[i][4 + j];
    if (det_out) *det_out = det;
    return true;
}

// d x / d y at fixed w in snake coordinates (L806)
double snake_delta(const rt_metric &mt, double y) { return mt.snake_A * mt.snake_k * PI * std::cos(mt.snake_k * PI * y); }

// covariant metric in logical coordinates
void metric_at(const rt_metric &mt, const double x[3], double g[4][4]) {
    zero44(g);
    if (mt.kind == RT_USER) { mt.g_fn(x, g, mt.user); return; }
    if (mt.kind != RT_KS_MKS && mt.kind != RT_BL_MKS) {
        g[0][0] = -1; g[1][1] = g[2][2] = g[3][3] = 1;
        if (mt.kind == RT_SNAKE) {   // x = w + A sin(k pi y):  dx = dw + delta dy  =>  ds^2 = -dt^2 + (dw + delta dy)^2 + dy^2 + dz^2
            const double dl = snake_delta(mt, x[1]);
            g[1][2] = g[2][1] = dl;
            g[2][2] += dl * dl;
        }
        return;
    }
    const double a = mt.a, h = mt.hslope;
    const double r = std::exp(x[0]);
    const double th = PI * x[1] + 0.5 * (1.0 - h) * std::sin(2 * PI * x[1]);
    const double J1 = r, J2 = PI + PI * (1.0 - h) * std::cos(2 * PI * x[1]);
    const double st = std::sin(th), ct = std::cos(th), s2 = st * st;
    const double Sig = r * r + a * a * ct * ct, H = 2.0 * r / Sig;
    if (mt.kind == RT_BL_MKS) {   // Boyer-Lindquist (section 4.7); the Gram-Schmidt below gives the zero-angular-momentum frame
        const double Del = r * r - 2.0 * r + a * a;
        g[0][0] = -1.0 + H;
        g[0][3] = g[3][0] = -a * H * s2;
        g[1][1] = Sig / Del * J1 * J1;
        g[2][2] = Sig * J2 * J2;
        g[3][3] = s2 * (r * r + a * a + a * a * H * s2);
        return;
    }
    g[0][0] = -1.0 + H;
    g[0][1] = g[1][0] = H * J1;
    g[0][3] = g[3][0] = -a * H * s2;
    g[1][1] = (1.0 + H) * J1 * J1;
    g[1][3] = g[3][1] = -a * s2 * (1.0 + H) * J1;
    g[2][2] = Sig * J2 * J2;
    g[3][3] = s2 * (Sig + a * a * s2 * (1.0 + H));
}

double gdot(const double g[4][4], const double u[4], const double v[4]) {
    double s = 0;
    for (int i = 1; i < 4; ++i) for (int j = 1; j < 4; ++j) s += g[i][j] * u[i] * v[j];
    return s;
}

}  // namespace

void eval_point(const rt_metric &mt, const double x[3], PointGeom &o) {
    metric_at(mt, x, o.g);
    zero44(o.e);
    zero44(o.einv);
    o.dead = false;
    double ginv[4][4], det;
    bool ok = invert44(o.g, ginv, &det);
    o.sqrtg = (ok && det < 0) ? std::sqrt(-det) : 0.0;
    if (mt.kind == RT_MINKOWSKI_CART) {
        for (int i = 0; i < 4; ++i) o.e[i][i] = o.einv[i][i] = 1.0;
        return;
    }
    if (mt.kind == RT_MINK_CYL_TETRAD) {  // flat space, rotating tetrad e_1 = R-hat, e_2 = phi-hat, e_3 = z-hat
        const double R = std::sqrt(x[0] * x[0] + x[1] * x[1]);
        o.e[0][0] = 1; o.e[3][3] = 1;
        o.e[1][1] = x[0] / R; o.e[2][1] = x[1] / R;
        o.e[1][2] = -x[1] / R; o.e[2][2] = x[0] / R;
        for (int a = 0; a < 4; ++a) for (int mu = 0; mu < 4; ++mu) o.einv[a][mu] = o.e[mu][a];
        return;
    }
    if (mt.kind == RT_SNAKE) {   // the Cartesian frame written in (w, y, z): d_x = d_w, d_y|_x = d_y - delta d_w
        const double dl = snake_delta(mt, x[1]);
        for (int i = 0; i < 4; ++i) o.e[i][i] = o.einv[i][i] = 1.0;
        o.e[1][2] = -dl;      // e^w_{y-hat}
        o.einv[1][2] = dl;    // e^{x-hat}_y:  dx = dw + delta dy
        return;
    }
    if (!ok || !(o.sqrtg > 1e-300) || !(o.g[3][3] > 0)) {  // polar axis: gamma_phiphi = 0
        o.dead = true;
        o.sqrtg = 0.0;
        return;
    }
    if (mt.kind == RT_USER && mt.e_fn) {
        mt.e_fn(x, o.e, mt.user);   // the caller's tetrad
    } else {
        // e_0 from Eq 4
        const double lapse_inv = std::sqrt(-ginv[0][0]);
        for (int mu = 0; mu < 4; ++mu) o.e[mu][0] = -ginv[0][mu] / lapse_inv;
        // Gram-Schmidt of d_3, d_2, d_1 with the spatial metric
        double leg[4][4] = {{0}};  // leg[a][mu]
        for (int a = 3; a >= 1; --a) {
            double v[4] = {0, 0, 0, 0};
            v[a] = 1.0;
            for (int b = 3; b > a; --b) {
                double pr = gdot(o.g, v, leg[b]);
                for (int mu = 1; mu < 4; ++mu) v[mu] -= pr * leg[b][mu];
            }
            double nrm = std::sqrt(gdot(o.g, v, v));
            for (int mu = 1; mu < 4; ++mu) leg[a][mu] = v[mu] / nrm;
        }
        for (int a = 1; a < 4; ++a) for (int mu = 0; mu < 4; ++mu) o.e[mu][a] = leg[a][mu];
    }
    // e^a_mu = eta^{ab} g_{mu nu} e^nu_b
    for (int a = 0; a < 4; ++a)
        for (int mu = 0; mu < 4; ++mu) {
            double s = 0;
            for (int nu = 0; nu < 4; ++nu) s += o.g[mu][nu] * o.e[nu][a];
            o.einv[a][mu] = (a == 0 ? -s : s);
        }
}

void eval_omega(const rt_metric &mt, const double x[3], double omega[4][4][4]) {
    std::memset(omega, 0, sizeof(double) * 64);
    if (mt.kind == RT_MINKOWSKI_CART) return;
    PointGeom c;
    eval_point(mt, x, c);
    if (c.dead) return;
    double ginv[4][4];
    invert44(c.g, ginv, nullptr);
    // dg[mu][s][l] = d_mu g_{sl}, de[mu][b][d] = d_mu e^b_d  (d_0 = 0: stationary, L79)
    // 6th-order central differences (reading S15: the paper says only "finite difference", L109): truncation h^6 f^(7) / 140,
    // round-off ~ 1.5 eps |f| / h; with h = 5e-4 this implementation and the oracle's agree to ~1e-12 and both are that close
    // to the exact coefficients
    static const double wgt[6] = {-1.0, 9.0, -45.0, 45.0, -9.0, 1.0};
    static const double off[6] = {-3.0, -2.0, -1.0, 1.0, 2.0, 3.0};
    double dg[4][4][4] = {{{0}}}, de[4][4][4] = {{{0}}};
    for (int i = 0; i < 3; ++i)
        for (int q = 0; q < 6; ++q) {
            double xx[3] = {x[0], x[1], x[2]};
            xx[i] += off[q] * FD_H;
            PointGeom p;
            eval_point(mt, xx, p);
            for (int s = 0; s < 4; ++s)
                for (int l = 0; l < 4; ++l) {
                    dg[i + 1][s][l] += wgt[q] * p.g[s][l] / (60.0 * FD_H);
                    de[i + 1][s][l] += wgt[q] * p.e[s][l] / (60.0 * FD_H);
                }
        }
    double Gam[4][4][4];  // Gamma^b_{m l}
    for (int b = 0; b < 4; ++b)
        for (int m = 0; m < 4; ++m)
            for (int l = 0; l < 4; ++l) {
                double s = 0;
                for (int q = 0; q < 4; ++q) s += ginv[b][q] * (dg[m][q][l] + dg[l][q][m] - dg[q][m][l]);
                Gam[b][m][l] = 0.5 * s;
            }
    double nab[4][4][4];  // nabla_mu e^b_d
    for (int mu = 0; mu < 4; ++mu)
        for (int b = 0; b < 4; ++b)
            for (int d = 0; d < 4; ++d) {
                double s = de[mu][b][d];
                for (int l = 0; l < 4; ++l) s += Gam[b][mu][l] * c.e[l][d];
                nab[mu][b][d] = s;
            }
    for (int a = 0; a < 4; ++a)
        for (int cc = 0; cc < 4; ++cc)
            for (int d = 0; d < 4; ++d) {
                double s = 0;
                for (int b = 0; b < 4; ++b)
                    for (int mu = 0; mu < 4; ++mu) s += c.einv[a][b] * c.e[mu][cc] * nab[mu][b][d];
                omega[a][cc][d] = s;
            }
}

}  // namespace rt
