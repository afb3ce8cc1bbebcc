// Angular flux with minimum-angle plane reconstruction (MAPR) for librt_b200 (sm_100a).
//
// PAPER.md L227 names MAPR (Christov & Popov 2008) for the reconstruction of I at the edges of the geodesic cells but
// does not describe it; reading S6 (O4'): in the tangent plane at n_s (log map), for every pair of
// consecutive neighbours (t_e, t_{e+1}) fit the plane through (0, I_s), (xi_e, I_e), (xi_{e+1}, I_{e+1}); keep the
// candidate gradient of smallest norm (ties -> lowest e); edge value I_s + grad . xi(m_e).  Flux: Eq 19 upwinded on the
// total normal angular velocity (S5).  PARITY UNPINNED beyond linear exactness (the oracle's O4' has no external pin).
//
// The arg-min over candidate planes is the only discontinuous branch of the scheme, so the squared norms are formed
// with explicitly rounded operations in the oracle's order (no FMA contraction): a near-tie resolves the same way.
//
// One CTA per column, thread = direction s, marching x3; per plane: stage the cell in shared memory, every thread
// computes its own gradient, stages it, then builds the two edge states of each of its 5/6 edges.
#include "rt_kernels.cuh"

namespace rt {
namespace {

__global__ void k_angular_mapr(KParams p, const double *__restrict__ I_in, double *I_io, double dt) {
    extern __shared__ double sm[];
    double *sI = sm, *sG = sm + p.pitch;   // sG[3][pitch]
    const int s = threadIdx.x, col = blockIdx.x, P = p.pitch;
    const int i = col % p.n1, j = col / p.n1;
    const bool live = s < p.nd, inrow = s < P;
    double coef[6];
    int nb[6], bk[6], nn = 0;
    unsigned up = 0;
    double scale = 0.0;
    bool zero = true;
    if (live) {
        const double nx = p.nhat[s], ny = p.nhat[P + s], nz = p.nhat[2 * P + s];
        const double *cen = p.cen + (long long)col * CEN_STRIDE;
        const double n0c = cen[0] + cen[1] * nx + cen[2] * ny + cen[3] * nz;
        const double nup = cen[4] + cen[5] * nx + cen[6] * ny + cen[7] * nz;
        scale = dt / (nup * n0c);
        const bool band_ij = (i < p.zlo[0] || i >= p.n1 - p.zhi[0] || j < p.zlo[1] || j >= p.n2 - p.zhi[1]);
        zero = band_ij || n0c > -p.n0_floor;
        nn = p.mapr_nnb[s];
        up = p.angup[(long long)col * P + s];
        for (int e = 0; e < 6; ++e) {
            coef[e] = p.angraw[((long long)col * 6 + e) * P + s];
            nb[e] = p.nb[e * P + s];
            bk[e] = p.mapr_back[e * P + s];
        }
    }
    const long long kstride = (long long)p.ncol * P;
    const double *pin = I_in + (long long)col * P + s;
    double *pio = I_io + (long long)col * P + s;
    for (int k = 0; k < p.n3; ++k, pin += kstride, pio += kstride) {
        const double v = inrow ? __ldg(pin) : 0.0;
        if (inrow) sI[s] = v;
        __syncthreads();
        double g0 = 0.0, g1 = 0.0, g2 = 0.0;
        if (live) {
            double dI[6];
#pragma unroll
            for (int e = 0; e < 6; ++e) dI[e] = (e < nn) ? sI[nb[e]] - v : 0.0;
            double best = __longlong_as_double(0x7ff0000000000000LL);
#pragma unroll
            for (int e = 0; e < 6; ++e) {
                if (e < nn) {
                    const int e2 = (e + 1 == nn) ? 0 : e + 1;
                    const double d1 = dI[e], d2 = (e + 1 == nn) ? dI[0] : dI[e + 1];
                    const double a11 = __ldg(p.mapr_a + (e * 4 + 0) * P + s), a12 = __ldg(p.mapr_a + (e * 4 + 1) * P + s);
                    const double a22 = __ldg(p.mapr_a + (e * 4 + 2) * P + s), det = __ldg(p.mapr_a + (e * 4 + 3) * P + s);
                    const double c1 = __ddiv_rn(__dsub_rn(__dmul_rn(d1, a22), __dmul_rn(d2, a12)), det);
                    const double c2 = __ddiv_rn(__dsub_rn(__dmul_rn(d2, a11), __dmul_rn(d1, a12)), det);
                    double G[3], nrm = 0.0;
#pragma unroll
                    for (int x = 0; x < 3; ++x) {
                        G[x] = __dadd_rn(__dmul_rn(c1, __ldg(p.mapr_xi + (e * 3 + x) * P + s)),
                                         __dmul_rn(c2, __ldg(p.mapr_xi + (e2 * 3 + x) * P + s)));
                        nrm = __dadd_rn(nrm, __dmul_rn(G[x], G[x]));
                    }
                    // ties (to round-off: equal masked neighbours tie structurally) -> lowest e
                    if (nrm < __dmul_rn(best, 1.0 - 1e-12)) { best = nrm; g0 = G[0]; g1 = G[1]; g2 = G[2]; }
                }
            }
        }
        if (inrow) { sG[s] = g0; sG[P + s] = g1; sG[2 * P + s] = g2; }
        __syncthreads();
        if (live) {
            double D = 0.0;
#pragma unroll
            for (int e = 0; e < 6; ++e) {
                if (e < nn) {
                    double val;
                    if ((up >> e) & 1u) {   // V > 0: the own reconstruction is upwind
                        val = v + (g0 * __ldg(p.mapr_xim + (e * 3 + 0) * P + s) + g1 * __ldg(p.mapr_xim + (e * 3 + 1) * P + s) +
                                   g2 * __ldg(p.mapr_xim + (e * 3 + 2) * P + s));
                    } else {
                        const int t = nb[e], be = bk[e];
                        val = sI[t] + (sG[t] * __ldg(p.mapr_xim + (be * 3 + 0) * P + t) + sG[P + t] * __ldg(p.mapr_xim + (be * 3 + 1) * P + t) +
                                       sG[2 * P + t] * __ldg(p.mapr_xim + (be * 3 + 2) * P + t));
                    }
                    D += coef[e] * val;
                }
            }
            const bool band_k = (k < p.zlo[2] || k >= p.n3 - p.zhi[2]);
            *pio = (zero || band_k) ? 0.0 : *pio - scale * D;
        } else if (inrow) {
            *pio = 0.0;
        }
        __syncthreads();
    }
}

}  // namespace

cudaError_t launch_angular_mapr(const KParams &p, const double *I_in, double *I_io, double dt, cudaStream_t st, long long *launches) {
    const int threads = ((p.pitch + 31) / 32) * 32;
    k_angular_mapr<<<p.ncol, threads, 4 * p.pitch * sizeof(double), st>>>(p, I_in, I_io, dt);
    ++*launches;
    return cudaGetLastError();
}

}  // namespace rt
