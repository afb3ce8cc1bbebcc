// Cell-local kernels of librt_b200 (sm_100a): implicit radiation-fluid source step (O6) fused with the moment
// reduction (O7) and the 4-force (Eq 36/48).
//
// PAPER.md: fluid-frame boost Eq 5 (L85) with I/nu^4 and nu^2 dOmega invariance (S17); angular sums Eq 33, 41
// (L344, L388-390); temperature equations Eq 42 / 43 / 46 (L396-426; S19: A' = alpha_- dt A); intensity update
// Eq 35 (L352) with the coefficients the T-equation was built from (S19b); density floor L468; moments Eq 13
// (L141); G_nu = -(R^0_nu after - before)/dt (Eq 36, 48).
//
// Design: one warp per cell; the cell's N_d intensities live in registers (MAXV per lane, s = lane + 32 v, so
// every load/store is a 256-byte coalesced row); all angular sums are butterfly warp reductions (fixed order =>
// bit-reproducible); the scalar temperature solve runs redundantly on all lanes (no divergence, no broadcast).
// Moments are accumulated in the TETRAD frame, M^{ab} = sum_s w_s I_s n^a n^b (10 sums with constant n-hat), and
// rotated once per cell: R^mu_nu = e^mu_a M^{ab} (e^lam_b g_{lam nu}).
#include <cmath>

#include "rt_kernels.cuh"

namespace rt {
namespace {

constexpr double FOURPI = 12.566370614359172953850573533118;

// T^-3.5 = (1/T)^3 sqrt(1/T): a reciprocal and a square root instead of pow()
__device__ __forceinline__ double t_m35(double T) {
    const double r = __drcp_rn(T);
    return r * r * r * sqrt(r);
}
__device__ __forceinline__ double warp_sum(double v) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}

// Sums of the ten moment components over the 32 lanes through shared memory: every lane stores its ten partial sums
// (row c at scr[c * 33 + lane]), three lanes add up each row (11 + 11 + 10 entries, combined by two shuffles), the
// ten totals are written behind the rows and read back by all lanes.  ~45 instructions per lane instead of the 150 of
// ten butterfly reductions; fixed order => bit-reproducible.  scr: WSUM_DOUBLES doubles owned by the warp.
constexpr int WSUM_DOUBLES = 10 * 33 + 10;
__device__ __forceinline__ void warp_sum10(double M[10], double *scr, int lane) {
#pragma unroll
    for (int c = 0; c < 10; ++c) scr[c * 33 + lane] = M[c];
    __syncwarp();
    const int c = lane / 3, q = lane - 3 * c;
    double t = 0.0;
    if (lane < 30) {
        const double *r = scr + c * 33 + q * 11;
#pragma unroll
        for (int m = 0; m < 10; ++m) t += r[m];
        if (q < 2) t += r[10];
    }
    const double t1 = __shfl_down_sync(0xffffffffu, t, 1), t2 = __shfl_down_sync(0xffffffffu, t, 2);
    if (lane < 30 && q == 0) scr[330 + c] = (t + t1) + t2;
    __syncwarp();
#pragma unroll
    for (int k = 0; k < 10; ++k) M[k] = scr[330 + k];
    __syncwarp();
}

struct TEq {
    int method;
    double a4, b1, c0;             // methods 1, 2: a4 g(T) + b1 T + c0
    double k45, k4, k35, k1, k0;   // method 3: coefficients of Eq 46
};
// residual and derivative of the temperature equation; sqrt(T) and 1/sqrt(T) from one rsqrt (no division)
__device__ __forceinline__ void teq_eval(const TEq &q, double T, double &f, double &df) {
    if (q.method == 1) {
        const double T3 = T * T * T;
        f = q.a4 * T3 * T + q.b1 * T + q.c0;
        df = 4.0 * q.a4 * T3 + q.b1;
    } else if (q.method == 2) {
        const double ir = rsqrt(T), r = T * ir;
        f = q.a4 * r + q.b1 * T + q.c0;
        df = 0.5 * q.a4 * ir + q.b1;
    } else {
        const double ir = rsqrt(T), r = T * ir, T3 = T * T * T, T35 = T3 * r, T4 = T3 * T, T45 = T4 * r;
        f = -(q.k45 * T45 + q.k4 * T4 + q.k35 * T35 + q.k1 * T + q.k0);
        df = -(4.5 * q.k45 * T35 + 4.0 * q.k4 * T3 + 3.5 * q.k35 * T3 * ir + q.k1);
    }
}
// Root of the temperature equation on (0, W/Y] (S20).  Existence is decided as the reading says (the residual is negative at
// 0+ and non-negative at W/Y; otherwise the cell keeps T_- and is counted).  Method 2 (Eq 43) is a quadratic in x = sqrt(T),
// a4 x + b1 x^2 + c0 = 0 with b1 > 0 > c0, and is solved in closed form, written so that nothing cancels:
//     x = 2 |c0| / (a4 + sqrt(a4^2 + 4 b1 |c0|)).
// Methods 1 and 3 (Eq 42: quartic, Eq 46: degree 9 in x) use Newton-Raphson (L399) from T_-, kept inside the bracket; the
// Newton step multiplies by a reciprocal instead of dividing, so the iterates differ from a division-based solver's in
// the last bits while the root they converge to (|dT| <= 1e-14 T) does not.
__device__ __forceinline__ bool solve_T(const TEq &q, double Tm, double Thi, double &Tp) {
    double lo = 0.0, hi = Thi, f, df;
    if (!(Thi > 0.0)) return false;
    teq_eval(q, hi, f, df);
    if (!(f >= 0.0)) return false;
    if (q.method != 3 && !(q.c0 < 0.0)) return false;
    if (q.method == 2) {
        const double x = 2.0 * -q.c0 / (q.a4 + sqrt(fma(q.a4, q.a4, 4.0 * q.b1 * -q.c0)));
        Tp = x * x;
        return true;
    }
    double T = (Tm > lo && Tm < hi) ? Tm : 0.5 * (lo + hi);
    for (int it = 0; it < 100; ++it) {
        teq_eval(q, T, f, df);
        if (f < 0) lo = T; else hi = T;
        double Tn = T - f * __drcp_rn(df);
        if (!(Tn > 0.0 && Tn >= lo && Tn <= hi)) Tn = 0.5 * (lo + hi);   // closed bracket (S20): a root at an end is kept
        const double d = Tn - T;
        T = Tn;
        if (fabs(d) <= 1e-14 * T) break;
    }
    Tp = T;
    return true;
}

// 10 independent components of M^{ab}: 00 01 02 03 11 12 13 22 23 33
__device__ __forceinline__ void mom_accumulate(double M[10], double wI, double nx, double ny, double nz) {
    M[0] += wI;
    M[1] += wI * nx; M[2] += wI * ny; M[3] += wI * nz;
    M[4] += wI * nx * nx; M[5] += wI * nx * ny; M[6] += wI * nx * nz;
    M[7] += wI * ny * ny; M[8] += wI * ny * nz; M[9] += wI * nz * nz;
}
__device__ __forceinline__ double mom_get(const double M[10], int a, int b) {
    if (a > b) { int t = a; a = b; b = t; }
    const int base[4] = {0, 4, 7, 9};
    return M[base[a] + (b - a)];
}
// R^mu_nu for (mu, nu) from tetrad-frame M, e^mu_a (ecen) and L[b][nu] (cen + 28)
__device__ __forceinline__ double rotate(const double M[10], const double *__restrict__ ecen, const double *__restrict__ L, int mu, int nu) {
    double r = 0.0;
    for (int a = 0; a < 4; ++a) {
        double t = 0.0;
        for (int b = 0; b < 4; ++b) t += mom_get(M, a, b) * L[4 * b + nu];
        r += ecen[4 * mu + a] * t;
    }
    return r;
}

// source-step variants: 128 registers, 16 warps per SM (80 registers x 24 warps spills and is 2-3 % slower)
constexpr int CELL_THREADS = 128, CELL_MINB = 4;
// moments-only instantiation (kept for completeness; the moments-only passes run in rt_moments_mma.cu)
constexpr int MOM_THREADS = 256, MOM_MINB = 4;
template <int MAXV, bool SRC, bool MOM, bool LIST>
__global__ void __launch_bounds__(SRC ? CELL_THREADS : MOM_THREADS, (SRC ? CELL_MINB : (MAXV > 6 ? MOM_MINB - 2 : MOM_MINB)))   // moments-only, 362 directions: 12 values per lane, 128 registers
k_cell(KParams p, double *I, double *T, double dt, int *n_fail, double *R_out, double *G_out) {
    extern __shared__ double tab[];   // nx[pitch] ny[pitch] nz[pitch] w[pitch], then one warp_sum10 scratch per warp
    for (int t = threadIdx.x; t < 3 * p.pitch; t += blockDim.x) tab[t] = p.nhat[t];
    for (int t = threadIdx.x; t < p.pitch; t += blockDim.x) tab[3 * p.pitch + t] = p.w[t];
    __syncthreads();
    const double *snx = tab, *sny = tab + p.pitch, *snz = tab + 2 * p.pitch, *sw = tab + 3 * p.pitch;
    const int lane = threadIdx.x & 31;
    double *scr = tab + 4 * p.pitch + (threadIdx.x >> 5) * WSUM_DOUBLES;
    const long long warp0 = (blockIdx.x * (long long)blockDim.x + threadIdx.x) >> 5;
    const long long nwarps = ((long long)gridDim.x * blockDim.x) >> 5;

    // LIST: the warp index runs over the compact list of cells above the density floor (built by rt_set_fluid)
    const long long nwork = LIST ? (long long)__ldg(p.nsel) : p.ncell;
    for (long long widx = warp0; widx < nwork; widx += nwarps) {
        const long long cell = LIST ? (long long)p.srclist[widx] : widx;
        if (!SRC && widx + nwarps < nwork) {   // moments-only passes stream: next cell of this warp, one 128-byte line per lane, into L2/L1
            const long long nc = LIST ? (long long)p.srclist[widx + nwarps] : widx + nwarps;
            const char *nx = reinterpret_cast<const char *>(I + nc * p.pitch) + lane * 128;
            if (lane * 128 < p.pitch * 8) asm volatile("prefetch.global.L1 [%0];" ::"l"(nx));
        }
        const int col = int((unsigned)cell % (unsigned)p.ncol);   // cell < 2^31 (the lists hold ints)
        const double *cen = p.cen + (long long)col * CEN_STRIDE;
        double *Ic = I + cell * p.pitch;
        // all independent loads first: the cell's intensities (needed for every cell only when moments are wanted)
        // and its fluid state
        double val[MAXV];
        if (MOM) {
#pragma unroll
            for (int v = 0; v < MAXV; ++v) {
                const int s = lane + 32 * v;
                val[v] = (s < p.nd) ? Ic[s] : 0.0;
            }
        }
        double alpha = 0.0, aa = 0.0, as = 0.0, rho = 0.0, Tm = 0.0, u0 = 1.0, u1 = 0.0, u2 = 0.0, u3 = 0.0;
        if (SRC) {
            rho = p.rho[cell];
            Tm = T[cell];
            u0 = p.u4[cell]; u1 = p.u4[p.ncell + cell]; u2 = p.u4[2 * p.ncell + cell]; u3 = p.u4[3 * p.ncell + cell];
            if (rho >= p.rho_floor) {
                aa = (p.kappa_a0 != 0.0) ? p.kappa_a0 * rho * rho * t_m35(Tm) : 0.0;
                as = p.kappa_s * rho;
            }
            alpha = aa + as;
        }
        const bool interact = SRC && p.method != 0 && alpha != 0.0;
        if (!interact && !MOM) continue;
        if (!MOM) {
#pragma unroll
            for (int v = 0; v < MAXV; ++v) {
                const int s = lane + 32 * v;
                val[v] = (s < p.nd) ? Ic[s] : 0.0;
            }
        }
        const double *ecen = p.ecen + (long long)col * 16, *L = cen + 28;
        double Rb = 0.0;          // lanes 0..3: R^0_nu before the source step
        bool updated = false;
        if (interact) {
            const double uh0 = cen[12] * u0 + cen[13] * u1 + cen[14] * u2 + cen[15] * u3;
            const double uh1 = cen[16] * u0 + cen[17] * u1 + cen[18] * u2 + cen[19] * u3;
            const double uh2 = cen[20] * u0 + cen[21] * u1 + cen[22] * u2 + cen[23] * u3;
            const double uh3 = cen[24] * u0 + cen[25] * u1 + cen[26] * u2 + cen[27] * u3;
            if (MOM && G_out) {   // moments before the update (only where the update can change them)
                double Mb[10] = {0, 0, 0, 0, 0, 0, 0, 0, 0, 0};
#pragma unroll
                for (int v = 0; v < MAXV; ++v) {
                    const int s = lane + 32 * v;
                    if (s < p.nd) mom_accumulate(Mb, sw[s] * val[v], snx[s], sny[s], snz[s]);
                }
                warp_sum10(Mb, scr, lane);
                if (lane < 4) Rb = rotate(Mb, ecen, L, 0, lane);
            }
            double E = 0.0, A1 = 0.0, A2 = 0.0;
            const double g0 = __ldg(cen), g1 = __ldg(cen + 1), g2 = __ldg(cen + 2), g3 = __ldg(cen + 3);       // -> n_0
            const double e0 = __ldg(cen + 4), e1 = __ldg(cen + 5), e2 = __ldg(cen + 6), e3 = __ldg(cen + 7);   // -> n^0
            const double adt = alpha * dt;
            // kept for the update loop below: ca = n^0/d (0 marks a masked or pad entry), cb = 1/(d nbar^3)
            double ca[MAXV], cb[MAXV];
#pragma unroll
            for (int v = 0; v < MAXV; ++v) {
                const int s = lane + 32 * v;
                ca[v] = 0.0; cb[v] = 0.0;
                if (s < p.nd) {
                    const double nx = snx[s], ny = sny[s], nz = snz[s], ws = sw[s];
                    const double n0c = g0 + g1 * nx + g2 * ny + g3 * nz;
                    if (!(n0c > -p.n0_floor)) {
                        const double nup = e0 + e1 * nx + e2 * ny + e3 * nz;
                        const double nbar = uh0 - (uh1 * nx + uh2 * ny + uh3 * nz);       // Eq 5, first row
                        // 1/d and 1/nbar from one reciprocal: 1/(d nbar) times nbar, times d
                        const double d = nup + nbar * adt, r = __drcp_rn(d * nbar);
                        const double rd = r * nbar, rn = r * d;
                        const double IbdOm = nbar * nbar * val[v] * ws;                     // Ibar dOmegabar (S17)
                        E += IbdOm;                                                         // Eq 33
                        A1 += nup * rd * IbdOm;                                             // Eq 41a
                        A2 += ws * rn * rd;                                                 // Eq 41b
                        ca[v] = nup * rd;
                        cb[v] = rd * (rn * rn * rn);
                    }
                }
            }
            E = warp_sum(E); A1 = warp_sum(A1); A2 = warp_sum(A2) * (dt / FOURPI);
            const double Y = p.Y_over_rho * rho, W = E + Y * Tm, Nbar = p.kappa_a0 * rho * rho;
            TEq q;
            q.method = p.method;
            q.a4 = (p.method == 1) ? A2 * aa * p.a_rad : A2 * Nbar * p.a_rad;
            q.b1 = Y * (1.0 - A2 * as);
            q.c0 = A1 - Y * (1.0 - A2 * as) * Tm - (1.0 - A2 * as) * E;
            if (p.method == 3) {
                const double A1p = alpha * dt * A1, A2p = alpha * dt * A2;
                q.k45 = Y * as * (A2p - dt);
                q.k4 = -A2p * Nbar * p.a_rad;
                q.k35 = -(A2p * as * W + A1p - W * as * dt);
                q.k1 = -Y * Nbar * dt;
                q.k0 = W * Nbar * dt;
            }
            double Tp;
            if (solve_T(q, Tm, W / Y, Tp)) {
                const double Ep = W - Y * Tp;                                               // Eq 39
                const double emis = (p.method == 1) ? aa * p.a_rad * Tp * Tp * Tp * Tp : Nbar * p.a_rad * sqrt(Tp);
                const double scale = (p.method == 3) ? alpha / (as + Nbar * t_m35(Tp)) : 1.0;
                const double Sdt = (emis + as * Ep) * (dt / FOURPI);
#pragma unroll
                for (int v = 0; v < MAXV; ++v) {
                    if (ca[v] != 0.0) {   // (n^0/d > 0 for every unmasked direction)
                        // Eq 35 divided by nbar^4 (L432): I+ = [n^0/d] I- + [nbar dt/(4 pi d)] S / nbar^4
                        val[v] = scale * (ca[v] * val[v] + Sdt * cb[v]);
                        Ic[lane + 32 * v] = val[v];
                    }
                }
                if (lane == 0) T[cell] = Tp;
                updated = true;
            } else if (lane == 0 && n_fail) {
                atomicAdd(n_fail, 1);
            }
        }
        if (MOM) {
            double Ma[10] = {0, 0, 0, 0, 0, 0, 0, 0, 0, 0};
#pragma unroll
            for (int v = 0; v < MAXV; ++v) {
                const int s = lane + 32 * v;
                if (s < p.nd) mom_accumulate(Ma, sw[s] * val[v], snx[s], sny[s], snz[s]);
            }
            warp_sum10(Ma, scr, lane);
            if (lane < 16) {
                const int mu = lane >> 2, nu = lane & 3;
                const double Ra = rotate(Ma, ecen, L, mu, nu);
                if (R_out) R_out[lane * p.ncell + cell] = Ra;
                if (G_out && mu == 0) G_out[nu * p.ncell + cell] = updated ? -(Ra - Rb) / dt : 0.0;
            }
        }
    }
}

template <bool SRC, bool MOM, bool LIST>
cudaError_t launch_cell(const KParams &p, double *I, double *T, double dt, int *n_fail, double *R, double *G, cudaStream_t st) {
    const int threads = SRC ? CELL_THREADS : MOM_THREADS;
    // a list's length is only known on the device: a fixed grid, the kernel strides over whatever the list holds
    const long long nwork = p.ncell;
    long long want = (nwork + threads / 32 - 1) / (threads / 32);
    const int blocks = (int)(want < 148LL * 8 * 4 ? want : 148LL * 8 * 4);
    if (blocks == 0) return cudaSuccess;
    const size_t smem = (4 * p.pitch + (threads / 32) * WSUM_DOUBLES) * sizeof(double);
    if (p.nd <= 64) k_cell<2, SRC, MOM, LIST><<<blocks, threads, smem, st>>>(p, I, T, dt, n_fail, R, G);
    else if (p.nd <= 192) k_cell<6, SRC, MOM, LIST><<<blocks, threads, smem, st>>>(p, I, T, dt, n_fail, R, G);
    else if (p.nd <= 384) k_cell<12, SRC, MOM, LIST><<<blocks, threads, smem, st>>>(p, I, T, dt, n_fail, R, G);
    else if (p.nd <= 672) k_cell<21, SRC, MOM, LIST><<<blocks, threads, smem, st>>>(p, I, T, dt, n_fail, R, G);
    else return cudaErrorInvalidValue;
    return cudaGetLastError();
}

}  // namespace

// Source step on the cells of the interaction list, with their moments (R after, G from before / after) when wanted;
// G is zero elsewhere; R of the cells not on the list comes from a second, source-free pass over the complement list.
cudaError_t launch_source(const KParams &p, double *I, double *T, double dt, int *n_fail, double *R_after, double *G,
                          cudaStream_t st, long long *launches) {
    cudaError_t e = cudaSuccess;
    if (G) e = cudaMemsetAsync(G, 0, 4 * p.ncell * sizeof(double), st);
    const bool listed = p.method != 0 && p.srclist != nullptr;   // (the list may still be empty: its kernels then find nothing to do)
    if (e == cudaSuccess && listed) {
        ++*launches;
        // with moments wanted the listed cells get theirs here (R after, G from before/after); the rest below
        e = (G || R_after) ? launch_cell<true, true, true>(p, I, T, dt, n_fail, R_after, G, st)
                           : launch_cell<true, false, true>(p, I, T, dt, n_fail, nullptr, nullptr, st);
    }
    if (e == cudaSuccess && R_after) {   // cells the source step did not visit: the tensor-pipe moments pass (rt_moments_mma.cu)
        ++*launches;
        e = launch_moments_mma(p, I, R_after, listed, st);   // listed: the complement of the list; else every cell
    }
    return e;
}

cudaError_t launch_moments(const KParams &p, const double *I, double *R, cudaStream_t st, long long *launches) {
    ++*launches;
    return launch_moments_mma(p, I, R, false, st);
}

}  // namespace rt
