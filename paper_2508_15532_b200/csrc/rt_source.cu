// Cell-local kernel of librt_b200 (sm_100a): the implicit radiation-fluid source step (O6).
//
// PAPER.md: fluid-frame boost Eq 5 (L85) with I/nu^4 and nu^2 dOmega invariance (S17); angular sums Eq 33, 41
// (L344, L388-390); temperature equations Eq 42 / 43 / 46 (L396-426; S19: A' = alpha_- dt A); intensity update
// Eq 35 (L352) with the coefficients the T-equation was built from (S19b); density floor L468.
// The moments (Eq 13) and the 4-force G_nu = -(R^0_nu after - before)/dt (Eq 36, 48) come from the tensor-pipe pass of
// rt_moments_mma.cu, run before and after this kernel on the same cells (launch_source below).
//
// Design: a warp takes CB cells of the interaction list per trip; a cell's N_d intensities live in registers (MAXV per
// lane, s = lane + 32 v, so every load/store is a 256-byte coalesced row); the angular sums are added in a fixed order
// (bit-reproducible); see k_cell_batch.
#include <cmath>
#include <type_traits>

#include "rt_kernels.cuh"

namespace rt {
namespace {

constexpr double FOURPI = 12.566370614359172953850573533118;

// T^-3.5 = (1/T)^3 sqrt(1/T): a reciprocal and a square root instead of pow()
__device__ __forceinline__ double t_m35(double T) {
    const double r = __drcp_rn(T);
    return r * r * r * sqrt(r);
}

// 1 / x for the positive, well-scaled x = d nbar of a direction: the hardware's reciprocal seed (rcp.approx.ftz.f64, ~20 bits) and two
// Newton steps (4 dependent FMAs, relative error < 2^-52 before the last rounding) instead of the correctly rounded __drcp_rn
// (its special-case handling and longer dependent chain cost ~5 instructions and ~25 cycles of latency per direction)
__device__ __forceinline__ double rcp_pos(double x) {
    double y;
    asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(x));
    double e = fma(-x, y, 1.0);
    y = fma(y, e, y);
    e = fma(-x, y, 1.0);
    return fma(y, e, y);
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

constexpr int CELL_THREADS = 128, CELL_MINB = 4;   // 128 registers, 16 warps per SM

// ---- the source step, CB cells per warp trip -----------------------------------------------------------------------------
// With one cell per warp trip (round 1) about half of the ~760 instructions per cell (162 directions) were scalar work every
// lane repeats (fluid-frame velocity, opacities, the temperature solve with its dependent reciprocal chain), and the warp's
// instruction stream was one long dependent chain.  Here a warp takes CB listed cells per trip:
//   phase 0  lane l does the scalar set-up of cell l mod CB (loads, opacities, u-hat): once per trip, not once per cell;
//   phase 1  cell by cell, lanes over directions: nbar, d, the three angular sums of Eq 33 / 41 as per-lane partials, and the
//            two coefficients of Eq 35 (n^0 I / d stays in the value's register, 1 / (d nbar^3) goes to shared memory);
//            the CB cells' loops are independent instruction streams the scheduler can overlap;
//   sums     the 3 CB rows of partials are added through shared memory in a fixed order (two lanes per row);
//   phase 2  lane l solves the temperature equation of cell l mod CB: ONE solve stream for the CB cells;
//   phase 3  cell by cell: Eq 35, store.
template <int MAXV>
struct CellBatch { static constexpr int CB = MAXV <= 3 ? 8 : (24 / MAXV > 0 ? 24 / MAXV : 1); };

// LITERAL: rt_options.source_literal with Method 2 or 3 -- Eq 35 with every opacity at T_+ (L432 taken literally, S19b's option):
// phase 3 forms d_s again with alpha(T_+) (an instantiation of its own: the default path pays nothing for the option)
template <int MAXV, bool LITERAL>
__global__ void __launch_bounds__(CELL_THREADS, CELL_MINB)
k_cell_batch(KParams p, double *I, double *T, double dt, int *n_fail) {
    constexpr int CB = CellBatch<MAXV>::CB;
    constexpr int PART = CB * 3 * 33 + CB * 3;                                   // partial sums [CB * 3][33], totals [CB * 3]
    constexpr int SCR = MAXV * 32 * CB + PART;
    extern __shared__ double tab[];   // nx[pitch] ny[pitch] nz[pitch] w[pitch], then one scratch area per warp
    for (int t = threadIdx.x; t < 3 * p.pitch; t += blockDim.x) tab[t] = p.nhat[t];
    for (int t = threadIdx.x; t < p.pitch; t += blockDim.x) tab[3 * p.pitch + t] = p.w[t];
    __syncthreads();
    const double *snx = tab, *sny = tab + p.pitch, *snz = tab + 2 * p.pitch, *sw = tab + 3 * p.pitch;
    const int lane = threadIdx.x & 31;
    double *cbs = tab + 4 * p.pitch + (threadIdx.x >> 5) * SCR;   // [CB][MAXV * 32]: 1 / (d nbar^3) of every direction
    double *part = cbs + MAXV * 32 * CB;
    const long long warp0 = (blockIdx.x * (long long)blockDim.x + threadIdx.x) >> 5;
    const long long nwarps = ((long long)gridDim.x * blockDim.x) >> 5;
    const long long nwork = (long long)__ldg(p.nsel);
    const int myc = lane % CB;   // the cell of the trip whose scalars this lane holds

    for (long long w0 = warp0 * CB; w0 < nwork; w0 += nwarps * CB) {
        const int ncb = (int)((nwork - w0) < CB ? (nwork - w0) : CB);
        // ---- phase 0: scalars of cell myc ----
        const bool have = myc < ncb;
        const long long mycell = have ? (long long)__ldg(p.srclist + w0 + myc) : 0;
        double rho = 0.0, Tm = 1.0, aa = 0.0, as = 0.0, alpha = 0.0, uh0 = 1.0, uh1 = 0.0, uh2 = 0.0, uh3 = 0.0;
        if (have) {
            rho = p.rho[mycell];
            Tm = T[mycell];
            const double u0 = p.u4[mycell], u1 = p.u4[p.ncell + mycell], u2 = p.u4[2 * p.ncell + mycell], u3 = p.u4[3 * p.ncell + mycell];
            const double *cen = p.cen + (long long)((unsigned)mycell % (unsigned)p.ncol) * CEN_STRIDE;
            uh0 = cen[12] * u0 + cen[13] * u1 + cen[14] * u2 + cen[15] * u3;
            uh1 = cen[16] * u0 + cen[17] * u1 + cen[18] * u2 + cen[19] * u3;
            uh2 = cen[20] * u0 + cen[21] * u1 + cen[22] * u2 + cen[23] * u3;
            uh3 = cen[24] * u0 + cen[25] * u1 + cen[26] * u2 + cen[27] * u3;
            if (rho >= p.rho_floor) {
                aa = (p.kappa_a0 != 0.0) ? p.kappa_a0 * rho * rho * t_m35(Tm) : 0.0;
                as = p.kappa_s * rho;
            }
            alpha = aa + as;
        }
        const bool interact = have && p.method != 0 && alpha != 0.0;
        const double adt = alpha * dt;

        {   // the NEXT trip's operands towards the SM now: the rows of its cells and their fluid state (a trip is ~15 us of work per warp;
            // otherwise its first loads -- list entry, then density, then intensities -- are three dependent trips to DRAM)
            const long long wn = w0 + nwarps * CB + myc;
            if (wn < nwork) {
                const long long cn = (long long)__ldg(p.srclist + wn);
                const char *row = reinterpret_cast<const char *>(I + cn * p.pitch);
                for (int line = lane / CB; line * 128 < p.pitch * 8; line += 32 / CB)
                    asm volatile("prefetch.global.L1 [%0];" ::"l"(row + line * 128));
                if (lane < CB) {
                    asm volatile("prefetch.global.L1 [%0];" ::"l"(p.rho + cn));
                    asm volatile("prefetch.global.L1 [%0];" ::"l"(T + cn));
#pragma unroll
                    for (int m = 0; m < 4; ++m) asm volatile("prefetch.global.L1 [%0];" ::"l"(p.u4 + m * p.ncell + cn));
                }
            }
        }
        // ---- phase 1: per cell, lanes over directions ----
        double val[CB][MAXV];          // I, then n^0 I / d for the cells that interact
        unsigned livebits = 0u;        // bit c * MAXV + v: direction v of cell c is updated (not masked, not a pad entry)
#pragma unroll
        for (int c = 0; c < CB; ++c) {
            const long long cell = __shfl_sync(0xffffffffu, mycell, c);
            const bool inter_c = __shfl_sync(0xffffffffu, (int)interact, c) != 0;
            const bool there = c < ncb;
            const double *Ic = I + cell * p.pitch;
#pragma unroll
            for (int v = 0; v < MAXV; ++v) {
                const int s = lane + 32 * v;
                val[c][v] = (there && s < p.nd) ? Ic[s] : 0.0;
            }
            double E = 0.0, A1 = 0.0, A2 = 0.0;
            if (inter_c) {
                const double b0 = __shfl_sync(0xffffffffu, uh0, c), b1 = __shfl_sync(0xffffffffu, uh1, c);
                const double b2 = __shfl_sync(0xffffffffu, uh2, c), b3 = __shfl_sync(0xffffffffu, uh3, c);
                const double adt_c = __shfl_sync(0xffffffffu, adt, c);
                const double *cen = p.cen + (long long)((unsigned)cell % (unsigned)p.ncol) * CEN_STRIDE;
                const double g0 = __ldg(cen), g1 = __ldg(cen + 1), g2 = __ldg(cen + 2), g3 = __ldg(cen + 3);       // -> n_0
                const double e0 = __ldg(cen + 4), e1 = __ldg(cen + 5), e2 = __ldg(cen + 6), e3 = __ldg(cen + 7);   // -> n^0
#pragma unroll
                for (int v = 0; v < MAXV; ++v) {
                    const int s = lane + 32 * v;
                    double cb = 0.0, ca = 0.0;
                    if (s < p.nd) {
                        const double nx = snx[s], ny = sny[s], nz = snz[s], ws = sw[s];
                        const double n0c = g0 + g1 * nx + g2 * ny + g3 * nz;
                        if (!(n0c > -p.n0_floor)) {
                            const double nup = e0 + e1 * nx + e2 * ny + e3 * nz;
                            const double nbar = b0 - (b1 * nx + b2 * ny + b3 * nz);        // Eq 5, first row
                            // 1/d and 1/nbar from one reciprocal: 1/(d nbar) times nbar, times d
                            const double d = nup + nbar * adt_c, r = rcp_pos(d * nbar);
                            const double rd = r * nbar, rn = r * d;
                            const double IbdOm = nbar * nbar * val[c][v] * ws;               // Ibar dOmegabar (S17)
                            E += IbdOm;                                                     // Eq 33
                            A1 += nup * rd * IbdOm;                                         // Eq 41a
                            A2 += ws * rn * rd;                                             // Eq 41b
                            ca = nup * rd;                                                  // n^0 / d
                            cb = rd * (rn * rn * rn);                                       // 1 / (d nbar^3)
                            livebits |= 1u << (c * MAXV + v);
                        }
                    }
                    val[c][v] = ca * val[c][v];
                    cbs[(c * MAXV + v) * 32 + lane] = cb;
                }
            }
            part[(c * 3 + 0) * 33 + lane] = E; part[(c * 3 + 1) * 33 + lane] = A1; part[(c * 3 + 2) * 33 + lane] = A2;
        }
        __syncwarp();
        // ---- the 3 CB sums: LPR lanes per row, each over its entries in index order, then one exchange ----
        {
            constexpr int LPR = (6 * CB <= 32) ? 2 : 1, NPL = 32 / LPR;
            double t = 0.0;
            if (lane < 3 * CB * LPR) {
                const double *r = part + (lane / LPR) * 33 + (lane % LPR) * NPL;
#pragma unroll
                for (int m = 0; m < NPL; ++m) t += r[m];
            }
            if (LPR == 2) t += __shfl_xor_sync(0xffffffffu, t, 1);   // (the even lane adds first half + second half)
            if (lane < 3 * CB * LPR && (lane % LPR) == 0) part[CB * 3 * 33 + lane / LPR] = t;
        }
        __syncwarp();
        // ---- phase 2: lane l solves the temperature equation of cell l mod CB ----
        bool ok = false;
        double Tp = Tm, scale = 1.0, Sdt = 0.0, adtp = 0.0;
        if (interact) {
            const double *tot = part + CB * 3 * 33 + myc * 3;
            const double E = tot[0], A1 = tot[1], A2 = tot[2] * (dt / FOURPI);
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
            ok = solve_T(q, Tm, W / Y, Tp);
            if (ok) {
                const double Ep = W - Y * Tp;                                               // Eq 39
                const double emis = (p.method == 1) ? aa * p.a_rad * Tp * Tp * Tp * Tp : Nbar * p.a_rad * sqrt(Tp);
                scale = (p.method == 3 && !LITERAL) ? alpha / (as + Nbar * t_m35(Tp)) : 1.0;
                if (LITERAL) adtp = (as + Nbar * t_m35(Tp)) * dt;
                Sdt = (emis + as * Ep) * (dt / FOURPI);
                if (lane < CB) T[mycell] = Tp;
            } else if (lane < CB && n_fail) {
                atomicAdd(n_fail, 1);
            }
        }
        __syncwarp();

        // ---- phase 3: Eq 35 divided by nbar^4 (L432): I+ = [n^0/d] I- + [nbar dt/(4 pi d)] S / nbar^4 ----
#pragma unroll
        for (int c = 0; c < CB; ++c) {
            if (c >= ncb) break;
            const long long cell = __shfl_sync(0xffffffffu, mycell, c);
            const bool ok_c = __shfl_sync(0xffffffffu, (int)ok, c) != 0;
            double *Ic = I + cell * p.pitch;
            if (ok_c) {
                const double sc = __shfl_sync(0xffffffffu, scale, c), sd = __shfl_sync(0xffffffffu, Sdt, c);
                if (LITERAL) {
                    // val holds (n^0 / d_-) I_-: times d_- / d_+, and the source term with 1 / (d_+ nbar^3)
                    const double b0 = __shfl_sync(0xffffffffu, uh0, c), b1 = __shfl_sync(0xffffffffu, uh1, c);
                    const double b2 = __shfl_sync(0xffffffffu, uh2, c), b3 = __shfl_sync(0xffffffffu, uh3, c);
                    const double am = __shfl_sync(0xffffffffu, adt, c), ap = __shfl_sync(0xffffffffu, adtp, c);
                    const double *cen = p.cen + (long long)((unsigned)cell % (unsigned)p.ncol) * CEN_STRIDE;
                    const double e0 = __ldg(cen + 4), e1 = __ldg(cen + 5), e2 = __ldg(cen + 6), e3 = __ldg(cen + 7);
#pragma unroll
                    for (int v = 0; v < MAXV; ++v) {
                        if ((livebits >> (c * MAXV + v)) & 1u) {
                            const int s = lane + 32 * v;
                            const double nx = snx[s], ny = sny[s], nz = snz[s];
                            const double nup = e0 + e1 * nx + e2 * ny + e3 * nz;
                            const double nbar = b0 - (b1 * nx + b2 * ny + b3 * nz);
                            const double dm = nup + nbar * am, dp = nup + nbar * ap, r = rcp_pos(dp * nbar);
                            const double rd = r * nbar, rn = r * dp;
                            val[c][v] = val[c][v] * (dm * rd) + sd * (rd * (rn * rn * rn));
                            Ic[s] = val[c][v];
                        }
                    }
                } else {
#pragma unroll
                    for (int v = 0; v < MAXV; ++v) {
                        if ((livebits >> (c * MAXV + v)) & 1u) {
                            val[c][v] = sc * (val[c][v] + sd * cbs[(c * MAXV + v) * 32 + lane]);
                            Ic[lane + 32 * v] = val[c][v];
                        }
                    }
                }
            }
        }
        __syncwarp();
    }
}

cudaError_t launch_cell_batch(const KParams &p, double *I, double *T, double dt, int *n_fail, cudaStream_t st) {
    const int threads = CELL_THREADS, warps = threads / 32;
    auto go = [&](auto maxv_tag) -> cudaError_t {
        constexpr int MAXV = decltype(maxv_tag)::value;
        constexpr int CB = CellBatch<MAXV>::CB;
        constexpr int PART = CB * 3 * 33 + CB * 3;
        const size_t scr = MAXV * 32 * CB + PART;
        const size_t smem = (4 * p.pitch + warps * scr) * sizeof(double);
        // a list's length is only known on the device: a fixed grid, the kernel strides over whatever the list holds
        long long want = (p.ncell + (long long)warps * CB - 1) / ((long long)warps * CB);
        const int blocks = (int)(want < 148LL * 8 * 4 ? want : 148LL * 8 * 4);
        if (blocks == 0) return cudaSuccess;
        const bool literal = p.source_literal && p.method != 1;   // (Method 1 does not update its opacities, L432)
        cudaError_t e = literal ? cudaFuncSetAttribute(k_cell_batch<MAXV, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem)
                                : cudaFuncSetAttribute(k_cell_batch<MAXV, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e != cudaSuccess) return e;
        if (literal) k_cell_batch<MAXV, true><<<blocks, threads, smem, st>>>(p, I, T, dt, n_fail);
        else k_cell_batch<MAXV, false><<<blocks, threads, smem, st>>>(p, I, T, dt, n_fail);
        return cudaGetLastError();
    };
    if (p.nd <= 64) return go(std::integral_constant<int, 2>());
    if (p.nd <= 192) return go(std::integral_constant<int, 6>());
    if (p.nd <= 384) return go(std::integral_constant<int, 12>());
    if (p.nd <= 672) return go(std::integral_constant<int, 21>());
    return cudaErrorInvalidValue;
}

}  // namespace

// Source step on the cells of the interaction list.  Moments, where wanted, come from the tensor-pipe pass (rt_moments_mma.cu)
// run over the same intensities: R^0_nu of the listed cells before the step (parked in G), R of the listed cells after it with
// G_nu = -(R^0_nu after - before) / dt (Eq 36, 48), and R of the cells the step does not visit; G is zero there.
cudaError_t launch_source(const KParams &p, double *I, double *T, double dt, int *n_fail, double *R_after, double *G,
                          cudaStream_t st, long long *launches) {
    cudaError_t e = cudaSuccess;
    if (G) e = cudaMemsetAsync(G, 0, 4 * p.ncell * sizeof(double), st);
    const bool listed = p.method != 0 && p.srclist != nullptr;   // (the list may still be empty: its kernels then find nothing to do)
    if (e == cudaSuccess && listed) {
        if (G) { ++*launches; e = launch_moments_mma(p, I, nullptr, G, 1, 1, dt, st); }
        if (e == cudaSuccess) { ++*launches; e = launch_cell_batch(p, I, T, dt, n_fail, st); }
        if (e == cudaSuccess && (G || R_after)) { ++*launches; e = launch_moments_mma(p, I, R_after, G, 1, G ? 2 : 0, dt, st); }
    }
    if (e == cudaSuccess && R_after) {   // cells the source step did not visit (all of them without a list)
        ++*launches;
        e = launch_moments_mma(p, I, R_after, nullptr, listed ? 2 : 0, 0, dt, st);
    }
    return e;
}

cudaError_t launch_moments(const KParams &p, const double *I, double *R, cudaStream_t st, long long *launches) {
    ++*launches;
    return launch_moments_mma(p, I, R, nullptr, 0, 0, 1.0, st);
}

}  // namespace rt
