// Transport kernels of librt_b200 (sm_100a): face coefficients, spatial transport (O3 + O5), angular flux (O4 + O5).
//
// PAPER.md: Eq 18 (L193) finite-volume update of n^0 n_0 I; PLI reconstruction per direction (L225); vacuum flux
// Eq 20 (L245); non-vacuum flux Eq 21-23 (L252-278) with readings S8-S13 of DESIGN.md; n_0 gate and mask
// (L280-284, S14); angular flux Eq 19 (L239-241) upwinded on the total normal angular velocity (S5).
//
// Design: one thread owns one (column (i,j), direction s) pair and marches along x^3.  The
// geometry of every built-in metric is x^3-independent, so all per-(face, s) coefficients (sqrt(-g) n^a_f, n_{0,f},
// gate) are formed ONCE per thread from 12-double per-column face rows and stay in registers for the whole march;
// the x^3 stencil lives in a 5-deep register window; x^1/x^2 neighbours are coalesced loads (s fastest, 32 lanes =
// 256 contiguous bytes) served by L1/L2.
#include <cmath>

#include "rt_transport_dev.cuh"

namespace rt {
namespace {

// ---- per-face, direction-independent coefficients of Eq 23 ---------------------------------------------------
// fcoef[a][face] = (1/2 e^-tau, 1/2 f(tau), (1-e^-tau) wL, (1-e^-tau) wR); vacuum face (tau == 0): y = -1.
__global__ void k_facecoef(KParams p, const double *__restrict__ T, double dt, int a, double4 *__restrict__ out) {
    const int e1 = p.n1 + (a == 0), e2 = p.n2 + (a == 1), e3 = p.n3 + (a == 2);
    long long f = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    if (f >= (long long)e1 * e2 * e3) return;
    int q[3] = {int(f % e1), int((f / e1) % e2), int(f / ((long long)e1 * e2))};
    const int N[3] = {p.n1, p.n2, p.n3};
    long long cell[4];
    for (int o = -2; o <= 1; ++o) {   // cells L-1, L, R, R+1 with R = q
        int c[3] = {q[0], q[1], q[2]};
        c[a] = fluid_idx(q[a] + o, N[a], p.bc_lo[a], p.bc_hi[a]);
        cell[o + 2] = ((long long)c[2] * p.n2 + c[1]) * p.n1 + c[0];
    }
    const double aL = alpha_total(p, p.rho[cell[1]], T[cell[1]]), aR = alpha_total(p, p.rho[cell[2]], T[cell[2]]);
    const double tau = p.abar * 0.5 * (aL + aR) * dt;
    double4 r;
    if (tau == 0.0) {
        r = make_double4(0.5, -1.0, 0.0, 0.0);
    } else {
        const double et = exp(-tau);
        const double ft = sqrt(-expm1(-tau * tau)) * __drcp_rn(tau);   // f(tau) = sqrt(1 - e^(-tau^2)) / tau
        double v[4];
        for (int o = 0; o < 4; ++o)
            v[o] = mirror_sign(q[a] + o - 2, N[a], p.bc_lo[a], p.bc_hi[a]) * (p.u4[(1 + a) * p.ncell + cell[o]] * __drcp_rn(p.u4[cell[o]]));   // (reciprocal, not a division)
        const double vL = v[1] + 0.5 * slope_rt(p.limiter, v[1] - v[0], v[2] - v[1]);
        const double vR = v[2] - 0.5 * slope_rt(p.limiter, v[2] - v[1], v[3] - v[2]);
        double wL, wR;
        if (vL > 0 && vR > 0) { wL = vL; wR = 0.0; }
        else if (vL < 0 && vR < 0) { wL = 0.0; wR = vR; }
        else { wL = vL; wR = vR; }
        r = make_double4(0.5 * et, 0.5 * ft, (1.0 - et) * wL, (1.0 - et) * wR);
    }
    out[f] = r;
}


// column flags: bit 0 = the column has a cell with a non-vacuum face, bit 1 = it has an all-vacuum cell
// column masks (32-bit words behind the flags, colmask_offset()): bit (k & 31) of word [(k >> 5) * ncol + col] = cell
// flag of (col, k).  The marching kernels test a bit per step and load one word per 32 steps: a per-step flag load sat
// in front of every step's branch and exposed its L2 latency (it was 70 % of the vacuum kernel's long-scoreboard stalls).
// One warp per column, lane = x3 index within a 32-cell word: the cell flags (any of the six faces non-vacuum) are formed
// from the face coefficients and go straight into the ballot that makes the mask word; no per-cell flag array.
__global__ void k_colflag(KParams p, const double4 *__restrict__ fc0, const double4 *__restrict__ fc1,
                          const double4 *__restrict__ fc2, unsigned char *__restrict__ colflag) {
    const int col = (int)((blockIdx.x * (long long)blockDim.x + threadIdx.x) >> 5), lane = threadIdx.x & 31;
    if (col >= p.ncol) return;
    const int i = col % p.n1, j = col / p.n1;
    unsigned *cmask = reinterpret_cast<unsigned *>(colflag + colmask_offset(p.ncol, p.n3));
    int m = 0;
    for (int k0 = 0; k0 < p.n3; k0 += 32) {
        const int k = k0 + lane;
        const bool in = k < p.n3;
        bool f = false;
        if (in) {
            const long long x = ((long long)k * p.n2 + j) * (p.n1 + 1) + i, y = ((long long)k * (p.n2 + 1) + j) * p.n1 + i,
                            c = (long long)k * p.ncol + col;
            f = fc0[x].y >= 0 || fc0[x + 1].y >= 0 || fc1[y].y >= 0 || fc1[y + p.n1].y >= 0 || fc2[c].y >= 0 || fc2[c + p.ncol].y >= 0;
        }
        const unsigned mw = __ballot_sync(0xffffffffu, f), valid = __ballot_sync(0xffffffffu, in);
        if (mw) m |= 1;
        if (valid & ~mw) m |= 2;
        if (lane == 0) cmask[(long long)(k0 >> 5) * p.ncol + col] = mw;
    }
    if (lane == 0) colflag[col] = (unsigned char)m;
}

// ---- spatial transport ------------------------------------------------------------------------------------------
// One thread = one (column, s); marches x3.  The work is split over two kernels that write disjoint (cell, s) sets:
//   k_transport_vac  all-vacuum cells (Eq 20 on all six faces) of threads whose n^a has one sign across the cell:
//                    lean upwind path, carried x3 flux, software-pipelined loads;
//   k_transport_gen  everything else: cells with a non-vacuum (Eq 23) face, threads with a sign change of n^a
//                    inside the cell, threads next to a ZERO / FIXED boundary.
// Block order of the marching kernels: a 1-D grid walked in bands of TILE_ROWS x2-rows with x2 fastest inside a band,
// so that the CTAs resident at the same time cover a compact (x1, x2) patch and their transverse neighbours are
// read from L2 instead of DRAM (row-major order re-reads ~4 halo rows per wave of ~5 rows).
// how many x3-planes beyond its two-plane register pipeline the angular kernel prefetches (0 = off)
constexpr int ANG_PF = 4;
// how many x3-planes beyond the register pipeline the vacuum kernel prefetches its operands (0 = off)
constexpr int VAC_PF = 2;
constexpr int TILE_ROWS = 24;
constexpr int VAC_THREADS = 128, VAC_MINB = 5;
__device__ __forceinline__ void tile_block(const KParams &p, int &bx, int &by) {
    const int nbx = (p.n1 * p.pitch + (int)blockDim.x - 1) / (int)blockDim.x;
    const int lin = blockIdx.x, band = lin / (nbx * TILE_ROWS), r = lin - band * nbx * TILE_ROWS;
    const int th = min(TILE_ROWS, p.n2 - band * TILE_ROWS);
    bx = r / th;
    by = band * TILE_ROWS + (r - bx * th);
}


// Per-(column, s) class byte, computed once at rt_init: bit 0 = dead (pad lane, masked direction, zero band in x1/x2),
// bit 1 = general (sign change of n^a inside the cell, or next to a ZERO / FIXED boundary).  Both transport kernels
// read it, so they always agree on which of them owns a thread.
__global__ void k_classify(const __grid_constant__ KParams p, unsigned char *__restrict__ cls) {
    const int e = blockIdx.x * blockDim.x + threadIdx.x;
    if (e >= p.n1 * p.pitch) return;
    ColSetup c;
    col_setup(p, 1.0, c, e / p.pitch, blockIdx.y, e % p.pitch);
    cls[(long long)c.col * p.pitch + c.s] = (unsigned char)((c.dead ? 1 : 0) | (c.general ? 2 : 0));
}

// Upwind path for vacuum faces (Eq 20): the flux only needs the UPWIND PLI state, and the upwind side of a face is a
// per-thread constant (the sign of n^a_f).  With (a, b, c, d) = four cells of a dim ordered along the propagation
// direction (c = this cell) the flux difference is K_bc S_bc + K_cd S_cd, S_bc = b + slope(b-a, c-b)/2,
// S_cd = c + slope(c-b, d-c)/2: 3 loads and 2 slopes per transverse dim; x3: 1 load, 1 slope, the lower flux carried.
template <int LIM, bool MATTER, bool SAME_BASE>
__global__ void __launch_bounds__(VAC_THREADS, VAC_MINB)
k_transport_vac(const __grid_constant__ KParams p, const double *__restrict__ I_in, const double *I_base, double *I_out,
                const unsigned char *__restrict__ colflag, double dt) {
    int bx, by;
    tile_block(p, bx, by);
    const int e0 = bx * blockDim.x + threadIdx.x;
    if (e0 >= p.n1 * p.pitch) return;
    const long long kstride = (long long)p.ncol * p.pitch;
    const int n3 = p.n3, ncol = p.ncol;
    {
        const long long q = (long long)by * p.n1 * p.pitch + e0;
        const int cl = p.cls[q];
        if (cl & 1) {   // dead: this kernel keeps those entries zero
            for (int k = 0; k < n3; ++k) I_out[q + k * kstride] = 0.0;
            return;
        }
        if (cl & 2) return;
        if (MATTER && !(colflag[by * p.n1 + e0 / p.pitch] & 2)) return;
    }
    ColSetup c;
    col_setup(p, dt, c, e0 / p.pitch, by, e0 % p.pitch);
    const long long pos0 = (long long)c.col * p.pitch + c.s;
    double *out = I_out + pos0;
    const int i = c.i, j = c.j, s = c.s;
    const bool xpos = c.xl.pos, ypos = c.yl.pos, zpos = c.zf.pos;
    const int oxa = xpos ? c.oxm2 : c.oxp2, oxb = xpos ? c.oxm1 : c.oxp1, oxd = xpos ? c.oxp1 : c.oxm1;
    const int oya = ypos ? c.oym2 : c.oyp2, oyb = ypos ? c.oym1 : c.oyp1, oyd = ypos ? c.oyp1 : c.oym1;
    const double Kxbc = xpos ? -c.xl.A : c.xh.A, Kxcd = xpos ? c.xh.A : -c.xl.A;
    const double Kybc = ypos ? -c.yl.A : c.yh.A, Kycd = ypos ? c.yh.A : -c.yl.A;
    const double zA = c.zf.A, zhalf = zpos ? 0.5 : -0.5;
    const double *pk = I_in + pos0;
    auto ldk = [&](int kk) -> double {
        return (kk >= 0 && kk < n3) ? __ldg(pk + kk * kstride) : slow_ld(p, I_in, 2, i, j, kk, s);
    };
    double w1 = ldk(-1), w2 = ldk(0), w3 = ldk(1), Flo;
    {
        const double w0 = ldk(-2);
        const double sg = slope_k<LIM>(w2 - w1, zpos ? (w1 - w0) : (w3 - w2));
        Flo = zA * fma(zhalf, sg, zpos ? w1 : w2);
    }
    const double *pb = I_base + pos0;
    const unsigned *pmask = reinterpret_cast<const unsigned *>(colflag + colmask_offset(ncol, n3)) + c.col;
    const int zlo = p.zlo[2], zhi = n3 - p.zhi[2];
    unsigned mcur = MATTER ? __ldg(pmask) : 0u, mnext = (MATTER && n3 > 32) ? __ldg(pmask + ncol) : 0u;
    double qxa = __ldg(pk + oxa), qxb = __ldg(pk + oxb), qxd = __ldg(pk + oxd);
    double qya = __ldg(pk + oya), qyb = __ldg(pk + oyb), qyd = __ldg(pk + oyd);
    double qw4 = ldk(2);
    double qbase = SAME_BASE ? 0.0 : *pb;
    for (int k = 0; k < n3; ++k) {
        const double xa = qxa, xb = qxb, xd = qxd, ya = qya, yb = qyb, yd = qyd, w4 = qw4, cbase = qbase;
        const bool mat = MATTER && ((mcur >> (k & 31)) & 1u);
        if (k + 1 < n3) {   // request the operands of step k + 1 before computing step k
            const double *pn = pk + kstride;
            if (!SAME_BASE) qbase = pb[kstride];
            qxa = __ldg(pn + oxa); qxb = __ldg(pn + oxb); qxd = __ldg(pn + oxd);
            qya = __ldg(pn + oya); qyb = __ldg(pn + oyb); qyd = __ldg(pn + oyd);
            qw4 = (k + 3 < n3) ? __ldg(pn + 2 * kstride) : slow_ld(p, I_in, 2, i, j, k + 3, s);
            if (k + VAC_PF + 1 < n3) {   // operands of step k + 1 + VAC_PF: pulled towards the SM now (no registers held)
                const double *pf = pn + VAC_PF * kstride;
                pf_l1(pf + oxa); pf_l1(pf + oxb); pf_l1(pf + oxd);
                pf_l1(pf + oya); pf_l1(pf + oyb); pf_l1(pf + oyd);
                if (k + VAC_PF + 3 < n3) pf_l1(pf + 2 * kstride);
                if (!SAME_BASE) pf_l1(pb + (VAC_PF + 1) * kstride);
            }
        }
        // x3: upwind state at the upper face (always formed: it is the next cell's lower flux if that cell is vacuum)
        const double sz = slope_k<LIM>(w3 - w2, zpos ? (w2 - w1) : (w4 - w3));
        const double Fhi = zA * fma(zhalf, sz, zpos ? w2 : w3);
        if (!mat) {
            double D = Fhi - Flo;
            {
                const double d1 = xb - xa, d2 = w2 - xb, d3 = xd - w2;
                D = fma(Kxbc, fma(0.5, slope_k<LIM>(d1, d2), xb), D);
                D = fma(Kxcd, fma(0.5, slope_k<LIM>(d2, d3), w2), D);
            }
            {
                const double d1 = yb - ya, d2 = w2 - yb, d3 = yd - w2;
                D = fma(Kybc, fma(0.5, slope_k<LIM>(d1, d2), yb), D);
                D = fma(Kycd, fma(0.5, slope_k<LIM>(d2, d3), w2), D);
            }
            const double base = SAME_BASE ? w2 : cbase;
            *out = base - D;      // Eq 18 (O5), dt/(n^0 n_0 sqrt(-g) dx) folded in; the x3 zero band is reset below
        }
        Flo = Fhi;
        w1 = w2; w2 = w3; w3 = w4;
        pk += kstride; pb += kstride; out += kstride;
        if (MATTER && (k & 31) == 31) {   // next mask word (requested 32 steps ago)
            mcur = mnext;
            pmask += ncol;
            mnext = (k + 33 < n3) ? __ldg(pmask + ncol) : 0u;
        }
    }
    if (zlo > 0 || zhi < n3) {   // zero band in x3 (L709): reset after the march instead of a select in every step
        double *o = I_out + pos0;
        for (int k = 0; k < n3; ++k)
            if (k < zlo || k >= zhi) o[k * kstride] = 0.0;
    }
}

// General path: full 5-point stencils, both PLI states at all six faces, Eq 20 or Eq 23 per face.  Marches x3 with a
// 5-deep register window; computes only the steps it owns (cells with a non-vacuum face, or every cell of a
// "general" thread).
constexpr int GEN_THREADS = 128, GEN_MINB = 4;   // 128 x 4 and 256 x 2 hold the same 16 warps per SM at 128 registers; the smaller CTA is 1-2 % faster
template <int LIM, bool MATTER, bool LIST>
__global__ void __launch_bounds__(GEN_THREADS, GEN_MINB)
k_transport_gen(const __grid_constant__ KParams p, const double *__restrict__ I_in, const double *I_base, double *I_out,
                const double4 *__restrict__ fc0, const double4 *__restrict__ fc1, const double4 *__restrict__ fc2,
                const unsigned char *__restrict__ colflag, double dt) {
    // LIST = false: the non-general threads of columns that hold a cell with a non-vacuum face (grid over (i, s) x j).
    // LIST = true:  the "general" (column, s) pairs, from the compact list built at rt_init (one thread per entry).
    int ci, cj, cs;
    const bool general = LIST;
    if (LIST) {
        const int t = blockIdx.x * blockDim.x + threadIdx.x;
        if (t >= p.ngen) return;
        const int q = p.genlist[t];
        const int col = q / p.pitch;
        cs = q - col * p.pitch; ci = col % p.n1; cj = col / p.n1;
    } else {
        int bx, by;
        tile_block(p, bx, by);
        const int e0 = bx * blockDim.x + threadIdx.x;
        if (e0 >= p.n1 * p.pitch) return;
        if (p.cls[(long long)by * p.n1 * p.pitch + e0] != 0) return;      // dead or general
        ci = e0 / p.pitch; cs = e0 - ci * p.pitch; cj = by;
        if (!(MATTER && (colflag[cj * p.n1 + ci] & 1))) return;
    }
    ColSetup c;
    col_setup(p, dt, c, ci, cj, cs);
    const int i = c.i, j = c.j, s = c.s, n3 = p.n3, ncol = p.ncol, n1 = p.n1;
    // the list kernel splits x3 into gridDim.y chunks (few threads: more of them in flight); the column kernel marches all of it
    const int kchunk = LIST ? (n3 + (int)gridDim.y - 1) / (int)gridDim.y : n3;
    const int k0 = LIST ? (int)blockIdx.y * kchunk : 0, k1 = min(n3, k0 + kchunk);
    if (k0 >= k1) return;
    const long long kstride = (long long)ncol * p.pitch;
    const long long pos0 = (long long)c.col * p.pitch + s;
    const double *pin = I_in + pos0;
    const double *pk = pin + k0 * kstride;
    const double4 vac = make_double4(0.5, -1.0, 0.0, 0.0);
    auto ldk = [&](int kk) -> double {
        return (kk >= 0 && kk < n3) ? __ldg(pin + kk * kstride) : slow_ld(p, I_in, 2, i, j, kk, s);
    };
    double w0 = ldk(k0 - 2), w1 = ldk(k0 - 1), w2 = ldk(k0), w3 = ldk(k0 + 1);
    const double *pb = I_base + pos0 + k0 * kstride;
    double *out = I_out + pos0 + k0 * kstride;
    const bool same_base = (I_base == I_in);
    const int sx = p.n2 * (n1 + 1), sy = (p.n2 + 1) * n1;
    const unsigned *pmask = reinterpret_cast<const unsigned *>(colflag + colmask_offset(ncol, n3)) + c.col + (long long)(k0 >> 5) * ncol;
    const double4 *px = fc0 + ((long long)j * (n1 + 1) + i) + (long long)k0 * sx, *py = fc1 + ((long long)j * n1 + i) + (long long)k0 * sy,
                  *pz = fc2 + c.col + (long long)k0 * ncol;
    const int zlo = p.zlo[2], zhi = n3 - p.zhi[2];
    const bool special = c.special;
    // software pipeline: transverse neighbours, x3 look-ahead and cell flag of step k+1 are requested during step k
    // (special threads load through slow_ld inside the step instead)
    const int oxm2 = special ? 0 : c.oxm2, oxm1 = special ? 0 : c.oxm1, oxp1 = special ? 0 : c.oxp1, oxp2 = special ? 0 : c.oxp2;
    const int oym2 = special ? 0 : c.oym2, oym1 = special ? 0 : c.oym1, oyp1 = special ? 0 : c.oyp1, oyp2 = special ? 0 : c.oyp2;
    double qxm2 = __ldg(pk + oxm2), qxm1 = __ldg(pk + oxm1), qxp1 = __ldg(pk + oxp1), qxp2 = __ldg(pk + oxp2);
    double qym2 = __ldg(pk + oym2), qym1 = __ldg(pk + oym1), qyp1 = __ldg(pk + oyp1), qyp2 = __ldg(pk + oyp2);
    double qw4 = ldk(k0 + 2);
    double qbase = same_base ? 0.0 : *pb;
    unsigned mcur = MATTER ? __ldg(pmask) : 0u, mnext = (MATTER && (k0 | 31) + 1 < k1) ? __ldg(pmask + ncol) : 0u;
    for (int k = k0; k < k1; ++k) {
        double xm2 = qxm2, xm1 = qxm1, xp1 = qxp1, xp2 = qxp2, ym2 = qym2, ym1 = qym1, yp1 = qyp1, yp2 = qyp2;
        const double w4 = qw4, cbase = qbase;
        const bool mat = MATTER && ((mcur >> (k & 31)) & 1u);
        if (k + 1 < k1) {
            if (!same_base) qbase = pb[kstride];
            const double *pn = pk + kstride;
            qxm2 = __ldg(pn + oxm2); qxm1 = __ldg(pn + oxm1); qxp1 = __ldg(pn + oxp1); qxp2 = __ldg(pn + oxp2);
            qym2 = __ldg(pn + oym2); qym1 = __ldg(pn + oym1); qyp1 = __ldg(pn + oyp1); qyp2 = __ldg(pn + oyp2);
            qw4 = (k + 3 < n3) ? __ldg(pn + 2 * kstride) : slow_ld(p, I_in, 2, i, j, k + 3, s);
            if (MATTER) {
                // the per-face coefficients of the next step: pulled into L1 now (no registers held), so that the
                // ld4() of step k+1 do not expose an L2 round trip in front of the flux evaluation
                asm volatile("prefetch.global.L1 [%0];" ::"l"(px + sx));
                asm volatile("prefetch.global.L1 [%0];" ::"l"(py + sy));
                asm volatile("prefetch.global.L1 [%0];" ::"l"(py + sy + n1));
                asm volatile("prefetch.global.L1 [%0];" ::"l"(pz + 2 * ncol));
            }
        }
        if (mat || general) {
            if (special) {
                xm2 = slow_ld(p, I_in, 0, i - 2, j, k, s); xm1 = slow_ld(p, I_in, 0, i - 1, j, k, s);
                xp1 = slow_ld(p, I_in, 0, i + 1, j, k, s); xp2 = slow_ld(p, I_in, 0, i + 2, j, k, s);
                ym2 = slow_ld(p, I_in, 1, i, j - 2, k, s); ym1 = slow_ld(p, I_in, 1, i, j - 1, k, s);
                yp1 = slow_ld(p, I_in, 1, i, j + 1, k, s); yp2 = slow_ld(p, I_in, 1, i, j + 2, k, s);
            }
            double D;
            if (mat) {
                D = flux_diff<LIM, MATTER>(w0, w1, w2, w3, w4, c.zf, c.zf, ld4(pz), ld4(pz + ncol));
                D += flux_diff<LIM, MATTER>(xm2, xm1, w2, xp1, xp2, c.xl, c.xh, ld4(px), ld4(px + 1));
                D += flux_diff<LIM, MATTER>(ym2, ym1, w2, yp1, yp2, c.yl, c.yh, ld4(py), ld4(py + n1));
            } else {
                D = flux_diff<LIM, false>(w0, w1, w2, w3, w4, c.zf, c.zf, vac, vac);
                D += flux_diff<LIM, false>(xm2, xm1, w2, xp1, xp2, c.xl, c.xh, vac, vac);
                D += flux_diff<LIM, false>(ym2, ym1, w2, yp1, yp2, c.yl, c.yh, vac, vac);
            }
            const double base = same_base ? w2 : cbase;
            *out = (k < zlo || k >= zhi) ? 0.0 : base - D;
        }
        w0 = w1; w1 = w2; w2 = w3; w3 = w4;
        pk += kstride; pb += kstride; out += kstride; px += sx; py += sy; pz += ncol;
        if (MATTER && (k & 31) == 31) {   // next mask word (requested 32 steps ago)
            mcur = mnext;
            pmask += ncol;
            mnext = (k + 33 < k1) ? __ldg(pmask + ncol) : 0u;
        }
    }
}

// ---- angular flux (donor cell) ------------------------------------------------------------------------------------
// One block per column; thread s keeps its 7 coefficients in registers over the x3 march; the cell's N_d intensities
// are staged in shared memory for the neighbour gather.  Two planes per barrier, stored INTERLEAVED ([s][plane]): thread s
// writes its two values with one 16-byte store and takes each neighbour's two values with one 16-byte load; every shared
// address is a 32-bit shared-space offset formed once (the first version spent 27 % of its instructions on generic-address
// and stride arithmetic, 190 per two planes for 16 fp64 operations, and issued at 66 % while moving 5.2 TB/s).
__device__ __forceinline__ double2 lds2(unsigned addr) {
    double2 v;
    asm volatile("ld.shared.v2.f64 {%0, %1}, [%2];" : "=d"(v.x), "=d"(v.y) : "r"(addr));
    return v;
}
__device__ __forceinline__ void sts2(unsigned addr, double a, double b) {
    asm volatile("st.shared.v2.f64 [%0], {%1, %2};" ::"r"(addr), "d"(a), "d"(b) : "memory");
}
// TB: upper bound of the block size (a bucket: 256 covers up to 256 directions, 1024 the rest); the small bucket is held to 64
// registers (both buckets: four blocks of 256, one of 1024)
template <int TB>
__global__ void __launch_bounds__(TB, TB <= 256 ? 4 : 1) k_angular(KParams p, const double *__restrict__ I_in, double *I_io, double dt) {
    extern __shared__ __align__(16) double sI[];   // [2 buffers][pitch][2 planes]
    const int s = threadIdx.x, col = blockIdx.x;
    const int i = col % p.n1, j = col / p.n1;
    const bool live = s < p.nd;
    double c[ANG_SLOTS];
    unsigned ga[6];
    const unsigned sb = (unsigned)__cvta_generic_to_shared(sI), own = sb + 16u * (unsigned)s, BB = 16u * (unsigned)p.pitch;
    double scale = 0.0;
    bool zero = true;
#pragma unroll
    for (int e = 0; e < 6; ++e) ga[e] = own;
#pragma unroll
    for (int e = 0; e < ANG_SLOTS; ++e) c[e] = 0.0;
    if (live) {
        const double nx = p.nhat[s], ny = p.nhat[p.pitch + s], nz = p.nhat[2 * p.pitch + s];
        const double *cen = p.cen + (long long)col * CEN_STRIDE;
        const double n0c = centre_n0(cen, nx, ny, nz);
        const double nup = cen[4] + cen[5] * nx + cen[6] * ny + cen[7] * nz;
        scale = dt / (nup * n0c);
        const bool band_ij = (i < p.zlo[0] || i >= p.n1 - p.zhi[0] || j < p.zlo[1] || j >= p.n2 - p.zhi[1]);
        zero = band_ij || n0c > -p.n0_floor;
        for (int e = 0; e < ANG_SLOTS; ++e) c[e] = p.angcoef[((long long)col * ANG_SLOTS + e) * p.pitch + s];
        for (int e = 0; e < 6; ++e) ga[e] = sb + 16u * (unsigned)p.nb[e * p.pitch + s];
    }
    const long long kstride = (long long)p.n1 * p.n2 * p.pitch;
    const bool inrow = s < p.pitch;
    const double *pin = I_in + (long long)col * p.pitch + s;
    double *pio = I_io + (long long)col * p.pitch + s;
    // software pipeline over x3, two planes per barrier: the operands of planes k+2, k+3 are requested before planes
    // k, k+1 are computed; the staged cells are double-buffered in shared memory
    const bool upd = live && !zero;
    const int n3 = p.n3, klo = p.zlo[2], khi = n3 - p.zhi[2];   // planes [klo, khi) are not in the x3 zero band
    const long long o2 = 2 * kstride, o3 = 3 * kstride, o4 = (2 + ANG_PF) * kstride, o5 = (3 + ANG_PF) * kstride;
    double v0 = inrow ? __ldg(pin) : 0.0, v1 = (inrow && 1 < n3) ? __ldg(pin + kstride) : 0.0;
    double io0 = upd ? *pio : 0.0, io1 = (upd && 1 < n3) ? pio[kstride] : 0.0;
    unsigned boff = 0;
    for (int k = 0; k < n3; k += 2) {
        const bool two = k + 1 < n3;
        if (inrow) sts2(own + boff, v0, v1);
        double vn0 = 0.0, vn1 = 0.0, ion0 = 0.0, ion1 = 0.0;
        if (k + 2 < n3) {
            if (inrow) vn0 = __ldg(pin + o2);
            if (upd) ion0 = pio[o2];
            if (k + 3 < n3) {
                if (inrow) vn1 = __ldg(pin + o3);
                if (upd) ion1 = pio[o3];
            }
            if (k + 2 + ANG_PF + 1 < n3) {   // planes further ahead: towards the SM now, no registers held
                if (inrow) { pf_l1(pin + o4); pf_l1(pin + o5); }
                if (upd) { pf_l1(pio + o4); pf_l1(pio + o5); }
            }
        }
        __syncthreads();
        if (live) {
            double D0 = c[6] * v0, D1 = c[6] * v1;
#pragma unroll
            for (int e = 0; e < 6; ++e) {
                const double2 g = lds2(ga[e] + boff);
                D0 += c[e] * g.x; D1 += c[e] * g.y;
            }
            const bool w0 = !zero && k >= klo && k < khi, w1 = !zero && k + 1 >= klo && k + 1 < khi;
            pio[0] = w0 ? io0 - scale * D0 : 0.0;
            if (two) pio[kstride] = w1 ? io1 - scale * D1 : 0.0;
        } else if (inrow) {
            pio[0] = 0.0;
            if (two) pio[kstride] = 0.0;
        }
        v0 = vn0; v1 = vn1; io0 = ion0; io1 = ion1;
        pin += o2; pio += o2;
        boff ^= BB;
    }
}

}  // namespace

// ---- launchers ---------------------------------------------------------------------------------------------------
cudaError_t launch_facecoef(const KParams &p, const double *T, double dt, double *fcoef[3], unsigned char *colflag,
                            cudaStream_t st, long long *launches) {
    for (int a = 0; a < 3; ++a) {
        long long nf = (long long)(p.n1 + (a == 0)) * (p.n2 + (a == 1)) * (p.n3 + (a == 2));
        k_facecoef<<<(unsigned)((nf + 255) / 256), 256, 0, st>>>(p, T, dt, a, reinterpret_cast<double4 *>(fcoef[a]));
        ++*launches;
    }
    k_colflag<<<(unsigned)(((long long)p.ncol * 32 + 127) / 128), 128, 0, st>>>(p, reinterpret_cast<const double4 *>(fcoef[0]),
                                                                                   reinterpret_cast<const double4 *>(fcoef[1]),
                                                                                   reinterpret_cast<const double4 *>(fcoef[2]), colflag);
    *launches += 1;
    return cudaGetLastError();
}

template <int LIM>
static void launch_transport_lim(const KParams &p, const double *I_in, const double *I_base, double *I_out,
                                 double *const fcoef[3], const unsigned char *colflag, bool matter, bool tiled,
                                 double dt, cudaStream_t st) {
    dim3 grid(((p.n1 * p.pitch + GEN_THREADS - 1) / GEN_THREADS) * p.n2);   // walked in tiles, see tile_block()
    dim3 gvac(((p.n1 * p.pitch + VAC_THREADS - 1) / VAC_THREADS) * p.n2);
    const double4 *f0 = reinterpret_cast<const double4 *>(fcoef[0]), *f1 = reinterpret_cast<const double4 *>(fcoef[1]),
                  *f2 = reinterpret_cast<const double4 *>(fcoef[2]);
    if (matter) {
        if (!tiled) {
            if (I_base == I_in) k_transport_vac<LIM, true, true><<<gvac, VAC_THREADS, 0, st>>>(p, I_in, I_base, I_out, colflag, dt);
            else k_transport_vac<LIM, true, false><<<gvac, VAC_THREADS, 0, st>>>(p, I_in, I_base, I_out, colflag, dt);
        }
        if (!tiled) k_transport_gen<LIM, true, false><<<grid, GEN_THREADS, 0, st>>>(p, I_in, I_base, I_out, f0, f1, f2, colflag, dt);
        if (p.ngen) k_transport_gen<LIM, true, true><<<dim3((p.ngen + 127) / 128, 8), 128, 0, st>>>(p, I_in, I_base, I_out, f0, f1, f2, colflag, dt);
    } else {
        if (!tiled) {
            if (I_base == I_in) k_transport_vac<LIM, false, true><<<gvac, VAC_THREADS, 0, st>>>(p, I_in, I_base, I_out, colflag, dt);
            else k_transport_vac<LIM, false, false><<<gvac, VAC_THREADS, 0, st>>>(p, I_in, I_base, I_out, colflag, dt);
        }
        if (p.ngen) k_transport_gen<LIM, false, true><<<dim3((p.ngen + 127) / 128, 8), 128, 0, st>>>(p, I_in, I_base, I_out, f0, f1, f2, colflag, dt);
    }
}

cudaError_t launch_transport(const KParams &p, const double *I_in, const double *I_base, double *I_out,
                             double *const fcoef[3], const unsigned char *colflag, bool matter,
                             double dt, cudaStream_t st, long long *launches) {
    const bool tiled = p.variant == RT_TRANSPORT_TMA;
    if (tiled) {   // the non-"general" pairs through the two tile kernels: vacuum cells, then the cells with an Eq 23 face
        cudaError_t e = launch_transport_tile(p, p.tile, I_in, I_base, I_out, colflag, matter, dt, st, launches);
        if (e == cudaSuccess && matter) e = launch_transport_tile_gen(p, I_in, I_base, I_out, fcoef, colflag, dt, st, launches);
        if (e != cudaSuccess) return e;
    }
    switch (p.limiter) {
        case RT_LIM_MC: launch_transport_lim<RT_LIM_MC>(p, I_in, I_base, I_out, fcoef, colflag, matter, tiled, dt, st); break;
        case RT_LIM_MINMOD: launch_transport_lim<RT_LIM_MINMOD>(p, I_in, I_base, I_out, fcoef, colflag, matter, tiled, dt, st); break;
        case RT_LIM_NONE: launch_transport_lim<RT_LIM_NONE>(p, I_in, I_base, I_out, fcoef, colflag, matter, tiled, dt, st); break;
        default: launch_transport_lim<RT_LIM_VANLEER>(p, I_in, I_base, I_out, fcoef, colflag, matter, tiled, dt, st); break;
    }
    *launches += (tiled ? 0 : 1 + (matter ? 1 : 0)) + (p.ngen ? 1 : 0);
    return cudaGetLastError();
}

// ---- rt_transport_static: the transport launch with its per-stage scratch in a file-scope device array ------------------
// For callers that cannot call cudaMalloc (CUDA graph capture, tight serving loops).  The scratch of one transport launch --
// the per-face coefficients of Eq 23 for the three dims and the column / cell flags -- lives in this array instead of the
// context's cudaMalloc'ed buffers.  Every GPU that loads the library holds RT_STATIC_SCRATCH_BYTES until exit.  All calls
// share it and it keeps the last call's contents: k_facecoef and k_colflag overwrite every entry the transport kernels read
// (nothing has to start at zero), and two calls that overlap on the GPU (different streams, no ordering) race on it.
static __device__ __align__(256) unsigned char g_static_scratch[RT_STATIC_SCRATCH_BYTES];

// In host code `g_static_scratch` is a host-side stand-in, not a device address: the address the kernels get comes from
// cudaGetSymbolAddress, resolved once per device with that device current.
static cudaError_t static_scratch_ptr(unsigned char **out) {
    static unsigned char *cache[64] = {nullptr};
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    if (dev < 0 || dev >= 64) return cudaErrorInvalidDevice;
    if (!cache[dev]) {
        void *q = nullptr;
        e = cudaGetSymbolAddress(&q, g_static_scratch);
        if (e != cudaSuccess) return e;
        cache[dev] = static_cast<unsigned char *>(q);
    }
    *out = cache[dev];
    return cudaSuccess;
}

static size_t align256(size_t v) { return (v + 255) & ~(size_t)255; }
size_t transport_static_bytes(const KParams &p, bool matter) {
    if (!matter) return 0;
    size_t need = 0;
    for (int a = 0; a < 3; ++a) need += align256((size_t)(p.n1 + (a == 0)) * (p.n2 + (a == 1)) * (p.n3 + (a == 2)) * sizeof(double4));
    return need + align256(colflag_bytes(p.ncol, p.n3));
}

// cudaErrorMemoryValueTooLarge: the mesh needs more scratch than the array holds.  No cudaMalloc / cudaFree / allocating
// library call on this path.
cudaError_t launch_transport_static(const KParams &p, const double *T, const double *I_in, const double *I_base, double *I_out,
                                    bool matter, double dt, cudaStream_t st, long long *launches) {
    if (transport_static_bytes(p, matter) > RT_STATIC_SCRATCH_BYTES) return cudaErrorMemoryValueTooLarge;
    double *fcoef[3] = {nullptr, nullptr, nullptr};
    unsigned char *colflag = nullptr;
    if (matter) {
        unsigned char *base = nullptr;
        cudaError_t e = static_scratch_ptr(&base);
        if (e != cudaSuccess) return e;
        size_t off = 0;
        for (int a = 0; a < 3; ++a) {
            fcoef[a] = reinterpret_cast<double *>(base + off);
            off += align256((size_t)(p.n1 + (a == 0)) * (p.n2 + (a == 1)) * (p.n3 + (a == 2)) * sizeof(double4));
        }
        colflag = base + off;
        e = launch_facecoef(p, T, dt, fcoef, colflag, st, launches);
        if (e != cudaSuccess) return e;
    }
    return launch_transport(p, I_in, I_base, I_out, fcoef, colflag, matter, dt, st, launches);
}

cudaError_t launch_classify(const KParams &p, unsigned char *cls, cudaStream_t st) {
    dim3 grid((p.n1 * p.pitch + 255) / 256, p.n2);
    k_classify<<<grid, 256, 0, st>>>(p, cls);
    return cudaGetLastError();
}

cudaError_t launch_angular(const KParams &p, const double *I_in, double *I_io, double dt, cudaStream_t st, long long *launches) {
    const int threads = ((p.pitch + 31) / 32) * 32;
    if (threads <= 256) k_angular<256><<<p.ncol, threads, 4 * p.pitch * sizeof(double), st>>>(p, I_in, I_io, dt);   // [2 buffers][pitch][2 planes]
    else k_angular<1024><<<p.ncol, threads, 4 * p.pitch * sizeof(double), st>>>(p, I_in, I_io, dt);
    ++*launches;
    return cudaGetLastError();
}

}  // namespace rt
