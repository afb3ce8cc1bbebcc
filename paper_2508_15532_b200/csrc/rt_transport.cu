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

#include "rt_kernels.cuh"

namespace rt {
namespace {

__device__ __forceinline__ double minmod3(double a, double b, double c) {
    if (a > 0 && b > 0 && c > 0) return fmin(a, fmin(b, c));
    if (a < 0 && b < 0 && c < 0) return fmax(a, fmax(b, c));
    return 0.0;
}
template <int LIM>
__device__ __forceinline__ double slope(double dm, double dp) {
    if (LIM == RT_LIM_MC) return minmod3(2.0 * dm, 0.5 * (dm + dp), 2.0 * dp);
    if (LIM == RT_LIM_MINMOD) return (dm * dp > 0) ? (fabs(dm) < fabs(dp) ? dm : dp) : 0.0;
    if (LIM == RT_LIM_NONE) return 0.0;
    return (dm * dp > 0) ? 2.0 * dm * dp / (dm + dp) : 0.0;
}
__device__ __forceinline__ double slope_rt(int lim, double dm, double dp) {
    switch (lim) {
        case RT_LIM_MC: return slope<RT_LIM_MC>(dm, dp);
        case RT_LIM_MINMOD: return slope<RT_LIM_MINMOD>(dm, dp);
        case RT_LIM_NONE: return 0.0;
        default: return slope<RT_LIM_VANLEER>(dm, dp);
    }
}

// index of a fluid cell along one dim: periodic wraps, reflecting mirrors, everything else clamps (fluid ghosts)
__device__ __forceinline__ int fluid_idx(int c, int N, int bc_lo, int bc_hi) {
    if (c < 0) return bc_lo == RT_BC_PERIODIC ? ((c % N) + N) % N : (bc_lo == RT_BC_REFLECT ? -1 - c : 0);
    if (c >= N) return bc_hi == RT_BC_PERIODIC ? c % N : (bc_hi == RT_BC_REFLECT ? 2 * N - 1 - c : N - 1);
    return c;
}
// -1 for a mirror-image cell behind a reflecting boundary (its normal velocity is reversed), else +1
__device__ __forceinline__ double mirror_sign(int c, int N, int bc_lo, int bc_hi) {
    return ((c < 0 && bc_lo == RT_BC_REFLECT) || (c >= N && bc_hi == RT_BC_REFLECT)) ? -1.0 : 1.0;
}
__device__ __forceinline__ double alpha_total(const KParams &p, double rho, double T) {
    if (rho < p.rho_floor) return 0.0;   // L468 (i)
    double aa = (p.kappa_a0 != 0.0) ? p.kappa_a0 * rho * rho * pow(T, -3.5) : 0.0;
    return aa + p.kappa_s * rho;
}

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
        const double ft = sqrt(-expm1(-tau * tau) / (tau * tau));
        double v[4];
        for (int o = 0; o < 4; ++o)
            v[o] = mirror_sign(q[a] + o - 2, N[a], p.bc_lo[a], p.bc_hi[a]) * (p.u4[(1 + a) * p.ncell + cell[o]] / p.u4[cell[o]]);
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

// ---- intensity access with boundary conditions ----------------------------------------------------------------
// Base pointer of the direction vector of cell (i,j,k) where the index along dim a may be up to 2 out of range.
// nullptr = zero ghost.
__device__ __forceinline__ const double *cell_ptr(const KParams &p, const double *I, int a, int i, int j, int k) {
    int q[3] = {i, j, k};
    const int N = (a == 0) ? p.n1 : (a == 1) ? p.n2 : p.n3;
    int c = q[a];
    if (c < 0 || c >= N) {
        const int bc = (c < 0) ? p.bc_lo[a] : p.bc_hi[a];
        if (bc == RT_BC_PERIODIC) q[a] = ((c % N) + N) % N;   // N may be 1 or 2: a single wrap is not enough
        else if (bc == RT_BC_OUTFLOW) q[a] = (c < 0) ? 0 : N - 1;
        else if (bc == RT_BC_ZERO) return nullptr;
        else if (bc == RT_BC_REFLECT) q[a] = (c < 0) ? (-1 - c) : (2 * N - 1 - c);   // mirror image (slow_ld flips the direction)
        else {
            const int layer = (c < 0) ? (-1 - c) : (c - N), side = (c < 0) ? 0 : 1;
            long long fc, nface;
            if (a == 0) { fc = (long long)k * p.n2 + j; nface = (long long)p.n2 * p.n3; }
            else if (a == 1) { fc = (long long)k * p.n1 + i; nface = (long long)p.n1 * p.n3; }
            else { fc = (long long)j * p.n1 + i; nface = (long long)p.n1 * p.n2; }
            const double *g = p.ghost[a][side];
            return g ? g + (layer * nface + fc) * p.pitch : nullptr;
        }
    }
    return I + (((long long)q[2] * p.n2 + q[1]) * p.n1 + q[0]) * p.pitch;
}
__device__ __forceinline__ double ldI(const double *base, int s) { return base ? __ldg(base + s) : 0.0; }
__device__ __forceinline__ double4 ld4(const double4 *q) {
    const double2 a = __ldg(reinterpret_cast<const double2 *>(q)), b = __ldg(reinterpret_cast<const double2 *>(q) + 1);
    return make_double4(a.x, a.y, b.x, b.y);
}

struct FaceC { double P, Q, Z; };   // sqrt(-g) n^a_f, n_{0,f} (0 if gated or dead), sqrt(-g) n^0_f
__device__ __forceinline__ FaceC face_coef(const double *__restrict__ f, double nx, double ny, double nz) {
    FaceC c;
    c.P = f[0] + f[1] * nx + f[2] * ny + f[3] * nz;
    c.Q = f[4] + f[5] * nx + f[6] * ny + f[7] * nz;
    c.Z = f[8] + f[9] * nx + f[10] * ny + f[11] * nz;
    return c;
}
__device__ __forceinline__ double centre_n0(const double *__restrict__ c, double nx, double ny, double nz) {
    return c[0] + c[1] * nx + c[2] * ny + c[3] * nz;
}
__device__ __forceinline__ bool sign_differs(double a, double b) {
    return ((a > 0) - (a < 0)) != ((b > 0) - (b < 0));
}

// Monotonised-central slope, same value as minmod3(2 dm, (dm+dp)/2, 2 dp) bit for bit, with 5 fp64-pipe operations:
// equal signs => sign * min(2 min(|dm|,|dp|), |dm+dp|/2); opposite signs or a zero difference => 0.
__device__ __forceinline__ double slope_mc(double dm, double dp) {
    // With s = dm + dp and t = |dm| - |dp|:  |s| - |t| = 2 min(|dm|, |dp|) when dm, dp have equal signs and exactly 0
    // when they differ (then |s| and |t| are the same IEEE subtraction), so
    //     MC = copysign( min(|s| - |t|, |s| / 2), s )
    // needs no sign test and no zeroing select: 4 fp64 operations, one compare, two selects, one sign copy.  The
    // equal-sign identity holds to one rounding of s (1e-16 of max(|dm|,|dp|)), inside the parity budget.
    const double s = dm + dp;
    const double t = fabs(dm) - fabs(dp);
    const double m2 = fabs(s) - fabs(t);
    const double c = 0.5 * fabs(s);
    const double r = (m2 < c) ? m2 : c;
    return copysign(r, s);
}
template <int LIM>
__device__ __forceinline__ double slope_k(double dm, double dp) {
    return (LIM == RT_LIM_MC) ? slope_mc(dm, dp) : slope<LIM>(dm, dp);
}

// Per-face coefficients of one (column, s), with dt / (n^0 n_0 sqrt(-g_c) dx^a) folded in, so that
// I_out = I_base - sum_faces (+-) flux.   A = [..] n_0f sqrt(-g_f) n^a_f,  Zq = [..] n_0f sqrt(-g_f) n^0_f.
struct FaceK { double A, Zq; bool pos; };
__device__ __forceinline__ FaceK fold(const FaceC &c, double scale) {
    FaceK k;
    k.A = c.Q * c.P * scale;
    k.Zq = c.Q * c.Z * scale;
    k.pos = c.P > 0;
    return k;
}
// flux through one face.  IL/IR: PLI states; Il/Ir: cell-centre values left/right of the face.
template <bool MATTER>
__device__ __forceinline__ double face_flux(const FaceK &c, double IL, double IR, double Il, double Ir, const double4 &fc) {
    if (!MATTER || fc.y < 0.0) return c.A * (c.pos ? IL : IR);                                     // Eq 20
    const double B = c.pos ? c.A : -c.A;                                                           // [..] n_0 |n^a|
    return c.A * fc.x * (IL + IR) - B * fc.y * (Ir - Il) + c.Zq * (fc.z * IL + fc.w * IR);          // Eq 23
}
// flux difference of one transverse dim from the 5-point stencil (m2, m1, c0, p1, p2)
template <int LIM, bool MATTER>
__device__ __forceinline__ double flux_diff(double m2, double m1, double c0, double p1, double p2, const FaceK &lo,
                                            const FaceK &hi, const double4 &fclo, const double4 &fchi) {
    const double d0 = m1 - m2, d1 = c0 - m1, d2 = p1 - c0, d3 = p2 - p1;
    const double sm = slope_k<LIM>(d0, d1), s0 = slope_k<LIM>(d1, d2), sp = slope_k<LIM>(d2, d3);
    const double Flo = face_flux<MATTER>(lo, m1 + 0.5 * sm, c0 - 0.5 * s0, m1, c0, fclo);
    const double Fhi = face_flux<MATTER>(hi, c0 + 0.5 * s0, p1 - 0.5 * sp, c0, p1, fchi);
    return Fhi - Flo;
}

// generic (boundary-aware) load, kept out of line: only threads next to a ZERO / FIXED boundary come here
__device__ __noinline__ double slow_ld(const KParams &p, const double *I, int a, int i, int j, int k, int s) {
    // reflecting boundary (x2 only): the mirror image holds the direction with n-hat^2 flipped
    if (a == 1 && ((j < 0 && p.bc_lo[1] == RT_BC_REFLECT) || (j >= p.n2 && p.bc_hi[1] == RT_BC_REFLECT))) s = p.mirror[s];
    return ldI(cell_ptr(p, I, a, i, j, k), s);
}
// neighbour of coordinate c0 at offset d along a dim of extent N: interior index after periodic wrap / outflow
// clamp, or -1 if it is a ZERO / FIXED ghost
__device__ __forceinline__ int nb_index(int c, int N, int bc_lo, int bc_hi) {
    if (c >= 0 && c < N) return c;
    const int bc = (c < 0) ? bc_lo : bc_hi;
    if (bc == RT_BC_PERIODIC) return ((c % N) + N) % N;
    if (bc == RT_BC_OUTFLOW) return (c < 0) ? 0 : N - 1;
    return -1;
}

// column flags: bit 0 = the column has a cell with a non-vacuum face, bit 1 = it has an all-vacuum cell
// colflag[ncol + kc * ncol + col]: the x3 chunk [kc*GEN_KC, (kc+1)*GEN_KC) of the column has such a cell
// column masks (32-bit words behind the flags, colmask_offset()): bit (k & 31) of word [(k >> 5) * ncol + col] = cell
// flag of (col, k).  The marching kernels test a bit per step and load one word per 32 steps: a per-step flag load sat
// in front of every step's branch and exposed its L2 latency (it was 70 % of the vacuum kernel's long-scoreboard stalls).
constexpr int GEN_KC = 8;
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
        const int kc = (k0 / GEN_KC) + lane;   // lanes 0..3: the four x3 chunks of this word
        if (lane < 32 / GEN_KC && kc * GEN_KC < p.n3)
            colflag[p.ncol + (long long)kc * p.ncol + col] = ((mw >> (GEN_KC * lane)) & ((1u << GEN_KC) - 1u)) ? 1 : 0;
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
#ifndef ANG_PF
#define ANG_PF 2
#endif
// how many x3-planes beyond the register pipeline the vacuum kernel prefetches its operands (0 = off)
#ifndef VAC_PF
#define VAC_PF 2
#endif
__device__ __forceinline__ void pf_l1(const void *q) { asm volatile("prefetch.global.L1 [%0];" ::"l"(q)); }
constexpr int TILE_ROWS = 24;
#ifndef VAC_THREADS
#define VAC_THREADS 128
#define VAC_MINB 5
#endif
__device__ __forceinline__ void tile_block(const KParams &p, int &bx, int &by) {
    const int nbx = (p.n1 * p.pitch + (int)blockDim.x - 1) / (int)blockDim.x;
    const int lin = blockIdx.x, band = lin / (nbx * TILE_ROWS), r = lin - band * nbx * TILE_ROWS;
    const int th = min(TILE_ROWS, p.n2 - band * TILE_ROWS);
    bx = r / th;
    by = band * TILE_ROWS + (r - bx * th);
}

struct ColSetup {
    int i, j, s, col;
    bool dead, special, general;
    FaceK xl, xh, yl, yh, zf;
    int oxm2, oxm1, oxp1, oxp2, oym2, oym1, oyp1, oyp2;
};
__device__ __forceinline__ bool col_setup(const KParams &p, double dt, ColSetup &c, int i, int j, int s) {
    c.i = i; c.j = j; c.s = s;
    c.col = j * p.n1 + i;
    c.dead = s >= p.nd;   // pad lanes: keep the pad zero
    c.special = c.general = false;
    if (c.dead) return true;
    const double nx = __ldg(p.nhat + s), ny = __ldg(p.nhat + p.pitch + s), nz = __ldg(p.nhat + 2 * p.pitch + s);
    const double *cen = p.cen + (long long)c.col * CEN_STRIDE;
    const double n0c = centre_n0(cen, nx, ny, nz);
    const double nup = cen[4] + cen[5] * nx + cen[6] * ny + cen[7] * nz;
    const double scale = dt * cen[8] / (nup * n0c);
    const bool band_ij = (i < p.zlo[0] || i >= p.n1 - p.zhi[0] || j < p.zlo[1] || j >= p.n2 - p.zhi[1]);
    c.dead = band_ij || n0c > -p.n0_floor;   // masked direction (S14) or zero band (L709): stays zero, no work
    if (c.dead) return true;
    // transverse neighbours: element offsets inside the x3-plane, resolved once (periodic / outflow map to interior
    // cells); a ZERO / FIXED ghost makes the thread use the generic loader
    const int im2 = nb_index(i - 2, p.n1, p.bc_lo[0], p.bc_hi[0]), im1 = nb_index(i - 1, p.n1, p.bc_lo[0], p.bc_hi[0]);
    const int ip1 = nb_index(i + 1, p.n1, p.bc_lo[0], p.bc_hi[0]), ip2 = nb_index(i + 2, p.n1, p.bc_lo[0], p.bc_hi[0]);
    const int jm2 = nb_index(j - 2, p.n2, p.bc_lo[1], p.bc_hi[1]), jm1 = nb_index(j - 1, p.n2, p.bc_lo[1], p.bc_hi[1]);
    const int jp1 = nb_index(j + 1, p.n2, p.bc_lo[1], p.bc_hi[1]), jp2 = nb_index(j + 2, p.n2, p.bc_lo[1], p.bc_hi[1]);
    c.special = (im2 | im1 | ip1 | ip2 | jm2 | jm1 | jp1 | jp2) < 0;
    const int rowp = p.n1 * p.pitch;
    c.oxm2 = (im2 - i) * p.pitch; c.oxm1 = (im1 - i) * p.pitch; c.oxp1 = (ip1 - i) * p.pitch; c.oxp2 = (ip2 - i) * p.pitch;
    c.oym2 = (jm2 - j) * rowp; c.oym1 = (jm1 - j) * rowp; c.oyp1 = (jp1 - j) * rowp; c.oyp2 = (jp2 - j) * rowp;
    // face coefficients, formed once per column (geometry is x3-independent); n_0 gate (L280) applied here
    const double sx = scale * p.inv_dx[0], sy = scale * p.inv_dx[1], sz = scale * p.inv_dx[2];
    FaceC f;
    int in;
    f = face_coef(p.face[0] + ((long long)j * (p.n1 + 1) + i) * FACE_STRIDE, nx, ny, nz);
    in = (i > 0) ? i - 1 : (p.bc_lo[0] == RT_BC_PERIODIC ? p.n1 - 1 : -1);
    if (in >= 0 && sign_differs(n0c, centre_n0(p.cen + ((long long)j * p.n1 + in) * CEN_STRIDE, nx, ny, nz))) f.Q = 0.0;
    c.xl = fold(f, sx);
    f = face_coef(p.face[0] + ((long long)j * (p.n1 + 1) + i + 1) * FACE_STRIDE, nx, ny, nz);
    in = (i < p.n1 - 1) ? i + 1 : (p.bc_hi[0] == RT_BC_PERIODIC ? 0 : -1);
    if (in >= 0 && sign_differs(n0c, centre_n0(p.cen + ((long long)j * p.n1 + in) * CEN_STRIDE, nx, ny, nz))) f.Q = 0.0;
    c.xh = fold(f, sx);
    f = face_coef(p.face[1] + ((long long)j * p.n1 + i) * FACE_STRIDE, nx, ny, nz);
    in = (j > 0) ? j - 1 : (p.bc_lo[1] == RT_BC_PERIODIC ? p.n2 - 1 : -1);
    if (in >= 0 && sign_differs(n0c, centre_n0(p.cen + ((long long)in * p.n1 + i) * CEN_STRIDE, nx, ny, nz))) f.Q = 0.0;
    c.yl = fold(f, sy);
    f = face_coef(p.face[1] + ((long long)(j + 1) * p.n1 + i) * FACE_STRIDE, nx, ny, nz);
    in = (j < p.n2 - 1) ? j + 1 : (p.bc_hi[1] == RT_BC_PERIODIC ? 0 : -1);
    if (in >= 0 && sign_differs(n0c, centre_n0(p.cen + ((long long)in * p.n1 + i) * CEN_STRIDE, nx, ny, nz))) f.Q = 0.0;
    c.yh = fold(f, sy);
    c.zf = fold(face_coef(p.face[2] + (long long)c.col * FACE_STRIDE, nx, ny, nz), sz);
    c.general = c.special || (c.xl.pos != c.xh.pos) || (c.yl.pos != c.yh.pos);
    return true;
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
#if VAC_PF
            if (k + VAC_PF + 1 < n3) {   // operands of step k + 1 + VAC_PF: pulled towards the SM now (no registers held)
                const double *pf = pn + VAC_PF * kstride;
                pf_l1(pf + oxa); pf_l1(pf + oxb); pf_l1(pf + oxd);
                pf_l1(pf + oya); pf_l1(pf + oyb); pf_l1(pf + oyd);
                if (k + VAC_PF + 3 < n3) pf_l1(pf + 2 * kstride);
                if (!SAME_BASE) pf_l1(pb + (VAC_PF + 1) * kstride);
            }
#endif
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

// The same upwind path with the x2 stencil staged in shared memory.  k_transport_vac asks L2 for seven operands per
// cell-direction and step (L1 hit rate 14 %: the transverse neighbours belong to CTAs on other SMs) and is bound by the
// L2 -> L1 traffic that causes (6.4 GB per launch for 2 GB of compulsory DRAM traffic, lts / l1tex throughput 66-70 %).
// Here a CTA owns YS_TY consecutive x2-rows x 32 consecutive entries of the row (one warp per row) and keeps a ring of
// three x3-planes of that patch plus its two halo rows on each side in shared memory: the value every thread loads
// for its own x3 window (plane k + 2) is also stored into the ring, each warp loads one halo row, and the three x2
// operands of step k are read from the ring two steps later.  L2 requests per cell-direction and step: own + halo
// (4 / YS_TY) + three x1 operands = 5 instead of 7.  One barrier per step (4 warps).  Threads the kernel does not
// compute for (dead, general, matter-only columns, rows beyond n2) still load and store their row: they are the
// neighbours' operands.
constexpr int YS_TY = 4;
template <int LIM, bool MATTER, bool SAME_BASE>
__global__ void __launch_bounds__(32 * YS_TY, VAC_MINB)
k_transport_vac_ys(const __grid_constant__ KParams p, const double *__restrict__ I_in, const double *I_base, double *I_out,
                   const unsigned char *__restrict__ colflag, double dt) {
    static_assert(YS_TY == 4, "one halo row per warp: four warps, four halo rows");
    __shared__ double tile[3][YS_TY + 4][32];
    const int lane = threadIdx.x & 31, ty = threadIdx.x >> 5;
    // block -> (bx: 32-entry segment of the row, bg: group of YS_TY rows), bands of TILE_ROWS rows as in tile_block()
    const int rowlen = p.n1 * p.pitch;
    const int nbx = (rowlen + 31) / 32, ngy = (p.n2 + YS_TY - 1) / YS_TY;
    constexpr int GB = TILE_ROWS / YS_TY;
    const int lin = blockIdx.x, band = lin / (nbx * GB), rr = lin - band * nbx * GB;
    const int th = min(GB, ngy - band * GB);
    const int bx = rr / th, bg = band * GB + (rr - bx * th);
    const int e0 = bx * 32 + lane, j0 = bg * YS_TY, j = j0 + ty;
    const bool inrow = e0 < rowlen;
    const long long kstride = (long long)p.ncol * p.pitch;
    const int n3 = p.n3, ncol = p.ncol;
    // loader rows: the own slot (tile row ty + 2) and one halo slot (tile rows 0, 1, YS_TY + 2, YS_TY + 3)
    const int hr = (ty < 2) ? ty : YS_TY + ty;
    const int jown = nb_index(j, p.n2, p.bc_lo[1], p.bc_hi[1]), jhalo = nb_index(j0 - 2 + hr, p.n2, p.bc_lo[1], p.bc_hi[1]);
    const double *pown = (inrow && jown >= 0) ? I_in + (long long)jown * rowlen + e0 : nullptr;
    const double *phalo = (inrow && jhalo >= 0) ? I_in + (long long)jhalo * rowlen + e0 : nullptr;
    // role of the thread
    bool compute = inrow && j < p.n2;
    if (compute) {
        const long long q = (long long)j * rowlen + e0;
        const int cl = p.cls[q];
        if (cl & 1) {   // dead: this kernel keeps those entries zero
            for (int k = 0; k < n3; ++k) I_out[q + k * kstride] = 0.0;
            compute = false;
        } else if (cl & 2) {
            compute = false;
        } else if (MATTER && !(colflag[j * p.n1 + e0 / p.pitch] & 2)) {
            compute = false;
        }
    }
    ColSetup c;
    c.col = 0; c.s = 0; c.i = 0; c.j = 0;
    c.xl = c.xh = c.yl = c.yh = c.zf = FaceK{0.0, 0.0, true};
    c.oxm2 = c.oxm1 = c.oxp1 = c.oxp2 = 0;
    if (compute) col_setup(p, dt, c, e0 / p.pitch, j, e0 % p.pitch);
    const long long pos0 = compute ? (long long)c.col * p.pitch + c.s : 0;
    double *out = I_out + pos0;
    const int i = c.i, s = c.s;
    const bool xpos = c.xl.pos, ypos = c.yl.pos, zpos = c.zf.pos;
    const int oxa = xpos ? c.oxm2 : c.oxp2, oxb = xpos ? c.oxm1 : c.oxp1, oxd = xpos ? c.oxp1 : c.oxm1;
    const double Kxbc = xpos ? -c.xl.A : c.xh.A, Kxcd = xpos ? c.xh.A : -c.xl.A;
    const double Kybc = ypos ? -c.yl.A : c.yh.A, Kycd = ypos ? c.yh.A : -c.yl.A;
    const double zA = c.zf.A, zhalf = zpos ? 0.5 : -0.5;
    // tile rows of the x2 operands (a, b: two and one cell upwind, d: one cell downwind)
    const double *tya = &tile[0][ty + 2 + (ypos ? -2 : 2)][lane], *tyb = &tile[0][ty + 2 + (ypos ? -1 : 1)][lane],
                 *tyd = &tile[0][ty + 2 + (ypos ? 1 : -1)][lane];
    double *town = &tile[0][ty + 2][lane], *thalo = &tile[0][hr][lane];
    constexpr int SLOT = (YS_TY + 4) * 32;   // doubles per ring slot
    const double *pk = I_in + pos0;          // compute threads only
    // own-row value of plane kk: the x3 window of a compute thread (with the x3 boundary behind it) and the ring entry
    auto ldown = [&](int kk) -> double {
        if (kk >= 0 && kk < n3) return pown ? __ldg(pown + kk * kstride) : 0.0;
        return compute ? slow_ld(p, I_in, 2, i, j, kk, s) : 0.0;
    };
    auto ldhalo = [&](int kk) -> double { return (phalo && kk < n3) ? __ldg(phalo + kk * kstride) : 0.0; };
    double w1 = ldown(-1), w2 = ldown(0), w3 = ldown(1), Flo;
    {
        const double w0 = ldown(-2);
        const double sg = slope_k<LIM>(w2 - w1, zpos ? (w1 - w0) : (w3 - w2));
        Flo = zA * fma(zhalf, sg, zpos ? w1 : w2);
    }
    // ring prologue: planes 0 and 1
    town[0] = w2; thalo[0] = ldhalo(0);
    town[SLOT] = w3; thalo[SLOT] = ldhalo(1);
    __syncthreads();
    const double *pb = I_base + pos0;
    const unsigned *pmask = reinterpret_cast<const unsigned *>(colflag + colmask_offset(ncol, n3)) + c.col;
    const int zlo = p.zlo[2], zhi = n3 - p.zhi[2];
    unsigned mcur = (MATTER && compute) ? __ldg(pmask) : 0u, mnext = (MATTER && compute && n3 > 32) ? __ldg(pmask + ncol) : 0u;
    // Prefetch plan: the rows the warp will ask for VAC_PF steps later (own row and halo row at plane k + VAC_PF + 3,
    // the four x1-neighbour rows and the base state at plane k + VAC_PF + 1) are 18 lines of 128 bytes; lane l asks for
    // line l, one prefetch instruction per step instead of six per lane.  pfp: the lane's line at step 0.
    const char *pfp = nullptr;
    int pf_kend = 0;   // the lane prefetches while k < pf_kend
#if VAC_PF
    {
        const unsigned cm = __ballot_sync(0xffffffffu, compute);
        const int lead = cm ? __ffs(cm) - 1 : 0;
        const bool nxm2 = __any_sync(0xffffffffu, compute && xpos), nxp2 = __any_sync(0xffffffffu, compute && !xpos);
        int off[4] = {c.oxm2, c.oxm1, c.oxp1, c.oxp2};
#pragma unroll
        for (int r = 0; r < 4; ++r) off[r] = __shfl_sync(0xffffffffu, off[r], lead);
        const long long lead_el = __shfl_sync(0xffffffffu, pos0, lead) - lead;   // plane-0 element of the warp's first entry (own row)
        if (lane < 2) {            // own row, plane k + VAC_PF + 3
            if (pown) { pfp = reinterpret_cast<const char *>(pown - lane + (VAC_PF + 3) * kstride) + 128 * lane; pf_kend = n3 - VAC_PF - 3; }
        } else if (lane < 4) {     // halo row
            if (phalo) { pfp = reinterpret_cast<const char *>(phalo - lane + (VAC_PF + 3) * kstride) + 128 * (lane - 2); pf_kend = n3 - VAC_PF - 3; }
        } else if (lane < 16) {    // x1 neighbours of the compute lanes, plane k + VAC_PF + 1
            const int r = (lane - 4) / 3, q = (lane - 4) - 3 * r;
            const bool need = cm != 0u && ((r == 0) ? nxm2 : (r == 3) ? nxp2 : true);
            const int o = (r == 0) ? off[0] : (r == 1) ? off[1] : (r == 2) ? off[2] : off[3];
            if (need) {
                const long long el = ((lead_el + o) & ~15LL) + 16 * q + (VAC_PF + 1) * kstride;
                pfp = reinterpret_cast<const char *>(I_in + el); pf_kend = n3 - VAC_PF - 1;
            }
        } else if (!SAME_BASE && lane < 18) {
            if (cm != 0u) { pfp = reinterpret_cast<const char *>(I_base + (lead_el & ~15LL) + 16 * (lane - 16) + (VAC_PF + 1) * kstride); pf_kend = n3 - VAC_PF - 1; }
        }
    }
#endif
    const long long kbytes = kstride * (long long)sizeof(double);
    // software pipeline: the operands of step k + 1 are requested before step k is computed
    double qxa = 0.0, qxb = 0.0, qxd = 0.0, qbase = 0.0;
    if (compute) {
        qxa = __ldg(pk + oxa); qxb = __ldg(pk + oxb); qxd = __ldg(pk + oxd);
        if (!SAME_BASE) qbase = *pb;
    }
    double qw4 = ldown(2), qh4 = ldhalo(2);
    int rd = 0, wr = 2 * SLOT;   // ring offsets (doubles) of plane k and plane k + 2
#pragma unroll 1
    for (int k = 0; k < n3; ++k) {
        const double xa = qxa, xb = qxb, xd = qxd, w4 = qw4, cbase = qbase;
        const bool mat = MATTER && ((mcur >> (k & 31)) & 1u);
        town[wr] = w4; thalo[wr] = qh4;   // plane k + 2 into the ring (read by the neighbours at step k + 2)
        if (k + 1 < n3) {
            qw4 = ldown(k + 3); qh4 = ldhalo(k + 3);
            if (compute) {
                const double *pn = pk + kstride;
                if (!SAME_BASE) qbase = pb[kstride];
                qxa = __ldg(pn + oxa); qxb = __ldg(pn + oxb); qxd = __ldg(pn + oxd);
            }
#if VAC_PF
            if (k < pf_kend) pf_l1(pfp);
#endif
        }
        pfp += kbytes;
        if (compute) {
            // x3: upwind state at the upper face (always formed: it is the next cell's lower flux if that cell is vacuum)
            const double sz = slope_k<LIM>(w3 - w2, zpos ? (w2 - w1) : (w4 - w3));
            const double Fhi = zA * fma(zhalf, sz, zpos ? w2 : w3);
            if (!mat) {
                const double ya = tya[rd], yb = tyb[rd], yd = tyd[rd];
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
            pk += kstride; pb += kstride; out += kstride;
            if (MATTER && (k & 31) == 31) {   // next mask word (requested 32 steps ago)
                mcur = mnext;
                pmask += ncol;
                mnext = (k + 33 < n3) ? __ldg(pmask + ncol) : 0u;
            }
        }
        w1 = w2; w2 = w3; w3 = w4;
        rd = (rd == 2 * SLOT) ? 0 : rd + SLOT;
        wr = (wr == 2 * SLOT) ? 0 : wr + SLOT;
        __syncthreads();
    }
    if (compute && (zlo > 0 || zhi < n3)) {   // zero band in x3 (L709): reset after the march instead of a select in every step
        double *o = I_out + pos0;
        for (int k = 0; k < n3; ++k)
            if (k < zlo || k >= zhi) o[k * kstride] = 0.0;
    }
}

// General path: full 5-point stencils, both PLI states at all six faces, Eq 20 or Eq 23 per face.  Marches x3 with a
// 5-deep register window; computes only the steps it owns (cells with a non-vacuum face, or every cell of a
// "general" thread).
#ifndef GEN_THREADS
#define GEN_THREADS 128   // 128 x 4 and 256 x 2 hold the same 16 warps per SM at 128 registers; the smaller CTA is 1-2 % faster
#define GEN_MINB 4
#endif
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
// are staged in shared memory for the neighbour gather.
__global__ void k_angular(KParams p, const double *__restrict__ I_in, double *I_io, double dt) {
    extern __shared__ double sI[];
    const int s = threadIdx.x, col = blockIdx.x;
    const int i = col % p.n1, j = col / p.n1;
    const bool live = s < p.nd;
    double c[ANG_SLOTS];
    int nb[6];
    double scale = 0.0;
    bool zero = true;
    if (live) {
        const double nx = p.nhat[s], ny = p.nhat[p.pitch + s], nz = p.nhat[2 * p.pitch + s];
        const double *cen = p.cen + (long long)col * CEN_STRIDE;
        const double n0c = centre_n0(cen, nx, ny, nz);
        const double nup = cen[4] + cen[5] * nx + cen[6] * ny + cen[7] * nz;
        scale = dt / (nup * n0c);
        const bool band_ij = (i < p.zlo[0] || i >= p.n1 - p.zhi[0] || j < p.zlo[1] || j >= p.n2 - p.zhi[1]);
        zero = band_ij || n0c > -p.n0_floor;
        for (int e = 0; e < ANG_SLOTS; ++e) c[e] = p.angcoef[((long long)col * ANG_SLOTS + e) * p.pitch + s];
        for (int e = 0; e < 6; ++e) nb[e] = p.nb[e * p.pitch + s];
    }
    const long long kstride = (long long)p.n1 * p.n2 * p.pitch;
    const bool inrow = s < p.pitch;
    const double *pin = I_in + (long long)col * p.pitch + s;
    double *pio = I_io + (long long)col * p.pitch + s;
    // software pipeline over x3, two planes per barrier: the operands of planes k+2, k+3 are requested before planes
    // k, k+1 are computed; the staged cells are double-buffered in shared memory (4 x pitch doubles)
    const bool upd = live && !zero;
    const int n3 = p.n3;
    double v0 = inrow ? __ldg(pin) : 0.0, v1 = (inrow && 1 < n3) ? __ldg(pin + kstride) : 0.0;
    double io0 = upd ? *pio : 0.0, io1 = (upd && 1 < n3) ? pio[kstride] : 0.0;
    for (int k = 0; k < n3; k += 2) {
        double *buf0 = sI + ((k >> 1) & 1) * 2 * p.pitch, *buf1 = buf0 + p.pitch;
        const bool two = k + 1 < n3;
        if (inrow) { buf0[s] = v0; buf1[s] = v1; }
        double vn0 = 0.0, vn1 = 0.0, ion0 = 0.0, ion1 = 0.0;
        if (k + 2 < n3) {
            if (inrow) vn0 = __ldg(pin + 2 * kstride);
            if (upd) ion0 = pio[2 * kstride];
            if (k + 3 < n3) {
                if (inrow) vn1 = __ldg(pin + 3 * kstride);
                if (upd) ion1 = pio[3 * kstride];
            }
#if ANG_PF
            if (k + 2 + ANG_PF + 1 < n3) {   // planes further ahead: towards the SM now, no registers held
                if (inrow) { pf_l1(pin + (2 + ANG_PF) * kstride); pf_l1(pin + (3 + ANG_PF) * kstride); }
                if (upd) { pf_l1(pio + (2 + ANG_PF) * kstride); pf_l1(pio + (3 + ANG_PF) * kstride); }
            }
#endif
        }
        __syncthreads();
        if (live) {
            double D0 = c[6] * v0, D1 = c[6] * v1;
#pragma unroll
            for (int e = 0; e < 6; ++e) { D0 += c[e] * buf0[nb[e]]; D1 += c[e] * buf1[nb[e]]; }
            const bool b0 = (k < p.zlo[2] || k >= n3 - p.zhi[2]), b1 = (k + 1 < p.zlo[2] || k + 1 >= n3 - p.zhi[2]);
            pio[0] = (zero || b0) ? 0.0 : io0 - scale * D0;
            if (two) pio[kstride] = (zero || b1) ? 0.0 : io1 - scale * D1;
        } else if (inrow) {
            pio[0] = 0.0;
            if (two) pio[kstride] = 0.0;
        }
        v0 = vn0; v1 = vn1; io0 = ion0; io1 = ion1;
        pin += 2 * kstride; pio += 2 * kstride;
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
                                 double *const fcoef[3], const unsigned char *colflag, bool matter,
                                 double dt, cudaStream_t st) {
    dim3 grid(((p.n1 * p.pitch + GEN_THREADS - 1) / GEN_THREADS) * p.n2);   // walked in tiles, see tile_block()
    dim3 gvac(((p.n1 * p.pitch + VAC_THREADS - 1) / VAC_THREADS) * p.n2);
    dim3 gys(((p.n1 * p.pitch + 31) / 32) * ((p.n2 + YS_TY - 1) / YS_TY));   // RT_TRANSPORT_SMEM_X2
    const double4 *f0 = reinterpret_cast<const double4 *>(fcoef[0]), *f1 = reinterpret_cast<const double4 *>(fcoef[1]),
                  *f2 = reinterpret_cast<const double4 *>(fcoef[2]);
    if (matter) {
        if (I_base == I_in) { if (p.vac_smem) k_transport_vac_ys<LIM, true, true><<<gys, 32 * YS_TY, 0, st>>>(p, I_in, I_base, I_out, colflag, dt); else k_transport_vac<LIM, true, true><<<gvac, VAC_THREADS, 0, st>>>(p, I_in, I_base, I_out, colflag, dt); }
        else { if (p.vac_smem) k_transport_vac_ys<LIM, true, false><<<gys, 32 * YS_TY, 0, st>>>(p, I_in, I_base, I_out, colflag, dt); else k_transport_vac<LIM, true, false><<<gvac, VAC_THREADS, 0, st>>>(p, I_in, I_base, I_out, colflag, dt); }
        k_transport_gen<LIM, true, false><<<grid, GEN_THREADS, 0, st>>>(p, I_in, I_base, I_out, f0, f1, f2, colflag, dt);
        if (p.ngen) k_transport_gen<LIM, true, true><<<dim3((p.ngen + 127) / 128, 8), 128, 0, st>>>(p, I_in, I_base, I_out, f0, f1, f2, colflag, dt);
    } else {
        if (I_base == I_in) { if (p.vac_smem) k_transport_vac_ys<LIM, false, true><<<gys, 32 * YS_TY, 0, st>>>(p, I_in, I_base, I_out, colflag, dt); else k_transport_vac<LIM, false, true><<<gvac, VAC_THREADS, 0, st>>>(p, I_in, I_base, I_out, colflag, dt); }
        else { if (p.vac_smem) k_transport_vac_ys<LIM, false, false><<<gys, 32 * YS_TY, 0, st>>>(p, I_in, I_base, I_out, colflag, dt); else k_transport_vac<LIM, false, false><<<gvac, VAC_THREADS, 0, st>>>(p, I_in, I_base, I_out, colflag, dt); }
        if (p.ngen) k_transport_gen<LIM, false, true><<<dim3((p.ngen + 127) / 128, 8), 128, 0, st>>>(p, I_in, I_base, I_out, f0, f1, f2, colflag, dt);
    }
}

cudaError_t launch_transport(const KParams &p, const double *I_in, const double *I_base, double *I_out,
                             double *const fcoef[3], const unsigned char *colflag, bool matter,
                             double dt, cudaStream_t st, long long *launches) {
    switch (p.limiter) {
        case RT_LIM_MC: launch_transport_lim<RT_LIM_MC>(p, I_in, I_base, I_out, fcoef, colflag, matter, dt, st); break;
        case RT_LIM_MINMOD: launch_transport_lim<RT_LIM_MINMOD>(p, I_in, I_base, I_out, fcoef, colflag, matter, dt, st); break;
        case RT_LIM_NONE: launch_transport_lim<RT_LIM_NONE>(p, I_in, I_base, I_out, fcoef, colflag, matter, dt, st); break;
        default: launch_transport_lim<RT_LIM_VANLEER>(p, I_in, I_base, I_out, fcoef, colflag, matter, dt, st); break;
    }
    *launches += 1 + (matter ? 1 : 0) + (p.ngen ? 1 : 0);
    return cudaGetLastError();
}

cudaError_t launch_classify(const KParams &p, unsigned char *cls, cudaStream_t st) {
    dim3 grid((p.n1 * p.pitch + 255) / 256, p.n2);
    k_classify<<<grid, 256, 0, st>>>(p, cls);
    return cudaGetLastError();
}

cudaError_t launch_angular(const KParams &p, const double *I_in, double *I_io, double dt, cudaStream_t st, long long *launches) {
    const int threads = ((p.pitch + 31) / 32) * 32;
    k_angular<<<p.ncol, threads, 4 * p.pitch * sizeof(double), st>>>(p, I_in, I_io, dt);
    ++*launches;
    return cudaGetLastError();
}

}  // namespace rt
