// Device helpers shared by the transport kernels of librt_b200 (rt_transport.cu, rt_transport_tile.cu): limiters, boundary
// index maps, per-(column, s) face coefficients.  PAPER.md: PLI reconstruction L225 (S7), Eq 20 (L245), Eq 21-23
// (L252-278, S8-S13), n_0 gate and mask L280-284 (S14), Eq 18 (L193).
#pragma once
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
    double aa = 0.0;
    if (p.kappa_a0 != 0.0) {   // T^-3.5 = (1/T)^3 sqrt(1/T): a reciprocal and a square root instead of pow() (~100 instructions)
        const double r = __drcp_rn(T);
        aa = p.kappa_a0 * rho * rho * (r * r * r * sqrt(r));
    }
    return aa + p.kappa_s * rho;
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

__device__ __forceinline__ void pf_l1(const void *q) { asm volatile("prefetch.global.L1 [%0];" ::"l"(q)); }

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

}  // namespace
}  // namespace rt
