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

// index of a fluid cell along one dim: periodic wraps, everything else clamps (fluid ghosts)
__device__ __forceinline__ int fluid_idx(int c, int N, int bc_lo, int bc_hi) {
    if (c < 0) return bc_lo == RT_BC_PERIODIC ? ((c % N) + N) % N : 0;
    if (c >= N) return bc_hi == RT_BC_PERIODIC ? c % N : N - 1;
    return c;
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
        for (int o = 0; o < 4; ++o) v[o] = p.u4[(1 + a) * p.ncell + cell[o]] / p.u4[cell[o]];
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

// flux through one face, times sqrt(-g_f).  IL/IR: PLI states; Il/Ir: cell-centre values left/right of the face.
template <bool MATTER>
__device__ __forceinline__ double face_flux(const FaceC &c, double IL, double IR, double Il, double Ir, const double4 &fc) {
    if (!MATTER || fc.y < 0.0) return c.Q * c.P * (c.P > 0 ? IL : IR);                       // Eq 20
    return c.Q * (c.P * fc.x * (IL + IR) - fabs(c.P) * fc.y * (Ir - Il) + c.Z * (fc.z * IL + fc.w * IR));   // Eq 23
}

// both fluxes of one dim from the 5-point stencil (m2, m1, c0, p1, p2): lo = face (m1|c0), hi = face (c0|p1)
template <int LIM, bool MATTER>
__device__ __forceinline__ double flux_diff(double m2, double m1, double c0, double p1, double p2, const FaceC &lo,
                                            const FaceC &hi, const double4 &fclo, const double4 &fchi) {
    const double d0 = m1 - m2, d1 = c0 - m1, d2 = p1 - c0, d3 = p2 - p1;
    const double sm = slope<LIM>(d0, d1), s0 = slope<LIM>(d1, d2), sp = slope<LIM>(d2, d3);
    const double Flo = face_flux<MATTER>(lo, m1 + 0.5 * sm, c0 - 0.5 * s0, m1, c0, fclo);
    const double Fhi = face_flux<MATTER>(hi, c0 + 0.5 * s0, p1 - 0.5 * sp, c0, p1, fchi);
    return Fhi - Flo;
}

// ---- spatial transport ------------------------------------------------------------------------------------------
template <int LIM, bool MATTER>
__global__ void __launch_bounds__(256)
k_transport(KParams p, const double *__restrict__ I_in, const double *I_base, double *I_out,
            const double4 *__restrict__ fc0, const double4 *__restrict__ fc1, const double4 *__restrict__ fc2, double dt) {
    const int e = blockIdx.x * blockDim.x + threadIdx.x;
    if (e >= p.n1 * p.pitch) return;
    const int i = e / p.pitch, s = e - i * p.pitch, j = blockIdx.y;
    const long long col = (long long)j * p.n1 + i;
    const long long kstride = (long long)p.n1 * p.n2 * p.pitch;
    double *out = I_out + col * p.pitch + s;
    if (s >= p.nd) {   // pad lanes: keep the pad zero
        for (int k = 0; k < p.n3; ++k) out[k * kstride] = 0.0;
        return;
    }
    const double nx = __ldg(p.nhat + s), ny = __ldg(p.nhat + p.pitch + s), nz = __ldg(p.nhat + 2 * p.pitch + s);
    const double *cen = p.cen + col * CEN_STRIDE;
    const double n0c = centre_n0(cen, nx, ny, nz);
    const double nup = cen[4] + cen[5] * nx + cen[6] * ny + cen[7] * nz;
    const double n0n0 = nup * n0c, inv_n0n0 = 1.0 / n0n0, inv_sg = cen[8];
    const bool band_ij = (i < p.zlo[0] || i >= p.n1 - p.zhi[0] || j < p.zlo[1] || j >= p.n2 - p.zhi[1]);
    if (band_ij || n0c > -p.n0_floor) {   // masked direction (S14) or zero band (L709): stays zero, no work
        for (int k = 0; k < p.n3; ++k) out[k * kstride] = 0.0;
        return;
    }
    // face coefficients, formed once per column (geometry is x3-independent)
    FaceC xl = face_coef(p.face[0] + ((long long)j * (p.n1 + 1) + i) * FACE_STRIDE, nx, ny, nz);
    FaceC xh = face_coef(p.face[0] + ((long long)j * (p.n1 + 1) + i + 1) * FACE_STRIDE, nx, ny, nz);
    FaceC yl = face_coef(p.face[1] + ((long long)j * p.n1 + i) * FACE_STRIDE, nx, ny, nz);
    FaceC yh = face_coef(p.face[1] + ((long long)(j + 1) * p.n1 + i) * FACE_STRIDE, nx, ny, nz);
    FaceC zf = face_coef(p.face[2] + col * FACE_STRIDE, nx, ny, nz);
    // n_0 gate (L280): no flux between two mesh cells whose n_0 differ in sign
    {
        int in;
        in = (i > 0) ? i - 1 : (p.bc_lo[0] == RT_BC_PERIODIC ? p.n1 - 1 : -1);
        if (in >= 0 && sign_differs(n0c, centre_n0(p.cen + ((long long)j * p.n1 + in) * CEN_STRIDE, nx, ny, nz))) xl.Q = 0.0;
        in = (i < p.n1 - 1) ? i + 1 : (p.bc_hi[0] == RT_BC_PERIODIC ? 0 : -1);
        if (in >= 0 && sign_differs(n0c, centre_n0(p.cen + ((long long)j * p.n1 + in) * CEN_STRIDE, nx, ny, nz))) xh.Q = 0.0;
        in = (j > 0) ? j - 1 : (p.bc_lo[1] == RT_BC_PERIODIC ? p.n2 - 1 : -1);
        if (in >= 0 && sign_differs(n0c, centre_n0(p.cen + ((long long)in * p.n1 + i) * CEN_STRIDE, nx, ny, nz))) yl.Q = 0.0;
        in = (j < p.n2 - 1) ? j + 1 : (p.bc_hi[1] == RT_BC_PERIODIC ? 0 : -1);
        if (in >= 0 && sign_differs(n0c, centre_n0(p.cen + ((long long)in * p.n1 + i) * CEN_STRIDE, nx, ny, nz))) yh.Q = 0.0;
    }
    const double cx = p.inv_dx[0] * inv_sg, cy = p.inv_dx[1] * inv_sg, cz = p.inv_dx[2] * inv_sg;

    // x3 register window: I_in at k-2 .. k+2
    double w0 = ldI(cell_ptr(p, I_in, 2, i, j, -2), s), w1 = ldI(cell_ptr(p, I_in, 2, i, j, -1), s);
    double w2 = ldI(cell_ptr(p, I_in, 2, i, j, 0), s), w3 = ldI(cell_ptr(p, I_in, 2, i, j, 1), s);
    const double4 vac = make_double4(0.5, -1.0, 0.0, 0.0);
    for (int k = 0; k < p.n3; ++k) {
        const double w4 = ldI(cell_ptr(p, I_in, 2, i, j, k + 2), s);
        const double xm2 = ldI(cell_ptr(p, I_in, 0, i - 2, j, k), s), xm1 = ldI(cell_ptr(p, I_in, 0, i - 1, j, k), s);
        const double xp1 = ldI(cell_ptr(p, I_in, 0, i + 1, j, k), s), xp2 = ldI(cell_ptr(p, I_in, 0, i + 2, j, k), s);
        const double ym2 = ldI(cell_ptr(p, I_in, 1, i, j - 2, k), s), ym1 = ldI(cell_ptr(p, I_in, 1, i, j - 1, k), s);
        const double yp1 = ldI(cell_ptr(p, I_in, 1, i, j + 1, k), s), yp2 = ldI(cell_ptr(p, I_in, 1, i, j + 2, k), s);
        double4 fxl = vac, fxh = vac, fyl = vac, fyh = vac, fzl = vac, fzh = vac;
        if (MATTER) {
            fxl = ld4(fc0 + ((long long)k * p.n2 + j) * (p.n1 + 1) + i);
            fxh = ld4(fc0 + ((long long)k * p.n2 + j) * (p.n1 + 1) + i + 1);
            fyl = ld4(fc1 + ((long long)k * (p.n2 + 1) + j) * p.n1 + i);
            fyh = ld4(fc1 + ((long long)k * (p.n2 + 1) + j + 1) * p.n1 + i);
            fzl = ld4(fc2 + ((long long)k * p.n2 + j) * p.n1 + i);
            fzh = ld4(fc2 + ((long long)(k + 1) * p.n2 + j) * p.n1 + i);
        }
        double D = cx * flux_diff<LIM, MATTER>(xm2, xm1, w2, xp1, xp2, xl, xh, fxl, fxh);
        D += cy * flux_diff<LIM, MATTER>(ym2, ym1, w2, yp1, yp2, yl, yh, fyl, fyh);
        D += cz * flux_diff<LIM, MATTER>(w0, w1, w2, w3, w4, zf, zf, fzl, fzh);
        const long long off = k * kstride;
        const double base = (I_base == I_in) ? w2 : I_base[col * p.pitch + s + off];
        const bool band_k = (k < p.zlo[2] || k >= p.n3 - p.zhi[2]);
        out[off] = band_k ? 0.0 : (n0n0 * base - dt * D) * inv_n0n0;          // Eq 18 (O5)
        w0 = w1; w1 = w2; w2 = w3; w3 = w4;
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
    for (int k = 0; k < p.n3; ++k) {
        const long long off = (long long)col * p.pitch + s + k * kstride;
        double v = 0.0;
        if (s < p.pitch) { v = I_in[off]; sI[s] = v; }
        __syncthreads();
        if (live) {
            double D = c[6] * v;
#pragma unroll
            for (int e = 0; e < 6; ++e) D += c[e] * sI[nb[e]];
            const bool band_k = (k < p.zlo[2] || k >= p.n3 - p.zhi[2]);
            I_io[off] = (zero || band_k) ? 0.0 : I_io[off] - scale * D;
        } else if (s < p.pitch) {
            I_io[off] = 0.0;
        }
        __syncthreads();
    }
}

}  // namespace

// ---- launchers ---------------------------------------------------------------------------------------------------
cudaError_t launch_facecoef(const KParams &p, const double *T, double dt, double *fcoef[3], cudaStream_t st, long long *launches) {
    for (int a = 0; a < 3; ++a) {
        long long nf = (long long)(p.n1 + (a == 0)) * (p.n2 + (a == 1)) * (p.n3 + (a == 2));
        k_facecoef<<<(unsigned)((nf + 255) / 256), 256, 0, st>>>(p, T, dt, a, reinterpret_cast<double4 *>(fcoef[a]));
        ++*launches;
    }
    return cudaGetLastError();
}

template <int LIM>
static void launch_transport_lim(const KParams &p, const double *I_in, const double *I_base, double *I_out,
                                 double *const fcoef[3], bool matter, double dt, cudaStream_t st) {
    dim3 grid((p.n1 * p.pitch + 255) / 256, p.n2);
    const double4 *f0 = reinterpret_cast<const double4 *>(fcoef[0]), *f1 = reinterpret_cast<const double4 *>(fcoef[1]),
                  *f2 = reinterpret_cast<const double4 *>(fcoef[2]);
    if (matter) k_transport<LIM, true><<<grid, 256, 0, st>>>(p, I_in, I_base, I_out, f0, f1, f2, dt);
    else k_transport<LIM, false><<<grid, 256, 0, st>>>(p, I_in, I_base, I_out, f0, f1, f2, dt);
}

cudaError_t launch_transport(const KParams &p, const double *I_in, const double *I_base, double *I_out,
                             double *const fcoef[3], bool matter, double dt, cudaStream_t st, long long *launches) {
    switch (p.limiter) {
        case RT_LIM_MC: launch_transport_lim<RT_LIM_MC>(p, I_in, I_base, I_out, fcoef, matter, dt, st); break;
        case RT_LIM_MINMOD: launch_transport_lim<RT_LIM_MINMOD>(p, I_in, I_base, I_out, fcoef, matter, dt, st); break;
        case RT_LIM_NONE: launch_transport_lim<RT_LIM_NONE>(p, I_in, I_base, I_out, fcoef, matter, dt, st); break;
        default: launch_transport_lim<RT_LIM_VANLEER>(p, I_in, I_base, I_out, fcoef, matter, dt, st); break;
    }
    ++*launches;
    return cudaGetLastError();
}

cudaError_t launch_angular(const KParams &p, const double *I_in, double *I_io, double dt, cudaStream_t st, long long *launches) {
    const int threads = ((p.pitch + 31) / 32) * 32;
    k_angular<<<p.ncol, threads, p.pitch * sizeof(double), st>>>(p, I_in, I_io, dt);
    ++*launches;
    return cudaGetLastError();
}

}  // namespace rt
