// Moments pass of librt_b200 (sm_100a) on the fp64 tensor pipe: R^mu_nu (and the 4-force G_nu around a source step).
//
// PAPER.md Eq 13 (L141): R^mu_nu = sum_s w_s I_s n^mu n_nu.  In the tetrad frame the ten independent sums
//     M^{ab}(cell) = sum_s I(cell, s) W(s, ab),      W(s, ab) = w_s nhat^a_s nhat^b_s     (nhat^0 = 1)
// are a dense contraction of the intensity with a CONSTANT [N_d x 10] matrix -- the one place on this path where a matrix
// unit applies (the paper itself singles this reduction out, L776).  One warp takes 8 cells at a time and runs
// mma.sync.m8n8k4.f64 over the direction axis (A = 8 cells x 4 directions straight from global memory, one 16-byte load per
// lane per two k-steps; B = W in fragment order from shared memory; two 8-wide column tiles hold the 10 components), then
// rotates M to R^mu_nu = e^mu_a M^{ab} (e^lam_b g_{lam nu}) with the per-column rows.  About 40 warp-instructions per
// cell instead of the ~350 of a lane-per-direction accumulation with warp reductions (round 1): the pass is a stream over
// the intensity.  The sums run in a fixed order, so the result is bit-reproducible; it differs from the oracle's sequential
// sum in the last bits, inside the 1e-10 parity budget like every other reduction here.
#include "rt_kernels.cuh"

namespace rt {
namespace {

constexpr int MM_WARPS = 8;   // warps per CTA

__device__ __forceinline__ void dmma884(double &d0, double &d1, double a, double b) {
    asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0, %1}, {%2}, {%3}, {%0, %1};" : "+d"(d0), "+d"(d1) : "d"(a), "d"(b));
}

// component c of the ten: 00 01 02 03 11 12 13 22 23 33 
__device__ __forceinline__ double wcomp(int c, double w, double nx, double ny, double nz) {
    switch (c) {
        case 0: return w;
        case 1: return w * nx; case 2: return w * ny; case 3: return w * nz;
        case 4: return w * nx * nx; case 5: return w * nx * ny; case 6: return w * nx * nz;
        case 7: return w * ny * ny; case 8: return w * ny * nz; case 9: return w * nz * nz;
        default: return 0.0;
    }
}
__device__ __forceinline__ double mget(const double *M, int a, int b) {
    if (a > b) { const int t = a; a = b; b = t; }
    const int base[4] = {0, 4, 7, 9};
    return M[base[a] + (b - a)];
}

// Direction order of the contraction: k-step 2 jj takes the directions 8 jj + 2 t, k-step 2 jj + 1 the directions
// 8 jj + 2 t + 1 (t = lane % 4), so that a lane's two A values are adjacent in memory; a tail of (pitch % 8) / 4 single steps.
// part: 0 = every cell, 1 = the cells of the interaction list, 2 = the others (LIST kernels only).
// gmode: 0 = R only; 1 = R^0_nu into G (the moments BEFORE a source step; R untouched); 2 = R (if given), and
// G_nu = -(R^0_nu - G_nu) / dt (Eq 36 / 48: G holds the moments before, left there by a gmode-1 pass over the same cells; a cell
// the source step did not change gets exactly 0: both passes add the same numbers in the same order).
// WIDE: rows of more than 256 directions (see NB below)
template <bool LIST, bool WIDE>
__global__ void __launch_bounds__(32 * MM_WARPS, WIDE ? 2 : 4)
k_moments_mma(const __grid_constant__ KParams p, const double *__restrict__ I, double *__restrict__ R, double *__restrict__ G,
              int part, int gmode, double inv_dt) {
    extern __shared__ double sm[];
    const int nks = p.pitch / 4;                       // k-steps (pitch is a multiple of 4)
    double *bfrag = sm;                                // [nks][2 tiles][32 lanes]
    double *mout = sm + (size_t)nks * 64;              // per warp: [8 cells][10]
    for (int q = threadIdx.x; q < nks * 64; q += blockDim.x) {
        const int ks = q >> 6, tile = (q >> 5) & 1, ln = q & 31;
        const int t = ln & 3, n = (ln >> 2) + 8 * tile;
        const int npair = (p.pitch / 8) * 2;
        const int s = ks < npair ? 8 * (ks >> 1) + 2 * t + (ks & 1) : 4 * ks + t;
        bfrag[q] = (s < p.nd && n < 10) ? wcomp(n, p.w[s], p.nhat[s], p.nhat[p.pitch + s], p.nhat[2 * p.pitch + s]) : 0.0;
    }
    __syncthreads();
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int g = lane >> 2, t = lane & 3;
    double *mo = mout + warp * 80;
    // LIST: the interaction list srclist[0 .. *nsel) or its complement srclist[*nsel .. ncell) (the length lives on the device)
    const long long nsel = LIST ? (long long)__ldg(p.nsel) : 0;
    const int *list = LIST ? p.srclist + (part == 2 ? nsel : 0) : nullptr;
    const long long nwork = LIST ? (part == 2 ? p.ncell - nsel : nsel) : p.ncell;
    const long long ngroups = (nwork + 7) / 8;
    const long long gw = (long long)blockIdx.x * MM_WARPS + warp, gstride = (long long)gridDim.x * MM_WARPS;
    const int npair = p.pitch / 8;
    // Software pipeline over (group, batch): the loads run a batch of NB pairs (NB x 512 bytes per warp) ahead of the MMAs that
    // consume them, double-buffered, and the last batch of a group already fetches the first batch of the warp's next group
    // (whose cell indices were looked up at the start of this one).  Without this every loop trip exposed a full memory latency
    // (long-scoreboard stalls of 41 cycles per issue, 3 TB/s).  Which side of the trade wins depends on the row length (measured):
    // at 162 directions four blocks of 64 registers per SM (32 warps) with a short batch beat two blocks of 128 registers with
    // NB = 8 by 13 %; at 362 directions (a group is 23 KB, the B fragments 47 KB per block) the deep batch wins by 40 %.
    constexpr int NB = WIDE ? 8 : 2;
    auto lookup = [&](long long grp_, bool &valid_) -> long long {
        const long long wi = grp_ * 8 + g;
        valid_ = grp_ < ngroups && wi < nwork;
        return valid_ ? (LIST ? (long long)__ldg(list + wi) : wi) : 0;
    };
    bool valid;
    long long cell = lookup(gw, valid);
    double2 cur[NB], nxt[NB];
    {
        const double2 *rp0 = reinterpret_cast<const double2 *>(I + cell * p.pitch + 2 * t);
#pragma unroll
        for (int q = 0; q < NB; ++q) cur[q] = (valid && q < npair) ? __ldg(rp0 + 4 * q) : make_double2(0.0, 0.0);
    }
    for (long long grp = gw; grp < ngroups; grp += gstride) {
        const double *row = I + cell * p.pitch;
        bool valid_n;
        const long long cell_n = lookup(grp + gstride, valid_n);
        // two accumulator sets (even / odd pairs of k-steps): the dependent DMMA chain is half as long
        double c0 = 0.0, c1 = 0.0, c2 = 0.0, c3 = 0.0, d0 = 0.0, d1 = 0.0, d2 = 0.0, d3 = 0.0;
        const double *bf = bfrag + lane;
        const double2 *rp = reinterpret_cast<const double2 *>(row + 2 * t);   // pair jj at rp[4 jj]
        double atail = 0.0;
        if (2 * npair < nks) atail = valid ? __ldg(row + 8 * npair + t) : 0.0;     // (pitch % 8 == 4: one single k-step at the end)
        for (int j0 = 0; j0 < npair; j0 += NB) {
            if (j0 + NB < npair) {
#pragma unroll
                for (int q = 0; q < NB; ++q) nxt[q] = (valid && j0 + NB + q < npair) ? __ldg(rp + 4 * (j0 + NB + q)) : make_double2(0.0, 0.0);
            } else {
                const double2 *rn = reinterpret_cast<const double2 *>(I + cell_n * p.pitch + 2 * t);
#pragma unroll
                for (int q = 0; q < NB; ++q) nxt[q] = (valid_n && q < npair) ? __ldg(rn + 4 * q) : make_double2(0.0, 0.0);
            }
#pragma unroll
            for (int q = 0; q < NB; ++q) {
                if (j0 + q < npair) {
                    if (q & 1) { dmma884(d0, d1, cur[q].x, bf[0]); dmma884(d2, d3, cur[q].x, bf[32]); dmma884(d0, d1, cur[q].y, bf[64]); dmma884(d2, d3, cur[q].y, bf[96]); }
                    else { dmma884(c0, c1, cur[q].x, bf[0]); dmma884(c2, c3, cur[q].x, bf[32]); dmma884(c0, c1, cur[q].y, bf[64]); dmma884(c2, c3, cur[q].y, bf[96]); }
                    bf += 128;
                }
            }
#pragma unroll
            for (int q = 0; q < NB; ++q) cur[q] = nxt[q];
        }
        if (2 * npair < nks) { dmma884(d0, d1, atail, bf[0]); dmma884(d2, d3, atail, bf[32]); }
        c0 += d0; c1 += d1; c2 += d2; c3 += d3;
        // C fragment: row g (cell), columns 2 t, 2 t + 1 of each tile -> shared memory [cell][comp]
        mo[g * 10 + 2 * t] = c0; mo[g * 10 + 2 * t + 1] = c1;
        if (t == 0) { mo[g * 10 + 8] = c2; mo[g * 10 + 9] = c3; }
        __syncwarp();
        // rotate: lane = (cell cl = lane % 8, column nu = lane / 8): T_a = sum_b M^{ab} L_{b nu}, then R^mu_nu = sum_a e^mu_a T_a
        // for the four mu; a store instruction writes one component of eight consecutive cells (full sectors)
        {
            const int cl = lane & 7, nu = lane >> 3;
            const long long wj = grp * 8 + cl;
            if (wj < nwork) {
                const long long cj = LIST ? (long long)list[wj] : wj;
                const int col = int((unsigned)cj % (unsigned)p.ncol);
                const double *ecen = p.ecen + (long long)col * 16, *L = p.cen + (long long)col * CEN_STRIDE + 28;
                const double *M = mo + cl * 10;
                const double l0 = __ldg(L + nu), l1 = __ldg(L + 4 + nu), l2 = __ldg(L + 8 + nu), l3 = __ldg(L + 12 + nu);
                double T[4];
#pragma unroll
                for (int a2 = 0; a2 < 4; ++a2) T[a2] = mget(M, a2, 0) * l0 + mget(M, a2, 1) * l1 + mget(M, a2, 2) * l2 + mget(M, a2, 3) * l3;
#pragma unroll
                for (int mu = 0; mu < 4; ++mu) {
                    if (mu > 0 && gmode == 1) break;
                    const double2 ea = __ldg(reinterpret_cast<const double2 *>(ecen + 4 * mu)), eb = __ldg(reinterpret_cast<const double2 *>(ecen + 4 * mu + 2));
                    const double r = ea.x * T[0] + ea.y * T[1] + eb.x * T[2] + eb.y * T[3];
                    if (gmode != 1 && R) R[(long long)(4 * mu + nu) * p.ncell + cj] = r;
                    if (mu == 0 && gmode != 0) {
                        double *g = G + (long long)nu * p.ncell + cj;
                        *g = (gmode == 1) ? r : -(r - *g) * inv_dt;
                    }
                }
            }
        }
        __syncwarp();
        cell = cell_n; valid = valid_n;
    }
}

}  // namespace

// Moments of every cell (part 0), of the listed cells (1) or of the others (2); see the kernel for gmode
cudaError_t launch_moments_mma(const KParams &p, const double *I, double *R, double *G, int part, int gmode, double dt, cudaStream_t st) {
    const size_t smem = ((size_t)(p.pitch / 4) * 64 + MM_WARPS * 80) * sizeof(double);
    const long long groups = (p.ncell + 7) / 8;
    long long blocks = (groups + MM_WARPS - 1) / MM_WARPS;
    if (blocks > 148LL * 8) blocks = 148LL * 8;
    const double inv_dt = gmode == 2 ? 1.0 / dt : 0.0;
    cudaError_t e = cudaSuccess;
#define RT_MM_LAUNCH(L, W)                                                                                              \
    do {                                                                                                                \
        e = cudaFuncSetAttribute(k_moments_mma<L, W>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);          \
        if (e == cudaSuccess) k_moments_mma<L, W><<<(unsigned)blocks, 32 * MM_WARPS, smem, st>>>(p, I, R, G, part, gmode, inv_dt); \
    } while (0)
    const bool wide = p.pitch > 256;
    if (part != 0) { if (wide) RT_MM_LAUNCH(true, true); else RT_MM_LAUNCH(true, false); }
    else { if (wide) RT_MM_LAUNCH(false, true); else RT_MM_LAUNCH(false, false); }
#undef RT_MM_LAUNCH
    return e != cudaSuccess ? e : cudaGetLastError();
}

}  // namespace rt
