// Tiled spatial transport of librt_b200 (sm_100a): O3 + O5 with the stencil operands staged in shared memory by TMA.
//
// PAPER.md: Eq 18 (L193), PLI reconstruction (L225, S7: monotonised central), vacuum flux Eq 20 (L245), non-vacuum flux
// Eq 21-23 (L252-278, S8-S13), n_0 gate and mask (L280-284, S14), polar zero band (L709).
//
// Why: the per-thread-load kernels of rt_transport.cu ask L2 for seven operands per cell-direction (own x3 window, three
// x1 and three x2 neighbours) and are bound by that L2 -> L1 traffic (profiles/r01_v20: 6.5 GB per launch for 2 GB of
// compulsory DRAM traffic).  Here a CTA owns a tile of TX x TY columns x a chunk of DCH directions and marches x3.  A
// producer warp streams every x3-plane of the tile, with its two-cell x1/x2 halos, ONCE into a ring of shared-memory
// slots (cp.async.bulk.tensor boxes [DCH x W cells], completion on an mbarrier per slot); 16 consumer warps take all
// seven (vacuum, upwind-only) or thirteen (Eq 23) operands from the ring.  L2 requests per cell-direction fall from 7 to
// (TY (TX + 4) + 4 TX) / (TX TY) (2.3-2.7 for the tiles used), and the march has no global loads, no prefetches and no
// 64-bit address arithmetic left except the store.
//
// Thread mapping: the tile's (column, s) pairs are numbered q = (lj TX + c) DCH + d; consumer thread t owns the pairs
// t, t + NT, .. (RP of them; RP = 1 as built).  As in rt_transport.cu everything geometric of a pair (folded face coefficients, upwind sides, operand offsets
// inside a slot) is formed once (the geometry is x3-independent) and lives in registers for the whole march, and the x3
// stencil is a register window.  Pairs of the "general" class (sign change of n^a inside the cell, ZERO / FIXED /
// REFLECT ghosts) stay with the list kernel of rt_transport.cu; the arithmetic is the same, in the same order, as in
// k_transport_vac / k_transport_gen, so the three variants agree bit for bit.
#include <cuda.h>

#include <cstdint>
#include <cstring>

#include "rt_transport_dev.cuh"

namespace rt {
namespace {

constexpr int NT = 736;               // consumer threads (23 warps) + warp 23, the producer: 24 warps of <= 85 registers.  One pair per thread and
                                      // 23 warps beat two pairs per thread and 15 warps of 128 registers by 4-5 % (the kernel is issue-bound: more warps to pick from)
constexpr int RP = 1;                   // pairs per consumer thread (the kernel is written for any RP)
constexpr int NS = 8;                // ring slots: planes k, k+1, k+2 in use, five in flight (a load takes about two steps)
constexpr int SLOT_STRIDE = 20480;   // bytes between ring slots (compile-time: every operand load is LDS [R + imm])
constexpr int BSLOT_STRIDE = RP * NT * 8 + 128;   // base ring: own cells only (+ the zero word, see ZERO_OFF)
constexpr int ZERO_OFF = SLOT_STRIDE - 8;   // a double behind each slot's data that holds 0.0: the operand of every pair that is not live

// ---- mbarrier / TMA primitives (PTX) ------------------------------------------------------------------------------
__device__ __forceinline__ uint32_t smem_u32(const void *q) { return (uint32_t)__cvta_generic_to_shared(q); }
__device__ __forceinline__ void mbar_init(uint32_t bar, int count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint32_t bar, uint32_t bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint32_t bar) {
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(bar) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t parity) {
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "WAIT_%=:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
        "@p bra DONE_%=;\n"
        "bra WAIT_%=;\n"
        "DONE_%=:\n"
        "}\n" ::"r"(bar), "r"(parity) : "memory");
}
// one non-blocking probe; the blocking wait is only entered if it fails (hides the probe's latency behind the step before)
__device__ __forceinline__ bool mbar_test(uint32_t bar, uint32_t parity) {
    uint32_t ok;
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n"
        "selp.u32 %0, 1, 0, p;\n"
        "}\n" : "=r"(ok) : "r"(bar), "r"(parity) : "memory");
    return ok != 0;
}
__device__ __forceinline__ void tma_box(uint32_t dst, const CUtensorMap *map, uint32_t bar, int c0, int c1, int c2, int c3) {
    asm volatile("cp.async.bulk.tensor.4d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4, %5, %6}], [%2];"
                 ::"r"(dst), "l"(map), "r"(bar), "r"(c0), "r"(c1), "r"(c2), "r"(c3) : "memory");
}
__device__ __forceinline__ double lds(uint32_t addr) {
    double v;
    asm volatile("ld.shared.f64 %0, [%1];" : "=d"(v) : "r"(addr));
    return v;
}

__device__ __forceinline__ double4 lds4(uint32_t addr) {
    double4 v;
    asm volatile("ld.shared.v2.f64 {%0, %1}, [%2];" : "=d"(v.x), "=d"(v.y) : "r"(addr));
    asm volatile("ld.shared.v2.f64 {%0, %1}, [%2+16];" : "=d"(v.z), "=d"(v.w) : "r"(addr));
    return v;
}

// x3-plane p (may be out of range by the stencil reach) -> source plane under a PERIODIC / OUTFLOW boundary
__device__ __forceinline__ int plane_src(int pl, int n3, int bc_lo, int bc_hi) { return nb_index(pl, n3, bc_lo, bc_hi); }

// ---- the kernel ------------------------------------------------------------------------------------------------------
// Shared memory: [barriers][ring: NS slots of the halo'd plane][base ring: NS slots, own cells][matter extras].
// A slot holds, each block starting on a 128-byte boundary (TMA destination) and written by ONE box per plane:
//   own   TY rows x (TX + 4) cells: columns i0-2 .. i0+TX+1 of rows j0 .. j0+TY-1            box [DCH, TX+4, TY]
//   Hlo   2 rows x TX cells: rows j0-2, j0-1;   Hhi: rows j0+TY, j0+TY+1                     box [DCH, TX, 2]
//   Gx    (x1 PERIODIC only) TY rows x 2 cells: the wrapped columns n1-2, n1-1 (lo) and 0, 1 (hi)   box [DCH, 2, TY]
//   Gy    (x2 PERIODIC only) 2 rows x TX cells: the wrapped rows n2-2, n2-1 (lo) and 0, 1 (hi)      box [DCH, TX, 2]
// Boxes that reach outside the mesh are zero-filled by TMA; nobody reads those cells: an OUTFLOW ghost is read from the
// edge cell it copies, a PERIODIC ghost from the G blocks, and pairs next to ZERO / FIXED / REFLECT ghosts are "general".
struct TileParams {
    int TX, TY, DCH, nch, ntx, nty;
    int cellB, rowB;                                   // bytes of one cell (DCH doubles), of one own row
    int oHlo, oHhi, oGxlo, oGxhi, oGylo, oGyhi;        // block offsets in a slot (own block at 0)
    int slotB, bslotB;
    int off_ring, off_base;
    int slotStride, bslotStride, zeroOff, bzeroOff;   // run-time ring geometry (k_transport_tile_gen; the vacuum kernel's is compile-time)
    int oCx, oCy, oCz, coefB;                          // k_transport_tile_gen: per-face coefficient blocks of a slot (x1 faces, x2 faces, x3 faces), their bytes
    int split;   // opacities present: tiles without an all-vacuum cell are skipped (see the kernel)
};

// ---- per-(column, s) table of everything geometric the tile kernel needs, built once by rt_init ----------------------------
// [ncol * pitch][8] doubles: Q P of the faces xl, xh, yl, yh, z (n_0 gate applied), 1 / sqrt(-g_c), n^0 n_0 at the centre,
// and a flag word (bit 0 dead, bit 1 general: the class byte of k_classify; bits 2-4: sqrt(-g) n^a_f > 0 for a = 1, 2, 3).
// The tile kernel folds dt / (n^0 n_0 sqrt(-g_c) dx^a) in exactly as col_setup() does, so its coefficients carry the same
// bits as those of the per-thread-load kernels; what it saves is col_setup's ~900 instructions and dependent loads per pair.
__global__ void k_paircoef(const __grid_constant__ KParams p, double *__restrict__ out, double *__restrict__ outz) {
    const int e = blockIdx.x * blockDim.x + threadIdx.x;
    if (e >= p.n1 * p.pitch) return;
    const int i = e / p.pitch, s = e - i * p.pitch, j = blockIdx.y, col = j * p.n1 + i;
    double4 *o = reinterpret_cast<double4 *>(out + ((long long)col * p.pitch + s) * 8);
    const int cl = p.cls[(long long)col * p.pitch + s];
    double qp[5] = {0, 0, 0, 0, 0}, qz[5] = {0, 0, 0, 0, 0}, c8 = 1.0, den = 1.0;
    unsigned flags = (unsigned)cl;
    if (!(cl & 1)) {
        const double nx = __ldg(p.nhat + s), ny = __ldg(p.nhat + p.pitch + s), nz = __ldg(p.nhat + 2 * p.pitch + s);
        const double *cen = p.cen + (long long)col * CEN_STRIDE;
        const double n0c = centre_n0(cen, nx, ny, nz);
        const double nup = cen[4] + cen[5] * nx + cen[6] * ny + cen[7] * nz;
        c8 = cen[8]; den = nup * n0c;
        FaceC f;
        int in;
        f = face_coef(p.face[0] + ((long long)j * (p.n1 + 1) + i) * FACE_STRIDE, nx, ny, nz);
        in = (i > 0) ? i - 1 : (p.bc_lo[0] == RT_BC_PERIODIC ? p.n1 - 1 : -1);
        if (in >= 0 && sign_differs(n0c, centre_n0(p.cen + ((long long)j * p.n1 + in) * CEN_STRIDE, nx, ny, nz))) f.Q = 0.0;
        qp[0] = f.Q * f.P; qz[0] = f.Q * f.Z; if (f.P > 0) flags |= 4u;
        f = face_coef(p.face[0] + ((long long)j * (p.n1 + 1) + i + 1) * FACE_STRIDE, nx, ny, nz);
        in = (i < p.n1 - 1) ? i + 1 : (p.bc_hi[0] == RT_BC_PERIODIC ? 0 : -1);
        if (in >= 0 && sign_differs(n0c, centre_n0(p.cen + ((long long)j * p.n1 + in) * CEN_STRIDE, nx, ny, nz))) f.Q = 0.0;
        qp[1] = f.Q * f.P; qz[1] = f.Q * f.Z;
        f = face_coef(p.face[1] + ((long long)j * p.n1 + i) * FACE_STRIDE, nx, ny, nz);
        in = (j > 0) ? j - 1 : (p.bc_lo[1] == RT_BC_PERIODIC ? p.n2 - 1 : -1);
        if (in >= 0 && sign_differs(n0c, centre_n0(p.cen + ((long long)in * p.n1 + i) * CEN_STRIDE, nx, ny, nz))) f.Q = 0.0;
        qp[2] = f.Q * f.P; qz[2] = f.Q * f.Z; if (f.P > 0) flags |= 8u;
        f = face_coef(p.face[1] + ((long long)(j + 1) * p.n1 + i) * FACE_STRIDE, nx, ny, nz);
        in = (j < p.n2 - 1) ? j + 1 : (p.bc_hi[1] == RT_BC_PERIODIC ? 0 : -1);
        if (in >= 0 && sign_differs(n0c, centre_n0(p.cen + ((long long)in * p.n1 + i) * CEN_STRIDE, nx, ny, nz))) f.Q = 0.0;
        qp[3] = f.Q * f.P; qz[3] = f.Q * f.Z;
        f = face_coef(p.face[2] + (long long)col * FACE_STRIDE, nx, ny, nz);
        qp[4] = f.Q * f.P; qz[4] = f.Q * f.Z; if (f.P > 0) flags |= 16u;
    }
    o[0] = make_double4(qp[0], qp[1], qp[2], qp[3]);
    o[1] = make_double4(qp[4], c8, den, __longlong_as_double((long long)flags));
    if (outz) {   // sqrt(-g) n_0 n^0 at the five faces: the advective term of Eq 23 (only with opacities)
        double4 *oz = reinterpret_cast<double4 *>(outz + ((long long)col * p.pitch + s) * 8);
        oz[0] = make_double4(qz[0], qz[1], qz[2], qz[3]);
        oz[1] = make_double4(qz[4], 0.0, 0.0, 0.0);
    }
}

// One x3 step of the pairs of a thread.  U = k mod NS is a compile-time constant of the unrolled march, so all ring
// offsets are immediates.
struct PairK { double Kxbc, Kxcd, Kybc, Kycd, zA, zhalf; };

template <bool SAME_BASE, bool MASK, int RP>
__global__ void __launch_bounds__(NT + 32, 1)
k_transport_tile(const __grid_constant__ KParams p, const __grid_constant__ TileParams tp,
                 const __grid_constant__ CUtensorMap mapA, const __grid_constant__ CUtensorMap mapH,
                 const __grid_constant__ CUtensorMap mapG, const __grid_constant__ CUtensorMap mapD, double *I_out,
                 const unsigned char *__restrict__ colflag, double dt) {
    extern __shared__ __align__(1024) unsigned char smem[];
    const uint32_t sbase = smem_u32(smem);
    // barriers: full[NS], empty[NS], fullB[NS], emptyB[NS]
    const uint32_t bar_full = sbase, bar_empty = sbase + 8 * NS, bar_fullB = sbase + 16 * NS, bar_emptyB = sbase + 24 * NS;
    const uint32_t ring = sbase + tp.off_ring, ringB = sbase + tp.off_base;

    // block -> (direction chunk fastest, then tiles in bands of 6 tile rows with x2 fastest inside a band)
    const int ch = blockIdx.x % tp.nch, tile = blockIdx.x / tp.nch;
    constexpr int BAND = 6;
    const int band = tile / (tp.ntx * BAND), rr = tile - band * tp.ntx * BAND;
    const int th = min(BAND, tp.nty - band * BAND);
    const int tx = rr / th, ty = band * BAND + (rr - tx * th);
    const int i0 = tx * tp.TX, j0 = ty * tp.TY, s0 = ch * tp.DCH;
    const int n3 = p.n3, warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const bool perx = p.bc_lo[0] == RT_BC_PERIODIC && p.n1 >= 2, pery = p.bc_lo[1] == RT_BC_PERIODIC && p.n2 >= 2;
    if (tp.split) {
        // With opacities the cells that have an Eq 23 face are recomputed afterwards by k_transport_gen; a tile without a single
        // all-vacuum cell (column flag bit 1 clear everywhere, k_colflag) has nothing to do here.
        int has = 0;
        if ((int)threadIdx.x < tp.TX * tp.TY) {
            const int i = i0 + (int)threadIdx.x % tp.TX, j = j0 + (int)threadIdx.x / tp.TX;
            if (i < p.n1 && j < p.n2) has = colflag[j * p.n1 + i] & 2;
        }
        if (__syncthreads_or(has) == 0) {   // only the dead entries (masked directions, zero bands, pad) are this kernel's: keep them zero
            if ((int)threadIdx.x < NT)
                for (int r = 0; r < RP; ++r) {
                    const int q = (int)threadIdx.x + r * NT, rowpairs = tp.TX * tp.DCH;
                    if (q >= rowpairs * tp.TY) continue;
                    const int lj = q / rowpairs, rem = q - lj * rowpairs, c = rem / tp.DCH, d = rem - c * tp.DCH;
                    const int i = i0 + c, j = j0 + lj, sdir = s0 + d;
                    if (i >= p.n1 || j >= p.n2 || sdir >= p.pitch) continue;
                    const long long e = (long long)(j * p.n1 + i) * p.pitch + sdir;
                    if (p.cls[e] & 1)
                        for (int k = 0; k < n3; ++k) I_out[e + k * (long long)p.ncol * p.pitch] = 0.0;
                }
            return;
        }
    }

    // ---- producer role (one lane at a time): plane m of the ring sequence = x3-plane m - 2 of I_in; base plane k ----
    const bool hlo = j0 >= 1, hhi = j0 + tp.TY < p.n2;
    const bool gxlo = perx && i0 < 2, gxhi = perx && i0 + tp.TX >= p.n1 - 1;
    const bool gylo = pery && j0 < 2, gyhi = pery && j0 + tp.TY >= p.n2 - 1;
    const uint32_t bA = (uint32_t)(tp.TY * tp.rowB), bH = (uint32_t)(2 * tp.TX * tp.cellB), bG = (uint32_t)(2 * tp.TY * tp.cellB);
    const uint32_t bytes = bA + (hlo ? bH : 0) + (hhi ? bH : 0) + (gxlo ? bG : 0) + (gxhi ? bG : 0) + (gylo ? bH : 0) + (gyhi ? bH : 0);
    const uint32_t bytesB = (uint32_t)(tp.TY * tp.TX * tp.cellB);
    auto issue_plane = [&](int m) {   // caller: one lane; the slot's previous plane has been released (or m < NS)
        const int slot = m % NS;
        if (m >= NS) mbar_wait(bar_empty + 8 * slot, ((m / NS) & 1) ^ 1);
        const int ks = plane_src(m - 2, n3, p.bc_lo[2], p.bc_hi[2]);
        const uint32_t dst = ring + slot * SLOT_STRIDE, bar = bar_full + 8 * slot;
        mbar_expect_tx(bar, bytes);
        tma_box(dst, &mapA, bar, s0, i0 - 2, j0, ks);
        if (hlo) tma_box(dst + tp.oHlo, &mapH, bar, s0, i0, j0 - 2, ks);
        if (hhi) tma_box(dst + tp.oHhi, &mapH, bar, s0, i0, j0 + tp.TY, ks);
        if (gxlo) tma_box(dst + tp.oGxlo, &mapG, bar, s0, p.n1 - 2, j0, ks);
        if (gxhi) tma_box(dst + tp.oGxhi, &mapG, bar, s0, 0, j0, ks);
        if (gylo) tma_box(dst + tp.oGylo, &mapH, bar, s0, i0, p.n2 - 2, ks);
        if (gyhi) tma_box(dst + tp.oGyhi, &mapH, bar, s0, i0, 0, ks);
    };
    auto issue_base = [&](int k) {
        const int slot = k % NS;
        if (k >= NS) mbar_wait(bar_emptyB + 8 * slot, ((k / NS) & 1) ^ 1);
        mbar_expect_tx(bar_fullB + 8 * slot, bytesB);
        tma_box(ringB + slot * BSLOT_STRIDE, &mapD, bar_fullB + 8 * slot, s0, i0, j0, k);
    };

    // the geometry rows of this thread's pairs: requested first (one exposed memory latency for all of them, overlapped with the
    // barrier set-up and the producer's first boxes); a slot that holds no pair of the mesh reads row 0 and ignores it
    const int rowpairs = tp.TX * tp.DCH, npairs = rowpairs * tp.TY;
    int pi[RP], pj[RP], pc[RP], plj[RP], pd[RP];
    bool pvalid[RP];
    double4 tq0[RP], tq1[RP];
#pragma unroll
    for (int r = 0; r < RP; ++r) {
        const int q = (int)threadIdx.x + r * NT;
        const int lj = q / rowpairs, rem = q - lj * rowpairs, c = rem / tp.DCH, d = rem - c * tp.DCH;
        plj[r] = lj; pc[r] = c; pd[r] = d; pi[r] = i0 + c; pj[r] = j0 + lj;
        pvalid[r] = (int)threadIdx.x < NT && q < npairs && pi[r] < p.n1 && pj[r] < p.n2 && s0 + d < p.pitch;
        const long long row = pvalid[r] ? (long long)(pj[r] * p.n1 + pi[r]) * p.pitch + s0 + d : 0;
        const double4 *tq = reinterpret_cast<const double4 *>(p.paircoef + row * 8);
        tq0[r] = ld4(tq); tq1[r] = ld4(tq + 1);
    }

    if (threadIdx.x == NT) {
        for (int q = 0; q < NS; ++q) {
            mbar_init(bar_full + 8 * q, 1); mbar_init(bar_empty + 8 * q, NT / 32);
            mbar_init(bar_fullB + 8 * q, 1); mbar_init(bar_emptyB + 8 * q, NT / 32);
        }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    if ((int)threadIdx.x < NS) {
        *reinterpret_cast<double *>(smem + tp.off_ring + threadIdx.x * SLOT_STRIDE + ZERO_OFF) = 0.0;
        if (!SAME_BASE) *reinterpret_cast<double *>(smem + tp.off_base + threadIdx.x * BSLOT_STRIDE + RP * NT * 8) = 0.0;
    }
    __syncthreads();

    if (warp == NT / 32) {
        // ===== producer warp: one lane streams the planes; base plane k goes out just before ring plane k + 4, which the
        // consumers need together with it =====
        if (lane == 0)
            for (int m = 0; m < n3 + 4; ++m) {
                if (!SAME_BASE && m >= 4) issue_base(m - 4);
                issue_plane(m);
            }
        return;
    }

    const int t = threadIdx.x;
    // per-pair constants
    uint32_t a_own[RP], a_xa[RP], a_xb[RP], a_xd[RP], a_ya[RP], a_yb[RP], a_yd[RP], a_base[RP];
    PairK K[RP];
    int pos0[RP];
    bool wr[RP], live[RP], zpos[RP];
    // MASK (opacities present): bit (k & 31) of the column's mask word = the cell has an Eq 23 face and belongs to
    // k_transport_gen, which reads its base state from I_base: this kernel must not touch it (I_out may alias I_base)
    const unsigned *cmask = reinterpret_cast<const unsigned *>(colflag + colmask_offset(p.ncol, n3));
    int mcol[RP];
    unsigned mcur[RP], mnext[RP];
#pragma unroll
    for (int r = 0; r < RP; ++r) {
        wr[r] = live[r] = false; zpos[r] = true;
        mcol[r] = -1; mcur[r] = mnext[r] = 0u;
        a_own[r] = a_xa[r] = a_xb[r] = a_xd[r] = a_ya[r] = a_yb[r] = a_yd[r] = ring + ZERO_OFF; a_base[r] = ringB + RP * NT * 8;   // zero words
        K[r] = PairK{0.0, 0.0, 0.0, 0.0, 0.0, 0.5};
        pos0[r] = 0;
        {
            const int lj = plj[r], c = pc[r], d = pd[r], i = pi[r], j = pj[r], s = s0 + d;
            if (pvalid[r]) {
                const int col = j * p.n1 + i;
                const double4 t0 = tq0[r], t1 = tq1[r];
                const unsigned fl = (unsigned)__double_as_longlong(t1.w);
                wr[r] = !(fl & 2u);
                live[r] = (fl & 3u) == 0u;
                pos0[r] = col * p.pitch + s;
                if (MASK && wr[r]) {
                    mcol[r] = col;
                    mcur[r] = __ldg(cmask + col);
                    mnext[r] = n3 > 32 ? __ldg(cmask + p.ncol + col) : 0u;
                }
                if (live[r]) {
                    // the folding of col_setup() / fold(): A = (Q P) * (dt / (n^0 n_0 sqrt(-g_c)) / dx^a)
                    const double scale = dt * t1.y / t1.z;
                    const double sx = scale * p.inv_dx[0], sy = scale * p.inv_dx[1], sz = scale * p.inv_dx[2];
                    const double Axl = t0.x * sx, Axh = t0.y * sx, Ayl = t0.z * sy, Ayh = t0.w * sy;
                    const bool xpos = (fl & 4u) != 0u, ypos = (fl & 8u) != 0u;
                    zpos[r] = (fl & 16u) != 0u;
                    K[r].Kxbc = xpos ? -Axl : Axh; K[r].Kxcd = xpos ? Axh : -Axl;
                    K[r].Kybc = ypos ? -Ayl : Ayh; K[r].Kycd = ypos ? Ayh : -Ayl;
                    K[r].zA = t1.x * sz; K[r].zhalf = zpos[r] ? 0.5 : -0.5;
                    const int din = d * 8;
                    auto xo = [&](int o) -> uint32_t {
                        int gi = i + o;
                        if (gi < 0 || gi >= p.n1) {
                            const int bc = gi < 0 ? p.bc_lo[0] : p.bc_hi[0];
                            if (bc == RT_BC_OUTFLOW) gi = gi < 0 ? 0 : p.n1 - 1;        // the edge cell itself
                            else if (bc == RT_BC_PERIODIC && perx)
                                return (gi < 0 ? tp.oGxlo + (gi + 2) * tp.cellB : tp.oGxhi + (gi - p.n1) * tp.cellB) + lj * 2 * tp.cellB + din;
                            else gi = i;   // a single periodic column wraps onto itself ("general" pairs do not come here)
                        }
                        return lj * tp.rowB + (gi - i0 + 2) * tp.cellB + din;
                    };
                    auto yo = [&](int o) -> uint32_t {
                        int gj = j + o;
                        if (gj < 0 || gj >= p.n2) {
                            const int bc = gj < 0 ? p.bc_lo[1] : p.bc_hi[1];
                            if (bc == RT_BC_OUTFLOW) gj = gj < 0 ? 0 : p.n2 - 1;
                            else if (bc == RT_BC_PERIODIC && pery)
                                return (gj < 0 ? tp.oGylo + (gj + 2) * tp.TX * tp.cellB : tp.oGyhi + (gj - p.n2) * tp.TX * tp.cellB) + c * tp.cellB + din;
                            else gj = j;
                        }
                        const int lr = gj - j0;
                        if (lr < 0) return tp.oHlo + ((lr + 2) * tp.TX + c) * tp.cellB + din;
                        if (lr >= tp.TY) return tp.oHhi + ((lr - tp.TY) * tp.TX + c) * tp.cellB + din;
                        return lr * tp.rowB + (c + 2) * tp.cellB + din;
                    };
                    a_own[r] = ring + xo(0);
                    a_xa[r] = ring + xo(xpos ? -2 : 2); a_xb[r] = ring + xo(xpos ? -1 : 1); a_xd[r] = ring + xo(xpos ? 1 : -1);
                    a_ya[r] = ring + yo(ypos ? -2 : 2); a_yb[r] = ring + yo(ypos ? -1 : 1); a_yd[r] = ring + yo(ypos ? 1 : -1);
                    a_base[r] = ringB + (lj * tp.TX + c) * tp.cellB + din;
                }
            }
        }
    }
    const long long kstride = (long long)p.ncol * p.pitch;
    const int zlo = p.zlo[2], zhi = n3 - p.zhi[2];

    // prologue: planes -2 .. 1 (ring sequence m = 0 .. 3) -> register windows
    double w1[RP], w2[RP], w3[RP], Flo[RP];
#pragma unroll
    for (int m = 0; m < 4; ++m) {
        mbar_wait(bar_full + 8 * m, 0);
#pragma unroll
        for (int r = 0; r < RP; ++r) {
            const double v = lds(a_own[r] + m * SLOT_STRIDE);
            if (m == 0) Flo[r] = v; else if (m == 1) w1[r] = v; else if (m == 2) w2[r] = v; else w3[r] = v;   // Flo: plane -2 for now
        }
        if (m < 2) {   // planes -2, -1 are not read again
            __syncwarp();
            if (lane == 0) mbar_arrive(bar_empty + 8 * m);
        }
    }
#pragma unroll
    for (int r = 0; r < RP; ++r) {
        const double sg = slope_k<RT_LIM_MC>(w2[r] - w1[r], zpos[r] ? (w1[r] - Flo[r]) : (w3[r] - w2[r]));
        Flo[r] = K[r].zA * fma(K[r].zhalf, sg, zpos[r] ? w1[r] : w2[r]);
    }
    double *outk = I_out;

    // One x3 step; in the unrolled march u, so, sk, sb are compile-time constants (every operand load is LDS [R + imm]).  A pair
    // that is not live reads the zero words with zero coefficients: its result is +0.0, which is what a dead entry holds.
    bool ready = false;   // outcome of the probe of this step's barriers, made during the step before
    auto step = [&](int k, int u, uint32_t par0) {
        const int uo = (u + 4) % NS, uk = (u + 2) % NS;
        const uint32_t so = (uint32_t)(uo * SLOT_STRIDE), sk = (uint32_t)(uk * SLOT_STRIDE), sb = (uint32_t)(u * BSLOT_STRIDE);
        if (!ready) {
            mbar_wait(bar_full + 8 * uo, par0 ^ (uint32_t)((u + 4) / NS & 1));
            if (!SAME_BASE) mbar_wait(bar_fullB + 8 * u, par0);
        }
        double w4[RP], cbase[RP], xa[RP], xb[RP], xd[RP], ya[RP], yb[RP], yd[RP];
#pragma unroll
        for (int r = 0; r < RP; ++r) {
            w4[r] = lds(a_own[r] + so);
            cbase[r] = SAME_BASE ? w2[r] : lds(a_base[r] + sb);
            xa[r] = lds(a_xa[r] + sk); xb[r] = lds(a_xb[r] + sk); xd[r] = lds(a_xd[r] + sk);
            ya[r] = lds(a_ya[r] + sk); yb[r] = lds(a_yb[r] + sk); yd[r] = lds(a_yd[r] + sk);
        }
        if (k + 1 < n3) {   // probe the next step's barriers now; the answer is there when the arithmetic below is done
            const int u1 = (u + 1) % NS;
            const uint32_t par1 = par0 ^ (uint32_t)(u + 1 == NS);
            ready = mbar_test(bar_full + 8 * ((u1 + 4) % NS), par1 ^ (uint32_t)((u1 + 4) / NS & 1));
            if (!SAME_BASE) ready = mbar_test(bar_fullB + 8 * u1, par1) && ready;
        }
#pragma unroll
        for (int r = 0; r < RP; ++r) {
            // x3: upwind state at the upper face (it is the next cell's lower flux)
            const double sz = slope_k<RT_LIM_MC>(w3[r] - w2[r], zpos[r] ? (w2[r] - w1[r]) : (w4[r] - w3[r]));
            const double Fhi = K[r].zA * fma(K[r].zhalf, sz, zpos[r] ? w2[r] : w3[r]);
            double D = Fhi - Flo[r];
            {
                const double d1 = xb[r] - xa[r], d2 = w2[r] - xb[r], d3 = xd[r] - w2[r];
                D = fma(K[r].Kxbc, fma(0.5, slope_k<RT_LIM_MC>(d1, d2), xb[r]), D);
                D = fma(K[r].Kxcd, fma(0.5, slope_k<RT_LIM_MC>(d2, d3), w2[r]), D);
            }
            {
                const double d1 = yb[r] - ya[r], d2 = w2[r] - yb[r], d3 = yd[r] - w2[r];
                D = fma(K[r].Kybc, fma(0.5, slope_k<RT_LIM_MC>(d1, d2), yb[r]), D);
                D = fma(K[r].Kycd, fma(0.5, slope_k<RT_LIM_MC>(d2, d3), w2[r]), D);
            }
            // Eq 18 (O5), dt / (n^0 n_0 sqrt(-g) dx) folded in; the x3 zero band is reset below
            if (wr[r] && !(MASK && live[r] && ((mcur[r] >> (k & 31)) & 1u))) outk[pos0[r]] = cbase[r] - D;   // (dead entries are always this kernel's)
            Flo[r] = Fhi;
            w1[r] = w2[r]; w2[r] = w3[r]; w3[r] = w4[r];
        }
        outk += kstride;
        __syncwarp();
        if (lane == 0) {
            mbar_arrive(bar_empty + 8 * uk);
            if (!SAME_BASE) mbar_arrive(bar_emptyB + 8 * u);
        }
        if (MASK && (k & 31) == 31) {   // next mask word (requested 32 steps ago)
#pragma unroll
            for (int r = 0; r < RP; ++r) {
                mcur[r] = mnext[r];
                mnext[r] = (mcol[r] >= 0 && k + 33 < n3) ? __ldg(cmask + (long long)((k >> 5) + 2) * p.ncol + mcol[r]) : 0u;
            }
        }
    };
    int k0 = 0;
    for (; k0 + NS <= n3; k0 += NS) {   // full ring rounds, unrolled
        const uint32_t par0 = (uint32_t)((k0 / NS) & 1);   // parity of the ring round that holds the sequence m = k0 .. k0 + NS - 1
#pragma unroll
        for (int u = 0; u < NS; ++u) step(k0 + u, u, par0);
    }
#pragma unroll 1
    for (int k = k0; k < n3; ++k) step(k, k - k0, (uint32_t)((k0 / NS) & 1));   // the last, partial round
    if (zlo > 0 || zhi < n3)   // zero band in x3 (L709): reset after the march instead of a select in every step
#pragma unroll
        for (int r = 0; r < RP; ++r)
            if (wr[r])
                for (int k = 0; k < n3; ++k)
                    if ((k < zlo || k >= zhi) && !(MASK && live[r] && ((__ldg(cmask + (long long)(k >> 5) * p.ncol + mcol[r]) >> (k & 31)) & 1u))) I_out[pos0[r] + k * kstride] = 0.0;
}

// ---- the Eq 23 cells through the same ring --------------------------------------------------------------------------------
// Cells with a non-vacuum face (mask bit of k_colflag) of the non-"general" pairs: full five-point stencils in all three
// dims, both PLI states at the six faces, Eq 20 or Eq 23 per face from the per-face coefficients of k_facecoef -- the
// arithmetic of k_transport_gen (rt_transport.cu) with the thirteen operands taken from the ring instead of thirteen global
// loads, except that the x3 face flux and slope a step has formed are carried to the next step instead of being formed again
// (the results agree with k_transport_gen's to rounding).  The per-face coefficients of k_facecoef (five double4 per cell and step,
// the same for all directions of a cell) ride in the ring as well: three more TMA boxes per plane ([4 x (TX+1) x TY] x1 faces,
// [4 x TX x (TY+1)] x2 faces, [4 x TX x TY] x3 faces k+1/2) on the slot's barrier, read by the consumers as shared-memory
// broadcasts.  Through global memory (L1, prefetched a step ahead, 71-79 % hits) they were the kernel's long-scoreboard stalls:
// 27 % of its time on the all-matter configs.  One pair per thread (the Eq 23 path holds ten face coefficients and a five-deep x3 window);
// tiles without such a cell leave at once; steps whose cell is all-vacuum only shift the window.
constexpr int NTG = 480;     // consumer threads of k_transport_tile_gen (+ one producer warp)
template <bool SAME_BASE>
__global__ void __launch_bounds__(NTG + 32, 1)
k_transport_tile_gen(const __grid_constant__ KParams p, const __grid_constant__ TileParams tp,
                     const __grid_constant__ CUtensorMap mapA, const __grid_constant__ CUtensorMap mapH,
                     const __grid_constant__ CUtensorMap mapG, const __grid_constant__ CUtensorMap mapD,
                     const __grid_constant__ CUtensorMap mapCx, const __grid_constant__ CUtensorMap mapCy, const __grid_constant__ CUtensorMap mapCz,
                     double *I_out, const double4 *__restrict__ fc2, const unsigned char *__restrict__ colflag, double dt) {
    constexpr int RP = 1;
    extern __shared__ __align__(1024) unsigned char smem[];
    const uint32_t sbase = smem_u32(smem);
    // barriers: full[NS], empty[NS], fullB[NS], emptyB[NS]
    const uint32_t bar_full = sbase, bar_empty = sbase + 8 * NS, bar_fullB = sbase + 16 * NS, bar_emptyB = sbase + 24 * NS;
    const uint32_t ring = sbase + tp.off_ring, ringB = sbase + tp.off_base;

    // block -> (direction chunk fastest, then tiles in bands of 6 tile rows with x2 fastest inside a band)
    const int ch = blockIdx.x % tp.nch, tile = blockIdx.x / tp.nch;
    constexpr int BAND = 6;
    const int band = tile / (tp.ntx * BAND), rr = tile - band * tp.ntx * BAND;
    const int th = min(BAND, tp.nty - band * BAND);
    const int tx = rr / th, ty = band * BAND + (rr - tx * th);
    const int i0 = tx * tp.TX, j0 = ty * tp.TY, s0 = ch * tp.DCH;
    const int n3 = p.n3, warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const bool perx = p.bc_lo[0] == RT_BC_PERIODIC && p.n1 >= 2, pery = p.bc_lo[1] == RT_BC_PERIODIC && p.n2 >= 2;
    {
        int has = 0;
        if ((int)threadIdx.x < tp.TX * tp.TY) {
            const int i = i0 + (int)threadIdx.x % tp.TX, j = j0 + (int)threadIdx.x / tp.TX;
            if (i < p.n1 && j < p.n2) has = colflag[j * p.n1 + i] & 1;
        }
        if (__syncthreads_or(has) == 0) return;
    }

    // ---- producer role (one lane at a time): plane m of the ring sequence = x3-plane m - 2 of I_in; base plane k ----
    const bool hlo = j0 >= 1, hhi = j0 + tp.TY < p.n2;
    const bool gxlo = perx && i0 < 2, gxhi = perx && i0 + tp.TX >= p.n1 - 1;
    const bool gylo = pery && j0 < 2, gyhi = pery && j0 + tp.TY >= p.n2 - 1;
    const uint32_t bA = (uint32_t)(tp.TY * tp.rowB), bH = (uint32_t)(2 * tp.TX * tp.cellB), bG = (uint32_t)(2 * tp.TY * tp.cellB);
    const uint32_t bytes = bA + (hlo ? bH : 0) + (hhi ? bH : 0) + (gxlo ? bG : 0) + (gxhi ? bG : 0) + (gylo ? bH : 0) + (gyhi ? bH : 0);
    const uint32_t bytesB = (uint32_t)(tp.TY * tp.TX * tp.cellB);
    auto issue_plane = [&](int m) {   // caller: one lane; the slot's previous plane has been released (or m < NS)
        const int slot = m % NS;
        if (m >= NS) mbar_wait(bar_empty + 8 * slot, ((m / NS) & 1) ^ 1);
        const int ks = plane_src(m - 2, n3, p.bc_lo[2], p.bc_hi[2]);
        const uint32_t dst = ring + slot * tp.slotStride, bar = bar_full + 8 * slot;
        const int kp = m - 2;                               // the plane itself (coefficients exist for 0 <= kp < n3 only)
        const bool coef = kp >= 0 && kp < n3;
        mbar_expect_tx(bar, bytes + (coef ? (uint32_t)tp.coefB : 0u));
        if (coef) {
            tma_box(dst + tp.oCx, &mapCx, bar, 0, i0, j0, kp);
            tma_box(dst + tp.oCy, &mapCy, bar, 0, i0, j0, kp);
            tma_box(dst + tp.oCz, &mapCz, bar, 0, i0, j0, kp + 1);
        }
        tma_box(dst, &mapA, bar, s0, i0 - 2, j0, ks);
        if (hlo) tma_box(dst + tp.oHlo, &mapH, bar, s0, i0, j0 - 2, ks);
        if (hhi) tma_box(dst + tp.oHhi, &mapH, bar, s0, i0, j0 + tp.TY, ks);
        if (gxlo) tma_box(dst + tp.oGxlo, &mapG, bar, s0, p.n1 - 2, j0, ks);
        if (gxhi) tma_box(dst + tp.oGxhi, &mapG, bar, s0, 0, j0, ks);
        if (gylo) tma_box(dst + tp.oGylo, &mapH, bar, s0, i0, p.n2 - 2, ks);
        if (gyhi) tma_box(dst + tp.oGyhi, &mapH, bar, s0, i0, 0, ks);
    };
    auto issue_base = [&](int k) {
        const int slot = k % NS;
        if (k >= NS) mbar_wait(bar_emptyB + 8 * slot, ((k / NS) & 1) ^ 1);
        mbar_expect_tx(bar_fullB + 8 * slot, bytesB);
        tma_box(ringB + slot * tp.bslotStride, &mapD, bar_fullB + 8 * slot, s0, i0, j0, k);
    };

    // the geometry rows of this thread's pair, requested first
    const int rowpairs = tp.TX * tp.DCH, npairs = rowpairs * tp.TY;
    const int q_ = (int)threadIdx.x;
    const int lj = q_ / rowpairs, rem_ = q_ - lj * rowpairs, c = rem_ / tp.DCH, d = rem_ - c * tp.DCH;
    const int i = i0 + c, j = j0 + lj, s = s0 + d;
    const bool pvalid = q_ < NTG && q_ < npairs && i < p.n1 && j < p.n2 && s < p.pitch;
    const int col = pvalid ? j * p.n1 + i : 0;
    const long long trow = pvalid ? (long long)col * p.pitch + s : 0;
    const double4 *tq = reinterpret_cast<const double4 *>(p.paircoef + trow * 8), *tz = reinterpret_cast<const double4 *>(p.paircoefz + trow * 8);
    const double4 t0 = ld4(tq), t1 = ld4(tq + 1), z0 = ld4(tz), z1 = ld4(tz + 1);
    const unsigned *cmask = reinterpret_cast<const unsigned *>(colflag + colmask_offset(p.ncol, n3));
    unsigned mcur = pvalid ? __ldg(cmask + col) : 0u, mnext = (pvalid && n3 > 32) ? __ldg(cmask + p.ncol + col) : 0u;

    if (threadIdx.x == NTG) {
        for (int q = 0; q < NS; ++q) {
            mbar_init(bar_full + 8 * q, 1); mbar_init(bar_empty + 8 * q, NTG / 32);
            mbar_init(bar_fullB + 8 * q, 1); mbar_init(bar_emptyB + 8 * q, NTG / 32);
        }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    if ((int)threadIdx.x < NS) {
        *reinterpret_cast<double *>(smem + tp.off_ring + threadIdx.x * tp.slotStride + tp.zeroOff) = 0.0;
        if (!SAME_BASE) *reinterpret_cast<double *>(smem + tp.off_base + threadIdx.x * tp.bslotStride + tp.bzeroOff) = 0.0;
    }
    __syncthreads();

    if (warp == NTG / 32) {
        // ===== producer warp: one lane streams the planes; base plane k goes out just before ring plane k + 4, which the
        // consumers need together with it =====
        if (lane == 0)
            for (int m = 0; m < n3 + 4; ++m) {
                if (!SAME_BASE && m >= 4) issue_base(m - 4);
                issue_plane(m);
            }
        return;
    }

    const int t = threadIdx.x;
    const unsigned fl = (unsigned)__double_as_longlong(t1.w);
    const bool live = pvalid && (fl & 3u) == 0u;          // dead entries belong to the vacuum kernel, general pairs to the list kernel
    if (!live) mcur = mnext = 0u;
    uint32_t a_own = ring + tp.zeroOff, a_x[4], a_y[4], a_base = ringB + tp.bzeroOff;
#pragma unroll
    for (int o = 0; o < 4; ++o) a_x[o] = a_y[o] = ring + tp.zeroOff;
    FaceK xl, xh, yl, yh, zf;
    xl = xh = yl = yh = zf = FaceK{0.0, 0.0, true};
    if (live) {
        const double scale = dt * t1.y / t1.z;              // the folding of col_setup() / fold()
        const double sx = scale * p.inv_dx[0], sy = scale * p.inv_dx[1], sz = scale * p.inv_dx[2];
        const bool xpos = (fl & 4u) != 0u, ypos = (fl & 8u) != 0u, zpos = (fl & 16u) != 0u;
        xl = FaceK{t0.x * sx, z0.x * sx, xpos}; xh = FaceK{t0.y * sx, z0.y * sx, xpos};
        yl = FaceK{t0.z * sy, z0.z * sy, ypos}; yh = FaceK{t0.w * sy, z0.w * sy, ypos};
        zf = FaceK{t1.x * sz, z1.x * sz, zpos};
        const int din = d * 8;
        auto xo = [&](int o) -> uint32_t {
            int gi = i + o;
            if (gi < 0 || gi >= p.n1) {
                const int bc = gi < 0 ? p.bc_lo[0] : p.bc_hi[0];
                if (bc == RT_BC_OUTFLOW) gi = gi < 0 ? 0 : p.n1 - 1;        // the edge cell itself
                else if (bc == RT_BC_PERIODIC && perx)
                    return (gi < 0 ? tp.oGxlo + (gi + 2) * tp.cellB : tp.oGxhi + (gi - p.n1) * tp.cellB) + lj * 2 * tp.cellB + din;
                else gi = i;   // a single periodic column wraps onto itself ("general" pairs do not come here)
            }
            return lj * tp.rowB + (gi - i0 + 2) * tp.cellB + din;
        };
        auto yo = [&](int o) -> uint32_t {
            int gj = j + o;
            if (gj < 0 || gj >= p.n2) {
                const int bc = gj < 0 ? p.bc_lo[1] : p.bc_hi[1];
                if (bc == RT_BC_OUTFLOW) gj = gj < 0 ? 0 : p.n2 - 1;
                else if (bc == RT_BC_PERIODIC && pery)
                    return (gj < 0 ? tp.oGylo + (gj + 2) * tp.TX * tp.cellB : tp.oGyhi + (gj - p.n2) * tp.TX * tp.cellB) + c * tp.cellB + din;
                else gj = j;
            }
            const int lr = gj - j0;
            if (lr < 0) return tp.oHlo + ((lr + 2) * tp.TX + c) * tp.cellB + din;
            if (lr >= tp.TY) return tp.oHhi + ((lr - tp.TY) * tp.TX + c) * tp.cellB + din;
            return lr * tp.rowB + (c + 2) * tp.cellB + din;
        };
        a_own = ring + xo(0);
        a_x[0] = ring + xo(-2); a_x[1] = ring + xo(-1); a_x[2] = ring + xo(1); a_x[3] = ring + xo(2);
        a_y[0] = ring + yo(-2); a_y[1] = ring + yo(-1); a_y[2] = ring + yo(1); a_y[3] = ring + yo(2);
        a_base = ringB + (lj * tp.TX + c) * tp.cellB + din;
    }
    const long long kstride = (long long)p.ncol * p.pitch;
    const int zlo = p.zlo[2], zhi = n3 - p.zhi[2], ncol = p.ncol, n1 = p.n1;
    const double4 *pz = fc2 + col;       // (only for the x3 low face at the start of a run of Eq 23 cells)
    if (!pvalid) pz = fc2;
    // this pair's per-face coefficients inside a slot
    const uint32_t cxl = ring + (uint32_t)(tp.oCx + (lj * (tp.TX + 1) + c) * 32), cyl = ring + (uint32_t)(tp.oCy + (lj * tp.TX + c) * 32);
    const uint32_t cyh = cyl + (uint32_t)tp.TX * 32u, czh = ring + (uint32_t)(tp.oCz + (lj * tp.TX + c) * 32);
    (void)n1;

    // prologue: planes -2 .. 1 (ring sequence m = 0 .. 3) -> the x3 window
    double w0, w1, w2, w3;
#pragma unroll
    for (int m = 0; m < 4; ++m) {
        mbar_wait(bar_full + 8 * m, 0);
        const double v = lds(a_own + m * tp.slotStride);
        if (m == 0) w0 = v; else if (m == 1) w1 = v; else if (m == 2) w2 = v; else w3 = v;
        if (m < 2) {   // planes -2, -1 are not read again
            __syncwarp();
            if (lane == 0) mbar_arrive(bar_empty + 8 * m);
        }
    }
    double *outk = I_out + (live ? trow : 0);
    double dz2 = w3 - w2, s0z = slope_mc(w2 - w1, dz2), Fzl = 0.0;   // x3 carries: I_{k+1} - I_k, slope of cell k, flux through its low face
    bool zcarry = false;

    // The march is NOT unrolled over the ring (the body is ~400 instructions: eight copies overflow the instruction cache and
    // spill); the slot offsets are run-time values, three adds per step.
    bool ready = false;
    int u = 0;                     // k mod NS
    uint32_t par0 = 0;             // parity of the ring round that holds the sequence m = k - u .. k - u + NS - 1
#pragma unroll 1
    for (int k = 0; k < n3; ++k) {
        const int uo = u + 4 < NS ? u + 4 : u + 4 - NS, uk = u + 2 < NS ? u + 2 : u + 2 - NS;
        const uint32_t so = (uint32_t)(uo * tp.slotStride), sk = (uint32_t)(uk * tp.slotStride), sb = (uint32_t)(u * tp.bslotStride);
        if (!ready) {
            mbar_wait(bar_full + 8 * uo, par0 ^ (uint32_t)(u + 4 >= NS));
            if (!SAME_BASE) mbar_wait(bar_fullB + 8 * u, par0);
        }
        const double w4 = lds(a_own + so);
        const bool mat = (mcur >> (k & 31)) & 1u;
        // x3: the slope of cell k + 1 is formed every step and carried (it is the next step's own slope)
        const double dz3 = w4 - w3, spz = slope_mc(dz2, dz3);
        if (mat) {
            const double4 fzh = lds4(czh + sk), fxl = lds4(cxl + sk), fxh = lds4(cxl + sk + 32u), fyl = lds4(cyl + sk), fyh = lds4(cyh + sk);
            const double xm2 = lds(a_x[0] + sk), xm1 = lds(a_x[1] + sk), xp1 = lds(a_x[2] + sk), xp2 = lds(a_x[3] + sk);
            const double ym2 = lds(a_y[0] + sk), ym1 = lds(a_y[1] + sk), yp1 = lds(a_y[2] + sk), yp2 = lds(a_y[3] + sk);
            const double cbase = SAME_BASE ? w2 : lds(a_base + sb);
            // x3: the flux through the low face is the one the step before sent through its high face (same thread, same
            // folded coefficients: the geometry does not depend on x3); formed afresh only at the start of a run of such cells
            if (!zcarry) Fzl = face_flux<true>(zf, w1 + 0.5 * slope_mc(w1 - w0, w2 - w1), w2 - 0.5 * s0z, w1, w2, ld4(pz));
            const double Fzh = face_flux<true>(zf, w2 + 0.5 * s0z, w3 - 0.5 * spz, w2, w3, fzh);
            double D = Fzh - Fzl;
            D += flux_diff<RT_LIM_MC, true>(xm2, xm1, w2, xp1, xp2, xl, xh, fxl, fxh);
            D += flux_diff<RT_LIM_MC, true>(ym2, ym1, w2, yp1, yp2, yl, yh, fyl, fyh);
            *outk = (k < zlo || k >= zhi) ? 0.0 : cbase - D;      // Eq 18 (O5), dt / (n^0 n_0 sqrt(-g) dx) folded in
            Fzl = Fzh;
        }
        zcarry = mat;
        const int u1 = u + 1 < NS ? u + 1 : 0;
        const uint32_t par1 = par0 ^ (uint32_t)(u + 1 == NS);
        if (k + 1 < n3) {   // probe the next step's barriers; the answer is there when it is needed
            const int uo1 = u1 + 4 < NS ? u1 + 4 : u1 + 4 - NS;
            ready = mbar_test(bar_full + 8 * uo1, par1 ^ (uint32_t)(u1 + 4 >= NS));
            if (!SAME_BASE) ready = mbar_test(bar_fullB + 8 * u1, par1) && ready;
        }
        w0 = w1; w1 = w2; w2 = w3; w3 = w4; dz2 = dz3; s0z = spz;
        outk += kstride; pz += ncol;
        __syncwarp();
        if (lane == 0) {
            mbar_arrive(bar_empty + 8 * uk);
            if (!SAME_BASE) mbar_arrive(bar_emptyB + 8 * u);
        }
        if ((k & 31) == 31) {   // next mask word (requested 32 steps ago)
            mcur = mnext;
            mnext = (live && k + 33 < n3) ? __ldg(cmask + (long long)((k >> 5) + 2) * ncol + col) : 0u;
        }
        u = u1; par0 = par1;
    }
    (void)t;
}

// ---- host side: tensor maps ------------------------------------------------------------------------------------------
typedef CUresult (*EncodeTiledFn)(CUtensorMap *, CUtensorMapDataType, cuuint32_t, void *, const cuuint64_t *, const cuuint64_t *,
                                  const cuuint32_t *, const cuuint32_t *, CUtensorMapInterleave, CUtensorMapSwizzle,
                                  CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
EncodeTiledFn encode_fn() {
    static EncodeTiledFn fn = nullptr;
    static bool tried = false;
    if (!tried) {
        tried = true;
        void *q = nullptr;
        cudaDriverEntryPointQueryResult st;
        if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &q, cudaEnableDefault, &st) == cudaSuccess && st == cudaDriverEntryPointSuccess)
            fn = reinterpret_cast<EncodeTiledFn>(q);
    }
    return fn;
}
// I[k][j][i][s] as a rank-4 fp64 tensor (s innermost), box = [DCH directions x w cells x h rows x 1 plane]
bool make_map(CUtensorMap *m, const double *I, const KParams &p, int dch, int w, int h) {
    EncodeTiledFn fn = encode_fn();
    if (!fn) return false;
    const cuuint64_t dims[4] = {(cuuint64_t)p.pitch, (cuuint64_t)p.n1, (cuuint64_t)p.n2, (cuuint64_t)p.n3};
    const cuuint64_t strides[3] = {(cuuint64_t)p.pitch * 8, (cuuint64_t)p.n1 * p.pitch * 8, (cuuint64_t)p.ncol * p.pitch * 8};
    const cuuint32_t box[4] = {(cuuint32_t)dch, (cuuint32_t)w, (cuuint32_t)h, 1}, es[4] = {1, 1, 1, 1};
    return fn(m, CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 4, const_cast<double *>(I), dims, strides, box, es, CU_TENSOR_MAP_INTERLEAVE_NONE,
              CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_128B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
}

// per-face coefficients fc[e3][e2][e1] of double4 as a rank-4 fp64 tensor (4 innermost), box = [4 x w faces x h rows x 1 plane]
bool make_map_fc(CUtensorMap *m, const double4 *fc, int e1, int e2, int e3, int w, int h) {
    EncodeTiledFn fn = encode_fn();
    if (!fn) return false;
    const cuuint64_t dims[4] = {4, (cuuint64_t)e1, (cuuint64_t)e2, (cuuint64_t)e3};
    const cuuint64_t strides[3] = {32, (cuuint64_t)e1 * 32, (cuuint64_t)e1 * e2 * 32};
    const cuuint32_t box[4] = {4, (cuuint32_t)w, (cuuint32_t)h, 1}, es[4] = {1, 1, 1, 1};
    return fn(m, CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 4, const_cast<double4 *>(fc), dims, strides, box, es, CU_TENSOR_MAP_INTERLEAVE_NONE,
              CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_128B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
}

int align_up(int v, int a) { return (v + a - 1) / a * a; }

// shared-memory layout of a tile (see the kernel) for a kernel with rp pairs per thread; returns the dynamic shared memory it needs
size_t tile_layout(const KParams &p, const int tile[3], bool same, TileParams &t) {
    std::memset(&t, 0, sizeof t);
    t.TX = tile[0]; t.TY = tile[1]; t.DCH = tile[2];
    t.nch = (p.pitch + t.DCH - 1) / t.DCH;
    t.ntx = (p.n1 + t.TX - 1) / t.TX; t.nty = (p.n2 + t.TY - 1) / t.TY;
    t.cellB = t.DCH * 8;
    t.rowB = (t.TX + 4) * t.cellB;
    const int bH = align_up(2 * t.TX * t.cellB, 128), bG = align_up(2 * t.TY * t.cellB, 128);
    int o = align_up(t.TY * t.rowB, 128);
    t.oHlo = o; o += bH;
    t.oHhi = o; o += bH;
    if (p.bc_lo[0] == RT_BC_PERIODIC) { t.oGxlo = o; o += bG; t.oGxhi = o; o += bG; }
    if (p.bc_lo[1] == RT_BC_PERIODIC) { t.oGylo = o; o += bH; t.oGyhi = o; o += bH; }
    t.slotB = o;   // must fit SLOT_STRIDE
    t.bslotB = t.TY * t.TX * t.cellB;
    t.off_ring = 1024;
    t.off_base = t.off_ring + NS * SLOT_STRIDE;
    return (size_t)t.off_base + (same ? 0 : NS * BSLOT_STRIDE);
}
// the same for k_transport_tile_gen: its own ring with run-time strides fitted to its tile (one pair per thread: a smaller tile
// than the vacuum kernel's), each slot followed by the per-face coefficient blocks of its plane
size_t tile_layout_gen(const KParams &p, const int tile[3], bool same, TileParams &t) {
    tile_layout(p, tile, same, t);
    t.zeroOff = t.slotB;
    // the per-face coefficients of Eq 23 ride in the same slot as the plane they belong to: [TY][TX+1] x1 faces, [TY+1][TX] x2 faces
    // of plane k and [TY][TX] x3 faces k+1/2, one double4 each, as three more TMA boxes on the slot's barrier
    t.oCx = align_up(t.slotB + 8, 128);
    t.oCy = t.oCx + align_up(t.TY * (t.TX + 1) * 32, 128);
    t.oCz = t.oCy + align_up((t.TY + 1) * t.TX * 32, 128);
    t.coefB = (t.TY * (t.TX + 1) + (t.TY + 1) * t.TX + t.TY * t.TX) * 32;
    t.slotStride = align_up(t.oCz + t.TY * t.TX * 32, 1024);
    t.bzeroOff = t.bslotB;
    t.bslotStride = align_up(t.bslotB + 8, 128);
    t.off_base = t.off_ring + NS * t.slotStride;
    return (size_t)t.off_base + (same ? 0 : NS * t.bslotStride);
}
constexpr size_t SMEM_MAX = 227 * 1024;

}  // namespace

// Tile shape for a mesh: TX x TY columns x DCH directions with TX TY DCH <= RP NT pairs.  DCH is even (TMA: the inner box
// extent is a multiple of 16 bytes) and chosen so that ceil(pitch / DCH) chunks waste few lanes; (TX, TY) minimise the halo'd
// cells loaded per cell computed, (TY (TX + 4) + 4 TX) / (TX TY), with the ragged tiles of this mesh counted.
static void choose_tile_rp(const KParams &p, int rp, int out[3], int dch_min = 8, int nt = NT) {
    double best = 1e300;
    out[0] = 2; out[1] = 1; out[2] = 8;
    for (int dch = dch_min; dch <= 64; dch += 2) {
        const int nch = (p.pitch + dch - 1) / dch;
        const double wd = (double)nch * dch / p.nd;   // lanes per real direction
        const int cells = rp * nt / dch;
        for (int ty = 1; ty <= 8; ++ty)
            for (int tx = 2; tx <= 16; ++tx) {
                if (tx * ty > cells) continue;
                const int tl[3] = {tx, ty, dch};
                TileParams t;
                if (tile_layout(p, tl, false, t) > SMEM_MAX || t.slotB > ZERO_OFF) continue;
                const double use = (double)(tx * ty * dch) / (rp * nt);    // consumer slots in use
                const double rag = ((double)((p.n1 + tx - 1) / tx) * tx / p.n1) * ((double)((p.n2 + ty - 1) / ty) * ty / p.n2);
                const double X = (double)(ty * (tx + 4) + 4 * tx) / (tx * ty);
                // short box rows (under 192 bytes) cost TMA throughput: measured 3 % at 80-byte rows against 192-byte rows
                const double rowpen = 1.0 + 0.25 * (dch * 8 < 192 ? (192.0 - dch * 8) / 192.0 : 0.0);
                const double cost = wd * rag / use * (1.0 + 0.12 * (X - 1.0)) * rowpen;
                if (cost < best) { best = cost; out[0] = tx; out[1] = ty; out[2] = dch; }
            }
    }
}

cudaError_t launch_paircoef(const KParams &p, double *out, double *outz, cudaStream_t st) {
    dim3 grid((p.n1 * p.pitch + 255) / 256, p.n2);
    k_paircoef<<<grid, 256, 0, st>>>(p, out, outz);
    return cudaGetLastError();
}

void choose_tile(const KParams &p, const int req[3], int out[3]) {
    if (req && req[0] > 0 && req[1] > 0 && req[2] > 0) { out[0] = req[0]; out[1] = req[1]; out[2] = req[2]; return; }
    choose_tile_rp(p, RP, out);
}
// (at least 16 directions per chunk: a warp then spans at most two cells and its per-face coefficient loads are near-broadcasts)
void choose_tile_gen(const KParams &p, int out[3]) { choose_tile_rp(p, 1, out, 16, NTG); }

bool tile_eligible(const KParams &p) {
    return p.limiter == RT_LIM_MC && (p.bc_lo[2] == RT_BC_PERIODIC || p.bc_lo[2] == RT_BC_OUTFLOW) &&
           (p.bc_hi[2] == RT_BC_PERIODIC || p.bc_hi[2] == RT_BC_OUTFLOW) && (long long)p.ncol * p.pitch < (1LL << 31) && encode_fn() != nullptr;
}

// The vacuum update (Eq 20 on all six faces) of the non-"general" pairs through the tile kernel.  With opacities, tiles
// without an all-vacuum cell are skipped, and the cells that have an Eq 23 face are recomputed afterwards by
// k_transport_gen (rt_transport.cu), which overwrites them.
cudaError_t launch_transport_tile(const KParams &p, const int tile[3], const double *I_in, const double *I_base, double *I_out,
                                  const unsigned char *colflag, bool matter, double dt, cudaStream_t st, long long *launches) {
    TileParams t;
    const bool same = (I_base == I_in);
    const size_t smem = tile_layout(p, tile, same, t);
    t.split = matter ? 1 : 0;
    if (smem > SMEM_MAX || t.slotB > ZERO_OFF || t.TX * t.TY * t.DCH > RP * NT || (t.DCH & 1) || t.TX < 2 || t.TX + 4 > 256 || t.DCH > 256)
        return cudaErrorInvalidConfiguration;
    CUtensorMap mA, mH, mG, mD;
    if (!make_map(&mA, I_in, p, t.DCH, t.TX + 4, t.TY) || !make_map(&mH, I_in, p, t.DCH, t.TX, 2) || !make_map(&mG, I_in, p, t.DCH, 2, t.TY) ||
        !make_map(&mD, I_base, p, t.DCH, t.TX, t.TY))
        return cudaErrorInvalidValue;
    const unsigned grid = (unsigned)(t.ntx * t.nty * t.nch);
    cudaError_t e = cudaSuccess;
#define RT_TILE_LAUNCH(S, M)                                                                                            \
    do {                                                                                                                \
        e = cudaFuncSetAttribute(k_transport_tile<S, M, RP>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);  \
        if (e == cudaSuccess) k_transport_tile<S, M, RP><<<grid, NT + 32, smem, st>>>(p, t, mA, mH, mG, mD, I_out, colflag, dt); \
    } while (0)
    if (same) { if (matter) RT_TILE_LAUNCH(true, true); else RT_TILE_LAUNCH(true, false); }
    else { if (matter) RT_TILE_LAUNCH(false, true); else RT_TILE_LAUNCH(false, false); }
#undef RT_TILE_LAUNCH
    ++*launches;
    return e != cudaSuccess ? e : cudaGetLastError();
}

// The Eq 23 cells of the non-"general" pairs through k_transport_tile_gen (it overwrites what the vacuum kernel left alone).
cudaError_t launch_transport_tile_gen(const KParams &p, const double *I_in, const double *I_base, double *I_out, double *const fcoef[3],
                                      const unsigned char *colflag, double dt, cudaStream_t st, long long *launches) {
    TileParams t;
    const bool same = (I_base == I_in);
    const size_t smem = tile_layout_gen(p, p.tile_gen, same, t);
    if (smem > SMEM_MAX || t.TX * t.TY * t.DCH > NTG || (t.DCH & 1) || t.TX < 2 || t.TX + 4 > 256 || t.DCH > 256)
        return cudaErrorInvalidConfiguration;
    CUtensorMap mA, mH, mG, mD, mCx, mCy, mCz;
    const double4 *f0 = reinterpret_cast<const double4 *>(fcoef[0]), *f1 = reinterpret_cast<const double4 *>(fcoef[1]),
                  *f2 = reinterpret_cast<const double4 *>(fcoef[2]);
    if (!make_map(&mA, I_in, p, t.DCH, t.TX + 4, t.TY) || !make_map(&mH, I_in, p, t.DCH, t.TX, 2) || !make_map(&mG, I_in, p, t.DCH, 2, t.TY) ||
        !make_map(&mD, I_base, p, t.DCH, t.TX, t.TY) || !make_map_fc(&mCx, f0, p.n1 + 1, p.n2, p.n3, t.TX + 1, t.TY) ||
        !make_map_fc(&mCy, f1, p.n1, p.n2 + 1, p.n3, t.TX, t.TY + 1) || !make_map_fc(&mCz, f2, p.n1, p.n2, p.n3 + 1, t.TX, t.TY))
        return cudaErrorInvalidValue;
    const unsigned grid = (unsigned)(t.ntx * t.nty * t.nch);
    cudaError_t e;
    if (same) {
        e = cudaFuncSetAttribute(k_transport_tile_gen<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e == cudaSuccess) k_transport_tile_gen<true><<<grid, NTG + 32, smem, st>>>(p, t, mA, mH, mG, mD, mCx, mCy, mCz, I_out, f2, colflag, dt);
    } else {
        e = cudaFuncSetAttribute(k_transport_tile_gen<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e == cudaSuccess) k_transport_tile_gen<false><<<grid, NTG + 32, smem, st>>>(p, t, mA, mH, mG, mD, mCx, mCy, mCz, I_out, f2, colflag, dt);
    }
    ++*launches;
    return e != cudaSuccess ? e : cudaGetLastError();
}

}  // namespace rt
