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
// Thread mapping: the tile's (column, s) pairs are numbered q = (lj TX + c) DCH + d; consumer thread t owns pairs t and
// t + NT.  As in rt_transport.cu everything geometric of a pair (folded face coefficients, upwind sides, operand offsets
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

constexpr int NT = 480;              // consumer threads (15 warps); warp 15 is the producer: 16 warps = 128 registers each
constexpr int RP = 2;                // pairs per consumer thread
#ifndef NS_X
#define NS_X 5
#endif
constexpr int NS = NS_X;             // ring slots: planes k, k+1, k+2 in use, two in flight
constexpr int SLOT_STRIDE = 24576;   // bytes between ring slots (compile-time: every operand load is LDS [R + imm])
constexpr int BSLOT_STRIDE = RP * NT * 8;   // base ring: own cells only

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
__device__ __forceinline__ void tma_box(uint32_t dst, const CUtensorMap *map, uint32_t bar, int c0, int c1, int c2, int c3) {
    asm volatile("cp.async.bulk.tensor.4d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4, %5, %6}], [%2];"
                 ::"r"(dst), "l"(map), "r"(bar), "r"(c0), "r"(c1), "r"(c2), "r"(c3) : "memory");
}
__device__ __forceinline__ double lds(uint32_t addr) {
    double v;
    asm volatile("ld.shared.f64 %0, [%1];" : "=d"(v) : "r"(addr));
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
    int split;   // opacities present: tiles without an all-vacuum cell are skipped (see the kernel)
};

// One x3 step of the pairs of a thread.  U = k mod NS is a compile-time constant of the unrolled march, so all ring
// offsets are immediates.
struct PairK { double Kxbc, Kxcd, Kybc, Kycd, zA, zhalf; };

template <bool SAME_BASE, int RP>
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

    if (threadIdx.x == NT) {
        for (int q = 0; q < NS; ++q) {
            mbar_init(bar_full + 8 * q, 1); mbar_init(bar_empty + 8 * q, NT / 32);
            mbar_init(bar_fullB + 8 * q, 1); mbar_init(bar_emptyB + 8 * q, NT / 32);
        }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
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
    const int rowpairs = tp.TX * tp.DCH, npairs = rowpairs * tp.TY;
    // per-pair constants
    uint32_t a_own[RP], a_xa[RP], a_xb[RP], a_xd[RP], a_ya[RP], a_yb[RP], a_yd[RP], a_base[RP];
    PairK K[RP];
    int pos0[RP];
    bool wr[RP], live[RP], zpos[RP];
#pragma unroll
    for (int r = 0; r < RP; ++r) {
        const int q = t + r * NT;
        wr[r] = live[r] = false; zpos[r] = true;
        a_own[r] = a_xa[r] = a_xb[r] = a_xd[r] = a_ya[r] = a_yb[r] = a_yd[r] = ring; a_base[r] = ringB;
        K[r] = PairK{0.0, 0.0, 0.0, 0.0, 0.0, 0.5};
        pos0[r] = 0;
        if (q < npairs) {
            const int lj = q / rowpairs, rem = q - lj * rowpairs, c = rem / tp.DCH, d = rem - c * tp.DCH;
            const int i = i0 + c, j = j0 + lj, s = s0 + d;
            if (i < p.n1 && j < p.n2 && s < p.pitch) {
                const int col = j * p.n1 + i;
                const int cl = p.cls[(long long)col * p.pitch + s];
                wr[r] = !(cl & 2);
                live[r] = cl == 0;
                pos0[r] = col * p.pitch + s;
                if (live[r]) {
                    ColSetup cs;
                    col_setup(p, dt, cs, i, j, s);
                    const bool xpos = cs.xl.pos, ypos = cs.yl.pos;
                    zpos[r] = cs.zf.pos;
                    K[r].Kxbc = xpos ? -cs.xl.A : cs.xh.A; K[r].Kxcd = xpos ? cs.xh.A : -cs.xl.A;
                    K[r].Kybc = ypos ? -cs.yl.A : cs.yh.A; K[r].Kycd = ypos ? cs.yh.A : -cs.yl.A;
                    K[r].zA = cs.zf.A; K[r].zhalf = cs.zf.pos ? 0.5 : -0.5;
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

    for (int k0 = 0; k0 < n3; k0 += NS) {
        const uint32_t par0 = (uint32_t)((k0 / NS) & 1);   // parity of the ring round that holds plane sequence m = k0 .. k0 + NS - 1
#pragma unroll
        for (int u = 0; u < NS; ++u) {
            const int k = k0 + u;
            if (k >= n3) break;
            // ring sequence: operands of plane k sit at m = k + 2, the new x3-window value at m = k + 4
            const int uo = (u + 4) % NS, uk = (u + 2) % NS;
            const uint32_t so = (uint32_t)(uo * SLOT_STRIDE), sk = (uint32_t)(uk * SLOT_STRIDE), sb = (uint32_t)(u * BSLOT_STRIDE);
            mbar_wait(bar_full + 8 * uo, par0 ^ (uint32_t)((u + 4) / NS & 1));
            if (!SAME_BASE) mbar_wait(bar_fullB + 8 * u, par0);
            const bool band = (k < zlo || k >= zhi);
            // straight-line code for both pairs (a pair that is not live computes on zero coefficients and address 0; only its
            // store is predicated), so that the two dependency chains interleave
#pragma unroll
            for (int r = 0; r < RP; ++r) {
                double res;
                {
                    const double w4 = lds(a_own[r] + so);
                    const double cbase = SAME_BASE ? w2[r] : lds(a_base[r] + sb);
                    // x3: upwind state at the upper face (always formed: it is the next cell's lower flux if that cell is vacuum)
                    const double sz = slope_k<RT_LIM_MC>(w3[r] - w2[r], zpos[r] ? (w2[r] - w1[r]) : (w4 - w3[r]));
                    const double Fhi = K[r].zA * fma(K[r].zhalf, sz, zpos[r] ? w2[r] : w3[r]);
                    const double xa = lds(a_xa[r] + sk), xb = lds(a_xb[r] + sk), xd = lds(a_xd[r] + sk);
                    const double ya = lds(a_ya[r] + sk), yb = lds(a_yb[r] + sk), yd = lds(a_yd[r] + sk);
                    double D = Fhi - Flo[r];
                    {
                        const double d1 = xb - xa, d2 = w2[r] - xb, d3 = xd - w2[r];
                        D = fma(K[r].Kxbc, fma(0.5, slope_k<RT_LIM_MC>(d1, d2), xb), D);
                        D = fma(K[r].Kxcd, fma(0.5, slope_k<RT_LIM_MC>(d2, d3), w2[r]), D);
                    }
                    {
                        const double d1 = yb - ya, d2 = w2[r] - yb, d3 = yd - w2[r];
                        D = fma(K[r].Kybc, fma(0.5, slope_k<RT_LIM_MC>(d1, d2), yb), D);
                        D = fma(K[r].Kycd, fma(0.5, slope_k<RT_LIM_MC>(d2, d3), w2[r]), D);
                    }
                    res = (band || !live[r]) ? 0.0 : cbase - D;   // Eq 18 (O5), dt / (n^0 n_0 sqrt(-g) dx) folded in
                    Flo[r] = Fhi;
                    w1[r] = w2[r]; w2[r] = w3[r]; w3[r] = w4;
                }
                if (wr[r]) outk[pos0[r]] = res;
            }
            outk += kstride;
            __syncwarp();
            if (lane == 0) {
                mbar_arrive(bar_empty + 8 * uk);
                if (!SAME_BASE) mbar_arrive(bar_emptyB + 8 * u);
            }
        }
    }
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
constexpr size_t SMEM_MAX = 227 * 1024;

}  // namespace

// Tile shape for a mesh: TX x TY columns x DCH directions with TX TY DCH <= RP NT pairs.  DCH is even (TMA: the inner box
// extent is a multiple of 16 bytes) and chosen so that ceil(pitch / DCH) chunks waste few lanes; (TX, TY) minimise the halo'd
// cells loaded per cell computed, (TY (TX + 4) + 4 TX) / (TX TY), with the ragged tiles of this mesh counted.
void choose_tile(const KParams &p, const int req[3], int out[3]) {
    if (req && req[0] > 0 && req[1] > 0 && req[2] > 0) { out[0] = req[0]; out[1] = req[1]; out[2] = req[2]; return; }
    double best = 1e300;
    out[0] = 2; out[1] = 1; out[2] = 8;
    for (int dch = 8; dch <= 64; dch += 2) {
        const int nch = (p.pitch + dch - 1) / dch;
        const double wd = (double)nch * dch / p.nd;   // lanes per real direction
        const int cells = RP * NT / dch;
        for (int ty = 1; ty <= 8; ++ty)
            for (int tx = 2; tx <= 16; ++tx) {
                if (tx * ty > cells) continue;
                const int tl[3] = {tx, ty, dch};
                TileParams t;
                if (tile_layout(p, tl, false, t) > SMEM_MAX || t.slotB > SLOT_STRIDE) continue;
                const double use = (double)(tx * ty * dch) / (RP * NT);    // consumer slots in use
                const double rag = ((double)((p.n1 + tx - 1) / tx) * tx / p.n1) * ((double)((p.n2 + ty - 1) / ty) * ty / p.n2);
                const double X = (double)(ty * (tx + 4) + 4 * tx) / (tx * ty);
                const double cost = wd * rag / use * (1.0 + 0.12 * (X - 1.0));
                if (cost < best) { best = cost; out[0] = tx; out[1] = ty; out[2] = dch; }
            }
    }
}

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
    if (smem > SMEM_MAX || t.slotB > SLOT_STRIDE || t.TX * t.TY * t.DCH > RP * NT || (t.DCH & 1) || t.TX < 2 || t.TX + 4 > 256 || t.DCH > 256)
        return cudaErrorInvalidConfiguration;
    CUtensorMap mA, mH, mG, mD;
    if (!make_map(&mA, I_in, p, t.DCH, t.TX + 4, t.TY) || !make_map(&mH, I_in, p, t.DCH, t.TX, 2) || !make_map(&mG, I_in, p, t.DCH, 2, t.TY) ||
        !make_map(&mD, I_base, p, t.DCH, t.TX, t.TY))
        return cudaErrorInvalidValue;
    const unsigned grid = (unsigned)(t.ntx * t.nty * t.nch);
    cudaError_t e;
    if (same) {
        e = cudaFuncSetAttribute(k_transport_tile<true, RP>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e == cudaSuccess) k_transport_tile<true, RP><<<grid, NT + 32, smem, st>>>(p, t, mA, mH, mG, mD, I_out, colflag, dt);
    } else {
        e = cudaFuncSetAttribute(k_transport_tile<false, RP>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e == cudaSuccess) k_transport_tile<false, RP><<<grid, NT + 32, smem, st>>>(p, t, mA, mH, mG, mD, I_out, colflag, dt);
    }
    ++*launches;
    return e != cudaSuccess ? e : cudaGetLastError();
}

}  // namespace rt
