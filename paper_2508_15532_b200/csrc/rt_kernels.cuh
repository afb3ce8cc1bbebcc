// Device-side parameter block and launcher declarations shared by the .cu files of librt_b200.
#pragma once
#include <cuda_runtime.h>

#include "rt_internal.h"

namespace rt {

constexpr int FACE_STRIDE = 12;  // doubles per face entry   (see DeviceTables::face)
constexpr int CEN_STRIDE = 44;   // doubles per centre entry (see below)
// centre entry: [0..3] g_{0mu}e^mu_b (-> n_0)  [4..7] e^0_b (-> n^0)  [8] 1/sqrt(-g_c)  [9..11] unused
//               [12..27] e^a_mu ([a][mu], -> u^a-hat)   [28..43] L[b][nu] = e^lam_b g_{lam nu} (-> n_nu)
constexpr int ANG_SLOTS = 7;     // 6 neighbour coefficients + 1 self coefficient per (column, s)

struct KParams {
    int n1, n2, n3, nd, pitch;
    int ncol;
    long long ncell;
    double inv_dx[3];
    int bc_lo[3], bc_hi[3];
    int zlo[3], zhi[3];
    int limiter, method, source_literal;
    int variant;    // RT_TRANSPORT_TMA only if tile_eligible(), else RT_TRANSPORT_L2
    int tile[3];    // RT_TRANSPORT_TMA: TX, TY, DCH of the vacuum tile kernel
    int tile_gen[3];   // ... of the Eq 23 tile kernel (one pair per thread)
    double n0_floor, rho_floor, kappa_a0, kappa_s, a_rad, Y_over_rho, abar;
    const double *face[3];
    const double *cen;
    const double *ecen;
    const double *angcoef;
    const double *nhat;
    const double *w;
    const int *nb;
    const unsigned char *cls;   // [ncol][pitch] class byte (k_classify)
    const double *paircoef;     // [ncol][pitch][8] geometry of a (column, s) pair for the tile kernels (k_paircoef), RT_TRANSPORT_TMA only
    const double *paircoefz;    // [ncol][pitch][8] the Q Z products of the five faces (Eq 23's advective term), only with opacities
    // MAPR tables (only when angular_recon == RT_ANG_MAPR): grid-only tables are [slot][..][pitch]
    const double *mapr_xi;    // [6][3][pitch]  log map of neighbour e in the tangent plane at n_s
    const double *mapr_xim;   // [6][3][pitch]  log map of the centre of edge e
    const double *mapr_a;     // [6][4][pitch]  a11, a12, a22, det of the pair (e, e+1)
    const int *mapr_back;     // [6][pitch]     slot of s in neighbour e's list
    const int *mapr_nnb;      // [pitch]        5 or 6
    const double *angraw;     // [ncol][6][pitch] dlam n_0e V / w per edge (gated)
    const unsigned char *angup;   // [ncol][pitch] bit e: V_e > 0
    const int *genlist;         // compact list of the "general" (column * pitch + s) entries
    int ngen;
    const double *ghost[3][2];
    const int *mirror;        // [pitch] RT_BC_REFLECT (x2 only): index of the direction with n-hat^2 flipped
    const double *rho, *u4;  // library-owned fluid copies
    // interaction list (rt_set_fluid, cub partition): srclist[0 .. *nsel) = cells with rho >= rho_floor in ascending order (the only
    // ones the source step can touch), srclist[*nsel .. ncell) = the others.  The length stays on the DEVICE (no read-back, no
    // synchronisation in rt_set_fluid): list kernels read *nsel and run grid-stride.  srclist == nullptr: no list (no opacity or
    // no source step).
    const int *srclist;
    const int *nsel;
};

// Layout of the column-flag buffer: [ncol] column flags, then (4-byte aligned)
// [ceil(n3/32)][ncol] 32-bit cell-flag masks (see k_colflag).
__host__ __device__ inline size_t colmask_offset(int ncol, int n3) {
    (void)n3;
    return ((size_t)ncol + 3) & ~(size_t)3;
}
__host__ __device__ inline size_t colflag_bytes(int ncol, int n3) {
    return colmask_offset(ncol, n3) + sizeof(unsigned) * (size_t)ncol * ((n3 + 31) / 32);
}

// launchers (rt_transport.cu, rt_source.cu); every launch increments *launches
cudaError_t launch_facecoef(const KParams &p, const double *T, double dt, double *fcoef[3], unsigned char *colflag,
                            cudaStream_t st, long long *launches);
cudaError_t launch_transport(const KParams &p, const double *I_in, const double *I_base, double *I_out,
                             double *const fcoef[3], const unsigned char *colflag, bool matter,
                             double dt, cudaStream_t st, long long *launches);
// rt_transport_tile.cu: the non-"general" pairs through the TMA tile kernel
void choose_tile(const KParams &p, const int req[3], int out[3]);
bool tile_eligible(const KParams &p);
cudaError_t launch_paircoef(const KParams &p, double *out, double *outz, cudaStream_t st);
void choose_tile_gen(const KParams &p, int out[3]);
cudaError_t launch_transport_tile_gen(const KParams &p, const double *I_in, const double *I_base, double *I_out, double *const fcoef[3],
                                      const unsigned char *colflag, double dt, cudaStream_t st, long long *launches);
cudaError_t launch_transport_tile(const KParams &p, const int tile[3], const double *I_in, const double *I_base, double *I_out,
                                  const unsigned char *colflag, bool matter, double dt, cudaStream_t st, long long *launches);
// rt_transport.cu: the transport launch with its scratch in a file-scope device array (rt_transport_static)
size_t transport_static_bytes(const KParams &p, bool matter);
cudaError_t launch_transport_static(const KParams &p, const double *T, const double *I_in, const double *I_base, double *I_out,
                                    bool matter, double dt, cudaStream_t st, long long *launches);
cudaError_t launch_angular_mapr(const KParams &p, const double *I_in, double *I_io, double dt, cudaStream_t st, long long *launches);
cudaError_t launch_classify(const KParams &p, unsigned char *cls, cudaStream_t st);
cudaError_t launch_angular(const KParams &p, const double *I_in, double *I_io, double dt, cudaStream_t st, long long *launches);
// source step; if R_after != nullptr also writes moments after the update; if G != nullptr writes
// G_nu = -(R^0_nu after - before)/dt.
cudaError_t launch_source(const KParams &p, double *I, double *T, double dt, int *n_fail, double *R_after, double *G,
                          cudaStream_t st, long long *launches);
// rt_moments_mma.cu: R^mu_nu on the fp64 tensor pipe; part: 0 all cells, 1 interaction list, 2 its complement; gmode: see the kernel
cudaError_t launch_moments_mma(const KParams &p, const double *I, double *R, double *G, int part, int gmode, double dt, cudaStream_t st);
cudaError_t launch_moments(const KParams &p, const double *I, double *R, cudaStream_t st, long long *launches);

}  // namespace rt
