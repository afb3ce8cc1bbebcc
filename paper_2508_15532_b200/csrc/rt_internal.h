// Internal declarations of librt_b200: host-side table builders and the device-side context.
// Not part of the ABI (include/rt.h is).
#pragma once
#include <cstdint>
#include <vector>

#include "../../include/rt.h"

namespace rt {

// ---- geodesic angular grid (PAPER.md 3.3, L207-217) ---------------------------------------------------------
struct AngularGrid {
    int nd = 0;
    std::vector<double> nhat;  // [nd][3]
    std::vector<double> w;     // [nd] solid angle of the Voronoi cell
    std::vector<int> nnb;      // [nd] 5 or 6
    std::vector<int> nb;       // [nd][6] neighbour per edge slot (ccw, lowest index first), -1 padded
    std::vector<int> back;     // [nd][6] slot of s in the neighbour's list
    std::vector<double> dlam;  // [nd][6] edge length
    std::vector<double> emid;  // [nd][6][3] edge centre
    std::vector<double> eun;   // [nd][6][3] outward unit normal of the edge, tangent at emid
};
// axis: direction the pole is turned to, boost: velocity of the frame in which the grid is regular (L215); zero vectors / NULL = none
bool build_angular_grid(int level, const double axis[3], const double boost[3], AngularGrid &g);

// ---- geometry at one point (PAPER.md 2.1, Eq 1-4, Eq 8, App. A) ----------------------------------------------
struct PointGeom {
    double g[4][4];     // g_{mu nu}
    double e[4][4];     // e^mu_a   [mu][a]
    double einv[4][4];  // e^a_mu   [a][mu]
    double sqrtg;       // sqrt(-g)
    bool dead;          // zero-area location (polar axis): tetrad undefined, no flux crosses
};
void eval_point(const rt_metric &m, const double x[3], PointGeom &out);
// omega^a_{cd} (Eq 8) by 6th-order central differences, h = 5e-4 (S15)
void eval_omega(const rt_metric &m, const double x[3], double omega[4][4][4]);

// ---- device context -----------------------------------------------------------------------------------------
// Per-column tables (geometry is x3-independent for every built-in metric; column = j*N1 + i).
struct DeviceTables {
    // faces: lower face of column (i,j) along dim a; extents (N1 + [a==0]) x (N2 + [a==1]); 12 doubles per face:
    //   [0..3]  sqrt(-g_f) e^a_{b}   (b = 0..3)   -> P = sqrt(-g) n^a_f
    //   [4..7]  g_{0 mu} e^mu_{b}                 -> Q = n_{0,f}
    //   [8..11] sqrt(-g_f) e^0_{b}                -> Z = sqrt(-g) n^0_f
    double *face[3];
    // centres, 44 doubles per column:
    //   [0..3] g_{0 mu} e^mu_b (n_0)   [4..7] e^0_b (n^0)   [8] 1/sqrt(-g_c)  [9..11] pad
    //   [12..27] e^a_mu (einv, [a][mu])   [28..43] L_{b nu} = e^lam_b g_{lam nu}  ... see rt_api.cu
    double *cen;
    double *ecen;     // [ncol][16] e^mu_a, for the moment transform
    double *angcoef;  // [ncol][6][pitch]  dlam_e n_0e V_e / w_s, gated (0 across an n_0 sign change / missing slot)
    double *nhat;     // [3][pitch] direction cosines, component-major (pad = 0)
    int *mirror;      // [pitch] direction with n-hat^2 flipped (RT_BC_REFLECT on x2), nullptr if unused
    double *w;        // [pitch] solid angles (pad = 0)
    int *nb;          // [6][pitch] neighbour per slot (pad / missing slot = own index)
};

}  // namespace rt
