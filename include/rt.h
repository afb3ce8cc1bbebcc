/* rt.h -- C ABI of the B200-native radiation hot path of arxiv 2508.15532 (cuHARM radiation module).
 *
 * Per spatial cell x per direction update of the gray tetrad-frame intensity I(x, n) on a geodesic angular grid:
 *   (a) conservative spatial transport   PAPER.md Eq 18 (L193), PLI L225, Eq 20 (L245), Eq 21-23 (L252-278)
 *   (b) angular fluxes                   Eq 19 (L239-241) with Eq 7-8 (L99-109)
 *   (c) implicit radiation-fluid source  Eq 35 (L352), Eq 39-46 (L377-430), Eq 5 (L85)
 *   (d) moments R^mu_nu and 4-force      Eq 13 (L141), Eq 36/48 (L361, L442)
 *   predictor-corrector driver           L448-456
 * Readings of silent/garbled passages: DESIGN.md (S1-S26).
 *
 * Conventions
 *  - All array arguments named *_dev are DEVICE pointers (fp64), owned by the caller, unless marked host.
 *  - Intensity layout I[k][j][i][s]: interior cells only, s (direction) fastest, cell pitch = rt_ndir_padded()
 *    doubles (N_d rounded up to a multiple of 4; pad entries are ignored on input and written as 0).
 *  - Cell fields (rho, T, ...) are [k][j][i]; multi-component cell fields are component-major: u4[4][N_c],
 *    R[16][N_c] (R^mu_nu at index 4*mu+nu), G[4][N_c] (G_nu).
 *  - `stream` is a cudaStream_t passed as void* (NULL = default stream).  Calls enqueue work and return; they do
 *    not synchronise.
 *  - Every call returns RT_OK (0) or a negative RT_E* code; nothing is printed, nothing aborts.  Numerical
 *    failure of a cell's temperature solve is NOT an error: the cell keeps T_-, skips the update and is counted.
 *  - Same inputs => bit-identical outputs (no atomics in reductions).
 */
#ifndef RT_H_
#define RT_H_

#ifdef __cplusplus
extern "C" {
#endif

#define RT_OK 0
#define RT_EINVAL (-1)  /* bad argument */
#define RT_ECUDA (-2)   /* a CUDA runtime call failed (rt_last_cuda_error() has the code) */
#define RT_ENOMEM (-3)
#define RT_ESTATE (-4)  /* call order: fluid / boundary not set */
#define RT_ETOOBIG (-5) /* rt_transport_static: the mesh needs more scratch than RT_STATIC_SCRATCH_BYTES */

enum { RT_BC_PERIODIC = 0, RT_BC_OUTFLOW = 1, RT_BC_ZERO = 2, RT_BC_FIXED = 3,
       RT_BC_REFLECT = 4 /* "symmetric" boundary (L709, DESIGN S23): ghost = mirror-image cell read in the direction with the
                            normal tetrad component flipped, normal fluid velocity reversed.  Only on x^2 boundaries: the
                            geodesic grid (pole along 3-hat, a vertex at azimuth 0) is mirror symmetric across 2-hat
                            only; rt_init returns RT_EINVAL for the other dims */ };
enum { RT_MINKOWSKI_CART = 0, RT_MINK_CYL_TETRAD = 1, RT_KS_MKS = 2, RT_SNAKE = 3,
       RT_BL_MKS = 4 /* Boyer-Lindquist, same logical map as RT_KS_MKS, zero-angular-momentum tetrad (photon-orbit test, L563-592);
                        the mesh must stay outside the horizon */,
       RT_USER = 5 /* metric (and, optionally, tetrad) from the caller's host functions, called by rt_init only */ };
enum { RT_LIM_MC = 0, RT_LIM_MINMOD = 1, RT_LIM_VANLEER = 2, RT_LIM_NONE = 3 };
enum { RT_ANG_DONOR = 0, RT_ANG_MAPR = 1 };
/* how the vacuum (Eq 20) spatial transport gets its stencil operands.  RT_TRANSPORT_TMA (default): a CTA owns a tile of
 * columns x a chunk of directions, a producer warp streams each x3-plane of the tile with its halos once into a ring of
 * shared-memory slots (cp.async.bulk.tensor + mbarrier), 23 consumer warps read all operands from the ring.  Needs the
 * monotonised-central limiter and a PERIODIC or OUTFLOW x3 boundary; otherwise, and with RT_TRANSPORT_L2, one thread
 * per (column, direction) loads its operands itself through L1/L2 (the round-1 kernel).  Same arithmetic in the same
 * order: results are bit-identical.  Cells with an Eq 23 face go through k_transport_gen either way. */
enum { RT_TRANSPORT_TMA = 0, RT_TRANSPORT_L2 = 1 };
/* rt_get_geometry selectors (host output, for table-level parity of the init precompute) */
enum { RT_GEOM_G_C = 0,     /* g_{mu nu} at centres        [E3][N2][N1][4][4]            */
       RT_GEOM_E_C = 1,     /* e^mu_a at centres           [E3][N2][N1][4 mu][4 a]       */
       RT_GEOM_EINV_C = 2,  /* e^a_mu at centres           [E3][N2][N1][4 a][4 mu]       */
       RT_GEOM_SQRTG_C = 3, /* sqrt(-g) at centres         [E3][N2][N1]                  */
       RT_GEOM_OMEGA_C = 4, /* omega^a_{cd} at centres     [E3][N2][N1][4][4][4]         */
       RT_GEOM_N0_C = 5,    /* n_0 per (cell, s)           [E3][N2][N1][N_d]             */
       RT_GEOM_ANGCOEF = 6  /* Delta-lambda_e n_0e V_e / w_s per (cell, edge slot, s)  [E3][N2][N1][6][N_d] */ };
/* E3 = 1 when the geometry is x3-symmetric, else N3. */

typedef struct rt_ctx rt_ctx; /* opaque; owns all precomputed tables and one scratch copy of I on the device */

/* Logical uniform mesh (L201): interior cells n[0..2] along x^1, x^2, x^3; cell i spans x0 + [i, i+1] dx. */
typedef struct {
    int n[3];
    double x0[3], dx[3];
    int bc_lo[3], bc_hi[3];     /* RT_BC_*; ghost depth is 2 (PLI) */
    int zero_lo[3], zero_hi[3]; /* bands of interior cells next to a boundary whose I is reset to 0 after every
                                   update ("zero the specific intensity in the four cells closest to the poles", L709) */
} rt_grid;

/* Metric + tetrad (L57-79, App. A).  x3_symmetric: geometry independent of x^3 (tables stored per (x1,x2) column,
 * the paper's own optimisation, L776); required for RT_KS_MKS, ignored (constant geometry) for RT_MINKOWSKI_CART. */
typedef struct {
    int kind;         /* RT_MINKOWSKI_CART | RT_MINK_CYL_TETRAD | RT_KS_MKS | RT_SNAKE | RT_BL_MKS | RT_USER */
    double a, hslope; /* RT_KS_MKS, RT_BL_MKS: spin, theta-map parameter h: r = exp(x1), theta = pi x2 + (1-h)/2 sin(2 pi x2), phi = x3 */
    int x3_symmetric;
    double snake_A, snake_k; /* RT_SNAKE (App A.1): flat space in (t, w, y, z), w = x - A sin(k pi y); metric Eq A1,
                                Cartesian-aligned tetrad (Eq A2 read as the co-frame, DESIGN S27): omega = 0, n^w = n^x - delta n^y */
    /* RT_USER (L57-79: any stationary metric with an orthonormal tetrad whose e_0 is normal to t = const, Eq 4).  HOST functions,
     * called only inside rt_init, at cell centres, face centres and the finite-difference points of Eq 8 (x = logical x1, x2,
     * x3; must not depend on x3, x3_symmetric = 1 is required):
     *   g_fn  fills the covariant metric g[mu][nu] (symmetric, signature - + + +); required;
     *   e_fn  fills e[mu][a] = e^mu_a-hat (orthonormal, e_0 along -grad t: Eq 4); NULL = the library builds the tetrad as for
     *         RT_KS_MKS (e_0 from Eq 4, then Gram-Schmidt of d_3, d_2, d_1 in the 3-metric);
     *   user  is handed back to both.  A point with sqrt(-g) = 0 (coordinate axis) is a zero-area location: no flux crosses it. */
    void (*g_fn)(const double x[3], double g[4][4], void *user);
    void (*e_fn)(const double x[3], double e[4][4], void *user);
    void *user;
} rt_metric;

typedef struct {
    int limiter;       /* RT_LIM_* (S7: monotonised central by default) */
    int angular_recon; /* RT_ANG_DONOR (first order, L227) | RT_ANG_MAPR (minimum-angle plane reconstruction, reading S6) */
    int source_method; /* 0 = no source step; 1, 2, 3 = Methods 1-3 of section 3.6.2 */
    double n0_floor;   /* mask directions with n_0 > -n0_floor (L284; 0.1) */
    double rho_floor;  /* no interaction below this density (L468; 5e-4) */
    double kappa_a0;   /* absorption: alpha^a = kappa_a0 rho^2 T^-3.5 (L403) */
    double kappa_s;    /* scattering: alpha^s = kappa_s rho */
    double a_rad;      /* radiation constant in code units */
    double Y_over_rho; /* k_B / ((Gamma-1) mu m_p), so that Y = Y_over_rho * rho (L399) */
    double abar;       /* a-bar of tau = abar alpha dt (L262; 1) */
    int transport_variant; /* RT_TRANSPORT_* (0) */
    int transport_tile[3]; /* RT_TRANSPORT_TMA tile: columns along x1, along x2, directions per chunk (even); all 0 = chosen by
                              rt_init for the mesh */
    /* L215: the geodesic grid "can be deformed in advance by performing a Lorentz transformation of its directions" and
     * "oriented along a pre-defined direction".  grid_axis: direction (tetrad components 1-3, any length) the grid's pole is
     * turned to; grid_boost: velocity (c = 1, |beta| < 1) of the frame in which the grid is the regular one -- the cells crowd
     * around +beta.  Zero vectors = the regular grid with its pole along tetrad axis 3 (S2).  Numbering and neighbour lists do
     * not change; areas, edges and the angular coefficients are those of the deformed cells.  A grid without the x-z mirror
     * symmetry cannot serve RT_BC_REFLECT (rt_init returns RT_EINVAL). */
    double grid_axis[3], grid_boost[3];
    int angflux_split;     /* 0: the angular flux of Eq 19 is upwinded on the total normal velocity of the edge (reading S5, the
                              default); 1: term by term as printed (L239), the zeta-hat and psi-hat parts of the velocity each
                              upwinded on its own sign.  Donor-cell reconstruction only (rt_init returns RT_EINVAL with MAPR). */
    int source_literal;    /* 0: the intensity update (Eq 35) uses the coefficients the temperature equation was built from, so
                              that the updated intensities add up to E_+ of Eq 39 (reading S19b, the default); 1: "the opacities
                              must be updated and are therefore recalculated for the new value of T_+" (L432) taken literally for
                              source Methods 2 and 3: every opacity of Eq 35 at T_+ (energy then balances to O(alpha_+ - alpha_-)) */
} rt_options;

/* Build the angular grid with N_d = 10 angle_level^2 + 2 directions (L207-213; angle_level = 2^generation is the
 * paper's rule, other levels by the extension S1), tetrads and Ricci rotation coefficients (Eq 8, 6th-order finite
 * differences, h = 5e-4), and every per-column table; upload them.  Host-side, not timed.  *out is owned by the
 * library until rt_free. */
int rt_init(const rt_grid *grid, const rt_metric *metric, int angle_level, const rt_options *opt, rt_ctx **out);
int rt_free(rt_ctx *ctx);
int rt_ndir(const rt_ctx *ctx);
int rt_ndir_padded(const rt_ctx *ctx);

/* Angular tables to HOST buffers: nhat[N_d][3], w[N_d] (solid angles, sum = 4 pi), nnb[N_d] (5 or 6),
 * nb[N_d][6] (neighbour per edge slot, -1 padded).  Any pointer may be NULL. */
int rt_get_directions(const rt_ctx *ctx, double *nhat_host, double *w_host, int *nnb_host, int *nb_host);
/* Geometry tables to a HOST buffer (shapes above). */
int rt_get_geometry(const rt_ctx *ctx, int which, double *host_out);
/* Time-step bounds to HOST: out[0] = half the light-crossing time of the smallest cell (L464), out[1] = the
 * angular-flux bound dt * (outflow rate of an angular cell) <= 1/2 (S14; +inf when omega = 0). */
int rt_cfl_dt(const rt_ctx *ctx, double out_host[2]);

/* RT_BC_FIXED ghost values for side (0 lo, 1 hi) of dim: device array [2 layers][face cells][pitch], layer 0
 * next to the interior, face cell index = (other dims, lower dim fastest).  The pointer is kept, not copied. */
int rt_set_boundary(rt_ctx *ctx, int dim, int side, const double *ghost_dev);
/* Fluid state: rho[N_c], T[N_c], u4[4][N_c] coordinate-frame u^mu (NULL = tetrad rest frame e_0).  Copied into
 * library-owned buffers on `stream`; T is the temperature used for the transport opacities of rt_transport.  Also
 * rebuilds the interaction list (cells with rho >= rho_floor, L468) on the device; nothing is read back and the stream is not
 * synchronised, so the call may be made every step (coupled GRMHD use, L448-456). */
int rt_set_fluid(rt_ctx *ctx, const double *rho_dev, const double *T_dev, const double *u4_dev, void *stream);

/* I_out = (n^0 n_0 I_base - dt D_x[I_in]) / (n^0 n_0), then mask + zero bands (O3 + O5).  I_out may alias I_base
 * but not I_in.  I_base may equal I_in. */
int rt_transport(rt_ctx *ctx, const double *I_in_dev, const double *I_base_dev, double *I_out_dev, double dt, void *stream);
/* rt_transport for callers that cannot allocate (code under CUDA graph capture, tight serving loops, harnesses that forbid
 * cudaMalloc): same arguments, same result bit for bit, but the scratch of the launch (the per-face coefficients of Eq 23 and
 * the column / cell flags; rt_transport keeps them in buffers rt_init allocated) lives in ONE file-scope device array of
 * RT_STATIC_SCRATCH_BYTES that every GPU loading the library holds until exit.  The call makes no cudaMalloc, cudaFree or
 * allocating library call (its first use on a device resolves the array's address with cudaGetSymbolAddress).  A mesh whose
 * faces need more (32 bytes per face of the three dims + the flag words; about 85 000 cells fit) is refused with RT_ETOOBIG;
 * without opacities no scratch is needed and any mesh is accepted.  The array is shared by all contexts and keeps the last
 * call's contents (every entry that is read is rewritten first, nothing needs clearing): calls that OVERLAP on the GPU --
 * different streams without ordering, different contexts -- race on it; serialise them. */
#define RT_STATIC_SCRATCH_BYTES (8u << 20)
int rt_transport_static(rt_ctx *ctx, const double *I_in_dev, const double *I_base_dev, double *I_out_dev, double dt, void *stream);
/* I_inout -= dt D_Omega[I_in] / (n^0 n_0), then mask + zero bands (O4 + O5).  No-op when omega = 0. */
int rt_angular_flux(rt_ctx *ctx, const double *I_in_dev, double *I_inout_dev, double dt, void *stream);
/* Implicit source step O6 in place on (I, T); *n_fail_dev (device int, may be NULL) += cells whose solve failed. */
int rt_source_implicit(rt_ctx *ctx, double *I_inout_dev, double *T_inout_dev, double dt, int *n_fail_dev, void *stream);
/* R[16][N_c] = R^mu_nu (O7). */
int rt_moments(rt_ctx *ctx, const double *I_dev, double *R_dev, void *stream);
/* One predictor-corrector step O8 in place on (I, T).  R_out[16][N_c] = moments after the step (may be NULL),
 * G_out[4][N_c] = G_nu = -(R^0_nu after - before the corrector's source step)/dt (may be NULL).
 * n_fail_dev as above.  The fluid (rho, u4) is the one last given to rt_set_fluid; T comes from T_inout. */
int rt_step(rt_ctx *ctx, double *I_inout_dev, double *T_inout_dev, double *R_out_dev, double *G_out_dev, double dt,
            int *n_fail_dev, void *stream);

/* rt_step with HOST buffers (pinned memory, or the copies cannot overlap): I[N_c][pitch] and T[N_c] are updated in place, R[16][N_c]
 * and G[4][N_c] (may be NULL) are written; the call returns after everything has landed on the host.  *n_fail_host (may be
 * NULL) receives the number of cells whose temperature solve failed.  Meshes with N3 >= 16 and no FIXED boundary are cut
 * into N3 / 8 x3-slabs with a 4-plane halo (the domain of dependence of one step): every plane crosses PCIe once, a slab is
 * stepped by the plain rt_step as soon as its planes have arrived and its owned planes go back while later slabs arrive or
 * compute (three internal streams, ordered after `stream`); other meshes go H2D -> rt_step -> D2H back to back.  Either way
 * the result is rt_step's, bit for bit.  The slab contexts and device buffers are built on the first call. */
int rt_step_host(rt_ctx *ctx, double *I_inout_host, double *T_inout_host, double *R_out_host, double *G_out_host, double dt,
                 int *n_fail_host, void *stream);

/* Per-kernel device timing (bench.py's roofline): while enabled, every kernel launch is bracketed by CUDA events
 * on its stream.  rt_profile_read synchronises on the last event, returns the accumulated milliseconds and launch
 * counts per kernel class (HOST arrays of RT_K_COUNT entries) and resets the accumulators. */
enum { RT_K_FACECOEF = 0, RT_K_TRANSPORT = 1, RT_K_ANGULAR = 2, RT_K_SOURCE = 3, RT_K_MOMENTS = 4, RT_K_COUNT = 5 };
int rt_profile_enable(rt_ctx *ctx, int on);
int rt_profile_read(rt_ctx *ctx, double *ms_host, long long *count_host);

/* One step of a rank's slab in a multi-GPU decomposition along x3, the planes its neighbours need FIRST (L778: "treating the boundaries
 * first and overlapping the transfer with the interior").  `ctx` is the rank's EXTENDED slab: RT_SLAB_MARGIN = 4 planes of halo on every
 * cut side (the domain of dependence of one predictor-corrector step), OUTFLOW there.  On `halo_stream` the library steps, per cut
 * side, a sub-slab of 3 x RT_SLAB_MARGIN planes with a context of its own and leaves in the caller's DEVICE send buffers the
 * RT_SLAB_MARGIN owned planes next to the cut as they will be after this step, bit for bit: send_lo_I [4][ncol][pitch], send_lo_T
 * [4][ncol] = planes 4..7 of the slab (NULL, both: no cut below), send_hi_* = planes n3-8 .. n3-5 (NULL: no cut above).  On `stream` the
 * whole slab is stepped exactly as by rt_step (I, T in place; R, G, n_fail as there).  The caller sends / receives on `halo_stream`
 * (ordered after the library's work there) while `stream` computes, and copies what it received into the halo planes (planes 0..3 and
 * n3-4 .. n3-1: contiguous) once `stream` has finished the step.  Costs 3 x RT_SLAB_MARGIN extra planes of compute per cut side; not
 * available with RT_BC_FIXED boundaries (RT_EINVAL).  With all four buffers NULL it is rt_step. */
#define RT_SLAB_MARGIN 4
int rt_step_slab(rt_ctx *ctx, double *I_inout_dev, double *T_inout_dev, double *R_out_dev, double *G_out_dev, double dt, int *n_fail_dev,
                 double *send_lo_I_dev, double *send_lo_T_dev, double *send_hi_I_dev, double *send_hi_T_dev, void *stream, void *halo_stream);

/* Which spatial transport path rt_init selected, to HOST: out[0] = RT_TRANSPORT_* actually used (RT_TRANSPORT_L2 when the
 * tile kernel's conditions do not hold), out[1..3] = the tile in the order of rt_options.transport_tile. */
int rt_transport_info(const rt_ctx *ctx, int out_host[4]);

/* number of kernels the library launched since rt_init (for bench.py's gpu_launches) */
long long rt_launch_count(const rt_ctx *ctx);
int rt_last_cuda_error(void);
const char *rt_strerror(int code);

#ifdef __cplusplus
}
#endif
#endif /* RT_H_ */
