// C ABI of librt_b200 (include/rt.h): context, init-time precompute (a0), and the rt_* entry points.
#include <climits>
#include <cmath>
#include <cstring>
#include <limits>
#include <new>
#include <vector>

#include <cub/device/device_partition.cuh>
#include <cub/iterator/counting_input_iterator.cuh>

#include "rt_kernels.cuh"

using namespace rt;

struct rt_ctx {
    rt_grid grid;
    rt_metric metric;
    rt_options opt;
    int level, nd, pitch, ncol;
    long long ncell;
    bool curved;   // omega != 0 somewhere: the angular-flux kernel has work to do
    bool matter;   // any opacity: Eq 23 faces may exist
    bool fluid_set;
    AngularGrid ang;
    // host copies of the geometry tables (rt_get_geometry, rt_cfl_dt)
    std::vector<double> h_g, h_e, h_einv, h_sqrtg, h_omega, h_n0, h_angcoef;
    DeviceTables tab;
    double *d_rho, *d_u4, *d_T, *d_Th, *d_Ih, *d_fcoef[3];
    int *d_genlist, *d_srclist;   // d_srclist: [ncell] listed cells first (ascending), the rest behind them; d_nsel: how many are listed
    int *d_nsel; void *d_part_tmp; size_t part_tmp_bytes;   // interaction-list partition (cub) scratch
    double *d_hI, *d_hT, *d_hR, *d_hG;   // device staging of rt_step_host (allocated on first use)
    int *d_hfail;
    // rt_step_host pipeline (x3 slabs with a 4-plane halo, each its own context over the same metric): built on first use
    struct HostSlab { rt_ctx *sub; int k0, k1, ext_lo, ext_hi, n3l; double *I, *T, *R, *G, *rho, *u4; cudaEvent_t done; };
    std::vector<HostSlab> hslabs;
    HostSlab bslab[2];                 // rt_step_slab: the boundary sub-slabs (3 margins of planes) at the low / high x3 end
    cudaEvent_t bev_in, bev_cloned; long long bslab_fluid_version; int *d_bfail;
    cudaStream_t hs_in, hs_cmp, hs_out;
    std::vector<cudaEvent_t> hev;      // one event per uploaded chunk
    cudaEvent_t hev_start, hev_end[3];
    long long fluid_version, hslab_fluid_version;
    bool is_sub;                       // a slab context of another context's pipeline
    double *d_mapr_xi, *d_mapr_xim, *d_mapr_a, *d_angraw;
    int *d_mapr_back, *d_mapr_nnb;
    unsigned char *d_angup;
    unsigned char *d_cls;     // per (column, s): dead / general class (k_classify)
    double *d_paircoef, *d_paircoefz;   // per (column, s): geometry tables of the tile kernels (k_paircoef)
    bool u4_rest;             // d_u4 holds the tetrad rest frame (rt_set_fluid with u4 == NULL)
    unsigned char *d_colflag; // per column: bit 0 has such a cell, bit 1 has an all-vacuum cell
    KParams kp;
    long long launches;
    bool profiling;
    struct Span { int cls; cudaEvent_t a, b; };
    std::vector<Span> spans;
};

// brackets one launcher call with events when profiling is on
struct ProfScope {
    rt_ctx *c; int cls; cudaStream_t st; cudaEvent_t a, b; bool on;
    ProfScope(rt_ctx *c_, int cls_, cudaStream_t st_) : c(c_), cls(cls_), st(st_), on(c_->profiling) {
        if (on) { cudaEventCreate(&a); cudaEventCreate(&b); cudaEventRecord(a, st); }
    }
    ~ProfScope() {
        if (on) { cudaEventRecord(b, st); c->spans.push_back({cls, a, b}); }
    }
};

static int g_last_cuda = 0;
#define CK(call)                                                       \
    do {                                                               \
        cudaError_t e_ = (call);                                       \
        if (e_ != cudaSuccess) { g_last_cuda = (int)e_; return RT_ECUDA; } \
    } while (0)

template <typename T>
static cudaError_t upload(T **dst, const std::vector<T> &src) {
    cudaError_t e = cudaMalloc((void **)dst, src.size() * sizeof(T));
    if (e != cudaSuccess) return e;
    return cudaMemcpy(*dst, src.data(), src.size() * sizeof(T), cudaMemcpyHostToDevice);
}

static void fill_face_entry(double *f, const PointGeom &g, int a) {
    for (int q = 0; q < FACE_STRIDE; ++q) f[q] = 0.0;
    if (g.dead || !(g.sqrtg > 0)) return;
    for (int b = 0; b < 4; ++b) {
        f[b] = g.sqrtg * g.e[1 + a][b];
        double c = 0;
        for (int mu = 0; mu < 4; ++mu) c += g.g[0][mu] * g.e[mu][b];
        f[4 + b] = c;
        f[8 + b] = g.sqrtg * g.e[0][b];
    }
}

extern "C" int rt_init(const rt_grid *grid, const rt_metric *metric, int angle_level, const rt_options *opt, rt_ctx **out) {
    if (!grid || !metric || !opt || !out) return RT_EINVAL;
    for (int a = 0; a < 3; ++a) {
        if (grid->n[a] < 1 || !(grid->dx[a] > 0)) return RT_EINVAL;
        if (grid->bc_lo[a] < 0 || grid->bc_lo[a] > RT_BC_REFLECT || grid->bc_hi[a] < 0 || grid->bc_hi[a] > RT_BC_REFLECT) return RT_EINVAL;
        if (a != 1 && (grid->bc_lo[a] == RT_BC_REFLECT || grid->bc_hi[a] == RT_BC_REFLECT)) return RT_EINVAL;   // no mirror symmetry of the angular grid there
        if ((grid->bc_lo[a] == RT_BC_PERIODIC) != (grid->bc_hi[a] == RT_BC_PERIODIC)) return RT_EINVAL;
        if (grid->zero_lo[a] < 0 || grid->zero_hi[a] < 0) return RT_EINVAL;
    }
    if (metric->kind < 0 || metric->kind > RT_USER) return RT_EINVAL;
    if (metric->kind == RT_USER && (!metric->g_fn || !metric->x3_symmetric)) return RT_EINVAL;
    if (opt->angflux_split && opt->angular_recon != 0) return RT_EINVAL;
    if ((metric->kind == RT_KS_MKS || metric->kind == RT_BL_MKS) && (!metric->x3_symmetric || std::fabs(metric->a) >= 1.0)) return RT_EINVAL;
    if (metric->kind == RT_BL_MKS && !(std::exp(grid->x0[0]) > 1.0 + std::sqrt(1.0 - metric->a * metric->a))) return RT_EINVAL;   // outside the horizon only
    if (opt->angular_recon != RT_ANG_DONOR && opt->angular_recon != RT_ANG_MAPR) return RT_EINVAL;
    if (opt->limiter < 0 || opt->limiter > 3 || opt->source_method < 0 || opt->source_method > 3) return RT_EINVAL;
    if (opt->transport_variant != RT_TRANSPORT_TMA && opt->transport_variant != RT_TRANSPORT_L2) return RT_EINVAL;
    if (opt->source_method != 0 && !(opt->Y_over_rho > 0)) return RT_EINVAL;

    rt_ctx *c = new (std::nothrow) rt_ctx();
    if (!c) return RT_ENOMEM;
    c->grid = *grid; c->metric = *metric; c->opt = *opt; c->level = angle_level;
    c->launches = 0; c->fluid_set = false; c->profiling = false;
    c->hs_in = c->hs_cmp = c->hs_out = nullptr; c->hev_start = nullptr; c->hev_end[0] = c->hev_end[1] = c->hev_end[2] = nullptr;
    c->fluid_version = 0; c->hslab_fluid_version = -1; c->is_sub = false;
    if (!build_angular_grid(angle_level, opt->grid_axis, opt->grid_boost, c->ang)) { delete c; return RT_EINVAL; }
    const int nd = c->nd = c->ang.nd;
    const int pitch = c->pitch = (nd + 3) / 4 * 4;
    const int n1 = grid->n[0], n2 = grid->n[1], n3 = grid->n[2];
    const int ncol = c->ncol = n1 * n2;
    c->ncell = (long long)ncol * n3;
    // limits of the kernels (32-bit element offsets inside an x3-plane and cell indices in the lists; one thread per
    // direction in the angular kernels; at most 21 values per lane in the per-cell kernels): refused here, not at the first step
    if ((long long)n1 * n2 > INT_MAX || nd > 672 || pitch > 1024 || c->ncell > INT_MAX || (long long)ncol * pitch > INT_MAX) { delete c; return RT_EINVAL; }
    c->matter = (opt->kappa_a0 != 0.0 || opt->kappa_s != 0.0);
    const double x3c = grid->x0[2] + 0.5 * grid->dx[2];

    // ---- geometry at centres and faces ----
    std::vector<double> cen((size_t)ncol * CEN_STRIDE, 0.0), ecen((size_t)ncol * 16);
    c->h_g.resize((size_t)ncol * 16); c->h_e.resize((size_t)ncol * 16); c->h_einv.resize((size_t)ncol * 16);
    c->h_sqrtg.resize(ncol); c->h_omega.resize((size_t)ncol * 64); c->h_n0.resize((size_t)ncol * nd);
    c->h_angcoef.assign((size_t)ncol * 6 * nd, 0.0);
    std::vector<double> face[3];
    face[0].resize((size_t)(n1 + 1) * n2 * FACE_STRIDE);
    face[1].resize((size_t)n1 * (n2 + 1) * FACE_STRIDE);
    face[2].resize((size_t)ncol * FACE_STRIDE);
    std::vector<double> angc((size_t)ncol * ANG_SLOTS * pitch, 0.0);
    const bool mapr = opt->angular_recon == RT_ANG_MAPR;
    std::vector<double> angraw(mapr ? (size_t)ncol * 6 * pitch : 0, 0.0);
    std::vector<unsigned char> angup(mapr ? (size_t)ncol * pitch : 0, 0);
    double omax = 0.0;
    for (int j = 0; j < n2; ++j)
        for (int i = 0; i < n1; ++i) {
            const size_t col = (size_t)j * n1 + i;
            const double x[3] = {grid->x0[0] + (i + 0.5) * grid->dx[0], grid->x0[1] + (j + 0.5) * grid->dx[1], x3c};
            PointGeom g;
            eval_point(*metric, x, g);
            if (g.dead) { delete c; return RT_EINVAL; }   // a cell centre on the polar axis
            double om[4][4][4];
            eval_omega(*metric, x, om);
            std::memcpy(&c->h_g[col * 16], g.g, 128); std::memcpy(&c->h_e[col * 16], g.e, 128);
            std::memcpy(&c->h_einv[col * 16], g.einv, 128); std::memcpy(&c->h_omega[col * 64], om, 512);
            c->h_sqrtg[col] = g.sqrtg;
            double *ce = &cen[col * CEN_STRIDE];
            for (int b = 0; b < 4; ++b) {
                double s0 = 0;
                for (int mu = 0; mu < 4; ++mu) s0 += g.g[0][mu] * g.e[mu][b];
                ce[b] = s0;
                ce[4 + b] = g.e[0][b];
                for (int nu = 0; nu < 4; ++nu) {
                    double l = 0;
                    for (int lam = 0; lam < 4; ++lam) l += g.e[lam][b] * g.g[lam][nu];
                    ce[28 + 4 * b + nu] = l;
                }
            }
            ce[8] = 1.0 / g.sqrtg;
            std::memcpy(ce + 12, g.einv, 128);
            std::memcpy(&ecen[col * 16], g.e, 128);
            fill_face_entry(&face[2][col * FACE_STRIDE], g, 2);
            // per-direction n_0 and per-edge angular coefficients
            const AngularGrid &A = c->ang;
            for (int s = 0; s < nd; ++s)
                c->h_n0[col * nd + s] = ce[0] + ce[1] * A.nhat[3 * s] + ce[2] * A.nhat[3 * s + 1] + ce[3] * A.nhat[3 * s + 2];
            for (int s = 0; s < nd; ++s) {
                double self = 0.0;
                for (int e = 0; e < A.nnb[s]; ++e) {
                    const double *m3 = &A.emid[3 * (6 * s + e)], *u3 = &A.eun[3 * (6 * s + e)];
                    const double m[4] = {1.0, m3[0], m3[1], m3[2]};
                    double V = 0.0, a3[3];
                    for (int ii = 1; ii < 4; ++ii) {
                        double q = 0.0;
                        for (int cc = 0; cc < 4; ++cc) for (int d = 0; d < 4; ++d) q += om[ii][cc][d] * m[cc] * m[d];
                        a3[ii - 1] = -q;
                        V -= u3[ii - 1] * q;                                     // a(m_e) . u_e  (Eq 7-8, S4)
                    }
                    // Eq 19 as printed (L239): the zeta-hat and psi-hat parts of the normal velocity, upwinded one by one
                    double Vout = V > 0 ? V : 0.0, Vin = V > 0 ? 0.0 : V;        // what multiplies the own / the neighbour's value
                    if (opt->angflux_split) {
                        const double sz = std::sqrt(m3[0] * m3[0] + m3[1] * m3[1]);
                        const double cp = sz > 0 ? m3[0] / sz : 1.0, sp = sz > 0 ? m3[1] / sz : 0.0;
                        const double ez[3] = {m3[2] * cp, m3[2] * sp, -sz}, ep[3] = {-sp, cp, 0.0};
                        const double Vz = (a3[0] * ez[0] + a3[1] * ez[1] + a3[2] * ez[2]) * (u3[0] * ez[0] + u3[1] * ez[1] + u3[2] * ez[2]);
                        const double Vp = (a3[0] * ep[0] + a3[1] * ep[1] + a3[2] * ep[2]) * (u3[0] * ep[0] + u3[1] * ep[1] + u3[2] * ep[2]);
                        Vout = std::fmax(Vz, 0.0) + std::fmax(Vp, 0.0);
                        Vin = std::fmin(Vz, 0.0) + std::fmin(Vp, 0.0);
                    }
                    omax = std::fmax(omax, std::fabs(V));
                    const double n0e = ce[0] + ce[1] * m3[0] + ce[2] * m3[1] + ce[3] * m3[2];
                    const int t = A.nb[6 * s + e];
                    const double n0s = c->h_n0[col * nd + s], n0t = c->h_n0[col * nd + t];
                    const bool gate = ((n0s > 0) - (n0s < 0)) != ((n0t > 0) - (n0t < 0));   // L280
                    const double c0 = gate ? 0.0 : A.dlam[6 * s + e] * n0e / A.w[s];
                    const double coef = c0 * V;                                 // Eq 19 / Eq 18
                    c->h_angcoef[(col * 6 + e) * nd + s] = coef;
                    if (mapr) {
                        angraw[(col * 6 + e) * pitch + s] = coef;
                        if (V > 0) angup[col * pitch + s] |= (unsigned char)(1u << e);
                    }
                    self += c0 * Vout;                                          // upwind: own value (S5)
                    angc[(col * ANG_SLOTS + e) * pitch + s] = c0 * Vin;         // upwind: neighbour's value
                }
                angc[(col * ANG_SLOTS + 6) * pitch + s] = self;
            }
        }
    for (int j = 0; j < n2; ++j)
        for (int i = 0; i <= n1; ++i) {
            const double x[3] = {grid->x0[0] + i * grid->dx[0], grid->x0[1] + (j + 0.5) * grid->dx[1], x3c};
            PointGeom g;
            eval_point(*metric, x, g);
            fill_face_entry(&face[0][((size_t)j * (n1 + 1) + i) * FACE_STRIDE], g, 0);
        }
    for (int j = 0; j <= n2; ++j)
        for (int i = 0; i < n1; ++i) {
            const double x[3] = {grid->x0[0] + (i + 0.5) * grid->dx[0], grid->x0[1] + j * grid->dx[1], x3c};
            PointGeom g;
            eval_point(*metric, x, g);
            fill_face_entry(&face[1][((size_t)j * n1 + i) * FACE_STRIDE], g, 1);
        }
    c->curved = omax > 0.0;

    // ---- angular tables, padded ----
    std::vector<double> nh(3 * (size_t)pitch, 0.0), w(pitch, 0.0);
    std::vector<int> nb(6 * (size_t)pitch, 0);
    for (int s = 0; s < pitch; ++s)
        for (int e = 0; e < 6; ++e) nb[e * pitch + s] = (s < nd && c->ang.nb[6 * s + e] >= 0) ? c->ang.nb[6 * s + e] : (s < nd ? s : 0);
    for (int s = 0; s < nd; ++s) {
        for (int q = 0; q < 3; ++q) nh[q * pitch + s] = c->ang.nhat[3 * s + q];
        w[s] = c->ang.w[s];
    }

    // reflecting x2 boundary: the permutation s -> direction with n-hat^2 flipped (the x-z plane is a mirror plane of the
    // grid: pole along 3-hat, a vertex at azimuth 0).  Looked up by nearest direction and verified.
    std::vector<int> mir;
    if (grid->bc_lo[1] == RT_BC_REFLECT || grid->bc_hi[1] == RT_BC_REFLECT) {
        mir.assign(pitch, 0);
        bool ok = true;
        for (int s = 0; s < nd; ++s) {
            int best = -1;
            double bd = 1e300;
            for (int t2 = 0; t2 < nd; ++t2) {
                const double dxn = c->ang.nhat[3 * t2] - c->ang.nhat[3 * s], dyn = c->ang.nhat[3 * t2 + 1] + c->ang.nhat[3 * s + 1],
                             dzn = c->ang.nhat[3 * t2 + 2] - c->ang.nhat[3 * s + 2];
                const double d = dxn * dxn + dyn * dyn + dzn * dzn;
                if (d < bd) { bd = d; best = t2; }
            }
            if (!(bd < 1e-18)) ok = false;
            mir[s] = best;
        }
        for (int s = 0; s < nd && ok; ++s) ok = mir[mir[s]] == s;
        if (!ok) { delete c; return RT_EINVAL; }
    }

    // ---- upload ----
    DeviceTables &t = c->tab;
    std::memset(&t, 0, sizeof t);
    cudaError_t e = cudaSuccess;
    if (!mir.empty()) e = upload(&t.mirror, mir);
    for (int a = 0; a < 3 && e == cudaSuccess; ++a) e = upload(&t.face[a], face[a]);
    if (e == cudaSuccess) e = upload(&t.cen, cen);
    if (e == cudaSuccess) e = upload(&t.ecen, ecen);
    if (e == cudaSuccess) e = upload(&t.angcoef, angc);
    if (e == cudaSuccess) e = upload(&t.nhat, nh);
    if (e == cudaSuccess) e = upload(&t.w, w);
    if (e == cudaSuccess) e = upload(&t.nb, nb);
    const size_t nI = (size_t)c->ncell * pitch;
    c->d_rho = c->d_u4 = c->d_T = c->d_Th = c->d_Ih = nullptr;
    c->d_fcoef[0] = c->d_fcoef[1] = c->d_fcoef[2] = nullptr;
    c->u4_rest = false; c->d_colflag = nullptr; c->d_cls = nullptr; c->d_paircoef = nullptr; c->d_paircoefz = nullptr; c->d_genlist = nullptr; c->d_srclist = nullptr; c->d_nsel = nullptr; c->d_part_tmp = nullptr; c->part_tmp_bytes = 0;
    c->d_hI = c->d_hT = c->d_hR = c->d_hG = nullptr; c->d_hfail = nullptr;
    std::memset(c->bslab, 0, sizeof c->bslab); c->bev_in = c->bev_cloned = nullptr; c->bslab_fluid_version = -1; c->d_bfail = nullptr;
    c->d_mapr_xi = c->d_mapr_xim = c->d_mapr_a = c->d_angraw = nullptr; c->d_mapr_back = c->d_mapr_nnb = nullptr; c->d_angup = nullptr;
    if (e == cudaSuccess) e = cudaMalloc((void **)&c->d_cls, (size_t)ncol * pitch);
    if (e == cudaSuccess) e = cudaMalloc((void **)&c->d_colflag, colflag_bytes(c->ncol, n3));   // column flags, x3-chunk flags, cell-flag masks
    if (e == cudaSuccess) e = cudaMalloc((void **)&c->d_rho, c->ncell * sizeof(double));
    if (e == cudaSuccess) e = cudaMalloc((void **)&c->d_u4, 4 * c->ncell * sizeof(double));
    if (e == cudaSuccess) e = cudaMalloc((void **)&c->d_T, c->ncell * sizeof(double));
    if (e == cudaSuccess) e = cudaMalloc((void **)&c->d_Th, c->ncell * sizeof(double));
    if (e == cudaSuccess) e = cudaMalloc((void **)&c->d_Ih, nI * sizeof(double));
    for (int a = 0; a < 3 && e == cudaSuccess; ++a) {
        size_t nf = (size_t)(n1 + (a == 0)) * (n2 + (a == 1)) * (n3 + (a == 2));
        e = cudaMalloc((void **)&c->d_fcoef[a], nf * 4 * sizeof(double));
    }
    if (e != cudaSuccess) { g_last_cuda = (int)e; rt_free(c); return e == cudaErrorMemoryAllocation ? RT_ENOMEM : RT_ECUDA; }

    KParams &k = c->kp;
    std::memset(&k, 0, sizeof k);
    k.n1 = n1; k.n2 = n2; k.n3 = n3; k.nd = nd; k.pitch = pitch; k.ncol = ncol; k.ncell = c->ncell;
    for (int a = 0; a < 3; ++a) {
        k.inv_dx[a] = 1.0 / grid->dx[a];
        k.bc_lo[a] = grid->bc_lo[a]; k.bc_hi[a] = grid->bc_hi[a];
        k.zlo[a] = grid->zero_lo[a]; k.zhi[a] = grid->zero_hi[a];
        k.face[a] = t.face[a];
    }
    k.limiter = opt->limiter; k.method = opt->source_method; k.source_literal = opt->source_literal;
    k.n0_floor = opt->n0_floor; k.rho_floor = opt->rho_floor; k.kappa_a0 = opt->kappa_a0; k.kappa_s = opt->kappa_s;
    k.a_rad = opt->a_rad; k.Y_over_rho = opt->Y_over_rho; k.abar = opt->abar;
    k.cen = t.cen; k.ecen = t.ecen; k.angcoef = t.angcoef; k.nhat = t.nhat; k.w = t.w; k.nb = t.nb; k.mirror = t.mirror;
    k.rho = c->d_rho; k.u4 = c->d_u4;
    k.cls = c->d_cls;
    if (mapr) {   // grid-only MAPR tables (S6): log maps of the neighbours and of the edge centres, pair matrices
        const AngularGrid &A = c->ang;
        std::vector<double> xi(18 * (size_t)pitch, 0.0), xim(18 * (size_t)pitch, 0.0), am(24 * (size_t)pitch, 0.0);
        std::vector<int> back(6 * (size_t)pitch, 0), nnb(pitch, 0);
        auto logmap = [](const double *c0, const double *q, double out[3]) {
            const double dot = c0[0] * q[0] + c0[1] * q[1] + c0[2] * q[2];
            const double pv[3] = {q[0] - dot * c0[0], q[1] - dot * c0[1], q[2] - dot * c0[2]};
            const double pn = std::sqrt(pv[0] * pv[0] + pv[1] * pv[1] + pv[2] * pv[2]);
            const double ang = std::atan2(pn, dot);
            for (int x = 0; x < 3; ++x) out[x] = ang * pv[x] / pn;
        };
        for (int s = 0; s < nd; ++s) {
            nnb[s] = A.nnb[s];
            double x6[6][3];
            for (int e = 0; e < A.nnb[s]; ++e) {
                logmap(&A.nhat[3 * s], &A.nhat[3 * A.nb[6 * s + e]], x6[e]);
                double xm[3];
                logmap(&A.nhat[3 * s], &A.emid[3 * (6 * s + e)], xm);
                for (int x = 0; x < 3; ++x) { xi[(e * 3 + x) * pitch + s] = x6[e][x]; xim[(e * 3 + x) * pitch + s] = xm[x]; }
                back[e * pitch + s] = A.back[6 * s + e];
            }
            for (int e = 0; e < A.nnb[s]; ++e) {
                const int e2 = (e + 1) % A.nnb[s];
                double a11 = 0, a12 = 0, a22 = 0;
                for (int x = 0; x < 3; ++x) { a11 += x6[e][x] * x6[e][x]; a12 += x6[e][x] * x6[e2][x]; a22 += x6[e2][x] * x6[e2][x]; }
                am[(e * 4 + 0) * pitch + s] = a11; am[(e * 4 + 1) * pitch + s] = a12; am[(e * 4 + 2) * pitch + s] = a22;
                am[(e * 4 + 3) * pitch + s] = a11 * a22 - a12 * a12;
            }
        }
        e = upload(&c->d_mapr_xi, xi);
        if (e == cudaSuccess) e = upload(&c->d_mapr_xim, xim);
        if (e == cudaSuccess) e = upload(&c->d_mapr_a, am);
        if (e == cudaSuccess) e = upload(&c->d_mapr_back, back);
        if (e == cudaSuccess) e = upload(&c->d_mapr_nnb, nnb);
        if (e == cudaSuccess) e = upload(&c->d_angraw, angraw);
        if (e == cudaSuccess) e = upload(&c->d_angup, angup);
        if (e != cudaSuccess) { g_last_cuda = (int)e; rt_free(c); return RT_ECUDA; }
        k.mapr_xi = c->d_mapr_xi; k.mapr_xim = c->d_mapr_xim; k.mapr_a = c->d_mapr_a; k.mapr_back = c->d_mapr_back;
        k.mapr_nnb = c->d_mapr_nnb; k.angraw = c->d_angraw; k.angup = c->d_angup;
    }
    k.variant = (opt->transport_variant == RT_TRANSPORT_TMA && tile_eligible(k)) ? RT_TRANSPORT_TMA : RT_TRANSPORT_L2;
    choose_tile(k, opt->transport_tile, k.tile);
    e = launch_classify(k, c->d_cls, 0);
    if (e == cudaSuccess && k.variant == RT_TRANSPORT_TMA) {
        e = cudaMalloc((void **)&c->d_paircoef, (size_t)ncol * pitch * 8 * sizeof(double));
        if (e == cudaSuccess && c->matter) e = cudaMalloc((void **)&c->d_paircoefz, (size_t)ncol * pitch * 8 * sizeof(double));
        k.paircoef = c->d_paircoef; k.paircoefz = c->d_paircoefz;
        choose_tile_gen(k, k.tile_gen);
        if (e == cudaSuccess) e = launch_paircoef(k, c->d_paircoef, c->d_paircoefz, 0);
    }
    if (e == cudaSuccess) e = cudaDeviceSynchronize();
    if (e == cudaSuccess) {   // compact list of the general (column, s) pairs, in memory order
        std::vector<unsigned char> hc((size_t)ncol * pitch);
        e = cudaMemcpy(hc.data(), c->d_cls, hc.size(), cudaMemcpyDeviceToHost);
        std::vector<int> gl;
        for (size_t q = 0; q < hc.size(); ++q)
            if ((hc[q] & 2) && !(hc[q] & 1)) gl.push_back((int)q);
        k.ngen = (int)gl.size();
        if (e == cudaSuccess && k.ngen) { e = upload(&c->d_genlist, gl); k.genlist = c->d_genlist; }
    }
    if (e != cudaSuccess) { g_last_cuda = (int)e; rt_free(c); return RT_ECUDA; }
    *out = c;
    return RT_OK;
}

extern "C" int rt_free(rt_ctx *c) {
    if (!c) return RT_EINVAL;
    for (auto &h : c->hslabs) {
        if (h.sub) rt_free(h.sub);
        cudaFree(h.I); cudaFree(h.T); cudaFree(h.R); cudaFree(h.G); cudaFree(h.rho); cudaFree(h.u4);
        if (h.done) cudaEventDestroy(h.done);
    }
    for (auto &h : c->bslab) {
        if (h.sub) rt_free(h.sub);
        cudaFree(h.I); cudaFree(h.T); cudaFree(h.rho); cudaFree(h.u4);
    }
    if (c->bev_in) cudaEventDestroy(c->bev_in);
    if (c->bev_cloned) cudaEventDestroy(c->bev_cloned);
    cudaFree(c->d_bfail);
    for (auto e : c->hev) cudaEventDestroy(e);
    if (c->hev_start) cudaEventDestroy(c->hev_start);
    for (int q = 0; q < 3; ++q) if (c->hev_end[q]) cudaEventDestroy(c->hev_end[q]);
    if (c->hs_in) cudaStreamDestroy(c->hs_in);
    if (c->hs_cmp) cudaStreamDestroy(c->hs_cmp);
    if (c->hs_out) cudaStreamDestroy(c->hs_out);
    for (int a = 0; a < 3; ++a) { cudaFree(c->tab.face[a]); cudaFree(c->d_fcoef[a]); }
    cudaFree(c->tab.cen); cudaFree(c->tab.ecen); cudaFree(c->tab.angcoef); cudaFree(c->tab.nhat); cudaFree(c->tab.w);
    cudaFree(c->tab.nb); cudaFree(c->tab.mirror); cudaFree(c->d_colflag); cudaFree(c->d_cls); cudaFree(c->d_paircoef); cudaFree(c->d_paircoefz); cudaFree(c->d_genlist); cudaFree(c->d_srclist); cudaFree(c->d_nsel); cudaFree(c->d_part_tmp); cudaFree(c->d_hI); cudaFree(c->d_hT); cudaFree(c->d_hR); cudaFree(c->d_hG); cudaFree(c->d_hfail); cudaFree(c->d_mapr_xi); cudaFree(c->d_mapr_xim); cudaFree(c->d_mapr_a);
    cudaFree(c->d_angraw); cudaFree(c->d_mapr_back); cudaFree(c->d_mapr_nnb); cudaFree(c->d_angup); cudaFree(c->d_rho); cudaFree(c->d_u4); cudaFree(c->d_T); cudaFree(c->d_Th); cudaFree(c->d_Ih);
    delete c;
    return RT_OK;
}

extern "C" int rt_ndir(const rt_ctx *c) { return c ? c->nd : RT_EINVAL; }
extern "C" int rt_ndir_padded(const rt_ctx *c) { return c ? c->pitch : RT_EINVAL; }
extern "C" long long rt_launch_count(const rt_ctx *c) { return c ? c->launches : -1; }
extern "C" int rt_last_cuda_error(void) { return g_last_cuda; }

extern "C" int rt_transport_info(const rt_ctx *c, int out[4]) {
    if (!c || !out) return RT_EINVAL;
    out[0] = c->kp.variant;
    for (int q = 0; q < 3; ++q) out[1 + q] = c->kp.tile[q];
    return RT_OK;
}

extern "C" int rt_profile_enable(rt_ctx *c, int on) {
    if (!c) return RT_EINVAL;
    c->profiling = on != 0;
    return RT_OK;
}

extern "C" int rt_profile_read(rt_ctx *c, double *ms, long long *count) {
    if (!c || !ms || !count) return RT_EINVAL;
    for (int q = 0; q < RT_K_COUNT; ++q) { ms[q] = 0.0; count[q] = 0; }
    if (!c->spans.empty()) CK(cudaEventSynchronize(c->spans.back().b));
    for (auto &sp : c->spans) {
        float t = 0.f;
        CK(cudaEventElapsedTime(&t, sp.a, sp.b));
        ms[sp.cls] += t;
        count[sp.cls] += 1;
        cudaEventDestroy(sp.a); cudaEventDestroy(sp.b);
    }
    c->spans.clear();
    return RT_OK;
}

extern "C" const char *rt_strerror(int code) {
    switch (code) {
        case RT_OK: return "ok";
        case RT_EINVAL: return "invalid argument";
        case RT_ECUDA: return "CUDA runtime error (see rt_last_cuda_error)";
        case RT_ENOMEM: return "out of memory";
        case RT_ESTATE: return "call order: fluid or boundary data not set";
        case RT_ETOOBIG: return "mesh too large for the static scratch array (RT_STATIC_SCRATCH_BYTES)";
        default: return "unknown error";
    }
}

extern "C" int rt_get_directions(const rt_ctx *c, double *nhat, double *w, int *nnb, int *nb) {
    if (!c) return RT_EINVAL;
    if (nhat) std::memcpy(nhat, c->ang.nhat.data(), sizeof(double) * 3 * c->nd);
    if (w) std::memcpy(w, c->ang.w.data(), sizeof(double) * c->nd);
    if (nnb) std::memcpy(nnb, c->ang.nnb.data(), sizeof(int) * c->nd);
    if (nb) std::memcpy(nb, c->ang.nb.data(), sizeof(int) * 6 * c->nd);
    return RT_OK;
}

extern "C" int rt_get_geometry(const rt_ctx *c, int which, double *out) {
    if (!c || !out) return RT_EINVAL;
    const std::vector<double> *v = nullptr;
    switch (which) {
        case RT_GEOM_G_C: v = &c->h_g; break;
        case RT_GEOM_E_C: v = &c->h_e; break;
        case RT_GEOM_EINV_C: v = &c->h_einv; break;
        case RT_GEOM_SQRTG_C: v = &c->h_sqrtg; break;
        case RT_GEOM_OMEGA_C: v = &c->h_omega; break;
        case RT_GEOM_N0_C: v = &c->h_n0; break;
        case RT_GEOM_ANGCOEF: v = &c->h_angcoef; break;
        default: return RT_EINVAL;
    }
    std::memcpy(out, v->data(), v->size() * sizeof(double));
    return RT_OK;
}

extern "C" int rt_cfl_dt(const rt_ctx *c, double out[2]) {
    if (!c || !out) return RT_EINVAL;
    const double INF = std::numeric_limits<double>::infinity();
    double dts = INF, dta = INF;
    const rt_grid &G = c->grid;
    const AngularGrid &A = c->ang;
    const int nd = c->nd;
    for (int j = 0; j < G.n[1]; ++j)
        for (int i = 0; i < G.n[0]; ++i) {
            if (i < G.zero_lo[0] || i >= G.n[0] - G.zero_hi[0] || j < G.zero_lo[1] || j >= G.n[1] - G.zero_hi[1]) continue;
            const size_t col = (size_t)j * G.n[0] + i;
            const double *e = &c->h_e[col * 16];
            for (int s = 0; s < nd; ++s) {
                const double n0 = c->h_n0[col * nd + s];
                if (n0 > -c->opt.n0_floor) continue;
                const double *nh = &A.nhat[3 * s];
                double n[4];
                for (int mu = 0; mu < 4; ++mu) n[mu] = e[4 * mu] + e[4 * mu + 1] * nh[0] + e[4 * mu + 2] * nh[1] + e[4 * mu + 3] * nh[2];
                for (int a = 0; a < 3; ++a)
                    if (n[1 + a] != 0.0) dts = std::fmin(dts, 0.5 * G.dx[a] * n[0] / std::fabs(n[1 + a]));   // L464
                double rate = 0.0;   // sum over edges with V > 0 of V |n_0e| dlam / w  (coef = dlam n_0e V / w)
                for (int q = 0; q < A.nnb[s]; ++q) {
                    const double *m3 = &A.emid[3 * (6 * s + q)], *u3 = &A.eun[3 * (6 * s + q)];
                    const double m[4] = {1.0, m3[0], m3[1], m3[2]};
                    const double *om = &c->h_omega[col * 64];
                    double V = 0.0;
                    for (int ii = 1; ii < 4; ++ii) {
                        double qq = 0.0;
                        for (int cc = 0; cc < 4; ++cc) for (int d = 0; d < 4; ++d) qq += om[(ii * 4 + cc) * 4 + d] * m[cc] * m[d];
                        V -= u3[ii - 1] * qq;
                    }
                    if (c->opt.angflux_split) {   // what leaves through this edge when the two terms are upwinded one by one
                        double a3[3];
                        for (int ii = 1; ii < 4; ++ii) {
                            double qq = 0.0;
                            for (int cc = 0; cc < 4; ++cc) for (int d = 0; d < 4; ++d) qq += om[(ii * 4 + cc) * 4 + d] * m[cc] * m[d];
                            a3[ii - 1] = -qq;
                        }
                        const double sz = std::sqrt(m3[0] * m3[0] + m3[1] * m3[1]);
                        const double cp = sz > 0 ? m3[0] / sz : 1.0, sp = sz > 0 ? m3[1] / sz : 0.0;
                        const double ez[3] = {m3[2] * cp, m3[2] * sp, -sz}, ep[3] = {-sp, cp, 0.0};
                        const double Vz = (a3[0] * ez[0] + a3[1] * ez[1] + a3[2] * ez[2]) * (u3[0] * ez[0] + u3[1] * ez[1] + u3[2] * ez[2]);
                        const double Vp = (a3[0] * ep[0] + a3[1] * ep[1] + a3[2] * ep[2]) * (u3[0] * ep[0] + u3[1] * ep[1] + u3[2] * ep[2]);
                        V = std::fmax(Vz, 0.0) + std::fmax(Vp, 0.0);
                    }
                    if (V > 0) {
                        const double *g0 = &c->h_g[col * 16];
                        double n0e = 0.0;
                        for (int mu = 0; mu < 4; ++mu)
                            n0e += g0[mu] * (e[4 * mu] + e[4 * mu + 1] * m3[0] + e[4 * mu + 2] * m3[1] + e[4 * mu + 3] * m3[2]);
                        rate += V * std::fabs(n0e) * A.dlam[6 * s + q] / A.w[s];
                    }
                }
                if (rate > 0) dta = std::fmin(dta, 0.5 * std::fabs(n[0] * n0) / rate);                        // S14
            }
        }
    out[0] = dts; out[1] = dta;
    return RT_OK;
}

extern "C" int rt_set_boundary(rt_ctx *c, int dim, int side, const double *ghost_dev) {
    if (!c || dim < 0 || dim > 2 || side < 0 || side > 1) return RT_EINVAL;
    c->kp.ghost[dim][side] = ghost_dev;
    return RT_OK;
}

namespace {
// tetrad rest frame u^mu = e^mu_0 of every cell (rt_set_fluid with u4 == NULL)
__global__ void k_rest_frame(const double *__restrict__ ecen, double *__restrict__ u4, long long ncell, int ncol) {
    const long long cell = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    if (cell >= ncell) return;
    const double *e = ecen + (cell % ncol) * 16;
    for (int mu = 0; mu < 4; ++mu) u4[mu * ncell + cell] = e[4 * mu];
}
struct AboveFloor {   // L468 (i): cells at or above the density floor interact
    const double *rho; double floor;
    __device__ bool operator()(int q) const { return rho[q] >= floor; }
};
}  // namespace

extern "C" int rt_set_fluid(rt_ctx *c, const double *rho, const double *T, const double *u4, void *stream) {
    if (!c || !rho || !T) return RT_EINVAL;
    cudaStream_t st = (cudaStream_t)stream;
    const size_t nb = c->ncell * sizeof(double);
    CK(cudaMemcpyAsync(c->d_rho, rho, nb, cudaMemcpyDeviceToDevice, st));
    CK(cudaMemcpyAsync(c->d_T, T, nb, cudaMemcpyDeviceToDevice, st));
    if (u4) {
        CK(cudaMemcpyAsync(c->d_u4, u4, 4 * nb, cudaMemcpyDeviceToDevice, st));
        c->u4_rest = false;
    } else if (!c->u4_rest) {   // tetrad rest frame u^mu = e^mu_0 (built once, on the device: it does not depend on the call)
        c->u4_rest = true;
        k_rest_frame<<<(unsigned)((c->ncell + 255) / 256), 256, 0, st>>>(c->tab.ecen, c->d_u4, c->ncell, c->ncol);
        CK(cudaGetLastError());
    }
    // interaction list: cells at or above the density floor (L468 (i)); below it alpha = 0 whatever T is.  Built on the device
    // (cub partition of the cell indices: listed cells first in ascending order, the rest behind them); its length STAYS on
    // the device, so a caller who hands over a new fluid state every step (the coupled GRMHD use, L448-456) pays no
    // read-back and no synchronisation here.
    {
        c->kp.srclist = nullptr; c->kp.nsel = nullptr;
        if (c->matter && c->opt.source_method != 0) {
            const int n = (int)c->ncell;
            cub::CountingInputIterator<int> idx(0);
            AboveFloor sel{c->d_rho, c->opt.rho_floor};
            if (!c->d_part_tmp) {   // first use; on any failure nothing half-allocated is left behind
                cudaError_t e = cudaMalloc((void **)&c->d_srclist, (size_t)n * sizeof(int));
                if (e == cudaSuccess) e = cudaMalloc((void **)&c->d_nsel, sizeof(int));
                if (e == cudaSuccess) e = cub::DevicePartition::If(nullptr, c->part_tmp_bytes, idx, c->d_srclist, c->d_nsel, n, sel, st);
                if (e == cudaSuccess) e = cudaMalloc(&c->d_part_tmp, c->part_tmp_bytes ? c->part_tmp_bytes : 1);
                if (e != cudaSuccess) {
                    cudaFree(c->d_srclist); cudaFree(c->d_nsel);
                    c->d_srclist = nullptr; c->d_nsel = nullptr; c->d_part_tmp = nullptr;
                    g_last_cuda = (int)e;
                    return e == cudaErrorMemoryAllocation ? RT_ENOMEM : RT_ECUDA;
                }
            }
            size_t tmp = c->part_tmp_bytes;
            CK(cub::DevicePartition::If(c->d_part_tmp, tmp, idx, c->d_srclist, c->d_nsel, n, sel, st));
            c->kp.srclist = c->d_srclist; c->kp.nsel = c->d_nsel;
        }
    }
    c->fluid_set = true;
    ++c->fluid_version;
    return RT_OK;
}

static bool fixed_bc_missing(const rt_ctx *c) {
    for (int a = 0; a < 3; ++a) {
        if (c->grid.bc_lo[a] == RT_BC_FIXED && !c->kp.ghost[a][0]) return true;
        if (c->grid.bc_hi[a] == RT_BC_FIXED && !c->kp.ghost[a][1]) return true;
    }
    return false;
}

extern "C" int rt_transport(rt_ctx *c, const double *I_in, const double *I_base, double *I_out, double dt, void *stream) {
    if (!c || !I_in || !I_base || !I_out || I_in == I_out) return RT_EINVAL;
    if (fixed_bc_missing(c) || (c->matter && !c->fluid_set)) return RT_ESTATE;
    cudaStream_t st = (cudaStream_t)stream;
    if (c->matter) { ProfScope ps(c, RT_K_FACECOEF, st); CK(launch_facecoef(c->kp, c->d_T, dt, c->d_fcoef, c->d_colflag, st, &c->launches)); }
    { ProfScope ps(c, RT_K_TRANSPORT, st); CK(launch_transport(c->kp, I_in, I_base, I_out, c->d_fcoef, c->d_colflag, c->matter, dt, st, &c->launches)); }
    return RT_OK;
}

extern "C" int rt_transport_static(rt_ctx *c, const double *I_in, const double *I_base, double *I_out, double dt, void *stream) {
    if (!c || !I_in || !I_base || !I_out || I_in == I_out) return RT_EINVAL;
    if (fixed_bc_missing(c) || (c->matter && !c->fluid_set)) return RT_ESTATE;
    if (transport_static_bytes(c->kp, c->matter) > RT_STATIC_SCRATCH_BYTES) return RT_ETOOBIG;
    CK(launch_transport_static(c->kp, c->d_T, I_in, I_base, I_out, c->matter, dt, (cudaStream_t)stream, &c->launches));
    return RT_OK;
}

extern "C" int rt_angular_flux(rt_ctx *c, const double *I_in, double *I_io, double dt, void *stream) {
    if (!c || !I_in || !I_io || I_in == I_io) return RT_EINVAL;
    if (!c->curved) return RT_OK;
    { ProfScope ps(c, RT_K_ANGULAR, (cudaStream_t)stream); CK((c->opt.angular_recon == RT_ANG_MAPR ? launch_angular_mapr : launch_angular)(c->kp, I_in, I_io, dt, (cudaStream_t)stream, &c->launches)); }
    return RT_OK;
}

extern "C" int rt_source_implicit(rt_ctx *c, double *I, double *T, double dt, int *n_fail, void *stream) {
    if (!c || !I || !T) return RT_EINVAL;
    if (!c->fluid_set) return RT_ESTATE;
    if (c->opt.source_method == 0) return RT_OK;
    { ProfScope ps(c, RT_K_SOURCE, (cudaStream_t)stream); CK(launch_source(c->kp, I, T, dt, n_fail, nullptr, nullptr, (cudaStream_t)stream, &c->launches)); }
    return RT_OK;
}

extern "C" int rt_moments(rt_ctx *c, const double *I, double *R, void *stream) {
    if (!c || !I || !R) return RT_EINVAL;
    { ProfScope ps(c, RT_K_MOMENTS, (cudaStream_t)stream); CK(launch_moments(c->kp, I, R, (cudaStream_t)stream, &c->launches)); }
    return RT_OK;
}

// one stage of the predictor-corrector (L448-456): I* = O5(I_base; fluxes of I_flux, opacities at T_flux; delta),
// then O6 on (I*, T) with T_- = T_base
static int stage(rt_ctx *c, const double *I_flux, const double *T_flux, const double *I_base, double *I_out, double *T_io,
                 double delta, int *n_fail, double *R, double *G, cudaStream_t st) {
    if (c->matter) { ProfScope ps(c, RT_K_FACECOEF, st); CK(launch_facecoef(c->kp, T_flux, delta, c->d_fcoef, c->d_colflag, st, &c->launches)); }
    { ProfScope ps(c, RT_K_TRANSPORT, st); CK(launch_transport(c->kp, I_flux, I_base, I_out, c->d_fcoef, c->d_colflag, c->matter, delta, st, &c->launches)); }
    if (c->curved) { ProfScope ps(c, RT_K_ANGULAR, st); CK((c->opt.angular_recon == RT_ANG_MAPR ? launch_angular_mapr : launch_angular)(c->kp, I_flux, I_out, delta, st, &c->launches)); }
    if (c->opt.source_method != 0 || R || G) {
        ProfScope ps(c, RT_K_SOURCE, st);
        CK(launch_source(c->kp, I_out, T_io, delta, n_fail, R, G, st, &c->launches));
    }
    return RT_OK;
}

extern "C" int rt_step(rt_ctx *c, double *I, double *T, double *R_out, double *G_out, double dt, int *n_fail, void *stream) {
    if (!c || !I || !T) return RT_EINVAL;
    if (!c->fluid_set || fixed_bc_missing(c)) return RT_ESTATE;
    cudaStream_t st = (cudaStream_t)stream;
    CK(cudaMemcpyAsync(c->d_Th, T, c->ncell * sizeof(double), cudaMemcpyDeviceToDevice, st));
    int rc = stage(c, I, T, I, c->d_Ih, c->d_Th, 0.5 * dt, n_fail, nullptr, nullptr, st);     // predictor
    if (rc != RT_OK) return rc;
    return stage(c, c->d_Ih, c->d_Th, I, I, T, dt, n_fail, R_out, G_out, st);               // corrector
}

// ---- rt_step_slab: one step of a rank's slab with the planes its neighbours need stepped first ---------------------------------------
// PAPER.md L778 lists "treating the boundaries first and overlapping the transfer with the interior" as missing from cuHARM's radiation
// module.  This context is a rank's EXTENDED slab of an x3 decomposition (RT_SLAB_MARGIN planes of halo on every cut side, OUTFLOW
// there).  On halo_stream a sub-slab of 3 margins of planes at each cut end (halo, the planes to send, as many again: the domain of
// dependence of one step) is copied out and stepped by a context of its own, and its middle planes -- the owned planes next to the
// cut as they will be after this step, bit for bit -- land in the caller's send buffers; on `stream` the whole slab is stepped as by
// rt_step.  The caller sends / receives on halo_stream meanwhile and copies what it received into the halo planes once `stream` is done.
static int bslab_build(rt_ctx *c, int side) {
    rt_ctx::HostSlab &h = c->bslab[side];
    const rt_grid &G = c->grid;
    const int n3l = 3 * RT_SLAB_MARGIN;
    std::memset(&h, 0, sizeof h);
    h.n3l = n3l;
    h.k0 = side == 0 ? 0 : G.n[2] - n3l;     // first plane of the sub-slab in this context
    rt_grid g = G;
    g.n[2] = n3l;
    g.x0[2] = G.x0[2] + h.k0 * G.dx[2];
    g.bc_lo[2] = g.bc_hi[2] = RT_BC_OUTFLOW;
    g.zero_lo[2] = g.zero_hi[2] = 0;
    int rc = rt_init(&g, &c->metric, c->level, &c->opt, &h.sub);
    if (rc != RT_OK) return rc;
    h.sub->is_sub = true;
    const size_t pc = (size_t)c->ncol, pi = pc * c->pitch;
    cudaError_t e = cudaMalloc((void **)&h.I, n3l * pi * sizeof(double));
    if (e == cudaSuccess) e = cudaMalloc((void **)&h.T, n3l * pc * sizeof(double));
    if (e == cudaSuccess) e = cudaMalloc((void **)&h.rho, n3l * pc * sizeof(double));
    if (e == cudaSuccess) e = cudaMalloc((void **)&h.u4, 4 * n3l * pc * sizeof(double));
    if (e != cudaSuccess) { g_last_cuda = (int)e; return e == cudaErrorMemoryAllocation ? RT_ENOMEM : RT_ECUDA; }
    return RT_OK;
}

extern "C" int rt_step_slab(rt_ctx *c, double *I, double *T, double *R_out, double *G_out, double dt, int *n_fail,
                            double *send_lo_I, double *send_lo_T, double *send_hi_I, double *send_hi_T, void *stream, void *halo_stream) {
    if (!c || !I || !T || (!send_lo_I != !send_lo_T) || (!send_hi_I != !send_hi_T)) return RT_EINVAL;
    if (!c->fluid_set || fixed_bc_missing(c)) return RT_ESTATE;
    const int M = RT_SLAB_MARGIN, n3 = c->grid.n[2];
    const bool lo = send_lo_I != nullptr, hi = send_hi_I != nullptr;
    if ((lo || hi) && n3 < 3 * M) return RT_EINVAL;                       // the sub-slab must fit
    for (int a = 0; a < 3; ++a)                                           // caller-supplied ghost data is not cut into the sub-slabs
        if ((lo || hi) && (c->grid.bc_lo[a] == RT_BC_FIXED || c->grid.bc_hi[a] == RT_BC_FIXED)) return RT_EINVAL;
    cudaStream_t st = (cudaStream_t)stream, hs = (cudaStream_t)halo_stream;
    const size_t pc = (size_t)c->ncol, pi = pc * c->pitch;
    if (lo || hi) {
        if (!c->bev_in) {
            CK(cudaEventCreateWithFlags(&c->bev_in, cudaEventDisableTiming));
            CK(cudaEventCreateWithFlags(&c->bev_cloned, cudaEventDisableTiming));
            CK(cudaMalloc((void **)&c->d_bfail, sizeof(int)));
        }
        for (int side = 0; side < 2; ++side)
            if ((side == 0 ? lo : hi) && !c->bslab[side].sub) { int rc = bslab_build(c, side); if (rc != RT_OK) return rc; }
        CK(cudaEventRecord(c->bev_in, st));                                // I, T and the fluid state are current on `stream`
        CK(cudaStreamWaitEvent(hs, c->bev_in, 0));
        const bool refluid = c->bslab_fluid_version != c->fluid_version;
        for (int side = 0; side < 2; ++side) {
            if (!(side == 0 ? lo : hi)) continue;
            rt_ctx::HostSlab &h = c->bslab[side];
            CK(cudaMemcpyAsync(h.I, I + (size_t)h.k0 * pi, h.n3l * pi * sizeof(double), cudaMemcpyDeviceToDevice, hs));
            CK(cudaMemcpyAsync(h.T, T + (size_t)h.k0 * pc, h.n3l * pc * sizeof(double), cudaMemcpyDeviceToDevice, hs));
            if (refluid || !h.sub->fluid_set) {
                CK(cudaMemcpyAsync(h.rho, c->d_rho + (size_t)h.k0 * pc, h.n3l * pc * sizeof(double), cudaMemcpyDeviceToDevice, hs));
                for (int m = 0; m < 4; ++m)
                    CK(cudaMemcpyAsync(h.u4 + (size_t)m * h.n3l * pc, c->d_u4 + (size_t)m * c->ncell + (size_t)h.k0 * pc, h.n3l * pc * sizeof(double),
                                       cudaMemcpyDeviceToDevice, hs));
                int rc = rt_set_fluid(h.sub, h.rho, h.T, h.u4, hs);
                if (rc != RT_OK) return rc;
            }
        }
        c->bslab_fluid_version = c->fluid_version;
        CK(cudaEventRecord(c->bev_cloned, hs));
        for (int side = 0; side < 2; ++side) {
            if (!(side == 0 ? lo : hi)) continue;
            rt_ctx::HostSlab &h = c->bslab[side];
            int rc = rt_step(h.sub, h.I, h.T, nullptr, nullptr, dt, c->d_bfail, hs);
            if (rc != RT_OK) return rc;
            double *sI = side == 0 ? send_lo_I : send_hi_I, *sT = side == 0 ? send_lo_T : send_hi_T;
            CK(cudaMemcpyAsync(sI, h.I + (size_t)M * pi, M * pi * sizeof(double), cudaMemcpyDeviceToDevice, hs));
            CK(cudaMemcpyAsync(sT, h.T + (size_t)M * pc, M * pc * sizeof(double), cudaMemcpyDeviceToDevice, hs));
        }
        CK(cudaStreamWaitEvent(st, c->bev_cloned, 0));                     // the whole-slab step must not overwrite what is being copied out
    }
    return rt_step(c, I, T, R_out, G_out, dt, n_fail, stream);
}

// H2D -> rt_step -> D2H back to back on one stream (meshes too thin to cut, FIXED boundaries)
static int step_host_simple(rt_ctx *c, double *I_h, double *T_h, double *R_h, double *G_h, double dt, int *n_fail_h, void *stream) {
    cudaStream_t st = (cudaStream_t)stream;
    const size_t nI = (size_t)c->ncell * c->pitch * sizeof(double), nC = (size_t)c->ncell * sizeof(double);
    if (!c->d_hI) {
        CK(cudaMalloc((void **)&c->d_hI, nI));
        CK(cudaMalloc((void **)&c->d_hT, nC));
        CK(cudaMalloc((void **)&c->d_hR, 16 * nC));
        CK(cudaMalloc((void **)&c->d_hG, 4 * nC));
        CK(cudaMalloc((void **)&c->d_hfail, sizeof(int)));
    }
    CK(cudaMemcpyAsync(c->d_hI, I_h, nI, cudaMemcpyHostToDevice, st));
    CK(cudaMemcpyAsync(c->d_hT, T_h, nC, cudaMemcpyHostToDevice, st));
    CK(cudaMemsetAsync(c->d_hfail, 0, sizeof(int), st));
    const int rc = rt_step(c, c->d_hI, c->d_hT, R_h ? c->d_hR : nullptr, G_h ? c->d_hG : nullptr, dt, c->d_hfail, stream);
    if (rc != RT_OK) return rc;
    CK(cudaMemcpyAsync(I_h, c->d_hI, nI, cudaMemcpyDeviceToHost, st));
    CK(cudaMemcpyAsync(T_h, c->d_hT, nC, cudaMemcpyDeviceToHost, st));
    if (R_h) CK(cudaMemcpyAsync(R_h, c->d_hR, 16 * nC, cudaMemcpyDeviceToHost, st));
    if (G_h) CK(cudaMemcpyAsync(G_h, c->d_hG, 4 * nC, cudaMemcpyDeviceToHost, st));
    if (n_fail_h) CK(cudaMemcpyAsync(n_fail_h, c->d_hfail, sizeof(int), cudaMemcpyDeviceToHost, st));
    CK(cudaStreamSynchronize(st));
    return RT_OK;
}

// ---- rt_step_host as a pipeline ---------------------------------------------------------------------------------------
// The mesh is cut into x3 slabs with a 4-plane halo on every cut side: one rt_step (two stages x a 2-cell stencil) has a
// domain of dependence of +-4 cells, so the plain rt_step on the extended slab (OUTFLOW on the cut faces) gives the exact
// single-domain result on the planes the slab owns (the decomposition of DESIGN.md section 8, here on one GPU).  Every
// plane of the input state crosses PCIe once, into a full-size device copy; a slab starts as soon as its planes are there
// and its owned planes go back while later slabs are still arriving or computing: H2D, compute and D2H on three streams
// (PCIe is full duplex).  Same kernels on the same values: the result equals rt_step's bit for bit.
static const int HS_MARGIN = 4;

static int hslab_build(rt_ctx *c, int nslab) {
    const rt_grid &G = c->grid;
    const int n3 = G.n[2];
    const bool per = G.bc_lo[2] == RT_BC_PERIODIC;
    const size_t plane_c = (size_t)c->ncol, plane_i = plane_c * c->pitch;
    for (int r = 0; r < nslab; ++r) {
        rt_ctx::HostSlab h;
        std::memset(&h, 0, sizeof h);
        const int base = n3 / nslab, rem = n3 % nslab;
        h.k0 = r * base + (r < rem ? r : rem);
        h.k1 = h.k0 + base + (r < rem ? 1 : 0);
        const bool lo_cut = per || r > 0, hi_cut = per || r < nslab - 1;
        h.ext_lo = lo_cut ? HS_MARGIN : 0; h.ext_hi = hi_cut ? HS_MARGIN : 0;
        h.n3l = h.k1 - h.k0 + h.ext_lo + h.ext_hi;
        rt_grid g = G;
        g.n[2] = h.n3l;
        g.x0[2] = G.x0[2] + (h.k0 - h.ext_lo) * G.dx[2];
        g.bc_lo[2] = lo_cut ? RT_BC_OUTFLOW : G.bc_lo[2];
        g.bc_hi[2] = hi_cut ? RT_BC_OUTFLOW : G.bc_hi[2];
        if (per) g.bc_lo[2] = g.bc_hi[2] = RT_BC_OUTFLOW;
        if (lo_cut) g.zero_lo[2] = 0;
        if (hi_cut) g.zero_hi[2] = 0;
        int rc = rt_init(&g, &c->metric, c->level, &c->opt, &h.sub);
        if (rc != RT_OK) { c->hslabs.push_back(h); return rc; }
        h.sub->is_sub = true;
        cudaError_t e = cudaMalloc((void **)&h.I, h.n3l * plane_i * sizeof(double));
        if (e == cudaSuccess) e = cudaMalloc((void **)&h.T, h.n3l * plane_c * sizeof(double));
        if (e == cudaSuccess) e = cudaMalloc((void **)&h.R, 16 * h.n3l * plane_c * sizeof(double));
        if (e == cudaSuccess) e = cudaMalloc((void **)&h.G, 4 * h.n3l * plane_c * sizeof(double));
        if (e == cudaSuccess) e = cudaMalloc((void **)&h.rho, h.n3l * plane_c * sizeof(double));
        if (e == cudaSuccess) e = cudaMalloc((void **)&h.u4, 4 * h.n3l * plane_c * sizeof(double));
        if (e == cudaSuccess) e = cudaEventCreateWithFlags(&h.done, cudaEventDisableTiming);
        c->hslabs.push_back(h);
        if (e != cudaSuccess) { g_last_cuda = (int)e; return e == cudaErrorMemoryAllocation ? RT_ENOMEM : RT_ECUDA; }
    }
    return RT_OK;
}

// local planes [0, n3l) of a slab <- global planes (k0 - ext_lo + l) mod n3 of `src`, as the fewest contiguous copies
static cudaError_t hslab_gather(const rt_ctx::HostSlab &h, int n3, double *dst, const double *src, size_t per_plane, cudaStream_t st) {
    int l = 0;
    while (l < h.n3l) {
        const int g0 = ((h.k0 - h.ext_lo + l) % n3 + n3) % n3;
        int len = 1;
        while (l + len < h.n3l && g0 + len < n3) ++len;
        cudaError_t e = cudaMemcpyAsync(dst + (size_t)l * per_plane, src + (size_t)g0 * per_plane, (size_t)len * per_plane * sizeof(double),
                                        cudaMemcpyDeviceToDevice, st);
        if (e != cudaSuccess) return e;
        l += len;
    }
    return cudaSuccess;
}

// the parent's fluid state cut into the slabs' contexts (only when it changed since the last call)
static int hslab_fluid(rt_ctx *c, cudaStream_t st) {
    const int n3 = c->grid.n[2];
    const size_t pc = (size_t)c->ncol;
    for (auto &h : c->hslabs) {
        CK(hslab_gather(h, n3, h.rho, c->d_rho, pc, st));
        CK(hslab_gather(h, n3, h.T, c->d_T, pc, st));
        for (int m = 0; m < 4; ++m) CK(hslab_gather(h, n3, h.u4 + (size_t)m * h.n3l * pc, c->d_u4 + (size_t)m * c->ncell, pc, st));
        const int rc = rt_set_fluid(h.sub, h.rho, h.T, h.u4, st);
        if (rc != RT_OK) return rc;
    }
    c->hslab_fluid_version = c->fluid_version;
    return RT_OK;
}

static int step_host_pipelined(rt_ctx *c, int nslab, double *I_h, double *T_h, double *R_h, double *G_h, double dt, int *n_fail_h, cudaStream_t cur) {
    const int n3 = c->grid.n[2];
    const size_t pc = (size_t)c->ncol, pi = pc * c->pitch;
    const size_t nI = (size_t)c->ncell * c->pitch * sizeof(double), nC = (size_t)c->ncell * sizeof(double);
    if (c->hslabs.empty()) {
        if (!c->d_hI) {
            CK(cudaMalloc((void **)&c->d_hI, nI));
            CK(cudaMalloc((void **)&c->d_hT, nC));
            CK(cudaMalloc((void **)&c->d_hfail, sizeof(int)));
        }
        CK(cudaStreamCreateWithFlags(&c->hs_in, cudaStreamNonBlocking));
        CK(cudaStreamCreateWithFlags(&c->hs_cmp, cudaStreamNonBlocking));
        CK(cudaStreamCreateWithFlags(&c->hs_out, cudaStreamNonBlocking));
        CK(cudaEventCreateWithFlags(&c->hev_start, cudaEventDisableTiming));
        for (int q = 0; q < 3; ++q) CK(cudaEventCreateWithFlags(&c->hev_end[q], cudaEventDisableTiming));
        const int rc = hslab_build(c, nslab);
        if (rc != RT_OK) return rc;
    }
    CK(cudaEventRecord(c->hev_start, cur));
    CK(cudaStreamWaitEvent(c->hs_in, c->hev_start, 0));
    CK(cudaStreamWaitEvent(c->hs_cmp, c->hev_start, 0));
    CK(cudaStreamWaitEvent(c->hs_out, c->hev_start, 0));
    if (c->hslab_fluid_version != c->fluid_version) {
        const int rc = hslab_fluid(c, c->hs_cmp);
        if (rc != RT_OK) return rc;
    }
    CK(cudaMemsetAsync(c->d_hfail, 0, sizeof(int), c->hs_cmp));
    // upload order: what slab 0 needs first (under a periodic x3 its lower halo is the top of the mesh), then upwards,
    // in chunks of a slab's worth of planes so that the first slab can start early
    const bool per = c->grid.bc_lo[2] == RT_BC_PERIODIC;
    const int chunk = (n3 + nslab - 1) / nslab;
    std::vector<int> arrival(n3, -1);
    int nchunk = 0;
    auto upload = [&](int a, int b) -> cudaError_t {
        cudaError_t e = cudaMemcpyAsync(c->d_hI + (size_t)a * pi, I_h + (size_t)a * pi, (size_t)(b - a) * pi * sizeof(double), cudaMemcpyHostToDevice, c->hs_in);
        if (e == cudaSuccess) e = cudaMemcpyAsync(c->d_hT + (size_t)a * pc, T_h + (size_t)a * pc, (size_t)(b - a) * pc * sizeof(double), cudaMemcpyHostToDevice, c->hs_in);
        if (e != cudaSuccess) return e;
        if ((int)c->hev.size() <= nchunk) {
            cudaEvent_t ev;
            e = cudaEventCreateWithFlags(&ev, cudaEventDisableTiming);
            if (e != cudaSuccess) return e;
            c->hev.push_back(ev);
        }
        e = cudaEventRecord(c->hev[nchunk], c->hs_in);
        for (int q = a; q < b; ++q) arrival[q] = nchunk;
        ++nchunk;
        return e;
    };
    const int top = per ? n3 - HS_MARGIN : n3;
    if (per) CK(upload(top, n3));
    for (int a = 0; a < top; a += chunk) CK(upload(a, a + chunk < top ? a + chunk : top));
    for (auto &h : c->hslabs) {
        int need = 0;
        for (int l = 0; l < h.n3l; ++l) {
            const int g = ((h.k0 - h.ext_lo + l) % n3 + n3) % n3;
            if (arrival[g] > need) need = arrival[g];
        }
        CK(cudaStreamWaitEvent(c->hs_cmp, c->hev[need], 0));
        CK(hslab_gather(h, n3, h.I, c->d_hI, pi, c->hs_cmp));
        CK(hslab_gather(h, n3, h.T, c->d_hT, pc, c->hs_cmp));
        const long long l0 = h.sub->launches;
        const int rc = rt_step(h.sub, h.I, h.T, R_h ? h.R : nullptr, G_h ? h.G : nullptr, dt, c->d_hfail, c->hs_cmp);
        if (rc != RT_OK) return rc;
        c->launches += h.sub->launches - l0;
        CK(cudaEventRecord(h.done, c->hs_cmp));
        CK(cudaStreamWaitEvent(c->hs_out, h.done, 0));
        const int own = h.k1 - h.k0;
        CK(cudaMemcpyAsync(I_h + (size_t)h.k0 * pi, h.I + (size_t)h.ext_lo * pi, (size_t)own * pi * sizeof(double), cudaMemcpyDeviceToHost, c->hs_out));
        CK(cudaMemcpyAsync(T_h + (size_t)h.k0 * pc, h.T + (size_t)h.ext_lo * pc, (size_t)own * pc * sizeof(double), cudaMemcpyDeviceToHost, c->hs_out));
        const size_t lc = (size_t)h.n3l * pc;
        if (R_h) for (int m = 0; m < 16; ++m)
            CK(cudaMemcpyAsync(R_h + (size_t)m * c->ncell + (size_t)h.k0 * pc, h.R + m * lc + (size_t)h.ext_lo * pc, (size_t)own * pc * sizeof(double), cudaMemcpyDeviceToHost, c->hs_out));
        if (G_h) for (int m = 0; m < 4; ++m)
            CK(cudaMemcpyAsync(G_h + (size_t)m * c->ncell + (size_t)h.k0 * pc, h.G + m * lc + (size_t)h.ext_lo * pc, (size_t)own * pc * sizeof(double), cudaMemcpyDeviceToHost, c->hs_out));
    }
    if (n_fail_h) CK(cudaMemcpyAsync(n_fail_h, c->d_hfail, sizeof(int), cudaMemcpyDeviceToHost, c->hs_cmp));
    cudaStream_t ss[3] = {c->hs_in, c->hs_cmp, c->hs_out};
    for (int q = 0; q < 3; ++q) {
        CK(cudaEventRecord(c->hev_end[q], ss[q]));
        CK(cudaStreamWaitEvent(cur, c->hev_end[q], 0));
    }
    CK(cudaStreamSynchronize(cur));
    return RT_OK;
}

extern "C" int rt_step_host(rt_ctx *c, double *I_h, double *T_h, double *R_h, double *G_h, double dt, int *n_fail_h, void *stream) {
    if (!c || !I_h || !T_h) return RT_EINVAL;
    if (!c->fluid_set || fixed_bc_missing(c)) return RT_ESTATE;
    const int n3 = c->grid.n[2];
    bool fixed = false;
    for (int a = 0; a < 3; ++a) fixed = fixed || c->grid.bc_lo[a] == RT_BC_FIXED || c->grid.bc_hi[a] == RT_BC_FIXED;
    const int nslab = n3 / 8;   // slabs of >= 8 owned planes: at most 8 / 8 redundant planes of compute
    if (nslab < 2 || fixed || c->is_sub) return step_host_simple(c, I_h, T_h, R_h, G_h, dt, n_fail_h, stream);
    return step_host_pipelined(c, nslab, I_h, T_h, R_h, G_h, dt, n_fail_h, (cudaStream_t)stream);
}
