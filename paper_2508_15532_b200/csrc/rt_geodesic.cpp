// Geodesic angular grid for librt_b200 (host, init-time only).
//
// PAPER.md section 3.3 (L207-217): icosahedron inscribed in the unit sphere; every Delaunay edge bisected, the new
// points projected on the sphere, repeated per generation; the angular cells are the Voronoi cells of the final
// triangulation (12 pentagons, the rest hexagons), N = 2 + 10 * 4^generation.
// DESIGN.md readings: S1 (level n = 2^a m: a bisections then one frequency-m subdivision, so n = 6 gives 362),
// S2 (pole along tetrad axis 3; order: z descending, then azimuth ascending), S3 (weights = exact cell areas).
// Edge data for the angular flux (L235-241): length, centre, outward normal tangent to the sphere.
#include <algorithm>
#include <array>
#include <cmath>
#include <map>
#include <tuple>

#include "rt_internal.h"

namespace rt {
namespace {

struct V3 {
    double x, y, z;
};
inline V3 operator+(V3 a, V3 b) { return {a.x + b.x, a.y + b.y, a.z + b.z}; }
inline V3 operator-(V3 a, V3 b) { return {a.x - b.x, a.y - b.y, a.z - b.z}; }
inline V3 operator*(double s, V3 a) { return {s * a.x, s * a.y, s * a.z}; }
inline double dot(V3 a, V3 b) { return a.x * b.x + a.y * b.y + a.z * b.z; }
inline V3 cross(V3 a, V3 b) { return {a.y * b.z - a.z * b.y, a.z * b.x - a.x * b.z, a.x * b.y - a.y * b.x}; }
inline double norm(V3 a) { return std::sqrt(dot(a, a)); }
inline V3 unit(V3 a) { return (1.0 / norm(a)) * a; }

using Tri = std::array<int, 3>;

struct Mesh {
    std::vector<V3> v;
    std::vector<Tri> t;
};

Mesh icosahedron() {
    const double PI = 3.14159265358979323846;
    Mesh m;
    const double lat = std::atan(0.5), cl = std::cos(lat), sl = std::sin(lat);
    m.v.push_back({0, 0, 1});
    for (int k = 0; k < 5; ++k) m.v.push_back({cl * std::cos(2 * PI * k / 5), cl * std::sin(2 * PI * k / 5), sl});
    for (int k = 0; k < 5; ++k)
        m.v.push_back({cl * std::cos(2 * PI * k / 5 + PI / 5), cl * std::sin(2 * PI * k / 5 + PI / 5), -sl});
    m.v.push_back({0, 0, -1});
    for (int k = 0; k < 5; ++k) {
        int u0 = 1 + k, u1 = 1 + (k + 1) % 5, l0 = 6 + k, l1 = 6 + (k + 1) % 5;
        m.t.push_back({0, u0, u1});
        m.t.push_back({u0, l0, u1});
        m.t.push_back({l0, l1, u1});
        m.t.push_back({11, l1, l0});
    }
    return m;
}

// frequency-f subdivision of every triangle; shared edge points are created once per (edge, position)
Mesh subdivide(const Mesh &in, int f) {
    Mesh out;
    out.v = in.v;
    std::map<std::tuple<int, int, int>, int> edge_pt;
    auto on_edge = [&](int a, int b, int q) {  // q/f of the way from a to b, 0 < q < f
        int lo = std::min(a, b), hi = std::max(a, b), qq = (a < b) ? q : f - q;
        auto key = std::make_tuple(lo, hi, qq);
        auto it = edge_pt.find(key);
        if (it != edge_pt.end()) return it->second;
        V3 p = (double(f - qq) / f) * in.v[lo] + (double(qq) / f) * in.v[hi];
        out.v.push_back(unit(p));
        return edge_pt[key] = int(out.v.size()) - 1;
    };
    for (const Tri &t : in.t) {
        const int a = t[0], b = t[1], c = t[2];
        std::vector<std::vector<int>> id(f + 1, std::vector<int>(f + 1, -1));
        for (int i = 0; i <= f; ++i)
            for (int j = 0; i + j <= f; ++j) {
                int k = f - i - j;
                if (i == 0 && j == 0) id[i][j] = a;
                else if (i == f) id[i][j] = b;
                else if (j == f) id[i][j] = c;
                else if (j == 0) id[i][j] = on_edge(a, b, i);
                else if (i == 0) id[i][j] = on_edge(a, c, j);
                else if (k == 0) id[i][j] = on_edge(b, c, j);
                else {
                    V3 p = (double(k) / f) * in.v[a] + (double(i) / f) * in.v[b] + (double(j) / f) * in.v[c];
                    out.v.push_back(unit(p));
                    id[i][j] = int(out.v.size()) - 1;
                }
            }
        for (int i = 0; i < f; ++i)
            for (int j = 0; i + j < f; ++j) {
                out.t.push_back({id[i][j], id[i + 1][j], id[i][j + 1]});
                if (i + j < f - 1) out.t.push_back({id[i + 1][j], id[i + 1][j + 1], id[i][j + 1]});
            }
    }
    return out;
}

double tri_solid_angle(V3 a, V3 b, V3 c) {  // Van Oosterom & Strackee, unit vectors
    return 2.0 * std::atan2(std::fabs(dot(a, cross(b, c))), 1.0 + dot(a, b) + dot(b, c) + dot(c, a));
}

// L215: "to account for strong anisotropies of the radiation because of the Lorentz boost, the grid can be deformed in advance by
// performing a Lorentz transformation of its directions.  It can also be easily oriented along a pre-defined direction".
// Both act on the cell centres of the regular grid in its canonical order; numbering and neighbour lists stay (a Lorentz
// transformation maps circles on the sphere to circles: the Delaunay triangles of the deformed centres are the same).
// turn the pole (0,0,1) to `axis` about the direction perpendicular to both
V3 orient(V3 v, const double axis[3]) {
    V3 a = unit({axis[0], axis[1], axis[2]});
    const V3 z = {0, 0, 1};
    V3 k = cross(z, a);
    const double sn = norm(k), cs = dot(z, a);
    if (sn < 1e-15) return cs > 0 ? v : V3{v.x, -v.y, -v.z};
    k = (1.0 / sn) * k;
    return cs * v + sn * cross(k, v) + ((1.0 - cs) * dot(k, v)) * k;   // Rodrigues
}
// direction of the null vector (1, n) of a frame moving with velocity beta, seen from the frame it moves in
V3 aberrate(V3 n, const double beta[3]) {
    const V3 b = {beta[0], beta[1], beta[2]};
    const double gam = 1.0 / std::sqrt(1.0 - dot(b, b)), bn = dot(b, n);
    const double k0 = gam * (1.0 + bn);
    const V3 ks = n + (gam + gam * gam / (gam + 1.0) * bn) * b;
    return (1.0 / k0) * ks;
}

}  // namespace

bool build_angular_grid(int level, const double axis[3], const double boost[3], AngularGrid &g) {
    if (level < 1 || level > 64) return false;
    int a = 0, m = level;
    while (m % 2 == 0) { m /= 2; ++a; }
    Mesh mesh = icosahedron();
    for (int q = 0; q < a; ++q) mesh = subdivide(mesh, 2);
    if (m > 1) mesh = subdivide(mesh, m);
    const int nd = int(mesh.v.size());
    if (nd != 10 * level * level + 2) return false;

    // canonical order (S2)
    const double TOL = 1e-9, TWO_PI = 6.283185307179586476925286766559;
    std::vector<double> az(nd);
    for (int i = 0; i < nd; ++i) {
        double p = std::atan2(mesh.v[i].y, mesh.v[i].x);
        if (p < -TOL) p += TWO_PI;
        if (std::fabs(p) <= TOL) p = 0.0;
        az[i] = p;
    }
    std::vector<int> order(nd);
    for (int i = 0; i < nd; ++i) order[i] = i;
    std::sort(order.begin(), order.end(), [&](int p, int q) { return mesh.v[p].z > mesh.v[q].z; });
    for (int i = 0; i < nd;) {  // group equal z (within TOL of the previous one), sort each group by azimuth
        int j = i + 1;
        while (j < nd && std::fabs(mesh.v[order[j]].z - mesh.v[order[j - 1]].z) <= TOL) ++j;
        std::sort(order.begin() + i, order.begin() + j, [&](int p, int q) { return az[p] < az[q]; });
        i = j;
    }
    std::vector<int> rank(nd);
    for (int i = 0; i < nd; ++i) rank[order[i]] = i;
    std::vector<V3> n(nd);
    for (int i = 0; i < nd; ++i) n[i] = unit(mesh.v[order[i]]);
    if (axis && (axis[0] != 0 || axis[1] != 0 || axis[2] != 0))
        for (int i = 0; i < nd; ++i) n[i] = unit(orient(n[i], axis));
    if (boost && (boost[0] != 0 || boost[1] != 0 || boost[2] != 0)) {
        if (!(boost[0] * boost[0] + boost[1] * boost[1] + boost[2] * boost[2] < 1.0)) return false;
        for (int i = 0; i < nd; ++i) n[i] = unit(aberrate(n[i], boost));
    }
    std::vector<Tri> tris;
    for (const Tri &t : mesh.t) {
        Tri r = {rank[t[0]], rank[t[1]], rank[t[2]]};
        // orient counter-clockwise seen from outside
        if (dot(cross(n[r[1]] - n[r[0]], n[r[2]] - n[r[0]]), n[r[0]]) < 0) std::swap(r[1], r[2]);
        tris.push_back(r);
    }
    // Voronoi corners = circumcentres of the Delaunay triangles
    std::vector<V3> cc(tris.size());
    for (size_t ti = 0; ti < tris.size(); ++ti) {
        const Tri &t = tris[ti];
        cc[ti] = unit(cross(n[t[1]] - n[t[0]], n[t[2]] - n[t[0]]));
    }
    // fan around every vertex: triangle (s, p, q) ccw => q follows p; corner between p and q is that triangle's
    std::vector<std::map<int, std::pair<int, int>>> next(nd);  // next[s][p] = (q, triangle)
    for (size_t ti = 0; ti < tris.size(); ++ti)
        for (int c = 0; c < 3; ++c) {
            int s = tris[ti][c], p = tris[ti][(c + 1) % 3], q = tris[ti][(c + 2) % 3];
            next[s][p] = {q, int(ti)};
        }
    g = AngularGrid();
    g.nd = nd;
    g.nhat.assign(3 * nd, 0.0);
    g.w.assign(nd, 0.0);
    g.nnb.assign(nd, 0);
    g.nb.assign(6 * nd, -1);
    g.back.assign(6 * nd, -1);
    g.dlam.assign(6 * nd, 0.0);
    g.emid.assign(18 * nd, 0.0);
    g.eun.assign(18 * nd, 0.0);
    for (int s = 0; s < nd; ++s) {
        g.nhat[3 * s] = n[s].x; g.nhat[3 * s + 1] = n[s].y; g.nhat[3 * s + 2] = n[s].z;
        const int cnt = int(next[s].size());
        if (cnt != 5 && cnt != 6) return false;
        g.nnb[s] = cnt;
        int p = next[s].begin()->first;  // lowest neighbour index (std::map is ordered)
        int tri_prev = -1;
        for (auto &kv : next[s])
            if (kv.second.first == p) tri_prev = kv.second.second;  // triangle whose fan step ENDS at p
        double area = 0.0;
        for (int e = 0; e < cnt; ++e) {
            // edge between s and p: its two corners are the circumcentres of the triangles before and after p
            int tri_next = next[s][p].second;
            V3 c1 = cc[tri_prev], c2 = cc[tri_next];
            g.nb[6 * s + e] = p;
            g.dlam[6 * s + e] = std::atan2(norm(cross(c1, c2)), dot(c1, c2));
            V3 mid = unit(c1 + c2);
            V3 tt = n[p] - dot(n[p], mid) * mid, ss = n[s] - dot(n[s], mid) * mid;
            V3 u = unit(tt - ss);
            double *pm = &g.emid[3 * (6 * s + e)], *pu = &g.eun[3 * (6 * s + e)];
            pm[0] = mid.x; pm[1] = mid.y; pm[2] = mid.z;
            pu[0] = u.x; pu[1] = u.y; pu[2] = u.z;
            area += tri_solid_angle(n[s], c1, c2);
            tri_prev = tri_next;
            p = next[s][p].first;
        }
        g.w[s] = area;
    }
    for (int s = 0; s < nd; ++s)
        for (int e = 0; e < g.nnb[s]; ++e) {
            int t = g.nb[6 * s + e];
            for (int q = 0; q < g.nnb[t]; ++q)
                if (g.nb[6 * t + q] == s) g.back[6 * s + e] = q;
            if (g.back[6 * s + e] < 0) return false;
        }
    return true;
}

}  // namespace rt
