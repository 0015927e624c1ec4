// host_grid.cpp -- R2Bk icosahedral C-grid generator of the library (host, C++17 + OpenMP).
//
// Topology is derived HIERARCHICALLY: every level carries explicit cell->edge and edge->vertex
// tables, each edge spawns its midpoint vertex and two half edges, each cell three interior
// edges, so no hash map or sort is needed to find shared midpoints. The canonical first-touch
// numbering of readings P-3/P-5 is then a relabelling sweep over plain
// arrays. Cites: icosahedral-triangular C-grid PAPER.md:56; dual grid with 12 pentagons and the
// index arrays PAPER.md:186; coefficient tables as static read-only inputs PAPER.md:164-167.
#include "host_grid.hpp"

#include <algorithm>
#include <cmath>
#include <numeric>

namespace icon {
namespace {

constexpr double kEarthRadius = 6.371e6;   // a [m]
constexpr double kOmega = 7.29212e-5;      // [1/s]
constexpr double kPi = 3.14159265358979323846;

struct V3 {
    double x, y, z;
};
inline V3 operator+(V3 a, V3 b) { return {a.x + b.x, a.y + b.y, a.z + b.z}; }
inline V3 operator-(V3 a, V3 b) { return {a.x - b.x, a.y - b.y, a.z - b.z}; }
inline V3 operator*(double s, V3 a) { return {s * a.x, s * a.y, s * a.z}; }
inline double dot(V3 a, V3 b) { return a.x * b.x + a.y * b.y + a.z * b.z; }
inline V3 cross(V3 a, V3 b) { return {a.y * b.z - a.z * b.y, a.z * b.x - a.x * b.z, a.x * b.y - a.y * b.x}; }
inline double len(V3 a) { return std::sqrt(dot(a, a)); }
inline V3 unit(V3 a) {
    double n = len(a);
    return {a.x / n, a.y / n, a.z / n};
}
inline V3 ld3(const std::vector<double>& v, int64_t i) { return {v[3 * i], v[3 * i + 1], v[3 * i + 2]}; }
inline void st3(std::vector<double>& v, int64_t i, V3 a) {
    v[3 * i] = a.x;
    v[3 * i + 1] = a.y;
    v[3 * i + 2] = a.z;
}
inline double arc(V3 p, V3 q) { return std::atan2(len(cross(p, q)), dot(p, q)); }
inline double tri_area(V3 p, V3 q, V3 r) {
    return 2.0 * std::atan2(std::fabs(dot(p, cross(q, r))), 1.0 + dot(p, q) + dot(q, r) + dot(r, p));
}

// One refinement level: provisional numbering, explicit edges.
struct Level {
    int64_t nv = 0, nc = 0, ne = 0;
    std::vector<double> xyz;       // [nv][3]
    std::vector<int32_t> c2v;      // [nc][3]
    std::vector<int32_t> c2e;      // [nc][3] slot j joins vertex slots j, j+1
    std::vector<int32_t> e2v;      // [ne][2]
};

// P-1: base icosahedron
void base_level(Level& L) {
    L.nv = 12;
    L.nc = 20;
    L.ne = 30;
    L.xyz.assign(36, 0.0);
    const double lat = std::atan(0.5);
    st3(L.xyz, 0, {0.0, 0.0, 1.0});
    for (int i = 0; i < 5; ++i) {
        double lon = (72.0 * i) * kPi / 180.0, lon2 = (36.0 + 72.0 * i) * kPi / 180.0;
        st3(L.xyz, 1 + i, {std::cos(lat) * std::cos(lon), std::cos(lat) * std::sin(lon), std::sin(lat)});
        st3(L.xyz, 6 + i, {std::cos(-lat) * std::cos(lon2), std::cos(-lat) * std::sin(lon2), std::sin(-lat)});
    }
    st3(L.xyz, 11, {0.0, 0.0, -1.0});
    L.c2v.resize(60);
    for (int i = 0; i < 5; ++i) {
        int j = (i + 1) % 5;
        const int32_t f[4][3] = {{0, 1 + i, 1 + j}, {1 + i, 6 + i, 1 + j}, {6 + i, 6 + j, 1 + j}, {11, 6 + j, 6 + i}};
        for (int q = 0; q < 4; ++q)
            for (int s = 0; s < 3; ++s) L.c2v[3 * (4 * i + q) + s] = f[q][s];
    }
    // 30 base edges: tiny, so a linear search over the edges found so far is enough
    L.c2e.assign(60, -1);
    L.e2v.clear();
    for (int c = 0; c < 20; ++c)
        for (int j = 0; j < 3; ++j) {
            int32_t a = L.c2v[3 * c + j], b = L.c2v[3 * c + (j + 1) % 3];
            int found = -1;
            for (size_t e = 0; e < L.e2v.size() / 2; ++e)
                if ((L.e2v[2 * e] == a && L.e2v[2 * e + 1] == b) || (L.e2v[2 * e] == b && L.e2v[2 * e + 1] == a)) found = (int)e;
            if (found < 0) {
                found = (int)(L.e2v.size() / 2);
                L.e2v.push_back(a);
                L.e2v.push_back(b);
            }
            L.c2e[3 * c + j] = found;
        }
}

// P-2: one bisection, derived from the parent's explicit edges.
// children 4p+0=(a,ab,ca) 4p+1=(ab,b,bc) 4p+2=(ca,bc,c) 4p+3=(ab,bc,ca)
void refine(const Level& P, Level& C, bool need_e2v) {
    C.nv = P.nv + P.ne;
    C.nc = 4 * P.nc;
    C.ne = 2 * P.ne + 3 * P.nc;
    C.xyz.resize(3 * (size_t)C.nv);
    std::copy(P.xyz.begin(), P.xyz.end(), C.xyz.begin());
#pragma omp parallel for schedule(static)
    for (int64_t e = 0; e < P.ne; ++e) {
        V3 m = unit(ld3(P.xyz, P.e2v[2 * e]) + ld3(P.xyz, P.e2v[2 * e + 1]));
        st3(C.xyz, P.nv + e, m);
    }
    if (need_e2v) {
        C.e2v.resize(2 * (size_t)C.ne);
#pragma omp parallel for schedule(static)
        for (int64_t e = 0; e < P.ne; ++e) {
            int32_t m = (int32_t)(P.nv + e);
            C.e2v[4 * e] = P.e2v[2 * e];
            C.e2v[4 * e + 1] = m;
            C.e2v[4 * e + 2] = m;
            C.e2v[4 * e + 3] = P.e2v[2 * e + 1];
        }
    }
    C.c2v.resize(3 * (size_t)C.nc);
    C.c2e.resize(3 * (size_t)C.nc);
#pragma omp parallel for schedule(static)
    for (int64_t p = 0; p < P.nc; ++p) {
        const int32_t a = P.c2v[3 * p], b = P.c2v[3 * p + 1], c = P.c2v[3 * p + 2];
        const int32_t E0 = P.c2e[3 * p], E1 = P.c2e[3 * p + 1], E2 = P.c2e[3 * p + 2];
        const int32_t ab = (int32_t)(P.nv + E0), bc = (int32_t)(P.nv + E1), ca = (int32_t)(P.nv + E2);
        // half of parent edge E that touches vertex x
        auto half = [&](int32_t E, int32_t x) { return (int32_t)(2 * (int64_t)E + (P.e2v[2 * E] == x ? 0 : 1)); };
        const int32_t i_abca = (int32_t)(2 * P.ne + 3 * p), i_abbc = i_abca + 1, i_bcca = i_abca + 2;
        int32_t* v = &C.c2v[12 * p];
        int32_t* e = &C.c2e[12 * p];
        v[0] = a;  v[1] = ab; v[2] = ca;   e[0] = half(E0, a);  e[1] = i_abca;       e[2] = half(E2, a);
        v[3] = ab; v[4] = b;  v[5] = bc;   e[3] = half(E0, b);  e[4] = half(E1, b);  e[5] = i_abbc;
        v[6] = ca; v[7] = bc; v[8] = c;    e[6] = i_bcca;       e[7] = half(E1, c);  e[8] = half(E2, c);
        v[9] = ab; v[10] = bc; v[11] = ca; e[9] = i_abbc;       e[10] = i_bcca;      e[11] = i_abca;
        if (need_e2v) {
            C.e2v[2 * (int64_t)i_abca] = ab; C.e2v[2 * (int64_t)i_abca + 1] = ca;
            C.e2v[2 * (int64_t)i_abbc] = ab; C.e2v[2 * (int64_t)i_abbc + 1] = bc;
            C.e2v[2 * (int64_t)i_bcca] = bc; C.e2v[2 * (int64_t)i_bcca + 1] = ca;
        }
    }
}

// counter-based mixer of reading P-7; oracle/ has its own copy
inline uint64_t mix64(uint64_t seed, uint64_t stream, uint64_t i) {
    uint64_t z = seed + 0x9E3779B97F4A7C15ULL * (i + 1) + 0xD1B54A32D192ED03ULL * (stream + 1);
    z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9ULL;
    z = (z ^ (z >> 27)) * 0x94D049BB133111EBULL;
    return z ^ (z >> 31);
}
std::vector<int32_t> rank_permutation(uint64_t seed, uint64_t stream, int64_t n) {
    std::vector<uint64_t> key((size_t)n);
#pragma omp parallel for schedule(static)
    for (int64_t i = 0; i < n; ++i) key[i] = mix64(seed, stream, (uint64_t)i);
    std::vector<int32_t> order((size_t)n);
    std::iota(order.begin(), order.end(), 0);
    std::sort(order.begin(), order.end(), [&](int32_t a, int32_t b) { return key[a] != key[b] ? key[a] < key[b] : a < b; });
    std::vector<int32_t> new_of_old((size_t)n);
#pragma omp parallel for schedule(static)
    for (int64_t r = 0; r < n; ++r) new_of_old[order[r]] = (int32_t)r;
    return new_of_old;
}
template <class T>
void permute_rows(std::vector<T>& tab, int cols, const std::vector<int32_t>& row_map, const std::vector<int32_t>* entry_map) {
    std::vector<T> out(tab.size());
    const int64_t n = (int64_t)row_map.size();
#pragma omp parallel for schedule(static)
    for (int64_t i = 0; i < n; ++i)
        for (int s = 0; s < cols; ++s) {
            T x = tab[i * cols + s];
            out[(int64_t)row_map[i] * cols + s] = entry_map ? (T)(*entry_map)[(size_t)x] : x;
        }
    tab.swap(out);
}

// 4x4 symmetric positive definite solve by Cholesky factorisation (RBF interpolation matrix)
void solve_spd4(const double M[4][4], const double b[4], double x[4]) {
    double Lm[4][4] = {};
    for (int i = 0; i < 4; ++i)
        for (int j = 0; j <= i; ++j) {
            double s = M[i][j];
            for (int q = 0; q < j; ++q) s -= Lm[i][q] * Lm[j][q];
            Lm[i][j] = (i == j) ? std::sqrt(s) : s / Lm[j][j];
        }
    double y[4];
    for (int i = 0; i < 4; ++i) {
        double s = b[i];
        for (int q = 0; q < i; ++q) s -= Lm[i][q] * y[q];
        y[i] = s / Lm[i][i];
    }
    for (int i = 3; i >= 0; --i) {
        double s = y[i];
        for (int q = i + 1; q < 4; ++q) s -= Lm[q][i] * x[q];
        x[i] = s / Lm[i][i];
    }
}

void build_geometry(HostGrid& g) {
    const double a = kEarthRadius;
    const int64_t nc = g.nc, ne = g.ne, nv = g.nv;
    g.cell_xyz.resize(3 * (size_t)nc);
    g.a_c.resize((size_t)nc);
    g.edge_xyz.resize(3 * (size_t)ne);
    g.edge_normal.resize(3 * (size_t)ne);
    g.l_e.resize((size_t)ne);
    g.d_e.resize((size_t)ne);
    g.inv_d_e.resize((size_t)ne);
    g.f_e.resize((size_t)ne);
    g.c_lin.resize(2 * (size_t)ne);
    g.cgrad.resize(2 * (size_t)ne);
    g.rbf.resize(4 * (size_t)ne);
    g.bln.resize(3 * (size_t)nc);
    g.adv_c.resize(3 * (size_t)nc);
    g.geofac_div.resize(3 * (size_t)nc);
    g.a_v.resize((size_t)nv);
    g.geofac_rot.resize(6 * (size_t)nv);

    // P-8: circumcentres and spherical-excess areas
#pragma omp parallel for schedule(static)
    for (int64_t c = 0; c < nc; ++c) {
        V3 p0 = ld3(g.vert_xyz, g.c2v[3 * c]), p1 = ld3(g.vert_xyz, g.c2v[3 * c + 1]), p2 = ld3(g.vert_xyz, g.c2v[3 * c + 2]);
        st3(g.cell_xyz, c, unit(cross(p1 - p0, p2 - p0)));
        g.a_c[c] = tri_area(p0, p1, p2) * a * a;
    }
    // P-4, P-8, P-9: midpoints, normals, lengths, Coriolis, linear cell->edge weights
#pragma omp parallel for schedule(static)
    for (int64_t e = 0; e < ne; ++e) {
        V3 p0 = ld3(g.vert_xyz, g.e2v[2 * e]), p1 = ld3(g.vert_xyz, g.e2v[2 * e + 1]);
        V3 c0 = ld3(g.cell_xyz, g.e2c[2 * e]), c1 = ld3(g.cell_xyz, g.e2c[2 * e + 1]);
        V3 x = unit(p0 + p1);
        V3 n = cross(unit(p1 - p0), x);
        st3(g.edge_xyz, e, x);
        st3(g.edge_normal, e, n);
        double de = arc(c0, c1);
        g.l_e[e] = arc(p0, p1) * a;
        g.d_e[e] = de * a;
        g.inv_d_e[e] = 1.0 / (de * a);
        g.f_e[e] = 2.0 * kOmega * x.z;
        g.c_lin[2 * e] = arc(x, c1) / de;
        g.c_lin[2 * e + 1] = arc(x, c0) / de;
        // P-20 distance-weighted KE-gradient coefficients, from the two linear weights: c_lin0 / c_lin1 = a1 / a0
        g.cgrad[2 * e] = (g.c_lin[2 * e] / g.c_lin[2 * e + 1]) * g.inv_d_e[e];
        g.cgrad[2 * e + 1] = (g.c_lin[2 * e + 1] / g.c_lin[2 * e]) * g.inv_d_e[e];
    }
    // folded divergence factor and P-10 bilinear (gnomonic-plane) weights
#pragma omp parallel for schedule(static)
    for (int64_t c = 0; c < nc; ++c) {
        V3 cc = ld3(g.cell_xyz, c);
        V3 p0 = ld3(g.vert_xyz, g.c2v[3 * c]);
        V3 e1 = unit(p0 - dot(p0, cc) * cc);
        V3 e2 = cross(cc, e1);
        double xi[3], eta[3];
        for (int j = 0; j < 3; ++j) {
            int32_t e = g.c2e[3 * c + j];
            g.geofac_div[3 * c + j] = g.l_e[e] * (double)g.c_os[3 * c + j] / g.a_c[c];
            V3 x = ld3(g.edge_xyz, e);
            V3 P = (1.0 / dot(x, cc)) * x - cc;
            xi[j] = dot(P, e1);
            eta[j] = dot(P, e2);
        }
        // weights with sum 1 and vanishing first moments: w_j proportional to the signed area of
        // the triangle formed by the origin and the other two points
        double w0 = xi[1] * eta[2] - xi[2] * eta[1];
        double w1 = xi[2] * eta[0] - xi[0] * eta[2];
        double w2 = xi[0] * eta[1] - xi[1] * eta[0];
        double s = w0 + w1 + w2;
        g.bln[3 * c] = w0 / s;
        g.bln[3 * c + 1] = w1 / s;
        g.bln[3 * c + 2] = w2 / s;
        // P-19 normal-component reconstruction weights: sum_j a_j n_j n_j^T = I. With n_j = (cos t_j, sin t_j),
        // n n^T = (I + R(2 t_j)) / 2, so the conditions are sum a_j = 2 and sum a_j z_j = 0 for the doubled-angle points
        // z_j = (cos 2t_j, sin 2t_j): the barycentric weights of the origin in the triangle z_0 z_1 z_2, times 2.
        double zx[3], zy[3];
        for (int j = 0; j < 3; ++j) {
            V3 n = ld3(g.edge_normal, g.c2e[3 * c + j]);
            const double px = dot(n, e1), py = dot(n, e2), r2 = px * px + py * py;
            zx[j] = (px * px - py * py) / r2;
            zy[j] = 2.0 * px * py / r2;
        }
        const double b0 = zx[1] * zy[2] - zx[2] * zy[1], b1 = zx[2] * zy[0] - zx[0] * zy[2], b2 = zx[0] * zy[1] - zx[1] * zy[0];
        const double bs = 0.5 * (b0 + b1 + b2);
        g.adv_c[3 * c] = b0 / bs;
        g.adv_c[3 * c + 1] = b1 / bs;
        g.adv_c[3 * c + 2] = b2 / bs;
    }
    // P-8 dual areas, folded rotation factor
#pragma omp parallel for schedule(static)
    for (int64_t v = 0; v < nv; ++v) {
        const int deg = g.v_deg[v];
        V3 pv = ld3(g.vert_xyz, v);
        double area = 0.0;
        for (int i = 0; i < deg; ++i) {
            V3 xa = ld3(g.edge_xyz, g.v2e[6 * v + i]);
            V3 xb = ld3(g.edge_xyz, g.v2e[6 * v + (i + 1) % deg]);
            V3 cc = ld3(g.cell_xyz, g.v2c[6 * v + i]);
            area += tri_area(pv, xa, cc);
            area += tri_area(pv, cc, xb);
        }
        g.a_v[v] = area * a * a;
        for (int i = 0; i < 6; ++i)
            g.geofac_rot[6 * v + i] = i < deg ? g.d_e[g.v2e[6 * v + i]] * (double)g.v_os[6 * v + i] / g.a_v[v] : 0.0;
    }
    // P-11 RBF reconstruction weights, Gaussian kernel, eps = 4*sqrt(4*pi/Nc)
    const double eps = 4.0 * std::sqrt(4.0 * kPi / (double)nc);
#pragma omp parallel for schedule(static)
    for (int64_t e = 0; e < ne; ++e) {
        V3 xe = ld3(g.edge_xyz, e);
        V3 te = cross(ld3(g.edge_normal, e), xe);
        V3 xs[4], ns[4];
        for (int i = 0; i < 4; ++i) {
            xs[i] = ld3(g.edge_xyz, g.e2e4[4 * e + i]);
            ns[i] = ld3(g.edge_normal, g.e2e4[4 * e + i]);
        }
        double M[4][4], b[4], c[4];
        for (int i = 0; i < 4; ++i) {
            for (int j = 0; j <= i; ++j) {
                double r = arc(xs[i], xs[j]) / eps;
                M[i][j] = M[j][i] = std::exp(-(r * r)) * dot(ns[i], ns[j]);
            }
            double r = arc(xs[i], xe) / eps;
            b[i] = std::exp(-(r * r)) * dot(ns[i], te);
        }
        solve_spd4(M, b, c);
        double s = 0.0;
        for (int i = 0; i < 4; ++i) s += c[i] * dot(ns[i], te);
        for (int i = 0; i < 4; ++i) g.rbf[4 * e + i] = c[i] / s;
    }
}

}  // namespace

std::string build_host_grid(int k, uint64_t seed, bool permute, HostGrid& g) {
    if (k < 0 || k > 9) return "bisections_k must be in 0..9";
    Level cur, nxt;
    base_level(cur);
    for (int b = 0; b <= k; ++b) {
        refine(cur, nxt, /*need_e2v=*/b < k);
        std::swap(cur, nxt);
        nxt = Level();
    }
    const int64_t nc = cur.nc, ne = cur.ne, nv = cur.nv;
    g.level_k = k;
    g.nc = nc;
    g.ne = ne;
    g.nv = nv;
    g.permuted = permute;

    // P-3: canonical ids = first touch in the sweep over cells and slots
    std::vector<int32_t> vnew((size_t)nv, -1), enew((size_t)ne, -1);
    std::vector<int32_t> v_first_cell((size_t)nv);
    std::vector<int8_t> v_first_slot((size_t)nv);
    g.c2v.resize(3 * (size_t)nc);
    g.c2e.resize(3 * (size_t)nc);
    g.e2v.resize(2 * (size_t)ne);
    g.e2c.resize(2 * (size_t)ne);
    int32_t next_v = 0, next_e = 0;
    for (int64_t c = 0; c < nc; ++c) {
        for (int j = 0; j < 3; ++j) {
            int32_t pv = cur.c2v[3 * c + j];
            if (vnew[pv] < 0) {
                v_first_cell[next_v] = (int32_t)c;
                v_first_slot[next_v] = (int8_t)j;
                vnew[pv] = next_v++;
            }
            g.c2v[3 * c + j] = vnew[pv];
        }
        for (int j = 0; j < 3; ++j) {
            int32_t pe = cur.c2e[3 * c + j];
            if (enew[pe] < 0) {
                enew[pe] = next_e;
                g.e2v[2 * (int64_t)next_e] = g.c2v[3 * c + j];
                g.e2v[2 * (int64_t)next_e + 1] = g.c2v[3 * c + (j + 1) % 3];
                g.e2c[2 * (int64_t)next_e] = (int32_t)c;
                ++next_e;
            } else {
                g.e2c[2 * (int64_t)enew[pe] + 1] = (int32_t)c;
            }
            g.c2e[3 * c + j] = enew[pe];
        }
    }
    if (next_v != nv || next_e != ne) return "internal error: first-touch numbering did not cover the grid";
    g.vert_xyz.resize(3 * (size_t)nv);
#pragma omp parallel for schedule(static)
    for (int64_t pv = 0; pv < nv; ++pv) st3(g.vert_xyz, vnew[pv], ld3(cur.xyz, pv));
    cur = Level();
    vnew.clear();
    vnew.shrink_to_fit();
    enew.clear();
    enew.shrink_to_fit();

    // P-4: orientation of a cell with respect to its edges, by slot
    g.c_os.resize(3 * (size_t)nc);
#pragma omp parallel for schedule(static)
    for (int64_t h = 0; h < 3 * nc; ++h) g.c_os[h] = g.e2c[2 * (int64_t)g.c2e[h]] == (int32_t)(h / 3) ? 1 : -1;

    // P-5: fans, counter-clockwise from the first-touch cell
    g.v2e.resize(6 * (size_t)nv);
    g.v2c.resize(6 * (size_t)nv);
    g.v_os.resize(6 * (size_t)nv);
    g.v_deg.resize((size_t)nv);
    int fan_error = 0;
#pragma omp parallel for schedule(static)
    for (int64_t v = 0; v < nv; ++v) {
        int32_t c = v_first_cell[v];
        int j = v_first_slot[v];
        int deg = 0;
        while (true) {
            g.v2c[6 * v + deg] = c;
            g.v2e[6 * v + deg] = g.c2e[3 * (int64_t)c + j];
            ++deg;
            int32_t en = g.c2e[3 * (int64_t)c + (j + 2) % 3];
            int32_t cn = g.e2c[2 * (int64_t)en] == c ? g.e2c[2 * (int64_t)en + 1] : g.e2c[2 * (int64_t)en];
            if (cn == v_first_cell[v]) break;
            if (deg == 6) { fan_error = 1; break; }
            c = cn;
            j = g.c2v[3 * (int64_t)c] == v ? 0 : (g.c2v[3 * (int64_t)c + 1] == v ? 1 : 2);
        }
        g.v_deg[v] = deg;
        for (int i = 0; i < 6; ++i) {
            if (i < deg) {
                g.v_os[6 * v + i] = g.e2v[2 * (int64_t)g.v2e[6 * v + i]] == (int32_t)v ? -1 : 1;
            } else {
                g.v2e[6 * v + i] = g.v2e[6 * v];
                g.v2c[6 * v + i] = g.v2c[6 * v];
                g.v_os[6 * v + i] = 0;
            }
        }
    }
    if (fan_error) return "internal error: vertex fan with more than 6 cells";

    // P-6: the four other edges of the two cells of an edge
    g.e2e4.resize(4 * (size_t)ne);
#pragma omp parallel for schedule(static)
    for (int64_t e = 0; e < ne; ++e)
        for (int side = 0; side < 2; ++side) {
            const int32_t* ce = &g.c2e[3 * (int64_t)g.e2c[2 * e + side]];
            int j = ce[0] == e ? 0 : (ce[1] == e ? 1 : 2);
            g.e2e4[4 * e + 2 * side] = ce[(j + 1) % 3];
            g.e2e4[4 * e + 2 * side + 1] = ce[(j + 2) % 3];
        }

    // P-7: seeded renumbering; rows move, entries are renumbered, slot order is kept
    if (permute) {
        std::vector<int32_t> pc = rank_permutation(seed, 0, nc), pe = rank_permutation(seed, 1, ne), pv = rank_permutation(seed, 2, nv);
        permute_rows(g.c2v, 3, pc, &pv);
        permute_rows(g.c2e, 3, pc, &pe);
        permute_rows(g.e2c, 2, pe, &pc);
        permute_rows(g.e2v, 2, pe, &pv);
        permute_rows(g.e2e4, 4, pe, &pe);
        permute_rows(g.v2e, 6, pv, &pe);
        permute_rows(g.v2c, 6, pv, &pc);
        permute_rows(g.v_deg, 1, pv, nullptr);
        permute_rows(g.c_os, 3, pc, nullptr);
        permute_rows(g.v_os, 6, pv, nullptr);
        permute_rows(g.vert_xyz, 3, pv, nullptr);
        g.user_of_pos_c.swap(pc);
        g.user_of_pos_e.swap(pe);
        g.user_of_pos_v.swap(pv);
    }
    build_geometry(g);
    return std::string();
}

}  // namespace icon
