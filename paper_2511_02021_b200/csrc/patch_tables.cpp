// patch_tables.cpp -- builds the tile / patch work-list of the fused kernels from the public
// connectivity (see patch_tables.hpp for the local topology). Everything is derived from the
// user-id tables c2v/c2e/e2c/e2e4/v2e and the generation order, and every structural assumption
// is checked, so a table that does not describe a 4-child bisection patch is an error, never a
// silently wrong stencil.
//
// Neighbour order of the nine tangential-wind stencils (reading P-6/P-11: vt = sum_j rbf_j vn_j):
//   i0: b0 b5 i1 i2     i1: b1 b2 i2 i0     i2: b3 b4 i0 i1
//   b0: i0 b5 om0 oc0   b1: b2 i1 om1 oc1   b2: b1 i1 om2 oc2
//   b3: i2 b4 om3 oc3   b4: i2 b3 om4 oc4   b5: b0 i0 om5 oc5
// Fan order of the three midpoint vorticities (reading P-5: zeta = sum_j geofac_rot_j vn_j):
//   ab: b0 b1 i0 i1 om0 om1     bc: b2 b3 i1 i2 om2 om3     ca: b4 b5 i2 i0 om4 om5
// Owned edges and their (L, H) cells, gradK = (KE(H) - KE(L)) * s_inv_d:
//   i0:(T0,T3) i1:(T1,T3) i2:(T2,T3) b0:(T0,X0) b2:(T1,X2) b4:(T2,X4)
// Every boundary half edge is owned by exactly one of its two patches: the one for which it is the
// FIRST half of the parent side in counter-clockwise order (the neighbour walks the side the other
// way round, so its first half is our second half).
#include "patch_tables.hpp"

#include <algorithm>
#include <atomic>

namespace icon {
namespace {

struct Ctx {
    const HostGrid& g;
    std::vector<int32_t> pos_c;   // generation position of a user cell id (identity if not permuted)
    explicit Ctx(const HostGrid& grid) : g(grid) {
        if (!g.user_of_pos_c.empty()) {
            pos_c.resize((size_t)g.nc);
#pragma omp parallel for schedule(static)
            for (int64_t p = 0; p < g.nc; ++p) pos_c[(size_t)g.user_of_pos_c[p]] = (int32_t)p;
        }
    }
    int32_t user_cell(int64_t pos) const { return g.user_of_pos_c.empty() ? (int32_t)pos : g.user_of_pos_c[(size_t)pos]; }
    int64_t pos_of_cell(int32_t user) const { return pos_c.empty() ? user : pos_c[(size_t)user]; }
    int32_t other_cell(int32_t e, int32_t c) const {
        return g.e2c[2 * (int64_t)e] == c ? g.e2c[2 * (int64_t)e + 1] : g.e2c[2 * (int64_t)e];
    }
    bool edge_has_vertex(int32_t e, int32_t v) const { return g.e2v[2 * (int64_t)e] == v || g.e2v[2 * (int64_t)e + 1] == v; }
    // rbf coefficient of edge x that multiplies neighbour n; NaN flag through `ok`
    double rbf_for(int32_t x, int32_t n, bool& ok) const {
        for (int q = 0; q < 4; ++q)
            if (g.e2e4[4 * (int64_t)x + q] == n) return g.rbf[4 * (int64_t)x + q];
        ok = false;
        return 0.0;
    }
    double rot_for(int32_t v, int32_t e, bool& ok) const {
        for (int q = 0; q < g.v_deg[(size_t)v]; ++q)
            if (g.v2e[6 * (int64_t)v + q] == e) return g.geofac_rot[6 * (int64_t)v + q];
        ok = false;
        return 0.0;
    }
};

struct PatchLocal {
    int32_t T[4], ei[3], eb[6], om[6], oc[6], X[6];
    int32_t va, vb, vc, vab, vbc, vca;
};

bool patch_local(const Ctx& c, int64_t p, PatchLocal& L) {
    const HostGrid& g = c.g;
    for (int j = 0; j < 4; ++j) L.T[j] = c.user_cell(4 * p + j);
    auto ce = [&](int j, int s) { return g.c2e[3 * (int64_t)L.T[j] + s]; };
    auto cv = [&](int j, int s) { return g.c2v[3 * (int64_t)L.T[j] + s]; };
    L.eb[0] = ce(0, 0); L.ei[0] = ce(0, 1); L.eb[5] = ce(0, 2);
    L.eb[1] = ce(1, 0); L.eb[2] = ce(1, 1); L.ei[1] = ce(1, 2);
    L.ei[2] = ce(2, 0); L.eb[3] = ce(2, 1); L.eb[4] = ce(2, 2);
    if (ce(3, 0) != L.ei[1] || ce(3, 1) != L.ei[2] || ce(3, 2) != L.ei[0]) return false;
    L.va = cv(0, 0); L.vab = cv(0, 1); L.vca = cv(0, 2);
    L.vb = cv(1, 1); L.vbc = cv(1, 2); L.vc = cv(2, 2);
    if (cv(1, 0) != L.vab || cv(2, 0) != L.vca || cv(2, 1) != L.vbc) return false;
    if (cv(3, 0) != L.vab || cv(3, 1) != L.vbc || cv(3, 2) != L.vca) return false;
    const int inside[6] = {0, 1, 1, 2, 2, 0};                                  // cell of the patch that holds bj
    const int32_t mid[6] = {L.vab, L.vab, L.vbc, L.vbc, L.vca, L.vca};         // midpoint end of bj
    const int32_t cor[6] = {L.va, L.vb, L.vb, L.vc, L.vc, L.va};               // corner end of bj
    for (int j = 0; j < 6; ++j) {
        const int32_t e = L.eb[j];
        if (!c.edge_has_vertex(e, mid[j]) || !c.edge_has_vertex(e, cor[j])) return false;
        const int32_t x = c.other_cell(e, L.T[inside[j]]);
        L.X[j] = x;
        L.om[j] = L.oc[j] = -1;
        for (int s = 0; s < 3; ++s) {
            const int32_t o = g.c2e[3 * (int64_t)x + s];
            if (o == e) continue;
            if (c.edge_has_vertex(o, mid[j])) L.om[j] = o;
            else if (c.edge_has_vertex(o, cor[j])) L.oc[j] = o;
        }
        if (L.om[j] < 0 || L.oc[j] < 0) return false;
    }
    return true;
}

}  // namespace

std::string build_patch_tables(const HostGrid& g, PatchTables& t) {
    if (g.nc % 4) return "patch tables: cell count is not a multiple of 4";
    Ctx c(g);
    const int64_t np = g.nc / 4;
    const int64_t nt = (np + kPatchesPerTile - 1) / kPatchesPerTile;
    t.n_patches = np;
    t.n_tiles = nt;
    t.patch_ids.assign((size_t)np * kPatchIdWords, 0);
    t.patch_coef.assign((size_t)np * kPatchCoefWords, 0.0);
    t.tile_hdr.assign((size_t)nt * 4, 0);
    t.mid_store.assign((size_t)np, 0);
    t.mid_vertex.assign((size_t)np * 4, 0);

    // ---- per patch: ids and coefficients in local slot order --------------------------------
    std::atomic<int> bad(0);
#pragma omp parallel for schedule(static)
    for (int64_t p = 0; p < np; ++p) {
        PatchLocal L;
        if (!patch_local(c, p, L)) {
            bad = 1;
            continue;
        }
        int32_t* id = &t.patch_ids[(size_t)p * kPatchIdWords];
        double* cf = &t.patch_coef[(size_t)p * kPatchCoefWords];
        for (int j = 0; j < 3; ++j) id[PID_I0 + j] = L.ei[j];
        for (int j = 0; j < 6; ++j) {
            id[PID_B0 + j] = L.eb[j];
            id[PID_OM0 + j] = L.om[j];
            id[PID_OC0 + j] = L.oc[j];
        }
        for (int j = 0; j < 4; ++j) id[PID_T0 + j] = L.T[j];
        bool ok = true;
        const int32_t *I = L.ei, *B = L.eb, *M = L.om, *O = L.oc;
        const int32_t nb[9][4] = {
            {B[0], B[5], I[1], I[2]}, {B[1], B[2], I[2], I[0]}, {B[3], B[4], I[0], I[1]},
            {I[0], B[5], M[0], O[0]}, {B[2], I[1], M[1], O[1]}, {B[1], I[1], M[2], O[2]},
            {I[2], B[4], M[3], O[3]}, {I[2], B[3], M[4], O[4]}, {B[0], I[0], M[5], O[5]}};
        const int32_t self[9] = {I[0], I[1], I[2], B[0], B[1], B[2], B[3], B[4], B[5]};
        for (int x = 0; x < 9; ++x)
            for (int q = 0; q < 4; ++q) cf[PCF_RBF + 4 * x + q] = c.rbf_for(self[x], nb[x][q], ok);
        for (int j = 0; j < 4; ++j)
            for (int s = 0; s < 3; ++s) cf[PCF_BLN + 3 * j + s] = g.bln[3 * (int64_t)L.T[j] + s];
        const int32_t midv[3] = {L.vab, L.vbc, L.vca};
        const int32_t fan[3][6] = {{B[0], B[1], I[0], I[1], M[0], M[1]},
                                   {B[2], B[3], I[1], I[2], M[2], M[3]},
                                   {B[4], B[5], I[2], I[0], M[4], M[5]}};
        for (int m = 0; m < 3; ++m) {
            if (g.v_deg[(size_t)midv[m]] != 6) ok = false;
            for (int q = 0; q < 6; ++q) cf[PCF_ROT + 6 * m + q] = c.rot_for(midv[m], fan[m][q], ok);
            t.mid_vertex[(size_t)p * 4 + m] = midv[m];
        }
        // owned edges: i0 i1 i2 b0 b2 b4 with their (L, H) cells
        const int32_t own[6] = {I[0], I[1], I[2], B[0], B[2], B[4]};
        const int32_t lo[6] = {L.T[0], L.T[1], L.T[2], L.T[0], L.T[1], L.T[2]};
        const int32_t hi[6] = {L.T[3], L.T[3], L.T[3], L.X[0], L.X[2], L.X[4]};
        for (int x = 0; x < 6; ++x) {
            const int64_t e = own[x];
            const int32_t c0 = g.e2c[2 * e], c1 = g.e2c[2 * e + 1];
            double* o = cf + PCF_EDGE + 4 * x;
            if (c0 == lo[x] && c1 == hi[x]) {
                o[0] = g.inv_d_e[e]; o[2] = g.c_lin[2 * e]; o[3] = g.c_lin[2 * e + 1];
            } else if (c0 == hi[x] && c1 == lo[x]) {
                o[0] = -g.inv_d_e[e]; o[2] = g.c_lin[2 * e + 1]; o[3] = g.c_lin[2 * e];
            } else {
                ok = false;
            }
            o[1] = g.f_e[e];
        }
        // midpoint vertex j is stored (div/vort call) by the patch with the smaller generation
        // position of the two patches that share the parent side
        const int side_edge[3] = {0, 2, 4};
        int ms = 0;
        for (int m = 0; m < 3; ++m) {
            const int64_t q = c.pos_of_cell(L.X[side_edge[m]]) / 4;
            if (q == p) ok = false;
            if (p < q) ms |= 1 << m;
        }
        t.mid_store[(size_t)p] = ms;
        if (!ok) bad = 1;
    }
    if (bad) return "patch tables: the grid is not a 4-child bisection hierarchy in generation order";

    // ---- per tile: halo cells (outer cells of owned boundary edges outside the tile) and corner
    //      vertices; exchange slots ---------------------------------------------------------------
    std::vector<std::vector<int32_t>> halo_of((size_t)nt), vert_of((size_t)nt);
#pragma omp parallel for schedule(dynamic, 64)
    for (int64_t tl = 0; tl < nt; ++tl) {
        auto& hl = halo_of[(size_t)tl];
        auto& vl = vert_of[(size_t)tl];
        const int64_t p0 = tl * kPatchesPerTile, p1 = std::min(np, p0 + kPatchesPerTile);
        for (int64_t p = p0; p < p1; ++p) {
            PatchLocal L;
            patch_local(c, p, L);
            int32_t* id = &t.patch_ids[(size_t)p * kPatchIdWords];
            const int ob[3] = {0, 2, 4};
            for (int x = 0; x < 3; ++x) {
                const int32_t X = L.X[ob[x]];
                const int64_t px = c.pos_of_cell(X);
                int slot;
                if (px / (4 * kPatchesPerTile) == tl) {
                    slot = 3 * (int)((px / 4) % kPatchesPerTile) + (int)(px % 4);   // px%4 != 3: T3 has no boundary edge
                } else {
                    auto it = std::find(hl.begin(), hl.end(), X);
                    if (it == hl.end()) {
                        hl.push_back(X);
                        it = hl.end() - 1;
                    }
                    slot = 3 * kPatchesPerTile + (int)(it - hl.begin());
                }
                id[PID_XSLOT + x] = slot;
            }
            const int32_t cor[3] = {L.va, L.vb, L.vc};
            for (int x = 0; x < 3; ++x) {
                auto it = std::find(vl.begin(), vl.end(), cor[x]);
                if (it == vl.end()) {
                    vl.push_back(cor[x]);
                    it = vl.end() - 1;
                }
                id[PID_VSLOT + x] = (int)(it - vl.begin());
            }
        }
    }
    int64_t nh = 0, nvt = 0;
    t.max_halo = t.max_vert = 0;
    for (int64_t tl = 0; tl < nt; ++tl) {
        int32_t* h = &t.tile_hdr[(size_t)tl * 4];
        h[0] = (int32_t)nh; h[1] = (int32_t)halo_of[(size_t)tl].size();
        h[2] = (int32_t)nvt; h[3] = (int32_t)vert_of[(size_t)tl].size();
        nh += h[1]; nvt += h[3];
        t.max_halo = std::max(t.max_halo, (int)h[1]);
        t.max_vert = std::max(t.max_vert, (int)h[3]);
    }
    if (nh > INT32_MAX || nvt > INT32_MAX) return "patch tables: task lists exceed int32";
    t.halo_ids.assign((size_t)nh * kHaloIdWords, 0);
    t.halo_coef.assign((size_t)nh * kHaloCoefWords, 0.0);
    t.vert_ids.assign((size_t)nvt * kVertIdWords, 0);
    t.vert_coef.assign((size_t)nvt * kVertCoefWords, 0.0);
    t.vert_store.assign((size_t)nvt, 0);
    // a corner vertex is stored (div/vort call) by the first tile in generation order that lists it
    std::vector<int32_t> first_tile((size_t)g.nv, INT32_MAX);
    for (int64_t tl = 0; tl < nt; ++tl)
        for (int32_t v : vert_of[(size_t)tl]) first_tile[(size_t)v] = std::min(first_tile[(size_t)v], (int32_t)tl);
#pragma omp parallel for schedule(dynamic, 64)
    for (int64_t tl = 0; tl < nt; ++tl) {
        const int32_t* h = &t.tile_hdr[(size_t)tl * 4];
        for (int i = 0; i < h[1]; ++i) {
            const int32_t X = halo_of[(size_t)tl][(size_t)i];
            int32_t* id = &t.halo_ids[((size_t)h[0] + i) * kHaloIdWords];
            double* cf = &t.halo_coef[((size_t)h[0] + i) * kHaloCoefWords];
            bool ok = true;
            int32_t e[3];
            for (int j = 0; j < 3; ++j) e[j] = id[j] = g.c2e[3 * (int64_t)X + j];
            for (int j = 0; j < 3; ++j) {
                const int32_t far_c = c.other_cell(e[j], X);
                int n = 0;
                int32_t far[2] = {-1, -1};
                for (int s = 0; s < 3; ++s) {
                    const int32_t o = g.c2e[3 * (int64_t)far_c + s];
                    if (o != e[j] && n < 2) far[n++] = o;
                }
                id[3 + 2 * j] = far[0];
                id[4 + 2 * j] = far[1];
                cf[4 * j + 0] = c.rbf_for(e[j], e[(j + 1) % 3], ok);
                cf[4 * j + 1] = c.rbf_for(e[j], e[(j + 2) % 3], ok);
                cf[4 * j + 2] = c.rbf_for(e[j], far[0], ok);
                cf[4 * j + 3] = c.rbf_for(e[j], far[1], ok);
                cf[12 + j] = g.bln[3 * (int64_t)X + j];
            }
            id[9] = X;
            if (!ok) bad = 1;
        }
        for (int i = 0; i < h[3]; ++i) {
            const int32_t v = vert_of[(size_t)tl][(size_t)i];
            int32_t* id = &t.vert_ids[((size_t)h[2] + i) * kVertIdWords];
            double* cf = &t.vert_coef[((size_t)h[2] + i) * kVertCoefWords];
            for (int q = 0; q < 6; ++q) {
                id[q] = g.v2e[6 * (int64_t)v + q];          // pentagon pad: valid id, coefficient 0 (P-5)
                cf[q] = g.geofac_rot[6 * (int64_t)v + q];
            }
            id[6] = v;
            t.vert_store[(size_t)h[2] + i] = first_tile[(size_t)v] == (int32_t)tl ? 1 : 0;
        }
    }
    if (bad) return "patch tables: halo stencil does not match e2e4";
    return std::string();
}

}  // namespace icon
