// sc_tables.cpp -- builds the self-contained patch records (sc_tables.hpp) from the public
// connectivity. Every structural assumption is checked: a record that does not describe a 4-child
// bisection patch with its outer ring is an error, never a silently wrong stencil.
#include "sc_tables.hpp"

#include <atomic>

namespace icon {
namespace {

struct View {
    const HostGrid& g;
    explicit View(const HostGrid& grid) : g(grid) {}
    int32_t user_cell(int64_t pos) const { return g.user_of_pos_c.empty() ? (int32_t)pos : g.user_of_pos_c[(size_t)pos]; }
    int32_t other_cell(int32_t e, int32_t c) const {
        return g.e2c[2 * (int64_t)e] == c ? g.e2c[2 * (int64_t)e + 1] : g.e2c[2 * (int64_t)e];
    }
    bool touches(int32_t e, int32_t v) const { return g.e2v[2 * (int64_t)e] == v || g.e2v[2 * (int64_t)e + 1] == v; }
    // the two edges of cell c other than e: `with_v` = the one touching vertex v, `without_v` = the other
    bool split_cell(int32_t c, int32_t e, int32_t v, int32_t& with_v, int32_t& without_v) const {
        with_v = without_v = -1;
        for (int s = 0; s < 3; ++s) {
            const int32_t o = g.c2e[3 * (int64_t)c + s];
            if (o == e) continue;
            if (touches(o, v) && with_v < 0) with_v = o;
            else without_v = o;
        }
        return with_v >= 0 && without_v >= 0;
    }
    // coefficients of stencil row `x` (4 entries of e2e4 / rbf) re-ordered to the slots nb[0..3]
    bool rbf_row(int32_t x, const int32_t nb[4], double out[4]) const {
        bool used[4] = {false, false, false, false};
        for (int s = 0; s < 4; ++s) {
            int hit = -1;
            for (int q = 0; q < 4; ++q)
                if (!used[q] && g.e2e4[4 * (int64_t)x + q] == nb[s]) { hit = q; break; }
            if (hit < 0) return false;
            used[hit] = true;
            out[s] = g.rbf[4 * (int64_t)x + hit];
        }
        return true;
    }
    // geofac_rot of vertex v re-ordered to the slots fan[0..n-1]; unmatched slots get 0, every
    // fan edge of v must land in exactly one slot
    bool rot_row(int32_t v, const int32_t* fan, int n, double scale, double* out) const {
        const int deg = g.v_deg[(size_t)v];
        for (int s = 0; s < n; ++s) out[s] = 0.0;
        bool used[6] = {false, false, false, false, false, false};
        for (int q = 0; q < deg; ++q) {
            const int32_t e = g.v2e[6 * (int64_t)v + q];
            int hit = -1;
            for (int s = 0; s < n; ++s)
                if (!used[s] && fan[s] == e) { hit = s; break; }
            if (hit < 0) return false;
            used[hit] = true;
            out[hit] = scale * g.geofac_rot[6 * (int64_t)v + q];
        }
        return true;
    }
    // geofac_div of cell c re-ordered to the edge slots e[0..2]
    bool div_row(int32_t c, const int32_t e[3], double out[3]) const {
        bool used[3] = {false, false, false};
        for (int s = 0; s < 3; ++s) {
            int hit = -1;
            for (int q = 0; q < 3; ++q)
                if (!used[q] && g.c2e[3 * (int64_t)c + q] == e[s]) { hit = q; break; }
            if (hit < 0) return false;
            used[hit] = true;
            out[s] = g.geofac_div[3 * (int64_t)c + hit];
        }
        return true;
    }
    // adv_c(c,.) * inv_d_e of the edge, re-ordered to the edge slots e[0..2], signed so that the advection term of cell c
    // reads out * vn_ie * (w(cell across the edge) - w(c)): + if c is e2c[.][0] of the edge, - if it is e2c[.][1] (P-19)
    bool adv_row(int32_t c, const int32_t e[3], double out[3]) const {
        bool used[3] = {false, false, false};
        for (int s = 0; s < 3; ++s) {
            int hit = -1;
            for (int q = 0; q < 3; ++q)
                if (!used[q] && g.c2e[3 * (int64_t)c + q] == e[s]) { hit = q; break; }
            if (hit < 0) return false;
            used[hit] = true;
            const int64_t ed = e[s];
            const double sign = g.e2c[2 * ed] == c ? 1.0 : -1.0;
            out[s] = sign * g.adv_c[3 * (int64_t)c + hit] * g.inv_d_e[ed];
        }
        return true;
    }
    bool bln_row(int32_t c, const int32_t e[3], double scale, double out[3]) const {
        bool used[3] = {false, false, false};
        for (int s = 0; s < 3; ++s) {
            int hit = -1;
            for (int q = 0; q < 3; ++q)
                if (!used[q] && g.c2e[3 * (int64_t)c + q] == e[s]) { hit = q; break; }
            if (hit < 0) return false;
            used[hit] = true;
            out[s] = scale * g.bln[3 * (int64_t)c + hit];
        }
        return true;
    }
};

struct Local {
    int32_t T[4], ei[3], eb[6], om[6], oc[6], X[6];
    int32_t va, vb, vc, vab, vbc, vca;
};

bool local_topology(const View& c, int64_t p, Local& L) {
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
    const int inside[6] = {0, 1, 1, 2, 2, 0};
    const int32_t mid[6] = {L.vab, L.vab, L.vbc, L.vbc, L.vca, L.vca};
    const int32_t cor[6] = {L.va, L.vb, L.vb, L.vc, L.vc, L.va};
    for (int j = 0; j < 6; ++j) {
        const int32_t e = L.eb[j];
        if (!c.touches(e, mid[j]) || !c.touches(e, cor[j])) return false;
        L.X[j] = c.other_cell(e, L.T[inside[j]]);
        // om touches the midpoint end, oc the corner end
        if (!c.split_cell(L.X[j], e, mid[j], L.om[j], L.oc[j])) return false;
        if (!c.touches(L.oc[j], cor[j])) return false;
    }
    return true;
}

}  // namespace

std::string build_sc_tables(const HostGrid& g, ScTables& t) {
    if (g.nc % 4) return "sc tables: cell count is not a multiple of 4";
    View c(g);
    const int64_t np = g.nc / 4;
    t.n_patches = np;
    t.ids.assign((size_t)np * kScIdWords, 0);
    t.coef.assign((size_t)np * kScCoefWords, 0.0);
    std::atomic<int> bad(0);
#pragma omp parallel for schedule(static)
    for (int64_t p = 0; p < np; ++p) {
        Local L;
        if (!local_topology(c, p, L)) {
            bad = 1;
            continue;
        }
        int32_t* id = &t.ids[(size_t)p * kScIdWords];
        double* cf = &t.coef[(size_t)p * kScCoefWords];
        const int32_t *I = L.ei, *B = L.eb, *M = L.om, *O = L.oc;
        for (int j = 0; j < 3; ++j) id[SID_I0 + j] = I[j];
        for (int j = 0; j < 6; ++j) {
            id[SID_B0 + j] = B[j];
            id[SID_OM0 + j] = M[j];
            id[SID_OC0 + j] = O[j];
        }
        for (int j = 0; j < 4; ++j) id[SID_T0 + j] = L.T[j];
        bool ok = true;
        // nine tangential-wind stencils of the patch (fixed neighbour order, see build_sc_tables)
        const int32_t nb[9][4] = {
            {B[0], B[5], I[1], I[2]}, {B[1], B[2], I[2], I[0]}, {B[3], B[4], I[0], I[1]},
            {I[0], B[5], M[0], O[0]}, {B[2], I[1], M[1], O[1]}, {B[1], I[1], M[2], O[2]},
            {I[2], B[4], M[3], O[3]}, {I[2], B[3], M[4], O[4]}, {B[0], I[0], M[5], O[5]}};
        const int32_t self[9] = {I[0], I[1], I[2], B[0], B[1], B[2], B[3], B[4], B[5]};
        for (int x = 0; x < 9; ++x) ok &= c.rbf_row(self[x], nb[x], cf + SCF_RBF + 4 * x);
        const int32_t cell_e[4][3] = {{B[0], I[0], B[5]}, {B[1], B[2], I[1]}, {I[2], B[3], B[4]}, {I[1], I[2], I[0]}};
        for (int j = 0; j < 4; ++j) ok &= c.bln_row(L.T[j], cell_e[j], 0.5, cf + SCF_BLN + 3 * j);
        for (int j = 0; j < 4; ++j) ok &= c.div_row(L.T[j], cell_e[j], cf + SCF_DIV + 3 * j);
        for (int j = 0; j < 4; ++j) ok &= c.adv_row(L.T[j], cell_e[j], cf + SCF_ADV + 3 * j);
        for (int x = 0; x < 3; ++x) id[SID_XW0 + x] = L.X[2 * x + 1];
        {
            const int32_t vs[6] = {L.vab, L.vbc, L.vca, L.va, L.vb, L.vc};
            for (int j = 0; j < 6; ++j) id[SID_V0 + j] = vs[j];
        }
        const int32_t midv[3] = {L.vab, L.vbc, L.vca};
        const int32_t fan[3][6] = {{B[0], B[1], I[0], I[1], M[0], M[1]},
                                   {B[2], B[3], I[1], I[2], M[2], M[3]},
                                   {B[4], B[5], I[2], I[0], M[4], M[5]}};
        for (int m = 0; m < 3; ++m) {
            if (g.v_deg[(size_t)midv[m]] != 6) ok = false;
            ok &= c.rot_row(midv[m], fan[m], 6, 0.5, cf + SCF_ROT + 6 * m);
        }
        // owned edges with their (L, H) cells: gradK = (KE(H) - KE(L)) * s_inv_d
        const int32_t own[6] = {I[0], I[1], I[2], B[0], B[2], B[4]};
        const int32_t lo[6] = {L.T[0], L.T[1], L.T[2], L.T[0], L.T[1], L.T[2]};
        const int32_t hi[6] = {L.T[3], L.T[3], L.T[3], L.X[0], L.X[2], L.X[4]};
        for (int x = 0; x < 6; ++x) {
            const int64_t e = own[x];
            const int32_t c0 = g.e2c[2 * e], c1 = g.e2c[2 * e + 1];
            double* o = cf + SCF_EDGE + 4 * x;
            double* m = cf + SCF_CGRAD + 4 * x;     // P-20: cgrad(e,1) KE_c(c1) - cgrad(e,0) KE_c(c0) + KE_e (cgrad(e,0) - cgrad(e,1))
            if (c0 == lo[x] && c1 == hi[x]) {
                o[0] = g.inv_d_e[e]; o[2] = g.c_lin[2 * e]; o[3] = g.c_lin[2 * e + 1];
                m[0] = g.cgrad[2 * e]; m[1] = g.cgrad[2 * e + 1];
            } else if (c0 == hi[x] && c1 == lo[x]) {
                o[0] = -g.inv_d_e[e]; o[2] = g.c_lin[2 * e + 1]; o[3] = g.c_lin[2 * e];
                m[0] = -g.cgrad[2 * e + 1]; m[1] = -g.cgrad[2 * e];
            } else {
                ok = false;
            }
            m[2] = 0.5 * (m[0] - m[1]);
            m[3] = 0.0;
            o[1] = g.f_e[e];
        }
        // the outer ring of the three owned boundary edges
        const int32_t cor[3] = {L.va, L.vb, L.vc};
        for (int x = 0; x < 3; ++x) {
            const int j = 2 * x, jp = (j + 5) % 6;
            const int32_t X = L.X[j], C = cor[x];
            id[SID_XC0 + x] = X;
            int32_t* ex = id + SID_X0 + 5 * x;
            // cell across om_j: its two other edges, in c2e order
            const int32_t Wc = c.other_cell(M[j], X);
            int n = 0;
            for (int s = 0; s < 3; ++s) {
                const int32_t o = g.c2e[3 * (int64_t)Wc + s];
                if (o != M[j] && n < 2) ex[n++] = o;
            }
            if (n != 2) ok = false;
            // cell Z1 across oc_j: n1 touches the corner, pcf does not
            const int32_t Z1 = c.other_cell(O[j], X);
            int32_t n1, pcf;
            if (!c.split_cell(Z1, O[j], C, n1, pcf)) ok = false;
            int32_t n2 = n1;
            const int deg = g.v_deg[(size_t)C];
            if (ok && deg == 6) {
                const int32_t Z2 = c.other_cell(n1, Z1);
                int32_t rest;
                if (!c.split_cell(Z2, n1, C, n2, rest)) ok = false;
            }
            ex[2] = pcf; ex[3] = n1; ex[4] = n2;
            if (!ok) continue;
            const int32_t nm[4] = {B[j], O[j], ex[0], ex[1]};
            const int32_t no[4] = {B[j], M[j], n1, pcf};
            ok &= c.rbf_row(M[j], nm, cf + SCF_XRM + 4 * x);
            ok &= c.rbf_row(O[j], no, cf + SCF_XRO + 4 * x);
            const int32_t xe[3] = {B[j], M[j], O[j]};
            ok &= c.bln_row(X, xe, 0.5, cf + SCF_XBL + 3 * x);
            const int32_t cfan[6] = {B[j], O[j], n1, n2, O[jp], B[jp]};
            if (deg == 6) {
                ok &= c.rot_row(C, cfan, 6, 0.5, cf + SCF_XROT + 6 * x);
            } else {
                // pentagon: fan is b_j, oc_j, n1, oc_jp, b_jp; slot n2 keeps coefficient 0
                double tmp[5];
                const int32_t pfan[5] = {B[j], O[j], n1, O[jp], B[jp]};
                ok &= deg == 5 && c.rot_row(C, pfan, 5, 0.5, tmp);
                double* r = cf + SCF_XROT + 6 * x;
                r[0] = tmp[0]; r[1] = tmp[1]; r[2] = tmp[2]; r[3] = 0.0; r[4] = tmp[3]; r[5] = tmp[4];
            }
        }
        if (!ok) bad = 1;
    }
    if (bad) return "sc tables: the grid is not a 4-child bisection hierarchy with a regular outer ring";
    // vertex ownership: the lowest patch that has the vertex as a midpoint or a corner stores its vorticity
    {
        std::vector<int64_t> owner((size_t)g.nv, np);
        for (int64_t p = 0; p < np; ++p)
            for (int j = 0; j < 6; ++j) {
                const int32_t v = t.ids[(size_t)p * kScIdWords + SID_V0 + j];
                if (v < 0 || v >= g.nv) return "sc tables: bad vertex id";
                if (owner[(size_t)v] > p) owner[(size_t)v] = p;
            }
        for (int64_t v = 0; v < g.nv; ++v)
            if (owner[(size_t)v] == np) return "sc tables: a vertex is neither a midpoint nor a corner of any patch";
#pragma omp parallel for schedule(static)
        for (int64_t p = 0; p < np; ++p)
            for (int j = 0; j < 6; ++j) {
                int32_t& v = t.ids[(size_t)p * kScIdWords + SID_V0 + j];
                if (owner[(size_t)v] != p) { v = -1; continue; }
                for (int i = 0; i < j; ++i)          // a pentagon corner may appear twice in one patch? keep the first
                    if (t.ids[(size_t)p * kScIdWords + SID_V0 + i] == v) { v = -1; break; }
            }
    }
    return std::string();
}

}  // namespace icon
