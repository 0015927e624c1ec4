// partition.cpp -- see partition.hpp. Host code only; everything is integer work on the patch records.
#include "partition.hpp"

#include <algorithm>
#include <utility>

namespace icon {

namespace {

// P-21: ranks own contiguous ranges of patches, floor(r P / R) <= p < floor((r+1) P / R)
struct Ranges {
    std::vector<int64_t> hi;        // [R] exclusive upper bound of rank r
    Ranges(int64_t n_patches, int n_parts) : hi((size_t)n_parts) {
        for (int r = 0; r < n_parts; ++r) hi[(size_t)r] = ((int64_t)(r + 1) * n_patches) / n_parts;
    }
    int rank_of(int64_t p) const { return (int)(std::upper_bound(hi.begin(), hi.end(), p) - hi.begin()); }
    int64_t lo(int r) const { return r == 0 ? 0 : hi[(size_t)r - 1]; }
};

// the column slots of a record: 36 edges, then 10 cells (sc_tables.hpp)
constexpr int kEdgeSlots = SID_T0;              // 36
constexpr int kCellSlots = SID_PAD - SID_T0;    // 10

}  // namespace

std::string build_partition(const ScTables& sc, int64_t nc, int64_t ne, int64_t nv, int n_parts, int part,
                            ScTables& local_sc, PartTables& pt) {
    const int64_t P = sc.n_patches;
    if (n_parts < 1 || part < 0 || part >= n_parts) return "partition: need 0 <= part < n_parts";
    if (P * 4 != nc) return "partition: the patch records do not cover the cells";
    if (n_parts > P) return "partition: more parts than parent triangles";
    const Ranges rg(P, n_parts);

    // ---- owner patch of every point ---------------------------------------------------------------------------------
    std::vector<int32_t> own_e((size_t)ne, -1), own_v((size_t)nv, -1);
    for (int64_t p = 0; p < P; ++p) {
        const int32_t* id = &sc.ids[(size_t)p * kScIdWords];
        for (int x = 0; x < 4; ++x)
            if (id[SID_T0 + x] / 4 != p) return "partition: the grid is not in the hierarchical numbering (children of parent p must be 4p .. 4p+3)";
        for (int x = 0; x < 6; ++x) {
            const int32_t e = x < 3 ? id[SID_I0 + x] : id[SID_B0 + 2 * (x - 3)];
            if (e < 0 || e >= ne || own_e[(size_t)e] != -1) return "partition: an edge has no owner or two";
            own_e[(size_t)e] = (int32_t)p;
        }
        for (int x = 0; x < 6; ++x) {
            const int32_t v = id[SID_V0 + x];
            if (v < 0) continue;
            if (v >= nv || own_v[(size_t)v] != -1) return "partition: a vertex has two owners";
            own_v[(size_t)v] = (int32_t)p;
        }
    }
    for (int64_t e = 0; e < ne; ++e)
        if (own_e[(size_t)e] < 0) return "partition: an edge has no owner";
    for (int64_t v = 0; v < nv; ++v)
        if (own_v[(size_t)v] < 0) return "partition: a vertex has no owner";

    pt = PartTables();
    pt.n_parts = n_parts;
    pt.part = part;
    pt.patch_lo = rg.lo(part);
    pt.patch_hi = rg.hi[(size_t)part];
    pt.nc_global = nc; pt.ne_global = ne; pt.nv_global = nv;

    // ---- local numbering: owned first (ascending global id), halo grouped by owner rank -----------------------------
    std::vector<int32_t> g2l_e((size_t)ne, -1), g2l_c((size_t)nc, -1), g2l_v((size_t)nv, -1);
    for (int64_t e = 0; e < ne; ++e)
        if (rg.rank_of(own_e[(size_t)e]) == part) { g2l_e[(size_t)e] = (int32_t)pt.l2g_e.size(); pt.l2g_e.push_back((int32_t)e); }
    for (int64_t c = 4 * pt.patch_lo; c < 4 * pt.patch_hi; ++c) { g2l_c[(size_t)c] = (int32_t)pt.l2g_c.size(); pt.l2g_c.push_back((int32_t)c); }
    for (int64_t v = 0; v < nv; ++v)
        if (rg.rank_of(own_v[(size_t)v]) == part) { g2l_v[(size_t)v] = (int32_t)pt.l2g_v.size(); pt.l2g_v.push_back((int32_t)v); }
    pt.ne_owned = (int64_t)pt.l2g_e.size();
    pt.nc_owned = (int64_t)pt.l2g_c.size();
    pt.nv_owned = (int64_t)pt.l2g_v.size();

    // the columns a range of patches reads and another rank owns: (owner rank, global id), sorted, unique
    auto halo_of = [&](int r, int kind, int only_owner, std::vector<std::pair<int32_t, int32_t>>& out) {
        out.clear();
        for (int64_t p = rg.lo(r); p < rg.hi[(size_t)r]; ++p) {
            const int32_t* id = &sc.ids[(size_t)p * kScIdWords] + (kind == 0 ? 0 : SID_T0);
            const int n = kind == 0 ? kEdgeSlots : kCellSlots;
            for (int i = 0; i < n; ++i) {
                const int32_t x = id[i];
                const int o = rg.rank_of(kind == 0 ? own_e[(size_t)x] : x / 4);
                if (o == r || (only_owner >= 0 && o != only_owner)) continue;
                out.emplace_back((int32_t)o, x);
            }
        }
        std::sort(out.begin(), out.end());
        out.erase(std::unique(out.begin(), out.end()), out.end());
    };

    std::vector<std::pair<int32_t, int32_t>> h;
    for (int kind = 0; kind < 2; ++kind) {
        halo_of(part, kind, -1, h);
        std::vector<int32_t>& l2g = kind == 0 ? pt.l2g_e : pt.l2g_c;
        std::vector<int32_t>& g2l = kind == 0 ? g2l_e : g2l_c;
        std::vector<int64_t>& rb = pt.recv_begin[kind];
        rb.assign((size_t)n_parts + 1, 0);
        size_t at = 0;
        for (int q = 0; q < n_parts; ++q) {
            rb[(size_t)q] = (int64_t)l2g.size();
            while (at < h.size() && h[at].first == q) {
                g2l[(size_t)h[at].second] = (int32_t)l2g.size();
                l2g.push_back(h[at].second);
                ++at;
            }
        }
        rb[(size_t)n_parts] = (int64_t)l2g.size();
    }
    pt.ne_local = (int64_t)pt.l2g_e.size();
    pt.nc_local = (int64_t)pt.l2g_c.size();

    // ---- what every other rank reads of mine, in ITS halo order (ascending global id) -------------------------------
    for (int kind = 0; kind < 2; ++kind) {
        const std::vector<int32_t>& g2l = kind == 0 ? g2l_e : g2l_c;
        pt.send_begin[kind].assign((size_t)n_parts + 1, 0);
        for (int q = 0; q < n_parts; ++q) {
            pt.send_begin[kind][(size_t)q] = (int64_t)pt.send_ids[kind].size();
            if (q == part) continue;
            halo_of(q, kind, part, h);
            for (const auto& x : h) pt.send_ids[kind].push_back(g2l[(size_t)x.second]);
        }
        pt.send_begin[kind][(size_t)n_parts] = (int64_t)pt.send_ids[kind].size();
    }

    // ---- local records ----------------------------------------------------------------------------------------------
    local_sc = ScTables();
    local_sc.n_patches = pt.patch_hi - pt.patch_lo;
    local_sc.ids.assign(sc.ids.begin() + (size_t)pt.patch_lo * kScIdWords, sc.ids.begin() + (size_t)pt.patch_hi * kScIdWords);
    local_sc.coef.assign(sc.coef.begin() + (size_t)pt.patch_lo * kScCoefWords, sc.coef.begin() + (size_t)pt.patch_hi * kScCoefWords);
    for (int64_t p = 0; p < local_sc.n_patches; ++p) {
        int32_t* id = &local_sc.ids[(size_t)p * kScIdWords];
        for (int i = 0; i < kEdgeSlots; ++i) {
            id[i] = g2l_e[(size_t)id[i]];
            if (id[i] < 0) return "partition: internal error, an edge column has no local id";
        }
        for (int i = 0; i < kCellSlots; ++i) {
            id[SID_T0 + i] = g2l_c[(size_t)id[SID_T0 + i]];
            if (id[SID_T0 + i] < 0) return "partition: internal error, a cell column has no local id";
        }
        for (int i = 0; i < 6; ++i) {
            int32_t& v = id[SID_V0 + i];
            if (v >= 0) v = g2l_v[(size_t)v];
        }
        for (int x = 0; x < 6; ++x) {       // every output row is an owned row
            const int32_t e = x < 3 ? id[SID_I0 + x] : id[SID_B0 + 2 * (x - 3)];
            if (e >= pt.ne_owned) return "partition: internal error, an output edge is not owned";
        }
    }
    return std::string();
}

}  // namespace icon
