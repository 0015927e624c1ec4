// partition.hpp -- horizontal domain decomposition of the sweep (reading P-21 in
// DESIGN.md): the LOCAL patch records of one rank, its local numbering and its halo lists. Internal header.
//
// Rank r of R owns the patches (parent triangles of the hierarchical numbering) floor(r P / R) <= p < floor((r+1) P / R).
// A point (edge, cell, vertex) is owned by the rank of the patch that STORES it in the fused step (sc_tables.hpp: the
// six owned edges, the four cells, the vertices of SID_V0 >= 0), so every output of the grid has exactly one owner.
// Local numbering of a rank, for edges and for cells alike:
//     [0, n_owned)            the owned points, ascending global id (the locality of the hierarchical numbering,
//                             and with it the run merging of the column-cache schedule, is kept)
//     [n_owned, n_local)      the halo = the columns the rank's patches read and do not own, grouped by owner rank
//                             ascending, ascending global id within a group
// so the halo columns one peer sends are ONE contiguous block of rows of the local field: a receive lands in place,
// nothing is unpacked. The sender gathers the rows of `send_ids` (its local ids, in the receiver's order) into a
// contiguous buffer (k_halo_pack). Vertices carry outputs only: the local vertices are the owned ones.
#pragma once
#include <cstdint>
#include <string>
#include <vector>

#include "sc_tables.hpp"

namespace icon {

struct PartTables {
    int n_parts = 0;                    // 0: the grid is not a partition
    int part = -1;
    int64_t patch_lo = 0, patch_hi = 0;
    int64_t nc_global = 0, ne_global = 0, nv_global = 0;
    int64_t nc_owned = 0, ne_owned = 0, nv_owned = 0;
    int64_t nc_local = 0, ne_local = 0;                 // owned + halo
    std::vector<int32_t> l2g_c, l2g_e, l2g_v;           // local id -> global id
    // kind 0 = edges (vn), kind 1 = cells (w); [n_parts + 1] each
    std::vector<int64_t> recv_begin[2];                 // rows [recv_begin[q], recv_begin[q+1]) of the local field come from rank q
    std::vector<int64_t> send_begin[2];                 // send_ids[send_begin[q] .. send_begin[q+1]) go to rank q
    std::vector<int32_t> send_ids[2];                   // local ids of owned rows, the receiver's order
};

// Derives the local records of `part` (ids in the LOCAL numbering, coefficients copied) and the tables above from the
// GLOBAL patch records of an unpermuted grid. Returns an empty string on success, else an error message.
std::string build_partition(const ScTables& global_sc, int64_t nc, int64_t ne, int64_t nv, int n_parts, int part,
                            ScTables& local_sc, PartTables& pt);

}  // namespace icon
