// host_grid.hpp -- host-side R2Bk grid, connectivity and coefficient tables of the library.
// Internal header of libicon_dycore (never shared with oracle/).
#pragma once
#include <cstdint>
#include <string>
#include <vector>

namespace icon {

struct HostGrid {
    int level_k = 0;
    int64_t nc = 0, ne = 0, nv = 0;
    bool permuted = false;
    // public tables, rows and entries in USER ids
    std::vector<int32_t> c2v, c2e, e2c, e2v, e2e4, v2e, v2c, v_deg;
    std::vector<int8_t> c_os, v_os;
    // geometry / coefficients (G2)
    std::vector<double> vert_xyz, cell_xyz, edge_xyz, edge_normal;
    std::vector<double> l_e, d_e, inv_d_e, f_e, c_lin, rbf, a_c, bln, a_v, geofac_div, geofac_rot, adv_c, cgrad;
    // generation (hierarchical, spatially local) order: user id of the entity at canonical
    // position p. Empty when the user numbering IS the canonical one.
    std::vector<int32_t> user_of_pos_c, user_of_pos_e, user_of_pos_v;
};

// Builds everything above. Returns an empty string on success, else an error message.
std::string build_host_grid(int k, uint64_t seed, bool permute, HostGrid& g);

}  // namespace icon
