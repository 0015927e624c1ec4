// patch_tables.hpp -- work-list of the fused tendency kernel (internal header of libicon_dycore).
//
// The R2Bk grid is a recursive bisection (reading P-2), so four sibling cells
// 4p..4p+3 of the generation order always form one PATCH with a fixed local topology:
//
//                    c                 parent (a,b,c), midpoints ab, bc, ca
//                   / \                T0=(a,ab,ca) T1=(ab,b,bc) T2=(ca,bc,c) T3=(ab,bc,ca)
//                 b4   b3              interior edges  i0=(ab,ca) i1=(ab,bc) i2=(bc,ca)
//                 / T2  \              boundary edges  b0=(a,ab) b1=(ab,b) b2=(b,bc) b3=(bc,c)
//               ca--i2---bc                            b4=(c,ca) b5=(ca,a)
//               / \ T3  / \            outer cell Xj lies across bj; its two other edges are
//             b5  i0   i1  b2          omj (touches the midpoint end of bj) and ocj (touches the
//             / T0  \ /  T1 \          corner end of bj)
//            a--b0---ab--b1--b
//
// One warp evaluates one patch with every one of these 21 edge columns in registers; the tables
// below give the warp the USER ids of the 21 edges / 4 cells and the coefficients re-ordered to
// the fixed local slots, so the kernel's dataflow is compile-time while the ids stay arbitrary
// (seeded permutation included: the tile walk is the locality work-list of SURVEY.md 8(a) G3).
// Sixteen consecutive patches (64 cells = one triangle three levels up) form a TILE = one CTA.
#pragma once
#include <cstdint>
#include <string>
#include <vector>

#include "host_grid.hpp"

namespace icon {

constexpr int kPatchesPerTile = 16;
constexpr int kPatchIdWords = 32;     // int32 per patch record
constexpr int kPatchCoefWords = 96;   // floating-point words per patch record (90 used)
constexpr int kHaloIdWords = 12;      // 3 own edges, 3x2 far edges, cell id, 2 pad
constexpr int kHaloCoefWords = 16;    // 3x4 rbf, 3 bln, 1 pad
constexpr int kVertIdWords = 8;       // 6 fan edges, 2 pad
constexpr int kVertCoefWords = 8;     // 6 geofac_rot, 2 pad

// slots of the patch id record
enum {
    PID_I0 = 0,      // i0 i1 i2
    PID_B0 = 3,      // b0..b5
    PID_OM0 = 9,     // om0..om5
    PID_OC0 = 15,    // oc0..oc5
    PID_T0 = 21,     // T0..T3 cell ids
    PID_XSLOT = 25,  // exchange slots of the outer cells X0, X2, X4 (owned boundary edges b0, b2, b4)
    PID_VSLOT = 28,  // exchange slots of the corner vertices a, b, c
    PID_PAD = 31
};
// slots of the patch coefficient record
enum {
    PCF_RBF = 0,     // [9][4] order i0 i1 i2 b0..b5, neighbour order documented in patch_tables.cpp
    PCF_BLN = 36,    // [4][3] T0..T3, slot order of c2e
    PCF_ROT = 48,    // [3][6] midpoints ab, bc, ca
    PCF_EDGE = 66,   // [6][4] owned edges i0 i1 i2 b0 b2 b4: s_inv_d, f_e, c_lin(L), c_lin(H)
    PCF_USED = 90
};

struct PatchTables {
    int64_t n_patches = 0, n_tiles = 0;
    int max_halo = 0, max_vert = 0;          // largest per-tile task counts (sizes the exchange buffers)
    std::vector<int32_t> patch_ids;          // [n_patches][kPatchIdWords]
    std::vector<double> patch_coef;          // [n_patches][kPatchCoefWords]
    std::vector<int32_t> tile_hdr;           // [n_tiles][4]: halo_off, n_halo, vert_off, n_vert
    std::vector<int32_t> halo_ids;           // [n_halo_total][kHaloIdWords]
    std::vector<double> halo_coef;           // [n_halo_total][kHaloCoefWords]
    std::vector<int32_t> vert_ids;           // [n_vert_total][kVertIdWords]
    std::vector<double> vert_coef;           // [n_vert_total][kVertCoefWords]
    // div/vort ownership: which tile task stores which vertex (every vertex exactly once)
    std::vector<int32_t> vert_store;         // [n_vert_total] 1 = this tile stores the corner vertex
    std::vector<int32_t> mid_store;          // [n_patches] bit j = this patch stores midpoint j (ab, bc, ca)
    std::vector<int32_t> mid_vertex;         // [n_patches][4] user ids of ab, bc, ca (+pad)
};

// Derives the tables from the public connectivity of `g` and checks the local topology of every
// patch while doing so. Returns an empty string on success, else an error message.
std::string build_patch_tables(const HostGrid& g, PatchTables& t);

}  // namespace icon
