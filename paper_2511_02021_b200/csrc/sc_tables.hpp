// sc_tables.hpp -- patch records, the work-list of the column-cache kernel (kernels_cc.cu) and of the
// self-contained patch kernel (kernels_sc.cu); internal header.
//
// The grid is a recursive bisection, so the four sibling cells T0..T3 of the generation order always form one
// PATCH with a fixed local topology: interior edges i0..i2, boundary edges b0..b5, outer cells X0..X5 with
// their edges om_j / oc_j. A patch record carries everything its six owned edges (i0 i1 i2 b0 b2 b4) need, so one
// warp finishes a patch without exchanging anything with other warps:
//
//   for each owned boundary edge b_j (j = 0, 2, 4; x = j/2) with outer cell X_j and corner vertex
//   C_x (a, b, c):
//     pm0, pm1   the two other edges of the cell across om_j     -> vt(om_j)
//     n1, pcf    the two other edges of the cell Z1 across oc_j  -> vt(oc_j); n1 touches C_x
//     n2         the next fan edge of C_x after n1 (hexagon); pentagon: n2 = n1, coefficient 0
//   so KE_c(X_j) = bln . (KE_e(b_j), KE_e(om_j), KE_e(oc_j)) and
//   zeta(C_x)   = rot . (b_j, oc_j, n1, n2, oc_jp, b_jp), jp = (j+5) mod 6, are local.
//
// The same columns also give div of the four cells and zeta at the three midpoints and three corners,
// so a record also carries geofac_div and the vertices the patch owns (every vertex of the grid is
// a midpoint or a corner of some patch; the lowest patch index owns it) -- dycore_step.
// 36 edge columns and 7 cell columns per patch; coefficients re-ordered to these fixed slots
// with the factors 1/2 of KE_e = (vn^2+vt^2)/2 and zeta_e = (zeta(v0)+zeta(v1))/2 folded in
// (exact: scaling by a power of two commutes with every rounding).
#pragma once
#include <cstdint>
#include <string>
#include <vector>

#include "host_grid.hpp"

namespace icon {

constexpr int kScIdWords = 56;      // int32 per patch: 36 edges, 10 cells, 2 pad, 6 vertices, 2 pad (224 B)
constexpr int kScCoefWords = 196;   // floating-point words per patch; every group starts on a multiple of 4 words

enum {                // id slots
    SID_I0 = 0,       // i0 i1 i2
    SID_B0 = 3,       // b0..b5
    SID_OM0 = 9,      // om0..om5
    SID_OC0 = 15,     // oc0..oc5
    SID_X0 = 21,      // [3][5]: pm0 pm1 pcf n1 n2 of owned boundary edges b0, b2, b4
    SID_T0 = 36,      // T0..T3
    SID_XC0 = 40,     // X0 X2 X4
    SID_XW0 = 43,     // X1 X3 X5: the other three outer cells, read by the vertical-wind tendency only
    SID_PAD = 46,     // number of column slots: 36 vn (edges) then 10 w (cells)
    SID_V0 = 48       // vertices ab bc ca a b c whose vorticity THIS patch stores (fused step), -1 = another patch does
};
enum {                // coefficient slots
    SCF_RBF = 0,      // [9][4] i0 i1 i2 b0..b5, fixed neighbour order, see build_sc_tables
    SCF_BLN = 36,     // [4][3] T0..T3 (x 1/2)
    SCF_ROT = 48,     // [3][6] midpoints ab bc ca (x 1/2)
    SCF_EDGE = 68,    // [6][4] owned i0 i1 i2 b0 b2 b4: s_inv_d, f_e, c_lin(L), c_lin(H)
    SCF_XRM = 92,     // [3][4] rbf of om_j over (b_j, oc_j, pm0, pm1)
    SCF_XRO = 104,   // [3][4] rbf of oc_j over (b_j, om_j, n1, pcf)
    SCF_XBL = 116,    // [3][3] bln of X_j over (b_j, om_j, oc_j) (x 1/2)
    SCF_XROT = 128,   // [3][6] rot of C_x over (b_j, oc_j, n1, n2, oc_jp, b_jp) (x 1/2)
    SCF_USED = 146,
    SCF_DIV = 148,    // [4][3] geofac_div of T0..T3 over the cell edges in the order of SCF_BLN
    SCF_ADV = 160,    // [4][3] +-adv_c * inv_d_e of T0..T3 over the same edges (P-19); sign such that the term is
                      //        coefficient * vn_ie * (w(cell across the edge) - w(this cell))
    SCF_CGRAD = 172   // [6][4] owned i0 i1 i2 b0 b2 b4 (P-20): gL, gH, gE, pad with
                      //        gradK = gH KE_c(H) - gL KE_c(L) + gE (vn^2 + vt^2), gE = (gL - gH) / 2
};

struct ScTables {
    int64_t n_patches = 0;
    std::vector<int32_t> ids;     // [n_patches][kScIdWords]
    std::vector<double> coef;     // [n_patches][kScCoefWords]
};

// Derives the records from the public connectivity of `g`, checking the local topology of every
// patch. Returns an empty string on success, else an error message.
std::string build_sc_tables(const HostGrid& g, ScTables& t);

}  // namespace icon
