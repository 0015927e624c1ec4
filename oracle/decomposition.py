"""ORACLE -- test infrastructure, not the product.

Horizontal domain decomposition of the sweep (reading P-21 in DESIGN.md section 3).

The paper says only that the model exchanges halos point to point between neighbouring subdomains of the horizontal
grid and that it scales down to about 10,800 cells per GPU; it prints no rule for
the subdomains. Reading P-21: the subdomain of rank r of R is a contiguous range of PARENT triangles of the
hierarchical numbering (the four children of parent q are the cells 4q .. 4q+3), parents floor(r P / R) <= q <
floor((r+1) P / R) with P = Nc / 4. What a rank must hold besides what it owns follows from the definitions S1-S7
 alone: the columns the outputs at its owned points read. This file states exactly that, in sets
of ids, straight from the connectivity tables: no blocking, no patch records, no tables of the library.

Which rank owns an edge shared by two subdomains, or a vertex shared by several, is a free choice; what is fixed is
that every point has exactly one owner and that the owner owns a cell adjacent to it (`check_ownership`).

Pins (tests/test_oracle_pins.py): the read sets against a brute-force perturbation of the oracle's own operator on
R2B1 (every column is perturbed in turn; the outputs that change are the ones that read it), the 15 distinct edges of
the `ddt_vn` stencil SURVEY.md 8(e) states, and the closed forms of the ranges.
"""
import numpy as np


def part_range(n_parents, n_parts, r):
    """P-21: parents [lo, hi) of rank r"""
    return (r * n_parents) // n_parts, ((r + 1) * n_parents) // n_parts


def cell_owner(nc, n_parts):
    """rank that owns each cell, [nc] int32"""
    n_parents = nc // 4
    bounds = np.array([part_range(n_parents, n_parts, r)[1] for r in range(n_parts)], dtype=np.int64)
    parent = np.arange(nc, dtype=np.int64) // 4
    return np.searchsorted(bounds, parent, side="right").astype(np.int32)


# ---- what one output point reads (S1-S7 written out as sets) --------------------------------------------------------
def vt_reads(t, e):
    """S3: vt(e) reads vn at the four edges e2e4[e]"""
    return {int(x) for x in t.e2e4[e]}


def ke_e_reads(t, e):
    """S4: KE_e(e) = (vn(e)^2 + vt(e)^2) / 2"""
    return {int(e)} | vt_reads(t, e)


def ke_c_reads(t, c):
    """S4: KE_c(c) = sum_j bln(c, j) KE_e(c2e[c][j])"""
    s = set()
    for e in t.c2e[c]:
        s |= ke_e_reads(t, e)
    return s


def vort_reads(t, v):
    """S2: zeta(v) reads vn at the v_deg[v] fan edges (the pentagon's pad entry carries coefficient 0: not a read)"""
    return {int(t.v2e[v][j]) for j in range(int(t.v_deg[v]))}


def div_reads(t, c):
    """S1"""
    return {int(x) for x in t.c2e[c]}


def ddt_vn_reads(t, e):
    """S5-S7: (vn edges, w cells) that ddt_vn(e, :) reads"""
    s = {int(e)} | vt_reads(t, e)                  # vn(e) (vertical term, KE gradient correction), vt(e)
    for c in t.e2c[e]:
        s |= ke_c_reads(t, c)                      # KE_c of both cells
    for v in t.e2v[e]:
        s |= vort_reads(t, v)                      # zeta at both vertices
    return s, {int(c) for c in t.e2c[e]}


def required_columns(t, owned_edges, owned_cells, owned_verts):
    """(sorted vn edge ids, sorted w cell ids) that dycore_step reads to produce ddt_vn at `owned_edges`, div at
    `owned_cells` and zeta at `owned_verts`"""
    edges, cells = set(), set()
    for e in owned_edges:
        a, b = ddt_vn_reads(t, e)
        edges |= a
        cells |= b
    for c in owned_cells:
        edges |= div_reads(t, c)
    for v in owned_verts:
        edges |= vort_reads(t, v)
    return np.array(sorted(edges), dtype=np.int64), np.array(sorted(cells), dtype=np.int64)


def check_ownership(t, n_parts, edge_owner, vert_owner):
    """the free choices of a decomposition are valid: every edge (vertex) has one owner, and that owner owns a cell
    adjacent to it. Returns a list of violations (empty = valid)."""
    co = cell_owner(t.nc, n_parts)
    bad = []
    edge_owner = np.asarray(edge_owner)
    vert_owner = np.asarray(vert_owner)
    if edge_owner.shape != (t.ne,) or vert_owner.shape != (t.nv,):
        return ["shape"]
    ok_e = (edge_owner == co[t.e2c[:, 0]]) | (edge_owner == co[t.e2c[:, 1]])
    bad += ["edge %d" % e for e in np.nonzero(~ok_e)[0][:5]]
    for v in range(t.nv):
        owners = {int(co[t.v2c[v][j]]) for j in range(int(t.v_deg[v]))}
        if int(vert_owner[v]) not in owners:
            bad.append("vertex %d" % v)
            if len(bad) > 10:
                break
    return bad
