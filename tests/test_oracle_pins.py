"""Pins for the oracle (CPU only): what the paper and the mathematics fix, independent of the
oracle's own formulas. SURVEY.md section 8(c) table "What pins the oracle"; DESIGN.md section 5.

A plausible mistake anywhere in oracle/icon_oracle.c (dropped term, wrong sign or index,
transposed operand, wrong tangent orientation) fails at least one test here."""
import numpy as np
import pytest

import seeded_inputs as si
from conftest import read_golden

A = 6.371e6
OMEGA = 7.29212e-5


# ----------------------------------------------------------------------------------------------
# counts, structure
# ----------------------------------------------------------------------------------------------
@pytest.mark.parametrize("k", [0, 1, 2, 3, 4, 5])
def test_counts_and_structure(oracle_grid, k):
    g = oracle_grid(k)
    nc = 20 * 4 ** (k + 1)                       # north_star: cells = 20*4^(k+1)
    assert (g.nc, g.ne, g.nv) == (nc, 3 * nc // 2, nc // 2 + 2)
    deg = g.v_deg
    assert (deg == 5).sum() == 12 and (deg == 6).sum() == g.nv - 12     # exactly 12 pentagons
    assert (g.e2c[:, 0] != g.e2c[:, 1]).all()
    assert (g.e2c[:, 0] < g.e2c[:, 1]).all()     # canonical numbering: first touch is the lower cell
    e = np.arange(g.ne)[:, None]
    assert (g.e2e4 != e).all()
    # every edge appears in exactly two c2e rows, once with each sign
    cnt = np.bincount(g.c2e.ravel(), minlength=g.ne)
    assert (cnt == 2).all()
    sgn = np.zeros(g.ne, dtype=np.int64)
    np.add.at(sgn, g.c2e.ravel(), g.c_os.ravel().astype(np.int64))
    assert (sgn == 0).all()
    # every edge appears in exactly two fans, with opposite signs
    real = g.v_os != 0
    cntv = np.bincount(g.v2e[real], minlength=g.ne)
    assert (cntv == 2).all()
    sgv = np.zeros(g.ne, dtype=np.int64)
    np.add.at(sgv, g.v2e[real], g.v_os[real].astype(np.int64))
    assert (sgv == 0).all()
    # pentagon pads repeat slot 0
    pent = deg == 5
    assert (g.v2e[pent, 5] == g.v2e[pent, 0]).all() and (g.v_os[pent, 5] == 0).all()
    assert (g.geofac_rot[pent, 5] == 0).all()


def test_table_checksums(oracle_grid):
    for row in read_golden("table_checksums.txt"):
        k = int(row[0])
        g = oracle_grid(k)
        got = [int(g.table(n).astype(np.int64).sum()) for n in ("c2e", "e2c", "e2v", "e2e4", "v2e")]
        assert got == [int(x) for x in row[1:]], "R2B%d" % k


def test_r2b0_table_rows(oracle_grid):
    g = oracle_grid(0)
    for row in read_golden("r2b0_tables.txt"):
        name, first = row[0], int(row[1])
        vals = np.array([int(x) for x in row[3:]])
        tab = g.table(name)
        cols = tab.shape[1]
        got = tab[first:first + vals.size // cols].ravel()
        assert (got == vals).all(), name


def test_r2b0_geometry_values(oracle_grid):
    g = oracle_grid(0)
    # closed forms for the icosahedron's first bisection
    assert abs(0.5 * np.arccos(1 / np.sqrt(5)) - 0.553574358897) < 1e-12
    assert abs(np.pi / 5 - 0.628318530718) < 1e-12
    scale = {"l_e": A, "d_e": A, "a_c": A * A, "a_v": A * A}
    want = {}
    for name, val, mult in read_golden("r2b0_geometry.txt"):
        want.setdefault(name, []).append((float(val), int(mult)))
    for name, items in want.items():
        x = g.table(name) / scale[name]
        vals = np.array([v for v, _ in items])
        nearest = np.abs(x[:, None] - vals[None, :]).argmin(1)
        assert np.abs(x - vals[nearest]).max() < 1e-12, name
        for j, (_, mult) in enumerate(items):
            assert (nearest == j).sum() > 0
            if mult > 0:
                assert (nearest == j).sum() == mult, (name, j)


# ----------------------------------------------------------------------------------------------
# brute force: an independent dict-based construction of P-1..P-6 in pure Python
# ----------------------------------------------------------------------------------------------
def _brute_topology(k):
    lat = np.arctan(0.5)
    P = [(0.0, 0.0, 1.0)]
    for i in range(5):
        lon = np.deg2rad(72.0 * i)
        P.append((np.cos(lat) * np.cos(lon), np.cos(lat) * np.sin(lon), np.sin(lat)))
    for i in range(5):
        lon = np.deg2rad(36.0 + 72.0 * i)
        P.append((np.cos(lat) * np.cos(lon), np.cos(lat) * np.sin(lon), -np.sin(lat)))
    P.append((0.0, 0.0, -1.0))
    P = [np.array(p) for p in P]
    cells = []
    for i in range(5):
        j = (i + 1) % 5
        cells += [(0, 1 + i, 1 + j), (1 + i, 6 + i, 1 + j), (6 + i, 6 + j, 1 + j), (11, 6 + j, 6 + i)]
    for _ in range(k + 1):
        mid = {}

        def m(a, b):
            key = (min(a, b), max(a, b))
            if key not in mid:
                p = P[a] + P[b]
                P.append(p / np.sqrt((p * p).sum()))
                mid[key] = len(P) - 1
            return mid[key]
        new = []
        for (a, b, c) in cells:
            ab, bc, ca = m(a, b), m(b, c), m(c, a)
            new += [(a, ab, ca), (ab, b, bc), (ca, bc, c), (ab, bc, ca)]
        cells = new
    vid, c2v = {}, []
    for cell in cells:
        row = []
        for v in cell:
            if v not in vid:
                vid[v] = len(vid)
            row.append(vid[v])
        c2v.append(row)
    xyz = np.zeros((len(vid), 3))
    for old, new in vid.items():
        xyz[new] = P[old]
    eid, e2v, e2c, c2e = {}, [], [], []
    for c, (a, b, d) in enumerate(c2v):
        row = []
        for (p, q) in ((a, b), (b, d), (d, a)):
            key = (min(p, q), max(p, q))
            if key not in eid:
                eid[key] = len(eid)
                e2v.append([p, q])
                e2c.append([c, -1])
            else:
                e2c[eid[key]][1] = c
            row.append(eid[key])
        c2e.append(row)
    e2e4 = []
    for e, (c0, c1) in enumerate(e2c):
        row = []
        for c in (c0, c1):
            j = c2e[c].index(e)
            row += [c2e[c][(j + 1) % 3], c2e[c][(j + 2) % 3]]
        e2e4.append(row)
    return np.array(c2v), np.array(c2e), np.array(e2c), np.array(e2v), np.array(e2e4), xyz


@pytest.mark.parametrize("k", [0, 1, 2])
def test_brute_force_topology(oracle_grid, k):
    g = oracle_grid(k)
    c2v, c2e, e2c, e2v, e2e4, xyz = _brute_topology(k)
    assert (g.c2v == c2v).all() and (g.c2e == c2e).all() and (g.e2c == e2c).all()
    assert (g.e2v == e2v).all() and (g.e2e4 == e2e4).all()
    assert np.abs(g.vert_xyz - xyz).max() < 1e-15
    # fans: CCW order means consecutive fan edges bound the listed cell, and the geometric angle
    # of the fan edges around the vertex increases counter-clockwise seen from outside
    for v in range(g.nv):
        d = g.v_deg[v]
        p = g.vert_xyz[v]
        for i in range(d):
            ea, eb, c = g.v2e[v, i], g.v2e[v, (i + 1) % d], g.v2c[v, i]
            assert ea in g.c2e[c] and eb in g.c2e[c] and v in g.c2v[c]
            xa, xb = g.edge_xyz[ea] - p, g.edge_xyz[eb] - p
            assert np.dot(np.cross(xa, xb), p) > 0            # CCW about the outward normal
        assert len(set(g.v2e[v, :d])) == d


def test_orientation_conventions(oracle_grid):
    """P-4: n_e points from e2c[e][0] to e2c[e][1]; t_e = n_e x x_e = -tau_e."""
    g = oracle_grid(3)
    dc = g.cell_xyz[g.e2c[:, 1]] - g.cell_xyz[g.e2c[:, 0]]
    assert ((dc * g.edge_normal).sum(1) > 0).all()
    tau = g.vert_xyz[g.e2v[:, 1]] - g.vert_xyz[g.e2v[:, 0]]
    tau /= np.linalg.norm(tau, axis=1)[:, None]
    t = np.cross(g.edge_normal, g.edge_xyz)
    assert np.abs(t + tau).max() < 1e-14
    assert np.abs(np.linalg.norm(g.edge_normal, axis=1) - 1).max() < 1e-14
    assert np.abs((g.edge_normal * g.edge_xyz).sum(1)).max() < 1e-14
    # cell centres are circumcentres: equidistant from the three vertices
    d = np.stack([np.linalg.norm(g.cell_xyz - g.vert_xyz[g.c2v[:, j]], axis=1) for j in range(3)], 1)
    assert np.abs(d - d[:, :1]).max() < 1e-14
    # C-grid orthogonality: the dual arc passes through the edge midpoint
    lin = g.c_lin.sum(1)
    assert np.abs(lin - 1).max() < 1e-12
    assert (g.c_lin > 0).all()
    assert np.abs(g.inv_d_e * g.d_e - 1).max() < 1e-15
    assert np.abs(g.f_e - 2 * OMEGA * g.edge_xyz[:, 2]).max() == 0


# ----------------------------------------------------------------------------------------------
# invariants of the discretisation
# ----------------------------------------------------------------------------------------------
@pytest.mark.parametrize("k", [0, 1, 2, 3, 4])
def test_area_closure(oracle_grid, k):
    g = oracle_grid(k)
    assert abs(g.a_c.sum() / (4 * np.pi * A * A) - 1) < 1e-15 * (1 + k) * 4
    assert abs(g.a_v.sum() / (4 * np.pi * A * A) - 1) < 1e-15 * (1 + k) * 4


@pytest.mark.parametrize("k,flags", [(0, 0), (2, 0), (4, 0), (3, 1)])
def test_discrete_gauss(oracle_grid, k, flags):
    """sum_c A_c div_c = 0 on the closed sphere, to round-off, for random vn"""
    g = oracle_grid(k, 7, flags)
    rng = np.random.default_rng(11)
    vn = rng.standard_normal((g.ne, 3))
    div, _ = g.div_vort(vn, 3)
    num = np.abs((g.a_c[:, None] * div).sum(0))
    den = (np.abs(vn) * g.l_e[:, None]).sum(0)
    assert (num / den).max() < 1e-16


@pytest.mark.parametrize("k,flags", [(0, 0), (2, 0), (4, 0), (3, 1)])
def test_curl_of_gradient_vanishes(oracle_grid, k, flags):
    """rot(grad_n psi) = 0 (mimetic identity); pins v_os against the e2c order"""
    g = oracle_grid(k, 7, flags)
    rng = np.random.default_rng(12)
    psi = rng.standard_normal((g.nc, 2))
    gradn = (psi[g.e2c[:, 1]] - psi[g.e2c[:, 0]]) * g.inv_d_e[:, None]
    _, vort = g.div_vort(gradn, 2)
    h = np.sqrt(g.a_c.mean())
    assert np.abs(vort).max() / (np.abs(gradn).max() / h) < 1e-15
    # and the same identity with a wrong-signed fan entry must be far from zero (the pin bites)
    bad = gradn.copy()
    bad[g.v2e[5, 0]] *= -1
    _, vort_bad = g.div_vort(bad, 2)
    assert np.abs(vort_bad).max() / (np.abs(gradn).max() / h) > 1e-3


@pytest.mark.parametrize("k", [0, 2, 4])
def test_weights(oracle_grid, k):
    g = oracle_grid(k)
    assert np.abs(g.bln.sum(1) - 1).max() < 1e-15 * 4
    assert (g.bln > 0.2).all() and (g.bln < 0.55).all()
    # bln reproduces linear functions in the gnomonic plane of the cell centre: the gnomonic image
    # of the cell centre itself is the origin, so sum_j bln_j * P(x_j) = 0
    cc = g.cell_xyz
    acc = np.zeros_like(cc)
    for j in range(3):
        x = g.edge_xyz[g.c2e[:, j]]
        Pj = x / (x * cc).sum(1)[:, None] - cc
        acc += g.bln[:, j:j + 1] * Pj
    assert np.abs(acc).max() < 1e-15
    # RBF normalisation identity (P-11): a locally uniform flow along t_e is returned exactly
    t = np.cross(g.edge_normal, g.edge_xyz)
    s = np.zeros(g.ne)
    for j in range(4):
        s += g.rbf[:, j] * (g.edge_normal[g.e2e4[:, j]] * t).sum(1)
    assert np.abs(s - 1).max() < 1e-14
    assert np.abs(g.rbf).sum(1).max() < 1.3
    # a uniform flow along n_e has (nearly) no tangential component
    s = np.zeros(g.ne)
    for j in range(4):
        s += g.rbf[:, j] * (g.edge_normal[g.e2e4[:, j]] * g.edge_normal).sum(1)
    assert np.abs(s).max() < 0.2
    # folded factors
    le = g.l_e[g.c2e]
    assert np.abs(g.geofac_div - le * g.c_os / g.a_c[:, None]).max() / np.abs(g.geofac_div).max() < 1e-15
    de = g.d_e[g.v2e]
    assert np.abs(g.geofac_rot - de * g.v_os / g.a_v[:, None]).max() / np.abs(g.geofac_rot).max() < 1e-15


# ----------------------------------------------------------------------------------------------
# solid-body rotation closed forms (first-order convergence values of SURVEY 8(c))
# ----------------------------------------------------------------------------------------------
def _solid_body(g, u0=20.0):
    x, n = g.edge_xyz, g.edge_normal
    vel = np.stack([-x[:, 1], x[:, 0], np.zeros(g.ne)], 1) * u0
    return vel, (vel * n).sum(1)


def _solid_body_errors(g):
    u0 = 20.0
    omp = u0 / A
    vel, vn_sb = _solid_body(g, u0)
    K = 6
    zh = si.z_half_levels(K)
    zf = 0.5 * (zh[:-1] + zh[1:])
    vn = np.repeat(vn_sb[:, None], K, 1)
    div, vort = g.div_vort(vn, K)
    err = {}
    err["zeta"] = np.abs(vort - 2 * omp * g.vert_xyz[:, 2:3]).max() / (2 * omp)
    err["div"] = np.abs(div).max() / omp
    out = g.velocity_tendencies(vn, np.zeros((g.nc, K + 1)), zh, K)
    t = np.cross(g.edge_normal, g.edge_xyz)
    err["vt"] = np.abs(out["vt"] - (vel * t).sum(1)[:, None]).max() / u0
    cos2 = 1 - g.cell_xyz[:, 2] ** 2
    err["ke_c"] = np.abs(out["ke_c"] - 0.5 * u0 * u0 * cos2[:, None]).max() / (0.5 * u0 * u0)
    gam, w0 = 1e-5, 0.1
    prof = 1 + gam * zf
    vn = vn_sb[:, None] * prof[None, :]
    w = np.full((g.nc, K + 1), w0)
    out = g.velocity_tendencies(vn, w, zh, K)
    x = g.edge_xyz
    sinp = x[:, 2]
    cosp = np.sqrt(1 - sinp ** 2)
    north = (np.array([0, 0, 1.0])[None, :] - sinp[:, None] * x) / cosp[:, None]
    nn = (north * g.edge_normal).sum(1)
    exact = -((prof[None, :] ** 2 * (u0 * u0 / A) + prof[None, :] * 2 * OMEGA * u0) * (sinp * cosp * nn)[:, None]) \
        - w0 * gam * vn_sb[:, None]
    err["tendency"] = np.abs(out["ddt_vn"] - exact).max() / np.abs(exact).max()
    out0 = g.velocity_tendencies(vn, np.zeros_like(w), zh, K)
    dv = (out["ddt_vn"] - out0["ddt_vn"]) + w0 * gam * vn_sb[:, None]
    err["vertical"] = np.abs(dv).max() / np.abs(w0 * gam * vn_sb).max()
    return err


def test_solid_body_closed_forms(oracle_grid):
    gold = {r[0]: ([float(x) for x in r[1:6]], float(r[6])) for r in read_golden("solid_body_errors.txt")}
    for k in range(5):
        err = _solid_body_errors(oracle_grid(k))
        for name, (vals, tol) in gold.items():
            assert abs(err[name] / vals[k] - 1) < tol, (name, k, err[name], vals[k])
        # P-14: the vertical term is exact for profiles linear in z
        assert err["vertical"] < 1e-12


def test_vertical_term_exact_for_linear_profiles(oracle_grid):
    """w d(vn)/dz with vn = a + b z at every edge, arbitrary (stretched) levels, incl. both ends"""
    g = oracle_grid(1)
    K = 9
    zh = si.z_half_levels(K)
    zf = 0.5 * (zh[:-1] + zh[1:])
    rng = np.random.default_rng(3)
    b = rng.standard_normal(g.ne) * 1e-3
    vn = 1.0 + b[:, None] * zf[None, :]
    w = rng.standard_normal((g.nc, K + 1))
    o1 = g.velocity_tendencies(vn, w, zh, K)
    o0 = g.velocity_tendencies(vn, np.zeros_like(w), zh, K)
    wf = 0.5 * (w[:, :-1] + w[:, 1:])
    w_e = g.c_lin[:, :1] * wf[g.e2c[:, 0]] + g.c_lin[:, 1:] * wf[g.e2c[:, 1]]
    want = -w_e * b[:, None]
    got = o1["ddt_vn"] - o0["ddt_vn"]
    assert np.abs(got - want).max() / np.abs(want).max() < 1e-11


def _arc(p, q):
    """great-circle distance of unit vectors, atan2(|p x q|, p . q) (reading P-8), numpy"""
    return np.arctan2(np.linalg.norm(np.cross(p, q), axis=1), (p * q).sum(1))


@pytest.mark.parametrize("k,seed,flags", [(0, 0, 0), (2, 0, 0), (4, 0, 0), (3, 4, 1)])
def test_c_lin_slot_order_from_geometry(oracle_grid, k, seed, flags):
    """P-9 pins the SLOT ORDER of c_lin from geometry alone: slot 0 multiplies the value at e2c[e][0] and is
    arc(x_e, c1)/d_e, so that linear interpolation along the dual arc holds: with signed abscissae s0 = -arc(x_e, c0),
    s1 = +arc(x_e, c1) the weights satisfy c_lin0 * s0 + c_lin1 * s1 = 0 and the NEARER cell weighs more. Swapping the
    two assignments in oracle/icon_oracle.c (c_lin[2e] <-> c_lin[2e+1]) fails both assertions on every unoptimised
    grid, where the two distances differ by per cent (checked on a scratch copy of the oracle)."""
    g = oracle_grid(k, seed, flags)
    x, c0, c1 = g.edge_xyz, g.cell_xyz[g.e2c[:, 0]], g.cell_xyz[g.e2c[:, 1]]
    a0, a1 = _arc(x, c0), _arc(x, c1)
    d = g.d_e / A
    assert np.abs(a0 + a1 - d).max() < 1e-14                 # the dual arc passes through x_e (P-8)
    assert np.abs(a0 - a1).max() / d.max() > 1e-3            # the pin has teeth: the distances do differ
    resid = g.c_lin[:, 0] * (-a0) + g.c_lin[:, 1] * a1
    assert np.abs(resid).max() < 1e-15
    differ = np.abs(a0 - a1) > 1e-9 * d
    assert ((g.c_lin[:, 0] > g.c_lin[:, 1]) == (a0 < a1))[differ].all()
    assert np.abs(g.c_lin[:, 0] - a1 / d).max() < 1e-14 and np.abs(g.c_lin[:, 1] - a0 / d).max() < 1e-14


def test_vertical_term_uses_c_lin_slot0_for_cell0(oracle_grid):
    """Operator-level pin of P-9 / S6: vn = a + b z per edge and a NON-uniform w. Expected -w_e b with w_e assembled
    from numpy arc distances (never from g.c_lin): w_e = [arc(x_e,c1) w_f(c0) + arc(x_e,c0) w_f(c1)] / d_e, i.e. the
    value linearly interpolated along the dual arc to the edge midpoint. Swapping the two factors in og_ddt_vn (or the
    two table assignments) gives a relative error of order 1e-2 here (checked on a scratch copy of the oracle)."""
    g = oracle_grid(2)
    K = 7
    zh = si.z_half_levels(K)
    zf = 0.5 * (zh[:-1] + zh[1:])
    rng = np.random.default_rng(11)
    b = (1.0 + rng.random(g.ne)) * 1e-3
    vn = 2.0 + b[:, None] * zf[None, :]
    # w linear in a Cartesian coordinate: the exact interpolant along the (short) dual arc is nearly linear in arc
    # length, and the two cells of an edge get clearly different values
    w = np.repeat((1.0 + 50.0 * g.cell_xyz[:, 0] + 30.0 * g.cell_xyz[:, 2])[:, None], K + 1, axis=1)
    w *= (1.0 + 0.1 * np.arange(K + 1))[None, :]
    x, c0, c1 = g.edge_xyz, g.cell_xyz[g.e2c[:, 0]], g.cell_xyz[g.e2c[:, 1]]
    a0, a1 = _arc(x, c0), _arc(x, c1)
    wf = 0.5 * (w[:, :-1] + w[:, 1:])
    w_e = (a1[:, None] * wf[g.e2c[:, 0]] + a0[:, None] * wf[g.e2c[:, 1]]) / (a0 + a1)[:, None]
    want = -w_e * b[:, None]
    got = g.velocity_tendencies(vn, w, zh, K)["ddt_vn"] - g.velocity_tendencies(vn, np.zeros_like(w), zh, K)["ddt_vn"]
    assert np.abs(got - want).max() / np.abs(want).max() < 1e-11
    # teeth: the swapped association differs from `want` by far more than the tolerance
    w_swapped = (a0[:, None] * wf[g.e2c[:, 0]] + a1[:, None] * wf[g.e2c[:, 1]]) / (a0 + a1)[:, None]
    assert np.abs(w_swapped - w_e).max() / np.abs(w_e).max() > 1e-3


def test_tolerance_scale_is_the_sum_of_absolute_terms(oracle_grid):
    """P-16: M(p) is EXACTLY the sum of the absolute values of the terms entering p -- two-sided, so an inflated
    scale (which would loosen every parity test) fails as surely as a deflated one. Re-assembled with numpy from the
    oracle's intermediate outputs and numpy arc distances."""
    g = oracle_grid(2)
    K = 6
    rng = np.random.default_rng(17)
    vn = rng.standard_normal((g.ne, K)) * 5
    w = rng.standard_normal((g.nc, K + 1))
    zh = si.z_half_levels(K)
    o = g.velocity_tendencies(vn, w, zh, K, with_scale=True)
    dz = zh[:-1] - zh[1:]
    zf = 0.5 * (zh[:-1] + zh[1:])
    vn_ie = np.zeros((g.ne, K + 1))
    gk = dz[:-1] / (dz[:-1] + dz[1:])
    vn_ie[:, 1:K] = gk * vn[:, 1:] + (1 - gk) * vn[:, :-1]
    vn_ie[:, 0] = vn[:, 0] + (vn[:, 0] - vn[:, 1]) * (zh[0] - zf[0]) / (zf[0] - zf[1])
    vn_ie[:, K] = vn[:, K - 1] + (vn[:, K - 1] - vn[:, K - 2]) * (zh[K] - zf[K - 1]) / (zf[K - 1] - zf[K - 2])
    x, c0, c1 = g.edge_xyz, g.cell_xyz[g.e2c[:, 0]], g.cell_xyz[g.e2c[:, 1]]
    a0, a1 = _arc(x, c0), _arc(x, c1)
    wf = 0.5 * (w[:, :-1] + w[:, 1:])
    w_e = (a1[:, None] * wf[g.e2c[:, 0]] + a0[:, None] * wf[g.e2c[:, 1]]) / (a0 + a1)[:, None]
    kc, vt, zeta = o["ke_c"], o["vt"], o["vort"]
    m = (np.abs(kc[g.e2c[:, 1]]) + np.abs(kc[g.e2c[:, 0]])) / g.d_e[:, None] \
        + np.abs(vt) * (np.abs(g.f_e)[:, None] + 0.5 * (np.abs(zeta[g.e2v[:, 0]]) + np.abs(zeta[g.e2v[:, 1]]))) \
        + np.abs(w_e) * (np.abs(vn_ie[:, :-1]) + np.abs(vn_ie[:, 1:])) / dz
    assert (o["m_ddt"] <= 1.0000001 * m).all() and (o["m_ddt"] >= 0.9999999 * m).all()
    assert (np.abs(o["ddt_vn"]) <= 1.0000001 * m).all()
    div, vort, md, mv = g.div_vort(vn, K, with_scale=True)
    m_div = sum(np.abs(g.geofac_div[:, j:j + 1] * vn[g.c2e[:, j]]) for j in range(3))
    m_vort = sum(np.abs(g.geofac_rot[:, j:j + 1] * vn[g.v2e[:, j]]) for j in range(6))
    assert (md <= 1.0000001 * m_div).all() and (md >= 0.9999999 * m_div).all()
    assert (mv <= 1.0000001 * m_vort).all() and (mv >= 0.9999999 * m_vort).all()


# ----------------------------------------------------------------------------------------------
# special cases that reduce to library routines; internal consistency of the two evaluation paths
# ----------------------------------------------------------------------------------------------
def test_operators_equal_sparse_matrix_products(oracle_grid):
    """div, vort, vt, KE_c are (sparse matrix) x (field): re-evaluate with scipy.sparse"""
    import scipy.sparse as sp
    g = oracle_grid(2)
    K = 5
    rng = np.random.default_rng(5)
    vn = rng.standard_normal((g.ne, K))
    w = rng.standard_normal((g.nc, K + 1))
    zh = si.z_half_levels(K)

    def mat(idx, coef, ncols):
        r = np.repeat(np.arange(idx.shape[0]), idx.shape[1])
        return sp.csr_matrix((coef.ravel(), (r, idx.ravel())), shape=(idx.shape[0], ncols))
    D = mat(g.c2e, g.geofac_div, g.ne)
    R = mat(g.v2e, g.geofac_rot, g.ne)
    T = mat(g.e2e4, g.rbf, g.ne)
    B = mat(g.c2e, g.bln, g.ne)
    div, vort = g.div_vort(vn, K)
    out = g.velocity_tendencies(vn, w, zh, K)
    assert np.abs(div - D @ vn).max() < 1e-15 * abs(D).max() * 10
    assert np.abs(vort - R @ vn).max() < 1e-15 * abs(R).max() * 10
    vt = T @ vn
    assert np.abs(out["vt"] - vt).max() < 1e-14
    ke_c = B @ (0.5 * (vn * vn + vt * vt))
    assert np.abs(out["ke_c"] - ke_c).max() < 1e-13
    assert np.abs(out["vort"] - vort).max() == 0
    # the tendency, re-assembled with numpy from the definition (S5-S7), all levels incl. the ends
    dz = zh[:-1] - zh[1:]
    zf = 0.5 * (zh[:-1] + zh[1:])
    vn_ie = np.zeros((g.ne, K + 1))
    gk = dz[:-1] / (dz[:-1] + dz[1:])
    vn_ie[:, 1:K] = gk * vn[:, 1:] + (1 - gk) * vn[:, :-1]
    vn_ie[:, 0] = vn[:, 0] + (vn[:, 0] - vn[:, 1]) * (zh[0] - zf[0]) / (zf[0] - zf[1])
    vn_ie[:, K] = vn[:, K - 1] + (vn[:, K - 1] - vn[:, K - 2]) * (zh[K] - zf[K - 1]) / (zf[K - 1] - zf[K - 2])
    wf = 0.5 * (w[:, :-1] + w[:, 1:])
    w_e = g.c_lin[:, :1] * wf[g.e2c[:, 0]] + g.c_lin[:, 1:] * wf[g.e2c[:, 1]]
    H = (ke_c[g.e2c[:, 1]] - ke_c[g.e2c[:, 0]]) * g.inv_d_e[:, None] \
        + vt * (g.f_e[:, None] + 0.5 * (vort[g.e2v[:, 0]] + vort[g.e2v[:, 1]]))
    V = w_e * (vn_ie[:, :-1] - vn_ie[:, 1:]) / dz
    ref = -(H + V)
    m = g.velocity_tendencies(vn, w, zh, K, with_scale=True)["m_ddt"]
    assert (np.abs(out["ddt_vn"] - ref) <= 1e-14 * m).all()


@pytest.mark.parametrize("k,flags", [(2, 0), (3, 1)])
def test_sampled_evaluation_matches_full_arrays(oracle_grid, k, flags):
    g = oracle_grid(k, 7, flags)
    K = 7
    rng = np.random.default_rng(8)
    vn = rng.standard_normal((g.ne, K + 2))      # ldk > nlev
    w = rng.standard_normal((g.nc, K + 3))
    zh = si.z_half_levels(K)
    full = g.velocity_tendencies(vn, w, zh, K, with_scale=True)
    div, vort, md, mv = g.div_vort(vn, K, with_scale=True)
    for what, arr, m, n in (("ddt_vn", full["ddt_vn"], full["m_ddt"], g.ne), ("div", div, md, g.nc),
                            ("vort", vort, mv, g.nv)):
        idx, lev = si.sample_points(1, n, K, 500)
        val, ms = g.sample(what, idx, lev, vn, K, w=w, z_half=zh)
        assert (np.abs(val - arr[idx, lev]) <= 1e-14 * m[idx, lev]).all(), what
        assert np.abs(ms - m[idx, lev]).max() <= 1e-14 * np.abs(m).max()


# ----------------------------------------------------------------------------------------------
# vertical-wind tendency ddt_w (reading P-19)
# ----------------------------------------------------------------------------------------------
def _numpy_ddt_w(g, vn, w, zh, K):
    """the definition of P-19 re-assembled with numpy (independent of og_ddt_w's loops)"""
    dz = zh[:-1] - zh[1:]
    gk = dz[:-1] / (dz[:-1] + dz[1:])
    vn_ie = np.zeros((g.ne, K + 1))
    vn_ie[:, 1:K] = gk * vn[:, 1:K] + (1 - gk) * vn[:, :K - 1]
    gradw = (w[g.e2c[:, 1]] - w[g.e2c[:, 0]]) * g.inv_d_e[:, None]
    hadv = sum(g.adv_c[:, j:j + 1] * (vn_ie * gradw)[g.c2e[:, j]] for j in range(3))
    out = np.zeros((g.nc, K + 1))
    dz2 = zh[:-2] - zh[2:]
    out[:, 1:K] = -(hadv[:, 1:K] + w[:, 1:K] * (w[:, :K - 1] - w[:, 2:K + 1]) / dz2)
    return out


@pytest.mark.parametrize("k,seed,flags", [(0, 0, 0), (2, 0, 0), (4, 0, 0), (3, 4, 1)])
def test_adv_c_reconstructs_the_identity(oracle_grid, k, seed, flags):
    """P-19: the three weights of a cell satisfy sum_j adv_c(c,j) n_j n_j^T = I in the tangent plane at the cell centre
    (so that sum_j adv_c (u.n_j)(grad s.n_j) = u.grad s), hence also sum_j adv_c = trace I = 2. Checked with numpy from the
    exported positions and normals in a basis of its own (the identity does not depend on the basis)."""
    g = oracle_grid(k, seed, flags)
    cc = g.cell_xyz
    ref = np.where(np.abs(cc[:, :1]) < 0.9, np.array([[1.0, 0, 0]]), np.array([[0, 1.0, 0]]))
    e1 = np.cross(cc, ref)
    e1 /= np.linalg.norm(e1, axis=1)[:, None]
    e2 = np.cross(cc, e1)
    S = np.zeros((g.nc, 2, 2))
    for j in range(3):
        n = g.edge_normal[g.c2e[:, j]]
        p = np.stack([(n * e1).sum(1), (n * e2).sum(1)], 1)
        p /= np.linalg.norm(p, axis=1)[:, None]
        S += g.adv_c[:, j, None, None] * p[:, :, None] * p[:, None, :]
    assert np.abs(S - np.eye(2)[None]).max() < 1e-13
    assert np.abs(g.adv_c.sum(1) - 2).max() < 1e-13
    assert (g.adv_c > 0.3).all() and (g.adv_c < 1.0).all()          # 2/3 each on an equilateral triangle


def test_ddt_w_definition_and_special_cases(oracle_grid):
    g = oracle_grid(2)
    K = 7
    zh = si.z_half_levels(K)
    rng = np.random.default_rng(21)
    vn = rng.standard_normal((g.ne, K)) * 10
    w = rng.standard_normal((g.nc, K + 1))
    got, m = g.w_tendency(vn, w, zh, K, with_scale=True)
    want = _numpy_ddt_w(g, vn, w, zh, K)
    assert (np.abs(got - want) <= 1e-14 * np.maximum(m, 1e-300))[:, 1:K].all()
    assert (got[:, 0] == 0).all() and (got[:, K] == 0).all()          # top and surface: boundary conditions of w
    # horizontally uniform w: no horizontal advection whatever vn; w linear in z: -w dw/dz exactly
    b, c0 = 2.0e-4, 0.3
    wl = np.repeat((c0 + b * zh)[None, :], g.nc, axis=0)
    got = g.w_tendency(vn, wl, zh, K)
    assert np.abs(got[:, 1:K] + (wl * b)[:, 1:K]).max() < 1e-13 * np.abs(wl * b).max()
    # vn = 0: only the vertical part, for any w
    got = g.w_tendency(np.zeros_like(vn), w, zh, K)
    dz2 = zh[:-2] - zh[2:]
    assert np.abs(got[:, 1:K] + w[:, 1:K] * (w[:, :K - 1] - w[:, 2:]) / dz2).max() < 1e-13
    # two-sided pin of the tolerance scale
    gradw_abs = (np.abs(w[g.e2c[:, 1]]) + np.abs(w[g.e2c[:, 0]])) * g.inv_d_e[:, None]
    dz = zh[:-1] - zh[1:]
    gk = dz[:-1] / (dz[:-1] + dz[1:])
    vie = np.zeros((g.ne, K + 1))
    vie[:, 1:K] = gk * vn[:, 1:K] + (1 - gk) * vn[:, :K - 1]
    mm = sum(np.abs(g.adv_c[:, j:j + 1]) * (np.abs(vie) * gradw_abs)[g.c2e[:, j]] for j in range(3))
    mm[:, 1:K] += np.abs(w[:, 1:K]) * (np.abs(w[:, :K - 1]) + np.abs(w[:, 2:])) / dz2
    assert (m[:, 1:K] <= 1.0000001 * mm[:, 1:K]).all() and (m[:, 1:K] >= 0.9999999 * mm[:, 1:K]).all()
    # sampled evaluation = full arrays
    idx, lev = si.sample_points(5, g.nc, K + 1, 400)
    val, ms = g.sample("ddt_w", idx, lev, vn, K, w=w, z_half=zh)
    full, mfull = g.w_tendency(vn, w, zh, K, with_scale=True)
    assert np.abs(val - full[idx, lev]).max() == 0 and np.abs(ms - mfull[idx, lev]).max() == 0


def test_ddt_w_converges_to_the_advection_of_a_tilted_solid_body_flow(oracle_grid):
    """Closed form: w(x) = w0 (x.z_hat) carried by the solid-body rotation u = a Omega' x x about a TILTED axis has
    -u.grad w = -w0 (Omega' x x).z_hat at every level (uniform in z, so the vertical part vanishes). The discrete
    ddt_w converges to it at first order; a weight set that does not reproduce u.grad s (e.g. bln in place of adv_c: half
    the value) stays at an error of order one."""
    om = 2.0e-6 * np.array([np.sin(0.7), 0.0, np.cos(0.7)])          # rad/s, tilted by 0.7 rad
    w0, K = 0.5, 4
    zh = si.z_half_levels(K)
    errs = []
    for k in (2, 3, 4):
        g = oracle_grid(k)
        u = np.cross(om[None, :], g.edge_xyz) * A                     # m/s at edge midpoints
        vn = np.repeat((u * g.edge_normal).sum(1)[:, None], K, axis=1)
        w = np.repeat((w0 * g.cell_xyz[:, 2])[:, None], K + 1, axis=1)
        exact = -w0 * np.cross(om[None, :], g.cell_xyz)[:, 2]
        got = g.w_tendency(vn, w, zh, K)
        errs.append(np.abs(got[:, 1:K] - exact[:, None]).max() / np.abs(exact).max())
    assert errs[2] < 0.03, errs
    assert 1.6 < errs[0] / errs[1] < 4.6 and 1.6 < errs[1] / errs[2] < 4.6, errs
    # teeth: the edge-to-cell interpolation weights bln (sum 1 instead of 2) give half the advection
    g = oracle_grid(3)
    u = np.cross(om[None, :], g.edge_xyz) * A
    vn = np.repeat((u * g.edge_normal).sum(1)[:, None], K, axis=1)
    w = np.repeat((w0 * g.cell_xyz[:, 2])[:, None], K + 1, axis=1)
    gradw = (w[g.e2c[:, 1]] - w[g.e2c[:, 0]]) * g.inv_d_e[:, None]
    half = -sum(g.bln[:, j:j + 1] * (vn[:, :1] * gradw[:, :1])[g.c2e[:, j]] for j in range(3))[:, 0]
    exact = -w0 * np.cross(om[None, :], g.cell_xyz)[:, 2]
    assert np.abs(half - exact).max() / np.abs(exact).max() > 0.3


# ----------------------------------------------------------------------------------------------
# metric variant (reading P-20): weighted KE gradient, per-edge vertical metrics,
# contravariant correction of w
# ----------------------------------------------------------------------------------------------
def _tilted_setup(g, K, h_top, h0, gam, u0, w0):
    """A hybrid terrain-following grid z(x, k) = zflat_k + h(x) (1 - zflat_k / h_top), h = h0 (x . p), flat at the top;
    vn = (1 + gam z) vn_solid_body sampled at the heights of every edge column, w = w0. All analytic, numpy only."""
    zflat = si.z_half_levels(K, h_top=h_top)
    zf = 0.5 * (zflat[:-1] + zflat[1:])
    p = np.array([np.sin(0.9) * np.cos(0.4), np.sin(0.9) * np.sin(0.4), np.cos(0.9)])
    x = g.edge_xyz
    h = h0 * (x @ p)
    zh_e = zflat[None, :] + h[:, None] * (1 - zflat[None, :] / h_top)
    zfull_e = zf[None, :] + h[:, None] * (1 - zf[None, :] / h_top)
    gradh = h0 * (p[None, :] - (x @ p)[:, None] * x) / A             # horizontal gradient of h on the sphere of radius A
    t = np.cross(g.edge_normal, x)                                    # t_e = n_e x x_e (P-4)
    zn = (gradh * g.edge_normal).sum(1)[:, None] * (1 - zf[None, :] / h_top)
    zt = (gradh * t).sum(1)[:, None] * (1 - zf[None, :] / h_top)
    vn_sb = si.solid_body_vn(x, g.edge_normal, u0)
    vt_sb = (u0 * np.cross(np.array([0, 0, 1.0])[None, :], x) * t).sum(1)
    prof = 1 + gam * zfull_e
    sinp = x[:, 2]
    cosp = np.sqrt(1 - sinp ** 2)
    north = (np.array([0, 0, 1.0])[None, :] - sinp[:, None] * x) / cosp[:, None]
    nn = (north * g.edge_normal).sum(1)
    exact = -((prof ** 2 * (u0 * u0 / A) + prof * 2 * OMEGA * u0) * (sinp * cosp * nn)[:, None]) - w0 * gam * vn_sb[:, None]
    return dict(zflat=zflat, zh_e=zh_e, zn=zn, zt=zt, vn=prof * vn_sb[:, None], w=np.full((g.nc, K + 1), w0), vn_sb=vn_sb,
                vt_sb=vt_sb, prof=prof, exact=exact)


@pytest.mark.parametrize("k,seed,flags", [(0, 0, 0), (2, 0, 0), (4, 0, 0), (3, 4, 1)])
def test_cgrad_is_second_order_from_geometry(oracle_grid, k, seed, flags):
    """P-20: gradK = cgrad1 K(c1) - cgrad0 K(c0) + K(x_e) (cgrad0 - cgrad1) is exact for K constant (by construction), linear
    AND quadratic along the dual arc: with signed abscissae -a0, +a1 (numpy arc distances, metres)
    cgrad1 a1 + cgrad0 a0 = 1 and cgrad1 a1^2 - cgrad0 a0^2 = 0. Swapping the two columns fails the second identity wherever
    a0 != a1; the plain centred difference (1/d_e, 1/d_e) fails it too."""
    g = oracle_grid(k, seed, flags)
    x, c0, c1 = g.edge_xyz, g.cell_xyz[g.e2c[:, 0]], g.cell_xyz[g.e2c[:, 1]]
    a0, a1 = _arc(x, c0) * A, _arc(x, c1) * A
    assert np.abs(g.cgrad[:, 1] * a1 + g.cgrad[:, 0] * a0 - 1).max() < 1e-13
    assert np.abs(g.cgrad[:, 1] * a1 ** 2 - g.cgrad[:, 0] * a0 ** 2).max() < 1e-13 * (a0 + a1).max()
    swapped = np.abs(g.cgrad[:, 0] * a1 ** 2 - g.cgrad[:, 1] * a0 ** 2).max() / (a0 + a1).max()
    assert swapped > 1e-3
    assert np.abs(g.cgrad[:, 0] - (a1 / a0) / g.d_e).max() < 1e-13 / g.d_e.min()


def test_metric_from_zhalf_and_vertical_exactness_per_edge(oracle_mod, oracle_grid):
    """per-edge level heights: weights and inverse thicknesses against numpy; the vertical term is exact for vn linear in z
    in every column although every column has its own heights, both ends included"""
    g = oracle_grid(1)
    K = 7
    rng = np.random.default_rng(31)
    zflat = si.z_half_levels(K)
    zh_e = zflat[None, :] * (1 + 0.3 * rng.random((g.ne, 1))) + 50.0 * rng.random((g.ne, 1))       # stretched and shifted per edge
    wgt, inv = oracle_mod.metric_from_zhalf(zh_e, K, K)
    dz = zh_e[:, :-1] - zh_e[:, 1:]
    assert np.abs(inv * dz - 1).max() < 1e-15
    assert np.abs(wgt[:, 1:K] - dz[:, :-1] / (dz[:, :-1] + dz[:, 1:])).max() < 1e-15
    assert np.abs(wgt[:, 0] - dz[:, 0] / (dz[:, 0] + dz[:, 1])).max() < 1e-15
    assert np.abs(wgt[:, K] - dz[:, K - 1] / (dz[:, K - 1] + dz[:, K - 2])).max() < 1e-15
    zf = 0.5 * (zh_e[:, :-1] + zh_e[:, 1:])
    b = (1.0 + rng.random(g.ne)) * 1e-3
    vn = 2.0 + b[:, None] * zf
    w = np.repeat((1.0 + 50.0 * g.cell_xyz[:, 0])[:, None], K + 1, axis=1) * (1.0 + 0.1 * np.arange(K + 1))[None, :]
    zero = np.zeros((g.ne, K))
    o1 = g.velocity_tendencies_metric(vn, w, wgt, inv, zero, zero, K)["ddt_vn"]
    o0 = g.velocity_tendencies_metric(vn, np.zeros_like(w), wgt, inv, zero, zero, K)["ddt_vn"]
    x, c0, c1 = g.edge_xyz, g.cell_xyz[g.e2c[:, 0]], g.cell_xyz[g.e2c[:, 1]]
    a0, a1 = _arc(x, c0), _arc(x, c1)
    wf = 0.5 * (w[:, :-1] + w[:, 1:])
    w_e = (a1[:, None] * wf[g.e2c[:, 0]] + a0[:, None] * wf[g.e2c[:, 1]]) / (a0 + a1)[:, None]
    want = -w_e * b[:, None]
    assert np.abs((o1 - o0) - want).max() / np.abs(want).max() < 1e-10


def test_metric_variant_on_flat_levels_differs_only_by_the_weighted_gradient(oracle_mod, oracle_grid):
    """flat levels, zero slopes: ddt_metric - ddt_plain = -(weighted gradK - centred gradK), re-assembled with numpy from
    the oracle's KE_c and a numpy KE_e; the tolerance scale M(p) is the sum of the absolute terms (two-sided)"""
    g = oracle_grid(2)
    K = 6
    rng = np.random.default_rng(33)
    vn = rng.standard_normal((g.ne, K)) * 8
    w = rng.standard_normal((g.nc, K + 1))
    zh = si.z_half_levels(K)
    wgt, inv = oracle_mod.metric_from_zhalf(np.repeat(zh[None, :], g.ne, axis=0), K, K)
    zero = np.zeros((g.ne, K))
    om = g.velocity_tendencies_metric(vn, w, wgt, inv, zero, zero, K, with_scale=True)
    op = g.velocity_tendencies(vn, w, zh, K, with_scale=True)
    ke_e = 0.5 * (vn * vn + op["vt"] ** 2)
    kc = op["ke_c"]
    c0, c1 = g.e2c[:, 0], g.e2c[:, 1]
    gw = g.cgrad[:, 1:] * kc[c1] - g.cgrad[:, :1] * kc[c0] + ke_e * (g.cgrad[:, :1] - g.cgrad[:, 1:])
    gp = (kc[c1] - kc[c0]) * g.inv_d_e[:, None]
    assert (np.abs((om["ddt_vn"] - op["ddt_vn"]) + (gw - gp)) <= 1e-13 * (om["m_ddt"] + op["m_ddt"])).all()
    assert np.abs(gw - gp).max() > 1e-3 * np.abs(gp).max()            # the weighting is not a no-op on this grid
    m = g.cgrad[:, 1:] * np.abs(kc[c1]) + g.cgrad[:, :1] * np.abs(kc[c0]) + np.abs(ke_e) * np.abs(g.cgrad[:, :1] - g.cgrad[:, 1:]) \
        + (op["m_ddt"] - (np.abs(kc[c1]) + np.abs(kc[c0])) * g.inv_d_e[:, None])
    assert (om["m_ddt"] <= 1.000001 * m).all() and (om["m_ddt"] >= 0.999999 * m).all()


def test_metric_sampled_evaluation_matches_full_arrays(oracle_mod, oracle_grid):
    g = oracle_grid(3, 7, 1)
    K = 9
    rng = np.random.default_rng(41)
    vn = rng.standard_normal((g.ne, K + 1)) * 6          # ldk > nlev
    w = rng.standard_normal((g.nc, K + 3))
    zh_e, zn, zt = si.make_metric_heights(1, g.edge_xyz, g.edge_normal, K, K + 1, K + 3, pad_value=0.0)
    zn, zt = zn * 50, zt * 50                            # slopes of a few per cent
    wgt, inv = oracle_mod.metric_from_zhalf(zh_e, K, K + 1)
    wgt, inv = np.nan_to_num(wgt), np.nan_to_num(inv)
    full = g.velocity_tendencies_metric(vn, w, wgt, inv, zn, zt, K, with_scale=True)
    idx, lev = si.sample_points(2, g.ne, K, 600)
    val, ms = g.sample_metric(idx, lev, vn, w, wgt, inv, zn, zt, K)
    assert (np.abs(val - full["ddt_vn"][idx, lev]) <= 1e-14 * full["m_ddt"][idx, lev]).all()
    assert np.abs(ms - full["m_ddt"][idx, lev]).max() <= 1e-14 * np.abs(full["m_ddt"]).max()


def test_contravariant_correction_closed_form(oracle_mod, oracle_grid):
    """On coordinate surfaces z(x, k) the horizontal operators see (d/dn)|_s = (d/dn)|_z + z_n d/dz; collecting the metric
    terms of dK/dn and vt zeta gives exactly -(vn z_n + vt z_t) dvn/dz (P-20), i.e. vertical advection with the
    contravariant velocity w - vn z_n - vt z_t. Pin of that term alone: the difference of the oracle with and without the
    slopes equals +(vn z_n + vt z_t) gam vn_sb, with vt the ANALYTIC tangential wind; a wrong sign gives a relative
    error of 2, swapped slopes 2.3. Values: R2B2..4 3.3e-3, 1.8e-3, 1.3e-3 (the RBF reconstruction of vt)."""
    K, gam = 6, 4.0e-5
    errs = []
    for k in (2, 3, 4):
        g = oracle_grid(k)
        s = _tilted_setup(g, K, 3.0e4, 9.0e3, gam, 20.0, 0.1)
        wgt, inv = oracle_mod.metric_from_zhalf(s["zh_e"], K, K)
        a = g.velocity_tendencies_metric(s["vn"], s["w"], wgt, inv, s["zn"], s["zt"], K)["ddt_vn"]
        b = g.velocity_tendencies_metric(s["vn"], s["w"], wgt, inv, 0 * s["zn"], 0 * s["zt"], K)["ddt_vn"]
        want = (s["vn"] * s["zn"] + s["prof"] * s["vt_sb"][:, None] * s["zt"]) * gam * s["vn_sb"][:, None]
        errs.append(np.abs((a - b) - want).max() / np.abs(want).max())
        assert np.abs((a - b) + want).max() / np.abs(want).max() > 1.9
    assert errs[0] < 5e-3 and errs[1] < 3e-3 and errs[2] < 2e-3, errs


def test_metric_tendency_converges_on_a_tilted_grid(oracle_mod, oracle_grid):
    """the whole tendency on the tilted grid against the z-coordinate closed form of the flat pin (the physical field is the
    same, only the coordinate surfaces tilt): first-order convergence as on flat levels, and dropping the correction
    doubles the error at R2B4. Values with / without: R2B2 8.2e-3 / 8.3e-3, R2B3 4.3e-3 / 5.6e-3, R2B4 2.7e-3 / 5.7e-3."""
    K, gam = 6, 4.0e-5
    with_c, without = [], []
    for k in (2, 3, 4):
        g = oracle_grid(k)
        s = _tilted_setup(g, K, 3.0e4, 9.0e3, gam, 20.0, 0.1)
        wgt, inv = oracle_mod.metric_from_zhalf(s["zh_e"], K, K)
        a = g.velocity_tendencies_metric(s["vn"], s["w"], wgt, inv, s["zn"], s["zt"], K)["ddt_vn"]
        b = g.velocity_tendencies_metric(s["vn"], s["w"], wgt, inv, 0 * s["zn"], 0 * s["zt"], K)["ddt_vn"]
        scale = np.abs(s["exact"]).max()
        with_c.append(np.abs(a - s["exact"]).max() / scale)
        without.append(np.abs(b - s["exact"]).max() / scale)
    assert with_c[0] < 1.0e-2 and with_c[1] < 5.5e-3 and with_c[2] < 3.5e-3, with_c
    assert with_c[0] / with_c[2] > 2.4
    assert without[2] > 1.8 * with_c[2], (with_c, without)


# ----------------------------------------------------------------------------------------------
# seeded permutation (P-7)
# ----------------------------------------------------------------------------------------------
def _perm_from_positions(a_perm, a_canon, decimals=12):
    """new id of canonical entity i, recovered geometrically (unique positions)"""
    key = lambda a: [tuple(r) for r in np.round(a, decimals) + 0.0]
    pos = {t: i for i, t in enumerate(key(a_perm))}
    return np.array([pos[t] for t in key(a_canon)])


def test_permutation_equivariance(oracle_grid):
    k, seed = 2, 4
    g0, g1 = oracle_grid(k), oracle_grid(k, seed, 1)
    pv = _perm_from_positions(g1.vert_xyz, g0.vert_xyz)
    pe = _perm_from_positions(g1.edge_xyz, g0.edge_xyz)
    pc = _perm_from_positions(g1.cell_xyz, g0.cell_xyz)
    for p, n in ((pv, g0.nv), (pe, g0.ne), (pc, g0.nc)):
        assert sorted(p) == list(range(n))
        assert (p != np.arange(n)).mean() > 0.9          # it really is a shuffle
    # rows move, entries are renumbered, slot order is kept
    assert (g1.c2e[pc] == pe[g0.c2e]).all() and (g1.c2v[pc] == pv[g0.c2v]).all()
    assert (g1.e2c[pe] == pc[g0.e2c]).all() and (g1.e2v[pe] == pv[g0.e2v]).all()
    assert (g1.e2e4[pe] == pe[g0.e2e4]).all()
    assert (g1.v2e[pv] == pe[g0.v2e]).all() and (g1.v2c[pv] == pc[g0.v2c]).all()
    assert (g1.c_os[pc] == g0.c_os).all() and (g1.v_os[pv] == g0.v_os).all()
    # permuted-grid outputs, un-permuted, reproduce canonical-grid outputs
    K = 4
    rng = np.random.default_rng(2)
    vn0 = rng.standard_normal((g0.ne, K))
    w0 = rng.standard_normal((g0.nc, K + 1))
    zh = si.z_half_levels(K)
    vn1 = np.empty_like(vn0)
    vn1[pe] = vn0
    w1 = np.empty_like(w0)
    w1[pc] = w0
    o0 = g0.velocity_tendencies(vn0, w0, zh, K, with_scale=True)
    o1 = g1.velocity_tendencies(vn1, w1, zh, K)
    assert (np.abs(o1["ddt_vn"][pe] - o0["ddt_vn"]) <= 1e-13 * o0["m_ddt"]).all()
    # different seeds give different permutations; same seed the same
    g2 = oracle_grid(k, seed + 1, 1)
    assert not (g2.c2e == g1.c2e).all()


def test_mix64_reference_values(oracle_mod):
    """P-7 mixer restated in Python integers; ranks must reproduce the oracle's permutation"""
    M = (1 << 64) - 1

    def mix64(seed, stream, i):
        z = (seed + 0x9E3779B97F4A7C15 * (i + 1) + 0xD1B54A32D192ED03 * (stream + 1)) & M
        z ^= z >> 30
        z = (z * 0xBF58476D1CE4E5B9) & M
        z ^= z >> 27
        z = (z * 0x94D049BB133111EB) & M
        z ^= z >> 31
        return z
    seed, k = 4, 1
    g0, g1 = oracle_mod.Grid(k), oracle_mod.Grid(k, seed, 1)
    for stream, n, canon, perm in ((0, g0.nc, g0.cell_xyz, g1.cell_xyz), (1, g0.ne, g0.edge_xyz, g1.edge_xyz),
                                   (2, g0.nv, g0.vert_xyz, g1.vert_xyz)):
        keys = [(mix64(seed, stream, i), i) for i in range(n)]
        order = sorted(range(n), key=lambda i: keys[i])
        new_of_old = np.empty(n, dtype=np.int64)
        new_of_old[order] = np.arange(n)
        assert np.abs(perm[new_of_old] - canon).max() < 1e-12


def test_fp32_rounded_grid(oracle_grid):
    g = oracle_grid(2)
    r = g.rounded_f32()
    assert (r.c2e == g.c2e).all()
    for name in ("rbf", "bln", "geofac_div", "geofac_rot", "inv_d_e", "f_e", "c_lin"):
        assert (r.table(name) == g.table(name).astype(np.float32).astype(np.float64)).all()


# ----------------------------------------------------------------------------------------------
# domain decomposition (reading P-21): oracle/decomposition.py
# ----------------------------------------------------------------------------------------------
def _random_fields(g, nlev, seed):
    rng = np.random.default_rng(seed)
    vn = rng.normal(0.0, 10.0, (g.ne, nlev))
    w = rng.normal(0.0, 0.5, (g.nc, nlev + 1))
    return vn, w, si.z_half_levels(nlev)


def test_decomposition_read_sets_against_brute_force_perturbation(oracle_grid):
    """every vn column (then every w column) of R2B1 is perturbed in turn; the outputs of the oracle's operators that
    change are exactly the ones whose read set, written out from S1-S7, holds that column. A forgotten neighbour, a
    pentagon pad counted as a read, or e2c / e2v swapped fails here."""
    from oracle import decomposition as dd
    g = oracle_grid(1)
    nlev = 4
    vn, w, zh = _random_fields(g, nlev, 11)
    base = g.velocity_tendencies(vn, w, zh, nlev)["ddt_vn"][:, :nlev].copy()
    div0, vort0 = (a[:, :nlev].copy() for a in g.div_vort(vn, nlev))
    reads = [dd.ddt_vn_reads(g, e) for e in range(g.ne)]
    for col in range(g.ne):
        p = vn.copy()
        p[col] *= 1.5
        p[col] += 3.0
        got = set(np.nonzero(np.any(g.velocity_tendencies(p, w, zh, nlev)["ddt_vn"][:, :nlev] != base, axis=1))[0].tolist())
        want = {e for e in range(g.ne) if col in reads[e][0]}
        assert got == want, col
        div1, vort1 = g.div_vort(p, nlev)
        got_c = set(np.nonzero(np.any(div1[:, :nlev] != div0, axis=1))[0].tolist())
        got_v = set(np.nonzero(np.any(vort1[:, :nlev] != vort0, axis=1))[0].tolist())
        assert got_c == {c for c in range(g.nc) if col in dd.div_reads(g, c)}, col
        assert got_v == {v for v in range(g.nv) if col in dd.vort_reads(g, v)}, col
    for col in range(g.nc):
        p = w.copy()
        p[col] += 0.7
        got = set(np.nonzero(np.any(g.velocity_tendencies(vn, p, zh, nlev)["ddt_vn"][:, :nlev] != base, axis=1))[0].tolist())
        assert got == {e for e in range(g.ne) if col in reads[e][1]}, col


@pytest.mark.parametrize("k", [1, 3])
def test_decomposition_stencil_size(oracle_grid, k):
    """"the ddt_vn stencil spans 15 distinct edges" -- away from the pentagons; next to a pentagon the
    fan of one end vertex has one edge fewer"""
    from oracle import decomposition as dd
    g = oracle_grid(k)
    n = np.array([len(dd.ddt_vn_reads(g, e)[0]) for e in range(g.ne)])
    pent = np.nonzero(g.v_deg == 5)[0]
    near = np.zeros(g.ne, dtype=bool)
    near[g.v2e[pent, :5].ravel()] = True            # the five fan edges of each pentagon
    assert (n[~near] == 15).all()
    assert (n[near] == 14).all() and near.sum() == 60
    assert all(len(dd.ddt_vn_reads(g, e)[1]) == 2 for e in range(0, g.ne, 7))


def test_decomposition_ranges_closed_forms():
    from oracle import decomposition as dd
    for nc, R in ((80, 1), (80, 3), (320, 7), (1280, 8), (5120, 148)):
        P = nc // 4
        own = dd.cell_owner(nc, R)
        assert own.min() == 0 and own.max() == R - 1 and (np.diff(own) >= 0).all()       # contiguous, in rank order
        assert (own.reshape(-1, 4) == own[::4, None]).all()                                # whole parents
        sizes = np.bincount(own, minlength=R)
        assert sizes.sum() == nc and sizes.max() - sizes.min() <= 4                        # balanced to one parent
        for r in range(R):
            lo, hi = dd.part_range(P, R, r)
            assert (own[4 * lo:4 * hi] == r).all() and hi - lo == sizes[r] // 4
    # equal ranges where R divides P: rank r owns cells [r Nc / R, (r+1) Nc / R)
    own = dd.cell_owner(1280, 8)
    assert (own == np.arange(1280) // 160).all()


def test_decomposition_required_columns_and_ownership(oracle_grid):
    """the union over the owned points; with one rank it is every column; an ownership that gives an edge to a rank
    owning neither of its cells is reported"""
    from oracle import decomposition as dd
    g = oracle_grid(2)
    e_all, c_all = dd.required_columns(g, range(g.ne), range(g.nc), range(g.nv))
    assert (e_all == np.arange(g.ne)).all() and (c_all == np.arange(g.nc)).all()
    co = dd.cell_owner(g.nc, 4)
    eo = co[g.e2c[:, 0]]                                  # lower cell's rank owns the edge
    vo = np.array([co[g.v2c[v][:g.v_deg[v]]].min() for v in range(g.nv)])
    assert dd.check_ownership(g, 4, eo, vo) == []
    bad = eo.copy()
    interior = np.nonzero(co[g.e2c[:, 0]] == co[g.e2c[:, 1]])[0]
    bad[interior[0]] = (bad[interior[0]] + 1) % 4
    assert dd.check_ownership(g, 4, bad, vo) != []
    # the halo of rank 1: every required edge not owned lies within two cell rings of an owned cell
    mine = np.nonzero(eo == 1)[0]
    need_e, need_c = dd.required_columns(g, mine, np.nonzero(co == 1)[0], np.nonzero(vo == 1)[0])
    ring = set(np.nonzero(co == 1)[0].tolist())
    for _ in range(2):
        ring |= {int(c) for e in range(g.ne) if int(g.e2c[e][0]) in ring or int(g.e2c[e][1]) in ring for c in g.e2c[e]}
        ring |= {int(c) for v in range(g.nv) for c in g.v2c[v][:g.v_deg[v]]
                 if any(int(x) in ring for x in g.v2c[v][:g.v_deg[v]])}
    ring_edges = {int(e) for c in ring for e in g.c2e[c]}
    assert set(need_e.tolist()) <= ring_edges and set(need_c.tolist()) <= ring
    assert len(need_e) > len(mine) and set(mine.tolist()) <= set(need_e.tolist())
