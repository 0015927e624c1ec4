/*
 * icon_oracle.c -- ORACLE (test infrastructure, NOT the product).
 *
 * A plain, slow, obviously-correct CPU statement of the hot path of
 * arxiv/paper_2511_02021: the horizontal/vertical stencil sweep of ICON's
 * non-hydrostatic dynamical core on the icosahedral-triangular C-grid
 * (section 2: "icosahedral-triangular C grid"; PAPER.md:142-172,
 * section 3.2: the dycore and its one printed statement, the 3-term
 * e_bln_c_s-weighted edge->cell sum; the dual grid of hexagons
 * and exactly 12 pentagons, and the index-lookup arrays).
 *
 * The paper is silent on almost all of the discrete mathematics; the readings
 * P-1 ... P-17 of SURVEY.md section 8(c) (restated in DESIGN.md section 3) fix
 * them, and each function below names the reading it follows.
 *
 * Rules this file obeys:
 *   - fp64 everywhere, scalar loops "for entity / for level", every
 *     intermediate materialised in a full array, no blocking / fusion /
 *     reordering beyond what the definition states.
 *   - shares no code, header, table or constant generator with the CUDA
 *     library under paper_2511_02021_b200/csrc; neither includes the other.
 *   - only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
 *     --impl reference legs may load it.
 *   - build: gcc -O2 -ffp-contract=off -fopenmp -shared -fPIC (see oracle/__init__.py)
 *
 * Pins (tests/test_oracle_pins.py, -m "not gpu"): grid counts, area closure,
 * discrete Gauss, curl(grad)=0, weight sums, solid-body closed forms, the
 * linear-profile exactness of the vertical term, R2B0 brute-force values and
 * table rows, table checksums, permutation equivariance.
 * Parity UNPINNED (paper does not state them, ICON source not available):
 * agreement of bln / RBF kernel+scale / KE-gradient weights / vertical end
 * treatment with ICON's production coefficients.
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

#define OG_EARTH_RADIUS 6.371e6     /* a, metres (SURVEY 8 notation) */
#define OG_OMEGA 7.29212e-5         /* Omega, 1/s */
#define OG_PERMUTE 1u

typedef struct og_grid {
    int level_k;                    /* R2Bk */
    int64_t nc, ne, nv;
    /* G1: topology */
    int32_t *c2v;                   /* [nc][3] */
    int32_t *c2e;                   /* [nc][3] */
    int32_t *e2c;                   /* [ne][2] */
    int32_t *e2v;                   /* [ne][2] */
    int32_t *e2e4;                  /* [ne][4] */
    int32_t *v2e;                   /* [nv][6] */
    int32_t *v2c;                   /* [nv][6] */
    int32_t *v_deg;                 /* [nv] */
    int8_t *c_os;                   /* [nc][3] */
    int8_t *v_os;                   /* [nv][6] */
    /* G2: geometry (unit sphere positions; metres / square metres otherwise) */
    double *vert_xyz;               /* [nv][3] */
    double *cell_xyz;               /* [nc][3] */
    double *edge_xyz;               /* [ne][3] */
    double *edge_normal;            /* [ne][3] */
    double *l_e, *d_e, *inv_d_e, *f_e; /* [ne] */
    double *c_lin;                  /* [ne][2] */
    double *cgrad;                  /* [ne][2] reading P-20: distance-weighted KE-gradient coefficients */
    double *rbf;                    /* [ne][4] */
    double *a_c;                    /* [nc] */
    double *bln;                    /* [nc][3] */
    double *adv_c;                  /* [nc][3] reading P-19: sum_j adv_c(c,j) n_j n_j^T = I in the tangent plane of c */
    double *a_v;                    /* [nv] */
    double *geofac_div;             /* [nc][3] */
    double *geofac_rot;             /* [nv][6] */
} og_grid;

/* ------------------------------------------------------------------ */
/* small vector helpers                                                */
/* ------------------------------------------------------------------ */
static double dot3(const double *p, const double *q) { return p[0] * q[0] + p[1] * q[1] + p[2] * q[2]; }
static void cross3(const double *p, const double *q, double *r)
{
    r[0] = p[1] * q[2] - p[2] * q[1];
    r[1] = p[2] * q[0] - p[0] * q[2];
    r[2] = p[0] * q[1] - p[1] * q[0];
}
static double norm3(const double *p) { return sqrt(dot3(p, p)); }
static void normalize3(double *p)
{
    double n = norm3(p);
    p[0] /= n; p[1] /= n; p[2] /= n;
}
/* great-circle arc between unit vectors, P-8: atan2(|p x q|, p.q) */
static double arc3(const double *p, const double *q)
{
    double c[3];
    cross3(p, q, c);
    return atan2(norm3(c), dot3(p, q));
}
/* spherical triangle area (spherical excess), P-8:
 * 2*atan2(|p.(q x r)|, 1 + p.q + q.r + r.p) */
static double sph_tri_area(const double *p, const double *q, const double *r)
{
    double qr[3];
    cross3(q, r, qr);
    return 2.0 * atan2(fabs(dot3(p, qr)), 1.0 + dot3(p, q) + dot3(q, r) + dot3(r, p));
}

/* ------------------------------------------------------------------ */
/* half-edge key sort: "collect (min v, max v) keys and sort"           */
/* ------------------------------------------------------------------ */
typedef struct { uint64_t key; int64_t h; } og_hkey;
static int og_hkey_cmp(const void *a, const void *b)
{
    const og_hkey *x = (const og_hkey *)a, *y = (const og_hkey *)b;
    if (x->key < y->key) return -1;
    if (x->key > y->key) return 1;
    if (x->h < y->h) return -1;
    if (x->h > y->h) return 1;
    return 0;
}
/* For a closed triangulation c2v[nc][3]: fill keys for all 3*nc half-edges
 * (cell c, slot j joins vertex slots j and j+1) and sort them, so that the two
 * half-edges of every undirected edge are adjacent. */
static og_hkey *og_sorted_halfedges(const int32_t *c2v, int64_t nc)
{
    og_hkey *hk = (og_hkey *)malloc(sizeof(og_hkey) * (size_t)(3 * nc));
    if (!hk) return NULL;
    for (int64_t c = 0; c < nc; ++c)
        for (int j = 0; j < 3; ++j) {
            uint64_t a = (uint64_t)c2v[3 * c + j], b = (uint64_t)c2v[3 * c + (j + 1) % 3];
            uint64_t lo = a < b ? a : b, hi = a < b ? b : a;
            hk[3 * c + j].key = (lo << 32) | hi;
            hk[3 * c + j].h = 3 * c + j;
        }
    qsort(hk, (size_t)(3 * nc), sizeof(og_hkey), og_hkey_cmp);
    return hk;
}

/* ------------------------------------------------------------------ */
/* P-7: counter-based integer mixer for the seeded permutation          */
/* key_i = mix64(seed, stream, i); DESIGN.md section 3 states it once,   */
/* oracle and library each implement it.                                */
/* ------------------------------------------------------------------ */
static uint64_t og_mix64(uint64_t seed, uint64_t stream, uint64_t i)
{
    uint64_t z = seed + 0x9E3779B97F4A7C15ULL * (i + 1) + 0xD1B54A32D192ED03ULL * (stream + 1);
    z ^= z >> 30; z *= 0xBF58476D1CE4E5B9ULL;
    z ^= z >> 27; z *= 0x94D049BB133111EBULL;
    z ^= z >> 31;
    return z;
}
typedef struct { uint64_t key; int64_t i; } og_pkey;
static int og_pkey_cmp(const void *a, const void *b)
{
    const og_pkey *x = (const og_pkey *)a, *y = (const og_pkey *)b;
    if (x->key < y->key) return -1;
    if (x->key > y->key) return 1;
    if (x->i < y->i) return -1;
    if (x->i > y->i) return 1;
    return 0;
}
/* new id of old entity i = rank of key_i ascending, ties by i (P-7) */
static int32_t *og_perm_new_of_old(uint64_t seed, uint64_t stream, int64_t n)
{
    og_pkey *pk = (og_pkey *)malloc(sizeof(og_pkey) * (size_t)n);
    int32_t *new_of_old = (int32_t *)malloc(sizeof(int32_t) * (size_t)n);
    for (int64_t i = 0; i < n; ++i) { pk[i].key = og_mix64(seed, stream, (uint64_t)i); pk[i].i = i; }
    qsort(pk, (size_t)n, sizeof(og_pkey), og_pkey_cmp);
    for (int64_t r = 0; r < n; ++r) new_of_old[pk[r].i] = (int32_t)r;
    free(pk);
    return new_of_old;
}

/* ------------------------------------------------------------------ */
/* G1: topology                                                        */
/* ------------------------------------------------------------------ */

/* P-1: unit icosahedron, 12 vertices and 20 CCW faces in five strips */
static void og_base_icosahedron(double *xyz /*[12][3]*/, int32_t *c2v /*[20][3]*/)
{
    const double pi = 3.14159265358979323846;
    const double lat = atan(0.5);
    xyz[0] = 0.0; xyz[1] = 0.0; xyz[2] = 1.0;
    for (int i = 0; i < 5; ++i) {
        double lon = (72.0 * i) * pi / 180.0;
        xyz[3 * (1 + i) + 0] = cos(lat) * cos(lon);
        xyz[3 * (1 + i) + 1] = cos(lat) * sin(lon);
        xyz[3 * (1 + i) + 2] = sin(lat);
        double lon2 = (36.0 + 72.0 * i) * pi / 180.0;
        xyz[3 * (6 + i) + 0] = cos(-lat) * cos(lon2);
        xyz[3 * (6 + i) + 1] = cos(-lat) * sin(lon2);
        xyz[3 * (6 + i) + 2] = sin(-lat);
    }
    xyz[33] = 0.0; xyz[34] = 0.0; xyz[35] = -1.0;
    for (int i = 0; i < 5; ++i) {
        int j = (i + 1) % 5;
        int32_t f[4][3] = { {0, 1 + i, 1 + j}, {1 + i, 6 + i, 1 + j}, {6 + i, 6 + j, 1 + j}, {11, 6 + j, 6 + i} };
        for (int q = 0; q < 4; ++q)
            for (int s = 0; s < 3; ++s) c2v[3 * (4 * i + q) + s] = f[q][s];
    }
}

/* P-2: one bisection. New vertex = normalised sum of the two end points;
 * children 4p+0=(a,ab,ca) 4p+1=(ab,b,bc) 4p+2=(ca,bc,c) 4p+3=(ab,bc,ca). */
static int og_bisect(double **pxyz, int64_t *pnv, int32_t **pc2v, int64_t *pnc)
{
    int64_t nc = *pnc, nv = *pnv;
    int32_t *c2v = *pc2v;
    double *xyz = *pxyz;
    og_hkey *hk = og_sorted_halfedges(c2v, nc);
    if (!hk) return -1;
    int64_t nh = 3 * nc, ne = nh / 2;
    int32_t *mid = (int32_t *)malloc(sizeof(int32_t) * (size_t)nh);   /* midpoint vertex of half-edge h */
    double *nxyz = (double *)realloc(xyz, sizeof(double) * 3 * (size_t)(nv + ne));
    if (!mid || !nxyz) return -1;
    xyz = nxyz;
    int64_t next = nv;
    for (int64_t s = 0; s < nh; s += 2) {
        /* closed manifold: every key occurs exactly twice */
        uint64_t lo = hk[s].key >> 32, hi = hk[s].key & 0xFFFFFFFFu;
        double m[3] = { xyz[3 * lo] + xyz[3 * hi], xyz[3 * lo + 1] + xyz[3 * hi + 1], xyz[3 * lo + 2] + xyz[3 * hi + 2] };
        normalize3(m);
        xyz[3 * next] = m[0]; xyz[3 * next + 1] = m[1]; xyz[3 * next + 2] = m[2];
        mid[hk[s].h] = (int32_t)next;
        mid[hk[s + 1].h] = (int32_t)next;
        ++next;
    }
    free(hk);
    int32_t *n2v = (int32_t *)malloc(sizeof(int32_t) * 3 * (size_t)(4 * nc));
    if (!n2v) return -1;
    for (int64_t p = 0; p < nc; ++p) {
        int32_t a = c2v[3 * p], b = c2v[3 * p + 1], c = c2v[3 * p + 2];
        int32_t ab = mid[3 * p], bc = mid[3 * p + 1], ca = mid[3 * p + 2];
        int32_t ch[4][3] = { {a, ab, ca}, {ab, b, bc}, {ca, bc, c}, {ab, bc, ca} };
        for (int q = 0; q < 4; ++q)
            for (int s = 0; s < 3; ++s) n2v[3 * (4 * p + q) + s] = ch[q][s];
    }
    free(mid);
    free(c2v);
    *pxyz = xyz; *pnv = next; *pc2v = n2v; *pnc = 4 * nc;
    return 0;
}

static void og_free_fields(og_grid *g)
{
    free(g->c2v); free(g->c2e); free(g->e2c); free(g->e2v); free(g->e2e4);
    free(g->v2e); free(g->v2c); free(g->v_deg); free(g->c_os); free(g->v_os);
    free(g->vert_xyz); free(g->cell_xyz); free(g->edge_xyz); free(g->edge_normal);
    free(g->l_e); free(g->d_e); free(g->inv_d_e); free(g->f_e); free(g->c_lin); free(g->cgrad); free(g->rbf);
    free(g->a_c); free(g->bln); free(g->adv_c); free(g->a_v); free(g->geofac_div); free(g->geofac_rot);
}
void og_grid_destroy(og_grid *g)
{
    if (!g) return;
    og_free_fields(g);
    free(g);
}

/* P-3 .. P-6: canonical numbering and all index tables */
static int og_build_topology(og_grid *g, double *xyz_prov, int64_t nv, int32_t *c2v_prov, int64_t nc)
{
    int64_t ne = 3 * nc / 2;
    g->nc = nc; g->ne = ne; g->nv = nv;
    /* P-3 vertices: first touch in the sweep c = 0..nc-1, slots 0,1,2 */
    int32_t *vnew = (int32_t *)malloc(sizeof(int32_t) * (size_t)nv);
    int32_t *v_first_cell = (int32_t *)malloc(sizeof(int32_t) * (size_t)nv);
    int8_t *v_first_slot = (int8_t *)malloc((size_t)nv);
    for (int64_t v = 0; v < nv; ++v) vnew[v] = -1;
    g->c2v = (int32_t *)malloc(sizeof(int32_t) * 3 * (size_t)nc);
    int64_t nextv = 0;
    for (int64_t c = 0; c < nc; ++c)
        for (int j = 0; j < 3; ++j) {
            int32_t pv = c2v_prov[3 * c + j];
            if (vnew[pv] < 0) {
                vnew[pv] = (int32_t)nextv;
                v_first_cell[nextv] = (int32_t)c;
                v_first_slot[nextv] = (int8_t)j;
                ++nextv;
            }
            g->c2v[3 * c + j] = vnew[pv];
        }
    if (nextv != nv) return -1;
    g->vert_xyz = (double *)malloc(sizeof(double) * 3 * (size_t)nv);
    for (int64_t pv = 0; pv < nv; ++pv)
        for (int s = 0; s < 3; ++s) g->vert_xyz[3 * vnew[pv] + s] = xyz_prov[3 * pv + s];
    free(vnew);

    /* P-3 edges: partner half-edges via sorted keys, then first-touch sweep */
    og_hkey *hk = og_sorted_halfedges(g->c2v, nc);
    int64_t nh = 3 * nc;
    int64_t *partner = (int64_t *)malloc(sizeof(int64_t) * (size_t)nh);
    for (int64_t s = 0; s < nh; s += 2) {
        if (hk[s].key != hk[s + 1].key) return -2;
        partner[hk[s].h] = hk[s + 1].h;
        partner[hk[s + 1].h] = hk[s].h;
    }
    free(hk);
    g->c2e = (int32_t *)malloc(sizeof(int32_t) * 3 * (size_t)nc);
    g->e2c = (int32_t *)malloc(sizeof(int32_t) * 2 * (size_t)ne);
    g->e2v = (int32_t *)malloc(sizeof(int32_t) * 2 * (size_t)ne);
    for (int64_t h = 0; h < nh; ++h) g->c2e[h] = -1;
    int64_t nexte = 0;
    for (int64_t c = 0; c < nc; ++c)
        for (int j = 0; j < 3; ++j) {
            int64_t h = 3 * c + j;
            if (g->c2e[h] < 0) {           /* unseen: first touch */
                int64_t p = partner[h];
                g->c2e[h] = (int32_t)nexte;
                g->c2e[p] = (int32_t)nexte;
                g->e2v[2 * nexte] = g->c2v[3 * c + j];
                g->e2v[2 * nexte + 1] = g->c2v[3 * c + (j + 1) % 3];
                g->e2c[2 * nexte] = (int32_t)c;
                g->e2c[2 * nexte + 1] = (int32_t)(p / 3);   /* second touch */
                ++nexte;
            }
        }
    free(partner);
    if (nexte != ne) return -3;

    /* P-4: c_os by slot */
    g->c_os = (int8_t *)malloc(3 * (size_t)nc);
    for (int64_t c = 0; c < nc; ++c)
        for (int j = 0; j < 3; ++j)
            g->c_os[3 * c + j] = (g->e2c[2 * g->c2e[3 * c + j]] == c) ? 1 : -1;

    /* P-5: vertex fans, counter-clockwise from the first-touch cell */
    g->v2e = (int32_t *)malloc(sizeof(int32_t) * 6 * (size_t)nv);
    g->v2c = (int32_t *)malloc(sizeof(int32_t) * 6 * (size_t)nv);
    g->v_deg = (int32_t *)malloc(sizeof(int32_t) * (size_t)nv);
    g->v_os = (int8_t *)malloc(6 * (size_t)nv);
    for (int64_t v = 0; v < nv; ++v) {
        int32_t c = v_first_cell[v];
        int j = v_first_slot[v];
        int deg = 0;
        for (;;) {
            if (deg >= 6) { if (c != v_first_cell[v]) return -4; break; }
            g->v2c[6 * v + deg] = c;
            g->v2e[6 * v + deg] = g->c2e[3 * c + j];
            ++deg;
            int32_t en = g->c2e[3 * c + (j + 2) % 3];          /* next edge */
            int32_t cn = (g->e2c[2 * en] == c) ? g->e2c[2 * en + 1] : g->e2c[2 * en];
            if (cn == v_first_cell[v]) break;
            int jn = -1;
            for (int s = 0; s < 3; ++s) if (g->c2v[3 * cn + s] == v) jn = s;
            if (jn < 0) return -5;
            c = cn; j = jn;
        }
        g->v_deg[v] = deg;
        for (int i = 0; i < deg; ++i)
            g->v_os[6 * v + i] = (g->e2v[2 * g->v2e[6 * v + i]] == v) ? -1 : 1;
        for (int i = deg; i < 6; ++i) {     /* pentagon: slot 5 = slot 0, sign 0 */
            g->v2e[6 * v + i] = g->v2e[6 * v];
            g->v2c[6 * v + i] = g->v2c[6 * v];
            g->v_os[6 * v + i] = 0;
        }
    }
    free(v_first_cell); free(v_first_slot);

    /* P-6: e2e4 */
    g->e2e4 = (int32_t *)malloc(sizeof(int32_t) * 4 * (size_t)ne);
    for (int64_t e = 0; e < ne; ++e)
        for (int side = 0; side < 2; ++side) {
            int32_t c = g->e2c[2 * e + side];
            int j = -1;
            for (int s = 0; s < 3; ++s) if (g->c2e[3 * c + s] == e) j = s;
            if (j < 0) return -6;
            g->e2e4[4 * e + 2 * side] = g->c2e[3 * c + (j + 1) % 3];
            g->e2e4[4 * e + 2 * side + 1] = g->c2e[3 * c + (j + 2) % 3];
        }
    return 0;
}

/* P-7: rows move to their new row, entries are renumbered, slot order kept */
static void og_permute_rows_i32(int32_t **ptab, int64_t n, int cols, const int32_t *row_new_of_old,
                                const int32_t *entry_new_of_old)
{
    int32_t *old = *ptab;
    int32_t *t = (int32_t *)malloc(sizeof(int32_t) * (size_t)(n * cols));
    for (int64_t i = 0; i < n; ++i)
        for (int s = 0; s < cols; ++s) {
            int32_t x = old[i * cols + s];
            t[(int64_t)row_new_of_old[i] * cols + s] = entry_new_of_old ? entry_new_of_old[x] : x;
        }
    free(old);
    *ptab = t;
}
static void og_permute_rows_i8(int8_t **ptab, int64_t n, int cols, const int32_t *row_new_of_old)
{
    int8_t *old = *ptab;
    int8_t *t = (int8_t *)malloc((size_t)(n * cols));
    for (int64_t i = 0; i < n; ++i)
        for (int s = 0; s < cols; ++s) t[(int64_t)row_new_of_old[i] * cols + s] = old[i * cols + s];
    free(old);
    *ptab = t;
}
static void og_permute_rows_f64(double **ptab, int64_t n, int cols, const int32_t *row_new_of_old)
{
    double *old = *ptab;
    double *t = (double *)malloc(sizeof(double) * (size_t)(n * cols));
    for (int64_t i = 0; i < n; ++i)
        for (int s = 0; s < cols; ++s) t[(int64_t)row_new_of_old[i] * cols + s] = old[i * cols + s];
    free(old);
    *ptab = t;
}
static void og_apply_permutation(og_grid *g, uint64_t seed)
{
    int32_t *pc = og_perm_new_of_old(seed, 0, g->nc);
    int32_t *pe = og_perm_new_of_old(seed, 1, g->ne);
    int32_t *pv = og_perm_new_of_old(seed, 2, g->nv);
    og_permute_rows_i32(&g->c2v, g->nc, 3, pc, pv);
    og_permute_rows_i32(&g->c2e, g->nc, 3, pc, pe);
    og_permute_rows_i32(&g->e2c, g->ne, 2, pe, pc);
    og_permute_rows_i32(&g->e2v, g->ne, 2, pe, pv);
    og_permute_rows_i32(&g->e2e4, g->ne, 4, pe, pe);
    og_permute_rows_i32(&g->v2e, g->nv, 6, pv, pe);
    og_permute_rows_i32(&g->v2c, g->nv, 6, pv, pc);
    og_permute_rows_i32(&g->v_deg, g->nv, 1, pv, NULL);
    og_permute_rows_i8(&g->c_os, g->nc, 3, pc);
    og_permute_rows_i8(&g->v_os, g->nv, 6, pv);
    og_permute_rows_f64(&g->vert_xyz, g->nv, 3, pv);
    free(pc); free(pe); free(pv);
}

/* ------------------------------------------------------------------ */
/* G2: geometry and coefficients (computed AFTER the optional           */
/* permutation, from the tables as the user sees them)                  */
/* ------------------------------------------------------------------ */

/* solve the 4x4 system M c = b by Gaussian elimination with partial pivoting */
static void og_solve4(double M[4][4], double b[4], double c[4])
{
    double A[4][5];
    for (int i = 0; i < 4; ++i) { for (int j = 0; j < 4; ++j) A[i][j] = M[i][j]; A[i][4] = b[i]; }
    for (int col = 0; col < 4; ++col) {
        int piv = col;
        for (int r = col + 1; r < 4; ++r) if (fabs(A[r][col]) > fabs(A[piv][col])) piv = r;
        if (piv != col) for (int j = 0; j < 5; ++j) { double t = A[col][j]; A[col][j] = A[piv][j]; A[piv][j] = t; }
        for (int r = col + 1; r < 4; ++r) {
            double f = A[r][col] / A[col][col];
            for (int j = col; j < 5; ++j) A[r][j] -= f * A[col][j];
        }
    }
    for (int i = 3; i >= 0; --i) {
        double s = A[i][4];
        for (int j = i + 1; j < 4; ++j) s -= A[i][j] * c[j];
        c[i] = s / A[i][i];
    }
}

static void og_build_geometry(og_grid *g)
{
    const double a = OG_EARTH_RADIUS;
    int64_t nc = g->nc, ne = g->ne, nv = g->nv;
    g->cell_xyz = (double *)malloc(sizeof(double) * 3 * (size_t)nc);
    g->edge_xyz = (double *)malloc(sizeof(double) * 3 * (size_t)ne);
    g->edge_normal = (double *)malloc(sizeof(double) * 3 * (size_t)ne);
    g->l_e = (double *)malloc(sizeof(double) * (size_t)ne);
    g->d_e = (double *)malloc(sizeof(double) * (size_t)ne);
    g->inv_d_e = (double *)malloc(sizeof(double) * (size_t)ne);
    g->f_e = (double *)malloc(sizeof(double) * (size_t)ne);
    g->c_lin = (double *)malloc(sizeof(double) * 2 * (size_t)ne);
    g->cgrad = (double *)malloc(sizeof(double) * 2 * (size_t)ne);
    g->rbf = (double *)malloc(sizeof(double) * 4 * (size_t)ne);
    g->a_c = (double *)malloc(sizeof(double) * (size_t)nc);
    g->bln = (double *)malloc(sizeof(double) * 3 * (size_t)nc);
    g->adv_c = (double *)malloc(sizeof(double) * 3 * (size_t)nc);
    g->a_v = (double *)malloc(sizeof(double) * (size_t)nv);
    g->geofac_div = (double *)malloc(sizeof(double) * 3 * (size_t)nc);
    g->geofac_rot = (double *)malloc(sizeof(double) * 6 * (size_t)nv);
    const double *V = g->vert_xyz;

    /* P-8: cell centre = spherical circumcentre normalize((v1-v0)x(v2-v0)); area = excess */
#pragma omp parallel for schedule(static)
    for (int64_t c = 0; c < nc; ++c) {
        const double *p0 = V + 3 * g->c2v[3 * c], *p1 = V + 3 * g->c2v[3 * c + 1], *p2 = V + 3 * g->c2v[3 * c + 2];
        double u[3] = { p1[0] - p0[0], p1[1] - p0[1], p1[2] - p0[2] };
        double w[3] = { p2[0] - p0[0], p2[1] - p0[1], p2[2] - p0[2] };
        double n[3];
        cross3(u, w, n);
        normalize3(n);
        g->cell_xyz[3 * c] = n[0]; g->cell_xyz[3 * c + 1] = n[1]; g->cell_xyz[3 * c + 2] = n[2];
        g->a_c[c] = sph_tri_area(p0, p1, p2) * a * a;
    }
    /* P-4 / P-8 / P-9: edge midpoint, normal, lengths, Coriolis, c_lin */
#pragma omp parallel for schedule(static)
    for (int64_t e = 0; e < ne; ++e) {
        const double *p0 = V + 3 * g->e2v[2 * e], *p1 = V + 3 * g->e2v[2 * e + 1];
        const double *c0 = g->cell_xyz + 3 * g->e2c[2 * e], *c1 = g->cell_xyz + 3 * g->e2c[2 * e + 1];
        double x[3] = { p0[0] + p1[0], p0[1] + p1[1], p0[2] + p1[2] };
        normalize3(x);
        double tau[3] = { p1[0] - p0[0], p1[1] - p0[1], p1[2] - p0[2] };
        normalize3(tau);
        double n[3];
        cross3(tau, x, n);                       /* n_e = tau_e x x_e */
        for (int s = 0; s < 3; ++s) { g->edge_xyz[3 * e + s] = x[s]; g->edge_normal[3 * e + s] = n[s]; }
        double le = arc3(p0, p1), de = arc3(c0, c1);
        g->l_e[e] = le * a;
        g->d_e[e] = de * a;
        g->inv_d_e[e] = 1.0 / (de * a);
        g->f_e[e] = 2.0 * OG_OMEGA * x[2];
        g->c_lin[2 * e] = arc3(x, c1) / de;
        g->c_lin[2 * e + 1] = arc3(x, c0) / de;
        /* P-20: cgrad(e,0) = (a1/a0)/d_e multiplies KE_c(c0), cgrad(e,1) = (a0/a1)/d_e multiplies KE_c(c1),
         * a0 = arc(x_e,c0), a1 = arc(x_e,c1), d_e in metres */
        g->cgrad[2 * e] = (arc3(x, c1) / arc3(x, c0)) / (de * a);
        g->cgrad[2 * e + 1] = (arc3(x, c0) / arc3(x, c1)) / (de * a);
    }
    /* G2 folded factor: geofac_div = l_e * c_os / A_c */
#pragma omp parallel for schedule(static)
    for (int64_t c = 0; c < nc; ++c)
        for (int j = 0; j < 3; ++j)
            g->geofac_div[3 * c + j] = g->l_e[g->c2e[3 * c + j]] * (double)g->c_os[3 * c + j] / g->a_c[c];
    /* P-10: bln = weights reproducing constants and linear functions in the
     * gnomonic tangent plane at the cell centre */
#pragma omp parallel for schedule(static)
    for (int64_t c = 0; c < nc; ++c) {
        const double *cc = g->cell_xyz + 3 * c;
        const double *p0 = V + 3 * g->c2v[3 * c];
        double d0 = dot3(p0, cc);
        double e1[3] = { p0[0] - d0 * cc[0], p0[1] - d0 * cc[1], p0[2] - d0 * cc[2] };
        normalize3(e1);
        double e2[3];
        cross3(cc, e1, e2);
        double xi[3], eta[3];
        for (int j = 0; j < 3; ++j) {
            const double *x = g->edge_xyz + 3 * g->c2e[3 * c + j];
            double s = dot3(x, cc);
            double P[3] = { x[0] / s - cc[0], x[1] / s - cc[1], x[2] / s - cc[2] };
            xi[j] = dot3(P, e1);
            eta[j] = dot3(P, e2);
        }
        /* [1 1 1; xi; eta] w = (1,0,0)^T by Cramer's rule */
        double det = (xi[1] * eta[2] - xi[2] * eta[1]) - (xi[0] * eta[2] - xi[2] * eta[0]) + (xi[0] * eta[1] - xi[1] * eta[0]);
        g->bln[3 * c] = (xi[1] * eta[2] - xi[2] * eta[1]) / det;
        g->bln[3 * c + 1] = (xi[2] * eta[0] - xi[0] * eta[2]) / det;
        g->bln[3 * c + 2] = (xi[0] * eta[1] - xi[1] * eta[0]) / det;
    }
    /* P-19: adv_c = the three weights a_j with sum_j a_j n_j n_j^T = I (2x2 identity) in the tangent plane at
     * the cell centre, n_j = the edge normal projected onto that plane and normalised. With them
     * sum_j a_j (u.n_j)(grad s.n_j) = u.grad s for locally constant u and grad s: the advection of a cell scalar
     * by the normal wind components alone (no vertex values needed). Equilateral triangle: a_j = 2/3. */
#pragma omp parallel for schedule(static)
    for (int64_t c = 0; c < nc; ++c) {
        const double *cc = g->cell_xyz + 3 * c;
        const double *p0 = V + 3 * g->c2v[3 * c];
        double d0 = dot3(p0, cc);
        double e1[3] = { p0[0] - d0 * cc[0], p0[1] - d0 * cc[1], p0[2] - d0 * cc[2] };
        normalize3(e1);
        double e2[3];
        cross3(cc, e1, e2);
        double nx[3], ny[3];
        for (int j = 0; j < 3; ++j) {
            const double *nn = g->edge_normal + 3 * g->c2e[3 * c + j];
            double px = dot3(nn, e1), py = dot3(nn, e2);
            double len = sqrt(px * px + py * py);
            nx[j] = px / len; ny[j] = py / len;
        }
        /* rows: n_x^2, n_x n_y, n_y^2; right-hand side (1, 0, 1); Cramer's rule */
        double A[3][3], b[3] = { 1.0, 0.0, 1.0 };
        for (int j = 0; j < 3; ++j) { A[0][j] = nx[j] * nx[j]; A[1][j] = nx[j] * ny[j]; A[2][j] = ny[j] * ny[j]; }
        double det = A[0][0] * (A[1][1] * A[2][2] - A[1][2] * A[2][1]) - A[0][1] * (A[1][0] * A[2][2] - A[1][2] * A[2][0])
                   + A[0][2] * (A[1][0] * A[2][1] - A[1][1] * A[2][0]);
        for (int j = 0; j < 3; ++j) {
            double M[3][3];
            for (int r = 0; r < 3; ++r) for (int q = 0; q < 3; ++q) M[r][q] = (q == j) ? b[r] : A[r][q];
            double dj = M[0][0] * (M[1][1] * M[2][2] - M[1][2] * M[2][1]) - M[0][1] * (M[1][0] * M[2][2] - M[1][2] * M[2][0])
                      + M[0][2] * (M[1][0] * M[2][1] - M[1][1] * M[2][0]);
            g->adv_c[3 * c + j] = dj / det;
        }
    }
    /* P-8: dual area = sum over the fan of (v, x_e(i), c_i) and (v, c_i, x_e(i+1));
     * geofac_rot = d_e * v_os / A*_v (0 in the pentagon pad slot) */
#pragma omp parallel for schedule(static)
    for (int64_t v = 0; v < nv; ++v) {
        int deg = g->v_deg[v];
        const double *pv = V + 3 * v;
        double area = 0.0;
        for (int i = 0; i < deg; ++i) {
            const double *xa = g->edge_xyz + 3 * g->v2e[6 * v + i];
            const double *xb = g->edge_xyz + 3 * g->v2e[6 * v + (i + 1) % deg];
            const double *cc = g->cell_xyz + 3 * g->v2c[6 * v + i];
            area += sph_tri_area(pv, xa, cc);
            area += sph_tri_area(pv, cc, xb);
        }
        g->a_v[v] = area * a * a;
        for (int i = 0; i < 6; ++i)
            g->geofac_rot[6 * v + i] = (i < deg) ? g->d_e[g->v2e[6 * v + i]] * (double)g->v_os[6 * v + i] / g->a_v[v] : 0.0;
    }
    /* P-11: RBF vector reconstruction coefficients for the tangential wind.
     * Gaussian kernel phi(r)=exp(-(r/eps)^2), eps = 4*sqrt(4*pi/Nc);
     * t_e = n_e x x_e (P-4). */
    const double pi = 3.14159265358979323846;
    const double eps = 4.0 * sqrt(4.0 * pi / (double)nc);
#pragma omp parallel for schedule(static)
    for (int64_t e = 0; e < ne; ++e) {
        const double *xe = g->edge_xyz + 3 * e, *nn = g->edge_normal + 3 * e;
        double te[3];
        cross3(nn, xe, te);
        double M[4][4], b[4], c[4];
        for (int i = 0; i < 4; ++i) {
            int32_t si = g->e2e4[4 * e + i];
            const double *xi = g->edge_xyz + 3 * si, *ni = g->edge_normal + 3 * si;
            for (int j = 0; j < 4; ++j) {
                int32_t sj = g->e2e4[4 * e + j];
                const double *xj = g->edge_xyz + 3 * sj, *nj = g->edge_normal + 3 * sj;
                double r = arc3(xi, xj) / eps;
                M[i][j] = exp(-(r * r)) * dot3(ni, nj);
            }
            double r = arc3(xi, xe) / eps;
            b[i] = exp(-(r * r)) * dot3(ni, te);
        }
        og_solve4(M, b, c);
        double s = 0.0;
        for (int i = 0; i < 4; ++i) s += c[i] * dot3(g->edge_normal + 3 * g->e2e4[4 * e + i], te);
        for (int i = 0; i < 4; ++i) g->rbf[4 * e + i] = c[i] / s;
    }
}

/* R2Bk grid, k = 0..9. flags & OG_PERMUTE: seeded renumbering (P-7). */
og_grid *og_grid_create(int k, uint64_t seed, unsigned flags)
{
    if (k < 0 || k > 9) return NULL;
    og_grid *g = (og_grid *)calloc(1, sizeof(og_grid));
    if (!g) return NULL;
    g->level_k = k;
    int64_t nv = 12, nc = 20;
    double *xyz = (double *)malloc(sizeof(double) * 36);
    int32_t *c2v = (int32_t *)malloc(sizeof(int32_t) * 60);
    og_base_icosahedron(xyz, c2v);
    for (int b = 0; b < k + 1; ++b)          /* P-2: R2Bk = k+1 bisections */
        if (og_bisect(&xyz, &nv, &c2v, &nc) != 0) { og_grid_destroy(g); return NULL; }
    int rc = og_build_topology(g, xyz, nv, c2v, nc);
    free(xyz); free(c2v);
    if (rc != 0) { og_grid_destroy(g); return NULL; }
    if (flags & OG_PERMUTE) og_apply_permutation(g, seed);
    og_build_geometry(g);
    return g;
}

/* P-17: a copy of the grid whose floating-point coefficient arrays have been
 * rounded to fp32 once (and are held as fp64 again). Index tables are shared
 * by value (deep-copied) so both grids can be destroyed independently. */
static double *og_round_copy(const double *x, int64_t n)
{
    double *y = (double *)malloc(sizeof(double) * (size_t)n);
    for (int64_t i = 0; i < n; ++i) y[i] = (double)(float)x[i];
    return y;
}
static void *og_dup(const void *x, size_t bytes)
{
    void *y = malloc(bytes);
    memcpy(y, x, bytes);
    return y;
}
og_grid *og_grid_round_f32(const og_grid *s)
{
    og_grid *g = (og_grid *)calloc(1, sizeof(og_grid));
    int64_t nc = s->nc, ne = s->ne, nv = s->nv;
    g->level_k = s->level_k; g->nc = nc; g->ne = ne; g->nv = nv;
    g->c2v = (int32_t *)og_dup(s->c2v, 12 * (size_t)nc);
    g->c2e = (int32_t *)og_dup(s->c2e, 12 * (size_t)nc);
    g->e2c = (int32_t *)og_dup(s->e2c, 8 * (size_t)ne);
    g->e2v = (int32_t *)og_dup(s->e2v, 8 * (size_t)ne);
    g->e2e4 = (int32_t *)og_dup(s->e2e4, 16 * (size_t)ne);
    g->v2e = (int32_t *)og_dup(s->v2e, 24 * (size_t)nv);
    g->v2c = (int32_t *)og_dup(s->v2c, 24 * (size_t)nv);
    g->v_deg = (int32_t *)og_dup(s->v_deg, 4 * (size_t)nv);
    g->c_os = (int8_t *)og_dup(s->c_os, 3 * (size_t)nc);
    g->v_os = (int8_t *)og_dup(s->v_os, 6 * (size_t)nv);
    g->vert_xyz = og_round_copy(s->vert_xyz, 3 * nv);
    g->cell_xyz = og_round_copy(s->cell_xyz, 3 * nc);
    g->edge_xyz = og_round_copy(s->edge_xyz, 3 * ne);
    g->edge_normal = og_round_copy(s->edge_normal, 3 * ne);
    g->l_e = og_round_copy(s->l_e, ne);
    g->d_e = og_round_copy(s->d_e, ne);
    g->inv_d_e = og_round_copy(s->inv_d_e, ne);
    g->f_e = og_round_copy(s->f_e, ne);
    g->c_lin = og_round_copy(s->c_lin, 2 * ne);
    g->cgrad = og_round_copy(s->cgrad, 2 * ne);
    g->rbf = og_round_copy(s->rbf, 4 * ne);
    g->a_c = og_round_copy(s->a_c, nc);
    g->bln = og_round_copy(s->bln, 3 * nc);
    g->adv_c = og_round_copy(s->adv_c, 3 * nc);
    g->a_v = og_round_copy(s->a_v, nv);
    g->geofac_div = og_round_copy(s->geofac_div, 3 * nc);
    g->geofac_rot = og_round_copy(s->geofac_rot, 6 * nv);
    return g;
}

/* ------------------------------------------------------------------ */
/* Operators S1..S7; fields are level-contiguous          */
/* x[i*ldk + k], k = 0 at the top.                                     */
/* Coefficient arrays are passed explicitly so that a test can feed the  */
/* oracle either its own geometry or arrays exported by the library      */
/* (P-18).                                                              */
/* ------------------------------------------------------------------ */

/* S1: div(c,k) = sum_{j<3} geofac_div(c,j) * vn(c2e[c][j],k)
 * m_div = sum of |terms| (P-16 tolerance scale), may be NULL */
void og_divergence(int64_t nc, int nlev, int64_t ldk, const int32_t *c2e, const double *geofac_div,
                   const double *vn, double *div, double *m_div)
{
#pragma omp parallel for schedule(static)
    for (int64_t c = 0; c < nc; ++c)
        for (int k = 0; k < nlev; ++k) {
            double s = 0.0, m = 0.0;
            for (int j = 0; j < 3; ++j) {
                double t = geofac_div[3 * c + j] * vn[(int64_t)c2e[3 * c + j] * ldk + k];
                s += t; m += fabs(t);
            }
            div[c * ldk + k] = s;
            if (m_div) m_div[c * ldk + k] = m;
        }
}

/* S2: zeta(v,k) = sum_{j<6} geofac_rot(v,j) * vn(v2e[v][j],k); pentagon pad has coefficient 0 */
void og_vorticity(int64_t nv, int nlev, int64_t ldk, const int32_t *v2e, const double *geofac_rot,
                  const double *vn, double *vort, double *m_vort)
{
#pragma omp parallel for schedule(static)
    for (int64_t v = 0; v < nv; ++v)
        for (int k = 0; k < nlev; ++k) {
            double s = 0.0, m = 0.0;
            for (int j = 0; j < 6; ++j) {
                double t = geofac_rot[6 * v + j] * vn[(int64_t)v2e[6 * v + j] * ldk + k];
                s += t; m += fabs(t);
            }
            vort[v * ldk + k] = s;
            if (m_vort) m_vort[v * ldk + k] = m;
        }
}

/* S3: vt(e,k) = sum_{j<4} rbf(e,j) * vn(e2e4[e][j],k) */
void og_tangential_wind(int64_t ne, int nlev, int64_t ldk, const int32_t *e2e4, const double *rbf,
                        const double *vn, double *vt)
{
#pragma omp parallel for schedule(static)
    for (int64_t e = 0; e < ne; ++e)
        for (int k = 0; k < nlev; ++k) {
            double s = 0.0;
            for (int j = 0; j < 4; ++j) s += rbf[4 * e + j] * vn[(int64_t)e2e4[4 * e + j] * ldk + k];
            vt[e * ldk + k] = s;
        }
}

/* S4a: KE_e = 1/2 (vn^2 + vt^2) */
void og_kinetic_energy_edge(int64_t ne, int nlev, int64_t ldk, const double *vn, const double *vt, double *ke_e)
{
#pragma omp parallel for schedule(static)
    for (int64_t e = 0; e < ne; ++e)
        for (int k = 0; k < nlev; ++k) {
            double a = vn[e * ldk + k], b = vt[e * ldk + k];
            ke_e[e * ldk + k] = 0.5 * (a * a + b * b);
        }
}

/* S4b: KE_c(c,k) = sum_{j<3} bln(c,j) * KE_e(c2e[c][j],k)   -- PAPER.md:164-167
 * (z_ekinh = sum_j e_bln_c_s(jc,j,jb) * z_kin_hor_e(ieidx(jc,jb,j),jk,ieblk(jc,jb,j)), reading P-15) */
void og_kinetic_energy_cell(int64_t nc, int nlev, int64_t ldk, const int32_t *c2e, const double *bln,
                            const double *ke_e, double *ke_c)
{
#pragma omp parallel for schedule(static)
    for (int64_t c = 0; c < nc; ++c)
        for (int k = 0; k < nlev; ++k) {
            double s = 0.0;
            for (int j = 0; j < 3; ++j) s += bln[3 * c + j] * ke_e[(int64_t)c2e[3 * c + j] * ldk + k];
            ke_c[c * ldk + k] = s;
        }
}

/* P-14: vn interpolated to half level k (0..nlev) of one column.
 * interior: vn_ie(k) = g_k vn(k) + (1-g_k) vn(k-1), g_k = dz_{k-1}/(dz_{k-1}+dz_k);
 * ends: linear extrapolation in z from the two nearest full levels. */
static double og_vn_half(const double *col, int nlev, const double *z_half, int k)
{
    if (k == 0) {
        double zf0 = 0.5 * (z_half[0] + z_half[1]), zf1 = 0.5 * (z_half[1] + z_half[2]);
        return col[0] + (col[0] - col[1]) * (z_half[0] - zf0) / (zf0 - zf1);
    }
    if (k == nlev) {
        double zfa = 0.5 * (z_half[nlev - 1] + z_half[nlev]), zfb = 0.5 * (z_half[nlev - 2] + z_half[nlev - 1]);
        return col[nlev - 1] + (col[nlev - 1] - col[nlev - 2]) * (z_half[nlev] - zfa) / (zfa - zfb);
    }
    double dz_up = z_half[k - 1] - z_half[k], dz_dn = z_half[k] - z_half[k + 1];
    double g = dz_up / (dz_up + dz_dn);
    return g * col[k] + (1.0 - g) * col[k - 1];
}

/* S5 + S6 + S7:
 *   gradK  = (KE_c(c1,k) - KE_c(c0,k)) * inv_d_e
 *   zeta_e = 1/2 (zeta(v0,k) + zeta(v1,k))
 *   H      = gradK + vt * (f_e + zeta_e)
 *   w_f(c,k) = 1/2 (w(c,k) + w(c,k+1)); w_e = c_lin(e,0) w_f(c0,k) + c_lin(e,1) w_f(c1,k)
 *   V      = w_e * (vn_ie(e,k) - vn_ie(e,k+1)) / dz_k
 *   ddt_vn = -(H + V)
 * m_ddt (may be NULL) = P-16 scale:
 *   (|KE_c(c1)|+|KE_c(c0)|) inv_d_e + |vt| (|f_e| + 1/2(|zeta(v0)|+|zeta(v1)|))
 *   + |w_e| (|vn_ie(k)|+|vn_ie(k+1)|)/dz_k                                            */
void og_ddt_vn(int64_t ne, int nlev, int64_t ldk, int64_t ldk_w, const double *z_half,
               const int32_t *e2c, const int32_t *e2v, const double *inv_d_e, const double *f_e,
               const double *c_lin, const double *vn, const double *w, const double *vt,
               const double *ke_c, const double *vort, double *ddt_vn, double *m_ddt)
{
#pragma omp parallel for schedule(static)
    for (int64_t e = 0; e < ne; ++e) {
        int64_t c0 = e2c[2 * e], c1 = e2c[2 * e + 1], v0 = e2v[2 * e], v1 = e2v[2 * e + 1];
        const double *col = vn + e * ldk;
        for (int k = 0; k < nlev; ++k) {
            double gradk = (ke_c[c1 * ldk + k] - ke_c[c0 * ldk + k]) * inv_d_e[e];
            double zeta_e = 0.5 * (vort[v0 * ldk + k] + vort[v1 * ldk + k]);
            double H = gradk + vt[e * ldk + k] * (f_e[e] + zeta_e);
            double wf0 = 0.5 * (w[c0 * ldk_w + k] + w[c0 * ldk_w + k + 1]);
            double wf1 = 0.5 * (w[c1 * ldk_w + k] + w[c1 * ldk_w + k + 1]);
            double w_e = c_lin[2 * e] * wf0 + c_lin[2 * e + 1] * wf1;
            double up = og_vn_half(col, nlev, z_half, k), dn = og_vn_half(col, nlev, z_half, k + 1);
            double dz = z_half[k] - z_half[k + 1];
            double Vt = w_e * (up - dn) / dz;
            ddt_vn[e * ldk + k] = -(H + Vt);
            if (m_ddt)
                m_ddt[e * ldk + k] = (fabs(ke_c[c1 * ldk + k]) + fabs(ke_c[c0 * ldk + k])) * inv_d_e[e]
                    + fabs(vt[e * ldk + k]) * (fabs(f_e[e]) + 0.5 * (fabs(vort[v0 * ldk + k]) + fabs(vort[v1 * ldk + k])))
                    + fabs(w_e) * (fabs(up) + fabs(dn)) / dz;
        }
    }
}

/* Vertical-wind tendency, reading P-19 (the other half of the velocity-tendency routine of
 * the dycore; the paper prints none of it). w lives at cells on the nlev+1 half levels, k = 0 top.
 *   interior half levels k = 1 .. nlev-1:
 *     hadv(c,k) = sum_{j<3} adv_c(c,j) * vn_ie(e_j,k) * (w(c1(e_j),k) - w(c0(e_j),k)) * inv_d_e(e_j),  e_j = c2e[c][j]
 *                 (normal wind interpolated to the half level, P-14; both factors follow the edge's own orientation)
 *     vadv(c,k) = w(c,k) * (w(c,k-1) - w(c,k+1)) / (z_half[k-1] - z_half[k+1])
 *     ddt_w(c,k) = -(hadv + vadv)
 *   k = 0 and k = nlev (model top and surface: boundary conditions of w): ddt_w = 0.
 * m_w (may be NULL) = P-16 scale: sum_j |adv_c| |vn_ie| (|w(c1)|+|w(c0)|) inv_d_e + |w(k)| (|w(k-1)|+|w(k+1)|)/dz. */
void og_ddt_w(int64_t nc, int nlev, int64_t ldk, int64_t ldk_w, const double *z_half, const int32_t *c2e,
              const int32_t *e2c, const double *inv_d_e, const double *adv_c, const double *vn, const double *w,
              double *ddt_w, double *m_w)
{
#pragma omp parallel for schedule(static)
    for (int64_t c = 0; c < nc; ++c) {
        for (int k = 0; k <= nlev; ++k) {
            double val = 0.0, m = 0.0;
            if (k >= 1 && k <= nlev - 1) {
                double hadv = 0.0;
                for (int j = 0; j < 3; ++j) {
                    int64_t e = c2e[3 * c + j];
                    int64_t c0 = e2c[2 * e], c1 = e2c[2 * e + 1];
                    double vie = og_vn_half(vn + e * ldk, nlev, z_half, k);
                    double gw = (w[c1 * ldk_w + k] - w[c0 * ldk_w + k]) * inv_d_e[e];
                    hadv += adv_c[3 * c + j] * vie * gw;
                    m += fabs(adv_c[3 * c + j]) * fabs(vie) * (fabs(w[c1 * ldk_w + k]) + fabs(w[c0 * ldk_w + k])) * inv_d_e[e];
                }
                double dz2 = z_half[k - 1] - z_half[k + 1];
                double vadv = w[c * ldk_w + k] * (w[c * ldk_w + k - 1] - w[c * ldk_w + k + 1]) / dz2;
                m += fabs(w[c * ldk_w + k]) * (fabs(w[c * ldk_w + k - 1]) + fabs(w[c * ldk_w + k + 1])) / dz2;
                val = -(hadv + vadv);
            }
            ddt_w[c * ldk_w + k] = val;
            if (m_w) m_w[c * ldk_w + k] = m;
        }
    }
}

int og_w_tendency(const og_grid *g, int nlev, int64_t ldk, int64_t ldk_w, const double *z_half,
                  const double *vn, const double *w, double *ddt_w, double *m_w)
{
    if (!g || nlev < 2 || ldk < nlev || ldk_w < nlev + 1) return -1;
    for (int k = 0; k < nlev; ++k) if (!(z_half[k] > z_half[k + 1])) return -2;
    og_ddt_w(g->nc, nlev, ldk, ldk_w, z_half, g->c2e, g->e2c, g->inv_d_e, g->adv_c, vn, w, ddt_w, m_w);
    return 0;
}

/* sampled evaluation of ddt_w at (cell idx[i], half level lev[i]), same arithmetic as og_ddt_w */
void og_sample_ddt_w(const og_grid *g, int nlev, int64_t ldk, int64_t ldk_w, const double *z_half,
                     const double *vn, const double *w, int64_t n, const int64_t *idx, const int32_t *lev,
                     double *val, double *scale)
{
#pragma omp parallel for schedule(static)
    for (int64_t i = 0; i < n; ++i) {
        int64_t c = idx[i];
        int k = lev[i];
        double v = 0.0, m = 0.0;
        if (k >= 1 && k <= nlev - 1) {
            double hadv = 0.0;
            for (int j = 0; j < 3; ++j) {
                int64_t e = g->c2e[3 * c + j];
                int64_t c0 = g->e2c[2 * e], c1 = g->e2c[2 * e + 1];
                double vie = og_vn_half(vn + e * ldk, nlev, z_half, k);
                double gw = (w[c1 * ldk_w + k] - w[c0 * ldk_w + k]) * g->inv_d_e[e];
                hadv += g->adv_c[3 * c + j] * vie * gw;
                m += fabs(g->adv_c[3 * c + j]) * fabs(vie) * (fabs(w[c1 * ldk_w + k]) + fabs(w[c0 * ldk_w + k])) * g->inv_d_e[e];
            }
            double dz2 = z_half[k - 1] - z_half[k + 1];
            double vadv = w[c * ldk_w + k] * (w[c * ldk_w + k - 1] - w[c * ldk_w + k + 1]) / dz2;
            m += fabs(w[c * ldk_w + k]) * (fabs(w[c * ldk_w + k - 1]) + fabs(w[c * ldk_w + k + 1])) / dz2;
            v = -(hadv + vadv);
        }
        val[i] = v;
        if (scale) scale[i] = m;
    }
}

/* dycore_div_vort: S1 + S2 */
int og_div_vort(const og_grid *g, int nlev, int64_t ldk, const double *vn, double *div, double *vort,
                double *m_div, double *m_vort)
{
    if (!g || nlev < 1 || ldk < nlev) return -1;
    og_divergence(g->nc, nlev, ldk, g->c2e, g->geofac_div, vn, div, m_div);
    og_vorticity(g->nv, nlev, ldk, g->v2e, g->geofac_rot, vn, vort, m_vort);
    return 0;
}

/* dycore_velocity_tendencies: S3, S4, S2, S5-S7 in that order, every
 * intermediate in a full array. vt, ke_c, vort are caller-provided [n][ldk]
 * work/output arrays (never NULL here); ke_e is allocated internally. */
int og_velocity_tendencies(const og_grid *g, int nlev, int64_t ldk, int64_t ldk_w, const double *z_half,
                           const double *vn, const double *w, double *ddt_vn, double *vt, double *ke_c,
                           double *vort, double *m_ddt)
{
    if (!g || nlev < 2 || ldk < nlev || ldk_w < nlev + 1) return -1;
    for (int k = 0; k < nlev; ++k) if (!(z_half[k] > z_half[k + 1])) return -2;
    double *ke_e = (double *)malloc(sizeof(double) * (size_t)(g->ne * ldk));
    if (!ke_e) return -3;
    og_tangential_wind(g->ne, nlev, ldk, g->e2e4, g->rbf, vn, vt);
    og_kinetic_energy_edge(g->ne, nlev, ldk, vn, vt, ke_e);
    og_kinetic_energy_cell(g->nc, nlev, ldk, g->c2e, g->bln, ke_e, ke_c);
    og_vorticity(g->nv, nlev, ldk, g->v2e, g->geofac_rot, vn, vort, NULL);
    og_ddt_vn(g->ne, nlev, ldk, ldk_w, z_half, g->e2c, g->e2v, g->inv_d_e, g->f_e, g->c_lin,
              vn, w, vt, ke_c, vort, ddt_vn, m_ddt);
    free(ke_e);
    return 0;
}

/* ------------------------------------------------------------------ */
/* Reading P-20: the ICON-faithful metric variant of S5-S7 on the "terrain following hybrid
 * sigma height grid" of PAPER.md:56. The paper prints none of it; the reading is in DESIGN.md section 3.
 *
 * Metric columns per EDGE (inputs of the operator, static in a model run):
 *   wgt_e     [ne][ldk_w] half levels k = 0..nlev: k = 1..nlev-1 weight of vn(k) in vn_ie(k) (vn(k-1) gets 1 - wgt);
 *                         k = 0 and k = nlev: the ratios r of the two-point linear extrapolation
 *                         vn_ie(0) = vn(0) + r (vn(0) - vn(1)),  vn_ie(nlev) = vn(nlev-1) + r (vn(nlev-1) - vn(nlev-2))
 *   inv_ddqz_e[ne][ldk]   1 / layer thickness at the edge
 *   ddxn_z, ddxt_z [ne][ldk]  slopes dz/dn, dz/dt of the full-level coordinate surface at the edge midpoint
 *                             (n = n_e, t = t_e = n_e x x_e, reading P-4)
 * og_metric_from_zhalf derives the first two from the half-level heights of every edge column. */
void og_metric_from_zhalf(int64_t ne, int nlev, int64_t ldk, int64_t ldk_w, const double *z_half_e,
                          double *wgt_e, double *inv_ddqz_e)
{
#pragma omp parallel for schedule(static)
    for (int64_t e = 0; e < ne; ++e) {
        const double *zh = z_half_e + e * ldk_w;
        for (int k = 0; k < nlev; ++k) inv_ddqz_e[e * ldk + k] = 1.0 / (zh[k] - zh[k + 1]);
        for (int k = 1; k <= nlev - 1; ++k) {
            double up = zh[k - 1] - zh[k], dn = zh[k] - zh[k + 1];
            wgt_e[e * ldk_w + k] = up / (up + dn);
        }
        {   /* ends: (z_half - z_full) / (z_full - z_full of the next level inwards) = dz_0 / (dz_0 + dz_1) */
            double d0 = zh[0] - zh[1], d1 = zh[1] - zh[2];
            wgt_e[e * ldk_w] = d0 / (d0 + d1);
            double dl = zh[nlev - 1] - zh[nlev], dm = zh[nlev - 2] - zh[nlev - 1];
            wgt_e[e * ldk_w + nlev] = dl / (dl + dm);
        }
    }
}

/* vn at half level k of one edge column with per-edge weights (P-20) */
static double og_vn_half_metric(const double *col, int nlev, const double *wg, int k)
{
    if (k == 0) return col[0] + wg[0] * (col[0] - col[1]);
    if (k == nlev) return col[nlev - 1] + wg[nlev] * (col[nlev - 1] - col[nlev - 2]);
    return wg[k] * col[k] + (1.0 - wg[k]) * col[k - 1];
}

/* S5-S7, metric variant:
 *   gradK  = cgrad(e,1) KE_c(c1) - cgrad(e,0) KE_c(c0) + KE_e(e) (cgrad(e,0) - cgrad(e,1))      (second-order at x_e)
 *   H      = gradK + vt (f_e + 1/2 (zeta(v0) + zeta(v1)))
 *   w_cc   = vn ddxn_z + vt ddxt_z                  (contravariant correction: the wind's climb along the surface)
 *   V      = (w_e - w_cc) (vn_ie(k) - vn_ie(k+1)) inv_ddqz_e,   w_e as in S6
 *   ddt_vn = -(H + V)
 * m (may be NULL): sum of the absolute values of the terms. */
void og_ddt_vn_metric(int64_t ne, int nlev, int64_t ldk, int64_t ldk_w, const int32_t *e2c, const int32_t *e2v,
                      const double *cgrad, const double *f_e, const double *c_lin, const double *wgt_e,
                      const double *inv_ddqz_e, const double *ddxn_z, const double *ddxt_z, const double *vn,
                      const double *w, const double *vt, const double *ke_e, const double *ke_c, const double *vort,
                      double *ddt_vn, double *m_ddt)
{
#pragma omp parallel for schedule(static)
    for (int64_t e = 0; e < ne; ++e) {
        int64_t c0 = e2c[2 * e], c1 = e2c[2 * e + 1], v0 = e2v[2 * e], v1 = e2v[2 * e + 1];
        const double *col = vn + e * ldk, *wg = wgt_e + e * ldk_w;
        double g0 = cgrad[2 * e], g1 = cgrad[2 * e + 1];
        for (int k = 0; k < nlev; ++k) {
            int64_t i = e * ldk + k;
            double gradk = g1 * ke_c[c1 * ldk + k] - g0 * ke_c[c0 * ldk + k] + ke_e[i] * (g0 - g1);
            double zeta_e = 0.5 * (vort[v0 * ldk + k] + vort[v1 * ldk + k]);
            double H = gradk + vt[i] * (f_e[e] + zeta_e);
            double wf0 = 0.5 * (w[c0 * ldk_w + k] + w[c0 * ldk_w + k + 1]);
            double wf1 = 0.5 * (w[c1 * ldk_w + k] + w[c1 * ldk_w + k + 1]);
            double w_e = c_lin[2 * e] * wf0 + c_lin[2 * e + 1] * wf1;
            double w_cc = vn[i] * ddxn_z[i] + vt[i] * ddxt_z[i];
            double up = og_vn_half_metric(col, nlev, wg, k), dn = og_vn_half_metric(col, nlev, wg, k + 1);
            double Vt = (w_e - w_cc) * (up - dn) * inv_ddqz_e[i];
            ddt_vn[i] = -(H + Vt);
            if (m_ddt)
                m_ddt[i] = g1 * fabs(ke_c[c1 * ldk + k]) + g0 * fabs(ke_c[c0 * ldk + k]) + fabs(ke_e[i]) * fabs(g0 - g1)
                    + fabs(vt[i]) * (fabs(f_e[e]) + 0.5 * (fabs(vort[v0 * ldk + k]) + fabs(vort[v1 * ldk + k])))
                    + (fabs(w_e) + fabs(vn[i] * ddxn_z[i]) + fabs(vt[i] * ddxt_z[i])) * (fabs(up) + fabs(dn)) * inv_ddqz_e[i];
        }
    }
}

int og_velocity_tendencies_metric(const og_grid *g, int nlev, int64_t ldk, int64_t ldk_w, const double *wgt_e,
                                  const double *inv_ddqz_e, const double *ddxn_z, const double *ddxt_z,
                                  const double *vn, const double *w, double *ddt_vn, double *vt, double *ke_c,
                                  double *vort, double *m_ddt)
{
    if (!g || nlev < 3 || ldk < nlev || ldk_w < nlev + 1) return -1;
    double *ke_e = (double *)malloc(sizeof(double) * (size_t)(g->ne * ldk));
    if (!ke_e) return -3;
    og_tangential_wind(g->ne, nlev, ldk, g->e2e4, g->rbf, vn, vt);
    og_kinetic_energy_edge(g->ne, nlev, ldk, vn, vt, ke_e);
    og_kinetic_energy_cell(g->nc, nlev, ldk, g->c2e, g->bln, ke_e, ke_c);
    og_vorticity(g->nv, nlev, ldk, g->v2e, g->geofac_rot, vn, vort, NULL);
    og_ddt_vn_metric(g->ne, nlev, ldk, ldk_w, g->e2c, g->e2v, g->cgrad, g->f_e, g->c_lin, wgt_e, inv_ddqz_e, ddxn_z,
                     ddxt_z, vn, w, vt, ke_e, ke_c, vort, ddt_vn, m_ddt);
    free(ke_e);
    return 0;
}

/* ------------------------------------------------------------------ */
/* One-by-one evaluation of sampled outputs (full-size parity tests):   */
/* the same definitions, evaluated for a single (entity, level) without  */
/* any full-array intermediate.                                         */
/* ------------------------------------------------------------------ */
static double og_pt_vt(const og_grid *g, int64_t ldk, const double *vn, int64_t e, int k)
{
    double s = 0.0;
    for (int j = 0; j < 4; ++j) s += g->rbf[4 * e + j] * vn[(int64_t)g->e2e4[4 * e + j] * ldk + k];
    return s;
}
static double og_pt_ke_c(const og_grid *g, int64_t ldk, const double *vn, int64_t c, int k)
{
    double s = 0.0;
    for (int j = 0; j < 3; ++j) {
        int64_t e = g->c2e[3 * c + j];
        double a = vn[e * ldk + k], b = og_pt_vt(g, ldk, vn, e, k);
        s += g->bln[3 * c + j] * (0.5 * (a * a + b * b));
    }
    return s;
}
static double og_pt_vort(const og_grid *g, int64_t ldk, const double *vn, int64_t v, int k, double *m)
{
    double s = 0.0, mm = 0.0;
    for (int j = 0; j < 6; ++j) {
        double t = g->geofac_rot[6 * v + j] * vn[(int64_t)g->v2e[6 * v + j] * ldk + k];
        s += t; mm += fabs(t);
    }
    if (m) *m = mm;
    return s;
}
void og_sample_div(const og_grid *g, int nlev, int64_t ldk, const double *vn, int64_t n, const int64_t *idx,
                   const int32_t *lev, double *out, double *m_out)
{
    (void)nlev;
    for (int64_t i = 0; i < n; ++i) {
        int64_t c = idx[i]; int k = lev[i];
        double s = 0.0, m = 0.0;
        for (int j = 0; j < 3; ++j) {
            double t = g->geofac_div[3 * c + j] * vn[(int64_t)g->c2e[3 * c + j] * ldk + k];
            s += t; m += fabs(t);
        }
        out[i] = s; m_out[i] = m;
    }
}
void og_sample_vort(const og_grid *g, int nlev, int64_t ldk, const double *vn, int64_t n, const int64_t *idx,
                    const int32_t *lev, double *out, double *m_out)
{
    (void)nlev;
    for (int64_t i = 0; i < n; ++i) out[i] = og_pt_vort(g, ldk, vn, idx[i], lev[i], &m_out[i]);
}
void og_sample_ddt_vn(const og_grid *g, int nlev, int64_t ldk, int64_t ldk_w, const double *z_half,
                      const double *vn, const double *w, int64_t n, const int64_t *idx, const int32_t *lev,
                      double *out, double *m_out)
{
    for (int64_t i = 0; i < n; ++i) {
        int64_t e = idx[i]; int k = lev[i];
        int64_t c0 = g->e2c[2 * e], c1 = g->e2c[2 * e + 1], v0 = g->e2v[2 * e], v1 = g->e2v[2 * e + 1];
        double kc0 = og_pt_ke_c(g, ldk, vn, c0, k), kc1 = og_pt_ke_c(g, ldk, vn, c1, k);
        double z0 = og_pt_vort(g, ldk, vn, v0, k, NULL), z1 = og_pt_vort(g, ldk, vn, v1, k, NULL);
        double vt = og_pt_vt(g, ldk, vn, e, k);
        double gradk = (kc1 - kc0) * g->inv_d_e[e];
        double H = gradk + vt * (g->f_e[e] + 0.5 * (z0 + z1));
        double wf0 = 0.5 * (w[c0 * ldk_w + k] + w[c0 * ldk_w + k + 1]);
        double wf1 = 0.5 * (w[c1 * ldk_w + k] + w[c1 * ldk_w + k + 1]);
        double w_e = g->c_lin[2 * e] * wf0 + g->c_lin[2 * e + 1] * wf1;
        const double *col = vn + e * ldk;
        double up = og_vn_half(col, nlev, z_half, k), dn = og_vn_half(col, nlev, z_half, k + 1);
        double dz = z_half[k] - z_half[k + 1];
        out[i] = -(H + w_e * (up - dn) / dz);
        m_out[i] = (fabs(kc1) + fabs(kc0)) * g->inv_d_e[e] + fabs(vt) * (fabs(g->f_e[e]) + 0.5 * (fabs(z0) + fabs(z1)))
            + fabs(w_e) * (fabs(up) + fabs(dn)) / dz;
    }
}

/* metric variant (P-20), one point at a time: the definitions of og_ddt_vn_metric without any full-array intermediate */
void og_sample_ddt_vn_metric(const og_grid *g, int nlev, int64_t ldk, int64_t ldk_w, const double *wgt_e,
                             const double *inv_ddqz_e, const double *ddxn_z, const double *ddxt_z, const double *vn,
                             const double *w, int64_t n, const int64_t *idx, const int32_t *lev, double *out, double *m_out)
{
    for (int64_t i = 0; i < n; ++i) {
        int64_t e = idx[i]; int k = lev[i];
        int64_t c0 = g->e2c[2 * e], c1 = g->e2c[2 * e + 1], v0 = g->e2v[2 * e], v1 = g->e2v[2 * e + 1];
        double kc0 = og_pt_ke_c(g, ldk, vn, c0, k), kc1 = og_pt_ke_c(g, ldk, vn, c1, k);
        double z0 = og_pt_vort(g, ldk, vn, v0, k, NULL), z1 = og_pt_vort(g, ldk, vn, v1, k, NULL);
        double vt = og_pt_vt(g, ldk, vn, e, k);
        double vne = vn[e * ldk + k];
        double ke_e = 0.5 * (vne * vne + vt * vt);
        double g0 = g->cgrad[2 * e], g1 = g->cgrad[2 * e + 1];
        double gradk = g1 * kc1 - g0 * kc0 + ke_e * (g0 - g1);
        double H = gradk + vt * (g->f_e[e] + 0.5 * (z0 + z1));
        double wf0 = 0.5 * (w[c0 * ldk_w + k] + w[c0 * ldk_w + k + 1]);
        double wf1 = 0.5 * (w[c1 * ldk_w + k] + w[c1 * ldk_w + k + 1]);
        double w_e = g->c_lin[2 * e] * wf0 + g->c_lin[2 * e + 1] * wf1;
        int64_t j = e * ldk + k;
        double w_cc = vne * ddxn_z[j] + vt * ddxt_z[j];
        const double *col = vn + e * ldk, *wg = wgt_e + e * ldk_w;
        double up = og_vn_half_metric(col, nlev, wg, k), dn = og_vn_half_metric(col, nlev, wg, k + 1);
        out[i] = -(H + (w_e - w_cc) * (up - dn) * inv_ddqz_e[j]);
        m_out[i] = g1 * fabs(kc1) + g0 * fabs(kc0) + fabs(ke_e) * fabs(g0 - g1)
            + fabs(vt) * (fabs(g->f_e[e]) + 0.5 * (fabs(z0) + fabs(z1)))
            + (fabs(w_e) + fabs(vne * ddxn_z[j]) + fabs(vt * ddxt_z[j])) * (fabs(up) + fabs(dn)) * inv_ddqz_e[j];
    }
}

/* accessors for the Python wrapper (struct layout stays private to C) */
int64_t og_grid_nc(const og_grid *g) { return g->nc; }
int64_t og_grid_ne(const og_grid *g) { return g->ne; }
int64_t og_grid_nv(const og_grid *g) { return g->nv; }
const void *og_grid_table(const og_grid *g, const char *name)
{
#define T(n) if (!strcmp(name, #n)) return g->n
    T(c2v); T(c2e); T(e2c); T(e2v); T(e2e4); T(v2e); T(v2c); T(v_deg); T(c_os); T(v_os);
    T(vert_xyz); T(cell_xyz); T(edge_xyz); T(edge_normal); T(l_e); T(d_e); T(inv_d_e); T(f_e);
    T(c_lin); T(cgrad); T(rbf); T(a_c); T(bln); T(adv_c); T(a_v); T(geofac_div); T(geofac_rot);
#undef T
    return NULL;
}
