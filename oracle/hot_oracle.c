/*
 * hot_oracle.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * A plain, slow, double-precision CPU statement of what the hot path of 2HOT (Warren, SC'13,
 * arXiv:1310.4502; text in PAPER.md) computes: keys -> sort -> bucket oct-tree -> moments ->
 * per-sink-group walk with an opening criterion -> Plummer-softened particle-particle and
 * Cartesian-multipole particle-cell sums, plus the definition it approximates (direct sum, and
 * the direct Ewald sum for periodic boxes).
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
 * load this file.  It shares no code, header, table or constant generator with the CUDA library
 * under paper_1310_4502_b200/csrc, and neither includes the other.
 *
 * Every function cites the passage it follows.  The paper prints almost none of the hot-path
 * mechanics (it defers to WS93, ref [67]); the readings taken are those of SURVEY.md 8(c) and
 * are listed in DESIGN.md "Readings".  Pins (tests/test_oracle_*.py): two-body closed form,
 * antisymmetry / momentum, uniform-sphere and Plummer-sphere analytic fields, theta->0 tree ==
 * direct sum, finite differences of the Green's function tensors, the (b/r)^(p+1) order law
 * of Fig 6, coverage invariant, tree invariants, brute-force Z-order, and for the
 * periodic part: Ewald constants, lattice symmetry values, tree+images+far-field vs direct Ewald.
 *
 * PARITY UNPINNED against the paper itself (the paper prints no worked force value, key, or
 * list count): key bit order, NLEAF/NCRIT, the integer-geometry MAC, the far-field coefficient
 * route.  They are pinned only by the mathematics above.
 *
 * Build: gcc -O2 -std=c11 -fopenmp -ffp-contract=off -shared -fPIC hot_oracle.c -lm
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define ORC_MAXLEVEL 21
#define ORC_MAXORDER 8
#define ORC_NMOM_MAX 165 /* multi-indices (a,b,c), a+b+c <= 8 */
/* moments are kept through degree g_mom_order (4 unless orc_set_moment_order says 6 or 8: f-3, "through p=8") */
static int g_mom_order = 4;
static int nmom_of(int order) { return (order + 1) * (order + 2) * (order + 3) / 6; }
void orc_set_moment_order(int order) { if (order >= 4 && order <= ORC_MAXORDER) g_mom_order = order; }

typedef struct {
    int64_t n;
    double lo[3], size;
    int periodic, nleaf, ncrit;
    /* particles */
    uint64_t *key;  /* [n] body keys, caller's order */
    uint64_t *skey; /* [n] sorted keys */
    uint32_t *perm; /* [n] sorted position -> caller's index */
    double *x;      /* [n][3] positions in key order */
    double *m;      /* [n] masses in key order */
    /* cells, ascending numeric key (level-major, Morton within a level) */
    int64_t ncells, capcells;
    uint64_t *ckey;
    int32_t *clevel;
    int64_t *cfirst, *ccount;
    uint8_t *cmask;
    int64_t *cchild;  /* index of first child, -1 for a leaf */
    int64_t *cparent; /* -1 for the root */
    /* sink groups in particle order */
    int64_t ngroups;
    int64_t *gcell;
    /* moments about the centre of mass, eq (6): mom[c][k] = sum m d^alpha_k; com[c][3]; bmax[c] */
    int nmom;         /* moments per cell: nmom_of(order they were built through) */
    double *mom, *com, *bmax;
    double *bbound;   /* b_max as the upward pass can carry it: see build_bbound */
    uint8_t *bgdone;  /* lazy trees: 1 where bgmom of the cell is filled */
    double *bgmom;    /* f-1: moments about the cell CENTRE minus those of the uniform cube (build_bg_moments), [ncells][35] */
    int lazy;         /* moments computed on demand, only for the cells a requested group accepts */
    uint8_t *momdone; /* lazy: 1 where mom/com/bmax of the cell are filled */
    /* periodic far field (C-9 step 2), built on demand */
    int far_ready;
    double far_coef[165]; /* coefficient of x^a y^b z^c of psi_sm, a+b+c<=8 (odd ones zero) */
    double far_S[165];    /* global raw moments about the box centre */
} orc_t;

/* ------------------------------------------------------------------------------------------
 * multi-index tables: alpha_k = (a,b,c) ordered by degree, then lexicographic x>y>z:
 * degree 0: 000; degree 1: 100 010 001; degree 2: 200 110 101 020 011 002; ...
 * ---------------------------------------------------------------------------------------- */
static int MI_A[ORC_NMOM_MAX], MI_B[ORC_NMOM_MAX], MI_C[ORC_NMOM_MAX], MI_READY = 0;
static void mi_init(void) {
    if (MI_READY) return;
    int k = 0;
    for (int d = 0; d <= ORC_MAXORDER; ++d)
        for (int a = d; a >= 0; --a)
            for (int b = d - a; b >= 0; --b) {
                MI_A[k] = a; MI_B[k] = b; MI_C[k] = d - a - b; ++k;
            }
    MI_READY = 1;
}
static int g_with_dipole = 0; /* set while background-subtracted cells (expanded about cell centres, f-1) are evaluated */
#pragma omp threadprivate(g_with_dipole)
static int g_soft_kind = 0; /* softening kernel of every routine that takes eps: 0 Plummer, 1 cubic spline (f-4, below) */
static double factorial(int n) { double f = 1; for (int i = 2; i <= n; ++i) f *= i; return f; }

/* ------------------------------------------------------------------------------------------
 * C-2 keys ("mapping of spatial co-ordinates to integer keys described in WS93";
 * north_star: 63-bit Morton + placeholder bit).  The scaling to [0,1) is done in float with one
 * subtract and one multiply (no contraction: -ffp-contract=off), because that sequence is part
 * of the key's definition.  Returns 0, or -1 if a coordinate is outside.
 * ---------------------------------------------------------------------------------------- */
static int key_coords(const float *p, const float lo[3], float inv, uint32_t ic[3]) {
    for (int k = 0; k < 3; ++k) {
        volatile float d = p[k] - lo[k];
        volatile float t = d * inv;
        if (!(t >= 0.0f) || !(t < 1.0f)) return -1;
        float s = floorf(t * 2097152.0f);
        int64_t i = (int64_t)s;
        if (i < 0) i = 0;
        if (i > 2097151) i = 2097151;
        ic[k] = (uint32_t)i;
    }
    return 0;
}
static uint64_t morton_from_coords(const uint32_t ic[3]) {
    uint64_t mkey = 0;
    for (int b = 0; b < ORC_MAXLEVEL; ++b) {
        mkey |= (uint64_t)((ic[0] >> b) & 1u) << (3 * b + 2);
        mkey |= (uint64_t)((ic[1] >> b) & 1u) << (3 * b + 1);
        mkey |= (uint64_t)((ic[2] >> b) & 1u) << (3 * b);
    }
    return mkey | (1ull << 63);
}
int orc_keys(const float *pos, int64_t n, const float lo[3], float size, uint64_t *key) {
    float inv = 1.0f / size;
    for (int64_t i = 0; i < n; ++i) {
        uint32_t ic[3];
        if (key_coords(pos + 3 * i, lo, inv, ic)) return -1;
        key[i] = morton_from_coords(ic);
    }
    return 0;
}
/* integer corner of a cell key at a given level (C-2 step 4): key = 1<<3l | morton>>(63-3l) */
static void key_corner(uint64_t key, int level, int64_t o[3]) {
    uint64_t mort = key & ((1ull << (3 * level)) - 1ull); /* strip placeholder */
    uint32_t ic[3] = {0, 0, 0};
    for (int b = 0; b < level; ++b) {
        ic[0] |= (uint32_t)((mort >> (3 * b + 2)) & 1ull) << b;
        ic[1] |= (uint32_t)((mort >> (3 * b + 1)) & 1ull) << b;
        ic[2] |= (uint32_t)((mort >> (3 * b)) & 1ull) << b;
    }
    for (int k = 0; k < 3; ++k) o[k] = (int64_t)ic[k] << (ORC_MAXLEVEL - level);
}

/* ------------------------------------------------------------------------------------------
 * C-3 stable sort of (key, index): bottom-up merge sort, ties keep ascending original index.
 * ---------------------------------------------------------------------------------------- */
static void stable_sort_keys(const uint64_t *key, int64_t n, uint64_t *skey, uint32_t *perm) {
    uint64_t *ka = malloc(sizeof(uint64_t) * (size_t)n), *kb = malloc(sizeof(uint64_t) * (size_t)n);
    uint32_t *pa = malloc(sizeof(uint32_t) * (size_t)n), *pb = malloc(sizeof(uint32_t) * (size_t)n);
    for (int64_t i = 0; i < n; ++i) { ka[i] = key[i]; pa[i] = (uint32_t)i; }
    for (int64_t w = 1; w < n; w *= 2) {
        for (int64_t s = 0; s < n; s += 2 * w) {
            int64_t mid = s + w < n ? s + w : n, end = s + 2 * w < n ? s + 2 * w : n;
            int64_t i = s, j = mid, o = s;
            while (i < mid && j < end) {
                if (ka[j] < ka[i]) { kb[o] = ka[j]; pb[o++] = pa[j++]; } /* strict: left wins ties */
                else { kb[o] = ka[i]; pb[o++] = pa[i++]; }
            }
            while (i < mid) { kb[o] = ka[i]; pb[o++] = pa[i++]; }
            while (j < end) { kb[o] = ka[j]; pb[o++] = pa[j++]; }
        }
        uint64_t *tk = ka; ka = kb; kb = tk;
        uint32_t *tp = pa; pa = pb; pb = tp;
    }
    memcpy(skey, ka, sizeof(uint64_t) * (size_t)n);
    memcpy(perm, pa, sizeof(uint32_t) * (size_t)n);
    free(ka); free(kb); free(pa); free(pb);
}

/* ------------------------------------------------------------------------------------------
 * C-4 tree: the unique bucket oct-tree of the sorted keys.  Breadth-first with a queue, so the
 * cells come out in ascending numeric key order.  A cell is a leaf iff count <= NLEAF or it is
 * at level 21; otherwise its non-empty octants are its children.
 * ---------------------------------------------------------------------------------------- */
static void cells_reserve(orc_t *t, int64_t want) {
    if (want <= t->capcells) return;
    int64_t cap = t->capcells ? t->capcells : 1024;
    while (cap < want) cap *= 2;
    t->ckey = realloc(t->ckey, sizeof(uint64_t) * (size_t)cap);
    t->clevel = realloc(t->clevel, sizeof(int32_t) * (size_t)cap);
    t->cfirst = realloc(t->cfirst, sizeof(int64_t) * (size_t)cap);
    t->ccount = realloc(t->ccount, sizeof(int64_t) * (size_t)cap);
    t->cmask = realloc(t->cmask, (size_t)cap);
    t->cchild = realloc(t->cchild, sizeof(int64_t) * (size_t)cap);
    t->cparent = realloc(t->cparent, sizeof(int64_t) * (size_t)cap);
    t->capcells = cap;
}
static void build_tree(orc_t *t) {
    cells_reserve(t, 1);
    t->ncells = 1;
    t->ckey[0] = 1; t->clevel[0] = 0; t->cfirst[0] = 0; t->ccount[0] = t->n;
    t->cmask[0] = 0; t->cchild[0] = -1; t->cparent[0] = -1;
    for (int64_t c = 0; c < t->ncells; ++c) { /* the array is the queue */
        int level = t->clevel[c];
        if (t->ccount[c] <= t->nleaf || level == ORC_MAXLEVEL) continue; /* leaf */
        int64_t first = t->cfirst[c], end = first + t->ccount[c];
        int shift = 60 - 3 * level; /* next 3 key bits below this cell's prefix */
        int64_t i = first;
        t->cchild[c] = t->ncells;
        while (i < end) {
            int oct = (int)((t->skey[i] >> shift) & 7ull);
            int64_t j = i;
            while (j < end && (int)((t->skey[j] >> shift) & 7ull) == oct) ++j;
            cells_reserve(t, t->ncells + 1);
            int64_t d = t->ncells++;
            t->ckey[d] = (t->ckey[c] << 3) | (uint64_t)oct;
            t->clevel[d] = level + 1; t->cfirst[d] = i; t->ccount[d] = j - i;
            t->cmask[d] = 0; t->cchild[d] = -1; t->cparent[d] = c;
            t->cmask[c] |= (uint8_t)(1u << oct);
            i = j;
        }
    }
}
/* sink groups: count <= NCRIT (or level 21) and (root or parent count > NCRIT) */
static void build_groups(orc_t *t) {
    int64_t ng = 0;
    int64_t *tmp = malloc(sizeof(int64_t) * (size_t)t->ncells);
    for (int64_t c = 0; c < t->ncells; ++c) {
        int small = t->ccount[c] <= t->ncrit || t->clevel[c] == ORC_MAXLEVEL;
        int top = t->cparent[c] < 0 || t->ccount[t->cparent[c]] > t->ncrit;
        if (small && top) tmp[ng++] = c;
    }
    /* order by first particle (insertion into a position table: groups partition [0,n)) */
    int64_t *at = malloc(sizeof(int64_t) * (size_t)t->n);
    for (int64_t i = 0; i < t->n; ++i) at[i] = -1;
    for (int64_t g = 0; g < ng; ++g) at[t->cfirst[tmp[g]]] = tmp[g];
    t->gcell = malloc(sizeof(int64_t) * (size_t)(ng ? ng : 1));
    t->ngroups = 0;
    for (int64_t i = 0; i < t->n; ++i) if (at[i] >= 0) t->gcell[t->ngroups++] = at[i];
    free(at); free(tmp);
}

/* ------------------------------------------------------------------------------------------
 * C-5 upward pass, eq (6): raw moments about the centre of mass, directly from the
 * cell's particle range.  mom[k] = sum_j m_j dx^a dy^b dz^c for alpha_k = (a,b,c), |alpha| <= 4.
 * ---------------------------------------------------------------------------------------- */
static void cell_moments(orc_t *t, int64_t c) {
    int64_t f = t->cfirst[c], e = f + t->ccount[c];
    double M0 = 0, z[3] = {0, 0, 0};
    for (int64_t j = f; j < e; ++j) {
        M0 += t->m[j];
        for (int k = 0; k < 3; ++k) z[k] += t->m[j] * t->x[3 * j + k];
    }
    for (int k = 0; k < 3; ++k) z[k] /= M0;
    double *mo = t->mom + (size_t)c * t->nmom, bm = 0;
    for (int k = 0; k < t->nmom; ++k) mo[k] = 0;
    for (int64_t j = f; j < e; ++j) {
        double d[3];
        for (int k = 0; k < 3; ++k) d[k] = t->x[3 * j + k] - z[k];
        double r = sqrt(d[0] * d[0] + d[1] * d[1] + d[2] * d[2]);
        if (r > bm) bm = r;
        for (int k = 0; k < t->nmom; ++k)
            mo[k] += t->m[j] * pow(d[0], MI_A[k]) * pow(d[1], MI_B[k]) * pow(d[2], MI_C[k]);
    }
    for (int k = 0; k < 3; ++k) t->com[3 * c + k] = z[k];
    t->bmax[c] = bm;
}
/* b_max of Fig 3 ("sources are contained within a source cell V of radius b_max") as
 * an upward pass carries it (R-15): a leaf's value is the largest distance of one of
 * its bodies from the centre of mass; an internal cell takes, over its children,
 * max(|z_child - z| + b_child), which contains every body of the cell by the triangle
 * inequality.  bmax[] above is the exact radius (directly from the bodies); bbound >= bmax. */
static void build_bbound(orc_t *t) {
    t->bbound = calloc((size_t)t->ncells, sizeof(double));
    for (int64_t c = t->ncells - 1; c >= 0; --c) { /* children have larger indices than parents */
        if (t->cchild[c] < 0) { t->bbound[c] = t->bmax[c]; continue; }
        int nch = 0; for (int b = 0; b < 8; ++b) nch += (t->cmask[c] >> b) & 1;
        double bb = 0;
        for (int k = 0; k < nch; ++k) {
            int64_t d = t->cchild[c] + k;
            double s = 0;
            for (int q = 0; q < 3; ++q) { double u = t->com[3 * d + q] - t->com[3 * c + q]; s += u * u; }
            double v = sqrt(s) + t->bbound[d];
            if (v > bb) bb = v;
        }
        t->bbound[c] = bb;
    }
}
/* with_moments = 1: every cell; 2: none now, orc_tree_forces fills in the cells its groups accept
 * (same cell_moments; for the 2^27-body config, where all 2e7 cells would take hours) */
static void build_moments(orc_t *t, int lazy) {
    mi_init();
    t->nmom = nmom_of(g_mom_order);
    t->mom = calloc((size_t)t->ncells * t->nmom, sizeof(double));
    t->com = calloc((size_t)t->ncells * 3, sizeof(double));
    t->bmax = calloc((size_t)t->ncells, sizeof(double));
    t->lazy = lazy;
    if (lazy) { t->momdone = calloc((size_t)t->ncells, 1); return; }
#pragma omp parallel for schedule(dynamic, 64)
    for (int64_t c = 0; c < t->ncells; ++c) cell_moments(t, c);
    build_bbound(t);
}

/* ------------------------------------------------------------------------------------------
 * create / destroy
 * ---------------------------------------------------------------------------------------- */
void orc_destroy(orc_t *t) {
    if (!t) return;
    free(t->key); free(t->skey); free(t->perm); free(t->x); free(t->m);
    free(t->ckey); free(t->clevel); free(t->cfirst); free(t->ccount); free(t->cmask);
    free(t->cchild); free(t->cparent); free(t->gcell); free(t->mom); free(t->com); free(t->bmax);
    free(t->bbound); free(t->momdone); free(t->bgmom); free(t->bgdone);
    free(t);
}
orc_t *orc_create(const float *pos, const float *mass, int64_t n, const float lo[3], float size,
                  int periodic, int nleaf, int ncrit, int with_moments, int *status) {
    *status = 0;
    if (n < 1 || !(size > 0) || nleaf < 1 || ncrit < nleaf) { *status = -1; return NULL; }
    orc_t *t = calloc(1, sizeof(orc_t));
    t->n = n; t->size = size; t->periodic = periodic; t->nleaf = nleaf; t->ncrit = ncrit;
    for (int k = 0; k < 3; ++k) t->lo[k] = lo[k];
    t->key = malloc(sizeof(uint64_t) * (size_t)n);
    t->skey = malloc(sizeof(uint64_t) * (size_t)n);
    t->perm = malloc(sizeof(uint32_t) * (size_t)n);
    t->x = malloc(sizeof(double) * 3 * (size_t)n);
    t->m = malloc(sizeof(double) * (size_t)n);
    if (orc_keys(pos, n, lo, size, t->key)) { *status = -2; orc_destroy(t); return NULL; }
    stable_sort_keys(t->key, n, t->skey, t->perm);
    for (int64_t i = 0; i < n; ++i) {
        for (int k = 0; k < 3; ++k) t->x[3 * i + k] = (double)pos[3 * (int64_t)t->perm[i] + k];
        t->m[i] = (double)mass[t->perm[i]];
    }
    build_tree(t);
    build_groups(t);
    if (with_moments) build_moments(t, with_moments == 2);
    return t;
}

/* plain getters for the parity tests */
int64_t orc_n(const orc_t *t) { return t->n; }
int64_t orc_ncells(const orc_t *t) { return t->ncells; }
int64_t orc_ngroups(const orc_t *t) { return t->ngroups; }
void orc_get_keys(const orc_t *t, uint64_t *key, uint64_t *skey, uint32_t *perm) {
    if (key) memcpy(key, t->key, sizeof(uint64_t) * (size_t)t->n);
    if (skey) memcpy(skey, t->skey, sizeof(uint64_t) * (size_t)t->n);
    if (perm) memcpy(perm, t->perm, sizeof(uint32_t) * (size_t)t->n);
}
void orc_get_cells(const orc_t *t, uint64_t *key, int32_t *level, int64_t *first, int64_t *count,
                   uint8_t *mask, int64_t *child, int64_t *parent) {
    size_t nc = (size_t)t->ncells;
    if (key) memcpy(key, t->ckey, 8 * nc);
    if (level) memcpy(level, t->clevel, 4 * nc);
    if (first) memcpy(first, t->cfirst, 8 * nc);
    if (count) memcpy(count, t->ccount, 8 * nc);
    if (mask) memcpy(mask, t->cmask, nc);
    if (child) memcpy(child, t->cchild, 8 * nc);
    if (parent) memcpy(parent, t->cparent, 8 * nc);
}
void orc_get_groups(const orc_t *t, int64_t *gcell) {
    memcpy(gcell, t->gcell, sizeof(int64_t) * (size_t)t->ngroups);
}
void orc_get_bbound(const orc_t *t, double *bbound) { memcpy(bbound, t->bbound, 8 * (size_t)t->ncells); }
void orc_get_moments(const orc_t *t, double *mom, double *com, double *bmax) {
    size_t nc = (size_t)t->ncells;
    if (mom) memcpy(mom, t->mom, 8 * nc * (size_t)t->nmom);
    if (com) memcpy(com, t->com, 8 * nc * 3);
    if (bmax) memcpy(bmax, t->bmax, 8 * nc);
}
/* per sorted particle: index of the leaf cell that holds it (cell membership) */
void orc_get_leaf_of(const orc_t *t, int64_t *leaf) {
    for (int64_t c = 0; c < t->ncells; ++c)
        if (t->cchild[c] < 0)
            for (int64_t j = t->cfirst[c]; j < t->cfirst[c] + t->ccount[c]; ++j) leaf[j] = c;
}

/* ------------------------------------------------------------------------------------------
 * C-6 Green's function tensors.  g(R) = (|R|^2 + eps^2)^(-1/2) (Plummer).
 * d^alpha g is obtained from the chain rule exactly as it reads: each derivative either hits
 * the power of u = |R|^2+eps^2 (factor R_i, next D_k) or an R_j already brought down (delta_ij).
 * D_k = (-1)^k (2k-1)!! u^(-(2k+1)/2).  The recursion enumerates every pairing of the index
 * list once: the first remaining index is either unpaired (factor R) or paired with a later one.
 * ---------------------------------------------------------------------------------------- */
static double dg_rec(const int *idx, int nidx, int npairs, int ntot, const double R[3],
                     const double *D) {
    if (nidx == 0) return D[ntot - npairs];
    double s = R[idx[0]] * dg_rec(idx + 1, nidx - 1, npairs, ntot, R, D);
    int rest[12];
    for (int j = 1; j < nidx; ++j) {
        if (idx[j] != idx[0]) continue; /* delta_{i0,ij} */
        int q = 0;
        for (int k = 1; k < nidx; ++k) if (k != j) rest[q++] = idx[k];
        s += dg_rec(rest, nidx - 2, npairs + 1, ntot, R, D);
    }
    return s;
}
static double dg(int a, int b, int c, const double R[3], const double *D) {
    int idx[12], n = 0;
    for (int i = 0; i < a; ++i) idx[n++] = 0;
    for (int i = 0; i < b; ++i) idx[n++] = 1;
    for (int i = 0; i < c; ++i) idx[n++] = 2;
    return dg_rec(idx, n, 0, n, R, D);
}
static void make_D(double u, double *D, int kmax) {
    double dfact = 1; /* (2k-1)!! */
    for (int k = 0; k <= kmax; ++k) {
        if (k > 0) dfact *= (2 * k - 1);
        D[k] = ((k & 1) ? -1.0 : 1.0) * dfact * pow(u, -0.5 * (2 * k + 1));
    }
}
/* exported for the finite-difference pin */
double orc_dg(int a, int b, int c, const double R[3], double eps) {
    double D[12]; make_D(R[0] * R[0] + R[1] * R[1] + R[2] * R[2] + eps * eps, D, a + b + c);
    return dg(a, b, c, R, D);
}

/* eq (5) with Delta = 0 (cell-body), Green's function g, truncated at `order`:
 *   phi(x) = - sum_{|alpha|<=p} ((-1)^|alpha| / alpha!) d^alpha g(R) M_alpha,   R = x - z
 *   a_k(x) = - d_k phi = + sum ... d^(alpha+e_k) g(R) M_alpha
 * (the multi-index form of the n-fold outer product / tensor inner product of eq (5); the minus
 * sign makes phi the potential of attracting masses, G = 1).  The dipole vanishes about the
 * centre of mass; order 0 -> n=0; order 2 -> n=0,2; order 3 -> n<=3; order 4 -> n<=4.        */
static void cell_on_sink(const double *mo, const double z[3], int order, const double x[3],
                         double eps2, double acc[3], double *pot) {
    double R[3] = {x[0] - z[0], x[1] - z[1], x[2] - z[2]}, D[12];
    make_D(R[0] * R[0] + R[1] * R[1] + R[2] * R[2] + (g_soft_kind == 1 ? 0.0 : eps2), D, order + 1);
    for (int k = 0; k < nmom_of(order); ++k) {
        int a = MI_A[k], b = MI_B[k], c = MI_C[k], n = a + b + c;
        if (n > order) break;
        if (n == 1 && !g_with_dipole) continue; /* dipole about the centre of mass is zero by construction */
        double w = ((n & 1) ? -1.0 : 1.0) / (factorial(a) * factorial(b) * factorial(c)) * mo[k];
        *pot -= w * dg(a, b, c, R, D);
        acc[0] += w * dg(a + 1, b, c, R, D);
        acc[1] += w * dg(a, b + 1, c, R, D);
        acc[2] += w * dg(a, b, c + 1, R, D);
    }
}
/* f-4 ("Plummer or spline [50] kernel"): the cubic-spline kernel.  A body is a ball of radius h with
 * density W(u) = 8/(pi h^3) (1 - 6u^2 + 6u^3) for u = r/h <= 1/2, 16/(pi h^3) (1-u)^3 for u <= 1; its field at
 * distance r is  m (y - x) fac(r),  phi = m pot(r)  with, from integrating W (enclosed mass and outer shells):
 *   u <= 1/2: fac h^3 = 32/3 - 192/5 u^2 + 32 u^3,                      pot h = -14/5 + 16/3 u^2 - 48/5 u^4 + 32/5 u^5
 *   u <= 1  : fac h^3 = 64/3 - 48 u + 192/5 u^2 - 32/3 u^3 - 1/(15 u^3), pot h = -16/5 + 1/(15u) + 32/3 u^2 - 16 u^3 + 48/5 u^4 - 32/15 u^5
 *   u >  1  : Newtonian.   h = 2.8 eps makes phi(0) = -m/eps as for Plummer softening.
 * orc_set_softening(1) selects it for every routine that takes eps (direct sum, tree); expansions of accepted cells are
 * then Newtonian, and a cell is accepted only if its cube is farther than h from the group's cube (R-17). */
void orc_set_softening(int kind) { g_soft_kind = kind; }
void orc_spline_kernel(double r, double h, double *fac, double *pot) {
    double u = r / h;
    if (u >= 1.0) { *fac = 1.0 / (r * r * r); *pot = -1.0 / r; return; }
    double u2 = u * u, u3 = u2 * u, h3 = h * h * h;
    if (u <= 0.5) {
        *fac = (32.0 / 3.0 - 192.0 / 5.0 * u2 + 32.0 * u3) / h3;
        *pot = (-14.0 / 5.0 + 16.0 / 3.0 * u2 - 48.0 / 5.0 * u2 * u2 + 32.0 / 5.0 * u2 * u3) / h;
    } else {
        *fac = (64.0 / 3.0 - 48.0 * u + 192.0 / 5.0 * u2 - 32.0 / 3.0 * u3 - 1.0 / (15.0 * u3)) / h3;
        *pot = (-16.0 / 5.0 + 1.0 / (15.0 * u) + 32.0 / 3.0 * u2 - 16.0 * u3 + 48.0 / 5.0 * u2 * u2 - 32.0 / 15.0 * u2 * u3) / h;
    }
}
/* C-1 summand (eq (2) right-hand side, softened): source (y,m) on sink x */
static void body_on_sink(const double y[3], double m, const double x[3], double eps2,
                         double acc[3], double *pot) {
    double d[3] = {y[0] - x[0], y[1] - x[1], y[2] - x[2]};
    if (g_soft_kind == 1) {
        double r = sqrt(d[0] * d[0] + d[1] * d[1] + d[2] * d[2]), h = 2.8 * sqrt(eps2), fac, pp;
        if (r == 0 && h == 0) return; /* coincident, unsoftened: skipped like the self term */
        orc_spline_kernel(r, h, &fac, &pp);
        for (int k = 0; k < 3; ++k) acc[k] += m * d[k] * fac;
        *pot += m * pp;
        return;
    }
    double u = d[0] * d[0] + d[1] * d[1] + d[2] * d[2] + eps2;
    double ri = 1.0 / sqrt(u), ri3 = ri / u;
    for (int k = 0; k < 3; ++k) acc[k] += m * d[k] * ri3;
    *pot -= m * ri;
}
/* exported single interactions (pins O-1, O-7, O-8, O-9) */
void orc_cell_on_sink(const double *mom35, const double z[3], int order, const double x[3],
                      double eps, double acc[3], double *pot) {
    mi_init();
    acc[0] = acc[1] = acc[2] = 0; *pot = 0;
    cell_on_sink(mom35, z, order, x, eps * eps, acc, pot);
}
/* moments of an arbitrary particle set about its centre of mass (same definition as C-5) */
void orc_moments_of_order(const double *y, const double *m, int64_t n, int order, double *mom, double z[3]);
void orc_moments_of(const double *y, const double *m, int64_t n, double *mom35, double z[3]) { orc_moments_of_order(y, m, n, 4, mom35, z); }
void orc_moments_of_order(const double *y, const double *m, int64_t n, int order, double *mom35, double z[3]) {
    const int ORC_NMOM = nmom_of(order);
    mi_init();
    double M0 = 0; z[0] = z[1] = z[2] = 0;
    for (int64_t j = 0; j < n; ++j) { M0 += m[j]; for (int k = 0; k < 3; ++k) z[k] += m[j] * y[3 * j + k]; }
    for (int k = 0; k < 3; ++k) z[k] /= M0;
    for (int k = 0; k < ORC_NMOM; ++k) mom35[k] = 0;
    for (int64_t j = 0; j < n; ++j) {
        double d[3] = {y[3 * j] - z[0], y[3 * j + 1] - z[1], y[3 * j + 2] - z[2]};
        for (int k = 0; k < ORC_NMOM; ++k)
            mom35[k] += m[j] * pow(d[0], MI_A[k]) * pow(d[1], MI_B[k]) * pow(d[2], MI_C[k]);
    }
}

/* ------------------------------------------------------------------------------------------
 * C-1 direct sum over all sources for the listed sinks (caller's indices).  Self term skipped.
 * ---------------------------------------------------------------------------------------- */
void orc_direct(const float *pos, const float *mass, int64_t n, double eps, const int64_t *sinks,
                int64_t ns, double *acc, double *pot) {
    double eps2 = eps * eps;
#pragma omp parallel for schedule(static)
    for (int64_t s = 0; s < ns; ++s) {
        int64_t i = sinks ? sinks[s] : s;
        double x[3] = {pos[3 * i], pos[3 * i + 1], pos[3 * i + 2]}, a[3] = {0, 0, 0}, p = 0;
        for (int64_t j = 0; j < n; ++j) {
            if (j == i) continue;
            double y[3] = {pos[3 * j], pos[3 * j + 1], pos[3 * j + 2]};
            body_on_sink(y, (double)mass[j], x, eps2, a, &p);
        }
        acc[3 * s] = a[0]; acc[3 * s + 1] = a[1]; acc[3 * s + 2] = a[2]; pot[s] = p;
    }
}

/* ------------------------------------------------------------------------------------------
 * C-7 walk with the integer-geometry minimum-distance MAC.  Cells and groups are cubes on the
 * 2^21 grid; the source may be shifted by an image vector (units of 2^21).  Accept iff
 * (double)(sC*sC) < theta2 * (double)d2  with d2 the squared gap between the cubes.
 * ---------------------------------------------------------------------------------------- */
typedef struct {
    const orc_t *t; double theta2; int64_t go[3], gs; int64_t sh[3];
    int64_t npc, npp, covered;       /* counts */
    int64_t *pc, *pp; int64_t cap;   /* optional lists: accepted cells / rejected leaves */
    int64_t nleafrej;
    uint8_t *mark;                   /* optional: set to 1 for every accepted cell */
    double hreal;                    /* spline softening: h = 2.8 eps in the caller's units */
    double hgrid2;                   /* spline softening: (h / grid spacing)^2; an accepted cell lies beyond h (R-17) */
    int bgmode; int64_t klo[3], khi[3]; double rhobar; /* f-1: near cube K_G on the integer grid, mean density */
    int64_t nbg, nvirt;              /* f-1: background-subtracted accepted cells, accepted virtual (empty) cubes */
    double bgvol;                    /* f-1: volume of all subtracted cubes, in grid cells */
    uint8_t *markbg;                 /* optional: set to 1 for every accepted background-subtracted cell */
    int tolmode; double tol; double gc[3], gh; /* error-bound MAC: tolerance, group cube centre and half side */
    int64_t npc_o[3];                /* accepted cells by order: monopole, quadrupole, hexadecapole */
    /* evaluation */
    int eval, order; double eps2; double shx[3];
    int64_t gfirst, gcount; double *acc, *pot; /* [gcount][3], [gcount], group-local */
} walk_t;

static int mac_accept(const walk_t *w, int64_t c) {
    const orc_t *t = w->t;
    int level = t->clevel[c];
    int64_t o[3], s = (int64_t)1 << (ORC_MAXLEVEL - level);
    key_corner(t->ckey[c], level, o);
    uint64_t d2 = 0;
    for (int k = 0; k < 3; ++k) {
        int64_t oc = o[k] + w->sh[k];
        int64_t g1 = oc - (w->go[k] + w->gs), g2 = w->go[k] - (oc + s);
        int64_t g = g1 > g2 ? g1 : g2;
        if (g < 0) g = 0;
        d2 += (uint64_t)(g * g);
    }
    if (g_soft_kind == 1 && !((double)d2 > w->hgrid2)) return 0;
    return (double)((uint64_t)(s * s)) < w->theta2 * (double)d2;
}
/* ------------------------------------------------------------------------------------------
 * f-2: error-bound MAC with per-interaction order (Fig 3).  The paper
 * prints no formula (it cites refs [45, 68]); the reading taken is DESIGN.md R-16.  A cell with
 * expansion centre z (its centre of mass), radius b = bbound and absolute moments
 * B_n = sum_j m_j |y_j - z|^n, truncated after order p, evaluated at distance R > b from z, is off by
 *     |delta a| <= (p+2) B_(p+1) / (R^(p+1) (R - b)^2)
 * (the Legendre series of 1/|R - d| summed beyond order p, each term's gradient bounded by
 * (n+1) |d|^n / R^(n+2); the softened kernel is bounded by the same expression).  About the centre
 * of mass the dipole vanishes, so "monopole" is p = 1.  B_2 = trace M2 and B_4 = M4_iijj are exact
 * from the moments; B_3 <= sqrt(B_2 B_4) (Cauchy-Schwarz) and B_5 <= b B_4.
 * R is the distance from z to the nearest point of the sink group's cube.  The cheapest order in
 * {monopole, quadrupole, hexadecapole} whose bound is <= tol is taken; if none, the cell is opened.
 * Returns 0, 2 or 4, or -1 (open).
 * ---------------------------------------------------------------------------------------- */
double orc_mac_bound(const double *mom35, double b, double R, int p) {
    double B2 = mom35[4] + mom35[7] + mom35[9];
    double B4 = mom35[20] + mom35[30] + mom35[34] + 2.0 * (mom35[23] + mom35[25] + mom35[32]);
    if (!(R > b)) return INFINITY;
    double den = (R - b) * (R - b);
    if (p <= 1) return 3.0 * B2 / (R * R * den);
    if (p == 2) return 4.0 * sqrt(B2 * B4) / (R * R * R * den);
    return 6.0 * b * B4 / (R * R * R * R * R * den);
}
static int mac_tol(const walk_t *w, int64_t c) {
    const orc_t *t = w->t;
    double d2 = 0;
    for (int k = 0; k < 3; ++k) {
        double g = fabs(t->com[3 * c + k] + w->shx[k] - w->gc[k]) - w->gh;
        if (g > 0) d2 += g * g;
    }
    double R = sqrt(d2), b = t->bbound[c];
    if (g_soft_kind == 1 && !(R - b > w->hreal)) return -1; /* every body of the cell beyond h from every sink (R-17) */
    const double *mo = t->mom + (size_t)c * t->nmom;
    if (orc_mac_bound(mo, b, R, 1) <= w->tol) return 0;
    if (orc_mac_bound(mo, b, R, 2) <= w->tol) return 2;
    if (orc_mac_bound(mo, b, R, 4) <= w->tol) return 4;
    return -1;
}
static void walk_rec(walk_t *w, int64_t c) {
    const orc_t *t = w->t;
    int ord = w->order, acc_ = 0;
    if (w->tolmode) { ord = mac_tol(w, c); acc_ = ord >= 0; }
    else acc_ = mac_accept(w, c);
    if (acc_) {
        if (w->tolmode) w->npc_o[ord / 2]++;
        if (w->pc && w->npc < w->cap) w->pc[w->npc] = c;
        w->npc++; w->covered += t->ccount[c];
        if (w->mark) w->mark[c] = 1;
        if (w->eval)
            for (int64_t i = 0; i < w->gcount; ++i) {
                double z[3] = {t->com[3 * c] + w->shx[0], t->com[3 * c + 1] + w->shx[1], t->com[3 * c + 2] + w->shx[2]};
                cell_on_sink(t->mom + (size_t)c * t->nmom, z, ord, t->x + 3 * (w->gfirst + i),
                             w->eps2, w->acc + 3 * i, w->pot + i);
            }
    } else if (t->cchild[c] < 0) {
        if (w->pp && w->nleafrej < w->cap) w->pp[w->nleafrej] = c;
        w->nleafrej++; w->npp += t->ccount[c];
        if (w->eval)
            for (int64_t i = 0; i < w->gcount; ++i)
                for (int64_t j = t->cfirst[c]; j < t->cfirst[c] + t->ccount[c]; ++j) {
                    if (j == w->gfirst + i && w->sh[0] == 0 && w->sh[1] == 0 && w->sh[2] == 0) continue;
                    double y[3] = {t->x[3 * j] + w->shx[0], t->x[3 * j + 1] + w->shx[1], t->x[3 * j + 2] + w->shx[2]};
                    body_on_sink(y, t->m[j], t->x + 3 * (w->gfirst + i), w->eps2, w->acc + 3 * i, w->pot + i);
                }
    } else {
        int nch = 0; for (int b = 0; b < 8; ++b) nch += (t->cmask[c] >> b) & 1;
        for (int k = 0; k < nch; ++k) walk_rec(w, t->cchild[c] + k);
    }
}
static void walk_setup(walk_t *w, const orc_t *t, double theta, int64_t g) {
    memset(w, 0, sizeof(*w));
    w->t = t; w->theta2 = theta * theta;
    int64_t gc = t->gcell[g];
    key_corner(t->ckey[gc], t->clevel[gc], w->go);
    w->gs = (int64_t)1 << (ORC_MAXLEVEL - t->clevel[gc]);
    w->gfirst = t->cfirst[gc]; w->gcount = t->ccount[gc];
}
static int image_range(const orc_t *t) { return t->periodic ? 2 : 0; } /* ws = 2 */

/* list counts per group, summed over the (2ws+1)^3 images when periodic; covered = sum of
 * count(C) over accepted cells + L_pp, which must equal n * (number of images) */
void orc_walk_counts(const orc_t *t, double theta, const int64_t *groups, int64_t ng,
                     int64_t *Lpc, int64_t *Lpp, int64_t *covered) {
    int ws = image_range(t);
#pragma omp parallel for schedule(dynamic, 8)
    for (int64_t q = 0; q < ng; ++q) {
        int64_t g = groups ? groups[q] : q;
        int64_t npc = 0, npp = 0, cov = 0;
        for (int ix = -ws; ix <= ws; ++ix) for (int iy = -ws; iy <= ws; ++iy) for (int iz = -ws; iz <= ws; ++iz) {
            walk_t w; walk_setup(&w, t, theta, g);
            w.sh[0] = (int64_t)ix << ORC_MAXLEVEL; w.sh[1] = (int64_t)iy << ORC_MAXLEVEL; w.sh[2] = (int64_t)iz << ORC_MAXLEVEL;
            walk_rec(&w, 0);
            npc += w.npc; npp += w.npp; cov += w.covered;
        }
        Lpc[q] = npc; Lpp[q] = npp; if (covered) covered[q] = cov;
    }
}
/* the lists themselves for one group and one image (tiny N): accepted cell indices and rejected
 * leaf cell indices, in walk order; returns their numbers through npc / nleaf */
void orc_walk_lists(const orc_t *t, double theta, int64_t g, const int img[3], int64_t cap,
                    int64_t *pc, int64_t *npc, int64_t *leaves, int64_t *nleaf) {
    walk_t w; walk_setup(&w, t, theta, g);
    for (int k = 0; k < 3; ++k) w.sh[k] = (int64_t)img[k] << ORC_MAXLEVEL;
    w.pc = pc; w.pp = leaves; w.cap = cap;
    walk_rec(&w, 0);
    *npc = w.npc; *nleaf = w.nleafrej;
}

/* ------------------------------------------------------------------------------------------
 * C-9 periodic pieces.  psi(r): Green's function of a unit point mass in the unit box plus a
 * uniform neutralising background, zero box mean (Ewald form of ref [25]):
 *   psi(r) = sum_n erfc(alpha|r-n|)/|r-n| + (1/pi) sum_{h!=0} exp(-pi^2 h^2/alpha^2)/h^2 cos(2 pi h.r) - pi/alpha^2
 * alpha = 2, |n_k| <= 4, |h|^2 <= 49.  Positions in units of the box.
 * ---------------------------------------------------------------------------------------- */
#define EW_ALPHA 2.0
#define EW_NR 4
#define EW_H2 49
void orc_ewald_psi(const double r[3], double *psi, double grad[3]) {
    const double al = EW_ALPHA, PI = 3.14159265358979323846;
    double p = -PI / (al * al), g[3] = {0, 0, 0};
    for (int nx = -EW_NR; nx <= EW_NR; ++nx) for (int ny = -EW_NR; ny <= EW_NR; ++ny) for (int nz = -EW_NR; nz <= EW_NR; ++nz) {
        double d[3] = {r[0] - nx, r[1] - ny, r[2] - nz};
        double dd = sqrt(d[0] * d[0] + d[1] * d[1] + d[2] * d[2]);
        if (dd == 0) continue; /* caller handles the singular term */
        p += erfc(al * dd) / dd;
        double f = (erfc(al * dd) + 2 * al * dd / sqrt(PI) * exp(-al * al * dd * dd)) / (dd * dd * dd);
        for (int k = 0; k < 3; ++k) g[k] -= f * d[k];
    }
    int hm = 7;
    for (int hx = -hm; hx <= hm; ++hx) for (int hy = -hm; hy <= hm; ++hy) for (int hz = -hm; hz <= hm; ++hz) {
        int h2 = hx * hx + hy * hy + hz * hz;
        if (h2 == 0 || h2 > EW_H2) continue;
        double ph = 2 * PI * (hx * r[0] + hy * r[1] + hz * r[2]);
        double e = exp(-PI * PI * h2 / (al * al)) / h2;
        p += e / PI * cos(ph);
        double s = -2 * e * sin(ph);
        g[0] += s * hx; g[1] += s * hy; g[2] += s * hz;
    }
    *psi = p; if (grad) { grad[0] = g[0]; grad[1] = g[1]; grad[2] = g[2]; }
}
/* psi_sm(r) = psi(r) - sum_{|n|_inf<=2} 1/|r-n| : analytic for |r_k| < 3 (C-9 step 2) */
static double psi_smooth(const double r[3]) {
    double p; orc_ewald_psi(r, &p, NULL);
    for (int nx = -2; nx <= 2; ++nx) for (int ny = -2; ny <= 2; ++ny) for (int nz = -2; nz <= 2; ++nz) {
        double d[3] = {r[0] - nx, r[1] - ny, r[2] - nz};
        double dd = sqrt(d[0] * d[0] + d[1] * d[1] + d[2] * d[2]);
        if (dd == 0) { /* at r = 0 psi() left the whole n=0 term out; erfc(al r)/r - 1/r -> -2 al/sqrt(pi) */
            p -= 2 * EW_ALPHA / sqrt(3.14159265358979323846);
            continue;
        }
        p -= 1.0 / dd;
    }
    return p;
}
double orc_psi_smooth(const double r[3]) { return psi_smooth(r); }

double orc_ewald_xi(void);
/* direct Ewald sum (the ladder's bottom rung), C-9 "Definition": minimum image
 * softened with Plummer, all other images and the background through psi.  Units: box = size. */
void orc_ewald_direct(const float *pos, const float *mass, int64_t n, double size, double eps,
                      const int64_t *sinks, int64_t ns, double *acc, double *pot) {
    double xi = orc_ewald_xi(); /* lim_{r->0} psi(r) - 1/r */
    double eps1 = eps / size;
#pragma omp parallel for schedule(dynamic, 4)
    for (int64_t s = 0; s < ns; ++s) {
        int64_t i = sinks ? sinks[s] : s;
        double a[3] = {0, 0, 0}, p = 0;
        for (int64_t j = 0; j < n; ++j) {
            if (j == i) continue;
            double r[3], rt[3];
            for (int k = 0; k < 3; ++k) {
                r[k] = ((double)pos[3 * i + k] - (double)pos[3 * j + k]) / size;
                rt[k] = r[k] - floor(r[k] + 0.5);
            }
            double psi, g[3]; orc_ewald_psi(rt, &psi, g); /* psi is periodic: use the minimum image */
            double d2 = rt[0] * rt[0] + rt[1] * rt[1] + rt[2] * rt[2];
            double mj = (double)mass[j];
            if (d2 > 0) {
                double d1 = sqrt(d2), u = d2 + eps1 * eps1;
                p -= mj * (psi - 1.0 / d1 + 1.0 / sqrt(u));
                for (int k = 0; k < 3; ++k) a[k] += mj * (g[k] + rt[k] / (d1 * d2) - rt[k] / (u * sqrt(u)));
            } else { /* coincident distinct bodies: psi() left the singular n=0 term out, whose
                        regular part erfc(a r)/r - 1/r -> -2a/sqrt(pi) must be put back */
                p -= mj * (psi - 2 * EW_ALPHA / sqrt(3.14159265358979323846) + 1.0 / eps1);
                for (int k = 0; k < 3; ++k) a[k] += mj * g[k];
            }
        }
        p -= (double)mass[i] * xi;
        for (int k = 0; k < 3; ++k) acc[3 * s + k] = a[k] / (size * size);
        pot[s] = p / size;
    }
}
double orc_ewald_xi(void) {
    double r0[3] = {0, 0, 0}, p; orc_ewald_psi(r0, &p, NULL);
    return p - 2 * EW_ALPHA / sqrt(3.14159265358979323846);
}

/* far-field table (C-9 step 2; "sums the infinite series of each relevant
 * combination of powers of the co-ordinates ... pre-computed coefficients ... used in a local
 * expansion about the center of the volume", p = 8, ws = 2).  The coefficients are the Taylor
 * coefficients of psi_sm about r = 0 through total degree 8:  c_alpha = d^alpha psi_sm(0)/alpha!.
 * psi_sm = [erfc(al r)/r - 1/r]                      (A: = -erf(al r)/r, a power series in r^2)
 *        + sum_{n!=0} erfc(al|r-n|)/|r-n|            (B: radial function, tensor by the chain rule)
 *        + (1/pi) sum_h w_h cos(2 pi h.r)            (C: power series of the cosine)
 *        - pi/al^2                                   (D)
 *        - sum_{0<|n|_inf<=2} 1/|r-n|                (E: the 124 explicit cubes, eps = 0)
 * For a radial f(d) the chain-rule recursion dg_rec applies with D_k = (1/d d/dd)^k f:
 * for f = erfc(al d)/d, D_k = (-1)^k B_k, B_0 = f, B_k = ((2k-1) B_(k-1) + (2 al^2)^k e^(-al^2 d^2)/(al sqrt(pi)))/d^2.
 * far_coef is indexed over all (a,b,c), a+b+c<=8, degree-major; odd ones are zero by symmetry. */
static int far_index(int a, int b, int c) { /* position of (a,b,c) in degree-major order */
    int d = a + b + c, k = 0;
    for (int dd = 0; dd < d; ++dd) k += (dd + 1) * (dd + 2) / 2;
    for (int aa = d; aa > a; --aa) k += d - aa + 1;
    return k + (d - a - b);
}
static void far_build_table(orc_t *t) {
    const double al = EW_ALPHA, PI = 3.14159265358979323846;
    for (int k = 0; k < 165; ++k) t->far_coef[k] = 0;
    for (int deg = 0; deg <= 8; deg += 2)
        for (int a = deg; a >= 0; a -= 2) for (int b = deg - a; b >= 0; b -= 2) {
            int c = deg - a - b, m = deg / 2;
            double afac = factorial(a) * factorial(b) * factorial(c), co = 0;
            /* A */
            co += -(2 * al / sqrt(PI)) * ((m & 1) ? -1.0 : 1.0) * pow(al, 2 * m) / (factorial(m) * (2 * m + 1))
                  * factorial(m) / (factorial(a / 2) * factorial(b / 2) * factorial(c / 2));
            /* B and E */
            for (int nx = -EW_NR; nx <= EW_NR; ++nx) for (int ny = -EW_NR; ny <= EW_NR; ++ny) for (int nz = -EW_NR; nz <= EW_NR; ++nz) {
                if (!nx && !ny && !nz) continue;
                double R[3] = {-(double)nx, -(double)ny, -(double)nz};
                double d2 = R[0] * R[0] + R[1] * R[1] + R[2] * R[2], d = sqrt(d2), D[10];
                double B = erfc(al * d) / d, ex = exp(-al * al * d2) / (al * sqrt(PI));
                D[0] = B;
                for (int k = 1; k <= deg; ++k) { B = ((2 * k - 1) * B + pow(2 * al * al, k) * ex) / d2; D[k] = (k & 1) ? -B : B; }
                co += dg(a, b, c, R, D) / afac;
                if (abs(nx) <= 2 && abs(ny) <= 2 && abs(nz) <= 2) { make_D(d2, D, deg); co -= dg(a, b, c, R, D) / afac; }
            }
            /* C */
            for (int hx = -7; hx <= 7; ++hx) for (int hy = -7; hy <= 7; ++hy) for (int hz = -7; hz <= 7; ++hz) {
                int h2 = hx * hx + hy * hy + hz * hz;
                if (h2 == 0 || h2 > EW_H2) continue;
                double w = exp(-PI * PI * h2 / (al * al)) / h2 / PI;
                co += w * ((m & 1) ? -1.0 : 1.0) * pow(2 * PI, 2 * m) * pow(hx, a) * pow(hy, b) * pow(hz, c) / afac;
            }
            /* D */
            if (deg == 0) co -= PI / (al * al);
            t->far_coef[far_index(a, b, c)] = co;
        }
}
static void far_prepare(orc_t *t) {
    if (t->far_ready) return;
    far_build_table(t);
    /* global raw moments about the box centre, box units: S_abc = sum m (x-c)^a (y-c)^b (z-c)^c */
    for (int k = 0; k < 165; ++k) t->far_S[k] = 0;
    for (int64_t j = 0; j < t->n; ++j) {
        double d[3];
        for (int k = 0; k < 3; ++k) d[k] = (t->x[3 * j + k] - (t->lo[k] + 0.5 * t->size)) / t->size;
        for (int deg = 0, q = 0; deg <= 8; ++deg)
            for (int a = deg; a >= 0; --a) for (int b = deg - a; b >= 0; --b, ++q)
                t->far_S[q] += t->m[j] * pow(d[0], a) * pow(d[1], b) * pow(d[2], deg - a - b);
    }
    t->far_ready = 1;
}
void orc_far_table(orc_t *t, double *coef165) { far_prepare(t); memcpy(coef165, t->far_coef, sizeof(double) * 165); }
/* sum_j m_j psi_sm(x - x_j) and its gradient at x, by the binomial expansion of every monomial
 * (x - x_j)^alpha = sum_beta C(alpha,beta) (x-c)^(alpha-beta) (-(x_j-c))^beta  (C-9 step 2) */
static double binom(int n, int k) { return factorial(n) / (factorial(k) * factorial(n - k)); }
static void far_on_sink(const orc_t *t, const double x[3], double *val, double grad[3]) {
    double d[3];
    for (int k = 0; k < 3; ++k) d[k] = (x[k] - (t->lo[k] + 0.5 * t->size)) / t->size;
    double v = 0, g[3] = {0, 0, 0};
    for (int deg = 0, q = 0; deg <= 8; ++deg)
        for (int a = deg; a >= 0; --a) for (int b = deg - a; b >= 0; --b, ++q) {
            int c = deg - a - b; double co = t->far_coef[q];
            if (co == 0) continue;
            for (int i = 0; i <= a; ++i) for (int j = 0; j <= b; ++j) for (int k = 0; k <= c; ++k) {
                double S = t->far_S[far_index(i, j, k)];
                double w = co * binom(a, i) * binom(b, j) * binom(c, k) * (((i + j + k) & 1) ? -1.0 : 1.0) * S;
                int pa = a - i, pb = b - j, pc = c - k;
                v += w * pow(d[0], pa) * pow(d[1], pb) * pow(d[2], pc);
                if (pa) g[0] += w * pa * pow(d[0], pa - 1) * pow(d[1], pb) * pow(d[2], pc);
                if (pb) g[1] += w * pb * pow(d[0], pa) * pow(d[1], pb - 1) * pow(d[2], pc);
                if (pc) g[2] += w * pc * pow(d[0], pa) * pow(d[1], pb) * pow(d[2], pc - 1);
            }
        }
    *val = v; grad[0] = g[0]; grad[1] = g[1]; grad[2] = g[2];
}

/* ------------------------------------------------------------------------------------------
 * C-8 tree evaluation for the listed groups (all if groups == NULL).  Results go to acc[n][3],
 * pot[n] in the CALLER's particle order; entries of particles outside the listed groups are left
 * untouched.  Periodic: 125 explicit images (Plummer g on every explicit term) + far field
 * (a = +grad, phi = -value; the j = i term stays in, C-9 step 3).
 * ---------------------------------------------------------------------------------------- */
void orc_tree_forces(orc_t *t, double theta, double eps, int order, const int64_t *groups,
                     int64_t ng, double *acc, double *pot, int64_t *Lpc, int64_t *Lpp) {
    mi_init();
    int ws = image_range(t);
    if (t->periodic) far_prepare(t);
    if (!groups) ng = t->ngroups;
    if (t->lazy) { /* moments of the cells these groups accept: mark them (walk only), then fill them in */
        uint8_t *need = calloc((size_t)t->ncells, 1);
#pragma omp parallel for schedule(dynamic, 4)
        for (int64_t q = 0; q < ng; ++q)
            for (int ix = -ws; ix <= ws; ++ix) for (int iy = -ws; iy <= ws; ++iy) for (int iz = -ws; iz <= ws; ++iz) {
                walk_t w; walk_setup(&w, t, theta, groups ? groups[q] : q);
                w.sh[0] = (int64_t)ix << ORC_MAXLEVEL; w.sh[1] = (int64_t)iy << ORC_MAXLEVEL; w.sh[2] = (int64_t)iz << ORC_MAXLEVEL;
                w.mark = need; w.hreal = 2.8 * eps; w.hgrid2 = (w.hreal * 2097152.0 / t->size) * (w.hreal * 2097152.0 / t->size);
                walk_rec(&w, 0);
            }
#pragma omp parallel for schedule(dynamic, 1)
        for (int64_t c = 0; c < t->ncells; ++c)
            if (need[c] && !t->momdone[c]) { cell_moments(t, c); t->momdone[c] = 1; }
        free(need);
    }
#pragma omp parallel for schedule(dynamic, 4)
    for (int64_t q = 0; q < ng; ++q) {
        int64_t g = groups ? groups[q] : q;
        walk_t w; walk_setup(&w, t, theta, g);
        int64_t nG = w.gcount, npc = 0, npp = 0;
        double *a = calloc((size_t)nG * 3, sizeof(double)), *p = calloc((size_t)nG, sizeof(double));
        for (int ix = -ws; ix <= ws; ++ix) for (int iy = -ws; iy <= ws; ++iy) for (int iz = -ws; iz <= ws; ++iz) {
            walk_setup(&w, t, theta, g);
            w.sh[0] = (int64_t)ix << ORC_MAXLEVEL; w.sh[1] = (int64_t)iy << ORC_MAXLEVEL; w.sh[2] = (int64_t)iz << ORC_MAXLEVEL;
            w.shx[0] = ix * t->size; w.shx[1] = iy * t->size; w.shx[2] = iz * t->size;
            w.eval = 1; w.order = order; w.eps2 = eps * eps; w.acc = a; w.pot = p;
            w.hreal = 2.8 * eps; w.hgrid2 = (w.hreal * 2097152.0 / t->size) * (w.hreal * 2097152.0 / t->size);
            walk_rec(&w, 0);
            npc += w.npc; npp += w.npp;
        }
        if (Lpc) Lpc[q] = npc;
        if (Lpp) Lpp[q] = npp;
        for (int64_t i = 0; i < nG; ++i) {
            int64_t s = w.gfirst + i, o = (int64_t)t->perm[s];
            if (t->periodic) {
                double v, gr[3]; far_on_sink(t, t->x + 3 * s, &v, gr);
                p[i] -= v / t->size;
                for (int k = 0; k < 3; ++k) a[3 * i + k] += gr[k] / (t->size * t->size);
            }
            for (int k = 0; k < 3; ++k) acc[3 * o + k] = a[3 * i + k];
            pot[o] = p[i];
        }
        free(a); free(p);
    }
}

/* ------------------------------------------------------------------------------------------
 * f-1: per-cell background subtraction (Fig 2; reading DESIGN.md R-18).  Periodic
 * boxes only: rhobar = total mass / size^3.
 *  - For sink group G the NEAR CUBE K_G is the 5 x 5 x 5 block of cells of G's level centred on G.
 *    Inside it the walk is the usual one ("the bodies inside cell a interact with the bodies and cells
 *    inside the gray shaded area as usual").
 *  - A cell outside K_G that the criterion accepts interacts through its moments about the cell CENTRE
 *    minus those of a cube of density rhobar, through the same order p ("we only want to subtract the
 *    uniform background expansion up to the same order as the multipole expansion of the matter"); the
 *    dipole is present.  Empty octants of opened cells and the cubes of rejected leaves outside K_G
 *    ("empty cell c ... must have its background contribution subtracted as well") become VIRTUAL cubes
 *    carrying only the negative background; one that the criterion rejects is subdivided.  Cells that
 *    straddle K_G are opened (a straddling leaf: its bodies directly, its cube as a virtual cube whose
 *    parts inside K_G are dropped).  So the subtracted cubes tile exactly (5 size)^3 minus K_G.
 *  - "The background contribution of the gray shaded area ... is removed analytically": what was
 *    subtracted is added back in closed form, rhobar x [field of the homogeneous (5 size)^3 cube - field
 *    of the homogeneous cube K_G] (orc_cube_field: "the analytic expression for the force inside a
 *    uniform cube").
 * ---------------------------------------------------------------------------------------- */
static double cube_moment_1d(int a, double s) { return (a & 1) ? 0.0 : 2.0 * pow(0.5 * s, a + 1) / (a + 1); } /* int_{-s/2}^{s/2} x^a dx */
void orc_cube_moments(double side, double *mom35) { /* raw moments of a unit-density cube about its centre */
    mi_init();
    for (int k = 0; k < 35; ++k) mom35[k] = cube_moment_1d(MI_A[k], side) * cube_moment_1d(MI_B[k], side) * cube_moment_1d(MI_C[k], side);
}
static void bg_cell_moments(orc_t *t, int64_t c, double rhobar) {
    const double h = t->size / 2097152.0;
    int64_t o[3]; key_corner(t->ckey[c], t->clevel[c], o);
    double side = (double)((int64_t)1 << (ORC_MAXLEVEL - t->clevel[c])) * h, ctr[3], cube[35];
    for (int k = 0; k < 3; ++k) ctr[k] = t->lo[k] + (double)o[k] * h + 0.5 * side;
    orc_cube_moments(side, cube);
    double *mo = t->bgmom + (size_t)c * 35;
    for (int k = 0; k < 35; ++k) mo[k] = 0;
    for (int64_t j = t->cfirst[c]; j < t->cfirst[c] + t->ccount[c]; ++j) {
        double d[3]; for (int k = 0; k < 3; ++k) d[k] = t->x[3 * j + k] - ctr[k];
        for (int k = 0; k < 35; ++k) mo[k] += t->m[j] * pow(d[0], MI_A[k]) * pow(d[1], MI_B[k]) * pow(d[2], MI_C[k]);
    }
    for (int k = 0; k < 35; ++k) mo[k] -= rhobar * cube[k];
}
static double total_mass(const orc_t *t) { double M = 0; for (int64_t j = 0; j < t->n; ++j) M += t->m[j]; return M; }
static void build_bg_moments(orc_t *t) { /* every cell, or (lazy trees) none now: orc_tree_forces_bg fills in what its groups accept */
    if (t->bgmom) return;
    mi_init();
    t->bgmom = calloc((size_t)t->ncells * 35, sizeof(double));
    if (t->lazy) { t->bgdone = calloc((size_t)t->ncells, 1); return; }
    double rhobar = total_mass(t) / (t->size * t->size * t->size);
#pragma omp parallel for schedule(dynamic, 64)
    for (int64_t c = 0; c < t->ncells; ++c) bg_cell_moments(t, c, rhobar);
}
/* potential (= -int dy / |x - y|) and acceleration (towards the mass) at x of the homogeneous unit-density cube
 * [lo, lo + side)^3, inside or outside: sum over the corners (X,Y,Z) = corner - x with sign (-1)^(i+j+k) of
 *   F  = XY ln(Z+r) + YZ ln(X+r) + ZX ln(Y+r) - (X^2 atan(YZ/(Xr)) + Y^2 atan(ZX/(Yr)) + Z^2 atan(XY/(Zr))) / 2,
 *   dF = Y ln(Z+r) + Z ln(Y+r) - X atan(YZ/(Xr))     (x component; cyclic for y, z)
 * (refs [59, 46] of the paper; pinned by quadrature in tests/test_oracle_pins.py). */
static double cube_F_l(double a, double b, double c, double r) { return a * b == 0 ? 0.0 : a * b * log(c + r); }
static double cube_F_t(double a, double b, double c, double r) { return a == 0 ? 0.0 : 0.5 * a * a * atan(b * c / (a * r)); }
static double cube_dF(double X, double Y, double Z, double r) {
    return (Y == 0 ? 0.0 : Y * log(Z + r)) + (Z == 0 ? 0.0 : Z * log(Y + r)) - (X == 0 ? 0.0 : X * atan(Y * Z / (X * r)));
}
void orc_cube_field(const double x[3], const double lo[3], double side, double *phi, double acc[3]) {
    double f = 0, g[3] = {0, 0, 0};
    for (int i = 0; i < 2; ++i) for (int j = 0; j < 2; ++j) for (int k = 0; k < 2; ++k) {
        double X = lo[0] + i * side - x[0], Y = lo[1] + j * side - x[1], Z = lo[2] + k * side - x[2];
        double r = sqrt(X * X + Y * Y + Z * Z), sg = ((i + j + k) & 1) ? -1.0 : 1.0;
        f += sg * (cube_F_l(X, Y, Z, r) + cube_F_l(Y, Z, X, r) + cube_F_l(Z, X, Y, r) - cube_F_t(X, Y, Z, r) - cube_F_t(Y, Z, X, r) - cube_F_t(Z, X, Y, r));
        g[0] += sg * cube_dF(X, Y, Z, r); g[1] += sg * cube_dF(Y, Z, X, r); g[2] += sg * cube_dF(Z, X, Y, r);
    }
    *phi = f; acc[0] = g[0]; acc[1] = g[1]; acc[2] = g[2];
}
/* where a cube [o, o+s)^3 of the integer grid lies relative to K_G: 0 inside, 1 outside, 2 straddling */
static int bg_where(const walk_t *w, const int64_t o[3], int64_t s) {
    int inside = 1;
    for (int k = 0; k < 3; ++k) {
        if (o[k] + s <= w->klo[k] || o[k] >= w->khi[k]) return 1;
        if (o[k] < w->klo[k] || o[k] + s > w->khi[k]) inside = 0;
    }
    return inside ? 0 : 2;
}
static int bg_mac(const walk_t *w, const int64_t oc[3], int64_t s) { /* the criterion of R-7 on a cube given by corner (image shift applied) and side */
    uint64_t d2 = 0;
    for (int k = 0; k < 3; ++k) {
        int64_t g1 = oc[k] - (w->go[k] + w->gs), g2 = w->go[k] - (oc[k] + s);
        int64_t g = g1 > g2 ? g1 : g2;
        if (g < 0) g = 0;
        d2 += (uint64_t)(g * g);
    }
    return (double)((uint64_t)(s * s)) < w->theta2 * (double)d2;
}
/* a virtual cube: only the negative background.  level, corner o (unshifted; the image shift is w->sh) */
static void bg_virtual(walk_t *w, int level, const int64_t o[3]) {
    const orc_t *t = w->t;
    int64_t s = (int64_t)1 << (ORC_MAXLEVEL - level), oc[3] = {o[0] + w->sh[0], o[1] + w->sh[1], o[2] + w->sh[2]};
    int where = bg_where(w, oc, s);
    if (where == 0) return;
    if (where == 1 && (bg_mac(w, oc, s) || level == ORC_MAXLEVEL)) {
        w->nvirt++; w->bgvol += (double)s * (double)s * (double)s;
        if (w->eval) {
            double h = t->size / 2097152.0, side = (double)s * h, cube[35], ctr[3];
            orc_cube_moments(side, cube);
            for (int k = 0; k < 35; ++k) cube[k] *= -w->rhobar;
            for (int k = 0; k < 3; ++k) ctr[k] = t->lo[k] + (double)oc[k] * h + 0.5 * side;
            g_with_dipole = 1;
            for (int64_t i = 0; i < w->gcount; ++i)
                cell_on_sink(cube, ctr, w->order, t->x + 3 * (w->gfirst + i), w->eps2, w->acc + 3 * i, w->pot + i);
            g_with_dipole = 0;
        }
        return;
    }
    for (int q = 0; q < 8; ++q) {
        int64_t oo[3] = {o[0] + ((q >> 2) & 1) * (s / 2), o[1] + ((q >> 1) & 1) * (s / 2), o[2] + (q & 1) * (s / 2)};
        bg_virtual(w, level + 1, oo);
    }
}
static void walk_bg(walk_t *w, int64_t c) {
    const orc_t *t = w->t;
    int level = t->clevel[c];
    int64_t o[3], s = (int64_t)1 << (ORC_MAXLEVEL - level), oc[3];
    key_corner(t->ckey[c], level, o);
    for (int k = 0; k < 3; ++k) oc[k] = o[k] + w->sh[k];
    int where = bg_where(w, oc, s);
    int accept = where != 2 && mac_accept(w, c);
    if (accept) {
        w->npc++;
        if (where == 1) { w->nbg++; w->bgvol += (double)s * (double)s * (double)s; if (w->markbg) w->markbg[c] = 1; }
        else if (w->mark) w->mark[c] = 1;
        if (w->eval) {
            if (where == 1) { /* background-subtracted, about the cell centre, dipole included */
                double h = t->size / 2097152.0, side = (double)s * h, ctr[3];
                for (int k = 0; k < 3; ++k) ctr[k] = t->lo[k] + (double)oc[k] * h + 0.5 * side;
                g_with_dipole = 1;
                for (int64_t i = 0; i < w->gcount; ++i)
                    cell_on_sink(t->bgmom + (size_t)c * 35, ctr, w->order < 1 ? 1 : w->order, t->x + 3 * (w->gfirst + i), w->eps2, w->acc + 3 * i, w->pot + i); /* about the centre the dipole is the leading correction: order 0 keeps it */
                g_with_dipole = 0;
            } else
                for (int64_t i = 0; i < w->gcount; ++i) {
                    double z[3] = {t->com[3 * c] + w->shx[0], t->com[3 * c + 1] + w->shx[1], t->com[3 * c + 2] + w->shx[2]};
                    cell_on_sink(t->mom + (size_t)c * t->nmom, z, w->order, t->x + 3 * (w->gfirst + i), w->eps2, w->acc + 3 * i, w->pot + i);
                }
        }
        return;
    }
    if (t->cchild[c] < 0) { /* a rejected leaf: its bodies directly; outside K_G its cube's background separately */
        w->npp += t->ccount[c];
        if (w->eval)
            for (int64_t i = 0; i < w->gcount; ++i)
                for (int64_t j = t->cfirst[c]; j < t->cfirst[c] + t->ccount[c]; ++j) {
                    if (j == w->gfirst + i && w->sh[0] == 0 && w->sh[1] == 0 && w->sh[2] == 0) continue;
                    double y[3] = {t->x[3 * j] + w->shx[0], t->x[3 * j + 1] + w->shx[1], t->x[3 * j + 2] + w->shx[2]};
                    body_on_sink(y, t->m[j], t->x + 3 * (w->gfirst + i), w->eps2, w->acc + 3 * i, w->pot + i);
                }
        if (where != 0) bg_virtual(w, level, o);
        return;
    }
    int k = 0;
    for (int q = 0; q < 8; ++q) {
        if ((t->cmask[c] >> q) & 1) { walk_bg(w, t->cchild[c] + k); ++k; }
        else if (where != 0) { /* an empty octant outside (or across) K_G */
            int64_t oo[3] = {o[0] + ((q >> 2) & 1) * (s / 2), o[1] + ((q >> 1) & 1) * (s / 2), o[2] + (q & 1) * (s / 2)};
            bg_virtual(w, level + 1, oo);
        }
    }
}
void orc_tree_forces_bg(orc_t *t, double theta, double eps, int order, const int64_t *groups, int64_t ng,
                        double *acc, double *pot, int64_t *Lpc, int64_t *Lbg, int64_t *Lvirt, int64_t *Lpp, double *Vol) {
    mi_init();
    if (!t->periodic || order > 4) return;
    far_prepare(t);
    build_bg_moments(t);
    if (!groups) ng = t->ngroups;
    const double rhobar = total_mass(t) / (t->size * t->size * t->size), h = t->size / 2097152.0;
    if (t->lazy) { /* the moments (both kinds) of the cells these groups accept: mark them (walk only), then fill them in */
        uint8_t *need = calloc((size_t)t->ncells, 1), *needbg = calloc((size_t)t->ncells, 1);
#pragma omp parallel for schedule(dynamic, 4)
        for (int64_t q = 0; q < ng; ++q)
            for (int ix = -2; ix <= 2; ++ix) for (int iy = -2; iy <= 2; ++iy) for (int iz = -2; iz <= 2; ++iz) {
                walk_t w; walk_setup(&w, t, theta, groups ? groups[q] : q);
                w.sh[0] = (int64_t)ix << ORC_MAXLEVEL; w.sh[1] = (int64_t)iy << ORC_MAXLEVEL; w.sh[2] = (int64_t)iz << ORC_MAXLEVEL;
                w.bgmode = 1; w.mark = need; w.markbg = needbg;
                for (int k = 0; k < 3; ++k) { w.klo[k] = w.go[k] - 2 * w.gs; w.khi[k] = w.go[k] + 3 * w.gs; }
                walk_bg(&w, 0);
            }
#pragma omp parallel for schedule(dynamic, 1)
        for (int64_t c = 0; c < t->ncells; ++c) {
            if (need[c] && !t->momdone[c]) { cell_moments(t, c); t->momdone[c] = 1; }
            if (needbg[c] && !t->bgdone[c]) { bg_cell_moments(t, c, rhobar); t->bgdone[c] = 1; }
        }
        free(need); free(needbg);
    }
#pragma omp parallel for schedule(dynamic, 4)
    for (int64_t q = 0; q < ng; ++q) {
        int64_t g = groups ? groups[q] : q;
        walk_t w; walk_setup(&w, t, theta, g);
        int64_t nG = w.gcount, npc = 0, nbg = 0, nv = 0, npp = 0;
        double vol = 0;
        double *a = calloc((size_t)nG * 3, sizeof(double)), *p = calloc((size_t)nG, sizeof(double));
        for (int ix = -2; ix <= 2; ++ix) for (int iy = -2; iy <= 2; ++iy) for (int iz = -2; iz <= 2; ++iz) {
            walk_setup(&w, t, theta, g);
            w.sh[0] = (int64_t)ix << ORC_MAXLEVEL; w.sh[1] = (int64_t)iy << ORC_MAXLEVEL; w.sh[2] = (int64_t)iz << ORC_MAXLEVEL;
            w.shx[0] = ix * t->size; w.shx[1] = iy * t->size; w.shx[2] = iz * t->size;
            w.eval = acc != NULL; w.order = order; w.eps2 = eps * eps; w.acc = a; w.pot = p;
            w.bgmode = 1; w.rhobar = rhobar;
            for (int k = 0; k < 3; ++k) { w.klo[k] = w.go[k] - 2 * w.gs; w.khi[k] = w.go[k] + 3 * w.gs; }
            walk_bg(&w, 0);
            npc += w.npc; nbg += w.nbg; nv += w.nvirt; npp += w.npp; vol += w.bgvol;
        }
        if (Vol) Vol[q] = vol / (2097152.0 * 2097152.0 * 2097152.0); /* in units of the box volume */
        if (Lpc) Lpc[q] = npc;
        if (Lbg) Lbg[q] = nbg;
        if (Lvirt) Lvirt[q] = nv;
        if (Lpp) Lpp[q] = npp;
        if (acc) {
            double big_lo[3], k_lo[3], kside = 5.0 * (double)w.gs * h;
            for (int k = 0; k < 3; ++k) { big_lo[k] = t->lo[k] - 2.0 * t->size; k_lo[k] = t->lo[k] + (double)(w.go[k] - 2 * w.gs) * h; }
            for (int64_t i = 0; i < nG; ++i) {
                int64_t sidx = w.gfirst + i, o = (int64_t)t->perm[sidx];
                double v, gr[3]; far_on_sink(t, t->x + 3 * sidx, &v, gr);
                p[i] -= v / t->size;
                for (int k = 0; k < 3; ++k) a[3 * i + k] += gr[k] / (t->size * t->size);
                /* what was subtracted, added back in closed form: rhobar x (homogeneous (5 size)^3 cube - homogeneous K_G) */
                double pb, ab[3], pk, ak[3];
                orc_cube_field(t->x + 3 * sidx, big_lo, 5.0 * t->size, &pb, ab);
                orc_cube_field(t->x + 3 * sidx, k_lo, kside, &pk, ak);
                p[i] += rhobar * (pb - pk);
                for (int k = 0; k < 3; ++k) a[3 * i + k] += rhobar * (ab[k] - ak[k]);
                for (int k = 0; k < 3; ++k) acc[3 * o + k] = a[3 * i + k];
                pot[o] = p[i];
            }
        }
        free(a); free(p);
    }
}

/* f-2: the same evaluation with the error-bound MAC; list counts per order (summed over images) */
void orc_tree_forces_tol(orc_t *t, double tol, double eps, const int64_t *groups, int64_t ng,
                         double *acc, double *pot, int64_t *Lpc0, int64_t *Lpc2, int64_t *Lpc4, int64_t *Lpp) {
    mi_init();
    int ws = image_range(t);
    if (t->periodic) far_prepare(t);
    if (!groups) ng = t->ngroups;
#pragma omp parallel for schedule(dynamic, 4)
    for (int64_t q = 0; q < ng; ++q) {
        int64_t g = groups ? groups[q] : q;
        walk_t w; walk_setup(&w, t, 0.0, g);
        int64_t nG = w.gcount, n0 = 0, n2 = 0, n4 = 0, npp = 0;
        double *a = calloc((size_t)nG * 3, sizeof(double)), *p = calloc((size_t)nG, sizeof(double));
        for (int ix = -ws; ix <= ws; ++ix) for (int iy = -ws; iy <= ws; ++iy) for (int iz = -ws; iz <= ws; ++iz) {
            walk_setup(&w, t, 0.0, g);
            w.sh[0] = (int64_t)ix << ORC_MAXLEVEL; w.sh[1] = (int64_t)iy << ORC_MAXLEVEL; w.sh[2] = (int64_t)iz << ORC_MAXLEVEL;
            w.shx[0] = ix * t->size; w.shx[1] = iy * t->size; w.shx[2] = iz * t->size;
            w.eval = acc != NULL; w.eps2 = eps * eps; w.acc = a; w.pot = p;
            w.hreal = 2.8 * eps; w.hgrid2 = (w.hreal * 2097152.0 / t->size) * (w.hreal * 2097152.0 / t->size);
            w.tolmode = 1; w.tol = tol;
            double h = t->size / 2097152.0; /* grid spacing: the group's cube from its integer corner and side */
            w.gh = 0.5 * (double)w.gs * h;
            for (int k = 0; k < 3; ++k) w.gc[k] = t->lo[k] + ((double)w.go[k] + 0.5 * (double)w.gs) * h;
            walk_rec(&w, 0);
            n0 += w.npc_o[0]; n2 += w.npc_o[1]; n4 += w.npc_o[2]; npp += w.npp;
        }
        if (Lpc0) Lpc0[q] = n0;
        if (Lpc2) Lpc2[q] = n2;
        if (Lpc4) Lpc4[q] = n4;
        if (Lpp) Lpp[q] = npp;
        if (acc)
            for (int64_t i = 0; i < nG; ++i) {
                int64_t s = w.gfirst + i, o = (int64_t)t->perm[s];
                if (t->periodic) {
                    double v, gr[3]; far_on_sink(t, t->x + 3 * s, &v, gr);
                    p[i] -= v / t->size;
                    for (int k = 0; k < 3; ++k) a[3 * i + k] += gr[k] / (t->size * t->size);
                }
                for (int k = 0; k < 3; ++k) acc[3 * o + k] = a[3 * i + k];
                pot[o] = p[i];
            }
        free(a); free(p);
    }
}
/* f-4 (the "drift" and "kick" operators of the symplectic integrator; their time factors -- in a comoving
 * background integrals over the expansion history -- are the caller's): v <- v + a dtk, then x <- x + v dtd, in fp32 with
 * one fused multiply-add each (so that a GPU does the same bits); periodic boxes wrap x back into [lo, lo + size). */
void orc_kick_drift(float *pos, float *vel, const float *acc, int64_t n, float dtk, float dtd,
                    const float lo[3], float size, int periodic) {
    for (int64_t i = 0; i < 3 * n; ++i) {
        float v = fmaf(acc[i], dtk, vel[i]);
        float x = fmaf(v, dtd, pos[i]);
        if (periodic) {
            float l = lo[i % 3];
            volatile float t = x - l;
            volatile float q = floorf(t / size);
            x = fmaf(-q, size, t) + l;
            if (x >= l + size) x = l;          /* rounding may land on the upper face */
            if (x < l) x = l;
        }
        vel[i] = v; pos[i] = x;
    }
}
/* thread count of the OpenMP loops (bench.py times the oracle with 1 thread and with all cores) */
void orc_set_num_threads(int n) {
#ifdef _OPENMP
    if (n > 0) omp_set_num_threads(n);
#else
    (void)n;
#endif
}
int orc_num_threads(void) {
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}
