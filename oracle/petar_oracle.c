/*
 * petar_oracle.c -- fp64 CPU ORACLE for the long-range P3T force path of PeTar
 *                   (arxiv 2006.16560; citations are PAPER.md:<line>).
 *
 * THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT.  It is a plain, slow, obviously
 * correct restatement of what the path computes.  Only tests/, __graft_entry__.smoke()
 * and bench.py's cpu_baseline / --impl reference leg may call it.  It shares no
 * source, header, table or helper with the CUDA path under paper_2006_16560_b200/.
 *
 * Two halves:
 *  (A) DEFINITIONS (tree-free, the exact result):  Eq. 11 with the
 *      changeover functions of Eq. 15-17 and the pairwise maxima of the
 *      radii, as O(N^2) direct sums; the neighbour definition
 *      r_ij < max(r_out,i, r_out,j) (north_star "inside r_out").
 *  (B) ALGORITHM (theta > 0): Barnes-Hut tree with opening angle theta and
 *      centre-of-mass super-particles with multipoles.  The paper
 *      delegates the tree to FDPS and describes none of it, so the
 *      construction rules O1-O9 below are the readings listed in DESIGN.md.
 *
 * Pins (tests/test_oracle_*.py): Eq. 19 boundary values, Eq. 18 as a second formula,
 * long+short = Newton (Eq. 7), sum m_i a_i = 0, neighbour symmetry, theta=0 tree ==
 * direct sum, partition invariants of the walk, Plummer potential energy -1/2.
 * Part (C): Eq. 24 search radii, the Kepler-pericentre filter and the
 * clustering; pinned by conic closed forms (r_p = a(1-e), a(e-1), impact parameter), r_p <= r,
 * symmetry, C_V -> infinity == rule O9, tree == O(N^2) definition, components against scipy.
 * Part (D) (rank 4): short-range acceleration, jerk and potential over the neighbour rows; pinned by
 * the O(N^2) short-range definition of part (A), dK/dx against a difference quotient of Eq. 17, the
 * jerk against a difference quotient of the acceleration along x + v t, Newton's two-body jerk
 * inside r_in, and sum m a = sum m j = 0.
 * The acceptance RULE of the walk (visit(): l^2 < theta^2 d^2, l = cube edge, d = group box to centre of
 * mass, reading P8) is pinned by a hand-worked dyadic geometry in which the cell flips at theta = 4/sqrt(116.8125)
 * (tests/test_oracle_tree.py::test_opening_criterion_flips_at_hand_computed_theta).
 * Parity UNPINNED (the paper prints nothing to pin them to): the NUMBERS that follow from it on a real
 * workload -- interaction counts and force error at theta > 0 (only monotonicity sanity checks).
 *
 * Floating point: everything is IEEE double.  Build with -ffp-contract=off so that the
 * compiler fuses nothing; fma() is called explicitly where rule O5/O7/O9 says so.
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

typedef struct {
    double G;          /* gravitational constant (1 in Henon units)      */
    double theta;      /* opening angle                                        */
    double rho;        /* r_in / r_out, 0.1                                    */
    int32_t multipole; /* 1 monopole, 2 quadrupole                             */
    int32_t n_leaf;    /* leaf capacity (8)                                                   */
    int32_t n_group;   /* i-group capacity (64)                                               */
    int32_t pad;
} ora_params;

/* ------------------------------------------------------------------------------------ */
/* (A) changeover functions                                                             */
/* ------------------------------------------------------------------------------------ */

/* Eq. 16: f(x) = 1 + Lambda x^5 (14 - 28x + 20x^2 - 5x^3) */
double ora_f(double x, double Lam) {
    double x5 = x * x * x * x * x;
    return 1.0 + Lam * x5 * (14.0 - 28.0 * x + 20.0 * x * x - 5.0 * x * x * x);
}

/* Eq. 15: potential changeover W(x) (the SHORT-range weight) */
double ora_W(double x, double Lam) {
    if (x >= 1.0) return 0.0;
    if (x <= 0.0) return Lam * (1.0 - 2.0 * x);
    return Lam * (1.0 - 2.0 * x) - 1.0 + ora_f(x, Lam);
}

/* Eq. 17: force changeover K(x) (the SHORT-range weight) */
double ora_K(double x, double Lam) {
    if (x >= 1.0) return 0.0;
    if (x <= 0.0) return 1.0;
    double xm = x - 1.0;
    double xm4 = xm * xm * xm * xm;
    return xm4 * (1.0 + 4.0 * x + 10.0 * x * x + 20.0 * x * x * x + 35.0 * Lam * x * x * x * x);
}

/* One pair of Eq. 11 (reading P1: H_L = -sum_{i<j} G m_i m_j (1-W)/r_ij).
 * d = r_j - r_i.  Adds to a[3], *phi the LONG-range (wl=1) or SHORT-range (wl=0) part.
 * R_ij = max(r_out,i, r_out,j), r_in,ij = rho R_ij, x and Lambda per Eq. 16.
 * r = 0 (coincident particles, reading P4): no force; (1-W)/r -> 2/(R+r_in), W/r -> +inf
 * is not representable, so the short-range potential of a coincident pair is skipped.          */
static void pair_split(double dx, double dy, double dz, double mj, double Ri, double Rj,
                       const ora_params *p, int want_long, double *a, double *phi) {
    double R = Ri > Rj ? Ri : Rj;
    double rin = p->rho * R;
    double r2 = dx * dx + dy * dy + dz * dz;
    double r = sqrt(r2);
    double Lam = (R - rin) / (R + rin);
    double x = (r - rin) / (R - rin);
    if (r == 0.0) {
        if (want_long) *phi -= p->G * mj * 2.0 / (R + rin);
        return;
    }
    double K = ora_K(x, Lam), W = ora_W(x, Lam);
    double wf = want_long ? (1.0 - K) : K;
    double wp = want_long ? (1.0 - W) : W;
    double r3 = r2 * r;
    a[0] += p->G * mj * wf * dx / r3;
    a[1] += p->G * mj * wf * dy / r3;
    a[2] += p->G * mj * wf * dz / r3;
    *phi -= p->G * mj * wp / r;
}

/* Direct sums over all j != i for the targets tgt[0..nt) (tgt == NULL: targets are 0..nt-1).
 * which: 0 = Newtonian, 1 = long-range part, 2 = short-range part.  out arrays have length nt. */
void ora_direct(int64_t N, const double *x, const double *y, const double *z, const double *m,
                const double *rout, const ora_params *p, int which, int64_t nt, const int64_t *tgt,
                double *ax, double *ay, double *az, double *pot) {
#pragma omp parallel for schedule(dynamic, 16)
    for (int64_t t = 0; t < nt; ++t) {
        int64_t i = tgt ? tgt[t] : t;
        double a[3] = {0, 0, 0}, phi = 0;
        for (int64_t j = 0; j < N; ++j) {
            if (j == i) continue;
            double dx = x[j] - x[i], dy = y[j] - y[i], dz = z[j] - z[i];
            if (which == 0) {
                double r2 = dx * dx + dy * dy + dz * dz;
                if (r2 == 0.0) continue;
                double r = sqrt(r2);
                a[0] += p->G * m[j] * dx / (r2 * r);
                a[1] += p->G * m[j] * dy / (r2 * r);
                a[2] += p->G * m[j] * dz / (r2 * r);
                phi -= p->G * m[j] / r;
            } else {
                pair_split(dx, dy, dz, m[j], rout[i], rout[j], p, which == 1, a, &phi);
            }
        }
        ax[t] = a[0]; ay[t] = a[1]; az[t] = a[2]; pot[t] = phi;
    }
}

/* Neighbour definition, O(N^2): NB(i) = { j != i : r_ij < max(rs_i, rs_j) }, rs = search radius
 * (= r_out on this path).  r2 is formed as in rule O9.  Two-phase: indices == NULL => only counts.
 * offsets has N+1 entries; rows are in ascending j.                                              */
void ora_neighbors_direct(int64_t N, const double *x, const double *y, const double *z,
                          const double *rs, int64_t *offsets, int32_t *indices) {
    if (!indices) {
#pragma omp parallel for schedule(dynamic, 64)
        for (int64_t i = 0; i < N; ++i) {
            int64_t c = 0;
            for (int64_t j = 0; j < N; ++j) {
                if (j == i) continue;
                double dx = x[i] - x[j], dy = y[i] - y[j], dz = z[i] - z[j];
                double r2 = fma(dz, dz, fma(dy, dy, dx * dx));
                double R = rs[i] > rs[j] ? rs[i] : rs[j];
                if (r2 < R * R) ++c;
            }
            offsets[i + 1] = c;
        }
        offsets[0] = 0;
        for (int64_t i = 0; i < N; ++i) offsets[i + 1] += offsets[i];
        return;
    }
#pragma omp parallel for schedule(dynamic, 64)
    for (int64_t i = 0; i < N; ++i) {
        int64_t o = offsets[i];
        for (int64_t j = 0; j < N; ++j) {
            if (j == i) continue;
            double dx = x[i] - x[j], dy = y[i] - y[j], dz = z[i] - z[j];
            double r2 = fma(dz, dz, fma(dy, dy, dx * dx));
            double R = rs[i] > rs[j] ? rs[i] : rs[j];
            if (r2 < R * R) indices[o++] = (int32_t)j;
        }
    }
}

/* ------------------------------------------------------------------------------------ */
/* (B) the tree algorithm, rules O1-O9                            */
/* ------------------------------------------------------------------------------------ */

#define ORA_MAXLEVEL 21

typedef struct {
    int32_t level;
    int32_t leaf;
    int64_t begin, end;      /* range in sorted order */
    int32_t nchild;
    int32_t child[8];        /* indices into the node array (DFS order) */
    double M, S[3], com[3], lo[3], hi[3], rmax, Q[6]; /* Q: xx yy zz xy xz yz about com */
    double edge;             /* geometric edge of the cell's cube, 2h / 2^level */
    int64_t canon;           /* rank in (level, begin) order */
} ora_node;

typedef struct {
    int64_t begin, end;
    double lo[3], hi[3], rmax;
} ora_group;

typedef struct {
    ora_params p;
    int64_t N;
    double c[3], h;           /* root cube centre and half edge (O1) */
    uint64_t *key;            /* sorted keys */
    int32_t *perm;            /* sorted position -> original index */
    double *x, *y, *z, *m, *rout, *rs; /* sorted copies; rs = search radius */
    ora_node *node; int64_t n_node, cap_node;
    int64_t *canon2dfs;       /* canonical id -> DFS index */
    ora_group *grp; int64_t n_grp, cap_grp;
    int32_t *grp_of;          /* sorted position -> group */
} ora_tree;

static void *xmalloc(size_t n) { void *p = malloc(n ? n : 1); if (!p) abort(); return p; }

/* O3: 63-bit Morton key; bit 3b+2 = bit b of qx, 3b+1 of qy, 3b of qz. */
static uint64_t morton63(uint64_t qx, uint64_t qy, uint64_t qz) {
    uint64_t k = 0;
    for (int b = 0; b < ORA_MAXLEVEL; ++b) {
        k |= ((qx >> b) & 1ull) << (3 * b + 2);
        k |= ((qy >> b) & 1ull) << (3 * b + 1);
        k |= ((qz >> b) & 1ull) << (3 * b);
    }
    return k;
}

typedef struct { uint64_t key; int32_t idx; } keyidx;
static int cmp_keyidx(const void *a, const void *b) {
    const keyidx *p = (const keyidx *)a, *q = (const keyidx *)b;
    if (p->key != q->key) return p->key < q->key ? -1 : 1;
    return (p->idx > q->idx) - (p->idx < q->idx);      /* O4: ties by original index */
}

static int64_t new_node(ora_tree *t) {
    if (t->n_node == t->cap_node) {
        t->cap_node = t->cap_node ? 2 * t->cap_node : 1024;
        t->node = (ora_node *)realloc(t->node, (size_t)t->cap_node * sizeof(ora_node));
        if (!t->node) abort();
    }
    memset(&t->node[t->n_node], 0, sizeof(ora_node));
    return t->n_node++;
}

/* O5: node (level, [b,e)); leaf iff e-b <= n_leaf or level == 21; otherwise one child per distinct
 * next-3-bit value present, ascending.  Moments in the fixed order of O5.                         */
static int64_t build_node(ora_tree *t, int level, int64_t b, int64_t e) {
    int64_t id = new_node(t);
    ora_node nd; memset(&nd, 0, sizeof nd);
    nd.level = level; nd.begin = b; nd.end = e;
    nd.edge = ldexp(2.0 * t->h, -level);
    nd.leaf = (e - b <= t->p.n_leaf) || level == ORA_MAXLEVEL;
    for (int k = 0; k < 3; ++k) { nd.lo[k] = INFINITY; nd.hi[k] = -INFINITY; }
    if (nd.leaf) {
        double M = 0, S0 = 0, S1 = 0, S2 = 0, rmax = 0;
        for (int64_t i = b; i < e; ++i) {          /* members in sorted order */
            M = M + t->m[i];
            S0 = fma(t->m[i], t->x[i], S0);
            S1 = fma(t->m[i], t->y[i], S1);
            S2 = fma(t->m[i], t->z[i], S2);
            if (t->x[i] < nd.lo[0]) nd.lo[0] = t->x[i];
            if (t->y[i] < nd.lo[1]) nd.lo[1] = t->y[i];
            if (t->z[i] < nd.lo[2]) nd.lo[2] = t->z[i];
            if (t->x[i] > nd.hi[0]) nd.hi[0] = t->x[i];
            if (t->y[i] > nd.hi[1]) nd.hi[1] = t->y[i];
            if (t->z[i] > nd.hi[2]) nd.hi[2] = t->z[i];
            if (t->rs[i] > rmax) rmax = t->rs[i];
        }
        nd.M = M; nd.S[0] = S0; nd.S[1] = S1; nd.S[2] = S2; nd.rmax = rmax;
    } else {
        int shift = 3 * (ORA_MAXLEVEL - (level + 1));
        int64_t i = b;
        double M = 0, S0 = 0, S1 = 0, S2 = 0, rmax = 0;
        while (i < e) {
            uint64_t oct = (t->key[i] >> shift) & 7ull;
            int64_t j = i + 1;
            while (j < e && ((t->key[j] >> shift) & 7ull) == oct) ++j;
            int64_t c = build_node(t, level + 1, i, j);     /* may realloc t->node */
            nd.child[nd.nchild++] = (int32_t)c;
            const ora_node *cn = &t->node[c];
            M = M + cn->M;                                   /* children ascending */
            S0 = S0 + cn->S[0]; S1 = S1 + cn->S[1]; S2 = S2 + cn->S[2];
            for (int k = 0; k < 3; ++k) {
                if (cn->lo[k] < nd.lo[k]) nd.lo[k] = cn->lo[k];
                if (cn->hi[k] > nd.hi[k]) nd.hi[k] = cn->hi[k];
            }
            if (cn->rmax > rmax) rmax = cn->rmax;
            i = j;
        }
        nd.M = M; nd.S[0] = S0; nd.S[1] = S1; nd.S[2] = S2; nd.rmax = rmax;
    }
    if (nd.M != 0.0) {
        for (int k = 0; k < 3; ++k) nd.com[k] = nd.S[k] / nd.M;
    } else {                                        /* massless cell: centre of its cube */
        uint64_t prefix = level ? (t->key[b] >> (3 * (ORA_MAXLEVEL - level))) : 0;
        uint64_t q[3] = {0, 0, 0};
        for (int l = 0; l < level; ++l) {
            uint64_t d = (prefix >> (3 * (level - 1 - l))) & 7ull;
            q[0] = (q[0] << 1) | ((d >> 2) & 1); q[1] = (q[1] << 1) | ((d >> 1) & 1); q[2] = (q[2] << 1) | (d & 1);
        }
        for (int k = 0; k < 3; ++k) nd.com[k] = (t->c[k] - t->h) + ((double)q[k] + 0.5) * nd.edge;
    }
    /* quadrupole about com, Eq. 30: Q = sum m (x-com)(x-com)^T, summed over members */
    for (int64_t i = b; i < e; ++i) {
        double dx = t->x[i] - nd.com[0], dy = t->y[i] - nd.com[1], dz = t->z[i] - nd.com[2], mi = t->m[i];
        nd.Q[0] += mi * dx * dx; nd.Q[1] += mi * dy * dy; nd.Q[2] += mi * dz * dz;
        nd.Q[3] += mi * dx * dy; nd.Q[4] += mi * dx * dz; nd.Q[5] += mi * dy * dz;
    }
    t->node[id] = nd;
    return id;
}

static void add_group(ora_tree *t, int64_t b, int64_t e) {
    if (t->n_grp == t->cap_grp) {
        t->cap_grp = t->cap_grp ? 2 * t->cap_grp : 1024;
        t->grp = (ora_group *)realloc(t->grp, (size_t)t->cap_grp * sizeof(ora_group));
        if (!t->grp) abort();
    }
    ora_group g; g.begin = b; g.end = e; g.rmax = 0;
    for (int k = 0; k < 3; ++k) { g.lo[k] = INFINITY; g.hi[k] = -INFINITY; }
    for (int64_t i = b; i < e; ++i) {
        if (t->x[i] < g.lo[0]) g.lo[0] = t->x[i];
        if (t->y[i] < g.lo[1]) g.lo[1] = t->y[i];
        if (t->z[i] < g.lo[2]) g.lo[2] = t->z[i];
        if (t->x[i] > g.hi[0]) g.hi[0] = t->x[i];
        if (t->y[i] > g.hi[1]) g.hi[1] = t->y[i];
        if (t->z[i] > g.hi[2]) g.hi[2] = t->z[i];
        if (t->rs[i] > g.rmax) g.rmax = t->rs[i];
        t->grp_of[i] = (int32_t)t->n_grp;
    }
    t->grp[t->n_grp++] = g;
}

/* O6: top-down; a node with count <= n_group is a group; an over-full level-21 leaf is cut into
 * consecutive chunks of n_group; otherwise descend.  DFS visits ranges in ascending order, so
 * groups come out numbered by range start.                                                       */
static void make_groups(ora_tree *t, int64_t id) {
    const ora_node *nd = &t->node[id];
    int64_t cnt = nd->end - nd->begin;
    if (cnt <= t->p.n_group) { add_group(t, nd->begin, nd->end); return; }
    if (nd->leaf) {
        for (int64_t b = nd->begin; b < nd->end; b += t->p.n_group) {
            int64_t e = b + t->p.n_group < nd->end ? b + t->p.n_group : nd->end;
            add_group(t, b, e);
        }
        return;
    }
    for (int k = 0; k < nd->nchild; ++k) make_groups(t, t->node[id].child[k]);
}

typedef struct { int64_t lvl, beg, idx; } canon_key;
static int cmp_canon(const void *a, const void *b) {
    const canon_key *p = (const canon_key *)a, *q = (const canon_key *)b;
    if (p->lvl != q->lvl) return p->lvl < q->lvl ? -1 : 1;
    return (p->beg > q->beg) - (p->beg < q->beg);
}

void ora_tree_free(ora_tree *t) {
    if (!t) return;
    free(t->key); free(t->perm); free(t->x); free(t->y); free(t->z); free(t->m); free(t->rout); free(t->rs);
    free(t->node); free(t->canon2dfs); free(t->grp); free(t->grp_of); free(t);
}

ora_tree *ora_tree_build(int64_t N, const double *x, const double *y, const double *z, const double *m,
                         const double *rout, const double *rsearch, const ora_params *p) {
    ora_tree *t = (ora_tree *)calloc(1, sizeof(ora_tree));
    t->p = *p; t->N = N;
    if (N == 0) return t;
    /* O1: root cube. */
    const double *xs[3] = {x, y, z};
    double L = 0;
    for (int k = 0; k < 3; ++k) {
        double lo = xs[k][0], hi = xs[k][0];
        for (int64_t i = 1; i < N; ++i) { if (xs[k][i] < lo) lo = xs[k][i]; if (xs[k][i] > hi) hi = xs[k][i]; }
        t->c[k] = 0.5 * (lo + hi);
        if (hi - lo > L) L = hi - lo;
    }
    if (L == 0.0) t->h = 1.0;
    else { double v = 0.5 * L * (1.0 + ldexp(1.0, -20)); int e; (void)frexp(v, &e); t->h = ldexp(1.0, e); }
    /* O2 + O3: grid coordinates and keys. */
    double s = ldexp(2.0 * t->h, -ORA_MAXLEVEL);
    keyidx *ki = (keyidx *)xmalloc((size_t)N * sizeof(keyidx));
    for (int64_t i = 0; i < N; ++i) {
        uint64_t q[3];
        for (int k = 0; k < 3; ++k) {
            double o = t->c[k] - t->h;
            double g = floor((xs[k][i] - o) / s);
            int64_t qi = (int64_t)g;
            if (qi < 0) qi = 0;
            if (qi > (1ll << ORA_MAXLEVEL) - 1) qi = (1ll << ORA_MAXLEVEL) - 1;
            q[k] = (uint64_t)qi;
        }
        ki[i].key = morton63(q[0], q[1], q[2]); ki[i].idx = (int32_t)i;
    }
    /* O4: ascending (key, original index). */
    qsort(ki, (size_t)N, sizeof(keyidx), cmp_keyidx);
    t->key = (uint64_t *)xmalloc((size_t)N * 8); t->perm = (int32_t *)xmalloc((size_t)N * 4);
    t->x = (double *)xmalloc((size_t)N * 8); t->y = (double *)xmalloc((size_t)N * 8); t->z = (double *)xmalloc((size_t)N * 8);
    t->m = (double *)xmalloc((size_t)N * 8); t->rout = (double *)xmalloc((size_t)N * 8); t->rs = (double *)xmalloc((size_t)N * 8);
    for (int64_t i = 0; i < N; ++i) {
        int32_t o = ki[i].idx;
        t->key[i] = ki[i].key; t->perm[i] = o;
        t->x[i] = x[o]; t->y[i] = y[o]; t->z[i] = z[o]; t->m[i] = m[o]; t->rout[i] = rout[o];
        t->rs[i] = rsearch ? rsearch[o] : rout[o];
    }
    free(ki);
    /* O5, O6 */
    build_node(t, 0, 0, N);
    t->grp_of = (int32_t *)xmalloc((size_t)N * 4);
    make_groups(t, 0);
    /* canonical ids: rank in (level, begin) order */
    canon_key *ck = (canon_key *)xmalloc((size_t)t->n_node * sizeof(canon_key));
    for (int64_t i = 0; i < t->n_node; ++i) { ck[i].lvl = t->node[i].level; ck[i].beg = t->node[i].begin; ck[i].idx = i; }
    qsort(ck, (size_t)t->n_node, sizeof(canon_key), cmp_canon);
    t->canon2dfs = (int64_t *)xmalloc((size_t)t->n_node * 8);
    for (int64_t r = 0; r < t->n_node; ++r) { t->canon2dfs[r] = ck[r].idx; t->node[ck[r].idx].canon = r; }
    free(ck);
    return t;
}

int64_t ora_tree_n_nodes(const ora_tree *t) { return t->n_node; }
int64_t ora_tree_n_groups(const ora_tree *t) { return t->n_grp; }
void ora_tree_root(const ora_tree *t, double *c3_h) { c3_h[0] = t->c[0]; c3_h[1] = t->c[1]; c3_h[2] = t->c[2]; c3_h[3] = t->h; }
void ora_tree_keys(const ora_tree *t, uint64_t *key, int32_t *perm) {
    memcpy(key, t->key, (size_t)t->N * 8); memcpy(perm, t->perm, (size_t)t->N * 4);
}
/* Node table in canonical (level, begin) order.  dbl: 17 doubles per node
 * [M, com3, lo3, hi3, rmax, Q6]; integer: 5 int64 per node [level, begin, end, leaf, nchild].   */
void ora_tree_nodes(const ora_tree *t, int64_t *integer, double *dbl) {
    for (int64_t r = 0; r < t->n_node; ++r) {
        const ora_node *n = &t->node[t->canon2dfs[r]];
        int64_t *I = integer + 5 * r; double *D = dbl + 17 * r;
        I[0] = n->level; I[1] = n->begin; I[2] = n->end; I[3] = n->leaf; I[4] = n->nchild;
        D[0] = n->M; for (int k = 0; k < 3; ++k) { D[1 + k] = n->com[k]; D[4 + k] = n->lo[k]; D[7 + k] = n->hi[k]; }
        D[10] = n->rmax; for (int k = 0; k < 6; ++k) D[11 + k] = n->Q[k];
    }
}
/* Group table: 2 int64 [begin, end] and 7 doubles [lo3, hi3, rmax] per group. */
void ora_tree_groups(const ora_tree *t, int64_t *integer, double *dbl) {
    for (int64_t g = 0; g < t->n_grp; ++g) {
        integer[2 * g] = t->grp[g].begin; integer[2 * g + 1] = t->grp[g].end;
        for (int k = 0; k < 3; ++k) { dbl[7 * g + k] = t->grp[g].lo[k]; dbl[7 * g + 3 + k] = t->grp[g].hi[k]; }
        dbl[7 * g + 6] = t->grp[g].rmax;
    }
}

/* O7: the walk of one group.  A visitor receives accepted cells and opened leaves. */
typedef struct {
    int64_t n_sp, n_ep_ranges, n_ep;          /* cells accepted; leaf ranges; particles in them */
    int64_t *sp; int64_t cap_sp;              /* DFS indices of accepted cells (if collected) */
    int64_t *ep; int64_t cap_ep;              /* [begin, end, near] triples (if collected) */
    int collect;
} ora_list;

static void list_push_sp(ora_list *l, int64_t id) {
    if (l->collect) {
        if (l->n_sp == l->cap_sp) { l->cap_sp = l->cap_sp ? 2 * l->cap_sp : 256; l->sp = (int64_t *)realloc(l->sp, (size_t)l->cap_sp * 8); }
        l->sp[l->n_sp] = id;
    }
    l->n_sp++;
}
static void list_push_ep(ora_list *l, int64_t b, int64_t e, int near) {
    if (l->collect) {
        if (l->n_ep_ranges == l->cap_ep) { l->cap_ep = l->cap_ep ? 2 * l->cap_ep : 256; l->ep = (int64_t *)realloc(l->ep, (size_t)l->cap_ep * 24); }
        l->ep[3 * l->n_ep_ranges] = b; l->ep[3 * l->n_ep_ranges + 1] = e; l->ep[3 * l->n_ep_ranges + 2] = near;
    }
    l->n_ep_ranges++; l->n_ep += e - b;
}

static double max3(double a, double b, double c) { double m = a > b ? a : b; return m > c ? m : c; }

static void visit(const ora_tree *t, const ora_group *g, int64_t id, ora_list *out) {
    const ora_node *c = &t->node[id];
    double gap[3], pp[3];
    for (int k = 0; k < 3; ++k) {
        gap[k] = max3(0.0, c->lo[k] - g->hi[k], g->lo[k] - c->hi[k]);       /* box-box, per axis */
        pp[k] = max3(0.0, g->lo[k] - c->com[k], c->com[k] - g->hi[k]);      /* com to group box   */
    }
    double d2box = fma(gap[2], gap[2], fma(gap[1], gap[1], gap[0] * gap[0]));
    double R = g->rmax > c->rmax ? g->rmax : c->rmax;
    int near = d2box < R * R;
    double d2com = fma(pp[2], pp[2], fma(pp[1], pp[1], pp[0] * pp[0]));
    int far = (c->edge * c->edge) < (t->p.theta * t->p.theta) * d2com;
    if (!near && far) list_push_sp(out, id);
    else if (c->leaf) list_push_ep(out, c->begin, c->end, near);
    else for (int k = 0; k < c->nchild; ++k) visit(t, g, c->child[k], out);
}

/* Per-group counts: n_i, n_ep (particles), n_sp (cells), n_ep_ranges; and the totals
 * N_epep = sum n_i n_ep (self pairs counted), N_epsp = sum n_i n_sp.  out4 = n_grp x 4 int64.   */
void ora_walk_counts(const ora_tree *t, int64_t *out4, int64_t *totals2) {
    int64_t epep = 0, epsp = 0;
#pragma omp parallel for schedule(dynamic, 8) reduction(+ : epep, epsp)
    for (int64_t g = 0; g < t->n_grp; ++g) {
        ora_list l; memset(&l, 0, sizeof l);
        visit(t, &t->grp[g], 0, &l);
        int64_t ni = t->grp[g].end - t->grp[g].begin;
        out4[4 * g] = ni; out4[4 * g + 1] = l.n_ep; out4[4 * g + 2] = l.n_sp; out4[4 * g + 3] = l.n_ep_ranges;
        epep += ni * l.n_ep; epsp += ni * l.n_sp;
    }
    totals2[0] = epep; totals2[1] = epsp;
}

/* Lists of one group: sp = canonical node ids (cap_sp), ep = [begin,end,near] triples (cap_ep).
 * Returns counts in n2 = [n_sp, n_ep_ranges]; writes only if the capacities suffice.              */
void ora_walk_lists(const ora_tree *t, int64_t g, int64_t *sp, int64_t cap_sp, int64_t *ep, int64_t cap_ep, int64_t *n2) {
    ora_list l; memset(&l, 0, sizeof l); l.collect = 1;
    visit(t, &t->grp[g], 0, &l);
    n2[0] = l.n_sp; n2[1] = l.n_ep_ranges;
    if (l.n_sp <= cap_sp) for (int64_t k = 0; k < l.n_sp; ++k) sp[k] = t->node[l.sp[k]].canon;
    if (l.n_ep_ranges <= cap_ep) memcpy(ep, l.ep, (size_t)l.n_ep_ranges * 24);
    free(l.sp); free(l.ep);
}

/* O8 cell term.  r = x_i - com_c; A' = 1.5 Q - 0.5 tr(Q) I (Eq. 31);
 * phi = -G [ M/r + r^T A' r / r^5 ],  a = -grad phi = G [ -M r/r^3 + 2 A' r / r^5 - 5 (r^T A' r) r / r^7 ]. */
static void cell_term(const ora_tree *t, const ora_node *c, double xi, double yi, double zi, double *a, double *phi) {
    double r[3] = {xi - c->com[0], yi - c->com[1], zi - c->com[2]};
    double r2 = r[0] * r[0] + r[1] * r[1] + r[2] * r[2];
    double rr = sqrt(r2);
    double G = t->p.G;
    for (int k = 0; k < 3; ++k) a[k] += -G * c->M * r[k] / (r2 * rr);
    *phi += -G * c->M / rr;
    if (t->p.multipole >= 2) {
        double tr = c->Q[0] + c->Q[1] + c->Q[2];
        double A[3][3];
        A[0][0] = 1.5 * c->Q[0] - 0.5 * tr; A[1][1] = 1.5 * c->Q[1] - 0.5 * tr; A[2][2] = 1.5 * c->Q[2] - 0.5 * tr;
        A[0][1] = A[1][0] = 1.5 * c->Q[3]; A[0][2] = A[2][0] = 1.5 * c->Q[4]; A[1][2] = A[2][1] = 1.5 * c->Q[5];
        double Ar[3], rAr = 0;
        for (int k = 0; k < 3; ++k) { Ar[k] = A[k][0] * r[0] + A[k][1] * r[1] + A[k][2] * r[2]; rAr += r[k] * Ar[k]; }
        double r5 = r2 * r2 * rr, r7 = r5 * r2;
        for (int k = 0; k < 3; ++k) a[k] += G * (2.0 * Ar[k] / r5 - 5.0 * rAr * r[k] / r7);
        *phi += -G * rAr / r5;
    }
}

static void eval_group(const ora_tree *t, int64_t gb, int64_t ge, const ora_list *l, const int64_t *sp_dfs,
                       double *ax, double *ay, double *az, double *pot) {
    for (int64_t i = gb; i < ge; ++i) {
        double a[3] = {0, 0, 0}, phi = 0;
        for (int64_t r = 0; r < l->n_ep_ranges; ++r)
            for (int64_t j = l->ep[3 * r]; j < l->ep[3 * r + 1]; ++j) {
                if (j == i) continue;
                pair_split(t->x[j] - t->x[i], t->y[j] - t->y[i], t->z[j] - t->z[i], t->m[j], t->rout[i], t->rout[j],
                           &t->p, 1, a, &phi);
            }
        for (int64_t k = 0; k < l->n_sp; ++k) cell_term(t, &t->node[sp_dfs[k]], t->x[i], t->y[i], t->z[i], a, &phi);
        int32_t o = t->perm[i];
        ax[o] = a[0]; ay[o] = a[1]; az[o] = a[2]; pot[o] = phi;
    }
}

/* O7 + O8 with self-built lists ("mode 1") for groups sel[0..ns) (sel == NULL: all groups).
 * Results are written in the caller's ORIGINAL particle order; untouched entries stay as they were. */
void ora_tree_force(const ora_tree *t, int64_t ns, const int64_t *sel, double *ax, double *ay, double *az, double *pot) {
    int64_t n = sel ? ns : t->n_grp;
#pragma omp parallel for schedule(dynamic, 4)
    for (int64_t s = 0; s < n; ++s) {
        int64_t g = sel ? sel[s] : s;
        ora_list l; memset(&l, 0, sizeof l); l.collect = 1;
        visit(t, &t->grp[g], 0, &l);
        eval_group(t, t->grp[g].begin, t->grp[g].end, &l, l.sp, ax, ay, az, pot);
        free(l.sp); free(l.ep);
    }
}

/* "mode 2": evaluate IMPORTED lists for one i-range [gb, ge) of sorted positions:
 * sp = canonical node ids, ep = [begin, end] pairs of sorted positions.                          */
void ora_eval_lists(const ora_tree *t, int64_t gb, int64_t ge, int64_t n_sp, const int64_t *sp_canon,
                    int64_t n_ep_ranges, const int64_t *ep2, double *ax, double *ay, double *az, double *pot) {
    ora_list l; memset(&l, 0, sizeof l);
    l.n_sp = n_sp; l.n_ep_ranges = n_ep_ranges;
    l.ep = (int64_t *)xmalloc((size_t)n_ep_ranges * 24);
    for (int64_t r = 0; r < n_ep_ranges; ++r) { l.ep[3 * r] = ep2[2 * r]; l.ep[3 * r + 1] = ep2[2 * r + 1]; l.ep[3 * r + 2] = 0; }
    int64_t *dfs = (int64_t *)xmalloc((size_t)n_sp * 8);
    for (int64_t k = 0; k < n_sp; ++k) dfs[k] = t->canon2dfs[sp_canon[k]];
    eval_group(t, gb, ge, &l, dfs, ax, ay, az, pot);
    free(dfs); free(l.ep);
}

/* O9: neighbours from the walk's EP lists, fp64 test, ORIGINAL indices; rows sorted ascending.
 * Two-phase like the library: indices == NULL => offsets only.                                   */
static int cmp_i32(const void *a, const void *b) { int32_t p = *(const int32_t *)a, q = *(const int32_t *)b; return (p > q) - (p < q); }
void ora_tree_neighbors_sel(const ora_tree *t, int64_t ns, const int64_t *sel, int64_t *offsets, int32_t *indices);
void ora_tree_neighbors(const ora_tree *t, int64_t *offsets, int32_t *indices) { ora_tree_neighbors_sel(t, 0, NULL, offsets, indices); }
/* Same for the particles of groups sel[0..ns) only (sel == NULL: all groups); other rows stay empty. */
void ora_tree_neighbors_sel(const ora_tree *t, int64_t ns, const int64_t *sel, int64_t *offsets, int32_t *indices) {
    int64_t N = t->N;
    int64_t ng = sel ? ns : t->n_grp;
    if (!indices) memset(offsets, 0, (size_t)(N + 1) * 8);
#pragma omp parallel for schedule(dynamic, 4)
    for (int64_t gs = 0; gs < ng; ++gs) {
        int64_t g = sel ? sel[gs] : gs;
        ora_list l; memset(&l, 0, sizeof l); l.collect = 1;
        visit(t, &t->grp[g], 0, &l);
        for (int64_t i = t->grp[g].begin; i < t->grp[g].end; ++i) {
            int32_t oi = t->perm[i];
            int64_t c = 0, o = indices ? offsets[oi] : 0;
            for (int64_t r = 0; r < l.n_ep_ranges; ++r)
                for (int64_t j = l.ep[3 * r]; j < l.ep[3 * r + 1]; ++j) {
                    if (j == i) continue;
                    double dx = t->x[i] - t->x[j], dy = t->y[i] - t->y[j], dz = t->z[i] - t->z[j];
                    double r2 = fma(dz, dz, fma(dy, dy, dx * dx));
                    double R = t->rs[i] > t->rs[j] ? t->rs[i] : t->rs[j];
                    if (r2 < R * R) { if (indices) indices[o + c] = t->perm[j]; ++c; }
                }
            if (indices) qsort(indices + o, (size_t)c, 4, cmp_i32);
            else offsets[oi + 1] = c;
        }
        free(l.sp); free(l.ep);
    }
    if (!indices) for (int64_t i = 0; i < N; ++i) offsets[i + 1] += offsets[i];
}

/* ------------------------------------------------------------------------------------ */
/* (C) orbit-dependent neighbour criterion and clustering (:325-335)  */
/* ------------------------------------------------------------------------------------ */

/* Eq. 24: r_nb,i = r_out,i + C_r |v_i| dt_L.  Operation order (rule O10a):
 * v2 = fma(vz,vz, fma(vy,vy, vx*vx)); r_nb = r_out + (C_r * sqrt(v2)) * dt.                        */
void ora_search_radii(int64_t N, const double *vx, const double *vy, const double *vz, const double *rout,
                      double Cr, double dt, double *rnb) {
    for (int64_t i = 0; i < N; ++i) {
        double v2 = fma(vz[i], vz[i], fma(vy[i], vy[i], vx[i] * vx[i]));
        rnb[i] = rout[i] + (Cr * sqrt(v2)) * dt;
    }
}

/* Pericentre separation of the two-body Kepler orbit of a pair ("Kepler orbital
 * pericentre separation r_p,ij"): relative position d, relative velocity w, mu = G (m_i + m_j).
 * With h = d x w and 2 eps = w^2 - 2 mu / r the conic has r_p = h^2 / (mu + sqrt(mu^2 + 2 eps h^2))
 * (= p / (1 + e); valid for bound, parabolic and unbound orbits; mu = 0 gives the impact parameter
 * h / |w|).  Rule O10b, exactly these operations:
 *   r2 = fma(dz,dz, fma(dy,dy, dx*dx)); v2 likewise; hx = dy*wz - dz*wy; hy = dz*wx - dx*wz;
 *   hz = dx*wy - dy*wx; h2 = fma(hz,hz, fma(hy,hy, hx*hx)); r = sqrt(r2); r == 0 => r_p = 0;
 *   e2 = v2 - (2 mu) / r; disc = max(0, fma(e2, h2, mu*mu)); den = mu + sqrt(disc);
 *   r_p = den > 0 ? h2 / den : r.                                                                  */
double ora_pericentre(double dx, double dy, double dz, double wx, double wy, double wz, double mu) {
    double r2 = fma(dz, dz, fma(dy, dy, dx * dx));
    double v2 = fma(wz, wz, fma(wy, wy, wx * wx));
    double hx = dy * wz - dz * wy, hy = dz * wx - dx * wz, hz = dx * wy - dy * wx;
    double h2 = fma(hz, hz, fma(hy, hy, hx * hx));
    double r = sqrt(r2);
    if (r == 0.0) return 0.0;
    double e2 = v2 - (2.0 * mu) / r;
    double disc = fma(e2, h2, mu * mu);
    if (!(disc > 0.0)) disc = 0.0;
    double den = mu + sqrt(disc);
    return den > 0.0 ? h2 / den : r;
}

/* Two-stage criterion, rule O10c (reading P20).  j is a neighbour of i iff
 *   stage (i)  j != i and r_ij < R_s, R_s = max(r_nb,i, r_nb,j) (the symmetric candidate rule O9 with the
 *              Eq. 24 radii), and
 *   stage (ii) r_p,ij < C_V min(r_nb,i, r_nb,j) -- the paper's "r_p,ij < C_V r_nb,i" required from both
 *              sides, so that the relation stays symmetric (the clusters need a symmetric graph); with the
 *              max instead, r_p <= r_ij < R_s would make the test vacuous for C_V >= 1 --
 *              OR r_ij < R_o = max(r_out,i, r_out,j): a pair inside its changeover radius has a non-zero
 *              short-range force now and is always kept.                                            */
static int orbit_pair(double xi, double yi, double zi, double vxi, double vyi, double vzi, double mi, double ri, double roi,
                      double xj, double yj, double zj, double vxj, double vyj, double vzj, double mj, double rj, double roj,
                      double G, double Cv) {
    double dx = xi - xj, dy = yi - yj, dz = zi - zj;
    double r2 = fma(dz, dz, fma(dy, dy, dx * dx));
    double Rs = ri > rj ? ri : rj;
    if (!(r2 < Rs * Rs)) return 0;
    double Ro = roi > roj ? roi : roj;
    if (r2 < Ro * Ro) return 1;
    double rp = ora_pericentre(dx, dy, dz, vxi - vxj, vyi - vyj, vzi - vzj, G * (mi + mj));
    double Rm = ri < rj ? ri : rj;
    return rp < Cv * Rm;
}

/* O(N^2) definition of the filtered list; two-phase like ora_neighbors_direct; rows ascending.     */
void ora_neighbors_orbit_direct(int64_t N, const double *x, const double *y, const double *z,
                                const double *vx, const double *vy, const double *vz, const double *m,
                                const double *rnb, const double *rout, double G, double Cv, int64_t *offsets, int32_t *indices) {
#pragma omp parallel for schedule(dynamic, 64)
    for (int64_t i = 0; i < N; ++i) {
        int64_t c = 0, o = indices ? offsets[i] : 0;
        for (int64_t j = 0; j < N; ++j) {
            if (j == i) continue;
            if (orbit_pair(x[i], y[i], z[i], vx[i], vy[i], vz[i], m[i], rnb[i], rout[i],
                           x[j], y[j], z[j], vx[j], vy[j], vz[j], m[j], rnb[j], rout[j], G, Cv)) {
                if (indices) indices[o + c] = (int32_t)j;
                ++c;
            }
        }
        if (!indices) offsets[i + 1] = c;
    }
    if (!indices) { offsets[0] = 0; for (int64_t i = 0; i < N; ++i) offsets[i + 1] += offsets[i]; }
}

/* Tree version (rule O10): the candidates are the walk's EP lists of a tree built with r_search = r_nb
 * (so every pair inside R is an EP pair, rule O7); velocities vx, vy, vz are in the CALLER's order.
 * Rows hold original indices, ascending.  sel as in ora_tree_neighbors_sel.                         */
void ora_tree_neighbors_orbit_sel(const ora_tree *t, int64_t ns, const int64_t *sel, const double *vx, const double *vy,
                                  const double *vz, double Cv, int64_t *offsets, int32_t *indices) {
    int64_t N = t->N;
    int64_t ng = sel ? ns : t->n_grp;
    if (!indices) memset(offsets, 0, (size_t)(N + 1) * 8);
#pragma omp parallel for schedule(dynamic, 4)
    for (int64_t gs = 0; gs < ng; ++gs) {
        int64_t g = sel ? sel[gs] : gs;
        ora_list l; memset(&l, 0, sizeof l); l.collect = 1;
        visit(t, &t->grp[g], 0, &l);
        for (int64_t i = t->grp[g].begin; i < t->grp[g].end; ++i) {
            int32_t oi = t->perm[i];
            int64_t c = 0, o = indices ? offsets[oi] : 0;
            for (int64_t r = 0; r < l.n_ep_ranges; ++r)
                for (int64_t j = l.ep[3 * r]; j < l.ep[3 * r + 1]; ++j) {
                    if (j == i) continue;
                    int32_t oj = t->perm[j];
                    if (orbit_pair(t->x[i], t->y[i], t->z[i], vx[oi], vy[oi], vz[oi], t->m[i], t->rs[i], t->rout[i],
                                   t->x[j], t->y[j], t->z[j], vx[oj], vy[oj], vz[oj], t->m[j], t->rs[j], t->rout[j], t->p.G, Cv)) {
                        if (indices) indices[o + c] = oj;
                        ++c;
                    }
                }
            if (indices) qsort(indices + o, (size_t)c, 4, cmp_i32);
            else offsets[oi + 1] = c;
        }
        free(l.sp); free(l.ep);
    }
    if (!indices) for (int64_t i = 0; i < N; ++i) offsets[i + 1] += offsets[i];
}

/* Clustering: "any member in one cluster have all its neighbours inside the same
 * cluster" -- the clusters are the connected components of the (symmetric) neighbour graph.  Plain
 * union-find with path halving; label[i] = smallest index of i's component (a particle without
 * neighbours is its own cluster).  Returns the number of clusters.                                  */
static int64_t uf_find(int64_t *parent, int64_t a) {
    while (parent[a] != a) { parent[a] = parent[parent[a]]; a = parent[a]; }
    return a;
}
int64_t ora_clusters(int64_t N, const int64_t *offsets, const int32_t *indices, int32_t *label) {
    int64_t *parent = (int64_t *)xmalloc((size_t)N * 8);
    for (int64_t i = 0; i < N; ++i) parent[i] = i;
    for (int64_t i = 0; i < N; ++i)
        for (int64_t e = offsets[i]; e < offsets[i + 1]; ++e) {
            int64_t a = uf_find(parent, i), b = uf_find(parent, indices[e]);
            if (a < b) parent[b] = a; else if (b < a) parent[a] = b;     /* the smaller index stays root */
        }
    int64_t nc = 0;
    for (int64_t i = 0; i < N; ++i) { int64_t r = uf_find(parent, i); label[i] = (int32_t)r; nc += (r == i); }
    free(parent);
    return nc;
}

/* ------------------------------------------------------------------------------------ */
/* (D) short-range force, jerk and potential over the neighbour list  */
/* ------------------------------------------------------------------------------------ */

/* dK/dx of Eq. 17 for 0 < x < 1 (0 outside).  Differentiating Eq. 18,
 * K = f - (x+q) f', gives K' = -(x+q) f'' with f'' = 280 Lambda x^3 (1-x)^3 (from Eq. 16) and
 * q = r_in / (r_out - r_in); all of Eq. 19's boundary values follow from the x^3 (1-x)^3 factor.   */
double ora_dK(double x, double Lam, double q) {
    if (x <= 0.0 || x >= 1.0) return 0.0;
    double y = 1.0 - x;
    return -280.0 * Lam * (x + q) * (x * x * x) * (y * y * y);
}

/* H_S of Eq. 11 evaluated over the neighbour rows (the Hermite integrator's force
 * evaluation, Eq. 40 :639 needs the acceleration and its first time derivative):
 *   a_S,i   = -G sum_j m_j K(x) d / r^3,                       d = x_i - x_j, w = v_i - v_j
 *   j_S,i   = -G sum_j m_j { K [ w / r^3 - 3 (d.w) d / r^5 ] + K'(x) xdot d / r^3 },  xdot = (d.w) / (r (R - r_in))
 *   phi_S,i = -G sum_j m_j W(x) / r
 * with R = max(r_out,i, r_out,j), r_in = rho R, x = (r - r_in)/(R - r_in).  Pairs at r >= R contribute
 * nothing; coincident pairs (r = 0) are skipped (reading P4).  Rows are summed in list order.       */
void ora_short_range(int64_t N, const double *x, const double *y, const double *z, const double *vx, const double *vy,
                     const double *vz, const double *m, const double *rout, const int64_t *offsets, const int32_t *indices,
                     double G, double rho, double *ax, double *ay, double *az, double *jx, double *jy, double *jz, double *pot) {
    const double q = rho / (1.0 - rho);
#pragma omp parallel for schedule(dynamic, 256)
    for (int64_t i = 0; i < N; ++i) {
        double a[3] = {0, 0, 0}, jk[3] = {0, 0, 0}, phi = 0.0;
        for (int64_t e = offsets[i]; e < offsets[i + 1]; ++e) {
            int64_t j = indices[e];
            double dx = x[i] - x[j], dy = y[i] - y[j], dz = z[i] - z[j];
            double wx = vx[i] - vx[j], wy = vy[i] - vy[j], wz = vz[i] - vz[j];
            double r2 = dx * dx + dy * dy + dz * dz;
            double r = sqrt(r2);
            double R = rout[i] > rout[j] ? rout[i] : rout[j];
            if (r == 0.0 || r >= R) continue;
            double rin = rho * R;
            double Lam = (R - rin) / (R + rin);
            double xx = (r - rin) / (R - rin);
            double K = ora_K(xx, Lam), W = ora_W(xx, Lam), dK = ora_dK(xx, Lam, q);
            double dw = dx * wx + dy * wy + dz * wz;
            double r3 = r2 * r;
            double xdot = dw / (r * (R - rin));
            double c0 = -G * m[j] * K / r3;                       /* coefficient of d in a, of w in the jerk */
            double c1 = -G * m[j] * (-3.0 * K * dw / (r3 * r2) + dK * xdot / r3);
            a[0] += c0 * dx; a[1] += c0 * dy; a[2] += c0 * dz;
            jk[0] += c0 * wx + c1 * dx; jk[1] += c0 * wy + c1 * dy; jk[2] += c0 * wz + c1 * dz;
            phi -= G * m[j] * W / r;
        }
        ax[i] = a[0]; ay[i] = a[1]; az[i] = a[2];
        jx[i] = jk[0]; jy[i] = jk[1]; jz[i] = jk[2];
        pot[i] = phi;
    }
}

void ora_set_num_threads(int n) {
#ifdef _OPENMP
    if (n > 0) omp_set_num_threads(n);
#else
    (void)n;
#endif
}

int ora_num_threads(void) {
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}
