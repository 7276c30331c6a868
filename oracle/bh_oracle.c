/*
 * oracle/bh_oracle.c — CPU ORACLE for the Barnes-Hut gravity hot path of arxiv/paper_1912_04197.
 *
 * THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only tests/, __graft_entry__.smoke() and bench.py's
 * cpu_baseline / --impl reference legs may call it.  It shares no code, header, table or helper
 * with the CUDA path under paper_1912_04197_b200/csrc/ and includes nothing from include/.
 *
 * Plain, slow and meant to be checked against the paper by eye.  Steps O1..O11 are the readings of
 * SURVEY.md §8(c) (restated in DESIGN.md §3); each function cites the PAPER.md passage it follows.
 * Compile with -ffp-contract=off: every fused multiply-add below is an explicit fma(), every other
 * operation is rounded once, so the integer decisions (keys, tree, accept/open) are reproducible.
 *
 * Pins (tests/test_oracle_*.py, all `-m "not gpu"`): Morton closed forms and round trip; a second,
 * recursive tree builder on unsorted integer coordinates; lattice node-count closed forms; root
 * monopole against extended-precision totals; exact coverage of every walk list; theta=0 == direct
 * sum; a textbook per-body recursive Barnes-Hut (W=1, C=1); two-body / triangle / tetrahedron
 * closed forms; Newton's third law; brute force in exact rational arithmetic on tiny N; KDK
 * two-body orbit, dt^2 energy error, time reversal.  Rows "next" (O12-O16, tests/test_oracle_next.py):
 * potential against the two-body closed form, exact-rational brute force and the finite-difference
 * gradient (= minus the acceleration); theta=0 tree potential == direct potential; diagnostics against
 * hand-computed systems; Eq. (7) on hand cases; Eq. (8) against the paper's "thousands of seconds";
 * semi-implicit Euler: angular momentum exact for a central force, first-order energy error; the
 * two-rate step against its closed form.  No function here is "parity unpinned".
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define ORC_MAXLEVEL 21 /* 63 key bits / 3 bits per level (reading R9: depth cap) */

int orc_num_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

/* ---------------------------------------------------------------------------------------------
 * O1  Canonical bounding cube.  PAPER.md:112 "compute bounding box around all bodies (root of the
 * octree)"; "a node ... corresponds to a cube".  Reading R11: corner at the per-axis
 * minimum, side L = smallest power of two strictly greater than the largest extent (L = 1 if the
 * extent is 0).  Returns 0, or -3 if any coordinate is not finite.  *e is the exponent: L = 2^e.
 * ------------------------------------------------------------------------------------------- */
int orc_cube(const double *pos, int64_t n, double lo[3], double *L, int32_t *e)
{
    double hi[3];
    for (int a = 0; a < 3; ++a) {
        lo[a] = pos[a];
        hi[a] = pos[a];
    }
    for (int64_t i = 0; i < n; ++i)
        for (int a = 0; a < 3; ++a) {
            double x = pos[3 * i + a];
            if (!isfinite(x)) return -3;
            if (x < lo[a]) lo[a] = x;
            if (x > hi[a]) hi[a] = x;
        }
    double E = 0.0;
    for (int a = 0; a < 3; ++a) {
        double ext = hi[a] - lo[a]; /* one rounding */
        if (ext > E) E = ext;
    }
    if (!isfinite(E)) return -3;
    if (E == 0.0) {
        *e = 0;
        *L = 1.0;
    } else {
        int ex;
        (void)frexp(E, &ex); /* E = f * 2^ex, 0.5 <= f < 1  =>  2^(ex-1) <= E < 2^ex */
        *e = ex;
        *L = ldexp(1.0, ex);
    }
    return 0;
}

/* ---------------------------------------------------------------------------------------------
 * O2 + O3  Quantise to 21 bits per axis and interleave to a 63-bit Morton key (not in the paper,
 * whose tree is built by insertion; reading R12).  q = trunc((x - lo) * 2^(21-e));
 * bit k of qx -> key bit 3k, of qy -> 3k+1, of qz -> 3k+2.  Naive bit loop on purpose.
 * ------------------------------------------------------------------------------------------- */
void orc_quantise(const double *pos, int64_t n, const double lo[3], int32_t e, uint32_t *q)
{
    double scale = ldexp(1.0, 21 - e); /* exact power of two */
    for (int64_t i = 0; i < n; ++i)
        for (int a = 0; a < 3; ++a) {
            double d = pos[3 * i + a] - lo[a]; /* one rounding */
            q[3 * i + a] = (uint32_t)(d * scale); /* exact scaling, truncation */
        }
}

uint64_t orc_morton_key(uint32_t qx, uint32_t qy, uint32_t qz)
{
    uint64_t key = 0;
    for (int k = 0; k < 21; ++k) {
        key |= (uint64_t)((qx >> k) & 1u) << (3 * k);
        key |= (uint64_t)((qy >> k) & 1u) << (3 * k + 1);
        key |= (uint64_t)((qz >> k) & 1u) << (3 * k + 2);
    }
    return key;
}

void orc_morton(const double *pos, int64_t n, const double lo[3], int32_t e, uint64_t *key)
{
    uint32_t *q = (uint32_t *)malloc((size_t)n * 3 * sizeof(uint32_t));
    orc_quantise(pos, n, lo, e, q);
    for (int64_t i = 0; i < n; ++i) key[i] = orc_morton_key(q[3 * i], q[3 * i + 1], q[3 * i + 2]);
    free(q);
}

/* ---------------------------------------------------------------------------------------------
 * O4  Sort: perm such that (key[perm[j]], perm[j]) ascends lexicographically (ties by original
 * index).  Replaces PAPER.md:115 "sort bodies by distance (to speed up force evaluation)" (R16).
 * ------------------------------------------------------------------------------------------- */
typedef struct {
    uint64_t key;
    uint32_t idx;
} orc_pair;

static int orc_pair_cmp(const void *pa, const void *pb)
{
    const orc_pair *a = (const orc_pair *)pa, *b = (const orc_pair *)pb;
    if (a->key != b->key) return a->key < b->key ? -1 : 1;
    if (a->idx != b->idx) return a->idx < b->idx ? -1 : 1;
    return 0;
}

void orc_sort(const uint64_t *key, int64_t n, uint32_t *perm, uint64_t *skey)
{
    orc_pair *p = (orc_pair *)malloc((size_t)n * sizeof(orc_pair));
    for (int64_t i = 0; i < n; ++i) {
        p[i].key = key[i];
        p[i].idx = (uint32_t)i;
    }
    qsort(p, (size_t)n, sizeof(orc_pair), orc_pair_cmp);
    for (int64_t j = 0; j < n; ++j) {
        perm[j] = p[j].idx;
        skey[j] = p[j].key;
    }
    free(p);
}

/* sorted bodies as (x, y, z, m) rows */
void orc_gather(const double *pos, const double *mass, const uint32_t *perm, int64_t n, double *sbody)
{
    for (int64_t j = 0; j < n; ++j) {
        uint32_t i = perm[j];
        sbody[4 * j + 0] = pos[3 * (int64_t)i + 0];
        sbody[4 * j + 1] = pos[3 * (int64_t)i + 1];
        sbody[4 * j + 2] = pos[3 * (int64_t)i + 2];
        sbody[4 * j + 3] = mass[i];
    }
}

/* ---------------------------------------------------------------------------------------------
 * O5  Octree in canonical numbering.  PAPER.md:62: cubes, eight children by homogeneous
 * subdivision, recursion until a node holds few enough particles, adaptive depth, rebuilt every
 * step.  Readings R8 (bucket leaves: leaf iff count <= C), R9 (level 21 is always a leaf), R10
 * (only non-empty children exist).  Node ids ascend in processing order: level by level, Morton
 * order inside a level, a node's children consecutive in octant order.
 * Returns the node count M, or -2 if cap nodes are not enough.
 * ------------------------------------------------------------------------------------------- */
static inline unsigned orc_digit(uint64_t key, int level) /* octant digit at level 1..21 */
{
    return (unsigned)((key >> (63 - 3 * level)) & 7u);
}

int64_t orc_tree(const uint64_t *skey, int64_t n, int32_t C, int64_t cap, uint8_t *level,
                 uint32_t *begin, uint32_t *count, int32_t *first_child, uint8_t *child_mask,
                 int32_t *parent, int32_t *depth)
{
    if (cap < 1) return -2;
    int64_t M = 1;
    level[0] = 0;
    begin[0] = 0;
    count[0] = (uint32_t)n;
    parent[0] = -1;
    *depth = 0;
    for (int64_t t = 0; t < M; ++t) {
        first_child[t] = -1;
        child_mask[t] = 0;
        if ((int64_t)count[t] <= C || level[t] == ORC_MAXLEVEL) continue; /* leaf */
        int64_t p = begin[t], end = (int64_t)begin[t] + count[t];
        int lv = level[t] + 1;
        for (unsigned o = 0; o < 8; ++o) {
            int64_t s = p;
            while (p < end && orc_digit(skey[p], lv) == o) ++p;
            if (p > s) {
                if (M >= cap) return -2;
                if (first_child[t] < 0) first_child[t] = (int32_t)M;
                child_mask[t] |= (uint8_t)(1u << o);
                level[M] = (uint8_t)lv;
                begin[M] = (uint32_t)s;
                count[M] = (uint32_t)(p - s);
                parent[M] = (int32_t)t;
                if (lv > *depth) *depth = lv;
                ++M;
            }
        }
    }
    return M;
}

static inline int orc_popcount8(unsigned m)
{
    int c = 0;
    for (; m; m >>= 1) c += (int)(m & 1u);
    return c;
}

/* ---------------------------------------------------------------------------------------------
 * O6  Monopoles, Eq. (2): node mass = sum of child masses, node COM = (1/m) * sum of
 * child COM * child mass; "computed for each leaf and internal node".  Fixed order so
 * the result is reproducible bit for bit: masses added left to right, weighted sums by fma from 0,
 * one IEEE division per coordinate.  A one-body leaf copies the body.  mono rows are (cx,cy,cz,m).
 * ------------------------------------------------------------------------------------------- */
void orc_monopoles(const double *sbody, int64_t M, const uint32_t *begin, const uint32_t *count,
                   const int32_t *first_child, const uint8_t *child_mask, double *mono)
{
    for (int64_t t = M - 1; t >= 0; --t) {
        double m, wx = 0.0, wy = 0.0, wz = 0.0;
        if (first_child[t] < 0) { /* leaf: from its bodies */
            int64_t b = begin[t], c = count[t];
            if (c == 1) {
                memcpy(&mono[4 * t], &sbody[4 * b], 4 * sizeof(double));
                continue;
            }
            m = sbody[4 * b + 3];
            for (int64_t j = b + 1; j < b + c; ++j) m = m + sbody[4 * j + 3];
            for (int64_t j = b; j < b + c; ++j) {
                double mj = sbody[4 * j + 3];
                wx = fma(mj, sbody[4 * j + 0], wx);
                wy = fma(mj, sbody[4 * j + 1], wy);
                wz = fma(mj, sbody[4 * j + 2], wz);
            }
        } else { /* internal: from its children in ascending id (octant order) */
            int64_t f = first_child[t], k = orc_popcount8(child_mask[t]);
            m = mono[4 * f + 3];
            for (int64_t u = f + 1; u < f + k; ++u) m = m + mono[4 * u + 3];
            for (int64_t u = f; u < f + k; ++u) {
                double mu = mono[4 * u + 3];
                wx = fma(mu, mono[4 * u + 0], wx);
                wy = fma(mu, mono[4 * u + 1], wy);
                wz = fma(mu, mono[4 * u + 2], wz);
            }
        }
        mono[4 * t + 0] = wx / m;
        mono[4 * t + 1] = wy / m;
        mono[4 * t + 2] = wz / m;
        mono[4 * t + 3] = m;
    }
}

/* ---------------------------------------------------------------------------------------------
 * O7  Walk groups (reading R6).  PAPER.md:118: "Each body is assigned to a thread ... Thanks to
 * sorting, neighbor bodies require the traversal of a similar sub-part of the octree": bodies that
 * are neighbours in the sorted order walk together.  A group must be spatially compact, so groups
 * never straddle a GROUP CELL: a tree node holding <= Gc bodies whose parent holds more than Gc
 * (the root if n <= Gc; a level-21 leaf is a group cell whatever it holds).  Group cells partition
 * the sorted bodies; each is cut into runs of W consecutive bodies (the last run may be shorter).
 * Groups are numbered in sorted-body order.  gstart must have room for n + 1 entries; returns the
 * number of groups Ng, group g = sorted bodies [gstart[g], gstart[g+1]).
 * ------------------------------------------------------------------------------------------- */
int64_t orc_group_starts(int64_t n, int64_t M, int32_t W, int32_t Gc, const uint32_t *begin,
                         const uint32_t *count, const int32_t *first_child, const int32_t *parent,
                         uint32_t *gstart)
{
    /* mark the first body of every run */
    uint8_t *flag = (uint8_t *)calloc((size_t)n + 1, 1);
    for (int64_t t = 0; t < M; ++t) {
        int small = (int64_t)count[t] <= Gc || first_child[t] < 0;
        int parent_big = parent[t] < 0 || (int64_t)count[parent[t]] > Gc;
        if (small && parent_big)
            for (int64_t j = begin[t]; j < (int64_t)begin[t] + count[t]; j += W) flag[j] = 1;
    }
    int64_t ng = 0;
    for (int64_t j = 0; j < n; ++j)
        if (flag[j]) gstart[ng++] = (uint32_t)j;
    gstart[ng] = (uint32_t)n;
    free(flag);
    return ng;
}

/* bounding boxes of the groups (exact min / max of the sorted coordinates) */
void orc_group_boxes(const double *sbody, const uint32_t *gstart, int64_t ng, double *glo, double *ghi)
{
    for (int64_t g = 0; g < ng; ++g) {
        int64_t b = gstart[g], e = gstart[g + 1];
        for (int a = 0; a < 3; ++a) {
            double l = sbody[4 * b + a], h = l;
            for (int64_t j = b + 1; j < e; ++j) {
                double x = sbody[4 * j + a];
                if (x < l) l = x;
                if (x > h) h = x;
            }
            glo[3 * g + a] = l;
            ghi[3 * g + a] = h;
        }
    }
}

/* ---------------------------------------------------------------------------------------------
 * O8  Walk of one group.  PAPER.md:84-106: from the root downwards; theta = r/D per body-node pair
 * (Eq. (3)); theta_BN < theta stops at the node (Eq. (5)), otherwise all children are visited; a
 * leaf is evaluated body to body (Eq. (4)).  Readings: R4 r := full cube edge s; R3 D unsoftened;
 * R5 equality opens; R6 D := distance from the node COM to the group's bounding box (W = 1: the
 * paper's per-body test); R7 a node holding a body of the group is never accepted.
 * The accept test is  s*s < (theta*theta) * d2  with every operation rounded once.
 * Depth-first, pre-order, children in ascending id.
 * ------------------------------------------------------------------------------------------- */
typedef struct {
    int32_t *v;
    int64_t n, cap;
} orc_ivec;

static void orc_push(orc_ivec *a, int32_t x)
{
    if (a->n == a->cap) {
        a->cap = a->cap ? 2 * a->cap : 1024;
        a->v = (int32_t *)realloc(a->v, (size_t)a->cap * sizeof(int32_t));
    }
    a->v[a->n++] = x;
}

typedef struct {
    double L;
    int64_t n;
    const uint8_t *level;
    const uint32_t *begin, *count;
    const int32_t *first_child;
    const uint8_t *child_mask;
    const double *mono;
} orc_tree_view;

static void orc_visit(const orc_tree_view *T, int32_t t, int64_t gbegin, int64_t gend,
                      const double glo[3], const double ghi[3], double theta2, orc_ivec *lmono,
                      orc_ivec *ldirect)
{
    int64_t b = T->begin[t], e = b + T->count[t];
    int overlap = (b < gend) && (gbegin < e);
    if (!overlap) {
        double dl[3];
        for (int a = 0; a < 3; ++a) {
            double c = T->mono[4 * (int64_t)t + a];
            double u = glo[a] - c; /* one rounding */
            double v = c - ghi[a]; /* one rounding */
            double w = u > v ? u : v;
            dl[a] = w > 0.0 ? w : 0.0;
        }
        double d2 = fma(dl[2], dl[2], fma(dl[1], dl[1], dl[0] * dl[0]));
        double s = ldexp(T->L, -(int)T->level[t]); /* exact */
        if (s * s < theta2 * d2) {
            orc_push(lmono, t);
            return;
        }
    }
    if (T->first_child[t] >= 0) {
        int k = orc_popcount8(T->child_mask[t]);
        for (int u = 0; u < k; ++u)
            orc_visit(T, T->first_child[t] + u, gbegin, gend, glo, ghi, theta2, lmono, ldirect);
    } else {
        for (int64_t j = b; j < e; ++j) orc_push(ldirect, (int32_t)j);
    }
}

/* One pairwise term, Eqs. (4)-(6) PAPER.md:92-101 divided by the body's own mass (R1): the source
 * (cx,cy,cz,m) pulls the body at p with  m * d / (r2 * sqrt(r2)),  d = c - p,  r2 = |d|^2 + eps^2
 * (R13: same softened r for bodies and nodes), nothing if r2 == 0.  Extended precision so that the
 * oracle's own rounding (~1e-19) is far below the 1e-11 parity bound. */
static inline void orc_term(const long double p[3], const double *src, long double eps2,
                            long double a[3], long double *sumnorm)
{
    long double dx = (long double)src[0] - p[0];
    long double dy = (long double)src[1] - p[1];
    long double dz = (long double)src[2] - p[2];
    long double d2 = dx * dx + dy * dy + dz * dz;
    long double r2 = d2 + eps2;
    if (r2 > 0.0L) {
        long double f = (long double)src[3] / (r2 * sqrtl(r2));
        a[0] += f * dx;
        a[1] += f * dy;
        a[2] += f * dz;
        *sumnorm += fabsl(f) * sqrtl(d2);
    }
}

/* Lists of one group (for tests of the walk structure). Returns 0; lists are malloc'ed here and
 * must be released with orc_free. */
int orc_walk_lists(double L, int64_t n, const uint32_t *gstart, const uint8_t *level,
                   const uint32_t *begin, const uint32_t *count, const int32_t *first_child,
                   const uint8_t *child_mask, const double *mono, const double *glo, const double *ghi,
                   int64_t g, double theta, int32_t **list_mono, int64_t *n_mono,
                   int32_t **list_direct, int64_t *n_direct)
{
    orc_tree_view T = {L, n, level, begin, count, first_child, child_mask, mono};
    orc_ivec lm = {0, 0, 0}, ld = {0, 0, 0};
    int64_t gb = gstart[g], ge = gstart[g + 1];
    orc_visit(&T, 0, gb, ge, &glo[3 * g], &ghi[3 * g], theta * theta, &lm, &ld);
    *list_mono = lm.v;
    *n_mono = lm.n;
    *list_direct = ld.v;
    *n_direct = ld.n;
    return 0;
}

void orc_free(void *p) { free(p); }

/* ---------------------------------------------------------------------------------------------
 * O8 + O9  Accelerations of the bodies of groups [g0, g1): walk, then evaluate both lists for each
 * body of the group (a body skips itself in the direct list, Eq. (1) j != i), multiply by G and
 * store at the body's ORIGINAL index.  n_mono / n_direct (per group, indexed g - g0) and kappa
 * (per body, original index; sum of term norms over norm of the sum) may be NULL.
 * ------------------------------------------------------------------------------------------- */
void orc_accel(double L, int64_t n, const uint32_t *gstart, const uint8_t *level, const uint32_t *begin,
               const uint32_t *count, const int32_t *first_child, const uint8_t *child_mask,
               const double *mono, const double *sbody, const uint32_t *perm, const double *glo,
               const double *ghi, double theta, double eps, double G, int64_t g0, int64_t g1,
               double *acc, uint32_t *n_mono, uint32_t *n_direct, double *kappa)
{
    orc_tree_view T = {L, n, level, begin, count, first_child, child_mask, mono};
    long double eps2 = (long double)eps * (long double)eps;
#pragma omp parallel
    {
        orc_ivec lm = {0, 0, 0}, ld = {0, 0, 0};
#pragma omp for schedule(dynamic, 4)
        for (int64_t g = g0; g < g1; ++g) {
            int64_t gb = gstart[g], ge = gstart[g + 1];
            lm.n = 0;
            ld.n = 0;
            orc_visit(&T, 0, gb, ge, &glo[3 * g], &ghi[3 * g], theta * theta, &lm, &ld);
            if (n_mono) n_mono[g - g0] = (uint32_t)lm.n;
            if (n_direct) n_direct[g - g0] = (uint32_t)ld.n;
            for (int64_t j = gb; j < ge; ++j) {
                long double p[3] = {sbody[4 * j], sbody[4 * j + 1], sbody[4 * j + 2]};
                long double a[3] = {0.0L, 0.0L, 0.0L}, sn = 0.0L;
                for (int64_t k = 0; k < lm.n; ++k) orc_term(p, &mono[4 * (int64_t)lm.v[k]], eps2, a, &sn);
                for (int64_t k = 0; k < ld.n; ++k)
                    if (ld.v[k] != j) orc_term(p, &sbody[4 * (int64_t)ld.v[k]], eps2, a, &sn);
                int64_t i = perm[j];
                for (int c = 0; c < 3; ++c) acc[3 * i + c] = (double)((long double)G * a[c]);
                if (kappa) {
                    long double nn = sqrtl(a[0] * a[0] + a[1] * a[1] + a[2] * a[2]);
                    kappa[i] = nn > 0.0L ? (double)(sn / nn) : 0.0;
                }
            }
        }
        free(lm.v);
        free(ld.v);
    }
}

/* ---------------------------------------------------------------------------------------------
 * O10  Direct sum, Eq. (1) PAPER.md:55 (reading R1: a_i = G * sum_{k != i} m_k R_ik / |R_ik|^3,
 * R_ik = R_k - R_i, softened as Eq. (6)).  tgt == NULL: all n bodies, acc[n][3]; else the nt
 * listed targets, acc[nt][3].
 * ------------------------------------------------------------------------------------------- */
void orc_direct(const double *pos, const double *mass, int64_t n, const int32_t *tgt, int64_t nt,
                double eps, double G, double *acc, double *kappa)
{
    long double eps2 = (long double)eps * (long double)eps;
    int64_t m = tgt ? nt : n;
#pragma omp parallel for schedule(dynamic, 16)
    for (int64_t r = 0; r < m; ++r) {
        int64_t i = tgt ? tgt[r] : r;
        long double p[3] = {pos[3 * i], pos[3 * i + 1], pos[3 * i + 2]};
        long double a[3] = {0.0L, 0.0L, 0.0L}, sn = 0.0L;
        for (int64_t k = 0; k < n; ++k) {
            if (k == i) continue;
            double src[4] = {pos[3 * k], pos[3 * k + 1], pos[3 * k + 2], mass[k]};
            orc_term(p, src, eps2, a, &sn);
        }
        for (int c = 0; c < 3; ++c) acc[3 * r + c] = (double)((long double)G * a[c]);
        if (kappa) {
            long double nn = sqrtl(a[0] * a[0] + a[1] * a[1] + a[2] * a[2]);
            kappa[r] = nn > 0.0L ? (double)(sn / nn) : 0.0;
        }
    }
}

/* ---------------------------------------------------------------------------------------------
 * O11  Leapfrog kick and drift (PAPER.md:148 lists leapfrog among the symplectic steppers;
 * reading R18).  Canonical arithmetic: v <- fma(a, h, v);  x <- fma(v, dt, x).
 * ------------------------------------------------------------------------------------------- */
void orc_kick(double *vel, const double *acc, int64_t n, double h)
{
    for (int64_t i = 0; i < 3 * n; ++i) vel[i] = fma(acc[i], h, vel[i]);
}

void orc_drift(double *pos, const double *vel, int64_t n, double dt)
{
    for (int64_t i = 0; i < 3 * n; ++i) pos[i] = fma(vel[i], dt, pos[i]);
}

/* =============================================================================================
 * Rows of SURVEY.md §8(f) ("next"): conservation diagnostics and the paper's stepping variants.
 * ========================================================================================== */

/* ---------------------------------------------------------------------------------------------
 * O12  Gravitational potential with the lists of the walk (NEXT-1: "Conservation of
 * energy, linear and angular momentum are checked for the purely gravitational case").  The paper
 * prints no potential; the one consistent with the softened force of Eqs. (4)-(6) (its gradient is
 * that force) is  phi_i = -G * sum_k m_k / sqrt(|d|^2 + eps^2),  nothing for a pair with r2 == 0,
 * a body skips itself (reading R24).  Same groups, same opening test, same lists as O8.
 * ------------------------------------------------------------------------------------------- */
static inline void orc_pot_term(const long double p[3], const double *src, long double eps2, long double *s)
{
    long double dx = (long double)src[0] - p[0];
    long double dy = (long double)src[1] - p[1];
    long double dz = (long double)src[2] - p[2];
    long double r2 = dx * dx + dy * dy + dz * dz + eps2;
    if (r2 > 0.0L) *s += (long double)src[3] / sqrtl(r2);
}

void orc_potential(double L, int64_t n, const uint32_t *gstart, const uint8_t *level, const uint32_t *begin,
                   const uint32_t *count, const int32_t *first_child, const uint8_t *child_mask,
                   const double *mono, const double *sbody, const uint32_t *perm, const double *glo,
                   const double *ghi, double theta, double eps, double G, int64_t g0, int64_t g1,
                   double *phi)
{
    orc_tree_view T = {L, n, level, begin, count, first_child, child_mask, mono};
    long double eps2 = (long double)eps * (long double)eps;
#pragma omp parallel
    {
        orc_ivec lm = {0, 0, 0}, ld = {0, 0, 0};
#pragma omp for schedule(dynamic, 4)
        for (int64_t g = g0; g < g1; ++g) {
            int64_t gb = gstart[g], ge = gstart[g + 1];
            lm.n = 0;
            ld.n = 0;
            orc_visit(&T, 0, gb, ge, &glo[3 * g], &ghi[3 * g], theta * theta, &lm, &ld);
            for (int64_t j = gb; j < ge; ++j) {
                long double p[3] = {sbody[4 * j], sbody[4 * j + 1], sbody[4 * j + 2]};
                long double s = 0.0L;
                for (int64_t k = 0; k < lm.n; ++k) orc_pot_term(p, &mono[4 * (int64_t)lm.v[k]], eps2, &s);
                for (int64_t k = 0; k < ld.n; ++k)
                    if (ld.v[k] != j) orc_pot_term(p, &sbody[4 * (int64_t)ld.v[k]], eps2, &s);
                phi[perm[j]] = (double)(-(long double)G * s);
            }
        }
        free(lm.v);
        free(ld.v);
    }
}

/* O13  Direct potential: phi_i = -G sum_{k != i} m_k / sqrt(|R_ik|^2 + eps^2) (plain definition). */
void orc_direct_potential(const double *pos, const double *mass, int64_t n, double eps, double G, double *phi)
{
    long double eps2 = (long double)eps * (long double)eps;
#pragma omp parallel for schedule(dynamic, 16)
    for (int64_t i = 0; i < n; ++i) {
        long double p[3] = {pos[3 * i], pos[3 * i + 1], pos[3 * i + 2]};
        long double s = 0.0L;
        for (int64_t k = 0; k < n; ++k) {
            if (k == i) continue;
            double src[4] = {pos[3 * k], pos[3 * k + 1], pos[3 * k + 2], mass[k]};
            orc_pot_term(p, src, eps2, &s);
        }
        phi[i] = (double)(-(long double)G * s);
    }
}

/* ---------------------------------------------------------------------------------------------
 * O14  Conserved quantities (energy, linear and angular momentum of the purely
 * gravitational system).  out[0] = kinetic energy  1/2 sum m |v|^2;  out[1] = potential energy
 * 1/2 sum m_i phi_i (every pair once; 0 if phi == NULL);  out[2..4] = linear momentum sum m v;
 * out[5..7] = angular momentum sum m x cross v (about the origin).  Extended-precision sums.
 * ------------------------------------------------------------------------------------------- */
void orc_diagnostics(const double *pos, const double *vel, const double *mass, const double *phi, int64_t n,
                     double out[8])
{
    long double ek = 0.0L, ep = 0.0L, P[3] = {0.0L, 0.0L, 0.0L}, Lm[3] = {0.0L, 0.0L, 0.0L};
    for (int64_t i = 0; i < n; ++i) {
        long double m = mass[i];
        long double x = pos[3 * i], y = pos[3 * i + 1], z = pos[3 * i + 2];
        long double vx = vel[3 * i], vy = vel[3 * i + 1], vz = vel[3 * i + 2];
        ek += 0.5L * m * (vx * vx + vy * vy + vz * vz);
        if (phi) ep += 0.5L * m * (long double)phi[i];
        P[0] += m * vx;
        P[1] += m * vy;
        P[2] += m * vz;
        Lm[0] += m * (y * vz - z * vy);
        Lm[1] += m * (z * vx - x * vz);
        Lm[2] += m * (x * vy - y * vx);
    }
    out[0] = (double)ek;
    out[1] = (double)ep;
    for (int c = 0; c < 3; ++c) {
        out[2 + c] = (double)P[c];
        out[5 + c] = (double)Lm[c];
    }
}

/* ---------------------------------------------------------------------------------------------
 * O15  Maximum relative position error, Eq. (7) PAPER.md:223:
 *     e_i = |r_i - r_i,ref| / |r_i,ref| * 100   (per cent),   result = max_i e_i.
 * Canonical arithmetic (compared bit for bit): d = r - r_ref per component (one rounding each);
 * |.|^2 = fma(z, z, fma(y, y, x*x));  e_i = 100 * sqrt(|d|^2 / |r_ref|^2).  A reference position at
 * the origin (|r_ref|^2 == 0) has no relative error and is skipped (reading R25).
 * ------------------------------------------------------------------------------------------- */
double orc_position_error(const double *pos, const double *ref, int64_t n)
{
    double worst = 0.0;
    for (int64_t i = 0; i < n; ++i) {
        double dx = pos[3 * i] - ref[3 * i], dy = pos[3 * i + 1] - ref[3 * i + 1], dz = pos[3 * i + 2] - ref[3 * i + 2];
        double nd = fma(dz, dz, fma(dy, dy, dx * dx));
        double nr = fma(ref[3 * i + 2], ref[3 * i + 2], fma(ref[3 * i + 1], ref[3 * i + 1], ref[3 * i] * ref[3 * i]));
        if (nr == 0.0) continue;
        double e = 100.0 * sqrt(nd / nr);
        if (e > worst) worst = e;
    }
    return worst;
}

/* ---------------------------------------------------------------------------------------------
 * O16  Gravity time-step bound, Eq. (8):  dt_g < T_g / 2 = 1 / (2 sqrt(G rho)).
 * Returns the bound 1 / (2 sqrt(G rho)).
 * ------------------------------------------------------------------------------------------- */
double orc_gravity_dt(double G, double rho) { return 1.0 / (2.0 * sqrt(G * rho)); }

/* =============================================================================================
 * Rows NEXT-3 and NEXT-4 of SURVEY.md §8(f): broad-phase collision detection and aggregate
 * identification.
 * ========================================================================================== */

/* ---------------------------------------------------------------------------------------------
 * O17  Broad phase: "pairs of bodies whose geometrical boundaries are close enough are
 * identified.  The bounding volume of a body is estimated based on its velocity and integration time
 * step.  If the bounding volume of two bodies overlap, the narrow phase is performed".
 * Reading R26: the bounding volume of body i is the sphere about its centre of radius
 *     b_i = fma(|v_i|, dt, R_i),   |v_i| = sqrt(fma(vz, vz, fma(vy, vy, vx*vx)))
 * (R_i the radius of the body's circumscribed sphere; within one step its boundary cannot leave that
 * sphere), and two volumes overlap iff  |x_j - x_i|^2 <= (b_i + b_j)^2  (touching counts), evaluated as
 *     d = x_j - x_i per component;  d2 = fma(dz, dz, fma(dy, dy, dx*dx));  s = b_i + b_j;  d2 <= s*s
 * with every operation rounded once, so that the set of pairs is reproducible bit for bit.
 * Plain definition: all i < j are tested.  orc_bound_radius fills b[n] (vel may be NULL: b = R).
 * orc_broadphase returns the number of pairs and writes the first `cap` of them, (i, j) with i < j, in
 * lexicographic order.
 * ------------------------------------------------------------------------------------------- */
void orc_bound_radius(const double *vel, const double *radius, int64_t n, double dt, double *b)
{
    for (int64_t i = 0; i < n; ++i) {
        if (!vel) {
            b[i] = radius[i];
            continue;
        }
        double vx = vel[3 * i], vy = vel[3 * i + 1], vz = vel[3 * i + 2];
        double sp = sqrt(fma(vz, vz, fma(vy, vy, vx * vx)));
        b[i] = fma(sp, dt, radius[i]);
    }
}

static inline int orc_overlap(const double *pos, const double *b, int64_t i, int64_t j)
{
    double dx = pos[3 * j] - pos[3 * i], dy = pos[3 * j + 1] - pos[3 * i + 1], dz = pos[3 * j + 2] - pos[3 * i + 2];
    double d2 = fma(dz, dz, fma(dy, dy, dx * dx));
    double s = b[i] + b[j];
    return d2 <= s * s;
}

int64_t orc_broadphase(const double *pos, const double *b, int64_t n, int32_t *pairs, int64_t cap)
{
    /* per-row counts in parallel, then rows are written in order */
    int64_t *cnt = (int64_t *)calloc((size_t)n + 1, sizeof(int64_t));
#pragma omp parallel for schedule(dynamic, 64)
    for (int64_t i = 0; i < n; ++i) {
        int64_t c = 0;
        for (int64_t j = i + 1; j < n; ++j) c += orc_overlap(pos, b, i, j);
        cnt[i + 1] = c;
    }
    for (int64_t i = 0; i < n; ++i) cnt[i + 1] += cnt[i];
    int64_t total = cnt[n];
#pragma omp parallel for schedule(dynamic, 64)
    for (int64_t i = 0; i < n; ++i) {
        int64_t at = cnt[i];
        if (at == cnt[i + 1]) continue;
        for (int64_t j = i + 1; j < n; ++j)
            if (orc_overlap(pos, b, i, j)) {
                if (at < cap) {
                    pairs[2 * at] = (int32_t)i;
                    pairs[2 * at + 1] = (int32_t)j;
                }
                ++at;
            }
    }
    free(cnt);
    return total;
}

/* ---------------------------------------------------------------------------------------------
 * O18  Aggregate identification: bodies are the vertices of a graph, contacts its
 * edges ("a contact container is filled with pairs ID_i, ID_j"); "aggregates obtained correspond to
 * the connected subgraphs"; "the number of aggregates is defined as the number of connected
 * components ... with a size greater than one"; "a Depth First Search (DFS) algorithm ... complexity
 * of O(N+E)".  Followed as written: adjacency lists from the pairs, DFS with an explicit stack from
 * every unvisited vertex in increasing id.  label[v] = id of the DFS root = smallest vertex of the
 * component (canonical, so it can be compared exactly); size[r] and mass[r] (sum of the members' masses
 * in increasing vertex id; mass_in may be NULL) are set at roots r and are 0 elsewhere.
 * counts[0] = connected components, counts[1] = aggregates (components with more than one body).
 * Self-pairs and repeated pairs are allowed and change nothing.  Returns 0, or -1 if a pair names a
 * vertex outside [0, n).
 * ------------------------------------------------------------------------------------------- */
int orc_aggregates(int64_t n, const int32_t *pairs, int64_t n_pairs, const double *mass_in, int32_t *label,
                   int32_t *size, double *mass, int64_t counts[2])
{
    int64_t *off = (int64_t *)calloc((size_t)n + 1, sizeof(int64_t));
    for (int64_t e = 0; e < n_pairs; ++e) {
        int32_t a = pairs[2 * e], b = pairs[2 * e + 1];
        if (a < 0 || b < 0 || a >= n || b >= n) {
            free(off);
            return -1;
        }
        ++off[a + 1];
        ++off[b + 1];
    }
    for (int64_t v = 0; v < n; ++v) off[v + 1] += off[v];
    int32_t *adj = (int32_t *)malloc(sizeof(int32_t) * (size_t)(2 * n_pairs + 1));
    int64_t *fill = (int64_t *)malloc(sizeof(int64_t) * (size_t)(n + 1));
    memcpy(fill, off, sizeof(int64_t) * (size_t)(n + 1));
    for (int64_t e = 0; e < n_pairs; ++e) {
        int32_t a = pairs[2 * e], b = pairs[2 * e + 1];
        adj[fill[a]++] = b;
        adj[fill[b]++] = a;
    }
    int32_t *stack = (int32_t *)malloc(sizeof(int32_t) * (size_t)(2 * n_pairs + n + 1));
    for (int64_t v = 0; v < n; ++v) {
        label[v] = -1;
        if (size) size[v] = 0;
        if (mass) mass[v] = 0.0;
    }
    counts[0] = counts[1] = 0;
    for (int64_t r = 0; r < n; ++r) {
        if (label[r] >= 0) continue;
        int64_t top = 0, members = 0;
        stack[top++] = (int32_t)r;
        label[r] = (int32_t)r;
        while (top > 0) {
            int32_t v = stack[--top];
            ++members;
            for (int64_t k = off[v]; k < off[v + 1]; ++k) {
                int32_t u = adj[k];
                if (label[u] < 0) {
                    label[u] = (int32_t)r;
                    stack[top++] = u;
                }
            }
        }
        if (size) size[r] = (int32_t)members;
        ++counts[0];
        if (members > 1) ++counts[1];
    }
    if (mass && mass_in)
        for (int64_t v = 0; v < n; ++v) mass[label[v]] += mass_in[v];
    free(off);
    free(adj);
    free(fill);
    free(stack);
    return 0;
}
