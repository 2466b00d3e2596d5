/*
 * oracle/bltc_cpu.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * Plain CPU barycentric Lagrange treecode (BLTC), written step by step from Section 6 and
 * Algorithm 3 of arXiv 2003.01833, in the paper's order and notation.
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs
 * may build, link or call this file.  It shares no code with the CUDA path (it links only
 * oracle/direct_sum.c for the kernel function G).
 *
 * Steps (O-2 in DESIGN.md), each with the passage it follows:
 *
 *  1. Tree of source clusters: root = all source particles; every cluster's
 *     box is the minimal bounding box of its particles; a cluster with more than N_L
 *     particles is bisected at the box midpoint in each "long" dimension (2, 4 or 8
 *     children, aspect-ratio rule sqrt(2)); recursion until <= N_L particles.
 *     Readings R4 (leaf iff count <= N_L) and R5 (split rule) in DESIGN.md.
 *  2. Target batches: "N_B = N_L ... the target batches are equivalent to the
 *     leaf source clusters"; otherwise the leaves of a second tree over the targets with N_B.
 *  3. Geometry of the MAC (Eq. (36), Fig. 8): centre = box
 *     midpoint, radius = half the box diagonal, R = distance between centres (reading R6).
 *  4. Interpolation points (Eq. (37)): s_k = cos(pi k / n), k = 0..n, mapped
 *     linearly to each cluster's box, per axis.
 *  5. Approximation weights / proxy charges (Eq. (35) right; barycentric form
 *     PAPER.md:416 Eq. (38); weights b_k = (-1)^k delta_k PAPER.md:421 Eq. (39)):
 *       fhat_k = sum_{r_j in C} L_k1(r_j1) L_k2(r_j2) L_k3(r_j3) f_j w_j,
 *     and the same with w_j alone (what_k), so singularity subtraction is exact in the far
 *     field (reading R11).  Reading R7: L_k(t) = delta_{k,k'} when t == s_k' exactly.
 *     Reading R9: from the cluster's own particles, not child-to-parent.
 *  6. ComputePotential(B, C), Algorithm 3 lines 4-12 with the text
 *     PAPER.md:434:  MAC satisfied -> Eq. (35) left;  fails on (r_B+r_C)/R >= theta -> leaf:
 *     direct sum Eq. (34), else recurse into children;  fails on (n+1)^3 >= N_S -> direct
 *     sum with the whole cluster (reading R10).  As in the paper's implementation
 *     ("interaction lists are precomputed for each target batch") the
 *     traversal records the lists first; the sums then run in list (= traversal) order.
 *  7. out_i = -2 (far + near + f_i/k^2), Eq. (18),(20),(21) as in oracle/direct_sum.c.
 *
 * Arithmetic: IEEE double, libm, no fast-math, no FMA contraction (build with
 * -ffp-contract=off); every sum over particles or interpolation points in long double.
 */
#include <math.h>
#include <omp.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

#ifndef M_PI
#define M_PI 3.14159265358979323846
#endif

double oracle_kernel(int kind, double k, double tx, double ty, double tz,
                     double sx, double sy, double sz, int* skip);   /* oracle/direct_sum.c */

#define SQRT2 1.4142135623730951

/* ------------------------------------------------------------------ tree */
typedef struct {
    int64_t begin, end;      /* particle range in tree order */
    double lo[3], hi[3];     /* minimal bounding box */
    int parent, level, nchild;
    int child[8];
} cluster_t;

typedef struct {
    int64_t n;               /* particles */
    const double* c[3];      /* caller's coordinates (not owned) */
    int64_t* perm;           /* tree order -> caller index */
    cluster_t* cl; int ncl, cap;
    int* leaf; int nleaf;    /* leaf cluster ids in DFS order */
    int max_per_leaf;
} tree_t;

static int new_cluster(tree_t* t)
{
    if (t->ncl == t->cap) {
        t->cap = t->cap ? 2 * t->cap : 1024;
        t->cl = (cluster_t*)realloc(t->cl, (size_t)t->cap * sizeof(cluster_t));
    }
    memset(&t->cl[t->ncl], 0, sizeof(cluster_t));
    return t->ncl++;
}

/* recursive bisection with shrink-to-fit boxes.  Returns the cluster id. */
static int build(tree_t* t, int64_t b, int64_t e, int parent, int level, int64_t* scratch)
{
    int id = new_cluster(t);
    cluster_t C;  memset(&C, 0, sizeof C);
    C.begin = b; C.end = e; C.parent = parent; C.level = level;
    /* "each cluster is shrunk to the minimal bounding box containing its particles" */
    for (int d = 0; d < 3; ++d) {
        double lo = t->c[d][t->perm[b]], hi = lo;
        for (int64_t i = b + 1; i < e; ++i) {
            double v = t->c[d][t->perm[i]];
            if (v < lo) lo = v;
            if (v > hi) hi = v;
        }
        C.lo[d] = lo; C.hi[d] = hi;
    }
    int64_t count = e - b;
    int split[3] = {0, 0, 0}, nsplit = 0;
    if (count > t->max_per_leaf) {                          /* R4 */
        double l[3], lmax = 0.0;
        for (int d = 0; d < 3; ++d) { l[d] = C.hi[d] - C.lo[d]; if (l[d] > lmax) lmax = l[d]; }
        /* R5: bisect every dimension whose extent is within a factor sqrt(2) of the longest */
        for (int d = 0; d < 3; ++d)
            if (l[d] > 0.0 && l[d] * SQRT2 >= lmax) { split[d] = 1; ++nsplit; }
    }
    if (nsplit > 0) {
        double mid[3];
        for (int d = 0; d < 3; ++d) mid[d] = 0.5 * (C.lo[d] + C.hi[d]);
        int64_t cnt[8] = {0,0,0,0,0,0,0,0};
        /* child code: bit0 = x upper, bit1 = y upper, bit2 = z upper (split axes only) */
        for (int64_t i = b; i < e; ++i) {
            int64_t p = t->perm[i]; int code = 0;
            for (int d = 0; d < 3; ++d) if (split[d] && t->c[d][p] > mid[d]) code |= (1 << d);
            ++cnt[code];
        }
        int nonempty = 0;
        for (int q = 0; q < 8; ++q) if (cnt[q]) ++nonempty;
        if (nonempty > 1) {
            int64_t start[8], pos[8], acc = b;
            for (int q = 0; q < 8; ++q) { start[q] = acc; pos[q] = acc; acc += cnt[q]; }
            /* stable partition by child code */
            for (int64_t i = b; i < e; ++i) {
                int64_t p = t->perm[i]; int code = 0;
                for (int d = 0; d < 3; ++d) if (split[d] && t->c[d][p] > mid[d]) code |= (1 << d);
                scratch[pos[code]++] = p;
            }
            memcpy(t->perm + b, scratch + b, (size_t)(e - b) * sizeof(int64_t));
            t->cl[id] = C;
            for (int q = 0; q < 8; ++q) {
                if (!cnt[q]) continue;                       /* empty children dropped */
                int ch = build(t, start[q], start[q] + cnt[q], id, level + 1, scratch);
                t->cl[id].child[t->cl[id].nchild++] = ch;
            }
            return id;
        }
        /* all particles fell into one child (midpoint rounded onto a face): leaf */
    }
    t->cl[id] = C;
    return id;
}

static void collect_leaves(tree_t* t, int id)
{
    if (t->cl[id].nchild == 0) { t->leaf[t->nleaf++] = id; return; }
    for (int q = 0; q < t->cl[id].nchild; ++q) collect_leaves(t, t->cl[id].child[q]);
}

static int tree_build(tree_t* t, int64_t n, const double* x, const double* y, const double* z,
                      int max_per_leaf)
{
    memset(t, 0, sizeof *t);
    t->n = n; t->c[0] = x; t->c[1] = y; t->c[2] = z; t->max_per_leaf = max_per_leaf;
    t->perm = (int64_t*)malloc((size_t)n * sizeof(int64_t));
    int64_t* scratch = (int64_t*)malloc((size_t)n * sizeof(int64_t));
    if (!t->perm || !scratch) return -1;
    for (int64_t i = 0; i < n; ++i) t->perm[i] = i;
    build(t, 0, n, -1, 0, scratch);
    free(scratch);
    t->leaf = (int*)malloc((size_t)t->ncl * sizeof(int));
    t->nleaf = 0;
    collect_leaves(t, 0);
    return 0;
}

static void tree_free(tree_t* t) { free(t->perm); free(t->cl); free(t->leaf); }

/* ------------------------------------------------------------------ plan */
typedef struct {
    int* v; int64_t n, cap;
} ivec_t;

static void ipush(ivec_t* a, int x)
{
    if (a->n == a->cap) { a->cap = a->cap ? 2 * a->cap : 256; a->v = (int*)realloc(a->v, (size_t)a->cap * sizeof(int)); }
    a->v[a->n++] = x;
}

typedef struct oracle_plan {
    int64_t N, M;
    int same;                       /* targets are the sources */
    int shared_batches;             /* batches are the source leaves */
    double theta; int degree, P, leaf_size, batch_size;
    double *sx, *sy, *sz, *tx, *ty, *tz;   /* owned copies, caller order */
    tree_t src, tgt;                /* tgt unused when shared_batches */
    int nbatch;
    int64_t *bbegin, *bend;         /* batch ranges in target tree order */
    double *blo, *bhi;              /* [nbatch][3] */
    const int64_t* tperm;           /* target tree order -> caller index */
    ivec_t far, near;               /* concatenated lists */
    int64_t *far_ptr, *near_ptr;    /* CSR offsets [nbatch+1] */
    double* nodes;                  /* [ncl][3][n+1], Eq. (37) mapped to the box */
    int64_t far_evals, near_evals;
    int upward_mode;                /* 0: proxy charges from the cluster's own particles (reading R9, the default);
                                       1: parents from their children (reading R23) */
} oracle_plan;

static double box_radius(const double* lo, const double* hi)
{
    double lx = hi[0] - lo[0], ly = hi[1] - lo[1], lz = hi[2] - lo[2];
    return 0.5 * sqrt((lx * lx + ly * ly) + lz * lz);
}

/* Algorithm 3, function ComputePotential(Batch, Cluster): records the decision. */
static void compute_potential(oracle_plan* p, int b, int c)
{
    const cluster_t* C = &p->src.cl[c];
    const double* blo = p->blo + 3 * b; const double* bhi = p->bhi + 3 * b;
    double rB = box_radius(blo, bhi), rC = box_radius(C->lo, C->hi);
    double dx = 0.5 * (blo[0] + bhi[0]) - 0.5 * (C->lo[0] + C->hi[0]);
    double dy = 0.5 * (blo[1] + bhi[1]) - 0.5 * (C->lo[1] + C->hi[1]);
    double dz = 0.5 * (blo[2] + bhi[2]) - 0.5 * (C->lo[2] + C->hi[2]);
    double R = sqrt((dx * dx + dy * dy) + dz * dz);
    int64_t NS = C->end - C->begin;
    int geometric = (rB + rC) < p->theta * R;             /* Eq. (36) left, R6 */
    int size_ok = (int64_t)p->P < NS;                     /* Eq. (36) right */
    /* R8: a box that is flat in some dimension cannot carry the tensor grid */
    if (C->hi[0] == C->lo[0] || C->hi[1] == C->lo[1] || C->hi[2] == C->lo[2]) size_ok = 0;
    if (geometric && size_ok) {                           /* line 5: MAC satisfied */
        ipush(&p->far, c);
    } else if (!geometric) {                              /* line 7 */
        if (C->nchild == 0) ipush(&p->near, c);           /* line 8 */
        else for (int q = 0; q < C->nchild; ++q) compute_potential(p, b, C->child[q]);  /* line 9 */
    } else {                                              /* line 10: (n+1)^3 >= N_S */
        ipush(&p->near, c);                               /* line 11 */
    }
}

oracle_plan* oracle_plan_create(int64_t N, const double* sx, const double* sy, const double* sz,
                                int64_t M, const double* tx, const double* ty, const double* tz,
                                double theta, int degree, int leaf_size, int batch_size)
{
    if (N <= 0 || degree < 1 || leaf_size < 1 || batch_size < 1 || !(theta >= 0.0) || !(theta < 1.0))
        return NULL;
    oracle_plan* p = (oracle_plan*)calloc(1, sizeof *p);
    p->N = N; p->theta = theta; p->degree = degree; p->P = (degree + 1) * (degree + 1) * (degree + 1);
    p->leaf_size = leaf_size; p->batch_size = batch_size;
    p->same = (tx == NULL);
    p->M = p->same ? N : M;
    size_t nb = (size_t)N * sizeof(double);
    p->sx = (double*)malloc(nb); p->sy = (double*)malloc(nb); p->sz = (double*)malloc(nb);
    memcpy(p->sx, sx, nb); memcpy(p->sy, sy, nb); memcpy(p->sz, sz, nb);
    if (p->same) { p->tx = p->sx; p->ty = p->sy; p->tz = p->sz; }
    else {
        size_t mb = (size_t)M * sizeof(double);
        p->tx = (double*)malloc(mb); p->ty = (double*)malloc(mb); p->tz = (double*)malloc(mb);
        memcpy(p->tx, tx, mb); memcpy(p->ty, ty, mb); memcpy(p->tz, tz, mb);
    }
    /* line 1: tree of source clusters and set of target batches */
    tree_build(&p->src, N, p->sx, p->sy, p->sz, leaf_size);
    p->shared_batches = p->same && (batch_size == leaf_size);
    const tree_t* bt = &p->src;
    if (!p->shared_batches) { tree_build(&p->tgt, p->M, p->tx, p->ty, p->tz, batch_size); bt = &p->tgt; }
    p->tperm = bt->perm;
    p->nbatch = bt->nleaf;
    p->bbegin = (int64_t*)malloc((size_t)p->nbatch * sizeof(int64_t));
    p->bend = (int64_t*)malloc((size_t)p->nbatch * sizeof(int64_t));
    p->blo = (double*)malloc((size_t)p->nbatch * 3 * sizeof(double));
    p->bhi = (double*)malloc((size_t)p->nbatch * 3 * sizeof(double));
    for (int b = 0; b < p->nbatch; ++b) {
        const cluster_t* L = &bt->cl[bt->leaf[b]];
        p->bbegin[b] = L->begin; p->bend[b] = L->end;
        for (int d = 0; d < 3; ++d) { p->blo[3 * b + d] = L->lo[d]; p->bhi[3 * b + d] = L->hi[d]; }
    }
    /* Eq. (37): s_k = cos(pi k / n) mapped linearly to each cluster's box, per axis */
    int n = degree;
    p->nodes = (double*)malloc((size_t)p->src.ncl * 3 * (n + 1) * sizeof(double));
    for (int c = 0; c < p->src.ncl; ++c)
        for (int d = 0; d < 3; ++d) {
            double mid = 0.5 * (p->src.cl[c].lo[d] + p->src.cl[c].hi[d]);
            double half = 0.5 * (p->src.cl[c].hi[d] - p->src.cl[c].lo[d]);
            for (int k = 0; k <= n; ++k)
                p->nodes[((size_t)c * 3 + d) * (n + 1) + k] = mid + half * cos((M_PI * k) / n);
        }
    /* line 3 (decision part): for each target batch, ComputePotential(B, root) */
    p->far_ptr = (int64_t*)malloc((size_t)(p->nbatch + 1) * sizeof(int64_t));
    p->near_ptr = (int64_t*)malloc((size_t)(p->nbatch + 1) * sizeof(int64_t));
    for (int b = 0; b < p->nbatch; ++b) {
        p->far_ptr[b] = p->far.n; p->near_ptr[b] = p->near.n;
        compute_potential(p, b, 0);
        int64_t nt = p->bend[b] - p->bbegin[b];
        for (int64_t q = p->far_ptr[b]; q < p->far.n; ++q) p->far_evals += nt * p->P;
        for (int64_t q = p->near_ptr[b]; q < p->near.n; ++q)
            p->near_evals += nt * (p->src.cl[p->near.v[q]].end - p->src.cl[p->near.v[q]].begin);
    }
    p->far_ptr[p->nbatch] = p->far.n; p->near_ptr[p->nbatch] = p->near.n;
    return p;
}

void oracle_plan_destroy(oracle_plan* p)
{
    if (!p) return;
    if (!p->same) { free(p->tx); free(p->ty); free(p->tz); }
    free(p->sx); free(p->sy); free(p->sz);
    tree_free(&p->src); if (!p->shared_batches) tree_free(&p->tgt);
    free(p->bbegin); free(p->bend); free(p->blo); free(p->bhi);
    free(p->far.v); free(p->near.v); free(p->far_ptr); free(p->near_ptr); free(p->nodes);
    free(p);
}

/* sizes: [0]=clusters [1]=leaves [2]=batches [3]=far entries [4]=near entries
 *        [5]=far evaluations [6]=near evaluations [7]=shared_batches */
void oracle_plan_sizes(const oracle_plan* p, int64_t* s)
{
    s[0] = p->src.ncl; s[1] = p->src.nleaf; s[2] = p->nbatch; s[3] = p->far.n; s[4] = p->near.n;
    s[5] = p->far_evals; s[6] = p->near_evals; s[7] = p->shared_batches;
}

/* Export for structural comparison.  Any pointer may be NULL. */
void oracle_plan_export(const oracle_plan* p, int64_t* src_perm, int64_t* tgt_perm,
                        int64_t* cl_begin, int64_t* cl_end, double* cl_lo, double* cl_hi,
                        int32_t* cl_parent, int32_t* cl_nchild,
                        int64_t* b_begin, int64_t* b_end,
                        int64_t* far_ptr, int32_t* far_idx, int64_t* near_ptr, int32_t* near_idx)
{
    if (src_perm) memcpy(src_perm, p->src.perm, (size_t)p->N * sizeof(int64_t));
    if (tgt_perm) memcpy(tgt_perm, p->tperm, (size_t)p->M * sizeof(int64_t));
    for (int c = 0; c < p->src.ncl; ++c) {
        const cluster_t* C = &p->src.cl[c];
        if (cl_begin) cl_begin[c] = C->begin;
        if (cl_end) cl_end[c] = C->end;
        if (cl_lo) for (int d = 0; d < 3; ++d) cl_lo[3 * c + d] = C->lo[d];
        if (cl_hi) for (int d = 0; d < 3; ++d) cl_hi[3 * c + d] = C->hi[d];
        if (cl_parent) cl_parent[c] = C->parent;
        if (cl_nchild) cl_nchild[c] = C->nchild;
    }
    for (int b = 0; b < p->nbatch; ++b) {
        if (b_begin) b_begin[b] = p->bbegin[b];
        if (b_end) b_end[b] = p->bend[b];
    }
    if (far_ptr) memcpy(far_ptr, p->far_ptr, (size_t)(p->nbatch + 1) * sizeof(int64_t));
    if (near_ptr) memcpy(near_ptr, p->near_ptr, (size_t)(p->nbatch + 1) * sizeof(int64_t));
    if (far_idx) for (int64_t q = 0; q < p->far.n; ++q) far_idx[q] = p->far.v[q];
    if (near_idx) for (int64_t q = 0; q < p->near.n; ++q) near_idx[q] = p->near.v[q];
}

/* ------------------------------------------------------------------ Eq. (38)-(39) */
/* L_k(t), k = 0..n, for nodes s[0..n]:  L_k(t) = (b_k/(t-s_k)) / sum_m (b_m/(t-s_m)),
 * b_k = (-1)^k delta_k, delta = 1/2 at k = 0, n.  R7: if t == s_k exactly, L = e_k. */
static void lagrange_row(int n, const double* s, double t, double* L)
{
    for (int k = 0; k <= n; ++k)
        if (t == s[k]) { for (int m = 0; m <= n; ++m) L[m] = 0.0; L[k] = 1.0; return; }
    long double denom = 0.0L;
    for (int m = 0; m <= n; ++m) {
        double b = ((m % 2) ? -1.0 : 1.0) * ((m == 0 || m == n) ? 0.5 : 1.0);
        L[m] = b / (t - s[m]);
        denom += (long double)L[m];
    }
    double dn = (double)denom;
    for (int m = 0; m <= n; ++m) L[m] = L[m] / dn;
}

/* Eq. (35) right: modified charges of cluster c for charge vector q (tree order index via perm).
 * qhat[(k1*(n+1)+k2)*(n+1)+k3]. */
static void proxy_charges(const oracle_plan* p, int c, const double* q_caller, double* qhat)
{
    int n = p->degree, n1 = n + 1;
    const cluster_t* C = &p->src.cl[c];
    const double* s = p->nodes + (size_t)c * 3 * n1;
    long double* acc = (long double*)calloc((size_t)p->P, sizeof(long double));
    double* L = (double*)malloc((size_t)3 * n1 * sizeof(double));
    for (int64_t i = C->begin; i < C->end; ++i) {
        int64_t j = p->src.perm[i];
        lagrange_row(n, s, p->sx[j], L);
        lagrange_row(n, s + n1, p->sy[j], L + n1);
        lagrange_row(n, s + 2 * n1, p->sz[j], L + 2 * n1);
        double qj = q_caller[j];
        for (int k1 = 0; k1 < n1; ++k1)
            for (int k2 = 0; k2 < n1; ++k2)
                for (int k3 = 0; k3 < n1; ++k3)
                    acc[(k1 * n1 + k2) * n1 + k3] +=
                        (long double)(L[k1] * L[n1 + k2] * L[2 * n1 + k3] * qj);
    }
    for (int k = 0; k < p->P; ++k) qhat[k] = (double)acc[k];
    free(acc); free(L);
}

/* ------------------------------------------------------------------ child -> parent upward pass
 * SURVEY.md 8(f) NEXT-4 (a variant the paper does not spell out: Alg. 3 line 2 only says "computes the approximation
 * weights for each source cluster").  Reading R23: the proxy charges of a LEAF come from
 * its particles, Eq. (35) right; those of an INTERNAL cluster P are the same formula applied to its children's
 * proxy points carrying the children's proxy charges,
 *     qhat^P_K = sum over children c, sum over k'  L^P_K1(s^c_k1') L^P_K2(s^c_k2') L^P_K3(s^c_k3')  qhat^c_k'
 * (L^P = the barycentric basis of P's grid, Eq. (38)-(39), with the node-hit rule R7: children share box faces with
 * their parent, so endpoint nodes do coincide).  In exact arithmetic this gives the SAME charges as Eq. (35) applied
 * to P's own particles: sum_k' L^P_K(s^c_k') L^c_k'(y) is the degree-n interpolant of the degree-n polynomial L^P_K,
 * i.e. L^P_K(y) itself.  Only the rounding differs (and the cost: O(N P) instead of O(N P depth)).
 * A child whose box is degenerate on an axis (R8) has no grid; a parent with such a child takes its charges from
 * its own particles instead. */
void oracle_plan_set_upward(oracle_plan* p, int mode) { if (p) p->upward_mode = mode ? 1 : 0; }

static int box_is_flat(const cluster_t* C)
{
    return C->hi[0] == C->lo[0] || C->hi[1] == C->lo[1] || C->hi[2] == C->lo[2];
}

static int from_children(const oracle_plan* p, int c)
{
    const cluster_t* C = &p->src.cl[c];
    if (!p->upward_mode || C->nchild == 0) return 0;
    for (int q = 0; q < C->nchild; ++q) if (box_is_flat(&p->src.cl[C->child[q]])) return 0;
    return 1;
}

static void charges_from_children(const oracle_plan* p, int c, double* const* qall, double* qhat)
{
    int n = p->degree, n1 = n + 1, P = p->P;
    const cluster_t* C = &p->src.cl[c];
    const double* sP = p->nodes + (size_t)c * 3 * n1;
    long double* acc = (long double*)calloc((size_t)P, sizeof(long double));
    double* L = (double*)malloc((size_t)3 * n1 * n1 * sizeof(double));     /* L[d][k'][K] = L^P_K(s^c_{d,k'}) */
    for (int q = 0; q < C->nchild; ++q) {
        int ch = C->child[q];
        const double* sC = p->nodes + (size_t)ch * 3 * n1;
        const double* qc = qall[ch];
        for (int d = 0; d < 3; ++d)
            for (int kp = 0; kp < n1; ++kp)
                lagrange_row(n, sP + d * n1, sC[d * n1 + kp], L + ((size_t)d * n1 + kp) * n1);
        for (int a1 = 0; a1 < n1; ++a1)
            for (int a2 = 0; a2 < n1; ++a2)
                for (int a3 = 0; a3 < n1; ++a3) {
                    double qk = qc[(a1 * n1 + a2) * n1 + a3];
                    const double* L1 = L + ((size_t)0 * n1 + a1) * n1;
                    const double* L2 = L + ((size_t)1 * n1 + a2) * n1;
                    const double* L3 = L + ((size_t)2 * n1 + a3) * n1;
                    for (int k1 = 0; k1 < n1; ++k1)
                        for (int k2 = 0; k2 < n1; ++k2)
                            for (int k3 = 0; k3 < n1; ++k3)
                                acc[(k1 * n1 + k2) * n1 + k3] += (long double)(L1[k1] * L2[k2] * L3[k3] * qk);
                }
    }
    for (int k = 0; k < P; ++k) qhat[k] = (double)acc[k];
    free(acc); free(L);
}

/* Proxy charges of every cluster with need[c] != 0, in the plan's upward mode: out[c] = malloc'd double[P] (caller
 * frees all non-NULL entries; mode 1 also leaves the descendants it had to compute).  Levels are processed deepest
 * first; clusters of one level are independent. */
static void proxy_charges_needed(const oracle_plan* p, const char* need, const double* q_caller, double** out)
{
    int ncl = p->src.ncl, P = p->P;
    char* use = (char*)calloc((size_t)ncl, 1);
    int maxlevel = 0;
    for (int c = 0; c < ncl; ++c) {                         /* pre-order: parents before children */
        if (need[c]) use[c] = 1;
        if (use[c] && from_children(p, c))
            for (int q = 0; q < p->src.cl[c].nchild; ++q) use[p->src.cl[c].child[q]] = 1;
        if (p->src.cl[c].level > maxlevel) maxlevel = p->src.cl[c].level;
    }
    for (int level = maxlevel; level >= 0; --level) {
        int c;
#pragma omp parallel for schedule(dynamic, 1)
        for (c = 0; c < ncl; ++c) {
            if (!use[c] || p->src.cl[c].level != level) continue;
            out[c] = (double*)malloc((size_t)P * sizeof(double));
            if (from_children(p, c)) charges_from_children(p, c, out, out[c]);
            else proxy_charges(p, c, q_caller, out[c]);
        }
    }
    free(use);
}

/* Exposed for the pins: proxy charges (in the plan's upward mode) and nodes of one cluster. */
int oracle_plan_proxy(const oracle_plan* p, int c, const double* q_caller, double* qhat, double* nodes3)
{
    if (c < 0 || c >= p->src.ncl) return -1;
    char* need = (char*)calloc((size_t)p->src.ncl, 1);
    double** all = (double**)calloc((size_t)p->src.ncl, sizeof(double*));
    need[c] = 1;
    proxy_charges_needed(p, need, q_caller, all);
    memcpy(qhat, all[c], (size_t)p->P * sizeof(double));
    for (int i = 0; i < p->src.ncl; ++i) free(all[i]);
    free(all); free(need);
    if (nodes3) memcpy(nodes3, p->nodes + (size_t)c * 3 * (p->degree + 1), (size_t)3 * (p->degree + 1) * sizeof(double));
    return 0;
}

/* threads the parallel loops below use (reported beside the timed baseline) */
int oracle_max_threads(void) { return omp_get_max_threads(); }

/* wall-clock seconds of the last evaluation's two phases: [0] proxy charges (Alg. 3 line 2), [1] batch-cluster sums
 * (line 3).  Timing only -- bench.py scales a sampled run to the whole convolution phase by phase. */
static double g_phase_s[2];
void oracle_last_phase_seconds(double out[2]) { out[0] = g_phase_s[0]; out[1] = g_phase_s[1]; }

/* ------------------------------------------------------------------ evaluation */
/* One orbital.  w, f_src: [N] caller order.  f_tgt: [M] caller order (NULL unless subtract;
 * when targets are the sources pass f_tgt = f_src).  sel: batch ids to evaluate (NULL = all);
 * out[M] caller order, written only for targets of evaluated batches.
 * parts (optional, [2][M]): raw far and near sums S_far, S_near per target. */
int oracle_bltc_eval(const oracle_plan* p, int kind, const double* w, const double* f_src,
                     const double* f_tgt, double k, int subtract, int finalize,
                     int64_t nsel, const int64_t* sel, double* out, double* parts)
{
    if (!p || !w || !f_src || !out) return -1;
    if (subtract && !f_tgt) return -1;
    if (kind == 0 && !(k > 0.0)) return -1;
    int n1 = p->degree + 1, ncl = p->src.ncl;
    int64_t nb = sel ? nsel : p->nbatch;
    /* line 2: approximation weights, for the clusters the selected batches approximate */
    char* need = (char*)calloc((size_t)ncl, 1);
    for (int64_t s = 0; s < nb; ++s) {
        int64_t b = sel ? sel[s] : s;
        if (b < 0 || b >= p->nbatch) { free(need); return -1; }
        for (int64_t q = p->far_ptr[b]; q < p->far_ptr[b + 1]; ++q) need[p->far.v[q]] = 1;
    }
    double** fhat = (double**)calloc((size_t)ncl, sizeof(double*));
    double** what = (double**)calloc((size_t)ncl, sizeof(double*));
    double* fw = (double*)malloc((size_t)p->N * sizeof(double));
    for (int64_t j = 0; j < p->N; ++j) fw[j] = f_src[j] * w[j];
    int c;
    double t_phase0 = omp_get_wtime();
    proxy_charges_needed(p, need, fw, fhat);
    if (subtract) proxy_charges_needed(p, need, w, what);
    /* line 3: for each target batch, the recorded batch-cluster interactions */
    /* Targets are independent (each one's sums are accumulated by one thread, in the order written below), so the
     * threads share the flat list of the selected batches' targets -- a sample of a few batches keeps every core busy. */
    int64_t ntg = 0, u;
    for (int64_t s = 0; s < nb; ++s) { int64_t b = sel ? sel[s] : s; ntg += p->bend[b] - p->bbegin[b]; }
    int64_t* tg_it = (int64_t*)malloc((size_t)(ntg ? ntg : 1) * sizeof(int64_t));
    int64_t* tg_b = (int64_t*)malloc((size_t)(ntg ? ntg : 1) * sizeof(int64_t));
    ntg = 0;
    for (int64_t s = 0; s < nb; ++s) {
        int64_t b = sel ? sel[s] : s;
        for (int64_t it = p->bbegin[b]; it < p->bend[b]; ++it) { tg_it[ntg] = it; tg_b[ntg] = b; ++ntg; }
    }
    double t_phase1 = omp_get_wtime();
#pragma omp parallel for schedule(dynamic, 16)
    for (u = 0; u < ntg; ++u) {
        {
            int64_t b = tg_b[u], it = tg_it[u];
            int64_t i = p->tperm[it];
            double xi = p->tx[i], yi = p->ty[i], zi = p->tz[i];
            double fi = subtract ? f_tgt[i] : 0.0;
            long double Sfar = 0.0L, Snear = 0.0L;
            int skip;
            /* Eq. (35) left: sum_k G(r_i, s_k) fhat_k   [with subtraction: fhat_k - f_i what_k] */
            for (int64_t q = p->far_ptr[b]; q < p->far_ptr[b + 1]; ++q) {
                int cc = p->far.v[q];
                const double* sn = p->nodes + (size_t)cc * 3 * n1;
                for (int k1 = 0; k1 < n1; ++k1)
                    for (int k2 = 0; k2 < n1; ++k2)
                        for (int k3 = 0; k3 < n1; ++k3) {
                            int kk = (k1 * n1 + k2) * n1 + k3;
                            double G = oracle_kernel(kind, k, xi, yi, zi, sn[k1], sn[n1 + k2], sn[2 * n1 + k3], &skip);
                            if (skip) continue;
                            double qk = subtract ? (fhat[cc][kk] - fi * what[cc][kk]) : fhat[cc][kk];
                            Sfar += (long double)(G * qk);
                        }
            }
            /* Eq. (34): sum_{r_j in C} G(r_i, r_j) f_j w_j   [with subtraction: (f_j - f_i) w_j] */
            for (int64_t q = p->near_ptr[b]; q < p->near_ptr[b + 1]; ++q) {
                const cluster_t* C = &p->src.cl[p->near.v[q]];
                for (int64_t jt = C->begin; jt < C->end; ++jt) {
                    int64_t j = p->src.perm[jt];
                    double G = oracle_kernel(kind, k, xi, yi, zi, p->sx[j], p->sy[j], p->sz[j], &skip);
                    if (skip) continue;
                    double df = subtract ? (f_src[j] - fi) : f_src[j];
                    Snear += (long double)(G * w[j] * df);
                }
            }
            long double S = Sfar + Snear;
            if (parts) { parts[i] = (double)Sfar; parts[p->M + i] = (double)Snear; }
            if (finalize) {
                if (subtract) S += (long double)fi / ((long double)k * (long double)k);
                out[i] = (double)(-2.0L * S);
            } else out[i] = (double)S;
        }
    }
    g_phase_s[0] = t_phase1 - t_phase0; g_phase_s[1] = omp_get_wtime() - t_phase1;
    for (c = 0; c < ncl; ++c) { free(fhat[c]); free(what[c]); }
    free(fhat); free(what); free(fw); free(need); free(tg_it); free(tg_b);
    return 0;
}

/* ------------------------------------------------------------------ evaluation, Coulomb kernel
 * Hartree potential (Eq. (19)) through the same treecode, with the Gaussian singularity
 * subtraction of PAPER.md:220-224 Eq. (23)-(24) (O-3 in DESIGN.md; direct definition in
 * oracle/coulomb_sum.c).  "Singularity subtraction ... can be easily accommodated in the BLTC"
 * -- not shown; reading R21: the first integrand of Eq. (23) is the sum of two
 * convolutions, kernel 1/r with charges f_j w_j and kernel e^{-r^2/alpha^2}/r with charges w_j
 * (times -f_i), and each is approximated by Eq. (35) with its own proxy charges:
 *   far  = sum_k [ fhat_k / |x_i - s_k|  -  f_i what_k e^{-|x_i - s_k|^2/alpha^2} / |x_i - s_k| ]
 *   near = sum_{r_j in C, r_ij != 0} (f_j - f_i e^{-r_ij^2/alpha^2}) w_j / r_ij          (Eq. (34))
 *   V_i  = far + near + 2 pi alpha^2 f_i                                               (Eq. (24))
 * Same lists, same proxy charges, same order of the sums as oracle_bltc_eval. */
double oracle_coulomb_term(double tx, double ty, double tz, double sx, double sy, double sz,
                           double fi, double fj, double wj, double alpha, int subtract, int* skip);  /* oracle/coulomb_sum.c */

int oracle_bltc_eval_coulomb(const oracle_plan* p, const double* w, const double* f_src,
                             const double* f_tgt, double alpha, int subtract,
                             int64_t nsel, const int64_t* sel, double* out, double* parts)
{
    if (!p || !w || !f_src || !out) return -1;
    if (subtract && (!f_tgt || !(alpha > 0.0))) return -1;
    int n1 = p->degree + 1, ncl = p->src.ncl;
    int64_t nb = sel ? nsel : p->nbatch;
    char* need = (char*)calloc((size_t)ncl, 1);
    for (int64_t s = 0; s < nb; ++s) {
        int64_t b = sel ? sel[s] : s;
        if (b < 0 || b >= p->nbatch) { free(need); return -1; }
        for (int64_t q = p->far_ptr[b]; q < p->far_ptr[b + 1]; ++q) need[p->far.v[q]] = 1;
    }
    double** fhat = (double**)calloc((size_t)ncl, sizeof(double*));
    double** what = (double**)calloc((size_t)ncl, sizeof(double*));
    double* fw = (double*)malloc((size_t)p->N * sizeof(double));
    for (int64_t j = 0; j < p->N; ++j) fw[j] = f_src[j] * w[j];
    int c;
    double t_phase0 = omp_get_wtime();
    proxy_charges_needed(p, need, fw, fhat);
    if (subtract) proxy_charges_needed(p, need, w, what);
    /* Targets are independent (each one's sums are accumulated by one thread, in the order written below), so the
     * threads share the flat list of the selected batches' targets -- a sample of a few batches keeps every core busy. */
    int64_t ntg = 0, u;
    for (int64_t s = 0; s < nb; ++s) { int64_t b = sel ? sel[s] : s; ntg += p->bend[b] - p->bbegin[b]; }
    int64_t* tg_it = (int64_t*)malloc((size_t)(ntg ? ntg : 1) * sizeof(int64_t));
    int64_t* tg_b = (int64_t*)malloc((size_t)(ntg ? ntg : 1) * sizeof(int64_t));
    ntg = 0;
    for (int64_t s = 0; s < nb; ++s) {
        int64_t b = sel ? sel[s] : s;
        for (int64_t it = p->bbegin[b]; it < p->bend[b]; ++it) { tg_it[ntg] = it; tg_b[ntg] = b; ++ntg; }
    }
    double t_phase1 = omp_get_wtime();
#pragma omp parallel for schedule(dynamic, 16)
    for (u = 0; u < ntg; ++u) {
        {
            int64_t b = tg_b[u], it = tg_it[u];
            int64_t i = p->tperm[it];
            double xi = p->tx[i], yi = p->ty[i], zi = p->tz[i];
            double fi = subtract ? f_tgt[i] : 0.0;
            long double Sfar = 0.0L, Snear = 0.0L;
            for (int64_t q = p->far_ptr[b]; q < p->far_ptr[b + 1]; ++q) {
                int cc = p->far.v[q];
                const double* sn = p->nodes + (size_t)cc * 3 * n1;
                for (int k1 = 0; k1 < n1; ++k1)
                    for (int k2 = 0; k2 < n1; ++k2)
                        for (int k3 = 0; k3 < n1; ++k3) {
                            int kk = (k1 * n1 + k2) * n1 + k3;
                            double dx = xi - sn[k1], dy = yi - sn[n1 + k2], dz = zi - sn[2 * n1 + k3];
                            double r2 = dx * dx + dy * dy + dz * dz;
                            double r = sqrt(r2);
                            if (r == 0.0) continue;
                            double t = fhat[cc][kk] / r;
                            if (subtract) t -= fi * what[cc][kk] * exp(-r2 / (alpha * alpha)) / r;
                            Sfar += (long double)t;
                        }
            }
            for (int64_t q = p->near_ptr[b]; q < p->near_ptr[b + 1]; ++q) {
                const cluster_t* C = &p->src.cl[p->near.v[q]];
                for (int64_t jt = C->begin; jt < C->end; ++jt) {
                    int64_t j = p->src.perm[jt];
                    int skip;
                    double t = oracle_coulomb_term(xi, yi, zi, p->sx[j], p->sy[j], p->sz[j], fi, f_src[j], w[j],
                                                   alpha, subtract, &skip);
                    if (skip) continue;
                    Snear += (long double)t;
                }
            }
            long double S = Sfar + Snear;
            if (parts) { parts[i] = (double)Sfar; parts[p->M + i] = (double)Snear; }
            if (subtract) S += 2.0L * (long double)M_PI * (long double)alpha * (long double)alpha * (long double)fi;
            out[i] = (double)S;
        }
    }
    g_phase_s[0] = t_phase1 - t_phase0; g_phase_s[1] = omp_get_wtime() - t_phase1;
    for (c = 0; c < ncl; ++c) { free(fhat[c]); free(what[c]); }
    free(fhat); free(what); free(fw); free(need); free(tg_it); free(tg_b);
    return 0;
}
