/*
 * oracle/unifrac_oracle.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * Plain, slow, obviously-correct CPU oracle for the UniFrac all-pairs distance
 * (section II: "UniFrac ... assesses differences between pairs of microbiome
 * profiles ... account[s] for the evolutionary relationships between microbes"; both the
 * "unweighted and the weighted normalized versions").  PAPER.md prints no formula; the two
 * ratios are the ones BASELINE.json:5 (north_star) names -- "len*(x xor y) and len*(x or y)"
 * for unweighted, "len*|u-v| and len*(u+v)" for weighted-normalized -- see DESIGN.md
 * readings Q1, Q2, Q9.
 *
 * The method reaches exactly (up to rounding order) the definitional result, so this oracle
 * IS the definition, written out pair by pair:
 *
 *   1. per sample s: cnt_s[v] = sum of the counts of the tips below v, obtained by walking
 *      every observed tip up to (excluding) the root ("computes each pair
 *      directly from the UniFrac definition by walking the tree", BASELINE.json:5);
 *      T_s = sum of the sample's counts.
 *   2. unweighted:  d = sum_v len_v*[x_av != x_bv] / sum_v len_v*[x_av or x_bv],
 *                   x_sv = (cnt_s[v] > 0);
 *   3. weighted-normalized:  d = sum_v len_v*|u_av - u_bv| / sum_v len_v*(u_av + u_bv),
 *                   u_sv = cnt_s[v] / T_s  (long double quotient of exact integers);
 *      sums over all non-root nodes v, in long double with Neumaier compensation;
 *   4. denominator == 0  ->  d = 0 (reading Q3).
 *
 * No levels, no bit packing, no separable sums, no tiling, no identities: none of the CUDA
 * path's shortcuts.  Shares no code with paper_2107_05397_b200/csrc.  Only tests/,
 * __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may use it.
 *
 * Two drivers over the same definition:
 *   oracle_unifrac_all_pairs : dense cnt vectors, loops over every branch for every pair.
 *   oracle_unifrac_pair_list : for big inputs; per-sample sorted (node,cnt) lists of the
 *                              touched branches, merged per pair (branches touched by
 *                              neither sample contribute exactly 0 to both sums).
 * tests/test_oracle_pins.py pins both (hand-worked example, closed forms, scipy reductions,
 * brute force) and cross-checks them against each other.
 *
 * Build: gcc -O2 -fopenmp -shared -fPIC (oracle/oracle.py does it).  Parity: PINNED.
 */
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#include <math.h>
#ifdef _OPENMP
#include <omp.h>
#endif

enum { ORC_OK = 0, ORC_ERR_ARG = -1, ORC_ERR_TREE = -2, ORC_ERR_TABLE = -3, ORC_ERR_EMPTY_SAMPLE = -4,
       ORC_ERR_NOMEM = -5 };
enum { ORC_UNWEIGHTED = 0, ORC_WEIGHTED_NORMALIZED = 1 };

/* Neumaier-compensated accumulator in long double */
typedef struct { long double s, c; } nsum_t;
static inline void nsum_add(nsum_t *a, long double x)
{
    long double t = a->s + x;
    if (fabsl(a->s) >= fabsl(x)) a->c += (a->s - t) + x; else a->c += (x - t) + a->s;
    a->s = t;
}
static inline long double nsum_get(const nsum_t *a) { return a->s + a->c; }

/* ---- validation (readings Q4-Q8, Q10), written independently of the library ---- */
int oracle_validate(int32_t n_nodes, const int32_t *parent, const double *len, const int32_t *postorder,
                    int32_t n_samples, const int64_t *indptr, const int32_t *indices, const int32_t *counts)
{
    if (n_nodes < 1 || n_samples < 0 || !parent || !len || !postorder || !indptr) return ORC_ERR_ARG;
    int32_t root = -1;
    char *haschild = (char *)calloc((size_t)n_nodes, 1);
    int32_t *pos = (int32_t *)malloc(sizeof(int32_t) * (size_t)n_nodes);
    if (!haschild || !pos) { free(haschild); free(pos); return ORC_ERR_NOMEM; }
    int rc = ORC_OK;
    for (int32_t v = 0; v < n_nodes; ++v) {
        int32_t p = parent[v];
        if (p == -1) { if (root != -1) rc = ORC_ERR_TREE; root = v; }
        else if (p < 0 || p >= n_nodes || p == v) rc = ORC_ERR_TREE;
        else {
            haschild[p] = 1;
            if (!(len[v] >= 0.0) || isinf(len[v])) rc = ORC_ERR_TREE;   /* also rejects NaN */
        }
    }
    if (root == -1) rc = ORC_ERR_TREE;
    if (rc == ORC_OK) {
        for (int32_t v = 0; v < n_nodes; ++v) pos[v] = -1;
        for (int32_t k = 0; k < n_nodes; ++k) {
            int32_t v = postorder[k];
            if (v < 0 || v >= n_nodes || pos[v] != -1) { rc = ORC_ERR_TREE; break; }
            pos[v] = k;
        }
    }
    if (rc == ORC_OK) {
        if (postorder[n_nodes - 1] != root) rc = ORC_ERR_TREE;
        for (int32_t v = 0; v < n_nodes && rc == ORC_OK; ++v)
            if (parent[v] >= 0 && pos[v] >= pos[parent[v]]) rc = ORC_ERR_TREE;  /* children first => acyclic */
    }
    if (rc == ORC_OK) {
        if (indptr[0] != 0) rc = ORC_ERR_TABLE;
        for (int32_t s = 0; s < n_samples && rc == ORC_OK; ++s) {
            if (indptr[s + 1] < indptr[s]) { rc = ORC_ERR_TABLE; break; }
            int64_t tot = 0;
            for (int64_t k = indptr[s]; k < indptr[s + 1]; ++k) {
                int32_t t = indices[k];
                if (t < 0 || t >= n_nodes || haschild[t] || counts[k] < 0) { rc = ORC_ERR_TABLE; break; }
                if (k > indptr[s] && indices[k - 1] >= t) { rc = ORC_ERR_TABLE; break; }
                tot += counts[k];
            }
            if (rc == ORC_OK && tot == 0) rc = ORC_ERR_EMPTY_SAMPLE;
        }
    }
    free(haschild); free(pos);
    return rc;
}

/* step 1: cnt_s[v] by walking each observed tip to the root (root excluded) */
static int64_t walk_sample(const int32_t *parent, int64_t lo, int64_t hi, const int32_t *indices,
                           const int32_t *counts, int64_t *cnt /* zeroed [n_nodes] */)
{
    int64_t T = 0;
    for (int64_t k = lo; k < hi; ++k) {
        int64_t c = counts[k];
        if (c <= 0) continue;
        T += c;
        for (int32_t v = indices[k]; parent[v] >= 0; v = parent[v]) cnt[v] += c;
    }
    return T;
}

/* steps 2-4 for one pair given dense cnt vectors */
static double pair_dense(int32_t n_nodes, const int32_t *parent, const double *len, int variant,
                         const int64_t *ca, int64_t Ta, const int64_t *cb, int64_t Tb)
{
    nsum_t num = {0, 0}, den = {0, 0};
    for (int32_t v = 0; v < n_nodes; ++v) {
        if (parent[v] < 0) continue;                       /* the root has no branch (Q5) */
        long double l = (long double)len[v];
        if (variant == ORC_UNWEIGHTED) {
            int xa = ca[v] > 0, xb = cb[v] > 0;
            if (xa != xb) nsum_add(&num, l);
            if (xa || xb) nsum_add(&den, l);
        } else {
            long double u = (long double)ca[v] / (long double)Ta;
            long double w = (long double)cb[v] / (long double)Tb;
            nsum_add(&num, l * fabsl(u - w));
            nsum_add(&den, l * (u + w));
        }
    }
    long double D = nsum_get(&den);
    if (D == 0.0L) return 0.0;                              /* Q3 */
    return (double)(nsum_get(&num) / D);
}

/* ALL pairs, condensed row-major upper triangle (scipy squareform order). */
int oracle_unifrac_all_pairs(int32_t n_nodes, const int32_t *parent, const double *len,
                             int32_t n_samples, const int64_t *indptr, const int32_t *indices,
                             const int32_t *counts, int variant, double *out_condensed)
{
    if (variant != ORC_UNWEIGHTED && variant != ORC_WEIGHTED_NORMALIZED) return ORC_ERR_ARG;
    size_t nn = (size_t)n_nodes;
    int64_t *cnt = (int64_t *)calloc(nn * (size_t)n_samples, sizeof(int64_t));
    int64_t *T = (int64_t *)calloc((size_t)n_samples, sizeof(int64_t));
    if (!cnt || !T) { free(cnt); free(T); return ORC_ERR_NOMEM; }
    int rc = ORC_OK;
    for (int32_t s = 0; s < n_samples; ++s) {
        T[s] = walk_sample(parent, indptr[s], indptr[s + 1], indices, counts, cnt + nn * s);
        if (T[s] == 0) rc = ORC_ERR_EMPTY_SAMPLE;
    }
    if (rc == ORC_OK) {
        #pragma omp parallel for schedule(dynamic, 1)
        for (int32_t a = 0; a < n_samples; ++a) {
            int64_t base = (int64_t)a * (2LL * n_samples - a - 1) / 2;
            for (int32_t b = a + 1; b < n_samples; ++b)
                out_condensed[base + (b - a - 1)] =
                    pair_dense(n_nodes, parent, len, variant, cnt + nn * a, T[a], cnt + nn * b, T[b]);
        }
    }
    free(cnt); free(T);
    return rc;
}

/* d(a,b) for one ordered pair, including a == b (used for the d(a,a)=0 / symmetry pins). */
int oracle_unifrac_pair(int32_t n_nodes, const int32_t *parent, const double *len,
                        const int64_t *indptr, const int32_t *indices, const int32_t *counts,
                        int variant, int32_t a, int32_t b, double *out)
{
    size_t nn = (size_t)n_nodes;
    int64_t *ca = (int64_t *)calloc(nn, sizeof(int64_t)), *cb = (int64_t *)calloc(nn, sizeof(int64_t));
    if (!ca || !cb) { free(ca); free(cb); return ORC_ERR_NOMEM; }
    int64_t Ta = walk_sample(parent, indptr[a], indptr[a + 1], indices, counts, ca);
    int64_t Tb = walk_sample(parent, indptr[b], indptr[b + 1], indices, counts, cb);
    int rc = ORC_OK;
    if (Ta == 0 || Tb == 0) rc = ORC_ERR_EMPTY_SAMPLE;
    else *out = pair_dense(n_nodes, parent, len, variant, ca, Ta, cb, Tb);
    free(ca); free(cb);
    return rc;
}

/* ---- pair-list driver: sparse per-sample (node,cnt) lists, merged per pair ---- */
typedef struct { int32_t node; int64_t cnt; } ent_t;
static int ent_cmp(const void *x, const void *y)
{
    int32_t a = ((const ent_t *)x)->node, b = ((const ent_t *)y)->node;
    return (a > b) - (a < b);
}

static double pair_sparse(const double *len, int variant, const ent_t *ea, int64_t na, int64_t Ta,
                          const ent_t *eb, int64_t nb, int64_t Tb)
{
    nsum_t num = {0, 0}, den = {0, 0};
    int64_t i = 0, j = 0;
    while (i < na || j < nb) {
        int32_t v; int64_t ca = 0, cb = 0;
        if (j >= nb || (i < na && ea[i].node < eb[j].node)) { v = ea[i].node; ca = ea[i].cnt; ++i; }
        else if (i >= na || eb[j].node < ea[i].node)         { v = eb[j].node; cb = eb[j].cnt; ++j; }
        else { v = ea[i].node; ca = ea[i].cnt; cb = eb[j].cnt; ++i; ++j; }
        long double l = (long double)len[v];
        if (variant == ORC_UNWEIGHTED) {
            int xa = ca > 0, xb = cb > 0;
            if (xa != xb) nsum_add(&num, l);
            if (xa || xb) nsum_add(&den, l);
        } else {
            long double u = (long double)ca / (long double)Ta;
            long double w = (long double)cb / (long double)Tb;
            nsum_add(&num, l * fabsl(u - w));
            nsum_add(&den, l * (u + w));
        }
    }
    long double D = nsum_get(&den);
    if (D == 0.0L) return 0.0;
    return (double)(nsum_get(&num) / D);
}

int oracle_unifrac_pair_list(int32_t n_nodes, const int32_t *parent, const double *len,
                             int32_t n_samples, const int64_t *indptr, const int32_t *indices,
                             const int32_t *counts, int variant, int64_t n_pairs,
                             const int32_t *pair_a, const int32_t *pair_b, double *out)
{
    if (variant != ORC_UNWEIGHTED && variant != ORC_WEIGHTED_NORMALIZED) return ORC_ERR_ARG;
    char *used = (char *)calloc((size_t)n_samples, 1);
    ent_t **lists = (ent_t **)calloc((size_t)n_samples, sizeof(ent_t *));
    int64_t *nl = (int64_t *)calloc((size_t)n_samples, sizeof(int64_t));
    int64_t *T = (int64_t *)calloc((size_t)n_samples, sizeof(int64_t));
    if (!used || !lists || !nl || !T) { free(used); free(lists); free(nl); free(T); return ORC_ERR_NOMEM; }
    int rc = ORC_OK;
    for (int64_t k = 0; k < n_pairs; ++k) {
        if (pair_a[k] < 0 || pair_a[k] >= n_samples || pair_b[k] < 0 || pair_b[k] >= n_samples) rc = ORC_ERR_ARG;
        else { used[pair_a[k]] = 1; used[pair_b[k]] = 1; }
    }
    if (rc == ORC_OK) {
        #pragma omp parallel
        {
            int64_t *cnt = (int64_t *)calloc((size_t)n_nodes, sizeof(int64_t));
            int32_t *touched = (int32_t *)malloc(sizeof(int32_t) * (size_t)n_nodes);
            #pragma omp for schedule(dynamic, 8)
            for (int32_t s = 0; s < n_samples; ++s) {
                if (!used[s] || !cnt || !touched) continue;
                /* same walk as walk_sample, remembering which nodes were touched */
                int64_t nt = 0, Ts = 0;
                for (int64_t k = indptr[s]; k < indptr[s + 1]; ++k) {
                    int64_t c = counts[k];
                    if (c <= 0) continue;
                    Ts += c;
                    for (int32_t v = indices[k]; parent[v] >= 0; v = parent[v]) {
                        if (cnt[v] == 0) touched[nt++] = v;
                        cnt[v] += c;
                    }
                }
                ent_t *e = (ent_t *)malloc(sizeof(ent_t) * (size_t)(nt > 0 ? nt : 1));
                if (e) {
                    for (int64_t q = 0; q < nt; ++q) { e[q].node = touched[q]; e[q].cnt = cnt[touched[q]]; cnt[touched[q]] = 0; }
                    qsort(e, (size_t)nt, sizeof(ent_t), ent_cmp);
                }
                lists[s] = e; nl[s] = nt; T[s] = Ts;
            }
            free(cnt); free(touched);
        }
        for (int32_t s = 0; s < n_samples; ++s) if (used[s]) { if (!lists[s]) rc = ORC_ERR_NOMEM; else if (T[s] == 0) rc = ORC_ERR_EMPTY_SAMPLE; }
    }
    if (rc == ORC_OK) {
        #pragma omp parallel for schedule(dynamic, 64)
        for (int64_t k = 0; k < n_pairs; ++k) {
            int32_t a = pair_a[k], b = pair_b[k];
            out[k] = pair_sparse(len, variant, lists[a], nl[a], T[a], lists[b], nl[b], T[b]);
        }
    }
    for (int32_t s = 0; s < n_samples; ++s) free(lists[s]);
    free(used); free(lists); free(nl); free(T);
    return rc;
}

int oracle_num_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}
