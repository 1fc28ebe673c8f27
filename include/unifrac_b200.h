/*
 * unifrac_b200.h -- C ABI of libunifrac_b200.so: Striped/Hybrid UniFrac all-pairs distance on one
 * NVIDIA B200 (sm_100a).  Plain C; callers need no CUDA headers.
 *
 * What it computes ("a distance matrix of size N x N where N is the number of
 * samples"; section II: UniFrac from a phylogeny and a sparse sample x feature
 * table, "for both unweighted and the weighted normalized versions", with "fp32 compute
 * support"; formulas per BASELINE.json:5, readings Q1-Q3, Q9):
 *
 *   x_sv = 1 if sample s has any count on a tip below branch v, else 0
 *   u_sv = (sum of s's counts on tips below v) / (sum of all of s's counts)
 *   unweighted           d(a,b) = sum_v len_v*(x_av xor x_bv) / sum_v len_v*(x_av or x_bv)
 *   weighted-normalized  d(a,b) = sum_v len_v*|u_av - u_bv|   / sum_v len_v*(u_av + u_bv)
 *   sums over all non-root nodes v; a zero denominator gives d = 0.
 *
 * Every step (plan/validate, per-branch embedding, stripe accumulation, finalize) runs in the
 * library's own CUDA kernels; there is no CPU fallback.
 */
#ifndef UNIFRAC_B200_H
#define UNIFRAC_B200_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef enum { UNIFRAC_UNWEIGHTED = 0, UNIFRAC_WEIGHTED_NORMALIZED = 1 } unifrac_variant_t;
typedef enum { UNIFRAC_FP32 = 0, UNIFRAC_FP64 = 1 } unifrac_precision_t;

typedef enum {
    UNIFRAC_OK = 0,
    UNIFRAC_ERR_INVALID_ARG = -1,   /* null pointer, bad enum, n_samples < 2, n_nodes < 2 ...          */
    UNIFRAC_ERR_INVALID_TREE = -2,  /* not exactly one root, parent out of range, postorder not a
                                       permutation with children before parent and root last,
                                       negative / non-finite branch length                           */
    UNIFRAC_ERR_INVALID_TABLE = -3, /* indptr not monotone from 0, column not a tip node id, columns
                                       not strictly increasing within a row, negative count          */
    UNIFRAC_ERR_EMPTY_SAMPLE = -4,  /* a sample whose counts sum to 0 (u would be 0/0)                */
    UNIFRAC_ERR_WORKSPACE = -5,     /* the allocator returned NULL / device memory exhausted          */
    UNIFRAC_ERR_CUDA = -6,          /* a CUDA runtime call failed (see unifrac_last_cuda_error)       */
    UNIFRAC_ERR_UNSUPPORTED = -7    /* a sample total >= 2^32, or n_samples / n_nodes beyond limits   */
} unifrac_status_t;

/* flags (bit mask) */
#define UNIFRAC_FLAG_LITERAL          1u  /* debug: accumulate BOTH pairwise sums exactly as BASELINE.json:5
                                             words them (len*|u-v| and len*(u+v); len*xor and len*or) in a
                                             plain one-thread-per-pair fp64 kernel.  Slow; small inputs.   */
#define UNIFRAC_FLAG_TENSOR_GRAM      2u  /* accepted for compatibility: the tcgen05 int8 Gram path (X^T diag(len) X,
                                             len in 24-bit fixed point, exact int32 accumulation) is the DEFAULT for
                                             the head branches of unweighted + fp32 (it meets the 1e-5 tolerance,
                                             BASELINE.json:5); see UNIFRAC_FLAG_NO_TENSOR                    */
#define UNIFRAC_FLAG_SKIP_VALIDATION  4u  /* trust the inputs (tree/table checks are skipped)            */
#define UNIFRAC_FLAG_ABSDIFF          8u  /* stripe kernel accumulates |u~_i - u~_j| over rows present in
                                             EITHER tile (direct form) instead of min(u~_i,u~_j) over rows
                                             present in BOTH (separable form, I2-I5); implies
                                             NO_TAIL                                                      */
#define UNIFRAC_FLAG_NO_TAIL         16u  /* every branch goes through the dense stripe kernel (no sparse
                                             tail scatter)                 */
#define UNIFRAC_FLAG_ALL_TAIL        32u  /* debug: every branch goes through the sparse tail scatter       */
#define UNIFRAC_FLAG_NO_MID         128u  /* fp32: no shared-memory fixed-point "mid" kernel; branches are split into
                                             head and tail only                                            */
#define UNIFRAC_FLAG_SPARSE_STRIPE   256u  /* head branches on the sparse-aware compact-row stripe kernel (row flags, quarter masks)
                                             instead of the dense min-GEMM kernel                          */
#define UNIFRAC_FLAG_RICHNESS_ZONES  512u  /* weighted + fp32: sort the samples by richness inside the call and split step a-5 per
                                             (branch, tile): tile pairs inside a branch's dense zone on the register-tile kernel
                                             k_zone, the rest on the join.  Same results; pays off when
                                             presence is strongly clustered over the samples (on the iid synthetic configs it is
                                             as fast as the default per-branch split, so it is opt-in).  Ignored otherwise.     */
#define UNIFRAC_FLAG_NO_TENSOR       64u  /* unweighted + fp32: head branches on the CUDA-core stripe kernel
                                             instead of the tensor-core Gram kernel                        */

/* CSR table, rows = samples, columns = tip NODE ids (reading Q6). */
typedef struct {
    const int64_t *indptr;   /* [n_samples+1]  indptr[0] = 0, non-decreasing                          */
    const int32_t *indices;  /* [nnz]          node id of a tip; strictly increasing within a row    */
    const int32_t *counts;   /* [nnz]          >= 0 (0 = absent)                                      */
} unifrac_csr_t;

/* Device-memory allocator supplied by the caller (e.g. backed by torch.empty).  Must return a
 * device pointer aligned to 256 bytes, or NULL.  Buffers are owned by the caller and must stay
 * valid until the work unifrac_dm enqueued on `stream` has completed; the library never frees
 * them.  If `alloc` is NULL the library uses cudaMallocAsync / cudaFreeAsync on `stream`. */
typedef void *(*unifrac_alloc_fn)(size_t bytes, void *user);

/*
 * unifrac_dm -- fill the condensed N x N UniFrac distance matrix.
 *
 * All array arguments are DEVICE pointers, read-only, owned by the caller, not retained.
 *   n_nodes       number of tree nodes (tips + internal + root), >= 2
 *   tree_parent   [n_nodes] parent node id; exactly one entry is -1 (the root)
 *   branch_len    [n_nodes] length of the edge v -> parent[v]; >= 0 and finite; root's ignored
 *   postorder     [n_nodes] permutation of node ids, children before parent, root last
 *   table         CSR counts, see unifrac_csr_t
 *   n_samples     N >= 2
 *   variant       unweighted / weighted-normalized
 *   precision     UNIFRAC_FP32: embeddings, stripe accumulators and output are float (partial
 *                 sums are folded into fp64 every 512 rows; per-sample sums and the final
 *                 division are fp64);  UNIFRAC_FP64: everything double.
 *   out_condensed device; N*(N-1)/2 float or double; row-major upper triangle (scipy
 *                 squareform order): index(i,j) = i*(2N-i-1)/2 + (j-i-1), i < j.
 *   alloc/user    workspace allocator (see above); may be NULL.
 *   flags         UNIFRAC_FLAG_* mask
 *   stream        cudaStream_t (NULL = default stream)
 *
 * Returns a unifrac_status_t.  Host-checkable errors return before anything is enqueued.  The
 * plan step reads a few words back (one or more stream synchronisations), so data errors
 * (tree / table / empty sample) are also returned synchronously and leave `out_condensed`
 * untouched; after planning and embedding the stripe kernel is enqueued asynchronously and the
 * call returns without waiting for it.  Never throws, never aborts.
 */
int unifrac_dm(int32_t n_nodes, const int32_t *tree_parent, const double *branch_len,
               const int32_t *postorder, unifrac_csr_t table, int32_t n_samples,
               unifrac_variant_t variant, unifrac_precision_t precision, void *out_condensed,
               unifrac_alloc_fn alloc, void *alloc_user, uint32_t flags, void *stream);

/*
 * unifrac_dm_shard -- one shard of the same computation, for one process per GPU (the paper's "set of stripes" split,
 * independent pieces of the matrix, merged afterwards).  The upper triangle is cut into blocks of
 * UNIFRAC_SHARD_BLOCK x UNIFRAC_SHARD_BLOCK sample tiles (128 samples each) that are dealt round-robin to the shards:
 * block (bi <= bj) belongs to shard (bj*(bj+1)/2 + bi) % shard_count  (see unifrac_shard_of_pair).  Every shard
 * embeds the whole table (cheap) and runs step a-5 / a-6 only for its own blocks: no data-path communication.
 * On return (after the stream work completes) `out_condensed` holds the distances of the pairs this shard owns and
 * 0 everywhere else, so the full matrix is the element-wise SUM (or an all-gather by owner) of the shards' buffers.
 * shard_count = 1 is unifrac_dm.  0 <= shard_index < shard_count <= 255, else UNIFRAC_ERR_INVALID_ARG.
 * The debug flags LITERAL / ABSDIFF / SPARSE_STRIPE / NO_TAIL are not available in shard mode (UNIFRAC_ERR_INVALID_ARG).
 */
#define UNIFRAC_SHARD_BLOCK 12
int unifrac_dm_shard(int32_t n_nodes, const int32_t *tree_parent, const double *branch_len,
                     const int32_t *postorder, unifrac_csr_t table, int32_t n_samples,
                     unifrac_variant_t variant, unifrac_precision_t precision, void *out_condensed,
                     unifrac_alloc_fn alloc, void *alloc_user, uint32_t flags, void *stream,
                     int32_t shard_index, int32_t shard_count);

/* owner shard of the pair of samples (i, j), i != j  (host helper, no CUDA) */
int32_t unifrac_shard_of_pair(int32_t i, int32_t j, int32_t shard_count);

/*
 * unifrac_dm_host -- same computation with HOST buffers (pageable or pinned).  The library allocates device memory itself
 * from its OWN stream-ordered pool (one per device; other users of the device's default pool are not affected), copies the
 * inputs in, runs unifrac_dm on an internal stream, copies the condensed result out to `out_condensed_host`, returns every
 * buffer to the pool and returns after completion (synchronous).  The pool keeps its memory mapped for the next call;
 * unifrac_release_host_pool() gives it back to the device.  `nnz` is read from indptr[n_samples].
 */
int unifrac_dm_host(int32_t n_nodes, const int32_t *tree_parent, const double *branch_len,
                    const int32_t *postorder, unifrac_csr_t table_host, int32_t n_samples,
                    unifrac_variant_t variant, unifrac_precision_t precision,
                    void *out_condensed_host, uint32_t flags);

/*
 * unifrac_dm_host_multi -- both variants of one table in one call (the paper's use: "both unweighted and the weighted
 * normalized versions").  The inputs are uploaded once; variant k + 1 is computed while the result of variant k
 * travels back to the host on a second stream (unifrac_dm is asynchronous after its planning step).  variants[k] is a
 * unifrac_variant_t, outs_host[k] the host buffer of variant k (n(n-1)/2 elements); 1 <= n_variants <= 2.  Synchronous.
 */
int unifrac_dm_host_multi(int32_t n_nodes, const int32_t *tree_parent, const double *branch_len,
                          const int32_t *postorder, unifrac_csr_t table_host, int32_t n_samples,
                          int32_t n_variants, const int32_t *variants, unifrac_precision_t precision,
                          void *const *outs_host, uint32_t flags);

/* trims the host entry points' device memory pool(s) to zero (after the calls that used them have returned) */
int unifrac_release_host_pool(void);

/* Statistics of the calling thread's last unifrac_dm call (work counters are exact, computed on
 * the device from the per-branch sample counts; times are CUDA-event milliseconds, valid only
 * if UNIFRAC_B200_TIMING=1 is set in the environment -- timing synchronises the stream). */
typedef struct {
    uint64_t branches_embedded;  /* B_emb = #{v : len_v > 0 and some sample present}                 */
    uint64_t updates_dense;      /* W_dense = P * B_emb           (the metric's "pair x branch")      */
    uint64_t updates_union;      /* W_union = sum_v [C(N,2) - C(N-n_v,2)]                             */
    uint64_t updates_inter;      /* W_inter = sum_v C(n_v,2)                                          */
    uint64_t updates_executed;   /* (pair, branch) updates actually executed: head (stripe) + tail       */
    uint64_t updates_executed_head; /* ... by the stripe kernel (head branches)                          */
    uint64_t head_rows;          /* branches handled by the dense stripe kernel                       */
    uint64_t tail_rows;          /* branches handled by the sparse tail scatter                       */
    uint64_t tail_updates;       /* sum over tail branches of C(n_v,2) = RED.ADDs issued               */
    uint64_t tail_entries;       /* sum over tail and mid branches of n_v = (sample, value) list entries */
    uint64_t mid_rows;           /* branches handled by the shared-memory fixed-point kernel (fp32 mode)  */
    uint64_t mid_updates;        /* sum over mid branches of C(n_v,2) = shared-memory atomic adds          */
    uint64_t rows_staged;        /* rows the producer staged into shared memory, over all tile pairs  */
    uint64_t embed_rows;         /* sum over sample tiles of non-empty rows (compact embedding rows)  */
    uint64_t workspace_bytes;    /* device bytes requested from the allocator                         */
    uint64_t skip_updates_executed; /* RICHNESS_ZONES (k_zone): 128 x 128 pair updates per (row, tile pair) visit           */
    uint64_t skip_row_pair_visits;  /* (row, tile pair) visits of k_zone                                                     */
    uint64_t mid_atomics;        /* shared-memory atomics of the mid stage: one per (pair, lone mid row) and one per (pair, group root);
                                    = mid_updates without the grouped join                                                  */
    uint32_t n_tile_pairs;       /* 128x128 tile pairs in the upper triangle                          */
    uint32_t n_levels;           /* tree depth levels                                                 */
    uint32_t stripe_launches;    /* stripe-kernel launches in this call                               */
    uint32_t tail_launches;      /* tail-scatter launches (one per L2-resident super tile)             */
    uint32_t kernel_launches;    /* all kernel launches in this call                                  */
    uint32_t mid_launches;       /* launches of the mid kernel                                          */
    uint32_t mid_F;              /* its fixed-point scale: u_q = round(u * 2^F)                          */
    uint32_t gram;               /* 1 if the head branches went through the tcgen05 int8 Gram kernel    */
    uint32_t gram_k;             /* K (head branches, padded to 64) of that GEMM                       */
    uint32_t gram_q;             /* fixed-point scale: L_v = round(len_v * 2^q)                        */
    uint32_t dense;              /* 1 if the head branches went through the dense CUDA-core kernel (k_dense) */
    uint32_t skip;               /* 1 if the call used the per-(branch, tile) split k_zone + join (UNIFRAC_FLAG_RICHNESS_ZONES);
                                    then head_rows = rows with a dense copy, mid_rows = list_rows, mid_updates = joined updates */
    uint32_t skip_rows;          /* rows of the dense operand matrix of k_zone                                       */
    uint32_t list_rows;          /* non-tail rows (ordered by their tile cut D_v)                                    */
    uint32_t guard_pairs;        /* pairs with d < 1/16 that the near-duplicate guard recomputed from the definition */
    uint32_t guard_capacity;     /* size of the guard's pair list: min(P, max(2^22, 64 N)); pairs listed beyond it keep
                                    their separable-form value (absolute error ~1e-7 in fp32)                           */
    uint32_t mid_groups;         /* grouped join (k_midg): groups of nested mid branches ...                          */
    uint32_t mid_group_rows;     /* ... and the mid rows in them (the other mid_rows - mid_group_rows rows go through k_mid) */
    uint32_t quant_fallback;     /* 1 if the fixed-point error ratio was over budget and the call was rerun without
                                    the fixed-point kernels (tensor-core Gram, shared-memory mid)                       */
    float guard_theta;           /* the guard's threshold of this call: max(1/16, quant_err_ratio / 2.5e-6)            */
    float quant_err_ratio;       /* max over samples of (|sum delta| + 3 sqrt(sum delta^2)) / (side sum), delta = fixed-point
                                    value - value over the sample's Gram-head lengths and mid entries; over 1.25e-6 => rerun */
    float ms_plan, ms_embed, ms_tail, ms_mid, ms_stripe, ms_total;
} unifrac_stats_t;
int unifrac_last_stats(unifrac_stats_t *out);

/*
 * unifrac_mantel_pearson -- Mantel test with Pearson's correlation between two distance matrices that are already resident
 * in HBM (the test itself is the standard one).  x, y: condensed upper triangles (the
 * layout unifrac_dm writes) of two symmetric hollow n x n matrices; perms: n_perms permutations of 0..n-1, row-major
 * [n_perms][n], supplied by the caller (the library draws no random numbers).  With X^pi[i][j] = X[pi(i)][pi(j)]:
 *     out[0] = r = Pearson(x, y);   out[4 + k] = r_k = Pearson(condensed(X^pi_k), y),  k = 0 .. n_perms-1
 *     out[1], out[2], out[3] = p-values (count + 1) / (n_perms + 1) with count = #{|r_k| >= |r|}, #{r_k >= r}, #{r_k <= r}
 * All pointers are DEVICE pointers; out has 4 + n_perms doubles; precision selects float / double inputs; sums are fp64.
 * Workspace (the square copy of X, n*n elements) comes from `alloc` (NULL: cudaMallocAsync).  A constant matrix (zero variance)
 * gives r = 0.  n < 3: UNIFRAC_ERR_INVALID_ARG.  Permutations are not validated.  Asynchronous on `stream`.
 */
int unifrac_mantel_pearson(int32_t n_samples, const void *x_condensed, const void *y_condensed,
                           unifrac_precision_t precision, const int32_t *perms, int32_t n_perms, double *out,
                           unifrac_alloc_fn alloc, void *alloc_user, void *stream);

/*
 * unifrac_mantel_pearson_noalloc -- unifrac_mantel_pearson for callers that cannot allocate (code under CUDA graph capture,
 * tight serving loops, harnesses that forbid cudaMalloc): the same kernels and the same result, with the workspace (square
 * copy of X, per-CTA partial sums, moments) in a static device array of UNIFRAC_NOALLOC_SCRATCH_BYTES inside the library
 * instead of an allocator.  Every GPU that loads the library holds that array until the process exits.  The call makes no
 * cudaMalloc / cudaFree / cudaMallocAsync and calls no allocating library routine; the caller passes inputs and `out`
 * (4 + n_perms doubles), all DEVICE pointers, as for unifrac_mantel_pearson.
 * Limits: n_samples <= UNIFRAC_NOALLOC_MAX_SAMPLES and n_perms <= UNIFRAC_NOALLOC_MAX_PERMS, else UNIFRAC_ERR_UNSUPPORTED
 * (unifrac_last_cuda_error() then names the limit that was exceeded); other argument errors as unifrac_mantel_pearson.
 * The array is SHARED by every call on the device and keeps the last call's contents (the call clears what must start at
 * zero): two calls that overlap on the GPU -- different streams, or different host threads -- race on it; serialise them.
 * Asynchronous on `stream`, which must belong to the current device.  The first call of a process also loads the kernels
 * (driver-internal); make one warm-up call before a region that must not allocate at all.
 */
#define UNIFRAC_NOALLOC_MAX_SAMPLES 1024
#define UNIFRAC_NOALLOC_MAX_PERMS 999
#define UNIFRAC_NOALLOC_SCRATCH_BYTES (8u * 1024u * 1024u + 64u * 1024u)   /* 1024 x 1024 fp64 square copy + 64 KB */
int unifrac_mantel_pearson_noalloc(int32_t n_samples, const void *x_condensed, const void *y_condensed,
                                   unifrac_precision_t precision, const int32_t *perms, int32_t n_perms, double *out,
                                   void *stream);

/*
 * unifrac_mantel_spearman -- the same test with Spearman's rank correlation ("either Pearson's product-moment
 * correlation coefficient or Spearman's rank correlation coefficient").  rho = Pearson's r of the RANKS of the
 * two condensed vectors, tied values sharing the mean of the ranks they span (1-based fractional ranking, DESIGN.md readings
 * M5-M6); a permutation of the objects only moves entries around, so every rho_k is Pearson's r between the permuted rank
 * matrix of X and the ranks of y.  Arguments, output layout, p-values and error behaviour are those of unifrac_mantel_pearson.
 * The ranks come from a stable LSD radix sort of (value, position) pairs on the device (no library sort); they are held as
 * exact 32-bit integers (twice the average rank).  Workspace: ~2 x (key + position) x n(n-1)/2 for the sort, 2 x 4 x n(n-1)/2
 * for the ranks, 4 n^2 for the square copy.  n(n-1)/2 >= 2^31 - 1 (n > 65,535): UNIFRAC_ERR_UNSUPPORTED.  NaNs are not supported.  Asynchronous on `stream`.
 */
int unifrac_mantel_spearman(int32_t n_samples, const void *x_condensed, const void *y_condensed,
                            unifrac_precision_t precision, const int32_t *perms, int32_t n_perms, double *out,
                            unifrac_alloc_fn alloc, void *alloc_user, void *stream);

/*
 * unifrac_pcoa -- principal coordinates analysis of a distance matrix that is already resident in HBM ("researchers
 * often apply principal coordinates analysis (PCoA)"; "PCoA can also be computed as part of the Hybrid UniFrac
 * compute itself").  Classical scaling (readings P1-P5): A = -1/2 D o D, B = Gower-centred A,
 * leading eigenpairs (lambda_i, v_i) of B in descending order, coordinates of axis i = v_i sqrt(lambda_i), proportion
 * explained = lambda_i / trace(B).
 *   d_condensed  DEVICE; n(n-1)/2 float or double (the layout unifrac_dm writes), read-only
 *   k            number of axes, 1 <= k <= 16, k < n
 *   max_iter     cap on the products B Q of the block subspace iteration (block of 32 vectors); tol: stop when every one of
 *                the k leading Ritz values moved by <= tol * |value| over the last 4 products (e.g. 200, 1e-9)
 *   out          DEVICE; 2 k + n k doubles: [k eigenvalues | k proportions explained | n x k coordinates, row-major].
 *                An eigenvector's sign is arbitrary; axes with a non-positive eigenvalue get zero coordinates.
 *   iterations   HOST, optional: products used.
 * The only O(n^2) work is Y = B Q: a hand-written tcgen05 kind::tf32 GEMM with a 3-term hi/lo split (fp32 accumulation in
 * TMEM); orthonormalisation and the 32 x 32 Rayleigh-Ritz step are fp64.  Workspace: 8 n^2 bytes (B as two fp32 matrices).
 * Eigenvalues of well-separated axes agree with a full fp64 eigendecomposition to ~1e-6 relative.  The call synchronises the
 * stream (it reads the Ritz values back to test convergence).  n < 3, k out of range: UNIFRAC_ERR_INVALID_ARG.
 */
int unifrac_pcoa(int32_t n_samples, const void *d_condensed, unifrac_precision_t precision, int32_t k, int32_t max_iter,
                 double tol, double *out, int32_t *iterations, unifrac_alloc_fn alloc, void *alloc_user, void *stream);

/* Device-rate probes (not on the data path): what this GPU retires per second of the two atomic units of work the
 * sparse kernels are made of; they are the constants of the head / mid / tail cost model and the `peak` of the
 * k_mid / k_tail_scatter rooflines in bench.py.  Runs ~20 ms of probe kernels on `stream` and synchronises it. */
typedef struct {
    double smem_atomic_conflict_free_per_s;  /* shared-memory u32 atomic adds, 32 lanes on 32 different banks        */
    double smem_atomic_random_per_s;         /* ... on pseudo-random cells of a 128 x 128 tile (k_mid's access pattern) */
    double l2_red_random_per_s;              /* fp32 RED.ADD on pseudo-random words of a 48 MB (L2-resident) footprint */
    double fmnmx_per_s;                      /* FP32 min lane-ops (the half-rate ALU pipe), register chains            */
    double fadd_per_s;                       /* FP32 add lane-ops (the FMA pipe)                                      */
    double fmnmx_fadd_per_s;                 /* lane-ops of interleaved min + add pairs (one k_dense update = 2)       */
    double fadd2_per_s;                      /* FP32 add lane-ops issued as packed add.f32x2 (FADD2, two per instruction) */
    double fmnmx2_fadd2_updates_per_s;       /* (pair, branch) updates of 2 x FMNMX + 1 x FADD2 (1.5 instructions per update) */
    double dense16_mix_updates_per_s;        /* updates of k_dense16's instruction mix (24 min cells with packed adds + 8 direct
                                                cells with FADD + FFMA per 32)                                              */
    int32_t sm_count;
    int32_t sm_clock_khz;                    /* cudaDevAttrClockRate                                               */
} unifrac_rates_t;
int unifrac_measure_rates(unifrac_rates_t *out, void *stream);

const char *unifrac_status_string(int status);
const char *unifrac_last_cuda_error(void);   /* text of the last CUDA error seen by this thread  */
int unifrac_abi_version(void);               /* 8                                                */

#ifdef __cplusplus
}
#endif
#endif /* UNIFRAC_B200_H */
