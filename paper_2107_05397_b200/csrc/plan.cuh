// plan.cuh -- step a-0 of the hot path (SURVEY 8a / DESIGN.md "K0 plan"): validate the tree and the
// table, per-sample totals T_s, node depths (pointer jumping), per-depth lists of internal nodes,
// children CSR.  Integer work, O(n_nodes + nnz).  BASELINE.json:5 "propagates ... up the postorder
// tree level by level" needs exactly these level lists.
#pragma once
#include "common.cuh"

namespace ufb {

// parent range / single root / branch lengths / child counts
__global__ void k_tree_check(int n, const int32_t* __restrict__ parent, const double* __restrict__ len,
                             int32_t* __restrict__ child_count, PlanWords* pw, int validate)
{
    int v = blockIdx.x * blockDim.x + threadIdx.x;
    if (v >= n) return;
    int p = parent[v];
    if (p == -1) {
        atomicAdd(&pw->n_roots, 1);
        pw->root = v;
    } else if (p < 0 || p >= n || p == v) {
        atomicOr(&pw->err, ERRBIT_TREE);
    } else {
        atomicAdd(&child_count[p], 1);
        if (validate) {
            double l = len[v];
            if (!(l >= 0.0) || isinf(l)) atomicOr(&pw->err, ERRBIT_TREE);
        }
    }
}

__global__ void k_root_check(PlanWords* pw)
{
    if (pw->n_roots != 1) atomicOr(&pw->err, ERRBIT_TREE);
}

// postorder is a permutation (each node seen exactly once); remember positions
__global__ void k_post_check1(int n, const int32_t* __restrict__ postorder, int32_t* __restrict__ seen,
                              int32_t* __restrict__ pos, PlanWords* pw)
{
    int k = blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= n) return;
    int v = postorder[k];
    if (v < 0 || v >= n) { atomicOr(&pw->err, ERRBIT_TREE); return; }
    if (atomicAdd(&seen[v], 1) != 0) atomicOr(&pw->err, ERRBIT_TREE);
    pos[v] = k;
}

// children before parent, root last  (=> the parent array is acyclic)
__global__ void k_post_check2(int n, const int32_t* __restrict__ parent, const int32_t* __restrict__ postorder,
                              const int32_t* __restrict__ pos, PlanWords* pw)
{
    if (pw->err) return;   // parent[] / postorder[] may be out of range
    int v = blockIdx.x * blockDim.x + threadIdx.x;
    if (v >= n) return;
    int p = parent[v];
    if (p >= 0) { if (pos[v] >= pos[p]) atomicOr(&pw->err, ERRBIT_TREE); }
    else if (postorder[n - 1] != v) atomicOr(&pw->err, ERRBIT_TREE);
}

// per-sample totals + CSR validation; one warp per sample
__global__ void k_csr_check(int n, int n_samples, const int64_t* __restrict__ indptr,
                            const int32_t* __restrict__ indices, const int32_t* __restrict__ counts,
                            const int32_t* __restrict__ child_count, unsigned long long* __restrict__ T,
                            PlanWords* pw, int validate)
{
    if (pw->err & ERRBIT_TREE) return;
    int s = (blockIdx.x * blockDim.x + threadIdx.x) >> 5;
    int lane = threadIdx.x & 31;
    if (s >= n_samples) return;
    long long lo = indptr[s], hi = indptr[s + 1];
    if (validate) {
        if ((s == 0 && lo != 0) || hi < lo || lo < 0) { if (lane == 0) atomicOr(&pw->err, ERRBIT_TABLE); return; }
    }
    unsigned long long sum = 0;
    bool bad = false;
    for (long long k = lo + lane; k < hi; k += 32) {
        int t = indices[k];
        int c = counts[k];
        if (validate) {
            if (t < 0 || t >= n || c < 0) { bad = true; continue; }
            if (child_count[t] != 0) bad = true;                  // column must be a tip
            if (k > lo && indices[k - 1] >= t) bad = true;        // strictly increasing
        }
        sum += (unsigned long long)(c > 0 ? c : 0);
    }
    for (int o = 16; o; o >>= 1) sum += __shfl_xor_sync(0xffffffffu, sum, o);
    bad = __any_sync(0xffffffffu, bad);
    if (lane == 0) {
        T[s] = sum;
        if (bad) atomicOr(&pw->err, ERRBIT_TABLE);
        else if (sum == 0) atomicOr(&pw->err, ERRBIT_EMPTY);
        else if (sum >= (1ull << 32)) atomicOr(&pw->err, ERRBIT_UNSUPPORTED);
    }
}

// depth by pointer jumping: after ceil(log2 n) rounds anc = root, dist = depth
__global__ void k_jump_init(int n, const int32_t* __restrict__ parent, int32_t* anc, int32_t* dist)
{
    int v = blockIdx.x * blockDim.x + threadIdx.x;
    if (v >= n) return;
    int p = parent[v];
    anc[v] = p < 0 ? v : p;
    dist[v] = p < 0 ? 0 : 1;
}
__global__ void k_jump_round(int n, const int32_t* __restrict__ anc_in, const int32_t* __restrict__ dist_in,
                             int32_t* __restrict__ anc_out, int32_t* __restrict__ dist_out)
{
    int v = blockIdx.x * blockDim.x + threadIdx.x;
    if (v >= n) return;
    int a = anc_in[v];
    dist_out[v] = dist_in[v] + dist_in[a];
    anc_out[v] = anc_in[a];
}

// histogram of depths over internal non-root... (root included: it is skipped at propagation time)
__global__ void k_level_hist(int n, const int32_t* __restrict__ depth, const int32_t* __restrict__ child_count,
                             uint32_t* __restrict__ hist, PlanWords* pw)
{
    int v = blockIdx.x * blockDim.x + threadIdx.x;
    if (v >= n) return;
    atomicMax(&pw->max_depth, depth[v]);
    if (child_count[v] > 0) { atomicAdd(&hist[depth[v]], 1u); atomicAdd(&pw->n_internal, 1ull); }
}
__global__ void k_level_fill(int n, const int32_t* __restrict__ depth, const int32_t* __restrict__ child_count,
                             uint32_t* __restrict__ cursor, int32_t* __restrict__ level_nodes)
{
    int v = blockIdx.x * blockDim.x + threadIdx.x;
    if (v >= n) return;
    if (child_count[v] > 0) level_nodes[atomicAdd(&cursor[depth[v]], 1u)] = v;
}
__global__ void k_child_fill(int n, const int32_t* __restrict__ parent, uint32_t* __restrict__ cursor,
                             int32_t* __restrict__ child_idx)
{
    int v = blockIdx.x * blockDim.x + threadIdx.x;
    if (v >= n) return;
    int p = parent[v];
    if (p >= 0) child_idx[atomicAdd(&cursor[p], 1u)] = v;
}

// single-block exclusive scan (n up to a few million; plan step only).  out[n] = total.
template <typename TI>
__global__ void k_exclusive_scan(int n, const TI* __restrict__ in, uint32_t* __restrict__ out)
{
    __shared__ uint32_t part[1024];
    int t = threadIdx.x;
    long long chunk = ((long long)n + blockDim.x - 1) / blockDim.x;
    long long lo = t * chunk, hi = lo + chunk;
    if (hi > n) hi = n;
    uint32_t s = 0;
    for (long long k = lo; k < hi; ++k) s += (uint32_t)in[k];
    part[t] = s;
    __syncthreads();
    // Hillis-Steele inclusive scan over the 1024 partials
    for (int o = 1; o < (int)blockDim.x; o <<= 1) {
        uint32_t add = t >= o ? part[t - o] : 0;
        __syncthreads();
        part[t] += add;
        __syncthreads();
    }
    uint32_t run = t ? part[t - 1] : 0;
    for (long long k = lo; k < hi; ++k) { uint32_t x = (uint32_t)in[k]; out[k] = run; run += x; }
    if (t == (int)blockDim.x - 1) out[n] = part[t];
}

}  // namespace ufb
