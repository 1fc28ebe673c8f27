// perm.cuh -- richness ordering of the samples inside one unifrac_dm call (SURVEY 8a-5d(5) "sample re-ordering"
// "sparse-aware optimizations", mechanism ours -- DESIGN.md "richness order").  Presence of a branch is far from uniform over
// the samples: a sample with many features is present on many more branches than a poor one.  With the samples sorted by their
// number of table entries (ascending), every branch is sparse in the leading 128-sample tiles and dense in the trailing ones,
// and step a-5 can decide per (branch, tile) which kernel handles it (zone.cuh).  The call then runs on the permuted table in
// "position space" and the finished condensed matrix is un-permuted once at the end.
#pragma once
#include "common.cuh"

namespace ufb {

// key[s] = entries of sample s: an ascending stable sort gives ascending richness, ties in sample order.
// bad != 0: indptr is not a plausible CSR pointer array (the caller then skips the permutation and lets validation report it)
__global__ void k_perm_keys(int N, const int64_t* __restrict__ indptr, uint32_t* __restrict__ key, unsigned int* __restrict__ bad)
{
    const int s = blockIdx.x * blockDim.x + threadIdx.x;
    if (s >= N) return;
    const long long lo = indptr[s], hi = indptr[s + 1];
    if ((s == 0 && lo != 0) || hi < lo || hi - lo >= (1ll << 31)) { atomicOr(bad, 1u); key[s] = 0u; return; }
    key[s] = (uint32_t)(hi - lo);
}

// rowlen[pos] = entries of the sample at position pos; inv[sample] = position
__global__ void k_perm_rowlen(int N, const int64_t* __restrict__ indptr, const uint32_t* __restrict__ perm,
                              uint32_t* __restrict__ rowlen, uint32_t* __restrict__ inv)
{
    const int pos = blockIdx.x * blockDim.x + threadIdx.x;
    if (pos >= N) return;
    const uint32_t s = perm[pos];
    rowlen[pos] = (uint32_t)(indptr[s + 1] - indptr[s]);
    inv[s] = (uint32_t)pos;
}

// permuted CSR: one warp per position copies the sample's row; new_indptr from the exclusive scan of rowlen
__global__ void __launch_bounds__(256)
k_perm_gather(int N, const int64_t* __restrict__ indptr, const int32_t* __restrict__ indices, const int32_t* __restrict__ counts,
              const uint32_t* __restrict__ perm, const uint32_t* __restrict__ off, int64_t* __restrict__ new_indptr,
              int32_t* __restrict__ new_indices, int32_t* __restrict__ new_counts)
{
    const int pos = (int)(((long long)blockIdx.x * blockDim.x + threadIdx.x) >> 5), lane = threadIdx.x & 31;
    if (pos >= N) return;
    const uint32_t s = perm[pos];
    const long long lo = indptr[s], m = indptr[s + 1] - lo;
    const long long dst = off[pos];
    for (long long k = lane; k < m; k += 32) { new_indices[dst + k] = indices[lo + k]; new_counts[dst + k] = counts[lo + k]; }
    if (lane == 0) { new_indptr[pos] = dst; if (pos == N - 1) new_indptr[N] = dst + m; }
}

// out[idx(i, j)] = tmp[idx(pos_i, pos_j)] for every i < j (coalesced writes, gathered reads)
template <typename T>
__global__ void __launch_bounds__(256)
k_unpermute(long long N, const uint32_t* __restrict__ inv, const T* __restrict__ tmp, T* __restrict__ out)
{
    for (long long i = blockIdx.y; i < N - 1; i += gridDim.y) {
        const long long j = i + 1 + (long long)blockIdx.x * blockDim.x + threadIdx.x;
        if (j >= N) continue;
        const long long a = inv[i], b = inv[j];
        const long long lo = a < b ? a : b, hi = a < b ? b : a;
        out[i * (2 * N - i - 1) / 2 - i - 1 + j] = tmp[lo * (2 * N - lo - 1) / 2 - lo - 1 + hi];
    }
}

}  // namespace ufb
