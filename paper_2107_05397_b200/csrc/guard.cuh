// guard.cuh -- near-duplicate guard of the separable forms ("pairs with small d recomputed by the
// direct form"; PAPER.md:11 -- new sample collections placed into the context of existing data is where replicate /
// proportional samples occur).
//
// The a-5 kernels accumulate M_ab = sum_v min(u~_av, u~_bv) and the finalize step forms num = S_a + S_b - 2 M, whose
// relative error grows like (1 - d) / d.  Every pair whose distance comes out below GUARD_THETA is appended to a
// device list by the finalize epilogues (common.cuh: guard_note); this kernel recomputes exactly those pairs from
// the definition (BASELINE.json:5: "len*|u-v| and len*(u+v)" / "len*(x xor y) and len*(x or y)"), all terms
// non-negative, in fp64 from the exact integer counts -- so duplicated and proportional samples give exactly 0.
// No host round trip: the grid is fixed, each CTA takes listed pairs p = blockIdx.x, blockIdx.x + gridDim.x, ...
//
// Per pair (a, b), one CTA, three walks over the two samples' table rows (every observed tip up to the root):
//   1. cntA[v] += c, cntB[v] += c on every branch above the tip           (integer atomics in the CTA's own scratch)
//   2. the first thread to reach a branch claims it (seen[v]) and adds its term; a walk stops at a claimed branch,
//      whose claimer continues upward, so every touched branch is counted exactly once
//   3. the touched cells are reset to zero the same way (the scratch is zero between pairs and between calls)
#pragma once
#include "common.cuh"

namespace ufb {

constexpr int GUARD_THREADS = 512;

struct GuardParams {
    int n;                                  // tree nodes
    const int32_t* parent;
    const double* len;
    const int64_t* indptr;
    const int32_t* indices;
    const int32_t* counts;
    const unsigned long long* Tsum;         // [n_samples] total count of every sample (table row order)
    const int32_t* order;                   // position -> table row of the sample (NULL: identity)
    long long N;
    int weighted;
    GuardList list;
    unsigned int* done;                     // listed pairs already recomputed by an earlier launch of this call
    uint32_t* scratch;                      // [grid][3][n] zeroed: cntA, cntB, seen
    void* out;                              // condensed, T (in position space)
};

template <typename T>
__global__ void __launch_bounds__(GUARD_THREADS)
k_guard(const GuardParams P)
{
    __shared__ double red[2][GUARD_THREADS / 32];
    uint32_t* cntA = P.scratch + (size_t)blockIdx.x * 3 * P.n;
    uint32_t* cntB = cntA + P.n;
    uint32_t* seen = cntB + P.n;
    const uint32_t total = min(*P.list.count, P.list.cap);
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    for (uint32_t p = *P.done + blockIdx.x; p < total; p += gridDim.x) {
        const uint2 ab = P.list.pairs[p];
        const int sa = P.order ? P.order[ab.x] : (int)ab.x, sb = P.order ? P.order[ab.y] : (int)ab.y;
        // ---- 1. integer counts of both samples on every branch above their observed tips
        for (int side = 0; side < 2; ++side) {
            const int s = side ? sb : sa;
            uint32_t* cnt = side ? cntB : cntA;
            const long long lo = P.indptr[s], hi = P.indptr[s + 1];
            for (long long k = lo + threadIdx.x; k < hi; k += GUARD_THREADS) {
                const int c = P.counts[k];
                if (c <= 0) continue;
                for (int v = P.indices[k]; P.parent[v] >= 0; v = P.parent[v]) atomicAdd(&cnt[v], (uint32_t)c);
            }
        }
        __syncthreads();
        // ---- 2. the definition, each touched branch once
        const double Ta = (double)P.Tsum[sa], Tb = (double)P.Tsum[sb];
        double num = 0.0, den = 0.0;
        for (int side = 0; side < 2; ++side) {
            const int s = side ? sb : sa;
            const long long lo = P.indptr[s], hi = P.indptr[s + 1];
            for (long long k = lo + threadIdx.x; k < hi; k += GUARD_THREADS) {
                if (P.counts[k] <= 0) continue;
                for (int v = P.indices[k]; P.parent[v] >= 0 && atomicExch(&seen[v], 1u) == 0u; v = P.parent[v]) {
                    const double l = P.len[v];
                    const uint32_t ca = __ldcg(&cntA[v]), cb = __ldcg(&cntB[v]);     // written by L2 atomics: bypass L1
                    if (P.weighted) {
                        const double ua = (double)ca / Ta, ub = (double)cb / Tb;
                        num += l * fabs(ua - ub);
                        den += l * (ua + ub);
                    } else {
                        if ((ca > 0u) != (cb > 0u)) num += l;
                        den += l;
                    }
                }
            }
        }
        for (int o = 16; o; o >>= 1) { num += __shfl_xor_sync(0xffffffffu, num, o); den += __shfl_xor_sync(0xffffffffu, den, o); }
        if (lane == 0) { red[0][warp] = num; red[1][warp] = den; }
        __syncthreads();
        if (threadIdx.x == 0) {
            double n2 = 0.0, d2 = 0.0;
            for (int w = 0; w < GUARD_THREADS / 32; ++w) { n2 += red[0][w]; d2 += red[1][w]; }
            const long long gi = ab.x, gj = ab.y;
            reinterpret_cast<T*>(P.out)[gi * (2 * P.N - gi - 1) / 2 - gi - 1 + gj] = (T)(d2 > 0.0 ? n2 / d2 : 0.0);
        }
        // ---- 3. reset the touched cells
        for (int side = 0; side < 2; ++side) {
            const int s = side ? sb : sa;
            const long long lo = P.indptr[s], hi = P.indptr[s + 1];
            for (long long k = lo + threadIdx.x; k < hi; k += GUARD_THREADS) {
                if (P.counts[k] <= 0) continue;
                for (int v = P.indices[k]; P.parent[v] >= 0 && atomicExch(&seen[v], 0u) == 1u; v = P.parent[v]) {
                    cntA[v] = 0u; cntB[v] = 0u;
                }
            }
        }
        __syncthreads();
    }
}

// after a k_guard launch: everything listed so far has been recomputed
__global__ void k_guard_mark(GuardList list, unsigned int* done) { *done = min(*list.count, list.cap); }

}  // namespace ufb
