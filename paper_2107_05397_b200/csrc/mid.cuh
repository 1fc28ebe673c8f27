// mid.cuh -- step a-5 for the MID branches (fp32 mode): too sparse for the dense head kernels, too
// dense for the global RED.ADD scatter.  PAPER.md:23 "sparse-aware optimizations" (mechanism ours,
// DESIGN.md "head / mid / tail split").
//
// A mid branch v is a sorted list of (sample, u~) entries (same arrays as the tail lists).  For the
// 128 x 128 tile pair (I, J) only the n_I x n_J pairs of samples present on BOTH sides contribute
// min(u~_a, u~_b) to M_ab (identities I3 / I5).  One CTA owns the tile pair's 128 x 128 accumulators in
// shared memory as 32-bit FIXED-POINT integers and adds the contributions with native shared-memory
// integer atomics (ATOMS.ADD; measured 8.4 /clk/SM = 2.4e12 /s against 2.6 /clk/SM for the fp32 CAS loop
// and 1.9e11 /s for global RED.ADD, profiles/r01_ubench_atomics.txt).  Integer addition commutes, so the
// result does not depend on the order in which warps reach a cell.
//   u_q = round(u~ * 2^F),  F = 30 - ceil(log2(max_s R_s))   =>   acc <= min(R_a, R_b) * 2^F < 2^31
//   epilogue: out[idx(a,b)] += acc * 2^-F      (exclusive owner of the tile pair; tail REDs ran before)
// Row bookkeeping: seg[t][r] = offset (within row r's list) of the first entry with sample >= 128 t,
// stored tile-major so that the 32 lanes of a warp (32 consecutive mid rows) read coalesced words.
#pragma once
#include "common.cuh"
#include "tail.cuh"

namespace ufb {

constexpr int MID_THREADS = 512;
constexpr int MID_PITCH = TILE + 1;                 // accumulator row pitch: bank = (a + b) mod 32 for both lane orders
constexpr size_t MID_SMEM = (size_t)TILE * MID_PITCH * sizeof(uint32_t);
constexpr int MID_SMALL = 4;

// mid rows ordered by n_v (counting sort: histogram, scan, scatter) so that the rows a warp handles together
// have similar list lengths; mbase[r] = list offset of row r.  The order inside a bucket is arbitrary --
// harmless, integer accumulation commutes.
__global__ void k_mid_hist(int n, const uint8_t* __restrict__ cls, const uint32_t* __restrict__ nv, uint32_t* __restrict__ hist)
{
    int v = blockIdx.x * blockDim.x + threadIdx.x;
    if (v < n && cls[v] == CLS_MID) atomicAdd(&hist[nv[v]], 1u);
}
__global__ void k_mid_rows(int n, const uint8_t* __restrict__ cls, const uint32_t* __restrict__ nv, uint32_t* __restrict__ cursor,
                           const uint32_t* __restrict__ tptr, int32_t* __restrict__ mrows, uint32_t* __restrict__ mbase)
{
    int v = blockIdx.x * blockDim.x + threadIdx.x;
    if (v < n && cls[v] == CLS_MID) {
        uint32_t r = atomicAdd(&cursor[nv[v]], 1u);
        mrows[r] = v;
        mbase[r] = tptr[v];
    }
}

// seg[t][r] for t = 0..n_tiles (thread per (t, r), r fastest)
__global__ void k_mid_seg(uint32_t n_mid, const int32_t* __restrict__ mrows, const uint32_t* __restrict__ tptr,
                          const uint32_t* __restrict__ ts, int n_tiles, uint32_t* __restrict__ seg)
{
    long long gid = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    uint32_t t = (uint32_t)(gid / n_mid), r = (uint32_t)(gid - (long long)t * n_mid);
    if (t > (uint32_t)n_tiles) return;
    const int v = mrows[r];
    const uint32_t lo0 = tptr[v], hi0 = tptr[v + 1];
    uint32_t lo = lo0, hi = hi0;
    const uint32_t key = t * (uint32_t)TILE;
    while (lo < hi) {
        uint32_t mid = lo + ((hi - lo) >> 1);
        if (ts[mid] < key) lo = mid + 1; else hi = mid;
    }
    seg[(size_t)t * n_mid + r] = lo - lo0;
}

struct MidParams {
    const int2* pairs; uint32_t n_pairs;
    unsigned int* counter;        // dynamic tile-pair queue
    uint32_t n_mid;
    const uint32_t* mbase;        // [n_mid] list offset of the row
    const uint32_t* seg;          // [n_tiles+1][n_mid]
    const uint32_t* ts;
    const float* tv;
    int n_samples;
    float* out;
    float qscale;                 // 2^F
    double inv_qscale;            // 2^-F
};

__device__ __forceinline__ uint32_t mid_q(float v, float qscale) { return __float2uint_rn(v * qscale); }

__global__ void __launch_bounds__(MID_THREADS)
k_mid(const MidParams P)
{
    extern __shared__ uint32_t macc[];              // [128][129]
    __shared__ int s_pair;
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const long long N = P.n_samples;
    const uint32_t n_chunks = (P.n_mid + 31) >> 5;

    for (;;) {
        if (threadIdx.x == 0) s_pair = (int)atomicAdd(P.counter, 1u);
        for (int i = threadIdx.x; i < TILE * MID_PITCH; i += MID_THREADS) macc[i] = 0u;
        __syncthreads();
        const int pi = s_pair;
        if ((uint32_t)pi >= P.n_pairs) break;
        const int2 ij = P.pairs[pi];
        const bool diag = ij.x == ij.y;
        const uint32_t* segI0 = P.seg + (size_t)ij.x * P.n_mid;
        const uint32_t* segI1 = segI0 + P.n_mid;
        const uint32_t* segJ0 = P.seg + (size_t)ij.y * P.n_mid;
        const uint32_t* segJ1 = segJ0 + P.n_mid;
        const uint32_t sI = (uint32_t)ij.x * TILE, sJ = (uint32_t)ij.y * TILE;

        const int grp = lane >> 3, gl = lane & 7, gbase = lane & ~7;
        for (uint32_t ch = warp; ch < n_chunks; ch += MID_THREADS / 32) {
            const uint32_t r = ch * 32 + lane;
            uint32_t i0 = 0, i1 = 0, j0 = 0, j1 = 0, base = 0;
            if (r < P.n_mid) {
                i0 = segI0[r]; i1 = segI1[r];
                if (diag) { j0 = i0; j1 = i1; } else { j0 = segJ0[r]; j1 = segJ1[r]; }
                base = P.mbase[r];
            }
            const uint32_t nI = i1 - i0, nJ = j1 - j0;
            const uint32_t work = diag ? (nI * (nI - (nI ? 1u : 0u))) / 2u : nI * nJ;
            // ---- tiny cross products: one row per lane
            if (work && work <= (uint32_t)MID_SMALL) {
                for (uint32_t k = i0; k < i1; ++k) {
                    const uint32_t a = P.ts[base + k] - sI;
                    const uint32_t qa = mid_q(P.tv[base + k], P.qscale);
                    for (uint32_t l = diag ? k + 1 : j0; l < j1; ++l) {
                        const uint32_t b = P.ts[base + l] - sJ;
                        const uint32_t qb = mid_q(P.tv[base + l], P.qscale);
                        atomicAdd(&macc[a * MID_PITCH + b], qa < qb ? qa : qb);
                    }
                }
            }
            // ---- the rest: four rows at a time, one per 8-lane group (four rows' loads in flight per warp);
            //      lanes of a group over the longer list, loop over the shorter one
            uint32_t rem = __ballot_sync(0xffffffffu, work > (uint32_t)MID_SMALL);
            while (rem) {
                uint32_t m = rem;
                for (int t = 0; t < grp; ++t) m &= m - 1;
                const bool act = m != 0;
                const int src = act ? __ffs(m) - 1 : 0;
#pragma unroll
                for (int t = 0; t < 4; ++t) rem &= rem - 1;
                uint32_t bi0 = __shfl_sync(0xffffffffu, i0, src), bi1 = __shfl_sync(0xffffffffu, i1, src);
                uint32_t bj0 = __shfl_sync(0xffffffffu, j0, src), bj1 = __shfl_sync(0xffffffffu, j1, src);
                const uint32_t bb = __shfl_sync(0xffffffffu, base, src);
                if (!act) { bi0 = bi1 = bj0 = bj1 = 0; }
                const bool lanesJ = diag || (bj1 - bj0) >= (bi1 - bi0);
                const uint32_t p0 = lanesJ ? bj0 : bi0, p1 = lanesJ ? bj1 : bi1;   // lane list
                const uint32_t q0 = lanesJ ? bi0 : bj0, q1 = lanesJ ? bi1 : bj1;   // loop list
                const uint32_t sP = lanesJ ? sJ : sI, sQ = lanesJ ? sI : sJ;
                const uint32_t mulP = lanesJ ? 1u : (uint32_t)MID_PITCH, mulQ = lanesJ ? (uint32_t)MID_PITCH : 1u;
                for (uint32_t l0 = p0; __any_sync(0xffffffffu, l0 < p1); l0 += 8) {
                    const uint32_t l = l0 + gl;
                    const bool lv = l < p1;
                    const uint32_t offe = lv ? (P.ts[bb + l] - sP) * mulP : 0u;
                    const uint32_t qe = lv ? mid_q(P.tv[bb + l], P.qscale) : 0u;
                    const uint32_t kend = diag ? (l0 + 8 < q1 ? l0 + 8 : q1) : q1;     // diag: only k < l
                    for (uint32_t kb = q0; __any_sync(0xffffffffu, kb < kend); kb += 8) {
                        const uint32_t kk = kb + gl;
                        uint32_t offf = 0, qf = 0;
                        if (kk < kend) { offf = (P.ts[bb + kk] - sQ) * mulQ; qf = mid_q(P.tv[bb + kk], P.qscale); }
#pragma unroll
                        for (int t = 0; t < 8; ++t) {
                            const uint32_t of = __shfl_sync(0xffffffffu, offf, gbase + t);
                            const uint32_t qv = __shfl_sync(0xffffffffu, qf, gbase + t);
                            if (lv && kb + t < kend && (!diag || kb + t < l)) atomicAdd(&macc[offe + of], qe < qv ? qe : qv);
                        }
                    }
                }
            }
        }
        __syncthreads();
        // ---- epilogue: add the tile pair's fixed-point sums to the condensed matrix (exclusive owner)
        for (int e = threadIdx.x; e < TILE * TILE; e += MID_THREADS) {
            const int a = e >> 7, b = e & 127;
            const uint32_t q = macc[a * MID_PITCH + b];
            if (q) {
                const long long gi = (long long)sI + a, gj = (long long)sJ + b;
                if (gi < gj && gj < N) {
                    float* o = P.out + (gi * (2 * N - gi - 1) / 2 - gi - 1 + gj);
                    *o = (float)((double)*o + (double)q * P.inv_qscale);
                }
            }
        }
        __syncthreads();
    }
}

}  // namespace ufb
