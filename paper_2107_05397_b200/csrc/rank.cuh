// rank.cuh -- average-rank transform of a condensed distance vector, for the Spearman variant of the Mantel test
// ("... or Spearman's rank correlation coefficient"; "the Spearman variety requires about 18
// minutes", readings M5-M6).  Spearman's rho is Pearson's r of the RANKS, ties sharing the mean of the
// ranks they span, so the device path is: a stable LSD radix sort of (key, position) pairs -- hand-written, 8-bit digits,
// no cub / thrust --, a prefix-max scan that gives every sorted position the start of its run of equal keys, and a scatter
// of  2 x rank = 2 start + (run length - 1) + 2  (1-based average ranks are half-integers, so twice the rank is an exact uint32)
// back to the original positions.  k_mantel_perm (mantel.cuh) then runs unchanged on the two integer vectors (fp64 sums).
// Bound: HBM.  One pass moves 4 + 8 + 8 bytes per element (histogram read, scatter read + write of key and position).
#pragma once
#include "common.cuh"

namespace ufb {

constexpr int RADIX_THREADS = 256;
constexpr int RADIX_ITEMS = 16;                         // per thread and tile: warp w owns 512 consecutive elements
constexpr int RADIX_TILE = RADIX_THREADS * RADIX_ITEMS; // 4096
constexpr int RADIX_WARPS = RADIX_THREADS / 32;

template <typename T> struct RankKey;
template <> struct RankKey<float> {
    using K = uint32_t;
    static constexpr int PASSES = 4;
    // order-preserving map of IEEE floats to unsigned integers; -0 is folded onto +0 so that equal VALUES are equal KEYS
    __device__ static __forceinline__ K make(float v) {
        const uint32_t u = __float_as_uint(v + 0.0f);
        return u ^ ((u >> 31) ? 0xffffffffu : 0x80000000u);
    }
};
template <> struct RankKey<double> {
    using K = unsigned long long;
    static constexpr int PASSES = 8;
    __device__ static __forceinline__ K make(double v) {
        const unsigned long long u = (unsigned long long)__double_as_longlong(v + 0.0);
        return u ^ ((u >> 63) ? 0xffffffffffffffffull : 0x8000000000000000ull);
    }
};

// plain unsigned keys (sample / row orderings inside unifrac_dm: perm.cuh, zone.cuh)
template <> struct RankKey<uint32_t> {
    using K = uint32_t;
    static constexpr int PASSES = 4;
    __device__ static __forceinline__ K make(uint32_t v) { return v; }
};
template <> struct RankKey<unsigned long long> {
    using K = unsigned long long;
    static constexpr int PASSES = 8;
    __device__ static __forceinline__ K make(unsigned long long v) { return v; }
};

// block b owns the contiguous element range [b * per_block, min(P, (b + 1) * per_block)), per_block a multiple of RADIX_TILE
__device__ __forceinline__ void radix_range(unsigned long long P, unsigned long long per_block, unsigned long long& lo, unsigned long long& hi) {
    lo = (unsigned long long)blockIdx.x * per_block;
    hi = lo + per_block;
    if (lo > P) lo = P;
    if (hi > P) hi = P;
}

// hist[d * gridDim.x + b] = number of elements of block b's range whose digit (key >> shift) & 255 is d
template <typename T, bool FIRST>
__global__ void __launch_bounds__(RADIX_THREADS)
k_radix_hist(const T* __restrict__ raw, const typename RankKey<T>::K* __restrict__ keys, unsigned long long P,
             unsigned long long per_block, int shift, uint32_t* __restrict__ hist)
{
    using K = typename RankKey<T>::K;
    __shared__ uint32_t wh[RADIX_WARPS][256];                          // per-warp counts
    for (int w = 0; w < RADIX_WARPS; ++w) wh[w][threadIdx.x] = 0;
    __syncthreads();
    unsigned long long lo, hi;
    radix_range(P, per_block, lo, hi);
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    for (unsigned long long tile = lo; tile < hi; tile += RADIX_TILE) {
        // the same element -> (warp, round, lane) map as the scatter kernel; RADIX_ITEMS independent loads in flight per thread
        const unsigned long long wbase = tile + (unsigned long long)warp * (32 * RADIX_ITEMS) + lane;
        K k[RADIX_ITEMS];
        if (FIRST) {                                                   // all loads first, then the key map (a load inside the
            T v[RADIX_ITEMS];                                          // conditional conversion is not hoisted by the compiler)
#pragma unroll
            for (int r = 0; r < RADIX_ITEMS; ++r) { const unsigned long long e = wbase + (unsigned long long)r * 32; v[r] = e < hi ? raw[e] : T(0); }
#pragma unroll
            for (int r = 0; r < RADIX_ITEMS; ++r) k[r] = RankKey<T>::make(v[r]);
        } else {
#pragma unroll
            for (int r = 0; r < RADIX_ITEMS; ++r) { const unsigned long long e = wbase + (unsigned long long)r * 32; k[r] = e < hi ? keys[e] : K(0); }
        }
        // counting needs no order: shared-memory atomics on the warp's own histogram (one __match_any_sync per element, which
        // the scatter kernel needs for its stable ranks, made this kernel 6x slower: 5.0 -> 0.82 ms per pass at N = 50,000)
#pragma unroll
        for (int r = 0; r < RADIX_ITEMS; ++r)
            if (wbase + (unsigned long long)r * 32 < hi) atomicAdd(&wh[warp][(uint32_t)((k[r] >> shift) & 255u)], 1u);
    }
    __syncthreads();
    uint32_t t = 0;
    for (int w = 0; w < RADIX_WARPS; ++w) t += wh[w][threadIdx.x];
    hist[(size_t)threadIdx.x * gridDim.x + blockIdx.x] = t;
}

// stable scatter of one digit: offs = exclusive scan of hist (digit-major), i.e. the global position of the first element
// of block b with digit d.  Tiles of the block's range are processed in order; within a tile warp w owns 512 consecutive
// elements and handles them in 16 rounds of 32 (lane order = element order), so equal digits keep their input order.
// The tile is first put into digit order in shared memory (local position = digit's offset in the tile + rank inside the
// digit) and then written out by position: elements of one digit are adjacent there and go to adjacent global addresses, so
// the stores are runs of ~16 elements instead of 32 unrelated words per warp instruction.
template <typename K> constexpr size_t radix_scatter_smem() { return (size_t)RADIX_TILE * (sizeof(K) + sizeof(uint32_t)); }
template <typename T, bool FIRST>
__global__ void __launch_bounds__(RADIX_THREADS)
k_radix_scatter(const T* __restrict__ raw, const typename RankKey<T>::K* __restrict__ keys_in, const uint32_t* __restrict__ idx_in,
                unsigned long long P, unsigned long long per_block, int shift, const uint32_t* __restrict__ offs,
                typename RankKey<T>::K* __restrict__ keys_out, uint32_t* __restrict__ idx_out)
{
    using K = typename RankKey<T>::K;
    extern __shared__ __align__(16) unsigned char rsm[];
    K* skey = reinterpret_cast<K*>(rsm);
    uint32_t* sidx = reinterpret_cast<uint32_t*>(rsm + (size_t)RADIX_TILE * sizeof(K));
    __shared__ uint32_t gbase[256];               // global position of the block's next element of digit d
    __shared__ uint32_t gdelta[256];              // global position - local position of the tile's elements of digit d
    __shared__ uint32_t wh[RADIX_WARPS][256];
    __shared__ uint32_t wsum[RADIX_WARPS];
    gbase[threadIdx.x] = offs[(size_t)threadIdx.x * gridDim.x + blockIdx.x];
    unsigned long long lo, hi;
    radix_range(P, per_block, lo, hi);
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const uint32_t lt = (1u << lane) - 1u;
    for (unsigned long long tile = lo; tile < hi; tile += RADIX_TILE) {
        for (int w = 0; w < RADIX_WARPS; ++w) wh[w][threadIdx.x] = 0;
        __syncthreads();
        K k[RADIX_ITEMS];
        uint32_t id[RADIX_ITEMS];
        const unsigned long long wbase = tile + (unsigned long long)warp * (32 * RADIX_ITEMS) + lane;
        if (FIRST) {                                                   // all loads first, then the key map
            T v[RADIX_ITEMS];
#pragma unroll
            for (int r = 0; r < RADIX_ITEMS; ++r) { const unsigned long long e = wbase + (unsigned long long)r * 32; v[r] = e < hi ? raw[e] : T(0); }
#pragma unroll
            for (int r = 0; r < RADIX_ITEMS; ++r) { k[r] = RankKey<T>::make(v[r]); id[r] = (uint32_t)(wbase + (unsigned long long)r * 32); }
        } else {
#pragma unroll
            for (int r = 0; r < RADIX_ITEMS; ++r) {
                const unsigned long long e = wbase + (unsigned long long)r * 32;
                k[r] = e < hi ? keys_in[e] : K(0);
                id[r] = e < hi ? idx_in[e] : 0u;
            }
        }
        // per-warp digit counts (order does not matter here: shared-memory atomics on the warp's own histogram)
#pragma unroll
        for (int r = 0; r < RADIX_ITEMS; ++r)
            if (wbase + (unsigned long long)r * 32 < hi) atomicAdd(&wh[warp][(uint32_t)((k[r] >> shift) & 255u)], 1u);
        __syncthreads();
        {   // thread d: the tile's count of digit d -> exclusive scan over the digits = local offset of digit d in the tile;
            // wh[w][d] becomes the local position of warp w's first element of digit d
            uint32_t tc = 0;
            for (int w = 0; w < RADIX_WARPS; ++w) tc += wh[w][threadIdx.x];
            uint32_t incl = tc;
#pragma unroll
            for (int o = 1; o < 32; o <<= 1) { const uint32_t x = __shfl_up_sync(0xffffffffu, incl, o); if (lane >= o) incl += x; }
            if (lane == 31) wsum[warp] = incl;
            __syncthreads();
            uint32_t pre = 0;
            for (int w = 0; w < warp; ++w) pre += wsum[w];
            uint32_t run = pre + incl - tc;                                   // local offset of digit d
            gdelta[threadIdx.x] = gbase[threadIdx.x] - run;
            gbase[threadIdx.x] += tc;
            for (int w = 0; w < RADIX_WARPS; ++w) { const uint32_t t = wh[w][threadIdx.x]; wh[w][threadIdx.x] = run; run += t; }
        }
        __syncthreads();
        // the lanes with the same digit in each round: all RADIX_ITEMS matches are issued back to back (MATCH has a long
        // latency; one match followed by its dependent shared-memory update per round left the warp waiting 16 times)
        uint32_t pm[RADIX_ITEMS];
#pragma unroll
        for (int r = 0; r < RADIX_ITEMS; ++r) {
            const bool ok = wbase + (unsigned long long)r * 32 < hi;
            pm[r] = __match_any_sync(0xffffffffu, ok ? (uint32_t)((k[r] >> shift) & 255u) : 256u);
        }
#pragma unroll
        for (int r = 0; r < RADIX_ITEMS; ++r) {
            const bool ok = wbase + (unsigned long long)r * 32 < hi;
            const uint32_t d = ok ? (uint32_t)((k[r] >> shift) & 255u) : 256u;
            const uint32_t peers = pm[r];
            if (ok) {
                const uint32_t lp = wh[warp][d] + (uint32_t)__popc(peers & lt);
                skey[lp] = k[r];
                sidx[lp] = id[r];
            }
            __syncwarp();
            if (ok && lane == __ffs(peers) - 1) wh[warp][d] += (uint32_t)__popc(peers);
            __syncwarp();
        }
        __syncthreads();
        const uint32_t n_tile = (uint32_t)min((unsigned long long)RADIX_TILE, hi - tile);
        for (uint32_t p = threadIdx.x; p < n_tile; p += RADIX_THREADS) {
            const K kk = skey[p];
            const uint32_t pos = p + gdelta[(uint32_t)((kk >> shift) & 255u)];
            keys_out[pos] = kk;
            idx_out[pos] = sidx[p];
        }
        __syncthreads();
    }
}

// ---- runs of equal keys in the sorted order ---------------------------------------------------------------------------
// blast[b] = 1 + (last position in block b's range that starts a run), 0 if none
template <typename K>
__global__ void __launch_bounds__(RADIX_THREADS)
k_rank_block_heads(const K* __restrict__ keys, unsigned long long P, unsigned long long per_block, uint32_t* __restrict__ blast)
{
    __shared__ uint32_t best;
    if (threadIdx.x == 0) best = 0;
    __syncthreads();
    unsigned long long lo, hi;
    radix_range(P, per_block, lo, hi);
    uint32_t mine = 0;
    for (unsigned long long e = lo + threadIdx.x; e < hi; e += RADIX_THREADS)
        if (e == 0 || keys[e] != keys[e - 1]) mine = (uint32_t)e + 1u;
    atomicMax(&best, mine);
    __syncthreads();
    if (threadIdx.x == 0) blast[blockIdx.x] = best;
}

// start[p] = first position of the run of equal keys that p belongs to (prefix maximum of the run-start positions);
// the last element of every run also records the run's length at rlen[start].
template <typename K>
__global__ void __launch_bounds__(RADIX_THREADS)
k_rank_starts(const K* __restrict__ keys, unsigned long long P, unsigned long long per_block, const uint32_t* __restrict__ blast,
              uint32_t* __restrict__ start, uint32_t* __restrict__ rlen)
{
    __shared__ uint32_t wmax[RADIX_WARPS];
    __shared__ uint32_t carry_s;
    unsigned long long lo, hi;
    radix_range(P, per_block, lo, hi);
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    if (threadIdx.x == 0) {
        uint32_t c = 0;
        for (unsigned b = 0; b < blockIdx.x; ++b) c = max(c, blast[b]);
        carry_s = c;
    }
    __syncthreads();
    for (unsigned long long base = lo; base < hi; base += RADIX_THREADS) {
        const unsigned long long e = base + threadIdx.x;
        const bool ok = e < hi;
        uint32_t v = 0;                                                   // 1 + start position, 0 = not a run start
        if (ok && (e == 0 || keys[e] != keys[e - 1])) v = (uint32_t)e + 1u;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) { const uint32_t t = __shfl_up_sync(0xffffffffu, v, o); if (lane >= o) v = max(v, t); }
        if (lane == 31) wmax[warp] = v;
        __syncthreads();
        uint32_t pre = carry_s;
        for (int w = 0; w < warp; ++w) pre = max(pre, wmax[w]);
        v = max(v, pre);
        if (ok) {
            const uint32_t s = v - 1u;                                    // v >= 1: position 0 always starts a run
            start[e] = s;
            if (e + 1 == P || keys[e + 1] != keys[e]) rlen[s] = (uint32_t)e - s + 1u;
        }
        __syncthreads();
        if (threadIdx.x == RADIX_THREADS - 1) carry_s = v;                // inclusive maximum of everything so far
        __syncthreads();
    }
}

// val[p] = 2 * (average rank) of sorted position p = 2 start[p] + (rlen[start[p]] - 1) + 2     (1-based average ranks are
// half-integers: twice the rank is an exact 32-bit integer for n(n-1)/2 < 2^31 - 1, half the bytes of an fp64 rank, and
// Pearson's r does not see the factor 2)
__global__ void __launch_bounds__(256)
k_rank_value(const uint32_t* __restrict__ start, const uint32_t* __restrict__ rlen, unsigned long long P, uint32_t* __restrict__ val)
{
    for (unsigned long long p = (unsigned long long)blockIdx.x * blockDim.x + threadIdx.x; p < P; p += (unsigned long long)gridDim.x * blockDim.x) {
        const uint32_t s = start[p];
        val[p] = 2u * s + (rlen[s] - 1u) + 2u;
    }
}

// rank2[pos[p]] = val[p].  The caller has partitioned the (pos, val) pairs by the top bits of pos (one more radix scatter, on
// the positions), so the blocks that run together write into one window of rank2 that stays in L2 until its sectors are
// complete; scattering straight from the sorted order costs a 32-byte read-modify-write per 4-byte rank (56.7 ms per vector
// at N = 50,000 against 0.5 + 4.5 + 9.5 ms for histogram + partition + this kernel).
// NOT a grid-stride loop: block b owns the RANK_PLACE_PER_BLOCK pairs behind b * RANK_PLACE_PER_BLOCK and blocks are scheduled
// in order, so the blocks in flight stay within one or two windows (persistent blocks drift apart by several windows over
// 10^9 elements and the windows' sectors leave L2 half-written: 45 ms).
constexpr int RANK_PLACE_PER_BLOCK = 2048;
__global__ void __launch_bounds__(256)
k_rank_place(const uint32_t* __restrict__ pos, const uint32_t* __restrict__ val, unsigned long long P, uint32_t* __restrict__ rank2)
{
    const unsigned long long base = (unsigned long long)blockIdx.x * RANK_PLACE_PER_BLOCK + threadIdx.x;
    uint32_t q[RANK_PLACE_PER_BLOCK / 256], v[RANK_PLACE_PER_BLOCK / 256];
#pragma unroll
    for (int u = 0; u < RANK_PLACE_PER_BLOCK / 256; ++u) {
        const unsigned long long p = base + (unsigned long long)u * 256;
        q[u] = 0xffffffffu;
        if (p < P) { q[u] = pos[p]; v[u] = val[p]; }
    }
#pragma unroll
    for (int u = 0; u < RANK_PLACE_PER_BLOCK / 256; ++u)
        if (q[u] != 0xffffffffu) rank2[q[u]] = v[u];
}

}  // namespace ufb
