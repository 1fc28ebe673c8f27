// embed.cuh -- steps a-1 .. a-4 (SURVEY 8a / DESIGN.md "K1 embedding builder"; BASELINE.json:5
// subsystem (1): "a per-branch embedding builder that propagates each sample's normalised
// abundances ... up the postorder tree level by level").
//
// Per batch of Wb samples (Wb a multiple of 128): exact integer subtree counts cnt[v][s] are
// scattered at the tips (a-1) and summed children -> parent one depth level at a time (a-2).  The
// batch is then cut into 128-sample tiles; for every tile the non-empty rows (branches with len > 0
// and at least one present sample) are flagged, ranked and written as a compact row-major
// embedding E_t[rank][128] of pre-scaled values u~ = len * cnt / T_s (weighted) or len * [cnt > 0]
// (unweighted) (a-4), together with a 4-bit mask of its non-empty 32-sample quarters; the
// per-sample side sums R_s / S_s = sum_v u~_sv (fp64) and per-branch sample counts n_v come out
// of the same pass (a-3).
#pragma once
#include "common.cuh"

namespace ufb {

// a-1: one warp per sample of the batch
__global__ void k_tip_scatter(int s0, int s1, const int64_t* __restrict__ indptr, const int32_t* __restrict__ indices,
                              const int32_t* __restrict__ counts, uint32_t* __restrict__ cnt, int Wb)
{
    int s = s0 + ((blockIdx.x * blockDim.x + threadIdx.x) >> 5);
    int lane = threadIdx.x & 31;
    if (s >= s1) return;
    long long lo = indptr[s], hi = indptr[s + 1];
    for (long long k = lo + lane; k < hi; k += 32) {
        int c = counts[k];
        if (c > 0) cnt[(size_t)indices[k] * Wb + (s - s0)] = (uint32_t)c;
    }
}

// a-2: parents of one depth level pull their children's rows (uint4 = 4 samples per thread)
__global__ void k_level_pull(const int32_t* __restrict__ nodes, int n_nodes_level, int skip_node,
                             const uint32_t* __restrict__ child_off, const int32_t* __restrict__ child_idx,
                             uint32_t* __restrict__ cnt, int Wb)
{
    int chunks = Wb >> 2;
    long long gid = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    long long q = gid / chunks;
    int ch = (int)(gid - q * chunks);
    if (q >= n_nodes_level) return;
    int v = nodes[q];
    if (v == skip_node) return;        // the root has no branch
    uint4 acc = make_uint4(0, 0, 0, 0);
    for (uint32_t k = child_off[v]; k < child_off[v + 1]; ++k) {
        uint4 c = reinterpret_cast<const uint4*>(cnt + (size_t)child_idx[k] * Wb)[ch];
        acc.x += c.x; acc.y += c.y; acc.z += c.z; acc.w += c.w;
    }
    reinterpret_cast<uint4*>(cnt + (size_t)v * Wb)[ch] = acc;
}

// a-3: row flags.  One CTA (32 warps) = 32 consecutive nodes (one flag word) x one tile of the batch.
__global__ void __launch_bounds__(1024)
k_row_flags(int n, const int32_t* __restrict__ parent, const double* __restrict__ len,
            const uint32_t* __restrict__ cnt, int Wb, uint32_t* __restrict__ flags /*[tile][nwords]*/,
            uint32_t nwords, int tile0, uint8_t* __restrict__ qtmp /*[tiles_in_batch][n]*/,
            const uint8_t* __restrict__ cls /*[n] 1 = head row (stripe kernel), others are not flagged*/)
{
    __shared__ uint32_t q_sm[32];
    int w = blockIdx.x, tb = blockIdx.y;
    int wv = threadIdx.x >> 5, lane = threadIdx.x & 31;
    int v = w * 32 + wv;
    bool valid = v < n && cls[v] == 1;
    uint4 c = make_uint4(0, 0, 0, 0);
    if (valid) c = reinterpret_cast<const uint4*>(cnt + (size_t)v * Wb + (size_t)tb * TILE)[lane];
    int nz = (c.x != 0) + (c.y != 0) + (c.z != 0) + (c.w != 0);
    uint32_t b = __ballot_sync(0xffffffffu, nz != 0);
    uint32_t q = ((b & 0x000000ffu) ? 1u : 0u) | ((b & 0x0000ff00u) ? 2u : 0u) |
                 ((b & 0x00ff0000u) ? 4u : 0u) | ((b & 0xff000000u) ? 8u : 0u);
    if (lane == 0) {
        q_sm[wv] = q;
        if (v < n) qtmp[(size_t)tb * n + v] = (uint8_t)q;
    }
    __syncthreads();
    if (threadIdx.x < 32) {
        uint32_t word = __ballot_sync(0xffffffffu, q_sm[threadIdx.x] != 0);
        if (threadIdx.x == 0) flags[(size_t)(tile0 + tb) * nwords + w] = word;
    }
}

// rank[tile][w] = number of flagged rows of the tile in words < w; rows[tile] = total.  One CTA per tile.
__global__ void __launch_bounds__(1024)
k_rank_scan(const uint32_t* __restrict__ flags, uint32_t* __restrict__ rank, uint32_t nwords, int tile0,
            uint32_t* __restrict__ rows)
{
    __shared__ uint32_t part[1024];
    int tile = tile0 + blockIdx.x;
    const uint32_t* f = flags + (size_t)tile * nwords;
    uint32_t* r = rank + (size_t)tile * nwords;
    int t = threadIdx.x;
    uint32_t chunk = (nwords + 1023u) / 1024u;
    uint32_t lo = t * chunk, hi = lo + chunk;
    if (lo > nwords) lo = nwords;
    if (hi > nwords) hi = nwords;
    uint32_t s = 0;
    for (uint32_t k = lo; k < hi; ++k) s += __popc(f[k]);
    part[t] = s;
    __syncthreads();
    for (int o = 1; o < 1024; o <<= 1) {
        uint32_t add = t >= o ? part[t - o] : 0;
        __syncthreads();
        part[t] += add;
        __syncthreads();
    }
    uint32_t run = t ? part[t - 1] : 0;
    for (uint32_t k = lo; k < hi; ++k) { r[k] = run; run += __popc(f[k]); }
    if (t == 1023) rows[tile] = part[1023];
}

template <typename T> struct Vec4;
template <> struct Vec4<float>  { static __device__ __forceinline__ void store(float* p, double a, double b, double c, double d, double* back) {
    float4 v = make_float4((float)a, (float)b, (float)c, (float)d);
    *reinterpret_cast<float4*>(p) = v; back[0] = v.x; back[1] = v.y; back[2] = v.z; back[3] = v.w; } };
template <> struct Vec4<double> { static __device__ __forceinline__ void store(double* p, double a, double b, double c, double d, double* back) {
    reinterpret_cast<double2*>(p)[0] = make_double2(a, b); reinterpret_cast<double2*>(p)[1] = make_double2(c, d);
    back[0] = a; back[1] = b; back[2] = c; back[3] = d; } };

// a-4 + a-3: write the compact pre-scaled embedding rows of one batch and accumulate side sums.
// grid.x = chunks of CH flag words, grid.y = tile in batch; 8 warps per CTA, one row per warp-iteration.
constexpr int COMPACT_WORDS = 64;
template <typename T>
__global__ void __launch_bounds__(256)
k_compact(int n, const double* __restrict__ len, const uint32_t* __restrict__ cnt, int Wb,
          const uint32_t* __restrict__ flags, const uint32_t* __restrict__ rank, uint32_t nwords, int tile0,
          const unsigned long long* __restrict__ Tsum, int n_samples, int weighted,
          T* const* __restrict__ tileE, uint8_t* const* __restrict__ tileQ, const uint8_t* __restrict__ qtmp)
{
    int tb = blockIdx.y, tile = tile0 + tb;
    int wv = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const uint32_t* f = flags + (size_t)tile * nwords;
    const uint32_t* rk = rank + (size_t)tile * nwords;
    T* E = tileE[tile];
    uint8_t* Q = tileQ[tile];
    double Tl[4];
#pragma unroll
    for (int e = 0; e < 4; ++e) {
        int s = tile * TILE + lane * 4 + e;
        Tl[e] = s < n_samples ? (double)Tsum[s] : 1.0;
    }
    uint32_t w0 = blockIdx.x * COMPACT_WORDS;
    uint32_t w1 = w0 + COMPACT_WORDS; if (w1 > nwords) w1 = nwords;
    for (uint32_t w = w0; w < w1; ++w) {
        uint32_t word = f[w];
        uint32_t base = rk[w];
        // the 8 warps share the rows of this word round-robin
        uint32_t m = word;
        int k = 0;
        while (m) {
            int b = __ffs(m) - 1;
            m &= m - 1;
            if ((k++ & 7) != wv) continue;
            int v = (int)(w * 32 + b);
            uint32_t r = base + __popc(word & ((1u << b) - 1u));
            uint4 c = reinterpret_cast<const uint4*>(cnt + (size_t)v * Wb + (size_t)tb * TILE)[lane];
            double l = len[v];
            double x0, x1, x2, x3;
            if (weighted) {
                x0 = c.x ? l * ((double)c.x / Tl[0]) : 0.0;
                x1 = c.y ? l * ((double)c.y / Tl[1]) : 0.0;
                x2 = c.z ? l * ((double)c.z / Tl[2]) : 0.0;
                x3 = c.w ? l * ((double)c.w / Tl[3]) : 0.0;
            } else {
                x0 = c.x ? l : 0.0; x1 = c.y ? l : 0.0; x2 = c.z ? l : 0.0; x3 = c.w ? l : 0.0;
            }
            double back[4];
            Vec4<T>::store(E + (size_t)r * TILE + lane * 4, x0, x1, x2, x3, back);
            if (lane == 0) Q[r] = qtmp[(size_t)tb * n + v];
        }
    }
}

// work counters from the per-branch sample counts n_v: exact integers
__global__ void k_work_counts(int n, const uint32_t* __restrict__ nv, unsigned long long N,
                              unsigned long long* __restrict__ out /*[4]: B_emb, W_union, W_inter, sum n_v*/)
{
    int v = blockIdx.x * blockDim.x + threadIdx.x;
    unsigned long long b = 0, wu = 0, wi = 0, sn = 0;
    if (v < n) {
        unsigned long long k = nv[v];
        if (k) {
            b = 1; sn = k;
            wi = k * (k - 1) / 2;
            unsigned long long m = N - k;
            wu = N * (N - 1) / 2 - m * (m - 1) / 2;
        }
    }
    for (int o = 16; o; o >>= 1) {
        b += __shfl_xor_sync(0xffffffffu, b, o);  wu += __shfl_xor_sync(0xffffffffu, wu, o);
        wi += __shfl_xor_sync(0xffffffffu, wi, o); sn += __shfl_xor_sync(0xffffffffu, sn, o);
    }
    if ((threadIdx.x & 31) == 0 && b) {
        atomicAdd(&out[0], b); atomicAdd(&out[1], wu); atomicAdd(&out[2], wi); atomicAdd(&out[3], sn);
    }
}

}  // namespace ufb
