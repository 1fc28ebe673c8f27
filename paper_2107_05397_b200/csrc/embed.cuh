// embed.cuh -- steps a-1 .. a-4 (SURVEY 8a / DESIGN.md "K1 embedding builder"; BASELINE.json:5
// subsystem (1): "a per-branch embedding builder that propagates each sample's normalised
// abundances (weighted) or presence bits (unweighted, bit-packed in 32/64-sample words) up the
// postorder tree level by level").
//
// The embedding is SPARSE ("rank layout"): the bit-packed presence matrix bits[v][w] (tail.cuh,
// k_bits_scatter / k_bits_pull) says which samples are present below branch v, and the values of the
// present samples are stored contiguously, in sample order, at
//     entry(v, s) = eptr[v] + rank_v(s),   rank_v(s) = popcount(bits[v] below sample s).
//   a-1  k_csc_fill + k_tip_cnt : integer counts of the tips, through a by-tip (CSC) copy of the table
//   a-2  k_cnt_pull             : parents of one depth level sum their children's entries (exact
//                                 integers; the child entry of sample s is found by rank)
//   a-3  k_values               : per-sample side sums R_s / S_s (fp64), sample ids of the entries
//   a-4  k_values               : pre-scaled values u~ = len * cnt / T_s (weighted) or len (unweighted)
// Only the weighted variant needs counts; the unweighted variant works from the bits alone.
// Head rows of the CUDA-core stripe kernel are then expanded into compact dense per-tile rows
// E_t[rank][128] with 4-bit quarter masks (k_head_flags, k_rank_scan, k_head_pref, k_compact).
#pragma once
#include "common.cuh"

namespace ufb {

// inclusive warp scan
__device__ __forceinline__ uint32_t warp_incl_scan(uint32_t x, int lane)
{
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) { uint32_t t = __shfl_up_sync(0xffffffffu, x, o); if (lane >= o) x += t; }
    return x;
}

// ------------------------------------------------------------------ a-1: table by tip (CSC), unordered within a tip
// one warp per sample; cursor[t] counts the entries appended to tip t so far
__global__ void k_csc_fill(int n_samples, const int64_t* __restrict__ indptr, const int32_t* __restrict__ indices,
                           const int32_t* __restrict__ counts, const uint32_t* __restrict__ cptr,
                           uint32_t* __restrict__ cursor, uint32_t* __restrict__ csc_s, uint32_t* __restrict__ csc_c)
{
    int s = (blockIdx.x * blockDim.x + threadIdx.x) >> 5;
    int lane = threadIdx.x & 31;
    if (s >= n_samples) return;
    long long lo = indptr[s], hi = indptr[s + 1];
    for (long long k = lo + lane; k < hi; k += 32) {
        int c = counts[k];
        if (c > 0) {
            int t = indices[k];
            uint32_t p = cptr[t] + atomicAdd(&cursor[t], 1u);
            csc_s[p] = (uint32_t)s;
            csc_c[p] = (uint32_t)c;
        }
    }
}

// tipc[v] = number of table entries of tip v (0 for internal nodes); total[0] += their sum
__global__ void k_tip_mark(int n, const int32_t* __restrict__ child_count, const uint32_t* __restrict__ ne,
                           uint32_t* __restrict__ tipc, unsigned long long* __restrict__ total)
{
    int v = blockIdx.x * blockDim.x + threadIdx.x;
    unsigned long long c = 0;
    if (v < n) { c = child_count[v] == 0 ? ne[v] : 0u; tipc[v] = (uint32_t)c; }
    for (int o = 16; o; o >>= 1) c += __shfl_xor_sync(0xffffffffu, c, o);
    if ((threadIdx.x & 31) == 0 && c) atomicAdd(total, c);
}

// head rank -> node id
__global__ void k_head_rows(int n, const uint8_t* __restrict__ cls, const uint32_t* __restrict__ hrank, int32_t* __restrict__ hrows)
{
    int v = blockIdx.x * blockDim.x + threadIdx.x;
    if (v < n && cls[v] == 1) hrows[hrank[v]] = v;
}

// a-1: counts of the tips in rank layout.  One warp per tip at a time.  Tips seen in <= 32 samples: the
// rank of an entry is the number of smaller sample ids in the tip's own list (warp shuffles).  Otherwise the
// warp builds the word-prefix popcounts of the tip's bit row in shared memory (NW words per warp).
__global__ void __launch_bounds__(256)
k_tip_cnt(int n, const int32_t* __restrict__ child_count, const uint32_t* __restrict__ ne,
          const uint32_t* __restrict__ cptr, const uint32_t* __restrict__ csc_s, const uint32_t* __restrict__ csc_c,
          const uint32_t* __restrict__ bits, uint32_t NW, const uint32_t* __restrict__ eptr, uint32_t* __restrict__ cnt)
{
    extern __shared__ uint32_t pre_sm[];                 // [warps per block][NW]
    const int lane = threadIdx.x & 31, wib = threadIdx.x >> 5;
    uint32_t* pre = pre_sm + (size_t)wib * NW;
    const int warps = (gridDim.x * blockDim.x) >> 5;
    for (int t = (blockIdx.x * blockDim.x + threadIdx.x) >> 5; t < n; t += warps) {
        const uint32_t m = ne[t];
        if (m == 0 || child_count[t] != 0) continue;
        const uint32_t c0 = cptr[t], e0 = eptr[t];
        if (m <= 32) {
            uint32_t s = 0xffffffffu, c = 0;
            if ((uint32_t)lane < m) { s = csc_s[c0 + lane]; c = csc_c[c0 + lane]; }
            uint32_t rank = 0;
            for (uint32_t j = 0; j < m; ++j) { uint32_t sj = __shfl_sync(0xffffffffu, s, (int)j); rank += sj < s ? 1u : 0u; }
            if ((uint32_t)lane < m) cnt[e0 + rank] = c;
            continue;
        }
        const uint32_t* row = bits + (size_t)t * NW;
        uint32_t run = 0;
        for (uint32_t w0 = 0; w0 < NW; w0 += 32) {
            uint32_t w = w0 + lane;
            uint32_t word = w < NW ? row[w] : 0u;
            uint32_t c = __popc(word), incl = warp_incl_scan(c, lane);
            if (w < NW) pre[w] = run + incl - c;
            run += __shfl_sync(0xffffffffu, incl, 31);
        }
        __syncwarp();
        for (uint32_t k = lane; k < m; k += 32) {
            uint32_t s = csc_s[c0 + k];
            uint32_t word = row[s >> 5];
            cnt[e0 + pre[s >> 5] + __popc(word & ((1u << (s & 31)) - 1u))] = csc_c[c0 + k];
        }
        __syncwarp();
    }
}

// ------------------------------------------------------------------ a-2: level-by-level propagation in rank layout
// One warp per parent node of the level.  The warp walks the parent's bit row 32 words at a time keeping the
// running entry offsets of the parent and of each child; a present sample's count is the sum of the counts of
// the children in which it is present.
constexpr int PULL_MAX_CHILDREN = 4;      // children handled per pass (binary trees: one pass)
__global__ void __launch_bounds__(256)
k_cnt_pull(const int32_t* __restrict__ nodes, int n_nodes_level, int skip_node,
           const uint32_t* __restrict__ child_off, const int32_t* __restrict__ child_idx,
           const uint32_t* __restrict__ bits, uint32_t NW, const uint32_t* __restrict__ eptr, uint32_t* __restrict__ cnt)
{
    const int q = (blockIdx.x * blockDim.x + threadIdx.x) >> 5, lane = threadIdx.x & 31;
    if (q >= n_nodes_level) return;
    const int v = nodes[q];
    if (v == skip_node) return;
    const uint32_t* prow = bits + (size_t)v * NW;
    const uint32_t pe = eptr[v];
    const uint32_t k0 = child_off[v], k1 = child_off[v + 1];
    for (uint32_t kb = k0; kb < k1; kb += PULL_MAX_CHILDREN) {
        const int nc = (int)min((uint32_t)PULL_MAX_CHILDREN, k1 - kb);
        const uint32_t* crow[PULL_MAX_CHILDREN];
        uint32_t ce[PULL_MAX_CHILDREN], crun[PULL_MAX_CHILDREN];
#pragma unroll
        for (int j = 0; j < PULL_MAX_CHILDREN; ++j) {
            const int c = j < nc ? child_idx[kb + j] : 0;
            crow[j] = bits + (size_t)c * NW; ce[j] = j < nc ? eptr[c] : 0u; crun[j] = 0;
        }
        uint32_t prun = 0;
        const bool first = kb == k0;
        for (uint32_t w0 = 0; w0 < NW; w0 += 32) {
            const uint32_t w = w0 + lane;
            uint32_t pw = w < NW ? prow[w] : 0u;
            if (!__any_sync(0xffffffffu, pw != 0u)) continue;            // children are subsets of the parent
            const uint32_t pc = __popc(pw), pincl = warp_incl_scan(pc, lane);
            uint32_t ppos = pe + prun + pincl - pc;
            prun += __shfl_sync(0xffffffffu, pincl, 31);
            uint32_t cw[PULL_MAX_CHILDREN], cpos[PULL_MAX_CHILDREN];
#pragma unroll
            for (int j = 0; j < PULL_MAX_CHILDREN; ++j) {
                cw[j] = 0u; cpos[j] = 0u;
                if (j < nc) {                                              // warp-uniform
                    if (w < NW) cw[j] = crow[j][w];
                    const uint32_t cc = __popc(cw[j]), cincl = warp_incl_scan(cc, lane);
                    cpos[j] = ce[j] + crun[j] + cincl - cc;
                    crun[j] += __shfl_sync(0xffffffffu, cincl, 31);
                }
            }
            while (pw) {
                const uint32_t bit = pw & (0u - pw);
                pw ^= bit;
                uint32_t sum = first ? 0u : cnt[ppos];
#pragma unroll
                for (int j = 0; j < PULL_MAX_CHILDREN; ++j)
                    if (cw[j] & bit) sum += cnt[cpos[j]++];
                cnt[ppos++] = sum;
            }
        }
    }
}

// ------------------------------------------------------------------ a-3 / a-4: values, sample ids, side sums
// One warp per branch v with n_v > 0 (non-root, len > 0).  For every present sample s, in sample order:
//   u~ = len_v * cnt / T_s   (weighted; the quotient of exact integers, rounded once)    or
//   u~ = uval[v] (unweighted; the branch's embedded length: len_v, or its fixed-point value on the Gram path)
//   rounded to T;  sums[s] += (double)u~ (fp64 RED.ADD; every kernel of step a-5 sees exactly these rounded values, so
//   the side sums and the pairwise sums are sums of the same numbers);  rows that keep a list (tcnt[v] > 0: mid and
//   tail rows, and every row of the weighted variant) also get ts[e] = s, tv[e] = u~.
template <typename T>
__global__ void __launch_bounds__(256)
k_values(int n, const uint32_t* __restrict__ nv, const uint32_t* __restrict__ tcnt, const uint32_t* __restrict__ tptr,
         const double* __restrict__ len, const double* __restrict__ uval, const uint32_t* __restrict__ bits, uint32_t NW,
         const uint32_t* __restrict__ cnt /* weighted: counts in rank layout at tptr; else NULL */,
         const unsigned long long* __restrict__ Tsum, uint32_t* __restrict__ ts, T* __restrict__ tv,
         double* __restrict__ sums, const double* __restrict__ uerr /* per-branch (u~ - len) of the fixed point, or NULL */,
         double* __restrict__ qerr /* [2 * samples] per-sample sum and sum of squares of it */)
{
    const int v = (blockIdx.x * blockDim.x + threadIdx.x) >> 5, lane = threadIdx.x & 31;
    if (v >= n || nv[v] == 0) return;
    const bool list = tcnt[v] != 0;
    const double ev = uerr ? uerr[v] : 0.0;
    const uint32_t e0 = tptr[v];
    const double l = len[v];
    const T uconst = (T)(uval ? uval[v] : l);
    const uint32_t* row = bits + (size_t)v * NW;
    uint32_t run = 0;
    for (uint32_t w0 = 0; w0 < NW; w0 += 32) {
        const uint32_t w = w0 + lane;
        uint32_t word = w < NW ? row[w] : 0u;
        if (!__any_sync(0xffffffffu, word != 0u)) continue;
        const uint32_t c = __popc(word), incl = warp_incl_scan(c, lane);
        uint32_t e = e0 + run + incl - c;
        run += __shfl_sync(0xffffffffu, incl, 31);
        while (word) {
            const int b = __ffs(word) - 1;
            word &= word - 1;
            const uint32_t s = w * 32 + b;
            T val = uconst;
            if (cnt) val = (T)(l * ((double)cnt[e] / (double)Tsum[s]));
            if (list) { ts[e] = s; tv[e] = val; }
            atomicAdd(&sums[s], (double)val);
            if (ev != 0.0) { atomicAdd(&qerr[2 * s], ev); atomicAdd(&qerr[2 * s + 1], ev * ev); }
            ++e;
        }
    }
}

// ------------------------------------------------------------------ head rows of the CUDA-core stripe kernel
// row flags: flags[t][w] bit b <=> branch 32 w + b is a head row with a present sample in tile t.
// One warp per flag word (32 branches, one per lane), looping over the tiles of its branches' bit rows.
__global__ void __launch_bounds__(256)
k_head_flags(int n, const uint8_t* __restrict__ cls, const uint32_t* __restrict__ bits, uint32_t NW,
             int n_tiles, uint32_t* __restrict__ flags, uint32_t nwords)
{
    const uint32_t w = (blockIdx.x * blockDim.x + threadIdx.x) >> 5;
    const int lane = threadIdx.x & 31;
    if (w >= nwords) return;
    const int v = (int)(w * 32 + lane);
    const bool head = v < n && cls[v] == 1;
    if (!__any_sync(0xffffffffu, head)) {
        for (int t = lane; t < n_tiles; t += 32) flags[(size_t)t * nwords + w] = 0u;
        return;
    }
    const uint4* row = reinterpret_cast<const uint4*>(bits + (size_t)(head ? v : 0) * NW);
    for (int t = 0; t < n_tiles; ++t) {
        uint4 g = make_uint4(0, 0, 0, 0);
        if (head) g = row[t];
        const uint32_t word = __ballot_sync(0xffffffffu, (g.x | g.y | g.z | g.w) != 0u);
        if (lane == 0) flags[(size_t)t * nwords + w] = word;
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

// hpref[h][t] = number of present samples of head row h before tile t (= entry offset of the tile's first sample).
// One warp per head row.
__global__ void __launch_bounds__(256)
k_head_pref(uint32_t n_head, const int32_t* __restrict__ hrows, const uint32_t* __restrict__ bits, uint32_t NW,
            int n_tiles, uint32_t* __restrict__ hpref)
{
    const uint32_t h = (blockIdx.x * blockDim.x + threadIdx.x) >> 5;
    const int lane = threadIdx.x & 31;
    if (h >= n_head) return;
    const uint32_t* row = bits + (size_t)hrows[h] * NW;
    uint32_t run = 0;
    for (uint32_t w0 = 0; w0 < NW; w0 += 32) {
        const uint32_t w = w0 + lane;
        const uint32_t word = w < NW ? row[w] : 0u;
        const uint32_t c = __popc(word), incl = warp_incl_scan(c, lane);
        if ((w & 3u) == 0u && (int)(w >> 2) < n_tiles) hpref[(size_t)h * n_tiles + (w >> 2)] = run + incl - c;
        run += __shfl_sync(0xffffffffu, incl, 31);
    }
}

template <typename T> struct Vec4;
template <> struct Vec4<float>  { static __device__ __forceinline__ void store(float* p, float a, float b, float c, float d) {
    *reinterpret_cast<float4*>(p) = make_float4(a, b, c, d); } };
template <> struct Vec4<double> { static __device__ __forceinline__ void store(double* p, double a, double b, double c, double d) {
    reinterpret_cast<double2*>(p)[0] = make_double2(a, b); reinterpret_cast<double2*>(p)[1] = make_double2(c, d); } };

// compact dense rows of the head branches: E_t[r][128] (zeros where absent) and the 4-bit quarter mask Q_t[r].
// grid.x = chunks of COMPACT_WORDS flag words, grid.y = tile; 8 warps per CTA, one row per warp-iteration;
// lane l owns samples 4l .. 4l+3 of the tile.
constexpr int COMPACT_WORDS = 64;
template <typename T>
__global__ void __launch_bounds__(256)
k_compact(int n, const double* __restrict__ len, const uint32_t* __restrict__ bits, uint32_t NW,
          const uint32_t* __restrict__ flags, const uint32_t* __restrict__ rank, uint32_t nwords, int n_tiles,
          const uint32_t* __restrict__ tptr, const uint32_t* __restrict__ hrank, const uint32_t* __restrict__ hpref,
          const T* __restrict__ tv /* weighted: values in rank layout; else NULL */,
          T* const* __restrict__ tileE, uint8_t* const* __restrict__ tileQ)
{
    const int tile = blockIdx.y;
    const int wv = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const uint32_t* f = flags + (size_t)tile * nwords;
    const uint32_t* rk = rank + (size_t)tile * nwords;
    T* E = tileE[tile];
    uint8_t* Q = tileQ[tile];
    uint32_t w0 = blockIdx.x * COMPACT_WORDS;
    uint32_t w1 = w0 + COMPACT_WORDS; if (w1 > nwords) w1 = nwords;
    for (uint32_t w = w0; w < w1; ++w) {
        const uint32_t word = f[w];
        const uint32_t base = rk[w];
        uint32_t m = word;
        int k = 0;
        while (m) {
            const int b = __ffs(m) - 1;
            m &= m - 1;
            if ((k++ & 7) != wv) continue;                     // the 8 warps share the rows of this word round-robin
            const int v = (int)(w * 32 + b);
            const uint32_t r = base + __popc(word & ((1u << b) - 1u));
            const uint4 g = reinterpret_cast<const uint4*>(bits + (size_t)v * NW)[tile];
            const uint32_t gw[4] = {g.x, g.y, g.z, g.w};
            const int wi = lane >> 3, sh = (lane & 7) * 4;
            const uint32_t mine = gw[wi];
            const uint32_t m4 = (mine >> sh) & 15u;
            T x[4] = {(T)0, (T)0, (T)0, (T)0};
            if (tv) {
                uint32_t e = tptr[v] + hpref[(size_t)hrank[v] * n_tiles + tile] + __popc(mine & ((1u << sh) - 1u));
                if (wi > 0) e += __popc(gw[0]);
                if (wi > 1) e += __popc(gw[1]);
                if (wi > 2) e += __popc(gw[2]);
#pragma unroll
                for (int j = 0; j < 4; ++j) if (m4 & (1u << j)) x[j] = tv[e++];
            } else {
                const T l = (T)len[v];
#pragma unroll
                for (int j = 0; j < 4; ++j) if (m4 & (1u << j)) x[j] = l;
            }
            Vec4<T>::store(E + (size_t)r * TILE + lane * 4, x[0], x[1], x[2], x[3]);
            if (lane == 0) Q[r] = (uint8_t)((g.x ? 1u : 0u) | (g.y ? 2u : 0u) | (g.z ? 4u : 0u) | (g.w ? 8u : 0u));
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
