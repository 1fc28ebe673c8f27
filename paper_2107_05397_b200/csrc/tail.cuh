// tail.cuh -- the sparse half of the sparse-aware split ("sparse-aware optimizations";
// the mechanism is ours).
//
// Branches are classified by n_v = number of samples present below them:
//   head  (n_v large)  : dense enough that the register-tiled stripe kernel (stripe.cuh) is the
//                        cheaper way to cover all N(N-1)/2 pairs;
//   tail  (n_v small)  : only the C(n_v,2) pairs of samples that are BOTH present contribute
//                        min(u~_a, u~_b) to M_ab (identities I3/I5), so the branch is stored as a
//                        sorted list of (sample, u~) entries and its pair contributions are
//                        scattered straight into the condensed matrix with fp32/fp64 RED.ADD.
// The scatter is ordered by output "super tiles" (ranges of SUP samples x SUP samples whose
// condensed rows fit the L2 cache), one launch per super tile, so the atomics resolve in L2
// (measured: 1.9e11 RED/s L2-resident vs 2e10 RED/s when the footprint spills to HBM).
//
// Steps:  bit-packed presence up the tree (a-1/a-2 on bits, BASELINE.json:5 "presence bits,
// bit-packed in 32/64-sample words ... level by level")  ->  n_v (popcount)  ->  classification
// ->  sparse values / sample lists (embed.cuh, k_values)  ->  super-tile segment offsets  ->  scatter.
#pragma once
#include "common.cuh"

namespace ufb {

enum : uint8_t { CLS_NONE = 0, CLS_HEAD = 1, CLS_TAIL = 2, CLS_MID = 3 };

// ------------------------------------------------------------------ presence bits (all samples at once)
// bits[v][w] bit b  <=>  sample 32*w + b has a positive count on some tip below v
__global__ void k_bits_scatter(int n_samples, const int64_t* __restrict__ indptr, const int32_t* __restrict__ indices,
                               const int32_t* __restrict__ counts, uint32_t* __restrict__ bits, uint32_t NW)
{
    int s = (blockIdx.x * blockDim.x + threadIdx.x) >> 5;
    int lane = threadIdx.x & 31;
    if (s >= n_samples) return;
    long long lo = indptr[s], hi = indptr[s + 1];
    const uint32_t w = (uint32_t)s >> 5, m = 1u << (s & 31);
    for (long long k = lo + lane; k < hi; k += 32)
        if (counts[k] > 0) atomicOr(&bits[(size_t)indices[k] * NW + w], m);
}

// parents of one depth level OR their children's rows (uint4 = 128 samples per thread); NW4 = NW/4
__global__ void k_bits_pull(const int32_t* __restrict__ nodes, int n_nodes_level, int skip_node,
                            const uint32_t* __restrict__ child_off, const int32_t* __restrict__ child_idx,
                            uint4* __restrict__ bits, uint32_t NW4)
{
    long long gid = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    long long q = gid / NW4;
    uint32_t ch = (uint32_t)(gid - q * NW4);
    if (q >= n_nodes_level) return;
    int v = nodes[q];
    if (v == skip_node) return;
    uint4 acc = make_uint4(0, 0, 0, 0);
    for (uint32_t k = child_off[v]; k < child_off[v + 1]; ++k) {
        uint4 c = bits[(size_t)child_idx[k] * NW4 + ch];
        acc.x |= c.x; acc.y |= c.y; acc.z |= c.z; acc.w |= c.w;
    }
    bits[(size_t)v * NW4 + ch] = acc;
}

// ne[v] = popcount of row v (0 for the root); n_v = ne[v] if the branch has a positive length, else 0.  One warp per node.
__global__ void k_bits_count(int n, const int32_t* __restrict__ parent, const double* __restrict__ len,
                             const uint4* __restrict__ bits, uint32_t NW4, uint32_t* __restrict__ nv, uint32_t* __restrict__ ne)
{
    int v = (blockIdx.x * blockDim.x + threadIdx.x) >> 5;
    int lane = threadIdx.x & 31;
    if (v >= n) return;
    uint32_t c = 0;
    if (parent[v] >= 0) {
        for (uint32_t k = lane; k < NW4; k += 32) {
            uint4 x = bits[(size_t)v * NW4 + k];
            c += __popc(x.x) + __popc(x.y) + __popc(x.z) + __popc(x.w);
        }
    }
    for (int o = 16; o; o >>= 1) c += __shfl_xor_sync(0xffffffffu, c, o);
    if (lane == 0) { ne[v] = c; nv[v] = len[v] > 0.0 ? c : 0u; }
}

// max over a vector of non-negative doubles (bit patterns order like the values)
__global__ void k_max_positive(int n, const double* __restrict__ x, unsigned long long* __restrict__ out_bits)
{
    int i = blockIdx.x * blockDim.x + threadIdx.x;
    unsigned long long b = 0;
    if (i < n && x[i] > 0.0) b = (unsigned long long)__double_as_longlong(x[i]);
    for (int o = 16; o; o >>= 1) { unsigned long long t = __shfl_xor_sync(0xffffffffu, b, o); b = t > b ? t : b; }
    if ((threadIdx.x & 31) == 0 && b) atomicMax(out_bits, b);
}

// Fixed-point error ratio.  The fixed-point kernels (Gram head lengths, mid entries)
// replace embedded values u~ by u~ + delta; the side sums use the same replaced values, so the result is the exact distance
// of the perturbed embedding.  Per sample: B_s = sum of delta (systematic part: e.g. many branches of one length round the
// same way), V_s = sum of delta^2 (random part).  ratio = max_s (|B_s| + 3 sqrt(V_s)) / S_s bounds the relative change of
// any of the sample's branch-subset sums at 3 sigma; a pair with d >= 1/16 (smaller ones go through k_guard) moves by at
// most ~32 x ratio relative.  Bit pattern of a double >= 0.
__global__ void k_quant_ratio(int n, const double* __restrict__ qerr, const double* __restrict__ sums, unsigned long long* __restrict__ out_bits)
{
    int i = blockIdx.x * blockDim.x + threadIdx.x;
    unsigned long long b = 0;
    if (i < n && qerr[2 * i + 1] > 0.0) {
        const double e = fabs(qerr[2 * i]) + 3.0 * sqrt(qerr[2 * i + 1]);
        const double r = sums[i] > 0.0 ? e / sums[i] : 1.0;
        b = (unsigned long long)__double_as_longlong(r);
    }
    for (int o = 16; o; o >>= 1) { unsigned long long t = __shfl_xor_sync(0xffffffffu, b, o); b = t > b ? t : b; }
    if ((threadIdx.x & 31) == 0 && b) atomicMax(out_bits, b);
}

__global__ void k_mark_class(int n, const uint8_t* __restrict__ cls, uint8_t which, uint32_t* __restrict__ mark)
{
    int v = blockIdx.x * blockDim.x + threadIdx.x;
    if (v < n) mark[v] = cls[v] == which ? 1u : 0u;
}

// head / mid / tail rule, per branch (costs are additive over branches, so a per-branch rule is optimal):
//   C(n_v,2) >= c2_head            -> head  (dense kernel: cost per branch independent of n_v)
//   c2_mid <= C(n_v,2) < c2_head   -> mid   (pair contributions accumulated per 128 x 128 tile pair in shared memory, mid.cuh)
//   C(n_v,2) < c2_mid              -> tail  (pair contributions scattered with global RED.ADD, k_tail_scatter)
// mid and tail branches share one list format; tcnt[v] = n_v for both (0 for head rows), scanned into the
// list offsets.  counters[0..5] = head rows, tail rows, tail pair updates, list entries (all rows that keep a list), mid rows, mid pair updates; counters[9] = entries of the mid rows.
__global__ void k_classify(int n, const uint32_t* __restrict__ nv, const uint32_t* __restrict__ ne, int all_rows,
                           double c2_head, double c2_mid, uint32_t force,
                           uint8_t* __restrict__ cls, uint32_t* __restrict__ tcnt, unsigned long long* __restrict__ counters)
{
    int v = blockIdx.x * blockDim.x + threadIdx.x;
    unsigned long long h = 0, t = 0, tu = 0, te = 0, m = 0, mu = 0, me = 0;
    if (v < n) {
        unsigned long long k = nv[v];
        uint8_t c = CLS_NONE;
        if (k) {
            double c2 = 0.5 * (double)k * (double)(k - 1);
            c = force == 2 ? CLS_TAIL : force == 1 ? CLS_HEAD : c2 >= c2_head ? CLS_HEAD : c2 >= c2_mid ? CLS_MID : CLS_TAIL;
            if (c == CLS_TAIL) { t = 1; tu = k * (k - 1) / 2; }
            else if (c == CLS_MID) { m = 1; mu = k * (k - 1) / 2; me = k; }
            else h = 1;
        }
        cls[v] = c;
        // rows that keep an entry list: mid and tail rows; all_rows (weighted): every row with a present sample,
        // zero-length branches included (their counts still propagate to the parent)
        const uint32_t keep = all_rows ? ne[v] : ((c == CLS_TAIL || c == CLS_MID) ? (uint32_t)k : 0u);
        tcnt[v] = keep;
        te = keep;
    }
    for (int o = 16; o; o >>= 1) {
        h += __shfl_xor_sync(0xffffffffu, h, o);  t += __shfl_xor_sync(0xffffffffu, t, o);
        tu += __shfl_xor_sync(0xffffffffu, tu, o); te += __shfl_xor_sync(0xffffffffu, te, o);
        m += __shfl_xor_sync(0xffffffffu, m, o);  mu += __shfl_xor_sync(0xffffffffu, mu, o);
        me += __shfl_xor_sync(0xffffffffu, me, o);
    }
    if ((threadIdx.x & 31) == 0 && (h | t | m)) {
        atomicAdd(&counters[0], h); atomicAdd(&counters[1], t); atomicAdd(&counters[2], tu); atomicAdd(&counters[3], te);
        atomicAdd(&counters[4], m); atomicAdd(&counters[5], mu); atomicAdd(&counters[9], me);
    }
}

// ------------------------------------------------------------------ super-tile segments of the lists
// seg[v][k] = number of entries of row v with sample id < k*SUP, k = 0..nsup   (thread per (v,k))
__global__ void k_tail_seg(int n, const uint32_t* __restrict__ tptr, const uint32_t* __restrict__ ts,
                           int SUP, int nsup, uint32_t* __restrict__ seg)
{
    long long gid = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    long long v = gid / (nsup + 1);
    int k = (int)(gid - v * (nsup + 1));
    if (v >= n) return;
    const uint32_t lo0 = tptr[v], hi0 = tptr[v + 1];
    uint32_t lo = lo0, hi = hi0;
    const uint32_t key = (uint32_t)k * (uint32_t)SUP;
    while (lo < hi) {
        uint32_t mid = lo + ((hi - lo) >> 1);
        if (ts[mid] < key) lo = mid + 1; else hi = mid;
    }
    seg[(size_t)v * (nsup + 1) + k] = lo - lo0;
}

// ------------------------------------------------------------------ the scatter
// One launch per super tile (SI <= SJ).  A warp takes 32 consecutive nodes; rows whose cross product in
// this super tile is small are done one per lane, larger ones by the whole warp (lanes over the longer
// list).  out[idx(a,b)] += min(u~_a, u~_b)   for a in range SI, b in range SJ, a < b.
template <typename T>
__device__ __forceinline__ void red_add(T* p, T v) { atomicAdd(p, v); }

struct TailParams {
    const uint32_t* tptr;   // [n+1]
    const uint32_t* seg;    // [n][nsup+1]
    const uint32_t* ts;     // sample ids
    const void* tv;         // values (T)
    const uint8_t* cls;     // [n] only CLS_TAIL rows are scattered here
    int n, nsup, SI, SJ;
    long long N;
    void* out;
    unsigned int* counter;  // dynamic chunk queue (one word per launch)
    const uint8_t* owner;   // shard mode: owner[bj*(bj+1)/2 + bi] of every SHARD_BLOCK x SHARD_BLOCK block of tiles; NULL = all
    int shard;              // this shard's index
};

constexpr int SHARD_BLOCK = 12;          // == UNIFRAC_SHARD_BLOCK of the C header
// does this shard own the pair of samples a < b ?  (owner table lookups hit L1)
__device__ __forceinline__ bool tail_owns(const TailParams& P, long long a, long long b) {
    if (!P.owner) return true;
    const uint32_t bi = ((uint32_t)a >> 7) / SHARD_BLOCK, bj = ((uint32_t)b >> 7) / SHARD_BLOCK;
    return P.owner[bj * (bj + 1) / 2 + bi] == (uint8_t)P.shard;
}

constexpr int TAIL_SMALL = 8;

template <typename T>
__global__ void __launch_bounds__(256)
k_tail_scatter(const TailParams P)
{
    const int lane = threadIdx.x & 31;
    const T* tv = reinterpret_cast<const T*>(P.tv);
    T* out = reinterpret_cast<T*>(P.out);
    const long long N = P.N;
    const int nchunks = (P.n + 31) >> 5;
    const bool diag = P.SI == P.SJ;
    for (;;) {
        int chunk = 0;
        if (lane == 0) chunk = (int)atomicAdd(P.counter, 1u);
        chunk = __shfl_sync(0xffffffffu, chunk, 0);
        if (chunk >= nchunks) break;
        const int v = chunk * 32 + lane;
        uint32_t i0 = 0, i1 = 0, j0 = 0, j1 = 0, base = 0;
        if (v < P.n && P.cls[v] == CLS_TAIL) {
            const uint32_t* sg = P.seg + (size_t)v * (P.nsup + 1);
            i0 = sg[P.SI]; i1 = sg[P.SI + 1];
            if (diag) { j0 = i0; j1 = i1; } else { j0 = sg[P.SJ]; j1 = sg[P.SJ + 1]; }
            base = P.tptr[v];
        }
        const uint32_t nI = i1 - i0, nJ = j1 - j0;
        const uint32_t work = diag ? (nI * (nI - (nI ? 1u : 0u))) / 2u : nI * nJ;
        // ---- small rows: one per lane
        if (work && work <= (uint32_t)TAIL_SMALL) {
            for (uint32_t k = i0; k < i1; ++k) {
                const long long a = P.ts[base + k];
                const T va = tv[base + k];
                const long long rowoff = a * (2 * N - a - 1) / 2 - a - 1;
                for (uint32_t l = diag ? k + 1 : j0; l < j1; ++l) {
                    const T vb = tv[base + l];
                    const long long b = P.ts[base + l];
                    if (tail_owns(P, a, b)) red_add(out + rowoff + b, va < vb ? va : vb);
                }
            }
        }
        // ---- larger rows: whole warp, lanes over the longer list, loop over the shorter one
        uint32_t big = __ballot_sync(0xffffffffu, work > (uint32_t)TAIL_SMALL);
        while (big) {
            const int src = __ffs(big) - 1;
            big &= big - 1;
            const uint32_t bi0 = __shfl_sync(0xffffffffu, i0, src), bi1 = __shfl_sync(0xffffffffu, i1, src);
            const uint32_t bj0 = __shfl_sync(0xffffffffu, j0, src), bj1 = __shfl_sync(0xffffffffu, j1, src);
            const uint32_t bb = __shfl_sync(0xffffffffu, base, src);
            if (!diag) {
                // off-diagonal super tile: the nI x nJ products are dealt to the lanes as one flat list (product t = lane,
                // lane + 32, ...; (i, j) advanced incrementally), so short lists still fill the warp's RED instructions
                const uint32_t nI2 = bi1 - bi0, nJ2 = bj1 - bj0, tot = nI2 * nJ2;
                uint32_t i = (uint32_t)lane / nJ2, j = (uint32_t)lane - i * nJ2;
                const uint32_t di = 32u / nJ2, dj = 32u - di * nJ2;
                for (uint32_t t = lane; t < tot; t += 32) {
                    const long long sa = P.ts[bb + bi0 + i], sb = P.ts[bb + bj0 + j];
                    const T va = tv[bb + bi0 + i], vb = tv[bb + bj0 + j];
                    if (tail_owns(P, sa, sb)) red_add(out + (sa * (2 * N - sa - 1) / 2 - sa - 1) + sb, va < vb ? va : vb);
                    i += di; j += dj;
                    if (j >= nJ2) { j -= nJ2; ++i; }
                }
                continue;
            }
            const bool lanesJ = diag || (bj1 - bj0) >= (bi1 - bi0);       // lane entries are the b's (else the a's)
            const uint32_t p0 = lanesJ ? bj0 : bi0, p1 = lanesJ ? bj1 : bi1;   // lane list
            const uint32_t q0 = lanesJ ? bi0 : bj0, q1 = lanesJ ? bi1 : bj1;   // loop list
            for (uint32_t l0 = p0; l0 < p1; l0 += 32) {
                const uint32_t l = l0 + lane;
                const bool lv = l < p1;
                const long long se = lv ? (long long)P.ts[bb + l] : 0;
                const T ve = lv ? tv[bb + l] : (T)0;
                const long long rowoff_e = se * (2 * N - se - 1) / 2 - se - 1;    // used when the lane entry is the a
                const uint32_t kend = diag ? (l0 + 32 < q1 ? l0 + 32 : q1) : q1;  // diag: only k < l
                for (uint32_t k = q0; k < kend; ++k) {
                    const long long sf = P.ts[bb + k];        // warp-uniform (broadcast) loads
                    const T vf = tv[bb + k];
                    if (lv && (!diag || k < l) && (lanesJ ? tail_owns(P, sf, se) : tail_owns(P, se, sf))) {
                        const T m = ve < vf ? ve : vf;
                        if (lanesJ) red_add(out + (sf * (2 * N - sf - 1) / 2 - sf - 1) + se, m);
                        else        red_add(out + rowoff_e + sf, m);
                    }
                }
            }
        }
    }
}

}  // namespace ufb
