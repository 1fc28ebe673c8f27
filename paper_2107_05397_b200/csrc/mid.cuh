// mid.cuh -- step a-5 for the MID branches (fp32 mode): too sparse for the dense head kernels, too
// dense for the global RED.ADD scatter.  PAPER.md:23 "sparse-aware optimizations" (mechanism ours,
// DESIGN.md "head / mid / tail split").
//
// A mid branch v is a sorted list of (sample, u~) entries (same arrays as the tail lists).  For the
// 128 x 128 tile pair (I, J) only the n_I x n_J pairs of samples present on BOTH sides contribute
// min(u~_a, u~_b) to M_ab (identities I3 / I5).  One CTA owns the tile pair's 128 x 128 accumulators in
// shared memory as 32-bit FIXED-POINT integers and adds the contributions with native shared-memory
// integer atomics (ATOMS.ADD: 8.84 lane-ops/clk/SM = 2.57e12 /s on B200, the same for conflict-free and for random
// cells -- unifrac_measure_rates, rates.cuh -- against 2.6 /clk/SM for an fp32 CAS loop and 1.9e11 /s for global
// RED.ADD).  Integer addition commutes, so the
// result does not depend on the order in which warps reach a cell.
//   u_q = round(u~ * 2^F),  F = 31 - ceil(log2(max_s R^mid_s)), R^mid_s = sample s's sum over the mid rows
//   =>   acc <= min(R^mid_a, R^mid_b) * 2^F + (rounding) < 2^32   (unsigned 32-bit cells)
//   epilogue: out[idx(a,b)] += acc * 2^-F      (exclusive owner of the tile pair; tail REDs ran before)
// Row bookkeeping: seg[t][r] = offset (within row r's list) of the first entry with sample >= 128 t,
// stored tile-major so that the 32 lanes of a warp (32 consecutive mid rows) read coalesced words.
#pragma once
#include "common.cuh"
#include "tail.cuh"
#include "stripe.cuh"   // smem_u32

namespace ufb {

constexpr int MID_THREADS = 512;
constexpr int MID_MINB = 3;                         // CTAs per SM (3 x 64.5 KB of accumulators)
// accumulator cell (a, b) lives at word a * 128 + (b ^ (a & 31)): bank = (a ^ b) mod 32, and the byte address is
// one LOP3 away from the packed entry word:  (row_base(a) | (a & 31) << 2) ^ (b << 2)
constexpr size_t MID_SMEM = (size_t)TILE * TILE * sizeof(uint32_t) + 512 /*alignment*/;

// mid rows ordered by n_v (counting sort: histogram, scan, scatter) so that the rows a warp handles together
// have similar list lengths; mbase[r] = list offset of row r.  The order inside a bucket is arbitrary --
// harmless, integer accumulation commutes.
__global__ void k_mid_hist(int n, const uint8_t* __restrict__ cls, const uint32_t* __restrict__ nv, uint32_t* __restrict__ hist,
                           uint8_t want /* class of the rows: CLS_MID, or CLS_MIDG_ROOT (midg.cuh) */)
{
    int v = blockIdx.x * blockDim.x + threadIdx.x;
    if (v < n && cls[v] == want) atomicAdd(&hist[nv[v]], 1u);
}
__global__ void k_mid_rows(int n, const uint8_t* __restrict__ cls, const uint32_t* __restrict__ nv, uint32_t* __restrict__ cursor,
                           const uint32_t* __restrict__ tptr, int32_t* __restrict__ mrows, uint32_t* __restrict__ mbase,
                           uint32_t* __restrict__ mlen, uint8_t want)
{
    int v = blockIdx.x * blockDim.x + threadIdx.x;
    if (v < n && cls[v] == want) {
        uint32_t r = atomicAdd(&cursor[nv[v]], 1u);
        mrows[r] = v;
        mbase[r] = tptr[v];
        mlen[r] = nv[v];
    }
}

// seg[t][r] for t = 0..n_tiles = number of entries of row r with sample < 128 t.  One warp per mid row walks the row's
// sorted sample list; the lane that sees the first entry of a new tile fills the boundaries up to that tile.
__global__ void __launch_bounds__(256)
k_mid_seg(uint32_t n_mid, const int32_t* __restrict__ mrows, const uint32_t* __restrict__ tptr,
          const uint32_t* __restrict__ ts, int n_tiles, uint32_t* __restrict__ seg)
{
    const uint32_t r = (blockIdx.x * blockDim.x + threadIdx.x) >> 5;
    const int lane = threadIdx.x & 31;
    if (r >= n_mid) return;
    const int v = mrows[r];
    const uint32_t base = tptr[v], m = tptr[v + 1] - base;
    for (uint32_t k = lane; k < m; k += 32) {
        const int t1 = (int)(ts[base + k] >> 7);
        const int t0 = k ? (int)(ts[base + k - 1] >> 7) : -1;
        for (int t = t0 + 1; t <= t1; ++t) seg[(size_t)t * n_mid + r] = k;
    }
    const int tl = m ? (int)(ts[base + m - 1] >> 7) : -1;
    for (int t = tl + 1 + lane; t <= n_tiles; t += 32) seg[(size_t)t * n_mid + r] = m;
}

// off[t][r], r = 0..n_mid: offset (within tile t's packed entries) of row r's first entry in tile t;
// off[t][n_mid] = ttot[t] = number of packed entries of tile t.  One CTA per tile (exclusive scan over rows).
__global__ void __launch_bounds__(1024)
k_mid_off(uint32_t n_mid, const uint32_t* __restrict__ seg, uint32_t* __restrict__ off, uint32_t* __restrict__ ttot,
          const uint32_t* __restrict__ cut /* rows r < cut[0] are never joined (zone.cuh), or NULL */,
          uint32_t pad /* every (row, tile) list is padded to a multiple of this power of two: 2 (k_mid), 4 (k_midg) */)
{
    __shared__ uint32_t part[1024];
    const uint32_t t = blockIdx.x;
    const uint32_t* s0 = seg + (size_t)t * n_mid;
    const uint32_t* s1 = s0 + n_mid;
    uint32_t* o = off + (size_t)t * (n_mid + 1);
    const int th = threadIdx.x;
    const uint32_t r0 = cut ? cut[0] : 0u;       // rows below cut[0] are in the dense zone of every tile
    auto cnt = [&](uint32_t r) { return r >= r0 ? ((s1[r] - s0[r] + pad - 1u) & ~(pad - 1u)) : 0u; };
    const uint32_t chunk = (n_mid + 1023u) / 1024u;
    uint32_t lo = th * chunk, hi = lo + chunk;
    if (lo > n_mid) lo = n_mid;
    if (hi > n_mid) hi = n_mid;
    uint32_t s = 0;
    for (uint32_t r = lo; r < hi; ++r) s += cnt(r);
    part[th] = s;
    __syncthreads();
    for (int k = 1; k < 1024; k <<= 1) {
        uint32_t add = th >= k ? part[th - k] : 0;
        __syncthreads();
        part[th] += add;
        __syncthreads();
    }
    uint32_t run = th ? part[th - 1] : 0;
    for (uint32_t r = lo; r < hi; ++r) { o[r] = run; run += cnt(r); }
    if (th == 1023) { o[n_mid] = part[1023]; ttot[t] = part[1023]; }
}

// per-sample sums over the mid rows only (they bound the fixed-point accumulators: acc(a, b) <= min(midsum_a, midsum_b) * 2^F).
// One warp per mid row.
__global__ void __launch_bounds__(256)
k_mid_sums(uint32_t n_mid, const uint32_t* __restrict__ mbase, const uint32_t* __restrict__ mlen,
           const uint32_t* __restrict__ ts, const float* __restrict__ tv, double* __restrict__ midsum,
           const uint32_t* __restrict__ cut /* or NULL */)
{
    const uint32_t r = (blockIdx.x * blockDim.x + threadIdx.x) >> 5;
    const int lane = threadIdx.x & 31;
    if (r >= n_mid) return;
    const uint32_t base = mbase[r], m = mlen[r];
    for (uint32_t k = lane; k < m; k += 32) {
        const uint32_t s = ts[base + k];
        if (cut && r < cut[0]) continue;                       // this row is never joined
        atomicAdd(&midsum[s], (double)tv[base + k]);
    }
}

// packed tile-major entries: pk[tbase[t] + off[t][r] + k] = { r << 9 | (sample - 128 t) << 2,  q = round(u~ * 2^F) }
// One warp per mid row.  The side sum of the sample is corrected by (q * 2^-F - u~), so that S_s / R_s and the pairwise
// sums are sums of the SAME numbers (the result is then the exact distance of an embedding perturbed by <= 2^-(F+1) per
// entry); qerr[s] collects the sum and the sum of squares of (q * 2^-F - u~) for the error-ratio check (k_quant_ratio).
__global__ void __launch_bounds__(256)
k_mid_pack(uint32_t n_mid, const uint32_t* __restrict__ mbase, const uint32_t* __restrict__ mlen,
           const uint32_t* __restrict__ ts, const float* __restrict__ tv, const uint32_t* __restrict__ seg,
           const uint32_t* __restrict__ off, const uint32_t* __restrict__ tbase, float qscale, double inv_qscale,
           double* __restrict__ sums, double* __restrict__ qerr, uint2* __restrict__ pk, const uint32_t* __restrict__ cut /* or NULL */)
{
    const uint32_t r = (blockIdx.x * blockDim.x + threadIdx.x) >> 5;
    const int lane = threadIdx.x & 31;
    if (r >= n_mid) return;
    const uint32_t base = mbase[r], m = mlen[r];
    for (uint32_t k = lane; k < m; k += 32) {
        const uint32_t s = ts[base + k];
        const uint32_t t = s >> 7;
        if (cut && r < cut[0]) continue;
        const uint32_t g0 = seg[(size_t)t * n_mid + r], g1 = seg[(size_t)(t + 1) * n_mid + r];
        const uint32_t pos = tbase[t] + off[(size_t)t * (n_mid + 1) + r] + (k - g0);
        const uint32_t x = (r << 9) | ((s & 127u) << 2);
        const float u = tv[base + k];
        const uint32_t q = __float2uint_rn(u * qscale);
        pk[pos] = make_uint2(x, q);
        const double c = (double)q * inv_qscale - (double)u;
        if (c != 0.0) { atomicAdd(&sums[s], c); atomicAdd(&qerr[2 * s], c); atomicAdd(&qerr[2 * s + 1], c * c); }
        if (k + 1 == g1 && ((g1 - g0) & 1u)) pk[pos + 1] = make_uint2(x, 0u);    // padding entry: adds 0 to a valid cell
    }
}

struct MidParams {
    const int2* pairs; uint32_t n_pairs;
    unsigned int* counter;        // dynamic tile-pair queue
    uint32_t n_mid;
    const uint32_t* off;          // [n_tiles][n_mid+1]
    const uint32_t* tbase;        // [n_tiles+1]
    const uint2* pk;              // packed entries, tile-major, rows ascending within a tile
    const uint32_t* cut;          // pair (I, J) joins the rows r >= cut[I] only (zone.cuh); NULL = every row
    int n_samples;
    float* out;
    double inv_qscale;            // 2^-F
};

// The join: every entry (row r, sample a, q_a) of tile I meets the entries (r, b, q_b) of the same row in tile J.
// One lane per I entry, looping over the row's J entries; chunks of 32 consecutive I entries per warp, software
// pipelined (entry loads two chunks ahead, offset gathers one chunk ahead).
__device__ __forceinline__ void mid_red(uint32_t addr, uint32_t v) {
    asm volatile("red.shared.add.u32 [%0], %1;" ::"r"(addr), "r"(v) : "memory");
}

// the join of one tile pair into the CTA's accumulators (macc_s = shared-memory address of row 0); NWARP warps take the chunks
template <int NWARP>
__device__ __forceinline__ void mid_join_pair(const MidParams& P, const int2 ij, const uint32_t macc_s, const int warp, const int lane)
{
    const size_t pitch = (size_t)P.n_mid + 1;
    const uint2* __restrict__ pk = P.pk;
    const uint32_t eI1 = P.tbase[ij.x + 1], eJ0 = P.tbase[ij.y];
    const uint32_t eI0 = P.tbase[ij.x] + (P.cut ? P.off[(size_t)ij.x * pitch + P.cut[ij.x]] : 0u);
    const uint32_t* offJ = P.off + (size_t)ij.y * pitch;
    const uint32_t nchunk = (eI1 - eI0 + 31u) >> 5;

    // pipeline registers: stage A = entry of chunk c+2, stage B = entry + J range of chunk c+1, stage C = current
    uint2 entA = make_uint2(0u, 0u), entB = make_uint2(0u, 0u), entC;
    uint32_t jB0 = 0, jB1 = 0, jC0, jC1;
    bool vA = false, vB = false;
    auto load_ent = [&](uint32_t c, uint2& ent, bool& valid) {
        const uint32_t e = eI0 + c * 32u + lane;
        valid = c < nchunk && e < eI1;
        if (valid) ent = __ldg(pk + e);
    };
    auto load_range = [&](const uint2& ent, bool valid, uint32_t& j0, uint32_t& j1) {
        j0 = j1 = 0;
        if (valid && ent.y != 0u) {                      // q = 0 (padding entries) contributes nothing
            const uint32_t r = ent.x >> 9;
            j0 = eJ0 + offJ[r];                          // both even: 16-byte aligned pairs of entries
            j1 = eJ0 + offJ[r + 1];
        }
    };
    // The diagonal tile pair (I == J) walks the row's full list as well: cells with a >= b receive sums that the
    // epilogue never reads (it keeps gi < gj only).
    uint32_t c = warp;
    load_ent(c, entB, vB);
    load_range(entB, vB, jB0, jB1);
    load_ent(c + NWARP, entA, vA);
    for (; c < nchunk; c += NWARP) {
        entC = entB; jC0 = jB0; jC1 = jB1;
        entB = entA; vB = vA;
        load_range(entB, vB, jB0, jB1);
        load_ent(c + 2 * NWARP, entA, vA);
        const uint32_t a4 = entC.x & 0x1fcu;                                  // 4 a
        const uint32_t arow = (macc_s + (a4 << 7)) | (a4 & 0x7cu);            // row base | (a & 31) << 2
        const uint32_t qa = entC.y;
        uint32_t l = jC0;
        while (__any_sync(0xffffffffu, l < jC1)) {
            uint4 f0, f1;
            const bool p0 = l < jC1, p1 = l + 2u < jC1;
            if (p0) f0 = __ldg(reinterpret_cast<const uint4*>(pk + l));
            if (p1) f1 = __ldg(reinterpret_cast<const uint4*>(pk + l + 2));
            if (p0) { mid_red(arow ^ (f0.x & 0x1fcu), min(qa, f0.y)); mid_red(arow ^ (f0.z & 0x1fcu), min(qa, f0.w)); }
            if (p1) { mid_red(arow ^ (f1.x & 0x1fcu), min(qa, f1.y)); mid_red(arow ^ (f1.z & 0x1fcu), min(qa, f1.w)); }
            l += 4;
        }
    }
}

// epilogue of a tile pair: add its fixed-point sums to the condensed matrix (exclusive owner; the tail REDs ran before)
template <int NTHREADS>
__device__ __forceinline__ void mid_epilogue(const uint32_t* macc, const int2 ij, const long long N, float* __restrict__ out, const double inv_qscale)
{
    const uint32_t sI = (uint32_t)ij.x * TILE, sJ = (uint32_t)ij.y * TILE;
    for (int e = threadIdx.x; e < TILE * TILE; e += NTHREADS) {
        const int a = e >> 7, b = (e & 127) ^ (a & 31);
        const uint32_t q = macc[e];
        if (q) {
            const long long gi = (long long)sI + a, gj = (long long)sJ + b;
            if (gi < gj && gj < N) {
                float* o = out + (gi * (2 * N - gi - 1) / 2 - gi - 1 + gj);
                *o = (float)((double)*o + (double)q * inv_qscale);
            }
        }
    }
}

__global__ void __launch_bounds__(MID_THREADS, MID_MINB)
k_mid(const MidParams P)
{
    extern __shared__ uint32_t macc_raw[];
    __shared__ int s_pair;
    const uint32_t raw_s = smem_u32(macc_raw);
    const uint32_t macc_s = (raw_s + 511u) & ~511u;                    // 512-byte aligned rows: row a at macc_s + 512 a
    uint32_t* macc = macc_raw + ((macc_s - raw_s) >> 2);
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    for (;;) {
        if (threadIdx.x == 0) s_pair = (int)atomicAdd(P.counter, 1u);
        for (int i = threadIdx.x; i < TILE * TILE; i += MID_THREADS) macc[i] = 0u;
        __syncthreads();
        const int pi = s_pair;
        if ((uint32_t)pi >= P.n_pairs) break;
        const int2 ij = P.pairs[pi];
        mid_join_pair<MID_THREADS / 32>(P, ij, macc_s, warp, lane);
        __syncthreads();
        mid_epilogue<MID_THREADS>(macc, ij, P.n_samples, P.out, P.inv_qscale);
        __syncthreads();
    }
}

}  // namespace ufb
