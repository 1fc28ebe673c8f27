// midg.cuh -- step a-5 for the mid branches, GROUPED join (fp32 mode).  PAPER.md:23 "sparse-aware optimizations"; the
// mechanism is ours.
//
// The samples in which a branch is present are a SUBSET of the samples in which its parent branch is present (a-2: a parent's
// bit row is the OR of its children's, its counts their sum).  So for a group of mid branches below a group ROOT r -- r itself
// and up to MIDG_L - 1 descendants connected to it -- every pair of samples (a, b) that any member touches is a pair of r, and
//     sum over the members v of min(u~_va, u~_vb)        (u~ = 0 where v is absent: min(0, x) = 0 adds nothing)
// can be formed in registers and added to the tile pair's accumulator with ONE shared-memory atomic per pair of r instead of
// one per member.  The atomic unit is what bounds k_mid (8.8 lanes/clk/SM); at Large / weighted the groups chosen below need
// 0.38 of k_mid's atomics for the same sums (profiles/r02_summary.md 4d).
//
// Grouping (k_midg_level, top-down by tree level): a mid branch c whose parent belongs to the group of root r joins that group
// if n_c > theta n_r and the group still has a free slot; otherwise c starts a group of its own.  Groups that stay alone
// (one member) remain ordinary k_mid rows.  Which of several competing children gets the last slot depends on the order of
// atomics; the RESULT does not: all sums are exact integer sums of the same fixed-point values q = round(u~ 2^F) that k_mid uses.
//
// Layout: the root's entries are packed tile-major exactly like k_mid's rows (k_mid_seg / k_mid_off on the root list);
// position p holds  ex[p] = g << 9 | (sample - 128 t) << 2  and  eq[p] = the MIDG_L fixed-point values of the members at
// that sample (slot 0 = the root; 0 where a member is absent or the slot is unused).
#pragma once
#include "mid.cuh"

namespace ufb {

constexpr int MIDG_L = 4;            // members per group = fixed-point values per position (one uint4)
constexpr int MIDG_R = 2;            // I positions per lane of k_midg; every (group, tile) list is padded to a multiple of it
constexpr uint8_t CLS_MIDG_ROOT = 4, CLS_MIDG_MEMBER = 5;
constexpr int MIDG_THREADS = 384;       // x 3 CTAs per SM: 56 registers per thread
constexpr int MIDG_MINB = 3;
constexpr uint32_t MIDG_MASK0 = 0x200u;  // mask mode: bit 9 + slot of a position's 16-bit word = member `slot` is present there (bits 2..8: cell << 2)

// children of the internal nodes of one tree level: groot[c] = root of c's group, gslot[c] = its slot, gcnt[r] = members so far
__global__ void k_midg_level(uint32_t n_lv, const int32_t* __restrict__ level_nodes, const uint32_t* __restrict__ child_off,
                             const int32_t* __restrict__ child_idx, const uint8_t* __restrict__ cls, const uint32_t* __restrict__ nv,
                             uint32_t theta_256, int32_t* __restrict__ groot, uint8_t* __restrict__ gslot, uint32_t* __restrict__ gcnt)
{
    const uint32_t i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n_lv) return;
    const int u = level_nodes[i];
    const int r = cls[u] == CLS_MID ? groot[u] : -1;
    const unsigned long long lim = r >= 0 ? (unsigned long long)theta_256 * nv[r] : 0ull;
    for (uint32_t k = child_off[u]; k < child_off[u + 1]; ++k) {
        const int c = child_idx[k];
        if (cls[c] != CLS_MID) continue;
        int g = c; uint32_t slot = 0;
        if (r >= 0 && (unsigned long long)nv[c] * 256ull > lim) {
            slot = atomicAdd(&gcnt[r], 1u);
            if (slot < (uint32_t)MIDG_L) g = r; else slot = 0;
        }
        groot[c] = g;
        gslot[c] = (uint8_t)slot;
        if (g == c) gcnt[c] = 1u;
    }
}

// members of groups with at least two members leave the k_mid rows: cnt[0] += roots, cnt[1] += rows (roots + members),
// cnt[2] += entries of the roots, cnt[3] += sum of n_v (n_v - 1) / 2 over the rows that left, cnt[4] += the same over the roots only
__global__ void k_midg_classify(int n, uint8_t* __restrict__ cls, const uint32_t* __restrict__ nv, const int32_t* __restrict__ groot,
                                const uint32_t* __restrict__ gcnt, unsigned long long* __restrict__ cnt)
{
    const int v = blockIdx.x * blockDim.x + threadIdx.x;
    if (v >= n || cls[v] != CLS_MID) return;
    const int r = groot[v];
    if (gcnt[r] < 2u) return;
    const bool is_root = r == v;
    cls[v] = is_root ? CLS_MIDG_ROOT : CLS_MIDG_MEMBER;
    const unsigned long long k = nv[v];
    if (is_root) { atomicAdd(&cnt[0], 1ull); atomicAdd(&cnt[2], k); atomicAdd(&cnt[4], k * (k - 1) / 2); }
    atomicAdd(&cnt[1], 1ull);
    atomicAdd(&cnt[3], k * (k - 1) / 2);
}

// per-sample sums over the grouped rows (they count toward the bound of the fixed-point accumulators like k_mid's rows)
__global__ void __launch_bounds__(256)
k_midg_sums(int n, const uint8_t* __restrict__ cls, const uint32_t* __restrict__ tptr, const uint32_t* __restrict__ nv,
            const uint32_t* __restrict__ ts, const float* __restrict__ tv, double* __restrict__ midsum)
{
    const int v = (int)((blockIdx.x * (unsigned)blockDim.x + threadIdx.x) >> 5);
    const int lane = threadIdx.x & 31;
    if (v >= n || (cls[v] != CLS_MIDG_ROOT && cls[v] != CLS_MIDG_MEMBER)) return;
    const uint32_t base = tptr[v], m = nv[v];
    for (uint32_t k = lane; k < m; k += 32) atomicAdd(&midsum[ts[base + k]], (double)tv[base + k]);
}

__global__ void k_midg_index(uint32_t n_g, const int32_t* __restrict__ grows, int32_t* __restrict__ rootidx)
{
    const uint32_t g = blockIdx.x * blockDim.x + threadIdx.x;
    if (g < n_g) rootidx[grows[g]] = (int32_t)g;
}

// fixed-point value of an entry and the correction of the sample's side sum (the same bookkeeping as k_mid_pack)
__device__ __forceinline__ uint32_t midg_quant(float u, uint32_t s, float qscale, double inv_qscale, double* __restrict__ sums,
                                               double* __restrict__ qerr)
{
    const uint32_t q = __float2uint_rn(u * qscale);
    const double c = (double)q * inv_qscale - (double)u;
    if (c != 0.0) { atomicAdd(&sums[s], c); atomicAdd(&qerr[2 * s], c); atomicAdd(&qerr[2 * s + 1], c * c); }
    return q;
}

// Position of sample a (0..127 within its tile) in the (group, tile) list of a root whose presence bits in the tile are the
// four words w[0..3] (bit r of w[j] = sample 32 j + r): the list is ordered by (a mod 32, a / 32), NOT by a.  A lane of k_midg
// owns two consecutive positions and one ATOMS covers every second position of up to 32 lanes, all in the same column b of the
// accumulator tile, whose bank is (a xor b) mod 32: in this order the rows a of one instruction differ mod 32 unless three
// samples of the list share a residue, so the lanes of a group hit different banks (sorted by a they collided 3-fold:
// ncu 3.06 shared-memory wavefronts per ATOMS).
__device__ __forceinline__ uint32_t midg_rank(const uint4 w, uint32_t a)
{
    const uint32_t r = a & 31u, j = a >> 5, lt = (1u << r) - 1u;
    uint32_t k = __popc(w.x & lt) + __popc(w.y & lt) + __popc(w.z & lt) + __popc(w.w & lt);
    if (j > 0) k += (w.x >> r) & 1u;
    if (j > 1) k += (w.y >> r) & 1u;
    if (j > 2) k += (w.z >> r) & 1u;
    return k;
}
__device__ __forceinline__ bool midg_has(const uint4 w, uint32_t a)
{
    const uint32_t j = a >> 5, x = j == 0 ? w.x : j == 1 ? w.y : j == 2 ? w.z : w.w;
    return (x >> (a & 31u)) & 1u;
}

// roots: one warp per group g.  Padding positions of a (group, tile) list: ex repeats a valid cell, eq = 0 (memset).
// bits4 = the presence bits of the tree nodes as uint4 (128 samples = one tile per element), NW4 elements per node.
__global__ void __launch_bounds__(256)
k_midg_pack_roots(uint32_t n_g, const int32_t* __restrict__ grows, const uint32_t* __restrict__ gbase, const uint32_t* __restrict__ glen,
                  const uint32_t* __restrict__ ts, const float* __restrict__ tv, const uint4* __restrict__ bits4, uint32_t NW4,
                  const uint32_t* __restrict__ off, const uint32_t* __restrict__ tbase, float qscale, double inv_qscale,
                  double* __restrict__ sums, double* __restrict__ qerr, uint32_t* __restrict__ ex, uint32_t* __restrict__ eq,
                  uint16_t* __restrict__ em, uint32_t* __restrict__ gq /* mask mode (unweighted), else NULL: see k_midg<true> */)
{
    const uint32_t g = (blockIdx.x * blockDim.x + threadIdx.x) >> 5;
    const int lane = threadIdx.x & 31;
    if (g >= n_g) return;
    const uint32_t base = gbase[g], m = glen[g];
    const uint4* __restrict__ wrow = bits4 + (size_t)grows[g] * NW4;
    for (uint32_t k = lane; k < m; k += 32) {
        const uint32_t s = ts[base + k];
        const uint32_t t = s >> 7, a = s & 127u;
        const uint4 w = wrow[t];
        const uint32_t len = __popc(w.x) + __popc(w.y) + __popc(w.z) + __popc(w.w);
        const uint32_t rk = midg_rank(w, a);
        const uint32_t pos = tbase[t] + off[(size_t)t * (n_g + 1) + g] + rk;
        const uint32_t x = (g << 9) | (a << 2);
        ex[pos] = x;
        const uint32_t q = midg_quant(tv[base + k], s, qscale, inv_qscale, sums, qerr);
        if (em) { em[pos] = (uint16_t)((a << 2) | MIDG_MASK0); gq[(size_t)g * MIDG_L] = q; }     // the same q for every entry of the row
        else eq[(size_t)pos * MIDG_L] = q;
        if (rk + 1 == len)
            for (uint32_t f = len; f & (MIDG_R - 1); ++f) { ex[pos + 1 + (f - len)] = x; if (em) em[pos + 1 + (f - len)] = (uint16_t)(a << 2); }
    }
}

// members: one warp per tree node (only CLS_MIDG_MEMBER nodes do anything).  Every sample of the member is a sample of its
// root: the position comes from the ROOT's presence bits; a miss (never, by the subset property) is counted.
__global__ void __launch_bounds__(256)
k_midg_pack_members(int n, const uint8_t* __restrict__ cls, const int32_t* __restrict__ groot, const uint8_t* __restrict__ gslot,
                    const int32_t* __restrict__ rootidx, const uint32_t* __restrict__ tptr, const uint32_t* __restrict__ nv,
                    const uint32_t* __restrict__ ts, const float* __restrict__ tv, const uint4* __restrict__ bits4, uint32_t NW4,
                    uint32_t n_g, const uint32_t* __restrict__ off, const uint32_t* __restrict__ tbase, float qscale, double inv_qscale,
                    double* __restrict__ sums, double* __restrict__ qerr, uint32_t* __restrict__ eq, unsigned long long* __restrict__ misses,
                    uint16_t* __restrict__ em, uint32_t* __restrict__ gq)
{
    const int v = (int)((blockIdx.x * (unsigned)blockDim.x + threadIdx.x) >> 5);
    const int lane = threadIdx.x & 31;
    if (v >= n || cls[v] != CLS_MIDG_MEMBER) return;
    const int r = groot[v];
    const uint32_t g = (uint32_t)rootidx[r], slot = gslot[v];
    const uint32_t base = tptr[v], m = nv[v];
    const uint4* __restrict__ wrow = bits4 + (size_t)r * NW4;
    for (uint32_t k = lane; k < m; k += 32) {
        const uint32_t s = ts[base + k];
        const uint32_t t = s >> 7, a = s & 127u;
        const uint4 w = wrow[t];
        if (!midg_has(w, a)) { atomicAdd(misses, 1ull); continue; }
        const uint32_t pos = tbase[t] + off[(size_t)t * (n_g + 1) + g] + midg_rank(w, a);
        const uint32_t q = midg_quant(tv[base + k], s, qscale, inv_qscale, sums, qerr);
        if (em) {                                                // set the member's bit in the position's 16-bit word
            atomicOr(reinterpret_cast<uint32_t*>(em) + (pos >> 1), (MIDG_MASK0 << slot) << (16u * (pos & 1u)));
            gq[(size_t)g * MIDG_L + slot] = q;
        } else eq[(size_t)pos * MIDG_L + slot] = q;
    }
}

struct MidgParams {
    const int2* pairs; uint32_t n_pairs;
    unsigned int* counter;        // dynamic tile-pair queue
    uint32_t n_g;
    const uint32_t* off;          // [n_tiles][n_g+1]
    const uint32_t* tbase;        // [n_tiles+1]
    const uint32_t* ex;           // packed positions, tile-major, groups ascending within a tile
    const uint4* eq;              // MIDG_L = 4 values per position
    int n_samples;
    float* out;
    double inv_qscale;            // 2^-F
    const uint16_t* em;           // mask mode (k_midg<true>, unweighted): per position cell << 2 | member mask << 9 ...
    const uint4* gq;              // ... and per group the members' (constant) fixed-point values
    MidParams rows;               // the mid rows that stayed alone: joined by the same CTA into the same accumulators (n_mid = 0: none)
};

__device__ __forceinline__ uint32_t midg_dot(const uint4& a, const uint4& b) {
    return min(a.x, b.x) + min(a.y, b.y) + min(a.z, b.z) + min(a.w, b.w);
}

// The grouped join: every position (group g, sample a, values qa[]) of tile I meets the positions (g, b, qb[]) of the same
// group in tile J.  A lane owns MIDG_R = 4 consecutive I positions (same group: the lists are padded to multiples of 4), a warp
// a chunk of 128; every J position a lane loads (20 bytes: cell + 4 values) feeds 4 atomics.  That ratio is the point: a
// warp-wide 16-byte load occupies the L1 data pipe for 4 cycles whether or not the lanes read the same address, and with
// one I position per lane those loads, not the atomics, bounded the kernel (ncu: data pipe 94 %, of it atomics 31 %).
// MASK = true (unweighted): a member's value is the same at every sample where it is present (u~ = the branch length), so a
// position carries 4 presence bits instead of 4 values -- 2 bytes per J position instead of 20 -- and the lane adds the group's
// values q[k] where both positions have the bit.
__device__ __forceinline__ uint32_t midg_sel(uint32_t m, const uint4& q) {
    return ((m & MIDG_MASK0) ? q.x : 0u) + ((m & (MIDG_MASK0 << 1)) ? q.y : 0u) + ((m & (MIDG_MASK0 << 2)) ? q.z : 0u) + ((m & (MIDG_MASK0 << 3)) ? q.w : 0u);
}
template <bool MASK>
__global__ void __launch_bounds__(MIDG_THREADS, MIDG_MINB)
k_midg(const MidgParams P)
{
    extern __shared__ uint32_t macc_raw[];
    __shared__ int s_pair;
    const uint32_t raw_s = smem_u32(macc_raw);
    const uint32_t macc_s = (raw_s + 511u) & ~511u;                    // 512-byte aligned rows: row a at macc_s + 512 a
    uint32_t* macc = macc_raw + ((macc_s - raw_s) >> 2);
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    constexpr int NWARP = MIDG_THREADS / 32;
    const long long N = P.n_samples;
    const size_t pitch = (size_t)P.n_g + 1;
    const uint32_t* __restrict__ ex = P.ex;
    const uint4* __restrict__ eq = P.eq;

    for (;;) {
        if (threadIdx.x == 0) s_pair = (int)atomicAdd(P.counter, 1u);
        for (int i = threadIdx.x; i < TILE * TILE; i += MIDG_THREADS) macc[i] = 0u;
        __syncthreads();
        const int pi = s_pair;
        if ((uint32_t)pi >= P.n_pairs) break;
        const int2 ij = P.pairs[pi];
        // the rows that are in no group first, into the same integer accumulators: one conversion to fp32 per pair, and a
        // result that does not depend on which rows the grouping picked (integer sums are exact)
        if (P.rows.n_mid) mid_join_pair<NWARP>(P.rows, ij, macc_s, warp, lane);
        const uint32_t eI0 = P.tbase[ij.x], eI1 = P.tbase[ij.x + 1], eJ0 = P.tbase[ij.y];
        const uint32_t* offJ = P.off + (size_t)ij.y * pitch;
        const uint32_t nchunk = (eI1 - eI0 + 32u * MIDG_R - 1u) / (32u * MIDG_R);

        // one chunk ahead: the cells of the lane and the J range of their group
        uint32_t xB[MIDG_R], xC[MIDG_R];
        uint32_t jB0 = 0, jB1 = 0, jC0, jC1;
        auto load_pos = [&](uint32_t c, uint32_t (&x)[MIDG_R], uint32_t& j0, uint32_t& j1) {
            const uint32_t e = eI0 + (c * 32u + lane) * MIDG_R;
            j0 = j1 = 0;
#pragma unroll
            for (int k = 0; k < MIDG_R; ++k) x[k] = 0u;
            if (c < nchunk && e < eI1) {
                if (MIDG_R == 4) { const uint4 t = __ldg(reinterpret_cast<const uint4*>(ex + e)); x[0] = t.x; x[1] = t.y; x[MIDG_R - 2] = t.z; x[MIDG_R - 1] = t.w; }
                else { const uint2 t = __ldg(reinterpret_cast<const uint2*>(ex + e)); x[0] = t.x; x[1] = t.y; }
                const uint32_t g = x[0] >> 9;
                j0 = eJ0 + offJ[g];                          // multiples of MIDG_R
                j1 = eJ0 + offJ[g + 1];
            }
        };
        uint32_t c = warp;
        load_pos(c, xB, jB0, jB1);
        for (; c < nchunk; c += NWARP) {
#pragma unroll
            for (int k = 0; k < MIDG_R; ++k) xC[k] = xB[k];
            jC0 = jB0; jC1 = jB1;
            const uint32_t e = eI0 + (c * 32u + lane) * MIDG_R;
            uint4 q[MIDG_R];
            uint32_t row[MIDG_R], mA[MIDG_R];
            if (MASK) {
                static_assert(MIDG_R == 2, "mask mode reads the lane's two 16-bit words as one 32-bit load");
                q[0] = make_uint4(0u, 0u, 0u, 0u);
                uint32_t w = 0u;
                if (jC0 < jC1) { q[0] = __ldg(P.gq + (xC[0] >> 9)); w = __ldg(reinterpret_cast<const uint32_t*>(P.em + e)); }
                mA[0] = w & 0x1e00u; mA[1] = (w >> 16) & 0x1e00u;
            }
#pragma unroll
            for (int k = 0; k < MIDG_R; ++k) {
                if (!MASK) { q[k] = make_uint4(0u, 0u, 0u, 0u); if (jC0 < jC1) q[k] = __ldg(eq + e + k); }
                const uint32_t a4 = xC[k] & 0x1fcu;
                row[k] = (macc_s + (a4 << 7)) | (a4 & 0x7cu);              // row base | (a & 31) << 2
            }
            load_pos(c + NWARP, xB, jB0, jB1);
            // 4 J positions per iteration (two independent pairs of loads in flight)
            if (MASK) {
                for (uint32_t l = jC0; __any_sync(0xffffffffu, l < jC1); l += 4) {
                    const bool p0 = l < jC1, p1 = l + 2u < jC1;
                    uint32_t w0 = 0u, w1 = 0u;
                    if (p0) w0 = __ldg(reinterpret_cast<const uint32_t*>(P.em + l));
                    if (p1) w1 = __ldg(reinterpret_cast<const uint32_t*>(P.em + l + 2));
                    if (p0) {
#pragma unroll
                        for (int k = 0; k < MIDG_R; ++k) {
                            mid_red(row[k] ^ (w0 & 0x1fcu), midg_sel(mA[k] & w0, q[0]));
                            mid_red(row[k] ^ ((w0 >> 16) & 0x1fcu), midg_sel(mA[k] & (w0 >> 16), q[0]));
                        }
                    }
                    if (p1) {
#pragma unroll
                        for (int k = 0; k < MIDG_R; ++k) {
                            mid_red(row[k] ^ (w1 & 0x1fcu), midg_sel(mA[k] & w1, q[0]));
                            mid_red(row[k] ^ ((w1 >> 16) & 0x1fcu), midg_sel(mA[k] & (w1 >> 16), q[0]));
                        }
                    }
                }
                continue;
            }
            for (uint32_t l = jC0; __any_sync(0xffffffffu, l < jC1); l += 4) {
                const bool p0 = l < jC1, p1 = l + 2u < jC1;
                uint2 xa, xb; uint4 b0, b1, b2, b3;
                if (p0) { xa = __ldg(reinterpret_cast<const uint2*>(ex + l)); b0 = __ldg(eq + l); b1 = __ldg(eq + l + 1); }
                if (p1) { xb = __ldg(reinterpret_cast<const uint2*>(ex + l + 2)); b2 = __ldg(eq + l + 2); b3 = __ldg(eq + l + 3); }
                if (p0) {
                    const uint32_t c0 = xa.x & 0x1fcu, c1 = xa.y & 0x1fcu;
#pragma unroll
                    for (int k = 0; k < MIDG_R; ++k) { mid_red(row[k] ^ c0, midg_dot(q[k], b0)); mid_red(row[k] ^ c1, midg_dot(q[k], b1)); }
                }
                if (p1) {
                    const uint32_t c0 = xb.x & 0x1fcu, c1 = xb.y & 0x1fcu;
#pragma unroll
                    for (int k = 0; k < MIDG_R; ++k) { mid_red(row[k] ^ c0, midg_dot(q[k], b2)); mid_red(row[k] ^ c1, midg_dot(q[k], b3)); }
                }
            }
        }
        __syncthreads();
        mid_epilogue<MIDG_THREADS>(macc, ij, N, P.out, P.inv_qscale);
        __syncthreads();
    }
}

}  // namespace ufb
