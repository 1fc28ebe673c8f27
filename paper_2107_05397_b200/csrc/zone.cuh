// zone.cuh -- step a-5 / a-6 for the weighted fp32 variant: a per-(branch, tile) split between the dense register-tile
// kernel and the shared-memory join ("sparse-aware optimizations", mechanism ours).
// The samples are in ascending richness order (perm.cuh), so a branch v is sparse in the leading (poor) 128-sample tiles and
// dense in the trailing (rich) ones.  Every non-tail branch gets a tile index D_v, its DENSE ZONE being the tiles >= D_v:
//     tile pair (I <= J) with I >= D_v (both tiles in the zone)  ->  k_zone : min-"GEMM" row of the 128 x 128 register tiles
//     every other tile pair                                      ->  k_mid  : join of the two sparse lists (~ n_vI * n_vJ / r_join)
// D_v minimises the modelled cost of the branch over all its tile pairs (k_row_cut).  Rows are ordered by (D_v ascending,
// n_v descending); cut[I] = #{rows with D_v <= I}, rounded down to whole 32-row stages, is the only thing the two kernels
// share: k_zone runs rows [0, cut[I]) of pair (I, J), k_mid rows [cut[I], n_list).  Any non-decreasing cut table gives a
// correct result; the model only decides how fast it is.
// (A variant that also skipped the absent samples of the poorer tile inside the register-tile kernel -- warp-uniform ballots,
//  one branch per sample -- was built and measured in this round: branch latency with 4 warps per scheduler made it slower
//  than both alternatives at every density.)
#pragma once
#include <cuda.h>
#include "common.cuh"
#include "tail.cuh"
#include "stripe.cuh"
#include "dense.cuh"

namespace ufb {

// list rows = every branch that is not left to the tail scatter
__global__ void k_list_compact(int n, const uint8_t* __restrict__ cls, int32_t* __restrict__ lnode, unsigned int* __restrict__ counter)
{
    const int v = blockIdx.x * blockDim.x + threadIdx.x;
    if (v < n && (cls[v] == CLS_HEAD || cls[v] == CLS_MID)) lnode[atomicAdd(counter, 1u)] = v;
}

struct CutModel { float c0, inv2rj, c_ent; };      // SM-clocks per (row, tile pair) of k_zone, 1 / (2 r_join), per (entry, tile pair) visit of the join

// One warp per list row: per-tile sample counts from the presence bits, then D_v = argmin over D of
//   c0 z (z + 1) / 2  +  (tot^2 - sfx(D)^2) inv2rj  +  c_ent pfx(D) (T - D / 2),
// z = T - D tiles in the zone, sfx(D) / pfx(D) = samples of the row inside / before the zone.
// key = (D_v << 48) | ((N - n_v) << 24) | (v & 0xffffff): ascending sort = rows by (D_v ascending, n_v descending)
constexpr int ROWCUT_WARPS = 8;
constexpr int ROWCUT_MAX_TILES = 1024;
__global__ void __launch_bounds__(ROWCUT_WARPS * 32)
k_row_cut(uint32_t n_list, const int32_t* __restrict__ lnode, const uint32_t* __restrict__ bits, uint32_t NW, int n_tiles,
          uint32_t N, CutModel M, unsigned long long* __restrict__ keys)
{
    __shared__ float pf[ROWCUT_WARPS][ROWCUT_MAX_TILES + 1];
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const uint32_t i = blockIdx.x * ROWCUT_WARPS + warp;
    if (i >= n_list) return;
    const int v = lnode[i];
    const uint4* row = reinterpret_cast<const uint4*>(bits + (size_t)v * NW);
    for (int t = lane; t < n_tiles; t += 32) {
        const uint4 g = row[t];
        pf[warp][t + 1] = (float)(__popc(g.x) + __popc(g.y) + __popc(g.z) + __popc(g.w));
    }
    __syncwarp();
    if (lane == 0) {
        float run = 0.f;
        pf[warp][0] = 0.f;
        for (int t = 1; t <= n_tiles; ++t) { run += pf[warp][t]; pf[warp][t] = run; }
        const float tot = pf[warp][n_tiles];
        // D = n_tiles: everything joined; every step down adds tile D to the dense zone
        float best = tot * tot * M.inv2rj + M.c_ent * tot * 0.5f * (float)n_tiles;
        int bestD = n_tiles;
        for (int D = n_tiles - 1; D >= 0; --D) {
            const float z = (float)(n_tiles - D);                            // tiles in the dense zone
            const float sfx = tot - pf[warp][D];                             // samples of the row in the zone
            const float dense = M.c0 * 0.5f * z * (z + 1.f);
            const float join = (tot * tot - sfx * sfx) * M.inv2rj + M.c_ent * pf[warp][D] * ((float)n_tiles - 0.5f * (float)D);
            const float c = dense + join;
            if (c < best) { best = c; bestD = D; }
        }
        const unsigned long long nvv = (unsigned long long)pf[warp][n_tiles];
        keys[i] = ((unsigned long long)bestD << 48) | (((unsigned long long)N - nvv) << 24) | ((unsigned long long)v & 0xffffffull);
    }
}

// sorted order -> mrows[r] (node), Dr[r], list offsets of the row
__global__ void k_rows_from_sort(uint32_t n_list, const uint32_t* __restrict__ idx, const unsigned long long* __restrict__ keys_sorted,
                                 const int32_t* __restrict__ lnode, const uint32_t* __restrict__ tptr, const uint32_t* __restrict__ nv,
                                 int32_t* __restrict__ mrows, uint32_t* __restrict__ Dr, uint32_t* __restrict__ mbase, uint32_t* __restrict__ mlen)
{
    const uint32_t r = blockIdx.x * blockDim.x + threadIdx.x;
    if (r >= n_list) return;
    const int v = lnode[idx[r]];
    mrows[r] = v;
    Dr[r] = (uint32_t)(keys_sorted[r] >> 48);
    mbase[r] = tptr[v];
    mlen[r] = nv[v];
}

// cut[I] = #{r : Dr[r] <= I} rounded down to a multiple of `gran` (Dr ascending); cut[n_tiles] = n_list (sentinel, unrounded)
__global__ void k_cut_table(int n_tiles, uint32_t n_list, const uint32_t* __restrict__ Dr, uint32_t gran, uint32_t* __restrict__ cut)
{
    const int J = blockIdx.x * blockDim.x + threadIdx.x;
    if (J > n_tiles) return;
    if (J == n_tiles) { cut[J] = n_list; return; }
    uint32_t lo = 0, hi = n_list;                       // first r with Dr[r] > J
    while (lo < hi) { const uint32_t mid = (lo + hi) >> 1; if (Dr[mid] <= (uint32_t)J) lo = mid + 1; else hi = mid; }
    cut[J] = lo / gran * gran;
}

// exact work counters of the split the cut table defines: counters[0] += joined pair updates, [1] += (row, tile pair) visits
// of k_zone.  One warp per list row.  A pair (I <= J) is dense iff r < cut[I]; cut is non-decreasing, so the row's zone is a
// suffix of the tiles.
__global__ void __launch_bounds__(256)
k_cut_stats(uint32_t n_list, const int32_t* __restrict__ mrows, const uint32_t* __restrict__ bits, uint32_t NW, int n_tiles,
            const uint32_t* __restrict__ cut, unsigned long long* __restrict__ counters)
{
    const uint32_t r = (blockIdx.x * blockDim.x + threadIdx.x) >> 5;
    const int lane = threadIdx.x & 31;
    if (r >= n_list) return;
    const uint4* row = reinterpret_cast<const uint4*>(bits + (size_t)mrows[r] * NW);
    unsigned long long tot = 0, zone = 0, ztiles = 0;
    for (int t = lane; t < n_tiles; t += 32) {
        const uint4 g = row[t];
        const unsigned long long c = (unsigned long long)(__popc(g.x) + __popc(g.y) + __popc(g.z) + __popc(g.w));
        tot += c;
        if (r < cut[t]) { zone += c; ++ztiles; }
    }
    for (int o = 16; o; o >>= 1) {
        tot += __shfl_xor_sync(0xffffffffu, tot, o); zone += __shfl_xor_sync(0xffffffffu, zone, o);
        ztiles += __shfl_xor_sync(0xffffffffu, ztiles, o);
    }
    if (lane == 0) {
        const unsigned long long c2t = tot ? tot * (tot - 1) / 2 : 0, c2z = zone ? zone * (zone - 1) / 2 : 0;
        atomicAdd(&counters[0], c2t - c2z);
        atomicAdd(&counters[1], ztiles * (ztiles + 1) / 2);
    }
}

// dense rows of the first K_E list rows: E[r][position] = u~ (E zeroed by the caller).  One warp per row.
__global__ void __launch_bounds__(256)
k_E_scatter(uint32_t K_E, const uint32_t* __restrict__ mbase, const uint32_t* __restrict__ mlen, const uint32_t* __restrict__ ts,
            const float* __restrict__ tv, float* __restrict__ E, size_t Npad)
{
    const uint32_t r = (blockIdx.x * blockDim.x + threadIdx.x) >> 5;
    const int lane = threadIdx.x & 31;
    if (r >= K_E) return;
    const uint32_t base = mbase[r], m = mlen[r];
    float* dst = E + (size_t)r * Npad;
    for (uint32_t k = lane; k < m; k += 32) dst[ts[base + k]] = tv[base + k];
}


// H[I][s] = sum over the rows r < cut[I] of E[r][s] (fp64): the half-sum k_zone's "direct" cells need back (see k_zone).
// One thread per sample column walks the rows in groups of 32 (cut[] are multiples of 32, non-decreasing in I).
__global__ void __launch_bounds__(128)
k_zone_hsum(const float* __restrict__ E, size_t Npad, int n_tiles, const uint32_t* __restrict__ cut, double* __restrict__ H)
{
    const size_t s = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (s >= Npad) return;
    double run = 0.0;
    uint32_t r = 0;
    for (int I = 0; I < n_tiles; ++I) {
        const uint32_t c = cut[I];
        for (; r < c; r += 32) {
            float v[32];
#pragma unroll
            for (int j = 0; j < 32; ++j) v[j] = E[(size_t)(r + j) * Npad + s];
            double g = 0.0;
#pragma unroll
            for (int j = 0; j < 32; ++j) g += (double)v[j];
            run += g;
        }
        H[(size_t)I * Npad + s] = run;
    }
}

// ------------------------------------------------------------------ k_zone
// Same TMA / mbarrier pipeline as k_dense16 (dense.cuh): one persistent CTA per SM, 16 consumer warps + 1 producer warp,
// BK = 32 rows of the two 128-sample column blocks per stage; the number of stages is per tile pair: cut[I] / 32.
// Consumer warp w owns the 8 samples 8w .. 8w+7 of tile I (rows of the output tile; two broadcast LDS.128 per staged row)
// against all 128 samples of tile J: lane l holds columns 4l .. 4l+3 (one LDS.128), acc[8][4]: 24 FMNMX (ALU pipe) + 12
// packed adds (add.f32x2 -> FADD2) + 8 FADD + 8 FFMA (direct cells) per staged row and warp; the epilogue writes 512
// contiguous bytes per row.
// The tile pairs of a CTA are a host-balanced list (least-loaded CTA first over cut[I] stages), cta_off[b] .. cta_off[b+1].
constexpr int ZONE_THREADS = 544;
constexpr int ZONE_BK = 32, ZONE_STAGES = 4, ZONE_FLUSH = 16, ZONE_FIRST_EVERY = 8;
constexpr size_t ZONE_SMEM = (size_t)ZONE_STAGES * ZONE_BK * 2 * TILE * sizeof(float) + 128 + 2 * ZONE_STAGES * 8;

struct ZoneParams {
    const int2* pairs; const uint32_t* cta_off;
    const uint32_t* cut;          // [n_tiles + 1] rows of pair (I, J) handled here: [0, cut[I]), multiples of ZONE_BK
    const double* sums;           // [n_tiles*128] R_s
    int n_samples;
    float* out;                   // condensed (position space); holds the join / tail sums when add_out
    int add_out;
    double* scratch;              // [grid][32][512] fp64 partial sums
    const double* H;              // [n_tiles][Npad] H[I][s] = sum_{r < cut[I]} E[r][s] (k_zone_hsum)
    size_t Npad;
    GuardList guard;
};

// the warp's samples 6 and 7 ("direct" cells, 8 of a thread's 32): acc += -1/2 |a - b|  (FADD + FFMA, both on the FMA pipe);
// min(p, q) = (p + q) / 2 - |p - q| / 2, so the epilogue adds (H[I][i] + H[I][j]) / 2 back.  The other 24 cells take FMNMX on
// the half-rate ALU pipe + packed adds: the same pipe balance as k_dense16 (dense.cuh).
__device__ __forceinline__ void zone_row4_direct(float (&acc)[4], float a, const float4& b) {
    acc[0] = fmaf(fabsf(a - b.x), -0.5f, acc[0]); acc[1] = fmaf(fabsf(a - b.y), -0.5f, acc[1]);
    acc[2] = fmaf(fabsf(a - b.z), -0.5f, acc[2]); acc[3] = fmaf(fabsf(a - b.w), -0.5f, acc[3]);
}
__device__ __forceinline__ constexpr bool zone_direct_row(int a) { return a >= 6; }

__device__ __forceinline__ void zone_row4(float (&acc)[4], float a, const float4& b) {
    add2(acc[0], acc[1], fminf(a, b.x), fminf(a, b.y));
    add2(acc[2], acc[3], fminf(a, b.z), fminf(a, b.w));
}

__global__ void __launch_bounds__(ZONE_THREADS, 1)
k_zone(const __grid_constant__ CUtensorMap tmE, const ZoneParams P)
{
    constexpr int BK = ZONE_BK, STAGES = ZONE_STAGES;
    constexpr uint32_t BOX_BYTES = BK * TILE * sizeof(float);
    extern __shared__ unsigned char zsm_raw[];
    const uint32_t raw = smem_u32(zsm_raw);
    const uint32_t base = (raw + 127u) & ~127u;
    float* ring = reinterpret_cast<float*>(zsm_raw + (base - raw));
    const uint32_t bar0 = base + STAGES * 2 * BOX_BYTES;
    auto full = [&](uint32_t s) { return bar0 + 8u * s; };
    auto empty = [&](uint32_t s) { return bar0 + 8u * (STAGES + s); };
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    if (threadIdx.x == 0) {
        for (int s = 0; s < STAGES; ++s) { mbar_init(full(s), 1); mbar_init(empty(s), 16); }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();
    const uint32_t p0 = P.cta_off[blockIdx.x], p1 = P.cta_off[blockIdx.x + 1];

    if (warp == 16) {
        if (lane == 0) {
            uint32_t stage = 0, phase = 0;
            for (uint32_t pi = p0; pi < p1; ++pi) {
                const int2 ij = P.pairs[pi];
                const uint32_t n_k = P.cut[ij.x] / BK;
                for (uint32_t kb = 0; kb < n_k; ++kb) {
                    mbar_wait(empty(stage), phase ^ 1u);
                    const uint32_t dst = base + stage * 2 * BOX_BYTES;
                    mbar_arrive_expect_tx(full(stage), 2 * BOX_BYTES);
                    tma_load_2d_box(dst, &tmE, ij.x * TILE, (int)(kb * BK), full(stage));
                    tma_load_2d_box(dst + BOX_BYTES, &tmE, ij.y * TILE, (int)(kb * BK), full(stage));
                    if (++stage == STAGES) { stage = 0; phase ^= 1u; }
                }
            }
        }
        return;
    }

    const int i_off = warp * 8;                       // the warp's 8 rows (samples of tile I)
    const int j_off = BK * TILE + lane * 4;           // the lane's 4 columns (samples of tile J)
    double* my_scratch = P.scratch + (size_t)blockIdx.x * 32 * 512 + threadIdx.x;
    float acc[8][4];
#pragma unroll
    for (int a = 0; a < 8; ++a)
#pragma unroll
        for (int b = 0; b < 4; ++b) acc[a][b] = 0.f;
    uint32_t stage = 0, phase = 0;

    for (uint32_t pi = p0; pi < p1; ++pi) {
        const int2 ij = P.pairs[pi];
        const uint32_t n_k = P.cut[ij.x] / BK;
        int since_flush = 0;
        bool scratch_live = false;
        for (uint32_t kb = 0; kb < n_k; ++kb) {
            mbar_wait(full(stage), phase);
            const float* sb = ring + (size_t)stage * 2 * BK * TILE;
#pragma unroll 4
            for (int r = 0; r < BK; ++r) {
                const float* row = sb + r * TILE;
                const float4 a0 = *reinterpret_cast<const float4*>(row + i_off);
                const float4 a1 = *reinterpret_cast<const float4*>(row + i_off + 4);
                const float4 b = *reinterpret_cast<const float4*>(row + j_off);
                zone_row4(acc[0], a0.x, b); zone_row4(acc[1], a0.y, b); zone_row4(acc[2], a0.z, b); zone_row4(acc[3], a0.w, b);
                zone_row4(acc[4], a1.x, b); zone_row4(acc[5], a1.y, b); zone_row4_direct(acc[6], a1.z, b); zone_row4_direct(acc[7], a1.w, b);
            }
            __syncwarp();
            if (lane == 0) mbar_arrive(empty(stage));
            if (++stage == STAGES) { stage = 0; phase ^= 1u; }
            // rows come in descending n_v order inside a zone class: the first stages hold the branches whose values are orders of
            // magnitude above the rest and are folded into fp64 after every stage; afterwards every ZONE_FLUSH stages
            if ((++since_flush >= ZONE_FLUSH || kb < ZONE_FIRST_EVERY) && kb + 1 < n_k) {
#pragma unroll
                for (int a = 0; a < 8; ++a)
#pragma unroll
                    for (int b = 0; b < 4; ++b) {
                        double* s = my_scratch + (size_t)(a * 4 + b) * 512;
                        double v = (double)acc[a][b];
                        if (scratch_live) v += *s;
                        *s = v;
                        acc[a][b] = 0.f;
                    }
                scratch_live = true;
                since_flush = 0;
            }
        }
        // ----------------------------------------------------------- a-6 finalize (epilogue of the tile pair)
        const long long N = P.n_samples;
        double sj[4], hj[4];
        const double* Hrow = P.H + (size_t)ij.x * P.Npad;            // sums over the rows [0, cut[I]) this pair ran
#pragma unroll
        for (int b = 0; b < 4; ++b) { sj[b] = P.sums[ij.y * TILE + lane * 4 + b]; hj[b] = Hrow[ij.y * TILE + lane * 4 + b]; }
#pragma unroll
        for (int a = 0; a < 8; ++a) {
            const long long gi = (long long)ij.x * TILE + i_off + a;
            const double si = P.sums[gi];
            const double hi = zone_direct_row(a) ? Hrow[gi] : 0.0;
            const long long rowbase = gi * (2 * N - gi - 1) / 2 - gi - 1;
#pragma unroll
            for (int b = 0; b < 4; ++b) {
                double tot = (double)acc[a][b];
                if (zone_direct_row(a)) tot += 0.5 * (hi + hj[b]);
                if (scratch_live) tot += my_scratch[(size_t)(a * 4 + b) * 512];
                acc[a][b] = 0.f;
                const long long gj = (long long)ij.y * TILE + lane * 4 + b;
                if (gi < gj && gj < N) {
                    const double ss = si + sj[b];
                    if (P.add_out) tot += (double)P.out[rowbase + gj];
                    double num = ss - 2.0 * tot;
                    if (num < 0.0) num = 0.0;
                    guard_note(P.guard, num, ss, (uint32_t)gi, (uint32_t)gj);
                    P.out[rowbase + gj] = (float)(ss > 0.0 ? num / ss : 0.0);
                }
            }
        }
    }
}

}  // namespace ufb
