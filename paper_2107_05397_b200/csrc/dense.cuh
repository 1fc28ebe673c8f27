// dense.cuh -- step a-5 for the HEAD branches on the CUDA cores (weighted variant, fp64, or unweighted with
// NO_TENSOR) and step a-6 (finalize) as its epilogue.  BASELINE.json:5 subsystems (2)+(3): "the
// stripe-accumulation kernel that, for batches of branches staged in shared memory via TMA/cp.async, updates
// register-resident tiles of per-pair ... accumulators"; PAPER.md:23,29 ("Striped UniFrac", "a set of stripes").
//
// Head branches are dense (a branch is "head" only if a large fraction of the samples is present below it,
// DESIGN.md "head / mid / tail split"), so their embedding is a plain row-major matrix E[K_pad][N_pad] of
// pre-scaled values u~ (zeros where absent) and the kernel is a min-plus-like "GEMM":
//     M[i][j] = sum_k min(E[k][i], E[k][j])          (identities I3 / I5 of DESIGN.md)
// One persistent CTA = 8 consumer warps + 1 producer warp; a CTA owns one 128 x 128 tile pair (I <= J) at a
// time (static round-robin over a cache-blocked pair list).  The producer's elected lane stages BK rows of the
// two 128-sample column blocks per pipeline stage with two TMA 2D tile loads (cp.async.bulk.tensor, mbarrier
// complete_tx).  Consumer warp w owns the 32 x 64 sub-tile (quarter w/2 of I, half w%2 of J) as an 8 x 8 register
// tile per thread: per staged row 4 x LDS.128 and 64 x (FMNMX + FADD).  Every FLUSH_STAGES stages the fp32
// register accumulators are folded into per-thread fp64 partial sums (blocked summation, DESIGN.md "fp32
// accuracy").  Epilogue (a-6): M_total = M_head + (mid / tail sums already in out[]),
//     weighted   : d = (R_i + R_j - 2 M) / (R_i + R_j)         unweighted : d = (S_i + S_j - 2 G) / (S_i + S_j - G)
#pragma once
#include <cuda.h>
#include "common.cuh"
#include "stripe.cuh"   // mbarrier helpers, VecLd

namespace ufb {

template <typename T> struct DenseCfg;
template <> struct DenseCfg<float>  { static constexpr int BK = 32, STAGES = 4, FLUSH_STAGES = 16, LAST_EVERY_STAGE = 8; };
template <> struct DenseCfg<double> { static constexpr int BK = 16, STAGES = 4, FLUSH_STAGES = 1 << 30, LAST_EVERY_STAGE = 0; };

constexpr int DENSE_THREADS = 288;       // 8 consumer warps + 1 producer warp

template <typename T>
constexpr size_t dense_smem_bytes() {
    return (size_t)DenseCfg<T>::STAGES * DenseCfg<T>::BK * 2 * TILE * sizeof(T) + 128 /*align*/ + 2 * DenseCfg<T>::STAGES * 8;
}

struct DenseParams {
    const int2* pairs; uint32_t n_pairs;
    uint32_t K_pad;               // head rows padded to a multiple of BK (padding rows are zero)
    const double* sums;           // [n_tiles*128] R_s or S_s
    int n_samples;
    int weighted;
    void* out;                    // condensed, T
    int add_out;                  // out[] already holds the mid / tail branches' sum of min(u~_a, u~_b)
    double* scratch;              // [grid][64][256] fp64 partial sums
    GuardList guard;              // pairs with d < GUARD_THETA are listed for k_guard (guard.cuh)
    const double* hsum;           // k_dense16: [n_tiles*128] Rh_s = sum over the head rows of E_ks
};

// head rows in ascending n_v order: keys for the stable radix sort, then the reordered row list
__global__ void k_head_keys(uint32_t n_head, const int32_t* __restrict__ hrows, const uint32_t* __restrict__ nv, uint32_t* __restrict__ key)
{
    const uint32_t h = blockIdx.x * blockDim.x + threadIdx.x;
    if (h < n_head) key[h] = nv[hrows[h]];
}
__global__ void k_head_reorder(uint32_t n_head, const int32_t* __restrict__ hrows, const uint32_t* __restrict__ idx, int32_t* __restrict__ out)
{
    const uint32_t h = blockIdx.x * blockDim.x + threadIdx.x;
    if (h < n_head) out[h] = hrows[idx[h]];
}

// dense head embedding: E[h][s] for head row h (node hrows[h]); one warp per (row, tile), lane l owns samples 4l..4l+3
template <typename T>
__global__ void __launch_bounds__(256)
k_head_dense(uint32_t n_head, const int32_t* __restrict__ hrows, const double* __restrict__ len,
             const uint32_t* __restrict__ bits, uint32_t NW, int n_tiles, const uint32_t* __restrict__ tptr,
             const uint32_t* __restrict__ hpref, const T* __restrict__ tv /* weighted: values in rank layout; else NULL */,
             T* __restrict__ E, size_t Npad, double* __restrict__ hsum /* per-sample sum of the head rows' values, or NULL */)
{
    const long long gw = ((long long)blockIdx.x * blockDim.x + threadIdx.x) >> 5;
    const int lane = threadIdx.x & 31;
    const uint32_t h = (uint32_t)(gw / n_tiles);
    const int tile = (int)(gw - (long long)h * n_tiles);
    if (h >= n_head) return;
    const int v = hrows[h];
    const uint4 g = reinterpret_cast<const uint4*>(bits + (size_t)v * NW)[tile];
    const uint32_t gw4[4] = {g.x, g.y, g.z, g.w};
    const int wi = lane >> 3, sh = (lane & 7) * 4;
    const uint32_t mine = gw4[wi];
    const uint32_t m4 = (mine >> sh) & 15u;
    T x[4] = {(T)0, (T)0, (T)0, (T)0};
    if (tv) {
        uint32_t e = tptr[v] + hpref[(size_t)h * n_tiles + tile] + __popc(mine & ((1u << sh) - 1u));
        if (wi > 0) e += __popc(gw4[0]);
        if (wi > 1) e += __popc(gw4[1]);
        if (wi > 2) e += __popc(gw4[2]);
#pragma unroll
        for (int j = 0; j < 4; ++j) if (m4 & (1u << j)) x[j] = tv[e++];
    } else {
        const T l = (T)len[v];
#pragma unroll
        for (int j = 0; j < 4; ++j) if (m4 & (1u << j)) x[j] = l;
    }
    if (hsum) {
#pragma unroll
        for (int j = 0; j < 4; ++j) if (m4 & (1u << j)) atomicAdd(&hsum[(size_t)tile * TILE + lane * 4 + j], (double)x[j]);
    }
    Vec4<T>::store(E + (size_t)h * Npad + (size_t)tile * TILE + lane * 4, x[0], x[1], x[2], x[3]);
}

__device__ __forceinline__ void tma_load_2d_box(uint32_t dst, const CUtensorMap* tm, int c0, int c1, uint32_t bar) {
    asm volatile("cp.async.bulk.tensor.2d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3}], [%4];"
                 ::"r"(dst), "l"(tm), "r"(c0), "r"(c1), "r"(bar) : "memory");
}

template <typename T>
__global__ void __launch_bounds__(DENSE_THREADS, 1)
k_dense(const __grid_constant__ CUtensorMap tmE, const DenseParams P)
{
    using Cfg = DenseCfg<T>;
    constexpr int BK = Cfg::BK, STAGES = Cfg::STAGES;
    constexpr int VEC = VecLd<T>::VEC, NV = 8 / VEC;
    constexpr uint32_t BOX_BYTES = BK * TILE * sizeof(T);

    extern __shared__ unsigned char dsm_raw[];
    const uint32_t raw = smem_u32(dsm_raw);
    const uint32_t base = (raw + 127u) & ~127u;
    T* ring = reinterpret_cast<T*>(dsm_raw + (base - raw));
    const uint32_t bar0 = base + STAGES * 2 * BOX_BYTES;
    auto full = [&](uint32_t s) { return bar0 + 8u * s; };
    auto empty = [&](uint32_t s) { return bar0 + 8u * (STAGES + s); };

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    if (threadIdx.x == 0) {
        for (int s = 0; s < STAGES; ++s) { mbar_init(full(s), 1); mbar_init(empty(s), 8); }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();
    const uint32_t n_k = P.K_pad / BK;

    if (warp == 8) {
        // =========================================================== producer
        if (lane == 0) {
            uint32_t stage = 0, phase = 0;
            for (uint32_t pi = blockIdx.x; pi < P.n_pairs; pi += gridDim.x) {
                const int2 ij = P.pairs[pi];
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

    // =============================================================== consumer warps
    const int wi = warp >> 1, wj = warp & 1;
    const int ty = lane >> 3, tx = lane & 7;
    // element a of the i side: local index  (a/VEC)*(4*VEC) + ty*VEC + a%VEC   within the warp's 32 rows
    // element b of the j side: local index  (b/VEC)*(8*VEC) + tx*VEC + b%VEC   within the warp's 64 columns
    const int i_off = wi * 32 + ty * VEC;
    const int j_off = BK * TILE + wj * 64 + tx * VEC;
    double* my_scratch = P.scratch + (size_t)blockIdx.x * 64 * 256 + threadIdx.x;

    T acc[8][8];
#pragma unroll
    for (int a = 0; a < 8; ++a)
#pragma unroll
        for (int b = 0; b < 8; ++b) acc[a][b] = (T)0;
    uint32_t stage = 0, phase = 0;

    for (uint32_t pi = blockIdx.x; pi < P.n_pairs; pi += gridDim.x) {
        int since_flush = 0;
        bool scratch_live = false;
        for (uint32_t kb = 0; kb < n_k; ++kb) {
            mbar_wait(full(stage), phase);
            const T* sb = ring + (size_t)stage * 2 * BK * TILE;
#pragma unroll 4
            for (int r = 0; r < BK; ++r) {
                const T* row = sb + r * TILE;
                T ai[8], bj[8];
#pragma unroll
                for (int k = 0; k < NV; ++k) {
                    VecLd<T>::ld(row + i_off + k * 4 * VEC, ai + k * VEC);
                    VecLd<T>::ld(row + j_off + k * 8 * VEC, bj + k * VEC);
                }
#pragma unroll
                for (int a = 0; a < 8; ++a)
#pragma unroll
                    for (int b = 0; b < 8; ++b) acc[a][b] += fmin(ai[a], bj[b]);
            }
            __syncwarp();
            if (lane == 0) mbar_arrive(empty(stage));
            if (++stage == STAGES) { stage = 0; phase ^= 1u; }
            // the last LAST_EVERY_STAGE stages hold the branches with the largest n_v (rows are in ascending n_v order):
            // their values are orders of magnitude above the rest and are folded after every stage
            if ((++since_flush >= Cfg::FLUSH_STAGES || kb + Cfg::LAST_EVERY_STAGE + 1 >= n_k) && kb + 1 < n_k) {
                // blocked summation: fold the fp32 partial sums into fp64 (per-thread slots, L2-resident)
#pragma unroll
                for (int a = 0; a < 8; ++a)
#pragma unroll
                    for (int b = 0; b < 8; ++b) {
                        double* s = my_scratch + (size_t)(a * 8 + b) * 256;
                        double v = (double)acc[a][b];
                        if (scratch_live) v += *s;
                        *s = v;
                        acc[a][b] = (T)0;
                    }
                scratch_live = true;
                since_flush = 0;
            }
        }
        // ----------------------------------------------------------- a-6 finalize (epilogue of the tile pair)
        const int2 ij = P.pairs[pi];
        const long long N = P.n_samples;
        double sj[8];
#pragma unroll
        for (int b = 0; b < 8; ++b) {
            int gj = ij.y * TILE + wj * 64 + (b / VEC) * (8 * VEC) + tx * VEC + (b % VEC);
            sj[b] = P.sums[gj];
        }
#pragma unroll
        for (int a = 0; a < 8; ++a) {
            const long long gi = (long long)ij.x * TILE + wi * 32 + (a / VEC) * (4 * VEC) + ty * VEC + (a % VEC);
            const double si = P.sums[gi];
            const long long rowbase = gi * (2 * N - gi - 1) / 2 - gi - 1;     // + gj gives the condensed index
#pragma unroll
            for (int b = 0; b < 8; ++b) {
                double tot = (double)acc[a][b];
                if (scratch_live) tot += my_scratch[(size_t)(a * 8 + b) * 256];
                acc[a][b] = (T)0;
                const long long gj = (long long)ij.y * TILE + wj * 64 + (b / VEC) * (8 * VEC) + tx * VEC + (b % VEC);
                if (gi < gj && gj < N) {
                    const double ss = si + sj[b];
                    if (P.add_out) tot += (double)reinterpret_cast<const T*>(P.out)[rowbase + gj];
                    double num = ss - 2.0 * tot;
                    const double den = P.weighted ? ss : ss - tot;
                    if (num < 0.0) num = 0.0;
                    guard_note(P.guard, num, den, (uint32_t)gi, (uint32_t)gj);
                    reinterpret_cast<T*>(P.out)[rowbase + gj] = (T)(den > 0.0 ? num / den : 0.0);
                }
            }
        }
    }
}

// ------------------------------------------------------------------ fp32 variant with 16 consumer warps, mixed forms
// Same pipeline as k_dense<float>, but the 128 x 128 tile pair is owned by 16 consumer warps (4 x 4 grid of 32 x 32
// sub-tiles, an 8 x 4 register tile per thread: 3 LDS.128 per 32 updates) so that every scheduler has four warps to pick
// from, and the two FP32 pipes are balanced (SURVEY 8a-5 table, rows "fp32 direct with FADD2" / "fp32 min-form"):
//   24 of a thread's 32 cells ("min cells"):    acc += min(E_ki, E_kj)              FMNMX on the half-rate ALU pipe, the adds
//                                               packed two per instruction (add.f32x2 -> FADD2, FMA pipe)
//   8 cells, a >= 4 and b >= 2 ("direct cells"): acc += -0.5 * |E_ki - E_kj|         FADD + FFMA, both on the FMA pipe
//   min(p, q) = (p + q) / 2 - |p - q| / 2, so with Rh_s = sum over the head rows of E_ks (fp64, k_head_dense) a direct cell
//   holds M_ij - (Rh_i + Rh_j) / 2 and the epilogue adds that half-sum back.
// A pure min-form row costs 32 ALU-pipe slots per 32 updates (that pipe's limit, 64 lanes/clk/SM); mixed, the ALU pipe
// carries 0.75 and the FMA pipe 1.25 lane-passes per update, interleaved instruction by instruction, and the kernel is
// bound by issue at 1.7 instructions per update instead of 2.1.
constexpr int DENSE16_THREADS = 544;     // 16 consumer warps + 1 producer warp
__device__ __forceinline__ constexpr bool dense16_direct_cell(int a, int b) { return a >= 4 && b >= 2; }

__device__ __forceinline__ void add2(float& x0, float& x1, float m0, float m1) {
    asm("{\n\t.reg .b64 p, q;\n\tmov.b64 p, {%0, %1};\n\tmov.b64 q, {%2, %3};\n\tadd.rn.f32x2 p, p, q;\n\tmov.b64 {%0, %1}, p;\n\t}"
        : "+f"(x0), "+f"(x1) : "f"(m0), "f"(m1));
}

__global__ void __launch_bounds__(DENSE16_THREADS, 1)
k_dense16(const __grid_constant__ CUtensorMap tmE, const DenseParams P)
{
    using T = float;
    using Cfg = DenseCfg<float>;
    constexpr int BK = Cfg::BK, STAGES = Cfg::STAGES;
    constexpr uint32_t BOX_BYTES = BK * TILE * sizeof(T);

    extern __shared__ unsigned char dsm_raw[];
    const uint32_t raw = smem_u32(dsm_raw);
    const uint32_t base = (raw + 127u) & ~127u;
    T* ring = reinterpret_cast<T*>(dsm_raw + (base - raw));
    const uint32_t bar0 = base + STAGES * 2 * BOX_BYTES;
    auto full = [&](uint32_t s) { return bar0 + 8u * s; };
    auto empty = [&](uint32_t s) { return bar0 + 8u * (STAGES + s); };

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    if (threadIdx.x == 0) {
        for (int s = 0; s < STAGES; ++s) { mbar_init(full(s), 1); mbar_init(empty(s), 16); }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();
    const uint32_t n_k = P.K_pad / BK;

    if (warp == 16) {
        if (lane == 0) {
            uint32_t stage = 0, phase = 0;
            for (uint32_t pi = blockIdx.x; pi < P.n_pairs; pi += gridDim.x) {
                const int2 ij = P.pairs[pi];
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

    const int wi = warp >> 2, wj = warp & 3;
    const int ty = lane >> 3, tx = lane & 7;
    // i side: element a at local row (a/4)*16 + ty*4 + a%4 of the warp's 32 rows; j side: element b at column tx*4 + b of its 32
    const int i_off = wi * 32 + ty * 4;
    const int j_off = BK * TILE + wj * 32 + tx * 4;
    double* my_scratch = P.scratch + (size_t)blockIdx.x * 64 * 256 + threadIdx.x;      // [32][512] per CTA

    float acc[8][4];
#pragma unroll
    for (int a = 0; a < 8; ++a)
#pragma unroll
        for (int b = 0; b < 4; ++b) acc[a][b] = 0.f;
    uint32_t stage = 0, phase = 0;

    for (uint32_t pi = blockIdx.x; pi < P.n_pairs; pi += gridDim.x) {
        int since_flush = 0;
        bool scratch_live = false;
        for (uint32_t kb = 0; kb < n_k; ++kb) {
            mbar_wait(full(stage), phase);
            const float* sb = ring + (size_t)stage * 2 * BK * TILE;
#pragma unroll 4
            for (int r = 0; r < BK; ++r) {
                const float* row = sb + r * TILE;
                float ai[8], bj[4];
                VecLd<float>::ld(row + i_off, ai);
                VecLd<float>::ld(row + i_off + 16, ai + 4);
                VecLd<float>::ld(row + j_off, bj);
#pragma unroll
                for (int a = 0; a < 8; ++a) {
                    add2(acc[a][0], acc[a][1], fminf(ai[a], bj[0]), fminf(ai[a], bj[1]));
                    if (!dense16_direct_cell(a, 2)) {
                        add2(acc[a][2], acc[a][3], fminf(ai[a], bj[2]), fminf(ai[a], bj[3]));
                    } else {
                        acc[a][2] = fmaf(fabsf(ai[a] - bj[2]), -0.5f, acc[a][2]);
                        acc[a][3] = fmaf(fabsf(ai[a] - bj[3]), -0.5f, acc[a][3]);
                    }
                }
            }
            __syncwarp();
            if (lane == 0) mbar_arrive(empty(stage));
            if (++stage == STAGES) { stage = 0; phase ^= 1u; }
            if ((++since_flush >= Cfg::FLUSH_STAGES || kb + Cfg::LAST_EVERY_STAGE + 1 >= n_k) && kb + 1 < n_k) {
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
        const int2 ij = P.pairs[pi];
        const long long N = P.n_samples;
        double sj[4], hj[4];
#pragma unroll
        for (int b = 0; b < 4; ++b) { sj[b] = P.sums[ij.y * TILE + wj * 32 + tx * 4 + b]; hj[b] = P.hsum[ij.y * TILE + wj * 32 + tx * 4 + b]; }
#pragma unroll
        for (int a = 0; a < 8; ++a) {
            const long long gi = (long long)ij.x * TILE + wi * 32 + (a / 4) * 16 + ty * 4 + (a % 4);
            const double si = P.sums[gi], hi = P.hsum[gi];
            const long long rowbase = gi * (2 * N - gi - 1) / 2 - gi - 1;
#pragma unroll
            for (int b = 0; b < 4; ++b) {
                double tot = (double)acc[a][b];
                if (dense16_direct_cell(a, b)) tot += 0.5 * (hi + hj[b]);
                if (scratch_live) tot += my_scratch[(size_t)(a * 4 + b) * 512];
                acc[a][b] = 0.f;
                const long long gj = (long long)ij.y * TILE + wj * 32 + tx * 4 + b;
                if (gi < gj && gj < N) {
                    const double ss = si + sj[b];
                    if (P.add_out) tot += (double)reinterpret_cast<const float*>(P.out)[rowbase + gj];
                    double num = ss - 2.0 * tot;
                    const double den = P.weighted ? ss : ss - tot;
                    if (num < 0.0) num = 0.0;
                    guard_note(P.guard, num, den, (uint32_t)gi, (uint32_t)gj);
                    reinterpret_cast<float*>(P.out)[rowbase + gj] = (float)(den > 0.0 ? num / den : 0.0);
                }
            }
        }
    }
}

}  // namespace ufb
