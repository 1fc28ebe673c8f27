// gram.cuh -- step a-5 for the HEAD branches of the UNWEIGHTED variant on the 5th-generation tensor
// cores (BASELINE.json:5: "Tensor cores are used only if the unweighted Gram-matrix reformulation
// (X^T diag(len) Y) meets the stated tolerance"; identity I5 of DESIGN.md).
//
//   G_ab = sum_{v in head} L_v x_av x_bv ,   L_v = m_v * 2^s_v ~ len_v * 2^q,  m_v < 2^24 = sum_d 256^d * digit_d(v),
//   s_v <= 7 (a per-row shift carried by the A operand: 24 significant bits for every head branch within a factor
//   2^7 of the longest one, fewer below that; the exact error sum is tracked per sample, see k_quant_ratio)
//   => G = sum_d 256^d * ( (2^s X)^T . (diag(digit_d) X) ) : three u8 x u8 -> s32 GEMMs, EXACT integer
//   accumulation in TMEM (128 * 255 * K < 2^31), recombined in int64, scaled by 2^-q in fp64.
//   d_U = (S_a + S_b - 2 G_tot) / (S_a + S_b - G_tot),  G_tot = G + (tail branches' sum, already in out[]).
//
// Operands in HBM (built from the bit-packed presence matrix by k_gram_expand), row-major
// [K_pad][N_pad] u8:  XA = x * 2^s,  XB_d = digit_d * x.  One CTA = one 128 x 128 tile pair at a time
// (static round-robin over a cache-blocked pair list); warp 0 lane 0 issues TMA 2D tile loads
// (128B swizzle) into a 6-stage ring, warp 1 lane 0 issues tcgen05.mma kind::i8 (M=128; N=256 for
// digits 0|1, N=128 for digit 2; both operands MN-major), warps 4..7 read the accumulators with
// tcgen05.ld and run the finalize step (a-6) for their 32 rows.
#pragma once
#include <cuda.h>
#include "common.cuh"
#include "stripe.cuh"   // mbarrier helpers

namespace ufb {

constexpr int GRAM_BK = 64;              // K rows per pipeline stage
constexpr int GRAM_STAGES = 6;
constexpr int GRAM_THREADS = 256;        // 8 warps: 0 TMA, 1 MMA, 2 TMEM alloc, 3 idle, 4..7 epilogue
constexpr uint32_t GRAM_OPB = GRAM_BK * TILE;                 // bytes of one operand tile per stage (8 KB)
constexpr uint32_t GRAM_STAGE_BYTES = 4 * GRAM_OPB;           // A, B0, B1, B2
constexpr size_t GRAM_SMEM = (size_t)GRAM_STAGES * GRAM_STAGE_BYTES + 1024 /*align*/ + 256 /*barriers*/;
constexpr uint32_t GRAM_TMEM_COLS = 512;

// ------------------------------------------------------------------ operand preparation
// max branch length over head rows (positive doubles order like their bit patterns)
__global__ void k_gram_lenmax(int n, const uint8_t* __restrict__ cls, const double* __restrict__ len,
                              unsigned long long* __restrict__ out_bits)
{
    int v = blockIdx.x * blockDim.x + threadIdx.x;
    unsigned long long b = 0;
    if (v < n && cls[v] == 1) b = (unsigned long long)__double_as_longlong(len[v]);
    for (int o = 16; o; o >>= 1) { unsigned long long t = __shfl_xor_sync(0xffffffffu, b, o); b = t > b ? t : b; }
    if ((threadIdx.x & 31) == 0 && b) atomicMax(out_bits, b);
}

// head rank -> node id, fixed-point length per head row, and the embedded value u~ of every branch for a present
// sample (what the side sums and the tail lists must use so that all parts agree):
//   head (Gram) rows: m_v * 2^(s_v - q)      other rows: (double)(float)len_v
// Fixed point with a per-row shift: len_v * 2^q ~ m_v * 2^s_v, m_v < 2^24 (three u8 digits, the B operands), s_v <= max_shift
// carried by the A operand (x * 2^s_v <= 128 fits its u8).  q is chosen so that the longest head branch uses s = max_shift
// and all 24 bits of m; a branch up to 2^max_shift times shorter still keeps 24 significant bits.
// Lq[r] = m | s << 24.
__global__ void k_gram_quant(int n, const uint8_t* __restrict__ cls, const uint32_t* __restrict__ hrank,
                             const double* __restrict__ len, int q, int max_shift, int32_t* __restrict__ hrows,
                             uint32_t* __restrict__ Lq, double* __restrict__ uval, double* __restrict__ uerr)
{
    int v = blockIdx.x * blockDim.x + threadIdx.x;
    if (v >= n) return;
    double l = len[v];
    if (cls[v] == 1) {
        const double Lf = ldexp(l, q);                       // < 2^(24 + max_shift)
        int s = 0;
        if (Lf >= 16777216.0) { int e; frexp(Lf, &e); s = e - 24; if (s > max_shift) s = max_shift; }
        long long m = llrint(ldexp(Lf, -s));
        if (m > 0xffffff) {                                  // rounded up to 2^24
            if (s < max_shift) { ++s; m = llrint(ldexp(Lf, -s)); } else m = 0xffffff;
        }
        uint32_t r = hrank[v];
        hrows[r] = v;
        Lq[r] = (uint32_t)m | ((uint32_t)s << 24);
        uval[v] = ldexp((double)m, s - q);
        uerr[v] = uval[v] - l;                               // what the fixed point changed (0 for most rows)
    } else {
        uval[v] = (double)(float)l;
        uerr[v] = 0.0;
    }
}

// bits -> u8 operand rows.  One thread = one 32-sample word of one head row: 32 bytes into each matrix.
__global__ void k_gram_expand(uint32_t K, uint32_t K_pad, const int32_t* __restrict__ hrows, const uint32_t* __restrict__ Lq,
                              const uint32_t* __restrict__ bits, uint32_t NW, uint8_t* __restrict__ XA,
                              uint8_t* __restrict__ XB0, uint8_t* __restrict__ XB1, uint8_t* __restrict__ XB2)
{
    long long gid = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    uint32_t r = (uint32_t)(gid / NW), w = (uint32_t)(gid - (long long)r * NW);
    if (r >= K_pad) return;
    uint32_t word = 0, L = 0;
    if (r < K) { word = bits[(size_t)hrows[r] * NW + w]; L = Lq[r]; }
    const uint32_t d0 = L & 255u, d1 = (L >> 8) & 255u, d2 = (L >> 16) & 255u, da = 1u << (L >> 24);
    const size_t off = (size_t)r * NW * 32 + (size_t)w * 32;
    uint32_t a[8], b0[8], b1[8], b2[8];
#pragma unroll
    for (int k = 0; k < 8; ++k) {
        uint32_t nib = (word >> (4 * k)) & 15u;
        uint32_t m = (nib & 1u) | ((nib & 2u) << 7) | ((nib & 4u) << 14) | ((nib & 8u) << 21);   // 4 bytes of 0/1
        a[k] = m * da; b0[k] = m * d0; b1[k] = m * d1; b2[k] = m * d2;
    }
    uint4* pa = reinterpret_cast<uint4*>(XA + off);   uint4* p0 = reinterpret_cast<uint4*>(XB0 + off);
    uint4* p1 = reinterpret_cast<uint4*>(XB1 + off);  uint4* p2 = reinterpret_cast<uint4*>(XB2 + off);
    pa[0] = make_uint4(a[0], a[1], a[2], a[3]);     pa[1] = make_uint4(a[4], a[5], a[6], a[7]);
    p0[0] = make_uint4(b0[0], b0[1], b0[2], b0[3]); p0[1] = make_uint4(b0[4], b0[5], b0[6], b0[7]);
    p1[0] = make_uint4(b1[0], b1[1], b1[2], b1[3]); p1[1] = make_uint4(b1[4], b1[5], b1[6], b1[7]);
    p2[0] = make_uint4(b2[0], b2[1], b2[2], b2[3]); p2[1] = make_uint4(b2[4], b2[5], b2[6], b2[7]);
}

// ------------------------------------------------------------------ PTX helpers (TMA tensor loads, tcgen05)
__device__ __forceinline__ void tma_load_2d(uint32_t dst, const CUtensorMap* tm, int c0, int c1, uint32_t bar) {
    asm volatile("cp.async.bulk.tensor.2d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3}], [%4];"
                 ::"r"(dst), "l"(tm), "r"(c0), "r"(c1), "r"(bar) : "memory");
}
__device__ __forceinline__ void tc_fence_before() { asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void tc_fence_after() { asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void tc_commit(uint32_t bar) {
    asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" ::"r"(bar) : "memory");
}
__device__ __forceinline__ void tc_mma_i8(uint32_t d_tmem, uint64_t adesc, uint64_t bdesc, uint32_t idesc, uint32_t accumulate) {
    asm volatile("{\n\t.reg .pred p;\n\tsetp.ne.b32 p, %4, 0;\n\t"
                 "tcgen05.mma.cta_group::1.kind::i8 [%0], %1, %2, %3, p;\n\t}"
                 ::"r"(d_tmem), "l"(adesc), "l"(bdesc), "r"(idesc), "r"(accumulate) : "memory");
}
__device__ __forceinline__ void tc_ld32(uint32_t taddr, uint32_t (&r)[32]) {
    asm volatile("tcgen05.ld.sync.aligned.32x32b.x32.b32 "
                 "{%0, %1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15, "
                 "%16, %17, %18, %19, %20, %21, %22, %23, %24, %25, %26, %27, %28, %29, %30, %31}, [%32];"
                 : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7]),
                   "=r"(r[8]), "=r"(r[9]), "=r"(r[10]), "=r"(r[11]), "=r"(r[12]), "=r"(r[13]), "=r"(r[14]), "=r"(r[15]),
                   "=r"(r[16]), "=r"(r[17]), "=r"(r[18]), "=r"(r[19]), "=r"(r[20]), "=r"(r[21]), "=r"(r[22]), "=r"(r[23]),
                   "=r"(r[24]), "=r"(r[25]), "=r"(r[26]), "=r"(r[27]), "=r"(r[28]), "=r"(r[29]), "=r"(r[30]), "=r"(r[31])
                 : "r"(taddr) : "memory");
}
__device__ __forceinline__ void tc_wait_ld() { asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory"); }

// shared-memory matrix descriptor, MN-major operand, 128B swizzle:
//   [0,14) start >> 4   [16,30) leading byte offset >> 4 (stride between 128-byte MN atoms)
//   [32,46) stride byte offset >> 4 (stride between 8-row K groups = 1024 B)   [46,48) version = 1   [61,64) layout = 2 (SW128)
__device__ __forceinline__ uint64_t umma_desc_mn_sw128(uint32_t smem_addr, uint32_t lbo_bytes) {
    uint64_t d = 0;
    d |= (uint64_t)((smem_addr & 0x3ffffu) >> 4);
    d |= (uint64_t)((lbo_bytes >> 4) & 0x3fffu) << 16;
    d |= (uint64_t)((1024u >> 4) & 0x3fffu) << 32;
    d |= (uint64_t)1 << 46;
    d |= (uint64_t)2 << 61;
    return d;
}
// instruction descriptor, kind::i8: D = s32, A = B = u8, both MN-major, M = 128, N given
__host__ __device__ constexpr uint32_t umma_idesc_i8(uint32_t N) {
    return (2u << 4) /*c: s32*/ | (0u << 7) /*a: u8*/ | (0u << 10) /*b: u8*/ | (1u << 15) /*a MN-major*/ |
           (1u << 16) /*b MN-major*/ | ((N >> 3) << 17) | ((128u >> 4) << 24);
}

struct GramParams {
    const int2* pairs; uint32_t n_pairs;
    uint32_t K_pad;               // multiple of GRAM_BK
    const double* sums;           // [n_tiles*128] S_s
    int n_samples;
    float* out;                   // condensed fp32
    int add_out;
    int q;                        // fixed-point scale
    // producer pacing (keeps the CTAs' K positions within two epochs of each other so that operand tiles shared by
    // the tile pairs of a block are still L2-resident when the slower CTAs reach them)
    unsigned int* epoch_cnt;      // [steps_per_cta >> epoch_shift + 1], zeroed per launch; NULL = no pacing
    uint32_t steps_per_cta;       // ceil(n_pairs / grid) * (K_pad / GRAM_BK): the same for every CTA
    uint32_t epoch_shift;         // epoch = 2^epoch_shift k-blocks
    GuardList guard;              // pairs with d < GUARD_THETA are listed for k_guard (guard.cuh)
};

// arrive at epoch e; before starting it, wait until every CTA has started epoch e - 1 (bounded spin: pacing only)
__device__ __forceinline__ void gram_epoch_sync(unsigned int* cnt, uint32_t e, uint32_t n_cta) {
    atomicAdd(cnt + e, 1u);
    if (e == 0) return;
    const volatile unsigned int* prev = cnt + (e - 1);
    for (uint32_t spin = 0; spin < (1u << 20); ++spin) {
        if (*prev >= n_cta) break;
        __nanosleep(64);
    }
}

__global__ void __launch_bounds__(GRAM_THREADS, 1)
k_gram(const __grid_constant__ CUtensorMap tmA, const __grid_constant__ CUtensorMap tmB0,
       const __grid_constant__ CUtensorMap tmB1, const __grid_constant__ CUtensorMap tmB2, const GramParams P)
{
    extern __shared__ unsigned char gsm_raw[];
    const uint32_t raw = smem_u32(gsm_raw);
    const uint32_t base = (raw + 1023u) & ~1023u;                       // SW128 tiles need 1024-byte alignment
    unsigned char* gsm = gsm_raw + (base - raw);
    const uint32_t bar0 = base + GRAM_STAGES * GRAM_STAGE_BYTES;        // barriers after the ring
    auto full = [&](int s) { return bar0 + 8u * s; };
    auto empty = [&](int s) { return bar0 + 8u * (GRAM_STAGES + s); };
    const uint32_t tmem_full = bar0 + 8u * (2 * GRAM_STAGES), tmem_empty = tmem_full + 8u;
    uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(gsm + GRAM_STAGES * GRAM_STAGE_BYTES + 8 * (2 * GRAM_STAGES + 2));

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    if (threadIdx.x == 0) {
        for (int s = 0; s < GRAM_STAGES; ++s) { mbar_init(full(s), 1); mbar_init(empty(s), 1); }
        mbar_init(tmem_full, 1); mbar_init(tmem_empty, 4);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    if (warp == 2) {
        asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_u32(tmem_slot)), "n"(GRAM_TMEM_COLS) : "memory");
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
    }
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const uint32_t tmem = *tmem_slot;
    const uint32_t n_k = P.K_pad / GRAM_BK;

    if (warp == 0) {
        // ======================================================= TMA producer
        if (lane == 0) {
            uint32_t stage = 0, phase = 0, g = 0;
            const uint32_t emask = (1u << P.epoch_shift) - 1u;
            for (uint32_t pi = blockIdx.x; pi < P.n_pairs; pi += gridDim.x) {
                const int2 ij = P.pairs[pi];
                for (uint32_t kb = 0; kb < n_k; ++kb, ++g) {
                    if (P.epoch_cnt && (g & emask) == 0u) gram_epoch_sync(P.epoch_cnt, g >> P.epoch_shift, gridDim.x);
                    mbar_wait(empty(stage), phase ^ 1u);
                    const uint32_t dst = base + stage * GRAM_STAGE_BYTES;
                    mbar_arrive_expect_tx(full(stage), GRAM_STAGE_BYTES);
                    const int row = (int)(kb * GRAM_BK);
                    tma_load_2d(dst, &tmA, ij.x * TILE, row, full(stage));
                    tma_load_2d(dst + GRAM_OPB, &tmB0, ij.y * TILE, row, full(stage));
                    tma_load_2d(dst + 2 * GRAM_OPB, &tmB1, ij.y * TILE, row, full(stage));
                    tma_load_2d(dst + 3 * GRAM_OPB, &tmB2, ij.y * TILE, row, full(stage));
                    if (++stage == GRAM_STAGES) { stage = 0; phase ^= 1u; }
                }
            }
            // CTAs with one tile pair fewer still arrive at the remaining epochs
            if (P.epoch_cnt)
                for (; g < P.steps_per_cta; ++g)
                    if ((g & emask) == 0u) atomicAdd(P.epoch_cnt + (g >> P.epoch_shift), 1u);
        }
    } else if (warp == 1) {
        // ======================================================= MMA issuer
        if (lane == 0) {
            uint32_t stage = 0, phase = 0, tphase = 0;
            constexpr uint32_t ID256 = umma_idesc_i8(256), ID128 = umma_idesc_i8(128);
            for (uint32_t pi = blockIdx.x; pi < P.n_pairs; pi += gridDim.x) {
                mbar_wait(tmem_empty, tphase ^ 1u);            // epilogue has drained the accumulators
                tc_fence_after();
                for (uint32_t kb = 0; kb < n_k; ++kb) {
                    mbar_wait(full(stage), phase);
                    tc_fence_after();
                    const uint32_t sa = base + stage * GRAM_STAGE_BYTES;
#pragma unroll
                    for (uint32_t ks = 0; ks < GRAM_BK / 32; ++ks) {
                        const uint32_t koff = ks * 32u * TILE;                       // 32 K rows of 128 bytes
                        const uint64_t da = umma_desc_mn_sw128(sa + koff, GRAM_OPB);
                        const uint64_t db01 = umma_desc_mn_sw128(sa + GRAM_OPB + koff, GRAM_OPB);   // N = 256: B0 | B1 atoms
                        const uint64_t db2 = umma_desc_mn_sw128(sa + 3 * GRAM_OPB + koff, GRAM_OPB);
                        const uint32_t acc = (kb | ks) ? 1u : 0u;
                        tc_mma_i8(tmem, da, db01, ID256, acc);
                        tc_mma_i8(tmem + 256, da, db2, ID128, acc);
                    }
                    tc_commit(empty(stage));                   // frees the smem stage when these MMAs retire
                    if (++stage == GRAM_STAGES) { stage = 0; phase ^= 1u; }
                }
                tc_commit(tmem_full);                          // accumulators complete
                tphase ^= 1u;
            }
        }
    } else if (warp >= 4) {
        // ======================================================= epilogue (a-6 finalize), 32 rows per warp
        const int e = warp - 4;                                // == warp % 4: TMEM lanes 32e .. 32e+31
        uint32_t tphase = 0;
        const long long N = P.n_samples;
        const double scale = ldexp(1.0, -P.q);
        for (uint32_t pi = blockIdx.x; pi < P.n_pairs; pi += gridDim.x) {
            const int2 ij = P.pairs[pi];
            mbar_wait(tmem_full, tphase);
            tc_fence_after();
            const long long gi = (long long)ij.x * TILE + e * 32 + lane;
            const double si = P.sums[gi];
            const long long rowbase = gi * (2 * N - gi - 1) / 2 - gi - 1;
            const uint32_t trow = tmem + ((uint32_t)(e * 32) << 16);
#pragma unroll 1
            for (int c0 = 0; c0 < TILE; c0 += 32) {
                uint32_t d0[32], d1[32], d2[32];
                tc_ld32(trow + c0, d0);
                tc_ld32(trow + 128 + c0, d1);
                tc_ld32(trow + 256 + c0, d2);
                tc_wait_ld();
#pragma unroll
                for (int c = 0; c < 32; ++c) {
                    const long long gj = (long long)ij.y * TILE + c0 + c;
                    if (gi < gj && gj < N) {
                        const long long g = (long long)(int)d0[c] + 256ll * (long long)(int)d1[c] + 65536ll * (long long)(int)d2[c];
                        double tot = (double)g * scale;
                        if (P.add_out) tot += (double)P.out[rowbase + gj];
                        const double ss = si + P.sums[gj];
                        double num = ss - 2.0 * tot, den = ss - tot;
                        if (num < 0.0) num = 0.0;
                        guard_note(P.guard, num, den, (uint32_t)gi, (uint32_t)gj);
                        P.out[rowbase + gj] = (float)(den > 0.0 ? num / den : 0.0);
                    }
                }
            }
            tc_fence_before();
            __syncwarp();
            if (lane == 0) mbar_arrive(tmem_empty);
            tphase ^= 1u;
        }
    }
    tc_fence_before();
    __syncthreads();
    if (warp == 2) {
        tc_fence_after();
        asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tmem), "n"(GRAM_TMEM_COLS) : "memory");
    }
}

}  // namespace ufb
