// pcoa.cuh -- principal coordinates analysis behind the distance matrix.  PAPER.md:13 "researchers often
// apply principal coordinates analysis (PCoA)"; "PCoA can also be computed as part of the Hybrid UniFrac compute
// itself ... virtually no additional memory usage".  The paper gives no formula; DESIGN.md "PCoA" readings P1-P5:
//     A = -1/2 D o D,   B = A - rowmean - colmean + mean (Gower),   B = V diag(lambda) V',   coordinates = V_k sqrt(lambda_k),
//     proportion explained = lambda_i / trace(B).
// Device path: the condensed matrix is expanded to the square B (fp32) once; the k leading eigenpairs come from block subspace
// iteration with Rayleigh-Ritz on a block of PCOA_NB = 32 vectors:  Y = B Q  (the only O(N^2) step: a 128 x 32 x N tcgen05
// GEMM per 128 rows, kind::tf32 with the 3-term split  B_hi Q_hi + B_lo Q_hi + B_hi Q_lo  so that the product carries ~2^-21
// relative error instead of tf32's 2^-11; fp32 accumulation in TMEM),  Q = orth(Y)  (Cholesky QR in fp64),  T = Q' B Q,
// eig(T) by cyclic Jacobi (fp64).  Bound: HBM -- every product streams B_hi and B_lo once (8 N^2 bytes).
#pragma once
#include <cuda.h>
#include "common.cuh"
#include "stripe.cuh"   // smem_u32, mbarrier helpers
#include "gram.cuh"     // tma_load_2d, tcgen05 helpers

namespace ufb {

constexpr int PCOA_NB = 32;                 // block size of the subspace iteration (columns of Q)
constexpr int PCOA_BK = 32;                 // K elements per pipeline stage: 32 floats = one 128-byte swizzle row
constexpr int PCOA_STAGES = 5;
constexpr uint32_t PCOA_A_BYTES = 128 * PCOA_BK * 4;      // 16 KB: 128 rows of B x 32 k
constexpr uint32_t PCOA_Q_BYTES = PCOA_NB * PCOA_BK * 4;  //  4 KB: 32 columns of Q x 32 k
constexpr uint32_t PCOA_STAGE_BYTES = 2 * PCOA_A_BYTES + 2 * PCOA_Q_BYTES;   // 40 KB
constexpr int PCOA_NACC = 4;                // TMEM accumulators (32 columns each) in flight
constexpr int PCOA_DRAIN = 2;               // k-blocks per accumulator before it is drained into the fp64 register sums
constexpr size_t PCOA_SMEM = (size_t)PCOA_STAGES * PCOA_STAGE_BYTES + 1024 /*align*/ + 8 * (2 * PCOA_STAGES + 2 * PCOA_NACC) + 16;
constexpr int PCOA_THREADS = 256;

// tf32 keeps the top 19 bits of an fp32 word
__device__ __forceinline__ float tf32_hi(float v) { return __uint_as_float(__float_as_uint(v) & 0xffffe000u); }

// A = -1/2 d^2 as a square fp32 matrix [Npad][Npad] (zero diagonal, zero padding) from the condensed upper triangle
template <typename T>
__global__ void __launch_bounds__(256)
k_pcoa_square(const T* __restrict__ d, int n, long long pitch, float* __restrict__ A)
{
    __shared__ float tile[32][33];
    const int bi = blockIdx.y, bj = blockIdx.x;
    if (bi > bj) return;
    const long long N = n;
    for (int r = threadIdx.y; r < 32; r += 8) {
        const long long i = (long long)bi * 32 + r, j = (long long)bj * 32 + threadIdx.x;
        float v = 0.f;
        if (i < N && j < N && i < j) { const double x = (double)d[i * (2 * N - i - 1) / 2 + (j - i - 1)]; v = (float)(-0.5 * x * x); }
        tile[r][threadIdx.x] = v;
        if (i < pitch && j < pitch && i <= j) A[i * pitch + j] = v;
    }
    __syncthreads();
    for (int r = threadIdx.y; r < 32; r += 8) {
        const long long j = (long long)bj * 32 + r, i = (long long)bi * 32 + threadIdx.x;
        if (i < pitch && j < pitch && i < j) A[j * pitch + i] = tile[threadIdx.x][r];
    }
}

// rs[i] = sum_j A[i][j] (fp64), one warp per row; tot += rs[i]
__global__ void __launch_bounds__(256)
k_pcoa_rowsum(const float* __restrict__ A, int n, long long pitch, double* __restrict__ rs, double* __restrict__ tot)
{
    const int row = (int)(((long long)blockIdx.x * blockDim.x + threadIdx.x) >> 5), lane = threadIdx.x & 31;
    if (row >= n) return;
    const float4* p = reinterpret_cast<const float4*>(A + (long long)row * pitch);
    double s = 0.0;
    for (long long c = lane; c < pitch / 4; c += 32) { const float4 v = p[c]; s += ((double)v.x + (double)v.y) + ((double)v.z + (double)v.w); }
    for (int o = 16; o; o >>= 1) s += __shfl_xor_sync(0xffffffffu, s, o);
    if (lane == 0) { rs[row] = s; atomicAdd(tot, s); }
}

// B = A - r_i/n - r_j/n + tot/n^2 inside the n x n block (padding stays 0), split for the tf32 product:
// Bhi = top 19 bits (overwrites A), Blo = B - Bhi (exact in fp32)
__global__ void __launch_bounds__(256)
k_pcoa_center(float* __restrict__ Bhi, float* __restrict__ Blo, int n, long long pitch, const double* __restrict__ rs,
              const double* __restrict__ tot)
{
    const long long q = (long long)blockIdx.x * blockDim.x + threadIdx.x;          // one float4 per thread
    const long long per_row = pitch / 4;
    const long long i = q / per_row, j0 = (q - i * per_row) * 4;
    if (i >= pitch) return;
    float4 a = reinterpret_cast<float4*>(Bhi + i * pitch)[j0 / 4];
    float v[4] = {a.x, a.y, a.z, a.w}, h[4], l[4];
    const double inv = 1.0 / (double)n, m = *tot * inv * inv;
    const double ri = i < n ? rs[i] * inv : 0.0;
#pragma unroll
    for (int t = 0; t < 4; ++t) {
        const long long j = j0 + t;
        float b = 0.f;
        if (i < n && j < n) b = (float)((double)v[t] - ri - rs[j] * inv + m);
        h[t] = tf32_hi(b);
        l[t] = b - h[t];
    }
    reinterpret_cast<float4*>(Bhi + i * pitch)[j0 / 4] = make_float4(h[0], h[1], h[2], h[3]);
    reinterpret_cast<float4*>(Blo + i * pitch)[j0 / 4] = make_float4(l[0], l[1], l[2], l[3]);
}

// start block: Y[r][c] = a fixed pseudo-random value in (-1, 1) (integer hash of (r, c); the result of the iteration does
// not depend on it), zero in the padding rows
__global__ void __launch_bounds__(256)
k_pcoa_init(float* __restrict__ Y, int n, long long n_pad)
{
    const long long q = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (q >= n_pad * PCOA_NB) return;
    const long long r = q / PCOA_NB;
    uint32_t x = (uint32_t)q * 2654435761u + 0x9e3779b9u;
    x ^= x >> 16; x *= 0x85ebca6bu; x ^= x >> 13; x *= 0xc2b2ae35u; x ^= x >> 16;
    Y[q] = r < n ? (float)((double)x * (2.0 / 4294967296.0) - 1.0) : 0.f;
}

// G[a][b] += sum_r U[r][a] * V[r][b]   (U, V row-major [n_pad][32] fp32; fp64 accumulation; G 32 x 32, zeroed by the caller)
__global__ void __launch_bounds__(1024)
k_pcoa_gram32(const float* __restrict__ U, const float* __restrict__ V, long long n_pad, double* __restrict__ G)
{
    __shared__ float su[32][33], sv[32][33];
    const int a = threadIdx.y, b = threadIdx.x;                  // 32 x 32 threads: thread (a, b) owns G[a][b]
    double acc = 0.0;
    for (long long r0 = (long long)blockIdx.x * 32; r0 < n_pad; r0 += (long long)gridDim.x * 32) {
        su[a][b] = U[(r0 + a) * PCOA_NB + b];
        sv[a][b] = V[(r0 + a) * PCOA_NB + b];
        __syncthreads();
#pragma unroll 8
        for (int r = 0; r < 32; ++r) acc += (double)su[r][a] * (double)sv[r][b];
        __syncthreads();
    }
    atomicAdd(&G[a * 32 + b], acc);
}

// single block, 32 threads: Cholesky G = R' R (upper R) and Rinv = R^-1, fp64.  A non-positive pivot (rank-deficient block,
// e.g. fewer than 32 non-zero directions) is replaced by a column that contributes nothing (Rinv column = 0).
__global__ void k_pcoa_chol(const double* __restrict__ G, double* __restrict__ Rinv)
{
    __shared__ double R[32][33];
    const int t = threadIdx.x;
    for (int i = 0; i < 32; ++i) R[i][t] = 0.0;
    __syncwarp();
    for (int j = 0; j < 32; ++j) {
        // column j of R: R[i][j] for i <= j  (thread t handles nothing special: sequential over i, dot products across lanes)
        for (int i = 0; i <= j; ++i) {
            double s = (t < i) ? R[t][i] * R[t][j] : 0.0;
            for (int o = 16; o; o >>= 1) s += __shfl_xor_sync(0xffffffffu, s, o);
            if (t == 0) {
                const double g = 0.5 * (G[i * 32 + j] + G[j * 32 + i]);
                if (i < j) R[i][j] = R[i][i] > 0.0 ? (g - s) / R[i][i] : 0.0;
                else { const double dgn = g - s; R[j][j] = dgn > 1e-300 && dgn > 1e-10 * g ? sqrt(dgn) : 0.0; }
            }
            __syncwarp();
        }
    }
    // Rinv by back substitution: column t of Rinv solves R x = e_t
    {
        double x[32];
        for (int i = 31; i >= 0; --i) {
            double s = (i == t) ? 1.0 : 0.0;
            for (int k2 = i + 1; k2 < 32; ++k2) s -= R[i][k2] * x[k2];
            x[i] = (i <= t && R[i][i] > 0.0 && R[t][t] > 0.0) ? s / R[i][i] : 0.0;
        }
        for (int i = 0; i < 32; ++i) Rinv[i * 32 + t] = x[i];
    }
}

// Q = Y Rinv (row-major [n_pad][32], fp64 arithmetic) and its transposed tf32 split Qt_hi / Qt_lo [32][n_pad] for the GEMM
__global__ void __launch_bounds__(256)
k_pcoa_apply(const float* __restrict__ Y, const double* __restrict__ Rinv, long long n_pad, float* __restrict__ Q,
             float* __restrict__ Qt_hi, float* __restrict__ Qt_lo)
{
    __shared__ double sR[32][32];
    __shared__ float sq[8][32][33];
    for (int e = threadIdx.x; e < 1024; e += 256) sR[e >> 5][e & 31] = Rinv[e];
    __syncthreads();
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    for (long long r0 = ((long long)blockIdx.x * 8 + warp) * 32; r0 < n_pad; r0 += (long long)gridDim.x * 8 * 32) {
        for (int r = 0; r < 32; ++r) {                                   // lane = output column
            const float yv = Y[(r0 + r) * PCOA_NB + lane];
            double s = 0.0;
#pragma unroll
            for (int c = 0; c < 32; ++c) s += (double)__shfl_sync(0xffffffffu, yv, c) * sR[c][lane];
            const float qv = (float)s;
            Q[(r0 + r) * PCOA_NB + lane] = qv;
            sq[warp][r][lane] = qv;
        }
        __syncwarp();
        for (int c = 0; c < 32; ++c) {                                   // lane = row: coalesced transposed stores
            const float qv = sq[warp][lane][c];
            const float h = tf32_hi(qv);
            Qt_hi[(long long)c * n_pad + r0 + lane] = h;
            Qt_lo[(long long)c * n_pad + r0 + lane] = qv - h;
        }
        __syncwarp();
    }
}

// ------------------------------------------------------------------ Y = B Q on the tensor cores (tcgen05, kind::tf32)
// shared-memory matrix descriptor, K-major operand, 128B swizzle: rows of 128 bytes (32 fp32 along K), 8-row groups 1024 B apart
//   [0,14) start >> 4   [16,30) leading byte offset >> 4 (unused for swizzled K-major: 1)   [32,46) stride byte offset >> 4
//   [46,48) version = 1   [61,64) layout = 2 (SW128).  A K step of 8 tf32 = 32 bytes advances the start address inside the row.
__device__ __forceinline__ uint64_t umma_desc_k_sw128(uint32_t smem_addr) {
    uint64_t d = 0;
    d |= (uint64_t)((smem_addr & 0x3ffffu) >> 4);
    d |= (uint64_t)1 << 16;
    d |= (uint64_t)((1024u >> 4) & 0x3fffu) << 32;
    d |= (uint64_t)1 << 46;
    d |= (uint64_t)2 << 61;
    return d;
}
// instruction descriptor, kind::tf32: D = f32, A = B = tf32, both K-major, M = 128, N given
__host__ __device__ constexpr uint32_t umma_idesc_tf32(uint32_t N) {
    return (1u << 4) /*c: f32*/ | (2u << 7) /*a: tf32*/ | (2u << 10) /*b: tf32*/ | ((N >> 3) << 17) | ((128u >> 4) << 24);
}
__device__ __forceinline__ void tc_mma_tf32(uint32_t d_tmem, uint64_t adesc, uint64_t bdesc, uint32_t idesc, uint32_t accumulate) {
    asm volatile("{\n\t.reg .pred p;\n\tsetp.ne.b32 p, %4, 0;\n\t"
                 "tcgen05.mma.cta_group::1.kind::tf32 [%0], %1, %2, %3, p;\n\t}"
                 ::"r"(d_tmem), "l"(adesc), "l"(bdesc), "r"(idesc), "r"(accumulate) : "memory");
}

// One CTA per 128 rows of B (grid = n_pad / 128), K = n_pad streamed in stages of 32 columns:
//   warp 0: TMA producer (B_hi, B_lo boxes of 128 rows x 32 k; Qt_hi, Qt_lo boxes of 32 rows x 32 k; 128B swizzle)
//   warp 1: MMA issuer: per stage 4 K steps x {B_hi Q_hi, B_lo Q_hi, B_hi Q_lo} into a 128 x 32 fp32 accumulator in TMEM
//   warp 2: TMEM allocation (4 accumulators x 32 columns)
//   warps 4-7: drain + epilogue.  The tensor core adds into its fp32 accumulator with truncation, a bias of ~2^-24 per add
//   that grows linearly with K (measured: eigenvalues 1.8e-5 low at N = 1000 with one accumulator over the whole K), so an
//   accumulator only collects PCOA_DRAIN k-blocks (24 adds); it is then read with tcgen05.ld and added into per-thread fp64
//   sums while the issuer fills the next one.  Y[row][0..31] = those sums.
__global__ void __launch_bounds__(PCOA_THREADS, 1)
k_pcoa_gemm(const __grid_constant__ CUtensorMap tmBhi, const __grid_constant__ CUtensorMap tmBlo,
            const __grid_constant__ CUtensorMap tmQhi, const __grid_constant__ CUtensorMap tmQlo, uint32_t n_pad, float* __restrict__ Y)
{
    extern __shared__ unsigned char psm_raw[];
    const uint32_t raw = smem_u32(psm_raw);
    const uint32_t base = (raw + 1023u) & ~1023u;
    unsigned char* psm = psm_raw + (base - raw);
    const uint32_t bar0 = base + PCOA_STAGES * PCOA_STAGE_BYTES;
    auto full = [&](int s) { return bar0 + 8u * s; };
    auto empty = [&](int s) { return bar0 + 8u * (PCOA_STAGES + s); };
    auto acc_full = [&](int a) { return bar0 + 8u * (2 * PCOA_STAGES + a); };
    auto acc_empty = [&](int a) { return bar0 + 8u * (2 * PCOA_STAGES + PCOA_NACC + a); };
    uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(psm + PCOA_STAGES * PCOA_STAGE_BYTES + 8 * (2 * PCOA_STAGES + 2 * PCOA_NACC));

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    if (threadIdx.x == 0) {
        for (int s = 0; s < PCOA_STAGES; ++s) { mbar_init(full(s), 1); mbar_init(empty(s), 1); }
        for (int a = 0; a < PCOA_NACC; ++a) { mbar_init(acc_full(a), 1); mbar_init(acc_empty(a), 4); }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    if (warp == 2) {
        asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_u32(tmem_slot)), "n"(32 * PCOA_NACC) : "memory");
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
    }
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const uint32_t tmem = *tmem_slot;
    const uint32_t n_k = n_pad / PCOA_BK;
    const int row0 = (int)blockIdx.x * 128;

    if (warp == 0) {
        if (lane == 0) {
            uint32_t stage = 0, phase = 0;
            for (uint32_t kb = 0; kb < n_k; ++kb) {
                mbar_wait(empty(stage), phase ^ 1u);
                const uint32_t dst = base + stage * PCOA_STAGE_BYTES;
                mbar_arrive_expect_tx(full(stage), PCOA_STAGE_BYTES);
                const int k0 = (int)(kb * PCOA_BK);
                tma_load_2d(dst, &tmBhi, k0, row0, full(stage));
                tma_load_2d(dst + PCOA_A_BYTES, &tmBlo, k0, row0, full(stage));
                tma_load_2d(dst + 2 * PCOA_A_BYTES, &tmQhi, k0, 0, full(stage));
                tma_load_2d(dst + 2 * PCOA_A_BYTES + PCOA_Q_BYTES, &tmQlo, k0, 0, full(stage));
                if (++stage == PCOA_STAGES) { stage = 0; phase ^= 1u; }
            }
        }
    } else if (warp == 1) {
        if (lane == 0) {
            uint32_t stage = 0, phase = 0;
            constexpr uint32_t ID = umma_idesc_tf32(PCOA_NB);
            for (uint32_t kb = 0; kb < n_k; ++kb) {
                const uint32_t chunk = kb / PCOA_DRAIN, acc = chunk % PCOA_NACC, first = (kb % PCOA_DRAIN) == 0u;
                if (first) { mbar_wait(acc_empty(acc), ((chunk / PCOA_NACC) & 1u) ^ 1u); tc_fence_after(); }
                const uint32_t tacc = tmem + acc * 32u;
                mbar_wait(full(stage), phase);
                tc_fence_after();
                const uint32_t sa = base + stage * PCOA_STAGE_BYTES;
#pragma unroll
                for (uint32_t ks = 0; ks < PCOA_BK / 8; ++ks) {
                    const uint64_t ahi = umma_desc_k_sw128(sa + ks * 32u);
                    const uint64_t alo = umma_desc_k_sw128(sa + PCOA_A_BYTES + ks * 32u);
                    const uint64_t qhi = umma_desc_k_sw128(sa + 2 * PCOA_A_BYTES + ks * 32u);
                    const uint64_t qlo = umma_desc_k_sw128(sa + 2 * PCOA_A_BYTES + PCOA_Q_BYTES + ks * 32u);
                    tc_mma_tf32(tacc, ahi, qhi, ID, (first && ks == 0u) ? 0u : 1u);
                    tc_mma_tf32(tacc, alo, qhi, ID, 1u);
                    tc_mma_tf32(tacc, ahi, qlo, ID, 1u);
                }
                tc_commit(empty(stage));
                if ((kb + 1) % PCOA_DRAIN == 0u || kb + 1 == n_k) tc_commit(acc_full(acc));
                if (++stage == PCOA_STAGES) { stage = 0; phase ^= 1u; }
            }
        }
    } else if (warp >= 4) {
        const int e = warp - 4;
        double sum[32];
#pragma unroll
        for (int c = 0; c < 32; ++c) sum[c] = 0.0;
        const uint32_t n_chunks = (n_k + PCOA_DRAIN - 1) / PCOA_DRAIN;
        for (uint32_t chunk = 0; chunk < n_chunks; ++chunk) {
            const uint32_t acc = chunk % PCOA_NACC;
            mbar_wait(acc_full(acc), (chunk / PCOA_NACC) & 1u);
            tc_fence_after();
            uint32_t v[32];
            tc_ld32(tmem + ((uint32_t)(e * 32) << 16) + acc * 32u, v);
            tc_wait_ld();
            tc_fence_before();
            __syncwarp();
            if (lane == 0) mbar_arrive(acc_empty(acc));
#pragma unroll
            for (int c = 0; c < 32; ++c) sum[c] += (double)__uint_as_float(v[c]);
        }
        float4* dst = reinterpret_cast<float4*>(Y + ((size_t)row0 + e * 32 + lane) * PCOA_NB);
#pragma unroll
        for (int c = 0; c < 8; ++c)
            dst[c] = make_float4((float)sum[4 * c], (float)sum[4 * c + 1], (float)sum[4 * c + 2], (float)sum[4 * c + 3]);
    }
    tc_fence_before();
    __syncthreads();
    if (warp == 2) {
        tc_fence_after();
        asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tmem), "n"(32 * PCOA_NACC) : "memory");
    }
}

// ------------------------------------------------------------------ Rayleigh-Ritz on the 32-dimensional block
// One warp.  T = (G + G') / 2 with G = Q' (B Q); cyclic Jacobi in fp64 (lane t owns row t of T and of the rotation product W);
// eigenvalues sorted in descending ALGEBRAIC order:  lam[0..31], W[c][a] = component c of eigenvector a.
__global__ void k_pcoa_jacobi(const double* __restrict__ G, double* __restrict__ lam, double* __restrict__ W)
{
    __shared__ double T[32][33], V[32][33];
    __shared__ int order[32];
    const int t = threadIdx.x;
    for (int c = 0; c < 32; ++c) { T[t][c] = 0.5 * (G[t * 32 + c] + G[c * 32 + t]); V[t][c] = t == c ? 1.0 : 0.0; }
    __syncwarp();
    for (int sweep = 0; sweep < 30; ++sweep) {
        double off = 0.0;
        for (int c = 0; c < 32; ++c) if (c != t) off += T[t][c] * T[t][c];
        double dg = T[t][t] * T[t][t];
        for (int o = 16; o; o >>= 1) { off += __shfl_xor_sync(0xffffffffu, off, o); dg += __shfl_xor_sync(0xffffffffu, dg, o); }
        if (off <= 1e-30 * dg || off == 0.0) break;
        for (int p = 0; p < 31; ++p)
            for (int q = p + 1; q < 32; ++q) {
                const double apq = T[p][q];
                if (apq != 0.0) {                                            // uniform: every lane reads the same cell
                    const double app = T[p][p], aqq = T[q][q];
                    const double theta = (aqq - app) / (2.0 * apq);
                    const double tt = (theta >= 0.0 ? 1.0 : -1.0) / (fabs(theta) + sqrt(theta * theta + 1.0));
                    const double cs = 1.0 / sqrt(tt * tt + 1.0), sn = tt * cs;
                    __syncwarp();
                    // columns p, q of T and V (lane t = row t), then rows p, q of T
                    const double tp = T[t][p], tq = T[t][q];
                    T[t][p] = cs * tp - sn * tq; T[t][q] = sn * tp + cs * tq;
                    const double vp = V[t][p], vq = V[t][q];
                    V[t][p] = cs * vp - sn * vq; V[t][q] = sn * vp + cs * vq;
                    __syncwarp();
                    const double rp = T[p][t], rq = T[q][t];
                    __syncwarp();
                    T[p][t] = cs * rp - sn * rq; T[q][t] = sn * rp + cs * rq;
                    __syncwarp();
                }
            }
    }
    __syncwarp();
    // rank of eigenvalue t in descending order (ties by index)
    const double mine = T[t][t];
    int rank = 0;
    for (int c = 0; c < 32; ++c) { const double o = T[c][c]; rank += (o > mine) || (o == mine && c < t); }
    order[rank] = t;
    __syncwarp();
    const int src = order[t];
    lam[t] = T[src][src];
    for (int c = 0; c < 32; ++c) W[c * 32 + t] = V[c][src];
}

// out = [k eigenvalues | k proportions | n x k coordinates (row-major)]:  coords[r][a] = sqrt(max(lam_a, 0)) * sum_c Q[r][c] W[c][a]
__global__ void __launch_bounds__(256)
k_pcoa_coords(const float* __restrict__ Q, const double* __restrict__ lam, const double* __restrict__ W, int n, int k,
              double trace, double* __restrict__ out)
{
    __shared__ double sW[32][32], sl[32];
    for (int e = threadIdx.x; e < 1024; e += 256) sW[e >> 5][e & 31] = W[e];
    if (threadIdx.x < 32) sl[threadIdx.x] = lam[threadIdx.x];
    __syncthreads();
    if (blockIdx.x == 0 && threadIdx.x < k) {
        out[threadIdx.x] = sl[threadIdx.x];
        out[k + threadIdx.x] = trace > 0.0 ? sl[threadIdx.x] / trace : 0.0;
    }
    const long long q = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (q >= (long long)n * k) return;
    const long long r = q / k;
    const int a = (int)(q - r * k);
    double s = 0.0;
    for (int c = 0; c < 32; ++c) s += (double)Q[r * PCOA_NB + c] * sW[c][a];
    out[2 * k + q] = s * sqrt(fmax(sl[a], 0.0));
}

}  // namespace ufb
