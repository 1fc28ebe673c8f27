// mantel.cuh -- Mantel test with Pearson's correlation on two resident distance matrices (PAPER.md:41-55:
// "The Mantel test is often used to check for correlations between two distance matrices ... Pearson's product-moment
// correlation coefficient"; "the application is likely mostly memory bound"; the authors did not port it to GPUs for lack
// of GPU memory -- 180 GB of HBM removes that reason).  The paper gives no formula; the test is the standard one
// (DESIGN.md "Mantel"): with x, y the condensed upper triangles of the symmetric hollow matrices X, Y,
//     r   = Pearson(x, y)
//     r_k = Pearson(condensed(X[pi_k, pi_k]), y)      for each given permutation pi_k of the N objects
//     p   = (#{k : |r_k| >= |r|} + 1) / (K + 1)       (two-sided; "greater" / "less" likewise)
// A permutation of the objects does not change the mean and the norm of x, so only S_k = sum_{i<j} X[pi_i, pi_j] y_ij
// differs between permutations.  Row pi_i of the SQUARE copy of X is staged in shared memory (it is gathered at the random
// columns pi_j), y's row i streams from HBM, pi_k stays in L2; fp64 accumulation.
// Bound: HBM -- 6 N^2 bytes per permutation for fp32 (X rows 4 N^2, y 2 N^2) against 4 N^2 algorithmic (both triangles once).
#pragma once
#include "common.cuh"
#include "stripe.cuh"   // mbarrier / bulk-copy helpers

namespace ufb {

// warp / block sum of doubles
__device__ __forceinline__ double warp_sum(double v) {
    for (int o = 16; o; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}

// moments over the condensed vectors, SHIFTED by the first elements x0 = x[0], y0 = y[0] (a constant vector then sums to
// exactly 0, and the variances below lose no digits to the mean):
//   out[0..4] += {sum (x - x0), sum (y - y0), sum (x - x0)^2, sum (y - y0)^2, sum (x - x0)(y - y0)}
template <typename T>
__global__ void __launch_bounds__(256)
k_mantel_moments(const T* __restrict__ x, const T* __restrict__ y, unsigned long long P, double* __restrict__ out)
{
    double s[5] = {0, 0, 0, 0, 0};
    const double x0 = (double)x[0], y0 = (double)y[0];
    const unsigned long long stride = (unsigned long long)gridDim.x * blockDim.x;
    unsigned long long k = (unsigned long long)blockIdx.x * blockDim.x + threadIdx.x;
    for (; k + 3 * stride < P; k += 4 * stride) {                    // 8 independent loads in flight per thread
        T xv[4], yv[4];
#pragma unroll
        for (int u = 0; u < 4; ++u) { xv[u] = x[k + u * stride]; yv[u] = y[k + u * stride]; }
#pragma unroll
        for (int u = 0; u < 4; ++u) {
            const double a = (double)xv[u] - x0, b = (double)yv[u] - y0;
            s[0] += a; s[1] += b; s[2] += a * a; s[3] += b * b; s[4] += a * b;
        }
    }
    for (; k < P; k += stride) {
        const double a = (double)x[k] - x0, b = (double)y[k] - y0;
        s[0] += a; s[1] += b; s[2] += a * a; s[3] += b * b; s[4] += a * b;
    }
    __shared__ double part[5][8];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
#pragma unroll
    for (int q = 0; q < 5; ++q) { s[q] = warp_sum(s[q]); if (lane == 0) part[q][warp] = s[q]; }
    __syncthreads();
    if (threadIdx.x < 5) {
        double t = 0;
        for (int w = 0; w < 8; ++w) t += part[threadIdx.x][w];
        atomicAdd(out + threadIdx.x, t);
    }
}

// square copy of X from its condensed upper triangle (zero diagonal): Xs[i][j] = Xs[j][i] = x[idx(i,j)]
// grid = (ceil(N/32), ceil(N/32)) tiles with bi <= bj, 32 x 8 threads: coalesced reads of rows i, coalesced writes of both.
template <typename T>
__global__ void __launch_bounds__(256)
k_mantel_square(const T* __restrict__ x, int n, long long pitch, T* __restrict__ Xs)
{
    __shared__ T tile[32][33];
    const int bi = blockIdx.y, bj = blockIdx.x;
    if (bi > bj) return;
    const long long N = n;
    for (int r = threadIdx.y; r < 32; r += 8) {
        const long long i = (long long)bi * 32 + r, j = (long long)bj * 32 + threadIdx.x;
        T v = (T)0;
        if (i < N && j < N && i < j) v = x[i * (2 * N - i - 1) / 2 + (j - i - 1)];
        tile[r][threadIdx.x] = v;
        if (i < N && j < N && i <= j) Xs[i * pitch + j] = v;
    }
    __syncthreads();
    for (int r = threadIdx.y; r < 32; r += 8) {
        const long long j = (long long)bj * 32 + r, i = (long long)bi * 32 + threadIdx.x;     // transposed element (j, i)
        if (i < N && j < N && i < j) Xs[j * pitch + i] = tile[threadIdx.x][r];
    }
}

__global__ void k_mantel_iota(int32_t* __restrict__ v, int n) { const int i = blockIdx.x * blockDim.x + threadIdx.x; if (i < n) v[i] = i; }

// S[k] += sum_{j > i} Xs[pi_k(i)][pi_k(j)] * y[idx(i, j)]   over the rows i = blockIdx.y, blockIdx.y + gridDim.y, ... of
// permutation k = blockIdx.x (k = 0: the identity = the statistic itself; k >= 1: perms[k-1]).  The permutation index is the
// FAST grid dimension: the CTAs resident at one time walk the same rows i for different permutations, so y's row i comes
// from HBM once and from L2 for the other permutations.
// Row pi_k(i) of the square copy (pitch elements, 16-byte aligned) is staged in shared memory in n_split column segments
// of seg elements through a two-buffer ring of TMA bulk copies (cp.async.bulk + mbarrier): while segment w is used, segment
// w+1 (the next segment, or the next row's first one) is in flight.  For every j > i the thread looks up c = pi_k(j); the
// product is taken if c falls into the staged segment.  The loads of pi_k(j) (L2-resident) and y_ij (streamed) of
// MANTEL_UNROLL elements per thread are issued together and unconditionally -- a y load that waited for the segment test
// would put two memory latencies in series, which is what bounded the first version of this loop.  fp64 accumulation.
constexpr int MANTEL_THREADS = 1024;             // 31 consumer warps + 1 producer warp
constexpr int MANTEL_CONSUMERS = MANTEL_THREADS - 32;
constexpr int MANTEL_UNROLL = 8;
constexpr uint32_t MANTEL_BULK = 32768;          // bytes per bulk copy
template <typename T, bool SPLIT>
__global__ void __launch_bounds__(MANTEL_THREADS, 1)
k_mantel_perm(const T* __restrict__ Xs, long long pitch, const T* __restrict__ y, const int32_t* __restrict__ perms,
              const int32_t* __restrict__ ident, int n, int seg, int n_split, int n_buf, int k_base, double* __restrict__ S)
{
    extern __shared__ __align__(128) unsigned char msm_raw[];
    __shared__ __align__(8) unsigned long long bars[4];              // full[0..1], empty[0..1]
    __shared__ double part[MANTEL_THREADS / 32];
    const uint32_t full[2] = {smem_u32(&bars[0]), smem_u32(&bars[1])};
    const uint32_t empty[2] = {smem_u32(&bars[2]), smem_u32(&bars[3])};
    const long long N = n;
    const int k = k_base + blockIdx.x;
    const int32_t* __restrict__ pi = k ? perms + (size_t)(k - 1) * n : ident;
    const long long n_rows = (N - 1 > (long long)blockIdx.y) ? (N - 1 - blockIdx.y + gridDim.y - 1) / gridDim.y : 0;
    const long long n_items = n_rows * n_split;
    const uint32_t useg = (uint32_t)seg;
    if (threadIdx.x == 0) {
        mbar_init(full[0], 1); mbar_init(full[1], 1);
        mbar_init(empty[0], MANTEL_CONSUMERS / 32); mbar_init(empty[1], MANTEL_CONSUMERS / 32);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        reinterpret_cast<T*>(msm_raw)[n_buf * seg] = (T)0;           // the zero element behind the buffers (SPLIT)
    }
    __syncthreads();
    double acc = 0.0;
    if (threadIdx.x >= MANTEL_CONSUMERS) {
        // ---- producer warp: one lane stages item w = (row, segment) into buffer w & 1 once every consumer warp has left
        // the item that used it before
        if (threadIdx.x == MANTEL_CONSUMERS) {
            for (long long w = 0; w < n_items; ++w) {
                const uint32_t b = n_buf == 2 ? (uint32_t)(w & 1) : 0u;
                const long long use = n_buf == 2 ? (w >> 1) : w;         // how often buffer b has been filled before
                if (use >= 1) mbar_wait(empty[b], (uint32_t)((use - 1) & 1));
                const long long i = blockIdx.y + (w / n_split) * gridDim.y;
                const long long src = pi[i];
                const long long lo = (long long)(w % n_split) * seg;
                const long long len = (pitch - lo < seg) ? pitch - lo : seg;
                const uint32_t bytes = (uint32_t)(len * sizeof(T));
                mbar_arrive_expect_tx(full[b], bytes);
                const unsigned char* g = reinterpret_cast<const unsigned char*>(Xs + src * pitch + lo);
                const uint32_t d = smem_u32(msm_raw) + b * useg * (uint32_t)sizeof(T);
                for (uint32_t off = 0; off < bytes; off += MANTEL_BULK)
                    bulk_g2s(d + off, g + off, bytes - off < MANTEL_BULK ? bytes - off : MANTEL_BULK, full[b]);
            }
        }
    } else {
        // ---- consumer warps: no block barrier between items -- a warp that is done with an item arrives on its buffer's
        // empty barrier and goes on to the next item (whose segment is already staged), so the load latency of one warp
        // overlaps the multiply-adds of the others across the end of a row
        const T* __restrict__ sm = reinterpret_cast<const T*>(msm_raw);  // indexed as shared memory (LDS), both buffers
        const uint32_t zero_at = (uint32_t)n_buf * useg;
        constexpr uint32_t BATCH = MANTEL_UNROLL * MANTEL_CONSUMERS;
        for (long long w = 0; w < n_items; ++w) {
            const long long i = blockIdx.y + (w / n_split) * gridDim.y;
            const uint32_t lo = (uint32_t)(w % n_split) * useg;
            const uint32_t b = n_buf == 2 ? (uint32_t)(w & 1) : 0u;
            const uint32_t phase = (uint32_t)((n_buf == 2 ? (w >> 1) : w) & 1);
            const uint32_t boff = b * useg;                          // staged element c (relative to lo) sits at sm[boff + c]
            const uint32_t rem = (uint32_t)(N - 1 - i);              // elements j = i + 1 + e, e < rem, of row i
            const T* __restrict__ yp = y + (i * (2 * N - i - 1) / 2) + threadIdx.x;  // y_ij of element e = threadIdx.x
            const int32_t* __restrict__ pp = pi + i + 1 + threadIdx.x;
            for (uint32_t e0 = 0; e0 < rem; e0 += BATCH, yp += BATCH, pp += BATCH) {
                uint32_t c[MANTEL_UNROLL]; T yv[MANTEL_UNROLL];
                if (e0 + BATCH <= rem) {
#pragma unroll
                    for (int u = 0; u < MANTEL_UNROLL; ++u) { c[u] = (uint32_t)pp[u * MANTEL_CONSUMERS] - lo; yv[u] = yp[u * MANTEL_CONSUMERS]; }
                } else {
#pragma unroll
                    for (int u = 0; u < MANTEL_UNROLL; ++u) {
                        const bool ok = e0 + threadIdx.x + u * MANTEL_CONSUMERS < rem;
                        c[u] = ok ? (uint32_t)pp[u * MANTEL_CONSUMERS] - lo : 0u;    // product with y = 0
                        yv[u] = ok ? yp[u * MANTEL_CONSUMERS] : (T)0;
                    }
                }
                // the first batch of an item is requested before its staged segment is waited for; later waits fall through
                mbar_wait(full[b], phase);
                // straight-line selects, no branches: membership of the segment is random per lane, so every warp executes
                // the load and the multiply-add anyway
#pragma unroll
                for (int u = 0; u < MANTEL_UNROLL; ++u) {
                    if (SPLIT) acc += (double)sm[c[u] < useg ? boff + c[u] : zero_at] * (double)yv[u];   // outside: the zero element
                    else acc += (double)sm[boff + c[u]] * (double)yv[u];
                }
            }
            __syncwarp();
            if ((threadIdx.x & 31) == 0) mbar_arrive(empty[b]);
        }
    }
    acc = warp_sum(acc);
    if ((threadIdx.x & 31) == 0) part[threadIdx.x >> 5] = acc;
    __syncthreads();
    if (threadIdx.x == 0) {
        double t = 0;
        for (int w = 0; w < MANTEL_CONSUMERS / 32; ++w) t += part[w];
        S[(size_t)k * gridDim.y + blockIdx.y] = t;                   // per-CTA partial: k_mantel_final adds them in a fixed order,
    }                                                                // so equal permutations give bit-equal statistics
}

// out[0] = r, out[1..3] = p two-sided / greater / less, out[4 + k] = r_k (k = 0 .. K-1)
// S[k][0..G) = per-CTA partial sums of the raw products x^pi y;  mom = the shifted moments of k_mantel_moments, (x0, y0) the shifts.
template <typename T>
__global__ void k_mantel_final(const double* __restrict__ mom, const double* __restrict__ Spart, int G, int K, double P,
                               const T* __restrict__ x, const T* __restrict__ y, double* __restrict__ out)
{
    auto Ssum = [&](int k) { double t = 0.0; for (int g = 0; g < G; ++g) t += Spart[(size_t)k * G + g]; return t; };
    const double x0 = (double)x[0], y0 = (double)y[0];
    const double dx = mom[0], dy = mom[1];                         // sum (x - x0), sum (y - y0)
    const double vx = mom[2] - dx * dx / P, vy = mom[3] - dy * dy / P;
    const double sx = dx + P * x0, sy = dy + P * y0;               // plain sums
    const double den = sqrt(vx * vy);
    auto corr = [&](double sxy) { return (vx > 0.0 && vy > 0.0 && den > 0.0) ? (sxy - sx * sy / P) / den : 0.0; };
    const double r = corr(Ssum(0));
    int two = 0, gr = 0, le = 0;
    for (int k = threadIdx.x; k < K; k += blockDim.x) {
        const double rk = corr(Ssum(1 + k));
        out[4 + k] = rk;
        two += fabs(rk) >= fabs(r); gr += rk >= r; le += rk <= r;
    }
    __shared__ int cnt[3];
    if (threadIdx.x == 0) { cnt[0] = cnt[1] = cnt[2] = 0; }
    __syncthreads();
    atomicAdd(&cnt[0], two); atomicAdd(&cnt[1], gr); atomicAdd(&cnt[2], le);
    __syncthreads();
    if (threadIdx.x == 0) {
        out[0] = r;
        out[1] = (cnt[0] + 1.0) / (K + 1.0); out[2] = (cnt[1] + 1.0) / (K + 1.0); out[3] = (cnt[2] + 1.0) / (K + 1.0);
    }
}

}  // namespace ufb
