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
    for (unsigned long long k = (unsigned long long)blockIdx.x * blockDim.x + threadIdx.x; k < P; k += (unsigned long long)gridDim.x * blockDim.x) {
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

// S[k] += sum_{j > i} Xs[pi_k(i)][pi_k(j)] * y[idx(i, j)]   over the rows i = blockIdx.x, blockIdx.x + gridDim.x, ... of
// permutation k = blockIdx.y (k = 0: identity = the statistic itself; k >= 1: perms[k-1]).
// Row pi_k(i) of the square copy (pitch elements, 16-byte aligned) is staged in shared memory in n_split column segments
// of seg elements through a two-buffer ring of TMA bulk copies (cp.async.bulk + mbarrier): while segment w is used, segment
// w+1 (the next segment, or the next row's first one) is in flight.  For every j > i the thread looks up c = pi_k(j); the
// product is taken if c falls into the staged segment.  y's row i is read once (only by the segment that owns c), pi_k
// stays L2-resident.  fp64 accumulation.
constexpr int MANTEL_THREADS = 1024;
constexpr uint32_t MANTEL_BULK = 32768;          // bytes per bulk copy
template <typename T>
__global__ void __launch_bounds__(MANTEL_THREADS, 1)
k_mantel_perm(const T* __restrict__ Xs, long long pitch, const T* __restrict__ y, const int32_t* __restrict__ perms, int n,
              int seg, int n_split, int k_base, double* __restrict__ S)
{
    extern __shared__ __align__(128) unsigned char msm_raw[];
    __shared__ __align__(8) unsigned long long bars[2];
    __shared__ double part[MANTEL_THREADS / 32];
    T* buf[2] = {reinterpret_cast<T*>(msm_raw), reinterpret_cast<T*>(msm_raw) + seg};
    const uint32_t bar[2] = {smem_u32(&bars[0]), smem_u32(&bars[1])};
    const long long N = n;
    const int k = k_base + blockIdx.y;
    const int32_t* pi = k ? perms + (size_t)(k - 1) * n : nullptr;
    const long long n_rows = (N - 1 > (long long)blockIdx.x) ? (N - 1 - blockIdx.x + gridDim.x - 1) / gridDim.x : 0;
    const long long n_items = n_rows * n_split;
    if (threadIdx.x == 0) {
        mbar_init(bar[0], 1); mbar_init(bar[1], 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();
    auto issue = [&](long long w) {                                  // one thread
        const long long i = blockIdx.x + (w / n_split) * gridDim.x;
        const int sgm = (int)(w % n_split);
        const long long src = pi ? pi[i] : i;
        const long long lo = (long long)sgm * seg;
        const long long len = (pitch - lo < seg) ? pitch - lo : seg;
        const uint32_t bytes = (uint32_t)(len * sizeof(T));
        const uint32_t b = bar[w & 1];
        mbar_arrive_expect_tx(b, bytes);
        const unsigned char* g = reinterpret_cast<const unsigned char*>(Xs + src * pitch + lo);
        const uint32_t d = smem_u32(buf[w & 1]);
        for (uint32_t off = 0; off < bytes; off += MANTEL_BULK)
            bulk_g2s(d + off, g + off, bytes - off < MANTEL_BULK ? bytes - off : MANTEL_BULK, b);
    };
    if (threadIdx.x == 0 && n_items > 0) issue(0);
    double acc = 0.0;
    for (long long w = 0; w < n_items; ++w) {
        if (threadIdx.x == 0 && w + 1 < n_items) issue(w + 1);       // its buffer was released by the barrier below (iteration w-1)
        mbar_wait(bar[w & 1], (uint32_t)((w >> 1) & 1));
        const long long i = blockIdx.x + (w / n_split) * gridDim.x;
        const long long lo = (long long)(w % n_split) * seg;
        const T* row = buf[w & 1];
        const T* yr = y + (i * (2 * N - i - 1) / 2 - i - 1);
#pragma unroll 4
        for (long long j = i + 1 + threadIdx.x; j < N; j += MANTEL_THREADS) {
            const long long c = (pi ? (long long)pi[j] : j) - lo;
            if ((unsigned long long)c < (unsigned long long)seg) acc += (double)row[c] * (double)yr[j];
        }
        __syncthreads();
    }
    acc = warp_sum(acc);
    if ((threadIdx.x & 31) == 0) part[threadIdx.x >> 5] = acc;
    __syncthreads();
    if (threadIdx.x == 0) {
        double t = 0;
        for (int w = 0; w < MANTEL_THREADS / 32; ++w) t += part[w];
        atomicAdd(S + k, t);
    }
}

// out[0] = r, out[1..3] = p two-sided / greater / less, out[4 + k] = r_k (k = 0 .. K-1)
// S[k] = sum of the raw products x^pi y;  mom = the shifted moments of k_mantel_moments, (x0, y0) the shifts.
template <typename T>
__global__ void k_mantel_final(const double* __restrict__ mom, const double* __restrict__ S, int K, double P, const T* __restrict__ x,
                               const T* __restrict__ y, double* __restrict__ out)
{
    const double x0 = (double)x[0], y0 = (double)y[0];
    const double dx = mom[0], dy = mom[1];                         // sum (x - x0), sum (y - y0)
    const double vx = mom[2] - dx * dx / P, vy = mom[3] - dy * dy / P;
    const double sx = dx + P * x0, sy = dy + P * y0;               // plain sums
    const double den = sqrt(vx * vy);
    auto corr = [&](double sxy) { return (vx > 0.0 && vy > 0.0 && den > 0.0) ? (sxy - sx * sy / P) / den : 0.0; };
    const double r = corr(S[0]);
    int two = 0, gr = 0, le = 0;
    for (int k = threadIdx.x; k < K; k += blockDim.x) {
        const double rk = corr(S[1 + k]);
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
