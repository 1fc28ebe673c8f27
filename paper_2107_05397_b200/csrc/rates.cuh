// rates.cuh -- device-rate probes behind the head / mid / tail cost model and
// behind the `peak` of the k_mid / k_tail_scatter rooflines: how many shared-memory integer atomics (the unit of work
// of k_mid) and L2-resident fp32 REDs (the unit of work of k_tail_scatter) this GPU retires per second.
// Launch shapes copy the kernels they stand for (k_mid: 3 CTAs/SM x 512 threads with 64 KB of accumulators each;
// k_tail_scatter: 8 CTAs/SM x 256 threads scattering into a 48 MB footprint).  Not on the data path.
#pragma once
#include "common.cuh"
#include "stripe.cuh"   // smem_u32

namespace ufb {

__device__ __forceinline__ uint32_t rate_hash(uint32_t x) {
    x ^= x >> 16; x *= 0x7feb352du; x ^= x >> 15; x *= 0x846ca68bu; x ^= x >> 16;
    return x;
}

// mode 0: the 32 lanes of a warp hit 32 different banks (conflict-free);  mode 1: pseudo-random cells of the 128 x 128
// tile (what k_mid's join produces);  8 independent atomics per loop iteration, addresses precomputed per iteration.
__global__ void __launch_bounds__(512, 3)
k_rate_atoms(int mode, int iters, unsigned int* __restrict__ sink)
{
    extern __shared__ uint32_t racc[];
    for (int i = threadIdx.x; i < 128 * 128; i += blockDim.x) racc[i] = 0u;
    __syncthreads();
    const uint32_t base = smem_u32(racc);
    const uint32_t lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    uint32_t h = rate_hash(blockIdx.x * 512u + threadIdx.x + 1u);
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int u = 0; u < 8; ++u) {
            h = h * 1664525u + 1013904223u;
            const uint32_t row = (h >> 8) & 127u;
            const uint32_t cell = mode == 0 ? (row * 128u + ((warp * 32u + lane) & 127u)) : ((h >> 15) & 16383u);
            asm volatile("red.shared.add.u32 [%0], %1;" ::"r"(base + cell * 4u), "r"(h & 255u) : "memory");
        }
    }
    __syncthreads();
    if (threadIdx.x == 0) atomicAdd(sink, racc[blockIdx.x & 16383]);     // keep the atomics observable
}

// pseudo-random fp32 RED.ADD into `cells` floats (L2-resident when cells * 4 B fits)
__global__ void __launch_bounds__(256)
k_rate_red(float* __restrict__ buf, uint32_t cells, int iters)
{
    uint32_t h = rate_hash(blockIdx.x * 256u + threadIdx.x + 1u);
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int u = 0; u < 4; ++u) {
            h = h * 1664525u + 1013904223u;
            atomicAdd(buf + (uint32_t)(((unsigned long long)(h >> 4) * cells) >> 28), 1.0f);
        }
    }
}

}  // namespace ufb
