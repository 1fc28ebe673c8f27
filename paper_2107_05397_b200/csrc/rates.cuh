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

// FP32-pipe probes behind the `"bound": "alu"` roofline of k_dense: 8 independent register chains per thread of
// mode 0: FMNMX (min.f32, the half-rate ALU pipe);  1: FADD (the FMA pipe);  2: FMNMX + FADD pairs (k_dense's update)
template <int mode>
__global__ void __launch_bounds__(256)
k_rate_alu(int iters, float* __restrict__ sink)
{
    float a[8], b[8];
#pragma unroll
    for (int k = 0; k < 8; ++k) { a[k] = 1.0f + threadIdx.x * 1e-3f + k; b[k] = 0.5f + k * 1e-2f + blockIdx.x * 1e-6f; }
#pragma unroll 4
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int k = 0; k < 8; ++k) {
            if (mode == 0) {                                    // min / max alternate so that the chain is not idempotent
                if (it & 1) asm volatile("min.f32 %0, %0, %1;" : "+f"(a[k]) : "f"(b[k]));
                else        asm volatile("max.f32 %0, %0, %1;" : "+f"(a[k]) : "f"(b[(k + 1) & 7]));
            }
            else if (mode == 1) asm volatile("add.f32 %0, %0, %1;" : "+f"(a[k]) : "f"(b[k]));
            else if (mode == 2) { float m; asm volatile("min.f32 %0, %1, %2;" : "=f"(m) : "f"(a[k]), "f"(b[k])); asm volatile("add.f32 %0, %0, %1;" : "+f"(b[k]) : "f"(m)); }
        }
        // packed adds (add.f32x2 -> FADD2): 3 = FADD2 alone (4 chains of pairs);  4 = two FMNMX + one FADD2 (the min cells of
        // k_dense16);  5 = k_dense16's mix for 8 updates: 3 x (2 FMNMX + FADD2) + 2 x (FADD + FFMA |d| * -0.5)
        if (mode == 3) {
#pragma unroll
            for (int k = 0; k < 8; k += 2)
                asm volatile("{\n\t.reg .b64 p, q;\n\tmov.b64 p, {%0, %1};\n\tmov.b64 q, {%2, %3};\n\tadd.rn.f32x2 p, p, q;\n\tmov.b64 {%0, %1}, p;\n\t}"
                             : "+f"(a[k]), "+f"(a[k + 1]) : "f"(b[k]), "f"(b[k + 1]));
        } else if (mode == 4 || mode == 5) {
#pragma unroll
            for (int k = 0; k < 8; k += 2) {
                if (mode == 5 && k == 6) {
                    float d0, d1;
                    asm volatile("sub.f32 %0, %1, %2;" : "=f"(d0) : "f"(a[k]), "f"(b[0]));
                    asm volatile("sub.f32 %0, %1, %2;" : "=f"(d1) : "f"(a[k + 1]), "f"(b[1]));
                    asm volatile("fma.rn.f32 %0, %1, 0fBF000000, %0;" : "+f"(b[k]) : "f"(fabsf(d0)));
                    asm volatile("fma.rn.f32 %0, %1, 0fBF000000, %0;" : "+f"(b[k + 1]) : "f"(fabsf(d1)));
                } else {
                    float m0, m1;
                    asm volatile("min.f32 %0, %1, %2;" : "=f"(m0) : "f"(a[k]), "f"(b[(k + 2) & 7]));
                    asm volatile("min.f32 %0, %1, %2;" : "=f"(m1) : "f"(a[k + 1]), "f"(b[(k + 3) & 7]));
                    asm volatile("{\n\t.reg .b64 p, q;\n\tmov.b64 p, {%0, %1};\n\tmov.b64 q, {%2, %3};\n\tadd.rn.f32x2 p, p, q;\n\tmov.b64 {%0, %1}, p;\n\t}"
                                 : "+f"(b[k]), "+f"(b[k + 1]) : "f"(m0), "f"(m1));
                }
            }
        }
    }
    float t = 0.f;
#pragma unroll
    for (int k = 0; k < 8; ++k) t += a[k] + b[k];
    if (t == 12345.678f) sink[0] = t;
}

}  // namespace ufb
