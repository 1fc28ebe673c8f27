// common.cuh -- shared declarations of the sm_100a UniFrac kernels (this library only).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace ufb {

constexpr int TILE = 128;          // samples per tile (stripe block edge), SURVEY 8a-5
constexpr int QUARTER = 32;        // sub-tile granularity of the sparse-aware row skipping

// device-side error word bits (plan step)
enum : uint32_t {
    ERRBIT_TREE = 1u,
    ERRBIT_TABLE = 2u,
    ERRBIT_EMPTY = 4u,
    ERRBIT_UNSUPPORTED = 8u,
};

// small block of words the plan step reads back
struct PlanWords {
    uint32_t err;          // ERRBIT_* mask
    int32_t n_roots;
    int32_t root;
    int32_t max_depth;
    unsigned long long n_internal;  // nodes with >= 1 child
};

__device__ __forceinline__ uint32_t lane_id() { return threadIdx.x & 31; }

}  // namespace ufb
