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

// Near-duplicate guard.  The separable forms finish with
// num = S_a + S_b - 2 M, which loses relative accuracy as d -> 0 (duplicated / proportional / replicate samples,
// PAPER.md:11 data reuse).  The finalize epilogues therefore append every pair whose distance comes out below
// GUARD_THETA to a device list, and k_guard (guard.cuh) recomputes exactly those pairs from the definition.
constexpr double GUARD_THETA = 0.0625;   // lowest threshold; the call raises it with the measured fixed-point error ratio
struct GuardList {
    uint2* pairs;            // (i, j) sample ids, i < j; NULL = guard off (debug forms)
    unsigned int* count;     // appended so far (may exceed cap; entries beyond cap are dropped)
    uint32_t cap;
    float theta;             // pairs with d < theta are listed
};
__device__ __forceinline__ void guard_note(const GuardList& g, double num, double den, uint32_t gi, uint32_t gj) {
    if (g.pairs && den > 0.0 && num < (double)g.theta * den) {
        const uint32_t k = atomicAdd(g.count, 1u);
        if (k < g.cap) g.pairs[k] = make_uint2(gi, gj);
    }
}

}  // namespace ufb
