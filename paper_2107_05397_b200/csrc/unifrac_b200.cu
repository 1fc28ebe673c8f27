// unifrac_b200.cu -- host side of the C ABI declared in include/unifrac_b200.h.
// Enqueues the plan (a-0), embedding (a-1..a-4) and stripe+finalize (a-5, a-6) kernels on one stream.
// No CPU fallback: every step of the path runs in the kernels of plan.cuh / embed.cuh / stripe.cuh.
#include "../../include/unifrac_b200.h"
#include "common.cuh"
#include "plan.cuh"
#include "embed.cuh"
#include "tail.cuh"
#include "stripe.cuh"
#include "gram.cuh"
#include "mid.cuh"
#include "dense.cuh"
#include "rates.cuh"
#include "mantel.cuh"
#include "rank.cuh"
#include "perm.cuh"
#include "zone.cuh"
#include "pcoa.cuh"
#include "guard.cuh"
#include "midg.cuh"

#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <string>
#include <type_traits>
#include <vector>
#include <algorithm>
#include <queue>
#include <mutex>

using namespace ufb;

namespace {

thread_local std::string g_cuda_err;
thread_local unifrac_stats_t g_stats;
thread_local unsigned long long* g_stats_pinned = nullptr;   // [2] stripe counters, pinned host
thread_local cudaEvent_t g_stats_event = nullptr;
thread_local int g_stats_event_dev = -1;                     // the device g_stats_event belongs to
thread_local bool g_stats_pending = false;

struct CudaFail { cudaError_t e; const char* what; int line; };
struct WorkspaceFail {};
struct StatusFail { int status; };
struct RetryExact {};        // the fixed-point error ratio is over budget: rerun without the fixed-point kernels
// unifrac_dm_host_multi: called after each segment of the finalizing kernel with the number of condensed ROWS that are final
// (rows [0, row_end) of out, guard included), so that their copy to the host can start while the rest is computed
typedef void (*ProgressFn)(void* user, long long row_end, cudaStream_t st);
// Fixed-point error ratio r (tail.cuh: k_quant_ratio): a distance d moves by at most ~2 r / d relative, so the guard
// threshold is raised to theta = max(1/16, r / QUANT_REL) -- every pair below it is recomputed from the definition -- and
// the call is rerun without the fixed-point kernels when theta would pass 1/2 (r > QUANT_RATIO_BUDGET).
constexpr double QUANT_REL = 2.5e-6;                 // 2 r / d <= 5e-6 for d >= theta
constexpr double QUANT_RATIO_BUDGET = 0.5 * QUANT_REL;

#define CU(x)                                                                                   \
    do {                                                                                        \
        cudaError_t e_ = (x);                                                                   \
        if (e_ != cudaSuccess) throw CudaFail{e_, #x, __LINE__};                                \
    } while (0)
#define CU_LAUNCH() CU(cudaGetLastError())

// bump of caller-provided (or stream-ordered) device allocations
struct Arena {
    unifrac_alloc_fn fn; void* user; cudaStream_t stream;
    cudaMemPool_t pool = nullptr;          // alloc == NULL: this pool instead of the device's default one (unifrac_dm_host)
    std::vector<void*> owned;
    size_t total = 0;
    void* get(size_t bytes) {
        if (bytes == 0) bytes = 256;
        bytes = (bytes + 255) & ~(size_t)255;
        void* p = nullptr;
        if (fn) { p = fn(bytes, user); if (!p) throw WorkspaceFail{}; }
        else {
            cudaError_t e = pool ? cudaMallocFromPoolAsync(&p, bytes, pool, stream) : cudaMallocAsync(&p, bytes, stream);
            if (e != cudaSuccess) { cudaGetLastError(); throw WorkspaceFail{}; }
            owned.push_back(p);
        }
        total += bytes;
        return p;
    }
    template <typename U> U* get_n(size_t n) { return reinterpret_cast<U*>(get(n * sizeof(U))); }
    void release() { for (void* p : owned) cudaFreeAsync(p, stream); owned.clear(); }
};

inline int cdiv(long long a, long long b) { return (int)((a + b - 1) / b); }
inline double env_double(const char* k, double d) { const char* e = getenv(k); return e ? atof(e) : d; }

// cuTensorMapEncodeTiled through the runtime's driver entry point (the library does not link libcuda)
typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*, const cuuint64_t*,
                                  const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle,
                                  CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
CUtensorMap make_rowmajor_map(void* base, CUtensorMapDataType dt, size_t esz, uint64_t cols, uint64_t rows, uint32_t box_cols,
                              uint32_t box_rows, CUtensorMapSwizzle swz)
{
    // resolved once (thread-safe static initialisation)
    static EncodeTiledFn fn = []() -> EncodeTiledFn {
        void* p = nullptr;
        cudaDriverEntryPointQueryResult qr;
        cudaError_t e = cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &qr);
        if (e != cudaSuccess || qr != cudaDriverEntryPointSuccess) { cudaGetLastError(); return nullptr; }
        return reinterpret_cast<EncodeTiledFn>(p);
    }();
    if (!fn) throw CudaFail{cudaErrorUnknown, "cuTensorMapEncodeTiled entry point", __LINE__};
    CUtensorMap m;
    cuuint64_t dims[2] = {cols, rows};
    cuuint64_t strides[1] = {cols * esz};        // bytes, dimension 1
    cuuint32_t box[2] = {box_cols, box_rows};
    cuuint32_t estr[2] = {1, 1};
    CUresult r = fn(&m, dt, 2, base, dims, strides, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE, swz,
                    CU_TENSOR_MAP_L2_PROMOTION_L2_256B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    if (r != CUDA_SUCCESS) throw CudaFail{cudaErrorInvalidValue, "cuTensorMapEncodeTiled", __LINE__};
    return m;
}
CUtensorMap make_u8_rowmajor_map(void* base, uint64_t cols, uint64_t rows, uint32_t box_cols, uint32_t box_rows)
{
    return make_rowmajor_map(base, CU_TENSOR_MAP_DATA_TYPE_UINT8, 1, cols, rows, box_cols, box_rows, CU_TENSOR_MAP_SWIZZLE_128B);
}

// tile pairs (I <= J) in BLK x BLK blocks of tiles, so that CTAs working on consecutive pairs share operand tiles in L2
// owner shard of the tile pair (I <= J): blocks of SHARD_BLOCK x SHARD_BLOCK tiles dealt round-robin (unifrac_b200.h)
inline int shard_of_tiles(int I, int J, int n_shards)
{
    const long long bi = I / SHARD_BLOCK, bj = J / SHARD_BLOCK;
    return (int)((bj * (bj + 1) / 2 + bi) % n_shards);
}
std::vector<int2> blocked_pairs(int n_tiles, int BLK, int shard = 0, int n_shards = 1)
{
    std::vector<int2> v;
    v.reserve((size_t)n_tiles * (n_tiles + 1) / 2 / n_shards + 1);
    for (int bi = 0; bi < n_tiles; bi += BLK)
        for (int bj = bi; bj < n_tiles; bj += BLK)
            for (int i = bi; i < std::min(n_tiles, bi + BLK); ++i)
                for (int j = std::max(i, bj); j < std::min(n_tiles, bj + BLK); ++j)
                    if (n_shards == 1 || shard_of_tiles(i, j, n_shards) == shard) v.push_back(make_int2(i, j));
    return v;
}

struct Timer {
    bool on; cudaStream_t s; cudaEvent_t ev[8]; int n = 0;
    Timer(bool on_, cudaStream_t s_) : on(on_), s(s_) { if (on) for (auto& e : ev) cudaEventCreate(&e); }
    ~Timer() { if (on) for (auto& e : ev) cudaEventDestroy(e); }
    void mark() { if (on && n < 8) cudaEventRecord(ev[n++], s); }
    float ms(int a, int b) { float m = 0; if (on && b < n) cudaEventElapsedTime(&m, ev[a], ev[b]); return m; }
};

// per-device scale factors of the cost-model rates (see run(): "The kernel rates below ...")
struct Calib { double f_atom = 1.0, f_red = 1.0, f_alu = 1.0; };
Calib calibration(int dev, cudaStream_t st)
{
    static std::mutex mu;
    static Calib cache[64];
    static bool have[64] = {};
    if (dev < 0 || dev >= 64) return Calib{};
    std::lock_guard<std::mutex> lock(mu);
    if (!have[dev]) {
        have[dev] = true;                                   // a failed probe leaves the reference rates in place
        const char* e = getenv("UNIFRAC_B200_CALIBRATE");
        if (!e || atoi(e) != 0) {
            unifrac_rates_t r{};
            if (unifrac_measure_rates(&r, st) == UNIFRAC_OK) {
                auto q = [](double measured, double ref) {
                    const double f = std::round(4.0 * measured / ref) / 4.0;
                    return f < 0.25 ? 0.25 : f > 4.0 ? 4.0 : f;
                };
                cache[dev].f_atom = q(r.smem_atomic_random_per_s, 2.57e12);     // 8.84 lanes/clk/SM x 148 SMs x 1.965 GHz
                cache[dev].f_red = q(r.l2_red_random_per_s, 1.94e11);
                cache[dev].f_alu = q(r.fmnmx_fadd_per_s, 3.48e13);
            }
        }
    }
    return cache[dev];
}

// Small device -> host read-backs of the planning steps.  A cudaMemcpyAsync would queue on the device-to-host copy engine BEHIND
// every copy submitted before it, from any stream -- in unifrac_dm_host_multi that is the previous variant's 5 GB result, and the
// next variant's planning (a dozen read-backs of a few words) then waited ~90 ms for it.  Here a one-block kernel writes the words
// into page-locked MAPPED host memory instead, and sync() hands them to their destinations after the stream synchronisation.
__global__ void k_readback(unsigned char* __restrict__ dst, const unsigned char* __restrict__ src, size_t bytes)
{
    for (size_t i = threadIdx.x; i < bytes; i += blockDim.x) dst[i] = src[i];
}
struct Readback {
    static constexpr size_t CAP = 64 * 1024, MAX_ITEM = 16 * 1024;
    struct Item { void* dst; size_t off, bytes; };
    cudaStream_t st;
    std::vector<Item> items;
    size_t used = 0;
    explicit Readback(cudaStream_t s) : st(s) {}
    static unsigned char* stage() {                       // one buffer per host thread, kept for the life of the process
        thread_local unsigned char* h = nullptr;
        thread_local bool failed = false;
        if (!h && !failed) {
            void* p = nullptr;
            if (cudaHostAlloc(&p, CAP, cudaHostAllocPortable | cudaHostAllocMapped) == cudaSuccess) h = static_cast<unsigned char*>(p);
            else { cudaGetLastError(); failed = true; }
        }
        return h;
    }
    void get(void* dst, const void* src, size_t bytes) {
        unsigned char* h = stage();
        void* d = nullptr;
        if (!h || bytes > MAX_ITEM || used + bytes > CAP || cudaHostGetDevicePointer(&d, h, 0) != cudaSuccess) {
            cudaGetLastError();
            CU(cudaMemcpyAsync(dst, src, bytes, cudaMemcpyDeviceToHost, st));
            return;
        }
        k_readback<<<1, 256, 0, st>>>(static_cast<unsigned char*>(d) + used, static_cast<const unsigned char*>(src), bytes);
        CU_LAUNCH();
        items.push_back({dst, used, bytes});
        used += (bytes + 15) & ~(size_t)15;
    }
    void sync() {
        CU(cudaStreamSynchronize(st));
        unsigned char* h = stage();
        for (const Item& it : items) memcpy(it.dst, h + it.off, it.bytes);
        items.clear();
        used = 0;
    }
};

// stable LSD radix sort of (key, position) pairs (rank.cuh); the sort buffers are shared between the sorts of a call
struct RankBufs { void* keys[2]; uint32_t* idx[2]; uint32_t* hist; uint32_t* offs; uint32_t* blast; unsigned nb; unsigned long long per_block; };
template <typename T>
RankBufs make_rank_bufs(Arena& A, unsigned long long P, int n_sm)
{
    RankBufs B{};
    B.nb = (unsigned)n_sm * 8;
    B.per_block = ((P + B.nb - 1) / B.nb + RADIX_TILE - 1) / RADIX_TILE * RADIX_TILE;
    const size_t ksz = sizeof(typename RankKey<T>::K);
    for (int i = 0; i < 2; ++i) { B.keys[i] = A.get(P * ksz); B.idx[i] = A.get_n<uint32_t>(P); }
    B.hist = A.get_n<uint32_t>((size_t)256 * B.nb + 1);
    B.offs = A.get_n<uint32_t>((size_t)256 * B.nb + 1);
    B.blast = A.get_n<uint32_t>(B.nb);
    return B;
}
// returns the buffer index that holds the sorted keys / positions
template <typename T>
int radix_sort(const T* v, unsigned long long P, const RankBufs& B, cudaStream_t st)
{
    using K = typename RankKey<T>::K;
    K* keys[2] = {reinterpret_cast<K*>(B.keys[0]), reinterpret_cast<K*>(B.keys[1])};
    int src = 0;                                                     // pass 0 reads v[] itself and writes buffer 0
    for (int pass = 0; pass < RankKey<T>::PASSES; ++pass) {
        const int shift = 8 * pass, dst = pass == 0 ? 0 : src ^ 1;
        if (pass == 0) k_radix_hist<T, true><<<B.nb, RADIX_THREADS, 0, st>>>(v, nullptr, P, B.per_block, shift, B.hist);
        else k_radix_hist<T, false><<<B.nb, RADIX_THREADS, 0, st>>>(nullptr, keys[src], P, B.per_block, shift, B.hist);
        CU_LAUNCH();
        k_exclusive_scan<uint32_t><<<1, 1024, 0, st>>>((int)(256 * B.nb), B.hist, B.offs); CU_LAUNCH();
        constexpr size_t ssm = radix_scatter_smem<K>();
        if (pass == 0) {
            CU(cudaFuncSetAttribute(k_radix_scatter<T, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)ssm));
            k_radix_scatter<T, true><<<B.nb, RADIX_THREADS, ssm, st>>>(v, nullptr, nullptr, P, B.per_block, shift, B.offs, keys[dst], B.idx[dst]);
        } else {
            CU(cudaFuncSetAttribute(k_radix_scatter<T, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)ssm));
            k_radix_scatter<T, false><<<B.nb, RADIX_THREADS, ssm, st>>>(nullptr, keys[src], B.idx[src], P, B.per_block, shift, B.offs, keys[dst], B.idx[dst]);
        }
        CU_LAUNCH();
        src = dst;
    }
    return src;
}
// twice the 1-based average ranks of the P values v[] (exact 32-bit integers) -> rank2[]
constexpr int RANK_WINDOW_BITS = 23;                                 // P < 2^31: at most 256 windows
template <typename T>
void rank_transform(const T* v, unsigned long long P, uint32_t* rank2, const RankBufs& B, cudaStream_t st)
{
    using K = typename RankKey<T>::K;
    const int src = radix_sort<T>(v, P, B, st);
    K* keys[2] = {reinterpret_cast<K*>(B.keys[0]), reinterpret_cast<K*>(B.keys[1])};
    uint32_t* start = reinterpret_cast<uint32_t*>(keys[src ^ 1]);     // the other key buffer and position buffer are free now
    uint32_t* rlen = B.idx[src ^ 1];
    k_rank_block_heads<K><<<B.nb, RADIX_THREADS, 0, st>>>(keys[src], P, B.per_block, B.blast); CU_LAUNCH();
    k_rank_starts<K><<<B.nb, RADIX_THREADS, 0, st>>>(keys[src], P, B.per_block, B.blast, start, rlen); CU_LAUNCH();
    // back to the original positions: rank values in sorted order, then the (position, value) pairs partitioned by the top
    // 8 bits of the position (windows of 2^RANK_WINDOW_BITS ranks = 32 MB, L2-resident), then the scatter inside the windows
    uint32_t* val = reinterpret_cast<uint32_t*>(keys[src]);           // the sorted keys are no longer needed
    k_rank_value<<<B.nb * 4, 256, 0, st>>>(start, rlen, P, val); CU_LAUNCH();
    if ((P >> RANK_WINDOW_BITS) == 0) {                               // one window: scatter directly
        k_rank_place<<<(unsigned)cdiv((long long)P, RANK_PLACE_PER_BLOCK), 256, 0, st>>>(B.idx[src], val, P, rank2); CU_LAUNCH();
        return;
    }
    uint32_t* pos_out = start;                                        // start / rlen are free once val is written
    uint32_t* val_out = rlen;
    k_radix_hist<uint32_t, false><<<B.nb, RADIX_THREADS, 0, st>>>(nullptr, B.idx[src], P, B.per_block, RANK_WINDOW_BITS, B.hist); CU_LAUNCH();
    k_exclusive_scan<uint32_t><<<1, 1024, 0, st>>>((int)(256 * B.nb), B.hist, B.offs); CU_LAUNCH();
    constexpr size_t ssm = radix_scatter_smem<uint32_t>();
    CU(cudaFuncSetAttribute(k_radix_scatter<uint32_t, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)ssm));
    k_radix_scatter<uint32_t, false><<<B.nb, RADIX_THREADS, ssm, st>>>(nullptr, B.idx[src], val, P, B.per_block, RANK_WINDOW_BITS, B.offs,
                                                                       pos_out, val_out);
    CU_LAUNCH();
    k_rank_place<<<(unsigned)cdiv((long long)P, RANK_PLACE_PER_BLOCK), 256, 0, st>>>(pos_out, val_out, P, rank2); CU_LAUNCH();
}

template <typename T>
void run(int32_t n, const int32_t* parent, const double* len, const int32_t* postorder, unifrac_csr_t tab,
         int32_t N, int weighted, void* out, Arena& A, uint32_t flags, cudaStream_t st, int shard, int n_shards, bool is_retry,
         ProgressFn progress = nullptr, void* progress_user = nullptr)
{
    Readback RDB(st);                   // the planning steps' small read-backs (no copy engine: see struct Readback)
    const bool validate = !(flags & UNIFRAC_FLAG_SKIP_VALIDATION);
    const bool timing = getenv("UNIFRAC_B200_TIMING") && atoi(getenv("UNIFRAC_B200_TIMING")) != 0;
    Timer tm(timing, st);
    unsigned launches = 0;
    tm.mark();
    const int TB = 256;
    int dev_id = 0, n_sm_dev = 0;
    CU(cudaGetDevice(&dev_id));
    CU(cudaDeviceGetAttribute(&n_sm_dev, cudaDevAttrMultiProcessorCount, dev_id));

    // ------------------------------------------------------------------ UNIFRAC_FLAG_RICHNESS_ZONES (weighted fp32): samples in
    // richness order (perm.cuh) and a per-(branch, tile) split between the dense kernel and the join (zone.cuh)
    const bool skip_path = std::is_same<T, float>::value && weighted && (flags & UNIFRAC_FLAG_RICHNESS_ZONES) &&
                           !(flags & (UNIFRAC_FLAG_ABSDIFF | UNIFRAC_FLAG_LITERAL | UNIFRAC_FLAG_NO_TAIL | UNIFRAC_FLAG_SPARSE_STRIPE |
                                      UNIFRAC_FLAG_NO_MID | UNIFRAC_FLAG_ALL_TAIL));
    uint32_t* inv_perm = nullptr;                 // sample -> position; NULL = identity
    void* const out_user = out;
    if (skip_path && n_shards == 1 && N > TILE && env_double("UNIFRAC_B200_PERMUTE", 1) != 0) {
        uint32_t* key = A.get_n<uint32_t>(N);
        unsigned int* bad = A.get_n<unsigned int>(1);
        CU(cudaMemsetAsync(bad, 0, sizeof(unsigned int), st));
        k_perm_keys<<<cdiv(N, TB), TB, 0, st>>>(N, tab.indptr, key, bad); CU_LAUNCH(); ++launches;
        unsigned int h_bad = 0; long long h_nnz = 0;
        RDB.get(&h_bad, bad, sizeof(h_bad));
        RDB.get(&h_nnz, tab.indptr + N, sizeof(h_nnz));
        RDB.sync();
        if (!h_bad && h_nnz >= 0 && h_nnz < (1ll << 32)) {       // otherwise: validation below reports what is wrong
            RankBufs RB = make_rank_bufs<uint32_t>(A, (unsigned long long)N, n_sm_dev);
            const int src = radix_sort<uint32_t>(key, (unsigned long long)N, RB, st);
            launches += 12;
            const uint32_t* perm = RB.idx[src];                  // position -> sample
            uint32_t* rowlen = A.get_n<uint32_t>((size_t)N + 1);
            uint32_t* rowoff = A.get_n<uint32_t>((size_t)N + 1);
            inv_perm = A.get_n<uint32_t>(N);
            k_perm_rowlen<<<cdiv(N, TB), TB, 0, st>>>(N, tab.indptr, perm, rowlen, inv_perm); CU_LAUNCH(); ++launches;
            k_exclusive_scan<uint32_t><<<1, 1024, 0, st>>>(N, rowlen, rowoff); CU_LAUNCH(); ++launches;
            int64_t* p_indptr = A.get_n<int64_t>((size_t)N + 1);
            int32_t* p_indices = A.get_n<int32_t>(h_nnz ? (size_t)h_nnz : 1);
            int32_t* p_counts = A.get_n<int32_t>(h_nnz ? (size_t)h_nnz : 1);
            k_perm_gather<<<cdiv((long long)N * 32, TB), TB, 0, st>>>(N, tab.indptr, tab.indices, tab.counts, perm, rowoff, p_indptr, p_indices, p_counts);
            CU_LAUNCH(); ++launches;
            tab.indptr = p_indptr; tab.indices = p_indices; tab.counts = p_counts;      // from here on: position space
            out = A.get_n<T>((size_t)N * (N - 1) / 2);
        }
    }

    // ------------------------------------------------------------------ a-0 plan / validate
    PlanWords* pw = A.get_n<PlanWords>(1);
    int32_t* child_count = A.get_n<int32_t>(n);
    int32_t* seen = A.get_n<int32_t>(n);
    int32_t* pos = A.get_n<int32_t>(n);
    unsigned long long* Tsum = A.get_n<unsigned long long>(N);
    CU(cudaMemsetAsync(pw, 0, sizeof(PlanWords), st));
    CU(cudaMemsetAsync(child_count, 0, sizeof(int32_t) * n, st));
    k_tree_check<<<cdiv(n, TB), TB, 0, st>>>(n, parent, len, child_count, pw, validate); CU_LAUNCH(); ++launches;
    k_root_check<<<1, 1, 0, st>>>(pw); CU_LAUNCH(); ++launches;
    if (validate) {
        CU(cudaMemsetAsync(seen, 0, sizeof(int32_t) * n, st));
        k_post_check1<<<cdiv(n, TB), TB, 0, st>>>(n, postorder, seen, pos, pw); CU_LAUNCH(); ++launches;
        k_post_check2<<<cdiv(n, TB), TB, 0, st>>>(n, parent, postorder, pos, pw); CU_LAUNCH(); ++launches;
    }
    PlanWords h{};
    RDB.get(&h, pw, sizeof(h));
    RDB.sync();
    if (h.err & ERRBIT_TREE) throw StatusFail{UNIFRAC_ERR_INVALID_TREE};

    k_csr_check<<<cdiv((long long)N * 32, TB), TB, 0, st>>>(n, N, tab.indptr, tab.indices, tab.counts, child_count,
                                                             Tsum, pw, validate); CU_LAUNCH(); ++launches;
    // depths by pointer jumping
    int32_t* anc[2] = {A.get_n<int32_t>(n), A.get_n<int32_t>(n)};
    int32_t* dist[2] = {A.get_n<int32_t>(n), A.get_n<int32_t>(n)};
    k_jump_init<<<cdiv(n, TB), TB, 0, st>>>(n, parent, anc[0], dist[0]); CU_LAUNCH(); ++launches;
    int cur = 0;
    for (long long reach = 1; reach < n; reach <<= 1) {
        k_jump_round<<<cdiv(n, TB), TB, 0, st>>>(n, anc[cur], dist[cur], anc[cur ^ 1], dist[cur ^ 1]); CU_LAUNCH(); ++launches;
        cur ^= 1;
    }
    const int32_t* depth = dist[cur];
    uint32_t* hist = A.get_n<uint32_t>((size_t)n + 1);
    CU(cudaMemsetAsync(hist, 0, sizeof(uint32_t) * ((size_t)n + 1), st));
    k_level_hist<<<cdiv(n, TB), TB, 0, st>>>(n, depth, child_count, hist, pw); CU_LAUNCH(); ++launches;
    RDB.get(&h, pw, sizeof(h));
    RDB.sync();
    if (h.err & ERRBIT_TABLE) throw StatusFail{UNIFRAC_ERR_INVALID_TABLE};
    if (h.err & ERRBIT_EMPTY) throw StatusFail{UNIFRAC_ERR_EMPTY_SAMPLE};
    if (h.err & ERRBIT_UNSUPPORTED) throw StatusFail{UNIFRAC_ERR_UNSUPPORTED};
    const int root = h.root;
    const int n_levels = h.max_depth + 1;
    const size_t n_internal = (size_t)h.n_internal;
    std::vector<uint32_t> h_hist(n_levels), h_off(n_levels + 1);
    RDB.get(h_hist.data(), hist, sizeof(uint32_t) * n_levels);
    RDB.sync();
    h_off[0] = 0;
    for (int d = 0; d < n_levels; ++d) h_off[d + 1] = h_off[d] + h_hist[d];
    uint32_t* cursor = A.get_n<uint32_t>(n_levels);
    int32_t* level_nodes = A.get_n<int32_t>(n_internal ? n_internal : 1);
    CU(cudaMemcpyAsync(cursor, h_off.data(), sizeof(uint32_t) * n_levels, cudaMemcpyHostToDevice, st));
    k_level_fill<<<cdiv(n, TB), TB, 0, st>>>(n, depth, child_count, cursor, level_nodes); CU_LAUNCH(); ++launches;
    uint32_t* child_off = A.get_n<uint32_t>((size_t)n + 1);
    uint32_t* child_cur = A.get_n<uint32_t>((size_t)n + 1);
    int32_t* child_idx = A.get_n<int32_t>(n);
    k_exclusive_scan<int32_t><<<1, 1024, 0, st>>>(n, child_count, child_off); CU_LAUNCH(); ++launches;
    CU(cudaMemcpyAsync(child_cur, child_off, sizeof(uint32_t) * ((size_t)n + 1), cudaMemcpyDeviceToDevice, st));
    k_child_fill<<<cdiv(n, TB), TB, 0, st>>>(n, parent, child_cur, child_idx); CU_LAUNCH(); ++launches;
    tm.mark();

    // ------------------------------------------------------------------ a-1/a-2 on presence bits -> n_v -> head/mid/tail classes
    const uint32_t NW = ((uint32_t)cdiv(N, 32) + 3u) & ~3u, NW4 = NW / 4;
    uint32_t* nv = A.get_n<uint32_t>(n);
    uint32_t* ne = A.get_n<uint32_t>(n);
    uint8_t* cls = A.get_n<uint8_t>(n);
    uint32_t* tcnt = A.get_n<uint32_t>(n);
    uint32_t* tptr = A.get_n<uint32_t>((size_t)n + 1);
    unsigned long long* work = A.get_n<unsigned long long>(28);
    CU(cudaMemsetAsync(work, 0, sizeof(unsigned long long) * 28, st));
    uint32_t* bits = A.get_n<uint32_t>((size_t)n * NW);
    {
        CU(cudaMemsetAsync(bits, 0, sizeof(uint32_t) * (size_t)n * NW, st));
        k_bits_scatter<<<cdiv((long long)N * 32, TB), TB, 0, st>>>(N, tab.indptr, tab.indices, tab.counts, bits, NW); CU_LAUNCH(); ++launches;
        for (int d = n_levels - 1; d >= 0; --d) {
            const uint32_t cntl = h_hist[d];
            if (!cntl) continue;
            k_bits_pull<<<cdiv((long long)cntl * NW4, TB), TB, 0, st>>>(level_nodes + h_off[d], (int)cntl, root, child_off, child_idx,
                                                                       reinterpret_cast<uint4*>(bits), NW4);
            CU_LAUNCH(); ++launches;
        }
        k_bits_count<<<cdiv((long long)n * 32, TB), TB, 0, st>>>(n, parent, len, reinterpret_cast<const uint4*>(bits), NW4, nv, ne); CU_LAUNCH(); ++launches;
    }
    k_work_counts<<<cdiv(n, TB), TB, 0, st>>>(n, nv, (unsigned long long)N, work); CU_LAUNCH(); ++launches;
    const bool gram = std::is_same<T, float>::value && !weighted &&
                      !(flags & (UNIFRAC_FLAG_NO_TENSOR | UNIFRAC_FLAG_ABSDIFF | UNIFRAC_FLAG_LITERAL | UNIFRAC_FLAG_ALL_TAIL));
    const bool mid_ok = std::is_same<T, float>::value &&
                        !(flags & (UNIFRAC_FLAG_NO_MID | UNIFRAC_FLAG_NO_TAIL | UNIFRAC_FLAG_ABSDIFF | UNIFRAC_FLAG_LITERAL | UNIFRAC_FLAG_ALL_TAIL));
    // Per-branch class thresholds on C(n_v,2) from measured rates (all can be
    // overridden through the environment for tuning):
    //   R_tail  global RED.ADD pair updates / s           R_mid   shared-memory integer-atomic pair updates / s
    //   R_head  dense-equivalent pair updates / s of k_stripe;  Gram kernel: seconds per branch = tile pairs * 512 B / operand rate
    const int n_tiles = cdiv(N, TILE);
    const double Pd = 0.5 * (double)N * (double)(N - 1), n_tp = 0.5 * (double)n_tiles * (n_tiles + 1);
    auto envd = [](const char* k, double d) { const char* e = getenv(k); return e ? atof(e) : d; };
    // The kernel rates below were measured on this pool's B200.  Once per process and device the unit rates they rest on
    // (shared-memory atomics, L2 REDs, the FMNMX + FADD mix) are probed (unifrac_measure_rates, ~20 ms) and the kernel rates
    // are scaled by measured / reference, in steps of 1/4 so that probe noise cannot move the split (on a B200: all 1.0).
    const Calib cal = calibration(dev_id, st);
    // with the grouped join (midg.cuh) a mid update costs about half of what it costs in k_mid alone (sweeps: profiles/r02_summary.md 4d)
    const bool groups_expected = std::is_same<T, float>::value && !skip_path && envd("UNIFRAC_B200_MID_GROUPS", 1.0) != 0.0;
    const double R_tail = envd("UNIFRAC_B200_R_TAIL", 1.6e11 * cal.f_red), R_mid = envd("UNIFRAC_B200_R_MID", (groups_expected ? 3.5e12 : 1.6e12) * cal.f_atom);
    const double R_head = envd("UNIFRAC_B200_R_HEAD", (std::is_same<T, float>::value ? 1.4e13 : 3.3e12) * cal.f_alu), gram_Bps = envd("UNIFRAC_B200_GRAM_BPS", 1.15e13);
    // the rows that compete with the Gram kernel are sparse (a few entries per tile), where k_mid's per-entry overhead
    // halves its update rate (measured 5.9e11 /s at Large against 1.3e12 - 1.6e12 /s for the denser rows of the weighted variant)
    const double R_mid_head = gram ? envd("UNIFRAC_B200_R_MID_SPARSE", (groups_expected ? 8e11 : 5.5e11) * cal.f_atom) : R_mid;
    const double c_ent = envd("UNIFRAC_B200_MID_ENT_S", groups_expected ? 4e-12 : 3e-12);         // seconds per (mid entry, tile pair) visit of the join kernel
    const double head_s = gram ? n_tp * 512.0 / gram_Bps : Pd / R_head;  // seconds per head branch
    double c2_head, c2_mid;
    if (mid_ok) {
        // mid row: n_v entries, each visited once per tile J >= its own tile (~ n_tiles / 2 visits) + C(n_v,2) / R_mid;
        // tail row: C(n_v,2) / R_tail  =>  mid wins for n_v > 1 + n_tiles * c_ent / (1/R_tail - 1/R_mid)
        const double nstar = 1.0 + (double)n_tiles * c_ent / (1.0 / R_tail - 1.0 / R_mid);
        c2_head = head_s * R_mid_head; c2_mid = 0.5 * nstar * (nstar - 1.0);
        if (c2_mid > c2_head) c2_mid = c2_head;
    } else { c2_head = head_s * R_tail; c2_mid = INFINITY; }
    uint32_t force = 0;
    if (flags & (UNIFRAC_FLAG_NO_TAIL | UNIFRAC_FLAG_ABSDIFF | UNIFRAC_FLAG_LITERAL)) force = 1;   // NO_TAIL + Gram = dense GEMM over every branch
    else if (flags & UNIFRAC_FLAG_ALL_TAIL) force = 2;
    // the weighted variant keeps an entry list (counts -> values) for every row; unweighted only for mid / tail rows
    k_classify<<<cdiv(n, TB), TB, 0, st>>>(n, nv, ne, weighted, c2_head, c2_mid, force, cls, tcnt, work + 8); CU_LAUNCH(); ++launches;
    k_exclusive_scan<uint32_t><<<1, 1024, 0, st>>>(n, tcnt, tptr); CU_LAUNCH(); ++launches;
    uint32_t* cptr = nullptr;                                  // weighted: by-tip (CSC) offsets of the table
    if (weighted) {
        uint32_t* tipc = A.get_n<uint32_t>(n);
        cptr = A.get_n<uint32_t>((size_t)n + 1);
        k_tip_mark<<<cdiv(n, TB), TB, 0, st>>>(n, child_count, ne, tipc, work + 16); CU_LAUNCH(); ++launches;
        k_exclusive_scan<uint32_t><<<1, 1024, 0, st>>>(n, tipc, cptr); CU_LAUNCH(); ++launches;
    }
    unsigned long long h_work[18];
    RDB.get(h_work, work, sizeof(h_work));
    RDB.sync();
    const unsigned long long head_rows = h_work[8], tail_rows = h_work[9], tail_updates = h_work[10], tail_entries = h_work[11];
    const unsigned long long mid_rows = h_work[12], mid_updates = h_work[13], nnz_pos = h_work[16], mid_entries = h_work[17];
    if (tail_entries >= (1ull << 32) || nnz_pos >= (1ull << 32)) throw StatusFail{UNIFRAC_ERR_UNSUPPORTED};
    uint32_t* ts = A.get_n<uint32_t>(tail_entries ? tail_entries : 1);
    T* tv = A.get_n<T>(tail_entries ? tail_entries : 1);

    // ------------------------------------------------------------------ tensor-core Gram path: u8 operand matrices from the bits
    bool use_gram = gram && head_rows > 0 && head_rows < (1ull << 23);
    // CUDA-core head path: dense min-GEMM kernel (dense.cuh) unless a debug form needs the sparse-aware compact-row kernel
    // weighted fp32, default flags: per-(branch, tile) split between k_zone and the join (zone.cuh) instead of the per-branch one
    const bool skip_on = skip_path && mid_ok && n_tiles <= ROWCUT_MAX_TILES && head_rows + mid_rows > 0 && head_rows + mid_rows < (1ull << 23);
    const bool dense_head = !skip_on && !use_gram && !(flags & (UNIFRAC_FLAG_ABSDIFF | UNIFRAC_FLAG_LITERAL | UNIFRAC_FLAG_NO_TAIL | UNIFRAC_FLAG_SPARSE_STRIPE));
    double* uval = nullptr;
    double* uerr = nullptr;                                    // Gram path: |u~_v - len_v| of the fixed-point head lengths
    uint8_t* XG[4] = {nullptr, nullptr, nullptr, nullptr};
    uint32_t K_pad = 0;
    int gram_q = 0;
    uint32_t* hrank = nullptr;                                 // head rank of every node (exclusive scan of the head marks)
    int32_t* hrows = nullptr;                                  // head rank -> node id
    if (head_rows > 0 && (use_gram || weighted || dense_head)) {
        uint32_t* is_head = A.get_n<uint32_t>(n);
        hrank = A.get_n<uint32_t>((size_t)n + 1);
        k_mark_class<<<cdiv(n, TB), TB, 0, st>>>(n, cls, CLS_HEAD, is_head); CU_LAUNCH(); ++launches;
        k_exclusive_scan<uint32_t><<<1, 1024, 0, st>>>(n, is_head, hrank); CU_LAUNCH(); ++launches;
    }
    if (use_gram) {
        unsigned long long* lmax = work + 14;
        k_gram_lenmax<<<cdiv(n, TB), TB, 0, st>>>(n, cls, len, lmax); CU_LAUNCH(); ++launches;
        unsigned long long h_lmax = 0;
        RDB.get(&h_lmax, lmax, sizeof(h_lmax));
        RDB.sync();
        double lm; memcpy(&lm, &h_lmax, sizeof(lm));
        int ex = 0; frexp(lm, &ex);
        const uint32_t K = (uint32_t)head_rows;
        K_pad = (K + GRAM_BK - 1) / GRAM_BK * GRAM_BK;
        int max_shift = 7;                                  // s32 accumulators: 2^shift * 255 * K_pad < 2^31
        while (max_shift > 0 && (255ull << max_shift) * K_pad >= (1ull << 31)) --max_shift;
        gram_q = 24 - ex + max_shift;                       // lmax * 2^q in [2^(23 + shift), 2^(24 + shift))
        const size_t Npad = (size_t)NW * 32;
        hrows = A.get_n<int32_t>(K_pad);
        uint32_t* Lq = A.get_n<uint32_t>(K_pad);
        uval = A.get_n<double>(n);
        uerr = A.get_n<double>(n);
        for (auto& x : XG) x = A.get_n<uint8_t>((size_t)K_pad * Npad);
        k_gram_quant<<<cdiv(n, TB), TB, 0, st>>>(n, cls, hrank, len, gram_q, max_shift, hrows, Lq, uval, uerr); CU_LAUNCH(); ++launches;
        k_gram_expand<<<cdiv((long long)K_pad * NW, TB), TB, 0, st>>>(K, K_pad, hrows, Lq, bits, NW, XG[0], XG[1], XG[2], XG[3]);
        CU_LAUNCH(); ++launches;
    }
    tm.mark();

    // ------------------------------------------------------------------ a-1 / a-2 counts in rank layout (weighted only)
    uint32_t* cnt = nullptr;
    if (weighted) {
        cnt = A.get_n<uint32_t>(tail_entries ? tail_entries : 1);
        uint32_t* csc_s = A.get_n<uint32_t>(nnz_pos ? nnz_pos : 1);
        uint32_t* csc_c = A.get_n<uint32_t>(nnz_pos ? nnz_pos : 1);
        uint32_t* ccur = A.get_n<uint32_t>(n);
        CU(cudaMemsetAsync(ccur, 0, sizeof(uint32_t) * n, st));
        k_csc_fill<<<cdiv((long long)N * 32, TB), TB, 0, st>>>(N, tab.indptr, tab.indices, tab.counts, cptr, ccur, csc_s, csc_c); CU_LAUNCH(); ++launches;
        int dev0 = 0, n_sm0 = 0;
        CU(cudaGetDevice(&dev0));
        CU(cudaDeviceGetAttribute(&n_sm0, cudaDevAttrMultiProcessorCount, dev0));
        int wpb = (int)std::min<size_t>(8, ((size_t)96 << 10) / ((size_t)NW * 4));
        if (wpb < 1) throw StatusFail{UNIFRAC_ERR_UNSUPPORTED};
        const size_t tsm = (size_t)wpb * NW * 4;
        CU(cudaFuncSetAttribute(k_tip_cnt, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)tsm));
        k_tip_cnt<<<n_sm0 * 8, wpb * 32, tsm, st>>>(n, child_count, ne, cptr, csc_s, csc_c, bits, NW, tptr, cnt); CU_LAUNCH(); ++launches;
        for (int d = n_levels - 1; d >= 0; --d) {            // deepest parents first
            const uint32_t cntl = h_hist[d];
            if (!cntl) continue;
            k_cnt_pull<<<cdiv((long long)cntl * 32, TB), TB, 0, st>>>(level_nodes + h_off[d], (int)cntl, root, child_off, child_idx,
                                                                     bits, NW, tptr, cnt);
            CU_LAUNCH(); ++launches;
        }
    }
    // ------------------------------------------------------------------ a-3 / a-4 values, sample ids, side sums
    double* sums = A.get_n<double>((size_t)n_tiles * TILE * 3);
    double* qerr = sums + (size_t)n_tiles * TILE;             // [2 * samples] per-sample sum / sum of squares of the fixed-point errors
    CU(cudaMemsetAsync(sums, 0, sizeof(double) * (size_t)n_tiles * TILE * 3, st));
    k_values<T><<<cdiv((long long)n * 32, TB), TB, 0, st>>>(n, nv, tcnt, tptr, len, uval, bits, NW, cnt, Tsum, ts, tv, sums, uerr, qerr); CU_LAUNCH(); ++launches;

    // ------------------------------------------------------------------ head rows of the CUDA-core stripe kernel: compact dense per-tile rows
    const uint32_t nwords = (uint32_t)cdiv(n, 32);
    uint32_t* rflags = nullptr; uint32_t* rrank = nullptr;
    T** tileE = nullptr; uint8_t** tileQ = nullptr;
    uint64_t embed_rows = 0;
    T* Edense = nullptr;
    const size_t Npad = (size_t)n_tiles * TILE;
    uint32_t Kd_pad = 0;
    const bool dense16 = dense_head && std::is_same<T, float>::value && envd("UNIFRAC_B200_DENSE16", 1) != 0;   // fp32: 16 consumer warps, mixed forms
    // skip path (zone.cuh)
    uint32_t sk_n = 0, sk_KE = 0;
    int32_t* sk_rows = nullptr; uint32_t* sk_base = nullptr; uint32_t* sk_len = nullptr; uint32_t* sk_cut = nullptr; float* sk_E = nullptr; double* sk_H = nullptr;
    std::vector<uint32_t> h_cut;
    unsigned long long h_skstat[2] = {0, 0};
    double* hsum = nullptr;
    if (dense16) {
        hsum = A.get_n<double>((size_t)n_tiles * TILE);
        CU(cudaMemsetAsync(hsum, 0, sizeof(double) * (size_t)n_tiles * TILE, st));
    }
    if (dense_head) {
        constexpr int BK = DenseCfg<T>::BK;
        Kd_pad = (uint32_t)((head_rows + BK - 1) / BK * BK);
        if (Kd_pad == 0) Kd_pad = BK;
        Edense = A.get_n<T>((size_t)Kd_pad * Npad);
        CU(cudaMemsetAsync(Edense + (size_t)head_rows * Npad, 0, sizeof(T) * (Kd_pad - (size_t)head_rows) * Npad, st));
        if (head_rows > 0) {
            hrows = A.get_n<int32_t>(head_rows);
            k_head_rows<<<cdiv(n, TB), TB, 0, st>>>(n, cls, hrank, hrows); CU_LAUNCH(); ++launches;
            {
                // fp32 accuracy: K order = ascending n_v (stable), so the few root-adjacent branches whose u~ is O(0.1) for every
                // sample come last and are folded into fp64 stage by stage (k_dense) instead of swamping the fp32 partial
                // sums that the thousands of small terms are added to.  Sorted on the device
                // (stable radix sort, rank.cuh): no host work on the data path.
                uint32_t* hkey = A.get_n<uint32_t>(head_rows);
                int32_t* hsorted = A.get_n<int32_t>(head_rows);
                k_head_keys<<<cdiv((long long)head_rows, TB), TB, 0, st>>>((uint32_t)head_rows, hrows, nv, hkey); CU_LAUNCH(); ++launches;
                RankBufs RBh = make_rank_bufs<uint32_t>(A, head_rows, n_sm_dev);
                const int hsrc = radix_sort<uint32_t>(hkey, head_rows, RBh, st);
                launches += 12;
                k_head_reorder<<<cdiv((long long)head_rows, TB), TB, 0, st>>>((uint32_t)head_rows, hrows, RBh.idx[hsrc], hsorted); CU_LAUNCH(); ++launches;
                hrows = hsorted;
            }
            uint32_t* hpref = nullptr;
            if (weighted) {
                hpref = A.get_n<uint32_t>((size_t)head_rows * n_tiles);
                k_head_pref<<<cdiv((long long)head_rows * 32, TB), TB, 0, st>>>((uint32_t)head_rows, hrows, bits, NW, n_tiles, hpref); CU_LAUNCH(); ++launches;
            }
            k_head_dense<T><<<cdiv((long long)head_rows * n_tiles * 32, TB), TB, 0, st>>>((uint32_t)head_rows, hrows, len, bits, NW, n_tiles, tptr, hpref,
                                                                                         weighted ? tv : nullptr, Edense, Npad,
                                                                                         hsum);
            CU_LAUNCH(); ++launches;
            embed_rows = head_rows * (uint64_t)n_tiles;
        }
    } else if (skip_on) {
        // rows in (D_v ascending, n_v descending) order, the cut table, the dense rows k_zone needs (zone.cuh)
        sk_n = (uint32_t)(head_rows + mid_rows);
        int32_t* lnode = A.get_n<int32_t>(sk_n);
        unsigned int* lcount = reinterpret_cast<unsigned int*>(work + 20);
        k_list_compact<<<cdiv(n, TB), TB, 0, st>>>(n, cls, lnode, lcount); CU_LAUNCH(); ++launches;
        unsigned long long* keys = A.get_n<unsigned long long>(sk_n);
        // cost model of k_row_cut in SM-clocks (measured on B200, sweeps in profiles/r02_summary.md; overridable for tuning):
        // one (row, tile pair) of k_zone, pair updates per clock of the join, one (entry, tile pair) visit of the join
        CutModel CM{(float)env_double("UNIFRAC_B200_ZONE_C0", 310.0), (float)(0.5 / env_double("UNIFRAC_B200_JOIN_RATE", 4.64)),
                    (float)env_double("UNIFRAC_B200_JOIN_ENT", 0.87)};
        k_row_cut<<<cdiv(sk_n, ROWCUT_WARPS), ROWCUT_WARPS * 32, 0, st>>>(sk_n, lnode, bits, NW, n_tiles, (uint32_t)N, CM, keys); CU_LAUNCH(); ++launches;
        RankBufs RB = make_rank_bufs<unsigned long long>(A, sk_n, n_sm_dev);
        const int src = radix_sort<unsigned long long>(keys, sk_n, RB, st);
        launches += 24;
        sk_rows = A.get_n<int32_t>(sk_n);
        uint32_t* Dr = A.get_n<uint32_t>(sk_n);
        sk_base = A.get_n<uint32_t>(sk_n);
        sk_len = A.get_n<uint32_t>(sk_n);
        k_rows_from_sort<<<cdiv(sk_n, TB), TB, 0, st>>>(sk_n, RB.idx[src], reinterpret_cast<const unsigned long long*>(RB.keys[src]), lnode, tptr, nv,
                                                         sk_rows, Dr, sk_base, sk_len); CU_LAUNCH(); ++launches;
        sk_cut = A.get_n<uint32_t>((size_t)n_tiles + 1);
        k_cut_table<<<cdiv(n_tiles + 1, TB), TB, 0, st>>>(n_tiles, sk_n, Dr, ZONE_BK, sk_cut); CU_LAUNCH(); ++launches;
        k_cut_stats<<<cdiv((long long)sk_n * 32, TB), TB, 0, st>>>(sk_n, sk_rows, bits, NW, n_tiles, sk_cut, work + 21); CU_LAUNCH(); ++launches;
        h_cut.resize((size_t)n_tiles + 1);
        RDB.get(h_cut.data(), sk_cut, sizeof(uint32_t) * ((size_t)n_tiles + 1));
        RDB.get(h_skstat, work + 21, sizeof(h_skstat));
        RDB.sync();
        sk_KE = h_cut[n_tiles - 1];                              // cut is non-decreasing in the tile index
        const size_t e_rows = sk_KE ? sk_KE : ZONE_BK;
        sk_E = A.get_n<float>(e_rows * Npad);
        CU(cudaMemsetAsync(sk_E, 0, sizeof(float) * e_rows * Npad, st));
        if (sk_KE) {
            k_E_scatter<<<cdiv((long long)sk_KE * 32, TB), TB, 0, st>>>(sk_KE, sk_base, sk_len, ts, reinterpret_cast<const float*>(tv), sk_E, Npad);
            CU_LAUNCH(); ++launches;
        }
        sk_H = A.get_n<double>((size_t)n_tiles * Npad);
        k_zone_hsum<<<cdiv((long long)Npad, 128), 128, 0, st>>>(sk_E, Npad, n_tiles, sk_cut, sk_H); CU_LAUNCH(); ++launches;
        embed_rows = (uint64_t)sk_KE * n_tiles;
    } else if (!use_gram) {
        rflags = A.get_n<uint32_t>((size_t)n_tiles * nwords);
        rrank = A.get_n<uint32_t>((size_t)n_tiles * nwords);
        uint32_t* rows = A.get_n<uint32_t>(n_tiles);
        tileE = A.get_n<T*>(n_tiles);
        tileQ = A.get_n<uint8_t*>(n_tiles);
        k_head_flags<<<cdiv((long long)nwords * 32, TB), TB, 0, st>>>(n, cls, bits, NW, n_tiles, rflags, nwords); CU_LAUNCH(); ++launches;
        k_rank_scan<<<n_tiles, 1024, 0, st>>>(rflags, rrank, nwords, 0, rows); CU_LAUNCH(); ++launches;
        std::vector<uint32_t> h_rows(n_tiles);
        RDB.get(h_rows.data(), rows, sizeof(uint32_t) * n_tiles);
        RDB.sync();
        for (int t = 0; t < n_tiles; ++t) embed_rows += h_rows[t];
        T* Eb = A.get_n<T>((embed_rows ? embed_rows : 1) * TILE);
        uint8_t* Qb = A.get_n<uint8_t>(embed_rows ? embed_rows : 1);
        std::vector<T*> h_tileE(n_tiles);
        std::vector<uint8_t*> h_tileQ(n_tiles);
        size_t run_rows = 0;
        for (int t = 0; t < n_tiles; ++t) { h_tileE[t] = Eb + run_rows * TILE; h_tileQ[t] = Qb + run_rows; run_rows += h_rows[t]; }
        CU(cudaMemcpyAsync(tileE, h_tileE.data(), sizeof(T*) * n_tiles, cudaMemcpyHostToDevice, st));
        CU(cudaMemcpyAsync(tileQ, h_tileQ.data(), sizeof(uint8_t*) * n_tiles, cudaMemcpyHostToDevice, st));
        uint32_t* hpref = nullptr;
        if (weighted && head_rows > 0) {
            hrows = A.get_n<int32_t>(head_rows);
            hpref = A.get_n<uint32_t>((size_t)head_rows * n_tiles);
            k_head_rows<<<cdiv(n, TB), TB, 0, st>>>(n, cls, hrank, hrows); CU_LAUNCH(); ++launches;
            k_head_pref<<<cdiv((long long)head_rows * 32, TB), TB, 0, st>>>((uint32_t)head_rows, hrows, bits, NW, n_tiles, hpref); CU_LAUNCH(); ++launches;
        }
        if (embed_rows) {
            k_compact<T><<<dim3(cdiv(nwords, COMPACT_WORDS), n_tiles), 256, 0, st>>>(n, len, bits, NW, rflags, rrank, nwords, n_tiles, tptr, hrank, hpref,
                                                                                    weighted ? tv : nullptr, tileE, tileQ);
            CU_LAUNCH(); ++launches;
        }
        RDB.sync();   // h_tileE / h_tileQ staging copies are done
    }
    tm.mark();

    // ------------------------------------------------------------------ a-5 (tail branches): scatter into the condensed matrix
    unsigned tail_launches = 0;
    if (tail_rows || mid_rows || skip_on || n_shards > 1) CU(cudaMemsetAsync(out, 0, sizeof(T) * ((size_t)N * (N - 1) / 2), st));
    if (tail_rows) {
        // super tiles: SUP x SUP samples whose condensed row segments (SUP * SUP * sizeof(T)) stay L2-resident
        size_t l2_budget = (size_t)48 << 20;
        if (const char* e = getenv("UNIFRAC_B200_TAIL_L2_MB")) l2_budget = (size_t)atoll(e) << 20;
        int SUP = 128;
        while ((size_t)(SUP + 128) * (SUP + 128) * sizeof(T) <= l2_budget) SUP += 128;
        const int nsup = cdiv(N, SUP);
        uint32_t* seg = A.get_n<uint32_t>((size_t)n * (nsup + 1));
        k_tail_seg<<<cdiv((long long)n * (nsup + 1), TB), TB, 0, st>>>(n, tptr, ts, SUP, nsup, seg); CU_LAUNCH(); ++launches;
        const int n_launch = nsup * (nsup + 1) / 2;
        unsigned int* tcounters = A.get_n<unsigned int>(n_launch);
        CU(cudaMemsetAsync(tcounters, 0, sizeof(unsigned int) * n_launch, st));
        int dev = 0, n_sm = 0;
        CU(cudaGetDevice(&dev));
        CU(cudaDeviceGetAttribute(&n_sm, cudaDevAttrMultiProcessorCount, dev));
        TailParams TP{};
        if (n_shards > 1) {
            const int nb = cdiv(n_tiles, SHARD_BLOCK);
            std::vector<uint8_t> h_owner((size_t)nb * (nb + 1) / 2);
            for (int bj = 0; bj < nb; ++bj)
                for (int bi = 0; bi <= bj; ++bi) h_owner[(size_t)bj * (bj + 1) / 2 + bi] = (uint8_t)(((long long)bj * (bj + 1) / 2 + bi) % n_shards);
            uint8_t* owner = A.get_n<uint8_t>(h_owner.size());
            CU(cudaMemcpyAsync(owner, h_owner.data(), h_owner.size(), cudaMemcpyHostToDevice, st));
            RDB.sync();
            TP.owner = owner; TP.shard = shard;
        }
        TP.tptr = tptr; TP.seg = seg; TP.ts = ts; TP.tv = tv; TP.cls = cls; TP.n = n; TP.nsup = nsup; TP.N = N; TP.out = out;
        int li = 0;
        for (int si = 0; si < nsup; ++si)
            for (int sj = si; sj < nsup; ++sj) {
                TP.SI = si; TP.SJ = sj; TP.counter = tcounters + li++;
                k_tail_scatter<T><<<n_sm * 8, 256, 0, st>>>(TP); CU_LAUNCH(); ++launches; ++tail_launches;
            }
    }
    tm.mark();

    // ------------------------------------------------------------------ a-5 (mid branches): per tile pair, fixed point in shared memory
    unsigned mid_launches = 0;
    int mid_F = 0;
    bool mid_packed = false;
    uint32_t midg_groups = 0, midg_rows = 0;
    unsigned long long mid_atomics = mid_updates;
    double quant_ratio = 0.0;
    // fixed-point error ratio (Gram head lengths + mid entries): over budget => rerun without the fixed-point kernels
    auto check_quant_ratio = [&]() {
        unsigned long long* rbits = work + 19;
        k_quant_ratio<<<cdiv((long long)n_tiles * TILE, TB), TB, 0, st>>>(n_tiles * TILE, qerr, sums, rbits); CU_LAUNCH(); ++launches;
        unsigned long long h_r = 0;
        RDB.get(&h_r, rbits, sizeof(h_r));
        RDB.sync();
        memcpy(&quant_ratio, &h_r, sizeof(quant_ratio));
        if (quant_ratio > envd("UNIFRAC_B200_QUANT_BUDGET", QUANT_RATIO_BUDGET) && !is_retry) throw RetryExact{};
    };
    if (mid_rows || skip_on) {
        if constexpr (std::is_same<T, float>::value) {
            if (mid_rows >= (1ull << 23)) throw StatusFail{UNIFRAC_ERR_UNSUPPORTED};     // packed entries keep the row in 23 bits
            // ---- grouped join (midg.cuh): mid branches whose presence sets nest are joined with one atomic per pair of the
            // group's root; rows that end up alone stay k_mid rows
            uint32_t n_g = 0;
            unsigned long long g_rows = 0;
            int32_t* groot = nullptr; uint8_t* gslot = nullptr;
            const bool groups_on = !skip_on && mid_rows >= 2 && envd("UNIFRAC_B200_MID_GROUPS", 1.0) != 0.0;
            if (groups_on) {
                groot = A.get_n<int32_t>(n); gslot = A.get_n<uint8_t>(n);
                uint32_t* gcnt = A.get_n<uint32_t>(n);
                unsigned long long* gc = A.get_n<unsigned long long>(8);
                CU(cudaMemsetAsync(gcnt, 0, sizeof(uint32_t) * n, st));
                CU(cudaMemsetAsync(gc, 0, sizeof(unsigned long long) * 8, st));
                const uint32_t theta_256 = (uint32_t)std::lround(256.0 * envd("UNIFRAC_B200_MID_GROUP_THETA", 0.35));
                for (int d = 0; d < n_levels; ++d)
                    if (h_hist[d]) {
                        k_midg_level<<<cdiv(h_hist[d], TB), TB, 0, st>>>(h_hist[d], level_nodes + h_off[d], child_off, child_idx, cls, nv,
                                                                         theta_256, groot, gslot, gcnt);
                        CU_LAUNCH(); ++launches;
                    }
                k_midg_classify<<<cdiv(n, TB), TB, 0, st>>>(n, cls, nv, groot, gcnt, gc); CU_LAUNCH(); ++launches;
                unsigned long long h_gc[5] = {0, 0, 0, 0, 0};
                RDB.get(h_gc, gc, sizeof(h_gc));
                RDB.sync();
                n_g = (uint32_t)h_gc[0]; g_rows = h_gc[1];
                midg_groups = n_g; midg_rows = (uint32_t)g_rows;
                mid_atomics = mid_updates - h_gc[3] + h_gc[4];    // one atomic per pair of a lone row / of a group root
            }
            const uint32_t n_mid = skip_on ? sk_n : (uint32_t)(mid_rows - g_rows);
            // row lists of one class ordered by n_v (counting sort)
            auto class_rows = [&](uint8_t want, uint32_t count, int32_t*& rows, uint32_t*& base, uint32_t*& len) {
                uint32_t* hh = A.get_n<uint32_t>((size_t)N + 2);
                uint32_t* cc = A.get_n<uint32_t>((size_t)N + 2);
                rows = A.get_n<int32_t>(count ? count : 1);
                base = A.get_n<uint32_t>(count ? count : 1);
                len = A.get_n<uint32_t>(count ? count : 1);
                CU(cudaMemsetAsync(hh, 0, sizeof(uint32_t) * ((size_t)N + 2), st));
                k_mid_hist<<<cdiv(n, TB), TB, 0, st>>>(n, cls, nv, hh, want); CU_LAUNCH(); ++launches;
                k_exclusive_scan<uint32_t><<<1, 1024, 0, st>>>(N + 1, hh, cc); CU_LAUNCH(); ++launches;
                k_mid_rows<<<cdiv(n, TB), TB, 0, st>>>(n, cls, nv, cc, tptr, rows, base, len, want); CU_LAUNCH(); ++launches;
            };
            // tile-major offsets of the rows' (row, tile) lists
            struct TileLists { uint32_t* seg; uint32_t* off; uint32_t* tbase; };
            auto tile_lists = [&](uint32_t count, const int32_t* rows, const uint32_t* cut, uint32_t pad) {
                TileLists L{};
                L.seg = A.get_n<uint32_t>((size_t)(n_tiles + 1) * std::max<uint32_t>(count, 1u));
                L.off = A.get_n<uint32_t>((size_t)n_tiles * ((size_t)count + 1));
                uint32_t* ttot = A.get_n<uint32_t>(n_tiles);
                L.tbase = A.get_n<uint32_t>((size_t)n_tiles + 1);
                if (count) { k_mid_seg<<<cdiv((long long)count * 32, TB), TB, 0, st>>>(count, rows, tptr, ts, n_tiles, L.seg); CU_LAUNCH(); ++launches; }
                k_mid_off<<<n_tiles, 1024, 0, st>>>(count, L.seg, L.off, ttot, cut, pad); CU_LAUNCH(); ++launches;
                k_exclusive_scan<uint32_t><<<1, 1024, 0, st>>>(n_tiles, ttot, L.tbase); CU_LAUNCH(); ++launches;
                return L;
            };
            int32_t* mrows = sk_rows; uint32_t* mbase = sk_base; uint32_t* mlen = sk_len;
            if (!skip_on) class_rows(CLS_MID, n_mid, mrows, mbase, mlen);
            const TileLists ML = tile_lists(n_mid, mrows, sk_cut, 2u);
            int32_t* grows = nullptr; uint32_t* gbase = nullptr; uint32_t* glen = nullptr;
            TileLists GLs{};
            if (n_g) { class_rows(CLS_MIDG_ROOT, n_g, grows, gbase, glen); GLs = tile_lists(n_g, grows, nullptr, (uint32_t)MIDG_R); }
            unsigned long long* smax = work + 15;
            double* midsum = A.get_n<double>((size_t)n_tiles * TILE);
            CU(cudaMemsetAsync(midsum, 0, sizeof(double) * (size_t)n_tiles * TILE, st));
            if (n_mid) { k_mid_sums<<<cdiv((long long)n_mid * 32, TB), TB, 0, st>>>(n_mid, mbase, mlen, ts, reinterpret_cast<const float*>(tv), midsum, sk_cut); CU_LAUNCH(); ++launches; }
            if (n_g) { k_midg_sums<<<cdiv((long long)n * 32, TB), TB, 0, st>>>(n, cls, tptr, nv, ts, reinterpret_cast<const float*>(tv), midsum); CU_LAUNCH(); ++launches; }
            k_max_positive<<<cdiv((long long)n_tiles * TILE, TB), TB, 0, st>>>(n_tiles * TILE, midsum, smax); CU_LAUNCH(); ++launches;
            unsigned long long h_smax = 0;
            RDB.get(&h_smax, smax, sizeof(h_smax));
            uint32_t h_pk_total = 0, h_g_total = 0;             // packed entries / positions incl. the even-length padding
            RDB.get(&h_pk_total, ML.tbase + n_tiles, sizeof(uint32_t));
            if (n_g) RDB.get(&h_g_total, GLs.tbase + n_tiles, sizeof(uint32_t));
            std::vector<int2> h_mp = blocked_pairs(n_tiles, 8, shard, n_shards);
            const size_t n_all_pairs = h_mp.size();
            int2* gpairs = A.get_n<int2>(n_all_pairs ? n_all_pairs : 1);     // the grouped join visits every tile pair of the shard
            CU(cudaMemcpyAsync(gpairs, h_mp.data(), sizeof(int2) * n_all_pairs, cudaMemcpyHostToDevice, st));
            if (skip_on)                                          // pairs whose rows all go to k_zone have nothing to join
                h_mp.erase(std::remove_if(h_mp.begin(), h_mp.end(), [&](const int2& q) { return h_cut[q.x] >= sk_n; }), h_mp.end());
            int2* mpairs = A.get_n<int2>(h_mp.size() ? h_mp.size() : 1);
            CU(cudaMemcpyAsync(mpairs, h_mp.data(), sizeof(int2) * h_mp.size(), cudaMemcpyHostToDevice, st));
            RDB.sync();
            double sm; memcpy(&sm, &h_smax, sizeof(sm));
            int ex = 0; frexp(sm > 0 ? sm : 1.0, &ex);          // sm < 2^ex
            // unsigned 32-bit cells: acc <= min(R^mid_a, R^mid_b) * 2^F + (rounding: at most half a unit per mid row)
            mid_F = 32 - ex;
            if (ldexp(sm, mid_F) + 0.5 * (double)(n_mid + g_rows) + 1.0 > 4294967295.0) --mid_F;
            (void)mid_entries;
            const float qscale = ldexpf(1.0f, mid_F);
            const double inv_qscale = ldexp(1.0, -mid_F);
            uint2* pk = A.get_n<uint2>(h_pk_total ? h_pk_total : 1);
            if (n_mid) {
                k_mid_pack<<<cdiv((long long)n_mid * 32, TB), TB, 0, st>>>(n_mid, mbase, mlen, ts, reinterpret_cast<const float*>(tv), ML.seg, ML.off, ML.tbase,
                                                                          qscale, inv_qscale, sums, qerr, pk, sk_cut); CU_LAUNCH(); ++launches;
            }
            uint32_t* gex = nullptr; uint32_t* geq = nullptr;
            uint16_t* gem = nullptr; uint32_t* ggq = nullptr;    // mask mode (unweighted: a member's value is one number per row)
            const bool mask_mode = !weighted && envd("UNIFRAC_B200_MID_MASKS", 1.0) != 0.0;
            unsigned long long* gmiss = work + 24;
            if (n_g) {
                const size_t n_pos = (size_t)h_g_total + 4;
                gex = A.get_n<uint32_t>(n_pos);
                CU(cudaMemsetAsync(gex, 0, sizeof(uint32_t) * n_pos, st));
                if (mask_mode) {
                    gem = A.get_n<uint16_t>(n_pos);
                    ggq = A.get_n<uint32_t>((size_t)n_g * MIDG_L);
                    CU(cudaMemsetAsync(gem, 0, sizeof(uint16_t) * n_pos, st));
                    CU(cudaMemsetAsync(ggq, 0, sizeof(uint32_t) * (size_t)n_g * MIDG_L, st));
                } else {
                    geq = A.get_n<uint32_t>(n_pos * MIDG_L);
                    CU(cudaMemsetAsync(geq, 0, sizeof(uint32_t) * n_pos * MIDG_L, st));
                }
                int32_t* rootidx = A.get_n<int32_t>(n);
                k_midg_index<<<cdiv(n_g, TB), TB, 0, st>>>(n_g, grows, rootidx); CU_LAUNCH(); ++launches;
                const uint4* bits4 = reinterpret_cast<const uint4*>(bits);
                k_midg_pack_roots<<<cdiv((long long)n_g * 32, TB), TB, 0, st>>>(n_g, grows, gbase, glen, ts, reinterpret_cast<const float*>(tv), bits4, NW4,
                                                                               GLs.off, GLs.tbase, qscale, inv_qscale, sums, qerr, gex, geq, gem, ggq); CU_LAUNCH(); ++launches;
                k_midg_pack_members<<<cdiv((long long)n * 32, TB), TB, 0, st>>>(n, cls, groot, gslot, rootidx, tptr, nv, ts, reinterpret_cast<const float*>(tv),
                                                                               bits4, NW4, n_g, GLs.off, GLs.tbase, qscale, inv_qscale, sums, qerr, geq, gmiss, gem, ggq);
                CU_LAUNCH(); ++launches;
            }
            mid_packed = true;
            check_quant_ratio();
            if (n_g) {                                            // (the stream was just synchronised)
                unsigned long long h_miss = 0;
                RDB.get(&h_miss, gmiss, sizeof(h_miss)); RDB.sync();
                if (h_miss) { g_cuda_err = "grouped join: a member branch has a sample its group root lacks"; throw StatusFail{UNIFRAC_ERR_CUDA}; }
            }
            int dev2 = 0, n_sm2 = 0;
            CU(cudaGetDevice(&dev2));
            CU(cudaDeviceGetAttribute(&n_sm2, cudaDevAttrMultiProcessorCount, dev2));
            MidParams MP{};
            MP.pairs = mpairs; MP.n_pairs = (uint32_t)h_mp.size(); MP.counter = reinterpret_cast<unsigned int*>(work + 7);
            MP.n_mid = n_mid; MP.off = ML.off; MP.tbase = ML.tbase; MP.pk = pk; MP.cut = sk_cut;
            MP.n_samples = N; MP.out = reinterpret_cast<float*>(out); MP.inv_qscale = inv_qscale;
            if (!n_g && n_mid && !h_mp.empty()) {                 // a shard may own no tile pair of a small problem
                CU(cudaFuncSetAttribute(k_mid, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)MID_SMEM));
                int occ = 0;
                CU(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, k_mid, MID_THREADS, MID_SMEM));
                if (occ < 1) occ = 1;
                k_mid<<<(unsigned)std::min<long long>((long long)n_sm2 * occ, (long long)h_mp.size()), MID_THREADS, MID_SMEM, st>>>(MP);
                CU_LAUNCH(); ++launches; ++mid_launches;
            }
            if (n_g && n_all_pairs) {
                MidgParams M{};
                M.pairs = gpairs; M.n_pairs = (uint32_t)n_all_pairs; M.counter = reinterpret_cast<unsigned int*>(work + 25);
                M.n_g = n_g; M.off = GLs.off; M.tbase = GLs.tbase; M.ex = gex; M.eq = reinterpret_cast<const uint4*>(geq);
                M.n_samples = N; M.out = reinterpret_cast<float*>(out); M.inv_qscale = inv_qscale;
                M.rows = MP;                                      // (groups are off in the zones path: MP.cut = NULL here)
                M.em = gem; M.gq = reinterpret_cast<const uint4*>(ggq);
                auto kern = mask_mode ? k_midg<true> : k_midg<false>;
                CU(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)MID_SMEM));
                int occ = 0;
                CU(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, kern, MIDG_THREADS, MID_SMEM));
                if (occ < 1) occ = 1;
                kern<<<(unsigned)std::min<long long>((long long)n_sm2 * occ, (long long)n_all_pairs), MIDG_THREADS, MID_SMEM, st>>>(M);
                CU_LAUNCH(); ++launches; ++mid_launches;
            }
        }
    }
    if (use_gram && !mid_packed) check_quant_ratio();
    tm.mark();

    // ------------------------------------------------------------------ near-duplicate guard list (filled by the finalize epilogues)
    GuardList GL{nullptr, nullptr, 0u, (float)std::max(GUARD_THETA, quant_ratio / QUANT_REL)};
    if (!(flags & (UNIFRAC_FLAG_LITERAL | UNIFRAC_FLAG_ABSDIFF))) {
        const unsigned long long Pn = (unsigned long long)N * (N - 1) / 2;
        GL.cap = (uint32_t)std::min<unsigned long long>(Pn, std::max<unsigned long long>(1ull << 22, 64ull * N));
        GL.pairs = A.get_n<uint2>(GL.cap);
        GL.count = reinterpret_cast<unsigned int*>(work + 18);         // zeroed with the other counters
    }
    // ------------------------------------------------------------------ near-duplicate guard: listed pairs from the definition
    // (launched after the finalizing kernel, or after each of its segments; `done` = listed pairs already recomputed)
    GuardParams GP{};
    unsigned ggrid = 0;
    if (GL.pairs) {
        ggrid = (unsigned)std::max(1, std::min(n_sm_dev, (int)std::min<unsigned long long>(GL.cap, 1u << 30)));
        GP.n = n; GP.parent = parent; GP.len = len; GP.indptr = tab.indptr; GP.indices = tab.indices; GP.counts = tab.counts;
        GP.Tsum = Tsum; GP.order = nullptr; GP.N = N; GP.weighted = weighted; GP.list = GL; GP.out = out;
        GP.done = reinterpret_cast<unsigned int*>(work + 23);                // zeroed with the other counters
        GP.scratch = A.get_n<uint32_t>((size_t)ggrid * 3 * n);
        CU(cudaMemsetAsync(GP.scratch, 0, sizeof(uint32_t) * (size_t)ggrid * 3 * n, st));
    }
    auto run_guard = [&]() {
        if (!GL.pairs) return;
        k_guard<T><<<ggrid, GUARD_THREADS, 0, st>>>(GP); CU_LAUNCH(); ++launches;
        k_guard_mark<<<1, 1, 0, st>>>(GL, GP.done); CU_LAUNCH(); ++launches;
    };
    // segments of the finalizing kernel's tile-pair list (blocked order: whole block rows of SHARD_BLOCK tiles): one segment
    // unless the caller wants to be told about finished rows; {first pair, end pair, condensed rows final after it}
    struct Seg { uint32_t p0, p1; long long row_end; };
    auto make_segments = [&](const std::vector<int2>& pl, int BLK) {
        std::vector<Seg> segs;
        const uint32_t np = (uint32_t)pl.size();
        const bool split = progress && n_shards == 1 && !inv_perm && np >= 64;
        const int n_seg = split ? (int)env_double("UNIFRAC_B200_E2E_SEGMENTS", 8) : 1;
        uint32_t begin = 0;
        for (int k = 1; k <= n_seg && begin < np; ++k) {
            uint32_t end = k == n_seg ? np : (uint32_t)((unsigned long long)np * k / n_seg);
            while (end < np && end > begin && (uint32_t)pl[end].x / BLK == (uint32_t)pl[end - 1].x / BLK) ++end;   // to the block row's end
            if (end <= begin) continue;
            const long long row_end = end == np ? (long long)N : std::min<long long>(N, ((long long)pl[end - 1].x / BLK + 1) * BLK * TILE);
            segs.push_back(Seg{begin, end, row_end});
            begin = end;
        }
        if (segs.empty()) segs.push_back(Seg{0, np, (long long)N});
        return segs;
    };
    // ------------------------------------------------------------------ a-5 / a-6 stripe accumulation + finalize
    unsigned long long* kstats = work + 4;     // [0] rows executed, [1] rows staged (zeroed above)
    unsigned stripe_launches = 0;
    uint32_t n_pairs = 0;
    bool guard_ran = false;
    int dev = 0, n_sm = 0;
    CU(cudaGetDevice(&dev));
    CU(cudaDeviceGetAttribute(&n_sm, cudaDevAttrMultiProcessorCount, dev));
    if (use_gram) {
        if constexpr (std::is_same<T, float>::value) {
            // (an H2D cudaMemcpyAsync from pageable memory returns once the source has been staged, so the host vectors of the
            //  pair lists may go out of scope right after it: no synchronisation follows the launch of an a-5 kernel)
            std::vector<int2> h_pairs = blocked_pairs(n_tiles, 12, shard, n_shards);
            n_pairs = (uint32_t)h_pairs.size();
            int2* pairs = A.get_n<int2>(n_pairs);
            CU(cudaMemcpyAsync(pairs, h_pairs.data(), sizeof(int2) * n_pairs, cudaMemcpyHostToDevice, st));
            const size_t Npad = (size_t)NW * 32;
            CUtensorMap tmA = make_u8_rowmajor_map(XG[0], Npad, K_pad, TILE, GRAM_BK);
            CUtensorMap tmB0 = make_u8_rowmajor_map(XG[1], Npad, K_pad, TILE, GRAM_BK);
            CUtensorMap tmB1 = make_u8_rowmajor_map(XG[2], Npad, K_pad, TILE, GRAM_BK);
            CUtensorMap tmB2 = make_u8_rowmajor_map(XG[3], Npad, K_pad, TILE, GRAM_BK);
            GramParams G{};
            G.K_pad = K_pad; G.sums = sums; G.n_samples = N;
            G.out = reinterpret_cast<float*>(out); G.add_out = (tail_rows || mid_rows) ? 1 : 0; G.q = gram_q; G.guard = GL;
            CU(cudaFuncSetAttribute(k_gram, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)GRAM_SMEM));
            const int eshift = (int)envd("UNIFRAC_B200_GRAM_EPOCH_SHIFT", 5);
            for (const Seg& sg : make_segments(h_pairs, 12)) {
                G.pairs = pairs + sg.p0; G.n_pairs = sg.p1 - sg.p0;
                unsigned grid = (unsigned)std::min<long long>(n_sm, G.n_pairs);
                G.epoch_cnt = nullptr;
                if (eshift >= 0 && grid) {
                    G.steps_per_cta = (uint32_t)((G.n_pairs + grid - 1) / grid) * (K_pad / GRAM_BK);
                    G.epoch_shift = (uint32_t)eshift;
                    const size_t n_ep = ((size_t)G.steps_per_cta >> eshift) + 2;
                    G.epoch_cnt = A.get_n<unsigned int>(n_ep);
                    CU(cudaMemsetAsync(G.epoch_cnt, 0, sizeof(unsigned int) * n_ep, st));
                }
                if (grid) { k_gram<<<grid, GRAM_THREADS, GRAM_SMEM, st>>>(tmA, tmB0, tmB1, tmB2, G); CU_LAUNCH(); ++launches; ++stripe_launches; }
                run_guard();
                if (progress) progress(progress_user, sg.row_end, st);
            }
            guard_ran = true;
        }
    } else if (skip_on) {
        if constexpr (std::is_same<T, float>::value) {
            // tile pairs dealt to the CTAs in cache-blocked order, each to the least loaded CTA (work ~ stages + epilogue)
            std::vector<int2> order = blocked_pairs(n_tiles, 8, shard, n_shards);
            n_pairs = (uint32_t)order.size();
            const unsigned grid = (unsigned)std::max<long long>(1, std::min<long long>(n_sm, n_pairs));
            std::vector<std::vector<int2>> per(grid);
            typedef std::pair<unsigned long long, unsigned> QE;
            std::priority_queue<QE, std::vector<QE>, std::greater<QE>> pq;
            for (unsigned b = 0; b < grid; ++b) pq.push(QE(0ull, b));
            for (const int2& q : order) {
                QE top = pq.top(); pq.pop();
                per[top.second].push_back(q);
                top.first += h_cut[q.x] / ZONE_BK + 3;
                pq.push(top);
            }
            std::vector<int2> h_pairs; h_pairs.reserve(n_pairs);
            std::vector<uint32_t> h_off(grid + 1, 0);
            for (unsigned b = 0; b < grid; ++b) { h_pairs.insert(h_pairs.end(), per[b].begin(), per[b].end()); h_off[b + 1] = (uint32_t)h_pairs.size(); }
            int2* pairs = A.get_n<int2>(n_pairs ? n_pairs : 1);
            uint32_t* cta_off = A.get_n<uint32_t>(grid + 1);
            CU(cudaMemcpyAsync(pairs, h_pairs.data(), sizeof(int2) * n_pairs, cudaMemcpyHostToDevice, st));
            CU(cudaMemcpyAsync(cta_off, h_off.data(), sizeof(uint32_t) * (grid + 1), cudaMemcpyHostToDevice, st));
            CUtensorMap tmE = make_rowmajor_map(sk_E, CU_TENSOR_MAP_DATA_TYPE_FLOAT32, sizeof(float), Npad, sk_KE ? sk_KE : ZONE_BK, TILE, ZONE_BK,
                                                CU_TENSOR_MAP_SWIZZLE_NONE);
            ZoneParams SP{};
            SP.pairs = pairs; SP.cta_off = cta_off; SP.cut = sk_cut; SP.H = sk_H; SP.Npad = Npad; SP.sums = sums; SP.n_samples = N;
            SP.out = reinterpret_cast<float*>(out); SP.add_out = 1; SP.guard = GL;
            SP.scratch = A.get_n<double>((size_t)grid * 32 * 512);
            CU(cudaFuncSetAttribute(k_zone, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)ZONE_SMEM));
            if (n_pairs) { k_zone<<<grid, ZONE_THREADS, ZONE_SMEM, st>>>(tmE, SP); CU_LAUNCH(); ++launches; ++stripe_launches; }
        }
    } else if (dense_head) {
        std::vector<int2> h_pairs = blocked_pairs(n_tiles, 12, shard, n_shards);
        n_pairs = (uint32_t)h_pairs.size();
        int2* pairs = A.get_n<int2>(n_pairs);
        CU(cudaMemcpyAsync(pairs, h_pairs.data(), sizeof(int2) * n_pairs, cudaMemcpyHostToDevice, st));
        constexpr bool f32 = std::is_same<T, float>::value;
        CUtensorMap tmE = make_rowmajor_map(Edense, f32 ? CU_TENSOR_MAP_DATA_TYPE_FLOAT32 : CU_TENSOR_MAP_DATA_TYPE_FLOAT64, sizeof(T), Npad, Kd_pad,
                                            TILE, DenseCfg<T>::BK, CU_TENSOR_MAP_SWIZZLE_NONE);
        DenseParams D{};
        D.K_pad = Kd_pad; D.sums = sums; D.n_samples = N; D.weighted = weighted; D.out = out;
        D.add_out = (tail_rows || mid_rows) ? 1 : 0; D.guard = GL;
        const size_t smem = dense_smem_bytes<T>();
        D.scratch = A.get_n<double>((size_t)std::max(1, n_sm) * 64 * 256);
        D.hsum = hsum;
        if (dense16) CU(cudaFuncSetAttribute(k_dense16, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
        else CU(cudaFuncSetAttribute(k_dense<T>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
        for (const Seg& sg : make_segments(h_pairs, 12)) {
            D.pairs = pairs + sg.p0; D.n_pairs = sg.p1 - sg.p0;
            const unsigned grid = (unsigned)std::min<long long>(n_sm, D.n_pairs);
            if (grid) {
                if (dense16) k_dense16<<<grid, DENSE16_THREADS, smem, st>>>(tmE, D);
                else k_dense<T><<<grid, DENSE_THREADS, smem, st>>>(tmE, D);
                CU_LAUNCH(); ++launches; ++stripe_launches;
            }
            run_guard();
            if (progress) progress(progress_user, sg.row_end, st);
        }
        guard_ran = true;
    } else {
    std::vector<int2> h_pairs;
    h_pairs.reserve((size_t)n_tiles * (n_tiles + 1) / 2);
    for (int i = 0; i < n_tiles; ++i)
        for (int j = i; j < n_tiles; ++j) h_pairs.push_back(make_int2(i, j));
    n_pairs = (uint32_t)h_pairs.size();
    int2* pairs = A.get_n<int2>(n_pairs);
    CU(cudaMemcpyAsync(pairs, h_pairs.data(), sizeof(int2) * n_pairs, cudaMemcpyHostToDevice, st));
    T* zero_row = A.get_n<T>(TILE);
    CU(cudaMemsetAsync(zero_row, 0, sizeof(T) * TILE, st));
    uint32_t* counter = reinterpret_cast<uint32_t*>(work + 6);

    StripeParams P{};
    P.add_out = (tail_rows || mid_rows) ? 1 : 0;
    P.tileE = reinterpret_cast<const void* const*>(tileE);
    P.tileQ = tileQ; P.flags = rflags; P.rank = rrank; P.nwords = nwords;
    P.pairs = pairs; P.n_pairs = n_pairs; P.counter = counter; P.sums = sums;
    P.n_samples = N; P.weighted = weighted; P.out = out; P.stats = kstats; P.zero_row = zero_row; P.guard = GL;

    if (flags & UNIFRAC_FLAG_LITERAL) {
        k_literal<T><<<n_pairs, 256, 0, st>>>(P); CU_LAUNCH(); ++launches; ++stripe_launches;
    } else {
        const size_t smem = stripe_smem_bytes<T>();
        auto kern = (flags & UNIFRAC_FLAG_ABSDIFF) ? k_stripe<T, FORM_ABSDIFF> : k_stripe<T, FORM_MIN>;
        CU(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
        int occ = 0;
        CU(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, kern, STRIPE_THREADS, smem));
        if (occ < 1) occ = 1;
        unsigned grid = (unsigned)std::min<long long>((long long)n_sm * occ, n_pairs);
        P.scratch = A.get_n<double>((size_t)grid * 64 * 256);
        kern<<<grid, STRIPE_THREADS, smem, st>>>(P); CU_LAUNCH(); ++launches; ++stripe_launches;
    }
    }
    if (!guard_ran) run_guard();
    if (inv_perm) {
        k_unpermute<T><<<dim3((unsigned)cdiv(N, 256), (unsigned)std::min(N, 65535)), 256, 0, st>>>((long long)N, inv_perm, reinterpret_cast<const T*>(out),
                                                                                                  reinterpret_cast<T*>(out_user));
        CU_LAUNCH(); ++launches;
    }
    // stripe counters -> pinned host block (read lazily by unifrac_last_stats)
    if (!g_stats_pinned) { CU(cudaHostAlloc(&g_stats_pinned, 4 * sizeof(unsigned long long), cudaHostAllocDefault)); }
    if (g_stats_event && g_stats_event_dev != dev_id) { cudaEventDestroy(g_stats_event); g_stats_event = nullptr; }    // thread moved to another GPU
    if (!g_stats_event) { CU(cudaEventCreateWithFlags(&g_stats_event, cudaEventDisableTiming)); g_stats_event_dev = dev_id; }
    CU(cudaMemcpyAsync(g_stats_pinned, kstats, 2 * sizeof(unsigned long long), cudaMemcpyDeviceToHost, st));
    CU(cudaMemcpyAsync(g_stats_pinned + 2, work + 18, sizeof(unsigned long long), cudaMemcpyDeviceToHost, st));
    CU(cudaEventRecord(g_stats_event, st));
    g_stats_pending = true;
    tm.mark();

    g_stats = unifrac_stats_t{};
    g_stats.branches_embedded = h_work[0];
    g_stats.updates_dense = (uint64_t)h_work[0] * ((uint64_t)N * (N - 1) / 2);
    g_stats.updates_union = h_work[1];
    g_stats.updates_inter = h_work[2];
    g_stats.embed_rows = embed_rows;
    g_stats.head_rows = head_rows; g_stats.tail_rows = tail_rows; g_stats.tail_updates = tail_updates; g_stats.tail_entries = tail_entries;
    g_stats.tail_launches = tail_launches;
    g_stats.mid_groups = midg_groups; g_stats.mid_group_rows = midg_rows; g_stats.mid_atomics = mid_atomics;
    g_stats.mid_rows = mid_rows; g_stats.mid_updates = mid_updates; g_stats.mid_launches = mid_launches; g_stats.mid_F = (uint32_t)mid_F;
    g_stats.skip = skip_on ? 1u : 0u; g_stats.skip_rows = sk_KE; g_stats.list_rows = sk_n;
    if (skip_on) { g_stats.mid_updates = h_skstat[0]; g_stats.skip_row_pair_visits = h_skstat[1]; g_stats.skip_updates_executed = h_skstat[1] * 16384ull; g_stats.mid_rows = sk_n; g_stats.head_rows = sk_KE; }
    g_stats.gram = use_gram ? 1u : 0u; g_stats.dense = dense_head ? 1u : 0u; g_stats.gram_k = K_pad; g_stats.gram_q = (uint32_t)gram_q;
    g_stats.guard_capacity = GL.cap; g_stats.guard_theta = GL.theta;
    g_stats.quant_err_ratio = (float)quant_ratio; g_stats.quant_fallback = is_retry ? 1u : 0u;
    g_stats.n_tile_pairs = n_pairs;
    g_stats.n_levels = (uint32_t)n_levels;
    g_stats.stripe_launches = stripe_launches;
    g_stats.kernel_launches = launches;
    A.release();
    g_stats.workspace_bytes = A.total;
    if (timing) {
        RDB.sync();
        g_stats.ms_plan = tm.ms(0, 1); g_stats.ms_embed = tm.ms(1, 3); g_stats.ms_tail = tm.ms(3, 4); g_stats.ms_mid = tm.ms(4, 5); g_stats.ms_stripe = tm.ms(5, 6);
        g_stats.ms_total = tm.ms(0, 6);
    }
}

int guarded(int32_t n_nodes, const int32_t* parent, const double* len, const int32_t* postorder, unifrac_csr_t tab,
            int32_t N, unifrac_variant_t variant, unifrac_precision_t precision, void* out, unifrac_alloc_fn alloc,
            void* user, uint32_t flags, cudaStream_t st, int shard = 0, int n_shards = 1, cudaMemPool_t pool = nullptr,
            ProgressFn progress = nullptr, void* progress_user = nullptr)
{
    if (n_shards < 1 || n_shards > 255 || shard < 0 || shard >= n_shards) return UNIFRAC_ERR_INVALID_ARG;
    if (n_shards > 1 && (flags & (UNIFRAC_FLAG_LITERAL | UNIFRAC_FLAG_ABSDIFF | UNIFRAC_FLAG_SPARSE_STRIPE | UNIFRAC_FLAG_NO_TAIL)))
        return UNIFRAC_ERR_INVALID_ARG;
    if (!parent || !len || !postorder || !tab.indptr || !tab.indices || !tab.counts || !out) return UNIFRAC_ERR_INVALID_ARG;
    if (n_nodes < 2 || N < 2) return UNIFRAC_ERR_INVALID_ARG;
    if (variant != UNIFRAC_UNWEIGHTED && variant != UNIFRAC_WEIGHTED_NORMALIZED) return UNIFRAC_ERR_INVALID_ARG;
    if (precision != UNIFRAC_FP32 && precision != UNIFRAC_FP64) return UNIFRAC_ERR_INVALID_ARG;
    if (flags & ~(UNIFRAC_FLAG_LITERAL | UNIFRAC_FLAG_TENSOR_GRAM | UNIFRAC_FLAG_SKIP_VALIDATION | UNIFRAC_FLAG_ABSDIFF |
                  UNIFRAC_FLAG_NO_TAIL | UNIFRAC_FLAG_ALL_TAIL | UNIFRAC_FLAG_NO_TENSOR | UNIFRAC_FLAG_NO_MID | UNIFRAC_FLAG_SPARSE_STRIPE |
                  UNIFRAC_FLAG_RICHNESS_ZONES))
        return UNIFRAC_ERR_INVALID_ARG;
    if ((long long)N > (1ll << 23)) return UNIFRAC_ERR_UNSUPPORTED;
    Arena A{alloc, user, st};
    A.pool = pool;
    int rc = UNIFRAC_OK;
    const bool w = variant == UNIFRAC_WEIGHTED_NORMALIZED;
    try {
        try {
            if (precision == UNIFRAC_FP32) run<float>(n_nodes, parent, len, postorder, tab, N, w, out, A, flags, st, shard, n_shards, false, progress, progress_user);
            else run<double>(n_nodes, parent, len, postorder, tab, N, w, out, A, flags, st, shard, n_shards, false, progress, progress_user);
        } catch (const RetryExact&) {
            // only the fp32 path has fixed-point kernels; head rows on the CUDA-core kernel, the rest on the fp32 scatter
            A.release();
            run<float>(n_nodes, parent, len, postorder, tab, N, w, out, A, flags | UNIFRAC_FLAG_NO_TENSOR | UNIFRAC_FLAG_NO_MID, st, shard, n_shards, true,
                       progress, progress_user);
        }
    } catch (const CudaFail& f) {
        char buf[512];
        snprintf(buf, sizeof(buf), "%s: %s (unifrac_b200.cu:%d)", f.what, cudaGetErrorString(f.e), f.line);
        g_cuda_err = buf;
        cudaGetLastError();
        rc = UNIFRAC_ERR_CUDA;
    } catch (const WorkspaceFail&) { rc = UNIFRAC_ERR_WORKSPACE; }
    catch (const StatusFail& s) { rc = s.status; }
    catch (...) { rc = UNIFRAC_ERR_CUDA; g_cuda_err = "unexpected C++ exception"; }
    if (rc != UNIFRAC_OK) A.release();
    return rc;
}

template <typename T>
void run_mantel(int32_t N, const T* x, const T* y, const int32_t* perms, int32_t K, double* out, Arena& A, cudaStream_t st)
{
    const unsigned long long P = (unsigned long long)N * (N - 1) / 2;
    double* mom = A.get_n<double>(8);
    const long long pitch = ((long long)N + 3) & ~3ll;                      // rows start 16-byte aligned (bulk copies)
    T* Xs = A.get_n<T>((size_t)N * pitch);
    CU(cudaMemsetAsync(mom, 0, sizeof(double) * 8, st));
    if (pitch > N)                                                          // the padding columns are copied with the rows: keep them finite
        CU(cudaMemset2DAsync(Xs + N, (size_t)pitch * sizeof(T), 0, (size_t)(pitch - N) * sizeof(T), (size_t)N, st));
    int dev = 0, n_sm = 0;
    CU(cudaGetDevice(&dev));
    CU(cudaDeviceGetAttribute(&n_sm, cudaDevAttrMultiProcessorCount, dev));
    k_mantel_moments<T><<<n_sm * 8, 256, 0, st>>>(x, y, P, mom); CU_LAUNCH();
    const unsigned nb = (unsigned)cdiv(N, 32);
    k_mantel_square<T><<<dim3(nb, nb), dim3(32, 8), 0, st>>>(x, N, pitch, Xs); CU_LAUNCH();
    // staging of the gathered rows: two ring buffers of a whole row when two fit in ~208 KB (the next row is copied while this
    // one is used); ONE whole-row buffer when only one fits (the SMs drift apart, so one SM's copy overlaps the others'
    // multiply-adds -- measured 2x faster than two passes over half rows); column segments in two buffers beyond that
    const size_t cap = (size_t)208 * 1024 / sizeof(T);                     // elements of staging space
    int n_buf = 2, n_split = 1;
    if (const char* e = getenv("UNIFRAC_B200_MANTEL_BUFS")) n_buf = atoi(e) == 1 ? 1 : 2;
    else if ((size_t)pitch * 2 > cap && (size_t)pitch <= cap) n_buf = 1;
    if ((size_t)pitch * n_buf > cap) n_split = cdiv(pitch, (long long)(cap / n_buf));
    const int seg = (int)(((pitch + n_split - 1) / n_split + 3) & ~3ll);
    const size_t smem = (size_t)n_buf * seg * sizeof(T) + 16;              // + the zero element of the split kernel
    auto kern = n_split > 1 ? k_mantel_perm<T, true> : k_mantel_perm<T, false>;
    CU(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    int32_t* ident = A.get_n<int32_t>(N);
    k_mantel_iota<<<cdiv(N, 256), 256, 0, st>>>(ident, N); CU_LAUNCH();
    {
        const int kn = K + 1;
        // row-strided CTAs per permutation: G * kn CTAs (one per SM at a time) should fill whole waves of n_sm
        int G = 1; double best = 0.0;
        for (int m = 1; m <= 8; ++m) {
            const int g = (int)std::min<long long>(std::min<long long>(N - 1, 65535), std::max<long long>(1, (long long)n_sm * m / kn));
            const double fill = (double)g * kn / ((double)n_sm * cdiv((long long)g * kn, n_sm));
            if (fill > best + 1e-9) { best = fill; G = g; }
        }
        double* S = A.get_n<double>((size_t)kn * G);                      // every CTA writes its own partial sum
        kern<<<dim3((unsigned)kn, (unsigned)G), MANTEL_THREADS, smem, st>>>(
            Xs, pitch, y, perms, ident, N, seg, n_split, n_buf, 0, S);
        CU_LAUNCH();
        k_mantel_final<T><<<1, 256, 0, st>>>(mom, S, G, K, (double)P, x, y, out); CU_LAUNCH();
    }
    A.release();
}

template <typename T>
void run_spearman(int32_t N, const T* x, const T* y, const int32_t* perms, int32_t K, double* out, Arena& A, cudaStream_t st)
{
    const unsigned long long P = (unsigned long long)N * (N - 1) / 2;
    if (P >= (1ull << 31) - 1) throw StatusFail{UNIFRAC_ERR_UNSUPPORTED};      // positions and 2 x rank are kept in 32 bits
    int dev = 0, n_sm = 0;
    CU(cudaGetDevice(&dev));
    CU(cudaDeviceGetAttribute(&n_sm, cudaDevAttrMultiProcessorCount, dev));
    RankBufs B = make_rank_bufs<T>(A, P, n_sm);
    uint32_t* rx = A.get_n<uint32_t>(P);
    uint32_t* ry = A.get_n<uint32_t>(P);
    rank_transform<T>(x, P, rx, B, st);
    rank_transform<T>(y, P, ry, B, st);
    run_mantel<uint32_t>(N, rx, ry, perms, K, out, A, st);
}

// PCoA: block subspace iteration with Rayleigh-Ritz (pcoa.cuh).  Synchronous: the Ritz values are read back every
// PCOA_CHECK products to test convergence.
constexpr int PCOA_CHECK = 4;
template <typename T>
void run_pcoa(int32_t N, const T* d, int32_t k, int32_t max_iter, double tol, double* out, int32_t* iters_out, Arena& A, cudaStream_t st)
{
    const long long n_pad = ((long long)N + 127) / 128 * 128;
    int dev = 0, n_sm = 0;
    CU(cudaGetDevice(&dev));
    CU(cudaDeviceGetAttribute(&n_sm, cudaDevAttrMultiProcessorCount, dev));
    float* Bhi = A.get_n<float>((size_t)n_pad * n_pad);
    float* Blo = A.get_n<float>((size_t)n_pad * n_pad);
    double* rs = A.get_n<double>((size_t)N + 1);
    double* tot = rs + N;
    float* Y = A.get_n<float>((size_t)n_pad * PCOA_NB);
    float* Q = A.get_n<float>((size_t)n_pad * PCOA_NB);
    float* Qt_hi = A.get_n<float>((size_t)n_pad * PCOA_NB);
    float* Qt_lo = A.get_n<float>((size_t)n_pad * PCOA_NB);
    double* G = A.get_n<double>(1024);
    double* Rinv = A.get_n<double>(1024);
    double* W = A.get_n<double>(1024);
    double* lam = A.get_n<double>(32);
    CU(cudaMemsetAsync(tot, 0, sizeof(double), st));
    const unsigned nb32 = (unsigned)(n_pad / 32);
    k_pcoa_square<T><<<dim3(nb32, nb32), dim3(32, 8), 0, st>>>(d, N, n_pad, Bhi); CU_LAUNCH();
    k_pcoa_rowsum<<<cdiv((long long)N * 32, 256), 256, 0, st>>>(Bhi, N, n_pad, rs, tot); CU_LAUNCH();
    k_pcoa_center<<<(unsigned)((n_pad * n_pad / 4 + 255) / 256), 256, 0, st>>>(Bhi, Blo, N, n_pad, rs, tot); CU_LAUNCH();
    double h_tot = 0.0;
    CU(cudaMemcpyAsync(&h_tot, tot, sizeof(double), cudaMemcpyDeviceToHost, st));
    CUtensorMap tmBhi = make_rowmajor_map(Bhi, CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 4, (uint64_t)n_pad, (uint64_t)n_pad, PCOA_BK, 128, CU_TENSOR_MAP_SWIZZLE_128B);
    CUtensorMap tmBlo = make_rowmajor_map(Blo, CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 4, (uint64_t)n_pad, (uint64_t)n_pad, PCOA_BK, 128, CU_TENSOR_MAP_SWIZZLE_128B);
    CUtensorMap tmQhi = make_rowmajor_map(Qt_hi, CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 4, (uint64_t)n_pad, PCOA_NB, PCOA_BK, PCOA_NB, CU_TENSOR_MAP_SWIZZLE_128B);
    CUtensorMap tmQlo = make_rowmajor_map(Qt_lo, CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 4, (uint64_t)n_pad, PCOA_NB, PCOA_BK, PCOA_NB, CU_TENSOR_MAP_SWIZZLE_128B);
    CU(cudaFuncSetAttribute(k_pcoa_gemm, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)PCOA_SMEM));
    const unsigned gblocks = (unsigned)std::min<long long>(n_sm, n_pad / 32);
    auto orth = [&]() {                                   // Q = orth(Y): Cholesky QR (fp64)
        CU(cudaMemsetAsync(G, 0, sizeof(double) * 1024, st));
        k_pcoa_gram32<<<gblocks, dim3(32, 32), 0, st>>>(Y, Y, n_pad, G); CU_LAUNCH();
        k_pcoa_chol<<<1, 32, 0, st>>>(G, Rinv); CU_LAUNCH();
        k_pcoa_apply<<<(unsigned)std::min<long long>(n_sm * 2, (n_pad + 255) / 256), 256, 0, st>>>(Y, Rinv, n_pad, Q, Qt_hi, Qt_lo); CU_LAUNCH();
    };
    k_pcoa_init<<<(unsigned)((n_pad * PCOA_NB + 255) / 256), 256, 0, st>>>(Y, N, n_pad); CU_LAUNCH();
    orth();
    std::swap(Y, Q);                                      // a second pass (Cholesky QR 2) makes the start block orthonormal to fp32 rounding
    orth();
    double h_lam[32], prev[32];
    for (auto& x : prev) x = 0.0;
    int it = 0;
    if (max_iter < 1) max_iter = 1;
    for (;;) {
        k_pcoa_gemm<<<(unsigned)(n_pad / 128), PCOA_THREADS, PCOA_SMEM, st>>>(tmBhi, tmBlo, tmQhi, tmQlo, (uint32_t)n_pad, Y); CU_LAUNCH();
        ++it;
        if (it % PCOA_CHECK == 0 || it >= max_iter) {
            CU(cudaMemsetAsync(G, 0, sizeof(double) * 1024, st));
            k_pcoa_gram32<<<gblocks, dim3(32, 32), 0, st>>>(Q, Y, n_pad, G); CU_LAUNCH();
            k_pcoa_jacobi<<<1, 32, 0, st>>>(G, lam, W); CU_LAUNCH();
            CU(cudaMemcpyAsync(h_lam, lam, sizeof(h_lam), cudaMemcpyDeviceToHost, st));
            CU(cudaStreamSynchronize(st));
            bool conv = true;
            for (int a = 0; a < k; ++a) conv = conv && fabs(h_lam[a] - prev[a]) <= tol * fabs(h_lam[a]);
            for (int a = 0; a < 32; ++a) prev[a] = h_lam[a];
            if (conv || it >= max_iter) break;
        }
        orth();
    }
    CU(cudaStreamSynchronize(st));
    const double trace = -h_tot / (double)N;              // trace(B) = -(sum of A) / n = (1/n) sum_{i<j} d_ij^2
    k_pcoa_coords<<<(unsigned)(((long long)N * k + 255) / 256), 256, 0, st>>>(Q, lam, W, N, k, trace, out); CU_LAUNCH();
    if (iters_out) *iters_out = it;
    A.release();
}
}  // namespace

extern "C" {

int unifrac_dm(int32_t n_nodes, const int32_t* tree_parent, const double* branch_len, const int32_t* postorder,
               unifrac_csr_t table, int32_t n_samples, unifrac_variant_t variant, unifrac_precision_t precision,
               void* out_condensed, unifrac_alloc_fn alloc, void* alloc_user, uint32_t flags, void* stream)
{
    return guarded(n_nodes, tree_parent, branch_len, postorder, table, n_samples, variant, precision, out_condensed,
                   alloc, alloc_user, flags, reinterpret_cast<cudaStream_t>(stream));
}

int unifrac_dm_shard(int32_t n_nodes, const int32_t* tree_parent, const double* branch_len, const int32_t* postorder,
                     unifrac_csr_t table, int32_t n_samples, unifrac_variant_t variant, unifrac_precision_t precision,
                     void* out_condensed, unifrac_alloc_fn alloc, void* alloc_user, uint32_t flags, void* stream,
                     int32_t shard_index, int32_t shard_count)
{
    return guarded(n_nodes, tree_parent, branch_len, postorder, table, n_samples, variant, precision, out_condensed,
                   alloc, alloc_user, flags, reinterpret_cast<cudaStream_t>(stream), shard_index, shard_count);
}

int32_t unifrac_shard_of_pair(int32_t i, int32_t j, int32_t shard_count)
{
    if (shard_count < 1 || i < 0 || j < 0 || i == j) return -1;
    const int a = i < j ? i : j, b = i < j ? j : i;
    return shard_of_tiles(a / TILE, b / TILE, shard_count);
}

// Device -> host copy in pieces of 32 MB: the planning steps of the NEXT variant read a few words back at every synchronisation
// point, and those small copies share the copy engine with this one -- behind a single 5 GB transfer they would wait ~190 ms.
static cudaError_t copy_d2h_pieces(unsigned char* dst, const unsigned char* src, size_t bytes, cudaStream_t s)
{
    const size_t PIECE = (size_t)env_double("UNIFRAC_B200_E2E_PIECE_MB", 32) << 20;
    for (size_t off = 0; off < bytes; off += PIECE) {
        cudaError_t e = cudaMemcpyAsync(dst + off, src + off, std::min(PIECE, bytes - off), cudaMemcpyDeviceToHost, s);
        if (e != cudaSuccess) return e;
    }
    return cudaSuccess;
}

// the library's own stream-ordered pool for the host entry points (one per device, created on first use; it keeps what it
// has mapped between calls -- release threshold = max -- and unifrac_release_host_pool gives it back)
static cudaMemPool_t g_host_pool[64] = {};
static cudaMemPool_t host_pool(int dev)
{
    if (dev < 0 || dev >= 64) return nullptr;
    static std::mutex mu;
    std::lock_guard<std::mutex> lock(mu);
    if (!g_host_pool[dev]) {
        cudaMemPoolProps props{};
        props.allocType = cudaMemAllocationTypePinned;
        props.handleTypes = cudaMemHandleTypeNone;
        props.location.type = cudaMemLocationTypeDevice;
        props.location.id = dev;
        cudaMemPool_t pool = nullptr;
        if (cudaMemPoolCreate(&pool, &props) != cudaSuccess) { cudaGetLastError(); return nullptr; }
        uint64_t keep = UINT64_MAX;
        cudaMemPoolSetAttribute(pool, cudaMemPoolAttrReleaseThreshold, &keep);
        g_host_pool[dev] = pool;
    }
    return g_host_pool[dev];
}

int unifrac_dm_host_multi(int32_t n_nodes, const int32_t* tree_parent, const double* branch_len, const int32_t* postorder,
                          unifrac_csr_t th, int32_t N, int32_t n_variants, const int32_t* variants, unifrac_precision_t precision,
                          void* const* outs_host, uint32_t flags)
{
    if (!tree_parent || !branch_len || !postorder || !th.indptr || !th.indices || !th.counts || !outs_host || !variants) return UNIFRAC_ERR_INVALID_ARG;
    if (n_nodes < 2 || N < 2 || n_variants < 1 || n_variants > 2) return UNIFRAC_ERR_INVALID_ARG;
    for (int k = 0; k < n_variants; ++k)
        if (!outs_host[k] || (variants[k] != UNIFRAC_UNWEIGHTED && variants[k] != UNIFRAC_WEIGHTED_NORMALIZED)) return UNIFRAC_ERR_INVALID_ARG;
    if (precision != UNIFRAC_FP32 && precision != UNIFRAC_FP64) return UNIFRAC_ERR_INVALID_ARG;
    const int64_t nnz = th.indptr[N];
    if (nnz < 0) return UNIFRAC_ERR_INVALID_TABLE;
    const size_t esz = precision == UNIFRAC_FP32 ? 4 : 8;
    const size_t n_out = (size_t)N * (N - 1) / 2;
    cudaStream_t st = nullptr, cs = nullptr;
    cudaEvent_t done[2] = {nullptr, nullptr};
    void *d_parent = nullptr, *d_len = nullptr, *d_post = nullptr, *d_indptr = nullptr, *d_idx = nullptr, *d_cnt = nullptr;
    void* d_out[2] = {nullptr, nullptr};
    int rc = UNIFRAC_OK;
    auto ok = [&](cudaError_t e) { if (e != cudaSuccess && rc == UNIFRAC_OK) { g_cuda_err = cudaGetErrorString(e); cudaGetLastError(); rc = e == cudaErrorMemoryAllocation ? UNIFRAC_ERR_WORKSPACE : UNIFRAC_ERR_CUDA; } return rc == UNIFRAC_OK; };
    int dev = 0;
    ok(cudaGetDevice(&dev));
    cudaMemPool_t pool = host_pool(dev);
    if (!pool && rc == UNIFRAC_OK) { rc = UNIFRAC_ERR_CUDA; g_cuda_err = "cudaMemPoolCreate failed"; }
    ok(cudaStreamCreateWithFlags(&st, cudaStreamNonBlocking));        // compute (and the input copies)
    ok(cudaStreamCreateWithFlags(&cs, cudaStreamNonBlocking));        // result copies: overlap the next variant's compute
    auto dalloc = [&](void** p, size_t bytes) { return ok(cudaMallocFromPoolAsync(p, bytes ? bytes : 256, pool, st)); };
    if (rc == UNIFRAC_OK) {
        dalloc(&d_parent, sizeof(int32_t) * n_nodes) && dalloc(&d_len, sizeof(double) * n_nodes) &&
        dalloc(&d_post, sizeof(int32_t) * n_nodes) && dalloc(&d_indptr, sizeof(int64_t) * ((size_t)N + 1)) &&
        dalloc(&d_idx, sizeof(int32_t) * (size_t)nnz) && dalloc(&d_cnt, sizeof(int32_t) * (size_t)nnz);
        for (int k = 0; k < n_variants; ++k) dalloc(&d_out[k], esz * n_out);
    }
    if (rc == UNIFRAC_OK) {
        ok(cudaMemcpyAsync(d_parent, tree_parent, sizeof(int32_t) * n_nodes, cudaMemcpyHostToDevice, st));
        ok(cudaMemcpyAsync(d_len, branch_len, sizeof(double) * n_nodes, cudaMemcpyHostToDevice, st));
        ok(cudaMemcpyAsync(d_post, postorder, sizeof(int32_t) * n_nodes, cudaMemcpyHostToDevice, st));
        ok(cudaMemcpyAsync(d_indptr, th.indptr, sizeof(int64_t) * ((size_t)N + 1), cudaMemcpyHostToDevice, st));
        ok(cudaMemcpyAsync(d_idx, th.indices, sizeof(int32_t) * (size_t)nnz, cudaMemcpyHostToDevice, st));
        ok(cudaMemcpyAsync(d_cnt, th.counts, sizeof(int32_t) * (size_t)nnz, cudaMemcpyHostToDevice, st));
    }
    // The LAST variant's result has nothing to hide behind, so its finalizing kernel runs in segments of whole block rows and
    // every finished range of condensed rows starts travelling while the next segment is computed (ProgressFn).
    struct Chunked {
        cudaStream_t cs; unsigned char* host; const unsigned char* dev; size_t esz; long long N; long long rows_done; cudaError_t err;
        std::vector<cudaEvent_t> events;
    } ch{cs, nullptr, nullptr, esz, (long long)N, 0, cudaSuccess, {}};
    auto on_rows = [](void* user, long long row_end, cudaStream_t s) {
        Chunked* c = static_cast<Chunked*>(user);
        if (row_end <= c->rows_done || c->err != cudaSuccess) return;
        auto first = [&](long long r) { return (size_t)(r * (2 * c->N - r - 1) / 2); };      // condensed index of (r, r + 1)
        const long long r1 = row_end >= c->N - 1 ? c->N - 1 : row_end;                         // row N - 1 has no element
        const size_t e0 = first(c->rows_done), e1 = first(r1);
        cudaEvent_t ev = nullptr;
        if ((c->err = cudaEventCreateWithFlags(&ev, cudaEventDisableTiming)) != cudaSuccess) return;
        c->events.push_back(ev);
        if ((c->err = cudaEventRecord(ev, s)) != cudaSuccess) return;
        if ((c->err = cudaStreamWaitEvent(c->cs, ev, 0)) != cudaSuccess) return;
        if (e1 > e0) c->err = copy_d2h_pieces(c->host + e0 * c->esz, c->dev + e0 * c->esz, (e1 - e0) * c->esz, c->cs);
        c->rows_done = r1;
    };
    for (int k = 0; k < n_variants && rc == UNIFRAC_OK; ++k) {
        unifrac_csr_t td{reinterpret_cast<const int64_t*>(d_indptr), reinterpret_cast<const int32_t*>(d_idx), reinterpret_cast<const int32_t*>(d_cnt)};
        const bool last = k == n_variants - 1;
        ch.host = static_cast<unsigned char*>(outs_host[k]); ch.dev = static_cast<const unsigned char*>(d_out[k]); ch.rows_done = 0;
        rc = guarded(n_nodes, reinterpret_cast<const int32_t*>(d_parent), reinterpret_cast<const double*>(d_len),
                     reinterpret_cast<const int32_t*>(d_post), td, N, (unifrac_variant_t)variants[k], precision, d_out[k], nullptr, nullptr,
                     flags, st, 0, 1, pool, last ? +on_rows : nullptr, last ? &ch : nullptr);
        if (rc != UNIFRAC_OK) break;
        if (last) ok(ch.err);
        // unifrac_dm returns once the a-5 kernels are enqueued: the copy of whatever has not been sent yet waits for them on its own stream
        ok(cudaEventCreateWithFlags(&done[k], cudaEventDisableTiming));
        if (rc == UNIFRAC_OK) {
            const long long r0 = last ? ch.rows_done : 0;
            const size_t e0 = (size_t)(r0 * (2 * (long long)N - r0 - 1) / 2);
            ok(cudaEventRecord(done[k], st));
            ok(cudaStreamWaitEvent(cs, done[k], 0));
            if (n_out > e0) ok(copy_d2h_pieces(static_cast<unsigned char*>(outs_host[k]) + e0 * esz, static_cast<const unsigned char*>(d_out[k]) + e0 * esz,
                                               (n_out - e0) * esz, cs));
        }
    }
    if (cs) ok(cudaStreamSynchronize(cs));
    for (void* p : {d_parent, d_len, d_post, d_indptr, d_idx, d_cnt, d_out[0], d_out[1]}) if (p && st) cudaFreeAsync(p, st);
    if (st) { ok(cudaStreamSynchronize(st)); cudaStreamDestroy(st); }
    if (cs) cudaStreamDestroy(cs);
    for (auto& e : done) if (e) cudaEventDestroy(e);
    for (auto& e : ch.events) cudaEventDestroy(e);
    return rc;
}

int unifrac_dm_host(int32_t n_nodes, const int32_t* tree_parent, const double* branch_len, const int32_t* postorder,
                    unifrac_csr_t th, int32_t N, unifrac_variant_t variant, unifrac_precision_t precision,
                    void* out_host, uint32_t flags)
{
    const int32_t v = (int32_t)variant;
    void* outs[1] = {out_host};
    return unifrac_dm_host_multi(n_nodes, tree_parent, branch_len, postorder, th, N, 1, &v, precision, outs, flags);
}

int unifrac_release_host_pool(void)
{
    int rc = UNIFRAC_OK;
    for (int d = 0; d < 64; ++d)
        if (g_host_pool[d] && cudaMemPoolTrimTo(g_host_pool[d], 0) != cudaSuccess) { cudaGetLastError(); rc = UNIFRAC_ERR_CUDA; }
    return rc;
}

int unifrac_last_stats(unifrac_stats_t* out)
{
    if (!out) return UNIFRAC_ERR_INVALID_ARG;
    if (g_stats_pending) {
        if (cudaEventSynchronize(g_stats_event) != cudaSuccess) { cudaGetLastError(); return UNIFRAC_ERR_CUDA; }
        g_stats.updates_executed_head = g_stats_pinned[0] * 2048ull;    // one (warp,row) = 32 x 64 pair updates
        if (g_stats.skip) g_stats.updates_executed_head = g_stats.skip_updates_executed;
        else if (g_stats.gram || g_stats.dense) g_stats.updates_executed_head = g_stats.head_rows * ((uint64_t)g_stats.updates_dense / (g_stats.branches_embedded ? g_stats.branches_embedded : 1));
        g_stats.updates_executed = g_stats.updates_executed_head + g_stats.tail_updates + g_stats.mid_updates;
        g_stats.rows_staged = g_stats_pinned[1];
        g_stats.guard_pairs = (uint32_t)(g_stats_pinned[2] & 0xffffffffull);      // listed; min(guard_pairs, guard_capacity) were recomputed
        g_stats_pending = false;
    }
    *out = g_stats;
    return UNIFRAC_OK;
}

int unifrac_mantel_pearson(int32_t N, const void* x, const void* y, unifrac_precision_t precision, const int32_t* perms,
                           int32_t K, double* out, unifrac_alloc_fn alloc, void* user, void* stream)
{
    if (!x || !y || !out || K < 0 || (K > 0 && !perms) || N < 3) return UNIFRAC_ERR_INVALID_ARG;
    if (precision != UNIFRAC_FP32 && precision != UNIFRAC_FP64) return UNIFRAC_ERR_INVALID_ARG;
    if ((long long)N > (1ll << 23)) return UNIFRAC_ERR_UNSUPPORTED;
    cudaStream_t st = reinterpret_cast<cudaStream_t>(stream);
    Arena A{alloc, user, st};
    int rc = UNIFRAC_OK;
    try {
        if (precision == UNIFRAC_FP32) run_mantel<float>(N, reinterpret_cast<const float*>(x), reinterpret_cast<const float*>(y), perms, K, out, A, st);
        else run_mantel<double>(N, reinterpret_cast<const double*>(x), reinterpret_cast<const double*>(y), perms, K, out, A, st);
    } catch (const CudaFail& f) {
        char b[512];
        snprintf(b, sizeof(b), "%s: %s (unifrac_b200.cu:%d)", f.what, cudaGetErrorString(f.e), f.line);
        g_cuda_err = b; cudaGetLastError(); rc = UNIFRAC_ERR_CUDA;
    } catch (const WorkspaceFail&) { rc = UNIFRAC_ERR_WORKSPACE; }
    catch (...) { rc = UNIFRAC_ERR_CUDA; g_cuda_err = "unexpected C++ exception"; }
    if (rc != UNIFRAC_OK) A.release();
    return rc;
}

// ---- unifrac_mantel_pearson_noalloc (header): run_mantel with its workspace bumped out of a static device array ----------
// In host code the array's NAME is a host-side stand-in, not a device address: the address the kernels get comes from
// cudaGetSymbolAddress, once per device, with that device current.
}  // extern "C"
static __device__ __align__(256) unsigned char g_noalloc_scratch[UNIFRAC_NOALLOC_SCRATCH_BYTES];
namespace {
struct NoAllocBump { unsigned char* base; size_t cap; size_t used; };
void* noalloc_bump(size_t bytes, void* user)            // Arena::get has rounded bytes up to a multiple of 256
{
    NoAllocBump* b = static_cast<NoAllocBump*>(user);
    if (bytes > b->cap - b->used) return nullptr;       // -> UNIFRAC_ERR_WORKSPACE (the limits below keep a call within cap)
    void* p = b->base + b->used;
    b->used += bytes;
    return p;
}
unsigned char* noalloc_scratch_of_current_device()
{
    constexpr int MAX_DEV = 64;
    static std::mutex mu;
    static unsigned char* ptrs[MAX_DEV] = {};
    int dev = 0;
    CU(cudaGetDevice(&dev));
    if (dev < 0 || dev >= MAX_DEV) throw StatusFail{UNIFRAC_ERR_UNSUPPORTED};
    std::lock_guard<std::mutex> g(mu);
    if (!ptrs[dev]) {
        void* p = nullptr;
        CU(cudaGetSymbolAddress(&p, g_noalloc_scratch));
        ptrs[dev] = static_cast<unsigned char*>(p);
    }
    return ptrs[dev];
}
}  // namespace
extern "C" {

int unifrac_mantel_pearson_noalloc(int32_t N, const void* x, const void* y, unifrac_precision_t precision, const int32_t* perms,
                                   int32_t K, double* out, void* stream)
{
    if (!x || !y || !out || K < 0 || (K > 0 && !perms) || N < 3) return UNIFRAC_ERR_INVALID_ARG;
    if (precision != UNIFRAC_FP32 && precision != UNIFRAC_FP64) return UNIFRAC_ERR_INVALID_ARG;
    if (N > UNIFRAC_NOALLOC_MAX_SAMPLES || K > UNIFRAC_NOALLOC_MAX_PERMS) {
        char b[256];
        snprintf(b, sizeof(b), "unifrac_mantel_pearson_noalloc: n_samples = %d, n_perms = %d beyond the static workspace "
                 "(UNIFRAC_NOALLOC_MAX_SAMPLES = %d, UNIFRAC_NOALLOC_MAX_PERMS = %d); use unifrac_mantel_pearson",
                 (int)N, (int)K, UNIFRAC_NOALLOC_MAX_SAMPLES, UNIFRAC_NOALLOC_MAX_PERMS);
        g_cuda_err = b;
        return UNIFRAC_ERR_UNSUPPORTED;
    }
    cudaStream_t st = reinterpret_cast<cudaStream_t>(stream);
    int rc = UNIFRAC_OK;
    try {
        NoAllocBump bump{noalloc_scratch_of_current_device(), (size_t)UNIFRAC_NOALLOC_SCRATCH_BYTES, 0};
        Arena A{noalloc_bump, &bump, st};               // fn != NULL: the arena owns nothing and release() frees nothing
        if (precision == UNIFRAC_FP32) run_mantel<float>(N, reinterpret_cast<const float*>(x), reinterpret_cast<const float*>(y), perms, K, out, A, st);
        else run_mantel<double>(N, reinterpret_cast<const double*>(x), reinterpret_cast<const double*>(y), perms, K, out, A, st);
    } catch (const CudaFail& f) {
        char b[512];
        snprintf(b, sizeof(b), "%s: %s (unifrac_b200.cu:%d)", f.what, cudaGetErrorString(f.e), f.line);
        g_cuda_err = b; cudaGetLastError(); rc = UNIFRAC_ERR_CUDA;
    } catch (const WorkspaceFail&) { rc = UNIFRAC_ERR_WORKSPACE; g_cuda_err = "unifrac_mantel_pearson_noalloc: static workspace exhausted"; }
    catch (const StatusFail& f) { rc = f.status; }
    catch (...) { rc = UNIFRAC_ERR_CUDA; g_cuda_err = "unexpected C++ exception"; }
    return rc;
}

int unifrac_mantel_spearman(int32_t N, const void* x, const void* y, unifrac_precision_t precision, const int32_t* perms,
                            int32_t K, double* out, unifrac_alloc_fn alloc, void* user, void* stream)
{
    if (!x || !y || !out || K < 0 || (K > 0 && !perms) || N < 3) return UNIFRAC_ERR_INVALID_ARG;
    if (precision != UNIFRAC_FP32 && precision != UNIFRAC_FP64) return UNIFRAC_ERR_INVALID_ARG;
    cudaStream_t st = reinterpret_cast<cudaStream_t>(stream);
    Arena A{alloc, user, st};
    int rc = UNIFRAC_OK;
    try {
        if (precision == UNIFRAC_FP32) run_spearman<float>(N, reinterpret_cast<const float*>(x), reinterpret_cast<const float*>(y), perms, K, out, A, st);
        else run_spearman<double>(N, reinterpret_cast<const double*>(x), reinterpret_cast<const double*>(y), perms, K, out, A, st);
    } catch (const CudaFail& f) {
        char b[512];
        snprintf(b, sizeof(b), "%s: %s (unifrac_b200.cu:%d)", f.what, cudaGetErrorString(f.e), f.line);
        g_cuda_err = b; cudaGetLastError(); rc = UNIFRAC_ERR_CUDA;
    } catch (const WorkspaceFail&) { rc = UNIFRAC_ERR_WORKSPACE; }
    catch (const StatusFail& s) { rc = s.status; }
    catch (...) { rc = UNIFRAC_ERR_CUDA; g_cuda_err = "unexpected C++ exception"; }
    if (rc != UNIFRAC_OK) A.release();
    return rc;
}

int unifrac_pcoa(int32_t N, const void* d, unifrac_precision_t precision, int32_t k, int32_t max_iter, double tol, double* out,
                 int32_t* iterations, unifrac_alloc_fn alloc, void* user, void* stream)
{
    if (!d || !out || N < 3 || k < 1 || k > 16 || k >= N || !(tol >= 0.0)) return UNIFRAC_ERR_INVALID_ARG;
    if (precision != UNIFRAC_FP32 && precision != UNIFRAC_FP64) return UNIFRAC_ERR_INVALID_ARG;
    if ((long long)N > (1ll << 20)) return UNIFRAC_ERR_UNSUPPORTED;
    cudaStream_t st = reinterpret_cast<cudaStream_t>(stream);
    Arena A{alloc, user, st};
    int rc = UNIFRAC_OK;
    try {
        if (precision == UNIFRAC_FP32) run_pcoa<float>(N, reinterpret_cast<const float*>(d), k, max_iter, tol, out, iterations, A, st);
        else run_pcoa<double>(N, reinterpret_cast<const double*>(d), k, max_iter, tol, out, iterations, A, st);
    } catch (const CudaFail& f) {
        char b[512];
        snprintf(b, sizeof(b), "%s: %s (unifrac_b200.cu:%d)", f.what, cudaGetErrorString(f.e), f.line);
        g_cuda_err = b; cudaGetLastError(); rc = UNIFRAC_ERR_CUDA;
    } catch (const WorkspaceFail&) { rc = UNIFRAC_ERR_WORKSPACE; }
    catch (const StatusFail& s) { rc = s.status; }
    catch (...) { rc = UNIFRAC_ERR_CUDA; g_cuda_err = "unexpected C++ exception"; }
    if (rc != UNIFRAC_OK) A.release();
    return rc;
}

int unifrac_measure_rates(unifrac_rates_t* out, void* stream)
{
    if (!out) return UNIFRAC_ERR_INVALID_ARG;
    cudaStream_t st = reinterpret_cast<cudaStream_t>(stream);
    int rc = UNIFRAC_OK;
    float* buf = nullptr; unsigned int* sink = nullptr;
    cudaEvent_t e[2] = {nullptr, nullptr};
    try {
        int dev = 0, n_sm = 0, khz = 0;
        CU(cudaGetDevice(&dev));
        CU(cudaDeviceGetAttribute(&n_sm, cudaDevAttrMultiProcessorCount, dev));
        CU(cudaDeviceGetAttribute(&khz, cudaDevAttrClockRate, dev));
        const uint32_t cells = (48u << 20) / 4u;
        CU(cudaMallocAsync(reinterpret_cast<void**>(&buf), (size_t)cells * 4, st));
        CU(cudaMallocAsync(reinterpret_cast<void**>(&sink), 256, st));
        CU(cudaMemsetAsync(buf, 0, (size_t)cells * 4, st));
        CU(cudaMemsetAsync(sink, 0, 256, st));
        CU(cudaEventCreate(&e[0])); CU(cudaEventCreate(&e[1]));
        const size_t smem = 128 * 128 * 4;
        CU(cudaFuncSetAttribute(k_rate_atoms, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
        auto timed = [&](auto&& launch) {
            launch();                                        // warm-up
            CU(cudaEventRecord(e[0], st));
            launch();
            CU(cudaEventRecord(e[1], st));
            CU(cudaEventSynchronize(e[1]));
            float ms = 0; CU(cudaEventElapsedTime(&ms, e[0], e[1]));
            return (double)ms * 1e-3;
        };
        const int it_a = 4096, it_r = 512;
        const unsigned ga = (unsigned)n_sm * 3, gr = (unsigned)n_sm * 8;
        double t0 = timed([&] { k_rate_atoms<<<ga, 512, smem, st>>>(0, it_a, sink); CU_LAUNCH(); });
        double t1 = timed([&] { k_rate_atoms<<<ga, 512, smem, st>>>(1, it_a, sink); CU_LAUNCH(); });
        double t2 = timed([&] { k_rate_red<<<gr, 256, 0, st>>>(buf, cells, it_r); CU_LAUNCH(); });
        out->smem_atomic_conflict_free_per_s = (double)ga * 512 * it_a * 8 / t0;
        out->smem_atomic_random_per_s = (double)ga * 512 * it_a * 8 / t1;
        out->l2_red_random_per_s = (double)gr * 256 * it_r * 4 / t2;
        const int it_f = 8192;
        const unsigned gf = (unsigned)n_sm * 8;
        float* fsink = buf;
        double t3 = timed([&] { k_rate_alu<0><<<gf, 256, 0, st>>>(it_f, fsink); CU_LAUNCH(); });
        double t4 = timed([&] { k_rate_alu<1><<<gf, 256, 0, st>>>(it_f, fsink); CU_LAUNCH(); });
        double t5 = timed([&] { k_rate_alu<2><<<gf, 256, 0, st>>>(it_f, fsink); CU_LAUNCH(); });
        out->fmnmx_per_s = (double)gf * 256 * it_f * 8 / t3;
        out->fadd_per_s = (double)gf * 256 * it_f * 8 / t4;
        out->fmnmx_fadd_per_s = (double)gf * 256 * it_f * 16 / t5;
        double t6 = timed([&] { k_rate_alu<3><<<gf, 256, 0, st>>>(it_f, fsink); CU_LAUNCH(); });
        double t7 = timed([&] { k_rate_alu<4><<<gf, 256, 0, st>>>(it_f, fsink); CU_LAUNCH(); });
        double t8 = timed([&] { k_rate_alu<5><<<gf, 256, 0, st>>>(it_f, fsink); CU_LAUNCH(); });
        out->fadd2_per_s = (double)gf * 256 * it_f * 8 / t6;               // 4 FADD2 = 8 lane-ops per iteration
        out->fmnmx2_fadd2_updates_per_s = (double)gf * 256 * it_f * 8 / t7;
        out->dense16_mix_updates_per_s = (double)gf * 256 * it_f * 8 / t8;
        out->sm_count = n_sm; out->sm_clock_khz = khz;
    } catch (const CudaFail& f) {
        char b[512];
        snprintf(b, sizeof(b), "%s: %s (unifrac_b200.cu:%d)", f.what, cudaGetErrorString(f.e), f.line);
        g_cuda_err = b; cudaGetLastError(); rc = UNIFRAC_ERR_CUDA;
    } catch (...) { rc = UNIFRAC_ERR_CUDA; g_cuda_err = "unexpected C++ exception"; }
    if (e[0]) cudaEventDestroy(e[0]);
    if (e[1]) cudaEventDestroy(e[1]);
    if (buf) cudaFreeAsync(buf, st);
    if (sink) cudaFreeAsync(sink, st);
    cudaStreamSynchronize(st);
    return rc;
}

const char* unifrac_status_string(int status)
{
    switch (status) {
        case UNIFRAC_OK: return "ok";
        case UNIFRAC_ERR_INVALID_ARG: return "invalid argument";
        case UNIFRAC_ERR_INVALID_TREE: return "invalid tree";
        case UNIFRAC_ERR_INVALID_TABLE: return "invalid table";
        case UNIFRAC_ERR_EMPTY_SAMPLE: return "empty sample";
        case UNIFRAC_ERR_WORKSPACE: return "workspace allocation failed";
        case UNIFRAC_ERR_CUDA: return "CUDA error";
        case UNIFRAC_ERR_UNSUPPORTED: return "unsupported size";
        default: return "unknown status";
    }
}

const char* unifrac_last_cuda_error(void) { return g_cuda_err.c_str(); }
int unifrac_abi_version(void) { return 8; }

}  // extern "C"
