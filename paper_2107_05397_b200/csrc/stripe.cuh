// stripe.cuh -- steps a-5 (stripe/tile accumulation, THE hot loop) and a-6 (finalize, fused as the
// epilogue).  BASELINE.json:5 subsystems (2)+(3); PAPER.md:23,29 ("Striped UniFrac", "a set of
// stripes").  DESIGN.md "K2 stripe kernel".
//
// One persistent CTA = 8 consumer warps + 1 producer warp.  A CTA owns one 128 x 128 tile pair
// (I, J), I <= J, of the upper triangle at a time (dynamic queue).  For that pair the producer warp
// walks the two tiles' row-flag bitmaps, and for every branch present in BOTH tiles (separable
// "min" form, identities I2-I5) or in EITHER tile (direct |u-v| form, flag ABSDIFF) stages the two
// 128-value embedding rows into a shared-memory ring with cp.async.bulk (TMA bulk copy, mbarrier
// complete_tx).  Consumer warp w owns the 32 x 64 sub-tile (quarter wi = w/2 of I, half wj = w%2
// of J) as an 8 x 8 register tile per thread and executes, per staged row it needs (4-bit
// quarter masks -> per-row 8-bit "need" byte),
//     acc[a][b] += min(u~_i[a], u~_j[b])        (FMNMX + FADD)      or
//     acc[a][b] += |u~_i[a] - u~_j[b]|           (FADD + FADD|.|)
// Every FLUSH_STAGES stages the fp32 register accumulators are folded into per-thread fp64 partial
// sums (blocked summation).  The epilogue (a-6) combines them with the
// per-sample side sums and writes the condensed matrix:
//     weighted   : d = (R_i + R_j - 2M) / (R_i + R_j)            [min form]   d = A / (R_i + R_j)        [direct]
//     unweighted : d = (S_i + S_j - 2G) / (S_i + S_j - G)        [min form]   d = 2A / (S_i + S_j + A)   [direct, I4]
#pragma once
#include "common.cuh"

namespace ufb {

// ------------------------------------------------------------------ PTX helpers (mbarrier, bulk copy)
__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(uint32_t bar, uint32_t count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint32_t bar) {
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(bar) : "memory");
}
__device__ __forceinline__ void mbar_arrive_expect_tx(uint32_t bar, uint32_t tx) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(tx) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t parity) {
    uint32_t ok;
    do {
        asm volatile("{\n\t.reg .pred p;\n\tmbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\t"
                     "selp.u32 %0, 1, 0, p;\n\t}"
                     : "=r"(ok) : "r"(bar), "r"(parity) : "memory");
    } while (!ok);
}
// TMA bulk copy global -> shared, completion signalled on an mbarrier (SASS: UBLKCP)
__device__ __forceinline__ void bulk_g2s(uint32_t dst, const void* src, uint32_t bytes, uint32_t bar) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                 ::"r"(dst), "l"(src), "r"(bytes), "r"(bar) : "memory");
}

// ------------------------------------------------------------------ configuration
template <typename T> struct StripeCfg;
template <> struct StripeCfg<float>  { static constexpr int RPS = 32, STAGES = 4, MINB = 1, FLUSH_STAGES = 16; };
template <> struct StripeCfg<double> { static constexpr int RPS = 16, STAGES = 4, MINB = 1, FLUSH_STAGES = 1 << 30; };

constexpr int STRIPE_THREADS = 288;      // 8 consumer warps + 1 producer warp
constexpr int PEND_CAP = 32 + 1024;
constexpr uint32_t ROW_NONE = 0xffffffffu;
constexpr int META_LAST = 1, META_DONE = 2;

enum StripeForm { FORM_MIN = 0, FORM_ABSDIFF = 1 };

struct StripeParams {
    const void* const* tileE;     // [n_tiles] compact embedding rows, [rows][128] of T
    const uint8_t* const* tileQ;  // [n_tiles] quarter masks per compact row
    const uint32_t* flags;        // [n_tiles][nwords] row-present bits
    const uint32_t* rank;         // [n_tiles][nwords] exclusive row ranks per word
    uint32_t nwords;
    const int2* pairs;            // tile pairs (I <= J)
    uint32_t n_pairs;
    uint32_t* counter;            // dynamic tile-pair queue
    const double* sums;           // [n_tiles*128] R_s or S_s
    int n_samples;
    int weighted;
    void* out;                    // condensed, T
    double* scratch;              // [grid][64][256] fp64 partial sums
    unsigned long long* stats;    // [0] rows executed by consumer warps, [1] rows staged
    const void* zero_row;         // 128 zero values of T (16-byte aligned)
    int add_out;                  // min form: out[] already holds the tail branches' sum of min(u~_a,u~_b) (tail.cuh)
    GuardList guard;              // min form: pairs with d < GUARD_THETA are listed for k_guard (guard.cuh)
};

template <typename T>
constexpr size_t stripe_smem_bytes() {
    return (size_t)StripeCfg<T>::STAGES * StripeCfg<T>::RPS * 2 * TILE * sizeof(T)   // ring
         + (size_t)StripeCfg<T>::STAGES * 32                                         // need bytes
         + (size_t)StripeCfg<T>::STAGES * 16                                         // meta
         + (size_t)StripeCfg<T>::STAGES * 2 * 8                                      // mbarriers
         + (size_t)PEND_CAP * 2 * 4;                                                 // pending row ranks
}

template <typename T> struct VecLd;
template <> struct VecLd<float> {
    static constexpr int VEC = 4;
    static __device__ __forceinline__ void ld(const float* p, float* d) { float4 v = *reinterpret_cast<const float4*>(p); d[0] = v.x; d[1] = v.y; d[2] = v.z; d[3] = v.w; }
};
template <> struct VecLd<double> {
    static constexpr int VEC = 2;
    static __device__ __forceinline__ void ld(const double* p, double* d) { double2 v = *reinterpret_cast<const double2*>(p); d[0] = v.x; d[1] = v.y; }
};

template <typename T, int FORM>
__global__ void __launch_bounds__(STRIPE_THREADS, StripeCfg<T>::MINB)
k_stripe(const StripeParams P)
{
    using Cfg = StripeCfg<T>;
    constexpr int RPS = Cfg::RPS, STAGES = Cfg::STAGES;
    constexpr int VEC = VecLd<T>::VEC, NV = 8 / VEC;
    constexpr uint32_t ROWBYTES = TILE * sizeof(T);

    extern __shared__ __align__(128) unsigned char smem[];
    T* ring = reinterpret_cast<T*>(smem);
    unsigned char* p = smem + (size_t)STAGES * RPS * 2 * TILE * sizeof(T);
    uint8_t* needb = p;                              p += STAGES * 32;
    int4* meta = reinterpret_cast<int4*>(p);         p += STAGES * 16;
    uint64_t* full = reinterpret_cast<uint64_t*>(p); p += STAGES * 8;
    uint64_t* empty = reinterpret_cast<uint64_t*>(p); p += STAGES * 8;
    uint32_t* pendI = reinterpret_cast<uint32_t*>(p); p += PEND_CAP * 4;
    uint32_t* pendJ = reinterpret_cast<uint32_t*>(p);

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;

    if (threadIdx.x == 0) {
        for (int s = 0; s < STAGES; ++s) { mbar_init(smem_u32(&full[s]), 1); mbar_init(smem_u32(&empty[s]), 8); }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();

    if (warp == 8) {
        // =========================================================== producer warp
        uint32_t stage = 0, phase = 0;
        unsigned long long staged = 0;
        int tile_pair = 0;
        uint32_t npend = 0;
        const T* EI = nullptr; const T* EJ = nullptr; const uint8_t* QI = nullptr; const uint8_t* QJ = nullptr;

        auto emit = [&](uint32_t head, uint32_t cnt, int mflags) {
            mbar_wait(smem_u32(&empty[stage]), phase ^ 1u);
            uint32_t ri = ROW_NONE, rj = ROW_NONE;
            if ((uint32_t)lane < cnt) {
                ri = pendI[head + lane]; rj = pendJ[head + lane];
                uint32_t qi = ri != ROW_NONE ? QI[ri] : 0u;
                uint32_t qj = rj != ROW_NONE ? QJ[rj] : 0u;
                uint32_t need = 0;
#pragma unroll
                for (int w = 0; w < 8; ++w) {
                    bool bi = (qi >> (w >> 1)) & 1u;
                    bool bj = ((qj >> ((w & 1) * 2)) & 3u) != 0u;
                    bool nd = FORM == FORM_MIN ? (bi && bj) : (bi || bj);
                    need |= (nd ? 1u : 0u) << w;
                }
                needb[stage * 32 + lane] = (uint8_t)need;
            }
            __syncwarp();
            if (lane == 0) {
                meta[stage] = make_int4((int)cnt, tile_pair, mflags, 0);
                if (cnt) mbar_arrive_expect_tx(smem_u32(&full[stage]), cnt * 2u * ROWBYTES);
                else mbar_arrive(smem_u32(&full[stage]));
            }
            __syncwarp();
            if ((uint32_t)lane < cnt) {
                T* dst = ring + ((size_t)stage * RPS + lane) * 2 * TILE;
                const void* si = ri != ROW_NONE ? (const void*)(EI + (size_t)ri * TILE) : P.zero_row;
                const void* sj = rj != ROW_NONE ? (const void*)(EJ + (size_t)rj * TILE) : P.zero_row;
                bulk_g2s(smem_u32(dst), si, ROWBYTES, smem_u32(&full[stage]));
                bulk_g2s(smem_u32(dst + TILE), sj, ROWBYTES, smem_u32(&full[stage]));
            }
            staged += cnt;
            if (++stage == STAGES) { stage = 0; phase ^= 1u; }
        };

        for (;;) {
            if (lane == 0) tile_pair = (int)atomicAdd(P.counter, 1u);
            tile_pair = __shfl_sync(0xffffffffu, tile_pair, 0);
            if ((uint32_t)tile_pair >= P.n_pairs) { emit(0, 0, META_DONE); break; }
            const int2 ij = P.pairs[tile_pair];
            const uint32_t* fI = P.flags + (size_t)ij.x * P.nwords;
            const uint32_t* fJ = P.flags + (size_t)ij.y * P.nwords;
            const uint32_t* rkI = P.rank + (size_t)ij.x * P.nwords;
            const uint32_t* rkJ = P.rank + (size_t)ij.y * P.nwords;
            EI = reinterpret_cast<const T*>(P.tileE[ij.x]); EJ = reinterpret_cast<const T*>(P.tileE[ij.y]);
            QI = P.tileQ[ij.x]; QJ = P.tileQ[ij.y];
            npend = 0;
            for (uint32_t w0 = 0; w0 < P.nwords; w0 += 32) {
                uint32_t w = w0 + lane;
                uint32_t fi = 0, fj = 0;
                if (w < P.nwords) { fi = fI[w]; fj = fJ[w]; }
                uint32_t m = FORM == FORM_MIN ? (fi & fj) : (fi | fj);
                uint32_t c = __popc(m), incl = c;
#pragma unroll
                for (int o = 1; o < 32; o <<= 1) { uint32_t t = __shfl_up_sync(0xffffffffu, incl, o); if (lane >= o) incl += t; }
                uint32_t total = __shfl_sync(0xffffffffu, incl, 31);
                if (total == 0) continue;
                uint32_t pos = npend + incl - c;
                if (m) {
                    uint32_t ri0 = rkI[w], rj0 = rkJ[w];
                    while (m) {
                        int b = __ffs(m) - 1;
                        m &= m - 1;
                        uint32_t below = (1u << b) - 1u;
                        pendI[pos] = ((fi >> b) & 1u) ? ri0 + __popc(fi & below) : ROW_NONE;
                        pendJ[pos] = ((fj >> b) & 1u) ? rj0 + __popc(fj & below) : ROW_NONE;
                        ++pos;
                    }
                }
                npend += total;
                __syncwarp();
                uint32_t head = 0;
                while (npend - head >= (uint32_t)RPS) { emit(head, RPS, 0); head += RPS; }
                uint32_t rem = npend - head;              // < RPS <= 32
                if (head) {
                    uint32_t vi = 0, vj = 0;
                    if ((uint32_t)lane < rem) { vi = pendI[head + lane]; vj = pendJ[head + lane]; }
                    __syncwarp();
                    if ((uint32_t)lane < rem) { pendI[lane] = vi; pendJ[lane] = vj; }
                    __syncwarp();
                }
                npend = rem;
            }
            emit(0, npend, META_LAST);
        }
        if (lane == 0 && staged) atomicAdd(&P.stats[1], staged);
        return;
    }

    // =============================================================== consumer warps
    const int wi = warp >> 1, wj = warp & 1;
    const int ty = lane >> 3, tx = lane & 7;
    // element a of the i side: local index  (a/VEC)*(4*VEC) + ty*VEC + a%VEC   within the warp's 32 rows
    // element b of the j side: local index  (b/VEC)*(8*VEC) + tx*VEC + b%VEC   within the warp's 64 columns
    const int i_off = wi * 32 + ty * VEC;
    const int j_off = TILE + wj * 64 + tx * VEC;
    double* my_scratch = P.scratch + (size_t)blockIdx.x * 64 * 256 + threadIdx.x;

    T acc[8][8];
#pragma unroll
    for (int a = 0; a < 8; ++a)
#pragma unroll
        for (int b = 0; b < 8; ++b) acc[a][b] = (T)0;
    uint32_t stage = 0, phase = 0;
    int since_flush = 0;
    bool scratch_live = false;
    unsigned long long rows_exec = 0;

    for (;;) {
        mbar_wait(smem_u32(&full[stage]), phase);
        const int4 m = meta[stage];
        if (m.z & META_DONE) break;
        uint32_t nb = lane < m.x ? (uint32_t)needb[stage * 32 + lane] : 0u;
        uint32_t mask = __ballot_sync(0xffffffffu, (nb >> warp) & 1u);
        rows_exec += __popc(mask);
        const T* base = ring + (size_t)stage * RPS * 2 * TILE;
        while (mask) {
            int r = __ffs(mask) - 1;
            mask &= mask - 1;
            const T* row = base + (size_t)r * 2 * TILE;
            T ai[8], bj[8];
#pragma unroll
            for (int k = 0; k < NV; ++k) {
                VecLd<T>::ld(row + i_off + k * 4 * VEC, ai + k * VEC);
                VecLd<T>::ld(row + j_off + k * 8 * VEC, bj + k * VEC);
            }
#pragma unroll
            for (int a = 0; a < 8; ++a)
#pragma unroll
                for (int b = 0; b < 8; ++b) {
                    if (FORM == FORM_MIN) acc[a][b] += fmin(ai[a], bj[b]);
                    else acc[a][b] += fabs(ai[a] - bj[b]);
                }
        }
        __syncwarp();
        if (lane == 0) mbar_arrive(smem_u32(&empty[stage]));
        if (++stage == STAGES) { stage = 0; phase ^= 1u; }

        const bool last = (m.z & META_LAST) != 0;
        if (!last) {
            if (++since_flush >= Cfg::FLUSH_STAGES) {
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
            continue;
        }

        // ----------------------------------------------------------- a-6 finalize (epilogue of the tile pair)
        const int2 ij = P.pairs[m.y];
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
                    double num, den;
                    if (FORM == FORM_MIN && P.add_out) tot += (double)reinterpret_cast<const T*>(P.out)[rowbase + gj];
                    if (FORM == FORM_MIN) {
                        num = ss - 2.0 * tot;
                        den = P.weighted ? ss : ss - tot;
                    } else {
                        num = P.weighted ? tot : 2.0 * tot;
                        den = P.weighted ? ss : ss + tot;
                    }
                    if (num < 0.0) num = 0.0;
                    if (FORM == FORM_MIN) guard_note(P.guard, num, den, (uint32_t)gi, (uint32_t)gj);
                    double d = den > 0.0 ? num / den : 0.0;
                    reinterpret_cast<T*>(P.out)[rowbase + gj] = (T)d;
                }
            }
        }
        scratch_live = false;
        since_flush = 0;
    }
    if (lane == 0 && rows_exec) atomicAdd(&P.stats[0], rows_exec);
}

// ------------------------------------------------------------------ literal debug kernel (flag LITERAL)
// One CTA per tile pair, one thread per pair, BOTH sums accumulated pairwise in fp64 exactly as
// BASELINE.json:5 words them.  Reads the compact embedding straight from global memory.
template <typename T>
__global__ void __launch_bounds__(256)
k_literal(const StripeParams P)
{
    const int2 ij = P.pairs[blockIdx.x];
    const uint32_t* fI = P.flags + (size_t)ij.x * P.nwords;
    const uint32_t* fJ = P.flags + (size_t)ij.y * P.nwords;
    const uint32_t* rkI = P.rank + (size_t)ij.x * P.nwords;
    const uint32_t* rkJ = P.rank + (size_t)ij.y * P.nwords;
    const T* EI = reinterpret_cast<const T*>(P.tileE[ij.x]);
    const T* EJ = reinterpret_cast<const T*>(P.tileE[ij.y]);
    const long long N = P.n_samples;
    for (int q = threadIdx.x; q < TILE * TILE; q += blockDim.x) {
        const int i = q >> 7, j = q & 127;
        const long long gi = (long long)ij.x * TILE + i, gj = (long long)ij.y * TILE + j;
        if (!(gi < gj && gj < N)) continue;
        double num = 0.0, den = 0.0;
        for (uint32_t w = 0; w < P.nwords; ++w) {
            const uint32_t fi = fI[w], fj = fJ[w];
            uint32_t m = fi | fj;
            while (m) {
                const int b = __ffs(m) - 1;
                m &= m - 1;
                const uint32_t below = (1u << b) - 1u;
                double x = 0.0, y = 0.0;
                if ((fi >> b) & 1u) x = (double)EI[(size_t)(rkI[w] + __popc(fi & below)) * TILE + i];
                if ((fj >> b) & 1u) y = (double)EJ[(size_t)(rkJ[w] + __popc(fj & below)) * TILE + j];
                num += fabs(x - y);                          // len*|u-v|   or   len*(x xor y)
                den += P.weighted ? (x + y) : fmax(x, y);    // len*(u+v)   or   len*(x or y)
            }
        }
        const double d = den > 0.0 ? num / den : 0.0;
        reinterpret_cast<T*>(P.out)[gi * (2 * N - gi - 1) / 2 + (gj - gi - 1)] = (T)d;
    }
}

}  // namespace ufb
