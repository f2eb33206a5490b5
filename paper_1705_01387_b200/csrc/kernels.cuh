// sm_100a kernels of the GPUQT hot path.  See include/gpuqt.h for the boundary and DESIGN.md for
// the layout, the byte model and the roofline of each kernel.
//
// Layout
//   vectors   complex fp64 [N][B] as double2: the B vectors of a row are contiguous (16*B bytes),
//             so one neighbour index serves one 16*B-byte gather (B = 8: one 128-byte line).
//   matrix    packed sliced ELL.  A slice is 32 consecutive rows; slice s of width w is ONE
//             contiguous record, column-major inside the record:
//                 double hre[w][32] (per-entry variants) | double him[w][32] (complex variant) |
//                 double onsite[32] | int32 col[w][32]
//             record bytes = 32 * (8 w nd + 8 + 4 w), nd = doubles per entry (0, 1, 2), a multiple
//             of 128.  Records are stored back to back; slice_off[s] is the byte offset of record
//             s.  Padding entries are (own row, hop 0.0); in the constant-hopping variant (nd = 0:
//             every stored hopping is the same real number, kept in Mat::hop_const) padding is
//             col = N: every vector buffer carries an all-zero row N (and x[N] = 0), so the walk
//             needs no guard.  One record = one 1-D TMA bulk copy.
//   warp      the unit of work is (consumer warp, slice).  A stage of a warp's shared-memory pipeline
//             holds everything the slice streams from HBM exactly once: the packed record, the
//             slice's own rows of T_{m-1} (and e_{m-1}) and of T_{m-2} (and e_{m-2}) -- each one
//             1-D TMA bulk copy (cp.async.bulk + mbarrier) issued by the CTA's producer warp one or
//             more slices ahead, so the DRAM streams never sit on a consumer's scoreboard and there
//             is no CTA-wide barrier in the loop.  A consumer walks the slice in rounds of 32/LPR
//             rows; a lane owns V = 2 consecutive vectors of a row (256-bit accesses) and LPR = B/V
//             lanes share a row.  Neighbours inside the slice are read from the staged rows in
//             shared memory; the others are gathered from global memory (L2 hits along the sweep
//             front), all gathers of a round issued back to back.  Stores of a warp are one
//             contiguous segment.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#ifndef GPUQT_THREADS
#define GPUQT_THREADS 256
#endif

#ifndef GPUQT_MINB
#define GPUQT_MINB 2
#endif
#ifndef GPUQT_MINB_MSD
#define GPUQT_MINB_MSD 1
#endif

// L2 policy experiments
#ifndef GPUQT_GATHER_POLICY   // 0: plain ld.global, 1: L2::evict_last
#define GPUQT_GATHER_POLICY 1
#endif
#ifndef GPUQT_IN_POLICY       // own rows of T_{m-1} by TMA: 0 no hint, 1 evict_last
#define GPUQT_IN_POLICY 0
#endif
#ifndef GPUQT_ST_POLICY       // stores of T_m / acc: 0 plain, 1 st.global.cs (evict-first)
#define GPUQT_ST_POLICY 0
#endif

namespace gpuqt {

constexpr int kThreads = GPUQT_THREADS;
constexpr int kWarps = kThreads / 32;
constexpr int kSlice = 32;
constexpr int kMaxStages = 4;

// nd = doubles stored per entry: 0 constant real hopping, 1 real, 2 complex
__host__ __device__ __forceinline__ long long record_bytes(int w, int nd) {
    return 32LL * (8LL * w * nd + 8 + 4LL * w);
}
__host__ __device__ __forceinline__ int record_width(long long bytes, int nd) {
    return (int)((bytes / 32 - 8) / (4 + 8 * nd));
}
// kHopConst16: constant hopping AND 16-bit columns -- the record is
//     double onsite[32] | int32 base[8] (first w used) | uint16 delta[w][32],   col = base[k] + delta[k][lane]
// (uniform tables without padding whose columns spread less than 65536 inside every (slice, k); lattices
// in natural order do).  288 + 64 w bytes instead of 256 + 128 w.
enum Hop : int { kHopReal = 0, kHopComplex = 1, kHopConst = 2, kHopConst16 = 3 };
__host__ __device__ constexpr bool hop_is_const(int hop) { return hop == kHopConst || hop == kHopConst16; }
__host__ __device__ constexpr int hop_doubles(int hop) { return hop_is_const(hop) ? 0 : hop == kHopComplex ? 2 : 1; }
__host__ __device__ __forceinline__ long long hop_record_bytes(int w, int hop) {
    return hop == kHopConst16 ? 288LL + 64LL * w : record_bytes(w, hop_doubles(hop));
}

struct Mat {
    const unsigned char* __restrict__ rec;      // packed slice records
    const long long* __restrict__ slice_off;    // [n_slices + 1] byte offsets (ragged variant)
    const double* __restrict__ x;               // [N + 1], x[N] = 0
    long long N;
    long long n_slices;
    int K;                                      // K_max
    int uniform;                                // every record has width K
    int cplx;
    int hop;                                    // Hop variant of the records
    double hop_const;                           // kHopConst: the one hopping value
    double inv_dE;
    double box;                                 // <= 0: open boundary
};

enum Mode : int {
    kModeDoubling = 0,   // T_new, dots |T_new|^2, Re<T_new|T_in>, |T_in|^2          (Eq. 28, 30)
    kModeLeft = 1,       // T_new, dot <phi_L|T_new>                                 (Eq. 29)
    kModeEvolve = 2,     // Clenshaw term b_k = c_k src + 2 H~ b_{k+1} - b_{k+2}      (Eq. 17, 21)
    kModeEvolveMsd = 3,  // the same for the (a, e) pair, [X,H~] weights in the walk (Eq. 18, 22)
};

// Operands of one recurrence step.  A launch performs one step, or two consecutive steps fused
// through L2 (see cheb_step_kernel): io[0] is T_m = 2 H~ T_{m-1} - T_{m-2}, io[1] is T_{m+1}.
struct StepIO {
    const double2* in;       // T_{m-1}: gathered and own row
    const double2* prev;     // T_{m-2}: own row (unused when first)
    double2* out;            // T_m (unused when !store)
    const double2* in_e;     // MSD pair: e_{m-1}
    const double2* prev_e;   //           e_{m-2}
    double2* out_e;          //           e_m
    // B >= 2: device addresses of the TMA tensor maps (CUtensorMap, 128-byte swizzle) of in / prev / in_e / prev_e
    const void *tm_in, *tm_prev, *tm_in_e, *tm_prev_e;
    double cr, ci;           // c_m
    double* result;          // [Q][B] reduced dots of this step
    int store;               // write T_m (0 on the last term of an evolve)
    int pad_;
};

struct StepArgs {
    StepIO io[2];
    const double2* __restrict__ src;     // evolve: the vector being evolved (psi; a; b), read-only
    const double2* __restrict__ src_e;   // evolve MSD: chi
    const double2* __restrict__ phiL;    // kModeLeft
    int first;                           // no T_{m-2} term (first launch of a recurrence); single-step launches only
    int half;                            // factor 1 instead of 2 on H~ (T_1 = H~ T_0; last Clenshaw term); single-step only
    int n_steps;                         // 1, or 2 (fused pair, scheduled by `sched`)
    int reverse;                         // sweep the slices from the top (L2 reuse between launches)
    int run;                             // consecutive slices one CTA walks before jumping (multiple of kWarps)
    int stages;                          // shared-memory stages per warp (<= kMaxStages)
    int stage_bytes;                     // bytes of one stage: record + staged vector rows
    int rec_bytes;                       // bytes reserved for the record inside a stage
    double* partials;                    // [grid][n_steps*Q*B]
    unsigned int* ticket;
    // fused pair: item t (taken by CTA t % G) = {run | step << 30 (run = kNoRun: nothing to do), -1};
    // a second-step item of run R waits until run_done[r] == kWarps for r in dep_list[dep_ptr[R] ..
    // dep_ptr[R+1]) (the first-step runs it gathers T_m from)
    const int2* sched;
    int n_items;
    unsigned int* run_done;              // [runs] warps that have finished the first step of the run
    const int* dep_ptr;
    const int* dep_list;
};
constexpr int kNoRun = (1 << 30) - 1;

// ------------------------------------------------------------------ PTX helpers (TMA / mbarrier)
__device__ __forceinline__ uint32_t smem_u32(const void* p) {
    return (uint32_t)__cvta_generic_to_shared(p);
}
__device__ __forceinline__ void mbar_init(uint64_t* bar, uint32_t count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count));
}
__device__ __forceinline__ void fence_mbar_init() {
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t* bar, uint32_t bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes)
                 : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t* bar, uint32_t parity) {
    asm volatile(
        "{\n"
        ".reg .pred P1;\n"
        "LAB_WAIT:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 P1, [%0], %1;\n"
        "@P1 bra DONE;\n"
        "bra LAB_WAIT;\n"
        "DONE:\n"
        "}" ::"r"(smem_u32(bar)),
        "r"(parity)
        : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint64_t* bar) {
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ bool mbar_test(uint64_t* bar, uint32_t parity) {
    uint32_t ok;
    asm volatile(
        "{\n"
        ".reg .pred P1;\n"
        "mbarrier.test_wait.parity.shared::cta.b64 P1, [%1], %2;\n"
        "selp.u32 %0, 1, 0, P1;\n"
        "}"
        : "=r"(ok)
        : "r"(smem_u32(bar)), "r"(parity)
        : "memory");
    return ok != 0;
}
__device__ __forceinline__ void prefetch_l2(const void* p) {
    asm volatile("prefetch.global.L2 [%0];" ::"l"(p));
}
__device__ __forceinline__ uint64_t policy_evict_first() {
    uint64_t p;
    asm volatile("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;" : "=l"(p));
    return p;
}
// 1-D bulk copy global -> shared through the TMA unit; completion is signalled on `bar`.
__device__ __forceinline__ void bulk_g2s(void* dst, const void* src, uint32_t bytes, uint64_t* bar,
                                         uint64_t policy) {
    asm volatile(
        "cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes.L2::cache_hint [%0], [%1], %2, [%3], %4;" ::
            "r"(smem_u32(dst)),
        "l"(src), "r"(bytes), "r"(smem_u32(bar)), "l"(policy)
        : "memory");
}

__device__ __forceinline__ void bulk_g2s_nohint(void* dst, const void* src, uint32_t bytes, uint64_t* bar) {
    asm volatile(
        "cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::
            "r"(smem_u32(dst)),
        "l"(src), "r"(bytes), "r"(smem_u32(bar))
        : "memory");
}

// 2-D tiled TMA copy global -> shared through a tensor map (box = one slice's rows of one vector set as
// 128-byte lines, 128-byte swizzle); completion is signalled on `bar`.  c1 = index of the first line.
__device__ __forceinline__ void tensor_g2s(void* dst, const void* tmap, int c1, uint64_t* bar) {
    asm volatile(
        "cp.async.bulk.tensor.2d.shared::cluster.global.tile.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3}], [%4];" ::
            "r"(smem_u32(dst)),
        "l"(tmap), "r"(0), "r"(c1), "r"(smem_u32(bar))
        : "memory");
}
__device__ __forceinline__ void tensor_g2s_hint(void* dst, const void* tmap, int c1, uint64_t* bar, uint64_t policy) {
    asm volatile(
        "cp.async.bulk.tensor.2d.shared::cluster.global.tile.mbarrier::complete_tx::bytes.L2::cache_hint [%0], [%1, {%2, %3}], [%4], %5;" ::
            "r"(smem_u32(dst)),
        "l"(tmap), "r"(0), "r"(c1), "r"(smem_u32(bar)), "l"(policy)
        : "memory");
}
// Staged vector rows are written by the TMA with the 128-byte swizzle (16-byte chunk index, address
// bits 4-6, ^= address bits 7-9; box rows are whole 128-byte lines): a lane's two 16-byte reads at a
// 32-byte lane stride then fall on distinct banks for every group of 8 lanes (without it: a 2-way
// bank conflict on every 128-bit read).  Uses the absolute shared address, as the TMA does.
__device__ __forceinline__ uint32_t swz32(uint32_t sa) { return sa ^ ((sa >> 3) & 0x70u); }

__device__ __forceinline__ uint64_t policy_evict_last() {
    uint64_t p;
    asm volatile("createpolicy.fractional.L2::evict_last.b64 %0, 1.0;" : "=l"(p));
    return p;
}
__device__ __forceinline__ void st_vec(double2* p, double2 v) {
#if GPUQT_ST_POLICY == 1
    __stcs(p, v);
#else
    *p = v;
#endif
}
__device__ __forceinline__ void red_release_gpu_inc(unsigned int* p) {
    asm volatile("red.release.gpu.global.add.u32 [%0], 1;" ::"l"(p) : "memory");
}
__device__ __forceinline__ double2 ldcs2(const double2* p) { return __ldcs(p); }

// minimum-image X_n - X_m  [A6]; pure add/sub so it is bit-identical to the oracle's
__device__ __forceinline__ double min_image(double d, double box) {
    if (box > 0.0) {
        if (d > 0.5 * box) d -= box;
        else if (d < -0.5 * box) d += box;
    }
    return d;
}

// Deterministic reduction of Q*B values per CTA.  A lane holds v[q * V + j] for vector
// b = (lane % (B / V)) * V + j.  Warp shuffle over lanes with equal b -> shared memory over warps ->
// per-block partial -> the last block to finish sums the per-block partials in a fixed order (no
// floating-point atomics, run-to-run identical).  result[q * B + b].
template <int B, int Q, int V = 1>
__device__ __forceinline__ void block_reduce_and_finish(double (&v)[Q * V], double* partials,
                                                        unsigned int* ticket, double* result) {
    constexpr int LPR = B / V;   // lanes per row
    __shared__ double s_part[kWarps][Q * B];
    __shared__ double s_tree[kThreads];
    __shared__ int s_last;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
#pragma unroll
    for (int q = 0; q < Q * V; ++q) {
#pragma unroll
        for (int off = 16; off >= LPR; off >>= 1) v[q] += __shfl_xor_sync(0xffffffffu, v[q], off);
    }
    if (lane < LPR) {
#pragma unroll
        for (int q = 0; q < Q; ++q)
#pragma unroll
            for (int j = 0; j < V; ++j) s_part[warp][q * B + lane * V + j] = v[q * V + j];
    }
    __syncthreads();
    if (tid < Q * B) {
        double s = 0.0;
#pragma unroll
        for (int w = 0; w < kWarps; ++w) s += s_part[w][tid];
        partials[(size_t)blockIdx.x * (Q * B) + tid] = s;
    }
    __threadfence();
    __syncthreads();
    if (tid == 0) {
        unsigned int t = atomicAdd(ticket, 1u);
        s_last = (t == gridDim.x - 1);
    }
    __syncthreads();
    if (!s_last) return;
    __threadfence();
    // fixed-shape sum over blocks: thread t handles value (t % P), blocks j, j + S, ...
    constexpr int P = Q * B;                 // <= 32
    constexpr int S = kThreads / P;          // strands per value
    const int pv = tid % P, strand = tid / P;
    double s = 0.0;
    if (strand < S)
        for (unsigned int g = strand; g < gridDim.x; g += S) s += __ldcg(&partials[(size_t)g * P + pv]);
    s_tree[tid] = (strand < S) ? s : 0.0;
    __syncthreads();
    if (tid < P) {
        double tot = 0.0;
        for (int j = 0; j < S; ++j) tot += s_tree[j * P + tid];
        result[tid] = tot;
    }
    if (tid == 0) *ticket = 0u;
}

template <int MODE>
struct ModeTraits {
    static constexpr int Q = (MODE == kModeDoubling) ? 3 : 2;
    static constexpr int kMinBlocks = (MODE == kModeEvolveMsd) ? GPUQT_MINB_MSD : GPUQT_MINB;   // register cap
};

// B = 8: a slice's rows are 4 KB per stream; staging T_{m-2} as well would leave room for one CTA per
// SM only, so T_{m-2} own rows are read by a streaming 256-bit load at the top of the round instead
// (the occupancy is worth more than the TMA staging there; at B <= 4 it is the other way round).
template <int B>
struct PrevDirect {
    static constexpr bool value = (B >= 8);
};

// Number of vector streams staged per slice: own rows of T_{m-1}, T_{m-2} (x2 for the (a, e) pair).
template <int MODE>
struct StagedStreams {
    static constexpr int value = (MODE == kModeEvolveMsd) ? 4 : 2;
};

// A lane owns V consecutive vectors of a row (V = 2 when B >= 2: one 256-bit access per operand).
template <int B>
struct LaneShape {
    static constexpr int V = B >= 2 ? 2 : 1;
    static constexpr int LPR = B / V;        // lanes per row
    static constexpr int RS = 32 / LPR;      // rows per round
    static constexpr int ROUNDS = LPR;       // rounds per slice
};

template <int V>
struct CV {   // V complex numbers
    double re[V], im[V];
};
template <int V>
__device__ __forceinline__ CV<V> cv_zero() {
    CV<V> z;
#pragma unroll
    for (int j = 0; j < V; ++j) z.re[j] = z.im[j] = 0.0;
    return z;
}
// shared memory, V consecutive double2
template <int V>
__device__ __forceinline__ CV<V> cv_lds(const double2* p) {
    CV<V> v;
#pragma unroll
    for (int j = 0; j < V; ++j) {
        const double2 t = p[j];
        v.re[j] = t.x;
        v.im[j] = t.y;
    }
    return v;
}
// shared memory written by a swizzled tensor copy: V consecutive double2 at shared address sa (V = 2)
__device__ __forceinline__ CV<2> cv_lds_swz(uint32_t sa) {
    const uint32_t p0 = swz32(sa);
    CV<2> v;
    asm volatile("ld.shared.v2.f64 {%0, %1}, [%2];" : "=d"(v.re[0]), "=d"(v.im[0]) : "r"(p0));
    asm volatile("ld.shared.v2.f64 {%0, %1}, [%2];" : "=d"(v.re[1]), "=d"(v.im[1]) : "r"(p0 ^ 16u));
    return v;
}
template <int V>
__device__ __forceinline__ CV<V> cv_lds_staged(const double2* p);
template <>
__device__ __forceinline__ CV<1> cv_lds_staged<1>(const double2* p) { return cv_lds<1>(p); }
template <>
__device__ __forceinline__ CV<2> cv_lds_staged<2>(const double2* p) { return cv_lds_swz(smem_u32(p)); }

// global memory, read once (evict-first)
template <int V>
__device__ __forceinline__ CV<V> cv_ld_stream(const double2* p);
template <>
__device__ __forceinline__ CV<1> cv_ld_stream<1>(const double2* p) {
    const double2 t = __ldcs(p);
    CV<1> v;
    v.re[0] = t.x;
    v.im[0] = t.y;
    return v;
}
template <>
__device__ __forceinline__ CV<2> cv_ld_stream<2>(const double2* p) {
    CV<2> v;
    asm volatile("ld.global.cs.v4.f64 {%0, %1, %2, %3}, [%4];"
                 : "=d"(v.re[0]), "=d"(v.im[0]), "=d"(v.re[1]), "=d"(v.im[1])
                 : "l"(p));
    return v;
}
template <int V>
__device__ __forceinline__ void cv_st(double2* p, const CV<V>& v);
template <>
__device__ __forceinline__ void cv_st<1>(double2* p, const CV<1>& v) {
    st_vec(p, make_double2(v.re[0], v.im[0]));
}
template <>
__device__ __forceinline__ void cv_st<2>(double2* p, const CV<2>& v) {
#if GPUQT_ST_POLICY == 1
    asm volatile("st.global.cs.v4.f64 [%0], {%1, %2, %3, %4};" ::"l"(p), "d"(v.re[0]), "d"(v.im[0]), "d"(v.re[1]), "d"(v.im[1])
                 : "memory");
#else
    asm volatile("st.global.v4.f64 [%0], {%1, %2, %3, %4};" ::"l"(p), "d"(v.re[0]), "d"(v.im[0]), "d"(v.re[1]), "d"(v.im[1])
                 : "memory");
#endif
}
// Gather of V consecutive vectors of row c of T_{m-1}: rows of the current slice come from the
// staged copy in shared memory, the others from global memory with an L2 evict_last hint (they are
// re-read by the neighbouring slices).  Both loads are predicated, so there is no branch.
//   g_l  = byte address of (row 0, the lane's first vector) in global memory
//   s_l  = shared-window address of the same element of the slice's staged rows, minus row0 * RB
//   RB   = bytes of one row (16 B)
template <int V>
__device__ __forceinline__ CV<V> cv_gather(const char* g_l, uint32_t s_l, int c, int row0, int RB);
template <>
__device__ __forceinline__ CV<1> cv_gather<1>(const char* g_l, uint32_t s_l, int c, int row0, int RB) {
    const unsigned d = (unsigned)(c - row0);
    const uint32_t sa = s_l + (uint32_t)(c * RB);
    const char* ga = g_l + (long long)c * RB;
    CV<1> v;
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "setp.lt.u32 p, %4, 32;\n"
        "@p ld.shared.v2.f64 {%0, %1}, [%2];\n"
        "@!p ld.global.v2.f64 {%0, %1}, [%3];\n"
        "}"
        : "=d"(v.re[0]), "=d"(v.im[0])
        : "r"(sa), "l"(ga), "r"(d));
    return v;
}
template <>
__device__ __forceinline__ CV<2> cv_gather<2>(const char* g_l, uint32_t s_l, int c, int row0, int RB) {
    const unsigned d = (unsigned)(c - row0);
    const uint32_t sa = swz32(s_l + (uint32_t)(c * RB));
    const uint32_t sb = sa ^ 16u;
    const char* ga = g_l + (long long)c * RB;
    CV<2> v;
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "setp.lt.u32 p, %6, 32;\n"
        "@p ld.shared.v2.f64 {%0, %1}, [%4];\n"
        "@p ld.shared.v2.f64 {%2, %3}, [%7];\n"
#if GPUQT_GATHER_POLICY == 1
        "@!p ld.global.L2::evict_last.v4.f64 {%0, %1, %2, %3}, [%5];\n"
#else
        "@!p ld.global.v4.f64 {%0, %1, %2, %3}, [%5];\n"
#endif
        "}"
        : "=d"(v.re[0]), "=d"(v.im[0]), "=d"(v.re[1]), "=d"(v.im[1])
        : "r"(sa), "l"(ga), "r"(d), "r"(sb));
    return v;
}

// acc += h * v for V vectors; h = (hr, hi)
template <int V, bool CPLX>
__device__ __forceinline__ void cv_fma(CV<V>& acc, double hr, double hi, const CV<V>& v) {
#pragma unroll
    for (int j = 0; j < V; ++j) {
        acc.re[j] = fma(hr, v.re[j], acc.re[j]);
        acc.im[j] = fma(hr, v.im[j], acc.im[j]);
        if (CPLX) {
            acc.re[j] = fma(-hi, v.im[j], acc.re[j]);
            acc.im[j] = fma(hi, v.re[j], acc.im[j]);
        }
    }
}

template <int V>
__device__ __forceinline__ void cv_add(CV<V>& acc, const CV<V>& v) {
#pragma unroll
    for (int j = 0; j < V; ++j) {
        acc.re[j] += v.re[j];
        acc.im[j] += v.im[j];
    }
}

// One round (RS rows) of one slice whose record and own rows sit in shared memory at `stage`.
// Rows past the end of the table (last slice only) are computed like the others on zero inputs
// (their staged self / prev are replaced by 0 and their entries are padding), so the dot products
// need no guard; only their stores are predicated off.
template <int B, int KT, int HOP, int MODE>
__device__ __forceinline__ void walk_round(const Mat& m, const StepArgs& a, const StepIO& io, const unsigned char* stage, int w,
                                           int row0, int rows_valid, int j, int lane, double scale,
                                           double (&red)[ModeTraits<MODE>::Q * LaneShape<B>::V],
                                           unsigned int* signal) {
    constexpr int V = LaneShape<B>::V, LPR = LaneShape<B>::LPR, RS = LaneShape<B>::RS;
    constexpr int KU = KT > 0 ? KT : 1;
    constexpr int RB = B * 16;   // bytes of one row of a vector set
    constexpr bool MSD = (MODE == kModeEvolveMsd);
    constexpr bool CPLX = (HOP == kHopComplex), CONST = hop_is_const(HOP), IDX16 = (HOP == kHopConst16);
    const int rl = lane / LPR, l = lane % LPR;
    const double* s_hre = reinterpret_cast<const double*>(stage);
    const double* s_him = s_hre + w * 32;
    const double* s_on = s_hre + w * 32 * hop_doubles(HOP);
    const int* s_col = reinterpret_cast<const int*>(s_on + 32);                        // int32 columns, or base[8]
    const unsigned short* s_d16 = reinterpret_cast<const unsigned short*>(s_col + 8);   // kHopConst16: deltas
    // staged vector rows: [in | (in_e) | prev | (prev_e)], each 32 * B double2
    const double2* s_in = reinterpret_cast<const double2*>(stage + a.rec_bytes);
    const double2* s_in_e = s_in + 32 * B;
    const double2* s_prev = s_in + (MSD ? 2 : 1) * 32 * B;
    const double2* s_prev_e = s_prev + 32 * B;
    // lane-relative bases of the gathers (see cv_gather)
    const uint32_t sl_in = smem_u32(s_in + l * V) - (uint32_t)(row0 * RB);
    const uint32_t sl_in_e = smem_u32(s_in_e + l * V) - (uint32_t)(row0 * RB);
    const char* gl_in = reinterpret_cast<const char*>(io.in + l * V);
    const char* gl_in_e = reinterpret_cast<const char*>(io.in_e + l * V);

    const int r = j * RS + rl;
    const bool ok = r < rows_valid;
    const int si_ = r * B + l * V;                                     // element inside the staged rows
    const size_t vi = (size_t)(row0 + (ok ? r : 0)) * B + l * V;       // element in global memory

    // streamed own-row operands (evolved vector / phi_L): issued first, consumed last
    CV<V> other = cv_zero<V>(), other_e = cv_zero<V>();
    if (MODE == kModeEvolve || MSD) other = cv_ld_stream<V>(&a.src[vi]);
    if (MSD) other_e = cv_ld_stream<V>(&a.src_e[vi]);
    if (MODE == kModeLeft) other = cv_ld_stream<V>(&a.phiL[vi]);
    double xm = 0.0;
    if (MSD) xm = m.x[row0 + (ok ? r : 0)];
    constexpr bool PD = PrevDirect<B>::value;
    CV<V> prev = cv_zero<V>(), prev_e = cv_zero<V>();
    if (PD && !a.first && ok) {         // rows past the end keep prev = 0 (their T_m must stay 0 for the dots)
        prev = cv_ld_stream<V>(&io.prev[vi]);
        if (MSD) prev_e = cv_ld_stream<V>(&io.prev_e[vi]);
    }

    const CV<V> self = ok ? cv_lds_staged<V>(s_in + si_) : cv_zero<V>();
    const CV<V> self_e = (MSD && ok) ? cv_lds_staged<V>(s_in_e + si_) : cv_zero<V>();
    const double on = s_on[r];

    CV<V> sum = cv_zero<V>(), sum_e = cv_zero<V>(), sum_x = cv_zero<V>();   // H T, H e, [X,H] T (unscaled)
    if (KT > 0) {
        // all gathers of the row first (independent loads in flight), then the arithmetic
        CV<V> v[KU], ve[MSD ? KU : 1];
        double xn[MSD ? KU : 1];
#pragma unroll
        for (int k = 0; k < KU; ++k) {
            const int c = IDX16 ? s_col[k] + (int)s_d16[k * 32 + r] : s_col[k * 32 + r];
            v[k] = cv_gather<V>(gl_in, sl_in, c, row0, RB);
            if (MSD) {
                ve[k] = cv_gather<V>(gl_in_e, sl_in_e, c, row0, RB);
                xn[k] = m.x[c];
            }
        }
        if (signal && lane == 0) red_release_gpu_inc(signal);           // see cheb_step_kernel, `pending`
#pragma unroll
        for (int k = 0; k < KU; ++k) {
            double hr = 1.0, hi = 0.0;                                  // CONST: the factor is applied once below
            if (!CONST) hr = s_hre[k * 32 + r];
            if (CPLX) hi = s_him[k * 32 + r];
            if (CONST) cv_add<V>(sum, v[k]);
            else cv_fma<V, CPLX>(sum, hr, hi, v[k]);
            if (MSD) {
                if (CONST) cv_add<V>(sum_e, ve[k]);
                else cv_fma<V, CPLX>(sum_e, hr, hi, ve[k]);
                // [X,H]_mn = (X_m - X_n) H_mn = -dx H_mn
                const double ndx = -min_image(xn[k] - xm, m.box);
                cv_fma<V, CPLX>(sum_x, ndx * hr, ndx * hi, v[k]);
            }
        }
    } else {
        if (signal && lane == 0) red_release_gpu_inc(signal);
        for (int k = 0; k < w; ++k) {
            const int c = IDX16 ? s_col[k] + (int)s_d16[k * 32 + r] : s_col[k * 32 + r];
            double hr = 1.0, hi = 0.0;
            if (!CONST) hr = s_hre[k * 32 + r];
            if (CPLX) hi = s_him[k * 32 + r];
            const CV<V> vv = cv_gather<V>(gl_in, sl_in, c, row0, RB);
            if (CONST) cv_add<V>(sum, vv);
            else cv_fma<V, CPLX>(sum, hr, hi, vv);
            if (MSD) {
                const CV<V> vve = cv_gather<V>(gl_in_e, sl_in_e, c, row0, RB);
                if (CONST) cv_add<V>(sum_e, vve);
                else cv_fma<V, CPLX>(sum_e, hr, hi, vve);
                const double ndx = -min_image(m.x[c] - xm, m.box);
                cv_fma<V, CPLX>(sum_x, ndx * hr, ndx * hi, vv);
            }
        }
    }
    if (!PD && !a.first && ok) {
        prev = cv_lds_staged<V>(s_prev + si_);
        if (MSD) prev_e = cv_lds_staged<V>(s_prev_e + si_);
    }
    const double hs = CONST ? scale * m.hop_const : scale;              // scale of the neighbour sums
    const double os = scale * on;                                       // scale of the on-site term
    CV<V> t, te;   // T_m (b_k) and e_m
#pragma unroll
    for (int q = 0; q < V; ++q) {
        t.re[q] = fma(hs, sum.re[q], fma(os, self.re[q], -prev.re[q]));
        t.im[q] = fma(hs, sum.im[q], fma(os, self.im[q], -prev.im[q]));
        if (MODE == kModeDoubling) {
            red[0 * V + q] += t.re[q] * t.re[q] + t.im[q] * t.im[q];
            red[1 * V + q] += t.re[q] * self.re[q] + t.im[q] * self.im[q];
            // <T_{m-1}|T_{m-1}> is only used from the first launch (C_0); later ones had it as <T_m|T_m>
            if (a.first) red[2 * V + q] += self.re[q] * self.re[q] + self.im[q] * self.im[q];
        } else if (MODE == kModeLeft) {   // conj(l) * t
            red[0 * V + q] += other.re[q] * t.re[q] + other.im[q] * t.im[q];
            red[1 * V + q] += other.re[q] * t.im[q] - other.im[q] * t.re[q];
        } else {
            // Clenshaw: b_k = c_k src + 2 H~ b_{k+1} - b_{k+2}; no accumulator is read or written
            t.re[q] += io.cr * other.re[q] - io.ci * other.im[q];
            t.im[q] += io.cr * other.im[q] + io.ci * other.re[q];
            if (MSD) {
                te.re[q] = fma(hs, sum_e.re[q] + sum_x.re[q], fma(os, self_e.re[q], -prev_e.re[q]));
                te.im[q] = fma(hs, sum_e.im[q] + sum_x.im[q], fma(os, self_e.im[q], -prev_e.im[q]));
                te.re[q] += io.cr * other_e.re[q] - io.ci * other_e.im[q];
                te.im[q] += io.cr * other_e.im[q] + io.ci * other_e.re[q];
            }
        }
    }
    if (ok && io.store) {
        cv_st<V>(&io.out[vi], t);
        if (MSD) cv_st<V>(&io.out_e[vi], te);
    }
}

// Dots of one warp: shuffle over lanes that hold the same vectors, then lanes < LPR add into the
// warp's shared-memory row dst[q * B + b]; the register accumulators restart from zero.
template <int B, int Q, int V>
__device__ __forceinline__ void warp_flush(double (&v)[Q * V], double* dst, int lane) {
    constexpr int LPR = B / V;
#pragma unroll
    for (int q = 0; q < Q * V; ++q) {
#pragma unroll
        for (int off = 16; off >= LPR; off >>= 1) v[q] += __shfl_xor_sync(0xffffffffu, v[q], off);
    }
    if (lane < LPR) {
#pragma unroll
        for (int q = 0; q < Q; ++q)
#pragma unroll
            for (int j = 0; j < V; ++j) dst[q * B + lane * V + j] += v[q * V + j];
    }
#pragma unroll
    for (int q = 0; q < Q * V; ++q) v[q] = 0.0;
    __syncwarp();
}

// Deterministic CTA / grid stage of the reduction: s_part[warp][P] -> per-block partial -> the last
// block to finish sums the per-block partials in a fixed order (no floating-point atomics).
// Value p < P0 goes to r0[p], the others to r1[p - P0] (second step of a fused pair).
__device__ __forceinline__ void block_finish(const double* s_part, int P, int P0, double* partials,
                                             unsigned int* ticket, double* r0, double* r1) {
    __shared__ double s_tree[kThreads + 32];   // the step kernel calls this with its producer warp as well
    __shared__ int s_last;
    const int tid = threadIdx.x;
    __syncthreads();
    if (tid < P) {
        double s = 0.0;
#pragma unroll
        for (int w = 0; w < kWarps; ++w) s += s_part[w * P + tid];
        partials[(size_t)blockIdx.x * P + tid] = s;
    }
    __threadfence();
    __syncthreads();
    if (tid == 0) {
        unsigned int t = atomicAdd(ticket, 1u);
        s_last = (t == gridDim.x - 1);
    }
    __syncthreads();
    if (!s_last) return;
    __threadfence();
    // fixed-shape sum over blocks: thread t handles value (t % P), blocks strand, strand + S, ...
    const int S = kThreads / P;              // strands per value
    const int pv = tid % P, strand = tid / P;
    double s = 0.0;
    if (strand < S)
        for (unsigned int g = strand; g < gridDim.x; g += S) s += __ldcg(&partials[(size_t)g * P + pv]);
    s_tree[tid] = (strand < S) ? s : 0.0;
    __syncthreads();
    if (tid < P) {
        double tot = 0.0;
        for (int j = 0; j < S; ++j) tot += s_tree[j * P + tid];
        if (tid < P0) r0[tid] = tot;
        else r1[tid - P0] = tot;
    }
    if (tid == 0) *ticket = 0u;
}

__device__ __forceinline__ unsigned int ld_acquire_gpu(const unsigned int* p) {
    unsigned int v;
    asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
    return v;
}


// One Chebyshev recurrence step fused with what consumes it (single-step launches; the default).
// Every warp issues its own TMA copies (lane 0) one or more slices ahead.  Persistent CTAs: the slices are cut
// into runs of a.run consecutive slices; CTA c walks runs c, c + G, c + 2G, ...; inside a run warp w
// takes slices w, w + kWarps, ...  A CTA therefore streams a contiguous band of rows and the grid
// sweeps the vector as a tight front, so gathers to nearby rows (the +-x, +-y, +-z neighbours of a
// lattice) are served by L1/L2.  All loop indices are kept incrementally (no divisions in the loop).
template <int B, int KT, int HOP, int MODE>
__global__ void __launch_bounds__(kThreads, ModeTraits<MODE>::kMinBlocks) cheb_step_kernel(const Mat m, const StepArgs a) {
    constexpr int Q = ModeTraits<MODE>::Q;
    constexpr int V = LaneShape<B>::V, ROUNDS = LaneShape<B>::ROUNDS;
    constexpr int RB = B * 16, QB = Q * B;
    constexpr bool DOTS = (MODE == kModeDoubling || MODE == kModeLeft);
    __shared__ double s_part[DOTS ? kWarps * QB : 1];
    const StepIO& io = a.io[0];
    constexpr int kPair = (MODE == kModeEvolveMsd) ? 2 : 1;
    extern __shared__ __align__(1024) unsigned char smem[];
    const int tid = threadIdx.x, lane = tid & 31;
    const int warp = __shfl_sync(0xffffffffu, tid >> 5, 0);   // warp-uniform for the compiler
    const int stages = a.stages;
    const int stage_bytes = a.stage_bytes;
    uint64_t* bars = reinterpret_cast<uint64_t*>(smem) + warp * kMaxStages;
    unsigned char* wstage = smem + 128 * ((kWarps * kMaxStages * 8 + 127) / 128) + (size_t)warp * stages * stage_bytes;

    double red[Q * V];
#pragma unroll
    for (int q = 0; q < Q * V; ++q) red[q] = 0.0;
    if (DOTS) {
        for (int i = lane; i < QB; i += 32) s_part[warp * QB + i] = 0.0;
    }
    const double scale = a.half ? m.inv_dE : 2.0 * m.inv_dE;

    const int N = (int)m.N, n_slices = (int)m.n_slices;
    const int per = a.run / kWarps;
    const int n_runs = (n_slices + a.run - 1) / a.run;
    const int G = gridDim.x;
    const int my_runs = (int)blockIdx.x < n_runs ? (n_runs - (int)blockIdx.x + G - 1) / G : 0;
    int n_my = 0;
    if (my_runs > 0) {
        const int last = blockIdx.x + (my_runs - 1) * G;
        const int rem = n_slices - last * a.run;          // slices in my last run (may be partial)
        const int in_last = rem >= a.run ? per : (warp < rem ? (rem - warp + kWarps - 1) / kWarps : 0);
        n_my = (my_runs - 1) * per + in_last;
    }
    uint64_t policy = 0;
    if (lane == 0) {
        for (int s = 0; s < stages; ++s) mbar_init(&bars[s], 1);
        fence_mbar_init();
        policy = policy_evict_first();
    }
    __syncwarp();

    // position of a pipeline cursor: slice (forward order), index inside the run, stage, phase
    struct Cursor {
        int s, k, st;
        uint32_t ph;
    };
    const int jump = G * a.run - (per - 1) * kWarps;     // last slice of a run -> first slice of my next run
    auto advance = [&](Cursor& c) {
        if (++c.k == per) {
            c.k = 0;
            c.s += jump;
        } else {
            c.s += kWarps;
        }
        if (++c.st == stages) {
            c.st = 0;
            c.ph ^= 1u;
        }
    };
    auto issue = [&](const Cursor& c) {   // lane 0 only: every HBM stream of the slice -> one stage, one mbarrier
        const int s = a.reverse ? n_slices - 1 - c.s : c.s;
        long long off;
        uint32_t bytes;
        if (KT > 0) {
            bytes = (uint32_t)hop_record_bytes(KT, HOP);
            off = (long long)s * bytes;
        } else {
            off = m.slice_off[s];
            bytes = (uint32_t)(m.slice_off[s + 1] - off);
        }
        const int left = N - s * 32;
        const uint32_t vbytes = (uint32_t)((left < 32 ? left : 32) * RB);
        // T_{m-1} rows include the all-zero row N when it falls into this slice's window (the
        // constant-hopping padding entries point at it)
        const uint32_t vbytes_in = (uint32_t)((left + 1 < 32 ? left + 1 : 32) * RB);
        const bool with_prev = !a.first && !PrevDirect<B>::value;
        unsigned char* dst = wstage + c.st * stage_bytes;
        unsigned char* vdst = dst + a.rec_bytes;
        if (B >= 2) {
            // tensor copies: always the full 32-row box (rows past the end of the buffer are zero-filled)
            const uint32_t total = bytes + (uint32_t)(32 * RB) * kPair * (with_prev ? 2u : 1u);
            const int unit = s * 4 * B;           // first 128-byte line of the slice
            mbar_expect_tx(&bars[c.st], total);
            bulk_g2s(dst, m.rec + off, bytes, &bars[c.st], policy);
            tensor_g2s(vdst, io.tm_in, unit, &bars[c.st]);
            if (MODE == kModeEvolveMsd) tensor_g2s(vdst + 512 * B, io.tm_in_e, unit, &bars[c.st]);
            if (with_prev) {
                tensor_g2s_hint(vdst + kPair * 512 * B, io.tm_prev, unit, &bars[c.st], policy);
                if (MODE == kModeEvolveMsd) tensor_g2s_hint(vdst + 3 * 512 * B, io.tm_prev_e, unit, &bars[c.st], policy);
            }
        } else {
            const uint32_t total = bytes + vbytes_in * kPair + (with_prev ? vbytes * kPair : 0u);
            const size_t voff = (size_t)s * 32 * B;
            mbar_expect_tx(&bars[c.st], total);
            bulk_g2s(dst, m.rec + off, bytes, &bars[c.st], policy);
            bulk_g2s_nohint(vdst, io.in + voff, vbytes_in, &bars[c.st]);
            if (MODE == kModeEvolveMsd) bulk_g2s_nohint(vdst + 512 * B, io.in_e + voff, vbytes_in, &bars[c.st]);
            if (with_prev) {
                bulk_g2s(vdst + kPair * 512 * B, io.prev + voff, vbytes, &bars[c.st], policy);
                if (MODE == kModeEvolveMsd) bulk_g2s(vdst + 3 * 512 * B, io.prev_e + voff, vbytes, &bars[c.st], policy);
            }
        }
    };

    Cursor prod{(int)blockIdx.x * a.run + warp, 0, 0, 0u}, cons = prod;
    int issued = 0;
    if (lane == 0) {
        for (; issued < stages - 1 && issued < n_my; ++issued) {
            issue(prod);
            advance(prod);
        }
    }
    for (int i = 0; i < n_my; ++i) {
        // the stage the producer cursor points at was consumed by the whole warp in the previous iteration
        if (lane == 0 && issued < n_my) {
            issue(prod);
            advance(prod);
            ++issued;
        }
        mbar_wait(&bars[cons.st], cons.ph);
        const unsigned char* stage = wstage + cons.st * stage_bytes;
        const int slice = a.reverse ? n_slices - 1 - cons.s : cons.s;
        int w = KT;
        if (KT == 0) w = record_width(m.slice_off[slice + 1] - m.slice_off[slice], hop_doubles(HOP));
        const int row0 = slice * 32;
        const int rows_valid = N - row0;          // >= 32 except in the last slice
#pragma unroll 1
        for (int j = 0; j < ROUNDS; ++j) walk_round<B, KT, HOP, MODE>(m, a, io, stage, w, row0, rows_valid, j, lane, scale, red, nullptr);
        advance(cons);
        __syncwarp();
    }
    if (DOTS) {
        warp_flush<B, Q, V>(red, s_part + warp * QB, lane);
        block_finish(s_part, QB, QB, a.partials, a.ticket, io.result, io.result);
    }
}


// TWO consecutive recurrence steps in one launch (a.n_steps == 2; opt-in, GPUQT_FUSE=1): the second
// step trails the first by a fixed slack of the work list so that it finds T_m, T_{m-1} and the matrix records in L2: per pair of steps DRAM then sees T_{m-1},
// T_{m-2} read and T_m, T_{m+1} written once each and the matrix once, instead of 6 vector passes
// and 2 matrix passes.
//
// Persistent, warp-specialised CTAs of kWarps consumer warps + 1 producer warp.  The slices are cut
// into runs of a.run consecutive slices; the work list is a sequence of items = (step, run); CTA c
// takes items c, c + G, c + 2G, ...; inside a run consumer warp w takes slices w, w + kWarps, ...
// Single-step launches use the arithmetic list item t = run t; fused launches read the list from
// a.sched (built on the host from the table's sparsity, host_util.h).
//   producer warp   walks the CTA's items; lane w < kWarps feeds consumer warp w: it waits for a
//                   free stage of that warp (mbarrier empty[w][st]), writes a 16-byte header
//                   {slice, step, flags, run} and issues the TMA bulk copies of the slice onto
//                   full[w][st].  Before a second-step item it checks, all 32 lanes at once with
//                   acquire loads, that the first-step runs the item gathers from are complete
//                   (run_done[r] == kWarps) and sleeps otherwise.  The consumers never touch the
//                   work list.
//   consumer warp   waits full[w][st], walks the slice, arrives on empty[w][st].  After the last
//                   slice of a first-step item it owes a release on run_done[run]; it pays one slice
//                   later, right after that slice's gathers have been issued (the fence then overlaps
//                   the gather latency), or at once when no slice is ready.
// An item depends only on earlier items of the list and every warp publishes what it owes before
// it blocks, so the scheme cannot deadlock as long as all CTAs are co-resident (the grid is sized
// by occupancy).
constexpr int kHdrBytes = 256;                    // per stage: the slice header (keeps the stages 256-byte aligned)
constexpr int kFlagEnd = 1, kFlagOwesRelease = 2;

template <int B, int KT, int HOP, int MODE>
__global__ void __launch_bounds__(kThreads + 32, ModeTraits<MODE>::kMinBlocks) cheb_pair_kernel(const Mat m, const StepArgs a) {
    constexpr int Q = ModeTraits<MODE>::Q;
    constexpr int V = LaneShape<B>::V, ROUNDS = LaneShape<B>::ROUNDS;
    constexpr int RB = B * 16, QB = Q * B;
    constexpr int kPair = (MODE == kModeEvolveMsd) ? 2 : 1;
    constexpr bool DOTS = (MODE == kModeDoubling || MODE == kModeLeft);
    extern __shared__ __align__(1024) unsigned char smem[];
    __shared__ double s_part[DOTS ? kWarps * 2 * QB : 1];
    const int tid = threadIdx.x, lane = tid & 31;
    const int warp = __shfl_sync(0xffffffffu, tid >> 5, 0);   // warp-uniform for the compiler
    const int stages = a.stages;
    const int stage_bytes = a.stage_bytes;                     // record | vector rows | header
    const int hdr_off = stage_bytes - kHdrBytes;
    uint64_t* full = reinterpret_cast<uint64_t*>(smem);        // [kWarps][kMaxStages]
    uint64_t* empty = full + kWarps * kMaxStages;              // [kWarps][kMaxStages]
    unsigned char* stage_base = smem + 128 * ((2 * kWarps * kMaxStages * 8 + 127) / 128);
    const int P = a.n_steps * QB;                 // dot values per block

    const int N = (int)m.N, n_slices = (int)m.n_slices;
    const int n_runs = (n_slices + a.run - 1) / a.run;
    const int G = gridDim.x;
    const bool fused = a.sched != nullptr;
    const int n_total = fused ? a.n_items : n_runs;

    if (warp < kWarps && lane == 0) {
        for (int s = 0; s < stages; ++s) {
            mbar_init(&full[warp * kMaxStages + s], 1);
            mbar_init(&empty[warp * kMaxStages + s], 1);
        }
        fence_mbar_init();
    }
    if (DOTS && warp < kWarps) {
        for (int i = lane; i < P; i += 32) s_part[warp * P + i] = 0.0;
    }
    __syncthreads();

    if (warp == kWarps) {
        // ------------------------------------------------------------------ producer warp
        const int cw = lane < kWarps ? lane : kWarps - 1;       // consumer warp this lane feeds
        const bool feeds = lane < kWarps;
        unsigned char* my_stages = stage_base + (size_t)cw * stages * stage_bytes;
        uint64_t* my_full = full + cw * kMaxStages;
        uint64_t* my_empty = empty + cw * kMaxStages;
        int st = 0;
        uint32_t ph = 0;
        const uint64_t policy = policy_evict_first();
        auto deps_done = [&](int run) {   // whole warp: have all first-step runs this run gathers from finished?
            const int b = a.dep_ptr[run], e = a.dep_ptr[run + 1];
            bool ok = true;
#pragma unroll 1
            for (int i0 = b; i0 < e; i0 += 32) {      // every lane acquires (lanes past the end re-read the last entry)
                const int i = i0 + lane < e ? i0 + lane : e - 1;
                ok = ok && (ld_acquire_gpu(a.run_done + a.dep_list[i]) >= (unsigned int)kWarps);
            }
            return __all_sync(0xffffffffu, ok) != 0;
        };
        for (int t = blockIdx.x; t < n_total; t += G) {
            int run = t, step = 0;
            if (fused) {
                const int2 e = a.sched[t];
                run = e.x & kNoRun;
                step = (e.x >> 30) & 1;
            }
            if (run == kNoRun) continue;
            if (fused && step == 1) {
                // rows stored through the generic proxy by other SMs, fenced and released at gpu scope
                // (they are in L2) and acquired here; the TMA reads below are issued behind the acquire
                // by control dependency and go to L2
                while (!deps_done(run)) __nanosleep(200);
            }
            const StepIO& io = a.io[step];
            int len = n_slices - run * a.run;
            len = len < a.run ? len : a.run;
            for (int k0 = 0; k0 < len; k0 += kWarps) {
                if (feeds && k0 + lane < len) {
                    const int vs = run * a.run + k0 + lane;                 // slice in sweep order
                    const int s = a.reverse ? n_slices - 1 - vs : vs;
                    mbar_wait(&my_empty[st], ph ^ 1u);                      // stage free (passes at once the first time round)
                    unsigned char* dst = my_stages + st * stage_bytes;
                    int flags = 0;
                    if (fused && step == 0 && k0 + lane + kWarps >= len) flags |= kFlagOwesRelease;
                    *reinterpret_cast<int4*>(dst + hdr_off) = make_int4(s, step, flags, run);
                    long long off;
                    uint32_t bytes;
                    if (KT > 0) {
                        bytes = (uint32_t)hop_record_bytes(KT, HOP);
                        off = (long long)s * bytes;
                    } else {
                        off = m.slice_off[s];
                        bytes = (uint32_t)(m.slice_off[s + 1] - off);
                    }
                    const int left = N - s * 32;
                    const uint32_t vbytes = (uint32_t)((left < 32 ? left : 32) * RB);
                    // T_{m-1} rows include the all-zero row N when it falls into this slice's window (the
                    // constant-hopping padding entries point at it)
                    const uint32_t vbytes_in = (uint32_t)((left + 1 < 32 ? left + 1 : 32) * RB);
                    const bool with_prev = !a.first && !PrevDirect<B>::value;
                    const uint32_t total = B >= 2 ? bytes + (uint32_t)(32 * RB) * kPair * (with_prev ? 2u : 1u)
                                                  : bytes + vbytes_in * kPair + (with_prev ? vbytes * kPair : 0u);
                    unsigned char* vdst = dst + a.rec_bytes;
                    const size_t voff = (size_t)s * 32 * B;
                    const int unit = s * 4 * B;           // first 128-byte line of the slice (tensor copies, B >= 2)
                    mbar_expect_tx(&my_full[st], total);
                    // the first step of a fused pair leaves the record in L2 for the second one
                    if (fused && step == 0) bulk_g2s_nohint(dst, m.rec + off, bytes, &my_full[st]);
                    else bulk_g2s(dst, m.rec + off, bytes, &my_full[st], policy);
                    if (B >= 2) {
                        tensor_g2s(vdst, io.tm_in, unit, &my_full[st]);
                        if (MODE == kModeEvolveMsd) tensor_g2s(vdst + 512 * B, io.tm_in_e, unit, &my_full[st]);
                        if (with_prev) {
                            tensor_g2s_hint(vdst + kPair * 512 * B, io.tm_prev, unit, &my_full[st], policy);
                            if (MODE == kModeEvolveMsd) tensor_g2s_hint(vdst + 3 * 512 * B, io.tm_prev_e, unit, &my_full[st], policy);
                        }
                    } else {
                        bulk_g2s_nohint(vdst, io.in + voff, vbytes_in, &my_full[st]);
                        if (MODE == kModeEvolveMsd) bulk_g2s_nohint(vdst + 512 * B, io.in_e + voff, vbytes_in, &my_full[st]);
                        if (with_prev) {
                            bulk_g2s(vdst + kPair * 512 * B, io.prev + voff, vbytes, &my_full[st], policy);
                            if (MODE == kModeEvolveMsd) bulk_g2s(vdst + 3 * 512 * B, io.prev_e + voff, vbytes, &my_full[st], policy);
                        }
                    }
                    if (++st == stages) {
                        st = 0;
                        ph ^= 1u;
                    }
                }
            }
            // consumer warps without a slice in this (short, last) run owe nothing: the producer counts for them
            if (fused && step == 0 && feeds && lane >= len) red_release_gpu_inc(a.run_done + run);
        }
        if (feeds) {   // end marker
            mbar_wait(&my_empty[st], ph ^ 1u);
            *reinterpret_cast<int4*>(my_stages + st * stage_bytes + hdr_off) = make_int4(0, 0, kFlagEnd, 0);
            mbar_arrive(&my_full[st]);
        }
    } else {
        // ------------------------------------------------------------------ consumer warps
        unsigned char* my_stages = stage_base + (size_t)warp * stages * stage_bytes;
        uint64_t* my_full = full + warp * kMaxStages;
        uint64_t* my_empty = empty + warp * kMaxStages;
        double* my_part = s_part + warp * P;
        double red[Q * V];
#pragma unroll
        for (int q = 0; q < Q * V; ++q) red[q] = 0.0;
        const double scale = a.half ? m.inv_dE : 2.0 * m.inv_dE;
        int st = 0;
        uint32_t ph = 0;
        int red_step = 0;                   // step whose dots the register accumulators hold
        unsigned int* pending = nullptr;    // release owed for a finished first-step item
        while (true) {
            if (pending && !mbar_test(&my_full[st], ph)) {     // nothing ready: pay now, then wait
                if (lane == 0) red_release_gpu_inc(pending);
                pending = nullptr;
            }
            mbar_wait(&my_full[st], ph);
            const unsigned char* stage = my_stages + st * stage_bytes;
            const int4 hdr = *reinterpret_cast<const int4*>(stage + hdr_off);
            if (hdr.z & kFlagEnd) break;
            const int slice = hdr.x, step = hdr.y;
            if (DOTS && step != red_step) {
                warp_flush<B, Q, V>(red, my_part + red_step * QB, lane);
                red_step = step;
            }
            int w = KT;
            if (KT == 0) w = record_width(m.slice_off[slice + 1] - m.slice_off[slice], hop_doubles(HOP));
            const int row0 = slice * 32;
            const int rows_valid = N - row0;          // >= 32 except in the last slice
            const StepIO& io = a.io[step];
#pragma unroll 1
            for (int j = 0; j < ROUNDS; ++j) {
                walk_round<B, KT, HOP, MODE>(m, a, io, stage, w, row0, rows_valid, j, lane, scale, red, pending);
                pending = nullptr;
            }
            __syncwarp();
            if (lane == 0) mbar_arrive(&my_empty[st]);
            if (hdr.z & kFlagOwesRelease) pending = a.run_done + hdr.w;
            if (++st == stages) {
                st = 0;
                ph ^= 1u;
            }
        }
        if (pending && lane == 0) red_release_gpu_inc(pending);
        if (DOTS) warp_flush<B, Q, V>(red, my_part + red_step * QB, lane);
    }
    if (DOTS) block_finish(s_part, P, QB, a.partials, a.ticket, a.io[0].result, a.io[1].result);
}

// Address of entry (row, k) pieces inside the packed records (plain global reads; used by the
// rarely-run kernels below).
struct RecView {
    const double* hre;
    const double* him;
    const double* on;
    const int* col;                  // int32 columns, or base[8] of the 16-bit variant
    const unsigned short* d16;       // 16-bit variant: deltas, else nullptr
    int w;
    __device__ __forceinline__ int col_at(int k, int r) const {
        return d16 ? col[k] + (int)d16[k * 32 + r] : col[k * 32 + r];
    }
};
__device__ __forceinline__ RecView record_view(const Mat& m, long long slice) {
    long long off, bytes;
    const int nd = hop_doubles(m.hop);
    if (m.uniform) {
        bytes = hop_record_bytes(m.K, m.hop);
        off = slice * bytes;
    } else {
        off = m.slice_off[slice];
        bytes = m.slice_off[slice + 1] - off;
    }
    RecView v;
    v.w = m.hop == kHopConst16 ? m.K : record_width(bytes, nd);     // the 16-bit variant is always uniform
    v.hre = reinterpret_cast<const double*>(m.rec + off);
    v.him = v.hre + (size_t)v.w * 32;
    v.on = v.hre + (size_t)v.w * 32 * nd;
    v.col = reinterpret_cast<const int*>(v.on + 32);
    v.d16 = m.hop == kHopConst16 ? reinterpret_cast<const unsigned short*>(v.col + 8) : nullptr;
    return v;
}

// out = V in,  V_mn = i (X_n - X_m) H_mn  (Eq. 34) — not scaled by 1/dE, no on-site.
// Runs once per VAC measurement (1 of N_m walks), so it reads the records straight from global.
template <int B>
__global__ void __launch_bounds__(kThreads) velocity_kernel(const Mat m, const double2* __restrict__ in,
                                                            double2* __restrict__ out) {
    constexpr int kRows = kThreads / B;
    const int tid = threadIdx.x, b = tid % B, rl = tid / B;
    const long long n_chunks = (m.N + kRows - 1) / kRows;
    for (long long chunk = blockIdx.x; chunk < n_chunks; chunk += gridDim.x) {
        const long long row = chunk * kRows + rl;
        if (row >= m.N) continue;
        const RecView rv = record_view(m, row >> 5);
        const int r = (int)(row & 31);
        const double xm = m.x[row];
        double sr = 0.0, si = 0.0;
        for (int k = 0; k < rv.w; ++k) {
            const int c = rv.col_at(k, r);                  // constant-hopping padding: the zero row N
            const double hr = hop_is_const(m.hop) ? m.hop_const : rv.hre[k * 32 + r];
            const double dx = min_image(m.x[c] - xm, m.box);
            const double wr = dx * hr;
            const double2 v = in[(size_t)c * B + b];
            sr = fma(wr, v.x, sr);
            si = fma(wr, v.y, si);
            if (m.cplx) {
                const double wi = dx * rv.him[k * 32 + r];
                sr = fma(-wi, v.y, sr);
                si = fma(wi, v.x, si);
            }
        }
        out[(size_t)row * B + b] = make_double2(-si, sr);   // multiply by i
    }
}

// <l|r> per vector: result[0][b] = Re, result[1][b] = Im
template <int B>
__global__ void __launch_bounds__(kThreads) dot_kernel(long long N, const double2* __restrict__ l,
                                                       const double2* __restrict__ r, double* partials,
                                                       unsigned int* ticket, double* result) {
    constexpr int kRows = kThreads / B;
    const int tid = threadIdx.x, b = tid % B, rl = tid / B;
    double red[2] = {0.0, 0.0};
    const long long n_chunks = (N + kRows - 1) / kRows;
    for (long long chunk = blockIdx.x; chunk < n_chunks; chunk += gridDim.x) {
        const long long row = chunk * kRows + rl;
        if (row >= N) continue;
        const double2 lv = l[(size_t)row * B + b], rv = r[(size_t)row * B + b];
        red[0] += lv.x * rv.x + lv.y * rv.y;
        red[1] += lv.x * rv.y - lv.y * rv.x;
    }
    block_reduce_and_finish<B, 2>(red, partials, ticket, result);
}

#ifndef GPUQT_PAIR_TU   // the non-template kernels below belong to gpuqt.cu's translation unit only
// [batch][N] (host order) <-> [N][B] (device order)
__global__ void to_device_layout(long long N, int B, const double2* __restrict__ src, double2* __restrict__ dst) {
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= N * B) return;
    const long long row = i / B;
    const int b = (int)(i % B);
    dst[i] = src[(size_t)b * N + row];
}
__global__ void from_device_layout(long long N, int B, const double2* __restrict__ src, double2* __restrict__ dst) {
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= N * B) return;
    const long long row = i / B;
    const int b = (int)(i % B);
    dst[(size_t)b * N + row] = src[i];
}
// out = c * in (complex): the start b_{N_p-1} = c_{N_p-1} psi of the Clenshaw recurrence
__global__ void scale_vec(long long n, double cr, double ci, const double2* __restrict__ in, double2* __restrict__ out) {
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    const double2 v = in[i];
    out[i] = make_double2(cr * v.x - ci * v.y, cr * v.y + ci * v.x);
}
__global__ void zero_vec(long long n, double2* __restrict__ v) {
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) v[i] = make_double2(0.0, 0.0);
}

// Doubling identity (T_2m = 2 T_m^2 - 1, T_2m+1 = 2 T_m+1 T_m - T_1):
// dots[j] = {<a_{j+1}|a_{j+1}>, Re<a_{j+1}|a_j>, <a_j|a_j> (j = 0 only)}[B]  ->  C[b][n]
//   C_0 = <a_0|a_0>, C_1 = <a_1|a_0>, C_{2j+2} = 2<a_{j+1}|a_{j+1}> - C_0, C_{2j+1} = 2<a_{j+1}|a_j> - C_1
__global__ void finalize_doubling(int B, int n_moments, int n_steps, const double* __restrict__ dots,
                                  double* __restrict__ C) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= B * n_moments) return;
    const int b = i / n_moments, n = i % n_moments;
    const double c0 = dots[(0 * 3 + 2) * B + b], c1 = dots[(0 * 3 + 1) * B + b];
    double v;
    if (n == 0) v = c0;
    else if (n == 1) v = c1;
    else if (n & 1) v = 2.0 * dots[((size_t)((n - 1) / 2) * 3 + 1) * B + b] - c1;
    else v = 2.0 * dots[((size_t)((n - 2) / 2) * 3 + 0) * B + b] - c0;
    C[(size_t)b * n_moments + n] = v;
}
// dots[n] = {Re, Im}[B] of <phi_L|T_n b>  ->  C[b][n] = Re
__global__ void finalize_left(int B, int n_moments, const double* __restrict__ dots, double* __restrict__ C) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= B * n_moments) return;
    const int b = i / n_moments, n = i % n_moments;
    C[(size_t)b * n_moments + n] = dots[((size_t)n * 2 + 0) * B + b];
}

// Jackson damping folded with the (2 - delta_n0) factor: mu_scale[n] = g_n (2 - delta_n0)  (Eq. 31)
__global__ void jackson_kernel(int n_moments, double* __restrict__ gs) {
    const int n = blockIdx.x * blockDim.x + threadIdx.x;
    if (n >= n_moments) return;
    const double alpha = 1.0 / (n_moments + 1.0);
    double s, c, s1, c1;
    sincospi(n * alpha, &s, &c);
    sincospi(alpha, &s1, &c1);
    const double g = (1.0 - n * alpha) * c + alpha * s * (c1 / s1);
    gs[n] = (n == 0) ? g : 2.0 * g;
}

// Energy transform by Clenshaw summation (Eq. 25-27): one thread per (set, energy)
__global__ void transform_kernel(int n_moments, int n_sets, int n_energies, const double* __restrict__ gs,
                                 const double* __restrict__ C, const double* __restrict__ energies,
                                 double inv_dE, double volume, double* __restrict__ out) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n_sets * n_energies) return;
    const int s = i / n_energies, j = i % n_energies;
    const double e = energies[j] * inv_dE;
    const double* c = C + (size_t)s * n_moments;
    double b1 = 0.0, b2 = 0.0;
    for (int k = n_moments - 1; k >= 1; --k) {
        const double bk = fma(2.0 * e, b1, gs[k] * c[k] - b2);
        b2 = b1;
        b1 = bk;
    }
    const double sum = gs[0] * c[0] + e * b1 - b2;
    const double pref = 2.0 * inv_dE / (3.14159265358979323846 * volume * sqrt(1.0 - e * e));
    out[i] = pref * sum;
}

// Running conductivity (units e = 1) from the transformed correlation functions, one thread per
// energy, a sequential walk over the time rows (PAPER.md:81 Eq. 2, :92 Eq. 5, :123 Eq. 11):
//   kind 0  in[k][j] = rho C_vv(E_j, t_k), t_k = sum_{i<k} dt_i:  sigma[k][j] = trapezoid integral to t_k  [A25]
//   kind 1  in[k][j] = rho dX^2(E_j, t_{k+1}), dX^2(0) = 0:        sigma[k][j] = (in[k] - in[k-1]) / (2 dt_k), the
//           value at the middle of step k [A26];  length[k][j] = 2 sqrt(in[k][j] / dos[j])
__global__ void conductivity_kernel(int kind, int n_t, int n_e, const double* __restrict__ in,
                                    const double* __restrict__ dos, const double* __restrict__ dt,
                                    double* __restrict__ sigma, double* __restrict__ length) {
    const int j = blockIdx.x * blockDim.x + threadIdx.x;
    if (j >= n_e) return;
    if (kind == 0) {
        double acc = 0.0, before = in[j];
        sigma[j] = 0.0;
        for (int k = 1; k < n_t; ++k) {
            const double now = in[(size_t)k * n_e + j];
            acc += 0.5 * (before + now) * dt[k - 1];
            sigma[(size_t)k * n_e + j] = acc;
            before = now;
        }
    } else {
        double before = 0.0;
        const double rho = dos ? dos[j] : 0.0;
        for (int k = 0; k < n_t; ++k) {
            const double now = in[(size_t)k * n_e + j];
            sigma[(size_t)k * n_e + j] = (now - before) / (2.0 * dt[k]);
            if (length) length[(size_t)k * n_e + j] = 2.0 * sqrt((rho > 0.0 && now > 0.0) ? now / rho : 0.0);
            before = now;
        }
    }
}

// Decode the packed records back to canonical padded row-major arrays (bit-exact check)
__global__ void decode_table(const Mat m, int32_t* __restrict__ col, double* __restrict__ re,
                             double* __restrict__ im, double* __restrict__ dx) {
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= m.N * m.K) return;
    const long long row = i / m.K;
    const int k = (int)(i % m.K);
    const RecView rv = record_view(m, row >> 5);
    const int r = (int)(row & 31);
    int c = (int)row;
    double hr = 0.0, hi = 0.0, d = 0.0;
    if (k < rv.w) {
        c = rv.col_at(k, r);
        if (hop_is_const(m.hop)) {
            hr = c < m.N ? m.hop_const : 0.0;
            c = c < m.N ? c : (int)row;
        } else {
            hr = rv.hre[k * 32 + r];
        }
        if (m.cplx) hi = rv.him[k * 32 + r];
        d = min_image(m.x[c] - m.x[row], m.box);
    }
    if (col) col[i] = c;
    if (re) re[i] = hr;
    if (im) im[i] = hi;
    if (dx) dx[i] = d;
}

#endif  // GPUQT_PAIR_TU

}  // namespace gpuqt

namespace gpuqt {

// ---------------------------------------------------------------------------------- small lattices
// Lattices whose matrix and four vector sets fit one SM's shared memory (config c1: 2304 orbitals) are
// launch-latency bound on the streaming kernels (one launch per recurrence term).  cheb_small_kernel
// runs a WHOLE recurrence in one launch of one CTA: matrix (decoded to plain arrays) and vectors live in
// shared memory, the terms are separated by __syncthreads(), the per-term dots are reduced in a fixed
// order (warp shuffle -> shared memory over warps) and written straight to dots[term].
//   MODE doubling : T_m from v0; dots {<T_m|T_m>, Re<T_m|T_{m-1}>, <T_{m-1}|T_{m-1}>} per term   (Eq. 28, 30)
//   MODE left     : T_n from v0; dots <aux|T_n> (Re, Im) per term                                  (Eq. 29)
//   MODE evolve   : out = sum_k c_k T_k(H~) aux by Clenshaw (v0 unused; coef[k] = c_k)             (Eq. 17)
constexpr int kSmallThreads = 1024;

struct SmallArgs {
    const double2* v0;      // doubling / left: T_0
    const double2* aux;     // left: phi_L; evolve: the vector being evolved
    double2* out;           // evolve: result
    const double2* coef;    // evolve: c_k, k < n_terms
    double* dots;           // doubling: [term-1][3][B]; left: [term][2][B]
    int n_terms;            // doubling / left: terms m = 1 .. n_terms-1; evolve: order
};

template <int B, int MODE>
__global__ void __launch_bounds__(kSmallThreads, 1) cheb_small_kernel(const Mat m, const SmallArgs a) {
    constexpr int Q = (MODE == kModeDoubling) ? 3 : 2;
    constexpr bool DOTS = (MODE == kModeDoubling || MODE == kModeLeft);
    extern __shared__ __align__(16) unsigned char sm_raw[];
    __shared__ double s_red[kSmallThreads / 32][Q * B];
    const int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5;
    const int N = (int)m.N, K = m.K, NB = N * B;
    const int nd = hop_doubles(m.hop);
    double2* vec = reinterpret_cast<double2*>(sm_raw);                  // 3 ring slots
    double2* aux = vec + 3 * (size_t)NB;
    double* on = reinterpret_cast<double*>(aux + NB);
    double* hre = on + N;                                               // [K][N] if nd >= 1
    double* him = hre + (nd >= 1 ? (size_t)K * N : 0);                  // [K][N] if nd == 2
    int* col = reinterpret_cast<int*>(him + (nd == 2 ? (size_t)K * N : 0));   // [K][N]; padding -> row itself, weight 0
    double* wpad = nullptr;
    (void)wpad;
    // decode the records into plain arrays
    for (int row = tid; row < N; row += kSmallThreads) {
        const RecView rv = record_view(m, row >> 5);
        const int r = row & 31;
        on[row] = rv.on[r];
        for (int k = 0; k < K; ++k) {
            int c = row;
            double hr = 0.0, hi = 0.0;
            if (k < rv.w) {
                c = rv.col_at(k, r);
                if (hop_is_const(m.hop)) {
                    hr = c < N ? m.hop_const : 0.0;
                    c = c < N ? c : row;
                } else {
                    hr = rv.hre[k * 32 + r];
                    if (nd == 2) hi = rv.him[k * 32 + r];
                }
            }
            col[k * N + row] = hop_is_const(m.hop) && hr == 0.0 ? -1 : c;   // const variant: -1 marks "no entry"
            if (nd >= 1) hre[k * N + row] = hr;
            if (nd == 2) him[k * N + row] = hi;
        }
    }
    const double2* src0 = (MODE == kModeEvolve) ? a.aux : a.v0;
    for (int i = tid; i < NB; i += kSmallThreads) {
        if (MODE == kModeEvolve) {
            const double2 s = a.aux[i], c = a.coef[a.n_terms - 1];
            aux[i] = s;
            vec[i] = make_double2(c.x * s.x - c.y * s.y, c.x * s.y + c.y * s.x);   // b_{order-1} = c_{order-1} src
        } else {
            vec[i] = src0[i];
            if (MODE == kModeLeft) aux[i] = a.aux[i];
        }
    }
    __syncthreads();
    if (MODE == kModeEvolve && a.n_terms == 1) {
        for (int i = tid; i < NB; i += kSmallThreads) a.out[i] = vec[i];
        return;
    }
    int cur = 0;                     // slot of x_{m-1}; x_{m-2} in (cur + 2) % 3; x_m goes to (cur + 1) % 3
    for (int t = 1; t < a.n_terms; ++t) {
        const double2* in = vec + (size_t)cur * NB;
        const double2* prev = vec + (size_t)((cur + 2) % 3) * NB;
        double2* out = vec + (size_t)((cur + 1) % 3) * NB;
        const bool first = (t == 1);
        const bool half = (MODE == kModeEvolve) ? (t == a.n_terms - 1) : first;
        const double scale = half ? m.inv_dE : 2.0 * m.inv_dE;
        double2 ck = make_double2(0.0, 0.0);
        if (MODE == kModeEvolve) ck = a.coef[a.n_terms - 1 - t];
        double red[Q];
#pragma unroll
        for (int q = 0; q < Q; ++q) red[q] = 0.0;
        for (int i = tid; i < NB; i += kSmallThreads) {
            const int row = i / B, b = i % B;
            const double2 self = in[i];
            double sr = on[row] * self.x, si = on[row] * self.y;
            for (int k = 0; k < K; ++k) {
                const int c = col[k * N + row];
                if (hop_is_const(m.hop)) {
                    if (c >= 0) {
                        const double2 v = in[c * B + b];
                        sr = fma(m.hop_const, v.x, sr);
                        si = fma(m.hop_const, v.y, si);
                    }
                } else {
                    const double2 v = in[c * B + b];
                    const double hr = hre[k * N + row];
                    sr = fma(hr, v.x, sr);
                    si = fma(hr, v.y, si);
                    if (nd == 2) {
                        const double hi = him[k * N + row];
                        sr = fma(-hi, v.y, sr);
                        si = fma(hi, v.x, si);
                    }
                }
            }
            double2 tt = make_double2(scale * sr, scale * si);
            if (!first) {
                const double2 p = prev[i];
                tt.x -= p.x;
                tt.y -= p.y;
            }
            if (MODE == kModeEvolve) {
                const double2 s = aux[i];
                tt.x += ck.x * s.x - ck.y * s.y;
                tt.y += ck.x * s.y + ck.y * s.x;
                if (half) a.out[i] = tt;
            } else if (MODE == kModeDoubling) {
                red[0] += tt.x * tt.x + tt.y * tt.y;
                red[1] += tt.x * self.x + tt.y * self.y;
                if (first) red[2] += self.x * self.x + self.y * self.y;
            } else {
                const double2 l = aux[i];
                red[0] += l.x * tt.x + l.y * tt.y;
                red[1] += l.x * tt.y - l.y * tt.x;
            }
            out[i] = tt;
        }
        if (DOTS) {
            // fixed-order reduction over the threads that hold vector b = tid % B
#pragma unroll
            for (int q = 0; q < Q; ++q) {
#pragma unroll
                for (int off = 16; off >= B; off >>= 1) red[q] += __shfl_xor_sync(0xffffffffu, red[q], off);
            }
            if (lane < B) {
#pragma unroll
                for (int q = 0; q < Q; ++q) s_red[wid][q * B + lane] = red[q];
            }
            __syncthreads();
            if (tid < Q * B) {
                double s = 0.0;
                for (int w = 0; w < kSmallThreads / 32; ++w) s += s_red[w][tid];
                const size_t base = (MODE == kModeDoubling) ? (size_t)(t - 1) * 3 * B : (size_t)t * 2 * B;
                a.dots[base + tid] = s;
            }
        }
        __syncthreads();
        cur = (cur + 1) % 3;
    }
}

}  // namespace gpuqt
