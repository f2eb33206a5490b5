// sm_100a kernels of the GPUQT hot path.  See include/gpuqt.h for the boundary and DESIGN.md for
// the layout, the byte model and the roofline of each kernel.
//
// Layout
//   vectors   complex fp64 [NV + 1][B] as double2: the B vectors of a row are contiguous (16*B bytes),
//             so one neighbour index serves one 16*B-byte gather (B = 8: one 128-byte line).  Row NV
//             of every buffer is all zero and never written (NV = N; a row slab of a decomposed lattice
//             keeps its halo rows N .. NV-1 in between, see Mat).
//   matrix    packed sliced ELL.  A slice is 32 consecutive rows; slice s of width w is ONE
//             contiguous record, column-major inside the record:
//                 double hre[w][32] (per-entry variants) | double him[w][32] (complex variant) |
//                 double onsite[32] | int32 col[w][32]
//             record bytes = 32 * (8 w nd + 8 + 4 w), nd = doubles per entry (0, 1, 2), a multiple
//             of 128.  Records are stored back to back; slice_off[s] is the byte offset of record
//             s.  Padding entries are (own row, hop 0.0); in the constant-hopping variants (nd = 0:
//             every stored hopping is the same real number, kept in Mat::hop_const) padding is
//             col = NV, the zero row (and x[NV] = 0), so the walk needs no guard.  The table is padded
//             with all-padding records up to a multiple of kTilePad slices, so a tile of several
//             slices is always one contiguous copy.
//   warp      the unit of work is (warp, tile); a tile is S consecutive slices (S = 2 at B = 1 on
//             the unrolled uniform tables, else 1).  A stage of a warp's shared-memory pipeline holds
//             everything the tile streams exactly once: the packed records and the tile's own rows
//             of x_{m-1} (and e_{m-1}) and of x_{m-2} (and e_{m-2}) -- TMA copies (cp.async.bulk +
//             mbarrier) issued by the warp's lane 0 one or more tiles ahead, so the streams never sit
//             on the warp's scoreboard and there is no CTA-wide barrier in the loop.  A warp walks the
//             tile in rounds of 32/LPR rows; a lane owns V consecutive vectors of a row (V = 1 at B = 1;
//             2 at B = 2, 4: one 256-bit access per operand; 4 at B = 8 in the KPM / evolve kernels: two)
//             and LPR = B/V lanes share a row; at B = 1 the two rounds of a tile are walked
//             together (all gathers of both first, then the arithmetic) for memory-level parallelism.
//             Neighbours inside the tile are read from the staged rows in shared memory; the others
//             are gathered from global memory (L2 hits along the sweep front).
//   launch    a launch performs the recurrence steps m_begin .. m_end-1.  Single-step launches are
//             plain launches; multi-step launches are cooperative (all CTAs co-resident) and separate
//             the steps by a grid-wide barrier, so a whole moment set or a whole time step is ONE
//             launch when the working set lives in L2 and the launch gaps would dominate.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#ifndef GPUQT_THREADS
#define GPUQT_THREADS 256
#endif

#ifndef GPUQT_MINB
#define GPUQT_MINB 2
#endif
#ifndef GPUQT_MINB_B1
#define GPUQT_MINB_B1 2
#endif
// (psi, chi) evolve kernel, experiment: two CTAs per SM -- a lane owns ONE vector of a row (128-bit accesses, half the
// registers of the 256-bit ownership) and x_{m-2}, e_{m-2} rows are read by streaming loads.  Measured: no gain
// (profiles/r2_ncu_summary.md), so it is off.
#ifndef GPUQT_MSD_V1
#define GPUQT_MSD_V1 0
#endif
// KPM / evolve kernels: a lane owns FOUR vectors of a row (two 256-bit accesses per operand) at B = 8 -- two lanes
// per row instead of four halve the per-row address / predicate / column / hopping reads; 180 registers, one CTA
// per SM (c5: kpm_left 1710 -> 1532 us per step).  GPUQT_V4 = 1 does the same at B = 4 (one lane per row, 224
// registers): the c4 KPM step goes from 157.5 to 190.8 us (8 warps per SM hide too little latency), so it is off.
#ifndef GPUQT_V4
#define GPUQT_V4 0
#endif
#ifndef GPUQT_V4_B8
#define GPUQT_V4_B8 1
#endif
// B = 8, KPM / evolve kernels: x_{m-2} rows by streaming loads (1) or staged by TMA (0).  With one CTA per SM the
// staged form fits (10.5 KB per stage) and wins: c5 kpm_left 1530.7 (direct) -> 1505.4 us (staged), 0.94 of the copy peak
#ifndef GPUQT_PD8
#define GPUQT_PD8 0
#endif
__host__ __device__ constexpr bool lane_owns_four(int B, int mode) {
    return mode != 3 /* kModeEvolveMsd */ && ((GPUQT_V4_B8 && B >= 8) || (GPUQT_V4 && B >= 4));
}
#ifndef GPUQT_MINB_MSD
#define GPUQT_MINB_MSD (GPUQT_MSD_V1 ? 2 : 1)
#endif

// -DGPUQT_CHECKED=1: range checks of every gathered column, staged-row offset and pipeline index inside the
// kernels (__trap() on violation -> the next CUDA call fails).  A test build: compute-sanitizer is not
// available on the GPU pool this was developed on (profiles/r2_sanitizers.md).
#ifndef GPUQT_CHECKED
#define GPUQT_CHECKED 0
#endif
#if GPUQT_CHECKED
#define GPUQT_CHECK(cond) do { if (!(cond)) __trap(); } while (0)
#else
#define GPUQT_CHECK(cond) do { } while (0)
#endif

namespace gpuqt {

constexpr int kThreads = GPUQT_THREADS;
constexpr int kWarps = kThreads / 32;
constexpr int kSlice = 32;
constexpr int kMaxStages = 4;
constexpr int kTilePad = 4;          // the record array is padded to a multiple of this many slices

// nd = doubles stored per entry: 0 constant real hopping, 1 real, 2 complex
__host__ __device__ __forceinline__ long long record_bytes(int w, int nd) {
    return 32LL * (8LL * w * nd + 8 + 4LL * w);
}
__host__ __device__ __forceinline__ int record_width(long long bytes, int nd) {
    return (int)((bytes / 32 - 8) / (4 + 8 * nd));
}
// kHopConst16 / kHopConst16P: constant hopping AND 16-bit columns -- the record is
//     double onsite[32] | int32 base[8] (first w used) | uint16 delta[w][32]
//     col = base[k] + delta[k][lane];  in the P variant delta == 0xffff stands for the zero row N
//     (tables with padding entries: vacancies, open boundaries)
// (uniform tables whose real columns spread less than 65535 inside every (slice, k); lattices in
// natural order do).  288 + 64 w bytes instead of 256 + 128 w.
// kHopStencil: constant hopping on a REGULAR lattice -- no index array is streamed at all (SURVEY 8(f) 3,
// "implicit stencil"; the paper's own examples are such lattices).  The columns of a
// slice RELATIVE to its first row, rel[k][lane] = col - 32 s, repeat from slice to slice on a regular lattice
// (they differ only where a periodic wrap falls inside the slice), so the table is stored as
//     record  s : double onsite[32]                         (256 bytes, streamed from HBM)
//     pid[s]    : int32 index of the slice's pattern        (4 bytes per slice)
//     dict[p]   : int32 rel[K][32]                          (a few hundred distinct patterns at most: L2 resident)
// and a stage of the pipeline is filled by two bulk copies per slice (record from HBM, pattern from L2) to the
// same image the kHopConst walk reads: onsite[32] | int32 rel[K][32];  col = 32 s + rel.
enum Hop : int { kHopReal = 0, kHopComplex = 1, kHopConst = 2, kHopConst16 = 3, kHopConst16P = 4, kHopStencil = 5 };
__host__ __device__ constexpr bool hop_is_16(int hop) { return hop == kHopConst16 || hop == kHopConst16P; }
__host__ __device__ constexpr bool hop_is_const(int hop) { return hop == kHopConst || hop_is_16(hop) || hop == kHopStencil; }
__host__ __device__ constexpr int hop_doubles(int hop) { return hop_is_const(hop) ? 0 : hop == kHopComplex ? 2 : 1; }
// bytes of one slice record as stored (and streamed from HBM)
__host__ __device__ __forceinline__ long long hop_record_bytes(int w, int hop) {
    return hop == kHopStencil ? 256LL : hop_is_16(hop) ? 288LL + 64LL * w : record_bytes(w, hop_doubles(hop));
}
// bytes one slice's record image takes inside a pipeline stage (kHopStencil: record + pattern)
__host__ __device__ __forceinline__ long long hop_stage_bytes(int w, int hop) {
    return hop == kHopStencil ? 256LL + 128LL * w : hop_record_bytes(w, hop);
}
constexpr unsigned kPad16 = 0xffffu;     // 16-bit delta that stands for the zero row N

struct Mat {
    const unsigned char* __restrict__ rec;      // packed slice records
    const long long* __restrict__ slice_off;    // [n_slices_padded + 1] byte offsets (ragged variant)
    const double* __restrict__ x;               // [NV + 1], x[NV] = 0
    const int* __restrict__ pid;                // kHopStencil: [n_slices_padded] pattern of each slice
    const int* __restrict__ dict;               // kHopStencil: [n_patterns][K][32] columns relative to the slice's first row
    long long N;                                // rows of the table = rows this device computes
    long long NV;                               // index of the all-zero row of every vector buffer (vector rows: NV + 1).
                                                // NV = N, except for a row slab of a decomposed lattice, whose vectors
                                                // carry the halo rows N .. NV-1 behind the owned rows (columns may point there)
    long long n_slices;                         // real slices, ceil(N / 32)
    int K;                                      // K_max
    int uniform;                                // every record has width K
    int cplx;
    int hop;                                    // Hop variant of the records
    double hop_const;                           // constant-hopping variants: the one hopping value
    double inv_dE;
    double box;                                 // <= 0: open boundary
};

enum Mode : int {
    kModeDoubling = 0,   // x_m, dots |x_m|^2, Re<x_m|x_{m-1}>, |x_{m-1}|^2            (Eq. 28, 30)
    kModeLeft = 1,       // x_m, dot <phi_L|x_m>                                      (Eq. 29)
    kModeEvolve = 2,     // Clenshaw term b_k = c_k src + 2 H~ b_{k+1} - b_{k+2}      (Eq. 17, 21)
    kModeEvolveMsd = 3,  // the same for the (a, e) pair, [X,H~] weights in the walk (Eq. 18, 22)
};

// One three-term recurrence x_m = 2 H~ x_{m-1} - x_{m-2} (+ c_k src), m = 1 .. terms-1, and the steps
// [m_begin, m_end) of it that this launch performs.  x_0 is given; x_m (m >= 1) lives in
// ring[(m - 1) % 3] (the last term optionally somewhere else).  Forward recurrences (moments) apply
// factor 1 instead of 2 in step 1 (T_1 = H~ T_0); Clenshaw recurrences (evolution) in the last step.
struct RecArgs {
    const double2* x0;           // x_0
    double2* ring[3];
    const double2* e0;           // MSD pair: e_0 and its ring
    double2* ring_e[3];
    // B >= 2: device addresses of the TMA tensor maps (CUtensorMap, 128-byte swizzle) of the buffers above
    const void* tm_x0;
    const void* tm_ring[3];
    const void* tm_e0;
    const void* tm_ring_e[3];
    double2* last_out;           // evolve: destination of x_{terms-1} (instead of its ring slot)
    double2* last_out_e;
    const double2* src;          // evolve: the vector being evolved (psi; a; b), read-only
    const double2* src_e;        // evolve MSD: chi
    const double2* phiL;         // kModeLeft
    const double* coef;          // evolve: c_k as (re, im) pairs, k < terms; step m adds c_{terms-1-m} src
    double* dots;                // step m writes its Q*B reduced dots at dots[(m - dot_m0) * Q*B ...]
    int terms;
    int m_begin, m_end;
    int clenshaw;
    int store_last;              // is x_{terms-1} written at all (moments: no)
    int dot_m0;
    int sweep0;                  // direction of step m_begin: 1 = from the top
    int alternate;               // the direction alternates from step to step (L2 reuse across the boundary)
    int run;                     // consecutive tiles one CTA walks before jumping (multiple of kWarps)
    int stages;                  // shared-memory stages per warp (<= kMaxStages)
    int stage_bytes;             // bytes of one stage: records + staged vector rows
    int rec_bytes;               // bytes reserved for the records inside a stage
    int multi;                   // cooperative multi-step launch: grid barrier between steps
    double* partials;            // [3][grid][Q*B] (multi-step launches: by step % 3)
    unsigned int* ticket;        // single-step launches: last-block detection
    unsigned int* barrier;       // multi-step launches: monotonically increasing arrival counter (zeroed by the host)
};

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
// Orders generic-proxy accesses (ordinary stores / loads) against async-proxy accesses (TMA) of the
// executing thread.  Used on both sides of the grid barrier of a multi-step launch: x_m is written by
// ordinary stores of one SM and read by TMA copies of another in the next step.
__device__ __forceinline__ void fence_proxy_async() { asm volatile("fence.proxy.async;" ::: "memory"); }

// Staged vector rows are written by the TMA with the 128-byte swizzle (16-byte chunk index, address bits 4-6,
// ^= address bits 7-9; box rows are whole 128-byte lines): a lane's two 16-byte reads at a 32-byte lane stride then
// fall on distinct banks for every group of 8 lanes when it reads its OWN row (without it: a 2-way bank conflict on
// every 128-bit read).  Uses the absolute shared address, as the TMA does.  An in-slice gather of the row one
// further on (the +-x neighbours of a lattice in natural order; 64 bytes at B = 4) still takes 6 instead of 4
// wavefronts: the 256 bytes a group reads then span half of line L, line L + 1 and half of line L + 2, and for
// lines L = 2, 6 (mod 8) the two halves collide under this swizzle (ncu, round 2: 20 % of the shared-memory
// wavefronts of the c4 step).  GPUQT_SWZ64 = 1 is the experiment that removes it -- 64-byte lines with the
// 64-byte swizzle, where address bit 6 keeps the halves apart: conflict-free and parity-green, but the TMA then
// moves 64-byte lines and the c4 step went from 156 to 164 us, so it is off.
#ifndef GPUQT_SWZ64
#define GPUQT_SWZ64 0
#endif
constexpr int kSwizzleLineBytes = GPUQT_SWZ64 ? 64 : 128;     // bytes of one line of the tensor maps
__device__ __forceinline__ uint32_t swz32(uint32_t sa) {
#if GPUQT_SWZ64
    return sa ^ ((sa >> 3) & 0x30u);
#else
    return sa ^ ((sa >> 3) & 0x70u);
#endif
}

__device__ __forceinline__ void st_vec(double2* p, double2 v) { *p = v; }
__device__ __forceinline__ unsigned int ld_acquire_gpu(const unsigned int* p) {
    unsigned int v;
    asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
    return v;
}
__device__ __forceinline__ void red_release_gpu_inc(unsigned int* p) {
    asm volatile("red.release.gpu.global.add.u32 [%0], 1;" ::"l"(p) : "memory");
}

// Grid-wide barrier of a cooperative launch (all CTAs co-resident), in two halves so that a CTA can do work that
// nobody waits for between its arrival and the completion (the deferred reduction of the previous step's dots).
// `counter` only ever grows; the e-th barrier of the launch completes when it reaches e * gridDim.x.
// Ordering: every thread's stores -> bar.sync -> thread 0's red.release.gpu (cumulative) ... thread 0's
// ld.acquire.gpu -> bar.sync -> every thread's loads: everything the CTA wrote before the barrier is visible to every
// CTA after it, without separate membar.gl fences; the proxy fences extend that to the TMA (async proxy) reads that
// follow x_m's ordinary stores.
__device__ __forceinline__ void grid_arrive(unsigned int* counter) {
    fence_proxy_async();
    __syncthreads();
    if (threadIdx.x == 0) red_release_gpu_inc(counter);
}
__device__ __forceinline__ void grid_wait(unsigned int* counter, unsigned int target) {
    if (threadIdx.x == 0) {
        while (ld_acquire_gpu(counter) < target) {
        }
    }
    __syncthreads();
    fence_proxy_async();
}

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
};
// resident CTAs per SM the register allocation aims at
__host__ __device__ constexpr int min_blocks(int B, int mode) {
    return mode == kModeEvolveMsd ? GPUQT_MINB_MSD : B == 1 ? GPUQT_MINB_B1 : lane_owns_four(B, mode) ? 1 : GPUQT_MINB;
}

// B = 8, (psi, chi) kernel: a slice's rows are 4 KB per stream and four staged streams do not fit two stages, so
// x_{m-2}, e_{m-2} own rows are read by streaming 256-bit loads at the top of the round instead.  (Round 1 did the
// same in the KPM kernels at B = 8 to keep two CTAs per SM; with four vectors per lane there is one CTA per SM and
// the staged form is back, see GPUQT_PD8.)
// The (psi, chi) evolve kernel does the same at every B when GPUQT_MSD_V1 is on (four staged
// streams would leave room for one CTA per SM).  Direct reads for it alone, at one CTA per SM, change nothing
// (c4: evolve_msd 195.3 vs 197.2 ms per 10 steps); GPUQT_PREV_DIRECT = 1 for every kernel costs the KPM kernels
// 7 % at B = 4 (158 -> 170 us per step).
#ifndef GPUQT_PREV_DIRECT     // experiment: x_{m-2} by streaming loads at every B
#define GPUQT_PREV_DIRECT 0
#endif
__host__ __device__ constexpr bool prev_direct(int B, int mode) {
    return (B >= 8 && (GPUQT_PD8 || mode == kModeEvolveMsd)) || GPUQT_PREV_DIRECT ||
           (GPUQT_MSD_V1 && mode == kModeEvolveMsd);
}

// slices per tile at B = 1 on the unrolled uniform tables (2 or 4; kTilePad is a multiple): a tile's bookkeeping
// (pipeline cursors, TMA issues, mbarrier wait: ~150 warp instructions) is paid once per tile
#ifndef GPUQT_B1_SLICES
#define GPUQT_B1_SLICES 2
#endif
// A lane owns V consecutive vectors of a row (V = 2 when B >= 2: one 256-bit access per operand).
// A tile is S consecutive slices and is walked in ROUNDS rounds of RS rows, U rounds at a time.
template <int B, int KT, int MODE = kModeDoubling>
struct LaneShape {
    static constexpr int V = lane_owns_four(B, MODE) ? 4
                             : (B >= 2 && !(GPUQT_MSD_V1 && MODE == kModeEvolveMsd)) ? 2 : 1;
    static constexpr bool SWZ = B >= 2;                    // staged rows are written by swizzled tensor copies
    static constexpr int LPR = B / V;                      // lanes per row
    static constexpr int RS = 32 / LPR;                    // rows per round
    static constexpr int S = (B == 1 && KT > 0) ? GPUQT_B1_SLICES : 1;   // slices per tile
    static constexpr int ROUNDS = S * LPR;                 // rounds per tile
    static constexpr int U = (B == 1 && KT > 0) ? 2 : 1;   // rounds walked together
};
__host__ __device__ constexpr int tile_slices(int B, int kt) { return (B == 1 && kt > 0) ? GPUQT_B1_SLICES : 1; }

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
template <int V, bool SWZ>
__device__ __forceinline__ CV<V> cv_lds_staged(const double2* p) {
    if constexpr (V == 4) {                 // 64 bytes, 64-byte aligned: the four chunks stay inside one half line
        const uint32_t p0 = swz32(smem_u32(p));
        CV<4> v;
#pragma unroll
        for (int j = 0; j < 4; ++j)
            asm volatile("ld.shared.v2.f64 {%0, %1}, [%2];" : "=d"(v.re[j]), "=d"(v.im[j]) : "r"(p0 ^ (16u * j)));
        return v;
    } else if constexpr (V == 2) {
        return cv_lds_swz(smem_u32(p));
    } else if constexpr (SWZ) {
        CV<1> v;
        asm volatile("ld.shared.v2.f64 {%0, %1}, [%2];" : "=d"(v.re[0]), "=d"(v.im[0]) : "r"(swz32(smem_u32(p))));
        return v;
    } else {
        return cv_lds<1>(p);
    }
}

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
template <>
__device__ __forceinline__ CV<4> cv_ld_stream<4>(const double2* p) {
    CV<4> v;
    asm volatile("ld.global.cs.v4.f64 {%0, %1, %2, %3}, [%4];"
                 : "=d"(v.re[0]), "=d"(v.im[0]), "=d"(v.re[1]), "=d"(v.im[1]) : "l"(p));
    asm volatile("ld.global.cs.v4.f64 {%0, %1, %2, %3}, [%4];"
                 : "=d"(v.re[2]), "=d"(v.im[2]), "=d"(v.re[3]), "=d"(v.im[3]) : "l"(p + 2));
    return v;
}
template <int V>
__device__ __forceinline__ void cv_st(double2* p, const CV<V>& v);
template <>
__device__ __forceinline__ void cv_st<4>(double2* p, const CV<4>& v) {
    asm volatile("st.global.v4.f64 [%0], {%1, %2, %3, %4};" ::"l"(p), "d"(v.re[0]), "d"(v.im[0]), "d"(v.re[1]), "d"(v.im[1]) : "memory");
    asm volatile("st.global.v4.f64 [%0], {%1, %2, %3, %4};" ::"l"(p + 2), "d"(v.re[2]), "d"(v.im[2]), "d"(v.re[3]), "d"(v.im[3]) : "memory");
}
template <>
__device__ __forceinline__ void cv_st<1>(double2* p, const CV<1>& v) {
    st_vec(p, make_double2(v.re[0], v.im[0]));
}
template <>
__device__ __forceinline__ void cv_st<2>(double2* p, const CV<2>& v) {
    asm volatile("st.global.v4.f64 [%0], {%1, %2, %3, %4};" ::"l"(p), "d"(v.re[0]), "d"(v.im[0]), "d"(v.re[1]), "d"(v.im[1])
                 : "memory");
}
// Gather of V consecutive vectors of row c of x_{m-1}: rows of the current tile come from the staged
// copy in shared memory, the others from global memory with an L2 evict_last hint (they are re-read
// by the neighbouring tiles).  Both loads are predicated, so there is no branch.
//   g_l  = byte address of (row 0, the lane's first vector) in global memory
//   s_l  = shared-window address of the same element of the tile's staged rows, minus row0 * RB
//          (mod 2^32: only rows of the tile are ever addressed through it)
//   RB   = bytes of one row (16 B);  TR = rows of a tile
template <int V, int TR, bool SWZ = false>
__device__ __forceinline__ CV<V> cv_gather(const char* g_l, uint32_t s_l, int c, int row0, int RB);
template <>
__device__ __forceinline__ CV<1> cv_gather<1, 32, true>(const char* g_l, uint32_t s_l, int c, int row0, int RB) {
    const unsigned d = (unsigned)(c - row0);
    const uint32_t sa = swz32(s_l + (uint32_t)c * (uint32_t)RB);
    const char* ga = g_l + (long long)c * RB;
    CV<1> v;
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "setp.lt.u32 p, %4, 32;\n"
        "@p ld.shared.v2.f64 {%0, %1}, [%2];\n"
        "@!p ld.global.v2.f64 {%0, %1}, [%3];\n"          // (the L2::evict_last qualifier exists for 256-bit loads only)
        "}"
        : "=d"(v.re[0]), "=d"(v.im[0])
        : "r"(sa), "l"(ga), "r"(d));
    return v;
}
// V = 1, plain (unswizzled) staged rows, any tile height
template <int TR>
__device__ __forceinline__ CV<1> cv_gather_plain(const char* g_l, uint32_t s_l, int c, int row0, int RB) {
    const unsigned d = (unsigned)(c - row0);
    const uint32_t sa = s_l + (uint32_t)c * (uint32_t)RB;
    const char* ga = g_l + (long long)c * RB;
    CV<1> v;
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "setp.lt.u32 p, %4, %5;\n"
        "@p ld.shared.v2.f64 {%0, %1}, [%2];\n"
        "@!p ld.global.v2.f64 {%0, %1}, [%3];\n"
        "}"
        : "=d"(v.re[0]), "=d"(v.im[0])
        : "r"(sa), "l"(ga), "r"(d), "n"(TR));
    return v;
}
template <>
__device__ __forceinline__ CV<1> cv_gather<1, 32, false>(const char* g_l, uint32_t s_l, int c, int row0, int RB) {
    return cv_gather_plain<32>(g_l, s_l, c, row0, RB);
}
template <>
__device__ __forceinline__ CV<1> cv_gather<1, 64, false>(const char* g_l, uint32_t s_l, int c, int row0, int RB) {
    return cv_gather_plain<64>(g_l, s_l, c, row0, RB);
}
template <>
__device__ __forceinline__ CV<1> cv_gather<1, 128, false>(const char* g_l, uint32_t s_l, int c, int row0, int RB) {
    return cv_gather_plain<128>(g_l, s_l, c, row0, RB);
}
template <>
__device__ __forceinline__ CV<4> cv_gather<4, 32, true>(const char* g_l, uint32_t s_l, int c, int row0, int RB) {
    const unsigned d = (unsigned)(c - row0);
    const uint32_t s0 = swz32(s_l + (uint32_t)c * (uint32_t)RB);
    const char* ga = g_l + (long long)c * RB;
    CV<4> v;
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "setp.lt.u32 p, %10, 32;\n"
        "@p ld.shared.v2.f64 {%0, %1}, [%8];\n"
        "@p ld.shared.v2.f64 {%2, %3}, [%11];\n"
        "@p ld.shared.v2.f64 {%4, %5}, [%12];\n"
        "@p ld.shared.v2.f64 {%6, %7}, [%13];\n"
        "@!p ld.global.L2::evict_last.v4.f64 {%0, %1, %2, %3}, [%9];\n"
        "@!p ld.global.L2::evict_last.v4.f64 {%4, %5, %6, %7}, [%9+32];\n"
        "}"
        : "=d"(v.re[0]), "=d"(v.im[0]), "=d"(v.re[1]), "=d"(v.im[1]), "=d"(v.re[2]), "=d"(v.im[2]), "=d"(v.re[3]), "=d"(v.im[3])
        : "r"(s0), "l"(ga), "r"(d), "r"(s0 ^ 16u), "r"(s0 ^ 32u), "r"(s0 ^ 48u));
    return v;
}
template <>
__device__ __forceinline__ CV<2> cv_gather<2, 32, true>(const char* g_l, uint32_t s_l, int c, int row0, int RB) {
    const unsigned d = (unsigned)(c - row0);
    const uint32_t sa = swz32(s_l + (uint32_t)c * (uint32_t)RB);
    const uint32_t sb = sa ^ 16u;
    const char* ga = g_l + (long long)c * RB;
    CV<2> v;
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "setp.lt.u32 p, %6, 32;\n"
        "@p ld.shared.v2.f64 {%0, %1}, [%4];\n"
        "@p ld.shared.v2.f64 {%2, %3}, [%7];\n"
        "@!p ld.global.L2::evict_last.v4.f64 {%0, %1, %2, %3}, [%5];\n"
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

// Operands of one recurrence step (derived from RecArgs at the top of the step, CTA-uniform)
struct StepCtx {
    const double2* in;       // x_{m-1}: gathered and own row
    const double2* prev;     // x_{m-2}: own row (unused when first)
    double2* out;            // x_m (unused when !store)
    const double2* in_e;     // MSD pair: e_{m-1}
    const double2* prev_e;   //           e_{m-2}
    double2* out_e;          //           e_m
    const void *tm_in, *tm_prev, *tm_in_e, *tm_prev_e;
    double cr, ci;           // c_k of this term (evolve)
    double scale;            // 2 / dE, or 1 / dE in the half step
    int first;               // no x_{m-2} term
    int store;               // write x_m
};

// Column of entry k of row rr of the slice whose record starts at s_col (int32 columns, or the base[8]
// table of the 16-bit variant with the deltas behind it)
template <int HOP>
__device__ __forceinline__ int col_of(const int* s_col, const unsigned short* s_d16, int k, int rr, int N) {
    if (hop_is_16(HOP)) {
        const unsigned d = s_d16[k * 32 + rr];
        if (HOP == kHopConst16P) return d == kPad16 ? N : s_col[k] + (int)d;
        return s_col[k] + (int)d;
    }
    return s_col[k * 32 + rr];
}

// U consecutive rounds (RS rows each) of one tile whose records and own rows sit in shared memory at
// `stage`.  Rows past the end of the table (last tile only) are computed like the others on zero
// inputs (their staged self / prev are replaced by 0 and their entries are padding), so the dot
// products need no guard; only their stores are predicated off.
template <int B, int KT, int HOP, int MODE>
__device__ __forceinline__ void walk_rounds(const Mat& m, const RecArgs& a, const StepCtx& io, const unsigned char* stage, int w,
                                            int row0, int rows_valid, int j0, int lane,
                                            double (&red)[ModeTraits<MODE>::Q * LaneShape<B, KT, MODE>::V]) {
    using LS = LaneShape<B, KT, MODE>;
    constexpr int V = LS::V, LPR = LS::LPR, RS = LS::RS, U = LS::U, TR = 32 * LS::S;
    constexpr int KU = KT > 0 ? KT : 1;
    constexpr int RB = B * 16;   // bytes of one row of a vector set
    constexpr bool MSD = (MODE == kModeEvolveMsd);
    constexpr bool CPLX = (HOP == kHopComplex), CONST = hop_is_const(HOP);
    constexpr bool STENCIL = (HOP == kHopStencil);
    constexpr int REC = KT > 0 ? (int)(STENCIL ? 256 + 128 * KT : hop_is_16(HOP) ? 288 + 64 * KT
                                                : 32 * (8 * KT * (CONST ? 0 : CPLX ? 2 : 1) + 8 + 4 * KT)) : 0;
    const int rl = lane / LPR, l = lane % LPR;
    // staged vector rows: [in | (in_e) | prev | (prev_e)], each TR * B double2
    const double2* s_in = reinterpret_cast<const double2*>(stage + a.rec_bytes);
    const double2* s_in_e = s_in + TR * B;
    const double2* s_prev = s_in + (MSD ? 2 : 1) * TR * B;
    const double2* s_prev_e = s_prev + TR * B;
    // lane-relative bases of the gathers (see cv_gather)
    const uint32_t sl_in = smem_u32(s_in + l * V) - (uint32_t)row0 * (uint32_t)RB;
    const uint32_t sl_in_e = smem_u32(s_in_e + l * V) - (uint32_t)row0 * (uint32_t)RB;
    const char* gl_in = reinterpret_cast<const char*>(io.in + l * V);
    const char* gl_in_e = reinterpret_cast<const char*>(io.in_e + l * V);
    constexpr bool PD = prev_direct(B, MODE);
    const int N = (int)m.NV;  // columns run over [0, NV]: owned rows, halo rows, the zero row

    int r[U];                 // row inside the tile
    bool ok[U];
    size_t vi[U];             // element in global memory
    const double* s_hre[U];
    const double* s_on[U];
    int srow0[U];             // kHopStencil: first row of the row's slice (the columns are relative to it)
    const int* s_col[U];
    const unsigned short* s_d16[U];
    CV<V> other[U], other_e[U], prev[U], prev_e[U], self[U], self_e[U];
    double xm[U];
#pragma unroll
    for (int u = 0; u < U; ++u) {
        r[u] = (j0 + u) * RS + rl;
        ok[u] = r[u] < rows_valid;
        vi[u] = (size_t)(row0 + (ok[u] ? r[u] : 0)) * B + l * V;
        const unsigned char* rec = stage + (LS::S > 1 ? (r[u] >> 5) * REC : 0);
        srow0[u] = STENCIL ? row0 + (LS::S > 1 ? (r[u] & ~31) : 0) : 0;
        s_hre[u] = reinterpret_cast<const double*>(rec);
        s_on[u] = s_hre[u] + w * 32 * hop_doubles(HOP);
        s_col[u] = reinterpret_cast<const int*>(s_on[u] + 32);                          // int32 columns, or base[8]
        s_d16[u] = reinterpret_cast<const unsigned short*>(s_col[u] + 8);                // kHopConst16: deltas
        // streamed own-row operands (evolved vector / phi_L): issued first, consumed last
        other[u] = cv_zero<V>();
        other_e[u] = cv_zero<V>();
        if (MODE == kModeEvolve || MSD) other[u] = cv_ld_stream<V>(&a.src[vi[u]]);
        if (MSD) other_e[u] = cv_ld_stream<V>(&a.src_e[vi[u]]);
        if (MODE == kModeLeft) other[u] = cv_ld_stream<V>(&a.phiL[vi[u]]);
        xm[u] = 0.0;
        if (MSD) xm[u] = m.x[row0 + (ok[u] ? r[u] : 0)];
        prev[u] = cv_zero<V>();
        prev_e[u] = cv_zero<V>();
        if (PD && !io.first && ok[u]) {         // rows past the end keep prev = 0 (their x_m must stay 0 for the dots)
            prev[u] = cv_ld_stream<V>(&io.prev[vi[u]]);
            if (MSD) prev_e[u] = cv_ld_stream<V>(&io.prev_e[vi[u]]);
        }
    }
#pragma unroll
    for (int u = 0; u < U; ++u) {
        const int si_ = r[u] * B + l * V;                                 // element inside the staged rows
        GPUQT_CHECK(si_ >= 0 && si_ + V <= TR * B && r[u] < TR);
        self[u] = ok[u] ? cv_lds_staged<V, LS::SWZ>(s_in + si_) : cv_zero<V>();
        self_e[u] = (MSD && ok[u]) ? cv_lds_staged<V, LS::SWZ>(s_in_e + si_) : cv_zero<V>();
    }

    CV<V> sum[U], sum_e[U], sum_x[U];   // H x, H e, [X,H] x (unscaled)
#pragma unroll
    for (int u = 0; u < U; ++u) sum[u] = sum_e[u] = sum_x[u] = cv_zero<V>();
    if (KT > 0) {
        // all gathers of the rows first (independent loads in flight), then the arithmetic
        constexpr int CH = KU;
#pragma unroll
        for (int k0 = 0; k0 < KU; k0 += CH) {
            CV<V> v[U][CH], ve[U][MSD ? CH : 1];
            double xn[U][MSD ? CH : 1];
#pragma unroll
            for (int u = 0; u < U; ++u) {
                const int rr = LS::S > 1 ? (r[u] & 31) : r[u];
#pragma unroll
                for (int kk = 0; kk < CH; ++kk) {
                    const int k = k0 + kk;
                    if (k < KU) {
                        const int c = col_of<HOP>(s_col[u], s_d16[u], k, rr, N) + srow0[u];
                        GPUQT_CHECK((unsigned)c <= (unsigned)N);
                        v[u][kk] = cv_gather<V, TR, LS::SWZ>(gl_in, sl_in, c, row0, RB);
                        if (MSD) {
                            ve[u][kk] = cv_gather<V, TR, LS::SWZ>(gl_in_e, sl_in_e, c, row0, RB);
                            xn[u][kk] = m.x[c];
                        }
                    }
                }
            }
#pragma unroll
            for (int u = 0; u < U; ++u) {
                const int rr = LS::S > 1 ? (r[u] & 31) : r[u];
#pragma unroll
                for (int kk = 0; kk < CH; ++kk) {
                    const int k = k0 + kk;
                    if (k < KU) {
                        double hr = 1.0, hi = 0.0;                              // CONST: the factor is applied once below
                        if (!CONST) hr = s_hre[u][k * 32 + rr];
                        if (CPLX) hi = (s_hre[u] + w * 32)[k * 32 + rr];
                        // constant hopping: the first neighbour starts the sum (no 0 + x additions)
                        if (CONST && k == 0) sum[u] = v[u][kk];
                        else if (CONST) cv_add<V>(sum[u], v[u][kk]);
                        else cv_fma<V, CPLX>(sum[u], hr, hi, v[u][kk]);
                        if (MSD) {
                            if (CONST && k == 0) sum_e[u] = ve[u][kk];
                            else if (CONST) cv_add<V>(sum_e[u], ve[u][kk]);
                            else cv_fma<V, CPLX>(sum_e[u], hr, hi, ve[u][kk]);
                            // [X,H]_mn = (X_m - X_n) H_mn = -dx H_mn
                            const double ndx = -min_image(xn[u][kk] - xm[u], m.box);
                            cv_fma<V, CPLX>(sum_x[u], ndx * hr, ndx * hi, v[u][kk]);
                        }
                    }
                }
            }
        }
    } else {
        const int rr = r[0] & 31;
        for (int k = 0; k < w; ++k) {
            const int c = col_of<HOP>(s_col[0], s_d16[0], k, rr, N) + srow0[0];
            GPUQT_CHECK((unsigned)c <= (unsigned)N);
            double hr = 1.0, hi = 0.0;
            if (!CONST) hr = s_hre[0][k * 32 + rr];
            if (CPLX) hi = (s_hre[0] + w * 32)[k * 32 + rr];
            const CV<V> vv = cv_gather<V, TR, LS::SWZ>(gl_in, sl_in, c, row0, RB);
            if (CONST) cv_add<V>(sum[0], vv);
            else cv_fma<V, CPLX>(sum[0], hr, hi, vv);
            if (MSD) {
                const CV<V> vve = cv_gather<V, TR, LS::SWZ>(gl_in_e, sl_in_e, c, row0, RB);
                if (CONST) cv_add<V>(sum_e[0], vve);
                else cv_fma<V, CPLX>(sum_e[0], hr, hi, vve);
                const double ndx = -min_image(m.x[c] - xm[0], m.box);
                cv_fma<V, CPLX>(sum_x[0], ndx * hr, ndx * hi, vv);
            }
        }
    }
    const double hs = CONST ? io.scale * m.hop_const : io.scale;          // scale of the neighbour sums
#pragma unroll
    for (int u = 0; u < U; ++u) {
        const int si_ = r[u] * B + l * V;
        if (!PD && !io.first && ok[u]) {
            prev[u] = cv_lds_staged<V, LS::SWZ>(s_prev + si_);
            if (MSD) prev_e[u] = cv_lds_staged<V, LS::SWZ>(s_prev_e + si_);
        }
        const double os = io.scale * s_on[u][LS::S > 1 ? (r[u] & 31) : r[u]];   // scale of the on-site term
        CV<V> t, te;   // x_m (b_k) and e_m
#pragma unroll
        for (int q = 0; q < V; ++q) {
            t.re[q] = fma(hs, sum[u].re[q], fma(os, self[u].re[q], -prev[u].re[q]));
            t.im[q] = fma(hs, sum[u].im[q], fma(os, self[u].im[q], -prev[u].im[q]));
            if (MODE == kModeDoubling) {
                red[0 * V + q] += t.re[q] * t.re[q] + t.im[q] * t.im[q];
                red[1 * V + q] += t.re[q] * self[u].re[q] + t.im[q] * self[u].im[q];
                // <x_{m-1}|x_{m-1}> is only used from the first step (C_0); later ones had it as <x_m|x_m>
                if (io.first) red[2 * V + q] += self[u].re[q] * self[u].re[q] + self[u].im[q] * self[u].im[q];
            } else if (MODE == kModeLeft) {   // conj(l) * t
                red[0 * V + q] += other[u].re[q] * t.re[q] + other[u].im[q] * t.im[q];
                red[1 * V + q] += other[u].re[q] * t.im[q] - other[u].im[q] * t.re[q];
            } else {
                // Clenshaw: b_k = c_k src + 2 H~ b_{k+1} - b_{k+2}; no accumulator is read or written
                t.re[q] += io.cr * other[u].re[q] - io.ci * other[u].im[q];
                t.im[q] += io.cr * other[u].im[q] + io.ci * other[u].re[q];
                if (MSD) {
                    te.re[q] = fma(hs, sum_e[u].re[q] + sum_x[u].re[q], fma(os, self_e[u].re[q], -prev_e[u].re[q]));
                    te.im[q] = fma(hs, sum_e[u].im[q] + sum_x[u].im[q], fma(os, self_e[u].im[q], -prev_e[u].im[q]));
                    te.re[q] += io.cr * other_e[u].re[q] - io.ci * other_e[u].im[q];
                    te.im[q] += io.cr * other_e[u].im[q] + io.ci * other_e[u].re[q];
                }
            }
        }
        if (ok[u] && io.store) {
            cv_st<V>(&io.out[vi[u]], t);
            if (MSD) cv_st<V>(&io.out_e[vi[u]], te);
        }
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
            for (int j = 0; j < V; ++j) dst[q * B + lane * V + j] = v[q * V + j];
    }
#pragma unroll
    for (int q = 0; q < Q * V; ++q) v[q] = 0.0;
    __syncwarp();
}

// Fixed-shape sum of the per-block partials [gridDim.x][P] (thread t handles value t % P, blocks
// strand, strand + S, ...; then the strands in order): every block computes the same bits for the
// same partials.  All kThreads threads of the CTA must call it.
__device__ __forceinline__ void sum_partials(const double* partials, int P, double* result) {
    __shared__ double s_tree[kThreads];
    const int tid = threadIdx.x;
    const int S = kThreads / P;              // strands per value
    const int pv = tid % P, strand = tid / P;
    double s = 0.0;
    if (strand < S) {
        // four independent loads in flight, added in the order of g (a missing block adds +0.0)
        for (unsigned int g = strand; g < gridDim.x; g += 4 * S) {
            double v[4];
#pragma unroll
            for (int j = 0; j < 4; ++j) {
                const unsigned int gg = g + j * S;
                v[j] = gg < gridDim.x ? __ldcg(&partials[(size_t)gg * P + pv]) : 0.0;
            }
#pragma unroll
            for (int j = 0; j < 4; ++j) s += v[j];
        }
    }
    s_tree[tid] = (strand < S) ? s : 0.0;
    __syncthreads();
    if (tid < P) {
        double tot = 0.0;
        for (int j = 0; j < S; ++j) tot += s_tree[j * P + tid];
        result[tid] = tot;
    }
    __syncthreads();
}

// CTA stage of the deterministic reduction: s_part[warp][P] -> partials[block][P]
__device__ __forceinline__ void block_partial(const double* s_part, int P, double* partials) {
    const int tid = threadIdx.x;
    __syncthreads();
    if (tid < P) {
        double s = 0.0;
#pragma unroll
        for (int w = 0; w < kWarps; ++w) s += s_part[w * P + tid];
        partials[(size_t)blockIdx.x * P + tid] = s;
    }
}

// Recurrence steps [a.m_begin, a.m_end), each x_m = 2 H~ x_{m-1} - x_{m-2} fused with what consumes it.
// Every warp issues its own TMA copies (lane 0) one or more tiles ahead.  Persistent CTAs: the tiles are
// cut into runs of a.run consecutive tiles; CTA c walks runs c, c + G, c + 2G, ...; inside a run warp w
// takes tiles w, w + kWarps, ...  A CTA therefore streams a contiguous band of rows and the grid
// sweeps the vector as a tight front, so gathers to nearby rows (the +-x, +-y, +-z neighbours of a
// lattice) are served by L1/L2.  All loop indices are kept incrementally (no divisions in the loop).
// Between the steps of a multi-step (cooperative) launch: per-block dot partials, a grid barrier, and
// block m % G sums the partials of step m in a fixed order while the others go on.
template <int B, int KT, int HOP, int MODE>
__global__ void __launch_bounds__(kThreads, min_blocks(B, MODE)) cheb_step_kernel(const Mat m, const RecArgs a) {
    using LS = LaneShape<B, KT, MODE>;
    constexpr int Q = ModeTraits<MODE>::Q;
    constexpr int V = LS::V, ROUNDS = LS::ROUNDS, U = LS::U, S = LS::S, TR = 32 * S;
    constexpr int RB = B * 16, QB = Q * B;
    constexpr bool DOTS = (MODE == kModeDoubling || MODE == kModeLeft);
    constexpr bool MSD = (MODE == kModeEvolveMsd);
    constexpr bool STENCIL = (HOP == kHopStencil);
    constexpr int kPair = MSD ? 2 : 1;
    __shared__ double s_part[DOTS ? kWarps * QB : 1];
    __shared__ int s_last;
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

    const int N = (int)m.N;
    const int n_tiles = ((int)m.n_slices + S - 1) / S;
    const int per = a.run / kWarps;
    const int n_runs = (n_tiles + a.run - 1) / a.run;
    const int G = gridDim.x;
    const int my_runs = (int)blockIdx.x < n_runs ? (n_runs - (int)blockIdx.x + G - 1) / G : 0;
    int n_my = 0;
    if (my_runs > 0) {
        const int last = blockIdx.x + (my_runs - 1) * G;
        const int rem = n_tiles - last * a.run;          // tiles in my last run (may be partial)
        const int in_last = rem >= a.run ? per : (warp < rem ? (rem - warp + kWarps - 1) / kWarps : 0);
        n_my = (my_runs - 1) * per + in_last;
    }
    const uint64_t policy = policy_evict_first();        // in every lane: the operands of the TMA issues stay warp-uniform
    if (lane == 0) {
        for (int s = 0; s < stages; ++s) mbar_init(&bars[s], 1);
        fence_mbar_init();
    }
    __syncwarp();

    const int jump = G * a.run - (per - 1) * kWarps;     // last tile of a run -> first tile of my next run
    // the stage ring and its mbarrier phases run on across the steps of the launch
    int p_st = 0, c_st = 0;
    uint32_t c_ph = 0;
    unsigned int epoch = 0;                               // grid barriers passed

    // operands of step mm (CTA-uniform)
    auto make_ctx = [&](int mm) {
        StepCtx io;
        const int last_term = a.terms - 1;
        io.first = (mm == 1);
        const bool half = a.clenshaw ? (mm == last_term) : (mm == 1);
        io.scale = half ? m.inv_dE : 2.0 * m.inv_dE;
        const int s_in = (mm + 1) % 3, s_prev = mm % 3, s_out = (mm + 2) % 3;      // (m-2)%3, (m-3)%3, (m-1)%3
        io.in = (mm == 1) ? a.x0 : a.ring[s_in];
        io.tm_in = (mm == 1) ? a.tm_x0 : a.tm_ring[s_in];
        io.prev = (mm == 2) ? a.x0 : a.ring[s_prev];
        io.tm_prev = (mm == 2) ? a.tm_x0 : a.tm_ring[s_prev];
        io.out = a.ring[s_out];
        io.in_e = io.prev_e = nullptr;
        io.out_e = nullptr;
        io.tm_in_e = io.tm_prev_e = nullptr;
        if (MSD) {
            io.in_e = (mm == 1) ? a.e0 : a.ring_e[s_in];
            io.tm_in_e = (mm == 1) ? a.tm_e0 : a.tm_ring_e[s_in];
            io.prev_e = (mm == 2) ? a.e0 : a.ring_e[s_prev];
            io.tm_prev_e = (mm == 2) ? a.tm_e0 : a.tm_ring_e[s_prev];
            io.out_e = a.ring_e[s_out];
        }
        io.store = 1;
        if (mm == last_term) {
            io.store = a.store_last;
            if (a.last_out) {
                io.out = a.last_out;
                io.out_e = a.last_out_e;
            }
        }
        io.cr = io.ci = 0.0;
        if (MODE == kModeEvolve || MSD) {
            io.cr = a.coef[2 * (last_term - mm)];
            io.ci = a.coef[2 * (last_term - mm) + 1];
        }
        return io;
    };
    int pp[S];                                 // kHopStencil: patterns of the tile the producer cursor points at (lane 0, or all lanes: UP)
#pragma unroll
    for (int j = 0; j < S; ++j) pp[j] = 0;
    // the record image of a tile -> dst: one bulk copy, or (kHopStencil) per slice the on-site record from HBM
    // and the slice's pattern from the dictionary
    auto copy_records = [&](unsigned char* dst, long long off, uint32_t bytes, uint64_t* bar) {
        if (STENCIL) {
#pragma unroll
            for (int j = 0; j < S; ++j) {
                unsigned char* d = dst + j * (256 + 128 * KT);
                bulk_g2s(d, m.rec + off + 256 * j, 256u, bar, policy);
                bulk_g2s_nohint(d + 256, m.dict + (size_t)pp[j] * (KT * 32), (uint32_t)(128 * KT), bar);
            }
        } else {
            bulk_g2s(dst, m.rec + off, bytes, bar, policy);
        }
    };
    // lane 0 only: every stream of tile t_virtual (sweep order) of the step `io` -> one stage, one mbarrier
    auto issue = [&](const StepCtx& io, int reverse, int t_virtual, int st) {
        const int t = reverse ? n_tiles - 1 - t_virtual : t_virtual;
        GPUQT_CHECK(t >= 0 && t < n_tiles && st >= 0 && st < stages);
        const int s = t * S;                   // first slice of the tile
        long long off;
        uint32_t bytes;
        if (KT > 0) {
            bytes = (uint32_t)hop_stage_bytes(KT, HOP) * S;         // the record array is padded to whole tiles
            off = (long long)s * (long long)hop_record_bytes(KT, HOP);
        } else {
            off = m.slice_off[s];
            bytes = (uint32_t)(m.slice_off[s + 1] - off);
        }
        const int left = N - s * 32;
        const uint32_t vbytes = (uint32_t)((left < TR ? left : TR) * RB);
        // x_{m-1} rows include the halo rows and the all-zero row NV when they fall into this tile's window
        // (columns of the last owned rows / the constant-hopping padding entries point at them)
        const int left_in = (int)m.NV + 1 - s * 32;
        const uint32_t vbytes_in = (uint32_t)((left_in < TR ? left_in : TR) * RB);
        const bool with_prev = !io.first && !prev_direct(B, MODE);
        unsigned char* dst = wstage + st * stage_bytes;
        unsigned char* vdst = dst + a.rec_bytes;
        if (B >= 2) {
            // tensor copies: always the full 32-row box (rows past the end of the buffer are zero-filled)
            const uint32_t total = bytes + (uint32_t)(32 * RB) * kPair * (with_prev ? 2u : 1u);
            const int unit = s * (512 / kSwizzleLineBytes) * B;    // first line of the slice
            mbar_expect_tx(&bars[st], total);
            copy_records(dst, off, bytes, &bars[st]);
            tensor_g2s(vdst, io.tm_in, unit, &bars[st]);
            if (MSD) tensor_g2s(vdst + 512 * B, io.tm_in_e, unit, &bars[st]);
            if (with_prev) {
                tensor_g2s_hint(vdst + kPair * 512 * B, io.tm_prev, unit, &bars[st], policy);
                if (MSD) tensor_g2s_hint(vdst + 3 * 512 * B, io.tm_prev_e, unit, &bars[st], policy);
            }
        } else {
            const uint32_t total = bytes + vbytes_in * kPair + (with_prev ? vbytes * kPair : 0u);
            const size_t voff = (size_t)s * 32 * B;
            mbar_expect_tx(&bars[st], total);
            copy_records(dst, off, bytes, &bars[st]);
            bulk_g2s_nohint(vdst, io.in + voff, vbytes_in, &bars[st]);
            if (MSD) bulk_g2s_nohint(vdst + TR * RB, io.in_e + voff, vbytes_in, &bars[st]);
            if (with_prev) {
                bulk_g2s(vdst + kPair * TR * RB, io.prev + voff, vbytes, &bars[st], policy);
                if (MSD) bulk_g2s(vdst + 3 * TR * RB, io.prev_e + voff, vbytes, &bars[st], policy);
            }
        }
    };
    // Producer cursor: tile in sweep order, index inside the run.  UP (uniform producer): every lane keeps the cursor
    // and only the issue itself is lane 0's, so the operands of the TMA instructions are warp-uniform and the
    // compiler issues them from uniform registers (no per-lane loop with R2UR broadcasts around each; 2008 -> 1624
    // SASS instructions).  Measured on c4, same box: evolve_msd 199.6 -> 192.2 ms per 10 steps, but kpm_doubling
    // 158.5 -> 164.0 us per step (c2, c3, c5 unchanged) -- so it is taken for the (psi, chi) kernel only; elsewhere
    // lane 0 alone keeps the cursor.
    constexpr bool UP = MSD;
    int p_t = 0, p_k = 0;
    int p_reverse = 0;                         // sweep direction of the step being issued
    auto p_patterns = [&]() {                  // kHopStencil: pattern ids of the tile at the cursor, one tile ahead of their use
        if (STENCIL) {
            const int t = p_reverse ? n_tiles - 1 - p_t : p_t;
            if (t >= 0 && t < n_tiles) {
#pragma unroll
                for (int j = 0; j < S; ++j) pp[j] = __ldg(&m.pid[t * S + j]);
            }
        }
    };
    auto p_reset = [&](int reverse) {
        p_t = (int)blockIdx.x * a.run + warp;
        p_k = 0;
        p_reverse = reverse;
        p_patterns();
    };
    auto p_advance = [&]() {
        if (++p_k == per) {
            p_k = 0;
            p_t += jump;
        } else {
            p_t += kWarps;
        }
        if (++p_st == stages) p_st = 0;
        p_patterns();
    };

    for (int mm = a.m_begin; mm < a.m_end; ++mm) {
        const StepCtx io = make_ctx(mm);
        const int reverse = a.alternate ? ((a.sweep0 + (mm - a.m_begin)) & 1) : a.sweep0;
        int c_t = (int)blockIdx.x * a.run + warp, c_k = 0;      // consumer cursor
        int issued = 0;
        if (UP || lane == 0) {
            p_reset(reverse);
            for (; issued < stages - 1 && issued < n_my; ++issued) {
                if (!UP || lane == 0) issue(io, reverse, p_t, p_st);
                p_advance();
            }
        }
        for (int i = 0; i < n_my; ++i) {
            // the stage the producer cursor points at was consumed by the whole warp in the previous iteration
            if ((UP || lane == 0) && issued < n_my) {
                if (!UP || lane == 0) issue(io, reverse, p_t, p_st);
                p_advance();
                ++issued;
            }
            mbar_wait(&bars[c_st], c_ph);
            const unsigned char* stage = wstage + c_st * stage_bytes;
            const int tile = reverse ? n_tiles - 1 - c_t : c_t;
            GPUQT_CHECK(c_st >= 0 && c_st < stages && tile >= 0 && tile < n_tiles);
            int w = KT;
            if (KT == 0) w = record_width(m.slice_off[tile + 1] - m.slice_off[tile], hop_doubles(HOP));
            const int row0 = tile * TR;
            const int rows_valid = N - row0;          // >= TR except in the last tile
#pragma unroll 1
            for (int j = 0; j < ROUNDS; j += U) walk_rounds<B, KT, HOP, MODE>(m, a, io, stage, w, row0, rows_valid, j, lane, red);
            if (++c_k == per) { c_k = 0; c_t += jump; } else c_t += kWarps;
            if (++c_st == stages) { c_st = 0; c_ph ^= 1u; }
            __syncwarp();
        }

        // ---- end of the step: dots, and the barrier before the next one
        double* result = DOTS ? a.dots + (size_t)(mm - a.dot_m0) * QB : nullptr;
        if (!a.multi) {
            if (DOTS) {
                warp_flush<B, Q, V>(red, s_part + warp * QB, lane);
                block_partial(s_part, QB, a.partials);
                __threadfence();
                __syncthreads();
                if (tid == 0) {
                    const unsigned int t = atomicAdd(a.ticket, 1u);
                    s_last = (t == gridDim.x - 1);
                }
                __syncthreads();
                if (s_last) {                       // CTA-uniform
                    __threadfence();
                    sum_partials(a.partials, QB, result);
                    if (tid == 0) *a.ticket = 0u;
                }
            }
        } else {
            // per-block partials of step mm -> buffer mm % 3; block (mm - 1) % G sums the partials of step mm - 1
            // (complete since the previous barrier) between its arrival at this barrier and the barrier's completion,
            // where nobody waits for it; the last step's partials are summed after the last barrier.  Three buffers:
            // buffer (mm - 1) % 3 is written again at the end of step mm + 2, after a barrier the summing block has
            // arrived at only after its sum.
            double* part = a.partials + (size_t)(mm % 3) * G * QB;
            if (DOTS) {
                warp_flush<B, Q, V>(red, s_part + warp * QB, lane);
                block_partial(s_part, QB, part);
            }
            ++epoch;
            grid_arrive(a.barrier);
            if (DOTS && mm > a.m_begin && (int)blockIdx.x == (mm - 1) % G)
                sum_partials(a.partials + (size_t)((mm - 1) % 3) * G * QB, QB, result - QB);
            grid_wait(a.barrier, epoch * (unsigned int)G);
            if (DOTS && mm + 1 == a.m_end && (int)blockIdx.x == mm % G) sum_partials(part, QB, result);
        }
    }
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
    int N;
    bool pad16;                      // 0xffff deltas stand for the zero row
    int add;                         // kHopStencil: first row of the slice (col[] is relative to it), else 0
    __device__ __forceinline__ int col_at(int k, int r) const {
        if (d16) {
            const unsigned d = d16[k * 32 + r];
            return (pad16 && d == kPad16) ? N : col[k] + (int)d;
        }
        return col[k * 32 + r] + add;
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
    v.N = (int)m.NV;
    v.w = (hop_is_16(m.hop) || m.hop == kHopStencil) ? m.K : record_width(bytes, nd);   // these variants are always uniform
    v.pad16 = m.hop == kHopConst16P;
    v.add = 0;
    v.hre = reinterpret_cast<const double*>(m.rec + off);
    v.him = v.hre + (size_t)v.w * 32;
    v.on = v.hre + (size_t)v.w * 32 * nd;
    v.col = reinterpret_cast<const int*>(v.on + 32);
    if (m.hop == kHopStencil) {
        v.col = m.dict + (size_t)m.pid[slice] * (m.K * 32);
        v.add = (int)(slice * 32);
    }
    v.d16 = hop_is_16(m.hop) ? reinterpret_cast<const unsigned short*>(v.col + 8) : nullptr;
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
            GPUQT_CHECK((unsigned)c <= (unsigned)m.NV);
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

#ifndef GPUQT_STEP_TU   // the non-template kernels below belong to gpuqt.cu's translation unit only
// [batch][N] (host order) <-> [N][B] (device order).  old_of_new != nullptr: the device rows are a permutation of the
// caller's sites (brick order of a recognised cubic lattice): device row `row` is the caller's site old_of_new[row].
__global__ void to_device_layout(long long N, int B, const double2* __restrict__ src, double2* __restrict__ dst,
                                 const int* __restrict__ old_of_new) {
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= N * B) return;
    const long long row = i / B;
    const int b = (int)(i % B);
    const long long site = old_of_new ? old_of_new[row] : row;
    dst[i] = src[(size_t)b * N + site];
}
__global__ void from_device_layout(long long N, int B, const double2* __restrict__ src, double2* __restrict__ dst,
                                   const int* __restrict__ old_of_new) {
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= N * B) return;
    const long long row = i / B;
    const int b = (int)(i % B);
    const long long site = old_of_new ? old_of_new[row] : row;
    dst[(size_t)b * N + site] = src[i];
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

// Damping factors folded with the (2 - delta_n0) factor: gs[n] = g_n (2 - delta_n0).
//   kind 0  Jackson, Eq. 31:  g_n = (1 - n a) cos(pi n a) + a sin(pi n a) cot(pi a), a = 1 / (N_m + 1)
//   kind 1  Lorentz (Weisse et al., the paper's ref. [33]):  g_n = sinh(lambda (1 - n / N_m)) / sinh(lambda)
//   kind 2  none (Dirichlet):  g_n = 1
__global__ void damping_kernel(int kind, double lambda, int n_moments, double* __restrict__ gs) {
    const int n = blockIdx.x * blockDim.x + threadIdx.x;
    if (n >= n_moments) return;
    double g = 1.0;
    if (kind == 0) {
        const double alpha = 1.0 / (n_moments + 1.0);
        double s, c, s1, c1;
        sincospi(n * alpha, &s, &c);
        sincospi(alpha, &s1, &c1);
        g = (1.0 - n * alpha) * c + alpha * s * (c1 / s1);
    } else if (kind == 1) {
        g = sinh(lambda * (1.0 - (double)n / (double)n_moments)) / sinh(lambda);
    }
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

// Localization length (Eq. 12) from the propagating length of Eq. 11, the limit read as the last measured
// time [A27]: xi[j] = L[n_t-1][j] / (2 pi); growth[j] = relative change of L over the last step (the saturation check).
__global__ void localization_kernel(int n_t, int n_e, const double* __restrict__ length, double* __restrict__ xi,
                                    double* __restrict__ growth) {
    const int j = blockIdx.x * blockDim.x + threadIdx.x;
    if (j >= n_e) return;
    const double last = length[(size_t)(n_t - 1) * n_e + j];
    xi[j] = last / (2.0 * 3.14159265358979323846);
    if (growth) growth[j] = last == 0.0 ? 0.0 : n_t == 1 ? 1.0 : (last - length[(size_t)(n_t - 2) * n_e + j]) / last;
}

// Decode the packed records back to canonical padded row-major arrays in the CALLER's site numbering (bit-exact
// check).  new_of_old / old_of_new: the row permutation of a reordered lattice, or nullptr.
__global__ void decode_table(const Mat m, int32_t* __restrict__ col, double* __restrict__ re,
                             double* __restrict__ im, double* __restrict__ dx, const int* __restrict__ new_of_old,
                             const int* __restrict__ old_of_new) {
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= m.N * m.K) return;
    const long long site = i / m.K;                               // the caller's row
    const int k = (int)(i % m.K);
    const long long row = new_of_old ? new_of_old[site] : site;   // where it is stored
    const RecView rv = record_view(m, row >> 5);
    const int r = (int)(row & 31);
    int c = (int)row;
    double hr = 0.0, hi = 0.0, d = 0.0;
    if (k < rv.w) {
        c = rv.col_at(k, r);
        if (hop_is_const(m.hop)) {
            hr = c < m.NV ? m.hop_const : 0.0;
            c = c < m.NV ? c : (int)row;
        } else {
            hr = rv.hre[k * 32 + r];
        }
        if (m.cplx) hi = rv.him[k * 32 + r];
        d = min_image(m.x[c] - m.x[row], m.box);
    }
    if (col) col[i] = old_of_new ? old_of_new[c] : c;
    if (re) re[i] = hr;
    if (im) im[i] = hi;
    if (dx) dx[i] = d;
}

#endif  // GPUQT_STEP_TU

// ---------------------------------------------------------------------------------- small lattices
// Lattices whose matrix and four vector sets fit one SM's shared memory (config c1: 2304 orbitals) are
// launch-latency bound on the streaming kernels.  cheb_small_kernel runs a WHOLE recurrence in one
// launch of one CTA: matrix (decoded to plain arrays) and vectors live in shared memory, the terms are
// separated by __syncthreads(), the per-term dots are reduced in a fixed order (warp shuffle -> shared
// memory over warps) and written straight to dots[term].
//   MODE doubling : T_m from v0; dots {<T_m|T_m>, Re<T_m|T_{m-1}>, <T_{m-1}|T_{m-1}>} per term   (Eq. 28, 30)
//   MODE left     : T_n from v0; dots <aux|T_n> (Re, Im) per term                                  (Eq. 29)
//   MODE evolve   : out = sum_k c_k T_k(H~) aux by Clenshaw (v0 unused; coef[k] = c_k)             (Eq. 17)
//   MODE evolve_msd: (out, out_e) = the same for the (psi, chi) pair with the block operator
//                   [[H~, 0], [[X,H~], H~]] (Eq. 18, 22, 24), see cheb_small_msd_kernel below
constexpr int kSmallThreads = 1024;

struct SmallArgs {
    const double2* v0;      // doubling / left: T_0
    const double2* aux;     // left: phi_L; evolve: the vector being evolved (psi)
    const double2* aux_e;   // evolve_msd: chi
    double2* out;           // evolve: result
    double2* out_e;         // evolve_msd: the new chi
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

// The (psi, chi) time step of a small lattice in one launch of one CTA (PAPER.md:156 Eq. 18, :170 Eq. 22,
// :176 Eq. 24; composition [A3]): Clenshaw recurrence of the pair
//     b_k = c_k psi + 2 H~ b_{k+1} - b_{k+2}
//     f_k = c_k chi + 2 H~ f_{k+1} - f_{k+2} + 2 [X,H~] b_{k+1},     [X,H~]_mn = (X_m - X_n) H_mn / dE
// with b, f in shared memory.  x_m only needs x_{m-2} at its OWN element, so it overwrites it: two ring
// slots per chain (4 N B double2 in all, as in cheb_small_kernel) and one __syncthreads() per term.  psi and
// chi are read from global memory each term (L1/L2 hits).
template <int B>
__global__ void __launch_bounds__(kSmallThreads, 1) cheb_small_msd_kernel(const Mat m, const SmallArgs a) {
    extern __shared__ __align__(16) unsigned char sm_raw[];
    const int tid = threadIdx.x;
    const int N = (int)m.N, K = m.K, NB = N * B;
    const int nd = hop_doubles(m.hop);
    double2* va = reinterpret_cast<double2*>(sm_raw);                   // b chain: 2 slots
    double2* ve = va + 2 * (size_t)NB;                                  // f chain: 2 slots
    double* on = reinterpret_cast<double*>(ve + 2 * (size_t)NB);
    double* xs = on + N;
    double* hre = xs + N;                                               // [K][N] if nd >= 1
    double* him = hre + (nd >= 1 ? (size_t)K * N : 0);                  // [K][N] if nd == 2
    int* col = reinterpret_cast<int*>(him + (nd == 2 ? (size_t)K * N : 0));   // [K][N]; -1 = no entry
    for (int row = tid; row < N; row += kSmallThreads) {
        const RecView rv = record_view(m, row >> 5);
        const int r = row & 31;
        on[row] = rv.on[r];
        xs[row] = m.x[row];
        for (int k = 0; k < K; ++k) {
            int c = -1;
            double hr = 0.0, hi = 0.0;
            if (k < rv.w) {
                c = rv.col_at(k, r);
                if (hop_is_const(m.hop)) {
                    hr = m.hop_const;
                    if (c >= N) c = -1;                                 // padding entry (the zero row)
                } else {
                    hr = rv.hre[k * 32 + r];
                    if (nd == 2) hi = rv.him[k * 32 + r];
                    if (hr == 0.0 && hi == 0.0) c = -1;                 // padding entry (own row, weight 0)
                }
            }
            col[k * N + row] = c;
            if (nd >= 1) hre[k * N + row] = hr;
            if (nd == 2) him[k * N + row] = hi;
        }
    }
    const double2 c_last = a.coef[a.n_terms - 1];
    for (int i = tid; i < NB; i += kSmallThreads) {
        const double2 p = a.aux[i], q = a.aux_e[i];
        va[i] = make_double2(c_last.x * p.x - c_last.y * p.y, c_last.x * p.y + c_last.y * p.x);
        ve[i] = make_double2(c_last.x * q.x - c_last.y * q.y, c_last.x * q.y + c_last.y * q.x);
    }
    __syncthreads();
    if (a.n_terms == 1) {
        for (int i = tid; i < NB; i += kSmallThreads) {
            a.out[i] = va[i];
            a.out_e[i] = ve[i];
        }
        return;
    }
    int cur = 0;                     // slot of x_{m-1}; x_{m-2} sits in the other slot and is overwritten by x_m
    for (int t = 1; t < a.n_terms; ++t) {
        const double2* in = va + (size_t)cur * NB;
        const double2* in_e = ve + (size_t)cur * NB;
        double2* out = va + (size_t)(cur ^ 1) * NB;
        double2* out_e = ve + (size_t)(cur ^ 1) * NB;
        const bool first = (t == 1), half = (t == a.n_terms - 1);
        const double scale = half ? m.inv_dE : 2.0 * m.inv_dE;
        const double2 ck = a.coef[a.n_terms - 1 - t];
        for (int i = tid; i < NB; i += kSmallThreads) {
            const int row = i / B, b = i % B;
            const double2 self = in[i], self_e = in_e[i];
            const double xm = xs[row];
            double sr = on[row] * self.x, si = on[row] * self.y;
            double er = on[row] * self_e.x, ei = on[row] * self_e.y;
            for (int k = 0; k < K; ++k) {
                const int c = col[k * N + row];
                if (c < 0) continue;
                const double2 v = in[c * B + b], w = in_e[c * B + b];
                const double hr = hop_is_const(m.hop) ? m.hop_const : hre[k * N + row];
                const double ndx = -min_image(xs[c] - xm, m.box);       // [X,H]_mn = (X_m - X_n) H_mn
                sr = fma(hr, v.x, sr);
                si = fma(hr, v.y, si);
                er = fma(hr, w.x, er);
                ei = fma(hr, w.y, ei);
                er = fma(ndx * hr, v.x, er);
                ei = fma(ndx * hr, v.y, ei);
                if (nd == 2) {
                    const double hi = him[k * N + row];
                    sr = fma(-hi, v.y, sr);
                    si = fma(hi, v.x, si);
                    er = fma(-hi, w.y, er);
                    ei = fma(hi, w.x, ei);
                    er = fma(-ndx * hi, v.y, er);
                    ei = fma(ndx * hi, v.x, ei);
                }
            }
            double2 ta = make_double2(scale * sr, scale * si), te = make_double2(scale * er, scale * ei);
            if (!first) {
                const double2 p = out[i], q = out_e[i];                 // x_{m-2}, own element only
                ta.x -= p.x; ta.y -= p.y;
                te.x -= q.x; te.y -= q.y;
            }
            const double2 s = a.aux[i], se = a.aux_e[i];
            ta.x += ck.x * s.x - ck.y * s.y;
            ta.y += ck.x * s.y + ck.y * s.x;
            te.x += ck.x * se.x - ck.y * se.y;
            te.y += ck.x * se.y + ck.y * se.x;
            if (half) {
                a.out[i] = ta;
                a.out_e[i] = te;
            } else {
                out[i] = ta;
                out_e[i] = te;
            }
        }
        __syncthreads();
        cur ^= 1;
    }
}

}  // namespace gpuqt
