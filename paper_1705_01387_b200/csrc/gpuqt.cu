// C-ABI of the B200-native GPUQT hot path (include/gpuqt.h): host logic + kernel launches.
#include <cuda.h>
#include <cuda_runtime.h>

#include <cstdio>
#include <cstdlib>
#include <string>
#include <vector>

#include "../../include/gpuqt.h"
#include "host_util.h"
#include "kernels.cuh"

using namespace gpuqt;

namespace gpuqt {
void* pair_kernel_fn(int mode, int B, int kt, int hop);   // pair_kernels.cu
}

namespace {

constexpr int kMaxGrid = 4096;
constexpr int kPartialDoubles = 64;   // n_steps*Q*B <= 48
constexpr int kRing = 4;              // recurrence ring: a fused pair reads two slots and writes two

struct PendingStat {
    int cls;
    cudaEvent_t start, stop;
    int64_t launches, steps;
};

}  // namespace

struct gpuqt_handle {
    int64_t N = 0;
    int32_t K = 0, B = 0;
    int modes = 0, cplx = 0, kt = 0, hop = 0;
    int max_blocks_per_sm = 0;          // GPUQT_BLOCKS_PER_SM (tuning override), 0 = occupancy limit
    int run = kWarps;                   // GPUQT_RUN: consecutive slices per CTA run (multiple of kWarps)
    int alternate = 1;                  // GPUQT_ALTERNATE: sweep direction alternates between launches
    int rec_bytes = 0;                  // bytes of one (widest) slice record
    int want_stages = 2;                // requested pipeline depth per warp
    // per launch configuration [mode + 4 * pair]: stages, bytes per stage, dynamic smem
    int mode_stages[8] = {0};
    int mode_stage_bytes[8] = {0};
    size_t mode_smem[8] = {0};
    std::vector<void*> smem_set;        // kernels whose dynamic-smem attribute has been raised
    double dE = 0, box = 0, volume = 0;
    cudaStream_t stream = nullptr;
    int n_sm = 0;
    Mat mat{};
    size_t vec_elems = 0;   // N * B double2
    // vectors (device, inside the caller's workspace)
    double2 *psi = nullptr, *chi = nullptr, *va = nullptr, *vb = nullptr, *phiL = nullptr;
    double2 *out0 = nullptr, *out1 = nullptr, *ring[kRing] = {nullptr, nullptr, nullptr, nullptr},
            *ringe[kRing] = {nullptr, nullptr, nullptr, nullptr};
    // fused pairs of steps: dependency structure of the table and the cached work lists
    int small = 1;                      // GPUQT_SMALL: one-CTA whole-recurrence kernel when everything fits one SM
    int fuse = 1, lag = 2;              // GPUQT_FUSE, GPUQT_LAG (slack of the second step in half rounds)
    std::vector<int> nbr_ptr, nbr_slices;
    struct DevSchedule {
        int G, reverse, n_items, n_runs;
        int2* items;
        int *dep_ptr, *dep_list;
        unsigned int* run_done;
    };
    std::vector<DevSchedule> schedules;
    // library-owned scratch for the small transform / table-decode calls: grown on demand, kept
    // (stream-ordered pool allocations can trim at every synchronisation and stall the step)
    char* scratch = nullptr;
    size_t scratch_bytes = 0;
    // B >= 2: one TMA tensor map (128-byte swizzle) per vector buffer, in device memory
    std::vector<const double2*> map_bufs;
    CUtensorMap* d_maps = nullptr;
    double *partials = nullptr, *dots = nullptr, *moments = nullptr;
    unsigned int* ticket = nullptr;
    int grid[8] = {0};                  // [mode + 4 * pair]
    int grid_aux = 0;
    int sweep = 0;                      // direction of the next step launch (reset per building block)
    bool state_set = false;
    std::string err;
    double stat_ms[GPUQT_KERNEL_CLASSES] = {0};
    int64_t stat_launches[GPUQT_KERNEL_CLASSES] = {0};
    int64_t stat_steps[GPUQT_KERNEL_CLASSES] = {0};     // recurrence steps (a fused launch does two)
    std::vector<PendingStat> pending;
    std::vector<cudaEvent_t> free_events;
};

namespace {

int fail(gpuqt_handle* h, int code, const std::string& msg) {
    if (h) h->err = msg;
    return code;
}
int cuda_fail(gpuqt_handle* h, cudaError_t e, const char* what) {
    return fail(h, GPUQT_ERR_CUDA, std::string(what) + ": " + cudaGetErrorString(e));
}
#define CU(call)                                                   \
    do {                                                           \
        cudaError_t e_ = (call);                                   \
        if (e_ != cudaSuccess) return cuda_fail(h, e_, #call);     \
    } while (0)

size_t align_up(size_t v, size_t a = 256) { return (v + a - 1) / a * a; }

int n_vectors(int modes) {
    int n = 2 + kRing;                              // psi, out0, ring
    if (modes & GPUQT_MODE_MSD) n += 2 + kRing;     // chi, out1, ringe
    if (modes & GPUQT_MODE_VAC) n += 3;             // a, b, phi_L
    return n;
}

struct Layout {
    size_t rec, slice_off, x, vectors, partials, dots, moments, ticket, total;
};

Layout make_layout(int64_t N, int32_t B, int modes, size_t rec_bytes) {
    Layout L{};
    size_t off = 0;
    auto take = [&](size_t bytes) {
        size_t o = off;
        off = align_up(off + bytes);
        return o;
    };
    const size_t n_slices = (size_t)((N + 31) / 32);
    L.rec = take(rec_bytes);
    L.slice_off = take((n_slices + 1) * sizeof(long long));
    L.x = take((size_t)(N + 1) * sizeof(double));
    // every vector buffer has N + 1 rows; row N stays zero for ever (nothing writes it)
    L.vectors = take((size_t)n_vectors(modes) * align_up((size_t)(N + 1) * B * sizeof(double2)));
    L.partials = take((size_t)kMaxGrid * kPartialDoubles * sizeof(double));
    L.dots = take((size_t)GPUQT_MAX_MOMENTS * 3 * 8 * sizeof(double));
    L.moments = take((size_t)GPUQT_MAX_MOMENTS * 8 * sizeof(double));
    L.ticket = take(256);
    L.total = off;
    return L;
}

// shared memory of one step-kernel CTA: mbarriers, then kWarps * stages record buffers
size_t step_smem_bytes(int stages, int stage_bytes, bool pair = false) {
    return 128 * (((pair ? 2 : 1) * (size_t)kWarps * kMaxStages * 8 + 127) / 128) + (size_t)kWarps * stages * stage_bytes;
}
constexpr size_t kSmemBudget = 200 * 1024;   // per CTA; leaves room for the static reduction buffers
constexpr size_t kSmemPerSm = 227 * 1024;

int env_int(const char* name, int dflt) {
    const char* v = getenv(name);
    return (v && *v) ? atoi(v) : dflt;
}

bool batch_ok(int B) { return B == 1 || B == 2 || B == 4 || B == 8; }

// ---------------------------------------------------------------- kernel dispatch
template <int MODE, int BB, int KK>
void* step_fn(int hop) {
    if (KK > 0 && hop == kHopConst16)      // 16-bit columns exist for the unrolled uniform tables only
        return (void*)cheb_step_kernel<BB, (KK > 0 ? KK : 3), kHopConst16, MODE>;
    return hop == kHopComplex ? (void*)cheb_step_kernel<BB, KK, kHopComplex, MODE>
           : hop == kHopConst ? (void*)cheb_step_kernel<BB, KK, kHopConst, MODE>
                              : (void*)cheb_step_kernel<BB, KK, kHopReal, MODE>;
}
template <int MODE, int BB>
void* step_fn_k(int kt, int hop) {
    switch (kt) {
    case 3: return step_fn<MODE, BB, 3>(hop);
    case 4: return step_fn<MODE, BB, 4>(hop);
    case 6: return step_fn<MODE, BB, 6>(hop);
    default: return step_fn<MODE, BB, 0>(hop);
    }
}
template <int MODE>
void* step_fn_b(int B, int kt, int hop) {
    switch (B) {
    case 1: return step_fn_k<MODE, 1>(kt, hop);
    case 2: return step_fn_k<MODE, 2>(kt, hop);
    case 4: return step_fn_k<MODE, 4>(kt, hop);
    default: return step_fn_k<MODE, 8>(kt, hop);
    }
}
void* step_kernel(const gpuqt_handle* h, int mode, bool pair) {
    if (pair) return pair_kernel_fn(mode, h->B, h->kt, h->hop);     // pair_kernels.cu
    switch (mode) {
    case kModeDoubling: return step_fn_b<kModeDoubling>(h->B, h->kt, h->hop);
    case kModeLeft: return step_fn_b<kModeLeft>(h->B, h->kt, h->hop);
    case kModeEvolve: return step_fn_b<kModeEvolve>(h->B, h->kt, h->hop);
    default: return step_fn_b<kModeEvolveMsd>(h->B, h->kt, h->hop);
    }
}

void* velocity_fn(const gpuqt_handle* h) {
    switch (h->B) {
    case 1: return (void*)velocity_kernel<1>;
    case 2: return (void*)velocity_kernel<2>;
    case 4: return (void*)velocity_kernel<4>;
    default: return (void*)velocity_kernel<8>;
    }
}
void* dot_fn(int B) {
    switch (B) {
    case 1: return (void*)dot_kernel<1>;
    case 2: return (void*)dot_kernel<2>;
    case 4: return (void*)dot_kernel<4>;
    default: return (void*)dot_kernel<8>;
    }
}

int grid_for(gpuqt_handle* h, void* fn, size_t smem, long long work_items, int threads = kThreads) {
    int per_sm = 0;
    if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, fn, threads, smem) != cudaSuccess || per_sm < 1)
        per_sm = 1;
    if (h->max_blocks_per_sm > 0 && per_sm > h->max_blocks_per_sm) per_sm = h->max_blocks_per_sm;
    long long g = (long long)per_sm * h->n_sm;
    if (g > work_items) g = work_items;
    if (g > kMaxGrid) g = kMaxGrid;
    if (g < 1) g = 1;
    return (int)g;
}

// bytes of one stage of a step kernel: the record plus the staged own rows of T_{m-1}, T_{m-2}
// (and e_{m-1}, e_{m-2} for the (a, e) pair)
int mode_stage_bytes_for(const gpuqt_handle* h, int mode, bool pair = false) {
    int streams = (mode == kModeEvolveMsd) ? 4 : 2;
    if (h->B >= 8) streams /= 2;   // PrevDirect<8>: T_{m-2} rows are not staged
    return h->rec_bytes + streams * 32 * h->B * (int)sizeof(double2) + (pair ? kHdrBytes : 0);
}

cudaError_t launch_step(gpuqt_handle* h, int mode, StepArgs& a) {
    const bool pair = a.n_steps == 2;
    const int cfg = mode + (pair ? 4 : 0);
    const int threads = pair ? kThreads + 32 : kThreads;     // the pair kernel has a producer warp
    void* fn = step_kernel(h, mode, pair);
    if (!h->grid[cfg]) {
        const int sb = mode_stage_bytes_for(h, mode, pair);
        int stages = h->want_stages;
        while (stages > 1 && step_smem_bytes(stages, sb, pair) > kSmemBudget) --stages;
        // prefer two resident CTAs per SM over a deeper pipeline
        while (stages > 2 && 2 * (step_smem_bytes(stages, sb, pair) + 4096) > kSmemPerSm) --stages;
        h->mode_stages[cfg] = stages;
        h->mode_stage_bytes[cfg] = sb;
        h->mode_smem[cfg] = step_smem_bytes(stages, sb, pair);
        if (h->mode_smem[cfg] > 48 * 1024) {
            cudaError_t e = cudaFuncSetAttribute(fn, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)h->mode_smem[cfg]);
            if (e != cudaSuccess) return e;
        }
        h->grid[cfg] = grid_for(h, fn, h->mode_smem[cfg], (h->mat.n_slices + h->run - 1) / h->run, threads);
    }
    a.sched = nullptr;
    a.n_items = 0;
    a.run_done = nullptr;
    a.dep_ptr = nullptr;
    a.dep_list = nullptr;
    if (a.n_steps == 2) {
        const int reverse = h->alternate ? (h->sweep & 1) : 0;
        const gpuqt_handle::DevSchedule* ds = nullptr;
        for (const auto& d : h->schedules)
            if (d.G == h->grid[cfg] && d.reverse == reverse) ds = &d;
        if (!ds) {
            FusedSchedule fs;
            build_fused_schedule((int)h->mat.n_slices, h->run, h->grid[cfg], reverse, std::max(1, h->lag * h->grid[cfg] / 2),
                                 kNoRun, h->nbr_ptr, h->nbr_slices, fs);
            gpuqt_handle::DevSchedule d{};
            d.G = h->grid[cfg];
            d.reverse = reverse;
            d.n_items = (int)(fs.items.size() / 2);
            d.n_runs = (int)fs.dep_ptr.size() - 1;
            auto up = [&](void** dst, const std::vector<int>& v) {
                cudaError_t e = cudaMalloc(dst, std::max<size_t>(v.size(), 1) * sizeof(int));
                if (e == cudaSuccess && !v.empty()) e = cudaMemcpy(*dst, v.data(), v.size() * sizeof(int), cudaMemcpyHostToDevice);
                return e;
            };
            cudaError_t e = up((void**)&d.items, fs.items);
            if (e == cudaSuccess) e = up((void**)&d.dep_ptr, fs.dep_ptr);
            if (e == cudaSuccess) e = up((void**)&d.dep_list, fs.dep_list);
            if (e == cudaSuccess) e = cudaMalloc((void**)&d.run_done, (size_t)d.n_runs * sizeof(unsigned int));
            if (e != cudaSuccess) return e;
            h->schedules.push_back(d);
            ds = &h->schedules.back();
        }
        cudaError_t e = cudaMemsetAsync(ds->run_done, 0, (size_t)ds->n_runs * sizeof(unsigned int), h->stream);
        if (e != cudaSuccess) return e;
        a.sched = ds->items;
        a.n_items = ds->n_items;
        a.run_done = ds->run_done;
        a.dep_ptr = ds->dep_ptr;
        a.dep_list = ds->dep_list;
    }
    a.stages = h->mode_stages[cfg];
    a.stage_bytes = h->mode_stage_bytes[cfg];
    a.rec_bytes = h->rec_bytes;
    a.partials = h->partials;
    a.ticket = h->ticket;
    a.reverse = h->alternate ? (h->sweep & 1) : 0;
    a.run = h->run;
    h->sweep ^= 1;
    void* args[] = {(void*)&h->mat, (void*)&a};
    return cudaLaunchKernel(fn, dim3(h->grid[cfg]), dim3(threads), args, h->mode_smem[cfg], h->stream);
}

cudaError_t launch_velocity(gpuqt_handle* h, const double2* in, double2* out) {
    void* fn = velocity_fn(h);
    if (!h->grid_aux) h->grid_aux = grid_for(h, fn, 0, (h->N * h->B + kThreads - 1) / kThreads);
    void* args[] = {(void*)&h->mat, (void*)&in, (void*)&out};
    return cudaLaunchKernel(fn, dim3(h->grid_aux), dim3(kThreads), args, 0, h->stream);
}

cudaError_t launch_dot(gpuqt_handle* h, const double2* l, const double2* r, double* result) {
    void* fn = dot_fn(h->B);
    if (!h->grid_aux) h->grid_aux = grid_for(h, velocity_fn(h), 0, (h->N * h->B + kThreads - 1) / kThreads);
    long long N = h->N;
    void* args[] = {(void*)&N, (void*)&l, (void*)&r, (void*)&h->partials, (void*)&h->ticket, (void*)&result};
    return cudaLaunchKernel(fn, dim3(h->grid_aux), dim3(kThreads), args, 0, h->stream);
}

// device address of the tensor map of a vector buffer (nullptr at B = 1, where plain bulk copies are used)
const void* tensor_map_of(const gpuqt_handle* h, const double2* buf) {
    if (!h->d_maps || !buf) return nullptr;
    for (size_t i = 0; i < h->map_bufs.size(); ++i)
        if (h->map_bufs[i] == buf) return h->d_maps + i;
    return nullptr;
}

// Tensor maps over the vector buffers: a buffer is seen as 128-byte lines (8 complex numbers; the last
// line may reach into the buffer's zeroed alignment padding); one box = the 4 * B lines of one slice,
// written to shared memory with the 128-byte swizzle; lines past the end are zero-filled.
int build_tensor_maps(gpuqt_handle* h) {
    if (h->B < 2) return GPUQT_OK;
    typedef CUresult (*EncodeFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*, const cuuint64_t*,
                                 const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle,
                                 CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
    void* fp = nullptr;
    cudaDriverEntryPointQueryResult qres;
    CU(cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fp, cudaEnableDefault, &qres));
    if (!fp || qres != cudaDriverEntryPointSuccess) return fail(h, GPUQT_ERR_CUDA, "cuTensorMapEncodeTiled is not available");
    EncodeFn encode = (EncodeFn)fp;
    std::vector<CUtensorMap> maps(h->map_bufs.size());
    for (size_t i = 0; i < maps.size(); ++i) {
        const cuuint64_t dims[2] = {16, ((cuuint64_t)(h->N + 1) * (cuuint64_t)h->B * 16 + 127) / 128};
        const cuuint64_t strides[1] = {128};
        const cuuint32_t box[2] = {16, (cuuint32_t)(4 * h->B)};
        const cuuint32_t estr[2] = {1, 1};
        CUresult r = encode(&maps[i], CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 2, (void*)h->map_bufs[i], dims, strides, box, estr,
                            CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_NONE,
                            CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
        if (r != CUDA_SUCCESS) return fail(h, GPUQT_ERR_CUDA, "cuTensorMapEncodeTiled failed with code " + std::to_string((int)r));
    }
    CU(cudaMalloc((void**)&h->d_maps, maps.size() * sizeof(CUtensorMap)));
    CU(cudaMemcpy(h->d_maps, maps.data(), maps.size() * sizeof(CUtensorMap), cudaMemcpyHostToDevice));
    return GPUQT_OK;
}

cudaError_t ensure_scratch(gpuqt_handle* h, size_t bytes) {
    if (bytes <= h->scratch_bytes) return cudaSuccess;
    cudaError_t e = cudaStreamSynchronize(h->stream);
    if (e != cudaSuccess) return e;
    if (h->scratch) cudaFree(h->scratch);
    h->scratch = nullptr;
    h->scratch_bytes = 0;
    const size_t want = bytes + bytes / 2;
    e = cudaMalloc((void**)&h->scratch, want);
    if (e == cudaSuccess) h->scratch_bytes = want;
    return e;
}

// ---------------------------------------------------------------- timing statistics
cudaEvent_t get_event(gpuqt_handle* h) {
    if (!h->free_events.empty()) {
        cudaEvent_t e = h->free_events.back();
        h->free_events.pop_back();
        return e;
    }
    cudaEvent_t e = nullptr;
    cudaEventCreate(&e);
    return e;
}
struct StatScope {
    gpuqt_handle* h;
    PendingStat p;
    StatScope(gpuqt_handle* hh, int cls) : h(hh) {
        p.cls = cls;
        p.launches = 0;
        p.steps = 0;
        p.start = get_event(h);
        p.stop = get_event(h);
        cudaEventRecord(p.start, h->stream);
    }
    void count(int64_t n = 1, int64_t steps = 1) {
        p.launches += n;
        p.steps += steps;
    }
    ~StatScope() {
        cudaEventRecord(p.stop, h->stream);
        h->pending.push_back(p);
    }
};
void flush_stats(gpuqt_handle* h) {
    for (auto& p : h->pending) {
        float ms = 0.f;
        if (cudaEventSynchronize(p.stop) == cudaSuccess && cudaEventElapsedTime(&ms, p.start, p.stop) == cudaSuccess) {
            h->stat_ms[p.cls] += ms;
            h->stat_launches[p.cls] += p.launches;
            h->stat_steps[p.cls] += p.steps;
        }
        h->free_events.push_back(p.start);
        h->free_events.push_back(p.stop);
    }
    h->pending.clear();
}

// ---------------------------------------------------------------- building blocks
// ---- small lattices: the whole recurrence in one launch of one CTA (kernels.cuh, cheb_small_kernel)
size_t small_smem_bytes(const gpuqt_handle* h) {
    const size_t NB = (size_t)h->N * h->B, KN = (size_t)h->K * h->N;
    return 4 * NB * sizeof(double2) + (size_t)h->N * 8 + KN * 8 * (size_t)hop_doubles(h->hop) + KN * 4 + 16;
}
bool small_ok(const gpuqt_handle* h) { return h->small && small_smem_bytes(h) <= 210 * 1024; }

template <int MODE>
void* small_fn(int B) {
    switch (B) {
    case 1: return (void*)cheb_small_kernel<1, MODE>;
    case 2: return (void*)cheb_small_kernel<2, MODE>;
    case 4: return (void*)cheb_small_kernel<4, MODE>;
    default: return (void*)cheb_small_kernel<8, MODE>;
    }
}
cudaError_t launch_small(gpuqt_handle* h, int mode, SmallArgs& a) {
    void* fn = mode == kModeDoubling ? small_fn<kModeDoubling>(h->B)
               : mode == kModeLeft   ? small_fn<kModeLeft>(h->B)
                                     : small_fn<kModeEvolve>(h->B);
    const size_t smem = small_smem_bytes(h);
    if (std::find(h->smem_set.begin(), h->smem_set.end(), fn) == h->smem_set.end()) {
        cudaError_t e = cudaFuncSetAttribute(fn, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e != cudaSuccess) return e;
        h->smem_set.push_back(fn);
    }
    void* args[] = {(void*)&h->mat, (void*)&a};
    return cudaLaunchKernel(fn, dim3(1), dim3(kSmallThreads), args, smem, h->stream);
}

// Driver of one three-term recurrence: launches m = 1 .. terms-1, each x_m = 2 H~ x_{m-1} - x_{m-2} (+ ...)
// (and the e-chain of the MSD pair).  Launch 1 has no x_{-1}.  Forward recurrences (moments) apply
// factor 1 in launch 1 (T_1 = H~ T_0); Clenshaw recurrences (evolution) apply factor 1 in the LAST
// launch.  In between two consecutive terms share one launch when fusing is on (kernels.cuh,
// cheb_pair_kernel).  fill(io, m) sets the per-term fields (coefficient, dot destination, store flag,
// output override).
template <class Fill>
int run_recurrence(gpuqt_handle* h, int mode, int cls, int terms, const double2* t0, const double2* e0,
                   const StepArgs& base, bool clenshaw, Fill fill) {
    StatScope s(h, cls);
    const double2 *tm1 = t0, *tm2 = nullptr, *em1 = e0, *em2 = nullptr;
    int slot = 0, m = 1;
    while (m < terms) {
        StepArgs a = base;
        a.first = (m == 1);
        a.half = clenshaw ? (m == terms - 1) : (m == 1);
        a.n_steps = (h->fuse && m >= 2 && m + 1 + (clenshaw ? 1 : 0) < terms) ? 2 : 1;
        for (int k = 0; k < a.n_steps; ++k) {
            StepIO& io = a.io[k];
            double2* tnew = h->ring[slot];
            io.in = tm1; io.prev = tm2; io.out = tnew;
            if (e0) {
                io.in_e = em1; io.prev_e = em2; io.out_e = h->ringe[slot];
            }
            slot = (slot + 1) % kRing;
            io.store = 1;
            io.tm_in = tensor_map_of(h, io.in);
            io.tm_prev = tensor_map_of(h, io.prev);
            io.tm_in_e = tensor_map_of(h, io.in_e);
            io.tm_prev_e = tensor_map_of(h, io.prev_e);
            fill(io, m + k);
            tm2 = tm1; tm1 = io.out;
            if (e0) {
                em2 = em1; em1 = io.out_e;
            }
        }
        CU(launch_step(h, mode, a));
        s.count(1, a.n_steps);
        m += a.n_steps;
    }
    return GPUQT_OK;
}

cudaError_t launch_scale(gpuqt_handle* h, double cr, double ci, const double2* in, double2* out) {
    const long long n = (long long)h->vec_elems;
    scale_vec<<<(int)((n + 255) / 256), 256, 0, h->stream>>>(n, cr, ci, in, out);
    return cudaGetLastError();
}

// out <- sum_{k<order} c_k T_k(H~) in  (Eq. 17, 21, 23) by Clenshaw's backward recurrence
//   b_{order-1} = c_{order-1} in,  b_k = c_k in + 2 H~ b_{k+1} - b_{k+2},  out = c_0 in + H~ b_1 - b_2:
// the same order - 1 SpMV launches as the forward form, but no accumulator is read-modified-written
// (64 instead of 80 bytes per row and term).  The same for the (psi, chi) pair with the block operator
// [[H~, 0], [[X,H~], H~]] (a_m = T_m psi, e_m = T_m chi + [X,T_m] psi, Eq. 18, 22, 24).
// `in` is left untouched; `out` must differ from in and from the ring buffers.
int evolve_clenshaw(gpuqt_handle* h, int mode, int cls, const double2* in, const double2* in_e, double2* out,
                    double2* out_e, const std::vector<double>& cr, const std::vector<double>& ci, int order) {
    if (!in_e && small_ok(h) && (size_t)order * 2 <= (size_t)GPUQT_MAX_MOMENTS * 8) {
        std::vector<double> c((size_t)order * 2);
        for (int k = 0; k < order; ++k) {
            c[(size_t)2 * k] = cr[(size_t)k];
            c[(size_t)2 * k + 1] = ci[(size_t)k];
        }
        CU(cudaMemcpyAsync(h->moments, c.data(), c.size() * sizeof(double), cudaMemcpyHostToDevice, h->stream));
        SmallArgs a{};
        a.aux = in; a.out = out; a.coef = (const double2*)h->moments; a.n_terms = order;
        StatScope s(h, cls);
        CU(launch_small(h, kModeEvolve, a));
        s.count(1, order > 1 ? order - 1 : 0);
        return GPUQT_OK;
    }
    if (order == 1) {
        StatScope s(h, cls);
        CU(launch_scale(h, cr[0], ci[0], in, out));
        if (in_e) CU(launch_scale(h, cr[0], ci[0], in_e, out_e));
        s.count(in_e ? 2 : 1, 0);
        return GPUQT_OK;
    }
    // b_{order-1} lives in the last ring slot: the recurrence writes slots 0, 1, 2, ... and needs it
    // only in its first two launches
    double2* b0 = h->ring[kRing - 1];
    double2* b0_e = in_e ? h->ringe[kRing - 1] : nullptr;
    {
        StatScope s(h, cls);       // counted as launches of the class, not as recurrence steps
        CU(launch_scale(h, cr[(size_t)order - 1], ci[(size_t)order - 1], in, b0));
        if (in_e) CU(launch_scale(h, cr[(size_t)order - 1], ci[(size_t)order - 1], in_e, b0_e));
        s.count(in_e ? 2 : 1, 0);
    }
    StepArgs base{};
    base.src = in;
    base.src_e = in_e;
    return run_recurrence(h, mode, cls, order, b0, b0_e, base, true, [&](StepIO& io, int m) {
        const int k = order - 1 - m;            // this launch produces b_k
        io.cr = cr[(size_t)k];
        io.ci = ci[(size_t)k];
        if (k == 0) {
            io.out = out;
            if (in_e) io.out_e = out_e;
        }
    });
}

int evolve_one(gpuqt_handle* h, const double2* in, double2* out, const std::vector<double>& cr,
               const std::vector<double>& ci, int order) {
    return evolve_clenshaw(h, kModeEvolve, GPUQT_KERNEL_EVOLVE, in, nullptr, out, nullptr, cr, ci, order);
}

// (psi, chi) <- (U psi, U chi + [X,U] psi)
int evolve_msd_pair(gpuqt_handle* h, const std::vector<double>& cr, const std::vector<double>& ci, int order) {
    int rc = evolve_clenshaw(h, kModeEvolveMsd, GPUQT_KERNEL_EVOLVE_MSD, h->psi, h->chi, h->out0, h->out1, cr, ci, order);
    if (rc) return rc;
    std::swap(h->psi, h->out0);
    std::swap(h->chi, h->out1);
    return GPUQT_OK;
}

// moments with the doubling identity: C_n = <v|T_n|v>, n < n_moments  -> h->moments [B][n]
int moments_doubling(gpuqt_handle* h, const double2* v, int n_moments) {
    const int n_steps = n_moments / 2;   // step j gives C_{2j+1}, C_{2j+2}
    if (small_ok(h)) {
        SmallArgs a{};
        a.v0 = v; a.dots = h->dots; a.n_terms = n_steps + 1;
        {
            StatScope s(h, GPUQT_KERNEL_KPM_DOUBLING);
            CU(launch_small(h, kModeDoubling, a));
            s.count(1, n_steps);
        }
        const int total = h->B * n_moments;
        finalize_doubling<<<(total + 255) / 256, 256, 0, h->stream>>>(h->B, n_moments, n_steps, h->dots, h->moments);
        CU(cudaGetLastError());
        return GPUQT_OK;
    }
    StepArgs base{};
    int rc = run_recurrence(h, kModeDoubling, GPUQT_KERNEL_KPM_DOUBLING, n_steps + 1, v, nullptr, base, false,
                            [&](StepIO& io, int m) {
                                io.store = (m < n_steps);
                                io.result = h->dots + (size_t)(m - 1) * 3 * h->B;
                            });
    if (rc) return rc;
    const int total = h->B * n_moments;
    finalize_doubling<<<(total + 255) / 256, 256, 0, h->stream>>>(h->B, n_moments, n_steps, h->dots, h->moments);
    CU(cudaGetLastError());
    return GPUQT_OK;
}

// C_n = <l|T_n|r>  -> h->moments [B][n] (real part)
int moments_left(gpuqt_handle* h, const double2* l, const double2* r, int n_moments) {
    CU(launch_dot(h, l, r, h->dots));
    if (small_ok(h)) {
        SmallArgs a{};
        a.v0 = r; a.aux = l; a.dots = h->dots; a.n_terms = n_moments;
        {
            StatScope s(h, GPUQT_KERNEL_KPM_LEFT);
            CU(launch_small(h, kModeLeft, a));
            s.count(1, n_moments - 1);
        }
        const int total = h->B * n_moments;
        finalize_left<<<(total + 255) / 256, 256, 0, h->stream>>>(h->B, n_moments, h->dots, h->moments);
        CU(cudaGetLastError());
        return GPUQT_OK;
    }
    StepArgs base{};
    base.phiL = l;
    int rc = run_recurrence(h, kModeLeft, GPUQT_KERNEL_KPM_LEFT, n_moments, r, nullptr, base, false, [&](StepIO& io, int n) {
        io.store = (n + 1 < n_moments);
        io.result = h->dots + (size_t)n * 2 * h->B;
    });
    if (rc) return rc;
    const int total = h->B * n_moments;
    finalize_left<<<(total + 255) / 256, 256, 0, h->stream>>>(h->B, n_moments, h->dots, h->moments);
    CU(cudaGetLastError());
    return GPUQT_OK;
}

int copy_moments_out(gpuqt_handle* h, int n_moments, double* out_host) {
    CU(cudaMemcpyAsync(out_host, h->moments, (size_t)h->B * n_moments * sizeof(double), cudaMemcpyDeviceToHost, h->stream));
    CU(cudaStreamSynchronize(h->stream));
    flush_stats(h);
    return GPUQT_OK;
}

int finish_set_state(gpuqt_handle* h) {
    // ring[0] holds phi in [batch][N] order
    const long long total = (long long)h->vec_elems;
    const int blocks = (int)((total + 255) / 256);
    to_device_layout<<<blocks, 256, 0, h->stream>>>(h->N, h->B, h->ring[0], h->psi);
    CU(cudaGetLastError());
    if (h->modes & GPUQT_MODE_MSD) {
        zero_vec<<<blocks, 256, 0, h->stream>>>(total, h->chi);
        CU(cudaGetLastError());
    }
    if (h->modes & GPUQT_MODE_VAC) {
        CU(cudaMemcpyAsync(h->va, h->psi, h->vec_elems * sizeof(double2), cudaMemcpyDeviceToDevice, h->stream));
        StatScope s(h, GPUQT_KERNEL_VELOCITY);
        CU(launch_velocity(h, h->psi, h->vb));
        s.count();
    }
    h->state_set = true;
    return GPUQT_OK;
}

}  // namespace

// =================================================================== C ABI
extern "C" {

size_t gpuqt_workspace_bytes(int64_t N, int32_t K_max, int is_complex, int32_t batch, int modes) {
    if (N <= 0 || K_max <= 0 || !batch_ok(batch)) return 0;
    // upper bound: every slice record padded to K_max
    const size_t rec = (size_t)((N + 31) / 32) * (size_t)record_bytes(K_max, is_complex ? 2 : 1);
    return make_layout(N, batch, modes, rec).total;
}

int gpuqt_validate(int64_t N, int32_t K_max, const int32_t* nbr_count, const int32_t* nbr_index,
                   const double* hop_re, const double* hop_im, const double* onsite,
                   const double* x, double box_length, double energy_scale) {
    std::string msg;
    return validate_inputs(N, K_max, nbr_count, nbr_index, hop_re, hop_im, onsite, x, box_length, energy_scale, msg);
}

int gpuqt_fused_schedule(int32_t n_slices, int32_t run, int32_t grid, int reverse, int32_t slack,
                         const int32_t* nbr_ptr, const int32_t* nbr_slices, int32_t* items, int32_t capacity,
                         int32_t* n_items, int32_t* dep_ptr, int32_t* dep_list, int32_t dep_capacity, int32_t* n_dep) {
    if (n_slices < 1 || run < 1 || grid < 1 || slack < 1 || !nbr_ptr || !nbr_slices || !n_items || !n_dep) return GPUQT_ERR_ARG;
    std::vector<int> np(nbr_ptr, nbr_ptr + n_slices + 1), ns(nbr_slices, nbr_slices + nbr_ptr[n_slices]);
    FusedSchedule fs;
    build_fused_schedule(n_slices, run, grid, reverse, slack, kNoRun, np, ns, fs);
    *n_items = (int32_t)(fs.items.size() / 2);
    *n_dep = (int32_t)fs.dep_list.size();
    if (items) {
        if (*n_items > capacity) return GPUQT_ERR_NOMEM;
        for (size_t i = 0; i < fs.items.size(); ++i) items[i] = fs.items[i];
    }
    if (dep_ptr && dep_list) {
        if (*n_dep > dep_capacity) return GPUQT_ERR_NOMEM;
        for (size_t i = 0; i < fs.dep_ptr.size(); ++i) dep_ptr[i] = fs.dep_ptr[i];
        for (size_t i = 0; i < fs.dep_list.size(); ++i) dep_list[i] = fs.dep_list[i];
    }
    return GPUQT_OK;
}

int gpuqt_bessel_coeffs(double energy_scale, double dt, int32_t order, double* c_re, double* c_im) {
    if (!(energy_scale > 0.0) || order < 1 || !c_re || !c_im) return GPUQT_ERR_ARG;
    std::vector<double> cr, ci;
    bessel_coeffs(energy_scale, dt, order, cr, ci);
    for (int m = 0; m < order; ++m) {
        c_re[m] = cr[(size_t)m];
        c_im[m] = ci[(size_t)m];
    }
    return GPUQT_OK;
}

int gpuqt_create(gpuqt_handle** out, int64_t N, int32_t K_max, const int32_t* nbr_count,
                 const int32_t* nbr_index, const double* hop_re, const double* hop_im,
                 const double* onsite, const double* x, double box_length, double volume,
                 double energy_scale, int32_t batch, int modes, void* workspace,
                 size_t workspace_bytes, void* cuda_stream) {
    if (!out) return GPUQT_ERR_ARG;
    *out = nullptr;
    if (!batch_ok(batch) || !workspace || !(volume > 0.0) || (modes & ~7)) return GPUQT_ERR_ARG;
    std::string msg;
    int rc = validate_inputs(N, K_max, nbr_count, nbr_index, hop_re, hop_im, onsite, x, box_length, energy_scale, msg);
    if (rc != GPUQT_OK) {
        fprintf(stderr, "gpuqt_create: %s\n", msg.c_str());
        return rc;
    }
    if ((reinterpret_cast<uintptr_t>(workspace) & 255u) != 0) return GPUQT_ERR_ARG;
    if (modes & GPUQT_MODE_MSD) modes |= GPUQT_MODE_PSI;
    gpuqt_handle* h = new (std::nothrow) gpuqt_handle();
    if (!h) return GPUQT_ERR_NOMEM;
    h->N = N; h->K = K_max; h->B = batch; h->modes = modes; h->cplx = hop_im ? 1 : 0;
    h->dE = energy_scale; h->box = box_length; h->volume = volume;
    h->stream = (cudaStream_t)cuda_stream;
    h->vec_elems = (size_t)N * batch;

    SellHost sell;
    build_sell(N, K_max, nbr_count, nbr_index, hop_re, hop_im, onsite, env_int("GPUQT_HOP_CONST", 1) != 0, sell);
    // 16-bit columns: only where the unrolled uniform kernels exist (K_max 3, 4, 6)
    if (env_int("GPUQT_IDX16", 1) != 0 && (K_max == 3 || K_max == 4 || K_max == 6)) try_idx16(sell, K_max);
    h->hop = sell.nd == 2 ? kHopComplex : sell.nd == 1 ? kHopReal : sell.idx16 ? kHopConst16 : kHopConst;
    const int stage_bytes = (int)align_up((size_t)hop_record_bytes(K_max, h->hop), 256);   // keeps the vector rows 256-byte aligned
    h->rec_bytes = stage_bytes;
    if (step_smem_bytes(1, mode_stage_bytes_for(h, kModeEvolveMsd, true), true) > kSmemBudget) {
        fprintf(stderr, "gpuqt_create: K_max = %d is too large: one slice record (%d bytes) per warp must fit in "
                        "shared memory\n", K_max, stage_bytes);
        delete h;
        return GPUQT_ERR_ARG;
    }
    const size_t rec_bytes = sell.rec.size();
    const Layout L = make_layout(N, batch, modes, rec_bytes);
    if (L.total > workspace_bytes) {
        delete h;
        return GPUQT_ERR_NOMEM;
    }
    int dev = 0;
    cudaError_t ce = cudaGetDevice(&dev);
    if (ce == cudaSuccess) ce = cudaDeviceGetAttribute(&h->n_sm, cudaDevAttrMultiProcessorCount, dev);
    if (ce != cudaSuccess) {
        fprintf(stderr, "gpuqt_create: no usable CUDA device: %s\n", cudaGetErrorString(ce));
        delete h;
        return GPUQT_ERR_CUDA;
    }
    char* base = (char*)workspace;
    unsigned char* d_rec = (unsigned char*)(base + L.rec);
    double* d_x = (double*)(base + L.x);
    long long* d_sp = (long long*)(base + L.slice_off);
    auto up = [&](void* d, const void* s, size_t bytes) {
        return bytes ? cudaMemcpyAsync(d, s, bytes, cudaMemcpyHostToDevice, h->stream) : cudaSuccess;
    };
    ce = up(d_rec, sell.rec.data(), rec_bytes);
    if (ce == cudaSuccess) ce = up(d_x, x, (size_t)N * sizeof(double));
    if (ce == cudaSuccess) ce = cudaMemsetAsync(d_x + N, 0, sizeof(double), h->stream);
    if (ce == cudaSuccess)
        ce = cudaMemsetAsync(base + L.vectors, 0, (size_t)n_vectors(modes) * align_up((size_t)(N + 1) * batch * sizeof(double2)),
                             h->stream);
    if (ce == cudaSuccess) ce = up(d_sp, sell.slice_off.data(), sell.slice_off.size() * sizeof(long long));
    if (ce == cudaSuccess) ce = cudaMemsetAsync(base + L.ticket, 0, 256, h->stream);
    if (ce == cudaSuccess) ce = cudaStreamSynchronize(h->stream);
    if (ce != cudaSuccess) {
        fprintf(stderr, "gpuqt_create: upload failed: %s\n", cudaGetErrorString(ce));
        delete h;
        return GPUQT_ERR_CUDA;
    }
    h->mat.rec = d_rec; h->mat.slice_off = d_sp; h->mat.x = d_x;
    h->mat.N = N; h->mat.n_slices = sell.n_slices; h->mat.K = K_max; h->mat.uniform = sell.uniform;
    h->mat.cplx = h->cplx; h->mat.hop = h->hop; h->mat.hop_const = sell.hop_const;
    h->mat.inv_dE = 1.0 / energy_scale; h->mat.box = box_length;
    h->kt = (sell.uniform && (K_max == 3 || K_max == 4 || K_max == 6)) ? K_max : 0;
    // Shared-memory stages per warp: one sub-step of a slice takes about one memory latency and a
    // slice has `batch` sub-steps, so small batches need a deeper prefetch.  Tuning overrides:
    // GPUQT_STAGES, GPUQT_BLOCKS_PER_SM, GPUQT_ALTERNATE.
    int stages = env_int("GPUQT_STAGES", batch == 1 ? 4 : batch == 2 ? 3 : 2);
    stages = std::max(1, std::min(stages, kMaxStages));
    h->want_stages = stages;
    h->max_blocks_per_sm = env_int("GPUQT_BLOCKS_PER_SM", 0);
    h->alternate = env_int("GPUQT_ALTERNATE", 1);
    h->run = std::max(1, env_int("GPUQT_RUN", 16) / kWarps) * kWarps;
    // two steps per launch (cheb_pair_kernel) are opt-in: they cut the DRAM bytes of a step pair by a
    // third but are time-neutral at best on B200 so far
    h->fuse = env_int("GPUQT_FUSE", 0);
    h->small = env_int("GPUQT_SMALL", 1);
    h->lag = std::max(1, env_int("GPUQT_LAG", 2));
    h->nbr_ptr.swap(sell.nbr_ptr);
    h->nbr_slices.swap(sell.nbr_slices);
    // without locality in the table (a slice gathering from very many others) a second step cannot
    // trail the first through L2: single-step launches only
    if (h->nbr_slices.size() > (size_t)24 * (size_t)sell.n_slices) h->fuse = 0;

    const size_t vstride = align_up((size_t)(N + 1) * batch * sizeof(double2));
    char* v = base + L.vectors;
    auto nextv = [&]() {
        double2* p = (double2*)v;
        v += vstride;
        h->map_bufs.push_back(p);
        return p;
    };
    h->psi = nextv(); h->out0 = nextv();
    for (int i = 0; i < kRing; ++i) h->ring[i] = nextv();
    if (modes & GPUQT_MODE_MSD) {
        h->chi = nextv(); h->out1 = nextv();
        for (int i = 0; i < kRing; ++i) h->ringe[i] = nextv();
    }
    if (modes & GPUQT_MODE_VAC) {
        h->va = nextv(); h->vb = nextv(); h->phiL = nextv();
    }
    h->partials = (double*)(base + L.partials);
    h->dots = (double*)(base + L.dots);
    h->moments = (double*)(base + L.moments);
    h->ticket = (unsigned int*)(base + L.ticket);
    rc = build_tensor_maps(h);
    if (rc != GPUQT_OK) {
        fprintf(stderr, "gpuqt_create: %s\n", h->err.c_str());
        gpuqt_destroy(h);
        return rc;
    }
    *out = h;
    return GPUQT_OK;
}

int gpuqt_set_state(gpuqt_handle* h, const double* phi_host) {
    if (!h || !phi_host) return fail(h, GPUQT_ERR_ARG, "null argument");
    CU(cudaMemcpyAsync(h->ring[0], phi_host, h->vec_elems * sizeof(double2), cudaMemcpyHostToDevice, h->stream));
    return finish_set_state(h);
}

int gpuqt_set_state_device(gpuqt_handle* h, const double* phi_device) {
    if (!h || !phi_device) return fail(h, GPUQT_ERR_ARG, "null argument");
    CU(cudaMemcpyAsync(h->ring[0], phi_device, h->vec_elems * sizeof(double2), cudaMemcpyDeviceToDevice, h->stream));
    return finish_set_state(h);
}

int gpuqt_dos_moments(gpuqt_handle* h, int32_t n_moments, double* out_host) {
    if (h) h->sweep = 0;
    if (!h || !out_host || n_moments < 2 || n_moments > GPUQT_MAX_MOMENTS) return fail(h, GPUQT_ERR_ARG, "bad n_moments or null output");
    if (!h->state_set) return fail(h, GPUQT_ERR_STATE, "gpuqt_set_state has not been called");
    int rc = moments_doubling(h, h->psi, n_moments);
    if (rc) return rc;
    return copy_moments_out(h, n_moments, out_host);
}

int gpuqt_msd(gpuqt_handle* h, int32_t n_moments, double* out_host) {
    if (h) h->sweep = 0;
    if (!h || !out_host || n_moments < 2 || n_moments > GPUQT_MAX_MOMENTS) return fail(h, GPUQT_ERR_ARG, "bad n_moments or null output");
    if (!(h->modes & GPUQT_MODE_MSD)) return fail(h, GPUQT_ERR_STATE, "handle was created without GPUQT_MODE_MSD");
    if (!h->state_set) return fail(h, GPUQT_ERR_STATE, "gpuqt_set_state has not been called");
    int rc = moments_doubling(h, h->chi, n_moments);
    if (rc) return rc;
    return copy_moments_out(h, n_moments, out_host);
}

int gpuqt_vac(gpuqt_handle* h, int32_t n_moments, double* out_host) {
    if (h) h->sweep = 0;
    if (!h || !out_host || n_moments < 2 || n_moments > GPUQT_MAX_MOMENTS) return fail(h, GPUQT_ERR_ARG, "bad n_moments or null output");
    if (!(h->modes & GPUQT_MODE_VAC)) return fail(h, GPUQT_ERR_STATE, "handle was created without GPUQT_MODE_VAC");
    if (!h->state_set) return fail(h, GPUQT_ERR_STATE, "gpuqt_set_state has not been called");
    {
        StatScope s(h, GPUQT_KERNEL_VELOCITY);
        CU(launch_velocity(h, h->va, h->phiL));   // phi_L = V a
        s.count();
    }
    int rc = moments_left(h, h->phiL, h->vb, n_moments);
    if (rc) return rc;
    return copy_moments_out(h, n_moments, out_host);
}

int gpuqt_evolve(gpuqt_handle* h, double dt, int32_t order) {
    if (h) h->sweep = 0;
    if (!h || order < 1 || !std::isfinite(dt)) return fail(h, GPUQT_ERR_ARG, "bad dt or order");
    if (!h->state_set) return fail(h, GPUQT_ERR_STATE, "gpuqt_set_state has not been called");
    std::vector<double> cr, ci;
    int rc;
    if (h->modes & (GPUQT_MODE_MSD | GPUQT_MODE_PSI)) {
        bessel_coeffs(h->dE, dt, order, cr, ci);
        if (h->modes & GPUQT_MODE_MSD) {
            rc = evolve_msd_pair(h, cr, ci, order);
            if (rc) return rc;
        } else {
            rc = evolve_one(h, h->psi, h->out0, cr, ci, order);
            if (rc) return rc;
            std::swap(h->psi, h->out0);
        }
    }
    if (h->modes & GPUQT_MODE_VAC) {
        bessel_coeffs(h->dE, -dt, order, cr, ci);   // both VAC branches step with U(-dt)  [A1]
        rc = evolve_one(h, h->va, h->out0, cr, ci, order);
        if (rc) return rc;
        std::swap(h->va, h->out0);
        rc = evolve_one(h, h->vb, h->out0, cr, ci, order);
        if (rc) return rc;
        std::swap(h->vb, h->out0);
    }
    return GPUQT_OK;
}

int gpuqt_kpm_transform(gpuqt_handle* h, const double* moments_host, int32_t n_moments,
                        int32_t n_sets, const double* energies_host, int32_t n_energies,
                        double* out_host) {
    if (!h || !moments_host || !energies_host || !out_host || n_moments < 1 || n_sets < 1 || n_energies < 1)
        return fail(h, GPUQT_ERR_ARG, "null or non-positive argument");
    for (int j = 0; j < n_energies; ++j)
        if (!(std::fabs(energies_host[j] / h->dE) < 1.0))
            return fail(h, GPUQT_ERR_ENERGY, "energy point outside (-energy_scale, energy_scale)");
    const size_t bm = (size_t)n_sets * n_moments * sizeof(double), be = (size_t)n_energies * sizeof(double),
                 bo = (size_t)n_sets * n_energies * sizeof(double), bg = (size_t)n_moments * sizeof(double);
    const size_t om = 0, oe = align_up(bm), oo = oe + align_up(be), og = oo + align_up(bo), tot = og + align_up(bg);
    CU(ensure_scratch(h, tot));
    char* s = h->scratch;
    cudaError_t e = cudaMemcpyAsync(s + om, moments_host, bm, cudaMemcpyHostToDevice, h->stream);
    if (e == cudaSuccess) e = cudaMemcpyAsync(s + oe, energies_host, be, cudaMemcpyHostToDevice, h->stream);
    if (e == cudaSuccess) {
        jackson_kernel<<<(n_moments + 255) / 256, 256, 0, h->stream>>>(n_moments, (double*)(s + og));
        const int total = n_sets * n_energies;
        transform_kernel<<<(total + 127) / 128, 128, 0, h->stream>>>(n_moments, n_sets, n_energies, (double*)(s + og),
                                                                     (double*)(s + om), (double*)(s + oe), 1.0 / h->dE,
                                                                     h->volume, (double*)(s + oo));
        e = cudaGetLastError();
    }
    if (e == cudaSuccess) e = cudaMemcpyAsync(out_host, s + oo, bo, cudaMemcpyDeviceToHost, h->stream);
    if (e == cudaSuccess) e = cudaStreamSynchronize(h->stream);
    if (e != cudaSuccess) return cuda_fail(h, e, "kpm_transform");
    flush_stats(h);
    return GPUQT_OK;
}

int gpuqt_running_conductivity(gpuqt_handle* h, int kind, const double* corr_host, const double* dos_host,
                               const double* dt_host, int32_t n_times, int32_t n_energies, double* sigma_host,
                               double* length_host) {
    if (!h || !corr_host || !dt_host || !sigma_host || n_times < 1 || n_energies < 1 ||
        (kind != GPUQT_SIGMA_FROM_VAC && kind != GPUQT_SIGMA_FROM_MSD))
        return fail(h, GPUQT_ERR_ARG, "null or non-positive argument");
    const int n_dt = kind == GPUQT_SIGMA_FROM_VAC ? n_times - 1 : n_times;
    for (int k = 0; k < n_dt; ++k)
        if (!(dt_host[k] > 0.0) || !std::isfinite(dt_host[k])) return fail(h, GPUQT_ERR_ARG, "time steps must be positive");
    const bool want_len = kind == GPUQT_SIGMA_FROM_MSD && length_host && dos_host;
    const size_t bc = (size_t)n_times * n_energies * sizeof(double), be = (size_t)n_energies * sizeof(double),
                 bt = (size_t)n_times * sizeof(double);
    const size_t oc = 0, od = align_up(bc), ot = od + align_up(be), os = ot + align_up(bt), ol = os + align_up(bc),
                 tot = ol + align_up(bc);
    CU(ensure_scratch(h, tot));
    char* s = h->scratch;
    cudaError_t e = cudaMemcpyAsync(s + oc, corr_host, bc, cudaMemcpyHostToDevice, h->stream);
    if (e == cudaSuccess && dos_host) e = cudaMemcpyAsync(s + od, dos_host, be, cudaMemcpyHostToDevice, h->stream);
    if (e == cudaSuccess && n_dt > 0) e = cudaMemcpyAsync(s + ot, dt_host, (size_t)n_dt * sizeof(double), cudaMemcpyHostToDevice, h->stream);
    if (e == cudaSuccess) {
        conductivity_kernel<<<(n_energies + 127) / 128, 128, 0, h->stream>>>(
            kind, n_times, n_energies, (const double*)(s + oc), dos_host ? (const double*)(s + od) : nullptr,
            (const double*)(s + ot), (double*)(s + os), want_len ? (double*)(s + ol) : nullptr);
        e = cudaGetLastError();
    }
    if (e == cudaSuccess) e = cudaMemcpyAsync(sigma_host, s + os, bc, cudaMemcpyDeviceToHost, h->stream);
    if (e == cudaSuccess && want_len) e = cudaMemcpyAsync(length_host, s + ol, bc, cudaMemcpyDeviceToHost, h->stream);
    if (e == cudaSuccess) e = cudaStreamSynchronize(h->stream);
    if (e != cudaSuccess) return cuda_fail(h, e, "running_conductivity");
    return GPUQT_OK;
}

int gpuqt_get_state(gpuqt_handle* h, int which, double* out_host) {
    if (!h || !out_host) return fail(h, GPUQT_ERR_ARG, "null argument");
    const double2* src = which == GPUQT_STATE_PSI ? h->psi : which == GPUQT_STATE_CHI ? h->chi
                       : which == GPUQT_STATE_VAC_A ? h->va : which == GPUQT_STATE_VAC_B ? h->vb : nullptr;
    if (!src) return fail(h, GPUQT_ERR_STATE, "state not available in this mode");
    const long long total = (long long)h->vec_elems;
    from_device_layout<<<(int)((total + 255) / 256), 256, 0, h->stream>>>(h->N, h->B, src, h->ring[0]);
    CU(cudaGetLastError());
    CU(cudaMemcpyAsync(out_host, h->ring[0], h->vec_elems * sizeof(double2), cudaMemcpyDeviceToHost, h->stream));
    CU(cudaStreamSynchronize(h->stream));
    flush_stats(h);
    return GPUQT_OK;
}

int gpuqt_get_table(gpuqt_handle* h, int32_t* col, double* re, double* im, double* dx) {
    if (!h) return GPUQT_ERR_ARG;
    const size_t nk = (size_t)h->N * h->K;
    // scratch: the ring buffers are free between calls (3 * N*B*16 bytes >= N*K*28 is not
    // guaranteed), so use a stream-ordered allocation
    const size_t oc = 0, orr = align_up(nk * 4), oi = orr + align_up(nk * 8), od = oi + align_up(nk * 8), tot = od + align_up(nk * 8);
    CU(ensure_scratch(h, tot));
    char* scratch = h->scratch;
    decode_table<<<(int)((nk + 255) / 256), 256, 0, h->stream>>>(h->mat, (int32_t*)(scratch + oc), (double*)(scratch + orr),
                                                                 (double*)(scratch + oi), (double*)(scratch + od));
    cudaError_t e = cudaGetLastError();
    if (e == cudaSuccess && col) e = cudaMemcpyAsync(col, scratch + oc, nk * 4, cudaMemcpyDeviceToHost, h->stream);
    if (e == cudaSuccess && re) e = cudaMemcpyAsync(re, scratch + orr, nk * 8, cudaMemcpyDeviceToHost, h->stream);
    if (e == cudaSuccess && im) e = cudaMemcpyAsync(im, scratch + oi, nk * 8, cudaMemcpyDeviceToHost, h->stream);
    if (e == cudaSuccess && dx) e = cudaMemcpyAsync(dx, scratch + od, nk * 8, cudaMemcpyDeviceToHost, h->stream);
    if (e == cudaSuccess) e = cudaStreamSynchronize(h->stream);
    if (e != cudaSuccess) return cuda_fail(h, e, "get_table");
    return GPUQT_OK;
}

int gpuqt_kernel_stats(gpuqt_handle* h, int kernel_class, double* ms, int64_t* launches) {
    if (!h || kernel_class < 0 || kernel_class >= GPUQT_KERNEL_CLASSES) return GPUQT_ERR_ARG;
    flush_stats(h);
    if (ms) *ms = h->stat_ms[kernel_class];
    if (launches) *launches = h->stat_launches[kernel_class];
    return GPUQT_OK;
}

int gpuqt_kernel_steps(gpuqt_handle* h, int kernel_class, int64_t* steps) {
    if (!h || !steps || kernel_class < 0 || kernel_class >= GPUQT_KERNEL_CLASSES) return GPUQT_ERR_ARG;
    flush_stats(h);
    *steps = h->stat_steps[kernel_class];
    return GPUQT_OK;
}

int gpuqt_reset_stats(gpuqt_handle* h) {
    if (!h) return GPUQT_ERR_ARG;
    flush_stats(h);
    for (int i = 0; i < GPUQT_KERNEL_CLASSES; ++i) {
        h->stat_ms[i] = 0;
        h->stat_launches[i] = 0;
        h->stat_steps[i] = 0;
    }
    return GPUQT_OK;
}

const char* gpuqt_last_error(const gpuqt_handle* h) { return h ? h->err.c_str() : "null handle"; }

void gpuqt_destroy(gpuqt_handle* h) {
    if (!h) return;
    cudaStreamSynchronize(h->stream);
    flush_stats(h);
    for (auto e : h->free_events) cudaEventDestroy(e);
    if (h->scratch) cudaFree(h->scratch);
    if (h->d_maps) cudaFree(h->d_maps);
    for (auto& d : h->schedules) {
        cudaFree(d.items);
        cudaFree(d.dep_ptr);
        cudaFree(d.dep_list);
        cudaFree(d.run_done);
    }
    delete h;
}

}  // extern "C"
