// C-ABI of the B200-native GPUQT hot path (include/gpuqt.h): host logic + kernel launches.
#include <cuda.h>
#include <cuda_runtime.h>

#include <cstdio>
#include <cstdlib>
#include <functional>
#include <map>
#include <mutex>
#include <string>
#include <vector>

#include "../../include/gpuqt.h"
#include "host_util.h"
#include "kernels.cuh"

using namespace gpuqt;

namespace gpuqt {
void* step_kernel_fn(int mode, int B, int kt, int hop);     // step_kernels.cu
}

namespace {

constexpr int kMaxGrid = 4096;
constexpr int kPartialDoubles = 96;   // 3 * Q*B <= 72 per block (three step buffers of a multi-step launch)
constexpr int kRing = 3;              // recurrence ring x_m -> ring[(m - 1) % 3]
constexpr int kCoefSlots = 8;         // Bessel-coefficient uploads in flight (pinned host ring + device mirror)

struct PendingStat {
    int cls;
    cudaEvent_t start, stop;
    int64_t launches, steps;
};

thread_local std::string g_create_error;   // gpuqt_last_error(NULL)

}  // namespace

struct gpuqt_handle {
    int64_t N = 0;                      // rows of the table (owned rows)
    int64_t NV = 0;                     // zero row of the vector buffers: N, or N + n_halo for a row slab
    int slab = 0;                       // member of a gpuqt_slab_group: one launch per step, no one-CTA kernels
    int32_t K = 0, B = 0;
    int modes = 0, cplx = 0, kt = 0, hop = 0;
    gpuqt_options opt{};
    int run = 16;                       // consecutive tiles per CTA run (multiple of kWarps)
    int rec_bytes = 0;                  // bytes reserved for the records of one tile inside a stage
    int want_stages = 2;                // requested pipeline depth per warp
    int persistent = 0;                 // whole recurrences as one cooperative launch
    int alternate = 1;                  // the sweep direction alternates from step to step
    int coop_ok = 0;                    // the device supports cooperative launches
    // per launch configuration [mode]: stages, bytes per stage, dynamic smem
    int mode_stages[4] = {0};
    int mode_stage_bytes[4] = {0};
    size_t mode_smem[4] = {0};
    double dE = 0, box = 0, volume = 0;
    cudaStream_t stream = nullptr;
    int n_sm = 0;
    Mat mat{};
    size_t vec_elems = 0;   // N * B double2
    size_t stored_matrix_bytes = 0, workspace_used = 0;
    int64_t stencil_patterns = 0;
    // vectors (device, inside the caller's workspace)
    double2 *psi = nullptr, *chi = nullptr, *va = nullptr, *vb = nullptr, *phiL = nullptr;
    double2 *out0 = nullptr, *out1 = nullptr, *ring[kRing] = {nullptr, nullptr, nullptr},
            *ringe[kRing] = {nullptr, nullptr, nullptr};
    // site reordering (recognised cubic lattices stored in bricks): device rows <-> the caller's sites; library-owned
    int32_t *d_new_of_old = nullptr, *d_old_of_new = nullptr;
    // gpuqt_prefetch_state: the next batch of random vectors, copied on the library's own stream while the
    // caller's stream computes
    double2* stage_in = nullptr;
    cudaStream_t copy_stream = nullptr;
    cudaEvent_t ev_copy_done = nullptr, ev_stage_free = nullptr;
    bool prefetched = false, stage_read = false;
    // library-owned scratch for the small transform / table-decode calls: grown on demand, kept
    // (stream-ordered pool allocations can trim at every synchronisation and stall the step)
    char* scratch = nullptr;
    size_t scratch_bytes = 0;
    // Bessel coefficients of the running time steps: pinned host ring -> device mirror
    double* coef_host = nullptr;
    double* coef_dev = nullptr;
    cudaEvent_t coef_event[kCoefSlots] = {nullptr};
    bool coef_used[kCoefSlots] = {false};
    int coef_next = 0;
    // B >= 2: one TMA tensor map (128-byte swizzle) per vector buffer, in device memory
    std::vector<const double2*> map_bufs;
    CUtensorMap* d_maps = nullptr;
    double *partials = nullptr, *dots = nullptr, *moments = nullptr;
    unsigned int *ticket = nullptr, *barrier = nullptr;
    int grid[4] = {0};                  // [mode]
    int grid_aux = 0;
    int sweep = 0;                      // direction of the next step (reset per building block)
    bool state_set = false;
    std::string err;
    double stat_ms[GPUQT_KERNEL_CLASSES] = {0};
    int64_t stat_launches[GPUQT_KERNEL_CLASSES] = {0};
    int64_t stat_steps[GPUQT_KERNEL_CLASSES] = {0};     // recurrence steps (a multi-step launch does many)
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
    int n = 3 + kRing;                              // psi, out0, ring, the staging buffer of gpuqt_prefetch_state
    if (modes & GPUQT_MODE_MSD) n += 2 + kRing;     // chi, out1, ringe
    if (modes & GPUQT_MODE_VAC) n += 3;             // a, b, phi_L
    return n;
}

struct Layout {
    size_t rec, slice_off, x, vectors, partials, dots, moments, ticket, total;
};

// N = rows of the vector buffers below the zero row (owned rows + halo rows of a slab)
Layout make_layout(int64_t N, int32_t B, int modes, size_t rec_bytes) {
    Layout L{};
    size_t off = 0;
    auto take = [&](size_t bytes) {
        size_t o = off;
        off = align_up(off + bytes);
        return o;
    };
    const size_t n_slices = (size_t)((N + 31) / 32) + kTilePad;
    L.rec = take(rec_bytes);
    L.slice_off = take((n_slices + 1) * sizeof(long long));
    L.x = take((size_t)(N + 1) * sizeof(double));
    // every vector buffer has N + 1 rows; row N stays zero for ever (nothing writes it)
    L.vectors = take((size_t)n_vectors(modes) * align_up((size_t)(N + 1) * B * sizeof(double2)));
    L.partials = take((size_t)kMaxGrid * kPartialDoubles * sizeof(double));
    L.dots = take((size_t)GPUQT_MAX_MOMENTS * 3 * 8 * sizeof(double));
    L.moments = take((size_t)GPUQT_MAX_MOMENTS * 8 * sizeof(double));
    L.ticket = take(256);                           // [0] last-block ticket, [32] grid-barrier counter
    L.total = off;
    return L;
}

// shared memory of one step-kernel CTA: mbarriers, then kWarps * stages tile buffers
size_t step_smem_bytes(int stages, int stage_bytes) {
    return 128 * (((size_t)kWarps * kMaxStages * 8 + 127) / 128) + (size_t)kWarps * stages * stage_bytes;
}
constexpr size_t kSmemBudget = 200 * 1024;   // per CTA; leaves room for the static reduction buffers
constexpr size_t kSmemPerSm = 227 * 1024;

bool batch_ok(int B) { return B == 1 || B == 2 || B == 4 || B == 8; }
bool unrolled_width(int K) { return K == 2 || K == 3 || K == 4 || K == 6; }

// cudaFuncAttributeMaxDynamicSharedMemorySize is a property of the kernel in this process, not of a
// handle: raise it (never lower it) under a lock, whichever handle asks
cudaError_t ensure_dynamic_smem(void* fn, size_t bytes) {
    static std::mutex mu;
    static std::map<void*, size_t> granted;
    // below 32 KB the default 48 KB limit holds even with the kernels' static shared memory (<= 9 KB) on top
    if (bytes <= 32 * 1024) return cudaSuccess;
    std::lock_guard<std::mutex> lock(mu);
    size_t& g = granted[fn];
    if (bytes <= g) return cudaSuccess;
    cudaError_t e = cudaFuncSetAttribute(fn, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bytes);
    if (e == cudaSuccess) g = bytes;
    return e;
}

constexpr int64_t kB200L2Bytes = 126LL << 20;

// Site reordering: a recognised simple-cubic lattice is stored in bricks of 4 x 4 x 2 sites (host_util.h,
// detect_cubic_bricks).  option 1: at batch >= 4 when a recurrence step's working set exceeds the L2 (the HBM-bound case
// it was measured to pay in, and the case in which the implicit stencil replaces the index array, whose 16-bit form the
// brick order would lose), 2: whenever the lattice is recognised (tests), 0: never.  On success the pointers are
// redirected to permuted copies held by `ro`.
struct ReorderedInputs {
    std::vector<int32_t> new_of_old, old_of_new, cnt, idx;
    std::vector<double> hre, him, ons, x;
};
void reorder_inputs(ReorderedInputs& ro, int option, int64_t l2_bytes, int64_t N, int32_t K_max, int batch,
                    const int32_t*& nbr_count, const int32_t*& nbr_index, const double*& hop_re, const double*& hop_im,
                    const double*& onsite, const double*& x) {
    const int64_t working_set = 3 * (N + 1) * (int64_t)batch * 16 + N * (8 + 2 * (int64_t)K_max);
    const bool want = option == 2 || (option == 1 && batch >= 4 && working_set > (l2_bytes > 0 ? l2_bytes : kB200L2Bytes));
    if (!want || !detect_cubic_bricks(N, K_max, nbr_count, nbr_index, ro.new_of_old, ro.old_of_new)) {
        ro.new_of_old.clear();
        ro.old_of_new.clear();
        return;
    }
    const size_t K = (size_t)K_max;
    ro.cnt.resize((size_t)N);
    ro.idx.resize((size_t)N * K);
    if (x) ro.x.resize((size_t)N);
    if (hop_re) ro.hre.resize((size_t)N * K);
    if (hop_im) ro.him.resize((size_t)N * K);
    if (onsite) ro.ons.resize((size_t)N);
    for (int64_t p = 0; p < N; ++p) {
        const size_t m = (size_t)ro.old_of_new[(size_t)p];
        ro.cnt[(size_t)p] = nbr_count[m];
        if (x) ro.x[(size_t)p] = x[m];
        if (onsite) ro.ons[(size_t)p] = onsite[m];
        for (size_t k = 0; k < K; ++k) {
            const int32_t n = nbr_index[m * K + k];
            ro.idx[(size_t)p * K + k] = (k < (size_t)nbr_count[m]) ? ro.new_of_old[(size_t)n] : n;
            if (hop_re) ro.hre[(size_t)p * K + k] = hop_re[m * K + k];
            if (hop_im) ro.him[(size_t)p * K + k] = hop_im[m * K + k];
        }
    }
    nbr_count = ro.cnt.data();
    nbr_index = ro.idx.data();
    if (x) x = ro.x.data();
    if (hop_re) hop_re = ro.hre.data();
    if (hop_im) hop_im = ro.him.data();
    if (onsite) onsite = ro.ons.data();
}

// The storage variant of a table: packed sliced ELL; no hopping array when every
// hopping is the same number; then the implicit stencil, else 16-bit columns, where the unrolled uniform
// kernels exist.  Returns the Hop variant; `sell` (and `sten`) hold the records to upload.
// The stencil saves HBM bytes and costs two more (small) TMA copies per slice: it is taken (option 1) only when
// a recurrence step's working set -- three vector sets and the table -- does not fit the L2, i.e. when the
// index array would really come from HBM every step (c2, 72 MB, is faster with the explicit array: 12.3 vs
// 20.0 us per step; c4, 786 MB, is faster with the stencil: 156 vs 162 us), and only at batch >= 4: at B = 1 a
// tile streams so few bytes that the two extra copies per slice cost more than the index bytes they save (the
// paper's example 5.1, a 2000 x 2000 square lattice with one vector: 1.57 s with explicit columns, 2.07 s with the
// stencil).
int choose_storage(int64_t N, int32_t K_max, const int32_t* nbr_count, const int32_t* nbr_index, const double* hop_re,
                   const double* hop_im, const double* onsite, const gpuqt_options& opt, int batch, int64_t l2_bytes,
                   SellHost& sell, StencilHost& sten, int64_t NV = -1) {
    if (NV < 0) NV = N;
    build_sell(N, K_max, nbr_count, nbr_index, hop_re, hop_im, onsite, opt.hop_const != 0, kTilePad, sell, NV);
    const int64_t working_set = 3 * (N + 1) * (int64_t)batch * 16 + (int64_t)sell.rec.size();
    const bool want_stencil = opt.stencil == 2 || (opt.stencil == 1 && batch >= 4 && working_set > (l2_bytes > 0 ? l2_bytes : kB200L2Bytes));
    const bool use_stencil = want_stencil && unrolled_width(K_max) && try_stencil(sell, K_max, N, opt.stencil == 2, sten);
    if (!use_stencil && opt.idx16 && unrolled_width(K_max)) try_idx16(sell, K_max, NV);
    return sell.nd == 2 ? kHopComplex : sell.nd == 1 ? kHopReal : use_stencil ? kHopStencil
           : sell.idx16 == 2 ? kHopConst16P : sell.idx16 ? kHopConst16 : kHopConst;
}
// bytes the table takes on the device: records (+ dictionary and pattern ids) + the x array
size_t stored_bytes_of(int64_t N, int hop, const SellHost& sell, const StencilHost& sten) {
    size_t rec = sell.rec.size();
    if (hop == kHopStencil) rec = align_up(rec) + sten.dict.size() * sizeof(int32_t) + sten.pid.size() * sizeof(int32_t);
    return rec + (size_t)(N + 1) * sizeof(double);
}
int create_handle(gpuqt_handle** out, int64_t N, int64_t n_halo, int32_t K_max, const int32_t* nbr_count,
                  const int32_t* nbr_index, const double* hop_re, const double* hop_im, const double* onsite,
                  const double* x, double box_length, double volume, double energy_scale, int32_t batch, int modes,
                  void* workspace, size_t workspace_bytes, void* cuda_stream, const gpuqt_options* options, bool is_slab);

// ---------------------------------------------------------------- kernel dispatch
// the cheb_step_kernel instantiations live in step_kernels.cu, one translation unit per Mode
void* step_kernel(const gpuqt_handle* h, int mode) { return gpuqt::step_kernel_fn(mode, h->B, h->kt, h->hop); }

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
    if (h->opt.blocks_per_sm > 0 && per_sm > h->opt.blocks_per_sm) per_sm = h->opt.blocks_per_sm;
    long long g = (long long)per_sm * h->n_sm;
    if (g > work_items) g = work_items;
    if (g > kMaxGrid) g = kMaxGrid;
    if (g < 1) g = 1;
    return (int)g;
}

// bytes of one stage of a step kernel: the records of a tile plus the staged own rows of x_{m-1},
// x_{m-2} (and e_{m-1}, e_{m-2} for the (a, e) pair)
int mode_stage_bytes_for(const gpuqt_handle* h, int mode) {
    int streams = (mode == kModeEvolveMsd) ? 4 : 2;
    if (prev_direct(h->B, mode)) streams /= 2;   // x_{m-2} rows are not staged
    return h->rec_bytes + streams * tile_slices(h->B, h->kt) * 32 * h->B * (int)sizeof(double2);
}

long long n_tiles_of(const gpuqt_handle* h) {
    const int S = tile_slices(h->B, h->kt);
    return (h->mat.n_slices + S - 1) / S;
}

cudaError_t configure_mode(gpuqt_handle* h, int mode) {
    if (h->grid[mode]) return cudaSuccess;
    void* fn = step_kernel(h, mode);
    const int sb = mode_stage_bytes_for(h, mode);
    int stages = h->want_stages;
    while (stages > 1 && step_smem_bytes(stages, sb) > kSmemBudget) --stages;
    // prefer two resident CTAs per SM over a deeper pipeline (where the registers allow two at all)
    while (min_blocks(h->B, mode) >= 2 && stages > 2 && 2 * (step_smem_bytes(stages, sb) + 4096) > kSmemPerSm) --stages;
    h->mode_stages[mode] = stages;
    h->mode_stage_bytes[mode] = sb;
    h->mode_smem[mode] = step_smem_bytes(stages, sb);
    cudaError_t e = ensure_dynamic_smem(fn, h->mode_smem[mode]);
    if (e != cudaSuccess) return e;
    h->grid[mode] = grid_for(h, fn, h->mode_smem[mode], (n_tiles_of(h) + h->run - 1) / h->run);
    return cudaSuccess;
}

// steps [a.m_begin, a.m_end) of a recurrence: a plain launch for one step, a cooperative launch for several
cudaError_t launch_steps(gpuqt_handle* h, int mode, RecArgs& a) {
    cudaError_t e = configure_mode(h, mode);
    if (e != cudaSuccess) return e;
    void* fn = step_kernel(h, mode);
    a.stages = h->mode_stages[mode];
    a.stage_bytes = h->mode_stage_bytes[mode];
    a.rec_bytes = h->rec_bytes;
    a.partials = h->partials;
    a.ticket = h->ticket;
    a.barrier = h->barrier;
    a.alternate = h->alternate;
    a.sweep0 = h->alternate ? (h->sweep & 1) : 0;
    a.run = h->run;
    const int n = a.m_end - a.m_begin;
    h->sweep += n;
    void* args[] = {(void*)&h->mat, (void*)&a};
    if (!a.multi) return cudaLaunchKernel(fn, dim3(h->grid[mode]), dim3(kThreads), args, h->mode_smem[mode], h->stream);
    e = cudaMemsetAsync(h->barrier, 0, sizeof(unsigned int), h->stream);
    if (e != cudaSuccess) return e;
    return cudaLaunchCooperativeKernel(fn, dim3(h->grid[mode]), dim3(kThreads), args, h->mode_smem[mode], h->stream);
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
// written to shared memory with the 128-byte swizzle; lines past the end are zero-filled.  (kSwizzleLineBytes = 64:
// the GPUQT_SWZ64 experiment of kernels.cuh.)
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
        constexpr cuuint64_t LB = kSwizzleLineBytes;
        const cuuint64_t dims[2] = {LB / 8, ((cuuint64_t)(h->NV + 1) * (cuuint64_t)h->B * 16 + LB - 1) / LB};
        const cuuint64_t strides[1] = {LB};
        const cuuint32_t box[2] = {(cuuint32_t)(LB / 8), (cuuint32_t)(512 / LB * h->B)};
        const cuuint32_t estr[2] = {1, 1};
        CUresult r = encode(&maps[i], CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 2, (void*)h->map_bufs[i], dims, strides, box, estr,
                            CU_TENSOR_MAP_INTERLEAVE_NONE, LB == 64 ? CU_TENSOR_MAP_SWIZZLE_64B : CU_TENSOR_MAP_SWIZZLE_128B,
                            CU_TENSOR_MAP_L2_PROMOTION_NONE, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
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

// The c_k of one time step -> device, through a ring of pinned host slots (no pageable copy, so the
// host never waits for the stream).  Returns the device address of (re, im) pairs, k < order.
cudaError_t upload_coefs(gpuqt_handle* h, const std::vector<double>& cr, const std::vector<double>& ci, int order,
                         const double** dev) {
    const int slot = h->coef_next;
    h->coef_next = (slot + 1) % kCoefSlots;
    cudaError_t e;
    if (h->coef_used[slot]) {
        e = cudaEventSynchronize(h->coef_event[slot]);      // the copy out of this pinned slot has run
        if (e != cudaSuccess) return e;
    }
    double* hs = h->coef_host + (size_t)slot * 2 * GPUQT_MAX_ORDER;
    double* ds = h->coef_dev + (size_t)slot * 2 * GPUQT_MAX_ORDER;
    for (int k = 0; k < order; ++k) {
        hs[2 * k] = cr[(size_t)k];
        hs[2 * k + 1] = ci[(size_t)k];
    }
    e = cudaMemcpyAsync(ds, hs, (size_t)order * 2 * sizeof(double), cudaMemcpyHostToDevice, h->stream);
    if (e != cudaSuccess) return e;
    e = cudaEventRecord(h->coef_event[slot], h->stream);
    if (e != cudaSuccess) return e;
    h->coef_used[slot] = true;
    *dev = ds;
    return cudaSuccess;
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
bool small_ok(const gpuqt_handle* h) { return h->opt.small && !h->slab && small_smem_bytes(h) <= 210 * 1024; }
// the (psi, chi) kernel keeps the x array in shared memory as well
size_t small_msd_smem_bytes(const gpuqt_handle* h) { return small_smem_bytes(h) + (size_t)h->N * 8; }
bool small_msd_ok(const gpuqt_handle* h) { return h->opt.small && !h->slab && small_msd_smem_bytes(h) <= 210 * 1024; }

template <int MODE>
void* small_fn(int B) {
    switch (B) {
    case 1: return (void*)cheb_small_kernel<1, MODE>;
    case 2: return (void*)cheb_small_kernel<2, MODE>;
    case 4: return (void*)cheb_small_kernel<4, MODE>;
    default: return (void*)cheb_small_kernel<8, MODE>;
    }
}
void* small_msd_fn(int B) {
    switch (B) {
    case 1: return (void*)cheb_small_msd_kernel<1>;
    case 2: return (void*)cheb_small_msd_kernel<2>;
    case 4: return (void*)cheb_small_msd_kernel<4>;
    default: return (void*)cheb_small_msd_kernel<8>;
    }
}
cudaError_t launch_small(gpuqt_handle* h, int mode, SmallArgs& a) {
    void* fn = mode == kModeDoubling ? small_fn<kModeDoubling>(h->B)
               : mode == kModeLeft   ? small_fn<kModeLeft>(h->B)
               : mode == kModeEvolve ? small_fn<kModeEvolve>(h->B)
                                     : small_msd_fn(h->B);
    const size_t smem = mode == kModeEvolveMsd ? small_msd_smem_bytes(h) : small_smem_bytes(h);
    cudaError_t e = ensure_dynamic_smem(fn, smem);
    if (e != cudaSuccess) return e;
    void* args[] = {(void*)&h->mat, (void*)&a};
    return cudaLaunchKernel(fn, dim3(1), dim3(kSmallThreads), args, smem, h->stream);
}

// Driver of one three-term recurrence x_m = 2 H~ x_{m-1} - x_{m-2} (+ ...), m = 1 .. terms-1 (and the
// e-chain of the MSD pair).  Forward recurrences (moments) apply factor 1 in step 1 (T_1 = H~ T_0);
// Clenshaw recurrences (evolution) in the LAST step.  One plain launch per step, or -- persistent
// mode -- the whole recurrence in one cooperative launch with grid barriers between the steps.
// ring buffers and tensor maps of a recurrence whose x_0 (e_0) the caller has set
void fill_rec_args(const gpuqt_handle* h, RecArgs& a) {
    for (int i = 0; i < kRing; ++i) {
        a.ring[i] = h->ring[i];
        a.tm_ring[i] = tensor_map_of(h, h->ring[i]);
        a.ring_e[i] = a.e0 ? h->ringe[i] : nullptr;
        a.tm_ring_e[i] = a.e0 ? tensor_map_of(h, h->ringe[i]) : nullptr;
    }
    a.tm_x0 = tensor_map_of(h, a.x0);
    a.tm_e0 = tensor_map_of(h, a.e0);
}

int run_recurrence(gpuqt_handle* h, int mode, int cls, RecArgs a) {
    StatScope s(h, cls);
    fill_rec_args(h, a);
    if (a.terms < 2) return GPUQT_OK;
    if (h->persistent) {
        a.multi = 1;
        a.m_begin = 1;
        a.m_end = a.terms;
        cudaError_t e = launch_steps(h, mode, a);
        if (e == cudaSuccess) {
            s.count(1, a.terms - 1);
            return GPUQT_OK;
        }
        if (e != cudaErrorCooperativeLaunchTooLarge && e != cudaErrorNotSupported) return cuda_fail(h, e, "cooperative launch");
        (void)cudaGetLastError();       // the device is shared (MPS, another context): fall back to one launch per step
        h->persistent = 0;
        h->sweep -= a.terms - 1;
    }
    a.multi = 0;
    for (int m = 1; m < a.terms; ++m) {
        a.m_begin = m;
        a.m_end = m + 1;
        CU(launch_steps(h, mode, a));
        s.count(1, 1);
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
// the same order - 1 SpMV steps as the forward form, but no accumulator is read-modified-written
// (64 instead of 80 bytes per row and term).  The same for the (psi, chi) pair with the block operator
// [[H~, 0], [[X,H~], H~]] (a_m = T_m psi, e_m = T_m chi + [X,T_m] psi, Eq. 18, 22, 24).
// `in` is left untouched; `out` must differ from in and from the ring buffers.
int evolve_clenshaw(gpuqt_handle* h, int mode, int cls, const double2* in, const double2* in_e, double2* out,
                    double2* out_e, const std::vector<double>& cr, const std::vector<double>& ci, int order) {
    if (order == 1) {
        StatScope s(h, cls);
        CU(launch_scale(h, cr[0], ci[0], in, out));
        if (in_e) CU(launch_scale(h, cr[0], ci[0], in_e, out_e));
        s.count(in_e ? 2 : 1, 0);
        return GPUQT_OK;
    }
    const double* coef = nullptr;
    CU(upload_coefs(h, cr, ci, order, &coef));
    if (in_e ? small_msd_ok(h) : small_ok(h)) {
        SmallArgs a{};
        a.aux = in; a.aux_e = in_e; a.out = out; a.out_e = out_e; a.coef = (const double2*)coef; a.n_terms = order;
        StatScope s(h, cls);
        CU(launch_small(h, in_e ? kModeEvolveMsd : kModeEvolve, a));
        s.count(1, order - 1);
        return GPUQT_OK;
    }
    // x_0 = b_{order-1} lives in the last ring slot: the recurrence writes slots 0, 1, 2, 0, ... and
    // needs x_0 only in its first two steps
    double2* b0 = h->ring[kRing - 1];
    double2* b0_e = in_e ? h->ringe[kRing - 1] : nullptr;
    {
        StatScope s(h, cls);       // counted as launches of the class, not as recurrence steps
        CU(launch_scale(h, cr[(size_t)order - 1], ci[(size_t)order - 1], in, b0));
        if (in_e) CU(launch_scale(h, cr[(size_t)order - 1], ci[(size_t)order - 1], in_e, b0_e));
        s.count(in_e ? 2 : 1, 0);
    }
    RecArgs a{};
    a.x0 = b0; a.e0 = b0_e;
    a.src = in; a.src_e = in_e;
    a.coef = coef;
    a.terms = order;
    a.clenshaw = 1;
    a.store_last = 1;
    a.last_out = out; a.last_out_e = out_e;
    return run_recurrence(h, mode, cls, a);
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
        StatScope s(h, GPUQT_KERNEL_KPM_DOUBLING);
        CU(launch_small(h, kModeDoubling, a));
        s.count(1, n_steps);
    } else {
        RecArgs a{};
        a.x0 = v;
        a.terms = n_steps + 1;
        a.dots = h->dots;        // step m -> dots[(m - 1) * 3 B]
        a.dot_m0 = 1;
        int rc = run_recurrence(h, kModeDoubling, GPUQT_KERNEL_KPM_DOUBLING, a);
        if (rc) return rc;
    }
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
        StatScope s(h, GPUQT_KERNEL_KPM_LEFT);
        CU(launch_small(h, kModeLeft, a));
        s.count(1, n_moments - 1);
    } else {
        RecArgs a{};
        a.x0 = r;
        a.phiL = l;
        a.terms = n_moments;
        a.dots = h->dots;        // step n -> dots[n * 2 B]
        a.dot_m0 = 0;
        int rc = run_recurrence(h, kModeLeft, GPUQT_KERNEL_KPM_LEFT, a);
        if (rc) return rc;
    }
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

int finish_set_state(gpuqt_handle* h, const double2* src) {
    // src holds phi in [batch][N] order
    const long long total = (long long)h->vec_elems;
    const int blocks = (int)((total + 255) / 256);
    to_device_layout<<<blocks, 256, 0, h->stream>>>(h->N, h->B, src, h->psi, h->d_old_of_new);
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

void gpuqt_default_options(gpuqt_options* o) {
    if (!o) return;
    o->struct_bytes = (int32_t)sizeof(gpuqt_options);
    o->stages = 0;
    o->blocks_per_sm = 0;
    o->run = 0;
    o->alternate = 1;
    o->hop_const = 1;
    o->idx16 = 1;
    o->small = 1;
    o->persistent = -1;
    o->stencil = 1;
    o->reorder = 1;
}

size_t gpuqt_workspace_bytes(int64_t N, int32_t K_max, int is_complex, int32_t batch, int modes) {
    if (N <= 0 || K_max <= 0 || !batch_ok(batch)) return 0;
    // upper bound: every slice record padded to K_max, per-entry hoppings, int32 columns
    const size_t rec = (size_t)((N + 31) / 32 + kTilePad) * (size_t)record_bytes(K_max, is_complex ? 2 : 1);
    return make_layout(N, batch, modes, rec).total;
}

int gpuqt_validate(int64_t N, int32_t K_max, const int32_t* nbr_count, const int32_t* nbr_index,
                   const double* hop_re, const double* hop_im, const double* onsite,
                   const double* x, double box_length, double energy_scale) {
    std::string msg;
    return validate_inputs(N, K_max, nbr_count, nbr_index, hop_re, hop_im, onsite, x, box_length, energy_scale, msg);
}

int gpuqt_plan_storage(int64_t N, int32_t K_max, const int32_t* nbr_count, const int32_t* nbr_index, const double* hop_re,
                       const double* hop_im, int32_t batch, int64_t l2_bytes, const gpuqt_options* options,
                       int32_t* hop_variant, int64_t* stored_matrix_bytes, int64_t* stencil_patterns) {
    if (N <= 0 || K_max <= 0 || N > 0x7fffffffLL || !nbr_count || !nbr_index || !batch_ok(batch) || l2_bytes < 0) return GPUQT_ERR_ARG;
    gpuqt_options opt;
    gpuqt_default_options(&opt);
    if (options) {
        if (options->struct_bytes < (int32_t)sizeof(int32_t) || options->struct_bytes > (int32_t)sizeof(gpuqt_options)) return GPUQT_ERR_ARG;
        std::memcpy(&opt, options, (size_t)options->struct_bytes);
    }
    for (int64_t m = 0; m < N; ++m) {
        if (nbr_count[m] < 0 || nbr_count[m] > K_max) return GPUQT_ERR_INDEX;
        for (int32_t k = 0; k < nbr_count[m]; ++k)
            if (nbr_index[(size_t)m * K_max + k] < 0 || nbr_index[(size_t)m * K_max + k] >= N) return GPUQT_ERR_INDEX;
    }
    ReorderedInputs ro;
    const double *no_onsite = nullptr, *no_x = nullptr;
    reorder_inputs(ro, opt.reorder, l2_bytes, N, K_max, batch, nbr_count, nbr_index, hop_re, hop_im, no_onsite, no_x);
    SellHost sell;
    StencilHost sten;
    const int hop = choose_storage(N, K_max, nbr_count, nbr_index, hop_re, hop_im, nullptr, opt, batch, l2_bytes, sell, sten);
    if (hop_variant) *hop_variant = hop;
    if (stored_matrix_bytes) *stored_matrix_bytes = (int64_t)stored_bytes_of(N, hop, sell, sten);
    if (stencil_patterns) *stencil_patterns = hop == kHopStencil ? sten.n_patterns : 0;
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
    return gpuqt_create_with_options(out, N, K_max, nbr_count, nbr_index, hop_re, hop_im, onsite, x, box_length, volume,
                                     energy_scale, batch, modes, workspace, workspace_bytes, cuda_stream, nullptr);
}

int gpuqt_create_with_options(gpuqt_handle** out, int64_t N, int32_t K_max, const int32_t* nbr_count,
                 const int32_t* nbr_index, const double* hop_re, const double* hop_im,
                 const double* onsite, const double* x, double box_length, double volume,
                 double energy_scale, int32_t batch, int modes, void* workspace,
                 size_t workspace_bytes, void* cuda_stream, const gpuqt_options* options) {
    return create_handle(out, N, 0, K_max, nbr_count, nbr_index, hop_re, hop_im, onsite, x, box_length, volume, energy_scale,
                         batch, modes, workspace, workspace_bytes, cuda_stream, options, false);
}
}  // extern "C"

namespace {
// gpuqt_create_with_options (n_halo = 0), or one row slab of a gpuqt_slab_group (n_halo >= 0 halo rows behind the
// N owned rows; x has N + n_halo entries)
int create_handle(gpuqt_handle** out, int64_t N, int64_t n_halo, int32_t K_max, const int32_t* nbr_count,
                  const int32_t* nbr_index, const double* hop_re, const double* hop_im, const double* onsite,
                  const double* x, double box_length, double volume, double energy_scale, int32_t batch, int modes,
                  void* workspace, size_t workspace_bytes, void* cuda_stream, const gpuqt_options* options, bool is_slab) {
    auto bad = [&](int code, const std::string& msg) {
        g_create_error = "gpuqt_create: " + msg;
        return code;
    };
    if (!out) return bad(GPUQT_ERR_ARG, "null output pointer");
    *out = nullptr;
    if (!batch_ok(batch)) return bad(GPUQT_ERR_ARG, "batch must be 1, 2, 4 or 8");
    if (!workspace || !(volume > 0.0) || (modes & ~7)) return bad(GPUQT_ERR_ARG, "null workspace, non-positive volume or unknown mode bits");
    gpuqt_options opt;
    gpuqt_default_options(&opt);
    if (options) {
        if (options->struct_bytes < (int32_t)sizeof(int32_t) || options->struct_bytes > (int32_t)sizeof(gpuqt_options))
            return bad(GPUQT_ERR_ARG, "gpuqt_options.struct_bytes does not match this library (use gpuqt_default_options)");
        std::memcpy(&opt, options, (size_t)options->struct_bytes);     // an older, shorter struct keeps the newer defaults
        opt.struct_bytes = (int32_t)sizeof(gpuqt_options);
    }
    if (opt.stages < 0 || opt.stages > kMaxStages || opt.blocks_per_sm < 0 || opt.run < 0 || opt.persistent < -1 || opt.persistent > 1 ||
        opt.stencil < 0 || opt.stencil > 2 || opt.reorder < 0 || opt.reorder > 2)
        return bad(GPUQT_ERR_ARG, "option out of range");
    std::string msg;
    int rc = validate_inputs(N, K_max, nbr_count, nbr_index, hop_re, hop_im, onsite, x, box_length, energy_scale, msg, n_halo);
    if (rc != GPUQT_OK) return bad(rc, msg);
    if ((reinterpret_cast<uintptr_t>(workspace) & 255u) != 0) return bad(GPUQT_ERR_ARG, "workspace must be 256-byte aligned");
    const int64_t NV = N + n_halo;
    if (is_slab) {              // the steps of a slab are separated by halo exchanges: one launch per step, streaming kernels
        opt.small = 0;
        opt.persistent = 0;
    }
    if (modes & GPUQT_MODE_MSD) modes |= GPUQT_MODE_PSI;
    gpuqt_handle* h = new (std::nothrow) gpuqt_handle();
    if (!h) return bad(GPUQT_ERR_NOMEM, "out of host memory");
    h->N = N; h->NV = NV; h->slab = is_slab ? 1 : 0; h->K = K_max; h->B = batch; h->modes = modes; h->cplx = hop_im ? 1 : 0;
    h->opt = opt;
    h->dE = energy_scale; h->box = box_length; h->volume = volume;
    h->stream = (cudaStream_t)cuda_stream;
    h->vec_elems = (size_t)N * batch;

    SellHost sell;
    StencilHost sten;
    int l2_bytes = 0;
    {
        int dev0 = 0;
        if (cudaGetDevice(&dev0) != cudaSuccess || cudaDeviceGetAttribute(&l2_bytes, cudaDevAttrL2CacheSize, dev0) != cudaSuccess) {
            (void)cudaGetLastError();
            l2_bytes = 0;                   // no device: gpuqt_create fails below with GPUQT_ERR_CUDA
        }
    }
    // Site reordering (reorder_inputs above): from here on every array is in the device numbering
    ReorderedInputs ro;
    reorder_inputs(ro, is_slab ? 0 : opt.reorder, l2_bytes, N, K_max, batch, nbr_count, nbr_index, hop_re, hop_im, onsite, x);
    std::vector<int32_t>& new_of_old = ro.new_of_old;
    std::vector<int32_t>& old_of_new = ro.old_of_new;
    h->hop = choose_storage(N, K_max, nbr_count, nbr_index, hop_re, hop_im, onsite, opt, batch, l2_bytes, sell, sten, NV);
    const bool use_stencil = h->hop == kHopStencil;
    h->stencil_patterns = use_stencil ? sten.n_patterns : 0;
    h->kt = (sell.uniform && unrolled_width(K_max)) ? K_max : 0;
    // bytes reserved for the record images of one tile inside a stage (keeps the vector rows 256-byte aligned)
    h->rec_bytes = (int)align_up((size_t)hop_stage_bytes(K_max, h->hop) * tile_slices(batch, h->kt), 256);
    if (step_smem_bytes(1, mode_stage_bytes_for(h, kModeEvolveMsd)) > kSmemBudget) {
        delete h;
        return bad(GPUQT_ERR_ARG, "K_max = " + std::to_string(K_max) + " is too large: one slice record per warp must fit in shared memory");
    }
    // the stencil dictionary lives behind the records
    const size_t dict_off = align_up(sell.rec.size()), dict_bytes = sten.dict.size() * sizeof(int32_t);
    const size_t rec_bytes = use_stencil ? dict_off + dict_bytes : sell.rec.size();
    const Layout L = make_layout(NV, batch, modes, rec_bytes);
    if (L.total > workspace_bytes) {
        delete h;
        return bad(GPUQT_ERR_NOMEM, "workspace too small: " + std::to_string(L.total) + " bytes needed");
    }
    h->workspace_used = L.total;
    h->stored_matrix_bytes = stored_bytes_of(NV, h->hop, sell, sten);
    int dev = 0;
    cudaError_t ce = cudaGetDevice(&dev);
    if (ce == cudaSuccess) ce = cudaDeviceGetAttribute(&h->n_sm, cudaDevAttrMultiProcessorCount, dev);
    if (ce == cudaSuccess) ce = cudaDeviceGetAttribute(&h->coop_ok, cudaDevAttrCooperativeLaunch, dev);
    if (ce != cudaSuccess) {
        delete h;
        return bad(GPUQT_ERR_CUDA, std::string("no usable CUDA device: ") + cudaGetErrorString(ce));
    }
    char* base = (char*)workspace;
    unsigned char* d_rec = (unsigned char*)(base + L.rec);
    double* d_x = (double*)(base + L.x);
    long long* d_sp = (long long*)(base + L.slice_off);
    auto up = [&](void* d, const void* s, size_t bytes) {
        return bytes ? cudaMemcpyAsync(d, s, bytes, cudaMemcpyHostToDevice, h->stream) : cudaSuccess;
    };
    ce = up(d_rec, sell.rec.data(), sell.rec.size());
    if (ce == cudaSuccess && use_stencil) ce = up(d_rec + dict_off, sten.dict.data(), dict_bytes);
    if (ce == cudaSuccess) ce = up(d_x, x, (size_t)NV * sizeof(double));
    if (ce == cudaSuccess) ce = cudaMemsetAsync(d_x + NV, 0, sizeof(double), h->stream);
    if (ce == cudaSuccess)
        ce = cudaMemsetAsync(base + L.vectors, 0, (size_t)n_vectors(modes) * align_up((size_t)(NV + 1) * batch * sizeof(double2)),
                             h->stream);
    // the slice_off slot holds the byte offsets of ragged tables, or the pattern ids of the stencil variant
    if (ce == cudaSuccess)
        ce = use_stencil ? up(d_sp, sten.pid.data(), sten.pid.size() * sizeof(int32_t))
                         : up(d_sp, sell.slice_off.data(), sell.slice_off.size() * sizeof(long long));
    if (ce == cudaSuccess) ce = cudaMemsetAsync(base + L.ticket, 0, 256, h->stream);
    if (ce == cudaSuccess) ce = cudaStreamSynchronize(h->stream);
    if (ce == cudaSuccess && !new_of_old.empty()) {
        ce = cudaMalloc((void**)&h->d_new_of_old, (size_t)N * sizeof(int32_t));
        if (ce == cudaSuccess) ce = cudaMalloc((void**)&h->d_old_of_new, (size_t)N * sizeof(int32_t));
        if (ce == cudaSuccess) ce = cudaMemcpy(h->d_new_of_old, new_of_old.data(), (size_t)N * sizeof(int32_t), cudaMemcpyHostToDevice);
        if (ce == cudaSuccess) ce = cudaMemcpy(h->d_old_of_new, old_of_new.data(), (size_t)N * sizeof(int32_t), cudaMemcpyHostToDevice);
    }
    if (ce == cudaSuccess) ce = cudaMallocHost((void**)&h->coef_host, (size_t)kCoefSlots * 2 * GPUQT_MAX_ORDER * sizeof(double));
    if (ce == cudaSuccess) ce = cudaMalloc((void**)&h->coef_dev, (size_t)kCoefSlots * 2 * GPUQT_MAX_ORDER * sizeof(double));
    for (int i = 0; i < kCoefSlots && ce == cudaSuccess; ++i) ce = cudaEventCreateWithFlags(&h->coef_event[i], cudaEventDisableTiming);
    if (ce != cudaSuccess) {
        const std::string why = cudaGetErrorString(ce);
        gpuqt_destroy(h);
        return bad(GPUQT_ERR_CUDA, "upload failed: " + why);
    }
    h->mat.rec = d_rec; h->mat.slice_off = d_sp; h->mat.x = d_x;
    h->mat.N = N; h->mat.NV = NV; h->mat.n_slices = sell.n_slices; h->mat.K = K_max; h->mat.uniform = sell.uniform;
    h->mat.cplx = h->cplx; h->mat.hop = h->hop; h->mat.hop_const = sell.hop_const;
    h->mat.inv_dE = 1.0 / energy_scale; h->mat.box = box_length;
    h->mat.pid = use_stencil ? (const int*)d_sp : nullptr;
    h->mat.dict = use_stencil ? (const int*)(d_rec + dict_off) : nullptr;
    // Shared-memory stages per warp: one round of a tile takes about one memory latency and a slice has
    // `batch / 2` rounds, so small batches need a deeper prefetch.
    int stages = opt.stages ? opt.stages : (batch == 1 ? 4 : batch == 2 ? 3 : 2);
    h->want_stages = std::max(1, std::min(stages, kMaxStages));
    // whole recurrences in one cooperative launch when a step is so short that launch gaps matter
    h->persistent = h->coop_ok && (opt.persistent == 1 || (opt.persistent == -1 && N * batch <= (int64_t)131072 * h->n_sm));
    h->alternate = opt.alternate;
    // tiles per CTA run: one tile per warp -- the finest granularity (load balance of short sweeps) and, measured,
    // never slower than longer runs (c4: 147.8 us per KPM step at 8, 149.2 at 16, 152.3 at 32; c5 indifferent)
    int run = opt.run ? opt.run : kWarps;
    h->run = std::max(1, run / kWarps) * kWarps;

    const size_t vstride = align_up((size_t)(NV + 1) * batch * sizeof(double2));
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
    h->stage_in = nextv();
    h->partials = (double*)(base + L.partials);
    h->dots = (double*)(base + L.dots);
    h->moments = (double*)(base + L.moments);
    h->ticket = (unsigned int*)(base + L.ticket);
    h->barrier = h->ticket + 32;
    rc = build_tensor_maps(h);
    if (rc != GPUQT_OK) {
        const std::string why = h->err;
        gpuqt_destroy(h);
        return bad(rc, why);
    }
    *out = h;
    return GPUQT_OK;
}
}  // namespace

extern "C" {

int gpuqt_set_state(gpuqt_handle* h, const double* phi_host) {
    if (!h || !phi_host) return fail(h, GPUQT_ERR_ARG, "null argument");
    CU(cudaMemcpyAsync(h->ring[0], phi_host, h->vec_elems * sizeof(double2), cudaMemcpyHostToDevice, h->stream));
    return finish_set_state(h, h->ring[0]);
}

int gpuqt_prefetch_state(gpuqt_handle* h, const double* phi_host) {
    if (!h || !phi_host) return fail(h, GPUQT_ERR_ARG, "null argument");
    if (!h->copy_stream) {
        CU(cudaStreamCreateWithFlags(&h->copy_stream, cudaStreamNonBlocking));
        CU(cudaEventCreateWithFlags(&h->ev_copy_done, cudaEventDisableTiming));
        CU(cudaEventCreateWithFlags(&h->ev_stage_free, cudaEventDisableTiming));
    }
    // the staging buffer may still be read by the layout kernel of the previous gpuqt_set_state_prefetched
    if (h->stage_read) CU(cudaStreamWaitEvent(h->copy_stream, h->ev_stage_free, 0));
    CU(cudaMemcpyAsync(h->stage_in, phi_host, h->vec_elems * sizeof(double2), cudaMemcpyHostToDevice, h->copy_stream));
    CU(cudaEventRecord(h->ev_copy_done, h->copy_stream));
    h->prefetched = true;
    return GPUQT_OK;
}

int gpuqt_set_state_prefetched(gpuqt_handle* h) {
    if (!h) return GPUQT_ERR_ARG;
    if (!h->prefetched) return fail(h, GPUQT_ERR_STATE, "gpuqt_prefetch_state has not been called since the last gpuqt_set_state_prefetched");
    CU(cudaStreamWaitEvent(h->stream, h->ev_copy_done, 0));
    int rc = finish_set_state(h, h->stage_in);
    if (rc) return rc;
    CU(cudaEventRecord(h->ev_stage_free, h->stream));     // psi = layout(stage_in) has been launched: the buffer is free after it
    h->stage_read = true;
    h->prefetched = false;
    return GPUQT_OK;
}

int gpuqt_set_state_device(gpuqt_handle* h, const double* phi_device) {
    if (!h || !phi_device) return fail(h, GPUQT_ERR_ARG, "null argument");
    CU(cudaMemcpyAsync(h->ring[0], phi_device, h->vec_elems * sizeof(double2), cudaMemcpyDeviceToDevice, h->stream));
    return finish_set_state(h, h->ring[0]);
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
    if (!h || order < 1 || order > GPUQT_MAX_ORDER || !std::isfinite(dt)) return fail(h, GPUQT_ERR_ARG, "bad dt or order");
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

int gpuqt_kpm_transform_damped(gpuqt_handle* h, int damping, double lambda, const double* moments_host,
                               int32_t n_moments, int32_t n_sets, const double* energies_host,
                               int32_t n_energies, double* out_host) {
    if (!h || !moments_host || !energies_host || !out_host || n_moments < 1 || n_sets < 1 || n_energies < 1)
        return fail(h, GPUQT_ERR_ARG, "null or non-positive argument");
    if (damping < GPUQT_DAMPING_JACKSON || damping > GPUQT_DAMPING_NONE ||
        (damping == GPUQT_DAMPING_LORENTZ && !(lambda > 0.0 && std::isfinite(lambda))))
        return fail(h, GPUQT_ERR_ARG, "unknown damping kernel or non-positive lambda");
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
        damping_kernel<<<(n_moments + 255) / 256, 256, 0, h->stream>>>(damping, lambda, n_moments, (double*)(s + og));
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

int gpuqt_kpm_transform(gpuqt_handle* h, const double* moments_host, int32_t n_moments,
                        int32_t n_sets, const double* energies_host, int32_t n_energies,
                        double* out_host) {
    return gpuqt_kpm_transform_damped(h, GPUQT_DAMPING_JACKSON, 0.0, moments_host, n_moments, n_sets, energies_host,
                                      n_energies, out_host);
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

int gpuqt_localization_length(gpuqt_handle* h, const double* length_host, int32_t n_times, int32_t n_energies,
                              double* xi_host, double* growth_host) {
    if (!h || !length_host || !xi_host || n_times < 1 || n_energies < 1) return fail(h, GPUQT_ERR_ARG, "null or non-positive argument");
    const size_t bl = (size_t)n_times * n_energies * sizeof(double), be = (size_t)n_energies * sizeof(double);
    const size_t ol = 0, ox = align_up(bl), og = ox + align_up(be), tot = og + align_up(be);
    CU(ensure_scratch(h, tot));
    char* s = h->scratch;
    cudaError_t e = cudaMemcpyAsync(s + ol, length_host, bl, cudaMemcpyHostToDevice, h->stream);
    if (e == cudaSuccess) {
        localization_kernel<<<(n_energies + 127) / 128, 128, 0, h->stream>>>(n_times, n_energies, (const double*)(s + ol),
                                                                             (double*)(s + ox), growth_host ? (double*)(s + og) : nullptr);
        e = cudaGetLastError();
    }
    if (e == cudaSuccess) e = cudaMemcpyAsync(xi_host, s + ox, be, cudaMemcpyDeviceToHost, h->stream);
    if (e == cudaSuccess && growth_host) e = cudaMemcpyAsync(growth_host, s + og, be, cudaMemcpyDeviceToHost, h->stream);
    if (e == cudaSuccess) e = cudaStreamSynchronize(h->stream);
    if (e != cudaSuccess) return cuda_fail(h, e, "localization_length");
    return GPUQT_OK;
}

int gpuqt_get_state(gpuqt_handle* h, int which, double* out_host) {
    if (!h || !out_host) return fail(h, GPUQT_ERR_ARG, "null argument");
    const double2* src = which == GPUQT_STATE_PSI ? h->psi : which == GPUQT_STATE_CHI ? h->chi
                       : which == GPUQT_STATE_VAC_A ? h->va : which == GPUQT_STATE_VAC_B ? h->vb : nullptr;
    if (!src) return fail(h, GPUQT_ERR_STATE, "state not available in this mode");
    const long long total = (long long)h->vec_elems;
    from_device_layout<<<(int)((total + 255) / 256), 256, 0, h->stream>>>(h->N, h->B, src, h->ring[0], h->d_old_of_new);
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
                                                                 (double*)(scratch + oi), (double*)(scratch + od),
                                                                 h->d_new_of_old, h->d_old_of_new);
    cudaError_t e = cudaGetLastError();
    if (e == cudaSuccess && col) e = cudaMemcpyAsync(col, scratch + oc, nk * 4, cudaMemcpyDeviceToHost, h->stream);
    if (e == cudaSuccess && re) e = cudaMemcpyAsync(re, scratch + orr, nk * 8, cudaMemcpyDeviceToHost, h->stream);
    if (e == cudaSuccess && im) e = cudaMemcpyAsync(im, scratch + oi, nk * 8, cudaMemcpyDeviceToHost, h->stream);
    if (e == cudaSuccess && dx) e = cudaMemcpyAsync(dx, scratch + od, nk * 8, cudaMemcpyDeviceToHost, h->stream);
    if (e == cudaSuccess) e = cudaStreamSynchronize(h->stream);
    if (e != cudaSuccess) return cuda_fail(h, e, "get_table");
    return GPUQT_OK;
}

int gpuqt_get_info(gpuqt_handle* h, int what, int64_t* value) {
    if (!h || !value) return GPUQT_ERR_ARG;
    switch (what) {
    case GPUQT_INFO_STORED_MATRIX_BYTES: *value = (int64_t)h->stored_matrix_bytes; break;
    case GPUQT_INFO_HOP_VARIANT: *value = h->hop; break;
    case GPUQT_INFO_UNIFORM: *value = h->mat.uniform; break;
    case GPUQT_INFO_UNROLLED_WIDTH: *value = h->kt; break;
    case GPUQT_INFO_SMALL_PATH: *value = small_ok(h) ? 1 : 0; break;
    case GPUQT_INFO_PERSISTENT: *value = h->persistent; break;
    case GPUQT_INFO_WORKSPACE_USED: *value = (int64_t)h->workspace_used; break;
    case GPUQT_INFO_SMALL_PATH_MSD: *value = small_msd_ok(h) ? 1 : 0; break;
    case GPUQT_INFO_STENCIL_PATTERNS: *value = h->stencil_patterns; break;
    case GPUQT_INFO_REORDERED: *value = h->d_old_of_new ? 1 : 0; break;
    default: return fail(h, GPUQT_ERR_ARG, "unknown info key");
    }
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

const char* gpuqt_last_error(const gpuqt_handle* h) { return h ? h->err.c_str() : g_create_error.c_str(); }

void gpuqt_destroy(gpuqt_handle* h) {
    if (!h) return;
    cudaStreamSynchronize(h->stream);
    flush_stats(h);
    for (auto e : h->free_events) cudaEventDestroy(e);
    for (auto e : h->coef_event)
        if (e) cudaEventDestroy(e);
    if (h->coef_host) cudaFreeHost(h->coef_host);
    if (h->coef_dev) cudaFree(h->coef_dev);
    if (h->scratch) cudaFree(h->scratch);
    if (h->d_maps) cudaFree(h->d_maps);
    if (h->d_new_of_old) cudaFree(h->d_new_of_old);
    if (h->d_old_of_new) cudaFree(h->d_old_of_new);
    if (h->copy_stream) {
        cudaStreamSynchronize(h->copy_stream);
        cudaStreamDestroy(h->copy_stream);
    }
    if (h->ev_copy_done) cudaEventDestroy(h->ev_copy_done);
    if (h->ev_stage_free) cudaEventDestroy(h->ev_stage_free);
    delete h;
}

}  // extern "C"

#include "slab_group.inl"
