// gpuqt_kpm_transform_static (include/gpuqt.h): the KPM damping + energy transform (Eq. 25-27,
// :203 Eq. 31) for callers that must not allocate device memory.
//
// Who this is for.  The ordinary gpuqt_kpm_transform keeps its working memory (staged inputs, the table of damping
// factors, the staged output) in a buffer the handle obtains with cudaMalloc and grows on demand.  That is a
// problem for a caller
//   * whose process has already handed the whole card to a memory pool or a framework's caching allocator, so a
//     cudaMalloc issued behind its back fails or pushes the pool into an out-of-memory retry;
//   * that runs inside a latency-sensitive loop (cudaMalloc and cudaFree serialise with all work on the device
//     and can stall other streams for milliseconds);
//   * that is confined to a fixed memory budget by its scheduler (MPS memory limits, MIG slices sized to the job)
//     and has to account for every byte before the run starts.
// Such a caller brings the inputs and the output as DEVICE buffers it already owns; the only memory the transform
// needs beyond them -- the table gs[n] = g_n (2 - delta_n0) that the damping kernel writes and the transform
// kernel reads, plus one status word -- lives in a file-scope `static __device__` array below.  Its size is fixed
// when the library is built: GPUQT_STATIC_MAX_MOMENTS doubles + 256 bytes = 128.25 KB, which every GPU that loads
// libgpuqt.so holds from module load until the process exits, whether this entry point is used or not.
//
// This file is self-contained on purpose: the array has internal linkage, so the kernels that use it, the host
// code that looks up its device address and the entry point all have to be in this one translation unit.  It
// shares no state with gpuqt.cu and needs no handle.
#include <cuda_runtime.h>

#include <cmath>
#include <cstdarg>
#include <cstdio>
#include <mutex>

#include "../../include/gpuqt.h"

namespace {

constexpr size_t kTableBytes = (size_t)GPUQT_STATIC_MAX_MOMENTS * sizeof(double);
constexpr size_t kStatusOffset = kTableBytes;          // one unsigned int, in a 256-byte line of its own
constexpr size_t kScratchBytes = kTableBytes + 256;

// The scratch.  In HOST code the name `g_static_scratch` is only a stand-in the runtime uses to identify the
// symbol; it is not a device address and must never be handed to a kernel.  Host code gets the real address
// from cudaGetSymbolAddress (scratch_address below).
static __device__ __align__(256) unsigned char g_static_scratch[kScratchBytes];

// Device address of g_static_scratch on each device, looked up once per device.
constexpr int kMaxDevices = 64;
std::mutex g_setup_mutex;
unsigned char* g_scratch_on_device[kMaxDevices] = {nullptr};

// Set-up, once per device, with that device current: ask the runtime where the array lives there.  Runs inside
// the first call of the entry point on a device.
cudaError_t scratch_address(unsigned char** out) {
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    if (dev < 0 || dev >= kMaxDevices) return cudaErrorInvalidDevice;
    std::lock_guard<std::mutex> lock(g_setup_mutex);
    if (!g_scratch_on_device[dev]) {
        void* p = nullptr;
        e = cudaGetSymbolAddress(&p, g_static_scratch);
        if (e != cudaSuccess) return e;
        if (!p) return cudaErrorInvalidSymbol;
        g_scratch_on_device[dev] = static_cast<unsigned char*>(p);
    }
    *out = g_scratch_on_device[dev];
    return cudaSuccess;
}

// gs[n] = g_n (2 - delta_n0) into the static table (same three kernels g_n as gpuqt_kpm_transform_damped), and the
// status word back to zero: the array keeps whatever the previous call left in it, and the transform kernel below
// only ever ORs bits into the word.  The table needs no clearing -- entries n < n_moments are all rewritten, the
// rest are not read.
__global__ void damping_static_kernel(int kind, double lambda, int n_moments, double* __restrict__ gs,
                                      unsigned int* __restrict__ status) {
    const int n = blockIdx.x * blockDim.x + threadIdx.x;
    if (n == 0) *status = 0u;
    if (n >= n_moments) return;
    double g = 1.0;
    if (kind == GPUQT_DAMPING_JACKSON) {                        // Eq. 31
        const double alpha = 1.0 / (n_moments + 1.0);
        double s, c, s1, c1;
        sincospi(n * alpha, &s, &c);
        sincospi(alpha, &s1, &c1);
        g = (1.0 - n * alpha) * c + alpha * s * (c1 / s1);
    } else if (kind == GPUQT_DAMPING_LORENTZ) {
        g = sinh(lambda * (1.0 - (double)n / (double)n_moments)) / sinh(lambda);
    }
    gs[n] = (n == 0) ? g : 2.0 * g;
}

// out[s][j] = 2 / (pi Omega dE sqrt(1 - e^2)) sum_n gs[n] T_n(e) C[s][n], e = E_j / dE, by Clenshaw summation
// (Eq. 25-27); one thread per (set, energy).  The energies are device data here, so the range check the ordinary
// call does on the host (|e| < 1) is done by the thread: it raises bit 0 of the status word and
// writes NaN.
__global__ void transform_static_kernel(int n_moments, int n_sets, int n_energies, const double* __restrict__ gs,
                                        const double* __restrict__ C, const double* __restrict__ energies,
                                        double inv_dE, double volume, double* __restrict__ out,
                                        unsigned int* __restrict__ status) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n_sets * n_energies) return;
    const int s = i / n_energies, j = i % n_energies;
    const double e = energies[j] * inv_dE;
    if (!(fabs(e) < 1.0)) {
        atomicOr(status, 1u);
        out[i] = nan("");
        return;
    }
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

int fail(char* err_text, size_t err_bytes, int code, const char* fmt, ...) {
    if (err_text && err_bytes) {
        va_list ap;
        va_start(ap, fmt);
        vsnprintf(err_text, err_bytes, fmt, ap);
        va_end(ap);
    }
    return code;
}

}  // namespace

extern "C" int gpuqt_kpm_transform_static(int damping, double lambda, const double* moments_device, int32_t n_moments,
                                          int32_t n_sets, const double* energies_device, int32_t n_energies,
                                          double energy_scale, double volume, double* out_device, void* cuda_stream,
                                          char* err_text, size_t err_text_bytes) {
    if (err_text && err_text_bytes) err_text[0] = '\0';
    if (!moments_device || !energies_device || !out_device || n_moments < 1 || n_sets < 1 || n_energies < 1)
        return fail(err_text, err_text_bytes, GPUQT_ERR_ARG, "null or non-positive argument");
    if (n_moments > GPUQT_STATIC_MAX_MOMENTS)
        return fail(err_text, err_text_bytes, GPUQT_ERR_NOMEM,
                    "n_moments = %d exceeds the static table of GPUQT_STATIC_MAX_MOMENTS = %d entries; use "
                    "gpuqt_kpm_transform (which allocates) or fewer moments", (int)n_moments, GPUQT_STATIC_MAX_MOMENTS);
    if ((long long)n_sets * n_energies > 0x7fffffffLL)
        return fail(err_text, err_text_bytes, GPUQT_ERR_ARG, "n_sets * n_energies must fit 31 bits");
    if (damping < GPUQT_DAMPING_JACKSON || damping > GPUQT_DAMPING_NONE ||
        (damping == GPUQT_DAMPING_LORENTZ && !(lambda > 0.0 && std::isfinite(lambda))))
        return fail(err_text, err_text_bytes, GPUQT_ERR_ARG, "unknown damping kernel or non-positive lambda");
    if (!(energy_scale > 0.0 && std::isfinite(energy_scale)) || !(volume > 0.0 && std::isfinite(volume)))
        return fail(err_text, err_text_bytes, GPUQT_ERR_ARG, "energy_scale and volume must be positive");

    unsigned char* scratch = nullptr;                          // DEVICE address of g_static_scratch on this device
    cudaError_t e = scratch_address(&scratch);
    if (e != cudaSuccess)
        return fail(err_text, err_text_bytes, GPUQT_ERR_CUDA, "cudaGetSymbolAddress(static scratch): %s", cudaGetErrorString(e));
    double* gs = reinterpret_cast<double*>(scratch);
    unsigned int* status = reinterpret_cast<unsigned int*>(scratch + kStatusOffset);

    cudaStream_t stream = static_cast<cudaStream_t>(cuda_stream);
    damping_static_kernel<<<(n_moments + 255) / 256, 256, 0, stream>>>(damping, lambda, n_moments, gs, status);
    const int total = n_sets * n_energies;
    transform_static_kernel<<<(total + 127) / 128, 128, 0, stream>>>(n_moments, n_sets, n_energies, gs, moments_device,
                                                                     energies_device, 1.0 / energy_scale, volume,
                                                                     out_device, status);
    e = cudaGetLastError();
    unsigned int raised = 0;                                   // four bytes to the caller's stack: no allocation
    if (e == cudaSuccess) e = cudaMemcpyAsync(&raised, status, sizeof(raised), cudaMemcpyDeviceToHost, stream);
    if (e == cudaSuccess) e = cudaStreamSynchronize(stream);
    if (e != cudaSuccess) return fail(err_text, err_text_bytes, GPUQT_ERR_CUDA, "kpm_transform_static: %s", cudaGetErrorString(e));
    if (raised & 1u)
        return fail(err_text, err_text_bytes, GPUQT_ERR_ENERGY, "energy point outside (-energy_scale, energy_scale)");
    return GPUQT_OK;
}
