// sm_100a kernels of the GPUQT hot path.  See include/gpuqt.h for the boundary and DESIGN.md for
// the layout, the byte model and the roofline of each kernel.
//
// Layout
//   vectors   complex fp64 [N][B] as double2: the B vectors of a row are contiguous (16*B bytes),
//             so one neighbour index serves one 16*B-byte gather (B = 8: one 128-byte line).
//   matrix    sliced ELL, slices of 32 rows, column-major inside a slice:
//             entry(row, k) = slice_ptr[row / 32] + k * 32 + row % 32
//             int32 col[], fp64 hre[], fp64 him[] (complex variant only), padding = (own row, 0).
//   thread    one thread per (row, b): tid -> row = tid / B, b = tid % B.  Own-row vector
//             loads/stores of a warp are one contiguous 512-byte segment.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace gpuqt {

constexpr int kThreads = 256;
constexpr int kSlice = 32;

struct Mat {
    const int32_t* __restrict__ col;
    const double* __restrict__ hre;
    const double* __restrict__ him;       // null in the real variant
    const double* __restrict__ onsite;    // [N]
    const double* __restrict__ x;         // [N]
    const long long* __restrict__ slice_ptr;  // [n_slices + 1], entry offsets (multiples of 32)
    long long N;
    int K;                                // K_max
    int uniform;                          // every slice has width K
    double inv_dE;
    double box;                           // <= 0: open boundary
};

enum Mode : int {
    kModeDoubling = 0,   // T_new, dots |T_new|^2, Re<T_new|T_in>, |T_in|^2          (Eq. 28, 30)
    kModeLeft = 1,       // T_new, dot <phi_L|T_new>                                 (Eq. 29)
    kModeEvolve = 2,     // T_new, acc += c T_new                                    (Eq. 17, 21)
    kModeEvolveMsd = 3,  // (a, e) pair with the [X,H~] weights in the same walk     (Eq. 18, 22)
};

struct StepArgs {
    const double2* __restrict__ in;      // T_{m-1}: gathered and own row
    const double2* __restrict__ prev;    // T_{m-2}: own row (unused when first)
    double2* __restrict__ out;           // T_m (unused when !store)
    const double2* __restrict__ in_e;    // MSD pair: e_{m-1}
    const double2* __restrict__ prev_e;  //           e_{m-2}
    double2* __restrict__ out_e;         //           e_m
    double2* __restrict__ acc;           // evolve: sum_m c_m T_m
    double2* __restrict__ acc_e;         // evolve MSD: sum_m c_m e_m
    const double2* __restrict__ phiL;    // kModeLeft
    double cr, ci;                       // c_m
    double c0r, c0i;                     // c_0, used when first (acc = c_0 T_0 + c_1 T_1)
    int first;                           // T_1 = H~ T_0 (no factor 2, no prev)
    int store;                           // write T_m (0 on the last term of an evolve)
    double* partials;                    // [grid][Q*B]
    unsigned int* ticket;
    double* result;                      // [Q][B] reduced dots of this launch
};

__device__ __forceinline__ double2 ldcs2(const double2* p) {
    return __ldcs(p);
}

// minimum-image X_n - X_m  [A6]; pure add/sub so it is bit-identical to the oracle's
__device__ __forceinline__ double min_image(double d, double box) {
    if (box > 0.0) {
        if (d > 0.5 * box) d -= box;
        else if (d < -0.5 * box) d += box;
    }
    return d;
}

// Deterministic reduction of Q*B per-thread values: warp shuffle over lanes with equal b ->
// shared memory over warps -> per-block partial -> the last block to finish sums the per-block
// partials in a fixed order (no floating-point atomics, run-to-run identical).
template <int B, int Q>
__device__ __forceinline__ void block_reduce_and_finish(double (&v)[Q], double* partials,
                                                        unsigned int* ticket, double* result) {
    constexpr int kWarps = kThreads / 32;
    __shared__ double s_part[kWarps][Q * B];
    __shared__ double s_tree[kThreads];
    __shared__ int s_last;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
#pragma unroll
    for (int q = 0; q < Q; ++q) {
#pragma unroll
        for (int off = 16; off >= B; off >>= 1) v[q] += __shfl_xor_sync(0xffffffffu, v[q], off);
    }
    if (lane < B) {
#pragma unroll
        for (int q = 0; q < Q; ++q) s_part[warp][q * B + lane] = v[q];
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

// One Chebyshev recurrence step fused with what consumes it.
template <int B, int KT, bool CPLX, int MODE>
__global__ void __launch_bounds__(kThreads) cheb_step_kernel(const Mat m, const StepArgs a) {
    constexpr int Q = (MODE == kModeDoubling) ? 3 : 2;
    constexpr int kRows = kThreads / B;
    const int tid = threadIdx.x;
    const int b = tid % B;
    const int rl = tid / B;
    double red[Q];
#pragma unroll
    for (int q = 0; q < Q; ++q) red[q] = 0.0;
    const long long n_chunks = (m.N + kRows - 1) / kRows;
    const double scale = a.first ? m.inv_dE : 2.0 * m.inv_dE;

    for (long long chunk = blockIdx.x; chunk < n_chunks; chunk += gridDim.x) {
        const long long row = chunk * kRows + rl;
        if (row >= m.N) continue;
        const size_t vi = (size_t)row * B + b;
        long long e0;
        int w;
        if (KT > 0) {
            e0 = (row >> 5) * (long long)(KT * kSlice) + (row & 31);
            w = KT;
        } else {
            const long long s0 = m.slice_ptr[row >> 5], s1 = m.slice_ptr[(row >> 5) + 1];
            e0 = s0 + (row & 31);
            w = (int)((s1 - s0) >> 5);
        }
        const double2 self = a.in[vi];
        const double u = __ldcs(&m.onsite[row]);
        double sr = u * self.x, si = u * self.y;
        double er = 0.0, ei = 0.0;     // H~ e_{m-1}
        double xr = 0.0, xi = 0.0;     // [X,H] a_{m-1}
        double2 self_e = make_double2(0.0, 0.0);
        double xm = 0.0;
        if (MODE == kModeEvolveMsd) {
            self_e = a.in_e[vi];
            er = u * self_e.x;
            ei = u * self_e.y;
            xm = m.x[row];
        }
        auto body = [&](int k) {
            const long long e = e0 + (long long)k * kSlice;
            const int c = __ldcs(&m.col[e]);
            const double hr = __ldcs(&m.hre[e]);
            double hi = 0.0;
            if (CPLX) hi = __ldcs(&m.him[e]);
            const double2 v = a.in[(size_t)c * B + b];
            sr = fma(hr, v.x, sr);
            si = fma(hr, v.y, si);
            if (CPLX) {
                sr = fma(-hi, v.y, sr);
                si = fma(hi, v.x, si);
            }
            if (MODE == kModeEvolveMsd) {
                const double2 ve = a.in_e[(size_t)c * B + b];
                er = fma(hr, ve.x, er);
                ei = fma(hr, ve.y, ei);
                if (CPLX) {
                    er = fma(-hi, ve.y, er);
                    ei = fma(hi, ve.x, ei);
                }
                // [X,H]_mn = (X_m - X_n) H_mn = -dx H_mn
                const double ndx = -min_image(m.x[c] - xm, m.box);
                const double wr = ndx * hr;
                xr = fma(wr, v.x, xr);
                xi = fma(wr, v.y, xi);
                if (CPLX) {
                    const double wi = ndx * hi;
                    xr = fma(-wi, v.y, xr);
                    xi = fma(wi, v.x, xi);
                }
            }
        };
        if (KT > 0) {
#pragma unroll
            for (int k = 0; k < KT; ++k) body(k);
        } else {
            for (int k = 0; k < w; ++k) body(k);
        }
        double2 t;   // T_m
        t.x = scale * sr;
        t.y = scale * si;
        if (!a.first) {
            const double2 p = ldcs2(&a.prev[vi]);
            t.x -= p.x;
            t.y -= p.y;
        }
        if (a.store) a.out[vi] = t;
        if (MODE == kModeDoubling) {
            red[0] += t.x * t.x + t.y * t.y;
            red[1] += t.x * self.x + t.y * self.y;
            red[2] += self.x * self.x + self.y * self.y;
        } else if (MODE == kModeLeft) {
            const double2 l = ldcs2(&a.phiL[vi]);
            red[0] += l.x * t.x + l.y * t.y;       // conj(l) * t
            red[1] += l.x * t.y - l.y * t.x;
        } else {
            double2 acc;
            if (a.first) {
                acc.x = a.c0r * self.x - a.c0i * self.y;
                acc.y = a.c0r * self.y + a.c0i * self.x;
            } else {
                acc = a.acc[vi];
            }
            acc.x += a.cr * t.x - a.ci * t.y;
            acc.y += a.cr * t.y + a.ci * t.x;
            a.acc[vi] = acc;
            if (MODE == kModeEvolveMsd) {
                double2 te;
                te.x = scale * (er + xr);
                te.y = scale * (ei + xi);
                if (!a.first) {
                    const double2 p = ldcs2(&a.prev_e[vi]);
                    te.x -= p.x;
                    te.y -= p.y;
                }
                if (a.store) a.out_e[vi] = te;
                double2 ae;
                if (a.first) {
                    ae.x = a.c0r * self_e.x - a.c0i * self_e.y;
                    ae.y = a.c0r * self_e.y + a.c0i * self_e.x;
                } else {
                    ae = a.acc_e[vi];
                }
                ae.x += a.cr * te.x - a.ci * te.y;
                ae.y += a.cr * te.y + a.ci * te.x;
                a.acc_e[vi] = ae;
            }
        }
    }
    if (MODE == kModeDoubling || MODE == kModeLeft)
        block_reduce_and_finish<B, Q>(red, a.partials, a.ticket, a.result);
}

// out = V in,  V_mn = i (X_n - X_m) H_mn  (Eq. 34) — not scaled by 1/dE, no on-site
template <int B, int KT, bool CPLX>
__global__ void __launch_bounds__(kThreads) velocity_kernel(const Mat m, const double2* __restrict__ in,
                                                            double2* __restrict__ out) {
    constexpr int kRows = kThreads / B;
    const int tid = threadIdx.x, b = tid % B, rl = tid / B;
    const long long n_chunks = (m.N + kRows - 1) / kRows;
    for (long long chunk = blockIdx.x; chunk < n_chunks; chunk += gridDim.x) {
        const long long row = chunk * kRows + rl;
        if (row >= m.N) continue;
        long long e0;
        int w;
        if (KT > 0) {
            e0 = (row >> 5) * (long long)(KT * kSlice) + (row & 31);
            w = KT;
        } else {
            const long long s0 = m.slice_ptr[row >> 5], s1 = m.slice_ptr[(row >> 5) + 1];
            e0 = s0 + (row & 31);
            w = (int)((s1 - s0) >> 5);
        }
        const double xm = m.x[row];
        double sr = 0.0, si = 0.0;
        auto body = [&](int k) {
            const long long e = e0 + (long long)k * kSlice;
            const int c = __ldcs(&m.col[e]);
            const double dx = min_image(m.x[c] - xm, m.box);
            const double wr = dx * __ldcs(&m.hre[e]);
            const double2 v = in[(size_t)c * B + b];
            sr = fma(wr, v.x, sr);
            si = fma(wr, v.y, si);
            if (CPLX) {
                const double wi = dx * __ldcs(&m.him[e]);
                sr = fma(-wi, v.y, sr);
                si = fma(wi, v.x, si);
            }
        };
        if (KT > 0) {
#pragma unroll
            for (int k = 0; k < KT; ++k) body(k);
        } else {
            for (int k = 0; k < w; ++k) body(k);
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
__global__ void zero_vec(long long n, double2* __restrict__ v) {
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) v[i] = make_double2(0.0, 0.0);
}

// Doubling identity (T_2m = 2 T_m^2 - 1, T_2m+1 = 2 T_m+1 T_m - T_1):
// dots[j] = {<a_{j+1}|a_{j+1}>, Re<a_{j+1}|a_j>, <a_j|a_j>}[B]  ->  C[b][n]
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

// Decode the sliced-ELL table back to canonical padded row-major arrays (bit-exact check)
__global__ void decode_table(const Mat m, int32_t* __restrict__ col, double* __restrict__ re,
                             double* __restrict__ im, double* __restrict__ dx) {
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= m.N * m.K) return;
    const long long row = i / m.K;
    const int k = (int)(i % m.K);
    const long long s0 = m.slice_ptr[row >> 5], s1 = m.slice_ptr[(row >> 5) + 1];
    const int w = (int)((s1 - s0) >> 5);
    int c = (int)row;
    double hr = 0.0, hi = 0.0, d = 0.0;
    if (k < w) {
        const long long e = s0 + (long long)k * kSlice + (row & 31);
        c = m.col[e];
        hr = m.hre[e];
        if (m.him) hi = m.him[e];
        d = min_image(m.x[c] - m.x[row], m.box);
    }
    if (col) col[i] = c;
    if (re) re[i] = hr;
    if (im) im[i] = hi;
    if (dx) dx[i] = d;
}

}  // namespace gpuqt
