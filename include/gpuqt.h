/*
 * gpuqt.h — C-ABI boundary of the B200-native GPUQT hot path (arXiv 1705.01387).
 *
 * One opaque handle owns a tight-binding Hamiltonian in sliced-ELL form on ONE GPU plus the state
 * vectors of a batch of random-phase vectors.  Every arithmetic step of the path (SpMV, Chebyshev
 * recurrences, commutator recursion, velocity apply, inner products, moment finalisation, Jackson
 * damping and energy transform) runs in hand-written sm_100a CUDA kernels; the host side only
 * validates, lays out memory, computes the N_p Bessel coefficients of one time step, and launches.
 * There is no CPU fallback: without a CUDA device every compute call returns GPUQT_ERR_CUDA.
 *
 * Citations are PAPER.md:<line> (= /root/reference/PAPER.md at build time, the text of the paper)
 * plus the equation.  Readings of silent points are marked [A#] and listed in DESIGN.md.
 *
 * Conventions
 *   N        number of orbitals (sites);  K_max  max neighbours per row
 *   batch    number of random vectors B processed together (B in {1, 2, 4, 8})
 *   dE       energy scale "energy_max", H~ = H / dE  (PAPER.md:160 Eq. 19, :329)
 *   hbar = 1
 *   complex vectors cross the ABI as interleaved doubles (re, im):  [batch][N][2]
 *   "host"   pointer to host memory (pageable or pinned);  "device" pointer to device memory
 *
 * Ownership: the caller owns every array it passes and the device workspace; gpuqt_create copies
 * the host inputs and keeps no host pointer.  Results are written to caller-allocated buffers and
 * are complete when the call returns (the call synchronises the stream).  All vectors and the
 * matrix live in the caller's workspace; the handle itself owns only small objects (the TMA tensor
 * maps of the vector buffers, a grow-on-demand device scratch buffer for gpuqt_kpm_transform /
 * gpuqt_running_conductivity / gpuqt_get_table, a few KB of pinned host memory and its device mirror
 * for the Bessel coefficients of a time step, the copy stream and two events of gpuqt_prefetch_state,
 * and -- for a lattice stored in brick order, gpuqt_options.reorder -- two int32[N] device arrays with
 * the site permutation), which gpuqt_destroy frees together with the handle; the workspace stays the
 * caller's.
 *
 * Errors: every call returns a gpuqt_status (0 = ok, < 0 = error); nothing throws, aborts or prints
 * across the ABI; the handle stays valid after an error; gpuqt_last_error(handle) gives text, and
 * gpuqt_last_error(NULL) the text of the last failed gpuqt_create on the calling thread.
 *
 * Threading: a handle is not thread-safe; all work is issued on the stream given at create.
 */
#ifndef GPUQT_H
#define GPUQT_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct gpuqt_handle gpuqt_handle;

typedef enum {
    GPUQT_OK = 0,
    GPUQT_ERR_ARG = -1,            /* null/negative/unsupported argument                          */
    GPUQT_ERR_INDEX = -2,          /* neighbour count or index out of range  [A11]                */
    GPUQT_ERR_NOT_HERMITIAN = -3,  /* H_nm != conj(H_mn) bit-exactly  [A10]                       */
    GPUQT_ERR_SCALE = -4,          /* Gershgorin bound of H exceeds dE  [A9]        */
    GPUQT_ERR_ENERGY = -5,         /* |E / dE| >= 1 in the transform  [A15]         */
    GPUQT_ERR_STATE = -6,          /* call order / mode not enabled at create                     */
    GPUQT_ERR_CUDA = -7,           /* CUDA runtime error or no device                             */
    GPUQT_ERR_NOMEM = -8,          /* workspace too small or host allocation failed               */
    GPUQT_ERR_POSITION = -9        /* |X_n - X_m| == box/2 on a non-zero hop: ambiguous image [A6]*/
} gpuqt_status;

/* modes (bit mask) — which branches gpuqt_evolve advances */
#define GPUQT_MODE_VAC 1   /* a = U(t)^dagger phi, b = U(t)^dagger V phi       (Eq. 29)  [A1]     */
#define GPUQT_MODE_MSD 2   /* psi = U(t) phi and chi = [X, U(t)] phi            (Eq. 30)  [A3]     */
#define GPUQT_MODE_PSI 4   /* psi = U(t) phi alone (implied by MSD; plain time evolution)         */

/* state selectors for gpuqt_get_state */
#define GPUQT_STATE_PSI 0
#define GPUQT_STATE_CHI 1
#define GPUQT_STATE_VAC_A 2
#define GPUQT_STATE_VAC_B 3

/* kernel classes for gpuqt_kernel_stats */
#define GPUQT_KERNEL_KPM_DOUBLING 0  /* fused SpMV + recurrence + 2 dots (DOS, MSD moments)       */
#define GPUQT_KERNEL_KPM_LEFT 1      /* fused SpMV + recurrence + <phi_L|.> (VAC moments)         */
#define GPUQT_KERNEL_EVOLVE 2        /* fused SpMV + Clenshaw recurrence with the Bessel weights   */
#define GPUQT_KERNEL_EVOLVE_MSD 3    /* the same for (psi, chi) with the [X,H~] walk fused in     */
#define GPUQT_KERNEL_VELOCITY 4      /* V apply                                                   */
#define GPUQT_KERNEL_CLASSES 5

#define GPUQT_MAX_MOMENTS 16384
#define GPUQT_MAX_ORDER 4096         /* largest N_p of one gpuqt_evolve call                          */

/* Tuning options of gpuqt_create_with_options.  gpuqt_default_options fills in the defaults, which are
 * what gpuqt_create uses and what bench.py times; nothing is read from the environment.
 *   struct_bytes   sizeof(gpuqt_options) as the caller compiled it (set by gpuqt_default_options)
 *   stages         shared-memory pipeline stages per warp, 1..4;            0 = by batch (4, 3, 2, 2)
 *   blocks_per_sm  cap on resident CTAs per SM;                             0 = what fits
 *   run            consecutive tiles a CTA walks before it jumps (rounded to a multiple of 8);   0 = 8
 *   alternate      1: the sweep direction alternates between recurrence steps (L2 reuse across the
 *                  step boundary)
 *   hop_const      1: store no hopping array when every listed hopping is the same real number
 *   idx16          1: 16-bit (base + delta) columns where the table allows it
 *   small          1: one-CTA whole-recurrence kernel when matrix and vectors fit one SM's shared memory
 *   persistent     whole recurrences in ONE cooperative launch with grid-wide barriers between the
 *                  steps: 1 always, 0 never, -1 when a whole recurrence is short enough to be one kernel
 *                  (N * batch <= 131072 rows per SM: a step of at most a few hundred microseconds)
 *   stencil        implicit stencil for constant-hopping tables of regular lattices ("all
 *                  hopping integrals ... are -1", the lattices of PAPER.md:359, :381): no index array is
 *                  streamed; the distinct per-slice patterns of relative columns are kept in a small
 *                  dictionary and a slice names its pattern.  1: when the dictionary is at most 1/16 of
 *                  the index array (and <= 8 MB) AND batch >= 4 AND a recurrence step's working set (three
 *                  vector sets + the table) exceeds the L2 cache, i.e. when the index array would come from
 *                  HBM in every step and a tile streams enough bytes to pay for the extra copies;
 *                  0: never; 2: whenever the table is uniform (tests)
 *   reorder        site reordering for locality: a simple-cubic periodic lattice in natural order (every row with its
 *                  six nearest neighbours, any order; Lx, Ly multiples of 4, Lz even -- the 3-D Anderson model of
 *                  PAPER.md:353-355) is stored in bricks of 4 x 4 x 2 sites per 32-row slice, so that four instead of
 *                  two of a row's six neighbours lie in its own slice.  Invisible at the boundary: states, tables and
 *                  moments are exchanged in the caller's numbering.  1: at batch >= 4 when a recurrence step's working
 *                  set exceeds the L2 (the rule of `stencil`); 0: never;
 *                  2: whenever the lattice is recognised (tests)                                          */
typedef struct gpuqt_options {
    int32_t struct_bytes;
    int32_t stages;
    int32_t blocks_per_sm;
    int32_t run;
    int32_t alternate;
    int32_t hop_const;
    int32_t idx16;
    int32_t small;
    int32_t persistent;
    int32_t stencil;
    int32_t reorder;
} gpuqt_options;
void gpuqt_default_options(gpuqt_options* opt);

/* Bytes of device workspace gpuqt_create needs for this problem (0 on invalid arguments): an upper
 * bound that holds for every storage variant (every slice record padded to K_max, per-entry fp64
 * hoppings, int32 columns).                                                                       */
size_t gpuqt_workspace_bytes(int64_t N, int32_t K_max, int is_complex, int32_t batch, int modes);

/* Host-only validation of the four input data sets: argument sanity, index range
 * [A11], bit-exact Hermiticity [A10], Gershgorin bound max_m(|U_m| + sum_k |H_mk|) <= dE [A9],
 * unambiguous minimum image [A6].  Uses no GPU.  Same checks gpuqt_create runs.                  */
int gpuqt_validate(int64_t N, int32_t K_max, const int32_t* nbr_count, const int32_t* nbr_index,
                   const double* hop_re, const double* hop_im, const double* onsite,
                   const double* x, double box_length, double energy_scale);

/* Host only, no GPU: the storage variant gpuqt_create would choose for this table and batch under `options`
 * (NULL = defaults) on a device with l2_bytes of L2 cache (0 = B200's 126 MB), and the bytes it takes on the
 * device ("waste memory" is about exactly this).
 * hop_variant as GPUQT_INFO_HOP_VARIANT, stored_matrix_bytes as
 * GPUQT_INFO_STORED_MATRIX_BYTES, stencil_patterns as GPUQT_INFO_STENCIL_PATTERNS; any output may be NULL.
 * Checks counts and index range only (GPUQT_ERR_INDEX); run gpuqt_validate for the full checks.     */
int gpuqt_plan_storage(int64_t N, int32_t K_max, const int32_t* nbr_count, const int32_t* nbr_index,
                       const double* hop_re, const double* hop_im, int32_t batch, int64_t l2_bytes,
                       const gpuqt_options* options, int32_t* hop_variant, int64_t* stored_matrix_bytes,
                       int64_t* stencil_patterns);

/* Build the model on the GPU.
 *   nbr_count  host [N]          number of neighbours of site m
 *   nbr_index  host [N*K_max]    row-major, 0-based; slots >= count ignored  PAPER.md:244 [A11]
 *   hop_re     host [N*K_max] or NULL => every hopping is -1
 *   hop_im     host [N*K_max] or NULL => real-hopping variant
 *   onsite     host [N] or NULL => 0
 *   x          host [N]          transport-direction coordinate X_m          PAPER.md:271, Eq. 33
 *   box_length length of the periodic box along x (<= 0: open boundary) and
 *   volume     Omega, the two numbers of line 1 of position.in
 *   energy_scale dE
 *   batch      B in {1,2,4,8};  modes: GPUQT_MODE_* mask
 *   workspace  device memory of at least gpuqt_workspace_bytes(...) bytes, 256-byte aligned,
 *              owned by the caller and alive until gpuqt_destroy
 *   cuda_stream a cudaStream_t (NULL = default stream)
 * Storage: slices of 32 rows, one packed record per slice, column-major inside it.
 * Per-entry variants: SoA fp64 hoppings (imaginary plane absent when hop_im == NULL) + int32 columns,
 * padding entries = (own row, 0.0).  When hop_im == NULL and every listed hopping has the same bit
 * pattern (the paper's default "all hoppings -1") no hopping array is stored and
 * padding entries point at an all-zero row N that every vector buffer carries; such a table keeps
 * its columns as int32 base + uint16 delta per (slice, k) when they spread less than 65535 there
 * (0xffff = the zero row, for tables with padding entries), or -- regular lattice, batch >= 4, working
 * set beyond the L2: gpuqt_options.stencil -- as no index array at all (per-slice pattern id + a small
 * dictionary of relative-column patterns).  gpuqt_plan_storage reports the choice without a GPU;
 * gpuqt_get_table decodes every variant back to the canonical padded table.
 * Errors: the gpuqt_validate codes; GPUQT_ERR_ARG (batch, volume, modes, alignment, K_max too large
 * for one record per warp in shared memory), GPUQT_ERR_NOMEM (workspace too small), GPUQT_ERR_CUDA.
 * On failure *out = NULL and gpuqt_last_error(NULL) describes it.                                */
int gpuqt_create(gpuqt_handle** out, int64_t N, int32_t K_max, const int32_t* nbr_count,
                 const int32_t* nbr_index, const double* hop_re, const double* hop_im,
                 const double* onsite, const double* x, double box_length, double volume,
                 double energy_scale, int32_t batch, int modes, void* workspace,
                 size_t workspace_bytes, void* cuda_stream);
/* The same with explicit tuning options (NULL = defaults).                                        */
int gpuqt_create_with_options(gpuqt_handle** out, int64_t N, int32_t K_max, const int32_t* nbr_count,
                 const int32_t* nbr_index, const double* hop_re, const double* hop_im,
                 const double* onsite, const double* x, double box_length, double volume,
                 double energy_scale, int32_t batch, int modes, void* workspace,
                 size_t workspace_bytes, void* cuda_stream, const gpuqt_options* options);

/* Load B random vectors (Eq. 13; generated by the caller [A7]) and reset time to 0:
 * psi = phi, chi = 0, a = phi, b = V phi (Eq. 34).  phi: [batch][N][2].
 * gpuqt_set_state ENQUEUES the upload and the set-up kernels on the handle's stream and returns without
 * synchronising (the exception to "complete when the call returns"; the next call on the handle is ordered
 * behind it).  With pageable phi_host the runtime has staged the data by then; with PINNED phi_host the copy
 * reads the buffer when the stream gets there, so keep it valid and unchanged until the stream has passed the
 * copy (a synchronising call on the handle -- any moment call, gpuqt_get_state -- or a stream synchronise).
 * gpuqt_slab_set_state behaves the same way.                                                      */
int gpuqt_set_state(gpuqt_handle* h, const double* phi_host);
int gpuqt_set_state_device(gpuqt_handle* h, const double* phi_device);
/* The same in two halves, for the loop over the N_r random vector sets of a run: the upload of
 * the NEXT batch overlaps the computation on the current one.  gpuqt_prefetch_state starts an asynchronous copy of
 * phi_host (pinned host memory, [batch][N][2]; must stay valid and unchanged until the matching
 * gpuqt_set_state_prefetched) into a staging buffer of the workspace on a stream the handle owns, and returns at
 * once; gpuqt_set_state_prefetched makes the handle's stream wait for that copy and then does what gpuqt_set_state
 * does after its copy.  GPUQT_ERR_STATE without a pending prefetch.                                           */
int gpuqt_prefetch_state(gpuqt_handle* h, const double* phi_host);
int gpuqt_set_state_prefetched(gpuqt_handle* h);

/* C_n^DOS = <psi|T_n(H~)|psi>, n < n_moments (Eq. 28) at the current psi (= phi when
 * called before any gpuqt_evolve).  out: host [batch][n_moments].  2 <= n_moments <= MAX.        */
int gpuqt_dos_moments(gpuqt_handle* h, int32_t n_moments, double* out_host);

/* One Chebyshev time step of N_p = order terms (Eq. 17-24) for every enabled
 * branch:  psi <- U(dt) psi;  chi <- U(dt) chi + [X,U(dt)] psi  [A3];  a <- U(-dt) a,
 * b <- U(-dt) b  [A1].  dt may differ from call to call and may be negative.
 * 1 <= order <= GPUQT_MAX_ORDER.                                                                  */
int gpuqt_evolve(gpuqt_handle* h, double dt, int32_t order);

/* C_n^VAC(t) = Re <V a|T_n(H~)|b> (Eq. 29) at the current time; does not advance it.
 * out: host [batch][n_moments].                                                                   */
int gpuqt_vac(gpuqt_handle* h, int32_t n_moments, double* out_host);

/* C_n^MSD(t) = <chi|T_n(H~)|chi> (Eq. 30) at the current time.                      */
int gpuqt_msd(gpuqt_handle* h, int32_t n_moments, double* out_host);

/* out[s][j] = 2 / (pi Omega dE sqrt(1 - E~_j^2)) sum_n g_n (2 - delta_n0) T_n(E~_j) C_n[s] with the
 * Jackson damping g_n (PAPER.md:184-188 Eq. 25-27, :203 Eq. 31).  moments: host [n_sets][n_moments];
 * energies: host [n_energies]; out: host [n_sets][n_energies].                                    */
int gpuqt_kpm_transform(gpuqt_handle* h, const double* moments_host, int32_t n_moments,
                        int32_t n_sets, const double* energies_host, int32_t n_energies,
                        double* out_host);

/* The same resummation with another damping kernel g_n of the kernel polynomial method (the paper's
 * ref. [33]; SURVEY 8(f) 5 -- the paper itself uses Jackson only):
 *   GPUQT_DAMPING_JACKSON    Eq. 31 (identical to gpuqt_kpm_transform; lambda ignored)
 *   GPUQT_DAMPING_LORENTZ    g_n = sinh(lambda (1 - n / N_m)) / sinh(lambda), lambda > 0 (typically 3..5):
 *                            Lorentzian broadening of half width ~ lambda dE / N_m (Green functions)
 *   GPUQT_DAMPING_NONE       g_n = 1 (plain truncated series, Gibbs oscillations)
 * Unknown kernel or lambda <= 0 for Lorentz => GPUQT_ERR_ARG.                                      */
#define GPUQT_DAMPING_JACKSON 0
#define GPUQT_DAMPING_LORENTZ 1
#define GPUQT_DAMPING_NONE 2
int gpuqt_kpm_transform_damped(gpuqt_handle* h, int damping, double lambda, const double* moments_host,
                               int32_t n_moments, int32_t n_sets, const double* energies_host,
                               int32_t n_energies, double* out_host);

/* The same resummation for callers that cannot allocate device memory -- no handle, no cudaMalloc, no cudaFree, no
 * allocating library routine anywhere in the call.  The calls above stage their arguments and keep the table of
 * damping factors in a buffer the handle obtains with cudaMalloc and grows on demand; that is unusable when the
 * process has already given the whole card to a memory pool or a framework's caching allocator (a cudaMalloc behind
 * its back fails, or triggers the pool's out-of-memory retry), when the call sits in a latency-critical loop
 * (cudaMalloc / cudaFree serialise with everything running on the device), or when a scheduler has fixed the job's
 * memory budget in advance (MPS limits, MIG slices).  Here the caller brings inputs and output as DEVICE buffers it
 * already owns:
 *   moments_device   device [n_sets][n_moments]    C_n, e.g. copied from gpuqt_dos_moments / gpuqt_vac / gpuqt_msd
 *   energies_device  device [n_energies]           E_j, |E_j| < energy_scale
 *   out_device       device [n_sets][n_energies]   the transformed function, as gpuqt_kpm_transform_damped
 *   energy_scale, volume   dE and Omega of the model; both > 0
 *   cuda_stream      a cudaStream_t of the CURRENT device (NULL = default stream); the three buffers live there too
 *   err_text         host buffer of err_text_bytes bytes for the message of a failed call, or NULL
 * and the table gs[n] = g_n (2 - delta_n0) plus one status word sit in a fixed `static __device__` array inside the
 * library: GPUQT_STATIC_MAX_MOMENTS doubles + 256 bytes = 128.25 KB of device memory that every GPU loading
 * libgpuqt.so holds until the process exits.  That fixed size is the limit: n_moments > GPUQT_STATIC_MAX_MOMENTS is
 * refused with GPUQT_ERR_NOMEM (n_sets and n_energies are not limited by it; inputs and output are the caller's).
 * The FIRST call on each device looks up the array's device address (cudaGetSymbolAddress, with that device
 * current) and remembers it; make that first call before you begin any stream capture on that device.
 * The array is shared by every call in the process and keeps the last call's contents: the call itself resets what
 * has to start at zero (the status word), and calls that overlap on the GPU -- different streams, different host
 * threads -- race on the table and the status word.  Issue them one at a time per device.
 * The call returns when out_device is complete (it synchronises cuda_stream to read the status word back).
 * Errors: GPUQT_ERR_ARG (null / non-positive argument, unknown damping, n_sets * n_energies >= 2^31),
 * GPUQT_ERR_NOMEM (n_moments beyond the static table), GPUQT_ERR_ENERGY (some |E_j| >= energy_scale, found on the
 * device: out_device then holds NaN at those energies and valid numbers elsewhere), GPUQT_ERR_CUDA.             */
#define GPUQT_STATIC_MAX_MOMENTS 16384
int gpuqt_kpm_transform_static(int damping, double lambda, const double* moments_device, int32_t n_moments,
                               int32_t n_sets, const double* energies_device, int32_t n_energies,
                               double energy_scale, double volume, double* out_device, void* cuda_stream,
                               char* err_text, size_t err_text_bytes);

/* Running conductivity sigma(E, t) in units e = 1 from the TRANSFORMED correlation functions
 * (outputs of gpuqt_kpm_transform), one row per time (PAPER.md:81 Eq. 2, :92 Eq. 5, :123 Eq. 11;
 * discretisation readings A25/A26 of DESIGN.md).  All arrays are host arrays.
 *   kind = GPUQT_SIGMA_FROM_VAC: corr[k][j] = rho(E_j) C_vv(E_j, t_k) with t_k = sum_{i<k} dt_i
 *          (measure, then evolve [A4]); dt has n_times - 1 entries;
 *          sigma[k][j] = integral_0^{t_k} rho C_vv dt by the trapezoid rule (sigma[0] = 0).
 *   kind = GPUQT_SIGMA_FROM_MSD: corr[k][j] = rho(E_j) dX^2(E_j, t_{k+1}) with t_{k+1} = sum_{i<=k} dt_i
 *          (evolve, then measure), dX^2(0) = 0; dt has n_times entries;
 *          sigma[k][j] = (corr[k][j] - corr[k-1][j]) / (2 dt_k), the running conductivity at the middle
 *          of step k; length[k][j] = 2 sqrt(corr[k][j] / dos[j]) (Eq. 11; 0 where dos <= 0 or corr < 0).
 * dos ([n_energies], Eq. 4) and length ([n_times][n_energies]) may be NULL.  Non-positive or
 * non-finite time steps => GPUQT_ERR_ARG.                                                         */
#define GPUQT_SIGMA_FROM_VAC 0
#define GPUQT_SIGMA_FROM_MSD 1
int gpuqt_running_conductivity(gpuqt_handle* h, int kind, const double* corr_host, const double* dos_host,
                               const double* dt_host, int32_t n_times, int32_t n_energies, double* sigma_host,
                               double* length_host);

/* Localization length xi(E) = lim_{t -> inf} L(E, t) / (2 pi)  (Eq. 12) from the propagating length
 * L(E, t) of Eq. 11 (the `length` output of gpuqt_running_conductivity, kind GPUQT_SIGMA_FROM_MSD).  The limit is read as
 * the last measured time [A27]:  xi[j] = length[n_times - 1][j] / (2 pi).  Eq. 12 holds once L has saturated
 * (PAPER.md:125); whether it has is reported as growth[j] = (L[n_times-1][j] - L[n_times-2][j]) / L[n_times-1][j], the
 * relative change over the last step (0 where L[n_times-1][j] == 0; 1 with a single row) -- the caller decides how small
 * is small enough.  length_host: host [n_times][n_energies]; xi_host, growth_host: host [n_energies]; growth_host may
 * be NULL.                                                                                                       */
int gpuqt_localization_length(gpuqt_handle* h, const double* length_host, int32_t n_times, int32_t n_energies,
                              double* xi_host, double* growth_host);

/* Copy a state back: host [batch][N][2].                                                          */
int gpuqt_get_state(gpuqt_handle* h, int which, double* out_host);

/* Decode the device sliced-ELL table back to canonical padded row-major [N*K_max] arrays
 * (padding = (own row, 0)); dx = minimum-image X_n - X_m as the kernels compute it [A6].
 * Any output pointer may be NULL.  Used for the bit-exact indexing check.                         */
int gpuqt_get_table(gpuqt_handle* h, int32_t* col, double* re, double* im, double* dx);

/* The N_p Bessel coefficients of one step, host only:
 * c_m = (2 - delta_0m) (-i sgn dt)^m J_m(dE |dt|), m < order   (Eq. 17).            */
int gpuqt_bessel_coeffs(double energy_scale, double dt, int32_t order, double* c_re, double* c_im);

/* Facts about the handle (what the builder chose), for reports and tests.                          */
#define GPUQT_INFO_STORED_MATRIX_BYTES 0   /* bytes of the packed records + the x array               */
#define GPUQT_INFO_HOP_VARIANT 1           /* 0 real per entry, 1 complex per entry, 2 constant hopping
                                              with int32 columns, 3 constant hopping with 16-bit columns,
                                              4 the same with padding entries (delta 0xffff = zero row),
                                              5 constant hopping, implicit stencil (pattern dictionary)  */
#define GPUQT_INFO_UNIFORM 2               /* 1: every record has width K_max                          */
#define GPUQT_INFO_UNROLLED_WIDTH 3        /* K_max when the unrolled walk is used (2, 3, 4, 6), else 0 */
#define GPUQT_INFO_SMALL_PATH 4            /* 1: the one-CTA whole-recurrence kernel is in use         */
#define GPUQT_INFO_PERSISTENT 5            /* 1: recurrences run as one cooperative multi-step launch  */
#define GPUQT_INFO_WORKSPACE_USED 6        /* bytes of the workspace actually carved up                */
#define GPUQT_INFO_SMALL_PATH_MSD 7        /* 1: the (psi, chi) time step is one launch of one CTA too    */
#define GPUQT_INFO_STENCIL_PATTERNS 8      /* patterns in the implicit-stencil dictionary (0: not in use)  */
#define GPUQT_INFO_REORDERED 9             /* 1: the sites are stored in brick order (gpuqt_options.reorder)  */
int gpuqt_get_info(gpuqt_handle* h, int what, int64_t* value);

/* Accumulated device time (CUDA events on the handle's stream around each run of launches) and
 * number of launches of one kernel class since the last reset.                                    */
int gpuqt_kernel_stats(gpuqt_handle* h, int kernel_class, double* ms, int64_t* launches);
/* Number of recurrence steps (Eq. 21/23 applications) those launches performed: a launch performs
 * one step, or a whole recurrence in the multi-step forms (persistent / one-CTA kernels).         */
int gpuqt_kernel_steps(gpuqt_handle* h, int kernel_class, int64_t* steps);
int gpuqt_reset_stats(gpuqt_handle* h);

/* Text of the last error on this handle; with h == NULL, of the last failed gpuqt_create on the
 * calling thread.  The pointer stays valid until the next failing call on the same handle / thread. */
const char* gpuqt_last_error(const gpuqt_handle* h);
void gpuqt_destroy(gpuqt_handle* h);

/* ------------------------------------------------------------------ row-slab decomposition
 * One lattice too large (or too slow) for one GPU is cut into SLABS of consecutive rows.  A slab owns n_own rows
 * of H and of every state vector; the columns of its rows that belong to other slabs are its n_halo HALO rows,
 * stored behind the owned rows (local index n_own + j), so a slab is an ordinary (rectangular) table for the
 * kernels above.  Every recurrence step x_m = 2 H~ x_{m-1} - x_{m-2} (Eq. 21) needs the halo rows of
 * x_{m-1}: after each step a slab PUSHES the owned rows its neighbours need straight into their halo rows (stores
 * to the peer's vector buffer: a local buffer, or a peer-mapped one over NVLink), and the next step starts when
 * every neighbour has pushed (same stream for slabs of one group; a release/acquire flag per sender at system
 * scope for slabs on other GPUs).  The paper is single-GPU and limited by one card's memory
 * (PAPER.md:51); this is the scale-out past that limit.  Inner products are partial sums over the owned rows:
 * every moment call returns the sum over the slabs of THIS group, and the caller adds the groups' results
 * (moments are linear in the partial sums).
 *
 * A gpuqt_slab_group is the set of slabs resident on one GPU (normally one; several emulate a multi-GPU
 * decomposition on one device, which is how the tests run).  All slabs of all groups must make the same
 * sequence of calls.  Slabs always run one launch per recurrence step (no cooperative / one-CTA forms).       */
typedef struct gpuqt_slab_group gpuqt_slab_group;
#define GPUQT_MAX_SLABS 64
typedef struct gpuqt_slab_desc {
    int32_t global_id;            /* id of this slab among all slabs of the decomposition, < GPUQT_MAX_SLABS   */
    int64_t n_own;                /* rows this slab owns (computes)                                            */
    int64_t n_halo;               /* halo rows, local indices n_own .. n_own + n_halo - 1                      */
    const int32_t* nbr_count;     /* host [n_own]                                                              */
    const int32_t* nbr_index;     /* host [n_own][K_max], LOCAL indices in [0, n_own + n_halo)                 */
    const double* hop_re;         /* host [n_own][K_max] or NULL (-1)                                          */
    const double* hop_im;         /* host [n_own][K_max] or NULL (real H)                                      */
    const double* onsite;         /* host [n_own] or NULL (0)                                                  */
    const double* x;              /* host [n_own + n_halo] positions (owned rows, then halo rows)              */
    int32_t n_sends;              /* segments of owned rows other slabs need                                   */
    const int32_t* send_peer;     /* host [n_sends] global id of the receiving slab                            */
    const int64_t* send_count;    /* host [n_sends] rows in the segment                                        */
    const int64_t* send_dst_row;  /* host [n_sends] first local row (>= the peer's n_own) it fills in the peer */
    const int32_t* send_rows;     /* host, the segments' local owned-row indices, concatenated                 */
    void* workspace;              /* device, 256-byte aligned, >= gpuqt_slab_workspace_bytes(...)              */
    size_t workspace_bytes;
} gpuqt_slab_desc;
size_t gpuqt_slab_workspace_bytes(int64_t n_own, int64_t n_halo, int32_t K_max, int is_complex, int32_t batch, int modes);
/* Builds the slabs (each validated like gpuqt_create; Hermiticity is checked for the owned-owned block only).
 * Sends to slabs of this group are connected here; sends to other groups need gpuqt_slab_connect.  Two local slabs
 * with the same global_id are refused (GPUQT_ERR_ARG).  Errors of this call: gpuqt_last_error(NULL).           */
int gpuqt_slab_create(gpuqt_slab_group** out, int32_t n_local, const gpuqt_slab_desc* slabs, int32_t K_max,
                      double box_length, double volume, double energy_scale, int32_t batch, int modes,
                      void* cuda_stream);
/* The same with explicit tuning options for every slab (NULL = defaults); small, persistent and reorder are
 * ignored for slabs (one launch per recurrence step, the caller's row order).                                  */
int gpuqt_slab_create_with_options(gpuqt_slab_group** out, int32_t n_local, const gpuqt_slab_desc* slabs, int32_t K_max,
                                   double box_length, double volume, double energy_scale, int32_t batch, int modes,
                                   void* cuda_stream, const gpuqt_options* options);
/* What another group needs to push into local slab `local_slab`: the device addresses of its vector buffers (in the
 * fixed order every slab uses; gpuqt_slab_buffer_count of them) and of its flag array, and its row counts n_own /
 * n_halo (either may be NULL).  The caller maps the addresses into the peer process (CUDA IPC) and hands the mapped
 * addresses and the two counts to gpuqt_slab_connect there, which refuses (GPUQT_ERR_INDEX) a send segment that does
 * not lie inside the peer's halo rows [peer_n_own, peer_n_own + peer_n_halo), and (GPUQT_ERR_ARG) a peer id that
 * belongs to the connecting group itself.  Every slab of another group that a local slab sends to must be connected
 * before the first compute call (GPUQT_ERR_STATE otherwise).                                                   */
int32_t gpuqt_slab_buffer_count(const gpuqt_slab_group* g);
int gpuqt_slab_export(gpuqt_slab_group* g, int32_t local_slab, void** buffers, void** flags, int64_t* n_own,
                      int64_t* n_halo);
int gpuqt_slab_connect(gpuqt_slab_group* g, int32_t peer_global_id, void* const* peer_buffers, void* peer_flags,
                       int64_t peer_n_own, int64_t peer_n_halo);
/* How long a halo exchange waits on the GPU for a slab of another group before it gives up (default 60 s; 0 <
 * seconds <= 3600).  A wait that gave up surfaces as GPUQT_ERR_STATE from the call's next synchronisation
 * (the moment calls, gpuqt_slab_get_state).  After that error, as after any error that strikes once a compute call
 * has started issuing work, the group's buffers and exchange counter no longer match its peers': every further call
 * returns GPUQT_ERR_STATE until the group is destroyed and rebuilt (on all ranks).                               */
int gpuqt_slab_set_wait_budget(gpuqt_slab_group* g, double seconds);
/* phi_host[i]: host [batch][n_own of local slab i][2].  chi = 0; VAC mode: a = phi, b = V phi.  Enqueued, not
 * synchronised: pinned phi_host buffers must stay valid and unchanged as for gpuqt_set_state.                  */
int gpuqt_slab_set_state(gpuqt_slab_group* g, const double* const* phi_host);
/* As gpuqt_dos_moments / gpuqt_evolve / gpuqt_vac / gpuqt_msd (gpuqt_slab_dos_moments answers in every mode, psi
 * being set in every mode); moments: host [batch][n_moments], the partial sums over this group's slabs.        */
int gpuqt_slab_dos_moments(gpuqt_slab_group* g, int32_t n_moments, double* out_host);
int gpuqt_slab_evolve(gpuqt_slab_group* g, double dt, int32_t order);
int gpuqt_slab_vac(gpuqt_slab_group* g, int32_t n_moments, double* out_host);
int gpuqt_slab_msd(gpuqt_slab_group* g, int32_t n_moments, double* out_host);
/* State of one local slab's owned rows: host [batch][n_own][2].                                               */
int gpuqt_slab_get_state(gpuqt_slab_group* g, int32_t local_slab, int which, double* out_host);
/* gpuqt_get_info (GPUQT_INFO_*) of one local slab: what the builder chose for its table.                      */
int gpuqt_slab_get_info(gpuqt_slab_group* g, int32_t local_slab, int what, int64_t* value);
const char* gpuqt_slab_last_error(const gpuqt_slab_group* g);
void gpuqt_slab_destroy(gpuqt_slab_group* g);

#ifdef __cplusplus
}
#endif
#endif /* GPUQT_H */
