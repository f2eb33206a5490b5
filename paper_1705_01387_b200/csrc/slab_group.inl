// Row-slab decomposition with halo exchange (include/gpuqt.h "row-slab decomposition").  Included at the
// end of gpuqt.cu: the slabs are ordinary gpuqt_handles (rectangular tables: n_own rows, n_own + n_halo vector rows) and
// the drivers below interleave their one-step launches with the halo pushes.
//
// Exchange of a vector buffer (identified by its index in gpuqt_handle::map_bufs, the same in every slab):
//   1. every local slab launches one halo_push_kernel per send segment: owned rows -> the peer's halo rows (plain stores;
//      the peer buffer is local, or a peer-mapped address of another GPU);
//   2. if there are remote peers: one halo_signal_kernel per slab publishes the exchange number to the remote receivers
//      (st.release.sys after a system fence; the pushes before it in the stream are complete), and one halo_wait_kernel
//      per slab spins (ld.acquire.sys) until every remote sender has published it.
// Slabs of one group share a stream, so their pushes are ordered before the next step without flags.  Write-after-read
// on a halo, remote case: a push of exchange e is issued after the sender's wait of exchange e-1, i.e. after the receiver
// published e-1, i.e. after everything the receiver ran BEFORE its exchange e-1.  Inside a recurrence push e goes to ring
// slot (e-1) % 3, whose previous contents (exchange e-3) were last read by the receiver's step e-2, before its exchange
// e-1: safe.  Across calls the same buffer could be exchanged twice with only one exchange in between and a reader after
// it (the last step of one recurrence, the first exchange of the next), so every top-level phase starts with
// slab_fence(): an exchange without pushes, after which every peer has finished all it ran before.

namespace {

__global__ void halo_push_kernel(int B, const double2* __restrict__ src, const int32_t* __restrict__ rows, long long n_rows,
                                 double2* __restrict__ dst, long long dst_row0) {
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n_rows * B) return;
    const long long r = i / B;
    const int b = (int)(i % B);
    dst[(dst_row0 + r) * B + b] = src[(long long)rows[r] * B + b];
}
// flags[k] points at word `me` of remote receiver k's flag array
__global__ void halo_signal_kernel(int n, unsigned int* const* __restrict__ flags, unsigned int epoch) {
    const int k = blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= n) return;
    __threadfence_system();
    asm volatile("st.release.sys.global.u32 [%0], %1;" ::"l"(flags[k]), "r"(epoch) : "memory");
}
// my_flags[sender[k]] >= epoch for every remote sender k.  The spin is bounded: a sender that has not published
// `epoch` within budget_ns (a peer that died, took an error path, or was never given the same sequence of calls)
// makes the thread give up and raise *timed_out, which the host turns into GPUQT_ERR_STATE at its next
// synchronisation instead of hanging the stream for ever.
__global__ void halo_wait_kernel(int n, const unsigned int* __restrict__ my_flags, const int* __restrict__ sender, unsigned int epoch,
                                 unsigned long long budget_ns, unsigned int* __restrict__ timed_out) {
    const int k = blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= n) return;
    unsigned long long t0, t;
    asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t0));
    unsigned int v;
    for (;;) {
        asm volatile("ld.acquire.sys.global.u32 %0, [%1];" : "=r"(v) : "l"(my_flags + sender[k]) : "memory");
        if ((int)(v - epoch) >= 0) break;
        asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t));
        if (t - t0 > budget_ns) {
            atomicExch(timed_out, 1u);
            break;
        }
    }
    __threadfence_system();
}
// dst[i] += src[i]: the partial dots of the slabs of a group
__global__ void add_dots_kernel(long long n, const double* __restrict__ src, double* __restrict__ dst) {
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) dst[i] += src[i];
}

struct SlabSend {
    int peer_global = -1;
    int peer_local = -1;            // index in the group, or -1: a slab of another group
    int64_t n_rows = 0, dst_row0 = 0;
    const int32_t* d_rows = nullptr;
};
struct SlabRemote {                 // a slab of another group that local slabs push to
    std::vector<double2*> bufs;     // its vector buffers, mapped into this process
    unsigned int* flags = nullptr;  // its flag array
};

}  // namespace

struct gpuqt_slab_group {
    std::vector<gpuqt_handle*> h;
    std::vector<int> global_id;
    std::vector<std::vector<SlabSend>> sends;       // [local slab]
    std::map<int, SlabRemote> remote;               // by global id
    std::vector<int32_t*> d_rows;                   // per local slab: all send rows (device)
    std::vector<unsigned int*> d_flags;             // per local slab: uint32[GPUQT_MAX_SLABS], written by remote senders,
                                                    // + one word [GPUQT_MAX_SLABS] a timed-out wait of this slab raises
    // per local slab, rebuilt by gpuqt_slab_connect: where to signal, whom to wait for
    std::vector<unsigned int**> d_signal;
    std::vector<int*> d_senders;
    std::vector<int> n_remote;
    unsigned int epoch = 0;
    unsigned long long wait_budget_ns = 60ull * 1000000000ull;     // gpuqt_slab_set_wait_budget
    cudaStream_t stream = nullptr;
    int B = 0, modes = 0;
    bool state_set = false;
    bool poisoned = false;                          // an error struck in the middle of a sequence: see slab_done
    std::string poison_reason;
    std::string err;
};

namespace {

int gfail(gpuqt_slab_group* g, int code, const std::string& msg) {
    if (g) g->err = msg;
    return code;
}
#define GCU(call)                                                                                   \
    do {                                                                                            \
        cudaError_t e_ = (call);                                                                    \
        if (e_ != cudaSuccess) return gfail(g, GPUQT_ERR_CUDA, std::string(#call) + ": " + cudaGetErrorString(e_)); \
    } while (0)

int buffer_index(const gpuqt_handle* h, const double2* p) {
    for (size_t i = 0; i < h->map_bufs.size(); ++i)
        if (h->map_bufs[i] == p) return (int)i;
    return -1;
}

// Halo exchange of one vector buffer per slab: bufs[i] is local slab i's buffer (the same buffer index in every slab)
int slab_exchange(gpuqt_slab_group* g, const std::vector<const double2*>& bufs) {
    const int n = (int)g->h.size();
    ++g->epoch;
    bool any_remote = false;
    for (int i = 0; i < n; ++i) {
        const int id = buffer_index(g->h[i], bufs[(size_t)i]);
        if (id < 0) return gfail(g, GPUQT_ERR_STATE, "halo exchange of an unknown buffer");
        for (const SlabSend& s : g->sends[(size_t)i]) {
            double2* dst = nullptr;
            if (s.peer_local >= 0) {
                dst = const_cast<double2*>(g->h[(size_t)s.peer_local]->map_bufs[(size_t)id]);
            } else {
                auto it = g->remote.find(s.peer_global);
                if (it == g->remote.end())
                    return gfail(g, GPUQT_ERR_STATE, "slab " + std::to_string(s.peer_global) + " is not connected (gpuqt_slab_connect)");
                dst = it->second.bufs[(size_t)id];
                any_remote = true;
            }
            const long long total = s.n_rows * g->B;
            if (total == 0) continue;
            halo_push_kernel<<<(unsigned)((total + 255) / 256), 256, 0, g->stream>>>(g->B, bufs[(size_t)i], s.d_rows, s.n_rows, dst, s.dst_row0);
            GCU(cudaGetLastError());
        }
    }
    if (any_remote) {
        for (int i = 0; i < n; ++i)
            if (g->n_remote[(size_t)i] > 0) {
                halo_signal_kernel<<<1, 64, 0, g->stream>>>(g->n_remote[(size_t)i], g->d_signal[(size_t)i], g->epoch);
                GCU(cudaGetLastError());
            }
        for (int i = 0; i < n; ++i)
            if (g->n_remote[(size_t)i] > 0) {
                halo_wait_kernel<<<1, 64, 0, g->stream>>>(g->n_remote[(size_t)i], g->d_flags[(size_t)i], g->d_senders[(size_t)i], g->epoch,
                                                          g->wait_budget_ns, g->d_flags[(size_t)i] + GPUQT_MAX_SLABS);
                GCU(cudaGetLastError());
            }
    }
    return GPUQT_OK;
}

// all remote peers have completed everything they issued before their matching slab_fence (no launches without remote
// peers).  The exchange number advances in every case, so that groups whose calls match keep matching numbers whatever
// the order of their gpuqt_slab_connect calls was.
int slab_fence(gpuqt_slab_group* g) {
    ++g->epoch;
    bool any = false;
    for (int r : g->n_remote) any = any || r > 0;
    if (!any) return GPUQT_OK;
    for (size_t i = 0; i < g->h.size(); ++i)
        if (g->n_remote[i] > 0) {
            halo_signal_kernel<<<1, 64, 0, g->stream>>>(g->n_remote[i], g->d_signal[i], g->epoch);
            GCU(cudaGetLastError());
        }
    for (size_t i = 0; i < g->h.size(); ++i)
        if (g->n_remote[i] > 0) {
            halo_wait_kernel<<<1, 64, 0, g->stream>>>(g->n_remote[i], g->d_flags[i], g->d_senders[i], g->epoch, g->wait_budget_ns,
                                                      g->d_flags[i] + GPUQT_MAX_SLABS);
            GCU(cudaGetLastError());
        }
    return GPUQT_OK;
}

// Before any work is issued: the group is usable and every slab of another group that a local slab sends to has been
// connected (an exchange that found a peer missing half way would leave the groups' exchange numbers apart).
int slab_ready(gpuqt_slab_group* g) {
    if (g->poisoned)
        return gfail(g, GPUQT_ERR_STATE, "the group is unusable after an earlier error in the middle of a sequence (" + g->poison_reason +
                                             "); destroy it and build a new one");
    for (size_t i = 0; i < g->h.size(); ++i)
        for (const SlabSend& s : g->sends[i])
            if (s.peer_local < 0 && g->remote.find(s.peer_global) == g->remote.end())
                return gfail(g, GPUQT_ERR_STATE, "slab " + std::to_string(s.peer_global) + " is not connected (gpuqt_slab_connect)");
    return GPUQT_OK;
}

// The end of a compute call that had started issuing work: after an error the states, the ring buffers and the
// exchange number no longer mean on this side what they mean on the peers' side, so the group refuses further work.
int slab_done(gpuqt_slab_group* g, int rc) {
    if (rc != GPUQT_OK && !g->poisoned) {
        g->poisoned = true;
        g->poison_reason = g->err;
    }
    return rc;
}

// Wait for the stream, then ask whether a wait for a remote sender gave up.
int slab_sync(gpuqt_slab_group* g) {
    GCU(cudaStreamSynchronize(g->stream));
    for (size_t i = 0; i < g->h.size(); ++i) {
        if (g->n_remote[i] == 0) continue;
        unsigned int gave_up = 0;
        GCU(cudaMemcpy(&gave_up, g->d_flags[i] + GPUQT_MAX_SLABS, sizeof(gave_up), cudaMemcpyDeviceToHost));
        if (gave_up)
            return gfail(g, GPUQT_ERR_STATE, "a slab of another group did not arrive at a halo exchange within " +
                                                 std::to_string((double)g->wait_budget_ns * 1e-9) + " s (gpuqt_slab_set_wait_budget)");
    }
    return GPUQT_OK;
}

template <class F>
std::vector<const double2*> each_buffer(gpuqt_slab_group* g, F sel) {      // sel(i) = the buffer of local slab i
    std::vector<const double2*> v;
    for (size_t i = 0; i < g->h.size(); ++i) v.push_back(sel(i));
    return v;
}

// Steps 1 .. terms-1 of one recurrence in every slab (args[i]: slab i, with x0 / e0 / src / coef / dots set), the halo
// rows of x_m (and e_m) exchanged after every step that another step follows; the halos of x_0 (e_0) first.
int slab_recurrence(gpuqt_slab_group* g, int mode, std::vector<RecArgs>& args) {
    const size_t n = g->h.size();
    const bool pair = args[0].e0 != nullptr;
    const int terms = args[0].terms;
    if (terms < 2) return GPUQT_OK;
    for (size_t i = 0; i < n; ++i) {
        fill_rec_args(g->h[i], args[i]);
        args[i].multi = 0;
    }
    int rc = slab_fence(g);
    if (rc == GPUQT_OK) rc = slab_exchange(g, each_buffer(g, [&](size_t i) { return args[i].x0; }));
    if (rc == GPUQT_OK && pair) rc = slab_exchange(g, each_buffer(g, [&](size_t i) { return args[i].e0; }));
    if (rc) return rc;
    for (int m = 1; m < terms; ++m) {
        for (size_t i = 0; i < n; ++i) {
            args[i].m_begin = m;
            args[i].m_end = m + 1;
            cudaError_t e = launch_steps(g->h[i], mode, args[i]);
            if (e != cudaSuccess) return gfail(g, GPUQT_ERR_CUDA, std::string("step launch: ") + cudaGetErrorString(e));
        }
        if (m + 1 < terms) {                      // x_m lives in ring slot (m - 1) % 3 (kernels.cuh, make_ctx)
            const int slot = (m - 1) % kRing;
            rc = slab_exchange(g, each_buffer(g, [&](size_t i) { return (const double2*)g->h[i]->ring[slot]; }));
            if (rc == GPUQT_OK && pair) rc = slab_exchange(g, each_buffer(g, [&](size_t i) { return (const double2*)g->h[i]->ringe[slot]; }));
            if (rc) return rc;
        }
    }
    return GPUQT_OK;
}

// Partial dots of slabs 1.. added into slab 0's, which then finalises the moments (the sums are linear)
int slab_sum_dots(gpuqt_slab_group* g, long long n_values) {
    for (size_t i = 1; i < g->h.size(); ++i) {
        add_dots_kernel<<<(unsigned)((n_values + 255) / 256), 256, 0, g->stream>>>(n_values, g->h[i]->dots, g->h[0]->dots);
        GCU(cudaGetLastError());
    }
    return GPUQT_OK;
}

int slab_copy_moments(gpuqt_slab_group* g, int n_moments, double* out_host) {
    GCU(cudaMemcpyAsync(out_host, g->h[0]->moments, (size_t)g->B * n_moments * sizeof(double), cudaMemcpyDeviceToHost, g->stream));
    const int rc = slab_sync(g);
    for (gpuqt_handle* h : g->h) flush_stats(h);
    return rc;
}

// C_n = <v|T_n|v> with the doubling identity, v = psi or chi of every slab
int slab_moments_doubling(gpuqt_slab_group* g, bool use_chi, int n_moments, double* out_host) {
    const int n_steps = n_moments / 2;
    std::vector<RecArgs> args(g->h.size());
    for (size_t i = 0; i < g->h.size(); ++i) {
        gpuqt_handle* h = g->h[i];
        h->sweep = 0;
        RecArgs a{};
        a.x0 = use_chi ? h->chi : h->psi;
        a.terms = n_steps + 1;
        a.dots = h->dots;
        a.dot_m0 = 1;
        args[i] = a;
    }
    int rc = slab_recurrence(g, kModeDoubling, args);
    if (rc) return rc;
    rc = slab_sum_dots(g, (long long)n_steps * 3 * g->B);
    if (rc) return rc;
    const int total = g->B * n_moments;
    finalize_doubling<<<(total + 255) / 256, 256, 0, g->stream>>>(g->B, n_moments, n_steps, g->h[0]->dots, g->h[0]->moments);
    GCU(cudaGetLastError());
    return slab_copy_moments(g, n_moments, out_host);
}

// (out, out_e) <- sum_k c_k T_k (in, in_e) in every slab (Clenshaw, as evolve_clenshaw)
using SlabIn = std::function<const double2*(size_t)>;
using SlabOut = std::function<double2*(size_t)>;
int slab_evolve_set(gpuqt_slab_group* g, int mode, SlabIn in_of, SlabIn in_e_of, SlabOut out_of, SlabOut out_e_of, double dt, int order) {
    const size_t n = g->h.size();
    const bool pair = mode == kModeEvolveMsd;
    std::vector<double> cr, ci;
    bessel_coeffs(g->h[0]->dE, dt, order, cr, ci);
    if (order == 1) {
        for (size_t i = 0; i < n; ++i) {
            GCU(launch_scale(g->h[i], cr[0], ci[0], in_of(i), out_of(i)));
            if (pair) GCU(launch_scale(g->h[i], cr[0], ci[0], in_e_of(i), out_e_of(i)));
        }
        return GPUQT_OK;
    }
    std::vector<RecArgs> args(n);
    for (size_t i = 0; i < n; ++i) {
        gpuqt_handle* h = g->h[i];
        h->sweep = 0;
        const double* coef = nullptr;
        GCU(upload_coefs(h, cr, ci, order, &coef));
        double2* b0 = h->ring[kRing - 1];
        double2* b0_e = pair ? h->ringe[kRing - 1] : nullptr;
        GCU(launch_scale(h, cr[(size_t)order - 1], ci[(size_t)order - 1], in_of(i), b0));
        if (pair) GCU(launch_scale(h, cr[(size_t)order - 1], ci[(size_t)order - 1], in_e_of(i), b0_e));
        RecArgs a{};
        a.x0 = b0; a.e0 = b0_e;
        a.src = in_of(i); a.src_e = pair ? in_e_of(i) : nullptr;
        a.coef = coef;
        a.terms = order;
        a.clenshaw = 1;
        a.store_last = 1;
        a.last_out = out_of(i); a.last_out_e = pair ? out_e_of(i) : nullptr;
        args[i] = a;
    }
    return slab_recurrence(g, mode, args);
}

}  // namespace

// =================================================================== C ABI of the slab groups
extern "C" {

size_t gpuqt_slab_workspace_bytes(int64_t n_own, int64_t n_halo, int32_t K_max, int is_complex, int32_t batch, int modes) {
    if (n_own <= 0 || n_halo < 0 || K_max <= 0 || !batch_ok(batch)) return 0;
    if (modes & GPUQT_MODE_MSD) modes |= GPUQT_MODE_PSI;
    const size_t rec = (size_t)((n_own + 31) / 32 + kTilePad) * (size_t)record_bytes(K_max, is_complex ? 2 : 1);
    return make_layout(n_own + n_halo, batch, modes, rec).total;
}

int gpuqt_slab_create(gpuqt_slab_group** out, int32_t n_local, const gpuqt_slab_desc* slabs, int32_t K_max,
                      double box_length, double volume, double energy_scale, int32_t batch, int modes,
                      void* cuda_stream) {
    return gpuqt_slab_create_with_options(out, n_local, slabs, K_max, box_length, volume, energy_scale, batch, modes,
                                          cuda_stream, nullptr);
}

int gpuqt_slab_create_with_options(gpuqt_slab_group** out, int32_t n_local, const gpuqt_slab_desc* slabs, int32_t K_max,
                                   double box_length, double volume, double energy_scale, int32_t batch, int modes,
                                   void* cuda_stream, const gpuqt_options* options) {
    auto bad = [&](int code, const std::string& msg) {
        g_create_error = "gpuqt_slab_create: " + msg;
        return code;
    };
    if (!out) return bad(GPUQT_ERR_ARG, "null output pointer");
    *out = nullptr;
    if (n_local < 1 || n_local > GPUQT_MAX_SLABS || !slabs) return bad(GPUQT_ERR_ARG, "1 .. GPUQT_MAX_SLABS local slabs");
    gpuqt_slab_group* g = new (std::nothrow) gpuqt_slab_group();
    if (!g) return bad(GPUQT_ERR_NOMEM, "out of host memory");
    g->stream = (cudaStream_t)cuda_stream;
    g->B = batch;
    g->modes = (modes & GPUQT_MODE_MSD) ? (modes | GPUQT_MODE_PSI) : modes;
    auto fail_create = [&](int code, const std::string& msg) {
        gpuqt_slab_destroy(g);
        return bad(code, msg);
    };
    for (int i = 0; i < n_local; ++i) {
        const gpuqt_slab_desc& d = slabs[i];
        if (d.global_id < 0 || d.global_id >= GPUQT_MAX_SLABS || d.n_sends < 0 || d.n_halo < 0 ||
            (d.n_sends > 0 && (!d.send_peer || !d.send_count || !d.send_dst_row || !d.send_rows)))
            return fail_create(GPUQT_ERR_ARG, "bad descriptor of local slab " + std::to_string(i));
        for (int j = 0; j < i; ++j)
            if (slabs[j].global_id == d.global_id)
                return fail_create(GPUQT_ERR_ARG, "global id " + std::to_string(d.global_id) + " is given to two local slabs");
        gpuqt_handle* h = nullptr;
        int rc = create_handle(&h, d.n_own, d.n_halo, K_max, d.nbr_count, d.nbr_index, d.hop_re, d.hop_im, d.onsite, d.x,
                               box_length, volume, energy_scale, batch, modes, d.workspace, d.workspace_bytes, cuda_stream,
                               options, true);
        if (rc != GPUQT_OK) {
            const std::string why = g_create_error;
            gpuqt_slab_destroy(g);
            g_create_error = "gpuqt_slab_create: slab " + std::to_string(i) + ": " + why;
            return rc;
        }
        g->h.push_back(h);
        g->global_id.push_back(d.global_id);
    }
    // send segments
    g->sends.resize((size_t)n_local);
    g->d_rows.assign((size_t)n_local, nullptr);
    g->d_flags.assign((size_t)n_local, nullptr);
    g->d_signal.assign((size_t)n_local, nullptr);
    g->d_senders.assign((size_t)n_local, nullptr);
    g->n_remote.assign((size_t)n_local, 0);
    for (int i = 0; i < n_local; ++i) {
        const gpuqt_slab_desc& d = slabs[i];
        int64_t total = 0;
        for (int s = 0; s < d.n_sends; ++s) {
            if (d.send_count[s] < 0) return fail_create(GPUQT_ERR_ARG, "negative send count");
            total += d.send_count[s];
        }
        for (int64_t r = 0; r < total; ++r)
            if (d.send_rows[r] < 0 || d.send_rows[r] >= d.n_own) return fail_create(GPUQT_ERR_INDEX, "send row is not an owned row");
        cudaError_t e = cudaSuccess;
        if (total > 0) {
            e = cudaMalloc((void**)&g->d_rows[(size_t)i], (size_t)total * sizeof(int32_t));
            if (e == cudaSuccess) e = cudaMemcpy(g->d_rows[(size_t)i], d.send_rows, (size_t)total * sizeof(int32_t), cudaMemcpyHostToDevice);
        }
        if (e == cudaSuccess) e = cudaMalloc((void**)&g->d_flags[(size_t)i], (GPUQT_MAX_SLABS + 1) * sizeof(unsigned int));
        if (e == cudaSuccess) e = cudaMemset(g->d_flags[(size_t)i], 0, (GPUQT_MAX_SLABS + 1) * sizeof(unsigned int));
        if (e == cudaSuccess) e = cudaMalloc((void**)&g->d_signal[(size_t)i], GPUQT_MAX_SLABS * sizeof(unsigned int*));
        if (e == cudaSuccess) e = cudaMalloc((void**)&g->d_senders[(size_t)i], GPUQT_MAX_SLABS * sizeof(int));
        if (e != cudaSuccess) return fail_create(GPUQT_ERR_CUDA, std::string("send lists: ") + cudaGetErrorString(e));
        int64_t off = 0;
        for (int s = 0; s < d.n_sends; ++s) {
            SlabSend snd;
            snd.peer_global = d.send_peer[s];
            snd.n_rows = d.send_count[s];
            snd.dst_row0 = d.send_dst_row[s];
            snd.d_rows = g->d_rows[(size_t)i] + off;
            off += d.send_count[s];
            if (snd.peer_global < 0 || snd.peer_global >= GPUQT_MAX_SLABS || snd.peer_global == d.global_id)
                return fail_create(GPUQT_ERR_ARG, "bad send peer");
            for (int j = 0; j < n_local; ++j)
                if (g->global_id[(size_t)j] == snd.peer_global) snd.peer_local = j;
            if (snd.peer_local >= 0) {       // the segment must lie inside the peer's halo rows
                const gpuqt_handle* p = g->h[(size_t)snd.peer_local];
                if (snd.dst_row0 < p->N || snd.dst_row0 + snd.n_rows > p->NV)
                    return fail_create(GPUQT_ERR_INDEX, "send segment outside the peer's halo rows");
            }
            g->sends[(size_t)i].push_back(snd);
        }
    }
    *out = g;
    return GPUQT_OK;
}

int32_t gpuqt_slab_buffer_count(const gpuqt_slab_group* g) { return g && !g->h.empty() ? (int32_t)g->h[0]->map_bufs.size() : 0; }

int gpuqt_slab_export(gpuqt_slab_group* g, int32_t local_slab, void** buffers, void** flags, int64_t* n_own, int64_t* n_halo) {
    if (!g || local_slab < 0 || local_slab >= (int32_t)g->h.size() || !buffers || !flags) return gfail(g, GPUQT_ERR_ARG, "bad argument");
    const gpuqt_handle* h = g->h[(size_t)local_slab];
    for (size_t i = 0; i < h->map_bufs.size(); ++i) buffers[i] = (void*)h->map_bufs[i];
    *flags = g->d_flags[(size_t)local_slab];
    if (n_own) *n_own = h->N;
    if (n_halo) *n_halo = h->NV - h->N;
    return GPUQT_OK;
}

int gpuqt_slab_connect(gpuqt_slab_group* g, int32_t peer_global_id, void* const* peer_buffers, void* peer_flags,
                       int64_t peer_n_own, int64_t peer_n_halo) {
    if (!g || !peer_buffers || !peer_flags || peer_global_id < 0 || peer_global_id >= GPUQT_MAX_SLABS || peer_n_own < 1 ||
        peer_n_halo < 0)
        return gfail(g, GPUQT_ERR_ARG, "bad argument");
    for (int id : g->global_id)
        if (id == peer_global_id) return gfail(g, GPUQT_ERR_ARG, "slab " + std::to_string(peer_global_id) + " belongs to this group");
    // every segment sent to this peer must land inside its halo rows (the pushes are plain stores into its memory)
    for (size_t i = 0; i < g->h.size(); ++i)
        for (const SlabSend& s : g->sends[i])
            if (s.peer_global == peer_global_id && (s.dst_row0 < peer_n_own || s.dst_row0 + s.n_rows > peer_n_own + peer_n_halo))
                return gfail(g, GPUQT_ERR_INDEX, "a send segment of local slab " + std::to_string(i) + " lies outside the halo rows of slab " +
                                                     std::to_string(peer_global_id));
    SlabRemote r;
    for (int32_t i = 0; i < gpuqt_slab_buffer_count(g); ++i) r.bufs.push_back((double2*)peer_buffers[i]);
    r.flags = (unsigned int*)peer_flags;
    g->remote[peer_global_id] = r;
    // per local slab: the remote slabs it sends to (= the remote slabs that send to it: H is Hermitian [A10]), each ONCE
    // however many segments go there -- at most GPUQT_MAX_SLABS - 1 entries, the size of d_signal / d_senders
    for (size_t i = 0; i < g->h.size(); ++i) {
        std::vector<unsigned int*> sig;
        std::vector<int> snd;
        for (const SlabSend& s : g->sends[i]) {
            if (s.peer_local >= 0) continue;
            auto it = g->remote.find(s.peer_global);
            if (it == g->remote.end()) continue;
            bool listed = false;
            for (int p : snd) listed = listed || p == s.peer_global;
            if (listed) continue;
            sig.push_back(it->second.flags + g->global_id[i]);
            snd.push_back(s.peer_global);
        }
        g->n_remote[i] = (int)sig.size();
        if (!sig.empty()) {
            GCU(cudaMemcpy(g->d_signal[i], sig.data(), sig.size() * sizeof(unsigned int*), cudaMemcpyHostToDevice));
            GCU(cudaMemcpy(g->d_senders[i], snd.data(), snd.size() * sizeof(int), cudaMemcpyHostToDevice));
        }
    }
    return GPUQT_OK;
}

int gpuqt_slab_set_wait_budget(gpuqt_slab_group* g, double seconds) {
    if (!g || !(seconds > 0.0) || !(seconds <= 3600.0)) return gfail(g, GPUQT_ERR_ARG, "the wait budget must lie in (0, 3600] seconds");
    g->wait_budget_ns = (unsigned long long)(seconds * 1e9);
    return GPUQT_OK;
}

static int slab_set_state_body(gpuqt_slab_group* g, const double* const* phi_host) {
    const size_t n = g->h.size();
    for (size_t i = 0; i < n; ++i) {
        gpuqt_handle* h = g->h[i];
        GCU(cudaMemcpyAsync(h->ring[0], phi_host[i], h->vec_elems * sizeof(double2), cudaMemcpyHostToDevice, g->stream));
        const long long total = (long long)h->vec_elems;
        const int blocks = (int)((total + 255) / 256);
        to_device_layout<<<blocks, 256, 0, g->stream>>>(h->N, h->B, h->ring[0], h->psi, nullptr);
        GCU(cudaGetLastError());
        if (g->modes & GPUQT_MODE_MSD) {
            zero_vec<<<blocks, 256, 0, g->stream>>>(total, h->chi);
            GCU(cudaGetLastError());
        }
        if (g->modes & GPUQT_MODE_VAC)
            GCU(cudaMemcpyAsync(h->va, h->psi, h->vec_elems * sizeof(double2), cudaMemcpyDeviceToDevice, g->stream));
        h->state_set = true;
    }
    if (g->modes & GPUQT_MODE_VAC) {          // b = V phi needs the halo rows of phi
        int rc = slab_fence(g);
        if (rc == GPUQT_OK) rc = slab_exchange(g, each_buffer(g, [&](size_t i) { return (const double2*)g->h[i]->psi; }));
        if (rc) return rc;
        for (size_t i = 0; i < n; ++i) GCU(launch_velocity(g->h[i], g->h[i]->psi, g->h[i]->vb));
    }
    g->state_set = true;
    return GPUQT_OK;
}

int gpuqt_slab_set_state(gpuqt_slab_group* g, const double* const* phi_host) {
    if (!g || !phi_host) return gfail(g, GPUQT_ERR_ARG, "null argument");
    for (size_t i = 0; i < g->h.size(); ++i)
        if (!phi_host[i]) return gfail(g, GPUQT_ERR_ARG, "null state of a slab");
    if (g->poisoned || (g->modes & GPUQT_MODE_VAC)) {          // b = V phi exchanges halos: every send peer must be there
        const int ready = slab_ready(g);
        if (ready) return ready;
    }
    return slab_done(g, slab_set_state_body(g, phi_host));
}

static int slab_check_moments(gpuqt_slab_group* g, int32_t n_moments, const double* out_host, int need_mode) {
    if (!g || !out_host || n_moments < 2 || n_moments > GPUQT_MAX_MOMENTS) return gfail(g, GPUQT_ERR_ARG, "bad n_moments or null output");
    if (need_mode && !(g->modes & need_mode)) return gfail(g, GPUQT_ERR_STATE, "group was created without the mode this call needs");
    if (!g->state_set) return gfail(g, GPUQT_ERR_STATE, "gpuqt_slab_set_state has not been called");
    return slab_ready(g);
}

// As gpuqt_dos_moments: psi is allocated and set in every mode, so a VAC-only group answers too.
int gpuqt_slab_dos_moments(gpuqt_slab_group* g, int32_t n_moments, double* out_host) {
    int rc = slab_check_moments(g, n_moments, out_host, 0);
    if (rc) return rc;
    return slab_done(g, slab_moments_doubling(g, false, n_moments, out_host));
}

int gpuqt_slab_msd(gpuqt_slab_group* g, int32_t n_moments, double* out_host) {
    int rc = slab_check_moments(g, n_moments, out_host, GPUQT_MODE_MSD);
    if (rc) return rc;
    return slab_done(g, slab_moments_doubling(g, true, n_moments, out_host));
}

static int slab_vac_body(gpuqt_slab_group* g, int32_t n_moments, double* out_host) {
    const size_t n = g->h.size();
    int rc;
    // phi_L = V a (needs the halo rows of a); C_0 = <phi_L|b>
    rc = slab_fence(g);
    if (rc == GPUQT_OK) rc = slab_exchange(g, each_buffer(g, [&](size_t i) { return (const double2*)g->h[i]->va; }));
    if (rc) return rc;
    std::vector<RecArgs> args(n);
    for (size_t i = 0; i < n; ++i) {
        gpuqt_handle* h = g->h[i];
        h->sweep = 0;
        GCU(launch_velocity(h, h->va, h->phiL));
        GCU(launch_dot(h, h->phiL, h->vb, h->dots));
        RecArgs a{};
        a.x0 = h->vb;
        a.phiL = h->phiL;
        a.terms = n_moments;
        a.dots = h->dots;
        a.dot_m0 = 0;
        args[i] = a;
    }
    rc = slab_recurrence(g, kModeLeft, args);
    if (rc) return rc;
    rc = slab_sum_dots(g, (long long)n_moments * 2 * g->B);
    if (rc) return rc;
    const int total = g->B * n_moments;
    finalize_left<<<(total + 255) / 256, 256, 0, g->stream>>>(g->B, n_moments, g->h[0]->dots, g->h[0]->moments);
    GCU(cudaGetLastError());
    return slab_copy_moments(g, n_moments, out_host);
}

int gpuqt_slab_vac(gpuqt_slab_group* g, int32_t n_moments, double* out_host) {
    int rc = slab_check_moments(g, n_moments, out_host, GPUQT_MODE_VAC);
    if (rc) return rc;
    return slab_done(g, slab_vac_body(g, n_moments, out_host));
}

static int slab_evolve_body(gpuqt_slab_group* g, double dt, int32_t order) {
    int rc;
    auto swap_all = [&](double2* gpuqt_handle::*a, double2* gpuqt_handle::*b) {
        for (gpuqt_handle* h : g->h) std::swap(h->*a, h->*b);
    };
    if (g->modes & GPUQT_MODE_MSD) {
        rc = slab_evolve_set(g, kModeEvolveMsd, [&](size_t i) { return (const double2*)g->h[i]->psi; },
                             [&](size_t i) { return (const double2*)g->h[i]->chi; }, [&](size_t i) { return g->h[i]->out0; },
                             [&](size_t i) { return g->h[i]->out1; }, dt, order);
        if (rc) return rc;
        swap_all(&gpuqt_handle::psi, &gpuqt_handle::out0);
        swap_all(&gpuqt_handle::chi, &gpuqt_handle::out1);
    } else if (g->modes & GPUQT_MODE_PSI) {
        rc = slab_evolve_set(g, kModeEvolve, [&](size_t i) { return (const double2*)g->h[i]->psi; },
                             [&](size_t i) { return (const double2*)nullptr; }, [&](size_t i) { return g->h[i]->out0; },
                             [&](size_t i) { return (double2*)nullptr; }, dt, order);
        if (rc) return rc;
        swap_all(&gpuqt_handle::psi, &gpuqt_handle::out0);
    }
    if (g->modes & GPUQT_MODE_VAC) {        // both VAC branches step with U(-dt)  [A1]
        rc = slab_evolve_set(g, kModeEvolve, [&](size_t i) { return (const double2*)g->h[i]->va; },
                             [&](size_t i) { return (const double2*)nullptr; }, [&](size_t i) { return g->h[i]->out0; },
                             [&](size_t i) { return (double2*)nullptr; }, -dt, order);
        if (rc) return rc;
        swap_all(&gpuqt_handle::va, &gpuqt_handle::out0);
        rc = slab_evolve_set(g, kModeEvolve, [&](size_t i) { return (const double2*)g->h[i]->vb; },
                             [&](size_t i) { return (const double2*)nullptr; }, [&](size_t i) { return g->h[i]->out0; },
                             [&](size_t i) { return (double2*)nullptr; }, -dt, order);
        if (rc) return rc;
        swap_all(&gpuqt_handle::vb, &gpuqt_handle::out0);
    }
    return GPUQT_OK;
}

int gpuqt_slab_evolve(gpuqt_slab_group* g, double dt, int32_t order) {
    if (!g || order < 1 || order > GPUQT_MAX_ORDER || !std::isfinite(dt)) return gfail(g, GPUQT_ERR_ARG, "bad dt or order");
    if (!g->state_set) return gfail(g, GPUQT_ERR_STATE, "gpuqt_slab_set_state has not been called");
    int rc = slab_ready(g);
    if (rc) return rc;
    return slab_done(g, slab_evolve_body(g, dt, order));
}

int gpuqt_slab_get_state(gpuqt_slab_group* g, int32_t local_slab, int which, double* out_host) {
    if (!g || local_slab < 0 || local_slab >= (int32_t)g->h.size() || !out_host) return gfail(g, GPUQT_ERR_ARG, "bad argument");
    if (g->poisoned) return slab_ready(g);
    gpuqt_handle* h = g->h[(size_t)local_slab];
    int rc = gpuqt_get_state(h, which, out_host);           // synchronises the stream
    if (rc) {
        g->err = h->err;
        return rc;
    }
    return slab_done(g, slab_sync(g));                      // a wait that gave up leaves halo rows, hence states, undefined
}

int gpuqt_slab_get_info(gpuqt_slab_group* g, int32_t local_slab, int what, int64_t* value) {
    if (!g || local_slab < 0 || local_slab >= (int32_t)g->h.size() || !value) return gfail(g, GPUQT_ERR_ARG, "bad argument");
    gpuqt_handle* h = g->h[(size_t)local_slab];
    const int rc = gpuqt_get_info(h, what, value);
    if (rc) g->err = h->err;
    return rc;
}

const char* gpuqt_slab_last_error(const gpuqt_slab_group* g) { return g ? g->err.c_str() : g_create_error.c_str(); }

void gpuqt_slab_destroy(gpuqt_slab_group* g) {
    if (!g) return;
    cudaStreamSynchronize(g->stream);
    for (gpuqt_handle* h : g->h) gpuqt_destroy(h);
    for (auto p : g->d_rows) if (p) cudaFree(p);
    for (auto p : g->d_flags) if (p) cudaFree(p);
    for (auto p : g->d_signal) if (p) cudaFree(p);
    for (auto p : g->d_senders) if (p) cudaFree(p);
    delete g;
}

}  // extern "C"
