#!/usr/bin/env python
"""bench.py — orbital-SpMV/s of the GPUQT hot path (Chebyshev evolution + KPM moments) on B200.

One "step" = one pass of the whole hot path over one batch of B random-phase vectors at one time
step of the workload: MSD configs: gpuqt_evolve(dt, N_p) (psi and chi with the fused commutator
walk) + gpuqt_msd(N_m) (doubling identity) + gpuqt_kpm_transform (Jackson + energy grid);
VAC configs: gpuqt_vac(N_m) + gpuqt_evolve(dt, N_p) + gpuqt_kpm_transform.

Unit: one orbital-SpMV = one row of one sparse matrix-vector walk for one vector, counted as the
CUDA path executes them: (N_p - 1) walks per evolved vector and N_m/2
(doubling) or N_m - 1 (VAC) walks per moment set.  The oracle legs are normalised to the SAME task
count, so value ratios are time ratios for the same job.

  python bench.py [--gpus N] [--steps K] [--warmup W] [--config c4] [--impl reference]
"""
import argparse
import json
import os
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

from workloads import configs  # noqa: E402

N_ENERGIES = 601      # PAPER.md:277-285, :359 (601 energy points)
FALLBACK_HBM_GBS = 6650.0


def walks_per_step(w, order):
    """(evolve walks, moment walks) per vector per step, as the CUDA path executes them."""
    if w.path == "msd":
        return 2 * (order - 1), w.n_moments // 2
    return 2 * (order - 1), 1 + (w.n_moments - 1)       # a and b branches; V a + N_m - 1 steps


L2_BYTES = 126e6      # B200 L2 (B200_PROFILING.md)


def contract_bytes_per_row(model, batch, kernel):
    """SURVEY 8(d)'s ELL-contract bytes one launch (= one recurrence step) moves per row: int32 index +
    fp64 (re, im) hopping per entry + on-site, and each vector element once per pass (evolve: with the
    read-modify-write of an accumulator the Clenshaw form does not have)."""
    cplx = model.hop_im is not None
    mat = model.K * (4 + (16 if cplx else 8)) + 8
    if kernel == "evolve_msd":                  # (psi, chi) pair: matrix once + x, two vector streams
        return mat + 8 + batch * 2 * 80
    return mat + batch * {"kpm_doubling": 48, "kpm_left": 64, "evolve": 80}[kernel]


def stored_bytes_per_row(model, batch, kernel, stored_matrix_bytes):
    """Bytes the stored layout must move per row and step: the packed records as gpuqt_create built
    them (no hopping array when the hopping is one constant, 16-bit columns where possible; from
    gpuqt_get_info), x for the commutator walk, and the vector streams the kernel really has
    (Clenshaw evolution: x_{m-1}, x_{m-2}, src read, x_m written = 64 B per vector)."""
    rec = (stored_matrix_bytes - 8 * (model.N + 1)) / model.N
    vec = {"kpm_doubling": 48, "kpm_left": 64, "evolve": 64, "evolve_msd": 128}[kernel] * batch
    return rec + vec + (8 if kernel == "evolve_msd" else 0)


def working_set_bytes(model, batch, kernel, stored_matrix_bytes):
    """Distinct bytes one step of the dominant kernel touches (what has to stay in L2 for the next step
    to find it there)."""
    streams = {"kpm_doubling": 3, "kpm_left": 4, "evolve": 4, "evolve_msd": 8}[kernel]
    return stored_matrix_bytes + streams * 16 * batch * model.N


def energies_for(model):
    e = 0.98 * model.energy_scale
    return np.linspace(-e, e, N_ENERGIES)


class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled during the timed region."""
    Q = ("clocks.sm,clocks.max.sm,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap,power.draw")

    def __init__(self, index):
        self.index, self.rows, self.proc = index, [], None

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits",
                                          "-lms", "100", "-i", str(self.index)], stdout=subprocess.PIPE, text=True)
            self.thread = threading.Thread(target=self._read, daemon=True)
            self.thread.start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append([c.strip() for c in line.split(",")])

    def stop(self):
        if not self.proc:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        self.thread.join(timeout=2)
        sm = [float(r[0]) for r in self.rows if len(r) >= 6 and r[0].replace(".", "").isdigit()]
        mx = [float(r[1]) for r in self.rows if len(r) >= 6 and r[1].replace(".", "").isdigit()]
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        reasons = [n for i, n in enumerate(names) if any(len(r) >= 6 and r[2 + i].startswith("Active") for r in self.rows)]
        pw = []
        for r in self.rows:
            try:
                pw.append(float(r[6]))
            except (IndexError, ValueError):
                pass
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "reasons": reasons, "samples": len(sm), "power_w": float(np.median(pw)) if pw else None}


TRAFFIC_SOURCES = ("paper_1705_01387_b200/csrc/kernels.cuh", "paper_1705_01387_b200/csrc/gpuqt.cu",
                   "paper_1705_01387_b200/csrc/step_kernels.cu", "paper_1705_01387_b200/csrc/host_util.h")


def kernel_source_hash():
    """sha256 over the sources of the step kernels and their launch logic: profiles/traffic.json carries the hash of the
    build its ncu captures were taken from, and its DRAM figures are quoted only while the sources still match."""
    import hashlib
    h = hashlib.sha256()
    for rel in TRAFFIC_SOURCES:
        with open(os.path.join(ROOT, rel), "rb") as f:
            h.update(f.read())
    return h.hexdigest()


def load_traffic():
    """(per-step DRAM bytes by 'config:kernel', stale?) from profiles/traffic.json; stale = the kernel sources have
    changed since the captures (then nothing is quoted)."""
    tp = os.path.join(ROOT, "profiles", "traffic.json")
    try:
        t = json.load(open(tp))
    except Exception:
        return {}, False
    if t.get("source_sha256") != kernel_source_hash():
        return {}, True
    return t, False


def measure_l2_gbs(torch, stream, reps=100):
    """L2-resident data rates for the configs whose recurrence step lives (partly) in the L2, measured in this run on
    the bench stream with CUDA events over `reps` back-to-back launches after 10 warm-up launches.  Candidates:
    device-to-device copies (read + write bytes) and read-only reductions (read bytes) over buffers that fit the 126 MB
    L2 with room to spare.  torch's copy / sum kernels serve as yardsticks only (as in MEASURED_PEAKS.json); they are
    not on the measured path.  Returns (best rate, {candidate: rate}): the best is the yardstick -- a LOWER bound of
    what the L2 can deliver (short launches, generic kernels), not a hardware ceiling."""
    out = {}

    def rate(fn, nbytes):
        with torch.cuda.stream(stream):
            for _ in range(10):
                fn()
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record(stream)
            for _ in range(reps):
                fn()
            e1.record(stream)
            stream.synchronize()
        return nbytes * reps / (e0.elapsed_time(e1) * 1e-3) / 1e9

    for mb in (24, 40):
        n = mb * 1000 * 1000 // 8
        with torch.cuda.stream(stream):
            a = torch.ones(n, dtype=torch.float64, device="cuda")
            b = torch.empty_like(a)
        out[f"copy_2x{mb}MB"] = rate(lambda: b.copy_(a), 2.0 * n * 8)
        del b
        out[f"sum_{mb}MB"] = rate(lambda: a.sum(), 1.0 * n * 8)
        del a
    with torch.cuda.stream(stream):
        a = torch.ones(80 * 1000 * 1000 // 8, dtype=torch.float64, device="cuda")
    out["sum_80MB"] = rate(lambda: a.sum(), 80e6)
    del a
    return max(out.values()), out


def residency(wset, stored, traffic):
    """'hbm-bound' / 'partly l2-resident' / 'l2-resident' for one recurrence step: from the measured DRAM bytes per
    step against the bytes the stored layout moves when an ncu capture of this build exists, else from the step's
    working set against the L2 size (a step that fits with room to spare stays; one well beyond it streams)."""
    if traffic:
        r = traffic / stored
        return "hbm-bound" if r > 0.85 else "l2-resident" if r < 0.25 else "partly l2-resident"
    return "hbm-bound" if wset > 1.5 * L2_BYTES else "l2-resident" if wset < 0.6 * L2_BYTES else "partly l2-resident"


def load_peak():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        try:
            return float(json.load(open(p))["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
        except Exception:
            pass
    return FALLBACK_HBM_GBS, "fallback (B200_PROFILING.md 6.65 TB/s)"


# ------------------------------------------------------------------------------------ oracle legs
def sample_moments(w, model):
    """Moments of the oracle's bounded sample: ~5e8 row-walks/s on 16 cores, aim at <= 1e10 row-walks."""
    return int(min(w.n_moments, max(16, (1e10 / model.N) // 2 * 2)))



def oracle_sample(w, model, order, seconds_hint=15.0):
    """Bounded sample of the workload's step on the CPU oracle: 1 vector, full N, the full evolve
    step, and a moment set sized for about 10-30 s of CPU work (the whole N_m when that fits).
    Returns (task-normalised orbital-SpMV, executed SpMV rows, seconds, cores, description)."""
    from oracle import oracle
    # ~5e8 row-walks/s on 16 cores: aim at <= 1e10 row-walks in the moment set
    nm_s = sample_moments(w, model)
    o = oracle.Oracle(model, batch=1, modes=oracle.MODE_MSD if w.path == "msd" else oracle.MODE_VAC)
    phi = w.phases(model)[:1]
    o.set_state(phi)
    t0 = time.perf_counter()
    if w.path == "msd":
        o.evolve(w.dt, order)
        o.msd(nm_s)
        task = model.N * (2 * (order - 1) + nm_s // 2)
        executed = model.N * (5 * (order - 1) + (nm_s - 1))      # U chi, U psi, [X,U] psi (3 walks) + moments
    else:
        o.vac(nm_s)
        o.evolve(w.dt, order)
        task = model.N * (2 * (order - 1) + nm_s)
        executed = model.N * (2 * (order - 1) + nm_s)
    dt = time.perf_counter() - t0
    cores = int(os.environ.get("OMP_NUM_THREADS", os.cpu_count() or 1))
    desc = (f"1 of {w.batch} vectors at full N={model.N}: one full evolve step (dt={w.dt}, N_p={order}) + a "
            f"{nm_s}-moment {w.path.upper()} set of {w.n_moments}; task-normalised count (same formula as the GPU leg)")
    o.close()
    return task, executed, dt, cores, desc


def oracle_one_thread(w, model, seconds_hint=8.0):
    """The oracle on ONE host thread ("once with 1 thread and once with all cores"): a short
    moment set of the workload's kind on 1 vector at full N, sized for about 10 s; executed row-walks / s."""
    import ctypes
    from oracle import oracle
    oracle.lib()
    gomp = ctypes.CDLL("libgomp.so.1")
    before = gomp.omp_get_max_threads()
    nm = int(max(4, min(w.n_moments, (seconds_hint * 3.5e7 / model.N) // 2 * 2)))
    o = oracle.Oracle(model, batch=1, modes=oracle.MODE_MSD if w.path == "msd" else oracle.MODE_VAC)
    o.set_state(w.phases(model)[:1])
    gomp.omp_set_num_threads(1)
    try:
        t0 = time.perf_counter()
        o.dos_moments(nm)                      # nm - 1 walks, no doubling
        dt = time.perf_counter() - t0
    finally:
        gomp.omp_set_num_threads(before)
    o.close()
    return model.N * (nm - 1) / dt, f"{nm}-moment DOS set on 1 vector at full N, {dt:.1f} s"


def run_reference(args, w):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    model = w.build()
    order = w.order
    times, task = [], 0
    for i in range(args.warmup + args.steps):
        task, executed, dt, cores, desc = oracle_sample(w, model, order)
        if i >= args.warmup:
            times.append(dt)
    total = sum(times)
    value = task * len(times) / total
    line = {"impl": "reference", "metric": "orbital-SpMV/s in Chebyshev evolution + KPM moments", "value": value,
            "unit": "orbital-SpMV/s", "n_gpus": args.gpus, "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": 1e3 * total / len(times), "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": w.key, "description": w.description, "N": model.N, "K": model.K,
                       "batch": 1, "n_moments_sampled": sample_moments(w, model), "order": order},
            "cpu_baseline": {"value": value, "unit": "orbital-SpMV/s", "cores": cores, "kind": "oracle", "sample": desc,
                             "executed_value": executed * len(times) / total},
            "e2e": {"value": value, "unit": "orbital-SpMV/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)



# ------------------------------------------------------------------------------------ CUDA leg
def run_ours(args, w):
    import torch
    import torch.distributed as dist
    import paper_1705_01387_b200 as gq
    from paper_1705_01387_b200 import binding

    from paper_1705_01387_b200 import replicas
    rank, local, world = replicas.world()
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))

    model = w.build()
    order = w.order
    modes = gq.MODE_MSD if w.path == "msd" else gq.MODE_VAC
    stream = torch.cuda.Stream()
    with torch.cuda.stream(stream):
        g = gq.GpuQT(model, batch=w.batch, modes=modes, stream=stream, options=args.options)
        # replicas over random vectors: rank r owns vectors [r*B, (r+1)*B)
        phi_host = torch.from_numpy(w.phases(model, first_vector=replicas.first_vector(rank, w.batch))).pin_memory()
        phi_dev = phi_host.to("cuda", non_blocking=True)
        mom_host = torch.empty((w.batch, w.n_moments), dtype=torch.float64).pin_memory()
        energies = energies_for(model)
        stream.synchronize()

        copy_ev = []                                # (start, stop) pairs around the e2e host->device load

        def step(e2e):
            if e2e:
                e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                e0.record(stream)
                if e2e == "serial":
                    g.set_state(phi_host)          # H2D of this step's input from pinned memory (+ layout change, V phi)
                else:
                    # the upload of this step's vectors was started one step ago on the library's copy stream
                    # (gpuqt_prefetch_state) and has overlapped that step's compute; start the next one now
                    g.set_state_prefetched()
                    g.prefetch_state(phi_host)
                e1.record(stream)
                copy_ev.append((e0, e1))
            if w.path == "msd":
                g.evolve(w.dt, order)
                g.msd(w.n_moments, out=mom_host)   # D2H of the step's result
            else:
                g.vac(w.n_moments, out=mom_host)
                g.evolve(w.dt, order)
            out = g.kpm_transform(mom_host.numpy(), energies)
            if e2e and world > 1:                  # the one exchange of the replicas scheme: all ranks' moment blocks
                replicas.gather_moments(mom_host.to("cuda", non_blocking=True))
            return out

        def barrier():
            if world > 1:
                dist.barrier()
            torch.cuda.synchronize()

        def timed(e2e):
            g.set_state_device(phi_dev)
            if e2e == "overlap":
                g.prefetch_state(phi_host)         # the first step's upload
            for _ in range(args.warmup):
                step(e2e)
            g.reset_stats()
            copy_ev.clear()
            barrier()
            ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            ev0.record(stream)
            for _ in range(args.steps):
                out = step(e2e)
            ev1.record(stream)
            barrier()
            ms = ev0.elapsed_time(ev1)
            return replicas.max_over_ranks(ms, device="cuda"), out

        sampler = ClockSampler(local)
        if not args.no_clock_sampler:
            sampler.start()
        ms, out = timed(False)
        clocks = sampler.stop()
        stats = {c: (g.kernel_stats(c)[0], g.kernel_steps(c), g.kernel_stats(c)[1]) for c in range(5)}   # (ms, steps, launches)
        n_launches = sum(stats[c][2] for c in range(5))
        ms_e2e_serial, _ = timed("serial")
        set_state_ms = sum(a.elapsed_time(b) for a, b in copy_ev) / max(len(copy_ev), 1)
        ms_e2e, _ = timed("overlap")
        # the bare pinned H2D copy of the same bytes, alone on the stream (for the PCIe rate)
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(stream)
        phi_dev.copy_(phi_host, non_blocking=True)
        e1.record(stream)
        stream.synchronize()
        h2d_ms = e0.elapsed_time(e1)
        info = {k: g.info(getattr(binding, "INFO_" + k)) for k in ("STORED_MATRIX_BYTES", "HOP_VARIANT", "SMALL_PATH", "PERSISTENT", "REORDERED")}

    ev_w, mom_w = walks_per_step(w, order)
    units_step = model.N * w.batch * (ev_w + mom_w) * world
    value = units_step * args.steps / (ms * 1e-3)
    e2e_value = units_step * args.steps / (ms_e2e * 1e-3)
    assert np.all(np.isfinite(out)), "non-finite result"

    if rank == 0:
        # one roofline entry per kernel class with >= 5 % of the timed region; the dominant one (most device time) on top
        names = {0: "kpm_doubling", 1: "kpm_left", 2: "evolve", 3: "evolve_msd"}
        peak, peak_src = load_peak()
        traffic_table, traffic_stale = load_traffic()
        l2_peak, l2_candidates = None, None

        def entry(c):
            nonlocal l2_peak, l2_candidates
            kernel = names[c]
            c_ms, c_steps, c_launches = stats[c]
            step_s = c_ms * 1e-3 / max(c_steps, 1)                 # one recurrence step of that kernel
            stored = stored_bytes_per_row(model, w.batch, kernel, info["STORED_MATRIX_BYTES"]) * model.N
            contract = contract_bytes_per_row(model, w.batch, kernel) * model.N
            wset = working_set_bytes(model, w.batch, kernel, info["STORED_MATRIX_BYTES"])
            traffic = traffic_table.get(f"{w.key}:{kernel}")
            where = residency(wset, stored, traffic)
            achieved = stored / step_s / 1e9
            e = {"kernel": kernel, "residency": where, "achieved": achieved, "unit": "GB/s",
                 "traffic": traffic, "bytes_per_launch": stored, "contract_bytes_per_launch": contract,
                 "contract_gbs": contract / step_s / 1e9,
                 "dram_gbs_from_ncu_traffic": (traffic / step_s / 1e9) if traffic else None,
                 "working_set_bytes": wset, "avg_step_us": step_s * 1e6, "steps": c_steps, "launches": c_launches,
                 "share_of_step": c_ms / ms}
            if where == "hbm-bound":
                e.update({"bound": "hbm", "peak": peak, "peak_source": peak_src, "frac": achieved / peak,
                          "contract_frac": contract / step_s / 1e9 / peak, "frac_of_nominal_8000": achieved / 8000.0,
                          "dram_frac_from_ncu_traffic": (traffic / step_s / 1e9 / peak) if traffic else None})
            else:           # the step is served (partly) from the L2: an HBM fraction would exceed 1 and say nothing
                if l2_peak is None:
                    l2_peak, l2_candidates = measure_l2_gbs(torch, stream)
                frac = achieved / l2_peak
                e.update({"bound": "l2", "peak": l2_peak, "frac": frac if frac <= 1.0 else None,
                          "peak_source": "measured in this run: the best of the L2-resident copy / read-only reduction rates "
                                         "in l2_yardsticks_gbs (bench.py measure_l2_gbs; torch kernels as yardsticks, a lower "
                                         "bound of the L2's rate, not a hardware ceiling)",
                          "l2_yardsticks_gbs": l2_candidates, "hbm_peak": peak, "hbm_peak_source": peak_src,
                          "dram_share_of_stored_bytes": (traffic / stored) if traffic else None})
                if frac > 1.0:
                    e["frac_note"] = ("the kernel moves its stored bytes %.2f x faster than the best L2 yardstick of this run: "
                                      "no ceiling is known for this step, so no fraction is quoted" % frac)
            return e

        big = sorted((c for c in names if stats[c][0] >= 0.05 * ms), key=lambda c: -stats[c][0]) or [max(names, key=lambda c: stats[c][0])]
        entries = [entry(c) for c in big]
        top = entries[0]
        wset = top["working_set_bytes"]
        l2_note = {"l2-resident": "working set of a recurrence step %.0f MB < 126 MB L2: the %d dependent steps of a moment set "
                                  "re-read it by construction (no flush is possible inside a step); the roofline is set against "
                                  "a measured L2 copy rate, not HBM" % (wset / 1e6, w.n_moments),
                   "partly l2-resident": "working set of a recurrence step %.0f MB is about the size of the 126 MB L2: part of "
                                         "it survives from step to step (no flush is possible inside a recurrence); the roofline "
                                         "is set against a measured L2 copy rate, the DRAM share is in roofline.traffic"
                                         % (wset / 1e6),
                   "hbm-bound": "inputs larger than L2: a recurrence step touches %.0f MB (vector set %.0f MB, stored matrix "
                                "%.0f MB) vs 126 MB L2; no flush" % (wset / 1e6, model.N * w.batch * 16 / 1e6,
                                                                      info["STORED_MATRIX_BYTES"] / 1e6)}[top["residency"]]
        launches = n_launches + args.steps * 3      # + finalize, damping, transform
        line = {"metric": "orbital-SpMV/s in Chebyshev evolution + KPM moments", "value": value,
                "unit": "orbital-SpMV/s", "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
                "ms_per_step": ms / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
                "dtype": "f64", "data": "synthetic",
                "config": {"workload": w.key, "description": w.description, "N": model.N, "K": model.K,
                           "batch_per_gpu": w.batch, "n_moments": w.n_moments, "order": order, "dt": w.dt,
                           "n_energies": N_ENERGIES, "path": w.path, "l2": l2_note,
                           "storage": {"hop_variant": ["real", "complex", "constant, int32 columns", "constant, 16-bit columns",
                                                       "constant, 16-bit columns with padding",
                                                       "constant, implicit stencil (pattern dictionary, no index array)"][info["HOP_VARIANT"]],
                                       "stored_matrix_bytes": info["STORED_MATRIX_BYTES"],
                                       "site_order": "bricks of 4 x 4 x 2 sites per slice (recognised cubic lattice)" if info["REORDERED"]
                                                     else "the caller's",
                                       "launch_form": "one-CTA whole-recurrence kernel" if info["SMALL_PATH"] else
                                                      "one cooperative launch per recurrence" if info["PERSISTENT"] else
                                                      "one launch per recurrence step"},
                           "parallelism": f"replicas-over-vectors x{world}",
                           "seconds_per_time_step": ms / args.steps * 1e-3,
                           **({"options": args.options} if args.options else {})},
                "clocks": clocks,
                "e2e": {"value": e2e_value, "unit": "orbital-SpMV/s", "ms_per_step": ms_e2e / args.steps,
                        "h2d_bytes_per_step": int(phi_host.numel() * 8 + (w.n_moments * w.batch + N_ENERGIES) * 8),
                        "d2h_bytes_per_step": int(mom_host.numel() * 8 + w.batch * N_ENERGIES * 8),
                        "set_state_ms_per_step": set_state_ms,
                        "value_without_overlap": units_step * args.steps / (ms_e2e_serial * 1e-3),
                        "ms_per_step_without_overlap": ms_e2e_serial / args.steps,
                        "overlap": "every step uploads one batch of random vectors from pinned host memory inside the timed "
                                   "region; the upload consumed by step k+1 is issued at the start of step k on the library's "
                                   "copy stream (gpuqt_prefetch_state / gpuqt_set_state_prefetched) and overlaps its compute; "
                                   "value_without_overlap is the same loop with gpuqt_set_state (copy, then compute)",
                        "h2d_copy_alone_ms": h2d_ms, "h2d_copy_alone_gbs": phi_host.numel() * 8 / (h2d_ms * 1e-3) / 1e9,
                        "note": "set_state_ms_per_step = gpuqt_set_state in the loop without overlap: pinned H2D copy of the B "
                                "random vectors + layout change (+ V phi in VAC mode), timed with its own CUDA events; the "
                                "bare copy is timed alone afterwards"},
                "gpu_launches": int(launches),
                "roofline": {**top,
                             "bytes_note": "achieved = bytes the STORED layout moves per recurrence step (records as built + "
                                           "vector streams) / average step time; the ELL contract of SURVEY 8(d) (int32 + fp64 "
                                           "per entry) is kept beside it as contract_*; traffic = DRAM bytes per step from the "
                                           "ncu captures named in profiles/traffic.json, quoted only while the kernel sources "
                                           "hash to the build they were taken from",
                             "traffic_stale": bool(traffic_stale),
                             "l2_resident": top["residency"] != "hbm-bound",
                             "kernels": entries,
                             "per_class_ms": {names[c]: stats[c][0] for c in names}},
                }
        if world == 1 and not args.no_cpu_baseline:
            task, executed, dt, cores, desc = oracle_sample(w, model, order)
            one, one_desc = oracle_one_thread(w, model)
            line["cpu_baseline"] = {"value": task / dt, "unit": "orbital-SpMV/s", "cores": cores, "kind": "oracle",
                                    "sample": desc, "seconds": dt, "executed_value": executed / dt,
                                    "executed_value_1_thread": one, "sample_1_thread": one_desc}
        print(json.dumps(line), flush=True)
    g.close()
    if world > 1:
        dist.destroy_process_group()


def run_slabs(args, w):
    """Secondary measurement (not the bench contract's line): the workload cut into --slabs row slabs, all resident
    on this one GPU (the multi-GPU decomposition emulated on one device: same launches and halo
    pushes, no cross-GPU flags).  Shows what the decomposition costs against the single-handle path."""
    import torch
    import paper_1705_01387_b200 as gq
    from paper_1705_01387_b200 import slab
    torch.cuda.set_device(0)
    model = w.build()
    order = w.order
    modes = gq.MODE_MSD if w.path == "msd" else gq.MODE_VAC
    stream = torch.cuda.Stream()
    with torch.cuda.stream(stream):
        slabs = slab.partition(model, args.slabs)
        g = slab.SlabGroup(model, slabs, batch=w.batch, modes=modes, stream=stream)
        g.set_state(w.phases(model))

        def step():
            if w.path == "msd":
                g.evolve(w.dt, order)
                return g.msd(w.n_moments, reduce=False)
            out = g.vac(w.n_moments, reduce=False)
            g.evolve(w.dt, order)
            return out

        for _ in range(args.warmup):
            step()
        torch.cuda.synchronize()
        ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        ev0.record(stream)
        for _ in range(args.steps):
            out = step()
        ev1.record(stream)
        torch.cuda.synchronize()
        ms = ev0.elapsed_time(ev1)
    ev_w, mom_w = walks_per_step(w, order)
    value = model.N * w.batch * (ev_w + mom_w) * args.steps / (ms * 1e-3)
    assert np.all(np.isfinite(out))
    print(json.dumps({"metric": "orbital-SpMV/s in Chebyshev evolution + KPM moments", "value": value, "unit": "orbital-SpMV/s",
                      "n_gpus": 1, "steps": args.steps, "warmup": args.warmup, "ms_per_step": ms / args.steps,
                      "higher_is_better": True, "dtype": "f64", "data": "synthetic",
                      "config": {"workload": w.key, "N": model.N, "batch_per_gpu": w.batch, "n_moments": w.n_moments,
                                 "order": order, "slabs": args.slabs, "slabs_resident_on_one_gpu": True,
                                 "rows_per_slab": [s.n_own for s in slabs], "halo_rows_per_slab": [s.n_halo for s in slabs],
                                 "note": "row-slab decomposition emulated on one device; no kpm_transform in this line"}}),
          flush=True)
    g.close()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", default="c4", choices=sorted(configs.WORKLOADS))
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-clock-sampler", action="store_true", help="diagnostic: do not poll nvidia-smi during the timed region")
    ap.add_argument("--opt", action="append", default=[], metavar="KEY=VALUE",
                    help="gpuqt_options override for tuning runs, e.g. --opt persistent=0 (default: the library defaults)")
    ap.add_argument("--slabs", type=int, default=0,
                    help="secondary measurement: cut the workload into this many row slabs resident on ONE GPU (SURVEY 8(f) 4)")
    args = ap.parse_args()
    args.options = {k: int(v) for k, v in (kv.split("=", 1) for kv in args.opt)}
    w = configs.WORKLOADS[args.config]
    from paper_1705_01387_b200 import replicas
    if args.impl == "ours" and args.slabs == 0 and replicas.needs_launch(args.gpus):
        # --gpus N without torchrun around it: start the N ranks ourselves (one process per GPU, NCCL), rank 0 prints
        import torch
        have = torch.cuda.device_count()
        if have < args.gpus:
            sys.exit(f"bench.py: --gpus {args.gpus} but {have} CUDA device(s) are visible")
        env = dict(os.environ)
        env.setdefault("NCCL_DEBUG", "INFO")          # the communicator lines (transport, NVLS) go to stderr
        cmd = replicas.launch_command(os.path.abspath(__file__), sys.argv[1:], args.gpus, replicas.free_port())
        sys.exit(subprocess.call(cmd, env=env))
    if args.impl == "ours" and args.slabs == 0 and args.gpus != replicas.world()[2]:
        sys.exit(f"bench.py: --gpus {args.gpus} does not match WORLD_SIZE={replicas.world()[2]}")
    if args.impl == "reference":
        run_reference(args, w)
    elif args.slabs > 0:
        run_slabs(args, w)
    else:
        run_ours(args, w)


if __name__ == "__main__":
    main()
