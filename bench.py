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


def bytes_per_orbital_spmv(model, batch, kind):
    """Algorithmic bytes of one orbital-SpMV from the sliced-ELL layout."""
    cplx = model.hop_im is not None
    mat = model.K * (4 + (16 if cplx else 8)) + 8
    vec = {"kpm_doubling": 48, "kpm_left": 64, "evolve": 80}[kind]
    return mat / batch + vec


def energies_for(model):
    e = 0.98 * model.energy_scale
    return np.linspace(-e, e, N_ENERGIES)


class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled during the timed region."""
    Q = ("clocks.sm,clocks.max.sm,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

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
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "reasons": reasons, "samples": len(sm)}


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


def run_reference(args, w):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    from paper_1705_01387_b200 import binding
    model = w.build()
    order = w.order or binding.choose_order(model.energy_scale, w.dt)
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
    order = w.order or binding.choose_order(model.energy_scale, w.dt)
    modes = gq.MODE_MSD if w.path == "msd" else gq.MODE_VAC
    stream = torch.cuda.Stream()
    with torch.cuda.stream(stream):
        g = gq.GpuQT(model, batch=w.batch, modes=modes, stream=stream)
        # replicas over random vectors: rank r owns vectors [r*B, (r+1)*B)
        phi_host = torch.from_numpy(w.phases(model, first_vector=replicas.first_vector(rank, w.batch))).pin_memory()
        phi_dev = phi_host.to("cuda", non_blocking=True)
        mom_host = torch.empty((w.batch, w.n_moments), dtype=torch.float64).pin_memory()
        energies = energies_for(model)
        stream.synchronize()

        def step(e2e):
            if e2e:
                g.set_state(phi_host)              # H2D of this step's input from pinned memory
            if w.path == "msd":
                g.evolve(w.dt, order)
                g.msd(w.n_moments, out=mom_host)   # D2H of the step's result
            else:
                g.vac(w.n_moments, out=mom_host)
                g.evolve(w.dt, order)
            return g.kpm_transform(mom_host.numpy(), energies)

        def barrier():
            if world > 1:
                dist.barrier()
            torch.cuda.synchronize()

        def timed(e2e):
            g.set_state_device(phi_dev)
            for _ in range(args.warmup):
                step(e2e)
            g.reset_stats()
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
        stats = {c: (g.kernel_stats(c)[0], g.kernel_steps(c)) for c in range(5)}       # (ms, recurrence steps)
        n_launches = sum(g.kernel_stats(c)[1] for c in range(5))
        ms_e2e, _ = timed(True)

    ev_w, mom_w = walks_per_step(w, order)
    units_step = model.N * w.batch * (ev_w + mom_w) * world
    value = units_step * args.steps / (ms * 1e-3)
    e2e_value = units_step * args.steps / (ms_e2e * 1e-3)
    assert np.all(np.isfinite(out)), "non-finite result"

    if rank == 0:
        # roofline of the dominant kernel class (most device time in the timed region)
        names = {0: "kpm_doubling", 1: "kpm_left", 2: "evolve", 3: "evolve_msd"}
        dom = max(names, key=lambda c: stats[c][0])
        kind = {0: "kpm_doubling", 1: "kpm_left", 2: "evolve", 3: "evolve"}[dom]
        bpo = bytes_per_orbital_spmv(model, w.batch, kind)
        if dom == 3:   # (psi, chi) pair: matrix read once + x, two vector streams
            cplx = model.hop_im is not None
            per_row_launch = (model.K * (4 + (16 if cplx else 8)) + 8 + 8) + w.batch * 2 * 80
        else:
            per_row_launch = bpo * w.batch
        # bytes the stored layout really holds per row (constant-hopping records carry no hop array)
        hop_const = model.hop_im is None and (model.hop_re is None or np.unique(
            model.hop_re.reshape(model.N, model.K)[np.arange(model.K)[None, :] < model.nbr_count[:, None]]).size <= 1)
        hop_const = hop_const and os.environ.get("GPUQT_HOP_CONST", "1") != "0"
        stored_row_launch = per_row_launch - (8 * model.K if hop_const else 0)
        # ... and 16-bit columns (base + delta) when the table is uniform, unpadded and N % 32 == 0
        if (hop_const and model.K in (3, 4, 6) and model.N % 32 == 0 and int(model.nbr_count.min()) == model.K
                and os.environ.get("GPUQT_IDX16", "1") != "0"):
            stored_row_launch -= 2 * model.K - 1
        dom_ms, dom_n = stats[dom]
        achieved = per_row_launch * model.N / (dom_ms * 1e-3 / max(dom_n, 1)) / 1e9
        peak, peak_src = load_peak()
        traffic = None
        tp = os.path.join(ROOT, "profiles", "traffic.json")
        if os.path.exists(tp):
            try:
                traffic = json.load(open(tp)).get(f"{w.key}:{names[dom]}")
            except Exception:
                traffic = None
        launches = n_launches + args.steps * 3      # + finalize, jackson, transform
        line = {"metric": "orbital-SpMV/s in Chebyshev evolution + KPM moments", "value": value,
                "unit": "orbital-SpMV/s", "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
                "ms_per_step": ms / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
                "dtype": "f64", "data": "synthetic",
                "config": {"workload": w.key, "description": w.description, "N": model.N, "K": model.K,
                           "batch_per_gpu": w.batch, "n_moments": w.n_moments, "order": order, "dt": w.dt,
                           "n_energies": N_ENERGIES, "path": w.path,
                           "l2": "inputs larger than L2 (each vector set %.0f MB, matrix %.0f MB vs 126 MB L2); no flush"
                                 % (model.N * w.batch * 16 / 1e6,
                                    model.N * (model.K * (20 if model.hop_im is not None else 12) + 8) / 1e6),
                           "parallelism": f"replicas-over-vectors x{world}",
                           "seconds_per_time_step": ms / args.steps * 1e-3},
                "clocks": clocks,
                "e2e": {"value": e2e_value, "unit": "orbital-SpMV/s", "ms_per_step": ms_e2e / args.steps,
                        "h2d_bytes_per_step": int(phi_host.numel() * 8 + (w.n_moments * w.batch + N_ENERGIES) * 8),
                        "d2h_bytes_per_step": int(mom_host.numel() * 8 + w.batch * N_ENERGIES * 8)},
                "gpu_launches": int(launches),
                "roofline": {"bound": "hbm", "kernel": names[dom], "achieved": achieved, "peak": peak,
                             "unit": "GB/s", "frac": achieved / peak, "traffic": traffic, "peak_source": peak_src,
                             "frac_of_nominal_8000": achieved / 8000.0,
                             "bytes_per_launch": per_row_launch * model.N,
                             "stored_bytes_per_launch": stored_row_launch * model.N,
                             "stored_gbs": stored_row_launch * model.N / (dom_ms * 1e-3 / max(dom_n, 1)) / 1e9,
                             "avg_launch_us": dom_ms * 1e3 / max(dom_n, 1), "launches": dom_n,
                             "note": "launches = recurrence steps; one step per kernel launch by default, two per "
                                     "launch with GPUQT_FUSE=1 (bytes and time are then both per step)",
                             "share_of_step": dom_ms / ms,
                             "per_class_ms": {names[c]: stats[c][0] for c in names}},
                }
        if world == 1 and not args.no_cpu_baseline:
            task, executed, dt, cores, desc = oracle_sample(w, model, order)
            line["cpu_baseline"] = {"value": task / dt, "unit": "orbital-SpMV/s", "cores": cores, "kind": "oracle",
                                    "sample": desc, "seconds": dt, "executed_value": executed / dt}
        print(json.dumps(line), flush=True)
    g.close()
    if world > 1:
        dist.destroy_process_group()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", default="c4", choices=sorted(configs.WORKLOADS))
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-clock-sampler", action="store_true", help="diagnostic: do not poll nvidia-smi during the timed region")
    args = ap.parse_args()
    w = configs.WORKLOADS[args.config]
    if args.impl == "reference":
        run_reference(args, w)
    else:
        run_ours(args, w)


if __name__ == "__main__":
    main()
