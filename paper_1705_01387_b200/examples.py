"""Run one of the paper's two examples end to end on the GPU and print a JSON
summary: `python -m paper_1705_01387_b200.examples e1 [--scale 0.25]`.

Inputs are the seeded synthetic lattices of workloads/configs.py (the paper's make_inputs.cpp is not
available); the printed observables are the ones the paper discusses for its figures.
"""
import argparse
import json
import os
import sys
import time

import numpy as np

sys.path.insert(0, os.path.dirname(os.path.dirname(os.path.abspath(__file__))))


def run_example(key, scale=1.0):
    import torch
    from workloads import configs
    from . import binding, transport
    ex = configs.EXAMPLES[key]
    model = ex.build(scale)
    modes = (binding.MODE_VAC if ex.vac else 0) | (binding.MODE_MSD if ex.msd else 0)
    g = binding.GpuQT(model, batch=ex.batch, modes=modes)
    phi = ex.phases(model)
    torch.cuda.synchronize()
    t0 = time.perf_counter()
    res = transport.run(g, phi, ex.dts, ex.n_moments, ex.energies(),
                        lambda dt: binding.choose_order(model.energy_scale, dt), vac=ex.vac, msd=ex.msd)
    torch.cuda.synchronize()
    res["seconds"] = time.perf_counter() - t0
    res["model"] = model
    g.close()
    return ex, res


def summary(ex, res):
    E = res["energies"]
    j0 = int(np.argmin(np.abs(E)))
    out = {"example": ex.key, "description": ex.description, "N": res["model"].N, "seconds": res["seconds"],
           "n_energies": int(E.size), "n_time_steps": len(ex.dts), "dos_at_0": float(res["dos"][j0]),
           "dos_integral": float(np.trapezoid(res["dos"], E))}
    if ex.vac:
        out["vac_at_0_over_time"] = (res["rho_vac"][:, j0] / res["dos"][j0]).tolist()
        out["sigma_vac_at_0"] = res["sigma_vac"][:, j0].tolist()
    if ex.msd:
        out["msd_at_0_over_time"] = (res["rho_msd"][:, j0] / res["dos"][j0]).tolist()
        out["sigma_msd_at_0"] = res["sigma_msd"][:, j0].tolist()
        out["length_at_0"] = res["length"][:, j0].tolist()
        out["xi_at_0"] = float(res["xi"][j0])                      # Eq. 12 at the last time; meaningful once xi_growth ~ 0
        out["xi_growth_at_0"] = float(res["xi_growth"][j0])
    return out


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("example", choices=["e1", "e2"])
    ap.add_argument("--scale", type=float, default=1.0, help="linear size factor (1 = the paper's size)")
    args = ap.parse_args()
    ex, res = run_example(args.example, args.scale)
    print(json.dumps(summary(ex, res)))


if __name__ == "__main__":
    main()
