"""The paper's simulation loop on top of the C-ABI calls (PAPER.md:134-205 section 3, :343-347 the
output rows, :359-409 the two examples): DOS, VAC and/or MSD at every time step on an energy grid,
averaged over the B random vectors of the handle, and the running conductivities of Eq. 2 / Eq. 5.

Call sequencing only -- every number is produced by libgpuqt.so's kernels (`engine` is a
`binding.GpuQT`; anything with the same methods works, which is how the tests drive the oracle
through the identical loop).
"""
import numpy as np


def time_axis(dts):
    """t_0 = 0, t_k = sum_{i<k} dt_i."""
    return np.concatenate([[0.0], np.cumsum(np.asarray(dts, np.float64))])


def run(engine, phi, dts, n_moments, energies, order_of, vac=True, msd=True, per_vector=False):
    """One pass of the method for the handle's B random vectors.

    phi       host [B][N][2] random-phase vectors
    dts       time steps (may be non-uniform)
    order_of  callable dt -> N_p (number of Chebyshev terms of that step, [A5])
    Row conventions [A4]: VAC row k is measured at t_k BEFORE step k (N_t rows, the last evolution of
    the VAC branches is skipped only if MSD is off); MSD row k is measured at t_{k+1} AFTER step k.
    Returns a dict of arrays averaged over the B vectors: dos [n_E], rho_vac / rho_msd [N_t][n_E]
    (= rho C_vv, rho dX^2), sigma_vac (at t_k), sigma_msd (at the middle of step k), length (Eq. 11), xi (Eq. 12 read
    at the last time) with xi_growth (relative change of the length over the last step: the saturation check).
    With per_vector=True nothing is averaged and no conductivity is formed: dos [B][n_E], rho_vac /
    rho_msd [N_t][B][n_E] -- the rows of the paper's dos.out / vac.out / msd.out.
    """
    dts = np.asarray(dts, np.float64)
    energies = np.ascontiguousarray(energies, np.float64)
    engine.set_state(phi)
    out = {"times": time_axis(dts), "energies": energies}
    avg = (lambda a: a) if per_vector else (lambda a: a.mean(axis=0))
    dos = avg(engine.kpm_transform(engine.dos_moments(n_moments), energies))
    out["dos"] = dos
    vac_rows, msd_rows = [], []
    for k, dt in enumerate(dts):
        if vac:
            vac_rows.append(avg(engine.kpm_transform(engine.vac(n_moments), energies)))
        if msd or k + 1 < len(dts):
            engine.evolve(float(dt), int(order_of(float(dt))))
        if msd:
            msd_rows.append(avg(engine.kpm_transform(engine.msd(n_moments), energies)))
    if vac:
        out["rho_vac"] = np.array(vac_rows).reshape((len(vac_rows),) + np.shape(dos))
    if msd:
        out["rho_msd"] = np.array(msd_rows).reshape((len(msd_rows),) + np.shape(dos))
    if per_vector:
        return out
    if vac:
        out["sigma_vac"], _ = engine.running_conductivity("vac", out["rho_vac"], dos, dts[:len(dts) - 1])
    if msd:
        out["sigma_msd"], out["length"] = engine.running_conductivity("msd", out["rho_msd"], dos, dts)
        out["xi"], out["xi_growth"] = engine.localization_length(out["length"])
    return out


def semiclassical(sigma):
    """sigma_sc(E) = max_t sigma(E, t)."""
    return np.max(np.asarray(sigma), axis=0)
