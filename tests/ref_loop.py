"""Test-side restatement of the paper's simulation loop (PAPER.md:333-347 output rows, reading [A4]) and of
the N_p tail rule [A5], written against the ORACLE only.  It shares no code with the product's
paper_1705_01387_b200/transport.py and binding.choose_order, which the tests compare with it.
"""
import numpy as np


def order_rule(oracle_mod, dE, dt, tol=1e-15):
    """Smallest N_p with |J_m(dE |dt|)| < tol for every m >= N_p, from the oracle's libm jn() table."""
    x = dE * abs(dt)
    n = int(x) + 100 + int(5 * np.sqrt(x + 1))
    c = oracle_mod.bessel_coeffs(dE, dt, n)            # c_m = (2 - delta_m0) (-i)^m J_m
    J = np.abs(c)
    J[1:] *= 0.5
    last = -1
    for m in range(n):
        if J[m] >= tol:
            last = m
    return last + 1 if last >= 0 else 1


def simulation_loop(oracle_mod, model, phi, dts, n_moments, energies, vac, msd):
    """DOS, then for every time step k: the VAC row at t_k = sum_{i<k} dt_i (BEFORE the step), the step,
    the MSD row at t_{k+1} (AFTER it).  Averages over the B vectors; conductivities by the oracle's
    running_conductivity.  Returns a dict with the names transport.run uses."""
    B = phi.shape[0]
    modes = (oracle_mod.MODE_VAC if vac else 0) | (oracle_mod.MODE_MSD if msd else 0)
    o = oracle_mod.Oracle(model, batch=B, modes=modes)
    o.set_state(phi)
    dE = model.energy_scale
    res = {"dos": o.kpm_transform(o.dos_moments(n_moments), energies).mean(axis=0)}
    rows_v, rows_m = [], []
    n_t = len(dts)
    k = 0
    while k < n_t:
        if vac:
            rows_v.append(o.kpm_transform(o.vac(n_moments), energies).mean(axis=0))
        last = (k == n_t - 1)
        if msd or not last:                     # the evolution after the last VAC row is never used
            o.evolve(float(dts[k]), order_rule(oracle_mod, dE, float(dts[k])))
        if msd:
            rows_m.append(o.kpm_transform(o.msd(n_moments), energies).mean(axis=0))
        k += 1
    if vac:
        res["rho_vac"] = np.array(rows_v)
        res["sigma_vac"], _ = oracle_mod.running_conductivity("vac", res["rho_vac"], res["dos"], np.asarray(dts[:n_t - 1], float))
    if msd:
        res["rho_msd"] = np.array(rows_m)
        res["sigma_msd"], res["length"] = oracle_mod.running_conductivity("msd", res["rho_msd"], res["dos"], np.asarray(dts, float))
        res["xi"], res["xi_growth"] = oracle_mod.localization_length(res["length"])
    o.close()
    return res


def per_vector_rows(oracle_mod, model, phi, dts, n_moments, energies, vac, msd):
    """The rows of the paper's dos.out / vac.out / msd.out, vector by vector, each vector
    run ALONE through the oracle: dos [B][n_E]; vac, msd [B][N_t][n_E] (VAC row k before step k, MSD row k
    after it)."""
    B, n_t = phi.shape[0], len(dts)
    modes = (oracle_mod.MODE_VAC if vac else 0) | (oracle_mod.MODE_MSD if msd else 0)
    dos, rv, rm = [], [], []
    for b in range(B):
        o = oracle_mod.Oracle(model, batch=1, modes=modes)
        o.set_state(phi[b:b + 1])
        dos.append(o.kpm_transform(o.dos_moments(n_moments), energies)[0])
        v_rows, m_rows = [], []
        for k in range(n_t):
            if vac:
                v_rows.append(o.kpm_transform(o.vac(n_moments), energies)[0])
            if msd or k < n_t - 1:
                o.evolve(float(dts[k]), order_rule(oracle_mod, model.energy_scale, float(dts[k])))
            if msd:
                m_rows.append(o.kpm_transform(o.msd(n_moments), energies)[0])
        rv.append(v_rows)
        rm.append(m_rows)
        o.close()
    return np.array(dos), np.array(rv), np.array(rm)
