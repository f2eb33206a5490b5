"""ctypes binding of the CPU oracle (oracle/gpuqt_oracle.c).  TEST INFRASTRUCTURE ONLY.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
import this module.  It never imports the CUDA package.
"""
import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "gpuqt_oracle.c")
# GPUQT_ORACLE_SANITIZE=1: a second build with -fsanitize=address,undefined (run the pins under it with
# LD_PRELOAD=$(gcc -print-file-name=libasan.so); summary in profiles/)
_SAN = os.environ.get("GPUQT_ORACLE_SANITIZE", "0") == "1"
_LIB = os.path.join(_HERE, "libgpuqt_oracle_san.so" if _SAN else "libgpuqt_oracle.so")

MODE_VAC, MODE_MSD = 1, 2
PSI, CHI, VAC_A, VAC_B = 0, 1, 2, 3


def build(force: bool = False) -> str:
    """Compile the oracle with gcc (plain C99 + OpenMP over rows)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        opt = ["-O1", "-g", "-fsanitize=address,undefined", "-fno-omit-frame-pointer"] if _SAN else ["-O2"]
        subprocess.check_call(["gcc"] + opt + ["-std=c99", "-D_DEFAULT_SOURCE", "-fPIC", "-shared",
                                               "-fopenmp", "-o", _LIB, _SRC, "-lm"])
    return _LIB


_lib = None


def lib():
    global _lib
    if _lib is None:
        _lib = C.CDLL(build())
    return _lib


def _p(a, t):
    return None if a is None else a.ctypes.data_as(C.POINTER(t))


def _d(a):
    return _p(a, C.c_double)


def _check(rc, what):
    if rc != 0:
        raise RuntimeError(f"oracle {what} failed with status {rc}")


class Oracle:
    """Thin wrapper: one oracle_model, states as numpy float64 [batch][N][2]."""

    def __init__(self, model, batch=1, modes=MODE_VAC | MODE_MSD):
        L = lib()
        self.N, self.K, self.batch, self.modes = model.N, model.K, batch, modes
        self.dE = model.energy_scale
        self._h = C.c_void_p()
        rc = L.oracle_create(C.byref(self._h), C.c_int64(model.N), C.c_int32(model.K),
                             _p(model.nbr_count, C.c_int32), _p(model.nbr_index, C.c_int32),
                             _d(model.hop_re), _d(model.hop_im), _d(model.onsite), _d(model.x),
                             C.c_double(model.box_length), C.c_double(model.volume),
                             C.c_double(model.energy_scale), C.c_int32(batch))
        _check(rc, "create")

    def close(self):
        if self._h:
            lib().oracle_destroy(self._h)
            self._h = C.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    # ---- table
    def get_table(self):
        nk = self.N * self.K
        col = np.empty(nk, np.int32)
        re, im, dx = (np.empty(nk, np.float64) for _ in range(3))
        _check(lib().oracle_get_table(self._h, _p(col, C.c_int32), _d(re), _d(im), _d(dx)), "get_table")
        return col, re, im, dx

    # ---- single-vector operators ([N][2] in, [N][2] out)
    def _op(self, fn, v):
        v = np.ascontiguousarray(v, np.float64)
        out = np.empty_like(v)
        _check(fn(self._h, _d(v), _d(out)), "apply")
        return out

    def apply_h(self, v):
        return self._op(lib().oracle_apply_h, v)

    def apply_v(self, v):
        return self._op(lib().oracle_apply_v, v)

    def apply_xh(self, v):
        return self._op(lib().oracle_apply_xh, v)

    def evolve_vec(self, v, dt, order):
        v = np.ascontiguousarray(v, np.float64)
        out = np.empty_like(v)
        _check(lib().oracle_evolve_vec(self._h, _d(v), _d(out), C.c_double(dt), C.c_int32(order)), "evolve_vec")
        return out

    def commutator_vec(self, v, dt, order):
        v = np.ascontiguousarray(v, np.float64)
        out = np.empty_like(v)
        _check(lib().oracle_commutator_vec(self._h, _d(v), _d(out), C.c_double(dt), C.c_int32(order)), "commutator_vec")
        return out

    def moments_vec(self, l, r, n):
        l = np.ascontiguousarray(l, np.float64)
        r = np.ascontiguousarray(r, np.float64)
        cre, cim = np.empty(n), np.empty(n)
        _check(lib().oracle_moments_vec(self._h, _d(l), _d(r), C.c_int32(n), _d(cre), _d(cim)), "moments_vec")
        return cre + 1j * cim

    # ---- the path
    def set_state(self, phi):
        phi = np.ascontiguousarray(phi, np.float64)
        assert phi.shape == (self.batch, self.N, 2)
        _check(lib().oracle_set_state(self._h, _d(phi)), "set_state")

    def evolve(self, dt, order):
        _check(lib().oracle_evolve(self._h, C.c_double(dt), C.c_int32(order), C.c_int(self.modes)), "evolve")

    def get_state(self, which):
        out = np.empty((self.batch, self.N, 2), np.float64)
        _check(lib().oracle_get_state(self._h, C.c_int(which), _d(out)), "get_state")
        return out

    def _moments(self, fn, n):
        out = np.empty((self.batch, n), np.float64)
        _check(fn(self._h, C.c_int32(n), _d(out)), "moments")
        return out

    def dos_moments(self, n):
        return self._moments(lib().oracle_dos_moments, n)

    def msd(self, n):
        return self._moments(lib().oracle_msd, n)

    def vac(self, n):
        return self._moments(lib().oracle_vac, n)

    def kpm_transform(self, moments, energies, damping=0, lam=0.0):
        """damping: 0 Jackson (Eq. 31), 1 Lorentz(lam), 2 none."""
        moments = np.ascontiguousarray(moments, np.float64)
        energies = np.ascontiguousarray(energies, np.float64)
        n_sets, n_m = moments.reshape(-1, moments.shape[-1]).shape
        out = np.empty((n_sets, energies.size), np.float64)
        _check(lib().oracle_kpm_transform_damped(self._h, C.c_int(damping), C.c_double(lam), _d(moments), C.c_int32(n_m),
                                                 C.c_int32(n_sets), _d(energies), C.c_int32(energies.size), _d(out)),
               "kpm_transform")
        return out


def bessel_coeffs(dE, dt, order):
    cr, ci = np.empty(order), np.empty(order)
    _check(lib().oracle_bessel_coeffs(C.c_double(dE), C.c_double(dt), C.c_int32(order), _d(cr), _d(ci)), "bessel")
    return cr + 1j * ci


def jackson(n):
    g = np.empty(n)
    _check(lib().oracle_jackson(C.c_int32(n), _d(g)), "jackson")
    return g


def damping(kind, lam, n):
    g = np.empty(n)
    _check(lib().oracle_damping(C.c_int(kind), C.c_double(lam), C.c_int32(n), _d(g)), "damping")
    return g


def running_conductivity(kind, corr, dos, dt):
    """oracle_running_conductivity: kind 'vac' or 'msd'; corr [n_t][n_E]; returns (sigma, length or None)."""
    corr = np.ascontiguousarray(corr, np.float64)
    dt = np.ascontiguousarray(dt, np.float64)
    n_t, n_e = corr.shape
    assert dt.size >= (n_t - 1 if kind == "vac" else n_t)
    sigma = np.empty_like(corr)
    length = np.empty_like(corr) if kind == "msd" else None
    dos_a = None if dos is None else np.ascontiguousarray(dos, np.float64)
    _check(lib().oracle_running_conductivity(C.c_int(0 if kind == "vac" else 1), _d(corr), _d(dos_a), _d(dt),
                                             C.c_int32(n_t), C.c_int32(n_e), _d(sigma), _d(length)), "running_conductivity")
    return sigma, length


def localization_length(length):
    """oracle_localization_length: length [n_t][n_E] (Eq. 11) -> (xi [n_E] of Eq. 12 at the last time, growth [n_E])."""
    length = np.ascontiguousarray(length, np.float64)
    n_t, n_e = length.shape
    xi, growth = np.empty(n_e), np.empty(n_e)
    _check(lib().oracle_localization_length(_d(length), C.c_int32(n_t), C.c_int32(n_e), _d(xi), _d(growth)),
           "localization_length")
    return xi, growth
