"""Thin Python binding of the C-ABI in include/gpuqt.h (argument marshalling only).

The functions below carry the same names as the C entry points; `GpuQT` is a small convenience
object around one handle.  PyTorch is used for device memory (the workspace), pinned host buffers
and the CUDA stream; every step of the path runs in libgpuqt.so's kernels.  There is no fallback:
if the library is missing or no CUDA device is present the calls raise.
"""
import ctypes as C
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.environ.get("GPUQT_LIB") or os.path.join(_HERE, "libgpuqt.so")

MODE_VAC, MODE_MSD, MODE_PSI = 1, 2, 4
STATE_PSI, STATE_CHI, STATE_VAC_A, STATE_VAC_B = 0, 1, 2, 3
KERNEL_KPM_DOUBLING, KERNEL_KPM_LEFT, KERNEL_EVOLVE, KERNEL_EVOLVE_MSD, KERNEL_VELOCITY = range(5)
MAX_MOMENTS = 16384
STATIC_MAX_MOMENTS = 16384     # GPUQT_STATIC_MAX_MOMENTS: the static table of gpuqt_kpm_transform_static
MAX_ORDER = 4096
DAMPING_JACKSON, DAMPING_LORENTZ, DAMPING_NONE = 0, 1, 2
(INFO_STORED_MATRIX_BYTES, INFO_HOP_VARIANT, INFO_UNIFORM, INFO_UNROLLED_WIDTH, INFO_SMALL_PATH, INFO_PERSISTENT,
 INFO_WORKSPACE_USED, INFO_SMALL_PATH_MSD, INFO_STENCIL_PATTERNS, INFO_REORDERED) = range(10)


class SlabDesc(C.Structure):
    """gpuqt_slab_desc (include/gpuqt.h)."""
    _fields_ = [("global_id", C.c_int32), ("n_own", C.c_int64), ("n_halo", C.c_int64),
                ("nbr_count", C.POINTER(C.c_int32)), ("nbr_index", C.POINTER(C.c_int32)),
                ("hop_re", C.POINTER(C.c_double)), ("hop_im", C.POINTER(C.c_double)), ("onsite", C.POINTER(C.c_double)),
                ("x", C.POINTER(C.c_double)), ("n_sends", C.c_int32), ("send_peer", C.POINTER(C.c_int32)),
                ("send_count", C.POINTER(C.c_int64)), ("send_dst_row", C.POINTER(C.c_int64)),
                ("send_rows", C.POINTER(C.c_int32)), ("workspace", C.c_void_p), ("workspace_bytes", C.c_size_t)]


class Options(C.Structure):
    """gpuqt_options (include/gpuqt.h)."""
    _fields_ = [(n, C.c_int32) for n in ("struct_bytes", "stages", "blocks_per_sm", "run", "alternate", "hop_const",
                                          "idx16", "small", "persistent", "stencil", "reorder")]


# overrides applied to every GpuQT() that does not pass its own `options` (the GPU tests run every
# small case on both the streaming and the one-CTA kernels this way); empty = the library defaults
DEFAULT_OPTIONS = {}

STATUS = {0: "GPUQT_OK", -1: "GPUQT_ERR_ARG", -2: "GPUQT_ERR_INDEX", -3: "GPUQT_ERR_NOT_HERMITIAN",
          -4: "GPUQT_ERR_SCALE", -5: "GPUQT_ERR_ENERGY", -6: "GPUQT_ERR_STATE", -7: "GPUQT_ERR_CUDA",
          -8: "GPUQT_ERR_NOMEM", -9: "GPUQT_ERR_POSITION"}

_dp = C.POINTER(C.c_double)
_ip = C.POINTER(C.c_int32)
_model_args = [C.c_int64, C.c_int32, _ip, _ip, _dp, _dp, _dp, _dp, C.c_double]

_SIGNATURES = {
    "gpuqt_workspace_bytes": (C.c_size_t, [C.c_int64, C.c_int32, C.c_int, C.c_int32, C.c_int]),
    "gpuqt_validate": (C.c_int, _model_args + [C.c_double]),
    "gpuqt_default_options": (None, [C.POINTER(Options)]),
    "gpuqt_plan_storage": (C.c_int, [C.c_int64, C.c_int32, _ip, _ip, _dp, _dp, C.c_int32, C.c_int64, C.POINTER(Options),
                                     C.POINTER(C.c_int32), C.POINTER(C.c_int64), C.POINTER(C.c_int64)]),
    "gpuqt_create": (C.c_int, [C.POINTER(C.c_void_p)] + _model_args + [C.c_double, C.c_double, C.c_int32, C.c_int,
                                                                       C.c_void_p, C.c_size_t, C.c_void_p]),
    "gpuqt_create_with_options": (C.c_int, [C.POINTER(C.c_void_p)] + _model_args + [
        C.c_double, C.c_double, C.c_int32, C.c_int, C.c_void_p, C.c_size_t, C.c_void_p, C.POINTER(Options)]),
    "gpuqt_set_state": (C.c_int, [C.c_void_p, C.c_void_p]),
    "gpuqt_set_state_device": (C.c_int, [C.c_void_p, C.c_void_p]),
    "gpuqt_prefetch_state": (C.c_int, [C.c_void_p, C.c_void_p]),
    "gpuqt_set_state_prefetched": (C.c_int, [C.c_void_p]),
    "gpuqt_dos_moments": (C.c_int, [C.c_void_p, C.c_int32, C.c_void_p]),
    "gpuqt_evolve": (C.c_int, [C.c_void_p, C.c_double, C.c_int32]),
    "gpuqt_vac": (C.c_int, [C.c_void_p, C.c_int32, C.c_void_p]),
    "gpuqt_msd": (C.c_int, [C.c_void_p, C.c_int32, C.c_void_p]),
    "gpuqt_kpm_transform": (C.c_int, [C.c_void_p, _dp, C.c_int32, C.c_int32, _dp, C.c_int32, _dp]),
    "gpuqt_kpm_transform_damped": (C.c_int, [C.c_void_p, C.c_int, C.c_double, _dp, C.c_int32, C.c_int32, _dp, C.c_int32, _dp]),
    "gpuqt_kpm_transform_static": (C.c_int, [C.c_int, C.c_double, C.c_void_p, C.c_int32, C.c_int32, C.c_void_p, C.c_int32,
                                             C.c_double, C.c_double, C.c_void_p, C.c_void_p, C.c_char_p, C.c_size_t]),
    "gpuqt_get_info": (C.c_int, [C.c_void_p, C.c_int, C.POINTER(C.c_int64)]),
    "gpuqt_running_conductivity": (C.c_int, [C.c_void_p, C.c_int, _dp, _dp, _dp, C.c_int32, C.c_int32, _dp, _dp]),
    "gpuqt_localization_length": (C.c_int, [C.c_void_p, _dp, C.c_int32, C.c_int32, _dp, _dp]),
    "gpuqt_get_state": (C.c_int, [C.c_void_p, C.c_int, C.c_void_p]),
    "gpuqt_get_table": (C.c_int, [C.c_void_p, _ip, _dp, _dp, _dp]),
    "gpuqt_bessel_coeffs": (C.c_int, [C.c_double, C.c_double, C.c_int32, _dp, _dp]),
    "gpuqt_kernel_stats": (C.c_int, [C.c_void_p, C.c_int, _dp, C.POINTER(C.c_int64)]),
    "gpuqt_kernel_steps": (C.c_int, [C.c_void_p, C.c_int, C.POINTER(C.c_int64)]),
    "gpuqt_reset_stats": (C.c_int, [C.c_void_p]),
    "gpuqt_last_error": (C.c_char_p, [C.c_void_p]),
    "gpuqt_destroy": (None, [C.c_void_p]),
    # row-slab decomposition
    "gpuqt_slab_workspace_bytes": (C.c_size_t, [C.c_int64, C.c_int64, C.c_int32, C.c_int, C.c_int32, C.c_int]),
    "gpuqt_slab_create": (C.c_int, [C.POINTER(C.c_void_p), C.c_int32, C.POINTER(SlabDesc), C.c_int32, C.c_double, C.c_double,
                                    C.c_double, C.c_int32, C.c_int, C.c_void_p]),
    "gpuqt_slab_buffer_count": (C.c_int32, [C.c_void_p]),
    "gpuqt_slab_create_with_options": (C.c_int, [C.POINTER(C.c_void_p), C.c_int32, C.POINTER(SlabDesc), C.c_int32, C.c_double,
                                                 C.c_double, C.c_double, C.c_int32, C.c_int, C.c_void_p, C.POINTER(Options)]),
    "gpuqt_slab_export": (C.c_int, [C.c_void_p, C.c_int32, C.POINTER(C.c_void_p), C.POINTER(C.c_void_p), C.POINTER(C.c_int64),
                                    C.POINTER(C.c_int64)]),
    "gpuqt_slab_connect": (C.c_int, [C.c_void_p, C.c_int32, C.POINTER(C.c_void_p), C.c_void_p, C.c_int64, C.c_int64]),
    "gpuqt_slab_set_wait_budget": (C.c_int, [C.c_void_p, C.c_double]),
    "gpuqt_slab_set_state": (C.c_int, [C.c_void_p, C.POINTER(C.c_void_p)]),
    "gpuqt_slab_dos_moments": (C.c_int, [C.c_void_p, C.c_int32, C.c_void_p]),
    "gpuqt_slab_evolve": (C.c_int, [C.c_void_p, C.c_double, C.c_int32]),
    "gpuqt_slab_vac": (C.c_int, [C.c_void_p, C.c_int32, C.c_void_p]),
    "gpuqt_slab_msd": (C.c_int, [C.c_void_p, C.c_int32, C.c_void_p]),
    "gpuqt_slab_get_state": (C.c_int, [C.c_void_p, C.c_int32, C.c_int, C.c_void_p]),
    "gpuqt_slab_get_info": (C.c_int, [C.c_void_p, C.c_int32, C.c_int, C.POINTER(C.c_int64)]),
    "gpuqt_slab_last_error": (C.c_char_p, [C.c_void_p]),
    "gpuqt_slab_destroy": (None, [C.c_void_p]),
}

_lib = None


def load():
    """Load libgpuqt.so (fails loudly if it has not been built)."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise RuntimeError(f"{LIB_PATH} is missing: run `python -m paper_1705_01387_b200.build` "
                               "(there is no CPU fallback)")
        lib = C.CDLL(LIB_PATH)
        for name, (res, args) in _SIGNATURES.items():
            fn = getattr(lib, name)
            fn.restype = res
            fn.argtypes = args
        _lib = lib
    return _lib


def __getattr__(name):          # gpuqt_* entry points under their C names
    if name in _SIGNATURES:
        return getattr(load(), name)
    raise AttributeError(name)


class GpuqtError(RuntimeError):
    def __init__(self, status, what, detail=""):
        self.status = status
        super().__init__(f"{what}: {STATUS.get(status, status)} {detail}".strip())


def _d(a):
    return None if a is None else a.ctypes.data_as(_dp)


def _i(a):
    return None if a is None else a.ctypes.data_as(_ip)


def _model_tuple(model):
    return (C.c_int64(model.N), C.c_int32(model.K), _i(model.nbr_count), _i(model.nbr_index),
            _d(model.hop_re), _d(model.hop_im), _d(model.onsite), _d(model.x), C.c_double(model.box_length))


def validate(model) -> int:
    """gpuqt_validate on a TBModel-like object; returns the status code (host only, no GPU)."""
    return load().gpuqt_validate(*_model_tuple(model), C.c_double(model.energy_scale))


def bessel_coeffs(dE, dt, order):
    cr, ci = np.empty(order), np.empty(order)
    rc = load().gpuqt_bessel_coeffs(dE, dt, order, _d(cr), _d(ci))
    if rc:
        raise GpuqtError(rc, "gpuqt_bessel_coeffs")
    return cr + 1j * ci


def choose_order(dE, dt, tol=1e-15):
    """Smallest N_p with |J_m(dE |dt|)| < tol for every m >= N_p (tail rule [A5]), from the
    library's own coefficient table."""
    x = dE * abs(dt)
    n = int(x) + 80 + int(4 * np.sqrt(x + 1))
    J = np.abs(bessel_coeffs(dE, dt, n)) / np.where(np.arange(n) == 0, 1.0, 2.0)
    big = np.nonzero(J >= tol)[0]
    return int(big[-1]) + 1 if big.size else 1


def default_options(**overrides) -> Options:
    """gpuqt_default_options, then the given fields overridden."""
    o = Options()
    load().gpuqt_default_options(C.byref(o))
    for k, v in overrides.items():
        if not hasattr(o, k):
            raise KeyError(f"unknown gpuqt option {k!r}")
        setattr(o, k, int(v))
    return o


def plan_storage(model, batch=1, options=None, l2_bytes=0):
    """gpuqt_plan_storage (host only): (hop_variant, stored_matrix_bytes, stencil_patterns) gpuqt_create would choose."""
    o = default_options(**(DEFAULT_OPTIONS if options is None else options))
    hop, nbytes, pats = C.c_int32(), C.c_int64(), C.c_int64()
    rc = load().gpuqt_plan_storage(model.N, model.K, _i(model.nbr_count), _i(model.nbr_index), _d(model.hop_re),
                                   _d(model.hop_im), batch, l2_bytes, C.byref(o), C.byref(hop), C.byref(nbytes), C.byref(pats))
    if rc != 0:
        raise GpuqtError(rc, "gpuqt_plan_storage")
    return hop.value, nbytes.value, pats.value


def kpm_transform_static(moments, energies, energy_scale, volume, damping=DAMPING_JACKSON, lam=0.0, out=None, stream=None):
    """gpuqt_kpm_transform_static: the damping + energy transform without a handle and without any device allocation
    inside the library -- for callers whose device memory is already spoken for (a pool or caching allocator owns the
    card, a fixed memory budget) or that cannot afford cudaMalloc's device-wide stall.  `moments` [n_sets][n_moments]
    and `energies` [n_energies] are CUDA float64 tensors the caller already holds; the result goes to `out`
    ([n_sets][n_energies], CUDA float64) -- pass one you own to keep this wrapper allocation-free as well, otherwise
    torch allocates it here, on the caller's side of the boundary.  At most STATIC_MAX_MOMENTS moments; one call at a
    time per device (every call shares one static scratch table inside the library)."""
    import torch
    assert moments.is_cuda and energies.is_cuda and moments.dtype == energies.dtype == torch.float64
    assert moments.is_contiguous() and energies.is_contiguous() and moments.dim() == 2 and energies.dim() == 1
    n_sets, n_moments = moments.shape
    if out is None:
        out = torch.empty((n_sets, energies.numel()), dtype=torch.float64, device=moments.device)
    assert out.is_cuda and out.is_contiguous() and out.dtype == torch.float64 and tuple(out.shape) == (n_sets, energies.numel())
    stream = stream if stream is not None else torch.cuda.current_stream()
    text = C.create_string_buffer(256)
    rc = load().gpuqt_kpm_transform_static(C.c_int(damping), C.c_double(lam), C.c_void_p(moments.data_ptr()),
                                           C.c_int32(n_moments), C.c_int32(n_sets), C.c_void_p(energies.data_ptr()),
                                           C.c_int32(energies.numel()), C.c_double(energy_scale), C.c_double(volume),
                                           C.c_void_p(out.data_ptr()), C.c_void_p(stream.cuda_stream), text, C.c_size_t(256))
    if rc:
        raise GpuqtError(rc, "gpuqt_kpm_transform_static", text.value.decode())
    return out


class GpuQT:
    """One gpuqt_handle on the current CUDA device; workspace and stream come from torch."""

    def __init__(self, model, batch=1, modes=MODE_VAC | MODE_MSD, stream=None, options=None):
        import torch
        if not torch.cuda.is_available():
            raise RuntimeError("gpuqt needs a CUDA device (no CPU fallback)")
        lib = load()
        self._torch = torch
        self.N, self.K, self.batch, self.modes = model.N, model.K, batch, modes
        nbytes = lib.gpuqt_workspace_bytes(model.N, model.K, int(model.hop_im is not None), batch, modes)
        if nbytes == 0:
            raise GpuqtError(-1, "gpuqt_workspace_bytes")
        self.workspace = torch.empty(nbytes, dtype=torch.uint8, device="cuda")
        self.stream = stream if stream is not None else torch.cuda.current_stream()
        self._h = C.c_void_p()
        self.options = default_options(**(DEFAULT_OPTIONS if options is None else options))
        rc = lib.gpuqt_create_with_options(C.byref(self._h), *_model_tuple(model), C.c_double(model.volume),
                                           C.c_double(model.energy_scale), C.c_int32(batch), C.c_int(modes),
                                           C.c_void_p(self.workspace.data_ptr()), C.c_size_t(nbytes),
                                           C.c_void_p(self.stream.cuda_stream), C.byref(self.options))
        if rc:
            self._h = C.c_void_p()
            raise GpuqtError(rc, "gpuqt_create", (lib.gpuqt_last_error(None) or b"").decode())

    def _ck(self, rc, what):
        if rc:
            raise GpuqtError(rc, what, (load().gpuqt_last_error(self._h) or b"").decode())

    def close(self):
        if getattr(self, "_h", None):
            load().gpuqt_destroy(self._h)
            self._h = C.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    # ---- state
    def set_state(self, phi):
        """phi: host [batch][N][2] float64 — numpy array or (pinned) CPU torch tensor."""
        if isinstance(phi, np.ndarray):
            phi = np.ascontiguousarray(phi, np.float64)
            assert phi.shape == (self.batch, self.N, 2)
            self._ck(load().gpuqt_set_state(self._h, C.c_void_p(phi.ctypes.data)), "gpuqt_set_state")
        else:
            assert phi.device.type == "cpu" and phi.is_contiguous() and phi.dtype == self._torch.float64
            assert tuple(phi.shape) == (self.batch, self.N, 2)
            self._ck(load().gpuqt_set_state(self._h, C.c_void_p(phi.data_ptr())), "gpuqt_set_state")

    def prefetch_state(self, phi):
        """Start the asynchronous upload of the next batch (pinned CPU torch tensor [batch][N][2]); keep it alive."""
        assert phi.device.type == "cpu" and phi.is_pinned() and phi.is_contiguous() and phi.dtype == self._torch.float64
        assert tuple(phi.shape) == (self.batch, self.N, 2)
        self._prefetch_keep = phi
        self._ck(load().gpuqt_prefetch_state(self._h, C.c_void_p(phi.data_ptr())), "gpuqt_prefetch_state")

    def set_state_prefetched(self):
        self._ck(load().gpuqt_set_state_prefetched(self._h), "gpuqt_set_state_prefetched")

    def set_state_device(self, phi):
        assert phi.is_cuda and phi.is_contiguous() and phi.dtype == self._torch.float64
        assert tuple(phi.shape) == (self.batch, self.N, 2)
        self._ck(load().gpuqt_set_state_device(self._h, C.c_void_p(phi.data_ptr())), "gpuqt_set_state_device")

    def get_state(self, which):
        out = np.empty((self.batch, self.N, 2), np.float64)
        self._ck(load().gpuqt_get_state(self._h, which, C.c_void_p(out.ctypes.data)), "gpuqt_get_state")
        return out

    def get_table(self):
        nk = self.N * self.K
        col = np.empty(nk, np.int32)
        re, im, dx = (np.empty(nk, np.float64) for _ in range(3))
        self._ck(load().gpuqt_get_table(self._h, _i(col), _d(re), _d(im), _d(dx)), "gpuqt_get_table")
        return col, re, im, dx

    # ---- the path
    def _moments(self, fn, what, n, out=None):
        if out is None:
            out = np.empty((self.batch, n), np.float64)
            ptr = out.ctypes.data
        else:                                   # pinned torch tensor
            ptr = out.data_ptr()
        self._ck(fn(self._h, C.c_int32(n), C.c_void_p(ptr)), what)
        return out

    def dos_moments(self, n, out=None):
        return self._moments(load().gpuqt_dos_moments, "gpuqt_dos_moments", n, out)

    def msd(self, n, out=None):
        return self._moments(load().gpuqt_msd, "gpuqt_msd", n, out)

    def vac(self, n, out=None):
        return self._moments(load().gpuqt_vac, "gpuqt_vac", n, out)

    def evolve(self, dt, order):
        self._ck(load().gpuqt_evolve(self._h, C.c_double(dt), C.c_int32(order)), "gpuqt_evolve")

    def kpm_transform(self, moments, energies, damping=None, lam=0.0):
        """gpuqt_kpm_transform (Jackson, Eq. 31), or gpuqt_kpm_transform_damped with damping = DAMPING_*."""
        moments = np.ascontiguousarray(moments, np.float64)
        energies = np.ascontiguousarray(energies, np.float64)
        m2 = moments.reshape(-1, moments.shape[-1])
        out = np.empty((m2.shape[0], energies.size), np.float64)
        if damping is None:
            self._ck(load().gpuqt_kpm_transform(self._h, _d(m2), C.c_int32(m2.shape[1]), C.c_int32(m2.shape[0]),
                                                _d(energies), C.c_int32(energies.size), _d(out)), "gpuqt_kpm_transform")
        else:
            self._ck(load().gpuqt_kpm_transform_damped(self._h, C.c_int(damping), C.c_double(lam), _d(m2),
                                                       C.c_int32(m2.shape[1]), C.c_int32(m2.shape[0]), _d(energies),
                                                       C.c_int32(energies.size), _d(out)), "gpuqt_kpm_transform_damped")
        return out

    def info(self, what):
        v = C.c_int64()
        self._ck(load().gpuqt_get_info(self._h, what, C.byref(v)), "gpuqt_get_info")
        return v.value

    def running_conductivity(self, kind, corr, dos, dt):
        """kind 'vac' or 'msd'; corr [n_t][n_E] from kpm_transform; returns (sigma, length or None)."""
        corr = np.ascontiguousarray(corr, np.float64)
        dt = np.ascontiguousarray(dt, np.float64)
        dos = None if dos is None else np.ascontiguousarray(dos, np.float64)
        n_t, n_e = corr.shape
        sigma = np.empty_like(corr)
        length = np.empty_like(corr) if (kind == "msd" and dos is not None) else None
        self._ck(load().gpuqt_running_conductivity(self._h, 0 if kind == "vac" else 1, _d(corr), _d(dos), _d(dt),
                                                   C.c_int32(n_t), C.c_int32(n_e), _d(sigma), _d(length)),
                 "gpuqt_running_conductivity")
        return sigma, length

    def localization_length(self, length):
        """gpuqt_localization_length: length [n_t][n_E] (Eq. 11) -> (xi [n_E] of Eq. 12 at the last time, growth [n_E])."""
        length = np.ascontiguousarray(length, np.float64)
        n_t, n_e = length.shape
        xi, growth = np.empty(n_e), np.empty(n_e)
        self._ck(load().gpuqt_localization_length(self._h, _d(length), C.c_int32(n_t), C.c_int32(n_e), _d(xi), _d(growth)),
                 "gpuqt_localization_length")
        return xi, growth

    # ---- timing
    def kernel_stats(self, cls):
        ms, n = C.c_double(), C.c_int64()
        self._ck(load().gpuqt_kernel_stats(self._h, cls, C.byref(ms), C.byref(n)), "gpuqt_kernel_stats")
        return ms.value, n.value

    def kernel_steps(self, cls):
        n = C.c_int64()
        self._ck(load().gpuqt_kernel_steps(self._h, cls, C.byref(n)), "gpuqt_kernel_steps")
        return n.value

    def reset_stats(self):
        self._ck(load().gpuqt_reset_stats(self._h), "gpuqt_reset_stats")
