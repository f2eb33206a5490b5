"""gpuqt_kpm_transform_static against gpuqt_kpm_transform_damped.

The static entry point exists for callers that cannot allocate device memory while they run: processes whose
whole card already belongs to a memory pool or a framework's caching allocator (a cudaMalloc inside the library
would fail or trip the pool's out-of-memory handling), latency-critical loops that cannot take cudaMalloc's
device-wide stall, and jobs held to a memory budget fixed before they start.  It keeps its only working memory --
the table of damping factors and a status word -- in a static device array inside libgpuqt.so, and every call
shares that array, which still holds what the previous call wrote.  So the check is made on calls IN A ROW: the
second transform uses fewer moments than the first (stale table entries lie behind its range), a refused call
with an out-of-range energy sits between two good ones (the status word it raised must not leak into the next
call), and the very first call of the process is the one that looks the array's address up.

The file name sorts last on purpose: pytest -x stops at the first failure, and a failure here should not hide the
parity tests.  It passes alone in a fresh process (first call = set-up call) and after the rest of the suite.
"""
import numpy as np
import pytest

from workloads import lattices as L

pytestmark = pytest.mark.gpu

TOL = 1e-10     # transform: max |d| / max |out|, the tolerance of tests/test_gpu_parity.py::test_transform


@pytest.fixture(scope="module")
def gq():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    import paper_1705_01387_b200 as g
    return g


def synthetic_moments(n_sets, n_moments, seed):
    """Seeded stand-in for KPM moments: bounded, slowly decaying, oscillating (no arithmetic of the method)."""
    rng = np.random.default_rng(seed)
    n = np.arange(n_moments)
    return rng.uniform(-1.0, 1.0, (n_sets, n_moments)) / (1.0 + 0.01 * n) + np.cos(0.3 * n)[None, :]


def rel_err(got, ref):
    return np.max(np.abs(got - ref)) / np.max(np.abs(ref))


def test_static_transform_matches_allocating_path_on_calls_in_a_row(gq):
    import torch
    model = L.square(12, 10, W=2.0, seed=3)
    dE, vol = model.energy_scale, model.volume
    g = gq.GpuQT(model, batch=1, modes=0)                 # the existing path needs a handle; the new one does not
    E = np.linspace(-0.98 * dE, 0.98 * dE, 601)
    E_dev = torch.from_numpy(E).cuda()
    out_dev = torch.empty((4, E.size), dtype=torch.float64, device="cuda")      # caller-owned output, reused
    calls = [   # (n_moments, damping, lambda): long table first, then shorter ones over its leftovers
        (1000, gq.DAMPING_JACKSON, 0.0),
        (257, gq.DAMPING_JACKSON, 0.0),
        (640, gq.DAMPING_LORENTZ, 4.0),
        (33, gq.DAMPING_NONE, 0.0),
    ]
    for i, (nm, kind, lam) in enumerate(calls):
        C = synthetic_moments(4, nm, seed=100 + i)
        ref = g.kpm_transform(C, E, damping=kind, lam=lam)
        got = gq.kpm_transform_static(torch.from_numpy(C).cuda(), E_dev, dE, vol, damping=kind, lam=lam, out=out_dev)
        assert got.data_ptr() == out_dev.data_ptr()
        assert rel_err(got.cpu().numpy(), ref) <= TOL, (nm, kind, lam)
        if i == 1:
            # a refused call in between: one energy on the band edge -> GPUQT_ERR_ENERGY, raised on the device ...
            bad = E.copy()
            bad[5] = dE
            with pytest.raises(gq.GpuqtError) as ei:
                gq.kpm_transform_static(torch.from_numpy(C).cuda(), torch.from_numpy(bad).cuda(), dE, vol, out=out_dev)
            assert ei.value.status == -5 and "energy" in str(ei.value)
            flagged = out_dev.cpu().numpy()
            assert np.all(np.isnan(flagged[:, 5])) and not np.any(np.isnan(np.delete(flagged, 5, axis=1)))
            # ... and the same good call again right after it: the raised status must not survive
            again = gq.kpm_transform_static(torch.from_numpy(C).cuda(), E_dev, dE, vol, damping=kind, lam=lam, out=out_dev)
            assert rel_err(again.cpu().numpy(), ref) <= TOL
    g.close()


def test_static_transform_refuses_what_does_not_fit(gq):
    import torch
    E_dev = torch.zeros(3, dtype=torch.float64, device="cuda")
    nm = gq.binding.STATIC_MAX_MOMENTS
    # the largest table that fits is accepted ...
    C = torch.from_numpy(synthetic_moments(1, nm, seed=7)).cuda()
    out = gq.kpm_transform_static(C, E_dev, 4.0, 10.0)
    assert bool(torch.isfinite(out).all())
    # ... one more moment is not, with a message that names the limit
    C = torch.zeros((1, nm + 1), dtype=torch.float64, device="cuda")
    with pytest.raises(gq.GpuqtError) as ei:
        gq.kpm_transform_static(C, E_dev, 4.0, 10.0)
    assert ei.value.status == -8 and str(nm) in str(ei.value)
    for kw in (dict(damping=gq.DAMPING_LORENTZ, lam=0.0), dict(damping=9)):
        with pytest.raises(gq.GpuqtError) as ei:
            gq.kpm_transform_static(C[:, :8].contiguous(), E_dev, 4.0, 10.0, **kw)
        assert ei.value.status == -1
