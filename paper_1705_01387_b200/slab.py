"""Row-slab decomposition with halo exchange (include/gpuqt.h "row-slab decomposition").

The paper's program is single-GPU and limited by one card's memory.  Here one
lattice is cut into slabs of consecutive rows; a slab owns its rows of H and of every vector and keeps the
rows of other slabs that its own rows reference as halo rows behind them.  This module is host plumbing
only (index bookkeeping, marshalling, the final sum of the partial moments); every arithmetic step runs in
libgpuqt.so (gpuqt_slab_*).

  partition(model, n_slabs)         -> list of Slab (pure numpy; tested without a GPU)
  SlabGroup(model, slabs, mine)     -> the slabs of `mine` resident on the current GPU
  SlabGroup.dos_moments / evolve / vac / msd / get_state

One process may hold all slabs (a multi-GPU decomposition emulated on one device: this is what the GPU parity
tests do), or one slab per rank with the slabs of other ranks connected through CUDA IPC (`connect_ranks`).
"""
import ctypes as C
from dataclasses import dataclass, field

import numpy as np

from . import binding


@dataclass
class Slab:
    """Rows [row0, row1) of the global lattice in local numbering: owned rows first, then the halo rows."""
    global_id: int
    row0: int
    row1: int
    halo_global: np.ndarray            # int64 [n_halo] global row of every halo row, ascending
    nbr_count: np.ndarray              # int32 [n_own]
    nbr_index: np.ndarray              # int32 [n_own * K] local indices (unused slots -1)
    hop_re: object
    hop_im: object
    onsite: object
    x: np.ndarray                      # float64 [n_own + n_halo]
    sends: list = field(default_factory=list)   # (peer global id, local owned rows int32[], first halo row in the peer)

    @property
    def n_own(self):
        return self.row1 - self.row0

    @property
    def n_halo(self):
        return int(self.halo_global.size)


def row_ranges(N, n_slabs):
    """Balanced consecutive row ranges, cut at multiples of 32 rows (a slab starts on a slice boundary)."""
    if n_slabs < 1 or n_slabs > 64:
        raise ValueError("1 .. 64 slabs")
    cuts = [0]
    for r in range(1, n_slabs):
        c = int(round(N * r / n_slabs / 32.0)) * 32
        cuts.append(min(max(c, cuts[-1]), N))
    cuts.append(N)
    if any(b <= a for a, b in zip(cuts, cuts[1:])):
        raise ValueError(f"{N} rows are too few for {n_slabs} slabs")
    return list(zip(cuts[:-1], cuts[1:]))


def partition(model, n_slabs):
    """Cut a TBModel-like object into `n_slabs` row slabs with their halo lists and send segments."""
    K = model.K
    ranges = row_ranges(model.N, n_slabs)
    idx = model.nbr_index.reshape(model.N, K)
    slabs = []
    for gid, (r0, r1) in enumerate(ranges):
        cnt = model.nbr_count[r0:r1]
        loc = idx[r0:r1].astype(np.int64)
        used = np.arange(K)[None, :] < cnt[:, None]
        remote = used & ((loc < r0) | (loc >= r1))
        halo = np.unique(loc[remote])                                   # ascending: grouped by owner automatically
        new = np.full(loc.shape, -1, np.int64)
        own = used & ~remote
        new[own] = loc[own] - r0
        new[remote] = (r1 - r0) + np.searchsorted(halo, loc[remote])
        sl = slice(r0 * K, r1 * K)
        slabs.append(Slab(global_id=gid, row0=r0, row1=r1, halo_global=halo,
                          nbr_count=np.ascontiguousarray(cnt, np.int32),
                          nbr_index=np.ascontiguousarray(new.reshape(-1), np.int32),
                          hop_re=None if model.hop_re is None else np.ascontiguousarray(model.hop_re[sl]),
                          hop_im=None if model.hop_im is None else np.ascontiguousarray(model.hop_im[sl]),
                          onsite=None if model.onsite is None else np.ascontiguousarray(model.onsite[r0:r1]),
                          x=np.ascontiguousarray(np.concatenate([model.x[r0:r1], model.x[halo]]), np.float64)))
    # send segments: the part of q's halo list that p owns, in q's halo order
    for q in slabs:
        for p in slabs:
            if p is q:
                continue
            lo, hi = np.searchsorted(q.halo_global, [p.row0, p.row1])
            if hi > lo:
                p.sends.append((q.global_id, np.ascontiguousarray(q.halo_global[lo:hi] - p.row0, np.int32), q.n_own + int(lo)))
    return slabs


class SlabGroup:
    """The slabs `mine` (global ids; default all) of a decomposition on the current CUDA device."""

    def __init__(self, model, slabs, mine=None, batch=1, modes=binding.MODE_VAC | binding.MODE_MSD, stream=None, options=None):
        import torch
        if not torch.cuda.is_available():
            raise RuntimeError("gpuqt needs a CUDA device (no CPU fallback)")
        lib = binding.load()
        self._torch = torch
        self.slabs = [s for s in slabs if mine is None or s.global_id in mine]
        self.batch, self.modes, self.K = batch, modes, model.K
        self.stream = stream if stream is not None else torch.cuda.current_stream()
        descs = (binding.SlabDesc * len(self.slabs))()
        self._keep = []
        self.workspaces = []
        cplx = int(model.hop_im is not None)
        for d, s in zip(descs, self.slabs):
            nbytes = lib.gpuqt_slab_workspace_bytes(s.n_own, s.n_halo, model.K, cplx, batch, modes)
            if nbytes == 0:
                raise binding.GpuqtError(-1, "gpuqt_slab_workspace_bytes")
            ws = torch.zeros(nbytes, dtype=torch.uint8, device="cuda")
            self.workspaces.append(ws)
            peers = np.array([p for p, _, _ in s.sends], np.int32)
            counts = np.array([r.size for _, r, _ in s.sends], np.int64)
            dst = np.array([d0 for _, _, d0 in s.sends], np.int64)
            rows = np.concatenate([r for _, r, _ in s.sends]).astype(np.int32) if s.sends else np.zeros(0, np.int32)
            self._keep += [peers, counts, dst, rows]
            d.global_id, d.n_own, d.n_halo = s.global_id, s.n_own, s.n_halo
            d.nbr_count, d.nbr_index = binding._i(s.nbr_count), binding._i(s.nbr_index)
            d.hop_re, d.hop_im, d.onsite, d.x = binding._d(s.hop_re), binding._d(s.hop_im), binding._d(s.onsite), binding._d(s.x)
            d.n_sends = len(s.sends)
            d.send_peer = peers.ctypes.data_as(C.POINTER(C.c_int32))
            d.send_count = counts.ctypes.data_as(C.POINTER(C.c_int64))
            d.send_dst_row = dst.ctypes.data_as(C.POINTER(C.c_int64))
            d.send_rows = rows.ctypes.data_as(C.POINTER(C.c_int32))
            d.workspace, d.workspace_bytes = ws.data_ptr(), nbytes
        self._g = C.c_void_p()
        self.options = binding.default_options(**(options or {}))
        rc = lib.gpuqt_slab_create_with_options(C.byref(self._g), len(self.slabs), descs, model.K, C.c_double(model.box_length),
                                                C.c_double(model.volume), C.c_double(model.energy_scale), batch, modes,
                                                C.c_void_p(self.stream.cuda_stream), C.byref(self.options))
        if rc:
            self._g = C.c_void_p()
            raise binding.GpuqtError(rc, "gpuqt_slab_create", (lib.gpuqt_last_error(None) or b"").decode())

    def _ck(self, rc, what):
        if rc:
            raise binding.GpuqtError(rc, what, (binding.load().gpuqt_slab_last_error(self._g) or b"").decode())

    def close(self):
        if getattr(self, "_g", None):
            binding.load().gpuqt_slab_destroy(self._g)
            self._g = C.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def info(self, i, what):
        """gpuqt_slab_get_info of local slab i (binding.INFO_*)."""
        v = C.c_int64()
        self._ck(binding.load().gpuqt_slab_get_info(self._g, i, what, C.byref(v)), "gpuqt_slab_get_info")
        return v.value

    def hop_variants(self):
        """The record variant (GPUQT_INFO_HOP_VARIANT) of every local slab."""
        return [self.info(i, binding.INFO_HOP_VARIANT) for i in range(len(self.slabs))]

    def set_wait_budget(self, seconds):
        """How long a halo exchange waits for a slab of another group before the call fails (gpuqt_slab_set_wait_budget)."""
        self._ck(binding.load().gpuqt_slab_set_wait_budget(self._g, C.c_double(seconds)), "gpuqt_slab_set_wait_budget")

    def export(self, i):
        """gpuqt_slab_export of local slab i: (buffer addresses, flag array address, n_own, n_halo)."""
        lib = binding.load()
        bufs, flags = (C.c_void_p * lib.gpuqt_slab_buffer_count(self._g))(), C.c_void_p()
        n_own, n_halo = C.c_int64(), C.c_int64()
        self._ck(lib.gpuqt_slab_export(self._g, i, bufs, C.byref(flags), C.byref(n_own), C.byref(n_halo)), "gpuqt_slab_export")
        return [int(b) for b in bufs], flags.value, n_own.value, n_halo.value

    def connect(self, peer_global_id, buffers, flags, n_own, n_halo):
        """gpuqt_slab_connect: addresses (valid in THIS process) and row counts of a slab held by another group."""
        ptrs = (C.c_void_p * len(buffers))(*buffers)
        self._ck(binding.load().gpuqt_slab_connect(self._g, peer_global_id, ptrs, C.c_void_p(flags), C.c_int64(n_own),
                                                   C.c_int64(n_halo)), "gpuqt_slab_connect")

    def set_state(self, phi):
        """phi: host [batch][N][2] of the GLOBAL lattice; every local slab takes its rows."""
        parts = [np.ascontiguousarray(phi[:, s.row0:s.row1, :], np.float64) for s in self.slabs]
        ptrs = (C.c_void_p * len(parts))(*[p.ctypes.data for p in parts])
        self._ck(binding.load().gpuqt_slab_set_state(self._g, ptrs), "gpuqt_slab_set_state")

    def get_state(self, which, N):
        """The local slabs' owned rows scattered into a global [batch][N][2] array (zeros elsewhere)."""
        out = np.zeros((self.batch, N, 2), np.float64)
        for i, s in enumerate(self.slabs):
            part = np.empty((self.batch, s.n_own, 2), np.float64)
            self._ck(binding.load().gpuqt_slab_get_state(self._g, i, which, C.c_void_p(part.ctypes.data)), "gpuqt_slab_get_state")
            out[:, s.row0:s.row1, :] = part
        return out

    def _moments(self, fn, what, n, reduce):
        out = np.empty((self.batch, n), np.float64)
        self._ck(fn(self._g, C.c_int32(n), C.c_void_p(out.ctypes.data)), what)
        return sum_over_ranks(out) if reduce else out

    def dos_moments(self, n, reduce=True):
        return self._moments(binding.load().gpuqt_slab_dos_moments, "gpuqt_slab_dos_moments", n, reduce)

    def vac(self, n, reduce=True):
        return self._moments(binding.load().gpuqt_slab_vac, "gpuqt_slab_vac", n, reduce)

    def msd(self, n, reduce=True):
        return self._moments(binding.load().gpuqt_slab_msd, "gpuqt_slab_msd", n, reduce)

    def evolve(self, dt, order):
        self._ck(binding.load().gpuqt_slab_evolve(self._g, C.c_double(dt), C.c_int32(order)), "gpuqt_slab_evolve")


def sum_over_ranks(partial, dist=None):
    """The groups' partial moments added up (moments are linear in the per-slab inner products): one all-reduce of
    [batch][N_m] doubles.  Without a process group the input is returned unchanged."""
    import torch
    if dist is None:
        import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return partial
    t = torch.from_numpy(np.ascontiguousarray(partial))
    if dist.get_backend() == "nccl":
        t = t.cuda()
    dist.all_reduce(t, op=dist.ReduceOp.SUM)
    return t.cpu().numpy()


def slabs_of_rank(n_slabs, rank, world):
    """Global slab ids rank `rank` holds when `n_slabs` slabs are dealt to `world` ranks in consecutive blocks."""
    per = (n_slabs + world - 1) // world
    return list(range(rank * per, min(n_slabs, (rank + 1) * per)))


# ------------------------------------------------------------------ slabs on other ranks: CUDA IPC
class _IpcHandle(C.Structure):
    """cudaIpcMemHandle_t: 64 opaque bytes.  Declared as unsigned bytes, not c_char: ctypes hands a c_char array back
    as a Python bytes object cut at the first NUL, and a handle is binary data full of NULs."""
    _fields_ = [("reserved", C.c_ubyte * 64)]


def _handle_to_bytes(h):
    """All 64 bytes of the handle, NULs included."""
    return C.string_at(C.addressof(h), 64)


def _handle_from_bytes(raw):
    """A handle structure holding exactly the 64 bytes `raw`."""
    if len(raw) != 64:
        raise ValueError(f"a CUDA IPC handle has 64 bytes, got {len(raw)}")
    h = _IpcHandle()
    C.memmove(C.addressof(h), raw, 64)
    return h


def _cuda_libs():
    rt = None
    for name in ("libcudart.so.12", "libcudart.so", "/usr/local/cuda/lib64/libcudart.so"):
        try:
            rt = C.CDLL(name)
            break
        except OSError:
            continue
    if rt is None:
        raise RuntimeError("libcudart not found (CUDA IPC needs it)")
    drv = C.CDLL("libcuda.so.1")
    rt.cudaIpcGetMemHandle.restype = C.c_int
    rt.cudaIpcGetMemHandle.argtypes = [C.POINTER(_IpcHandle), C.c_void_p]
    rt.cudaIpcOpenMemHandle.restype = C.c_int
    rt.cudaIpcOpenMemHandle.argtypes = [C.POINTER(C.c_void_p), _IpcHandle, C.c_uint]      # the handle goes by value
    drv.cuMemGetAddressRange_v2.restype = C.c_int
    drv.cuMemGetAddressRange_v2.argtypes = [C.POINTER(C.c_uint64), C.POINTER(C.c_size_t), C.c_uint64]
    return rt, drv


def _export_pointer(rt, drv, ptr):
    """(ipc handle bytes, offset of ptr inside its allocation)."""
    base, size = C.c_uint64(), C.c_size_t()
    if drv.cuMemGetAddressRange_v2(C.byref(base), C.byref(size), C.c_uint64(ptr)) != 0:
        raise RuntimeError("cuMemGetAddressRange failed")
    h = _IpcHandle()
    if rt.cudaIpcGetMemHandle(C.byref(h), C.c_void_p(base.value)) != 0:
        raise RuntimeError("cudaIpcGetMemHandle failed")
    return _handle_to_bytes(h), ptr - base.value


def connect_ranks(group, dist=None):
    """One slab group per rank, one rank per GPU: every rank publishes CUDA IPC handles of its slabs' vector buffers
    and flag arrays (all_gather_object), opens those of the slabs its own slabs send to, and hands the mapped
    addresses to gpuqt_slab_connect.  The pushes then go straight into the peer GPU's memory over NVLink.
    Host plumbing only.  Exercised by tests/test_gpu_slab_ipc.py, which needs two GPUs with peer access and is skipped
    on a one-GPU box (every box this repository has run on so far: the path below has not executed on hardware yet; the
    one-GPU tests keep all slabs in one group, which needs no connection -- see DESIGN.md "Multi-GPU")."""
    if dist is None:
        import torch.distributed as dist
    rt, drv = _cuda_libs()
    mine = {}
    for i, s in enumerate(group.slabs):
        bufs, flags, n_own, n_halo = group.export(i)
        mine[s.global_id] = ([_export_pointer(rt, drv, b) for b in bufs], _export_pointer(rt, drv, flags), n_own, n_halo)
    everyone = [None] * dist.get_world_size()
    dist.all_gather_object(everyone, mine)
    wanted = {peer for s in group.slabs for peer, _, _ in s.sends} - {s.global_id for s in group.slabs}
    opened = {}

    def open_(handle, offset):
        if handle not in opened:
            h, p = _handle_from_bytes(handle), C.c_void_p()
            if rt.cudaIpcOpenMemHandle(C.byref(p), h, C.c_uint(1)) != 0:       # cudaIpcMemLazyEnablePeerAccess
                raise RuntimeError("cudaIpcOpenMemHandle failed (peer access between the two GPUs is required)")
            opened[handle] = p.value
        return opened[handle] + offset

    for published in everyone:
        for gid, (bufs, flags, n_own, n_halo) in published.items():
            if gid in wanted:
                group.connect(gid, [open_(h, off) for h, off in bufs], open_(*flags), n_own, n_halo)
    group._ipc = opened
    dist.barrier()
