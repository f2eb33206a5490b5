"""Scale-out over random vectors: random-phase vectors are
independent, so every rank holds a replica of H and its own B vectors.  There is no data-path
collective; the only exchanges are the final gather of the `[B][N_m]` moment blocks and the
max-over-ranks of the device time.  Host plumbing only (torch.distributed), no method arithmetic.
"""
import os


def world():
    """(rank, local_rank, world_size) from the torchrun environment (1 process = 1 GPU)."""
    return (int(os.environ.get("RANK", "0")), int(os.environ.get("LOCAL_RANK", "0")),
            int(os.environ.get("WORLD_SIZE", "1")))


def launch_command(script, argv, n_ranks, port, python=None):
    """The command that starts `script argv...` as `n_ranks` ranks of one node, one process per GPU -- the same
    launch the bench contract uses (`python -m torch.distributed.run --nnodes=1 --nproc-per-node N --master-addr
    127.0.0.1 --master-port P script ...`).  bench.py re-executes itself with it when it is asked for --gpus N > 1
    outside a torchrun environment."""
    import sys
    return [python or sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={int(n_ranks)}",
            "--master-addr", "127.0.0.1", "--master-port", str(int(port)), script, *argv]


def needs_launch(n_gpus: int, env=None) -> bool:
    """True when more than one rank is wanted and this process was not started by torchrun (no WORLD_SIZE)."""
    env = os.environ if env is None else env
    return n_gpus > 1 and "WORLD_SIZE" not in env


def free_port() -> int:
    import socket
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def first_vector(rank: int, batch: int) -> int:
    """Rank r owns the global random vectors [r*B, (r+1)*B)."""
    return rank * batch


def vector_owner(vector: int, batch: int):
    """(rank, slot) that holds global random vector `vector`."""
    return vector // batch, vector % batch


def gather_moments(local, dist=None):
    """All ranks' `[B][N_m]` moment blocks -> `[world*B][N_m]` in global vector order (on every
    rank).  `local` is a CPU or CUDA torch tensor; with no process group it is returned as is."""
    import torch
    if dist is None:
        import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return local
    parts = [torch.empty_like(local) for _ in range(dist.get_world_size())]
    dist.all_gather(parts, local.contiguous())
    return torch.cat(parts, dim=0)


def mean_over_vectors(local, dist=None):
    """Average of the moments over all world*B vectors (the averaging over N_r
    random vectors is the caller's [A17]); one all-reduce of N_m doubles."""
    import torch
    if dist is None:
        import torch.distributed as dist
    s = local.sum(dim=0)
    n = torch.tensor([float(local.shape[0])], dtype=s.dtype, device=s.device)
    if dist.is_available() and dist.is_initialized() and dist.get_world_size() > 1:
        dist.all_reduce(s, op=dist.ReduceOp.SUM)
        dist.all_reduce(n, op=dist.ReduceOp.SUM)
    return s / n


def max_over_ranks(ms: float, device="cpu", dist=None) -> float:
    """Job time = slowest rank's device time."""
    import torch
    if dist is None:
        import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return float(ms)
    t = torch.tensor([ms], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())
