"""Seeded counter-based random numbers for the synthetic workloads.

splitmix64 in closed (counter) form: output i of a stream with state0 = seed is
mix(seed + (i+1)*GAMMA).  Vectorised with numpy uint64 wrap-around arithmetic.
This module holds no arithmetic of the GPUQT method; it only produces inputs.
Recipe: SURVEY.md §8(d) "RNG" / DESIGN.md "Input recipe".
"""
import numpy as np

_GAMMA = np.uint64(0x9E3779B97F4A7C15)
_M1 = np.uint64(0xBF58476D1CE4E5B9)
_M2 = np.uint64(0x94D049BB133111EB)
BASE_SEED = 170501387


def stream_seed(config: int, stream: int, vector: int = 0) -> int:
    """state0 = 170501387 xor (config << 32) xor (stream << 16) xor vector."""
    return (BASE_SEED ^ (int(config) << 32) ^ (int(stream) << 16) ^ int(vector)) & 0xFFFFFFFFFFFFFFFF


def splitmix64(seed: int, n: int, offset: int = 0) -> np.ndarray:
    """Outputs offset .. offset+n-1 of the splitmix64 stream started at `seed`."""
    with np.errstate(over="ignore"):
        ctr = np.arange(offset + 1, offset + n + 1, dtype=np.uint64)
        z = np.uint64(seed & 0xFFFFFFFFFFFFFFFF) + _GAMMA * ctr
        z = (z ^ (z >> np.uint64(30))) * _M1
        z = (z ^ (z >> np.uint64(27))) * _M2
        z = z ^ (z >> np.uint64(31))
    return z


def uniform01(seed: int, n: int, offset: int = 0) -> np.ndarray:
    """u = (next >> 11) * 2^-53 in [0, 1)."""
    return (splitmix64(seed, n, offset) >> np.uint64(11)).astype(np.float64) * (2.0 ** -53)
