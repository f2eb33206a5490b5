"""Build libgpuqt.so (sm_100a only) in-tree with nvcc.  `python -m paper_1705_01387_b200.build`.

Six translation units compiled in parallel and linked into one shared library: gpuqt.cu (the C-ABI,
host logic and the small kernels), step_kernels.cu once per Mode of the step kernel, and transform_static.cu
(the allocation-free energy transform with its static device scratch)."""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.environ.get("GPUQT_LIB") or os.path.join(HERE, "libgpuqt.so")
UNITS = [("gpuqt.cu", [])] + [("step_kernels.cu", [f"-DGPUQT_TU_MODE={m}"]) for m in range(4)] + [("transform_static.cu", [])]
DEPS = [os.path.join(CSRC, f) for f in ("gpuqt.cu", "step_kernels.cu", "kernels.cuh", "host_util.h", "slab_group.inl", "transform_static.cu")] + [
    os.path.join(os.path.dirname(HERE), "include", "gpuqt.h")]
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17",
              "-Xcompiler", "-fPIC"]


def needs_build() -> bool:
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    return any(os.path.getmtime(d) > t for d in DEPS)


def build(force: bool = False, verbose: bool = False) -> str:
    if force or needs_build():
        nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
        extra = os.environ.get("GPUQT_NVCC_EXTRA", "").split()      # e.g. -DGPUQT_MINB=1 (kernel tuning macros)
        flags = NVCC_FLAGS + extra + (["-Xptxas", "-v"] if verbose else [])
        objs, procs = [], []
        for i, (src, defs) in enumerate(UNITS):
            obj = f"{LIB}.{i}.o"
            objs.append(obj)
            procs.append(subprocess.Popen([nvcc] + flags + defs + ["-c", "-o", obj, os.path.join(CSRC, src)]))
        codes = [p.wait() for p in procs]
        if any(codes):
            raise subprocess.CalledProcessError(max(codes), "nvcc -c")
        subprocess.check_call([nvcc, "-shared", "-gencode", "arch=compute_100a,code=sm_100a", "-o", LIB] + objs)
        for o in objs:
            os.remove(o)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
