"""Build libtcp.so (the C-ABI CUDA library) in-tree with nvcc for sm_100a.

The fused step kernels are ~70 template instantiations; they live in four translation units
(precision x boundary kind x hydrodynamic lattice) that are compiled in parallel and linked with the host API.

Usage: python -m paper_2401_03041_b200.build [--force] [--verbose]
"""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
OBJ = os.path.join(HERE, "build")
LIB = os.path.join(HERE, "libtcp.so")
SOURCES = ["tcp_api.cu", "tcp_fused_f64_periodic.cu", "tcp_fused_f64_walls.cu", "tcp_fused_f32_periodic.cu",
           "tcp_fused_f32_walls.cu", "tcp_fused_f64_periodic_q19.cu", "tcp_fused_f64_walls_q19.cu",
           "tcp_fused_f32_periodic_q19.cu", "tcp_fused_f32_walls_q19.cu"]
HEADERS = ["tcp_lattice.cuh", "tcp_device.cuh", "tcp_kernels.cuh", "tcp_step.cuh", "tcp_rk.cuh",
           "tcp_launch.h", "tcp_launch.inl", "tcp_real.cuh", "tcp_pair.cuh", "tcp_halo.cuh"]
# IEEE division / sqrt kept (no fast-math); FMA contraction on
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-std=c++17", "-O3", "-lineinfo", "-fmad=true",
              "-Xcompiler", "-fPIC"]


def _stale() -> bool:
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    deps = [os.path.join(CSRC, f) for f in SOURCES + HEADERS] + [os.path.join(HERE, "..", "include", "tcp.h"), __file__]
    return any(os.path.getmtime(d) > t for d in deps)


def build(force: bool = False, verbose: bool = False) -> str:
    if not force and not _stale():
        return LIB
    nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
    os.makedirs(OBJ, exist_ok=True)
    extra = ["-Xptxas", "-v"] if verbose else []
    procs = []
    for src in SOURCES:
        obj = os.path.join(OBJ, src.replace(".cu", ".o"))
        cmd = [nvcc] + NVCC_FLAGS + extra + ["-c", "-o", obj, os.path.join(CSRC, src)]
        procs.append((src, obj, subprocess.Popen(cmd, stdout=subprocess.PIPE, stderr=subprocess.STDOUT, text=True)))
    objs, failed = [], []
    for src, obj, p in procs:
        out, _ = p.communicate()
        if verbose or p.returncode != 0:
            sys.stderr.write(out)
        if p.returncode != 0:
            failed.append(src)
        objs.append(obj)
    if failed:
        raise RuntimeError(f"nvcc failed on {failed}")
    subprocess.run([nvcc, "-shared", "-gencode", "arch=compute_100a,code=sm_100a", "-o", LIB] + objs, check=True)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="--verbose" in sys.argv))
