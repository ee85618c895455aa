"""Build libpinmpc.so in-tree with nvcc for sm_100a (no JIT cache: the .so travels with the repo)."""
from __future__ import annotations

import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libpinmpc.so")
SOURCES = ["pinmpc_api.cu", "pinmpc_dense.cu", "pinmpc_srb.cu", "pinmpc_tmem.cu", "pinmpc_landmarks.cu", "pinmpc_split.cu", "pinmpc_centroidal.cu"]
# bench-only helper (a register-resident FMA loop that measures the FP32 peak): its own library, not part of the product ABI
PROBE_SRC = "bench_probe.cu"
PROBE_LIB = os.path.join(HERE, "libpinmpc_benchprobe.so")
# --ftz=true: denormals flushed to zero (nothing here lives near 1e-38; the iteration kernel loses its denormal slow
# paths: 1.422 -> 1.407 ms); --prec-sqrt=false: the square roots of the assembly's Cholesky at 1-2 ulp (34 -> 31 us).
# Measured and parity-checked; --prec-div=false and -use_fast_math make the iteration kernel slower (1.44-1.45 ms).
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17", "--ftz=true", "--prec-sqrt=false",
              "-Xcompiler", "-fPIC", "-Xptxas", "-v"] + os.environ.get("PINMPC_NVCC_EXTRA", "").split()


def _stale() -> bool:
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    deps = [os.path.join(CSRC, f) for f in os.listdir(CSRC)] + [os.path.join(HERE, "..", "include", "pinmpc.h")]
    return any(os.path.getmtime(d) > t for d in deps)


def build(force: bool = False, verbose: bool = False) -> str:
    if not force and not _stale():
        return LIB
    nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
    objs = []
    procs = []
    for src in SOURCES:
        obj = os.path.join(CSRC, src.replace(".cu", ".o"))
        objs.append(obj)
        cmd = [nvcc] + NVCC_FLAGS + ["-c", os.path.join(CSRC, src), "-o", obj]
        procs.append((src, subprocess.Popen(cmd, stdout=subprocess.PIPE, stderr=subprocess.STDOUT, text=True)))
    log = []
    for src, p in procs:
        out, _ = p.communicate()
        log.append(f"== {src}\n{out}")
        if p.returncode:
            sys.stderr.write("\n".join(log))
            raise RuntimeError(f"nvcc failed on {src}")
    tmp = LIB + f".tmp{os.getpid()}"
    subprocess.check_call([nvcc, "-gencode", "arch=compute_100a,code=sm_100a", "-shared", "-o", tmp] + objs + ["-lcudart"])
    os.replace(tmp, LIB)
    tmp = PROBE_LIB + f".tmp{os.getpid()}"
    subprocess.check_call([nvcc, "-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-shared", "-Xcompiler", "-fPIC", "-o", tmp,
                           os.path.join(CSRC, PROBE_SRC), "-lcudart"])
    os.replace(tmp, PROBE_LIB)
    with open(LIB.replace(".so", ".ptxas.log"), "w") as f:      # register / spill report of the build (git-ignored)
        f.write("\n".join(log) + "\n")
    if verbose:
        print("\n".join(log))
    return LIB


if __name__ == "__main__":
    build(force="--force" in sys.argv, verbose=True)
