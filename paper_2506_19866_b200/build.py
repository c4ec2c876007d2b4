"""Builds libternary_sa.so in-tree with nvcc for sm_100a (cross-compiles without a GPU).

    python -m paper_2506_19866_b200.build [--force] [--verbose]
    python -m paper_2506_19866_b200.build --microbench      # only the stand-alone microbenchmarks, on request
"""
from __future__ import annotations

import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libternary_sa.so")
SOURCES = ["sa_api.cu", "sa_kernels.cu", "sa_peak.cu", "sa_plan.cpp", "sa_dense_plan.cpp", "sa_jit.cpp", "sa_static_aot.cu",
           "sa_dense_aot.cu", "sap_api.cu", "sap_plan.cpp", "sap_aot.cu"]
EMBED = {"sa_static_source.inc": ("sa_static_params.h", "sa_static_kernel.cu"),
         "sa_dense_source.inc": ("sa_dense_params.h", "sa_dense_kernel.cu"),
         "sap_source.inc": ("sap_params.h", "sap_kernel.cu")}
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17",
              "-Xcompiler", "-fPIC,-O2,-Wall", "--use_fast_math"]


def _nvcc() -> str:
    cand = os.path.join(os.environ.get("CUDA_HOME", "/usr/local/cuda"), "bin", "nvcc")
    return cand if os.path.exists(cand) else "nvcc"


def _deps():
    out = [os.path.join(HERE, "..", "include", "ternary_sa.h"), os.path.abspath(__file__)]
    for f in os.listdir(CSRC):
        out.append(os.path.join(CSRC, f))
    return out


def stale() -> bool:
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    return any(os.path.getmtime(d) > t for d in _deps())


def embed_static_source() -> None:
    """sa_static_source.inc = params header + kernel source as one C++ raw string literal: the
    text NVRTC compiles at run time (sa_jit.cpp)."""
    for inc, names in EMBED.items():
        parts = []
        for name in names:
            with open(os.path.join(CSRC, name)) as f:
                parts.append(f.read())
        text = 'R"TSASRC(' + "\n".join(parts) + ')TSASRC"\n'
        path = os.path.join(CSRC, inc)
        old = None
        if os.path.exists(path):
            with open(path) as f:
                old = f.read()
        if old != text:
            with open(path, "w") as f:
                f.write(text)


MICRO = os.path.join(CSRC, "microbench")
MICRO_OUT = os.path.join(HERE, "build")


def build_microbench(force: bool = False) -> None:
    """The stand-alone microbenchmarks behind the roofline (csrc/microbench/*.cu -> build/<name>, run by hand on a B200;
    profiles/r2c_microbench.md has their output).  Never part of build(): the library must not depend on them."""
    os.makedirs(MICRO_OUT, exist_ok=True)
    for f in sorted(os.listdir(MICRO)):
        if not f.endswith(".cu"):
            continue
        src, out = os.path.join(MICRO, f), os.path.join(MICRO_OUT, f[:-3])
        if force or not os.path.exists(out) or os.path.getmtime(src) > os.path.getmtime(out):
            subprocess.check_call([_nvcc(), "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O2", "-o", out, src])


def build(force: bool = False, verbose: bool = False) -> str:
    if not force and not stale():
        return LIB
    embed_static_source()
    tmp = LIB + ".tmp.%d" % os.getpid()
    cmd = [_nvcc()] + NVCC_FLAGS + (["-Xptxas", "-v"] if verbose else []) + ["-shared", "-o", tmp]
    cmd += [os.path.join(CSRC, s) for s in SOURCES] + ["-ldl"]
    if verbose:
        print(" ".join(cmd))
    subprocess.check_call(cmd)
    os.replace(tmp, LIB)
    return LIB


if __name__ == "__main__":
    if "--microbench" in sys.argv:
        build_microbench(force="--force" in sys.argv)
        print(MICRO_OUT)
        sys.exit(0)
    print(build(force="--force" in sys.argv, verbose="--verbose" in sys.argv))
