"""Build libwcras.so in-tree with nvcc for sm_100a (cross-compiles without a GPU)."""
from __future__ import annotations

import os
import subprocess
from concurrent.futures import ThreadPoolExecutor

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libwcras.so")
SOURCES = ["api.cu", "layout.cu", "dslash.cu", "solver.cu", "ras.cu", "ras_fused.cu", "ras_cta.cu", "ras_cta16.cu", "ras_cl16.cu", "ras_pair.cu", "ras_stream.cu", "noalloc.cu"]
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17",
              "-Xcompiler", "-fPIC", "--expt-relaxed-constexpr"]


def _stale(target: str, deps) -> bool:
    if not os.path.exists(target):
        return True
    t = os.path.getmtime(target)
    return any(os.path.getmtime(d) > t for d in deps)


def build(force: bool = False, verbose: bool = False) -> str:
    nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
    headers = [os.path.join(CSRC, f) for f in os.listdir(CSRC) if f.endswith((".cuh", ".h"))]
    headers.append(os.path.join(HERE, "..", "include", "wcras.h"))
    objdir = os.path.join(HERE, "build")
    os.makedirs(objdir, exist_ok=True)
    jobs = []
    objs = []
    for src in SOURCES:
        s = os.path.join(CSRC, src)
        o = os.path.join(objdir, src.replace(".cu", ".o"))
        objs.append(o)
        if force or _stale(o, [s] + headers):
            cmd = [nvcc] + NVCC_FLAGS + (["-Xptxas", "-v"] if verbose else []) + ["-c", s, "-o", o]
            jobs.append(cmd)

    def run(cmd):
        r = subprocess.run(cmd, capture_output=True, text=True)
        if r.returncode:
            raise RuntimeError("nvcc failed: %s\n%s\n%s" % (" ".join(cmd), r.stdout, r.stderr))
        return r.stderr

    with ThreadPoolExecutor(max_workers=6) as ex:
        logs = list(ex.map(run, jobs))
    if verbose:
        print("\n".join(logs))
    if jobs or not os.path.exists(LIB):
        run([nvcc, "-shared", "-o", LIB] + objs + ["-lcudart"])
    return LIB


def build_microbench() -> str:
    """The standalone packed-fp32 microbenchmark (csrc/microbench_f32x2.cu; results: profiles/r2_microbench.md)."""
    nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
    out = os.path.join(HERE, "build", "microbench_f32x2")
    os.makedirs(os.path.dirname(out), exist_ok=True)
    r = subprocess.run([nvcc, "-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-std=c++17", "--expt-relaxed-constexpr",
                        "-o", out, os.path.join(CSRC, "microbench_f32x2.cu")], capture_output=True, text=True)
    if r.returncode:
        raise RuntimeError("nvcc failed:\n%s\n%s" % (r.stdout, r.stderr))
    return out


def build_phase_profile() -> str:
    """A copy of the library whose persistent block solver (csrc/ras_cta16.cu, -DWC_CTA16_PROFILE) prints the cycles thread 0
    of CTA 0 spends in each phase of the domain loop; load it with WCRAS_LIB=<path> (results: profiles/r2_kernels.md)."""
    build()
    nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
    objdir = os.path.join(HERE, "build")
    obj = os.path.join(objdir, "ras_cta16_phase.o")
    out = os.path.join(objdir, "libwcras_phase.so")
    for cmd in ([nvcc] + NVCC_FLAGS + ["-DWC_CTA16_PROFILE", "-c", os.path.join(CSRC, "ras_cta16.cu"), "-o", obj],
                [nvcc, "-shared", "-o", out] + [os.path.join(objdir, s.replace(".cu", ".o")) for s in SOURCES if s != "ras_cta16.cu"] + [obj, "-lcudart"]):
        r = subprocess.run(cmd, capture_output=True, text=True)
        if r.returncode:
            raise RuntimeError("nvcc failed:\n%s\n%s" % (r.stdout, r.stderr))
    return out


if __name__ == "__main__":
    import sys
    if "--microbench" in sys.argv:
        print(build_microbench())
    elif "--phase-profile" in sys.argv:
        print(build_phase_profile())
    else:
        print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
