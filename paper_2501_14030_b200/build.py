"""Builds paper_2501_14030_b200/libhr_b200.so (the C-ABI library of include/hr.h) with nvcc for
sm_100a.  In-tree, so the .so travels to the GPU box with the repo snapshot."""
import os
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(HERE)
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libhr_b200.so")
SOURCES = ["hr_api.cu", "hr_kernels.cu", "hr_measure.cu"]
HEADERS = ["hr_internal.h", "fd_tables.cuh", "hr_march.cuh", os.path.join(ROOT, "include", "hr.h")]
NVCC_FLAGS = ["-O3", "-std=c++17", "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo",
              "-Xcompiler", "-fPIC", "-Xcompiler", "-fvisibility=hidden"]
# The ablation of PAPER.md:193, 301-321: the same sources with FMA contraction switched off
# (plain expressions compile to separate multiplies and adds; the explicit fma() of the reciprocal's Newton
# steps stays).  Loaded instead of the product library when HR_B200_LIB names it (binding.py).
LIB_NOFMAD = os.path.join(HERE, "libhr_b200_nofmad.so")


def _nvcc() -> str:
    for c in (os.environ.get("NVCC"), "/usr/local/cuda/bin/nvcc", "nvcc"):
        if c and (os.path.isabs(c) and os.path.exists(c) or not os.path.isabs(c)):
            return c
    return "nvcc"


def _stale() -> bool:
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    deps = [os.path.join(CSRC, s) for s in SOURCES] + [
        h if os.path.isabs(h) else os.path.join(CSRC, h) for h in HEADERS] + [__file__]
    return any(os.path.getmtime(d) > t for d in deps)


def _compile_all(jobs, verbose):
    """jobs: (library path, object suffix, extra flags); every translation unit of every job side by side."""
    procs = []
    for lib, suffix, extra in jobs:
        for src in SOURCES:
            obj = os.path.join(CSRC, src.replace(".cu", suffix + ".o"))
            # HR_NVCC_DEFS="-DHR_MARCH_D_F64=3 ...": tuning overrides of the macros in hr_internal.h
            cmd = [_nvcc(), *NVCC_FLAGS, *extra, *os.environ.get("HR_NVCC_DEFS", "").split(), "-c",
                   os.path.join(CSRC, src), "-o", obj]
            if verbose:
                cmd.insert(1, "-Xptxas=-v")
            procs.append((cmd, subprocess.Popen(cmd)))
    for cmd, pr in procs:
        if pr.wait() != 0:
            raise subprocess.CalledProcessError(pr.returncode, cmd)
    for lib, suffix, _ in jobs:
        objs = [os.path.join(CSRC, src.replace(".cu", suffix + ".o")) for src in SOURCES]
        tmp = lib + f".tmp{os.getpid()}"
        subprocess.run([_nvcc(), "-shared", "-gencode", "arch=compute_100a,code=sm_100a", *objs,
                        "-o", tmp], check=True)
        os.replace(tmp, lib)


def build(force: bool = False, verbose: bool = False, ablation: bool = True) -> str:
    """The product library (FMA contraction on, nvcc's default) and, with `ablation`, its --fmad=false twin."""
    if not force and not _stale() and (not ablation or os.path.exists(LIB_NOFMAD)):
        return LIB
    jobs = [(LIB, "", ["--fmad=true"])]
    if ablation:
        jobs.append((LIB_NOFMAD, "_nofmad", ["--fmad=false"]))
    _compile_all(jobs, verbose)
    return LIB


if __name__ == "__main__":
    import sys
    print(build(force=True, verbose="-v" in sys.argv, ablation="--no-ablation" not in sys.argv))
