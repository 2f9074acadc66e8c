"""Build the CPU oracle shared library (TEST INFRASTRUCTURE, see hr_oracle.h).

`python oracle/build.py` or `oracle.build.build()` compiles
    hr_oracle_setup.c            (fp64 set-up)
    hr_oracle_step.c  x 2        (ORC_REAL = double / float)
into oracle/liboracle_hr.so with gcc -O2, no -ffast-math, no FMA contraction, OpenMP on the
outermost loops only.  Nothing here touches the CUDA path.
"""
import os
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
LIB = os.path.join(HERE, "liboracle_hr.so")
SOURCES = ["hr_oracle_setup.c", "hr_oracle_step.c", "hr_oracle.h", "hr_oracle_internal.h"]
CFLAGS = ["-O2", "-std=gnu99", "-fPIC", "-fopenmp", "-ffp-contract=off", "-Wall", "-Wextra",
          "-Wno-unused-parameter"]


def _stale() -> bool:
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    return any(os.path.getmtime(os.path.join(HERE, s)) > t for s in SOURCES + ["build.py"])


def build(force: bool = False) -> str:
    if not force and not _stale():
        return LIB
    objs = []
    jobs = [
        ("hr_oracle_setup.c", "hr_oracle_setup.o", []),
        ("hr_oracle_step.c", "hr_oracle_step_f64.o", ["-DORC_REAL=double", "-DORC_SUF=_f64"]),
        ("hr_oracle_step.c", "hr_oracle_step_f32.o", ["-DORC_REAL=float", "-DORC_SUF=_f32"]),
    ]
    for src, obj, defs in jobs:
        cmd = ["gcc", *CFLAGS, *defs, "-c", os.path.join(HERE, src), "-o", os.path.join(HERE, obj)]
        subprocess.run(cmd, check=True)
        objs.append(os.path.join(HERE, obj))
    tmp = LIB + f".tmp{os.getpid()}"
    subprocess.run(["gcc", "-shared", "-fopenmp", *objs, "-o", tmp, "-lm"], check=True)
    os.replace(tmp, LIB)
    return LIB


if __name__ == "__main__":
    print(build(force=True))
