"""Build step for the oracle: compiles lwe_oracle.c into liblwe_oracle.so with gcc.

ORACLE -- test infrastructure.  Run as ``python -m oracle.build`` or call
``build()``.  OpenMP is used when the compiler has it (the loops are annotated the
way the paper's CPU baseline is); without it the same code runs
on one thread.
"""
from __future__ import annotations

import os
import shutil
import subprocess
from pathlib import Path

HERE = Path(__file__).resolve().parent
LIB = HERE / "liblwe_oracle.so"
SRC = [HERE / "lwe_oracle.c", HERE / "lwe_oracle.h"]


def _compilers():
    seen = []
    for cand in ("/usr/bin/gcc", shutil.which("gcc"), os.environ.get("CC"), shutil.which("cc")):
        if cand and cand not in seen and os.path.exists(cand):
            seen.append(cand)
    return seen


def needs_build() -> bool:
    if not LIB.exists():
        return True
    t = LIB.stat().st_mtime
    return any(p.stat().st_mtime > t for p in SRC)


def build(force: bool = False) -> Path:
    if not force and not needs_build():
        return LIB
    errors = []
    for cc in _compilers():
        for omp in (["-fopenmp"], []):
            cmd = [cc, "-O2", "-std=c11", "-Wall", "-Wextra", "-fPIC", *omp,
                   "-shared", "-o", str(LIB), str(SRC[0]), "-lm"]
            r = subprocess.run(cmd, capture_output=True, text=True)
            if r.returncode == 0:
                return LIB
            errors.append(f"{' '.join(cmd)}\n{r.stderr}")
    raise RuntimeError("could not build the oracle:\n" + "\n".join(errors))


if __name__ == "__main__":
    print(build(force=True))
