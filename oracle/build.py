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


SAN_LIB = HERE / "liblwe_oracle_san.so"
SAN_FLAGS = ["-fsanitize=address,undefined", "-fno-sanitize-recover=undefined", "-fno-omit-frame-pointer", "-g", "-O1"]


def build_sanitized(force: bool = False) -> Path:
    """The same source under AddressSanitizer + UndefinedBehaviorSanitizer (the only sanitizer that can
    run on this pool guards the checker every parity claim rests on).  No OpenMP (its runtime's own allocations
    only add noise); -fno-sanitize-recover makes any undefined behaviour abort instead of printing and going on.
    A process that loads this library must start with libasan preloaded -- tests/test_oracle_sanitized.py runs its
    checks in such a child process."""
    if not force and SAN_LIB.exists() and all(p.stat().st_mtime <= SAN_LIB.stat().st_mtime for p in SRC):
        return SAN_LIB
    errors = []
    for cc in _compilers():
        cmd = [cc, *SAN_FLAGS, "-std=c11", "-Wall", "-Wextra", "-fPIC", "-shared", "-o", str(SAN_LIB), str(SRC[0]), "-lm"]
        r = subprocess.run(cmd, capture_output=True, text=True)
        if r.returncode == 0:
            return SAN_LIB
        errors.append(f"{' '.join(cmd)}\n{r.stderr}")
    raise RuntimeError("could not build the sanitized oracle:\n" + "\n".join(errors))


def asan_runtime() -> str:
    """path of libasan.so for LD_PRELOAD (the sanitized library is loaded into an uninstrumented python)"""
    for cc in _compilers():
        r = subprocess.run([cc, "-print-file-name=libasan.so"], capture_output=True, text=True)
        path = r.stdout.strip()
        if r.returncode == 0 and os.path.isabs(path) and os.path.exists(path):
            return os.path.realpath(path)
    raise RuntimeError("libasan.so not found")


def build(force: bool = False) -> Path:
    if os.environ.get("LWE_ORACLE_SANITIZE") == "1":          # set by the sanitizer test's child process only
        return build_sanitized(force)
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
    import sys
    print(build_sanitized(force=True) if "--sanitize" in sys.argv else build(force=True))
