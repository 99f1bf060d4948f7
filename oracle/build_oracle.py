"""Compile oracle/emri_oracle.cpp into two shared libraries next to it.

  libemri_oracle.so     real = double        (the oracle)
  libemri_oracle_ld.so  real = long double   (conditioning diagnostics only)

TEST INFRASTRUCTURE.  `python -m oracle.build_oracle` or `build()`; rebuilds only when the source
is newer than the library.
"""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "emri_oracle.cpp")
LIB = os.path.join(HERE, "libemri_oracle.so")
LIB_LD = os.path.join(HERE, "libemri_oracle_ld.so")
# -ffp-contract=off: no FMA contraction, so the arithmetic is what the source says
FLAGS = ["-O2", "-ffp-contract=off", "-fopenmp", "-shared", "-fPIC", "-std=c++17"]
# EMRI_ORACLE_SANITIZE=1: AddressSanitizer + UndefinedBehaviorSanitizer build; load it with
#   LD_PRELOAD=$(gcc -print-file-name=libasan.so) ASAN_OPTIONS=detect_leaks=0 python -m pytest tests/test_oracle_pins.py
# and rebuild with --force afterwards (profiles/sanitizers_r3.md records the run)
if os.environ.get("EMRI_ORACLE_SANITIZE"):
    FLAGS += ["-g", "-fno-omit-frame-pointer", "-fsanitize=address,undefined", "-fno-sanitize-recover=undefined"]


def _stale(lib):
    return (not os.path.exists(lib)) or os.path.getmtime(lib) < os.path.getmtime(SRC)


def build(force=False):
    for lib, extra in ((LIB, []), (LIB_LD, ["-DEMRI_ORACLE_LONG_DOUBLE"])):
        if force or _stale(lib):
            cmd = ["g++"] + FLAGS + extra + [SRC, "-o", lib]
            subprocess.run(cmd, check=True)
    return LIB, LIB_LD


if __name__ == "__main__":
    print(build(force="--force" in sys.argv))
