"""Build the CPU oracle (test infrastructure) into oracle/libora.so.

g++ -O2 -ffp-contract=off: no FMA contraction, so the oracle is a fixed IEEE reference
(SURVEY.md §8(c)).  OpenMP only parallelises loops over independent cells/faces, so the
result is identical for any thread count.
"""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
LIB = os.path.join(HERE, "libora.so")
# Second build of the SAME sources with FMA contraction allowed: used only to measure how much
# the oracle's own result moves under a legal change of rounding (tests' sensitivity band).
LIB_FMA = os.path.join(HERE, "libora_fma.so")
# Third build of the SAME sources under AddressSanitizer + UndefinedBehaviorSanitizer:
# loaded only by tests/test_oracle_sanitizers.py in a child process with libasan preloaded.
LIB_ASAN = os.path.join(HERE, "libora_asan.so")
SOURCES = ["ora_capi.cpp"]
HEADERS = ["ora.h", "ora_core.hpp", "ora_solver.hpp", "ora_naive.hpp"]


def needs_build(lib=LIB):
    if not os.path.exists(lib):
        return True
    t = os.path.getmtime(lib)
    return any(os.path.getmtime(os.path.join(HERE, f)) > t for f in SOURCES + HEADERS + ["build.py"])


def build(force=False, variant="ref"):
    lib = {"ref": LIB, "fma": LIB_FMA, "asan": LIB_ASAN}[variant]
    if not force and not needs_build(lib):
        return lib
    fp = ["-ffp-contract=off"] if variant != "fma" else ["-ffp-contract=fast", "-mfma"]
    opt = ["-O2"]
    if variant == "asan":
        opt = ["-O1", "-g", "-fno-omit-frame-pointer", "-fsanitize=address,undefined", "-fno-sanitize-recover=all"]
    cmd = ["g++", "-std=c++17"] + opt + fp + ["-fopenmp", "-fPIC", "-shared",
           "-Wall", "-o", lib] + [os.path.join(HERE, s) for s in SOURCES]
    subprocess.check_call(cmd, cwd=HERE)
    return lib


def asan_runtime():
    """Path of the libasan the asan variant must be preloaded with (LD_PRELOAD), or None."""
    try:
        p = subprocess.check_output(["g++", "-print-file-name=libasan.so"], text=True).strip()
    except (OSError, subprocess.CalledProcessError):
        return None
    return os.path.realpath(p) if os.path.sep in p and os.path.exists(p) else None


if __name__ == "__main__":
    print(build(force="--force" in sys.argv))
    print(build(force="--force" in sys.argv, variant="fma"))
