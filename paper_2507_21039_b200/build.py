"""Build libmg5b200.so in-tree: run the emitter, then nvcc for sm_100a (cross-compiles without a GPU).

Usage: python -m paper_2507_21039_b200.build [--force] [--tune '<json>']

--tune is for tuning builds only: a JSON dict of emitter overrides (emitter/emit.py TUNING) plus an optional "nvcc_extra" list of
compiler flags.  A normal build reads neither the environment nor any file outside the package; the generated program
file records the overrides it was built with.
"""
import json
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
GEN = os.path.join(CSRC, "generated", "mg_programs.inc")
LIB = os.path.join(HERE, "libmg5b200.so")
SOURCES = [os.path.join(CSRC, "mg_lib.cu")]
DEPS = SOURCES + [os.path.join(CSRC, "mg_vm.cuh"), os.path.join(CSRC, "mg_pipes.cuh"), os.path.join(HERE, "..", "include", "mg5b200.h"),
                  os.path.join(HERE, "emitter", "emit.py"), os.path.join(HERE, "emitter", "program.py"),
                  os.path.join(HERE, "emitter", "diagrams.py")]
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17", "--shared",
              "-Xcompiler", "-fPIC", "-Xptxas", "-v"]


def build(force=False, verbose=False, tuning=None):
    newest = max(os.path.getmtime(p) for p in DEPS)
    if not force and os.path.exists(LIB) and os.path.getmtime(LIB) >= newest:
        return LIB
    from .emitter import emit
    tuning = dict(tuning or {})
    extra = list(tuning.pop("nvcc_extra", []))
    emit.main(GEN, tuning=tuning)
    nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
    cmd = [nvcc] + NVCC_FLAGS + extra + ["-o", LIB] + SOURCES
    res = subprocess.run(cmd, capture_output=True, text=True)
    log = res.stdout + res.stderr
    with open(os.path.join(HERE, "csrc", "generated", "build.log"), "w") as f:
        f.write(" ".join(cmd) + "\n" + log)
    if verbose or res.returncode != 0:
        print(log)
    if res.returncode != 0:
        raise RuntimeError("nvcc failed")
    return LIB


if __name__ == "__main__":
    tune = json.loads(sys.argv[sys.argv.index("--tune") + 1]) if "--tune" in sys.argv else None
    print(build(force="--force" in sys.argv or tune is not None, verbose=True, tuning=tune))
