"""Build libmadme.so (the C-ABI library of include/madme.h) in-tree with nvcc for sm_100a.

Step 1 regenerates csrc/generated/*.inc from the diagram generator (gen/), step 2 compiles csrc/madme.cu.
`python -m paper_2211_14056_b200.build [--force]`.  nvcc cross-compiles without a GPU.
"""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libmadme.so")
NVCC = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17", "-shared",
         "-Xcompiler", "-fPIC", "-Xptxas", "-v"]


def _sources():
    out = []
    for root, _, files in os.walk(CSRC):
        out += [os.path.join(root, f) for f in files if f.endswith((".cu", ".cuh", ".inc", ".h"))]
    out.append(os.path.join(os.path.dirname(HERE), "include", "madme.h"))
    return out


def build(force: bool = False, verbose: bool = False) -> str:
    from .gen import emit
    emit.emit_all()
    deps = _sources() + [os.path.join(HERE, "gen", "emit.py"), os.path.join(HERE, "gen", "diagrams.py")]
    if not force and os.path.exists(LIB) and all(os.path.getmtime(LIB) >= os.path.getmtime(d) for d in deps):
        return LIB
    cmd = [NVCC] + FLAGS + ["-o", LIB, os.path.join(CSRC, "madme.cu")]
    res = subprocess.run(cmd, capture_output=True, text=True)
    log = os.path.join(HERE, "build.log")
    with open(log, "w") as f:
        f.write(" ".join(cmd) + "\n" + res.stdout + res.stderr)
    if verbose or res.returncode:
        sys.stderr.write(res.stdout + res.stderr)
    if res.returncode:
        raise RuntimeError("nvcc failed, see " + log)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
