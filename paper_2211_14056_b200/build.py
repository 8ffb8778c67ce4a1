"""Build libmadme.so (the C-ABI library of include/madme.h) in-tree with nvcc for sm_100a.

Step 1 regenerates csrc/generated/*.inc from the diagram generator (gen/), step 2 compiles csrc/*.cu (in parallel).
`python -m paper_2211_14056_b200.build [--force]`.  nvcc cross-compiles without a GPU.
"""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libmadme.so")
NVCC = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
CFLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17",
          "-Xcompiler", "-fPIC", "-Xptxas", "-v"]


def _sources():
    out = []
    for root, _, files in os.walk(CSRC):
        out += [os.path.join(root, f) for f in files if f.endswith((".cu", ".cuh", ".inc", ".h"))]
    out.append(os.path.join(os.path.dirname(HERE), "include", "madme.h"))
    return out


PROCESSES = ["epem_mupmum", "gg_ttx", "gg_ttxg", "gg_ttxgg", "gg_ttxggg", "qqx_ttx", "qqx_ttxg", "qg_ttxq", "qqx_ttxgg", "qg_ttxqg", "qxg_ttxqx", "qxg_ttxqxg"]


def _compile(job):
    src, obj, defs = job
    cmd = [NVCC] + CFLAGS + defs + os.environ.get("MADME_NVCC_FLAGS", "").split() + ["-c", "-o", obj, os.path.join(CSRC, src)]
    res = subprocess.run(cmd, capture_output=True, text=True)
    return " ".join(cmd) + "\n" + res.stdout + res.stderr, res.returncode


def build(force: bool = False, verbose: bool = False) -> str:
    """Each process's kernels are their own translation units (proc_eval.cu / proc_vegas.cu with -DMADME_PROC=...),
    compiled in parallel, then linked with madme.cu into libmadme.so."""
    from concurrent.futures import ThreadPoolExecutor
    from .gen import emit
    emit.emit_all()
    deps = _sources() + [os.path.join(HERE, "gen", "emit.py"), os.path.join(HERE, "gen", "diagrams.py")]
    if not force and os.path.exists(LIB) and all(os.path.getmtime(LIB) >= os.path.getmtime(d) for d in deps):
        return LIB
    objdir = os.path.join(HERE, "build")
    os.makedirs(objdir, exist_ok=True)
    jobs = [("madme.cu", os.path.join(objdir, "madme.o"), []), ("unweight_static.cu", os.path.join(objdir, "unweight_static.o"), [])]
    for p in reversed(PROCESSES):   # the big ones first
        jobs.append(("proc_eval.cu", os.path.join(objdir, "eval_%s.o" % p), ["-DMADME_PROC=" + p]))
        jobs.append(("proc_vegas.cu", os.path.join(objdir, "vegas_%s.o" % p), ["-DMADME_PROC=" + p]))
    with ThreadPoolExecutor(max_workers=min(len(jobs), os.cpu_count() or 4)) as ex:
        results = list(ex.map(_compile, jobs))
    link = [NVCC, "-gencode", "arch=compute_100a,code=sm_100a", "-shared", "-o", LIB] + [j[1] for j in jobs]
    failed = any(rc for _, rc in results)
    text = "".join(t for t, _ in results)
    if not failed:
        res = subprocess.run(link, capture_output=True, text=True)
        text += " ".join(link) + "\n" + res.stdout + res.stderr
        failed = res.returncode != 0
    if not failed:   # the stand-alone measurement programs of csrc/probes (profiles/r2_probes.md), not linked into the library
        for name in sorted(os.listdir(os.path.join(CSRC, "probes"))):
            if name.endswith(".cu"):
                cmd = [NVCC, "-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-o", os.path.join(objdir, name[:-3]), os.path.join(CSRC, "probes", name)]
                res = subprocess.run(cmd, capture_output=True, text=True)
                text += " ".join(cmd) + "\n" + res.stdout + res.stderr
                failed = failed or res.returncode != 0
    log = os.path.join(HERE, "build.log")
    with open(log, "w") as f:
        f.write(text)
    if verbose or failed:
        sys.stderr.write(text)
    if failed:
        raise RuntimeError("nvcc failed, see " + log)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
