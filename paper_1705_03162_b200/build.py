"""Build libswept_b200.so in-tree with nvcc for sm_100a (no torch headers involved).

    python -m paper_1705_03162_b200.build [--force]

Flags: -fmad=false (every fused multiply-add in the kernels is explicit, so the GPU evaluates exactly the
expression trees of DESIGN.md §4), IEEE division/sqrt, no flush-to-zero, -lineinfo for ncu source pages.
"""
from __future__ import annotations

import concurrent.futures as cf
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
BUILD = os.path.join(HERE, "build")
LIB = os.path.join(HERE, "libswept_b200.so")
# (source, object stem, extra defines); the Euler swept kernels are compiled in four parallel slices, slowest first
SOURCES = [("kernels_euler_inst.cu", f"kernels_euler_i{i}r{r}", [f"-DSWEPT_INST={i}", f"-DSWEPT_RK2={r}"])
           for i in (1, 0) for r in (0, 1)]
SOURCES += [("swept_api.cu", "swept_api", []), ("probes.cu", "probes", []), ("flow_static.cu", "flow_static", []), ("shard_kernels.cu", "shard_kernels", []),
           ("kernels_heat.cu", "kernels_heat", []), ("kernels_ks.cu", "kernels_ks", []),
           ("kernels_ks3.cu", "kernels_ks3", []),
           ("kernels_euler.cu", "kernels_euler", [])]
NVCC_FLAGS = ["-std=c++17", "-O3", "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo",
              "-fmad=false", "-prec-div=true", "-prec-sqrt=true", "-ftz=false",
              "-Xcompiler", "-fPIC"]


def _nvcc() -> str:
    for cand in (os.environ.get("NVCC"), "/usr/local/cuda/bin/nvcc", "nvcc"):
        if cand and (os.path.sep not in cand or os.path.exists(cand)):
            return cand
    return "nvcc"


def _deps_mtime() -> float:
    t = 0.0
    for root in (CSRC, os.path.join(os.path.dirname(HERE), "include")):
        for f in os.listdir(root):
            t = max(t, os.path.getmtime(os.path.join(root, f)))
    return max(t, os.path.getmtime(__file__))


def _includes(path: str, seen: set) -> set:
    """Transitive closure of the quoted #include files of `path` (for per-object staleness)."""
    if path in seen or not os.path.exists(path):
        return seen
    seen.add(path)
    with open(path) as f:
        for line in f:
            line = line.strip()
            if line.startswith("#include \""):
                inc = line.split('"')[1]
                _includes(os.path.normpath(os.path.join(os.path.dirname(path), inc)), seen)
    return seen


def build(force: bool = False, verbose: bool = False) -> str:
    if not force and os.path.exists(LIB) and os.path.getmtime(LIB) >= _deps_mtime():
        return LIB
    os.makedirs(BUILD, exist_ok=True)
    nvcc = _nvcc()
    import time
    started = time.time()  # the library is stamped with the START of the build: a source edited while it ran is newer

    def compile_one(item) -> str:
        src, stem, defs = item
        obj = os.path.join(BUILD, stem + ".o")
        deps = _includes(os.path.join(CSRC, src), set()) | {os.path.abspath(__file__)}
        if not force and not verbose and os.path.exists(obj) and \
                os.path.getmtime(obj) >= max(os.path.getmtime(d) for d in deps):
            return obj
        cmd = [nvcc, *NVCC_FLAGS, *defs, "-c", os.path.join(CSRC, src), "-o", obj]
        if verbose:
            cmd.insert(1, "-Xptxas=-v")
        r = subprocess.run(cmd, capture_output=True, text=True)
        if r.returncode != 0:
            raise RuntimeError(f"nvcc failed for {stem}:\n{r.stdout}\n{r.stderr}")
        if verbose:
            sys.stderr.write(r.stderr)
        return obj

    with cf.ThreadPoolExecutor(max_workers=min(len(SOURCES), os.cpu_count() or 4)) as ex:
        objs = list(ex.map(compile_one, SOURCES))
    tmp = LIB + f".tmp{os.getpid()}"
    r = subprocess.run([nvcc, "-shared", "-o", tmp, *objs], capture_output=True, text=True)
    if r.returncode != 0:
        raise RuntimeError(f"link failed:\n{r.stdout}\n{r.stderr}")
    os.utime(tmp, (started, started))
    for o in objs:
        if os.path.getmtime(o) > started:
            os.utime(o, (started, started))
    os.replace(tmp, LIB)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
