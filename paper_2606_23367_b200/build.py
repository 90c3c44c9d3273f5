"""Builds the C-ABI library libprism.so IN-TREE with nvcc for sm_100a (no torch extension machinery, no JIT cache).

One object per translation unit of csrc/ (k_*.cu kernel families + prism.cu, the C ABI and host driver), compiled in
parallel, linked into paper_2606_23367_b200/libprism.so.  Objects go to paper_2606_23367_b200/_obj/ (git-ignored)."""
from __future__ import annotations

import os
import re
import subprocess
import sys
from concurrent.futures import ThreadPoolExecutor

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
OBJ = os.path.join(HERE, "_obj")
LIB = os.path.join(HERE, "libprism.so")
HEADER = os.path.join(os.path.dirname(HERE), "include", "prism.h")
FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17", "-Xcompiler", "-fPIC,-pthread,-fvisibility=hidden"]
FLAGS += os.environ.get("PRISM_NVCC_FLAGS", "").split()       # builder's switch, e.g. -DPRISM_STATS (pass counts of the root find)


def sources():
    return sorted(f for f in os.listdir(CSRC) if f.endswith(".cu"))


def _deps(path, seen=None):
    """Transitive quoted includes of a source file (inside csrc/ and include/)."""
    seen = set() if seen is None else seen
    if path in seen or not os.path.exists(path):
        return seen
    seen.add(path)
    with open(path) as f:
        for inc in re.findall(r'#include\s+"([^"]+)"', f.read()):
            _deps(os.path.normpath(os.path.join(os.path.dirname(path), inc)), seen)
    return seen


def _stale(target, deps):
    if not os.path.exists(target):
        return True
    t = os.path.getmtime(target)
    return any(os.path.getmtime(d) > t for d in deps)


def needs_build() -> bool:
    srcs = [os.path.join(CSRC, s) for s in sources()]
    alld = set()
    for s in srcs:
        alld |= _deps(s)
    return _stale(LIB, alld | {HEADER})


def build(force: bool = False, verbose: bool = False) -> str:
    if not force and not needs_build():
        return LIB
    nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
    os.makedirs(OBJ, exist_ok=True)
    jobs = []
    for s in sources():
        src = os.path.join(CSRC, s)
        obj = os.path.join(OBJ, s[:-3] + ".o")
        if force or _stale(obj, _deps(src) | {HEADER}):
            cmd = [nvcc] + FLAGS + (["-Xptxas=-v"] if verbose else []) + ["-c", src, "-o", obj]
            jobs.append((s, cmd))

    def run(job):
        name, cmd = job
        res = subprocess.run(cmd, capture_output=True, text=True)
        return name, res

    with ThreadPoolExecutor(max_workers=max(1, min(len(jobs), os.cpu_count() or 1))) as ex:
        for name, res in ex.map(run, jobs):
            if res.returncode != 0:
                raise RuntimeError(f"nvcc failed on {name}:\n" + res.stdout + res.stderr)
            if verbose:
                sys.stderr.write(f"---- {name}\n" + res.stderr)
    objs = [os.path.join(OBJ, s[:-3] + ".o") for s in sources()]
    res = subprocess.run([nvcc, "-gencode", "arch=compute_100a,code=sm_100a", "-shared", "-Xcompiler", "-fPIC,-pthread"] + objs + ["-o", LIB],
                         capture_output=True, text=True)
    if res.returncode != 0:
        raise RuntimeError("link failed:\n" + res.stdout + res.stderr)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
