"""Build libteuk.so in-tree with nvcc for sm_100a (cross-compiles without a GPU).

One object per translation unit under csrc/ (compiled in parallel, rebuilt only when the unit or a header changed),
linked into paper_1006_0663_b200/libteuk.so.  Objects live in csrc/build/ (git-ignored)."""
from __future__ import annotations

import os
import subprocess
import sys
from concurrent.futures import ThreadPoolExecutor

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
OBJ = os.path.join(CSRC, "build")
SO = os.path.join(HERE, "libteuk.so")
SOURCES = ["teuk.cu", "k_generic1.cu", "k_generic2.cu", "k_generic4.cu", "k_tma.cu", "k_tb2.cu", "k_march.cu"]
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17", "--fmad=true",
              "-Xcompiler", "-fPIC,-O2,-ffp-contract=off"]


def _compile(nvcc: str, src: str, obj: str, verbose: bool) -> None:
    tmp = obj + f".tmp{os.getpid()}"
    cmd = [nvcc, *NVCC_FLAGS, *(["-Xptxas", "-v"] if verbose else []), "-c", os.path.join(CSRC, src), "-o", tmp]
    subprocess.check_call(cmd)
    os.replace(tmp, obj)


def _deps(path: str, seen: set) -> set:
    """the file plus every quoted #include reachable from it (system headers are not tracked)"""
    path = os.path.normpath(path)
    if path in seen or not os.path.exists(path):
        return seen
    seen.add(path)
    with open(path) as f:
        for line in f:
            line = line.strip()
            if line.startswith("#include \""):
                _deps(os.path.join(os.path.dirname(path), line.split('"')[1]), seen)
    return seen


def build(force: bool = False, verbose: bool = False) -> str:
    nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
    os.makedirs(OBJ, exist_ok=True)
    objs, stale = [], []
    for s in SOURCES:
        o = os.path.join(OBJ, s[:-3] + ".o")
        objs.append(o)
        newest = max(os.path.getmtime(p) for p in _deps(os.path.join(CSRC, s), {os.path.normpath(__file__)}))
        if force or not os.path.exists(o) or os.path.getmtime(o) < newest:
            stale.append((s, o))
    if stale:
        with ThreadPoolExecutor(max_workers=min(len(stale), os.cpu_count() or 1)) as ex:
            for f in [ex.submit(_compile, nvcc, s, o, verbose) for s, o in stale]:
                f.result()
    if stale or not os.path.exists(SO) or os.path.getmtime(SO) < max(os.path.getmtime(o) for o in objs):
        tmp = SO + f".tmp{os.getpid()}"
        subprocess.check_call([nvcc, "-gencode", "arch=compute_100a,code=sm_100a", "-shared", *objs, "-o", tmp])
        os.replace(tmp, SO)
    return SO


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
