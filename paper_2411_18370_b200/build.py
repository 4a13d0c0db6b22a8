"""Build libfasttracks_b200.so in-tree with nvcc for sm_100a (no JIT cache: the .so travels with the repo).

Every .cu of csrc/ is compiled to an object under paper_2411_18370_b200/build/ (git-ignored), the
translation units in parallel, and only those whose source or any header changed; the objects are then
linked into the shared library."""
from __future__ import annotations

import os
import subprocess
import sys
from concurrent.futures import ThreadPoolExecutor

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
OBJ = os.path.join(HERE, "build")
SO = os.path.join(HERE, "libfasttracks_b200.so")
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17",
              "--extended-lambda", "-Xcompiler", "-fPIC"]


def _sources():
    return sorted(f for f in os.listdir(CSRC) if f.endswith(".cu"))


def _headers():
    return [os.path.join(CSRC, f) for f in os.listdir(CSRC) if f.endswith((".cuh", ".h"))] + [
        os.path.join(HERE, "..", "include", "fasttracks_b200.h"), os.path.abspath(__file__)]


def _stale() -> bool:
    if not os.path.exists(SO):
        return True
    t = os.path.getmtime(SO)
    deps = [os.path.join(CSRC, f) for f in os.listdir(CSRC)] + _headers()
    return any(os.path.getmtime(d) > t for d in deps)


def _compile_one(nvcc, src, verbose):
    obj = os.path.join(OBJ, src[:-3] + ".o")
    extra = os.environ.get("FT_NVCC_EXTRA", "").split()   # e.g. -DFT_K1_INT_CVT=0 (tuning experiments)
    cmd = [nvcc] + NVCC_FLAGS + extra + (["-Xptxas", "-v"] if verbose else []) + ["-c", os.path.join(CSRC, src), "-o", obj]
    r = subprocess.run(cmd, capture_output=True, text=True)
    return src, obj, r


def build(force: bool = False, verbose: bool = False) -> str:
    """Compile if missing or stale.  Safe under concurrent callers (one process per GPU): an exclusive
    file lock serialises them and the library is written to a temporary name, then renamed."""
    if not (force or _stale()):
        return SO
    import fcntl
    with open(SO + ".lock", "w") as lock:
        fcntl.flock(lock, fcntl.LOCK_EX)
        if force or _stale():  # another process may have built it while we waited
            nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
            os.makedirs(OBJ, exist_ok=True)
            t_hdr = max(os.path.getmtime(h) for h in _headers())
            todo, objs = [], []
            for src in _sources():
                obj = os.path.join(OBJ, src[:-3] + ".o")
                objs.append(obj)
                if force or verbose or not os.path.exists(obj) or \
                        os.path.getmtime(obj) < max(t_hdr, os.path.getmtime(os.path.join(CSRC, src))):
                    todo.append(src)
            with ThreadPoolExecutor(max_workers=min(8, max(1, len(todo)))) as ex:
                results = list(ex.map(lambda s: _compile_one(nvcc, s, verbose), todo))
            failed = False
            for src, obj, r in results:
                if verbose or r.returncode != 0:
                    sys.stderr.write(f"--- {src}\n" + r.stdout + r.stderr)
                if r.returncode != 0:
                    failed = True
                    if os.path.exists(obj):
                        os.remove(obj)
            if failed:
                raise RuntimeError("nvcc failed building libfasttracks_b200.so")
            tmp = f"{SO}.tmp.{os.getpid()}"
            r = subprocess.run([nvcc, "-shared", "-gencode", "arch=compute_100a,code=sm_100a"] + objs + ["-o", tmp],
                               capture_output=True, text=True)
            if r.returncode != 0:
                sys.stderr.write(r.stdout + r.stderr)
                if os.path.exists(tmp):
                    os.remove(tmp)
                raise RuntimeError("nvcc failed linking libfasttracks_b200.so")
            os.replace(tmp, SO)
    return SO


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
