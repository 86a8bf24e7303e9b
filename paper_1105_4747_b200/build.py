"""Build paper_1105_4747_b200/liblya.so (the C-ABI library of include/lya.h) with nvcc for sm_100a.

In-tree, explicit nvcc: the .so travels to the GPU box with the repo snapshot; nothing is JIT-compiled.
`python -m paper_1105_4747_b200.build [--force] [--verbose]`
"""
from __future__ import annotations

import hashlib
import os
import shutil
import subprocess
import sys

_HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(_HERE, "csrc")
LIB = os.path.join(_HERE, "liblya.so")
STAMP = LIB + ".sha256"
SOURCES = ["lya_api.cu", "gas.cu", "tau.cu", "normalize.cu", "forest_host.cu", "probe.cu", "observe.cu", "power.cu", "fields.cu"]
HEADERS = ["lya_internal.h", "root_iter.h", "gas_cell.h", "pdf_bin.h", os.path.join("..", "..", "include", "lya.h")]
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17",
              "-Xcompiler", "-fPIC"]
LINK_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-shared", "-Xcompiler", "-fPIC", "-ldl"]
OBJ_DIR = os.path.join(_HERE, "build")           # git-ignored; objects are cached per content hash


def nvcc() -> str:
    for cand in (shutil.which("nvcc"), "/usr/local/cuda/bin/nvcc"):
        if cand and os.path.exists(cand):
            return cand
    raise RuntimeError("nvcc not found: the CUDA library cannot be built (there is no CPU fallback)")


def _headers_digest() -> bytes:
    h = hashlib.sha256(" ".join(NVCC_FLAGS + LINK_FLAGS).encode())
    for d in sorted(HEADERS):
        with open(os.path.join(CSRC, d), "rb") as f:
            h.update(d.encode() + b"\0" + f.read())
    return h.digest()


def _source_digest(src: str, hdr: bytes) -> str:
    h = hashlib.sha256(hdr)
    with open(os.path.join(CSRC, src), "rb") as f:
        h.update(src.encode() + b"\0" + f.read())
    return h.hexdigest()


def _digest() -> str:
    hdr = _headers_digest()
    h = hashlib.sha256(hdr)
    for s in sorted(SOURCES):
        h.update(_source_digest(s, hdr).encode())
    return h.hexdigest()


def stale() -> bool:
    """Content hash, not mtimes: the repo snapshot on the GPU box does not keep mtimes."""
    if not (os.path.exists(LIB) and os.path.exists(STAMP)):
        return True
    with open(STAMP) as f:
        return f.read().strip() != _digest()


def build(force: bool = False, verbose: bool = False) -> str:
    """One nvcc -c per source, in parallel, each object cached under build/ by the hash of its source, the headers
    and the flags; then one link.  `force` recompiles everything."""
    if not force and not stale():
        return LIB
    from concurrent.futures import ThreadPoolExecutor
    os.makedirs(OBJ_DIR, exist_ok=True)
    hdr = _headers_digest()
    exe = nvcc()

    def compile_one(src: str):
        obj = os.path.join(OBJ_DIR, src.replace(".cu", "") + "." + _source_digest(src, hdr)[:16] + ".o")
        if os.path.exists(obj) and not force:
            return obj, None
        cmd = [exe] + NVCC_FLAGS + (["-Xptxas", "-v"] if verbose else []) + ["-c", "-o", obj, os.path.join(CSRC, src)]
        r = subprocess.run(cmd, capture_output=True, text=True)
        if r.returncode and os.path.exists(obj):
            os.remove(obj)
        return obj, (r, cmd)

    with ThreadPoolExecutor(max_workers=min(len(SOURCES), os.cpu_count() or 4)) as ex:
        results = list(ex.map(compile_one, SOURCES))
    for obj, out in results:
        if out is None:
            continue
        r, cmd = out
        if verbose or r.returncode:
            sys.stderr.write(r.stdout + r.stderr)
        if r.returncode:
            raise RuntimeError("nvcc failed: " + " ".join(cmd))
    keep = {obj for obj, _ in results}
    for f in os.listdir(OBJ_DIR):                                  # drop objects of older source versions
        if f.endswith(".o") and os.path.join(OBJ_DIR, f) not in keep:
            os.remove(os.path.join(OBJ_DIR, f))
    cmd = [exe] + LINK_FLAGS + ["-o", LIB] + [obj for obj, _ in results]
    r = subprocess.run(cmd, capture_output=True, text=True)
    if r.returncode:
        sys.stderr.write(r.stdout + r.stderr)
        raise RuntimeError("nvcc link failed: " + " ".join(cmd))
    with open(STAMP, "w") as f:
        f.write(_digest() + "\n")
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="--verbose" in sys.argv))
