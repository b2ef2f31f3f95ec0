"""Builds libomnimem.so (the C-ABI library of include/omnimem.h) in-tree with nvcc for sm_100a.

The compile flags are fixed here: no environment variable can change what the shipped library computes.  Staleness is
decided by content, not by time stamps: build/stamp.json records the SHA-256 of every source, header and of the linked
library together with the flags; anything that does not match (edited source, different flags, a library that some other
tool linked) triggers a rebuild.
"""
from __future__ import annotations

import hashlib
import json
import os
import subprocess
import sys
from concurrent.futures import ThreadPoolExecutor

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libomnimem.so")
OBJDIR = os.path.join(HERE, "build")
STAMP = os.path.join(OBJDIR, "stamp.json")
SOURCES = ["api.cu", "score_simt.cu", "score_tc.cu", "attend_tc.cu", "stages.cu", "redundancy_static.cu"]
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17", "-Xcompiler", "-fPIC",
              "-Xcompiler", "-fvisibility=hidden", "--expt-relaxed-constexpr"]
LINK_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-Xcompiler", "-fvisibility=hidden"]


def _sha(path: str) -> str:
    h = hashlib.sha256()
    with open(path, "rb") as f:
        for blk in iter(lambda: f.read(1 << 20), b""):
            h.update(blk)
    return h.hexdigest()


def _headers():
    hs = [os.path.join(CSRC, f) for f in sorted(os.listdir(CSRC)) if f.endswith((".cuh", ".h"))]
    hs.append(os.path.join(os.path.dirname(HERE), "include", "omnimem.h"))
    return hs


def _want_stamp() -> dict:
    srcs = [os.path.join(CSRC, s) for s in SOURCES]
    missing = [p for p in srcs if not os.path.exists(p)]
    if missing:   # a dropped entry would only show up later as an unresolved symbol at link or load time
        raise FileNotFoundError("sources listed in build.SOURCES are missing: " + ", ".join(missing))
    return {"flags": NVCC_FLAGS + LINK_FLAGS, "sources": {os.path.basename(p): _sha(p) for p in srcs},
            "headers": {os.path.basename(p): _sha(p) for p in _headers()}}


def build(force: bool = False, verbose: bool = False) -> str:
    nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
    os.makedirs(OBJDIR, exist_ok=True)
    want = _want_stamp()
    have = {}
    if os.path.exists(STAMP):
        try:
            have = json.load(open(STAMP))
        except Exception:
            have = {}
    objs = [os.path.join(OBJDIR, s.replace(".cu", ".o")) for s in want["sources"]]
    lib_ok = os.path.exists(LIB) and have.get("lib") == _sha(LIB)
    same_env = have.get("flags") == want["flags"] and have.get("headers") == want["headers"]
    jobs = []
    for src, o in zip(want["sources"], objs):
        fresh = same_env and os.path.exists(o) and have.get("sources", {}).get(src) == want["sources"][src] and \
            have.get("objects", {}).get(src) == _sha(o)
        if force or not fresh:
            jobs.append([nvcc] + NVCC_FLAGS + (["-Xptxas", "-v"] if verbose else []) + ["-c", os.path.join(CSRC, src), "-o", o])
    with ThreadPoolExecutor(max_workers=4) as ex:
        for r in ex.map(lambda c: subprocess.run(c, capture_output=True, text=True), jobs):
            if verbose or r.returncode:
                sys.stderr.write(r.stdout + r.stderr)
            if r.returncode:
                raise RuntimeError("nvcc failed: " + " ".join(r.args))
    if force or jobs or not lib_ok:
        r = subprocess.run([nvcc, "-shared", "-o", LIB] + objs + LINK_FLAGS, capture_output=True, text=True)
        if r.returncode:
            sys.stderr.write(r.stdout + r.stderr)
            raise RuntimeError("link failed")
        want["objects"] = {s: _sha(o) for s, o in zip(want["sources"], objs)}
        want["lib"] = _sha(LIB)
        json.dump(want, open(STAMP, "w"), indent=1)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
