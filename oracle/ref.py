"""ctypes front end of the fp64 CPU oracle (oracle/omnimem_ref.c).

TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only tests/, __graft_entry__.smoke() and bench.py's
cpu_baseline / --impl reference legs may import this module.  It never imports the CUDA package
(paper_2606_07577_b200) and the CUDA package never imports it.

Everything here is argument marshalling: inputs (torch or numpy, bf16/fp32/fp64) are widened exactly
to float64 numpy arrays and handed to the C functions, which follow PAPER.md Eq.1-14 step by step.
`compress_chunk` chains the steps in the paper's order.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
from dataclasses import dataclass

import dataclasses

from typing import Optional

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "omnimem_ref.c")
_SO = os.path.join(_HERE, "libomnimem_ref.so")


def build(force: bool = False) -> str:
    """Compile the oracle with gcc (plain C, OpenMP); returns the path of the shared object.
    OMNIMEM_REF_SANITIZE=1 builds (and loads) a separate AddressSanitizer + UBSan copy instead; the process must then
    run with LD_PRELOAD=$(gcc -print-file-name=libasan.so) (tests/test_oracle_pins.py does, in a subprocess)."""
    if os.environ.get("OMNIMEM_REF_SANITIZE") == "1":
        so = os.path.join(_HERE, "libomnimem_ref_san.so")
        if force or not os.path.exists(so) or os.path.getmtime(so) < os.path.getmtime(_SRC):
            cmd = ["gcc", "-O1", "-g", "-fsanitize=address,undefined", "-fno-sanitize-recover=undefined", "-fno-omit-frame-pointer",
                   "-fopenmp", "-fPIC", "-shared", "-o", so, _SRC, "-lm"]
            subprocess.run(cmd, check=True)
        return so
    # -march=native ties the object to the CPU it was built on, and the built file travels with the tree to other
    # machines: a stamp records source and CPU flags, and anything else triggers a rebuild
    stamp, want = _SO + ".stamp", _machine_stamp()
    have = open(stamp).read() if os.path.exists(stamp) else ""
    if force or not os.path.exists(_SO) or have != want:
        cmd = ["gcc", "-O2", "-march=native", "-fopenmp", "-fPIC", "-shared", "-o", _SO, _SRC, "-lm"]
        subprocess.run(cmd, check=True)
        with open(stamp, "w") as f:
            f.write(want)
    return _SO


def _machine_stamp() -> str:
    import hashlib
    flags = ""
    try:
        with open("/proc/cpuinfo") as f:
            for line in f:
                if line.startswith("flags"):
                    flags = line
                    break
    except OSError:
        pass
    with open(_SRC, "rb") as f:
        return hashlib.sha256(f.read() + flags.encode()).hexdigest()


class _Params(C.Structure):
    _fields_ = [
        ("L", C.c_int32), ("Hq", C.c_int32), ("Hkv", C.c_int32), ("D", C.c_int32),
        ("cache_cap", C.c_int32), ("Nn_v", C.c_int32), ("Nn_a", C.c_int32), ("causal", C.c_int32),
        ("sim_stride_v", C.c_int32), ("sim_stride_a", C.c_int32),
        ("seg_cap_v", C.c_int32), ("seg_cap_a", C.c_int32),
        ("scale", C.c_double), ("lam", C.c_double), ("ratio_r", C.c_double), ("temperature", C.c_double),
        ("budget_min", C.c_int64), ("budget_max", C.c_int64), ("chunk_modality", C.c_void_p),
    ]


@dataclass
class RefParams:
    L: int
    Hq: int
    Hkv: int
    D: int
    cache_cap: int
    Nn_v: int
    Nn_a: int
    causal: int = 1
    sim_stride_v: int = 1
    sim_stride_a: int = 1
    scale: float = 0.0          # 0 => 1/sqrt(D)  (R4)
    lam: float = 0.02
    ratio_r: float = 5.0
    temperature: float = 0.2
    budget_min: int = 0
    budget_max: int = 0
    chunk_modality: Optional[np.ndarray] = None   # [Nn] int32, 0 visual / 1 audio per chunk row (time-interleaved chunk)

    @property
    def Nn(self) -> int:
        return self.Nn_v + self.Nn_a

    @property
    def seg_cap_v(self) -> int:
        return self.cache_cap + self.Nn_v

    @property
    def seg_cap_a(self) -> int:
        return self.cache_cap + self.Nn_a

    def c(self) -> _Params:
        sc = self.scale if self.scale > 0 else 1.0 / float(np.sqrt(np.float64(self.D)))
        mod = None
        if self.chunk_modality is not None:
            self._mod = np.ascontiguousarray(self.chunk_modality, dtype=np.int32)   # kept alive by the dataclass instance
            assert self._mod.shape == (self.Nn,) and int((self._mod == 0).sum()) == self.Nn_v
            mod = self._mod.ctypes.data
        return _Params(self.L, self.Hq, self.Hkv, self.D, self.cache_cap, self.Nn_v, self.Nn_a, self.causal,
                       self.sim_stride_v, self.sim_stride_a, self.seg_cap_v, self.seg_cap_a,
                       sc, self.lam, self.ratio_r, self.temperature, self.budget_min, self.budget_max, mod)


_lib = None


def lib():
    global _lib
    if _lib is None:
        _lib = C.CDLL(build())
    return _lib


def f64(x) -> np.ndarray:
    """Exact widening of a torch / numpy array to a C-contiguous float64 numpy array."""
    if hasattr(x, "detach"):
        import torch
        x = x.detach().cpu().to(torch.float64).numpy()
    return np.ascontiguousarray(x, dtype=np.float64)


def i32(x) -> np.ndarray:
    if hasattr(x, "detach"):
        x = x.detach().cpu().numpy()
    return np.ascontiguousarray(x, dtype=np.int32)


def _p(a: np.ndarray):
    return a.ctypes.data_as(C.c_void_p)


def _check(rc: int, what: str):
    if rc != 0:
        raise RuntimeError(f"oracle {what} failed with status {rc}")


def num_threads() -> int:
    return int(lib().omnimem_ref_num_threads())


# ---- O2 ----------------------------------------------------------------------------------------
def attention(p: RefParams, cacheK, n, chunkK, Q, want_rowH: bool = True):
    """Eq.6 importance in logical key order + per-row LSE (+ row entropy).  Returns (a_log, lse, rowH)."""
    cacheK, chunkK, Q, n = f64(cacheK), f64(chunkK), f64(Q), i32(n)
    assert cacheK.shape == (p.L, p.Hkv, p.cache_cap, p.D), cacheK.shape
    assert chunkK.shape == (p.L, p.Hkv, p.Nn, p.D), chunkK.shape
    assert Q.shape == (p.L, p.Hq, p.Nn, p.D), Q.shape
    a_log = np.zeros((p.L, p.Hkv, p.cache_cap + p.Nn), np.float64)
    lse = np.zeros((p.L, p.Hq, p.Nn), np.float64)
    rowH = np.zeros((p.L, p.Hq, p.Nn), np.float64) if want_rowH else None
    cp = p.c()
    _check(lib().omnimem_ref_attention(C.byref(cp), _p(cacheK), _p(n), _p(chunkK), _p(Q), _p(a_log), _p(lse),
                                       _p(rowH) if want_rowH else None), "attention")
    return a_log, lse, rowH


def mhsa(p: RefParams, cacheK, cacheV, n, chunkK, chunkV, Q, want_abs: bool = False):
    """P:54 Eq.1: the chunk's attention output over [cached visual; cached audio; chunk] and its row LSE.
    Returns (Y [L,Hq,Nn,D], lse [L,Hq,Nn], absY or None)."""
    cacheK, cacheV, chunkK, chunkV, Q, n = f64(cacheK), f64(cacheV), f64(chunkK), f64(chunkV), f64(Q), i32(n)
    assert cacheK.shape == cacheV.shape == (p.L, p.Hkv, p.cache_cap, p.D), cacheK.shape
    assert chunkK.shape == chunkV.shape == (p.L, p.Hkv, p.Nn, p.D), chunkK.shape
    assert Q.shape == (p.L, p.Hq, p.Nn, p.D), Q.shape
    Y = np.zeros((p.L, p.Hq, p.Nn, p.D), np.float64)
    lse = np.zeros((p.L, p.Hq, p.Nn), np.float64)
    absY = np.zeros_like(Y) if want_abs else None
    cp = p.c()
    _check(lib().omnimem_ref_mhsa(C.byref(cp), _p(cacheK), _p(cacheV), _p(n), _p(chunkK), _p(chunkV), _p(Q), _p(Y), _p(lse),
                                  _p(absY) if want_abs else None), "mhsa")
    return Y, lse, absY


def split(p: RefParams, a_log, n_v, n):
    a_log, n_v, n = f64(a_log), i32(n_v), i32(n)
    a_v = np.zeros((p.L, p.Hkv, p.seg_cap_v), np.float64)
    a_a = np.zeros((p.L, p.Hkv, p.seg_cap_a), np.float64)
    cp = p.c()
    _check(lib().omnimem_ref_split(C.byref(cp), _p(a_log), _p(n_v), _p(n), _p(a_v), _p(a_a)), "split")
    return a_v, a_a


# ---- O3 ----------------------------------------------------------------------------------------
def redundancy(p: RefParams, cacheX, n_v, n, chunkX):
    cacheX, chunkX, n_v, n = f64(cacheX), f64(chunkX), i32(n_v), i32(n)
    s_v = np.zeros((p.L, p.Hkv, p.seg_cap_v), np.float64)
    s_a = np.zeros((p.L, p.Hkv, p.seg_cap_a), np.float64)
    cp = p.c()
    _check(lib().omnimem_ref_redundancy(C.byref(cp), _p(cacheX), _p(n_v), _p(n), _p(chunkX), _p(s_v), _p(s_a)),
           "redundancy")
    return s_v, s_a


def redundancy_hidden(p: RefParams, cacheH, n_v, n, chunkH):
    """Eq.7 in the paper's first form: the vectors are the layer's hidden states H_k, one row per token and
    layer (cacheH [L, cache_cap, d_model], chunkH [L, Nn, d_model]; reading R30).  The definition is the same adjacent
    cosine as on value rows, with one "head" of width d_model, so the same plain routine is called on that shape; the
    result [L, seg_cap_m] is the redundancy of the token in every KV head."""
    p1 = dataclasses.replace(p, Hq=1, Hkv=1, D=int(cacheH.shape[-1]))
    s_v, s_a = redundancy(p1, cacheH[:, None], n_v, n, chunkH[:, None])
    return np.repeat(s_v, p.Hkv, axis=1), np.repeat(s_a, p.Hkv, axis=1)


def compact_hidden(p: RefParams, cacheH, chunkH, n_v, n, idx_v, idx_a, M_v, M_a):
    """The retained hidden states follow the kept tokens; the layer's index set is head 0's (select_scope = 1)."""
    p1 = dataclasses.replace(p, Hq=1, Hkv=1, D=int(cacheH.shape[-1]))
    dst, _, _ = compact(p1, cacheH[:, None], chunkH[:, None], n_v, n, i32(idx_v)[:, :1], i32(idx_a)[:, :1], M_v, M_a)
    return dst[:, 0]


# ---- O4 ----------------------------------------------------------------------------------------
def psi(p: RefParams, n_v, n, a_v, a_a, s_v, s_a, select_scope: int = 0):
    """select_scope 0: Eq.8 per (layer, KV head); 1: once per layer, paper-literal index sets (R29)."""
    n_v, n = i32(n_v), i32(n)
    a_v, a_a, s_v, s_a = f64(a_v), f64(a_a), f64(s_v), f64(s_a)
    psi_v = np.zeros((p.L, p.Hkv, p.seg_cap_v), np.float32)
    psi_a = np.zeros((p.L, p.Hkv, p.seg_cap_a), np.float32)
    cp = p.c()
    fn = lib().omnimem_ref_psi_shared if select_scope == 1 else lib().omnimem_ref_psi
    _check(fn(C.byref(cp), _p(n_v), _p(n), _p(a_v), _p(a_a), _p(s_v), _p(s_a), _p(psi_v), _p(psi_a)), "psi")
    return psi_v, psi_a


# ---- O5 ----------------------------------------------------------------------------------------
STAT_NAMES = ("Hn_v", "Hn_a", "sbar_v", "sbar_a", "C_v", "C_a", "Hn_all", "sbar_all")


def stats(p: RefParams, n_v, n, a_v, a_a, s_v, s_a):
    n_v, n = i32(n_v), i32(n)
    a_v, a_a, s_v, s_a = f64(a_v), f64(a_a), f64(s_v), f64(s_a)
    st = np.zeros((p.L, 8), np.float64)
    cp = p.c()
    _check(lib().omnimem_ref_stats(C.byref(cp), _p(n_v), _p(n), _p(a_v), _p(a_a), _p(s_v), _p(s_a), _p(st)), "stats")
    return st


# ---- O6 ----------------------------------------------------------------------------------------
def layer_budgets(p: RefParams, st, total: int):
    st = f64(st)
    out = np.zeros((p.L,), np.int32)
    cp = p.c()
    _check(lib().omnimem_ref_layer_budgets(C.byref(cp), _p(st), C.c_int64(int(total)), _p(out)), "layer_budgets")
    return out


def calibrate_budgets(p: RefParams, stats_per_chunk, total: int):
    """Offline per-layer totals ("determined offline ... based on a small calibration set", reading R28):
    arithmetic mean over the calibration chunks of each layer's statistics, then Eq.13-14 on the means
    (C^(l) = mean Hn_all * (1 - mean sbar_all)).  stats_per_chunk: [n_chunks, L, 8].  Returns (B [L] int32, mean [L,8])."""
    st = np.asarray(stats_per_chunk, np.float64)
    mean = st.sum(axis=0) / st.shape[0]
    return layer_budgets(p, mean, total), mean


def allocate(p: RefParams, st, n_v, n, layer_budget):
    st, n_v, n, layer_budget = f64(st), i32(n_v), i32(n), i32(layer_budget)
    M_v = np.zeros((p.L,), np.int32)
    M_a = np.zeros((p.L,), np.int32)
    cp = p.c()
    _check(lib().omnimem_ref_allocate(C.byref(cp), _p(st), _p(n_v), _p(n), _p(layer_budget), _p(M_v), _p(M_a)),
           "allocate")
    return M_v, M_a


# ---- O7 ----------------------------------------------------------------------------------------
def select(p: RefParams, psi_v, psi_a, n_v, n, M_v, M_a):
    """Returns idx_v, idx_a int32 [L,Hkv,cache_cap], ascending segment-local indices, -1 padded."""
    psi_v = np.ascontiguousarray(psi_v, dtype=np.float32)
    psi_a = np.ascontiguousarray(psi_a, dtype=np.float32)
    n_v, n, M_v, M_a = i32(n_v), i32(n), i32(M_v), i32(M_a)
    idx_v = np.full((p.L, p.Hkv, p.cache_cap), -1, np.int32)
    idx_a = np.full((p.L, p.Hkv, p.cache_cap), -1, np.int32)
    cp = p.c()
    _check(lib().omnimem_ref_select(C.byref(cp), _p(psi_v), _p(psi_a), _p(n_v), _p(n), _p(M_v), _p(M_a), _p(idx_v),
                                    _p(idx_a), C.c_int32(p.cache_cap)), "select")
    return idx_v, idx_a


# ---- O8 ----------------------------------------------------------------------------------------
def _raw(x) -> np.ndarray:
    """Raw bytes of a tensor/array, shape [..., D*elem_size] uint8 (bf16 has no numpy dtype)."""
    if hasattr(x, "detach"):
        import torch
        x = x.detach().cpu().contiguous()
        return x.view(torch.uint8).numpy()
    x = np.ascontiguousarray(x)
    return x.view(np.uint8)


def compact(p: RefParams, cacheX, chunkX, n_v, n, idx_v, idx_a, M_v, M_a):
    """Byte-exact prune of one tensor (K or V).  Returns (dst raw uint8 [L,Hkv,cap,row_bytes], n_v', n')."""
    src, chk = _raw(cacheX), _raw(chunkX)
    row_bytes = src.shape[-1]
    assert src.shape[:3] == (p.L, p.Hkv, p.cache_cap) and chk.shape[:3] == (p.L, p.Hkv, p.Nn)
    n_v, n, M_v, M_a, idx_v, idx_a = i32(n_v), i32(n), i32(M_v), i32(M_a), i32(idx_v), i32(idx_a)
    dst = np.zeros_like(src)
    n_v_out = np.zeros((p.L,), np.int32)
    n_out = np.zeros((p.L,), np.int32)
    cp = p.c()
    _check(lib().omnimem_ref_compact(C.byref(cp), C.c_int64(row_bytes), _p(src), _p(chk), _p(n_v), _p(n), _p(idx_v),
                                     _p(idx_a), C.c_int32(idx_v.shape[-1]), _p(M_v), _p(M_a), _p(dst), _p(n_v_out),
                                     _p(n_out)), "compact")
    return dst, n_v_out, n_out


# ---- the whole step, in the paper's order ------------------------------------------------------------
def score(p: RefParams, cacheK, cacheV, n_v, n, chunkK, chunkV, Q, sim_source: int = 0, want_rowH: bool = False,
          select_scope: int = 0, hidden=None):
    """Stages 1-3a: a, s, psi, statistics (Eq.6-10, 13).  Returns a dict of numpy arrays."""
    a_log, lse, rowH = attention(p, cacheK, n, chunkK, Q, want_rowH)
    a_v, a_a = split(p, a_log, n_v, n)
    if sim_source == 0:
        s_v, s_a = redundancy(p, cacheV, n_v, n, chunkV)
    elif sim_source == 1:
        s_v, s_a = redundancy(p, cacheK, n_v, n, chunkK)
    else:
        s_v, s_a = redundancy_hidden(p, hidden[0], n_v, n, hidden[1])
    psi_v, psi_a = psi(p, n_v, n, a_v, a_a, s_v, s_a, select_scope)
    st = stats(p, n_v, n, a_v, a_a, s_v, s_a)
    return dict(a_log=a_log, lse=lse, rowH=rowH, a_v=a_v, a_a=a_a, s_v=s_v, s_a=s_a, psi_v=psi_v, psi_a=psi_a,
                stats=st)


def compress_chunk(p: RefParams, cacheK, cacheV, n_v, n, chunkK, chunkV, Q, layer_budget, sim_source: int = 0,
                   want_rowH: bool = False, select_scope: int = 0, hidden=None):
    """One full step: score -> allocate -> select -> compact.  `layer_budget` is an int array [L].
    hidden = (cacheH, chunkH) when sim_source == 2 (hidden-state redundancy, R30)."""
    out = score(p, cacheK, cacheV, n_v, n, chunkK, chunkV, Q, sim_source, want_rowH, select_scope, hidden)
    M_v, M_a = allocate(p, out["stats"], n_v, n, layer_budget)
    idx_v, idx_a = select(p, out["psi_v"], out["psi_a"], n_v, n, M_v, M_a)
    dstK, n_v2, n2 = compact(p, cacheK, chunkK, n_v, n, idx_v, idx_a, M_v, M_a)
    dstV, _, _ = compact(p, cacheV, chunkV, n_v, n, idx_v, idx_a, M_v, M_a)
    out.update(M_v=M_v, M_a=M_a, idx_v=idx_v, idx_a=idx_a, dstK=dstK, dstV=dstV, n_v_out=n_v2, n_out=n2)
    if hidden is not None:
        out["dstH"] = compact_hidden(p, hidden[0], hidden[1], n_v, n, idx_v, idx_a, M_v, M_a)
    return out
