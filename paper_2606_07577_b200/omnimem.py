"""Thin ctypes binding of the C-ABI library declared in include/omnimem.h.

Argument marshalling only: every step of the path runs in the CUDA kernels of libomnimem.so.  PyTorch provides
device memory and streams.  There is NO fallback: if libomnimem.so is missing or the device is not sm_100 the
calls raise.  This module never imports anything under oracle/.
"""
from __future__ import annotations

import ctypes as C
import os
from dataclasses import dataclass
from typing import Optional

import torch

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libomnimem.so")

OMNIMEM_FP32, OMNIMEM_BF16 = 0, 1
STAGES = ("lse", "colsum", "cosine", "finalize", "allocate", "select", "compact", "attend")
STAT_NAMES = ("Hn_v", "Hn_a", "sbar_v", "sbar_a", "C_v", "C_a", "Hn_all", "sbar_all")
EXPORTS = ("omnimem_create", "omnimem_destroy", "omnimem_workspace_bytes", "omnimem_seg_cap", "omnimem_strerror",
           "omnimem_last_cuda_error", "omnimem_score", "omnimem_allocate", "omnimem_select", "omnimem_compact",
           "omnimem_compress_chunk", "omnimem_compress_chunk_host", "omnimem_set_profiling", "omnimem_get_stage_ms",
           "omnimem_calibrate_accumulate", "omnimem_calibrate_budgets", "omnimem_attend", "omnimem_redundancy_static")
STATIC_SCRATCH_FLOATS = 1 << 20      # OMNIMEM_STATIC_SCRATCH_FLOATS of include/omnimem.h


class OmniMemError(RuntimeError):
    pass


class omnimem_config(C.Structure):
    _fields_ = [("n_layers", C.c_int32), ("n_q_heads", C.c_int32), ("n_kv_heads", C.c_int32), ("head_dim", C.c_int32),
                ("dtype", C.c_int32), ("cache_cap", C.c_int32), ("max_chunk_v", C.c_int32), ("max_chunk_a", C.c_int32),
                ("softmax_scale", C.c_float), ("lam", C.c_float), ("ratio_r", C.c_float), ("temperature", C.c_float),
                ("budget_min", C.c_int32), ("budget_max", C.c_int32), ("causal", C.c_int32), ("sim_source", C.c_int32),
                ("sim_stride_v", C.c_int32), ("sim_stride_a", C.c_int32), ("score_path", C.c_int32),
                ("select_scope", C.c_int32), ("d_model", C.c_int32), ("score_ctas", C.c_int32)]


class omnimem_cache(C.Structure):
    _fields_ = [("k", C.c_void_p), ("v", C.c_void_p), ("n_v", C.c_void_p), ("n", C.c_void_p), ("h", C.c_void_p)]


class omnimem_chunk(C.Structure):
    _fields_ = [("k", C.c_void_p), ("v", C.c_void_p), ("q", C.c_void_p), ("lse", C.c_void_p),
                ("Nn_v", C.c_int32), ("Nn_a", C.c_int32), ("h", C.c_void_p), ("modality", C.c_void_p)]


class omnimem_scores(C.Structure):
    _fields_ = [("a_v", C.c_void_p), ("a_a", C.c_void_p), ("s_v", C.c_void_p), ("s_a", C.c_void_p),
                ("psi_v", C.c_void_p), ("psi_a", C.c_void_p), ("lse_out", C.c_void_p), ("row_entropy", C.c_void_p),
                ("stats", C.c_void_p)]


_lib = None


def load_library() -> C.CDLL:
    """dlopen libomnimem.so (built in-tree by paper_2606_07577_b200/build.py).  Raises if it is missing."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise OmniMemError(f"{LIB_PATH} is missing: run `python -m paper_2606_07577_b200.build` "
                               "(there is no CPU fallback)")
        lib = C.CDLL(LIB_PATH)
        vp, i32, i64 = C.c_void_p, C.c_int32, C.c_int64
        lib.omnimem_create.argtypes = [C.POINTER(omnimem_config), C.POINTER(vp)]
        lib.omnimem_destroy.argtypes = [vp]
        lib.omnimem_workspace_bytes.argtypes = [vp]
        lib.omnimem_workspace_bytes.restype = C.c_size_t
        lib.omnimem_seg_cap.argtypes = [vp, i32]
        lib.omnimem_seg_cap.restype = i32
        lib.omnimem_strerror.argtypes = [C.c_int]
        lib.omnimem_strerror.restype = C.c_char_p
        lib.omnimem_last_cuda_error.argtypes = [vp]
        lib.omnimem_last_cuda_error.restype = C.c_char_p
        lib.omnimem_score.argtypes = [vp, C.POINTER(omnimem_cache), C.POINTER(omnimem_chunk), C.POINTER(omnimem_scores),
                                      vp, C.c_size_t, vp]
        lib.omnimem_attend.argtypes = [vp, C.POINTER(omnimem_cache), C.POINTER(omnimem_chunk), vp, vp, vp, C.c_size_t, vp]
        lib.omnimem_allocate.argtypes = [vp, vp, vp, vp, i32, i32, vp, i64, vp, vp, vp, vp]
        lib.omnimem_calibrate_accumulate.argtypes = [vp, vp, vp, vp]
        lib.omnimem_calibrate_budgets.argtypes = [vp, vp, i64, vp, vp, vp]
        lib.omnimem_select.argtypes = [vp, vp, vp, vp, vp, i32, i32, vp, vp, vp, vp, vp, C.c_size_t, vp]
        lib.omnimem_compact.argtypes = [vp, C.POINTER(omnimem_cache), C.POINTER(omnimem_chunk), vp, vp, vp, vp,
                                        C.POINTER(omnimem_cache), vp]
        lib.omnimem_compress_chunk.argtypes = [vp, C.POINTER(omnimem_cache), C.POINTER(omnimem_chunk), vp,
                                               C.POINTER(omnimem_cache), C.POINTER(omnimem_scores), vp, vp, vp, vp, vp,
                                               C.c_size_t, vp]
        lib.omnimem_compress_chunk_host.argtypes = [vp, C.POINTER(omnimem_cache), C.POINTER(omnimem_chunk),
                                                    C.POINTER(omnimem_chunk), vp, C.POINTER(omnimem_cache), vp, vp,
                                                    C.POINTER(i64), C.POINTER(i64), vp, C.c_size_t, vp]
        lib.omnimem_set_profiling.argtypes = [vp, i32]
        lib.omnimem_get_stage_ms.argtypes = [vp, C.POINTER(C.c_float), C.POINTER(i32)]
        lib.omnimem_redundancy_static.argtypes = [i32] * 9 + [vp, vp, vp, vp, i32, i32, vp, vp, vp]
        _lib = lib
    return _lib


def _ptr(t: Optional[torch.Tensor]):
    return None if t is None else C.c_void_p(t.data_ptr())


def _stream() -> C.c_void_p:
    return C.c_void_p(torch.cuda.current_stream().cuda_stream)


def redundancy_static(cache_x: torch.Tensor, n_v: torch.Tensor, n: torch.Tensor, chunk_x: Optional[torch.Tensor],
                      Nn_v: int, Nn_a: int, max_chunk_v: int, max_chunk_a: int, s_v: torch.Tensor, s_a: torch.Tensor,
                      sim_stride_v: int = 1, sim_stride_a: int = 1) -> None:
    """omnimem_redundancy_static: the Eq.7 redundancy s_v, s_a for callers that must not allocate device memory (a
    serving engine whose pool already owns all of HBM, an operator body that is handed its tensors and nothing else).
    No context and no workspace: the C call's intermediates live in a 4 MiB array inside the library, which is why
    L * Hkv * (2 * cache_cap + max_chunk_v + max_chunk_a) may not exceed STATIC_SCRATCH_FLOATS and why calls that can
    overlap on the GPU must be serialised by the caller.  This wrapper allocates nothing either: cache_x
    [L,Hkv,cache_cap,D], chunk_x [L,Hkv,Nn,D] (None when Nn = 0) and the outputs s_m float32 [L,Hkv,cache_cap+max_chunk_m]
    all come from the caller; work goes to torch's current stream of cache_x's device."""
    lib = load_library()
    L, Hkv, cache_cap, D = cache_x.shape
    dtype = OMNIMEM_FP32 if cache_x.dtype == torch.float32 else OMNIMEM_BF16
    with torch.cuda.device(cache_x.device):
        rc = lib.omnimem_redundancy_static(dtype, L, Hkv, D, cache_cap, max_chunk_v, max_chunk_a, sim_stride_v,
                                           sim_stride_a, _ptr(cache_x), _ptr(n_v), _ptr(n), _ptr(chunk_x), Nn_v, Nn_a,
                                           _ptr(s_v), _ptr(s_a), _stream())
    if rc != 0:
        raise OmniMemError(f"omnimem_redundancy_static failed ({rc}): {lib.omnimem_strerror(rc).decode()}")


@dataclass
class Cache:
    """One pooled KV cache on the device: k, v [L,Hkv,cache_cap,D]; n_v, n int32 [L]."""
    k: torch.Tensor
    v: torch.Tensor
    n_v: torch.Tensor
    n: torch.Tensor
    h: Optional[torch.Tensor] = None     # [L, cache_cap, d_model] retained hidden states (sim_source == 2)

    def c(self) -> omnimem_cache:
        return omnimem_cache(self.k.data_ptr(), self.v.data_ptr(), self.n_v.data_ptr(), self.n.data_ptr(),
                             None if self.h is None else self.h.data_ptr())


@dataclass
class Chunk:
    """One chunk: k, v [L,Hkv,Nn,D], q [L,Hq,Nn,D] (device, or pinned host for compress_chunk_host)."""
    k: torch.Tensor
    v: torch.Tensor
    q: torch.Tensor
    Nn_v: int
    Nn_a: int
    lse: Optional[torch.Tensor] = None
    h: Optional[torch.Tensor] = None     # [L, Nn, d_model] hidden states of the chunk's tokens (sim_source == 2)
    modality: Optional[torch.Tensor] = None   # int32 [Nn], 0 visual / 1 audio per row: time-interleaved chunk (R25')

    def c(self) -> omnimem_chunk:
        return omnimem_chunk(self.k.data_ptr(), self.v.data_ptr(), self.q.data_ptr(),
                             None if self.lse is None else self.lse.data_ptr(), self.Nn_v, self.Nn_a,
                             None if self.h is None else self.h.data_ptr(),
                             None if self.modality is None else self.modality.data_ptr())


@dataclass
class Scores:
    a_v: torch.Tensor
    a_a: torch.Tensor
    s_v: torch.Tensor
    s_a: torch.Tensor
    psi_v: torch.Tensor
    psi_a: torch.Tensor
    stats: torch.Tensor
    lse: Optional[torch.Tensor] = None
    row_entropy: Optional[torch.Tensor] = None

    def c(self) -> omnimem_scores:
        return omnimem_scores(self.a_v.data_ptr(), self.a_a.data_ptr(), self.s_v.data_ptr(), self.s_a.data_ptr(),
                              self.psi_v.data_ptr(), self.psi_a.data_ptr(),
                              None if self.lse is None else self.lse.data_ptr(),
                              None if self.row_entropy is None else self.row_entropy.data_ptr(), self.stats.data_ptr())


class OmniMem:
    """A context of the C library plus its workspace.  Method names mirror the C entry points."""

    def __init__(self, L: int, Hq: int, Hkv: int, D: int, dtype: str, cache_cap: int, max_chunk_v: int, max_chunk_a: int,
                 lam: float = 0.02, ratio_r: float = 5.0, temperature: float = 0.2, softmax_scale: float = 0.0,
                 budget_min: int = 0, budget_max: int = 0, causal: int = 1, sim_source: int = 0, sim_stride_v: int = 1,
                 sim_stride_a: int = 1, score_path: int = 0, select_scope: int = 0, d_model: int = 0, score_ctas: int = 0,
                 device: str = "cuda:0"):
        self.lib = load_library()
        if not torch.cuda.is_available():
            raise OmniMemError("no CUDA device: the OmniMem path has no CPU fallback")
        self.device = torch.device(device)
        self.L, self.Hq, self.Hkv, self.D = L, Hq, Hkv, D
        self.cache_cap, self.max_chunk_v, self.max_chunk_a = cache_cap, max_chunk_v, max_chunk_a
        self.d_model, self.sim_source = d_model, sim_source
        self.torch_dtype = torch.float32 if dtype == "fp32" else torch.bfloat16
        self.cfg = omnimem_config(L, Hq, Hkv, D, OMNIMEM_FP32 if dtype == "fp32" else OMNIMEM_BF16, cache_cap, max_chunk_v,
                                  max_chunk_a, softmax_scale, lam, ratio_r, temperature, budget_min, budget_max, causal,
                                  sim_source, sim_stride_v, sim_stride_a, score_path, select_scope, d_model, score_ctas)
        self.ctx = C.c_void_p()
        with torch.cuda.device(self.device):
            self._check(self.lib.omnimem_create(C.byref(self.cfg), C.byref(self.ctx)), "omnimem_create")
        self.seg_cap_v = int(self.lib.omnimem_seg_cap(self.ctx, 0))
        self.seg_cap_a = int(self.lib.omnimem_seg_cap(self.ctx, 1))
        self.ws_bytes = int(self.lib.omnimem_workspace_bytes(self.ctx))
        self.ws = torch.empty(self.ws_bytes, dtype=torch.uint8, device=self.device)

    @classmethod
    def for_workload(cls, wl, **kw) -> "OmniMem":
        args = dict(L=wl.L, Hq=wl.Hq, Hkv=wl.Hkv, D=wl.D, dtype=wl.dtype, cache_cap=wl.cache_cap, max_chunk_v=wl.Nn_v,
                    max_chunk_a=wl.Nn_a, sim_stride_v=wl.sim_stride_v, sim_stride_a=wl.sim_stride_a)
        args.update(kw)
        return cls(**args)

    def close(self):
        if getattr(self, "ctx", None) is not None and self.ctx.value:
            self.lib.omnimem_destroy(self.ctx)
            self.ctx = C.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def _check(self, rc: int, what: str):
        if rc != 0:
            msg = self.lib.omnimem_strerror(rc).decode()
            if rc == -4 and self.ctx.value:
                msg += ": " + self.lib.omnimem_last_cuda_error(self.ctx).decode()
            raise OmniMemError(f"{what} failed ({rc}): {msg}")

    # ---- allocation helpers (device memory comes from torch) --------------------------------------------------
    def new_cache(self) -> Cache:
        z = lambda *s, dt: torch.zeros(*s, dtype=dt, device=self.device)
        return Cache(z(self.L, self.Hkv, self.cache_cap, self.D, dt=self.torch_dtype),
                     z(self.L, self.Hkv, self.cache_cap, self.D, dt=self.torch_dtype),
                     z(self.L, dt=torch.int32), z(self.L, dt=torch.int32),
                     z(self.L, self.cache_cap, self.d_model, dt=self.torch_dtype) if self.sim_source == 2 else None)

    def new_scores(self, Nn: int, want_lse: bool = False, want_row_entropy: bool = False) -> Scores:
        f = lambda *s: torch.zeros(*s, dtype=torch.float32, device=self.device)
        return Scores(f(self.L, self.Hkv, self.seg_cap_v), f(self.L, self.Hkv, self.seg_cap_a),
                      f(self.L, self.Hkv, self.seg_cap_v), f(self.L, self.Hkv, self.seg_cap_a),
                      f(self.L, self.Hkv, self.seg_cap_v), f(self.L, self.Hkv, self.seg_cap_a),
                      torch.zeros(self.L, 8, dtype=torch.float64, device=self.device),
                      f(self.L, self.Hq, Nn) if want_lse else None, f(self.L, self.Hq, Nn) if want_row_entropy else None)

    def new_indices(self):
        mk = lambda: torch.full((self.L, self.Hkv, self.cache_cap), -1, dtype=torch.int32, device=self.device)
        return mk(), mk()

    # ---- the C entry points ------------------------------------------------------------------------------------------
    def score(self, src: Cache, chunk: Chunk, out: Optional[Scores] = None, want_lse: bool = False,
              want_row_entropy: bool = False) -> Scores:
        out = out or self.new_scores(chunk.Nn_v + chunk.Nn_a, want_lse, want_row_entropy)
        cs, cc, co = src.c(), chunk.c(), out.c()
        self._check(self.lib.omnimem_score(self.ctx, C.byref(cs), C.byref(cc), C.byref(co), _ptr(self.ws), self.ws_bytes,
                                           _stream()), "omnimem_score")
        return out

    def attend(self, src: Cache, chunk: Chunk, y: Optional[torch.Tensor] = None, lse: Optional[torch.Tensor] = None):
        """P:54 Eq.1: the chunk's attention output y [L,Hq,Nn,D] (context dtype) and its row LSE [L,Hq,Nn] (fp32, natural
        log: the array Chunk.lse takes)."""
        Nn = chunk.Nn_v + chunk.Nn_a
        if y is None:
            y = torch.empty(self.L, self.Hq, Nn, self.D, dtype=self.torch_dtype, device=self.device)
        if lse is None:
            lse = torch.empty(self.L, self.Hq, Nn, dtype=torch.float32, device=self.device)
        cs, cc = src.c(), chunk.c()
        self._check(self.lib.omnimem_attend(self.ctx, C.byref(cs), C.byref(cc), _ptr(y), _ptr(lse), _ptr(self.ws), self.ws_bytes,
                                            _stream()), "omnimem_attend")
        return y, lse

    def allocate(self, stats: torch.Tensor, n_v: torch.Tensor, n: torch.Tensor, Nn_v: int, Nn_a: int,
                 layer_budget: Optional[torch.Tensor] = None, total_budget: int = 0):
        M_v = torch.zeros(self.L, dtype=torch.int32, device=self.device)
        M_a = torch.zeros_like(M_v)
        B_out = torch.zeros_like(M_v)
        self._check(self.lib.omnimem_allocate(self.ctx, _ptr(stats), _ptr(n_v), _ptr(n), Nn_v, Nn_a, _ptr(layer_budget),
                                              int(total_budget), _ptr(M_v), _ptr(M_a), _ptr(B_out), _stream()),
                    "omnimem_allocate")
        return M_v, M_a, B_out

    def new_calibration(self) -> torch.Tensor:
        """Zeroed accumulator of omnimem_calibrate_accumulate: [(L+1)*8] doubles on the device."""
        return torch.zeros((self.L + 1) * 8, dtype=torch.float64, device=self.device)

    def calibrate_accumulate(self, stats: torch.Tensor, acc: torch.Tensor) -> torch.Tensor:
        self._check(self.lib.omnimem_calibrate_accumulate(self.ctx, _ptr(stats), _ptr(acc), _stream()),
                    "omnimem_calibrate_accumulate")
        return acc

    def calibrate_budgets(self, acc: torch.Tensor, total_budget: int):
        mean_stats = torch.zeros(self.L, 8, dtype=torch.float64, device=self.device)
        B = torch.zeros(self.L, dtype=torch.int32, device=self.device)
        self._check(self.lib.omnimem_calibrate_budgets(self.ctx, _ptr(acc), int(total_budget), _ptr(mean_stats), _ptr(B),
                                                       _stream()), "omnimem_calibrate_budgets")
        return B, mean_stats

    def select(self, psi_v: torch.Tensor, psi_a: torch.Tensor, n_v: torch.Tensor, n: torch.Tensor, Nn_v: int, Nn_a: int,
               M_v: torch.Tensor, M_a: torch.Tensor, idx_v: Optional[torch.Tensor] = None,
               idx_a: Optional[torch.Tensor] = None):
        if idx_v is None or idx_a is None:
            idx_v, idx_a = self.new_indices()
        self._check(self.lib.omnimem_select(self.ctx, _ptr(psi_v), _ptr(psi_a), _ptr(n_v), _ptr(n), Nn_v, Nn_a, _ptr(M_v),
                                            _ptr(M_a), _ptr(idx_v), _ptr(idx_a), _ptr(self.ws), self.ws_bytes, _stream()),
                    "omnimem_select")
        return idx_v, idx_a

    def compact(self, src: Cache, chunk: Chunk, idx_v: torch.Tensor, idx_a: torch.Tensor, M_v: torch.Tensor,
                M_a: torch.Tensor, dst: Cache) -> Cache:
        cs, cc, cd = src.c(), chunk.c(), dst.c()
        self._check(self.lib.omnimem_compact(self.ctx, C.byref(cs), C.byref(cc), _ptr(idx_v), _ptr(idx_a), _ptr(M_v),
                                             _ptr(M_a), C.byref(cd), _stream()), "omnimem_compact")
        return dst

    def compress_chunk(self, src: Cache, chunk: Chunk, layer_budget: torch.Tensor, dst: Cache,
                       out: Optional[Scores] = None, idx_v: Optional[torch.Tensor] = None,
                       idx_a: Optional[torch.Tensor] = None, M_v: Optional[torch.Tensor] = None,
                       M_a: Optional[torch.Tensor] = None) -> Cache:
        cs, cc, cd = src.c(), chunk.c(), dst.c()
        co = out.c() if out is not None else None
        self._check(self.lib.omnimem_compress_chunk(self.ctx, C.byref(cs), C.byref(cc), _ptr(layer_budget), C.byref(cd),
                                                    C.byref(co) if co is not None else None, _ptr(idx_v), _ptr(idx_a),
                                                    _ptr(M_v), _ptr(M_a), _ptr(self.ws), self.ws_bytes, _stream()),
                    "omnimem_compress_chunk")
        return dst

    def compress_chunk_host(self, src: Cache, host_chunk: Chunk, dev_chunk: Chunk, layer_budget: torch.Tensor, dst: Cache,
                            host_M_v: torch.Tensor, host_M_a: torch.Tensor):
        """End-to-end entry: chunk in (pinned) HOST memory -> device -> fused step -> budgets back on the host."""
        cs, ch, cdv, cd = src.c(), host_chunk.c(), dev_chunk.c(), dst.c()
        h2d, d2h = C.c_int64(0), C.c_int64(0)
        self._check(self.lib.omnimem_compress_chunk_host(self.ctx, C.byref(cs), C.byref(ch), C.byref(cdv), _ptr(layer_budget),
                                                         C.byref(cd), _ptr(host_M_v), _ptr(host_M_a), C.byref(h2d),
                                                         C.byref(d2h), _ptr(self.ws), self.ws_bytes, _stream()),
                    "omnimem_compress_chunk_host")
        return int(h2d.value), int(d2h.value)

    def set_profiling(self, enabled: bool):
        self._check(self.lib.omnimem_set_profiling(self.ctx, int(enabled)), "omnimem_set_profiling")

    def stage_ms(self):
        """Per-stage milliseconds and kernel-launch count of the most recent call (profiling must be enabled)."""
        out = (C.c_float * len(STAGES))()
        launches = C.c_int32(0)
        self._check(self.lib.omnimem_get_stage_ms(self.ctx, out, C.byref(launches)), "omnimem_get_stage_ms")
        return {s: float(out[i]) for i, s in enumerate(STAGES)}, int(launches.value)
