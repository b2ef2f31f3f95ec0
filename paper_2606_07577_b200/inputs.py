"""Seeded synthetic inputs for the OmniMem compression step (shared by the CUDA path and the oracle).

This module holds NONE of the method's arithmetic: it only draws K/V/Q tensors with the shapes, sizes
and value structure of BASELINE.json's five configs (the recipe table is in DESIGN.md section "Inputs").
The paper measures on VideoMME-long / LVBench / LV-Omni-Bench / StreamingBench streams through
video-SALMONN 2+ and Qwen2.5-Omni; neither the videos nor the weights exist here,
so these tensors stand in for them.

All randomness comes from CPU `torch.Generator`s seeded from (config, step, layer): the same bytes on
every machine.  Values are drawn in fp32, transformed, and cast ONCE to the config dtype; that tensor
is the single source for both sides.
"""
from __future__ import annotations

import dataclasses
import math
import os
from concurrent.futures import ThreadPoolExecutor
from dataclasses import dataclass

import torch


@dataclass(frozen=True)
class Workload:
    name: str
    S: int                  # config number - 1 (seed base)
    L: int
    Hq: int
    Hkv: int
    D: int
    dtype: str              # "fp32" | "bf16"
    n_v: int                # cached visual rows at step 0
    n_a: int                # cached audio rows at step 0
    Nn_v: int               # chunk visual rows
    Nn_a: int               # chunk audio rows
    budget: int             # per-layer budget B
    cache_cap: int          # rows per (layer, kv head) of the cache buffers
    recipe: str             # "ar1" | "mixture"
    sim_stride_v: int = 1
    sim_stride_a: int = 1
    frame: int = 1          # tokens per visual frame (ar1)
    rho: float = 0.0        # AR(1) coefficient across frames (ar1)
    audio_std: float = 1.0
    q_scale_lo: float = 1.0  # per (layer, q head) query scale ~ U[lo, hi]
    q_scale_hi: float = 1.0
    n_sinks: int = 0        # first cached visual rows with K x sink_scale (mixture)
    sink_scale: float = 8.0
    outlier_p: float = 0.0  # Bernoulli(p) per key: K x outlier_scale
    outlier_scale: float = 4.0
    steps: int = 1          # chunks in the stream (cfg5)

    @property
    def G(self) -> int:
        return self.Hq // self.Hkv

    @property
    def Nn(self) -> int:
        return self.Nn_v + self.Nn_a

    @property
    def torch_dtype(self) -> torch.dtype:
        return torch.float32 if self.dtype == "fp32" else torch.bfloat16

    @property
    def elem_bytes(self) -> int:
        return 4 if self.dtype == "fp32" else 2

    def replace(self, **kw) -> "Workload":
        return dataclasses.replace(self, **kw)


CFG1 = Workload("cfg1_tiny_fp32", 0, L=2, Hq=4, Hkv=2, D=64, dtype="fp32", n_v=512, n_a=64, Nn_v=112, Nn_a=16,
                budget=256, cache_cap=576, recipe="ar1", sim_stride_v=16, frame=16, rho=0.9, audio_std=0.5)
CFG2 = Workload("cfg2_qwen25omni7b", 1, L=28, Hq=28, Hkv=4, D=128, dtype="bf16", n_v=14336, n_a=2048, Nn_v=4096,
                Nn_a=1500, budget=16384, cache_cap=16384, recipe="mixture", n_sinks=4)
CFG3 = Workload("cfg3_8b", 2, L=36, Hq=32, Hkv=8, D=128, dtype="bf16", n_v=28672, n_a=4096, Nn_v=8192, Nn_a=3000,
                budget=32768, cache_cap=32768, recipe="ar1", sim_stride_v=256, frame=256, rho=0.95, audio_std=0.7,
                q_scale_lo=0.5, q_scale_hi=2.0)
CFG4 = Workload("cfg4_4b_tight", 3, L=36, Hq=32, Hkv=8, D=128, dtype="bf16", n_v=3413, n_a=683, Nn_v=4096, Nn_a=750,
                budget=4096, cache_cap=4096, recipe="ar1", sim_stride_v=256, frame=256, rho=0.98, audio_std=1.0,
                outlier_p=0.1)
CFG5 = Workload("cfg5_hour_stream", 4, L=28, Hq=28, Hkv=4, D=128, dtype="bf16", n_v=0, n_a=0, Nn_v=4096, Nn_a=1500,
                budget=32768, cache_cap=32768, recipe="mixture", n_sinks=4, steps=60)
CONFIGS = {1: CFG1, 2: CFG2, 3: CFG3, 4: CFG4, 5: CFG5}

N_VISUAL_CENTRES = 16
N_AUDIO_CENTRES = 4


def _gen(wl: Workload, step: int, layer: int, tid: int) -> torch.Generator:
    g = torch.Generator(device="cpu")
    g.manual_seed(((1_000_003 * wl.S + 1009 * step + tid) * 4099 + layer) & 0x7FFFFFFFFFFFFFFF)
    return g


def _randn(g, *shape):
    return torch.randn(*shape, generator=g, dtype=torch.float32)


def _ar1_frames(g, Hkv: int, n_frames: int, frame: int, D: int, rho: float) -> torch.Tensor:
    """x[f] = rho x[f-1] + sqrt(1-rho^2) eps, x[0] = eps, per token slot; returns [Hkv, n_frames*frame, D]."""
    if n_frames == 0:
        return torch.zeros(Hkv, 0, D)
    eps = _randn(g, n_frames, Hkv, frame, D)
    out = torch.empty_like(eps)
    out[0] = eps[0]
    c = math.sqrt(1.0 - rho * rho)
    for f in range(1, n_frames):
        out[f] = rho * out[f - 1] + c * eps[f]
    return out.permute(1, 0, 2, 3).reshape(Hkv, n_frames * frame, D)


def layer_inputs(wl: Workload, layer: int, step: int = 0, with_cache: bool = True) -> dict:
    """One layer's tensors in the config dtype.

    Returns cacheK/cacheV [Hkv, n_v+n_a, D] (visual rows then audio rows; only if with_cache),
    chunkK/chunkV [Hkv, Nn, D] (visual block then audio block) and Q [Hq, Nn, D].
    """
    Hkv, Hq, D, G = wl.Hkv, wl.Hq, wl.D, wl.G
    n_v, n_a = (wl.n_v, wl.n_a) if with_cache else (0, 0)
    aux = _gen(wl, 0, layer, 5)          # drawn once per layer, reused by every step (cfg5)
    gk, gv, gq, gm = _gen(wl, step, layer, 0), _gen(wl, step, layer, 1), _gen(wl, step, layer, 4), _gen(wl, step, layer, 3)
    out = {}
    if wl.recipe == "ar1":
        cache_frames = -(-n_v // wl.frame) if n_v else 0
        chunk_frames = -(-wl.Nn_v // wl.frame)
        lead = cache_frames * wl.frame - n_v      # cache = LAST n_v rows of its frames
        kv_vis = []
        for g in (gk, gv):
            x = _ar1_frames(g, Hkv, cache_frames + chunk_frames, wl.frame, D, wl.rho)
            kv_vis.append((x[:, lead:lead + n_v], x[:, cache_frames * wl.frame: cache_frames * wl.frame + wl.Nn_v]))
        aud = [(wl.audio_std * _randn(g, Hkv, n_a, D), wl.audio_std * _randn(g, Hkv, wl.Nn_a, D)) for g in (gk, gv)]
        cacheK = torch.cat([kv_vis[0][0], aud[0][0]], 1)
        cacheV = torch.cat([kv_vis[1][0], aud[1][0]], 1)
        chunkK = torch.cat([kv_vis[0][1], aud[0][1]], 1)
        chunkV = torch.cat([kv_vis[1][1], aud[1][1]], 1)
        Q = _randn(gq, Hq, wl.Nn, D)
    elif wl.recipe == "mixture":
        muK = _randn(aux, Hkv, N_VISUAL_CENTRES + N_AUDIO_CENTRES, D)
        muV = _randn(aux, Hkv, N_VISUAL_CENTRES + N_AUDIO_CENTRES, D)

        def assign(n_vis, n_aud):
            cv = torch.randint(0, N_VISUAL_CENTRES, (Hkv, n_vis), generator=gm)
            ca = torch.randint(N_VISUAL_CENTRES, N_VISUAL_CENTRES + N_AUDIO_CENTRES, (Hkv, n_aud), generator=gm)
            return torch.cat([cv, ca], 1)

        def draw(mu, c, g):
            centre = torch.gather(mu, 1, c.unsqueeze(-1).expand(-1, -1, D))
            return 0.7 * centre + 0.7 * _randn(g, Hkv, c.shape[1], D)

        c_cache, c_chunk = assign(n_v, n_a), assign(wl.Nn_v, wl.Nn_a)
        cacheK, cacheV = draw(muK, c_cache, gk), draw(muV, c_cache, gv)
        chunkK, chunkV = draw(muK, c_chunk, gk), draw(muV, c_chunk, gv)
        cq = c_chunk.repeat_interleave(G, 0)                       # query head j follows KV head j // G
        muKq = muK.repeat_interleave(G, 0)
        Q = 0.7 * torch.gather(muKq, 1, cq.unsqueeze(-1).expand(-1, -1, D)) + 0.7 * _randn(gq, Hq, wl.Nn, D)
        if wl.n_sinks:
            if n_v >= wl.n_sinks:
                cacheK[:, :wl.n_sinks] *= wl.sink_scale
            elif step == 0 and n_v == 0:
                chunkK[:, :wl.n_sinks] *= wl.sink_scale           # cfg5: sinks are the first rows of chunk 0
    else:
        raise ValueError(wl.recipe)
    if wl.q_scale_hi != wl.q_scale_lo:
        u = wl.q_scale_lo + (wl.q_scale_hi - wl.q_scale_lo) * torch.rand(Hq, 1, 1, generator=aux)
        Q = Q * u
    if wl.outlier_p > 0:
        mc = torch.rand(Hkv, n_v + n_a, 1, generator=gm) < wl.outlier_p
        mk = torch.rand(Hkv, wl.Nn, 1, generator=gm) < wl.outlier_p
        cacheK = torch.where(mc, cacheK * wl.outlier_scale, cacheK)
        chunkK = torch.where(mk, chunkK * wl.outlier_scale, chunkK)
    dt = wl.torch_dtype
    if with_cache:
        out["cacheK"], out["cacheV"] = cacheK.to(dt).contiguous(), cacheV.to(dt).contiguous()
    out["chunkK"], out["chunkV"], out["Q"] = chunkK.to(dt).contiguous(), chunkV.to(dt).contiguous(), Q.to(dt).contiguous()
    return out


def full_inputs(wl: Workload, step: int = 0, layers=None, with_cache: bool = True, pin: bool = False,
                workers: int | None = None) -> dict:
    """Stack `layers` (default all) into [L', ...] tensors; the cache is zero-padded to cache_cap rows.

    Returns cacheK, cacheV [L',Hkv,cache_cap,D], chunkK, chunkV [L',Hkv,Nn,D], Q [L',Hq,Nn,D],
    n_v, n int32 [L'] (rows valid per layer).  Layers have their own generators, so they are drawn by `workers`
    threads (default: up to 8) with bit-identical results.
    """
    layers = list(range(wl.L)) if layers is None else list(layers)
    Lp, dt = len(layers), wl.torch_dtype
    mk = (lambda *s: torch.zeros(*s, dtype=dt).pin_memory()) if pin else (lambda *s: torch.zeros(*s, dtype=dt))
    out = dict(chunkK=mk(Lp, wl.Hkv, wl.Nn, wl.D), chunkV=mk(Lp, wl.Hkv, wl.Nn, wl.D), Q=mk(Lp, wl.Hq, wl.Nn, wl.D))
    if with_cache:
        out["cacheK"] = torch.zeros(Lp, wl.Hkv, wl.cache_cap, wl.D, dtype=dt)
        out["cacheV"] = torch.zeros(Lp, wl.Hkv, wl.cache_cap, wl.D, dtype=dt)
    nc = (wl.n_v + wl.n_a) if with_cache else 0
    def fill(il):
        i, l = il
        x = layer_inputs(wl, l, step, with_cache)
        for k in ("chunkK", "chunkV", "Q"):
            out[k][i] = x[k]
        if with_cache:
            out["cacheK"][i, :, :nc] = x["cacheK"]
            out["cacheV"][i, :, :nc] = x["cacheV"]

    workers = min(8, os.cpu_count() or 1, Lp) if workers is None else workers
    if workers > 1:
        with ThreadPoolExecutor(max_workers=workers) as ex:
            list(ex.map(fill, enumerate(layers)))
    else:
        for il in enumerate(layers):
            fill(il)
    out["n_v"] = torch.full((Lp,), wl.n_v if with_cache else 0, dtype=torch.int32)
    out["n"] = torch.full((Lp,), nc, dtype=torch.int32)
    return out


def hidden_inputs(wl: Workload, d_model: int, step: int = 0, with_cache: bool = True) -> dict:
    """Synthetic hidden states for the hidden-state form of Eq.7 (NEXT-3): cacheH [L, cache_cap, d_model]
    (zero-padded) and chunkH [L, Nn, d_model] in the config dtype.  Generator tid 6.  Visual rows: AR(1) across frames
    of `wl.frame` tokens with the config's rho ("ar1" recipe), or a 16-centre mixture ("mixture"); audio rows i.i.d.
    N(0, audio_std^2).  One row per token and layer (hidden states have no head index)."""
    n_v, n_a = (wl.n_v, wl.n_a) if with_cache else (0, 0)
    dt = wl.torch_dtype
    cacheH = torch.zeros(wl.L, wl.cache_cap, d_model, dtype=dt)
    chunkH = torch.zeros(wl.L, wl.Nn, d_model, dtype=dt)
    for l in range(wl.L):
        g = _gen(wl, step, l, 6)
        if wl.recipe == "ar1":
            cache_frames = -(-n_v // wl.frame) if n_v else 0
            chunk_frames = -(-wl.Nn_v // wl.frame)
            lead = cache_frames * wl.frame - n_v
            x = _ar1_frames(g, 1, cache_frames + chunk_frames, wl.frame, d_model, wl.rho)[0]
            vis_c, vis_n = x[lead:lead + n_v], x[cache_frames * wl.frame: cache_frames * wl.frame + wl.Nn_v]
        else:
            mu = _randn(_gen(wl, 0, l, 7), N_VISUAL_CENTRES, d_model)
            c = torch.randint(0, N_VISUAL_CENTRES, (n_v + wl.Nn_v,), generator=g)
            x = 0.7 * mu[c] + 0.7 * _randn(g, n_v + wl.Nn_v, d_model)
            vis_c, vis_n = x[:n_v], x[n_v:]
        aud = wl.audio_std * _randn(g, n_a + wl.Nn_a, d_model)
        cacheH[l, :n_v], cacheH[l, n_v:n_v + n_a] = vis_c.to(dt), aud[:n_a].to(dt)
        chunkH[l, :wl.Nn_v], chunkH[l, wl.Nn_v:] = vis_n.to(dt), aud[n_a:].to(dt)
    return dict(cacheH=cacheH, chunkH=chunkH)


def modality_pattern(wl: Workload, groups: int) -> torch.Tensor:
    """Per-row modality map of a time-interleaved chunk (NEXT-4b, R25'): `groups` time slices (e.g. seconds), each holding
    its share of the visual rows followed by its share of the audio rows.  int32 [Nn], 0 = visual, 1 = audio."""
    groups = max(1, min(groups, max(wl.Nn_v, wl.Nn_a, 1)))
    out = []
    for g in range(groups):
        nv = (g + 1) * wl.Nn_v // groups - g * wl.Nn_v // groups
        na = (g + 1) * wl.Nn_a // groups - g * wl.Nn_a // groups
        out += [0] * nv + [1] * na
    return torch.tensor(out, dtype=torch.int32)


def interleave(x: dict, modality: torch.Tensor, Nn_v: int) -> dict:
    """Reorder the chunk tensors of a modality-blocked input dict (chunkK, chunkV, Q and chunkH if present; row axis -2)
    into the temporal order of `modality`: the j-th visual (audio) row of the result is blocked row j (Nn_v + j)."""
    m = modality.long()
    rank_v, rank_a = torch.cumsum(1 - m, 0) - 1, torch.cumsum(m, 0) - 1
    src = torch.where(m == 0, rank_v, Nn_v + rank_a)
    y = dict(x)
    for k in ("chunkK", "chunkV", "Q", "chunkH"):
        if k in x:
            y[k] = x[k].index_select(-2, src).contiguous()
    return y
