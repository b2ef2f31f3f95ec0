"""GPU parity: the CUDA path (through the C ABI) against the fp64 oracle on the same seeded inputs.

north_star matching rules: (a) scores, entropies, budgets within 2e-3 relative (1e-5 for fp32 inputs);
(b) selection and compaction bit-exact when fed the oracle's score array; (c) end-to-end kept-index sets
identical except where adjacent scores differ by less than that tolerance.
"""
import os

import numpy as np
import pytest
import torch

from oracle import ref
from paper_2606_07577_b200 import inputs as I
from tests.util import TOL, compare_scores, kept_sets_rule_c, ref_params, scores_to_numpy, seg_lens, to_device

pytestmark = pytest.mark.gpu


def engine_for(wl, **kw):
    from paper_2606_07577_b200.omnimem import OmniMem
    return OmniMem.for_workload(wl, **kw)


def dev_objs(x, wl):
    from paper_2606_07577_b200.omnimem import Cache, Chunk
    d = to_device(x)
    return Cache(d["cacheK"], d["cacheV"], d["n_v"], d["n"]), Chunk(d["chunkK"], d["chunkV"], d["Q"], wl.Nn_v, wl.Nn_a)


def check_step(wl, x=None, eng_kw=None, ref_kw=None, sim_source=0, check_rowH=True, stats_tol=None, select_scope=0,
               modality=None):
    """All of rules (a), (b), (c) for one step of workload `wl` (L = number of layers in x)."""
    eng_kw, ref_kw = dict(eng_kw or {}), dict(ref_kw or {})
    x = x if x is not None else I.full_inputs(wl)
    L = x["Q"].shape[0]
    wl = wl.replace(L=L)
    tol = TOL[wl.dtype]
    if modality is not None:                       # time-interleaved chunk: both sides get the reordered rows + the map
        x = I.interleave(x, modality, wl.Nn_v)
        ref_kw["chunk_modality"] = modality.numpy()
    p = ref_params(wl, L, **ref_kw)
    B = np.full((L,), wl.budget, np.int32)
    orc = ref.compress_chunk(p, x["cacheK"], x["cacheV"], x["n_v"], x["n"], x["chunkK"], x["chunkV"], x["Q"], B,
                             sim_source=sim_source, want_rowH=check_rowH, select_scope=select_scope)
    eng = engine_for(wl, sim_source=sim_source, select_scope=select_scope, **eng_kw)
    src, chunk = dev_objs(x, wl)
    if modality is not None:
        chunk.modality = modality.cuda()
    n_v, n = x["n_v"].numpy(), x["n"].numpy()
    Kv, Ka = seg_lens(wl, n_v, n)

    # ---- rule (a): scoring stages
    sc = eng.score(src, chunk, want_lse=True, want_row_entropy=check_rowH)
    torch.cuda.synchronize()
    g = scores_to_numpy(sc)
    compare_scores(wl, n_v, n, g, orc, tol, stats_tol)
    if check_rowH and wl.Nn:
        # row entropy (R16 diagnostic) at rule (a): H <= ln Nk, so tol * ln Nk is `tol` relative to the quantity's range
        np.testing.assert_allclose(g["rowH"], orc["rowH"], rtol=0, atol=tol * np.log(max(2, int(n.max()) + wl.Nn)))
    # softmax rows sum to one => sum_k a[l,h,k] = G * Nq
    tot = np.array([[g["a_v"][l, h, :Kv[l]].astype(np.float64).sum() + g["a_a"][l, h, :Ka[l]].astype(np.float64).sum()
                     for h in range(wl.Hkv)] for l in range(L)])
    np.testing.assert_allclose(tot, wl.G * wl.Nn, rtol=10 * tol, atol=1e-12)

    # ---- budgets from the ORACLE's statistics: exact
    dev = eng.device
    Bt = torch.from_numpy(B).to(dev)
    M_v, M_a, _ = eng.allocate(torch.from_numpy(orc["stats"]).to(dev), src.n_v, src.n, wl.Nn_v, wl.Nn_a, Bt)
    assert np.array_equal(M_v.cpu().numpy(), orc["M_v"]) and np.array_equal(M_a.cpu().numpy(), orc["M_a"])

    # ---- rule (b): selection + compaction fed the oracle's score array and budgets: bit-exact
    idx_v, idx_a = eng.select(torch.from_numpy(orc["psi_v"]).to(dev), torch.from_numpy(orc["psi_a"]).to(dev), src.n_v,
                              src.n, wl.Nn_v, wl.Nn_a, M_v, M_a)
    iv, ia = idx_v.cpu().numpy(), idx_a.cpu().numpy()
    for l in range(L):
        assert np.array_equal(iv[l, :, :orc["M_v"][l]], orc["idx_v"][l, :, :orc["M_v"][l]]), f"idx_v layer {l}"
        assert np.array_equal(ia[l, :, :orc["M_a"][l]], orc["idx_a"][l, :, :orc["M_a"][l]]), f"idx_a layer {l}"
    dst = eng.new_cache()
    eng.compact(src, chunk, idx_v, idx_a, M_v, M_a, dst)
    torch.cuda.synchronize()
    dK, dV = dst.k.cpu().view(torch.uint8).numpy(), dst.v.cpu().view(torch.uint8).numpy()
    for l in range(L):
        nl = int(orc["n_out"][l])
        assert np.array_equal(dK[l, :, :nl], orc["dstK"][l, :, :nl]) and np.array_equal(dV[l, :, :nl], orc["dstV"][l, :, :nl])
    assert np.array_equal(dst.n_v.cpu().numpy(), orc["n_v_out"]) and np.array_equal(dst.n.cpu().numpy(), orc["n_out"])

    # ---- rule (c): the fused step end to end
    dst2 = eng.new_cache()
    idx_v2, idx_a2 = eng.new_indices()
    M_v2 = torch.zeros(L, dtype=torch.int32, device=dev)
    M_a2 = torch.zeros_like(M_v2)
    eng.compress_chunk(src, chunk, Bt, dst2, idx_v=idx_v2, idx_a=idx_a2, M_v=M_v2, M_a=M_a2)
    torch.cuda.synchronize()
    mv, ma = M_v2.cpu().numpy(), M_a2.cpu().numpy()
    iv, ia = idx_v2.cpu().numpy(), idx_a2.cpu().numpy()
    n_diff = 0
    for l in range(L):
        assert mv[l] + ma[l] == min(wl.budget, Kv[l] + Ka[l])
        if mv[l] != orc["M_v"][l]:
            # rule (a) for an integer decided by a float: M_v = floor(w_v B + 1/2) may differ by ONE, and only when the
            # oracle's w_v B lies within the statistic tolerance of the rounding boundary (and never by more than half a
            # unit of slack: min(tol B, 0.5)); the kept sets are then judged against the GPU's own budgets below
            st = orc["stats"][l]
            r = float(eng.cfg.ratio_r)
            den = r * st[4] + st[5]
            wv = r * st[4] / den if den > 0 else r / (r + 1.0)
            x_ref = wv * wl.budget
            assert abs(int(mv[l]) - int(orc["M_v"][l])) == 1 and \
                abs(x_ref + 0.5 - round(x_ref + 0.5)) <= min(tol * wl.budget, 0.5), f"M_v[{l}] {mv[l]} vs {orc['M_v'][l]} (w_v B = {x_ref})"
            Mg_v, Mg_a = ref.select(ref_params(wl, 1, **ref_kw), orc["psi_v"][l:l + 1], orc["psi_a"][l:l + 1], n_v[l:l + 1], n[l:l + 1],
                                    mv[l:l + 1], ma[l:l + 1])
            for h in range(wl.Hkv):                               # oracle scores, the GPU's budgets
                n_diff += kept_sets_rule_c(f"v[{l},{h}]*", iv[l, h], Mg_v[0, h], int(mv[l]), orc["psi_v"][l, h, :Kv[l]], tol)
                n_diff += kept_sets_rule_c(f"a[{l},{h}]*", ia[l, h], Mg_a[0, h], int(ma[l]), orc["psi_a"][l, h, :Ka[l]], tol)
            continue
        for h in range(wl.Hkv):
            n_diff += kept_sets_rule_c(f"v[{l},{h}]", iv[l, h], orc["idx_v"][l, h], int(mv[l]), orc["psi_v"][l, h, :Kv[l]], tol)
            n_diff += kept_sets_rule_c(f"a[{l},{h}]", ia[l, h], orc["idx_a"][l, h], int(ma[l]), orc["psi_a"][l, h, :Ka[l]], tol)
    # whatever was kept, dst rows are byte-exact copies of the rows the GPU's indices name
    dK2 = dst2.k.cpu().view(torch.uint8).numpy()
    rawc, rawk = x["cacheK"].view(torch.uint8).numpy(), x["chunkK"].view(torch.uint8).numpy()
    for l in range(L):
        for h in range(wl.Hkv):
            mv_rows = np.arange(wl.Nn) < wl.Nn_v if modality is None else modality.numpy() == 0
            vis = np.concatenate([rawc[l, h, :n_v[l]], rawk[l, h][mv_rows]])
            aud = np.concatenate([rawc[l, h, n_v[l]:n[l]], rawk[l, h][~mv_rows]])
            assert np.array_equal(dK2[l, h, :mv[l]], vis[iv[l, h, :mv[l]]])
            assert np.array_equal(dK2[l, h, mv[l]:mv[l] + ma[l]], aud[ia[l, h, :ma[l]]])
    eng.close()
    return n_diff


# ---------------------------------------------------------------------------------------------- CFG1 (fp32, SIMT)
def test_cfg1_full():
    assert check_step(I.CFG1) == 0                 # fp32: the kept sets must be identical


def test_cfg1_paper_literal_stride_and_key_similarity():
    wl = I.CFG1.replace(sim_stride_v=1)
    check_step(wl)
    check_step(wl, sim_source=1)


# ---------------------------------------------------------------------------------------------- bf16, tcgen05 path
SMALL2 = I.CFG2.replace(L=2, Hq=4, Hkv=2, n_v=700, n_a=150, Nn_v=400, Nn_a=123, budget=850, cache_cap=850)
SMALL3 = I.CFG3.replace(L=2, Hq=4, Hkv=2, n_v=1024, n_a=200, Nn_v=512, Nn_a=100, budget=1224, cache_cap=1300)
SMALL4 = I.CFG4.replace(L=2, Hq=4, Hkv=1, n_v=333, n_a=67, Nn_v=512, Nn_a=70, budget=400, cache_cap=400)


@pytest.mark.parametrize("wl", [SMALL2, SMALL3, SMALL4], ids=lambda w: w.name)
def test_bf16_tcgen05_small(wl):
    check_step(wl)


@pytest.mark.parametrize("ctas", [1, 2, 3, 7])
def test_persistent_ctas_walk_several_items(ctas):
    """The tcgen05 scoring kernels are persistent: with `score_ctas` CTAs instead of one per SM, every CTA of these small
    shapes walks several work items, so ring positions and barrier phases carry across items, across skipped items
    (cache blocks beyond n), across ragged last blocks where one sub-tile's warps have nothing to do (they must not run
    ahead of the ring), the lse ring wraps inside and between items, and an empty cache leaves only chunk items.
    Results must not depend on the number of CTAs: rules (a)-(c) as everywhere."""
    for wl in (SMALL2, SMALL3, SMALL4):
        for n_v in (wl.n_v, wl.n_v - 37, 300, 0):
            check_step(wl.replace(n_v=n_v), eng_kw=dict(score_ctas=ctas), check_rowH=(n_v == 300))
    check_step(SMALL2, eng_kw=dict(score_ctas=ctas, causal=0), ref_kw=dict(causal=0))
    # layers of different length in one launch (what a ragged budget table leaves behind): full, 137 rows short, nearly empty, empty
    wl = SMALL3.replace(L=4)
    x = I.full_inputs(wl)
    x["n_v"] = x["n_v"].clone()
    x["n"] = x["n"].clone()
    for l, (dv, dn) in enumerate(((0, 0), (100, 137), (wl.n_v - 3, wl.n_v + wl.n_a - 5), (wl.n_v, wl.n_v + wl.n_a))):
        x["n_v"][l] -= dv
        x["n"][l] -= dn
    check_step(wl, x=x, eng_kw=dict(score_ctas=ctas))
    check_step(SMALL3.replace(Hq=14, Hkv=2), eng_kw=dict(score_ctas=ctas))          # G = 7: 35 query tiles per key block
    check_step(SMALL3, eng_kw=dict(score_ctas=ctas), modality=I.modality_pattern(SMALL3, 5))


@pytest.mark.parametrize("wl", [SMALL2, SMALL4], ids=lambda w: w.name)
def test_bf16_simt_path_small(wl):
    check_step(wl, eng_kw=dict(score_path=1))


def test_bf16_head_dim_64_simt():
    check_step(SMALL2.replace(D=64))


def test_noncausal_and_lambda_zero():
    check_step(SMALL2, eng_kw=dict(causal=0), ref_kw=dict(causal=0))
    check_step(SMALL3, eng_kw=dict(lam=0.0), ref_kw=dict(lam=0.0))      # cosine-only ablation
    check_step(I.CFG1, eng_kw=dict(causal=0, lam=1.0, ratio_r=2.0), ref_kw=dict(causal=0, lam=1.0, ratio_r=2.0))


def test_edge_shapes():
    check_step(SMALL2.replace(n_a=0, Nn_a=0))                     # single modality ("no split")
    check_step(SMALL2.replace(n_v=0, n_a=0))                      # empty cache (first chunk of a stream)
    check_step(SMALL2.replace(budget=2000, cache_cap=2000))       # nothing to evict: keep all, identity indices
    check_step(SMALL2.replace(Nn_v=1, Nn_a=0))                    # one-token chunk
    check_step(SMALL2.replace(n_v=128, n_a=128, Nn_v=128, Nn_a=128, budget=256, cache_cap=256))   # tile-aligned
    check_step(I.CFG1.replace(n_v=0, n_a=64, Nn_v=0, cache_cap=200, budget=40))                  # audio only


def test_empty_chunk_keeps_everything():
    wl = SMALL2.replace(Nn_v=0, Nn_a=0, budget=850)
    x = I.full_inputs(SMALL2)
    x["chunkK"], x["chunkV"], x["Q"] = x["chunkK"][:, :, :0], x["chunkV"][:, :, :0], x["Q"][:, :, :0]
    check_step(wl, x=x, check_rowH=False)


def test_supplied_lse_skips_pass1():
    """chunk.lse given (the model's attention forward already has it): pass 2 alone must reproduce a."""
    from paper_2606_07577_b200.omnimem import Chunk
    for wl, kw in ((SMALL3, {}), (I.CFG1, {})):
        x = I.full_inputs(wl)
        L = x["Q"].shape[0]
        p = ref_params(wl, L)
        orc = ref.score(p, x["cacheK"], x["cacheV"], x["n_v"], x["n"], x["chunkK"], x["chunkV"], x["Q"])
        eng = engine_for(wl.replace(L=L), **kw)
        src, chunk = dev_objs(x, wl)
        chunk = Chunk(chunk.k, chunk.v, chunk.q, wl.Nn_v, wl.Nn_a, lse=torch.from_numpy(orc["lse"]).float().cuda())
        eng.set_profiling(True)
        sc = eng.score(src, chunk)
        torch.cuda.synchronize()
        ms, _ = eng.stage_ms()
        assert ms["lse"] == 0.0 and ms["colsum"] > 0.0
        compare_scores(wl, x["n_v"].numpy(), x["n"].numpy(), scores_to_numpy(sc), orc, TOL[wl.dtype])
        eng.close()


# ---------------------------------------------------------------------------------------------- rule (b) at scale
def test_select_compact_bit_exact_with_ties_large():
    """Random fp32 scores with many ties and negative zeros, ragged per-layer budgets: select + compact are bit-exact."""
    from paper_2606_07577_b200.omnimem import Cache, Chunk
    wl = I.CFG2.replace(L=3, Hq=2, Hkv=2, n_v=20000, n_a=3000, Nn_v=4096, Nn_a=1500, cache_cap=23000, budget=16384)
    L = wl.L
    eng = engine_for(wl)
    p = ref_params(wl, L)
    g = np.random.default_rng(5)
    n_v = np.array([20000, 17000, 1], np.int32)
    n = np.array([23000, 18001, 3], np.int32)
    psi_v = np.round(g.random((L, wl.Hkv, p.seg_cap_v)), 3).astype(np.float32)       # ~1000 distinct values: heavy ties
    psi_a = (g.random((L, wl.Hkv, p.seg_cap_a)).astype(np.float32)) ** 8
    psi_a[0, 0, :50] = -0.0
    psi_a[0, 0, 50:100] = 0.0
    psi_v[1, 1] = 0.25                                                               # all equal
    Kv, Ka = seg_lens(wl, n_v, n)
    M_v = np.array([13000, 9999, 0], np.int32)
    M_a = np.array([3384, 2000, 700], np.int32)
    M_v[2] = Kv[2]                                                                   # keep every visual row
    iv_ref, ia_ref = ref.select(p, psi_v, psi_a, n_v, n, M_v, M_a)
    t = lambda a: torch.from_numpy(a).cuda()
    iv, ia = eng.select(t(psi_v), t(psi_a), t(n_v), t(n), wl.Nn_v, wl.Nn_a, t(M_v), t(M_a))
    iv, ia = iv.cpu().numpy(), ia.cpu().numpy()
    for l in range(L):
        assert np.array_equal(iv[l, :, :M_v[l]], iv_ref[l, :, :M_v[l]]) and np.array_equal(ia[l, :, :M_a[l]], ia_ref[l, :, :M_a[l]])
    gK = torch.Generator().manual_seed(1)
    cacheK = torch.randn(L, wl.Hkv, wl.cache_cap, wl.D, generator=gK).to(torch.bfloat16)
    cacheV = torch.randn(L, wl.Hkv, wl.cache_cap, wl.D, generator=gK).to(torch.bfloat16)
    chunkK = torch.randn(L, wl.Hkv, wl.Nn, wl.D, generator=gK).to(torch.bfloat16)
    chunkV = torch.randn(L, wl.Hkv, wl.Nn, wl.D, generator=gK).to(torch.bfloat16)
    dK_ref, nv2, n2 = ref.compact(p, cacheK, chunkK, n_v, n, iv_ref, ia_ref, M_v, M_a)
    dV_ref, _, _ = ref.compact(p, cacheV, chunkV, n_v, n, iv_ref, ia_ref, M_v, M_a)
    src = Cache(cacheK.cuda(), cacheV.cuda(), t(n_v), t(n))
    chunk = Chunk(chunkK.cuda(), chunkV.cuda(), chunkK.cuda(), wl.Nn_v, wl.Nn_a)
    dst = eng.new_cache()
    eng.compact(src, chunk, t(iv_ref), t(ia_ref), t(M_v), t(M_a), dst)
    torch.cuda.synchronize()
    dK, dV = dst.k.cpu().view(torch.uint8).numpy(), dst.v.cpu().view(torch.uint8).numpy()
    for l in range(L):
        assert np.array_equal(dK[l, :, :n2[l]], dK_ref[l, :, :n2[l]]) and np.array_equal(dV[l, :, :n2[l]], dV_ref[l, :, :n2[l]])
    assert np.array_equal(dst.n.cpu().numpy(), n2) and np.array_equal(dst.n_v.cpu().numpy(), nv2)
    eng.close()


def test_layer_budgets_eq14_on_device():
    """Eq.13-14 in omnimem_allocate (layer_budget == NULL) against the oracle on the 240 seeded cases that pin the oracle's
    clamp branch to the kappa water-filling form (tests/test_oracle_pins.py): one- and two-sided clamps, tight ranges,
    infeasible totals, no clamp.  The kernel finds kappa by a breakpoint search and integerises by rank; the oracle by
    its round-by-round rule: two procedures, one answer."""
    from tests.test_oracle_pins import eq14_cases
    t = lambda a: torch.from_numpy(a).cuda()
    n_checked = 0
    for i, (L, st, T, lo, hi, total) in enumerate(eq14_cases()):
        if i % 6 == 5:
            lo, hi = 0, 0                                                   # the unclamped branch
        cap = max(64, min(hi, total) if hi > 0 else total)                     # no share exceeds min(B_max, total)
        wl = I.CFG1.replace(L=L, Hq=1, Hkv=1, cache_cap=cap, n_v=0, n_a=0, Nn_v=8, Nn_a=8)   # workspace ~ 40 B x L x cap
        g = np.random.default_rng(i)
        st = st.copy()
        st[:, 4], st[:, 5] = g.uniform(0.1, 0.9, L), g.uniform(0.1, 0.9, L)
        n_v, n = np.full(L, 0, np.int32), np.full(L, 0, np.int32)
        eng = engine_for(wl, budget_min=lo, budget_max=hi, temperature=T)
        p = ref_params(wl, L, budget_min=lo, budget_max=hi, temperature=T)
        B_ref = ref.layer_budgets(p, st, total)
        M_v_ref, M_a_ref = ref.allocate(p, st, n_v, n, B_ref)
        M_v, M_a, B = eng.allocate(t(st), t(n_v), t(n), wl.Nn_v, wl.Nn_a, None, total)
        assert np.array_equal(B.cpu().numpy(), B_ref), f"case {i}: L={L} lo={lo} hi={hi} total={total}: {B.cpu().numpy()} vs {B_ref}"
        assert np.array_equal(M_v.cpu().numpy(), M_v_ref) and np.array_equal(M_a.cpu().numpy(), M_a_ref)
        n_checked += 1
        eng.close()
    assert n_checked == 240


def test_budget_above_capacity_is_clamped_not_written_out_of_bounds():
    """include/omnimem.h "Budgets": device-resident budgets cannot be rejected on the host, so they are clamped where they
    are consumed.  layer_budget = cache_cap + 1000 with K > cache_cap, and M_v / M_a above K and above cache_cap handed
    to select / compact directly: nothing may be written at or beyond row cache_cap of an idx or dst row block.  The
    buffers are over-allocated by guard rows holding a sentinel."""
    from paper_2606_07577_b200.omnimem import Cache, Chunk
    wl = SMALL2.replace(cache_cap=900, budget=900)                       # K = 850 + 523 = 1373 > cache_cap
    L, cap, G = wl.L, wl.cache_cap, 64                                   # G guard rows after each tensor
    x = I.full_inputs(wl)
    eng = engine_for(wl)
    src, chunk = dev_objs(x, wl)
    dt = wl.torch_dtype
    SENT = 0x7B7B

    def guarded(shape, dtype, fill):
        n = int(np.prod(shape))
        row = int(np.prod(shape[2:])) if len(shape) > 2 else 1
        buf = torch.full((n + G * row,), fill, dtype=dtype, device="cuda")
        return buf, buf[:n].view(*shape), buf[n:]

    kbuf, kview, kguard = guarded((L, wl.Hkv, cap, wl.D), torch.int16, SENT)
    vbuf, vview, vguard = guarded((L, wl.Hkv, cap, wl.D), torch.int16, SENT)
    ivbuf, ivview, ivguard = guarded((L, wl.Hkv, cap), torch.int32, -7)
    iabuf, iaview, iaguard = guarded((L, wl.Hkv, cap), torch.int32, -7)
    dst = Cache(kview.view(dt), vview.view(dt), torch.zeros(L, dtype=torch.int32, device="cuda"), torch.zeros(L, dtype=torch.int32, device="cuda"))
    B = torch.full((L,), cap + 1000, dtype=torch.int32, device="cuda")
    M_v = torch.zeros(L, dtype=torch.int32, device="cuda")
    M_a = torch.zeros_like(M_v)
    eng.compress_chunk(src, chunk, B, dst, idx_v=ivview, idx_a=iaview, M_v=M_v, M_a=M_a)
    torch.cuda.synchronize()
    assert bool((M_v + M_a == cap).all()), "an over-capacity total is clamped to cache_cap"
    assert torch.equal(dst.n, torch.full_like(dst.n, cap))
    for gd, fill in ((kguard, SENT), (vguard, SENT), (ivguard, -7), (iaguard, -7)):
        assert bool((gd == fill).all()), "wrote past the end of a buffer"
    # every head's rows [M_v + M_a, cap) of idx are untouched, and the next head's block starts intact
    mv, ma = M_v.cpu().numpy(), M_a.cpu().numpy()
    for l in range(L):
        assert bool((ivview[l, :, mv[l]:] == -7).all()) and bool((iaview[l, :, ma[l]:] == -7).all())
    # the public stage calls with budgets above K and above cache_cap
    sc = eng.score(src, chunk)
    big_v = torch.full((L,), 5000, dtype=torch.int32, device="cuda")     # > K_v = 1100 > cache_cap
    big_a = torch.full((L,), 5000, dtype=torch.int32, device="cuda")
    ivview.fill_(-7); iaview.fill_(-7); kview.fill_(SENT); vview.fill_(SENT)
    eng.select(sc.psi_v, sc.psi_a, src.n_v, src.n, wl.Nn_v, wl.Nn_a, big_v, big_a, idx_v=ivview, idx_a=iaview)
    eng.compact(src, chunk, ivview, iaview, big_v, big_a, dst)
    torch.cuda.synchronize()
    Kv = wl.n_v + wl.Nn_v
    want_v = min(Kv, cap)                                                # 5000 -> 900 visual rows, nothing left for audio
    assert torch.equal(dst.n_v, torch.full_like(dst.n_v, want_v)) and torch.equal(dst.n, torch.full_like(dst.n, cap))
    p = ref_params(wl, L)
    iv_ref, _ = ref.select(p, sc.psi_v.cpu().numpy(), sc.psi_a.cpu().numpy(), x["n_v"].numpy(), x["n"].numpy(),
                           np.full(L, want_v, np.int32), np.zeros(L, np.int32))
    assert np.array_equal(ivview[:, :, :want_v].cpu().numpy(), iv_ref[:, :, :want_v])    # the clamped M: a real top-900 of 1100
    assert bool((iaview == -7).all())
    for gd, fill in ((kguard, SENT), (vguard, SENT), (ivguard, -7), (iaguard, -7)):
        assert bool((gd == fill).all()), "wrote past the end of a buffer"
    neg = torch.full((L,), -5, dtype=torch.int32, device="cuda")
    eng.select(sc.psi_v, sc.psi_a, src.n_v, src.n, wl.Nn_v, wl.Nn_a, neg, neg, idx_v=ivview, idx_a=iaview)
    eng.compact(src, chunk, ivview, iaview, neg, neg, dst)
    torch.cuda.synchronize()
    assert int(dst.n.max()) == 0 and int(dst.n_v.max()) == 0
    eng.close()


@pytest.mark.parametrize("cap", [49152, 65536], ids=["48k_budget_smem_keys", "64k_global_keys"])
def test_select_at_the_papers_largest_budgets(cap):
    """P:266 sweeps the memory up to 48k per layer.  cache_cap 49152 + a 4096 + 1500 chunk is 53248 visual keys per
    segment: the shared-memory key path of select_kernel at its largest paper-stated size; 65536 forces the
    global-memory variant (select_kernel<false>, taken above 57600 keys).  Bit-exact against the oracle with heavy ties,
    signed zeros and an all-equal head (rule (b))."""
    wl = I.CFG2.replace(L=1, Hq=2, Hkv=2, n_v=cap - 6000, n_a=6000, Nn_v=4096, Nn_a=1500, cache_cap=cap, budget=cap)
    eng = engine_for(wl)
    p = ref_params(wl, 1)
    g = np.random.default_rng(cap)
    n_v, n = np.array([cap - 6000], np.int32), np.array([cap], np.int32)
    psi_v = np.round(g.random((1, 2, p.seg_cap_v)), 3).astype(np.float32)
    psi_a = (g.random((1, 2, p.seg_cap_a)).astype(np.float32)) ** 6
    psi_a[0, 0, :40] = -0.0
    psi_a[0, 0, 40:90] = 0.0
    psi_v[0, 1] = 0.5
    M_v, M_a = np.array([cap - 5000], np.int32), np.array([5000], np.int32)
    iv_ref, ia_ref = ref.select(p, psi_v, psi_a, n_v, n, M_v, M_a)
    t = lambda a: torch.from_numpy(a).cuda()
    iv, ia = eng.select(t(psi_v), t(psi_a), t(n_v), t(n), wl.Nn_v, wl.Nn_a, t(M_v), t(M_a))
    assert np.array_equal(iv.cpu().numpy()[0, :, :M_v[0]], iv_ref[0, :, :M_v[0]])
    assert np.array_equal(ia.cpu().numpy()[0, :, :M_a[0]], ia_ref[0, :, :M_a[0]])
    assert bool((iv[0, :, M_v[0]:] == -1).all()) and bool((ia[0, :, M_a[0]:] == -1).all())
    eng.close()


@pytest.mark.parametrize("mult", [12.0, 40.0])
def test_wide_logit_range(mult):
    """Logits far wider than the Gaussian test inputs give: the softmax scale is multiplied by 12 / 40 and three keys get
    64 x the norm -- one in the FIRST cache tile, one in the LAST cache tile and one in the chunk -- so that in pass 1 the
    running reference is re-based in the middle of a row with Z != 0 (the lazy-maximum vote fails mid-row), most
    probabilities underflow (the polynomial's exponent clamp, ex2.approx.ftz, flush-to-zero sums), 7 of 8 rows are taken
    by one key, and at x 40 more than half of the keys have an importance below 1e-30 (down to 1e-107 in the mixture
    input): those are recomputed in the log domain (R31).  Rules (a)-(c) unchanged, causal and not."""
    for wl in (SMALL2, SMALL3, SMALL4):
        x = I.full_inputs(wl)
        nc = wl.n_v + wl.n_a
        x["cacheK"][:, :, 5] *= 64.0
        x["cacheK"][:, :, nc - 3] *= 64.0
        x["chunkK"][:, :, wl.Nn // 2] *= 64.0
        c = mult / float(np.sqrt(wl.D))
        check_step(wl, x=x, eng_kw=dict(softmax_scale=c), ref_kw=dict(scale=c))
        check_step(wl, x=x, eng_kw=dict(softmax_scale=c, causal=0), ref_kw=dict(scale=c, causal=0))
    # (fp32 inputs are left out: logits of +-100 computed in fp32 carry an absolute error of ~1e-5, i.e. the whole 1e-5
    # tolerance of rule (a), before anything else is counted)
    check_step(SMALL2, eng_kw=dict(softmax_scale=c, score_path=1), ref_kw=dict(scale=c))        # bf16 SIMT path
    check_step(SMALL3.replace(Hq=8, Hkv=4), eng_kw=dict(softmax_scale=c), ref_kw=dict(scale=c), select_scope=1)   # log-sum over heads


def test_importance_below_fp32_range_is_recovered():
    """DESIGN.md R31: two cached keys point AGAINST every query (logit between -318 and -106 for all of them): every one of
    their softmax weights is below 2^-126, the fp32 column sum is exactly 0, and the true importance is about 1e-55.
    Eq.8 maps that to psi ~ 0.08 (1 - s), so it must not be lost: the key is recomputed in the log domain, psi matches the
    oracle at rule (a), and the published fp32 `a` holds what fp32 can (0)."""
    wl = SMALL3
    x = I.full_inputs(wl)
    e = torch.ones(wl.D) / float(np.sqrt(wl.D))                                  # a fixed unit direction
    x["Q"] = (x["Q"].float() + 12.0 * e).to(x["Q"].dtype)                        # <q, e> = 12 + N(0, u^2) in [6, 18], u <= 2
    dead = (-200.0 * e).to(x["cacheK"].dtype)                                    # c <q, dead> in [-318, -106] for every query
    x["cacheK"][:, :, 7] = dead
    x["cacheK"][:, :, 600] = dead
    L = wl.L
    p = ref_params(wl, L)
    orc = ref.score(p, x["cacheK"], x["cacheV"], x["n_v"], x["n"], x["chunkK"], x["chunkV"], x["Q"])
    assert orc["a_v"][:, :, 7].max() < 2.0 ** -140 and orc["a_v"][:, :, 7].min() > 0.0      # the oracle: tiny but positive
    assert orc["psi_v"][:, :, 7].min() > 1e-3
    eng = engine_for(wl)
    src, chunk = dev_objs(x, wl)
    sc = eng.score(src, chunk)
    torch.cuda.synchronize()
    for t in (7, 600):
        assert bool((sc.a_v[:, :, t] == 0).all())
    compare_scores(wl, x["n_v"].numpy(), x["n"].numpy(), scores_to_numpy(sc), orc, TOL[wl.dtype])
    eng.close()
    check_step(wl, x=x)


def test_rescue_cost_is_bounded_when_most_keys_are_flagged():
    """DESIGN.md R31, worst case.  With peaky logits (softmax scale x 40 on one layer of config 2's shape: 21 980 keys x 4 KV
    heads, 7 x 5596 queries each) most keys get less than 2^-100 from all queries together, so most of pass 2's 256-key items
    are redone in the log domain.  On the tensor-core path that is the scoring kernel once more over the flagged items
    (score_tc_kernel<3>), so the column-sum stage (pass 2 + rescue) must stay within a small multiple of its ordinary time
    (asserted: 4 x); the per-key SIMT recompute it replaces cost one warp G x Nn dot products per flagged key.  Parity at rules (a)-(c) against the oracle on the same
    inputs, with 1 CTA per SM and with 3 CTAs in all (every CTA then walks ~100 flagged items)."""
    wl = I.CFG2.replace(L=1)
    x = I.full_inputs(wl)
    c = 40.0 / float(np.sqrt(wl.D))
    check_step(wl, x=x, eng_kw=dict(softmax_scale=c), ref_kw=dict(scale=c), check_rowH=False)
    src, chunk = dev_objs(x, wl)
    ms, share = {}, {}
    for name, kw in (("plain", {}), ("peaky", dict(softmax_scale=c)), ("peaky3", dict(softmax_scale=c, score_ctas=3))):
        eng = engine_for(wl, **kw)
        eng.set_profiling(True)
        sc = eng.new_scores(wl.Nn)
        for _ in range(3):
            eng.score(src, chunk, out=sc)
            torch.cuda.synchronize()
        ms[name] = eng.stage_ms()[0]["colsum"]
        Kv, Ka = wl.n_v + wl.Nn_v, wl.n_a + wl.Nn_a
        tiny = int((sc.a_v[:, :, :Kv] < 2.0 ** -100).sum()) + int((sc.a_a[:, :, :Ka] < 2.0 ** -100).sum())
        share[name] = tiny / float(wl.L * wl.Hkv * (Kv + Ka))
        if name == "peaky":
            ref_psi = sc.psi_v.clone()
        if name == "peaky3":
            assert torch.equal(ref_psi, sc.psi_v)          # results do not depend on which CTA took which flagged item
        eng.close()
    print(f"colsum stage: plain {ms['plain']:.3f} ms, peaky {ms['peaky']:.3f} ms; keys below 2^-100: "
          f"{share['plain']:.3f} / {share['peaky']:.3f}")
    # measured on a B200: 21 % of the keys are below 2^-100 (spread over nearly every 256-key item, so nearly every item is
    # redone) and the stage takes 3.1 x its ordinary time here (2.8 x with all 28 layers, bench.py `rescue_worst`): pass 2
    # once, plus the log-domain pass at 1.8-2.1 x the cost of a pass-2 tile (every exponential on the MUFU, a running maximum)
    assert share["plain"] == 0.0 and share["peaky"] > 0.15
    assert ms["peaky"] <= 4.0 * ms["plain"], ms


# ---------------------------------------------------------------------------------------------- streaming (cfg5 shape logic at cfg1 size)
def test_streaming_free_running_small():
    """Sixty consecutive chunks from an empty cache (append-only steps, first eviction, steady state: the step count of
    BASELINE.json's config 5 at config-1 shapes), both sides free-running on their own state; fp32 so the
    kept sets must stay identical at every step."""
    from paper_2606_07577_b200.omnimem import Chunk
    wl = I.CFG1.replace(n_v=0, n_a=0, budget=300, cache_cap=300, steps=60, recipe="ar1")
    L = wl.L
    eng = engine_for(wl)
    p = ref_params(wl, L)
    B = np.full((L,), wl.budget, np.int32)
    Bt = torch.from_numpy(B).cuda()
    src, dst = eng.new_cache(), eng.new_cache()
    rK = np.zeros((L, wl.Hkv, wl.cache_cap, wl.D), np.float32)
    rV = np.zeros_like(rK)
    r_nv, r_n = np.zeros(L, np.int32), np.zeros(L, np.int32)
    for step in range(wl.steps):
        x = I.full_inputs(wl, step=step, with_cache=False)
        orc = ref.compress_chunk(p, rK, rV, r_nv, r_n, x["chunkK"], x["chunkV"], x["Q"], B)
        rK = orc["dstK"].view(np.float32).reshape(rK.shape)
        rV = orc["dstV"].view(np.float32).reshape(rV.shape)
        r_nv, r_n = orc["n_v_out"], orc["n_out"]
        chunk = Chunk(x["chunkK"].cuda(), x["chunkV"].cuda(), x["Q"].cuda(), wl.Nn_v, wl.Nn_a)
        eng.compress_chunk(src, chunk, Bt, dst)
        src, dst = dst, src
        torch.cuda.synchronize()
        assert np.array_equal(src.n.cpu().numpy(), r_n) and np.array_equal(src.n_v.cpu().numpy(), r_nv), f"step {step}"
        for l in range(L):
            assert np.array_equal(src.k[l, :, :r_n[l]].cpu().numpy(), rK[l, :, :r_n[l]]), f"step {step} layer {l}"
            assert np.array_equal(src.v[l, :, :r_n[l]].cpu().numpy(), rV[l, :, :r_n[l]])
    assert r_n.max() == wl.budget
    eng.close()


def test_error_codes():
    from paper_2606_07577_b200.omnimem import OmniMem, OmniMemError, Chunk
    with pytest.raises(OmniMemError):
        OmniMem(L=1, Hq=3, Hkv=2, D=64, dtype="fp32", cache_cap=8, max_chunk_v=4, max_chunk_a=4)     # Hq % Hkv
    with pytest.raises(OmniMemError):
        OmniMem(L=1, Hq=2, Hkv=2, D=96, dtype="fp32", cache_cap=8, max_chunk_v=4, max_chunk_a=4)     # head_dim
    wl = I.CFG1
    eng = engine_for(wl)
    x = I.full_inputs(wl)
    src, chunk = dev_objs(x, wl)
    big = Chunk(chunk.k, chunk.v, chunk.q, wl.Nn_v + 1, wl.Nn_a)
    with pytest.raises(OmniMemError, match="capacities"):
        eng.score(src, big)
    Bt = torch.full((wl.L,), wl.budget, dtype=torch.int32, device="cuda")
    with pytest.raises(OmniMemError, match="invalid"):
        eng.compress_chunk(src, chunk, Bt, src)                                                   # dst aliases src
    eng.close()


def test_host_entry_matches_device_entry():
    """omnimem_compress_chunk_host (chunk in pinned host memory, copied and compressed in layer groups on two streams)
    must give exactly what omnimem_compress_chunk gives on the same inputs; 9 layers -> groups of 2 with a ragged tail."""
    from paper_2606_07577_b200.omnimem import Chunk
    for wl in (SMALL2.replace(L=9), I.CFG1.replace(L=3)):
        x = I.full_inputs(wl, pin=True)
        eng = engine_for(wl)
        src, chunk = dev_objs(x, wl)
        B = torch.full((wl.L,), wl.budget, dtype=torch.int32, device="cuda")
        dst = eng.new_cache()
        M_v = torch.zeros(wl.L, dtype=torch.int32, device="cuda")
        M_a = torch.zeros_like(M_v)
        eng.compress_chunk(src, chunk, B, dst, M_v=M_v, M_a=M_a)
        host_chunk = Chunk(x["chunkK"], x["chunkV"], x["Q"], wl.Nn_v, wl.Nn_a)
        stage = Chunk(torch.zeros_like(chunk.k), torch.zeros_like(chunk.v), torch.zeros_like(chunk.q), wl.Nn_v, wl.Nn_a)
        dst2 = eng.new_cache()
        hM_v, hM_a = torch.zeros(wl.L, dtype=torch.int32).pin_memory(), torch.zeros(wl.L, dtype=torch.int32).pin_memory()
        for _ in range(2):                                   # twice: the staging buffers are reused across calls
            h2d, d2h = eng.compress_chunk_host(src, host_chunk, stage, B, dst2, hM_v, hM_a)
        assert h2d == sum(t.numel() * t.element_size() for t in (x["chunkK"], x["chunkV"], x["Q"])) and d2h == 8 * wl.L
        assert torch.equal(hM_v, M_v.cpu()) and torch.equal(hM_a, M_a.cpu())
        assert torch.equal(dst2.n, dst.n) and torch.equal(dst2.n_v, dst.n_v)
        for l in range(wl.L):
            nl = int(dst.n[l])
            assert torch.equal(dst2.k[l, :, :nl], dst.k[l, :, :nl]) and torch.equal(dst2.v[l, :, :nl], dst.v[l, :, :nl])
        eng.close()


def test_offline_calibration_and_ragged_layer_budgets():
    """NEXT-2 (R28): statistics of several calibration chunks are accumulated on the device, Eq.13-14 on their
    means give the per-layer table, and the fused step then runs with those RAGGED per-layer totals.  Layers get
    different redundancy (AR(1) rho) so that the table is far from uniform."""
    wl = I.CFG1.replace(L=6, cache_cap=700, budget=300)
    L, n_cal = wl.L, 3
    eng = engine_for(wl, budget_min=120, budget_max=520)
    p = ref_params(wl, L, budget_min=120, budget_max=520)
    acc = eng.new_calibration()
    ref_stats = []
    for c in range(n_cal):
        x = I.full_inputs(wl, step=c)
        for l in range(L):                                   # make the layers differ: a common offset raises the value
            x["cacheV"][l] += 0.3 * l                        # similarity, a larger query scale lowers the entropy
            x["chunkV"][l] += 0.3 * l
            x["Q"][l] *= 0.3 + 0.5 * l
        orc = ref.score(p, x["cacheK"], x["cacheV"], x["n_v"], x["n"], x["chunkK"], x["chunkV"], x["Q"])
        ref_stats.append(orc["stats"])
        src, chunk = dev_objs(x, wl)
        sc = eng.score(src, chunk)
        eng.calibrate_accumulate(sc.stats, acc)
    total = 300 * L
    B_ref, mean_ref = ref.calibrate_budgets(p, np.stack(ref_stats), total)
    B_gpu, mean_gpu = eng.calibrate_budgets(acc, total)
    torch.cuda.synchronize()
    np.testing.assert_allclose(mean_gpu.cpu().numpy()[:, 6:8], mean_ref[:, 6:8], rtol=1e-5, atol=1e-7)
    Bg = B_gpu.cpu().numpy()
    assert Bg.sum() == total == B_ref.sum() and Bg.min() >= 120 and Bg.max() <= 520
    assert np.abs(Bg - B_ref).max() <= 1, f"{Bg} vs {B_ref}"          # statistics agree to 1e-6: at most a rounding flip
    assert Bg.max() - Bg.min() > 50, "calibration inputs should give a visibly non-uniform table"
    # the fused step under the oracle's ragged table: kept sets identical (fp32)
    x = I.full_inputs(wl, step=n_cal)
    orc = ref.compress_chunk(p, x["cacheK"], x["cacheV"], x["n_v"], x["n"], x["chunkK"], x["chunkV"], x["Q"], B_ref)
    src, chunk = dev_objs(x, wl)
    dst = eng.new_cache()
    idx_v, idx_a = eng.new_indices()
    M_v = torch.zeros(L, dtype=torch.int32, device="cuda")
    M_a = torch.zeros_like(M_v)
    eng.compress_chunk(src, chunk, torch.from_numpy(B_ref).cuda(), dst, idx_v=idx_v, idx_a=idx_a, M_v=M_v, M_a=M_a)
    torch.cuda.synchronize()
    assert np.array_equal(M_v.cpu().numpy(), orc["M_v"]) and np.array_equal(dst.n.cpu().numpy(), orc["n_out"])
    assert np.array_equal(dst.n.cpu().numpy(), np.minimum(B_ref, x["n"].numpy() + wl.Nn))
    for l in range(L):
        nl = int(orc["n_out"][l])
        assert np.array_equal(idx_v[l, :, :orc["M_v"][l]].cpu().numpy(), orc["idx_v"][l, :, :orc["M_v"][l]])
        assert np.array_equal(dst.k[l, :, :nl].cpu().view(torch.uint8).numpy(), orc["dstK"][l, :, :nl])
    eng.close()


def test_shared_head_selection_paper_literal():
    """select_scope = 1 (R29: the index sets carry no head index): one score per token and layer, identical
    kept sets for every KV head; rules (a), (b), (c) as for the per-head mode."""
    for wl in (I.CFG1, SMALL2, SMALL3.replace(Hq=8, Hkv=4)):
        check_step(wl, select_scope=1)
    from paper_2606_07577_b200.omnimem import OmniMem
    wl = SMALL3.replace(Hq=8, Hkv=4)
    x = I.full_inputs(wl)
    eng = OmniMem.for_workload(wl, select_scope=1)
    src, chunk = dev_objs(x, wl)
    idx_v, idx_a = eng.new_indices()
    M_v = torch.zeros(wl.L, dtype=torch.int32, device="cuda")
    M_a = torch.zeros_like(M_v)
    dst = eng.new_cache()
    B = torch.full((wl.L,), wl.budget, dtype=torch.int32, device="cuda")
    eng.compress_chunk(src, chunk, B, dst, idx_v=idx_v, idx_a=idx_a, M_v=M_v, M_a=M_a)
    torch.cuda.synchronize()
    for l in range(wl.L):
        mv, ma = int(M_v[l]), int(M_a[l])
        for h in range(1, wl.Hkv):
            assert torch.equal(idx_v[l, h, :mv], idx_v[l, 0, :mv]) and torch.equal(idx_a[l, h, :ma], idx_a[l, 0, :ma])
    eng.close()


def check_hidden_variant(wl, d_model, steps=2):
    """`steps` free-running steps of the hidden-state variant (sim_source = 2, select_scope = 1) against the oracle; returns the
    number of kept indices that differ inside rule (c)'s band."""
    from paper_2606_07577_b200.omnimem import Cache, Chunk, OmniMem
    tol = TOL[wl.dtype]
    L = wl.L
    p = ref_params(wl, L)
    eng = OmniMem.for_workload(wl, select_scope=1, sim_source=2, d_model=d_model)
    B = np.full((L,), wl.budget, np.int32)
    x, hx = I.full_inputs(wl), I.hidden_inputs(wl, d_model)
    rK, rV, rH, r_nv, r_n = x["cacheK"], x["cacheV"], hx["cacheH"], x["n_v"].numpy(), x["n"].numpy()
    src = Cache(rK.cuda(), rV.cuda(), x["n_v"].cuda(), x["n"].cuda(), h=rH.cuda())
    dst = eng.new_cache()
    n_total = 0
    for step in range(steps):
        if step:
            x, hx = I.full_inputs(wl, step=step, with_cache=False), I.hidden_inputs(wl, d_model, step=step, with_cache=False)
        orc = ref.compress_chunk(p, rK, rV, r_nv, r_n, x["chunkK"], x["chunkV"], x["Q"], B, sim_source=2,
                                 select_scope=1, hidden=(rH, hx["chunkH"]))
        chunk = Chunk(x["chunkK"].cuda(), x["chunkV"].cuda(), x["Q"].cuda(), wl.Nn_v, wl.Nn_a, h=hx["chunkH"].cuda())
        sc = eng.new_scores(wl.Nn, want_lse=True)
        idx_v, idx_a = eng.new_indices()
        M_v = torch.zeros(L, dtype=torch.int32, device="cuda")
        M_a = torch.zeros_like(M_v)
        eng.compress_chunk(src, chunk, torch.from_numpy(B).cuda(), dst, out=sc, idx_v=idx_v, idx_a=idx_a, M_v=M_v, M_a=M_a)
        torch.cuda.synchronize()
        compare_scores(wl, r_nv, r_n, scores_to_numpy(sc), orc, tol)
        assert np.array_equal(M_v.cpu().numpy(), orc["M_v"])
        Kv, Ka = seg_lens(wl, r_nv, r_n)
        n_diff = 0
        for l in range(L):
            n_diff += kept_sets_rule_c(f"v[{l}]", idx_v[l, 0].cpu().numpy(), orc["idx_v"][l, 0], int(orc["M_v"][l]),
                                       orc["psi_v"][l, 0, :Kv[l]], tol)
            n_diff += kept_sets_rule_c(f"a[{l}]", idx_a[l, 0].cpu().numpy(), orc["idx_a"][l, 0], int(orc["M_a"][l]),
                                       orc["psi_a"][l, 0, :Ka[l]], tol)
        n_total += n_diff
        for l in range(L):
            nl = int(orc["n_out"][l])
            assert np.array_equal(dst.k[l, :, :nl].cpu().view(torch.uint8).numpy(), orc["dstK"][l, :, :nl])
            assert np.array_equal(dst.h[l, :nl].cpu().view(torch.uint8).numpy(), orc["dstH"][l, :nl]), f"hidden rows, layer {l}"
        # carry the ORACLE's state into the next step on both sides (byte-identical to the GPU's, just asserted)
        dt = wl.torch_dtype
        rK = torch.from_numpy(orc["dstK"].copy()).view(dt).reshape(x["chunkK"].shape[0], wl.Hkv, wl.cache_cap, wl.D)
        rV = torch.from_numpy(orc["dstV"].copy()).view(dt).reshape(rK.shape)
        rH = torch.from_numpy(orc["dstH"].copy()).view(dt).reshape(L, wl.cache_cap, d_model)
        r_nv, r_n = orc["n_v_out"], orc["n_out"]
        src, dst = dst, src
    eng.close()
    return n_total


def test_hidden_state_redundancy_variant():
    """NEXT-3 (R30): Eq.7 on the layer's hidden states (width d_model, one row per token and layer), the
    retained hidden states compacted with the kept tokens.  Needs select_scope = 1.  Rules (a)/(c) on the fused step,
    byte-exact K/V/H rows, and a second free-running step on the compacted state."""
    from paper_2606_07577_b200.omnimem import Cache, Chunk, OmniMem, OmniMemError
    for wl, d_model in ((I.CFG1, 96), (SMALL3.replace(Hq=8, Hkv=4), 328),        # 328 * 2 B = 656 B: ragged 512-byte steps
                        (SMALL2.replace(Hq=8, Hkv=4), 328), (SMALL2, 3584)):      # neighbour distance 1: the streaming kernel
        assert check_hidden_variant(wl, d_model) == 0, "these sizes are expected to agree exactly"
    with pytest.raises(OmniMemError):                          # hidden states have no head index: per-head sets are refused
        OmniMem.for_workload(I.CFG1, select_scope=0, sim_source=2, d_model=96)
    eng = OmniMem.for_workload(I.CFG1, select_scope=1, sim_source=2, d_model=96)
    x = I.full_inputs(I.CFG1)
    src, chunk = dev_objs(x, I.CFG1)
    with pytest.raises(OmniMemError, match="invalid"):
        eng.score(src, chunk)                                  # cache.h / chunk.h missing
    eng.close()


def test_time_interleaved_chunk():
    """NEXT-4b (R25'): chunk rows in true temporal order with a per-row modality map: causal mask by true position,
    segments gathered through the map.  All of rules (a), (b), (c) on the tcgen05, SIMT and fp32 paths, plus the host
    entry (the map travels from host memory)."""
    check_step(I.CFG1, modality=I.modality_pattern(I.CFG1, 7))
    check_step(SMALL2, modality=I.modality_pattern(SMALL2, 9))
    check_step(SMALL3, modality=I.modality_pattern(SMALL3, 1000))                  # alternating single rows
    check_step(SMALL2, modality=I.modality_pattern(SMALL2, 5), eng_kw=dict(score_path=1))
    check_step(SMALL4, modality=I.modality_pattern(SMALL4, 3), eng_kw=dict(causal=0), ref_kw=dict(causal=0))
    from paper_2606_07577_b200.omnimem import Chunk
    wl = SMALL2.replace(L=3)
    mod = I.modality_pattern(wl, 6)
    x = I.interleave(I.full_inputs(wl, pin=True), mod, wl.Nn_v)
    eng = engine_for(wl)
    src, chunk = dev_objs(x, wl)
    chunk.modality = mod.cuda()
    B = torch.full((wl.L,), wl.budget, dtype=torch.int32, device="cuda")
    dst, dst2 = eng.new_cache(), eng.new_cache()
    eng.compress_chunk(src, chunk, B, dst)
    host_chunk = Chunk(x["chunkK"].pin_memory(), x["chunkV"].pin_memory(), x["Q"].pin_memory(), wl.Nn_v, wl.Nn_a, modality=mod.pin_memory())
    stage = Chunk(torch.zeros_like(chunk.k), torch.zeros_like(chunk.v), torch.zeros_like(chunk.q), wl.Nn_v, wl.Nn_a,
                  modality=torch.zeros_like(chunk.modality))
    hM_v, hM_a = torch.zeros(wl.L, dtype=torch.int32).pin_memory(), torch.zeros(wl.L, dtype=torch.int32).pin_memory()
    eng.compress_chunk_host(src, host_chunk, stage, B, dst2, hM_v, hM_a)
    assert torch.equal(dst2.n, dst.n) and torch.equal(dst2.k, dst.k) and torch.equal(dst2.v, dst.v)
    eng.close()


@pytest.mark.parametrize("seed", range(int(os.environ.get("OMNIMEM_FUZZ_SEEDS", "8"))))
def test_random_shapes_fuzz(seed):
    """Seeded random shapes around the tile edges (128-row tiles, 256-row CTAs, the 16-slot lse ring, ragged caches,
    tiny budgets, strides, both modalities possibly empty, optional interleaving / shared selection): rules (a)-(c)."""
    g = np.random.default_rng(1000 + seed)
    for rep in range(4):
        bf16 = bool(g.integers(0, 2))
        Hkv = int(g.integers(1, 4))
        G = int(g.choice([1, 2, 4, 7]))
        big = rep == 3                                     # one larger case per seed: several CTAs along x, > 16 tiles
        Nn_v, Nn_a = int(g.integers(0, 1400 if big else 600)), int(g.integers(0, 200))
        if Nn_v + Nn_a == 0:
            Nn_v = 1
        n_v, n_a = int(g.integers(0, 2600 if big else 900)), int(g.integers(0, 300))
        cap = n_v + n_a + int(g.integers(0, 64))
        budget = int(g.integers(1, max(2, cap + 1)))
        cap = max(cap, budget, 1)
        base = SMALL3 if bf16 else I.CFG1
        wl = base.replace(L=int(g.integers(1, 3)), Hq=Hkv * G, Hkv=Hkv, n_v=n_v, n_a=n_a, Nn_v=Nn_v, Nn_a=Nn_a, budget=budget,
                          cache_cap=cap, sim_stride_v=int(g.choice([1, 1, 16, 256])), sim_stride_a=int(g.choice([1, 3])))
        causal = int(g.integers(0, 2))
        scope = int(g.integers(0, 2))
        mod = I.modality_pattern(wl, int(g.integers(1, 12))) if g.integers(0, 2) and Nn_v and Nn_a else None
        ctas = int(g.choice([0, 0, 1, 2, 5]))              # persistent scoring CTAs (0 = one per SM)
        check_step(wl, eng_kw=dict(causal=causal, score_ctas=ctas), ref_kw=dict(causal=causal), select_scope=scope, modality=mod,
                   check_rowH=bool(g.integers(0, 2)))


def test_fused_step_captures_into_a_cuda_graph():
    """The fused call only enqueues work on the given stream (no host synchronisation, no allocation): it can be
    captured once and replayed; the replay must reproduce the eager result byte for byte, also after the inputs changed."""
    for wl in (I.CFG1, SMALL2):
        eng = engine_for(wl)
        x = I.full_inputs(wl)
        src, chunk = dev_objs(x, wl)
        B = torch.full((wl.L,), wl.budget, dtype=torch.int32, device="cuda")
        dst_e, dst_g = eng.new_cache(), eng.new_cache()
        eng.compress_chunk(src, chunk, B, dst_g)                      # warm-up outside the capture (attributes, tensor maps)
        torch.cuda.synchronize()
        g = torch.cuda.CUDAGraph()
        with torch.cuda.graph(g):
            eng.compress_chunk(src, chunk, B, dst_g)
        for step in (0, 1):
            if step:                                                  # new chunk contents in the SAME buffers
                y = I.full_inputs(wl, step=1)
                chunk.k.copy_(y["chunkK"].cuda()); chunk.v.copy_(y["chunkV"].cuda()); chunk.q.copy_(y["Q"].cuda())
            dst_g.k.zero_(); dst_g.v.zero_()
            g.replay()
            eng.compress_chunk(src, chunk, B, dst_e)
            torch.cuda.synchronize()
            assert torch.equal(dst_g.n, dst_e.n) and torch.equal(dst_g.n_v, dst_e.n_v)
            for l in range(wl.L):
                nl = int(dst_e.n[l])
                assert torch.equal(dst_g.k[l, :, :nl], dst_e.k[l, :, :nl]) and torch.equal(dst_g.v[l, :, :nl], dst_e.v[l, :, :nl])
        eng.close()
