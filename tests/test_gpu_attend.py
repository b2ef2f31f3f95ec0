"""GPU parity of omnimem_attend (Eq.1) against the fp64 oracle's omnimem_ref_mhsa.

Tolerances: LSE at rule (a) (absolute tol: an LSE error is a relative error of every exp(z - lse)).
Y: the bf16 kernel rounds every weight p to bf16 before P V (bf16 keeps 8 significant bits: relative error <= 2^-8 just
above a power of two, 2^-9 just below) and rounds Y once to bf16 (<= 2^-8 |Y|), so the rigorous bound is
|Y_gpu - Y_ref| <= 2^-8 sum_k p_k |v_k| + 2^-8 |Y| <= 2^-7 * sum_k p_k |v_k| (the oracle returns that magnitude, absY);
it is attained when one key takes the whole row (p ~ 1, Y ~ v).  fp32 inputs: 1e-5 of the same magnitude.
Then the point of the row: attend -> compress_chunk(lse = ...) must keep what the two-pass step keeps.
"""
import os

import numpy as np
import pytest
import torch

from oracle import ref
from paper_2606_07577_b200 import inputs as I
from tests.test_gpu_parity import SMALL2, SMALL3, SMALL4, dev_objs, engine_for
from tests.util import TOL, compare_scores, ref_params, scores_to_numpy

pytestmark = pytest.mark.gpu

Y_TOL = {"fp32": 1e-5, "bf16": 2.0 ** -7}


def compare_attend(wl, y_gpu, lse_gpu, Y_ref, lse_ref, absY, what=""):
    tol = TOL[wl.dtype]
    err_l = np.abs(lse_gpu.astype(np.float64) - lse_ref)
    assert err_l.max() <= tol * np.maximum(1.0, np.abs(lse_ref)).max(), f"{what} lse: max err {err_l.max():.3e}"
    assert np.all(err_l <= tol * np.maximum(1.0, np.abs(lse_ref))), f"{what} lse: max err {err_l.max():.3e}"
    err = np.abs(y_gpu.astype(np.float64) - Y_ref)
    bound = Y_TOL[wl.dtype] * absY + 1e-30
    bad = err > bound
    if bad.any():
        i = np.unravel_index(np.argmax(err / bound), err.shape)
        raise AssertionError(f"{what} Y: {int(bad.sum())}/{bad.size} outside the bound; worst at {i}: got {y_gpu[i]!r} exp "
                             f"{Y_ref[i]!r} bound {bound[i]:.3e}")
    return float((err / bound).max())


def check_attend(wl, x=None, eng_kw=None, ref_kw=None, also_compress=True):
    eng_kw, ref_kw = dict(eng_kw or {}), dict(ref_kw or {})
    x = x if x is not None else I.full_inputs(wl)
    L = x["Q"].shape[0]
    wl = wl.replace(L=L)
    p = ref_params(wl, L, **ref_kw)
    Y_ref, lse_ref, absY = ref.mhsa(p, x["cacheK"], x["cacheV"], x["n"], x["chunkK"], x["chunkV"], x["Q"], want_abs=True)
    eng = engine_for(wl, **eng_kw)
    src, chunk = dev_objs(x, wl)
    y, lse = eng.attend(src, chunk)
    torch.cuda.synchronize()
    worst = compare_attend(wl, y.float().cpu().numpy(), lse.cpu().numpy(), Y_ref, lse_ref, absY, wl.name)
    if also_compress and wl.Nn:
        from paper_2606_07577_b200.omnimem import Chunk
        B = torch.full((L,), wl.budget, dtype=torch.int32, device="cuda")
        out = []
        for ch in (chunk, Chunk(chunk.k, chunk.v, chunk.q, wl.Nn_v, wl.Nn_a, lse=lse)):     # two-pass, then forward + one pass
            dst = eng.new_cache()
            iv, ia = eng.new_indices()
            sc = eng.new_scores(wl.Nn)
            M_v = torch.zeros(L, dtype=torch.int32, device="cuda")
            M_a = torch.zeros_like(M_v)
            eng.set_profiling(True)
            eng.compress_chunk(src, ch, B, dst, out=sc, idx_v=iv, idx_a=ia, M_v=M_v, M_a=M_a)
            torch.cuda.synchronize()
            ms, _ = eng.stage_ms()
            out.append((dst, iv, ia, M_v, M_a, sc, ms))
        assert out[0][6]["lse"] > 0.0 and out[1][6]["lse"] == 0.0                           # pass 1 really was skipped
        orc = ref.score(p, x["cacheK"], x["cacheV"], x["n_v"], x["n"], x["chunkK"], x["chunkV"], x["Q"])
        compare_scores(wl, x["n_v"].numpy(), x["n"].numpy(), scores_to_numpy(out[1][5]), orc, TOL[wl.dtype])
        assert torch.equal(out[0][3], out[1][3]) and torch.equal(out[0][4], out[1][4])
        same = 0
        for l in range(L):
            mv, ma = int(out[0][3][l]), int(out[0][4][l])
            same += int((out[0][1][l, :, :mv] != out[1][1][l, :, :mv]).sum()) + int((out[0][2][l, :, :ma] != out[1][2][l, :, :ma]).sum())
        assert same == 0, f"{same} kept indices differ between the two-pass step and forward + one pass"
    eng.close()
    return worst


def test_attend_cfg1_fp32():
    check_attend(I.CFG1)
    check_attend(I.CFG1, eng_kw=dict(causal=0), ref_kw=dict(causal=0))


@pytest.mark.parametrize("wl", [SMALL2, SMALL3, SMALL4], ids=lambda w: w.name)
def test_attend_bf16_tcgen05_small(wl):
    check_attend(wl)
    check_attend(wl, eng_kw=dict(causal=0), ref_kw=dict(causal=0))


@pytest.mark.parametrize("ctas", [1, 2, 5])
def test_attend_persistent_ctas_walk_several_items(ctas):
    """The tcgen05 forward is persistent: with `score_ctas` CTAs every CTA of these small shapes walks several items, so the
    K / V ring, the S / P / O barrier phases of each sub-tile, the Q-free and O-free hand-overs and the item queue carry
    across items, including ragged last blocks (one sub-tile without rows) and an empty cache."""
    for wl in (SMALL2, SMALL3, SMALL4):
        for n_v in (wl.n_v, wl.n_v - 37, 0):
            check_attend(wl.replace(n_v=n_v), eng_kw=dict(score_ctas=ctas), also_compress=(n_v == wl.n_v))
    check_attend(SMALL2, eng_kw=dict(score_ctas=ctas, causal=0), ref_kw=dict(causal=0), also_compress=False)
    check_attend(SMALL3.replace(n_v=1, n_a=0, Nn_v=257, Nn_a=0, cache_cap=300, budget=258), eng_kw=dict(score_ctas=ctas),
                 also_compress=False)


@pytest.mark.parametrize("seed", range(int(os.environ.get("OMNIMEM_FUZZ_SEEDS", "6"))))
def test_attend_random_shapes_fuzz(seed):
    """Seeded random shapes around the tile edges (128-row tiles, 256-row items, ragged caches, GQA widths), causal or not,
    with 1-5 persistent CTAs or one per SM: Y and LSE against the oracle."""
    g = np.random.default_rng(7000 + seed)
    for rep in range(3):
        Hkv = int(g.integers(1, 3))
        G = int(g.choice([1, 2, 4, 7]))
        Nn_v, Nn_a = int(g.integers(0, 700)), int(g.integers(0, 150))
        if Nn_v + Nn_a == 0:
            Nn_v = 1
        n_v, n_a = int(g.integers(0, 1200)), int(g.integers(0, 200))
        cap = n_v + n_a + int(g.integers(1, 64))
        wl = SMALL3.replace(L=int(g.integers(1, 3)), Hq=Hkv * G, Hkv=Hkv, n_v=n_v, n_a=n_a, Nn_v=Nn_v, Nn_a=Nn_a,
                            budget=max(1, cap // 2), cache_cap=cap)
        causal = int(g.integers(0, 2))
        check_attend(wl, eng_kw=dict(causal=causal, score_ctas=int(g.choice([0, 1, 2, 5]))), ref_kw=dict(causal=causal),
                     also_compress=False)


def test_attend_bf16_simt_paths():
    check_attend(SMALL2, eng_kw=dict(score_path=1))
    check_attend(SMALL2.replace(D=64))


def test_attend_edge_shapes():
    check_attend(SMALL2.replace(n_v=0, n_a=0))                                                  # empty cache: first chunk of a stream
    check_attend(SMALL2.replace(Nn_v=1, Nn_a=0))                                                # one-token chunk
    check_attend(SMALL2.replace(n_v=128, n_a=128, Nn_v=128, Nn_a=128, budget=256, cache_cap=256))   # tile-aligned everywhere
    check_attend(SMALL3.replace(n_v=1000, n_a=24, Nn_v=256, Nn_a=0, cache_cap=1100, budget=1100))   # one full CTA of queries
    check_attend(SMALL3.replace(n_v=1, n_a=0, Nn_v=257, Nn_a=0, cache_cap=300, budget=258))         # a second CTA with one row
    check_attend(SMALL3.replace(n_v=700, n_a=100, Nn_v=600, Nn_a=170, cache_cap=1700, budget=1000, Hq=14, Hkv=2))  # G = 7


def test_attend_needs_no_workspace():
    """omnimem_attend uses no scratch: NULL / 0 for ws is accepted (a model that only wants the forward and its LSE need not
    allocate the compression workspace) and gives bit-identical results to a call that passes one."""
    import ctypes as C
    for wl, kw in ((SMALL2, {}), (I.CFG1, {})):                 # tcgen05 and SIMT forward
        x = I.full_inputs(wl)
        eng = engine_for(wl, **kw)
        src, chunk = dev_objs(x, wl)
        y0, lse0 = eng.attend(src, chunk)
        y1, lse1 = torch.full_like(y0, float("nan")), torch.full_like(lse0, float("nan"))
        cs, cc = src.c(), chunk.c()
        rc = eng.lib.omnimem_attend(eng.ctx, C.byref(cs), C.byref(cc), C.c_void_p(y1.data_ptr()), C.c_void_p(lse1.data_ptr()),
                                    None, 0, C.c_void_p(torch.cuda.current_stream().cuda_stream))
        torch.cuda.synchronize()
        assert rc == 0
        assert torch.equal(y0, y1) and torch.equal(lse0, lse1)
        eng.close()


def test_attend_ignores_rows_beyond_n():
    """Rows n .. cache_cap of the cache buffers may hold anything (stale rows, NaN bit patterns): masked key columns are
    selected away and the value rows of the ragged last cache tile are zeroed in shared memory before P V."""
    wl = SMALL2.replace(cache_cap=1100)
    x = I.full_inputs(wl)
    nc = wl.n_v + wl.n_a
    x["cacheK"][:, :, nc:] = float("nan")
    x["cacheV"][:, :, nc:] = float("nan")
    x["cacheV"][:, :, nc + 1] = float("inf")
    L = wl.L
    p = ref_params(wl, L)
    clean = {k: (v.clone() if torch.is_tensor(v) else v) for k, v in x.items()}
    clean["cacheK"][:, :, nc:] = 0
    clean["cacheV"][:, :, nc:] = 0
    Y_ref, lse_ref, absY = ref.mhsa(p, clean["cacheK"], clean["cacheV"], x["n"], x["chunkK"], x["chunkV"], x["Q"], want_abs=True)
    eng = engine_for(wl)
    src, chunk = dev_objs(x, wl)
    y, lse = eng.attend(src, chunk)
    torch.cuda.synchronize()
    assert bool(torch.isfinite(y.float()).all()) and bool(torch.isfinite(lse).all())
    compare_attend(wl, y.float().cpu().numpy(), lse.cpu().numpy(), Y_ref, lse_ref, absY)
    eng.close()


@pytest.mark.parametrize("mult", [12.0, 40.0])
def test_attend_wide_logits_rebase_the_reference(mult):
    """Keys with 64 x the norm in the first cache tile, the last cache tile and the chunk, softmax scale x 12 / x 40: the
    lazy reference overflows in the middle of a row, the thread re-bases and rescales its O row in tensor memory."""
    for wl in (SMALL2, SMALL3):
        x = I.full_inputs(wl)
        nc = wl.n_v + wl.n_a
        x["cacheK"][:, :, 5] *= 64.0
        x["cacheK"][:, :, nc - 3] *= 64.0
        x["chunkK"][:, :, wl.Nn // 2] *= 64.0
        c = mult / float(np.sqrt(wl.D))
        check_attend(wl, x=x, eng_kw=dict(softmax_scale=c), ref_kw=dict(scale=c), also_compress=False)


def oracle_one_kv_head(wl, x, l, h):
    """The oracle's Eq.1 on the G query heads of KV head h of layer slot l (query heads are independent given their KV head)."""
    G = wl.G
    p = ref_params(wl.replace(Hq=G, Hkv=1), 1)
    sl = lambda t, a, b: t[l:l + 1, a:b]
    return ref.mhsa(p, sl(x["cacheK"], h, h + 1), sl(x["cacheV"], h, h + 1), x["n"][l:l + 1], sl(x["chunkK"], h, h + 1),
                    sl(x["chunkV"], h, h + 1), sl(x["Q"], h * G, (h + 1) * G), want_abs=True)


@pytest.mark.parametrize("wl,samples", [(I.CFG2, ((0, 0), (14, 3), (27, 1))), (I.CFG4, ((0, 7), (35, 2))), (I.CFG3, ((35, 5),))],
                         ids=["cfg2", "cfg4", "cfg3"])
def test_attend_full_size(wl, samples):
    """BASELINE.json's full sizes in the launch configuration bench.py times (one omnimem_attend over all layers): sampled
    (layer, KV head) units in full against the oracle; every row of every layer: finite, and the LSE equal to the one
    score pass 1 computes up to the two kernels' exponential error: each puts a different quarter of a row's terms on the
    degree-3 polynomial (relative error <= 7.5e-5, tc_ptx.cuh), so a row whose mass sits on one key (config 4's x4
    outliers) can differ by 2 x 7.5e-5 in ln Z, plus fp32 rounding of an LSE of ~15 (1.488e-4 is what config 4 shows).
    Rule (a) against the oracle (2e-3) is checked below on the sampled units."""
    from paper_2606_07577_b200.omnimem import Cache, Chunk, OmniMem
    x = I.full_inputs(wl)
    eng = OmniMem.for_workload(wl)
    dev = eng.device
    src = Cache(x["cacheK"].to(dev), x["cacheV"].to(dev), x["n_v"].to(dev), x["n"].to(dev))
    chunk = Chunk(x["chunkK"].to(dev), x["chunkV"].to(dev), x["Q"].to(dev), wl.Nn_v, wl.Nn_a)
    y, lse = eng.attend(src, chunk)
    torch.cuda.synchronize()
    assert bool(torch.isfinite(lse).all()) and bool(torch.isfinite(y.float()).all())
    sc = eng.score(src, chunk, want_lse=True)
    torch.cuda.synchronize()
    assert float((sc.lse - lse).abs().max()) < 2 * 7.5e-5 + 1e-5
    G = wl.G
    worst = 0.0
    for l, h in samples:
        Y_ref, lse_ref, absY = oracle_one_kv_head(wl, x, l, h)
        worst = max(worst, compare_attend(wl, y[l:l + 1, h * G:(h + 1) * G].float().cpu().numpy(),
                                          lse[l:l + 1, h * G:(h + 1) * G].cpu().numpy(), Y_ref, lse_ref, absY,
                                          f"{wl.name} layer {l} kv head {h}"))
    print(f"{wl.name}: worst |dY| / sum_k p_k |v_k| = {worst * Y_TOL[wl.dtype]:.3e} (bound {Y_TOL[wl.dtype]:.3e})")
    # the point of the row at full size: forward + one-pass compression keeps what the two-pass step keeps, on EVERY layer
    # (the two LSEs differ by up to 1.5e-4, i.e. psi by lambda x that = 3e-6 relative: only exact near-ties at the threshold
    # can flip, and rule (c) allows those)
    from paper_2606_07577_b200.omnimem import Chunk
    B = torch.full((wl.L,), wl.budget, dtype=torch.int32, device=dev)
    res = []
    for ch in (chunk, Chunk(chunk.k, chunk.v, chunk.q, wl.Nn_v, wl.Nn_a, lse=lse)):
        dst = eng.new_cache()
        iv, ia = eng.new_indices()
        M_v = torch.zeros(wl.L, dtype=torch.int32, device=dev)
        M_a = torch.zeros_like(M_v)
        sc2 = eng.new_scores(wl.Nn)
        eng.compress_chunk(src, ch, B, dst, out=sc2, idx_v=iv, idx_a=ia, M_v=M_v, M_a=M_a)
        torch.cuda.synchronize()
        res.append((iv, ia, M_v, M_a, sc2))
    assert torch.equal(res[0][2], res[1][2]) and torch.equal(res[0][3], res[1][3])
    n_flip, n_kept = 0, 0
    for l in range(wl.L):
        mv, ma = int(res[0][2][l]), int(res[0][3][l])
        for which, m in ((0, mv), (1, ma)):
            a_idx, b_idx = res[0][which][l, :, :m], res[1][which][l, :, :m]
            if torch.equal(a_idx, b_idx):
                n_kept += a_idx.numel()
                continue
            psi = (res[0][4].psi_v if which == 0 else res[0][4].psi_a)[l]
            for h in range(wl.Hkv):
                sa, sb = set(a_idx[h].tolist()), set(b_idx[h].tolist())
                diff = sorted(sa ^ sb)
                n_kept += len(sa)
                if diff:
                    tau = float(psi[h][torch.tensor(sorted(sa), device=dev)].min())
                    worst = float((psi[h][torch.tensor(diff, device=dev)] - tau).abs().max())
                    assert worst <= 2e-3 * tau, f"layer {l} head {h}: kept sets differ away from the threshold ({worst} vs tau {tau})"
                    n_flip += len(diff) // 2
    print(f"{wl.name}: forward + one pass vs two-pass: {n_flip} of {n_kept} kept indices differ (all within rule (c) of the threshold)")
    assert n_flip <= 1e-4 * n_kept
    eng.close()
