"""Pins of the fp64 oracle (oracle/omnimem_ref.c) against things other than itself.

Each test names the passage of PAPER.md (P:<line>) or the DESIGN.md reading (R<k>) it pins and the kind of
pin: a closed form, an invariant, a library routine on a special case, or brute force on a tiny input.
They are chosen so that a plausible slip in the oracle (dropped term, wrong sign or index, transposed
operand, wrong head mapping, off-by-one in the causal mask or in the segment maps) fails at least one.
"""
import itertools
import math
import os

import numpy as np
import pytest
import torch

from oracle import ref
from paper_2606_07577_b200 import inputs as I

GOLD = os.path.join(os.path.dirname(__file__), "golden")
torch.manual_seed(0)


def rnd(*shape, seed=0, scale=1.0):
    g = torch.Generator().manual_seed(seed)
    return (scale * torch.randn(*shape, generator=g, dtype=torch.float64)).numpy()


def make(L=1, Hq=4, Hkv=2, D=8, cap=12, n=(9,), n_v=(6,), Nn_v=5, Nn_a=3, seed=0, **kw):
    p = ref.RefParams(L=L, Hq=Hq, Hkv=Hkv, D=D, cache_cap=cap, Nn_v=Nn_v, Nn_a=Nn_a, **kw)
    x = dict(cacheK=rnd(L, Hkv, cap, D, seed=seed + 1), cacheV=rnd(L, Hkv, cap, D, seed=seed + 2),
             chunkK=rnd(L, Hkv, p.Nn, D, seed=seed + 3), chunkV=rnd(L, Hkv, p.Nn, D, seed=seed + 4),
             Q=rnd(L, Hq, p.Nn, D, seed=seed + 5), n=np.array(n, np.int32), n_v=np.array(n_v, np.int32))
    return p, x


# ------------------------------------------------------------------------------------------ O2 (Eq.6)
def torch_attention(p, x, l):
    """Library special case: torch fp64 softmax over the concatenated keys + causal mask, summed over rows."""
    Nc, Nn, G = int(x["n"][l]), p.Nn, p.Hq // p.Hkv
    a = torch.zeros(p.Hkv, Nc + Nn, dtype=torch.float64)
    lse = torch.zeros(p.Hq, Nn, dtype=torch.float64)
    ent = torch.zeros(p.Hq, Nn, dtype=torch.float64)
    for j in range(p.Hq):
        h = j // G
        K = torch.cat([torch.from_numpy(x["cacheK"][l, h, :Nc]), torch.from_numpy(x["chunkK"][l, h])], 0)
        z = torch.from_numpy(x["Q"][l, j]) @ K.T / math.sqrt(p.D)
        if p.causal:
            mask = torch.ones(Nn, Nc + Nn, dtype=torch.bool)
            mask[:, Nc:] = torch.tril(torch.ones(Nn, Nn, dtype=torch.bool))
            z = z.masked_fill(~mask, -float("inf"))
        P = torch.softmax(z, -1)
        a[h] += P.sum(0)
        lse[j] = torch.logsumexp(z, -1)
        ent[j] = -(torch.where(P > 0, P * torch.log(P), torch.zeros_like(P))).sum(-1)
    return a.numpy(), lse.numpy(), ent.numpy()


@pytest.mark.parametrize("causal", [1, 0])
@pytest.mark.parametrize("shape", [dict(), dict(Hq=6, Hkv=2, D=16, cap=20, n=(13,), n_v=(8,), Nn_v=7, Nn_a=2),
                                   dict(L=2, Hq=2, Hkv=2, D=4, cap=5, n=(5, 0), n_v=(2, 0), Nn_v=1, Nn_a=6)])
def test_attention_matches_torch_softmax(causal, shape):
    p, x = make(causal=causal, **shape)
    a_log, lse, rowH = ref.attention(p, x["cacheK"], x["n"], x["chunkK"], x["Q"])
    for l in range(p.L):
        a_t, lse_t, ent_t = torch_attention(p, x, l)
        Nk = int(x["n"][l]) + p.Nn
        np.testing.assert_allclose(a_log[l, :, :Nk], a_t, rtol=1e-12, atol=1e-14)
        assert np.all(a_log[l, :, Nk:] == 0)
        np.testing.assert_allclose(lse[l], lse_t, rtol=1e-12)
        np.testing.assert_allclose(rowH[l], ent_t, rtol=1e-10, atol=1e-13)


def test_attention_rows_sum_to_one():
    """Softmax rows sum to 1 => sum_k a[l,h,k] = G * Nq (NS invariant; Eq.6)."""
    p, x = make(Hq=6, Hkv=2, D=16, cap=40, n=(33,), n_v=(20,), Nn_v=11, Nn_a=4)
    a_log, _, _ = ref.attention(p, x["cacheK"], x["n"], x["chunkK"], x["Q"])
    np.testing.assert_allclose(a_log.sum(-1), (p.Hq // p.Hkv) * p.Nn, rtol=1e-13)


def test_attention_zero_query_harmonic_golden():
    """Closed form, tests/golden/harmonic_causal.txt (Q = 0, causal R3, GQA sum R5)."""
    line = [ln for ln in open(os.path.join(GOLD, "harmonic_causal.txt")) if not ln.startswith("#")][0]
    left, right = line.split("|")
    G, Nc, Nn = map(int, left.split())
    exp = np.array(list(map(float, right.split())))
    p, x = make(Hq=G, Hkv=1, D=4, cap=Nc + 2, n=(Nc,), n_v=(1,), Nn_v=Nn - 1, Nn_a=1)
    x["Q"][:] = 0
    a_log, lse, _ = ref.attention(p, x["cacheK"], x["n"], x["chunkK"], x["Q"])
    np.testing.assert_allclose(a_log[0, 0, :Nc], exp[0], rtol=1e-14)
    np.testing.assert_allclose(a_log[0, 0, Nc:Nc + Nn], exp[1:], rtol=1e-14)
    np.testing.assert_allclose(lse[0, 0], np.log(Nc + 1 + np.arange(Nn)), rtol=1e-14)


def test_attention_zero_query_noncausal_uniform():
    p, x = make(causal=0)
    x["Q"][:] = 0
    a_log, _, rowH = ref.attention(p, x["cacheK"], x["n"], x["chunkK"], x["Q"])
    Nk = 9 + p.Nn
    np.testing.assert_allclose(a_log[0, :, :Nk], (p.Hq // p.Hkv) * p.Nn / Nk, rtol=1e-14)
    np.testing.assert_allclose(rowH, math.log(Nk), rtol=1e-13)   # uniform attention: entropy = ln Nk


def test_attention_rational_golden():
    """Closed form, tests/golden/rational_softmax.txt: exact rational softmax, pins the causal off-by-one."""
    gold = {ln.split()[0]: np.array(list(map(float, ln.split()[1:])))
            for ln in open(os.path.join(GOLD, "rational_softmax.txt")) if not ln.startswith("#")}
    p = ref.RefParams(L=1, Hq=1, Hkv=1, D=1, cache_cap=1, Nn_v=1, Nn_a=1, scale=1.0)
    a_log, lse, rowH = ref.attention(p, np.zeros((1, 1, 1, 1)), np.array([1], np.int32),
                                     np.log(np.array([2.0, 3.0])).reshape(1, 1, 2, 1), np.ones((1, 1, 2, 1)))
    np.testing.assert_allclose(a_log[0, 0], gold["a"], rtol=1e-14)
    np.testing.assert_allclose(lse[0, 0], gold["lse"], rtol=1e-14)
    np.testing.assert_allclose(rowH[0, 0], gold["rowH"], rtol=1e-13)


def test_attention_dominant_key_takes_all_mass():
    p, x = make(causal=0)
    x["cacheK"][0, 1, 4] = 50.0 * np.sign(x["Q"][0, 2:4].sum((0, 1)))   # aligned with head 1's queries
    x["Q"][0, 2:4] = np.abs(x["Q"][0, 2:4]) * np.sign(x["cacheK"][0, 1, 4])
    a_log, _, _ = ref.attention(p, x["cacheK"], x["n"], x["chunkK"], x["Q"])
    assert abs(a_log[0, 1, 4] - 2 * p.Nn) < 1e-6


def test_attention_gqa_head_mapping():
    """R5: query head j reads KV head j // G.  Zeroing the queries of one group flattens only its KV head."""
    p, x = make(Hq=6, Hkv=3, causal=0)
    x["Q"][0, 2:4] = 0                                    # group of KV head 1
    a_log, _, _ = ref.attention(p, x["cacheK"], x["n"], x["chunkK"], x["Q"])
    Nk = 9 + p.Nn
    np.testing.assert_allclose(a_log[0, 1, :Nk], 2 * p.Nn / Nk, rtol=1e-14)
    assert np.std(a_log[0, 0, :Nk]) > 1e-3 and np.std(a_log[0, 2, :Nk]) > 1e-3


def test_attention_ignores_rows_beyond_n():
    p, x = make()
    a1, l1, _ = ref.attention(p, x["cacheK"], x["n"], x["chunkK"], x["Q"])
    x["cacheK"][:, :, 9:] = 1e6
    a2, l2, _ = ref.attention(p, x["cacheK"], x["n"], x["chunkK"], x["Q"])
    np.testing.assert_allclose(a1, a2, rtol=1e-13)     # thread-order rounding only
    assert np.array_equal(l1, l2)


# ------------------------------------------------------------------------------------------ A1 (Eq.1, NEXT-1)
def torch_mhsa(p, x, l):
    """Library special case: torch fp64 softmax(QK^T c + mask) @ V over the concatenated keys / values."""
    Nc, Nn, G = int(x["n"][l]), p.Nn, p.Hq // p.Hkv
    Y = torch.zeros(p.Hq, Nn, p.D, dtype=torch.float64)
    for j in range(p.Hq):
        h = j // G
        K = torch.cat([torch.from_numpy(x["cacheK"][l, h, :Nc]), torch.from_numpy(x["chunkK"][l, h])], 0)
        V = torch.cat([torch.from_numpy(x["cacheV"][l, h, :Nc]), torch.from_numpy(x["chunkV"][l, h])], 0)
        mask = torch.ones(Nn, Nc + Nn, dtype=torch.bool)
        if p.causal:
            mask[:, Nc:] = torch.tril(torch.ones(Nn, Nn, dtype=torch.bool))
        Y[j] = torch.nn.functional.scaled_dot_product_attention(torch.from_numpy(x["Q"][l, j])[None], K[None], V[None],
                                                                attn_mask=mask[None], scale=1.0 / math.sqrt(p.D))[0]
    return Y.numpy()


@pytest.mark.parametrize("causal", [1, 0])
@pytest.mark.parametrize("shape", [dict(), dict(Hq=6, Hkv=2, D=16, cap=20, n=(13,), n_v=(8,), Nn_v=7, Nn_a=2),
                                   dict(L=2, Hq=2, Hkv=2, D=4, cap=5, n=(5, 0), n_v=(2, 0), Nn_v=1, Nn_a=6)])
def test_mhsa_matches_torch_sdpa(causal, shape):
    """Eq.1: Y against torch's fp64 scaled_dot_product_attention with the explicit mask of R3; the LSE it returns
    is the one O2 returns (one routine cannot drift from the other); absY bounds |Y|."""
    p, x = make(causal=causal, **shape)
    Y, lse, absY = ref.mhsa(p, x["cacheK"], x["cacheV"], x["n"], x["chunkK"], x["chunkV"], x["Q"], want_abs=True)
    for l in range(p.L):
        np.testing.assert_allclose(Y[l], torch_mhsa(p, x, l), rtol=1e-12, atol=1e-13)
    _, lse2, _ = ref.attention(p, x["cacheK"], x["n"], x["chunkK"], x["Q"])
    np.testing.assert_allclose(lse, lse2, rtol=1e-14, atol=1e-14)
    assert np.all(np.abs(Y) <= absY + 1e-12)


def test_mhsa_rational_golden_and_closed_forms():
    """Golden worked by hand (tests/golden/mhsa_rational.txt).  Closed forms: q = 0 makes every visible key equally
    likely, so Y_i is the running mean of the visible value rows (causal); values that do not depend on the key pass
    through unchanged (rows sum to one); one key with a huge logit returns its value row; GQA: query head j reads the
    keys AND the values of KV head j // G."""
    p = ref.RefParams(L=1, Hq=1, Hkv=1, D=1, cache_cap=1, Nn_v=2, Nn_a=0, scale=1.0)
    cacheK, cacheV = np.array([[[[math.log(1.0)]]]]), np.array([[[[6.0]]]])
    chunkK, chunkV = np.log(np.array([2.0, 3.0])).reshape(1, 1, 2, 1), np.array([12.0, -6.0]).reshape(1, 1, 2, 1)
    Y, lse, _ = ref.mhsa(p, cacheK, cacheV, [1], chunkK, chunkV, np.ones((1, 1, 2, 1)))
    for line in open(os.path.join(GOLD, "mhsa_rational.txt")):
        if line.startswith("#") or not line.strip():
            continue
        i, y, el = line.split()
        assert abs(Y[0, 0, int(i), 0] - float(y)) < 1e-12 and abs(math.exp(lse[0, 0, int(i)]) - float(el)) < 1e-12
    p, x = make(Hq=4, Hkv=2, D=8, cap=12, n=(9,), n_v=(6,), Nn_v=5, Nn_a=3)
    Y, _, _ = ref.mhsa(p, x["cacheK"], x["cacheV"], x["n"], x["chunkK"], x["chunkV"], 0 * x["Q"])
    for h in range(2):
        V = np.concatenate([x["cacheV"][0, h, :9], x["chunkV"][0, h]], 0)
        for i in range(p.Nn):
            for g in range(2):
                np.testing.assert_allclose(Y[0, 2 * h + g, i], V[:9 + i + 1].mean(0), rtol=1e-13)     # running mean
    const = np.broadcast_to(rnd(1, 2, 1, 8, seed=9), (1, 2, 12, 8))
    Y, _, _ = ref.mhsa(p, x["cacheK"], const, x["n"], x["chunkK"], const[:, :, :8], x["Q"])
    np.testing.assert_allclose(Y[0, :, :, :], np.repeat(const[0, :, :1], 2, 0).repeat(8, 1), rtol=1e-13)
    xk = {k: v.copy() for k, v in x.items()}
    xk["cacheK"][0, 1, 4] = 60.0 * np.sign(x["Q"][0, 3, 2])                    # KV head 1, cached row 4 dominates for q head 3, query 2
    Y, _, _ = ref.mhsa(p, xk["cacheK"], x["cacheV"], x["n"], x["chunkK"], x["chunkV"], x["Q"])
    np.testing.assert_allclose(Y[0, 3, 2], x["cacheV"][0, 1, 4], atol=1e-9)
    np.testing.assert_allclose(Y[0, :2], ref.mhsa(p, x["cacheK"], x["cacheV"], x["n"], x["chunkK"], x["chunkV"], x["Q"])[0][0, :2])  # head 0 untouched


def test_mhsa_lse_feeds_the_column_sums():
    """The point of NEXT-1: the LSE that the attention forward emits, fed to Eq.6's column sums as exp(z - lse), gives
    the importance of O2 (the two-pass formulation and the forward + one-pass formulation are the same function)."""
    p, x = make(Hq=4, Hkv=2, D=8, cap=12, n=(9,), n_v=(6,), Nn_v=5, Nn_a=3)
    _, lse, _ = ref.mhsa(p, x["cacheK"], x["cacheV"], x["n"], x["chunkK"], x["chunkV"], x["Q"])
    a_log, _, _ = ref.attention(p, x["cacheK"], x["n"], x["chunkK"], x["Q"])
    a = np.zeros_like(a_log)
    for h in range(2):
        K = np.concatenate([x["cacheK"][0, h, :9], x["chunkK"][0, h]], 0)
        for g in range(2):
            z = x["Q"][0, 2 * h + g] @ K.T / math.sqrt(8)
            P = np.exp(z - lse[0, 2 * h + g][:, None])
            P[:, 9:] *= np.tril(np.ones((8, 8)))
            a[0, h, :17] += P.sum(0)
    np.testing.assert_allclose(a, a_log, rtol=1e-12, atol=1e-14)


def test_split_segment_maps():
    """O1 / Eq.3: visual = cached visual ++ new visual, audio = cached audio ++ new audio (R9)."""
    p, x = make()
    Nkcap = p.cache_cap + p.Nn
    a_log = np.arange(p.Hkv * Nkcap, dtype=np.float64).reshape(1, p.Hkv, Nkcap)
    a_v, a_a = ref.split(p, a_log, x["n_v"], x["n"])
    n_v, n = 6, 9
    for h in range(p.Hkv):
        base = a_log[0, h]
        np.testing.assert_array_equal(a_v[0, h, :n_v + p.Nn_v], np.r_[base[:n_v], base[n:n + p.Nn_v]])
        np.testing.assert_array_equal(a_a[0, h, :(n - n_v) + p.Nn_a], np.r_[base[n_v:n], base[n + p.Nn_v:n + p.Nn]])


# ------------------------------------------------------------------------------------------ O3 (Eq.7)
def seg_rows(p, x, l, h, m, which="V"):
    n_v, n = int(x["n_v"][l]), int(x["n"][l])
    c, k = x["cache" + which][l, h], x["chunk" + which][l, h]
    return np.concatenate([c[:n_v], k[:p.Nn_v]]) if m == 0 else np.concatenate([c[n_v:n], k[p.Nn_v:]])


@pytest.mark.parametrize("stride", [(1, 1), (2, 3)])
def test_redundancy_matches_torch_cosine(stride):
    p, x = make(sim_stride_v=stride[0], sim_stride_a=stride[1])
    s_v, s_a = ref.redundancy(p, x["cacheV"], x["n_v"], x["n"], x["chunkV"])
    for h in range(p.Hkv):
        for m, s, sg in ((0, s_v, stride[0]), (1, s_a, stride[1])):
            X = torch.from_numpy(seg_rows(p, x, 0, h, m))
            K = X.shape[0]
            c = torch.nn.functional.cosine_similarity(X[:-sg], X[sg:], dim=-1).numpy()   # c[t] = cos(x_t, x_{t+sg})
            for t in range(K):
                terms = ([c[t]] if t + sg < K else []) + ([c[t - sg]] if t - sg >= 0 else [])
                exp = float(np.mean(terms)) if terms else 0.0
                assert abs(s[0, h, t] - exp) < 1e-13
            assert np.all(s[0, h, K:] == 0)


def test_redundancy_special_values():
    """cos(x,x) = 1; duplicated neighbours => s = 1 => psi = 0 (Eq.7-8); orthogonal => 0; opposite => -1."""
    p = ref.RefParams(L=1, Hq=1, Hkv=1, D=4, cache_cap=4, Nn_v=4, Nn_a=0)
    e = np.eye(4)
    cache = np.stack([e[0], e[0], e[0], e[1]]).reshape(1, 1, 4, 4)          # dup dup dup | orth
    chunk = np.stack([-e[1], e[2], 3 * e[2], e[3]]).reshape(1, 1, 4, 4)     # opposite (junction) | orth | dup (scaled)
    n_v = np.array([4], np.int32)
    s_v, _ = ref.redundancy(p, cache, n_v, n_v, chunk)
    np.testing.assert_allclose(s_v[0, 0, :8], [1, 1, 0.5, -0.5, -0.5, 0.5, 0.5, 0], atol=1e-15)
    psi_v, _ = ref.psi(p, n_v, n_v, np.ones_like(s_v), np.zeros((1, 1, 4)), s_v, np.zeros((1, 1, 4)))
    assert psi_v[0, 0, 0] == 0 and psi_v[0, 0, 1] == 0


def test_redundancy_zero_vector_and_modalities_do_not_neighbour():
    p, x = make()
    x["cacheV"][0, 0, 2] = 0                                  # zero vector: cos = 0 / max(0, 1e-8) = 0 (R12)
    s_v, s_a = ref.redundancy(p, x["cacheV"], x["n_v"], x["n"], x["chunkV"])
    assert np.all(np.isfinite(s_v)) and np.all(np.isfinite(s_a))
    ref_v = s_v.copy()
    x["cacheV"][0, :, 6:9] = rnd(2, 3, p.D, seed=99)          # change cached AUDIO rows only
    x["chunkV"][0, :, p.Nn_v:] = rnd(2, p.Nn_a, p.D, seed=98)
    s_v2, s_a2 = ref.redundancy(p, x["cacheV"], x["n_v"], x["n"], x["chunkV"])
    assert np.array_equal(ref_v, s_v2) and not np.array_equal(s_a, s_a2)


@pytest.mark.parametrize("cfg,tol", [(I.CFG1, 0.03), (I.CFG4.replace(L=1, Hq=8, Hkv=2, n_v=1301, n_a=40, Nn_v=768, Nn_a=30,
                                                                   cache_cap=1400, outlier_p=0.0), 0.02)])
def test_redundancy_ar1_statistics(cfg, tol):
    """Statistical pin (DESIGN.md inputs): AR(1) rows with coefficient rho at the tested stride => E[s] ~ rho."""
    x = I.full_inputs(cfg)
    p = ref.RefParams(L=cfg.L, Hq=cfg.Hq, Hkv=cfg.Hkv, D=cfg.D, cache_cap=cfg.cache_cap, Nn_v=cfg.Nn_v, Nn_a=cfg.Nn_a,
                      sim_stride_v=cfg.sim_stride_v, sim_stride_a=cfg.sim_stride_a)
    s_v, s_a = ref.redundancy(p, x["cacheV"], x["n_v"], x["n"], x["chunkV"])
    Kv = cfg.n_v + cfg.Nn_v
    interior = s_v[:, :, cfg.frame:Kv - cfg.frame]
    assert abs(interior.mean() - cfg.rho) < tol
    assert abs(s_a[:, :, :cfg.n_a + cfg.Nn_a].mean()) < 0.05   # i.i.d. audio: no redundancy


# ------------------------------------------------------------------------------------------ O4 (Eq.8)
def test_psi_special_lambdas():
    p, x = make()
    a_v, a_a = np.abs(rnd(1, 2, p.seg_cap_v, seed=7)) * 3, np.abs(rnd(1, 2, p.seg_cap_a, seed=8))
    s_v, s_a = np.tanh(rnd(1, 2, p.seg_cap_v, seed=9)), np.tanh(rnd(1, 2, p.seg_cap_a, seed=10))
    Kv, Ka = 6 + p.Nn_v, 3 + p.Nn_a
    for lam, f in ((0.0, lambda a, s: 1 - s), (1.0, lambda a, s: a * (1 - s)), (0.5, lambda a, s: np.sqrt(a) * (1 - s))):
        p.lam = lam
        psi_v, psi_a = ref.psi(p, x["n_v"], x["n"], a_v, a_a, s_v, s_a)
        np.testing.assert_array_equal(psi_v[..., :Kv], f(a_v, s_v)[..., :Kv].astype(np.float32))
        np.testing.assert_array_equal(psi_a[..., :Ka], f(a_a, s_a)[..., :Ka].astype(np.float32))
        assert np.all(psi_v[..., Kv:] == 0)
    p.lam = 0.02
    a_v[0, 0, 0] = 0.0                                        # R13: 0^lambda = 0
    psi_v, _ = ref.psi(p, x["n_v"], x["n"], a_v, a_a, s_v, s_a)
    assert psi_v[0, 0, 0] == 0
    # monotone in a at fixed s, and ranking invariant under a -> kappa a (R5: sum vs mean over G)
    psi2, _ = ref.psi(p, x["n_v"], x["n"], 7.0 * a_v, a_a, s_v, s_a)
    o1, o2 = np.argsort(-psi_v[0, 1, :Kv].astype(np.float64), kind="stable"), np.argsort(-psi2[0, 1, :Kv].astype(np.float64), kind="stable")
    assert np.array_equal(o1, o2)


# ------------------------------------------------------------------------------------------ O5 (Eq.9-10, 13)
def test_stats_entropy_closed_forms():
    p, x = make()
    Kv, Ka = 6 + p.Nn_v, 3 + p.Nn_a
    a_v, a_a = np.zeros((1, 2, p.seg_cap_v)), np.zeros((1, 2, p.seg_cap_a))
    s_v, s_a = np.zeros_like(a_v), np.zeros_like(a_a)
    a_v[..., :Kv] = 0.37                                      # uniform => Hn = 1
    a_a[0, 0, 2] = 5.0                                        # one-hot => Hn = 0
    s_v[0, :, :Kv] = 0.25
    s_a[0, 0, :Ka], s_a[0, 1, :Ka] = 0.5, -0.1
    st = ref.stats(p, x["n_v"], x["n"], a_v, a_a, s_v, s_a)[0]
    assert abs(st[0] - 1.0) < 1e-14 and st[1] == 0.0
    assert abs(st[2] - 0.25) < 1e-15 and abs(st[3] - 0.2) < 1e-15
    assert abs(st[4] - 0.75) < 1e-14 and st[5] == 0.0          # C = Hn (1 - sbar)
    assert abs(st[7] - (0.25 * 2 * Kv + 0.4 * Ka) / (2 * (Kv + Ka))) < 1e-15


def test_stats_matches_scipy_entropy_and_identity():
    from scipy.stats import entropy
    p, x = make(Hq=6, Hkv=3)
    Kv, Ka = 6 + p.Nn_v, 3 + p.Nn_a
    a_v, a_a = np.abs(rnd(1, 3, p.seg_cap_v, seed=1)), np.abs(rnd(1, 3, p.seg_cap_a, seed=2))
    s_v, s_a = np.tanh(rnd(1, 3, p.seg_cap_v, seed=3)), np.tanh(rnd(1, 3, p.seg_cap_a, seed=4))
    st = ref.stats(p, x["n_v"], x["n"], a_v, a_a, s_v, s_a)[0]
    Av, Aa = a_v[0, :, :Kv].sum(0), a_a[0, :, :Ka].sum(0)       # R16: heads summed, then normalised per modality
    assert abs(st[0] - entropy(Av) / math.log(Kv)) < 1e-13
    assert abs(st[1] - entropy(Aa) / math.log(Ka)) < 1e-13
    assert abs(st[6] - entropy(np.r_[Av, Aa]) / math.log(Kv + Ka)) < 1e-13
    S = Av.sum()
    assert abs(st[0] * math.log(Kv) - (math.log(S) - (Av * np.log(Av)).sum() / S)) < 1e-12   # H = ln S - sum A ln A / S
    assert abs(st[2] - s_v[0, :, :Kv].mean()) < 1e-15 and abs(st[3] - s_a[0, :, :Ka].mean()) < 1e-15
    assert 0 <= st[0] <= 1 and 0 <= st[1] <= 1 and 0 <= st[6] <= 1


def test_stats_uniform_attention_end_to_end():
    """NS invariant: normalized entropy equals 1 for uniform attention (Q = 0, non-causal)."""
    p, x = make(causal=0)
    x["Q"][:] = 0
    out = ref.score(p, x["cacheK"], x["cacheV"], x["n_v"], x["n"], x["chunkK"], x["chunkV"], x["Q"])
    np.testing.assert_allclose(out["stats"][0, [0, 1, 6]], 1.0, rtol=1e-13)


# ------------------------------------------------------------------------------------------ O6 (Eq.11-14)
def stats_with(C_v, C_a, L=1):
    st = np.zeros((L, 8))
    st[:, 0], st[:, 1], st[:, 4], st[:, 5] = C_v, C_a, C_v, C_a
    return st


def test_allocate_budget_split_golden():
    """tests/golden/budget_split.txt: w_v = r/(r+1) at C_v = C_a (Eq.11-12; P:272 round figures)."""
    for ln in open(os.path.join(GOLD, "budget_split.txt")):
        if ln.startswith("#"):
            continue
        r, mv, ma = map(int, ln.split())
        p = ref.RefParams(L=1, Hq=1, Hkv=1, D=1, cache_cap=8000, Nn_v=0, Nn_a=0, ratio_r=float(r))
        M_v, M_a = ref.allocate(p, stats_with(0.4, 0.4), [6000], [8000], [4096])
        assert (int(M_v[0]), int(M_a[0])) == (mv, ma)


def test_allocate_formula_and_edges():
    p = ref.RefParams(L=4, Hq=1, Hkv=1, D=1, cache_cap=1000, Nn_v=100, Nn_a=50, ratio_r=5.0)
    st = np.zeros((4, 8))
    st[:, 4] = [0.9, 0.2, 0.0, 0.5]
    st[:, 5] = [0.3, 0.8, 0.0, 0.5]
    n_v, n = np.array([600, 600, 600, 10], np.int32), np.array([900, 900, 900, 20], np.int32)
    B = np.array([500, 500, 500, 500], np.int32)
    M_v, M_a = ref.allocate(p, st, n_v, n, B)
    for l in range(3):
        wv = 5 * st[l, 4] / (5 * st[l, 4] + st[l, 5]) if st[l, 4] + st[l, 5] > 0 else 5 / 6   # Eq.11; 0/0 -> prior
        assert M_v[l] == math.floor(wv * 500 + 0.5) and M_v[l] + M_a[l] == 500
    assert (M_v[3], M_a[3]) == (110, 60)                      # K_v + K_a <= B: keep all
    # a modality with fewer rows than its share: the surplus spills to the other one (R22)
    p2 = ref.RefParams(L=1, Hq=1, Hkv=1, D=1, cache_cap=1000, Nn_v=10, Nn_a=300, ratio_r=5.0)
    M_v, M_a = ref.allocate(p2, stats_with(0.5, 0.5), [90], [700], [600])
    assert (M_v[0], M_a[0]) == (100, 500)
    p3 = ref.RefParams(L=1, Hq=1, Hkv=1, D=1, cache_cap=1000, Nn_v=400, Nn_a=10, ratio_r=5.0)
    M_v, M_a = ref.allocate(p3, stats_with(0.01, 0.99), [500], [520], [600])
    assert (M_v[0], M_a[0]) == (570, 30)
    # r -> infinity: everything visual (up to availability)
    p4 = ref.RefParams(L=1, Hq=1, Hkv=1, D=1, cache_cap=1000, Nn_v=400, Nn_a=100, ratio_r=1e12)
    M_v, M_a = ref.allocate(p4, stats_with(0.3, 0.6), [500], [700], [600])
    assert (M_v[0], M_a[0]) == (600, 0)


def test_layer_budgets_invariants():
    """Eq.14 invariants: softmax sums to 1, T -> inf and equal C => uniform, exact sum, clamps (the clamp branch itself is
    pinned by test_layer_budgets_clamp_branch_is_kappa_waterfilling below)."""
    L = 7
    st = np.zeros((L, 8))
    st[:, 6] = np.linspace(0.5, 0.9, L)
    st[:, 7] = 0.1
    p = ref.RefParams(L=L, Hq=1, Hkv=1, D=1, cache_cap=1, Nn_v=0, Nn_a=0, temperature=0.2)
    b = ref.layer_budgets(p, st, 7 * 8192)
    assert b.sum() == 7 * 8192 and np.all(np.diff(b) > 0)
    C = st[:, 6] * 0.9
    pi = np.exp(C / 0.2) / np.exp(C / 0.2).sum()
    assert np.all(np.abs(b - pi * 7 * 8192) < 1.0)
    p.temperature = 1e9
    b = ref.layer_budgets(p, st, 7 * 8192 + 3)
    assert b.sum() == 7 * 8192 + 3 and b.max() - b.min() <= 1
    st[:, 6] = 0.7
    p.temperature = 0.2
    assert list(ref.layer_budgets(p, st, 7 * 100)) == [100] * 7
    assert list(ref.layer_budgets(p, st, 7 * 100 + 3)) == [101] * 3 + [100] * 4   # equal remainders: lowest layers first
    st[:, 6] = np.linspace(0.1, 0.9, L)
    p.budget_min, p.budget_max = 4096, 12288
    b = ref.layer_budgets(p, st, 7 * 8192)
    assert b.sum() == 7 * 8192 and b.min() >= 4096 and b.max() <= 12288
    assert b[0] == 4096 and b[-1] == 12288
    # two-sided clamp where both bounds bite: the total must survive (one side is fixed per round)
    g = np.random.default_rng(2)
    st9 = np.zeros((9, 8))
    st9[:, 6], st9[:, 7] = g.uniform(0.5, 0.95, 9), g.uniform(0.0, 0.5, 9)
    p9 = ref.RefParams(L=9, Hq=1, Hkv=1, D=1, cache_cap=1, Nn_v=0, Nn_a=0, temperature=0.2, budget_min=200, budget_max=320)
    b = ref.layer_budgets(p9, st9, 256 * 9)
    assert b.sum() == 256 * 9 and b.min() >= 200 and b.max() <= 320
    C9 = st9[:, 6] * (1 - st9[:, 7])
    assert np.all(np.diff(b[np.argsort(C9)]) >= 0)            # monotone in compressibility


# ---- Eq.14 with [B_min, B_max] ("constrained within the range of [B_min, B_max]"): independent pin (R20) -------
def kappa_waterfill(pi, lo, hi, total):
    """The bounded proportional split that the mathematics fixes: b_l = clip(kappa * pi_l, lo, hi) with the scalar kappa
    set by sum_l b_l = total (f(kappa) = sum clip(kappa pi) is continuous and non-decreasing, so kappa is unique wherever
    f is strictly increasing; on a flat part every kappa gives the same b).  Plain bisection on kappa: no loop over
    'violators', no re-splitting, nothing of the oracle's procedure."""
    f = lambda k: np.clip(k * pi, lo, hi).sum()
    if total >= hi * len(pi):
        return np.full(len(pi), float(hi))
    if total <= lo * len(pi):
        return np.full(len(pi), float(lo))
    k0, k1 = 0.0, 1.0
    while f(k1) < total:
        k1 *= 2.0
    for _ in range(200):
        km = 0.5 * (k0 + k1)
        if f(km) < total:
            k0 = km
        else:
            k1 = km
    return np.clip(0.5 * (k0 + k1) * pi, lo, hi)


def largest_remainder(b, total, hi):
    """numpy largest-remainder integerisation: floor, then +1 to the (total - sum floor) largest fractional parts, equal
    fractions to the lowest layer first, never above hi.  Returns (ints, gap) where gap is the distance between the
    last fraction that got a unit and the first that did not (a near-zero gap means the choice is rounding noise)."""
    fl = np.floor(b + 1e-9)                       # a clamped layer sits ON an integer bound; bisection leaves it 1e-13 short
    frac = np.where(fl + 1 <= hi, b - fl, -1.0)
    left = int(round(total - fl.sum()))
    order = np.argsort(-frac, kind="stable")      # stable: equal fractions keep ascending layer order
    out = fl.astype(np.int64)
    out[order[:left]] += 1
    gap = frac[order[left - 1]] - frac[order[left]] if 0 < left < len(b) else 1.0
    return out, gap


def eq14_cases(n_cases=240):
    g = np.random.default_rng(2014)
    for c in range(n_cases):
        L = int(g.integers(2, 41))
        st = np.zeros((L, 8))
        spread = [0.05, 0.3, 0.8][c % 3]                       # narrow to wide compressibility spread
        st[:, 6] = np.clip(0.6 + spread * g.standard_normal(L) * 0.5, 0.01, 1.0)
        st[:, 7] = g.uniform(0.0, 0.6, L)
        T = [0.2, 0.05, 1.0][(c // 3) % 3]
        mean_b = int(g.integers(64, 40000))
        kind = c % 5
        if kind == 0:
            lo, hi = int(0.8 * mean_b), int(1.25 * mean_b)      # both bounds bite
        elif kind == 1:
            lo, hi = 1, int(1.1 * mean_b)                       # upper bound only
        elif kind == 2:
            lo, hi = int(0.9 * mean_b), 100 * mean_b            # lower bound only
        elif kind == 3:
            lo, hi = int(0.5 * mean_b), int(2 * mean_b)         # mild
        else:
            lo, hi = int(0.97 * mean_b), int(1.03 * mean_b)     # tight: almost every layer is clamped
        total = mean_b * L + int(g.integers(-L, L + 1))
        if c % 40 == 7:
            total = hi * L + 5                                  # infeasible: every layer at B_max
        if c % 40 == 9:
            total = max(0, lo * L - 5)                          # infeasible: every layer at B_min
        yield L, st, T, lo, hi, total


def test_layer_budgets_clamp_branch_is_kappa_waterfilling():
    """R20 pin: omnimem_ref_layer_budgets with clamps == clip(kappa pi, B_min, B_max), sum = total, found by
    bisection in numpy, then integerised by a numpy largest-remainder.  240 seeded cases: one- and two-sided clamps,
    tight ranges, wide and narrow softmax spreads, infeasible totals."""
    n_clamped_lo = n_clamped_hi = n_both = checked = 0
    for L, st, T, lo, hi, total in eq14_cases():
        p = ref.RefParams(L=L, Hq=1, Hkv=1, D=1, cache_cap=1, Nn_v=0, Nn_a=0, temperature=T, budget_min=lo, budget_max=hi)
        got = ref.layer_budgets(p, st, total).astype(np.int64)
        C = st[:, 6] * (1.0 - st[:, 7])
        e = np.exp((C - C.max()) / T)
        pi = e / e.sum()
        b = kappa_waterfill(pi, lo, hi, total)
        assert got.min() >= lo and got.max() <= hi
        if total >= hi * L or total <= lo * L:
            assert np.all(got == (hi if total >= hi * L else lo))
            continue
        assert got.sum() == total
        assert np.all(np.abs(got - b) < 1.0 + 1e-6), f"not within one unit of the kappa form: {got} vs {b}"
        want, gap = largest_remainder(b, total, hi)
        if gap > 1e-6:                                           # else the last unit is decided by rounding noise
            assert np.array_equal(got, want), f"L={L} lo={lo} hi={hi} total={total}: {got} vs {want}"
            checked += 1
        at_lo, at_hi = (np.abs(b - lo) < 1e-9).sum(), (np.abs(b - hi) < 1e-9).sum()
        n_clamped_lo += at_lo > 0
        n_clamped_hi += at_hi > 0
        n_both += (at_lo > 0) and (at_hi > 0)
    assert checked >= 200 and n_both >= 40 and n_clamped_lo >= 80 and n_clamped_hi >= 80    # the cases do exercise the branch


def test_layer_budgets_pin_catches_a_wrong_redistribution():
    """The pin above discriminates: a plausible wrong rule -- clipped mass re-spread UNIFORMLY over the free layers
    instead of in proportion to pi -- departs from the kappa form by more than a unit on most clamped cases."""
    def uniform_respread(pi, lo, hi, total):
        b = np.clip(pi * total, lo, hi)
        for _ in range(100):
            free = (b > lo) & (b < hi)
            if not free.any() or abs(total - b.sum()) < 1e-9:
                break
            b[free] += (total - b.sum()) / free.sum()
            b = np.clip(b, lo, hi)
        return b
    caught = tried = 0
    for L, st, T, lo, hi, total in eq14_cases(120):
        if total >= hi * L or total <= lo * L:
            continue
        C = st[:, 6] * (1.0 - st[:, 7])
        e = np.exp((C - C.max()) / T)
        pi = e / e.sum()
        b = kappa_waterfill(pi, lo, hi, total)
        if not ((np.abs(b - lo) < 1e-9).any() or (np.abs(b - hi) < 1e-9).any()):
            continue
        tried += 1
        caught += np.abs(uniform_respread(pi, lo, hi, total) - b).max() > 1.0
    assert tried >= 60 and caught >= 0.6 * tried


def test_layer_budgets_two_layer_clamp_closed_form():
    """Two layers, upper clamp biting: B = (total - B_max, B_max) whatever pi says; three layers with one clamped:
    the other two split the rest in the ratio pi_0 : pi_1 = exp((C_0 - C_1)/T)."""
    p = ref.RefParams(L=2, Hq=1, Hkv=1, D=1, cache_cap=1, Nn_v=0, Nn_a=0, temperature=0.2, budget_min=10, budget_max=600)
    st = np.zeros((2, 8))
    st[:, 6] = [0.9, 0.3]
    assert list(ref.layer_budgets(p, st, 1000)) == [600, 400]
    p3 = ref.RefParams(L=3, Hq=1, Hkv=1, D=1, cache_cap=1, Nn_v=0, Nn_a=0, temperature=0.2, budget_min=0, budget_max=500000)
    st3 = np.zeros((3, 8))
    st3[:, 6] = [0.5, 0.6, 0.95]                     # pi_2 dominates: unclamped it would take ~80 %
    b = ref.layer_budgets(p3, st3, 10**6)
    assert b[2] == 500000 and b.sum() == 10**6
    assert abs(b[0] / b[1] - np.exp((0.5 - 0.6) / 0.2)) < 1e-4


def test_psi_shared_heads_paper_literal():
    """R29: one score per token and layer.  Pins: Hkv = 1 reduces to Eq.8 per head; identical heads give
    Hkv^lambda a^lambda (1 - s); permuting the heads changes nothing; every head's row carries the same score, so the
    stable top-M of every head is the same set; against the formula written out with numpy."""
    g = np.random.default_rng(4)
    L, Hkv, cap_v, cap_a = 2, 3, 9, 5
    p = ref.RefParams(L=L, Hq=Hkv, Hkv=Hkv, D=1, cache_cap=6, Nn_v=3, Nn_a=1, lam=0.3)
    n_v, n = np.array([6, 4], np.int32), np.array([6, 6], np.int32)          # K_v = 9, 7 ; K_a = 1, 3
    assert (p.seg_cap_v, p.seg_cap_a) == (cap_v, 7)
    a_v, a_a = g.uniform(0.1, 3, (L, Hkv, p.seg_cap_v)), g.uniform(0.1, 3, (L, Hkv, p.seg_cap_a))
    s_v, s_a = g.uniform(-0.5, 0.9, a_v.shape), g.uniform(-0.5, 0.9, a_a.shape)
    pv, pa = ref.psi(p, n_v, n, a_v, a_a, s_v, s_a, select_scope=1)
    want = (a_v.sum(1) ** 0.3 * (1 - s_v.mean(1))).astype(np.float32)
    for l, Kv in enumerate((9, 7)):
        for h in range(Hkv):
            np.testing.assert_array_equal(pv[l, h, :Kv], want[l, :Kv])
            assert np.all(pv[l, h, Kv:] == 0)
    perm = [2, 0, 1]
    pv2, pa2 = ref.psi(p, n_v, n, a_v[:, perm], a_a[:, perm], s_v[:, perm], s_a[:, perm], select_scope=1)
    np.testing.assert_allclose(pv2, pv, rtol=1e-6)
    np.testing.assert_allclose(pa2, pa, rtol=1e-6)
    same = np.repeat(a_v[:, :1], Hkv, 1), np.repeat(a_a[:, :1], Hkv, 1), np.repeat(s_v[:, :1], Hkv, 1), np.repeat(s_a[:, :1], Hkv, 1)
    ps, _ = ref.psi(p, n_v, n, *same, select_scope=1)
    ph, _ = ref.psi(p, n_v, n, *same, select_scope=0)
    np.testing.assert_allclose(ps[:, 0], ph[:, 0] * Hkv ** 0.3, rtol=1e-6)
    p1 = ref.RefParams(L=L, Hq=1, Hkv=1, D=1, cache_cap=6, Nn_v=3, Nn_a=1, lam=0.3)
    one = a_v[:, :1].copy(), a_a[:, :1].copy(), s_v[:, :1].copy(), s_a[:, :1].copy()
    np.testing.assert_array_equal(ref.psi(p1, n_v, n, *one, select_scope=1)[0], ref.psi(p1, n_v, n, *one, select_scope=0)[0])
    M_v, M_a = np.array([4, 3], np.int32), np.array([1, 2], np.int32)
    iv, ia = ref.select(p, pv, pa, n_v, n, M_v, M_a)
    for l in range(L):
        for h in range(1, Hkv):
            assert np.array_equal(iv[l, h, :M_v[l]], iv[l, 0, :M_v[l]]) and np.array_equal(ia[l, h, :M_a[l]], ia[l, 0, :M_a[l]])


def test_redundancy_hidden_states():
    """R30: Eq.7 on hidden states.  Pins: against torch cosine_similarity on the rows; the same value in
    every KV head; duplicate neighbours => 1; the compaction of H picks exactly the kept rows (numpy take)."""
    g = torch.Generator().manual_seed(3)
    L, cap, d = 2, 10, 24
    p = ref.RefParams(L=L, Hq=4, Hkv=2, D=8, cache_cap=cap, Nn_v=4, Nn_a=2)
    n_v, n = np.array([5, 3], np.int32), np.array([8, 6], np.int32)
    cacheH, chunkH = torch.randn(L, cap, d, generator=g, dtype=torch.float64), torch.randn(L, 6, d, generator=g, dtype=torch.float64)
    chunkH[0, 1] = chunkH[0, 0]                                  # duplicate neighbours
    s_v, s_a = ref.redundancy_hidden(p, cacheH, n_v, n, chunkH)
    assert s_v.shape == (L, 2, p.seg_cap_v) and np.array_equal(s_v[:, 0], s_v[:, 1]) and np.array_equal(s_a[:, 0], s_a[:, 1])
    cos = torch.nn.functional.cosine_similarity
    for l in range(L):
        vis = torch.cat([cacheH[l, :n_v[l]], chunkH[l, :4]])
        aud = torch.cat([cacheH[l, n_v[l]:n[l]], chunkH[l, 4:]])
        for seq, s in ((vis, s_v[l, 0]), (aud, s_a[l, 0])):
            c = cos(seq[:-1], seq[1:], dim=-1).numpy()
            want = np.empty(len(seq))
            want[0], want[-1] = c[0], c[-1]
            want[1:-1] = 0.5 * (c[:-1] + c[1:])
            np.testing.assert_allclose(s[:len(seq)], want, atol=1e-12)
    Kv0 = n_v[0] + 4
    assert abs(s_v[0, 0, n_v[0]] - 0.5 * (1.0 + cos(cacheH[0, n_v[0] - 1], chunkH[0, 0], dim=0).item())) < 1e-12 and Kv0 == 9
    idx_v = np.full((L, 2, cap), -1, np.int32)
    idx_a = np.full((L, 2, cap), -1, np.int32)
    idx_v[0, :, :3], idx_v[1, :, :2] = [0, 5, 8], [2, 6]
    idx_a[0, :, :2], idx_a[1, :, :1] = [1, 3], [4]
    M_v, M_a = np.array([3, 2], np.int32), np.array([2, 1], np.int32)
    dst = ref.compact_hidden(p, cacheH, chunkH, n_v, n, idx_v, idx_a, M_v, M_a).view(np.float64).reshape(L, cap, d)
    vis0 = np.concatenate([cacheH[0, :5].numpy(), chunkH[0, :4].numpy()])
    aud0 = np.concatenate([cacheH[0, 5:8].numpy(), chunkH[0, 4:].numpy()])
    np.testing.assert_array_equal(dst[0, :3], vis0[[0, 5, 8]])
    np.testing.assert_array_equal(dst[0, 3:5], aud0[[1, 3]])


def test_time_interleaved_chunk():
    """R25' (NEXT-4b): chunk rows in true temporal order with a per-row modality map.  Pins: (1) the attention itself
    does not know the map (torch softmax, causal by storage order = true position) and the split takes the map's rows;
    (2) Eq.7 neighbours are the adjacent tokens of the same modality, by torch cosine on sequences built with numpy;
    (3) without the causal mask an interleaved chunk is a row permutation of the blocked chunk: every segment output,
    the kept sets and the compacted bytes are the same."""
    mod = np.array([0, 0, 1, 0, 1, 1, 0, 0], np.int32)                      # Nn_v = 5, Nn_a = 3
    p, x = make(chunk_modality=mod)
    Nc, n_v = 9, 6
    out = ref.score(p, x["cacheK"], x["cacheV"], x["n_v"], x["n"], x["chunkK"], x["chunkV"], x["Q"])
    a_t = torch_attention(p, x, 0)[0]                                       # [Hkv, Nc + Nn], knows nothing of modalities
    vis = np.concatenate([a_t[:, :n_v], a_t[:, Nc:][:, mod == 0]], 1)
    aud = np.concatenate([a_t[:, n_v:Nc], a_t[:, Nc:][:, mod == 1]], 1)
    np.testing.assert_allclose(out["a_v"][0, :, :11], vis, rtol=1e-12)
    np.testing.assert_allclose(out["a_a"][0, :, :6], aud, rtol=1e-12)
    cos = torch.nn.functional.cosine_similarity
    for h in range(p.Hkv):
        seq = torch.from_numpy(np.concatenate([x["cacheV"][0, h, :n_v], x["chunkV"][0, h][mod == 0]]))
        c = cos(seq[:-1], seq[1:], dim=-1).numpy()
        want = np.concatenate([[c[0]], 0.5 * (c[:-1] + c[1:]), [c[-1]]])
        np.testing.assert_allclose(out["s_v"][0, h, :11], want, atol=1e-12)
    # (3) permutation invariance without the causal mask
    perm = np.concatenate([np.where(mod == 0)[0], np.where(mod == 1)[0]])   # interleaved row of each blocked row
    pi, xi = make(chunk_modality=mod, causal=0)
    pb, xb = make(causal=0)
    for k in ("chunkK", "chunkV", "Q"):
        xb[k] = np.ascontiguousarray(xi[k][:, :, perm])
    B = np.array([7], np.int32)
    oi = ref.compress_chunk(pi, xi["cacheK"], xi["cacheV"], xi["n_v"], xi["n"], xi["chunkK"], xi["chunkV"], xi["Q"], B)
    ob = ref.compress_chunk(pb, xb["cacheK"], xb["cacheV"], xb["n_v"], xb["n"], xb["chunkK"], xb["chunkV"], xb["Q"], B)
    for k in ("a_v", "a_a", "s_v", "s_a", "stats"):
        np.testing.assert_allclose(oi[k], ob[k], rtol=1e-12, atol=1e-15)
    assert np.array_equal(oi["M_v"], ob["M_v"]) and np.array_equal(oi["idx_v"], ob["idx_v"]) and np.array_equal(oi["idx_a"], ob["idx_a"])
    assert np.array_equal(oi["dstK"], ob["dstK"]) and np.array_equal(oi["dstV"], ob["dstV"])
    # with the causal mask the two layouts differ: an early audio row is seen by more queries than in the blocked order
    oc = ref.score(p, x["cacheK"], x["cacheV"], x["n_v"], x["n"], x["chunkK"], x["chunkV"], x["Q"])
    pbc, _ = make(causal=1)
    obc = ref.score(pbc, xb["cacheK"], xb["cacheV"], xb["n_v"], xb["n"], xb["chunkK"], xb["chunkV"], xb["Q"])
    assert not np.allclose(oc["a_a"], obc["a_a"])


def test_calibration_means_then_eq14():
    """R28: budgets from the MEANS of the two layer measures over the calibration chunks.  Pins: one chunk ==
    plain Eq.14; chunks that are permutations of each other give the same table; closed form of the two-layer case
    B_0 / B_1 = exp((C_0 - C_1) / T); identical layers => uniform."""
    L, total = 5, 5 * 1000
    g = np.random.default_rng(11)
    st = np.zeros((4, L, 8))
    st[:, :, 6], st[:, :, 7] = g.uniform(0.6, 0.95, (4, L)), g.uniform(0.0, 0.4, (4, L))
    p = ref.RefParams(L=L, Hq=1, Hkv=1, D=1, cache_cap=1, Nn_v=0, Nn_a=0, temperature=0.2)
    b1, m1 = ref.calibrate_budgets(p, st[:1], total)
    assert np.array_equal(b1, ref.layer_budgets(p, st[0], total)) and np.array_equal(m1, st[0])
    b, m = ref.calibrate_budgets(p, st, total)
    b_perm, _ = ref.calibrate_budgets(p, st[[2, 0, 3, 1]], total)
    assert np.array_equal(b, b_perm) and b.sum() == total
    np.testing.assert_allclose(m[:, 6], st[:, :, 6].mean(0), rtol=1e-15)
    C = st[:, :, 6].mean(0) * (1.0 - st[:, :, 7].mean(0))              # product of means, not mean of products
    pi = np.exp(C / 0.2) / np.exp(C / 0.2).sum()
    assert np.all(np.abs(b - pi * total) < 1.0)
    p2 = ref.RefParams(L=2, Hq=1, Hkv=1, D=1, cache_cap=1, Nn_v=0, Nn_a=0, temperature=0.2)
    st2 = np.zeros((3, 2, 8))
    st2[:, 0, 6], st2[:, 1, 6] = [0.9, 0.8, 0.7], [0.6, 0.7, 0.5]      # means 0.8 and 0.6, sbar = 0
    b2, _ = ref.calibrate_budgets(p2, st2, 10**6)
    assert abs(b2[0] / b2[1] - np.exp((0.8 - 0.6) / 0.2)) < 1e-4
    st[:, :, 6], st[:, :, 7] = 0.8, 0.3
    assert list(ref.calibrate_budgets(p, st, total)[0]) == [1000] * L


# ------------------------------------------------------------------------------------------ O7 (Eq.4-5)
def run_select(psi_row, M):
    K = len(psi_row)
    p = ref.RefParams(L=1, Hq=1, Hkv=1, D=1, cache_cap=K, Nn_v=0, Nn_a=0)
    psi_v = np.zeros((1, 1, p.seg_cap_v), np.float32)
    psi_v[0, 0, :K] = psi_row
    idx_v, _ = ref.select(p, psi_v, np.zeros((1, 1, p.seg_cap_a), np.float32), [K], [K], [M], [0])
    assert np.all(idx_v[0, 0, M:] == -1)
    return idx_v[0, 0, :M]


def test_select_brute_force_tiny():
    """Exhaustive: the kept set maximises sum(psi) and is the lexicographically smallest maximiser (ties -> lowest index)."""
    g = np.random.default_rng(0)
    for trial in range(30):
        K = int(g.integers(1, 10))
        psi_row = g.integers(0, 4, K).astype(np.float32) / 4      # many ties
        for M in range(K + 1):
            best = max(itertools.combinations(range(K), M), key=lambda c: (sum(psi_row[list(c)]), [-i for i in c]))
            assert list(run_select(psi_row, M)) == list(best)


def test_select_matches_stable_argsort_and_edges():
    g = np.random.default_rng(1)
    psi_row = np.round(g.random(500), 2).astype(np.float32)
    for M in (0, 1, 137, 499, 500):
        exp = np.sort(np.argsort(-psi_row.astype(np.float64), kind="stable")[:M])
        assert np.array_equal(run_select(psi_row, M), exp)
    assert list(run_select(np.full(9, 0.5, np.float32), 4)) == [0, 1, 2, 3]     # all equal: lowest indices


# ------------------------------------------------------------------------------------------ O8 + end to end
def test_compact_is_a_byte_exact_gather():
    p, x = make(L=2, cap=12, n=(9, 7), n_v=(6, 2), seed=5)
    cacheK = torch.from_numpy(x["cacheK"]).to(torch.bfloat16)
    chunkK = torch.from_numpy(x["chunkK"]).to(torch.bfloat16)
    M_v, M_a = np.array([4, 5], np.int32), np.array([3, 6], np.int32)
    g = np.random.default_rng(3)
    idx_v, idx_a = np.full((2, 2, 12), -1, np.int32), np.full((2, 2, 12), -1, np.int32)
    for l in range(2):
        for h in range(2):
            idx_v[l, h, :M_v[l]] = np.sort(g.choice(x["n_v"][l] + p.Nn_v, M_v[l], replace=False))
            idx_a[l, h, :M_a[l]] = np.sort(g.choice(x["n"][l] - x["n_v"][l] + p.Nn_a, M_a[l], replace=False))
    dst, n_v2, n2 = ref.compact(p, cacheK, chunkK, x["n_v"], x["n"], idx_v, idx_a, M_v, M_a)
    assert list(n_v2) == [4, 5] and list(n2) == [7, 11]
    raw_c, raw_k = cacheK.view(torch.uint8).numpy(), chunkK.view(torch.uint8).numpy()
    for l in range(2):
        n_v, n = int(x["n_v"][l]), int(x["n"][l])
        for h in range(2):
            vis = np.concatenate([raw_c[l, h, :n_v], raw_k[l, h, :p.Nn_v]])
            aud = np.concatenate([raw_c[l, h, n_v:n], raw_k[l, h, p.Nn_v:]])
            assert np.array_equal(dst[l, h, :M_v[l]], vis[idx_v[l, h, :M_v[l]]])
            assert np.array_equal(dst[l, h, M_v[l]:M_v[l] + M_a[l]], aud[idx_a[l, h, :M_a[l]]])


def run_step(wl, x):
    p = ref.RefParams(L=x["Q"].shape[0], Hq=wl.Hq, Hkv=wl.Hkv, D=wl.D, cache_cap=wl.cache_cap, Nn_v=wl.Nn_v, Nn_a=wl.Nn_a,
                      sim_stride_v=wl.sim_stride_v, sim_stride_a=wl.sim_stride_a)
    B = np.full((p.L,), wl.budget, np.int32)
    return p, ref.compress_chunk(p, x["cacheK"], x["cacheV"], x["n_v"], x["n"], x["chunkK"], x["chunkV"], x["Q"], B)


def test_end_to_end_cfg1_invariants():
    """CFG1 in full: budgets sum to B, kept rows are rows of the input, heads permute, re-compress keeps all."""
    wl = I.CFG1
    x = I.full_inputs(wl)
    p, out = run_step(wl, x)
    assert np.all(out["M_v"] + out["M_a"] == wl.budget) and np.all(out["n_out"] == wl.budget)
    G = wl.G
    np.testing.assert_allclose(out["a_v"].sum(-1) + out["a_a"].sum(-1), G * wl.Nn, rtol=1e-12)
    st = out["stats"]
    assert np.all((st[:, [0, 1, 6]] >= 0) & (st[:, [0, 1, 6]] <= 1))
    for l in range(wl.L):
        for h in range(wl.Hkv):
            iv = out["idx_v"][l, h, :out["M_v"][l]]
            assert np.all(np.diff(iv) > 0) and iv.min() >= 0 and iv.max() < wl.n_v + wl.Nn_v
    # permuting KV heads (and their query groups) permutes the per-head outputs
    perm = [1, 0]
    qperm = [h * G + g for h in perm for g in range(G)]
    x2 = dict(x)
    for k in ("cacheK", "cacheV", "chunkK", "chunkV"):
        x2[k] = x[k][:, perm]
    x2["Q"] = x["Q"][:, qperm]
    _, out2 = run_step(wl, x2)
    assert np.array_equal(out2["idx_v"], out["idx_v"][:, perm]) and np.array_equal(out2["dstK"], out["dstK"][:, perm])
    assert np.array_equal(out2["M_v"], out["M_v"])
    # a second step with an empty chunk and the same budget keeps everything, in place order
    wl0 = wl.replace(Nn_v=0, Nn_a=0)
    dt = wl.torch_dtype
    x3 = dict(cacheK=torch.from_numpy(out["dstK"]).view(dt), cacheV=torch.from_numpy(out["dstV"]).view(dt),
              chunkK=torch.zeros(wl.L, wl.Hkv, 0, wl.D, dtype=dt), chunkV=torch.zeros(wl.L, wl.Hkv, 0, wl.D, dtype=dt),
              Q=torch.zeros(wl.L, wl.Hq, 0, wl.D, dtype=dt), n_v=out["n_v_out"], n=out["n_out"])
    _, out3 = run_step(wl0, x3)
    assert np.array_equal(out3["dstK"], out["dstK"]) and np.array_equal(out3["n_v_out"], out["n_v_out"])


def test_duplicate_rows_are_evicted_first():
    """Eq.7-8: a run of identical value rows has s = 1, psi = 0 and loses to everything else."""
    wl = I.CFG1.replace(L=1)
    x = I.full_inputs(wl)
    x["cacheV"][0, :, 100:140] = x["cacheV"][0, :, 100:101].clone()   # with stride 16: rows 116..123 have both neighbours equal
    p, out = run_step(wl.replace(sim_stride_v=1), x)
    for h in range(wl.Hkv):
        kept = set(out["idx_v"][0, h, :out["M_v"][0]].tolist())
        assert not kept & set(range(101, 139))


def test_oracle_under_address_and_ub_sanitizers():
    """the oracle built with -fsanitize=address,undefined runs a whole step (blocked and interleaved
    chunk, shared selection, Eq.14 with clamps, ragged layers incl. an empty cache) without a report.  compute-sanitizer is
    closed on the GPU pool, so this is the sanitizer this repo can run."""
    import subprocess
    import sys
    asan = subprocess.run(["gcc", "-print-file-name=libasan.so"], capture_output=True, text=True).stdout.strip()
    if not os.path.isabs(asan) or not os.path.exists(asan):
        pytest.skip("libasan not installed")
    code = """
import numpy as np, torch
from oracle import ref
from paper_2606_07577_b200 import inputs as I
wl = I.CFG1.replace(L=3, cache_cap=600)
x = I.full_inputs(wl)
x['n'][1], x['n_v'][1] = 0, 0
x['n'][2], x['n_v'][2] = 77, 13
mod = I.modality_pattern(wl, 5)
for kw, scope in ((dict(), 0), (dict(chunk_modality=mod.numpy()), 1)):
    p = ref.RefParams(L=3, Hq=wl.Hq, Hkv=wl.Hkv, D=wl.D, cache_cap=wl.cache_cap, Nn_v=wl.Nn_v, Nn_a=wl.Nn_a,
                      sim_stride_v=16, budget_min=100, budget_max=300, **kw)
    sc = ref.score(p, x['cacheK'], x['cacheV'], x['n_v'], x['n'], x['chunkK'], x['chunkV'], x['Q'], want_rowH=True, select_scope=scope)
    B = ref.layer_budgets(p, sc['stats'], 3 * 200)
    out = ref.compress_chunk(p, x['cacheK'], x['cacheV'], x['n_v'], x['n'], x['chunkK'], x['chunkV'], x['Q'], B, select_scope=scope)
    assert out['n_out'].tolist() == np.minimum(B, x['n'].numpy() + wl.Nn).tolist()
print('sanitized oracle ok')
"""
    env = dict(os.environ, OMNIMEM_REF_SANITIZE="1", LD_PRELOAD=asan, ASAN_OPTIONS="detect_leaks=0:abort_on_error=0",
               UBSAN_OPTIONS="print_stacktrace=1", OMP_NUM_THREADS="2")
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    r = subprocess.run([sys.executable, "-c", code], env=env, cwd=root, capture_output=True, text=True, timeout=600)
    assert r.returncode == 0 and "sanitized oracle ok" in r.stdout, r.stdout[-2000:] + r.stderr[-4000:]
    assert "ERROR: AddressSanitizer" not in r.stderr and "runtime error" not in r.stderr, r.stderr[-4000:]
