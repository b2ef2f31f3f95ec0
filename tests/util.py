"""Helpers shared by the GPU parity tests: run both sides on the same seeded inputs and compare by NS's rules."""
from __future__ import annotations

import numpy as np
import torch

from oracle import ref
from paper_2606_07577_b200 import inputs as I

TOL = {"fp32": 1e-5, "bf16": 2e-3}   # north_star rule (a)


def ref_params(wl: I.Workload, L: int, **kw) -> ref.RefParams:
    args = dict(L=L, Hq=wl.Hq, Hkv=wl.Hkv, D=wl.D, cache_cap=wl.cache_cap, Nn_v=wl.Nn_v, Nn_a=wl.Nn_a,
                sim_stride_v=wl.sim_stride_v, sim_stride_a=wl.sim_stride_a)
    args.update(kw)
    return ref.RefParams(**args)


def seg_lens(wl, n_v, n):
    n_v, n = np.asarray(n_v), np.asarray(n)
    return n_v + wl.Nn_v, (n - n_v) + wl.Nn_a


def assert_close_rule_a(name, got, exp, tol, floor=0.0):
    """|got - exp| <= tol * max(|exp|, floor)."""
    got, exp = np.asarray(got, np.float64), np.asarray(exp, np.float64)
    bound = tol * np.maximum(np.abs(exp), floor)
    err = np.abs(got - exp)
    bad = err > bound
    if bad.any():
        i = np.unravel_index(np.argmax(err - bound), err.shape)
        raise AssertionError(f"{name}: {int(bad.sum())}/{bad.size} outside tol {tol}; worst at {i}: got {got[i]!r} "
                             f"exp {exp[i]!r} err {err[i]:.3e} bound {bound[i]:.3e}")


def compare_scores(wl, n_v, n, gpu: dict, orc: dict, tol: float, stats_tol=None):
    """Rule (a) on a, s, psi, lse, statistics.  gpu/orc: dicts of numpy arrays with the oracle's key names."""
    Kv, Ka = seg_lens(wl, n_v, n)
    L = len(Kv)
    for l in range(L):
        for key, K in (("a_v", Kv[l]), ("a_a", Ka[l])):
            e = orc[key][l, :, :K]
            if K:
                floor = 1e-6 * e.max(axis=-1, keepdims=True)
                assert_close_rule_a(f"{key}[{l}]", gpu[key][l, :, :K], e, tol, floor)
        for key, K in (("s_v", Kv[l]), ("s_a", Ka[l])):
            assert_close_rule_a(f"{key}[{l}]", gpu[key][l, :, :K], orc[key][l, :, :K], tol, 1.0)   # s in [-1,1]: absolute
        for key, K in (("psi_v", Kv[l]), ("psi_a", Ka[l])):
            if K:
                e = orc[key][l, :, :K].astype(np.float64)
                assert_close_rule_a(f"{key}[{l}]", gpu[key][l, :, :K], e, tol, 1e-6 * e.max())
    if "lse" in gpu and gpu["lse"] is not None:
        # LSE enters Eq.6 through exp(z - lse): an absolute error `tol` in lse is a relative error `tol` in a
        assert_close_rule_a("lse", gpu["lse"], orc["lse"], tol, 1.0)
    st = stats_tol or tol
    assert_close_rule_a("stats", gpu["stats"], orc["stats"], st, 1e-3)


def kept_sets_rule_c(name, idx_gpu, idx_ref, M, psi_ref_seg, tol):
    """Rule (c): index sets identical except where the oracle's score is within tol of the M-th largest score."""
    assert np.all(np.diff(idx_gpu[:M]) > 0), f"{name}: indices not ascending"      # the order is part of the contract
    g, r = set(idx_gpu[:M].tolist()), set(idx_ref[:M].tolist())
    diff = g ^ r
    if not diff:
        return 0
    K = len(psi_ref_seg)
    tau = np.sort(psi_ref_seg.astype(np.float64))[K - M] if M > 0 else 0.0
    for t in diff:
        if abs(float(psi_ref_seg[t]) - tau) > tol * max(abs(tau), 1e-30):
            raise AssertionError(f"{name}: index {t} differs and psi {psi_ref_seg[t]!r} is not within {tol} of tau {tau!r}")
    return len(diff)


def to_device(x: dict, device="cuda:0") -> dict:
    return {k: (v.to(device) if torch.is_tensor(v) else v) for k, v in x.items()}


def scores_to_numpy(sc) -> dict:
    f = lambda t: None if t is None else t.detach().cpu().numpy()
    return dict(a_v=f(sc.a_v), a_a=f(sc.a_a), s_v=f(sc.s_v), s_a=f(sc.s_a), psi_v=f(sc.psi_v), psi_a=f(sc.psi_a),
                stats=f(sc.stats), lse=f(sc.lse), rowH=f(sc.row_entropy))
