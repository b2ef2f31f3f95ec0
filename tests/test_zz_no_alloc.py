"""omnimem_redundancy_static, the entry point for callers that cannot allocate device memory, against the regular path.

Why the entry point exists: the regular calls need a context (omnimem_create calls cudaMalloc) and a caller-allocated
workspace.  A serving engine that gave all of HBM to its KV-cache pool at start-up, or an operator body that a host
runtime hands its tensors and forbids to allocate, has neither.  omnimem_redundancy_static computes the Eq.7 redundancy
with its intermediates in a 4 MiB array built into the library, so it allocates nothing -- and every call on a device
shares that one array, which keeps whatever the previous call left in it.

What is checked: its s_v, s_a equal those omnimem_score writes (the existing path: cosine_kernel + finalize_kernel through
the workspace) within the tolerance of rule (a) that every parity test here uses (tests/util.py TOL, absolute: s lies in
[-1, 1]) -- on TWO calls in a row on different inputs and shapes, so that a result which leaned on a fresh (zeroed) array,
or on what the previous call left behind, fails the second comparison; then the first inputs once more.  Also that sizes
beyond the built-in array are refused with their own status before anything is launched.

This file sorts last on purpose (`pytest --collect-only`): under `pytest -x` a failure here must not hide any other test.
It holds no state from other tests and passes alone in a fresh process as well as after the rest of the suite.
"""
import numpy as np
import pytest
import torch

from paper_2606_07577_b200 import inputs as I
from tests.util import TOL, seg_lens, to_device

pytestmark = pytest.mark.gpu

CASES = [
    # fp32 D = 64, neighbour distance 16 (visual) / 1 (audio): config 1 as it stands
    I.CFG1,
    # bf16 D = 128, two layers of a config-2-like shape with ragged lengths; different capacities from the case above, so
    # the same array cells hold different (layer, head, row) entries from one call to the next
    I.CFG2.replace(L=2, Hq=4, Hkv=2, n_v=700, n_a=150, Nn_v=400, Nn_a=123, budget=850, cache_cap=850),
    # paper-literal neighbour distance 1 on a bf16 D = 64 shape, empty audio cache
    I.CFG2.replace(L=3, Hq=2, Hkv=1, D=64, n_v=300, n_a=0, Nn_v=77, Nn_a=5, budget=400, cache_cap=400, sim_stride_v=1),
]


def existing_path(wl, x):
    """s_v, s_a from omnimem_score (context + workspace from torch's allocator)."""
    from paper_2606_07577_b200.omnimem import Cache, Chunk, OmniMem
    eng = OmniMem.for_workload(wl)
    d = to_device(x)
    sc = eng.score(Cache(d["cacheK"], d["cacheV"], d["n_v"], d["n"]), Chunk(d["chunkK"], d["chunkV"], d["Q"], wl.Nn_v, wl.Nn_a))
    torch.cuda.synchronize()
    out = sc.s_v.cpu().numpy(), sc.s_a.cpu().numpy()
    eng.close()
    return out


def static_path(wl, x, poison):
    """s_v, s_a from omnimem_redundancy_static; the outputs start as `poison` so untouched entries are visible."""
    from paper_2606_07577_b200 import omnimem
    d = to_device(x)
    L, Hkv = wl.L, wl.Hkv
    s_v = torch.full((L, Hkv, wl.cache_cap + wl.Nn_v), poison, dtype=torch.float32, device="cuda:0")
    s_a = torch.full((L, Hkv, wl.cache_cap + wl.Nn_a), poison, dtype=torch.float32, device="cuda:0")
    omnimem.redundancy_static(d["cacheV"], d["n_v"], d["n"], d["chunkV"], wl.Nn_v, wl.Nn_a, wl.Nn_v, wl.Nn_a, s_v, s_a,
                              sim_stride_v=wl.sim_stride_v, sim_stride_a=wl.sim_stride_a)
    torch.cuda.synchronize()
    return s_v.cpu().numpy(), s_a.cpu().numpy()


def compare(wl, x, got, exp, poison):
    Kv, Ka = seg_lens(wl, x["n_v"].numpy(), x["n"].numpy())
    tol = TOL[wl.dtype]
    for name, g, e, K in (("s_v", got[0], exp[0], Kv), ("s_a", got[1], exp[1], Ka)):
        for l in range(wl.L):
            err = np.abs(g[l, :, :K[l]].astype(np.float64) - e[l, :, :K[l]]).max() if K[l] else 0.0
            assert err <= tol, f"{wl.name} {name}[{l}]: {err:.3e} > {tol}"
            assert np.all(g[l, :, K[l]:] == poison), f"{wl.name} {name}[{l}]: wrote past K_m"


def test_static_scratch_entry_matches_the_workspace_path_on_calls_in_a_row():
    xs = [I.full_inputs(wl) for wl in CASES]
    for wl, x in zip(CASES, xs):   # ragged lengths: the second layer of every case is shorter than the first
        x["n_v"] = x["n_v"].clone()
        x["n"] = x["n"].clone()
        cut = min(29, int(x["n_v"][-1]))
        x["n_v"][-1] -= cut
        x["n"][-1] -= cut
    expected = [existing_path(wl, x) for wl, x in zip(CASES, xs)]
    # calls in a row, nothing in between that could reset the array; then the first case again on top of the others' leftovers
    order = list(range(len(CASES))) + [0]
    for k, i in enumerate(order):
        poison = 7.0 + k
        compare(CASES[i], xs[i], static_path(CASES[i], xs[i], poison), expected[i], poison)


def test_static_scratch_entry_refuses_what_does_not_fit():
    from paper_2606_07577_b200 import omnimem
    lib = omnimem.load_library()
    wl = I.CFG2                                    # all 28 layers at once: 28 * 4 * 38364 floats > 2^20
    assert wl.L * wl.Hkv * (2 * wl.cache_cap + wl.Nn_v + wl.Nn_a) > omnimem.STATIC_SCRATCH_FLOATS
    one = torch.zeros(1, dtype=torch.int32, device="cuda:0")   # never dereferenced: the size check comes first
    p = one.data_ptr()
    rc = lib.omnimem_redundancy_static(omnimem.OMNIMEM_BF16, wl.L, wl.Hkv, wl.D, wl.cache_cap, wl.Nn_v, wl.Nn_a, 1, 1,
                                       p, p, p, p, wl.Nn_v, wl.Nn_a, p, p, None)
    assert rc == -6 and b"OMNIMEM_STATIC_SCRATCH_FLOATS" in lib.omnimem_strerror(rc)
    # six layers of that shape do fit (what the header promises)
    assert 6 * wl.Hkv * (2 * wl.cache_cap + wl.Nn_v + wl.Nn_a) <= omnimem.STATIC_SCRATCH_FLOATS
    rc = lib.omnimem_redundancy_static(omnimem.OMNIMEM_BF16, 1, 1, 128, 16, 4, 4, 1, 1, None, p, p, p, 4, 4, p, p, None)
    assert rc == -1                                # NULL input
    rc = lib.omnimem_redundancy_static(omnimem.OMNIMEM_BF16, 1, 1, 128, 16, 4, 4, 1, 1, p, p, p, p, 5, 4, p, p, None)
    assert rc == -5                                # chunk larger than the stated maximum
