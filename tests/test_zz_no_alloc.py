"""tc_triples_energy_static: the energy call whose scratch is a static device array inside the library (no allocation on its path).

Collected last on purpose (the suite runs with pytest -x: a failure here must not hide the other tests).  Each test builds
its own context and inputs, so the file passes alone in a fresh process and after the rest of the suite.

The reference is the existing path (tc_triples_energy_slice with a caller-allocated workspace) on the same inputs: the same
kernels run on the same data, so E and every S_ijk must agree within the tolerance the parity tests use (in fact to the bit).
Two calls in a row on DIFFERENT problems: the second finds the first one's leftovers in the shared array.
"""
import numpy as np
import pytest

import harness
from paper_2512_01055_b200 import binding

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu

REL_TOL = 1e-9    # as tests/test_gpu_parity.py
ABS_TOL = 1e-10


def _dev(a):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def _problem(o, v, naux, seed, blocks):
    p = harness.make_problem(o, v, naux, seed, blocks=blocks)
    d = {k: _dev(getattr(p, k)) for k in ("eps_occ", "eps_vir", "t1", "t2", "Boo", "Bov", "Bvv")}
    if blocks:
        d.update({k: _dev(getattr(p, k)) for k in ("vvvo", "ovoo", "ovov")})
    return p, d


def _both_paths(ctx, p, d, use_df, first, count):
    kw = dict(df=(p.naux, d["Boo"], d["Bov"], d["Bvv"])) if use_df else dict(blocks=(d["vvvo"], d["ovoo"], d["ovov"]))
    args = (p.o, p.v, d["eps_occ"], d["eps_vir"], d["t1"], d["t2"])
    # existing path: caller-allocated workspace
    nb = ctx.workspace_bytes(p.o, p.v, p.naux if use_df else 0)
    assert nb <= binding.STATIC_SCRATCH_BYTES
    ws = torch.empty(nb, dtype=torch.uint8, device="cuda")
    S_ref = torch.full((count,), float("nan"), dtype=torch.float64, device="cuda")
    E_ref = ctx.triples_energy_slice(*args, workspace=ws, workspace_bytes=nb, first=first, count=count, S_dev=S_ref, **kw)
    # new path: no workspace argument at all
    S = torch.full((count,), float("nan"), dtype=torch.float64, device="cuda")
    E = ctx.triples_energy_static(*args, first=first, count=count, S_dev=S, **kw)
    assert ctx.get_stats()["kernel"] == binding.TC_KERNEL_TMA
    return E, S.cpu().numpy(), E_ref, S_ref.cpu().numpy()


def _assert_same(E, S, E_ref, S_ref):
    assert np.isfinite(S).all() and np.isfinite(S_ref).all()
    assert abs(E - E_ref) <= REL_TOL * abs(E_ref) + ABS_TOL, (E, E_ref)
    assert (np.abs(S - S_ref) <= REL_TOL * np.abs(S_ref) + ABS_TOL).all(), np.abs(S - S_ref).max()


def test_static_scratch_matches_workspace_path_on_two_calls_in_a_row():
    ctx = binding.Context(0)
    try:
        # call 1: cfg0-sized, DF input, all triplets (ragged v = 2 * 16 + 8)
        p1, d1 = _problem(8, 40, 120, 0, blocks=False)
        n1 = binding.triplet_count(p1.o)
        r1 = _both_paths(ctx, p1, d1, True, 0, n1)
        _assert_same(*r1)
        assert abs(r1[0]) > 1e-3                      # a real energy, not zeros
        # call 2, right after, on a different (smaller, odd-v, block-input) problem and a sub-range: other offsets into the
        # same array, which still holds call 1's data
        p2, d2 = _problem(5, 37, 30, 11, blocks=True)
        r2 = _both_paths(ctx, p2, d2, False, 3, 20)
        _assert_same(*r2)
        # and call 1 again: its result does not depend on what call 2 left behind
        r3 = _both_paths(ctx, p1, d1, True, 0, n1)
        assert r3[0] == r1[0] and (r3[1] == r1[1]).all()
    finally:
        ctx.close()


def test_static_scratch_rejects_problems_beyond_its_size():
    ctx = binding.Context(0)
    try:
        o, v, naux = 20, 200, 600                      # cfg1: 1.5 GB of scratch
        assert ctx.workspace_bytes(o, v, naux) > binding.STATIC_SCRATCH_BYTES
        z = torch.zeros(16, dtype=torch.float64, device="cuda")   # never read: the size check comes first
        with pytest.raises(binding.TcError) as ei:
            ctx.triples_energy_static(o, v, z, z, z, z, df=(naux, z, z, z), first=0, count=1)
        msg = str(ei.value)
        assert "static scratch" in msg and str(binding.STATIC_SCRATCH_BYTES) in msg, msg
    finally:
        ctx.close()
