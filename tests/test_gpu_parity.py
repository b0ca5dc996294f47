"""GPU parity: the CUDA path (through the C-ABI binding) against the CPU oracle, element by
element on the same seeded inputs.  Tolerances (BASELINE.json north_star): |dE| <= 1e-10 Eh and
relative error <= 1e-9; on inputs whose |E| is far above 1 Eh only the relative bound can hold
(one ulp of E exceeds 1e-10), so the absolute bound is asserted where
|E| < 10 Eh and on the scaled twins.
"""
import numpy as np
import pytest

import oracle
from paper_2512_01055_b200 import synth

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu

ABS_TOL = 1e-10
REL_TOL = 1e-9


@pytest.fixture(scope="module")
def ctx():
    from paper_2512_01055_b200 import binding
    c = binding.Context(0)
    yield c
    c.close()


def dev(a):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


class DevProblem:
    def __init__(self, p):
        self.p = p
        self.eps_occ, self.eps_vir, self.t1, self.t2 = dev(p.eps_occ), dev(p.eps_vir), dev(p.t1), dev(p.t2)
        self.Boo, self.Bov, self.Bvv = dev(p.Boo), dev(p.Bov), dev(p.Bvv)
        if p.vvvo is not None:
            self.vvvo, self.ovoo, self.ovov = dev(p.vvvo), dev(p.ovoo), dev(p.ovov)

    def blocks(self):
        return (self.vvvo, self.ovoo, self.ovov)

    def df(self):
        return (self.p.naux, self.Boo, self.Bov, self.Bvv)


def run_slice(ctx, dp, first, count, use_df=False):
    p = dp.p
    nb = ctx.workspace_bytes(p.o, p.v, p.naux if use_df else 0)
    ws = torch.empty(nb, dtype=torch.uint8, device="cuda")
    S = torch.full((max(count, 1),), float("nan"), dtype=torch.float64, device="cuda")
    kw = dict(df=dp.df()) if use_df else dict(blocks=dp.blocks())
    E = ctx.triples_energy_slice(p.o, p.v, dp.eps_occ, dp.eps_vir, dp.t1, dp.t2, workspace=ws, workspace_bytes=nb,
                                 first=first, count=count, S_dev=S, **kw)
    return E, S.cpu().numpy()[:count]


def assert_energy(E, E_ref):
    err = abs(E - E_ref)
    assert err <= REL_TOL * abs(E_ref) + (ABS_TOL if abs(E_ref) < 10 else 0.0), (E, E_ref, err)
    if abs(E_ref) < 10:
        assert err <= ABS_TOL, (E, E_ref, err)


# ---- W alone (steps a3 + a4), any order of i, j, k ------------------------------------------
@pytest.mark.parametrize("o,v,naux,seed", [(3, 4, 5, 11), (4, 19, 7, 12), (5, 37, 9, 13), (3, 48, 6, 14)])
def test_W_matches_oracle(ctx, o, v, naux, seed):
    p = synth.make_problem(o, v, naux, seed, sigma_B=0.3, blocks=True)
    dp = DevProblem(p)
    rng = np.random.default_rng(seed)
    trips = [(o - 1, 1, 0), (1, o - 1, 0), (0, 0, 1), (2, 2, 2)] + [tuple(rng.integers(0, o, 3)) for _ in range(3)]
    W = torch.empty((v, v, v), dtype=torch.float64, device="cuda")
    for (i, j, k) in trips:
        i, j, k = int(i), int(j), int(k)
        W.fill_(float("nan"))
        ctx.debug_W_triplet(o, v, i, j, k, dp.t2, dp.blocks(), W)
        W_ref = oracle.W_triplet(o, v, i, j, k, p.t2, p.vvvo[i], p.vvvo[j], p.vvvo[k], p.ovoo)
        got = W.cpu().numpy()
        scale = np.abs(W_ref).max()
        assert np.isfinite(got).all()
        assert np.abs(got - W_ref).max() <= 1e-13 * scale * max(v, 8), (i, j, k, np.abs(got - W_ref).max(), scale)


# ---- worked closed-form examples (tests/golden/p10_worked_values.txt via the oracle) -----------
@pytest.mark.parametrize("o,v,naux", [(3, 4, 5), (4, 6, 7), (2, 5, 3), (5, 3, 4)])
def test_closed_form_examples(ctx, o, v, naux):
    p = synth.closed_form_problem(o, v, naux)
    dp = DevProblem(p)
    n = oracle.triplet_count(o)
    E_ref, S_ref = oracle.triples_energy(p)
    E, S = run_slice(ctx, dp, 0, n)
    assert_energy(E, E_ref)
    assert np.abs(S - S_ref).max() <= ABS_TOL


# ---- random problems, ragged sizes, blocks and DF input ----------------------------------------
@pytest.mark.parametrize("o,v,naux,seed", [(1, 5, 3, 1), (2, 1, 3, 2), (3, 8, 4, 3), (4, 17, 6, 4), (5, 33, 8, 5), (6, 40, 20, 6)])
@pytest.mark.parametrize("use_df", [False, True])
def test_energy_small(ctx, o, v, naux, seed, use_df):
    p = synth.make_problem(o, v, naux, seed, sigma_B=0.25, blocks=True)
    dp = DevProblem(p)
    n = oracle.triplet_count(o)
    E_ref, S_ref = oracle.triples_energy(p)
    E, S = run_slice(ctx, dp, 0, n, use_df=use_df)
    tol = REL_TOL * max(np.abs(S_ref).max(), 1e-300)
    assert np.abs(S - S_ref).max() <= tol + (ABS_TOL if np.abs(S_ref).max() < 10 else 0), np.abs(S - S_ref).max()
    assert_energy(E, E_ref)


def test_cfg0_full(ctx):
    p = synth.make_config("cfg0", blocks=True)
    dp = DevProblem(p)
    n = oracle.triplet_count(p.o)
    E_ref, S_ref = oracle.triples_energy(p)
    for use_df in (False, True):
        E, S = run_slice(ctx, dp, 0, n, use_df=use_df)
        assert np.abs(S - S_ref).max() <= REL_TOL * np.abs(S_ref).max()
        assert_energy(E, E_ref)
    # the full-range call and a middle slice agree with the per-triplet values
    nb = ctx.workspace_bytes(p.o, p.v, 0)
    ws = torch.empty(nb, dtype=torch.uint8, device="cuda")
    E_full = ctx.triples_energy(p.o, p.v, dp.eps_occ, dp.eps_vir, dp.t1, dp.t2, blocks=dp.blocks(), workspace=ws,
                                workspace_bytes=nb)
    assert_energy(E_full, E_ref)
    E_mid, S_mid = run_slice(ctx, dp, 17, 40)
    assert np.abs(S_mid - S_ref[17:57]).max() <= REL_TOL * np.abs(S_ref).max()


def test_cfg0_scaled_twin_absolute_bound(ctx):
    """Same shapes as cfg0 with sigma_B reduced so that |E| ~ 1e-3 Eh: the absolute 1e-10 Eh bound binds."""
    p = synth.make_config("cfg0", blocks=True, sigma_B=0.02)
    dp = DevProblem(p)
    E_ref, S_ref = oracle.triples_energy(p)
    E, S = run_slice(ctx, dp, 0, oracle.triplet_count(p.o))
    assert abs(E_ref) < 1.0
    assert abs(E - E_ref) <= ABS_TOL and abs(E - E_ref) <= REL_TOL * abs(E_ref)
    assert np.abs(S - S_ref).max() <= ABS_TOL


@pytest.mark.parametrize("nslots", [3, 4, 7])
def test_slice_cache_blocked_schedule(ctx, nslots):
    """DF input with a workspace too small for all (vv|v.) slices: the blocked schedule with a slice cache
    (the cfg4 path) must give the same per-triplet S_ijk, on a full range and on a middle slice."""
    p = synth.make_problem(9, 24, 10, 41, sigma_B=0.25, blocks=True)
    dp = DevProblem(p)
    o, v, naux = p.o, p.v, p.naux
    n = oracle.triplet_count(o)
    E_ref, S_ref = oracle.triples_energy(p)
    full = ctx.workspace_bytes(o, v, naux)
    slice_bytes = (v ** 3 * 8 + 255) // 256 * 256
    budget = full - (o - nslots) * slice_bytes
    nb = ctx.workspace_bytes(o, v, naux, budget)
    assert nb <= budget < full
    ws = torch.empty(nb, dtype=torch.uint8, device="cuda")
    for first, count in ((0, n), (37, 61)):
        S = torch.full((count,), float("nan"), dtype=torch.float64, device="cuda")
        E = ctx.triples_energy_slice(o, v, dp.eps_occ, dp.eps_vir, dp.t1, dp.t2, df=dp.df(), workspace=ws, workspace_bytes=nb,
                                     first=first, count=count, S_dev=S)
        got = S.cpu().numpy()
        assert np.abs(got - S_ref[first:first + count]).max() <= REL_TOL * np.abs(S_ref).max()
        st = ctx.get_stats()
        assert st["slices_built"] >= min(o, 3)
    assert_energy(ctx.triples_energy_slice(o, v, dp.eps_occ, dp.eps_vir, dp.t1, dp.t2, df=dp.df(), workspace=ws,
                                           workspace_bytes=nb, first=0, count=n), E_ref)
    with pytest.raises(Exception):   # two slots cannot hold the three slices of a triplet
        ctx.workspace_bytes(o, v, naux, full - (o - 2) * slice_bytes)


def test_host_entry_point(ctx):
    p = synth.make_problem(4, 21, 9, 21, sigma_B=0.25, blocks=True)
    E_ref, _ = oracle.triples_energy(p)
    E, nbytes = ctx.triples_energy_host(p.o, p.v, p.naux, p.eps_occ, p.eps_vir, p.t1, p.t2, p.Boo, p.Bov, p.Bvv)
    assert_energy(E, E_ref)
    assert nbytes == 8 * (p.o + p.v + p.t1.size + p.t2.size + p.Boo.size + p.Bov.size + p.Bvv.size)


def test_build_blocks_matches_oracle(ctx):
    p = synth.make_problem(4, 21, 9, 31, blocks=False)
    dp = DevProblem(p)
    o, v, naux = p.o, p.v, p.naux
    vvvo = torch.empty((o, v, v, v), dtype=torch.float64, device="cuda")
    ovoo = torch.empty((o, o, o, v), dtype=torch.float64, device="cuda")
    ovov = torch.empty((o, o, v, v), dtype=torch.float64, device="cuda")
    ctx.build_blocks(o, v, naux, dp.Boo, dp.Bov, dp.Bvv, 0, o, vvvo, ovoo, ovov)
    torch.cuda.synchronize()
    for x in range(o):
        ref = oracle.build_vvvo_slice(o, v, naux, x, p.Bov, p.Bvv)
        assert np.abs(vvvo[x].cpu().numpy() - ref).max() <= 1e-14 * naux
    assert np.abs(ovoo.cpu().numpy() - oracle.build_ovoo(o, v, naux, p.Boo, p.Bov)).max() <= 1e-14 * naux
    assert np.abs(ovov.cpu().numpy() - oracle.build_ovov(o, v, naux, p.Bov)).max() <= 1e-14 * naux


def test_deterministic(ctx):
    p = synth.make_problem(5, 33, 8, 5, sigma_B=0.25, blocks=True)
    dp = DevProblem(p)
    n = oracle.triplet_count(p.o)
    E1, S1 = run_slice(ctx, dp, 0, n)
    E2, S2 = run_slice(ctx, dp, 0, n)
    assert E1 == E2 and (S1 == S2).all()


def test_argument_errors(ctx):
    from paper_2512_01055_b200.binding import TcError
    p = synth.make_problem(3, 8, 4, 3, blocks=True)
    dp = DevProblem(p)
    ws = torch.empty(1 << 20, dtype=torch.uint8, device="cuda")
    with pytest.raises(TcError):   # both blocks and df
        ctx.triples_energy(p.o, p.v, dp.eps_occ, dp.eps_vir, dp.t1, dp.t2, blocks=dp.blocks(), df=dp.df(), workspace=ws,
                           workspace_bytes=ws.numel())
    with pytest.raises(TcError):   # workspace too small
        ctx.triples_energy(p.o, p.v, dp.eps_occ, dp.eps_vir, dp.t1, dp.t2, blocks=dp.blocks(), workspace=ws, workspace_bytes=16)
    with pytest.raises(TcError):   # range outside
        ctx.triples_energy_slice(p.o, p.v, dp.eps_occ, dp.eps_vir, dp.t1, dp.t2, blocks=dp.blocks(), workspace=ws,
                                 workspace_bytes=ws.numel(), first=5, count=100)
    with pytest.raises(TcError):   # host pointer where a device pointer is required
        ctx.triples_energy(p.o, p.v, p.eps_occ.ctypes.data, dp.eps_vir, dp.t1, dp.t2, blocks=dp.blocks(), workspace=ws,
                           workspace_bytes=ws.numel())


def test_empty_range_and_fallback_kernel_on_even_v(ctx, monkeypatch):
    """count = 0 is a valid (empty) range; the cp.async fallback kernel (used for odd v) gives the same numbers as the
    TMA kernel on an even-v problem (TC_FORCE_CPASYNC is a testing aid of the library)."""
    p = synth.make_problem(4, 24, 6, 9, sigma_B=0.25, blocks=True)
    dp = DevProblem(p)
    n = oracle.triplet_count(p.o)
    E0, _ = run_slice(ctx, dp, 3, 0)
    assert E0 == 0.0
    E_ref, S_ref = oracle.triples_energy(p)
    E_tma, S_tma = run_slice(ctx, dp, 0, n)
    monkeypatch.setenv("TC_FORCE_CPASYNC", "1")
    E_cp, S_cp = run_slice(ctx, dp, 0, n)
    monkeypatch.delenv("TC_FORCE_CPASYNC")
    for E, S in ((E_tma, S_tma), (E_cp, S_cp)):
        assert np.abs(S - S_ref).max() <= REL_TOL * np.abs(S_ref).max()
        assert_energy(E, E_ref)
