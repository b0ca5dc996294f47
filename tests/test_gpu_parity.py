"""GPU parity: the CUDA path (through the C-ABI binding) against the CPU oracle, element by
element on the same seeded inputs.  Tolerances (BASELINE.json north_star): |dE| <= 1e-10 Eh and
relative error <= 1e-9; on inputs whose |E| is far above 1 Eh only the relative bound can hold
(one ulp of E exceeds 1e-10), so the absolute bound is asserted where
|E| < 10 Eh and on the scaled twins.
"""
import numpy as np
import pytest

import harness
import oracle
from paper_2512_01055_b200 import binding as binding_mod
from paper_2512_01055_b200 import synth

from paper_2512_01055_b200.binding import TC_KERNEL_TMA

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


def run_slice(ctx, dp, first, count, use_df=False, expect_kernel=None):
    p = dp.p
    nb = ctx.workspace_bytes(p.o, p.v, p.naux if use_df else 0)
    ws = torch.empty(nb, dtype=torch.uint8, device="cuda")
    S = torch.full((max(count, 1),), float("nan"), dtype=torch.float64, device="cuda")
    kw = dict(df=dp.df()) if use_df else dict(blocks=dp.blocks())
    E = ctx.triples_energy_slice(p.o, p.v, dp.eps_occ, dp.eps_vir, dp.t1, dp.t2, workspace=ws, workspace_bytes=nb,
                                 first=first, count=count, S_dev=S, **kw)
    if expect_kernel is not None and count > 0:
        assert ctx.get_stats()["kernel"] == expect_kernel, ctx.get_stats()
    return E, S.cpu().numpy()[:count]


def hole_chunks(o):
    return (o + 3) // 4


def chunks_per_step(o, v):
    """cps of csrc/tc_wbuild_tma.cu: the deferred flush is taken when cps >= 16."""
    return 2 * hole_chunks(o) + (v + 3) // 4


def assert_energy(E, E_ref):
    err = abs(E - E_ref)
    assert err <= REL_TOL * abs(E_ref) + (ABS_TOL if abs(E_ref) < 10 else 0.0), (E, E_ref, err)
    if abs(E_ref) < 10:
        assert err <= ABS_TOL, (E, E_ref, err)


# ---- W alone (steps a3 + a4), any order of i, j, k ------------------------------------------
# (5,64) and (9,50): deferred-flush sizes with 2 and 3 hole chunks, the second with ragged tiles (50 = 3*16 + 2)
@pytest.mark.parametrize("o,v,naux,seed", [(3, 4, 5, 11), (4, 19, 7, 12), (5, 37, 9, 13), (3, 48, 6, 14), (5, 64, 8, 15), (9, 50, 10, 16)])
def test_W_matches_oracle(ctx, o, v, naux, seed):
    p = harness.make_problem(o, v, naux, seed, sigma_B=0.3, blocks=True)
    dp = DevProblem(p)
    rng = np.random.default_rng(seed)
    trips = [(o - 1, 1, 0), (1, o - 1, 0), (0, 0, 1), (2, 2, 2)] + [tuple(rng.integers(0, o, 3)) for _ in range(3)]
    W = torch.empty((v, v, v), dtype=torch.float64, device="cuda")
    for (i, j, k) in trips:
        i, j, k = int(i), int(j), int(k)
        W.fill_(float("nan"))
        ctx.debug_W_triplet(o, v, i, j, k, dp.t2, dp.blocks(), W)
        assert ctx.get_stats()["kernel"] == TC_KERNEL_TMA          # every v takes the TMA kernel (odd v through padded copies)
        W_ref = oracle.W_triplet(o, v, i, j, k, p.t2, p.vvvo[i], p.vvvo[j], p.vvvo[k], p.ovoo)
        got = W.cpu().numpy()
        scale = np.abs(W_ref).max()
        assert np.isfinite(got).all()
        assert np.abs(got - W_ref).max() <= 1e-13 * scale * max(v, 8), (i, j, k, np.abs(got - W_ref).max(), scale)


# ---- worked closed-form examples (tests/golden/p10_worked_values.txt via the oracle) -----------
@pytest.mark.parametrize("o,v,naux", [(3, 4, 5), (4, 6, 7), (2, 5, 3), (5, 3, 4)])
def test_closed_form_examples(ctx, o, v, naux):
    p = harness.closed_form_problem(o, v, naux)
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
    p = harness.make_problem(o, v, naux, seed, sigma_B=0.25, blocks=True)
    dp = DevProblem(p)
    n = oracle.triplet_count(o)
    E_ref, S_ref = oracle.triples_energy(p)
    E, S = run_slice(ctx, dp, 0, n, use_df=use_df, expect_kernel=TC_KERNEL_TMA)
    assert ctx.get_stats()["padded"] == (v % 2)
    tol = REL_TOL * max(np.abs(S_ref).max(), 1e-300)
    assert np.abs(S - S_ref).max() <= tol + (ABS_TOL if np.abs(S_ref).max() < 10 else 0), np.abs(S - S_ref).max()
    assert_energy(E, E_ref)


# ---- the paths k_wbuild_tma takes at full size: deferred flush (cps >= 16) with every hole-chunk count,
#      full range in ONE multi-triplet launch, even v (ragged and not), blocks and DF input --------------------
DEFERRED_CASES = [(3, 64, 6, 21), (5, 64, 8, 22), (9, 50, 10, 23), (12, 40, 8, 24), (16, 72, 12, 25), (21, 56, 10, 26),
                  (7, 58, 9, 27)]   # nhc = 1, 2, 3 (ragged v), 3, 4 (ragged), 6, 2 (v mod 16 = 10)


@pytest.mark.parametrize("o,v,naux,seed", DEFERRED_CASES)
@pytest.mark.parametrize("use_df", [False, True])
def test_energy_deferred_flush_paths(ctx, o, v, naux, seed, use_df):
    assert chunks_per_step(o, v) >= 16 and v % 2 == 0
    p = harness.make_problem(o, v, naux, seed, sigma_B=0.25, blocks=True)
    dp = DevProblem(p)
    n = oracle.triplet_count(o)
    E_ref, S_ref = oracle.triples_energy(p)
    E, S = run_slice(ctx, dp, 0, n, use_df=use_df, expect_kernel=TC_KERNEL_TMA)
    st = ctx.get_stats()
    nb16 = (v + 15) // 16
    assert st["n_work_units"] == n * (nb16 * (nb16 + 1) * (nb16 + 2) // 6) and st["n_blocks"] == 0   # resident regime, one launch
    assert np.abs(S - S_ref).max() <= REL_TOL * np.abs(S_ref).max(), (np.abs(S - S_ref).max(), np.abs(S_ref).max())
    assert_energy(E, E_ref)


def test_odd_v_takes_the_same_kernel(ctx):
    """Odd v runs on the one W-builder there is (TMA / mbarrier / TMEM) through a zero-padded copy of t2 (row length
    v + 1); slices and (ov|oo)^T are laid out by the library, so nothing else depends on the parity of v."""
    p = harness.make_problem(6, 37, 9, 33, sigma_B=0.25, blocks=True)
    dp = DevProblem(p)
    n = oracle.triplet_count(p.o)
    E_ref, S_ref = oracle.triples_energy(p)
    for use_df in (False, True):
        E, S = run_slice(ctx, dp, 0, n, use_df=use_df, expect_kernel=TC_KERNEL_TMA)
        assert ctx.get_stats()["padded"] == 1
        assert np.abs(S - S_ref).max() <= REL_TOL * np.abs(S_ref).max()
        assert_energy(E, E_ref)


def test_misaligned_t2_is_rejected(ctx):
    """t2 is a TMA operand: a pointer that is not 16-byte aligned is an argument error, not a slow path."""
    p = harness.make_problem(4, 24, 6, 9, sigma_B=0.25, blocks=True)
    dp = DevProblem(p)
    n = oracle.triplet_count(p.o)
    buf = torch.empty(p.t2.size + 1, dtype=torch.float64, device="cuda")
    t2_off = buf[1:]                                   # 8 bytes past a 256-byte boundary
    t2_off.copy_(dp.t2.reshape(-1))
    assert t2_off.data_ptr() % 16 == 8
    nb = ctx.workspace_bytes(p.o, p.v, 0)
    ws = torch.empty(nb, dtype=torch.uint8, device="cuda")
    with pytest.raises(binding_mod.TcError) as e:
        ctx.triples_energy_slice(p.o, p.v, dp.eps_occ, dp.eps_vir, dp.t1, t2_off, blocks=dp.blocks(), workspace=ws,
                                 workspace_bytes=nb, first=0, count=n)
    assert e.value.status == 1
    # blocks whose base pointers are only 8-byte aligned are fine: the library re-lays them out itself
    E_ref, S_ref = oracle.triples_energy(p)
    vb = torch.empty(p.vvvo.size + 1, dtype=torch.float64, device="cuda")[1:]
    vb.copy_(dp.vvvo.reshape(-1))
    S = torch.empty(n, dtype=torch.float64, device="cuda")
    E = ctx.triples_energy_slice(p.o, p.v, dp.eps_occ, dp.eps_vir, dp.t1, dp.t2, blocks=(vb, dp.ovoo, dp.ovov), workspace=ws,
                                 workspace_bytes=nb, first=0, count=n, S_dev=S)
    assert np.abs(S.cpu().numpy() - S_ref).max() <= REL_TOL * np.abs(S_ref).max()
    assert_energy(E, E_ref)


def test_cfg0_full(ctx):
    p = harness.make_config("cfg0", blocks=True)
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
    p = harness.make_config("cfg0", blocks=True, sigma_B=0.02)
    dp = DevProblem(p)
    E_ref, S_ref = oracle.triples_energy(p)
    E, S = run_slice(ctx, dp, 0, oracle.triplet_count(p.o))
    assert abs(E_ref) < 1.0
    assert abs(E - E_ref) <= ABS_TOL and abs(E - E_ref) <= REL_TOL * abs(E_ref)
    assert np.abs(S - S_ref).max() <= ABS_TOL


@pytest.mark.parametrize("dims", [(9, 24, 10, 41), (8, 37, 9, 42), (9, 50, 10, 23)], ids=["v24", "v37-odd", "v50-deferred"])
@pytest.mark.parametrize("nslots", [3, 4, 7])
def test_slice_cache_blocked_schedule(ctx, nslots, dims):
    """DF input with a workspace too small for all (vv|v.) slices: the blocked schedule with a slice cache
    (the cfg4 path) must give the same per-triplet S_ijk, on a full range and on a middle slice."""
    assert nslots < dims[0]
    p = harness.make_problem(*dims, sigma_B=0.25, blocks=True)
    dp = DevProblem(p)
    o, v, naux = p.o, p.v, p.naux
    n = oracle.triplet_count(o)
    E_ref, S_ref = oracle.triples_energy(p)
    full = ctx.workspace_bytes(o, v, naux)
    slice_bytes = harness.tiled_slice_bytes(v)
    budget = full - (o - nslots) * slice_bytes
    nb = ctx.workspace_bytes(o, v, naux, budget)
    assert nb <= budget < full
    ws = torch.empty(nb, dtype=torch.uint8, device="cuda")
    for first, count in ((0, n), (n // 4, n // 3)):
        S = torch.full((count,), float("nan"), dtype=torch.float64, device="cuda")
        E = ctx.triples_energy_slice(o, v, dp.eps_occ, dp.eps_vir, dp.t1, dp.t2, df=dp.df(), workspace=ws, workspace_bytes=nb,
                                     first=first, count=count, S_dev=S)
        got = S.cpu().numpy()
        assert np.abs(got - S_ref[first:first + count]).max() <= REL_TOL * np.abs(S_ref).max()
        st = ctx.get_stats()
        plan = binding_mod.plan_summary(o, first, count, nslots)
        assert st["slices_built"] == plan["n_loads"] and st["n_blocks"] == plan["n_blocks"] and st["kernel"] == TC_KERNEL_TMA
        # a2 runs on the side stream: its interval lies inside the call and starts before the last W-builder ends
        assert 0.0 <= st["staging_first_ms"] <= st["staging_last_ms"] <= st["ms_total"]
        assert st["staging_first_ms"] < st["contraction_last_ms"]
    assert_energy(ctx.triples_energy_slice(o, v, dp.eps_occ, dp.eps_vir, dp.t1, dp.t2, df=dp.df(), workspace=ws,
                                           workspace_bytes=nb, first=0, count=n), E_ref)
    with pytest.raises(Exception):   # two slots cannot hold the three slices of a triplet
        ctx.workspace_bytes(o, v, naux, full - (o - 2) * slice_bytes)


def test_host_entry_point(ctx):
    p = harness.make_problem(4, 21, 9, 21, sigma_B=0.25, blocks=True)
    E_ref, _ = oracle.triples_energy(p)
    E, nbytes = ctx.triples_energy_host(p.o, p.v, p.naux, p.eps_occ, p.eps_vir, p.t1, p.t2, p.Boo, p.Bov, p.Bvv)
    assert_energy(E, E_ref)
    assert nbytes == 8 * (p.o + p.v + p.t1.size + p.t2.size + p.Boo.size + p.Bov.size + p.Bvv.size)


def test_build_blocks_matches_oracle(ctx):
    p = harness.make_problem(4, 21, 9, 31, blocks=False)
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


def test_deterministic_tma_kernel(ctx):
    """Bit-reproducibility of the TMA kernel on a deferred-flush size (cps >= 16), full range, four runs: the flush has
    no CTA barrier and rests on a ring-ordering argument -- a race would show up here first."""
    p = harness.make_problem(9, 50, 10, 23, sigma_B=0.25, blocks=True)
    assert chunks_per_step(p.o, p.v) >= 16
    dp = DevProblem(p)
    n = oracle.triplet_count(p.o)
    runs = [run_slice(ctx, dp, 0, n, use_df=(r % 2 == 1), expect_kernel=TC_KERNEL_TMA) for r in range(6)]
    for r in (2, 4):
        assert runs[r][0] == runs[0][0] and (runs[r][1] == runs[0][1]).all()
    for r in (3, 5):
        assert runs[r][0] == runs[1][0] and (runs[r][1] == runs[1][1]).all()


def test_deterministic_odd_v(ctx):
    p = harness.make_problem(5, 33, 8, 5, sigma_B=0.25, blocks=True)
    dp = DevProblem(p)
    n = oracle.triplet_count(p.o)
    E1, S1 = run_slice(ctx, dp, 0, n)
    E2, S2 = run_slice(ctx, dp, 0, n)
    assert E1 == E2 and (S1 == S2).all()


def test_workspace_canaries(ctx):
    """Bounds check of our own (compute-sanitizer is closed on this pool): guard bands before and after the workspace,
    around S_dev and copies of the read-only inputs must be untouched by the calls, resident and blocked regime."""
    p = harness.make_problem(9, 50, 10, 23, sigma_B=0.25, blocks=True)
    dp = DevProblem(p)
    o, v, naux = p.o, p.v, p.naux
    n = oracle.triplet_count(o)
    E_ref, S_ref = oracle.triples_energy(p)
    guard = 1 << 16
    full = ctx.workspace_bytes(o, v, naux)
    small = ctx.workspace_bytes(o, v, naux, full - (o - 4) * harness.tiled_slice_bytes(v))
    t2_copy, Bvv_copy = dp.t2.clone(), dp.Bvv.clone()
    for nb in (full, small):
        buf = torch.full((nb + 2 * guard,), 0xA5, dtype=torch.uint8, device="cuda")
        Sbuf = torch.full((n + 64,), 12345.0, dtype=torch.float64, device="cuda")
        ws = buf[guard:guard + nb]
        assert ws.data_ptr() % 256 == 0
        E = ctx.triples_energy_slice(o, v, dp.eps_occ, dp.eps_vir, dp.t1, dp.t2, df=dp.df(), workspace=ws, workspace_bytes=nb,
                                     first=0, count=n, S_dev=Sbuf[32:32 + n])
        assert_energy(E, E_ref)
        assert bool((buf[:guard] == 0xA5).all()) and bool((buf[guard + nb:] == 0xA5).all())
        assert bool((Sbuf[:32] == 12345.0).all()) and bool((Sbuf[32 + n:] == 12345.0).all())
        assert np.abs(Sbuf[32:32 + n].cpu().numpy() - S_ref).max() <= REL_TOL * np.abs(S_ref).max()
    assert torch.equal(t2_copy, dp.t2) and torch.equal(Bvv_copy, dp.Bvv)


def test_argument_errors(ctx):
    from paper_2512_01055_b200.binding import TcError
    p = harness.make_problem(3, 8, 4, 3, blocks=True)
    dp = DevProblem(p)
    ws = torch.empty(1 << 20, dtype=torch.uint8, device="cuda")
    with pytest.raises(TcError):   # both blocks and df
        ctx.triples_energy(p.o, p.v, dp.eps_occ, dp.eps_vir, dp.t1, dp.t2, blocks=dp.blocks(), df=dp.df(), workspace=ws,
                           workspace_bytes=ws.numel())
    with pytest.raises(TcError) as e:   # workspace too small
        ctx.triples_energy(p.o, p.v, dp.eps_occ, dp.eps_vir, dp.t1, dp.t2, blocks=dp.blocks(), workspace=ws, workspace_bytes=16)
    assert e.value.status == 3
    with pytest.raises(TcError) as e:   # workspace_bytes = 0 is "too small", never "unbounded" (blocks and DF input)
        ctx.triples_energy(p.o, p.v, dp.eps_occ, dp.eps_vir, dp.t1, dp.t2, blocks=dp.blocks(), workspace=ws, workspace_bytes=0)
    assert e.value.status == 3
    with pytest.raises(TcError) as e:
        ctx.triples_energy(p.o, p.v, dp.eps_occ, dp.eps_vir, dp.t1, dp.t2, df=dp.df(), workspace=ws, workspace_bytes=0)
    assert e.value.status == 3
    with pytest.raises(TcError):   # range outside
        ctx.triples_energy_slice(p.o, p.v, dp.eps_occ, dp.eps_vir, dp.t1, dp.t2, blocks=dp.blocks(), workspace=ws,
                                 workspace_bytes=ws.numel(), first=5, count=100)
    with pytest.raises(TcError):   # host pointer where a device pointer is required
        ctx.triples_energy(p.o, p.v, p.eps_occ.ctypes.data, dp.eps_vir, dp.t1, dp.t2, blocks=dp.blocks(), workspace=ws,
                           workspace_bytes=ws.numel())


def test_empty_range(ctx):
    """count = 0 is a valid (empty) range."""
    p = harness.make_problem(4, 24, 6, 9, sigma_B=0.25, blocks=True)
    dp = DevProblem(p)
    E0, _ = run_slice(ctx, dp, 3, 0)
    assert E0 == 0.0
    E0, _ = run_slice(ctx, dp, 3, 0, use_df=True)
    assert E0 == 0.0


# ---- NEXT-3: host-resident amplitudes streamed through a device ring of rows -----------------
@pytest.mark.parametrize("o,v,naux,seed,nslots", [(9, 24, 10, 41, 4), (9, 24, 10, 41, 9), (7, 37, 9, 42, 5), (12, 40, 8, 24, 6)])
def test_streamed_t2_from_host(ctx, o, v, naux, seed, nslots):
    p = harness.make_problem(o, v, naux, seed, sigma_B=0.25, blocks=True)
    dp = DevProblem(p)
    n = oracle.triplet_count(o)
    E_ref, S_ref = oracle.triples_energy(p)
    t2_host = torch.from_numpy(np.ascontiguousarray(p.t2)).pin_memory()
    full = ctx.workspace_bytes_streamed(o, v, naux)
    ldv = v + (v % 2)
    per_slot = harness.tiled_slice_bytes(v) + (o * v * ldv * 8 + 255) // 256 * 256
    budget = full - (o - nslots) * per_slot
    nb = ctx.workspace_bytes_streamed(o, v, naux, budget)
    assert nb <= budget <= full
    ws = torch.empty(nb, dtype=torch.uint8, device="cuda")
    for first, count in ((0, n), (n // 3, n // 2)):
        S = torch.full((count,), float("nan"), dtype=torch.float64, device="cuda")
        E = ctx.triples_energy_streamed(o, v, dp.eps_occ, dp.eps_vir, dp.t1, t2_host, df=dp.df(), workspace=ws,
                                        workspace_bytes=nb, first=first, count=count, S_dev=S)
        st = ctx.get_stats()
        plan = binding_mod.plan_summary(o, first, count, nslots)
        assert st["t2_rows_copied"] == plan["n_loads"] == st["slices_built"] and st["kernel"] == TC_KERNEL_TMA
        assert st["bytes_h2d"] == plan["n_loads"] * o * v * v * 8
        assert np.abs(S.cpu().numpy() - S_ref[first:first + count]).max() <= REL_TOL * np.abs(S_ref).max()
        if first == 0:
            assert_energy(E, E_ref)
    with pytest.raises(binding_mod.TcError):   # a device pointer where the host array is expected
        ctx.triples_energy_streamed(o, v, dp.eps_occ, dp.eps_vir, dp.t1, dp.t2, df=dp.df(), workspace=ws, workspace_bytes=nb,
                                    first=0, count=n)


# ---- NEXT-1: triplet ranges per rank behind the boundary, all ranks' ranges on this one GPU --------
@pytest.mark.parametrize("world", [2, 3])
def test_partitioned_ranges_sum_to_the_full_energy(ctx, world):
    p = harness.make_config("cfg0", blocks=True)
    dp = DevProblem(p)
    n = oracle.triplet_count(p.o)
    E_ref, S_ref = oracle.triples_energy(p)
    E_full, _ = run_slice(ctx, dp, 0, n, use_df=True)
    parts, covered = [], 0
    for rank in range(world):
        first, count = binding_mod.triplet_partition(p.o, world, rank)
        assert first == covered
        covered += count
        E_r, S_r = run_slice(ctx, dp, first, count, use_df=True)
        assert np.abs(S_r - S_ref[first:first + count]).max() <= REL_TOL * np.abs(S_ref).max()
        parts.append(E_r)
    assert covered == n
    assert_energy(sum(parts), E_ref)
    assert abs(sum(parts) - E_full) <= 1e-13 * abs(E_full)


# ---- NEXT-2: the paper's abcijk schedule -- tile orbits outer, all triplets inner, integrals rebuilt per tile ----
@pytest.mark.parametrize("o,v,naux,seed", [(4, 24, 6, 9), (5, 37, 9, 13), (6, 40, 20, 6), (9, 50, 10, 23)])
def test_abcijk_schedule(ctx, o, v, naux, seed):
    """Same kernels, the paper's own loop order: E against the oracle, and the per-orbit energies against the oracle's sums
    restricted to the points of each tile orbit (tco_S_from_W_tile_orbit); a sub-range of orbits sums its own orbits."""
    p = harness.make_problem(o, v, naux, seed, sigma_B=0.25, blocks=True)
    dp = DevProblem(p)
    E_ref, _ = oracle.triples_energy(p)
    Eorb_ref = oracle.orbit_energies(p, 16)
    norb = binding_mod.tile_orbit_count(v)
    assert norb == len(Eorb_ref) == len(oracle.tile_orbits(v, 16))
    nb = ctx.workspace_bytes_abcijk(o, v, naux)
    # O(o v T^2) of integrals instead of o v^3: at cfg1 size the footprint is under a third of the resident schedule's (two tile orbits per launch)
    assert ctx.workspace_bytes_abcijk(20, 200, 600) < 0.3 * ctx.workspace_bytes(20, 200, 600)
    ws = torch.empty(nb, dtype=torch.uint8, device="cuda")
    Eorb = torch.full((norb,), float("nan"), dtype=torch.float64, device="cuda")
    E = ctx.triples_energy_abcijk(o, v, dp.eps_occ, dp.eps_vir, dp.t1, dp.t2, df=dp.df(), workspace=ws, workspace_bytes=nb,
                                  E_orbit_dev=Eorb)
    st = ctx.get_stats()
    assert st["kernel"] == TC_KERNEL_TMA and st["n_blocks"] == norb and st["slices_built"] == norb * o
    assert_energy(E, E_ref)
    got = Eorb.cpu().numpy()
    assert np.abs(got - Eorb_ref).max() <= REL_TOL * np.abs(Eorb_ref).max(), (got, Eorb_ref)
    assert abs(got.sum() - E) <= 1e-12 * abs(E)
    # a middle range of orbits
    f0, cnt = norb // 3, max(1, norb // 2)
    E2 = ctx.triples_energy_abcijk(o, v, dp.eps_occ, dp.eps_vir, dp.t1, dp.t2, df=dp.df(), workspace=ws, workspace_bytes=nb,
                                   orbit_first=f0, orbit_count=cnt, E_orbit_dev=Eorb)
    assert abs(E2 - Eorb_ref[f0:f0 + cnt].sum()) <= REL_TOL * np.abs(Eorb_ref).max() * cnt
    assert np.abs(Eorb.cpu().numpy()[:cnt] - Eorb_ref[f0:f0 + cnt]).max() <= REL_TOL * np.abs(Eorb_ref).max()
    with pytest.raises(binding_mod.TcError):
        ctx.triples_energy_abcijk(o, v, dp.eps_occ, dp.eps_vir, dp.t1, dp.t2, df=dp.df(), workspace=ws, workspace_bytes=nb,
                                  orbit_first=norb, orbit_count=1)


# ---- stream semantics: "work is enqueued on `stream`; the side stream is forked and joined with events so the caller sees
#      single-stream semantics" (include/tc_triples.h) --------------------------------------------------------------------------
@pytest.mark.parametrize("regime", ["resident", "blocked", "abcijk", "static"])
def test_caller_stream_ordering(ctx, regime):
    """Every input is PRODUCED on a non-blocking caller stream right before the call (behind ~10 ms of other work on that
    stream), and holds NaN until then: a library that ran on another stream, or whose side stream did not wait for the fork
    event, would read the NaNs.  The result must equal the default-stream result to the bit."""
    p = harness.make_problem(9, 24, 10, 41, sigma_B=0.25, blocks=False)
    dp = DevProblem(p)
    o, v, naux = p.o, p.v, p.naux
    n = oracle.triplet_count(o)
    names = ("eps_occ", "eps_vir", "t1", "t2", "Boo", "Bov", "Bvv")
    if regime == "blocked":
        nb = ctx.workspace_bytes(o, v, naux, ctx.workspace_bytes(o, v, naux) - (o - 3) * harness.tiled_slice_bytes(v))
    elif regime == "abcijk":
        nb = ctx.workspace_bytes_abcijk(o, v, naux)
    else:
        nb = ctx.workspace_bytes(o, v, naux)
    ws = torch.empty(nb, dtype=torch.uint8, device="cuda")

    def call(t, stream):
        df = (naux, t["Boo"], t["Bov"], t["Bvv"])
        S = torch.full((n,), float("nan"), dtype=torch.float64, device="cuda")
        a = (o, v, t["eps_occ"], t["eps_vir"], t["t1"], t["t2"])
        if regime == "abcijk":
            return ctx.triples_energy_abcijk(*a, df=df, workspace=ws, workspace_bytes=nb, stream=stream), None
        if regime == "static":
            return ctx.triples_energy_static(*a, df=df, stream=stream, first=0, count=n, S_dev=S), S
        return ctx.triples_energy_slice(*a, df=df, workspace=ws, workspace_bytes=nb, stream=stream, first=0, count=n, S_dev=S), S

    ref = {k: getattr(dp, k) for k in names}
    E_ref, S_ref = call(ref, None)
    if regime == "blocked":
        assert ctx.get_stats()["n_blocks"] >= 2
    late = {k: torch.full_like(ref[k], float("nan")) for k in names}
    junk = torch.randn(4096, 4096, device="cuda")
    torch.cuda.synchronize()
    s = torch.cuda.Stream()                          # non-blocking: no implicit ordering with the legacy default stream
    with torch.cuda.stream(s):
        for _ in range(8):
            junk = junk @ junk * 1e-3                # keeps the stream busy while the host runs ahead
        for k in names:
            late[k].copy_(ref[k])
        E, S = call(late, s)
    assert E == E_ref, (regime, E, E_ref)
    if S is not None:
        assert (S.cpu().numpy() == S_ref.cpu().numpy()).all()
