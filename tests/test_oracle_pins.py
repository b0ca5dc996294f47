"""Pins of the CPU oracle (oracle/tc_oracle.c) to things other than itself.

P1..P10 of SURVEY.md section 8(c).  The independent formulas used here (the paper's
own eq. (1)/(2)/(5) form with the G index reading, and the spin-orbital textbook
(T) formula) are written with numpy einsum over full six-index tensors and share
nothing with the oracle's loops.  No GPU needed.
"""
import itertools
import os

import numpy as np
import pytest

import harness
import oracle
from paper_2512_01055_b200 import synth

GOLDEN = os.path.join(os.path.dirname(__file__), "golden", "p10_worked_values.txt")
IDX = lambda i, j, k: i * (i + 1) * (i + 2) // 6 + j * (j + 1) // 2 + k


# ----------------------------------------------------------------------------
# independent formulas (numpy, full tensors)
# ----------------------------------------------------------------------------
def full_eri(p):
    """(pq|rs) over all o+v orbitals from the DF factors, eq. (6)."""
    o, v = p.o, p.v
    N = o + v
    B = np.zeros((p.naux, N, N))
    B[:, :o, :o] = p.Boo
    B[:, :o, o:] = p.Bov
    B[:, o:, :o] = p.Bov.transpose(0, 2, 1)
    B[:, o:, o:] = p.Bvv
    return np.einsum("qpr,qst->prst", B, B)


def paper_form_energy(p):
    """Eqs. (1)-(5) exactly as printed with the G reading
    G_pq^rs = (rp|sq) (reading 2): virtual loop a>=b>=c with weight
    (2 - d_ab - d_bc), occupied-index permutations in the right factor."""
    o, v = p.o, p.v
    eri = full_eri(p)
    O, V = slice(0, o), slice(o, o + v)
    G_vovv = eri[V, O, V, V]        # (ai|bf)  [a,i,b,f]
    G_vooo = eri[V, O, O, O]        # (ai|lj)  [a,i,l,j]
    G_vovo = eri[V, O, V, O]        # (bj|ck)  [b,j,c,k]
    t2 = p.t2                       # [i,j,a,b]
    # A_ijk^abc = sum_f G_if^ab t_kj^cf - sum_l G_ij^al t_lk^bc
    A = (np.einsum("aibf,kjcf->ijkabc", G_vovv, t2)
         - np.einsum("ailj,lkbc->ijkabc", G_vooo, t2))
    # eq. (5): P A = A_ijk^abc + A_ikj^acb + A_jik^bac + A_jki^bca + A_kji^cba + A_kij^cab
    W = (A
         + A.transpose(0, 2, 1, 3, 5, 4)
         + A.transpose(1, 0, 2, 4, 3, 5)
         + np.einsum("jkibca->ijkabc", A)
         + np.einsum("kjicba->ijkabc", A)
         + np.einsum("kijcab->ijkabc", A))
    # eq. (3): V = t_i^a G_jk^bc + t_j^b G_ik^ac + t_k^c G_ij^ab, G_jk^bc = (bj|ck)
    Vd = (np.einsum("ia,bjck->ijkabc", p.t1, G_vovo)
          + np.einsum("jb,aick->ijkabc", p.t1, G_vovo)
          + np.einsum("kc,aibj->ijkabc", p.t1, G_vovo))
    eo, ev = p.eps_occ, p.eps_vir
    D = (eo[:, None, None, None, None, None] + eo[None, :, None, None, None, None]
         + eo[None, None, :, None, None, None] - ev[None, None, None, :, None, None]
         - ev[None, None, None, None, :, None] - ev[None, None, None, None, None, :])
    # eq. (1) right factor: occupied permutations at fixed abc
    Rr = (4 * W + np.einsum("jkiabc->ijkabc", W) + np.einsum("kijabc->ijkabc", W)
          - 2 * np.einsum("jikabc->ijkabc", W) - 2 * np.einsum("ikjabc->ijkabc", W)
          - 2 * np.einsum("kjiabc->ijkabc", W))
    X = ((W + Vd) * Rr / D).sum(axis=(0, 1, 2))      # [a,b,c]
    E = 0.0
    for a in range(v):
        for b in range(a + 1):
            for c in range(b + 1):
                E += (2 - (a == b) - (b == c)) * X[a, b, c]
    return E, W


def spin_orbital_energy(p):
    """Textbook spin-orbital (T): E = (1/36) sum t_c D (t_c + t_d) with
    D t_c = P(i/jk)P(a/bc)[ sum_e t_jk^ae <ei||bc> - sum_m t_im^bc <ma||jk> ],
    D t_d = P(i/jk)P(a/bc) t_i^a <jk||bc>,  P(p/qr) f(pqr) = f(pqr) - f(qpr) - f(rqp)."""
    o, v = p.o, p.v
    N = o + v
    eri = full_eri(p)                                  # chemists' (pq|rs), spatial
    # spin orbitals: index 2*p + s
    spat = np.repeat(np.arange(N), 2)
    spin = np.tile(np.arange(2), N)
    n = 2 * N
    chem = eri[np.ix_(spat, spat, spat, spat)] * (
        (spin[:, None, None, None] == spin[None, :, None, None])
        & (spin[None, None, :, None] == spin[None, None, None, :]))
    phys = chem.transpose(0, 2, 1, 3)                  # <pq|rs> = (pr|qs)
    anti = phys - phys.transpose(0, 1, 3, 2)           # <pq||rs>
    no, nv = 2 * o, 2 * v
    Os, Vs = slice(0, no), slice(no, n)
    so_o_spat, so_o_spin = spat[:no], spin[:no]
    so_v_spat, so_v_spin = spat[no:] - o, spin[no:]
    t1s = p.t1[np.ix_(so_o_spat, so_v_spat)] * (so_o_spin[:, None] == so_v_spin[None, :])
    t2sp = p.t2[np.ix_(so_o_spat, so_o_spat, so_v_spat, so_v_spat)]          # t_ij^ab spatial gathered
    t2sp_x = p.t2[np.ix_(so_o_spat, so_o_spat, so_v_spat, so_v_spat)].transpose(0, 1, 3, 2)
    d_ia_jb = ((so_o_spin[:, None, None, None] == so_v_spin[None, None, :, None])
               & (so_o_spin[None, :, None, None] == so_v_spin[None, None, None, :]))
    d_ib_ja = ((so_o_spin[:, None, None, None] == so_v_spin[None, None, None, :])
               & (so_o_spin[None, :, None, None] == so_v_spin[None, None, :, None]))
    t2s = t2sp * d_ia_jb - t2sp_x * d_ib_ja            # antisymmetrised spin-orbital doubles
    eps = np.concatenate([p.eps_occ, p.eps_vir])[spat]
    eo, ev = eps[:no], eps[no:]
    D = (eo[:, None, None, None, None, None] + eo[None, :, None, None, None, None]
         + eo[None, None, :, None, None, None] - ev[None, None, None, :, None, None]
         - ev[None, None, None, None, :, None] - ev[None, None, None, None, None, :])

    def P_perm(X):
        # P(i/jk): X(ijk) - X(jik) - X(kji) on axes 0,1,2 ; P(a/bc) on axes 3,4,5
        X = X - X.transpose(1, 0, 2, 3, 4, 5) - X.transpose(2, 1, 0, 3, 4, 5)
        X = X - X.transpose(0, 1, 2, 4, 3, 5) - X.transpose(0, 1, 2, 5, 4, 3)
        return X

    vovv = anti[Vs, Os, Vs, Vs]                        # <ei||bc> [e,i,b,c]
    ovoo = anti[Os, Vs, Os, Os]                        # <ma||jk> [m,a,j,k]
    oovv = anti[Os, Os, Vs, Vs]                        # <jk||bc>
    conn = P_perm(np.einsum("jkae,eibc->ijkabc", t2s, vovv)
                  - np.einsum("imbc,majk->ijkabc", t2s, ovoo))
    disc = P_perm(np.einsum("ia,jkbc->ijkabc", t1s, oovv))
    tc = conn / D
    td = disc / D
    return (tc * D * (tc + td)).sum() / 36.0


# ----------------------------------------------------------------------------
# P10: worked values
# ----------------------------------------------------------------------------
def _golden_rows():
    rows = []
    for line in open(GOLDEN):
        line = line.strip()
        if not line or line.startswith("#"):
            continue
        f = line.split()
        rows.append((f[0], int(f[1]), int(f[2]), int(f[3]), f[4:10], float(f[10])))
    return rows


@pytest.mark.parametrize("row", _golden_rows(), ids=lambda r: f"{r[0]}-{r[1]}{r[2]}{r[3]}-{''.join(r[4])}")
def test_p10_worked_values(row):
    kind, o, v, naux, ix, val = row
    p = harness.closed_form_problem(o, v, naux, t1_zero=(kind == "E_t1zero"))
    ii = [None if s == "-" else int(s) for s in ix]
    if kind in ("E", "E_t1zero"):
        got, _ = oracle.triples_energy(p)
    elif kind == "B000":
        got = p.Boo[0, 0, 0]
    elif kind == "ERI_bd_ck":
        k, b, c, d = ii[2], ii[4], ii[5], 1
        got = oracle.build_vvvo_slice(o, v, naux, k, p.Bov, p.Bvv)[d, b, c]
    elif kind == "T2":
        got = p.t2[ii[0], ii[1], ii[3], ii[4]]
    elif kind in ("W", "Y"):
        i, j, k, a, b, c = ii
        W = oracle.W_triplet(o, v, i, j, k, p.t2, p.vvvo[i], p.vvvo[j], p.vvvo[k], p.ovoo)
        if kind == "W":
            got = W[a, b, c]
        else:
            _, Y = oracle.S_from_W(o, v, i, j, k, p.eps_occ, p.eps_vir, p.t1, p.ovov, W, want_Y=True)
            got = Y[a, b, c]
    elif kind == "S":
        i, j, k = ii[:3]
        _, S = oracle.triples_energy(p, IDX(i, j, k), 1)
        got = S[0]
    else:
        raise AssertionError(kind)
    assert got == pytest.approx(val, rel=1e-12, abs=1e-15)


# ----------------------------------------------------------------------------
# P1 .. P7
# ----------------------------------------------------------------------------
@pytest.fixture(scope="module")
def small():
    return harness.make_problem(4, 6, 9, seed=11, blocks=True)


def test_p1_zero_amplitudes(small):
    import copy
    p = copy.copy(small)
    p.t1 = np.zeros_like(small.t1)
    p.t2 = np.zeros_like(small.t2)
    E, S = oracle.triples_energy(p)
    assert E == 0.0 and np.all(S == 0.0)


def test_p2_s2_scaling(small):
    import copy
    p = copy.copy(small)
    p.t1 = np.zeros_like(small.t1)
    E1, _ = oracle.triples_energy(p)
    p.t2 = 2.5 * small.t2
    E2, _ = oracle.triples_energy(p)
    assert E1 != 0.0
    assert E2 / E1 == pytest.approx(6.25, rel=1e-13)


def test_p3_W_simultaneous_permutation_symmetry(small):
    p = small
    o, v = p.o, p.v
    i, j, k = 3, 1, 2
    base = oracle.W_triplet(o, v, i, j, k, p.t2, p.vvvo[i], p.vvvo[j], p.vvvo[k], p.ovoo)
    occ = (i, j, k)
    for perm in itertools.permutations(range(3)):
        x, y, z = (occ[q] for q in perm)
        Wp = oracle.W_triplet(o, v, x, y, z, p.t2, p.vvvo[x], p.vvvo[y], p.vvvo[z], p.ovoo)
        # W_{perm(ijk)}^{perm(abc)} = W_ijk^abc: Wp[a_perm...] -> transpose back
        inv = np.argsort(perm)
        np.testing.assert_allclose(Wp.transpose(*inv), base, rtol=0, atol=1e-15)
    # the one north_star names explicitly: W_ijk^abc = W_jik^bac
    Wjik = oracle.W_triplet(o, v, j, i, k, p.t2, p.vvvo[j], p.vvvo[i], p.vvvo[k], p.ovoo)
    np.testing.assert_allclose(Wjik.transpose(1, 0, 2), base, rtol=0, atol=1e-15)


def _relabel(p, perm_o, perm_v):
    q = synth.Problem(p.o, p.v, p.naux,
                      p.eps_occ[perm_o].copy(), p.eps_vir[perm_v].copy(),
                      np.ascontiguousarray(p.t1[np.ix_(perm_o, perm_v)]),
                      np.ascontiguousarray(p.t2[np.ix_(perm_o, perm_o, perm_v, perm_v)]),
                      np.ascontiguousarray(p.Boo[:, perm_o][:, :, perm_o]),
                      np.ascontiguousarray(p.Bov[:, perm_o][:, :, perm_v]),
                      np.ascontiguousarray(p.Bvv[:, perm_v][:, :, perm_v]))
    return oracle.blocks.materialise_blocks(q)


def test_p4_relabelling_invariance(small):
    E0, _ = oracle.triples_energy(small)
    rng = np.random.default_rng(5)
    Eo, _ = oracle.triples_energy(_relabel(small, rng.permutation(small.o), np.arange(small.v)))
    Ev, _ = oracle.triples_energy(_relabel(small, np.arange(small.o), rng.permutation(small.v)))
    assert Eo == pytest.approx(E0, rel=1e-12)
    assert Ev == pytest.approx(E0, rel=1e-12)


def test_p5_restricted_equals_bruteforce(small):
    E, S = oracle.triples_energy(small)
    Eb = oracle.triples_energy_bruteforce(small)
    assert E == pytest.approx(Eb, rel=1e-12)
    # and the weights really are 2 - d_ij - d_jk on the colexicographic index
    acc = 0.0
    for idx in range(oracle.triplet_count(small.o)):
        i, j, k, w = oracle.triplet_decode(small.o, idx)
        assert i >= j >= k and idx == IDX(i, j, k)
        assert w == 2 - (i == j) - (j == k)
        acc += w * S[idx]
    assert acc == pytest.approx(E, rel=1e-14)


def test_p6_negative_semidefinite_when_t1_zero(small):
    import copy
    p = copy.copy(small)
    p.t1 = np.zeros_like(small.t1)
    E, S = oracle.triples_energy(p)
    assert E < 0.0
    assert np.all(S <= 1e-18)


def test_p7_degenerate_sizes():
    p = harness.make_problem(1, 5, 4, seed=3, blocks=True)
    E, S = oracle.triples_energy(p)
    assert abs(E) < 1e-18
    p = harness.make_problem(3, 1, 4, seed=3, blocks=True)
    E, S = oracle.triples_energy(p)
    assert abs(E) < 1e-18 and np.all(np.abs(S) < 1e-18)
    p = harness.make_problem(3, 4, 4, seed=3, blocks=True)
    _, S = oracle.triples_energy(p)
    for i in range(3):
        assert abs(S[IDX(i, i, i)]) < 1e-18 * max(1.0, np.abs(S).max()) + 1e-20


# ----------------------------------------------------------------------------
# P8, P9: independently written formulas
# ----------------------------------------------------------------------------
@pytest.mark.parametrize("dims", [(3, 4, 5), (2, 5, 3), (4, 3, 6)])
def test_p8_paper_printed_form(dims):
    p = harness.make_problem(*dims, seed=21, sigma_B=0.3, sigma_t1=0.05, blocks=True)
    E, _ = oracle.triples_energy(p)
    Ep, W6 = paper_form_energy(p)
    assert E == pytest.approx(Ep, rel=1e-12)
    # element-wise W (eq. (2) with the G reading) against the oracle's W
    o, v = p.o, p.v
    for (i, j, k) in [(0, 0, 0), (1, 0, 1), (o - 1, 0, 1), (o - 1, o - 1, 0)]:
        W = oracle.W_triplet(o, v, i, j, k, p.t2, p.vvvo[i], p.vvvo[j], p.vvvo[k], p.ovoo)
        np.testing.assert_allclose(W, W6[i, j, k], rtol=1e-12, atol=1e-15)


@pytest.mark.parametrize("dims", [(2, 3, 4), (3, 3, 5), (2, 4, 3)])
def test_p9_spin_orbital_textbook_formula(dims):
    p = harness.make_problem(*dims, seed=31, sigma_B=0.3, sigma_t1=0.05, blocks=True)
    E, _ = oracle.triples_energy(p)
    Es = spin_orbital_energy(p)
    assert E == pytest.approx(Es, rel=1e-11)


@pytest.mark.parametrize("o,v,naux", [(3, 4, 5), (4, 6, 7), (2, 5, 3), (5, 3, 4)])
def test_p9_closed_form_example(o, v, naux):
    """Every E in tests/golden/p10_worked_values.txt is re-derived here by two formulas that share nothing with the
    oracle (the spin-orbital textbook formula and the paper's own printed form), so the file stands on its own."""
    golden = {(r[1], r[2], r[3]): r[5] for r in _golden_rows() if r[0] == "E"}
    p = harness.closed_form_problem(o, v, naux)
    assert spin_orbital_energy(p) == pytest.approx(golden[(o, v, naux)], rel=1e-11)
    assert paper_form_energy(p)[0] == pytest.approx(golden[(o, v, naux)], rel=1e-11)


# ----------------------------------------------------------------------------
# DF builders against a library contraction, triplet index, slices entry
# ----------------------------------------------------------------------------
def test_df_builders_against_einsum():
    p = harness.make_problem(3, 5, 7, seed=2, blocks=True)
    o, v, naux = p.o, p.v, p.naux
    eri = full_eri(p)
    O, V = slice(0, o), slice(o, o + v)
    for x in range(o):
        I = oracle.build_vvvo_slice(o, v, naux, x, p.Bov, p.Bvv)
        ref = eri[V, V, V, x].transpose(1, 0, 2)     # (bd|cx) -> [d][b][c]
        np.testing.assert_allclose(I, ref, rtol=1e-13, atol=1e-15)
        np.testing.assert_allclose(p.vvvo[x], ref, rtol=1e-13, atol=1e-15)
    ovoo = oracle.build_ovoo(o, v, naux, p.Boo, p.Bov)
    np.testing.assert_allclose(ovoo, eri[O, O, O, V].transpose(1, 2, 0, 3), rtol=1e-13, atol=1e-15)  # (lj|kc)->[j][k][l][c]
    np.testing.assert_allclose(p.ovoo, ovoo, rtol=1e-13, atol=1e-15)
    ovov = oracle.build_ovov(o, v, naux, p.Bov)
    np.testing.assert_allclose(ovov, eri[O, V, O, V].transpose(0, 2, 1, 3), rtol=1e-13, atol=1e-15)  # (jb|kc)->[j][k][b][c]
    np.testing.assert_allclose(p.ovov, ovov, rtol=1e-13, atol=1e-15)


def test_pair_panels_and_amplitude_rows():
    """The restricted builders the large-size goldens use (only the panels / amplitude rows a few triplets touch)
    agree with the full ones."""
    p = harness.make_problem(5, 6, 7, seed=4, blocks=True)
    occ = [4, 1, 2]
    ovoo, ovov = oracle.blocks.ovoo_pairs(p, occ), oracle.blocks.ovov_pairs(p, occ)
    for x in occ:
        for y in occ:
            np.testing.assert_allclose(ovoo[x, y], p.ovoo[x, y], rtol=1e-13, atol=1e-16)
            np.testing.assert_allclose(ovov[x, y], p.ovov[x, y], rtol=1e-13, atol=1e-16)
    rows = synth.mp2_amplitude_rows(p.Bov, p.eps_occ, p.eps_vir, occ)
    for x in occ:
        np.testing.assert_allclose(rows[x], p.t2[x], rtol=1e-13, atol=1e-18)
    assert not rows[0].any() and not rows[3].any()
    # the oracle reads t2 only through rows whose first index is one of i, j, k
    idx = IDX(4, 2, 1)
    q = synth.Problem(p.o, p.v, p.naux, p.eps_occ, p.eps_vir, p.t1, rows, p.Boo, p.Bov, p.Bvv, None, ovoo, ovov)
    _, S_rows = oracle.triples_energy_slices(q, {x: p.vvvo[x] for x in occ}, idx, 1)
    _, S_full = oracle.triples_energy(p, idx, 1)
    assert S_rows[0] == pytest.approx(S_full[0], rel=1e-12)


def test_tile_orbit_sums_partition_S():
    """tco_S_from_W_tile_orbit (the per-tile sums of the abcijk scheme): the orbits partition the abc cube, so the restricted sums
    add up to tco_S_from_W; each one equals a numpy mask over Y R / D built from the oracle's own Y and W."""
    p = harness.make_problem(3, 7, 5, seed=8, sigma_B=0.3, sigma_t1=0.05, blocks=True)
    o, v, T = p.o, p.v, 3            # tiles of 3, 3, 1 virtual indices
    i, j, k = 2, 1, 0
    W = oracle.W_triplet(o, v, i, j, k, p.t2, p.vvvo[i], p.vvvo[j], p.vvvo[k], p.ovoo)
    S, Y = oracle.S_from_W(o, v, i, j, k, p.eps_occ, p.eps_vir, p.t1, p.ovov, W, want_Y=True)
    R = (4 * W + W.transpose(2, 0, 1) + W.transpose(1, 2, 0) - 2 * W.transpose(0, 2, 1) - 2 * W.transpose(2, 1, 0)
         - 2 * W.transpose(1, 0, 2))      # R[a,b,c] = 4W_abc + W_bca + W_cab - 2W_acb - 2W_cba - 2W_bac
    ev = p.eps_vir
    D = p.eps_occ[i] + p.eps_occ[j] + p.eps_occ[k] - ev[:, None, None] - ev[None, :, None] - ev[None, None, :]
    term = Y * R / D
    assert term.sum() == pytest.approx(S, rel=1e-13)
    tile = np.arange(v) // T
    total = 0.0
    orbs = oracle.tile_orbits(v, T)
    assert len(orbs) == 10 and orbs[0] == (0, 0, 0) and orbs[-1] == (2, 2, 2)
    for (A, B, C) in orbs:
        got = oracle.S_from_W_tile_orbit(o, v, i, j, k, p.eps_occ, p.eps_vir, p.t1, p.ovov, W, T, A, B, C)
        key = np.sort(np.stack(np.meshgrid(tile, tile, tile, indexing="ij"), -1), -1)[..., ::-1]
        mask = (key[..., 0] == A) & (key[..., 1] == B) & (key[..., 2] == C)
        assert got == pytest.approx(term[mask].sum(), rel=1e-12, abs=1e-18)
        total += got
    assert total == pytest.approx(S, rel=1e-13)
    E_orb = oracle.orbit_energies(p, T)
    E, _ = oracle.triples_energy(p)
    assert E_orb.sum() == pytest.approx(E, rel=1e-12)


def test_triplet_index_is_a_bijection():
    for o in (1, 2, 5, 9):
        seen = []
        for i in range(o):
            for j in range(i + 1):
                for k in range(j + 1):
                    seen.append((i, j, k))
        assert len(seen) == oracle.triplet_count(o)
        for idx, t in enumerate(seen):
            i, j, k, w = oracle.triplet_decode(o, idx)
            assert (i, j, k) == t
        with pytest.raises(ValueError):
            oracle.triplet_decode(o, len(seen))


def test_slices_entry_matches_blocks_entry(small):
    first, count = 7, 6
    E1, S1 = oracle.triples_energy(small, first, count)
    need = set()
    for idx in range(first, first + count):
        need.update(oracle.triplet_decode(small.o, idx)[:3])
    E2, S2 = oracle.triples_energy_slices(small, {x: small.vvvo[x] for x in need}, first, count)
    assert E1 == E2 and np.array_equal(S1, S2)


def test_t2_generator_symmetry():
    p = synth.make_problem(3, 4, 5, seed=9)
    assert np.array_equal(p.t2, p.t2.transpose(1, 0, 3, 2))
    assert np.array_equal(p.Bvv, p.Bvv.transpose(0, 2, 1))
    assert np.array_equal(p.Boo, p.Boo.transpose(0, 2, 1))
