"""Integral blocks from DF factors for the ORACLE side -- TEST INFRASTRUCTURE ONLY.

Eq. (6) of arxiv 2512.01055, ``(pq|rs) = sum_Q B^Q_pq B^Q_rs``, written with one numpy
contraction per block (a library matmul serving as the step "sum over Q"; no blocking or reordering beyond
it).  The plain-loop statement of the same equation is ``tco_build_*`` in tc_oracle.c; the two are pinned
against each other and against a full-ERI einsum in tests/test_oracle_pins.py
(``test_df_builders_against_einsum``), so these functions are not "parity unpinned".  They exist because the
plain loops need minutes per (vv|v.) slice at BASELINE.json's sizes.

Layouts (include/tc_triples.h): vvvo[x][d][b][c] = (bd|cx); ovoo[j][k][l][c] = (lj|kc); ovov[j][k][b][c] = (jb|kc).
The product path (paper_2512_01055_b200) never imports this module: on the CUDA side the same step is
``k_df_gemm`` (csrc/tc_stager.cu).
"""
from __future__ import annotations

import numpy as np


def vvvo_slice(prob, x: int) -> np.ndarray:
    """I_x[d][b][c] = (bd|cx) = sum_Q Bvv[Q][d][b] Bov[Q][x][c] for one occupied index x (v^3 doubles)."""
    naux, v = prob.naux, prob.v
    A = prob.Bvv.reshape(naux, v * v)                 # [Q][(d,b)]
    return (A.T @ prob.Bov[:, x, :]).reshape(v, v, v)


def ovoo_block(prob) -> np.ndarray:
    """ovoo[j][k][l][c] = (lj|kc) = sum_Q Boo[Q][l][j] Bov[Q][k][c]."""
    return np.ascontiguousarray(np.einsum("qlj,qkc->jklc", prob.Boo, prob.Bov, optimize=True))


def ovov_block(prob) -> np.ndarray:
    """ovov[j][k][b][c] = (jb|kc) = sum_Q Bov[Q][j][b] Bov[Q][k][c]."""
    return np.ascontiguousarray(np.einsum("qjb,qkc->jkbc", prob.Bov, prob.Bov, optimize=True))


def ovoo_pairs(prob, occ) -> np.ndarray:
    """The (ov|oo) panels ovoo[x][y][:][:] for x, y in ``occ`` only (everything else zero): what the oracle's
    loops touch for triplets drawn from ``occ`` (used where the full o^3 v block is too large to be worth building)."""
    o, v = prob.o, prob.v
    out = np.zeros((o, o, o, v))
    for x in occ:
        for y in occ:
            out[x, y] = np.einsum("ql,qc->lc", prob.Boo[:, :, x], prob.Bov[:, y, :])     # (lx|yc)
    return out


def ovov_pairs(prob, occ) -> np.ndarray:
    """The (ov|ov) panels ovov[x][y][:][:] for x, y in ``occ`` only (everything else zero)."""
    o, v = prob.o, prob.v
    out = np.zeros((o, o, v, v))
    for x in occ:
        for y in occ:
            out[x, y] = np.einsum("qb,qc->bc", prob.Bov[:, x, :], prob.Bov[:, y, :])     # (xb|yc)
    return out


def materialise_blocks(prob):
    """Fill prob.vvvo / ovoo / ovov from the DF factors; returns prob."""
    o, v = prob.o, prob.v
    vvvo = np.empty((o, v, v, v), dtype=np.float64)
    for x in range(o):
        vvvo[x] = vvvo_slice(prob, x)
    prob.vvvo = vvvo
    prob.ovoo = ovoo_block(prob)
    prob.ovov = ovov_block(prob)
    return prob
