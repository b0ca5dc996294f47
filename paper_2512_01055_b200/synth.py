"""Seeded synthetic inputs for the closed-shell (T) energy.

This module is shared by the oracle's tests and by the CUDA path's tests and
bench.  It holds NO arithmetic of the (T) method itself: it only draws the
problem inputs (DF factors, orbital energies, MP2 amplitudes).  The integral
blocks of eq. (6) -- step a2 of the method -- are NOT derived here: the oracle
side builds them in ``oracle/blocks.py``, the CUDA side in ``csrc/tc_stager.cu``.
It imports neither ``oracle`` nor the CUDA binding.

Recipe (BASELINE.json ``configs``):

* ``B^Q_pq ~ N(0, sigma_B^2)`` (sigma_B = 0.05), drawn for ``p <= q`` and
  mirrored, ``p, q`` over ``o+v`` orbitals with the occupied ones first, so
  that ``(pq|rs) = sum_Q B^Q_pq B^Q_rs`` exactly (eq. (6)).
* ``eps_occ ~ U[-2.0, -0.3]``, ``eps_vir ~ U[0.1, 5.0]``.
* ``t2`` = MP2 amplitudes ``(ia|jb) / (e_i + e_j - e_a - e_b)``, symmetrised
  bit-exactly so that ``t_ij^ab == t_ji^ba``.
* ``t1 ~ N(0, 0.01^2)``.

Random numbers come from a counter-based generator (splitmix64 of
``(seed, tensor id, flat index)`` then Box-Muller), so every element of every
tensor is a pure function of its index.

A second, closed-form input family (``closed_form_problem``) reproduces the
worked examples of SURVEY.md section 8(c) P10.
"""
from __future__ import annotations

import dataclasses
from typing import Optional

import numpy as np

_M64 = np.uint64(0xFFFFFFFFFFFFFFFF)
_GOLD = 0x9E3779B97F4A7C15
_MIX1 = 0xBF58476D1CE4E5B9
_MIX2 = 0x94D049BB133111EB

TENSOR_B = 1
TENSOR_EPS_OCC = 2
TENSOR_EPS_VIR = 3
TENSOR_T1 = 4

# BASELINE.json configs[0..4]: (o, v, naux, seed)
CONFIGS = {
    "cfg0": (8, 40, 120, 0),
    "cfg1": (20, 200, 600, 1),
    "cfg2": (40, 400, 1200, 2),
    "cfg3": (60, 500, 1500, 3),
    "cfg4": (100, 800, 2400, 4),
    # the paper's own shape, v/o ~ 4 -- sized like (H2O)14 / cc-pVDZ (336 AOs, PAPER.md:77-83,
    # Table 1; o and v are inferred, the paper does not print them); v = 266 = 16*16 + 10 is ragged
    "h2o14": (70, 266, 800, 5),
}


def _splitmix64(x: np.ndarray) -> np.ndarray:
    """One splitmix64 output for each 64-bit state in ``x`` (uint64 array)."""
    with np.errstate(over="ignore"):
        z = x + np.uint64(_GOLD)
        z = (z ^ (z >> np.uint64(30))) * np.uint64(_MIX1)
        z = (z ^ (z >> np.uint64(27))) * np.uint64(_MIX2)
        z = z ^ (z >> np.uint64(31))
    return z


def _uniform_pair(seed: int, tensor_id: int, idx: np.ndarray):
    """Two uniforms per counter: u1 in (0, 1], u2 in [0, 1)."""
    idx = np.asarray(idx, dtype=np.uint64)
    with np.errstate(over="ignore"):
        base = (np.uint64((seed * _GOLD) & 0xFFFFFFFFFFFFFFFF)
                ^ np.uint64((tensor_id * _MIX1) & 0xFFFFFFFFFFFFFFFF))
        ctr = base + np.uint64(2) * idx
        r1 = _splitmix64(ctr)
        r2 = _splitmix64(ctr + np.uint64(1))
    scale = 1.0 / 9007199254740992.0  # 2^-53
    u1 = ((r1 >> np.uint64(11)).astype(np.float64) + 1.0) * scale
    u2 = (r2 >> np.uint64(11)).astype(np.float64) * scale
    return u1, u2


def counter_normal(seed: int, tensor_id: int, idx, sigma: float) -> np.ndarray:
    u1, u2 = _uniform_pair(seed, tensor_id, idx)
    return sigma * np.sqrt(-2.0 * np.log(u1)) * np.cos(2.0 * np.pi * u2)


def counter_uniform(seed: int, tensor_id: int, idx, lo: float, hi: float) -> np.ndarray:
    _, u2 = _uniform_pair(seed, tensor_id, idx)
    return lo + (hi - lo) * u2


@dataclasses.dataclass
class Problem:
    """Inputs of one (T) calculation, all float64, C order (host numpy arrays).

    Layouts are those of include/tc_triples.h:
      Boo[Q][i][j], Bov[Q][i][a], Bvv[Q][a][b];
      t1[i][a]; t2[i][j][a][b] = t_ij^ab;
      vvvo[x][d][b][c] = (bd|cx); ovoo[j][k][l][c] = (lj|kc); ovov[j][k][b][c] = (jb|kc).
    The integral blocks are optional: None here; the tests fill them on the oracle side
    (``oracle.blocks.materialise_blocks``) or on the device (``tc_build_blocks``).
    """
    o: int
    v: int
    naux: int
    eps_occ: np.ndarray
    eps_vir: np.ndarray
    t1: np.ndarray
    t2: np.ndarray
    Boo: np.ndarray
    Bov: np.ndarray
    Bvv: np.ndarray
    vvvo: Optional[np.ndarray] = None
    ovoo: Optional[np.ndarray] = None
    ovov: Optional[np.ndarray] = None


def _split_B(B: np.ndarray, o: int):
    Boo = np.ascontiguousarray(B[:, :o, :o])
    Bov = np.ascontiguousarray(B[:, :o, o:])
    Bvv = np.ascontiguousarray(B[:, o:, o:])
    return Boo, Bov, Bvv


def mp2_amplitudes(Bov: np.ndarray, eps_occ: np.ndarray, eps_vir: np.ndarray) -> np.ndarray:
    """t2[i][j][a][b] = (ia|jb) / (e_i + e_j - e_a - e_b), made exactly symmetric
    under (i,a) <-> (j,b) by averaging with its own transpose."""
    naux, o, v = Bov.shape
    M = Bov.reshape(naux, o * v)
    iajb = (M.T @ M).reshape(o, v, o, v)              # (ia|jb)
    den = (eps_occ[:, None, None, None] - eps_vir[None, :, None, None]
           + eps_occ[None, None, :, None] - eps_vir[None, None, None, :])
    t = iajb / den                                    # [i][a][j][b]
    t = 0.5 * (t + t.transpose(2, 3, 0, 1))           # bit-exact t_ij^ab = t_ji^ba
    return np.ascontiguousarray(t.transpose(0, 2, 1, 3))   # [i][j][a][b]


def make_problem(o: int, v: int, naux: int, seed: int, sigma_B: float = 0.05,
                 sigma_t1: float = 0.01, with_t2: bool = True) -> Problem:
    """Draw one synthetic problem with the BASELINE.json recipe.  with_t2=False leaves ``t2`` None (the
    caller derives the MP2 amplitudes on the device with ``mp2_amplitudes_device``: at cfg4 size ``t2`` is 51 GB)."""
    N = o + v
    p = np.arange(N, dtype=np.uint64)
    lo = np.minimum(p[:, None], p[None, :])
    hi = np.maximum(p[:, None], p[None, :])
    pair = lo * np.uint64(N) + hi                    # (min, max) -> mirrored draw
    B = np.empty((naux, N, N), dtype=np.float64)
    for Q in range(naux):
        idx = np.uint64(Q) * np.uint64(N * N) + pair
        B[Q] = counter_normal(seed, TENSOR_B, idx, sigma_B)
    eps_occ = counter_uniform(seed, TENSOR_EPS_OCC, np.arange(o), -2.0, -0.3)
    eps_vir = counter_uniform(seed, TENSOR_EPS_VIR, np.arange(v), 0.1, 5.0)
    t1 = counter_normal(seed, TENSOR_T1, np.arange(o * v), sigma_t1).reshape(o, v)
    Boo, Bov, Bvv = _split_B(B, o)
    t2 = mp2_amplitudes(Bov, eps_occ, eps_vir) if with_t2 else None
    return Problem(o, v, naux, eps_occ, eps_vir, np.ascontiguousarray(t1), t2, Boo, Bov, Bvv)


def mp2_amplitudes_device(Bov, eps_occ, eps_vir):
    """``mp2_amplitudes`` with torch tensors on the device (input preparation for problems whose ``t2`` does not
    fit comfortably on the host): t2[i][j][a][b] = (ia|jb) / (e_i + e_j - e_a - e_b), then made bit-exactly
    symmetric under (i,a) <-> (j,b).  Works one occupied index at a time (temporaries of o*v*v doubles)."""
    import torch
    naux, o, v = Bov.shape
    t2 = torch.empty((o, o, v, v), dtype=torch.float64, device=Bov.device)
    Bflat = Bov.reshape(naux, o * v)
    ea = eps_vir.reshape(v, 1, 1)
    eb = eps_vir.reshape(1, 1, v)
    ej = eps_occ.reshape(1, o, 1)
    for i in range(o):
        iajb = (Bov[:, i, :].t().contiguous() @ Bflat).reshape(v, o, v)      # [a][j][b] = (ia|jb)
        iajb /= (eps_occ[i] + ej - ea - eb)
        t2[i] = iajb.permute(1, 0, 2)
        del iajb
    for i in range(o):                                                      # t_ij^ab <- (t_ij^ab + t_ji^ba) / 2
        avg = 0.5 * (t2[i] + t2[:, i].transpose(1, 2))
        t2[i] = avg
        t2[:, i] = avg.transpose(1, 2)
        del avg
    return t2


def mp2_amplitude_rows(Bov: np.ndarray, eps_occ: np.ndarray, eps_vir: np.ndarray, rows) -> np.ndarray:
    """``mp2_amplitudes`` restricted to the first occupied index in ``rows``: returns an (o, o, v, v) array whose rows
    t2[x] (x in rows) hold t_xl^ab for all l and whose other rows are untouched zeros (the array is calloc-backed, so
    at cfg4 size -- 51 GB in full -- only the requested rows cost memory)."""
    naux, o, v = Bov.shape
    Bflat = Bov.reshape(naux, o * v)
    t2 = np.zeros((o, o, v, v))
    ea = eps_vir.reshape(v, 1, 1)
    eb = eps_vir.reshape(1, 1, v)
    el = eps_occ.reshape(1, o, 1)
    for x in rows:
        Bx = np.ascontiguousarray(Bov[:, x, :])
        g1 = (Bx.T @ Bflat).reshape(v, o, v)                       # (xa|lb)  [a][l][b]
        g2 = (Bflat.T @ Bx).reshape(o, v, v).transpose(2, 0, 1)    # (lb|xa)  [a][l][b]
        d1 = eps_occ[x] - ea + el - eb                             # e_x - e_a + e_l - e_b
        d2 = el - eb + eps_occ[x] - ea                             # e_l - e_b + e_x - e_a
        t2[x] = (0.5 * (g1 / d1 + g2 / d2)).transpose(1, 0, 2)     # [l][a][b]
    return t2


def _splitmix64_torch(x):
    """``_splitmix64`` on int64 tensors (two's-complement wrap-around = uint64 arithmetic; logical shifts by masking)."""
    import torch

    def lsr(z, n):
        return (z >> n) & ((1 << (64 - n)) - 1)

    def c(u):   # uint64 constant as the int64 with the same bits
        return u - (1 << 64) if u >= (1 << 63) else u

    z = x + c(_GOLD)
    z = (z ^ lsr(z, 30)) * c(_MIX1)
    z = (z ^ lsr(z, 27)) * c(_MIX2)
    return z ^ lsr(z, 31)


def counter_normal_torch(seed: int, tensor_id: int, idx, sigma: float):
    """``counter_normal`` with torch tensors (idx: int64 tensor on any device): the same counters and the same
    Box-Muller formula, so every element agrees with the numpy generator up to the last bits of log/cos."""
    import torch
    base = ((seed * _GOLD) & 0xFFFFFFFFFFFFFFFF) ^ ((tensor_id * _MIX1) & 0xFFFFFFFFFFFFFFFF)
    base = base - (1 << 64) if base >= (1 << 63) else base
    ctr = 2 * idx + base
    r1 = _splitmix64_torch(ctr)
    r2 = _splitmix64_torch(ctr + 1)
    scale = 1.0 / 9007199254740992.0
    u1 = (((r1 >> 11) & ((1 << 53) - 1)).double() + 1.0) * scale
    u2 = ((r2 >> 11) & ((1 << 53) - 1)).double() * scale
    return sigma * torch.sqrt(-2.0 * torch.log(u1)) * torch.cos(2.0 * np.pi * u2)


def make_problem_device(o: int, v: int, naux: int, seed: int, device="cuda", sigma_B: float = 0.05, sigma_t1: float = 0.01):
    """``make_problem`` with the DF factors drawn on the device (bench.py's throughput legs at sizes where the host draw
    of B -- 15 GB at cfg4 -- would take minutes): dict of device tensors eps_occ, eps_vir, t1, t2, Boo, Bov, Bvv.
    Same counter-based recipe; values agree with ``make_problem`` up to the last bits of log/cos."""
    import torch
    N = o + v
    p = torch.arange(N, dtype=torch.int64, device=device)
    lo = torch.minimum(p[:, None], p[None, :])
    hi = torch.maximum(p[:, None], p[None, :])
    pair = lo * N + hi
    Boo = torch.empty((naux, o, o), dtype=torch.float64, device=device)
    Bov = torch.empty((naux, o, v), dtype=torch.float64, device=device)
    Bvv = torch.empty((naux, v, v), dtype=torch.float64, device=device)
    step = max(1, min(naux, (1 << 25) // (N * N)))
    for q0 in range(0, naux, step):
        q1 = min(naux, q0 + step)
        Q = torch.arange(q0, q1, dtype=torch.int64, device=device)[:, None, None]
        B = counter_normal_torch(seed, TENSOR_B, Q * (N * N) + pair[None], sigma_B)
        Boo[q0:q1] = B[:, :o, :o]
        Bov[q0:q1] = B[:, :o, o:]
        Bvv[q0:q1] = B[:, o:, o:]
        del B
    ho = make_small_host(o, v, seed, sigma_t1)
    d = {k: torch.from_numpy(x).to(device) for k, x in ho.items()}
    d.update(Boo=Boo, Bov=Bov, Bvv=Bvv)
    d["t2"] = mp2_amplitudes_device(Bov, d["eps_occ"], d["eps_vir"])
    return d


def make_small_host(o: int, v: int, seed: int, sigma_t1: float = 0.01):
    """eps_occ, eps_vir, t1 of the recipe (host numpy)."""
    return {"eps_occ": counter_uniform(seed, TENSOR_EPS_OCC, np.arange(o), -2.0, -0.3),
            "eps_vir": counter_uniform(seed, TENSOR_EPS_VIR, np.arange(v), 0.1, 5.0),
            "t1": np.ascontiguousarray(counter_normal(seed, TENSOR_T1, np.arange(o * v), sigma_t1).reshape(o, v))}


def config_sizes(name: str):
    """(o, v, naux, seed) of a named BASELINE.json config, or of an ad-hoc "o,v,naux,seed" string."""
    if name in CONFIGS:
        return CONFIGS[name]
    o, v, naux, seed = (int(x) for x in name.split(","))
    return o, v, naux, seed


def make_config(name: str, sigma_B: float = 0.05, with_t2: bool = True) -> Problem:
    o, v, naux, seed = config_sizes(name)
    return make_problem(o, v, naux, seed, sigma_B=sigma_B, with_t2=with_t2)


def closed_form_problem(o: int, v: int, naux: int, t1_zero: bool = False) -> Problem:
    """Closed-form inputs of the worked examples:
    B^Q_pq = 0.3 cos(0.7(Q+1) + 1.3(p+q) + 0.11 p q) / (1 + 0.1|p-q|),
    eps_occ[i] = -1.5 + 0.35 i, eps_vir[a] = 0.4 + 0.45 a,
    t1[i][a] = 0.02 sin(1 + 2i + 3a), t2 = MP2 from B."""
    N = o + v
    Q = np.arange(naux, dtype=np.float64)[:, None, None]
    p = np.arange(N, dtype=np.float64)[None, :, None]
    q = np.arange(N, dtype=np.float64)[None, None, :]
    B = 0.3 * np.cos(0.7 * (Q + 1.0) + 1.3 * (p + q) + 0.11 * p * q) / (1.0 + 0.1 * np.abs(p - q))
    eps_occ = -1.5 + 0.35 * np.arange(o, dtype=np.float64)
    eps_vir = 0.4 + 0.45 * np.arange(v, dtype=np.float64)
    ii = np.arange(o, dtype=np.float64)[:, None]
    aa = np.arange(v, dtype=np.float64)[None, :]
    t1 = 0.02 * np.sin(1.0 + 2.0 * ii + 3.0 * aa)
    if t1_zero:
        t1 = np.zeros_like(t1)
    Boo, Bov, Bvv = _split_B(B, o)
    t2 = mp2_amplitudes(Bov, eps_occ, eps_vir)
    return Problem(o, v, naux, eps_occ, eps_vir, np.ascontiguousarray(t1), t2, Boo, Bov, Bvv)
