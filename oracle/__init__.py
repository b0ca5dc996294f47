"""CPU ORACLE for the closed-shell (T) energy -- TEST INFRASTRUCTURE ONLY.

ctypes front end of oracle/tc_oracle.c (plain C loops, FP64; see tc_oracle.h for
the equations and PAPER.md citations).  Only tests/, ``__graft_entry__.smoke()``
and bench.py's ``cpu_baseline`` / ``--impl reference`` legs may import this
package; the product path (paper_2512_01055_b200) never does.
"""
from __future__ import annotations

import ctypes

import numpy as np

from . import build as _build

_lib = None
_dp = ctypes.POINTER(ctypes.c_double)


def _f64(a):
    a = np.ascontiguousarray(a, dtype=np.float64)
    return a, a.ctypes.data_as(_dp)


def lib():
    global _lib
    if _lib is None:
        L = ctypes.CDLL(_build.build())
        L.tco_triplet_count.restype = ctypes.c_longlong
        L.tco_triplet_count.argtypes = [ctypes.c_int]
        L.tco_triplet_decode.restype = ctypes.c_int
        L.tco_triplet_decode.argtypes = [ctypes.c_int, ctypes.c_longlong] + [ctypes.POINTER(ctypes.c_int)] * 3 + [_dp]
        L.tco_W_triplet.restype = None
        L.tco_W_triplet.argtypes = [ctypes.c_int] * 5 + [_dp] * 6
        L.tco_S_from_W.restype = ctypes.c_double
        L.tco_S_from_W.argtypes = [ctypes.c_int] * 5 + [_dp] * 6
        L.tco_S_from_W_tile_orbit.restype = ctypes.c_double
        L.tco_S_from_W_tile_orbit.argtypes = [ctypes.c_int] * 5 + [_dp] * 5 + [ctypes.c_int] * 4
        L.tco_triples_energy_blocks.restype = ctypes.c_int
        L.tco_triples_energy_blocks.argtypes = [ctypes.c_int] * 2 + [_dp] * 7 + [ctypes.c_longlong] * 2 + [_dp] * 2
        L.tco_triples_energy_slices.restype = ctypes.c_int
        L.tco_triples_energy_slices.argtypes = ([ctypes.c_int] * 2 + [_dp] * 4 + [ctypes.POINTER(_dp)]
                                                + [_dp] * 2 + [ctypes.c_longlong] * 2 + [_dp] * 2)
        L.tco_triples_energy_bruteforce.restype = ctypes.c_int
        L.tco_triples_energy_bruteforce.argtypes = [ctypes.c_int] * 2 + [_dp] * 7 + [_dp]
        L.tco_build_vvvo_slice.restype = None
        L.tco_build_vvvo_slice.argtypes = [ctypes.c_int] * 4 + [_dp] * 3
        L.tco_build_ovoo.restype = None
        L.tco_build_ovoo.argtypes = [ctypes.c_int] * 3 + [_dp] * 3
        L.tco_build_ovov.restype = None
        L.tco_build_ovov.argtypes = [ctypes.c_int] * 3 + [_dp] * 2
        L.tco_num_threads.restype = ctypes.c_int
        _lib = L
    return _lib


def num_threads() -> int:
    return int(lib().tco_num_threads())


def triplet_count(o: int) -> int:
    return int(lib().tco_triplet_count(o))


def triplet_decode(o: int, idx: int):
    i, j, k = ctypes.c_int(), ctypes.c_int(), ctypes.c_int()
    w = ctypes.c_double()
    rc = lib().tco_triplet_decode(o, idx, ctypes.byref(i), ctypes.byref(j), ctypes.byref(k), ctypes.byref(w))
    if rc:
        raise ValueError("triplet index out of range")
    return i.value, j.value, k.value, w.value


def W_triplet(o, v, i, j, k, t2, I_i, I_j, I_k, ovoo):
    """W[a][b][c] for one (i,j,k) (any order)."""
    t2, pt2 = _f64(t2)
    I_i, pi = _f64(I_i)
    I_j, pj = _f64(I_j)
    I_k, pk = _f64(I_k)
    ovoo, po = _f64(ovoo)
    W = np.empty((v, v, v), dtype=np.float64)
    lib().tco_W_triplet(o, v, i, j, k, pt2, pi, pj, pk, po, W.ctypes.data_as(_dp))
    return W


def S_from_W(o, v, i, j, k, eps_occ, eps_vir, t1, ovov, W, want_Y=False):
    eps_occ, pe = _f64(eps_occ)
    eps_vir, pv = _f64(eps_vir)
    t1, pt1 = _f64(t1)
    ovov, po = _f64(ovov)
    W, pW = _f64(W)
    Y = np.empty((v, v, v), dtype=np.float64) if want_Y else None
    pY = Y.ctypes.data_as(_dp) if want_Y else None
    S = lib().tco_S_from_W(o, v, i, j, k, pe, pv, pt1, po, pW, pY)
    return (S, Y) if want_Y else S


def S_from_W_tile_orbit(o, v, i, j, k, eps_occ, eps_vir, t1, ovov, W, T, A, B, C):
    """S_ijk restricted to the points (a,b,c) of the tile orbit A >= B >= C (tile edge T)."""
    eps_occ, pe = _f64(eps_occ)
    eps_vir, pv = _f64(eps_vir)
    t1, pt1 = _f64(t1)
    ovov, po = _f64(ovov)
    W, pW = _f64(W)
    return lib().tco_S_from_W_tile_orbit(o, v, i, j, k, pe, pv, pt1, po, pW, T, A, B, C)


def tile_orbits(v, T=16):
    """The orbits of virtual tiles in the order A >= B >= C, A slowest (the order of tc_triples_energy_abcijk)."""
    nb = (v + T - 1) // T
    return [(A, B, C) for A in range(nb) for B in range(A + 1) for C in range(B + 1)]


def orbit_energies(prob, T=16):
    """E_orbit = sum_{i>=j>=k} (2 - d_ij - d_jk) sum_{(a,b,c) in orbit} Y R / D for every tile orbit (numpy array, the
    order of tile_orbits): what the abcijk schedule produces per virtual tile, from the plain loops."""
    o, v = prob.o, prob.v
    orbs = tile_orbits(v, T)
    E = np.zeros(len(orbs))
    for idx in range(triplet_count(o)):
        i, j, k, w = triplet_decode(o, idx)
        if w == 0.0:
            continue
        W = W_triplet(o, v, i, j, k, prob.t2, prob.vvvo[i], prob.vvvo[j], prob.vvvo[k], prob.ovoo)
        for n, (A, B, C) in enumerate(orbs):
            E[n] += w * S_from_W_tile_orbit(o, v, i, j, k, prob.eps_occ, prob.eps_vir, prob.t1, prob.ovov, W, T, A, B, C)
    return E


def triples_energy(prob, first=0, count=None):
    """(E_partial, S[count]) over a range of the linear triplet index, from integral blocks."""
    o, v = prob.o, prob.v
    if count is None:
        count = triplet_count(o) - first
    arrs = [_f64(x) for x in (prob.eps_occ, prob.eps_vir, prob.t1, prob.t2, prob.vvvo, prob.ovoo, prob.ovov)]
    S = np.empty(max(count, 1), dtype=np.float64)
    E = ctypes.c_double()
    rc = lib().tco_triples_energy_blocks(o, v, *[p for _, p in arrs], first, count,
                                         S.ctypes.data_as(_dp), ctypes.cast(ctypes.byref(E), _dp))
    if rc:
        raise RuntimeError(f"oracle error {rc}")
    return E.value, S[:count]


def triples_energy_slices(prob, slices, first, count):
    """Same as triples_energy but with a dict {x: I_x (v^3 array)} of only the needed slices."""
    o, v = prob.o, prob.v
    keep = {x: _f64(s) for x, s in slices.items()}
    ptrs = (_dp * o)()
    for x in range(o):
        ptrs[x] = keep[x][1] if x in keep else None
    arrs = [_f64(x) for x in (prob.eps_occ, prob.eps_vir, prob.t1, prob.t2)]
    ovoo, povoo = _f64(prob.ovoo)
    ovov, povov = _f64(prob.ovov)
    S = np.empty(max(count, 1), dtype=np.float64)
    E = ctypes.c_double()
    rc = lib().tco_triples_energy_slices(o, v, *[p for _, p in arrs], ptrs, povoo, povov, first, count,
                                         S.ctypes.data_as(_dp), ctypes.cast(ctypes.byref(E), _dp))
    if rc:
        raise RuntimeError(f"oracle error {rc}")
    return E.value, S[:count]


def triples_energy_bruteforce(prob):
    o, v = prob.o, prob.v
    arrs = [_f64(x) for x in (prob.eps_occ, prob.eps_vir, prob.t1, prob.t2, prob.vvvo, prob.ovoo, prob.ovov)]
    E = ctypes.c_double()
    rc = lib().tco_triples_energy_bruteforce(o, v, *[p for _, p in arrs], ctypes.cast(ctypes.byref(E), _dp))
    if rc:
        raise RuntimeError(f"oracle error {rc}")
    return E.value


def build_vvvo_slice(o, v, naux, x, Bov, Bvv):
    Bov, pb = _f64(Bov)
    Bvv, pv = _f64(Bvv)
    I = np.empty((v, v, v), dtype=np.float64)
    lib().tco_build_vvvo_slice(o, v, naux, x, pb, pv, I.ctypes.data_as(_dp))
    return I


def build_ovoo(o, v, naux, Boo, Bov):
    Boo, p1 = _f64(Boo)
    Bov, p2 = _f64(Bov)
    out = np.empty((o, o, o, v), dtype=np.float64)
    lib().tco_build_ovoo(o, v, naux, p1, p2, out.ctypes.data_as(_dp))
    return out


def build_ovov(o, v, naux, Bov):
    Bov, p = _f64(Bov)
    out = np.empty((o, o, v, v), dtype=np.float64)
    lib().tco_build_ovov(o, v, naux, p, out.ctypes.data_as(_dp))
    return out
from . import blocks  # noqa: E402,F401  (numpy statement of eq. (6), pinned against the C loops)
