"""Thin ctypes binding of include/tc_triples.h -- argument marshalling only.

Every step of the (T) path runs in the CUDA library (``libtc_triples.so``, built in-tree by
``paper_2512_01055_b200.build``).  There is no Python or CPU fallback: if the library is missing
or no sm_100 device is present the calls raise.  Device arrays are passed as anything with a
``data_ptr()`` method (``torch.Tensor``) or as integer addresses; host arrays as C-contiguous
float64 numpy arrays.  Names follow the C header one to one.
"""
from __future__ import annotations

import ctypes
import os
from typing import Optional, Sequence

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.environ.get("TC_TRIPLES_LIB") or os.path.join(_HERE, "libtc_triples.so")   # override: a differently built copy

TC_OK = 0
TC_KERNEL_TMA = 1
_STATUS = {0: "TC_OK", 1: "TC_ERR_INVALID_ARG", 2: "TC_ERR_UNSUPPORTED_DEVICE", 3: "TC_ERR_WORKSPACE_TOO_SMALL",
           4: "TC_ERR_CUDA", 5: "TC_ERR_INTERNAL"}


class TcError(RuntimeError):
    def __init__(self, status: int, message: str):
        super().__init__(f"{_STATUS.get(status, status)}: {message}")
        self.status = status


class _IntBlocks(ctypes.Structure):
    _fields_ = [("vvvo", ctypes.c_void_p), ("ovoo", ctypes.c_void_p), ("ovov", ctypes.c_void_p)]


class _DfFactors(ctypes.Structure):
    _fields_ = [("naux", ctypes.c_int), ("Boo", ctypes.c_void_p), ("Bov", ctypes.c_void_p), ("Bvv", ctypes.c_void_p)]


class TcStats(ctypes.Structure):
    _fields_ = [("n_triplets", ctypes.c_longlong), ("n_work_units", ctypes.c_longlong),
                ("n_kernel_launches", ctypes.c_longlong), ("flop_contraction", ctypes.c_double),
                ("ms_total", ctypes.c_double), ("ms_contraction", ctypes.c_double), ("ms_staging", ctypes.c_double),
                ("slices_built", ctypes.c_longlong), ("kernel", ctypes.c_int), ("padded", ctypes.c_int),
                ("n_blocks", ctypes.c_longlong), ("t2_rows_copied", ctypes.c_longlong), ("bytes_h2d", ctypes.c_double),
                ("ms_kernels", ctypes.c_double), ("ms_staging_side", ctypes.c_double),
                ("staging_first_ms", ctypes.c_double), ("staging_last_ms", ctypes.c_double),
                ("contraction_first_ms", ctypes.c_double), ("contraction_last_ms", ctypes.c_double)]

    def as_dict(self):
        return {name: getattr(self, name) for name, _ in self._fields_}


STATIC_SCRATCH_BYTES = 64 << 20   # TC_STATIC_SCRATCH_BYTES of include/tc_triples.h

EXPORTS = [
    "tc_create", "tc_destroy", "tc_status_string", "tc_last_error",
    "tc_triplet_count", "tc_triplet_decode", "tc_triplet_index", "tc_triplet_partition",
    "tc_workspace_bytes", "tc_workspace_bytes_streamed", "tc_plan_summary", "tc_plan_dump", "tc_build_blocks",
    "tc_triples_energy", "tc_triples_energy_slice", "tc_triples_energy_static", "tc_triples_energy_streamed", "tc_triples_energy_host",
    "tc_tile_orbit_count", "tc_workspace_bytes_abcijk", "tc_triples_energy_abcijk",
    "tc_debug_W_triplet",
    "tc_get_stats", "tc_bench_dmma_peak", "tc_bench_dfma_peak", "tc_bench_copy_bw", "tc_bench_ring_peak",
]

_lib = None
_vp, _i, _ll, _d, _sz = ctypes.c_void_p, ctypes.c_int, ctypes.c_longlong, ctypes.c_double, ctypes.c_size_t
_P = ctypes.POINTER


def lib() -> ctypes.CDLL:
    """Load the CUDA library; raises if it has not been built (no fallback)."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise ImportError(f"{LIB_PATH} not found: build it with `python -m paper_2512_01055_b200.build` "
                          "(there is no CPU fallback)")
    L = ctypes.CDLL(LIB_PATH)
    L.tc_create.argtypes = [_P(_vp), _i]
    L.tc_destroy.argtypes = [_vp]
    L.tc_status_string.argtypes = [_i]
    L.tc_status_string.restype = ctypes.c_char_p
    L.tc_last_error.argtypes = [_vp]
    L.tc_last_error.restype = ctypes.c_char_p
    L.tc_triplet_count.argtypes = [_i]
    L.tc_triplet_count.restype = _ll
    L.tc_triplet_decode.argtypes = [_i, _ll, _P(_i), _P(_i), _P(_i), _P(_d)]
    L.tc_triplet_index.argtypes = [_i, _i, _i, _i]
    L.tc_triplet_index.restype = _ll
    L.tc_triplet_partition.argtypes = [_i, _i, _i, _P(_ll), _P(_ll)]
    L.tc_workspace_bytes.argtypes = [_vp, _i, _i, _i, _sz, _P(_sz)]
    L.tc_workspace_bytes_streamed.argtypes = [_vp, _i, _i, _i, _sz, _P(_sz)]
    L.tc_plan_summary.argtypes = [_i, _ll, _ll, _i, _P(_ll), _P(_ll), _P(_i), _P(_i), _P(_i)]
    L.tc_tile_orbit_count.argtypes = [_i]
    L.tc_tile_orbit_count.restype = _ll
    L.tc_workspace_bytes_abcijk.argtypes = [_vp, _i, _i, _i, _P(_sz)]
    L.tc_triples_energy_abcijk.argtypes = [_vp, _i, _i, _vp, _vp, _vp, _vp, _P(_DfFactors), _vp, _sz, _vp, _ll, _ll, _vp, _P(_d)]
    L.tc_plan_dump.argtypes = [_i, _ll, _ll, _i, _vp, _vp, _ll]
    L.tc_triples_energy_streamed.argtypes = [_vp, _i, _i, _vp, _vp, _vp, _vp, _P(_DfFactors), _vp, _sz, _vp, _ll, _ll, _vp, _P(_d)]
    L.tc_bench_ring_peak.argtypes = [_vp, _i, _d, _vp, _sz, _P(_d)]
    L.tc_build_blocks.argtypes = [_vp, _i, _i, _P(_DfFactors), _i, _i, _vp, _vp, _vp, _vp]
    L.tc_triples_energy.argtypes = [_vp, _i, _i, _vp, _vp, _vp, _vp, _P(_IntBlocks), _P(_DfFactors), _vp, _sz, _vp, _P(_d)]
    L.tc_triples_energy_slice.argtypes = [_vp, _i, _i, _vp, _vp, _vp, _vp, _P(_IntBlocks), _P(_DfFactors), _vp, _sz, _vp,
                                          _ll, _ll, _vp, _P(_d)]
    L.tc_triples_energy_static.argtypes = [_vp, _i, _i, _vp, _vp, _vp, _vp, _P(_IntBlocks), _P(_DfFactors), _vp, _ll, _ll, _vp, _P(_d)]
    L.tc_triples_energy_host.argtypes = [_vp, _i, _i, _i] + [_vp] * 7 + [_ll, _ll, _P(_d), _P(_sz)]
    L.tc_debug_W_triplet.argtypes = [_vp, _i, _i, _i, _i, _i, _vp, _P(_IntBlocks), _vp, _vp]
    L.tc_get_stats.argtypes = [_vp, _P(TcStats)]
    L.tc_bench_dmma_peak.argtypes = [_vp, _d, _P(_d), _P(_d)]
    L.tc_bench_dfma_peak.argtypes = [_vp, _d, _P(_d), _P(_d)]
    L.tc_bench_copy_bw.argtypes = [_vp, _vp, _vp, _sz, _i, _P(_d)]
    _lib = L
    return L


def _ptr(x) -> Optional[int]:
    if x is None:
        return None
    if hasattr(x, "data_ptr"):
        return int(x.data_ptr())
    return int(x)


def _host(a) -> np.ndarray:
    return np.ascontiguousarray(a, dtype=np.float64)


def _stream(stream) -> Optional[int]:
    if stream is None:
        return None
    return int(getattr(stream, "cuda_stream", stream))


class Context:
    """tc_ctx wrapper (tc_create / tc_destroy)."""

    def __init__(self, device: int = 0):
        self._h = _vp()
        rc = lib().tc_create(ctypes.byref(self._h), device)
        if rc != TC_OK:
            self._h = None
            raise TcError(rc, "tc_create failed (needs an sm_100 CUDA device; there is no fallback path)")

    def close(self):
        if getattr(self, "_h", None):
            lib().tc_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def _check(self, rc: int):
        if rc != TC_OK:
            raise TcError(rc, lib().tc_last_error(self._h).decode())

    # -- scheduler ---------------------------------------------------------------------------
    # (host-only helpers are module functions below)

    # -- workspace ---------------------------------------------------------------------------
    def workspace_bytes(self, o: int, v: int, naux_or_0: int = 0, hbm_budget: int = 0) -> int:
        out = _sz()
        self._check(lib().tc_workspace_bytes(self._h, o, v, naux_or_0, hbm_budget, ctypes.byref(out)))
        return int(out.value)

    def workspace_bytes_streamed(self, o: int, v: int, naux: int, hbm_budget: int = 0) -> int:
        out = _sz()
        self._check(lib().tc_workspace_bytes_streamed(self._h, o, v, naux, hbm_budget, ctypes.byref(out)))
        return int(out.value)

    # -- a2 ----------------------------------------------------------------------------------
    def build_blocks(self, o, v, naux, Boo, Bov, Bvv, x0=0, nx=None, vvvo_out=None, ovoo_out=None, ovov_out=None,
                     stream=None):
        df = _DfFactors(naux, _ptr(Boo), _ptr(Bov), _ptr(Bvv))
        nx = o - x0 if nx is None else nx
        self._check(lib().tc_build_blocks(self._h, o, v, ctypes.byref(df), x0, nx, _ptr(vvvo_out), _ptr(ovoo_out),
                                          _ptr(ovov_out), _stream(stream)))

    # -- a3..a7 ------------------------------------------------------------------------------
    @staticmethod
    def _ints(blocks, df):
        b = d = None
        if blocks is not None:
            b = _IntBlocks(*[_ptr(x) for x in blocks])
        if df is not None:
            d = _DfFactors(int(df[0]), _ptr(df[1]), _ptr(df[2]), _ptr(df[3]))
        return b, d, (ctypes.byref(b) if b is not None else None), (ctypes.byref(d) if d is not None else None)

    def triples_energy(self, o, v, eps_occ, eps_vir, t1, t2, *, workspace, workspace_bytes, blocks=None, df=None,
                       stream=None) -> float:
        """blocks = (vvvo, ovoo, ovov) or df = (naux, Boo, Bov, Bvv); all device arrays."""
        b, d, pb, pd = self._ints(blocks, df)
        E = _d()
        self._check(lib().tc_triples_energy(self._h, o, v, _ptr(eps_occ), _ptr(eps_vir), _ptr(t1), _ptr(t2), pb, pd,
                                            _ptr(workspace), workspace_bytes, _stream(stream), ctypes.byref(E)))
        return E.value

    def triples_energy_slice(self, o, v, eps_occ, eps_vir, t1, t2, *, workspace, workspace_bytes, blocks=None, df=None,
                             stream=None, first=0, count=0, S_dev=None) -> float:
        b, d, pb, pd = self._ints(blocks, df)
        E = _d()
        self._check(lib().tc_triples_energy_slice(self._h, o, v, _ptr(eps_occ), _ptr(eps_vir), _ptr(t1), _ptr(t2), pb, pd,
                                                  _ptr(workspace), workspace_bytes, _stream(stream), first, count,
                                                  _ptr(S_dev), ctypes.byref(E)))
        return E.value

    def triples_energy_static(self, o, v, eps_occ, eps_vir, t1, t2, *, blocks=None, df=None, stream=None, first=0, count=0,
                              S_dev=None) -> float:
        """As triples_energy_slice, with the scratch in the library's static device array (STATIC_SCRATCH_BYTES): no allocation."""
        b, d, pb, pd = self._ints(blocks, df)
        E = _d()
        self._check(lib().tc_triples_energy_static(self._h, o, v, _ptr(eps_occ), _ptr(eps_vir), _ptr(t1), _ptr(t2), pb, pd,
                                                   _stream(stream), first, count, _ptr(S_dev), ctypes.byref(E)))
        return E.value

    def triples_energy_streamed(self, o, v, eps_occ, eps_vir, t1, t2_host, *, df, workspace, workspace_bytes, stream=None,
                                first=0, count=0, S_dev=None) -> float:
        """t2_host: C-contiguous float64 HOST array (numpy, or a pinned torch CPU tensor); everything else on the device."""
        d = _DfFactors(int(df[0]), _ptr(df[1]), _ptr(df[2]), _ptr(df[3]))
        t2p = t2_host.ctypes.data if isinstance(t2_host, np.ndarray) else _ptr(t2_host)
        E = _d()
        self._check(lib().tc_triples_energy_streamed(self._h, o, v, _ptr(eps_occ), _ptr(eps_vir), _ptr(t1), t2p, ctypes.byref(d),
                                                     _ptr(workspace), workspace_bytes, _stream(stream), first, count,
                                                     _ptr(S_dev), ctypes.byref(E)))
        return E.value

    def workspace_bytes_abcijk(self, o: int, v: int, naux: int) -> int:
        out = _sz()
        self._check(lib().tc_workspace_bytes_abcijk(self._h, o, v, naux, ctypes.byref(out)))
        return int(out.value)

    def triples_energy_abcijk(self, o, v, eps_occ, eps_vir, t1, t2, *, df, workspace, workspace_bytes, stream=None,
                              orbit_first=0, orbit_count=None, E_orbit_dev=None) -> float:
        """The paper's abcijk schedule: tile orbits outer, all triplets inner (see the header)."""
        d = _DfFactors(int(df[0]), _ptr(df[1]), _ptr(df[2]), _ptr(df[3]))
        if orbit_count is None:
            orbit_count = tile_orbit_count(v) - orbit_first
        E = _d()
        self._check(lib().tc_triples_energy_abcijk(self._h, o, v, _ptr(eps_occ), _ptr(eps_vir), _ptr(t1), _ptr(t2), ctypes.byref(d),
                                                   _ptr(workspace), workspace_bytes, _stream(stream), orbit_first, orbit_count,
                                                   _ptr(E_orbit_dev), ctypes.byref(E)))
        return E.value

    def triples_energy_host(self, o, v, naux, eps_occ, eps_vir, t1, t2, Boo, Bov, Bvv, first=0, count=None):
        """HOST (numpy) inputs; returns (E, bytes copied host->device)."""
        arrs = [_host(x) for x in (eps_occ, eps_vir, t1, t2, Boo, Bov, Bvv)]
        if count is None:
            count = triplet_count(o) - first
        E, nb = _d(), _sz()
        self._check(lib().tc_triples_energy_host(self._h, o, v, naux, *[x.ctypes.data for x in arrs], first, count,
                                                 ctypes.byref(E), ctypes.byref(nb)))
        return E.value, int(nb.value)

    def debug_W_triplet(self, o, v, i, j, k, t2, blocks: Sequence, W_dev, stream=None):
        b = _IntBlocks(*[_ptr(x) for x in blocks])
        self._check(lib().tc_debug_W_triplet(self._h, o, v, i, j, k, _ptr(t2), ctypes.byref(b), _ptr(W_dev), _stream(stream)))

    def get_stats(self) -> dict:
        s = TcStats()
        self._check(lib().tc_get_stats(self._h, ctypes.byref(s)))
        return s.as_dict()

    # -- microbenchmarks ---------------------------------------------------------------------
    def bench_dmma_peak(self, seconds: float = 1.0):
        a, b = _d(), _d()
        self._check(lib().tc_bench_dmma_peak(self._h, seconds, ctypes.byref(a), ctypes.byref(b)))
        return a.value, b.value

    def bench_dfma_peak(self, seconds: float = 1.0):
        a, b = _d(), _d()
        self._check(lib().tc_bench_dfma_peak(self._h, seconds, ctypes.byref(a), ctypes.byref(b)))
        return a.value, b.value

    def bench_copy_bw(self, dst, src, nbytes: int, reps: int = 10) -> float:
        g = _d()
        self._check(lib().tc_bench_copy_bw(self._h, _ptr(dst), _ptr(src), nbytes, reps, ctypes.byref(g)))
        return g.value


    def bench_ring_peak(self, variant: int, seconds: float = 1.0, scratch=None, scratch_bytes: int = 0) -> float:
        g = _d()
        self._check(lib().tc_bench_ring_peak(self._h, variant, seconds, _ptr(scratch), scratch_bytes, ctypes.byref(g)))
        return g.value


def triplet_partition(o: int, world: int, rank: int):
    """(first, count) of the linear triplet index owned by `rank` of `world` (host only)."""
    f, c = _ll(), _ll()
    rc = lib().tc_triplet_partition(o, world, rank, ctypes.byref(f), ctypes.byref(c))
    if rc != TC_OK:
        raise TcError(rc, "bad partition arguments")
    return int(f.value), int(c.value)


def plan_summary(o: int, first: int, count: int, nslots: int) -> dict:
    """The blocked schedule for a triplet range with `nslots` operand slots (host only)."""
    nb, nl, bi, bj, bk = _ll(), _ll(), _i(), _i(), _i()
    rc = lib().tc_plan_summary(o, first, count, nslots, ctypes.byref(nb), ctypes.byref(nl), ctypes.byref(bi), ctypes.byref(bj),
                               ctypes.byref(bk))
    if rc != TC_OK:
        raise TcError(rc, "no plan (bad range, or fewer than three slots)")
    return {"n_blocks": int(nb.value), "n_loads": int(nl.value), "bi": bi.value, "bj": bj.value, "bk": bk.value}


def plan_dump(o: int, first: int, count: int, nslots: int):
    """(recs[count][8], loads[n_loads][4]) of the blocked schedule; see tc_plan_dump in the header."""
    n_loads = plan_summary(o, first, count, nslots)["n_loads"]
    recs = np.zeros((max(count, 1), 8), dtype=np.int32)
    loads = np.zeros((max(n_loads, 1), 4), dtype=np.int32)
    rc = lib().tc_plan_dump(o, first, count, nslots, recs.ctypes.data, loads.ctypes.data, n_loads)
    if rc != TC_OK:
        raise TcError(rc, "tc_plan_dump failed")
    return recs[:count], loads[:n_loads]


def tile_orbit_count(v: int) -> int:
    return int(lib().tc_tile_orbit_count(v))


def triplet_count(o: int) -> int:
    return int(lib().tc_triplet_count(o))


def triplet_index(o: int, i: int, j: int, k: int) -> int:
    return int(lib().tc_triplet_index(o, i, j, k))


def triplet_decode(o: int, idx: int):
    i, j, k, w = _i(), _i(), _i(), _d()
    rc = lib().tc_triplet_decode(o, idx, ctypes.byref(i), ctypes.byref(j), ctypes.byref(k), ctypes.byref(w))
    if rc != TC_OK:
        raise TcError(rc, "triplet index out of range")
    return i.value, j.value, k.value, w.value
