"""The C-ABI library loads on a machine without a GPU and exports every symbol include/tc_triples.h declares
(no compute calls here).  Host-only entry points (the triplet scheduler, a1) are exercised against the oracle's
independent implementation of the same index map; compute calls must fail loudly without an sm_100 device."""
import ctypes
import os
import re

import pytest

import oracle
from paper_2512_01055_b200 import binding

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _declared_symbols():
    text = open(os.path.join(ROOT, "include", "tc_triples.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(tc_[a-z_A-Z0-9]+)\s*\(", text)))


def test_every_declared_symbol_is_exported():
    lib = binding.lib()
    names = _declared_symbols()
    assert len(names) >= 16
    missing = [n for n in names if not hasattr(lib, n)]
    assert not missing, missing
    assert sorted(binding.EXPORTS) == names          # the binding covers exactly the header


def test_triplet_scheduler_matches_oracle():
    for o in (1, 2, 5, 20, 100):
        n = binding.triplet_count(o)
        assert n == oracle.triplet_count(o) == o * (o + 1) * (o + 2) // 6
        for idx in sorted({0, 1, n // 3, n // 2, n - 2, n - 1} & set(range(n))):
            got = binding.triplet_decode(o, idx)
            assert got == oracle.triplet_decode(o, idx)
            i, j, k, w = got
            assert i >= j >= k >= 0 and binding.triplet_index(o, i, j, k) == idx
            assert w == 2.0 - (i == j) - (j == k)
    assert binding.triplet_count(0) == -1
    assert binding.triplet_index(5, 2, 3, 1) == -1
    with pytest.raises(binding.TcError):
        binding.triplet_decode(4, 20)


def test_no_cpu_fallback():
    """Without an sm_100 device the context cannot be created: there is no CPU path behind the boundary."""
    try:
        import torch
        if torch.cuda.is_available():
            pytest.skip("a CUDA device is present")
    except ImportError:
        pass
    with pytest.raises(binding.TcError) as e:
        binding.Context(0)
    assert e.value.status == 2   # TC_ERR_UNSUPPORTED_DEVICE
    assert binding.lib().tc_status_string(2) == b"TC_ERR_UNSUPPORTED_DEVICE"
