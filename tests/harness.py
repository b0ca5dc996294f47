"""Test harness helpers shared by the CPU and GPU test modules: seeded problems (paper_2512_01055_b200.synth)
with the integral blocks of eq. (6) filled in on the oracle side (oracle.blocks, numpy), and the stored
large-size oracle values (tests/golden/S_*.txt, written by tests/golden/make_large_goldens.py from oracle/ only).
"""
import os

from oracle import blocks as oblocks
from paper_2512_01055_b200 import synth

GOLDEN_DIR = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden")


def make_problem(o, v, naux, seed, blocks=False, **kw):
    p = synth.make_problem(o, v, naux, seed, **kw)
    return oblocks.materialise_blocks(p) if blocks else p


def make_config(name, blocks=False, **kw):
    p = synth.make_config(name, **kw)
    return oblocks.materialise_blocks(p) if blocks else p


def closed_form_problem(o, v, naux, blocks=True, **kw):
    p = synth.closed_form_problem(o, v, naux, **kw)
    return oblocks.materialise_blocks(p) if blocks else p


def read_golden_S(name):
    """tests/golden/S_<name>.txt -> (dict idx -> (i, j, k, S), E or None).  Lines: `S idx i j k value`, `E value`."""
    path = os.path.join(GOLDEN_DIR, f"S_{name}.txt")
    rows, E = {}, None
    with open(path) as f:
        for line in f:
            t = line.split()
            if not t or t[0].startswith("#"):
                continue
            if t[0] == "S":
                rows[int(t[1])] = (int(t[2]), int(t[3]), int(t[4]), float(t[5]))
            elif t[0] == "E":
                E = float(t[1])
    return rows, E


def tiled_slice_bytes(v):
    """Bytes of one (vv|v.) slice slot in the library's workspace: the slice in the W-builder's tiled layout
    ([n1 tile][n2 tile][K chunk][2][16][4][8] doubles, zero padded, an even number of K chunks), rounded up to 256 (csrc/tc_energy.cu make_layout)."""
    nb, nkq = (v + 15) // 16, (v + 3) // 4
    nkq += nkq % 2          # K chunks per tile pair are rounded up to even
    return (nb * nb * nkq * 1024 * 8 + 255) // 256 * 256

