#!/usr/bin/env python
"""Write the stored oracle values for BASELINE.json's full-size configs: tests/golden/S_<name>.txt.

Imports ONLY ``oracle`` (the CPU oracle, plain C loops, and its numpy statement of eq. (6)) and
``paper_2512_01055_b200.synth`` (seeded input generators, no method arithmetic).  Nothing here touches the CUDA
path; the GPU parity tests (tests/test_gpu_large.py) and bench.py compare the CUDA results with these files.
SURVEY.md 8(d): "cache one long full-oracle run ... as a golden value".

  python tests/golden/make_large_goldens.py cfg1            # all 1540 S_ijk and E(T) of cfg1 (~25 min on 8 cores)
  python tests/golden/make_large_goldens.py cfg2 cfg3 h2o14 # sampled S_ijk (i>j>k, i=j>k, i>j=k, first, last)
  python tests/golden/make_large_goldens.py cfg4            # three triplets of the benchmark slice (i = 70), ~5 min each

File format: `# comment`, `S idx i j k value`, `E value`; values are Python reprs of the FP64 numbers
(they round-trip exactly).  Each file states its command line.
"""
import os
import sys
import time

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
sys.path.insert(0, ROOT)

import oracle                                   # noqa: E402
from oracle import blocks as oblocks            # noqa: E402
from paper_2512_01055_b200 import synth         # noqa: E402

HERE = os.path.dirname(os.path.abspath(__file__))
IDX = lambda i, j, k: i * (i + 1) * (i + 2) // 6 + j * (j + 1) // 2 + k


def sample_triplets(name, o):
    """The sampled triplets of a config: the first two indices, the last ones, i>j>k in the middle, i=j>k, i>j=k."""
    if name == "cfg4":      # inside the benchmark slice idx in [59640, 61640) (reading 14): i = 70, j <= 62
        return [(70, 31, 7), (70, 31, 31), (70, 62, 61)]
    trips = [(0, 0, 0), (1, 0, 0), (o - 1, o - 1, o - 2), (o - 1, o - 3, o - 3), (o - 1, o // 2, 1), (o // 2, o // 3, 2)]
    return sorted(set(trips), key=lambda t: IDX(*t))


def write(name, kind, rows, E, seconds, sizes):
    o, v, naux, seed = sizes
    path = os.path.join(HERE, f"S_{name}.txt")
    with open(path, "w") as f:
        f.write(f"# CPU-oracle values of the closed-shell (T) energy, config {name}: o={o} v={v} naux={naux} seed={seed}\n")
        f.write("# (BASELINE.json configs / DESIGN.md section 4; generators: paper_2512_01055_b200/synth.py).\n")
        f.write("# S_ijk = sum_abc (W+Vd) R / D for one triplet (eqs. (1)-(5), PAPER.md:33-53); E = sum_{i>=j>=k} (2-d_ij-d_jk) S_ijk.\n")
        f.write(f"# Written by: python tests/golden/make_large_goldens.py {name}   ({kind}; {seconds:.0f} s of oracle/ on "
                f"{oracle.num_threads()} threads; oracle/ and synth only)\n")
        f.write("# kind idx i j k value\n")
        for idx, (i, j, k, S) in sorted(rows.items()):
            f.write(f"S {idx} {i} {j} {k} {S!r}\n")
        if E is not None:
            f.write(f"E {E!r}\n")
    print(f"wrote {path}: {len(rows)} S values" + (f", E = {E!r}" if E is not None else ""), flush=True)


def run_full(name):
    sizes = synth.config_sizes(name)
    p = oblocks.materialise_blocks(synth.make_config(name))
    t0 = time.time()
    E, S = oracle.triples_energy(p)
    rows = {}
    for idx in range(oracle.triplet_count(p.o)):
        i, j, k, _ = oracle.triplet_decode(p.o, idx)
        rows[idx] = (i, j, k, float(S[idx]))
    write(name, "full range", rows, float(E), time.time() - t0, sizes)


def run_sampled(name):
    sizes = synth.config_sizes(name)
    o, v, naux, seed = sizes
    big = 8.0 * o * o * v * v > 8e9          # cfg4: t2 is 51 GB -- only the rows the sampled triplets touch
    p = synth.make_config(name, with_t2=not big)
    trips = sample_triplets(name, o)
    occ = sorted({x for t in trips for x in t})
    if big:
        p.t2 = synth.mp2_amplitude_rows(p.Bov, p.eps_occ, p.eps_vir, occ)
    p.ovoo = oblocks.ovoo_pairs(p, occ)
    p.ovov = oblocks.ovov_pairs(p, occ)
    rows = {}
    slices = {}
    t0 = time.time()
    for (i, j, k) in trips:
        for x in list(slices):
            if x not in (i, j, k):
                del slices[x]                # at most three slices live (4.1 GB each at cfg4)
        for x in (i, j, k):
            if x not in slices:
                slices[x] = oblocks.vvvo_slice(p, x)
        idx = IDX(i, j, k)
        _, S = oracle.triples_energy_slices(p, slices, idx, 1)
        rows[idx] = (i, j, k, float(S[0]))
        print(f"  {name} ({i},{j},{k}) idx {idx}: S = {float(S[0])!r}   [{time.time() - t0:.0f} s]", flush=True)
    write(name, "sampled triplets", rows, None, time.time() - t0, sizes)


def main():
    names = sys.argv[1:] or ["cfg1", "cfg2", "cfg3", "h2o14", "cfg4"]
    for name in names:
        if name in ("cfg0", "cfg1"):
            run_full(name)
        else:
            run_sampled(name)


if __name__ == "__main__":
    main()
