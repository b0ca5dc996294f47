"""Host logic of the blocked schedule (csrc/tc_plan.cu) and of the multi-GPU partition, without a GPU: every
triplet of the range is executed exactly once, the operands it reads are resident in the slots its record names,
no slot is overwritten while a block that still needs it may be running, and more slots never cost more loads."""
import numpy as np
import pytest

import oracle
from paper_2512_01055_b200 import binding


def _check_plan(o, first, count, nslots):
    summ = binding.plan_summary(o, first, count, nslots)
    recs, loads = binding.plan_dump(o, first, count, nslots)
    assert sorted(recs[:, 3].tolist()) == list(range(count))                  # each triplet once
    for r in recs:
        i, j, k, _ = oracle.triplet_decode(o, first + int(r[3]))
        assert (i, j, k) == tuple(int(x) for x in r[:3])
    assert np.all(np.diff(recs[:, 4]) >= 0)                                   # blocks in execution order
    owner = [-1] * min(nslots, o)
    last_use = [-1] * len(owner)
    by_block = {}
    for b, x, slot, wait in loads.tolist():
        by_block.setdefault(b, []).append((x, slot, wait))
    for b in range(summ["n_blocks"]):
        mine = recs[recs[:, 4] == b]
        assert len(mine) > 0
        need = set(mine[:, :3].ravel().tolist())
        assert len(need) <= len(owner)
        for x, slot, wait in by_block.get(b, []):
            assert owner[slot] not in need                                     # never evicts what the block needs
            assert last_use[slot] <= wait < b                                  # the side stream waits long enough
            owner[slot] = x
        for r in mine:
            for p in range(3):
                assert owner[int(r[5 + p])] == int(r[p])                       # operands resident where the record says
        for x in need:
            last_use[owner.index(x)] = b
    return summ


@pytest.mark.parametrize("o,first,count,nslots", [(9, 0, 165, 3), (9, 0, 165, 4), (9, 37, 61, 7), (9, 0, 165, 9), (9, 0, 165, 20),
                                                   (12, 100, 200, 5), (20, 0, 1540, 6), (20, 713, 400, 11), (5, 3, 0, 3)])
def test_plan_is_consistent(o, first, count, nslots):
    summ = _check_plan(o, first, count, nslots)
    distinct = set()
    for n in range(first, first + count):
        distinct.update(oracle.triplet_decode(o, n)[:3])
    assert summ["n_loads"] >= len(distinct)
    if nslots >= o:
        assert summ["n_loads"] == len(distinct)                                # everything fits: each operand once


def test_more_slots_never_cost_more_loads():
    o, n = 30, binding.triplet_count(30)
    loads = [binding.plan_summary(o, 0, n, s)["n_loads"] for s in (3, 4, 6, 9, 13, 20, 30)]
    assert all(a >= b for a, b in zip(loads, loads[1:])), loads
    assert loads[-1] == o
    # the i x j footprint of a streamed k operand: cfg4 with 13 slots needs < 0.05 loads per triplet
    s = binding.plan_summary(100, 0, binding.triplet_count(100), 13)
    assert s["n_loads"] < 0.05 * binding.triplet_count(100) and s["bi"] > 1


def test_plan_argument_errors():
    with pytest.raises(binding.TcError):
        binding.plan_summary(9, 0, 165, 2)          # a triplet needs three operands
    with pytest.raises(binding.TcError):
        binding.plan_summary(9, 100, 100, 5)        # range outside
    assert binding.plan_summary(2, 0, 4, 2)["n_loads"] == 2   # o = 2: two slots hold everything


def test_partition_tiles_the_index_range():
    for o in (1, 3, 8, 20):
        n = binding.triplet_count(o)
        for world in (1, 2, 3, 4, 8):
            at, sizes = 0, []
            for r in range(world):
                first, count = binding.triplet_partition(o, world, r)
                assert first == at and count >= 0
                at += count
                sizes.append(count)
            assert at == n and max(sizes) - min(sizes) <= 1
    with pytest.raises(binding.TcError):
        binding.triplet_partition(8, 2, 2)
