"""Pins T7, T8: binning (O3-O6) against the paper's Table 1 and against what a stable sort fixes."""
import os

import numpy as np

from oracle import axo
from paper_1405_3331_b200 import workloads as W


def test_T7_paper_table_1(golden_dir):
    cells, pairs, ranges = None, None, {}
    for ln in open(os.path.join(golden_dir, "table1.txt")):
        p = ln.split()
        if not p or p[0].startswith("#"):
            continue
        if p[0] == "cells":
            cells = [int(v) for v in p[1:]]
        elif p[0] == "sorted":
            pairs = [tuple(int(v) for v in q.split(",")) for q in p[1:]]
        elif p[0] == "range":
            ranges[int(p[1])] = (int(p[2]), int(p[3]))
    perm, ks, cs, ce = axo.bin_keys(cells, 16)
    assert list(zip((int(v) for v in ks), (int(v) for v in perm))) == pairs
    for c in range(16):
        assert (int(cs[c]), int(ce[c])) == ranges.get(c, (0, 0))


def _check_invariants(keys, perm, ks, cs, ce, cells):
    n = len(keys)
    assert np.array_equal(np.sort(perm), np.arange(n, dtype=np.uint32))          # a permutation
    assert np.array_equal(ks, keys[perm])
    assert np.all(ks[1:] >= ks[:-1])                                              # non-decreasing
    same = ks[1:] == ks[:-1]
    assert np.all(perm[1:][same] > perm[:-1][same])                               # ties keep pre-sort order
    assert np.array_equal(perm, np.argsort(keys, kind="stable").astype(np.uint32))  # library special case
    cnt = np.bincount(keys, minlength=cells)
    assert np.array_equal((ce.astype(np.int64) - cs.astype(np.int64)), cnt)       # per-cell counts; sum = n
    ne = np.nonzero(cnt)[0]
    assert np.all(ks[cs[ne]] == ne) and np.all(ks[ce[ne] - 1] == ne)
    assert np.all(cs[cnt == 0] == 0) and np.all(ce[cnt == 0] == 0)                # A-10
    first = cs[ne]
    assert np.all((first == 0) | (ks[np.maximum(first, 1) - 1] < ne))


def test_T8_invariants_random_keys():
    rng = np.random.default_rng(3)
    for n, cells in ((0, 8), (1, 8), (1000, 7), (5000, 4096), (20000, 100000), (4096, 1)):
        keys = rng.integers(0, cells, n).astype(np.uint32)
        if n > 100:
            keys[: n // 4] = keys[0]  # one very full cell
        perm, ks, cs, ce = axo.bin_keys(keys, cells)
        _check_invariants(keys, perm, ks, cs, ce, cells)


def test_T8_key_formula_and_reorder():
    grid = (7, 5, 3)
    x, y, z, sp, ids = W.random_particles(17, 3000, grid)
    o = axo.Oracle(grid, 0.5, 0, 2.0, 0.25, 0.1, 1)
    o.load_particles(x, y, z, sp, ids, next_id=3000, step=0)
    o.step_phase(axo.PHASE_BIN)
    key = o.read_state("PRE_KEY")
    # x fastest, then y, then z (A-8); floor of the coordinates
    expect = (np.floor(z).astype(np.int64) * 5 + np.floor(y).astype(np.int64)) * 7 + np.floor(x).astype(np.int64)
    assert np.array_equal(key.astype(np.int64), expect)
    assert key.max() < 7 * 5 * 3
    # a particle exactly on an upper face of a cell belongs to the next cell; the last representable coordinate below
    # the wall belongs to the last cell
    assert int(expect[np.argmax(x)]) % 7 == 6
    perm = o.read_state("PERM")
    _check_invariants(key, perm, o.read_state("KEYS_SORTED"), o.read_state("CELL_START"), o.read_state("CELL_END"), 105)
    for f, src in (("PART_X", x), ("PART_Y", y), ("PART_Z", z), ("PART_SPECIES", sp), ("PART_ID", ids)):
        assert np.array_equal(o.read_state(f), src[perm])
    # pre-sort arrays recoverable from the sorted ones: pre[perm[j]] = sorted[j]
    back = np.empty_like(x)
    back[perm] = o.read_state("PART_X")
    assert np.array_equal(back, x)
