"""Pins T16 of the oracle's connection formation, adjacency list and BFS (DESIGN.md readings
A-28..A-30; PAPER.md:223-233 §3.3 sphere-sphere test on squared distances, :239 growth stops at another neuron,
:241-247 compact adjacency list Va / Ea, :249-255 Fig. 5 level-synchronous BFS).

What they are pinned to (nothing here re-calls the oracle to check the oracle):
  T16a  the collision rule: hand-built cases with exactly representable distances (strict '<' at the threshold, the
        nearest soma wins, equal distances go to the lowest index, a cone never connects to its own neuron, frozen cones
        are not tested), the step at which a straight-growing axon must connect (closed form), and scipy's cKDTree
        ball query in float64 (a library routine) on 2 000 random neurons.
  T16b  the adjacency list: scipy.sparse's CSR of the same 0/1 matrix (indptr = Va, indices = Ea), directed and
        symmetric; mutual connections collapse to one entry.
  T16c  the BFS levels: scipy.sparse.csgraph.shortest_path (unweighted) on random graphs; closed forms on a path, a ring
        and a star; -1 for unreachable vertices.
"""
import numpy as np
import pytest
import scipy.sparse as sp
from scipy.sparse.csgraph import shortest_path
from scipy.spatial import cKDTree

from oracle import axo

NONE = axo.NO_TARGET


def _oracle(somata, heading=None, grid=(32, 32, 32), speed=0.25, noise=0.0, segs=64):
    o = axo.Oracle(grid, 0.5, 1, 2.0, speed, noise, 3)
    o.set_capacity(1 << 12, segs)
    o.place_neurons(np.asarray(somata, np.float32), heading)
    return o


def test_collision_rule_on_exact_distances():
    # somata 0..4; the cone tips are loaded separately (a cone's soma stays where the neuron was placed)
    somata = [[4, 4, 4], [10, 4, 4], [4, 10, 4], [20, 20, 20], [4, 4, 5.5]]
    o = _oracle(somata)
    o.set_connect(0.25, 0.5)                     # reach 0.75, threshold d^2 < 0.5625
    tips = np.array([
        [10, 4, 4.75],     # cone 0: soma 1 at d^2 = 0.5625 exactly -> NOT a collision (strict <)
        [4, 4, 4.5],       # cone 1: soma 0 at d^2 = 0.25 -> connects to 0
        [4, 4, 4.75],      # cone 2: somata 0 and 4 both at d^2 = 0.5625 -> none; see the next call for the tie
        [20, 20, 20.25],   # cone 3: only its OWN soma is in reach -> none
        [4, 10, 4.25],     # cone 4: soma 2 at 0.0625 -> connects to 2, but the cone is loaded as EXITED -> not tested
    ], np.float32)
    state = np.array([0, 0, 0, 0, 2], np.uint8)
    o.load_cones(tips, np.tile([0, 0, 1], (5, 1)).astype(np.float32), state, np.full(5, 2, np.uint32))   # tip = second polyline point: the soma (first point) stays
    o.step_phase(axo.PHASE_CONNECT)
    assert o.read_state("CONE_TARGET").tolist() == [NONE, 0, NONE, NONE, NONE]
    assert o.read_state("CONE_STATE").tolist() == [0, 3, 0, 0, 2]
    # ties and "nearest wins": cone 2 half-way between somata 0 and 4 (d^2 = 0.5625 each) with a larger reach
    o.set_connect(0.5, 0.5)                      # threshold 1.0
    tips2 = tips.copy()
    tips2[0] = [4, 4, 4.875]                     # soma 0 at 0.765625, soma 4 at 0.390625 -> the nearer one, 4
    state2 = np.array([0, 3, 0, 0, 2], np.uint8)
    o.load_cones(tips2, np.tile([0, 0, 1], (5, 1)).astype(np.float32), state2, np.full(5, 2, np.uint32))   # tip = second polyline point: the soma (first point) stays
    o.step_phase(axo.PHASE_CONNECT)
    t = o.read_state("CONE_TARGET").tolist()
    assert t[0] == 4 and t[2] == 0               # equal distances: the lowest index
    assert t[1] == 0 and t[3] == NONE            # an earlier connection is kept; own soma never counts
    assert o.counters()["connected"] == 3
    o.close()


def test_straight_axon_connects_at_the_step_the_geometry_fixes():
    """noise = 0 and no cue particles: the heading is kept, the tip is at z0 + k speed after k steps; it must
    connect at the first k with (L - k speed)^2 < reach^2 and not before, and then stop growing."""
    L, speed, reach = 6.0, 0.25, 1.0
    o = _oracle([[16, 16, 2], [16, 16, 2 + L], [3, 3, 3]], speed=speed)
    o.set_connect(0.5, 0.5)
    k_expect = int(np.floor((L - reach) / speed)) + 1      # (L - k s) < reach  <=>  k > (L - reach) / s
    for k in range(1, k_expect + 4):
        o.step(1)
        t, st, ln = o.read_state("CONE_TARGET"), o.read_state("CONE_STATE"), o.read_state("POLY_LEN")
        if k < k_expect:
            assert t[0] == NONE and st[0] == 0 and ln[0] == 1 + k
        else:
            assert t[0] == 1 and st[0] == 3 and ln[0] == 1 + k_expect      # frozen: no further segments
    assert o.read_state("CONE_TARGET")[2] == NONE
    o.close()


def test_all_pairs_rule_against_a_kd_tree_ball_query():
    rng = np.random.default_rng(160)
    n = 2000
    somata = rng.uniform(1, 31, (n, 3)).astype(np.float32)
    tips = (somata[rng.permutation(n)] + rng.normal(0, 0.8, (n, 3))).astype(np.float32)
    tips = np.clip(tips, 0.01, 31.99).astype(np.float32)
    state = (rng.uniform(size=n) < 0.1).astype(np.uint8) * 2            # a tenth of the cones frozen (EXITED)
    o = _oracle(somata, segs=4)
    r_c, r_s = np.float32(0.4), np.float32(0.6)
    o.set_connect(float(r_c), float(r_s))
    o.load_cones(tips, np.tile([0, 0, 1], (n, 1)).astype(np.float32), state, np.full(n, 2, np.uint32))
    o.step_phase(axo.PHASE_CONNECT)
    got = o.read_state("CONE_TARGET")
    reach = float(np.float32(r_c + r_s))
    tree = cKDTree(somata.astype(np.float64))
    n_conn = 0
    for c in range(n):
        if state[c]:
            assert got[c] == NONE
            continue
        near = [j for j in tree.query_ball_point(tips[c].astype(np.float64), reach + 1e-4) if j != c]
        d = np.array([np.sum((tips[c].astype(np.float64) - somata[j]) ** 2) for j in near])
        sure = [j for j, dj in zip(near, d) if dj < reach * reach - 1e-5]    # clear of fp32 rounding at the threshold
        maybe = [j for j, dj in zip(near, d) if dj < reach * reach + 1e-5]
        if not maybe:
            assert got[c] == NONE
        elif sure:
            assert got[c] != NONE
            dmin = d.min()
            # the winner is a nearest soma (within rounding); among exact ties the oracle takes the lowest index
            assert abs(np.sum((tips[c].astype(np.float64) - somata[got[c]]) ** 2) - dmin) < 1e-5
            n_conn += 1
    assert n_conn > 50
    assert (o.read_state("CONE_STATE") == 3).sum() == (got != NONE).sum()
    o.close()


def _random_targets(rng, n, p_connect=0.7, mutual=40):
    t = np.full(n, NONE, np.uint32)
    for i in np.flatnonzero(rng.uniform(size=n) < p_connect):
        j = int(rng.integers(0, n - 1))
        t[i] = j if j < i else j + 1
    for _ in range(mutual):                     # i -> j and j -> i: one entry each way, not two
        i, j = rng.choice(n, 2, replace=False)
        t[i], t[j] = j, i
    return t


@pytest.mark.parametrize("directed", [False, True])
def test_adjacency_list_is_the_csr_of_the_connection_matrix(directed):
    rng = np.random.default_rng(161)
    n = 5000
    t = _random_targets(rng, n)
    o = _oracle(rng.uniform(1, 31, (n, 3)), segs=2)
    o.load_targets(t)
    o.build_graph(directed)
    va, ea = o.read_state("GRAPH_VA"), o.read_state("GRAPH_EA")
    src = np.flatnonzero(t != NONE)
    m = sp.coo_matrix((np.ones(len(src)), (src, t[src].astype(np.int64))), shape=(n, n)).tocsr()
    if not directed:
        m = m + m.T
    m.data[:] = 1.0
    m.sum_duplicates()
    m.sort_indices()
    assert np.array_equal(va, m.indptr.astype(np.uint32))
    assert np.array_equal(ea, m.indices.astype(np.uint32))
    # round trip: the list back to a matrix is the matrix
    back = sp.csr_matrix((np.ones(len(ea)), ea.astype(np.int64), va.astype(np.int64)), shape=(n, n))
    assert (back != m).nnz == 0
    for i in range(n):                                  # ascending, no duplicates, no self loops
        row = ea[va[i]:va[i + 1]]
        assert (np.diff(row.astype(np.int64)) > 0).all() and i not in row
    o.close()


@pytest.mark.parametrize("directed", [False, True])
def test_bfs_levels_against_shortest_paths(directed):
    rng = np.random.default_rng(162)
    n = 3000
    t = _random_targets(rng, n, p_connect=0.9)
    o = _oracle(rng.uniform(1, 31, (n, 3)), segs=2)
    o.load_targets(t)
    o.build_graph(directed)
    va, ea = o.read_state("GRAPH_VA"), o.read_state("GRAPH_EA")
    m = sp.csr_matrix((np.ones(len(ea)), ea.astype(np.int64), va.astype(np.int64)), shape=(n, n))
    for root in (0, 17, int(np.argmax(np.diff(va)))):
        lev = o.bfs(root)
        d = shortest_path(m, directed=True, unweighted=True, indices=root)
        want = np.where(np.isinf(d), -1, d).astype(np.int32)
        assert np.array_equal(lev, want)
        assert lev[root] == 0
    o.close()


def test_bfs_closed_forms():
    n = 64
    o = _oracle(np.random.default_rng(1).uniform(1, 31, (n, 3)), segs=2)
    path = np.arange(1, n + 1, dtype=np.uint32)
    path[-1] = NONE                                     # 0 -> 1 -> ... -> n-1
    o.load_targets(path)
    o.build_graph(True)
    assert np.array_equal(o.bfs(0), np.arange(n))       # directed path from its head: level = index
    lev = o.bfs(10)
    assert (lev[:10] == -1).all() and np.array_equal(lev[10:], np.arange(n - 10))   # nothing upstream is reached
    o.build_graph(False)
    assert np.array_equal(o.bfs(10), np.abs(np.arange(n) - 10))
    ring = ((np.arange(n) + 1) % n).astype(np.uint32)
    o.load_targets(ring)
    o.build_graph(False)
    k = np.arange(n)
    assert np.array_equal(o.bfs(0), np.minimum(k, n - k))
    star = np.zeros(n, np.uint32)                       # every neuron connects to neuron 0
    star[0] = NONE
    o.load_targets(star)
    o.build_graph(False)
    assert np.array_equal(o.bfs(0), np.r_[0, np.ones(n - 1, int)])
    assert np.array_equal(o.bfs(5), np.r_[1, np.full(n - 1, 2)] * (np.arange(n) != 5))
    va = o.read_state("GRAPH_VA")
    assert va[1] - va[0] == n - 1 and (np.diff(va)[1:] == 1).all()
    o.close()
