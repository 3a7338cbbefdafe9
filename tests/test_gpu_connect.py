"""GPU-vs-oracle parity of connection formation, the adjacency list and the BFS (DESIGN.md
readings A-28..A-30; include/axg.h axg_set_connect / axg_build_graph / axg_bfs).  Everything here is an integer result:
bit-exact.  The collision test takes fp32 differences of cone and soma positions, so -- like the binning on particle
positions -- it is compared on identical cone positions: the oracle is handed the library's cones before the phase."""
import numpy as np
import pytest

from oracle import axo
from paper_1405_3331_b200 import workloads as W

import parity_util as pu

pytestmark = pytest.mark.gpu
NONE = axo.NO_TARGET


@pytest.fixture(scope="module")
def axg():
    from paper_1405_3331_b200 import axg as m
    m.lib()
    return m


def _hand_over_cones(g, o):
    o.load_cones(g.read_state("CONE_POS"), g.read_state("CONE_HEADING"), g.read_state("CONE_STATE"),
                 g.read_state("POLY_LEN"))


def test_chain_with_connection_formation(axg):
    """Whole steps phase by phase with cue particles, cones steering, and the connect phase after P5."""
    w = W.small(seed=31, grid=(24, 20, 16), n_cones=400, n_sources=3, rate=60)
    w.speed = 0.5
    g, o = pu.make_pair(w, axg)
    for s in (g, o):
        s.set_connect(0.4, 0.6)
    pu.load_same_particles(g, o, 5, 40_000, w.grid, step=0)
    connected = 0
    for t in range(8):
        g.step_phase(axg.PHASE_DIFFUSE | axg.PHASE_BIN)
        o.step_phase(axo.PHASE_DIFFUSE)
        pu.compare_presort(pu.pre_arrays(g), pu.pre_arrays(o), w.grid, w.emitted_per_step)
        pu.feed_gpu_presort_to_oracle(g, o, t)
        for ph in (axg.PHASE_SENSE, axg.PHASE_ADVANCE):
            g.step_phase(ph)
            o.step_phase(ph)
        pu.compare_sense(g, o)
        pu.compare_cones(g, o)
        _hand_over_cones(g, o)
        g.step_phase(axg.PHASE_CONNECT | axg.PHASE_COMMIT)
        o.step_phase(axo.PHASE_CONNECT | axo.PHASE_COMMIT)
        assert np.array_equal(g.read_state("CONE_TARGET"), o.read_state("CONE_TARGET"))
        assert np.array_equal(g.read_state("CONE_STATE"), o.read_state("CONE_STATE"))
        assert g.counters()["connected"] == o.counters()["connected"]
        connected = g.counters()["connected"]
    assert connected > 20
    for directed in (False, True):
        g.build_graph(directed)
        o.build_graph(directed)
        assert np.array_equal(g.read_state("GRAPH_VA"), o.read_state("GRAPH_VA"))
        assert np.array_equal(g.read_state("GRAPH_EA"), o.read_state("GRAPH_EA"))
        root = int(np.argmax(np.diff(o.read_state("GRAPH_VA").astype(np.int64))))
        assert np.array_equal(g.bfs(root), o.bfs(root))
    g.close()
    o.close()


def test_whole_steps_without_cues_are_bit_identical(axg):
    """No sources and noise 0: every cone keeps its heading, both sides add speed x heading with the same
    individually rounded operations, so positions -- hence connections, polylines and states -- agree bit for bit over
    whole axg_step calls (the connect phase rides on the side stream with P3..P5 there)."""
    rng = np.random.default_rng(41)
    n = 3000
    grid = (40, 36, 28)
    somata = np.stack([rng.uniform(1, 39, n), rng.uniform(1, 35, n), rng.uniform(1, 27, n)], 1).astype(np.float32)
    hd = rng.normal(size=(n, 3)).astype(np.float32)
    g = axg.Axg(grid, 0.5, 1, 2.0, 0.35, 0.0, 7)
    o = axo.Oracle(grid, 0.5, 1, 2.0, 0.35, 0.0, 7)
    for s in (g, o):
        s.set_capacity(1024, 64)
        s.set_connect(0.3, 0.5)
        s.place_neurons(somata, hd)
    for k in (1, 2, 7, 30):                       # plain enqueueing, the overlapped path, and the CUDA-graph path
        g.step(k)
        o.step(k)
        assert g.counters() == o.counters()
        for f in ("CONE_TARGET", "CONE_STATE", "POLY_LEN"):
            assert np.array_equal(g.read_state(f), o.read_state(f)), f
        for f in ("CONE_POS", "CONE_HEADING", "POLYLINE"):
            assert np.array_equal(g.read_state(f).view(np.uint32), o.read_state(f).view(np.uint32)), f
    c = g.counters()
    assert c["connected"] > 300 and c["exited"] > 300
    g.close()
    o.close()


def test_connect_phase_on_a_dense_given_state(axg):
    """20 000 neurons in a 64 x 48 x 40 box (several somata per soma-grid cell), tips scattered around other somata,
    on walls and in corners; a tenth frozen; three reaches (soma-grid cells of 1, 2 and 4 unit cells)."""
    rng = np.random.default_rng(43)
    n = 20_000
    grid = (64, 48, 40)
    hi = np.nextafter(np.asarray(grid, np.float32), np.float32(0))
    somata = (rng.uniform(0, 1, (n, 3)) * np.asarray(grid)).astype(np.float32)
    somata = np.minimum(somata, hi)
    tips = somata[rng.permutation(n)] + rng.normal(0, 0.9, (n, 3)).astype(np.float32)
    tips[:50] = somata[rng.permutation(n)[:50]]                    # exactly on another soma: d2 = 0
    tips = np.clip(tips, 0, hi).astype(np.float32)
    tips[50:60, 0] = 0.0
    tips[60:70] = hi
    state = (rng.uniform(size=n) < 0.1).astype(np.uint8) * 2
    hd = np.tile(np.array([0, 0, 1], np.float32), (n, 1))
    for r_c, r_s in ((0.25, 0.5), (0.75, 1.0), (1.5, 2.0)):
        g = axg.Axg(grid, 0.5, 1, 2.0, 0.25, 0.1, 3)
        o = axo.Oracle(grid, 0.5, 1, 2.0, 0.25, 0.1, 3)
        for s in (g, o):
            s.set_capacity(1024, 4)
            s.place_neurons(somata, None)
            s.set_connect(r_c, r_s)                                  # after the neurons: the soma grid is rebuilt
            s.load_cones(tips, hd, state, np.full(n, 2, np.uint32))
            s.step_phase(axg.PHASE_CONNECT)
        gt, ot = g.read_state("CONE_TARGET"), o.read_state("CONE_TARGET")
        assert np.array_equal(gt, ot), "reach %g: %d differ" % (r_c + r_s, int((gt != ot).sum()))
        assert np.array_equal(g.read_state("CONE_STATE"), o.read_state("CONE_STATE"))
        assert (gt != NONE).sum() > 1000
        g.close()
        o.close()


@pytest.mark.parametrize("directed", [False, True])
def test_graph_and_bfs_on_given_targets(axg, directed):
    """2e5 vertices: random connections, mutual pairs, a hub with 5 000 in-neighbours (rank-by-counting path of the list
    sort), one with 1 000 (bitonic path), one with 33 and one with 32 (the inline limit), isolated vertices."""
    rng = np.random.default_rng(47)
    n = 200_000
    t = np.full(n, NONE, np.uint32)
    pick = np.flatnonzero(rng.uniform(size=n) < 0.8)
    j = rng.integers(0, n - 1, len(pick))
    t[pick] = np.where(j < pick, j, j + 1).astype(np.uint32)
    perm = rng.permutation(n)
    at = 0
    for hub, deg in ((11, 5000), (12, 1000), (13, 33), (14, 32)):
        src = perm[at:at + deg]
        src = src[src != hub]
        t[src] = hub
        at += deg
    for _ in range(500):
        a, b = rng.choice(n, 2, replace=False)
        t[a], t[b] = b, a
    pos = rng.uniform(1, 63, (n, 3)).astype(np.float32)
    g = axg.Axg((64, 64, 64), 0.5, 1, 2.0, 0.25, 0.1, 3)
    o = axo.Oracle((64, 64, 64), 0.5, 1, 2.0, 0.25, 0.1, 3)
    for s in (g, o):
        s.set_capacity(1024, 2)
        s.place_neurons(pos, None)
        s.load_targets(t)
        s.build_graph(directed)
    va, ea = g.read_state("GRAPH_VA"), g.read_state("GRAPH_EA")
    assert np.array_equal(va, o.read_state("GRAPH_VA"))
    assert np.array_equal(ea, o.read_state("GRAPH_EA"))
    assert len(ea) == va[-1] and len(ea) > n // 2
    for root in (11, 0, int(perm[-1])):
        assert np.array_equal(g.bfs(root), o.bfs(root))
    g.close()
    o.close()


def test_bfs_on_a_long_path(axg):
    """3 000 levels: one kernel pair per level, 'repeated until frontier is empty'."""
    n = 3000
    t = np.arange(1, n + 1, dtype=np.uint32)
    t[-1] = NONE
    pos = np.random.default_rng(3).uniform(1, 31, (n, 3)).astype(np.float32)
    g = axg.Axg((32, 32, 32), 0.5, 1, 2.0, 0.25, 0.1, 3)
    g.set_capacity(1024, 2)
    g.place_neurons(pos, None)
    g.load_targets(t)
    g.build_graph(True)
    assert np.array_equal(g.bfs(0), np.arange(n))              # closed form: level = index
    lev = g.bfs(100)
    assert (lev[:100] == -1).all() and np.array_equal(lev[100:], np.arange(n - 100))
    g.build_graph(False)
    assert np.array_equal(g.bfs(100), np.abs(np.arange(n) - 100))
    with pytest.raises(axg.AxgError):
        g.bfs(n)
    g.close()
