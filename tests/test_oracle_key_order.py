"""Pin T15: the bricked cell order ("a Z-order curve ... potential optimization";
DESIGN.md reading A-27) of the oracle: the key is a bijection from the grid's cells into the padded key space, the cells
of one 8 x 4 x 4 brick are contiguous, x runs inside a brick are contiguous; binning under it equals numpy's stable
argsort of an independently written key; sensing through the bricked cell table equals the all-pairs form (which knows
no keys) and the linear order's sums; nothing but the order of the particle array depends on it."""
import numpy as np
import pytest

from oracle import axo
from paper_1405_3331_b200 import workloads as W


def _brick_key(ix, iy, iz, grid):
    """written from the definition: bricks in linear order, cells inside a brick in linear order, x fastest"""
    nbx, nby = -(-grid[0] // 8), -(-grid[1] // 4)
    return ((iz // 4 * nby + iy // 4) * nbx + ix // 8) * 128 + iz % 4 * 32 + iy % 4 * 8 + ix % 8


def _morton_key(ix, iy, iz, grid):
    """written from the definition (reading A-31): bit b of x, then of y, then of z, b = 0, 1, ...; an axis that needs
    fewer bits than the others drops out once its bits are used up"""
    nb = [int(np.ceil(np.log2(n))) if n > 1 else 0 for n in grid]
    key = np.zeros_like(np.asarray(ix, dtype=np.int64))
    out = 0
    for b in range(max(nb) if max(nb) else 0):
        for v, bits in zip((ix, iy, iz), nb):
            if b < bits:
                key |= ((np.asarray(v, dtype=np.int64) >> b) & 1) << out
                out += 1
    return key


def _setup(grid, order, n=6000, seed=3, R=2.0):
    o = axo.Oracle(grid, 0.5, 0, R, 0.25, 0.1, seed)
    o.set_key_order(order)
    o.add_source(1.0, 1.0, 1.0, 0, 1, 1)
    o.add_source(2.0, 2.0, 2.0, 1, -1, 1)
    rng = np.random.default_rng(seed)
    cones = np.stack([rng.uniform(0, grid[a], 60) for a in range(3)], 1).astype(np.float32)
    o.place_neurons(cones)
    x, y, z, sp, ids = W.random_particles(seed, n, grid)
    o.load_particles(x, y, z, sp, ids, next_id=n, step=0)
    return o, (x, y, z, sp, ids)


@pytest.mark.parametrize("grid", [(24, 20, 16), (13, 7, 5), (8, 4, 4), (40, 33, 21)])
def test_T15_key_is_a_bijection_with_contiguous_bricks(grid):
    o, (x, y, z, sp, ids) = _setup(grid, 1)
    o.step_phase(axo.PHASE_BIN)
    ix, iy, iz = x.astype(np.int64), y.astype(np.int64), z.astype(np.int64)
    want = _brick_key(ix, iy, iz, grid)
    perm = o.read_state("PERM")
    assert np.array_equal(o.read_state("KEYS_SORTED"), want[perm])
    assert np.array_equal(perm, np.argsort(want, kind="stable"))
    # all cells of the grid: distinct keys below the padded size, a brick = 128 consecutive keys
    gx, gy, gz = np.meshgrid(np.arange(grid[0]), np.arange(grid[1]), np.arange(grid[2]), indexing="ij")
    k = _brick_key(gx.ravel(), gy.ravel(), gz.ravel(), grid)
    size = -(-grid[0] // 8) * -(-grid[1] // 4) * -(-grid[2] // 4) * 128
    assert len(np.unique(k)) == len(k) and k.max() < size
    assert len(o.read_state("CELL_START")) == size
    same_brick = (gx.ravel() // 8 == 0) & (gy.ravel() // 4 == 0) & (gz.ravel() // 4 == 0)
    assert set(k[same_brick]) <= set(range(128))
    # cellStart / cellEnd against the sorted keys
    ks = want[perm]
    cs, ce = o.read_state("CELL_START"), o.read_state("CELL_END")
    for c in np.unique(ks)[::17]:
        assert (cs[c], ce[c]) == (np.searchsorted(ks, c), np.searchsorted(ks, c, side="right"))
    assert cs[np.setdiff1d(np.arange(size), ks)].sum() == 0


@pytest.mark.parametrize("grid,R", [((24, 20, 16), 2.0), ((13, 7, 5), 3.0), ((40, 33, 21), 2.5)])
def test_T15_sensing_does_not_depend_on_the_cell_order(grid, R):
    res = []
    for order in (0, 1, 2):
        o, _ = _setup(grid, order, R=R)
        o.step_phase(axo.PHASE_BIN | axo.PHASE_SENSE)
        cnt, mom = o.read_state("CONE_COUNTS"), o.read_state("CONE_MOMENT")
        bc, bm = o.sense_brute()                       # all pairs, no keys, no cell table
        assert np.array_equal(cnt, bc.ravel()) and np.array_equal(mom, bm.ravel())
        res.append((cnt, mom))
    for other in res[1:]:
        assert np.array_equal(res[0][0], other[0]) and np.array_equal(res[0][1], other[1]) and res[0][0].sum() > 0


def test_T15_only_the_order_of_the_particle_array_depends_on_it():
    w = W.small(seed=5, grid=(20, 18, 14), n_cones=30, n_sources=4, rate=50)
    out = []
    for order in (0, 1, 2):
        o = axo.Oracle(w.grid, w.D, w.emission, w.radius, w.speed, w.noise, w.seed)
        o.set_key_order(order)
        W.apply(o, w)
        o.step(12)
        ids = o.read_state("PART_ID")
        srt = np.argsort(ids)
        out.append((ids[srt], o.read_state("PART_X")[srt], o.read_state("PART_Z")[srt], o.read_state("CONE_POS"),
                    o.read_state("POLYLINE"), o.counters()))
    for other in out[1:]:
        for a, b in zip(out[0][:5], other[:5]):
            assert np.array_equal(a.view(np.uint32) if a.dtype == np.float32 else a,
                                  b.view(np.uint32) if b.dtype == np.float32 else b)
        assert out[0][5] == other[5]


@pytest.mark.parametrize("grid", [(16, 16, 16), (24, 20, 16), (13, 7, 5), (64, 8, 4), (3, 9, 33), (40, 33, 21)])
def test_T15_morton_key_is_the_z_order_curve(grid):
    o, (x, y, z, sp, ids) = _setup(grid, 2)
    o.step_phase(axo.PHASE_BIN)
    ix, iy, iz = x.astype(np.int64), y.astype(np.int64), z.astype(np.int64)
    want = _morton_key(ix, iy, iz, grid)
    perm = o.read_state("PERM")
    assert np.array_equal(o.read_state("KEYS_SORTED"), want[perm])
    assert np.array_equal(perm, np.argsort(want, kind="stable"))
    gx, gy, gz = np.meshgrid(np.arange(grid[0]), np.arange(grid[1]), np.arange(grid[2]), indexing="ij")
    k = _morton_key(gx.ravel(), gy.ravel(), gz.ravel(), grid)
    size = 1
    for n in grid:
        size *= 1 << (int(np.ceil(np.log2(n))) if n > 1 else 0)
    assert len(np.unique(k)) == len(k) and k.max() < size and len(o.read_state("CELL_START")) == size
    if grid == (16, 16, 16):
        # the textbook curve on a cube: the first eight cells are the 2 x 2 x 2 octant in x, y, z order, and every aligned
        # 2^j cube is one contiguous run of 8^j keys
        first8 = [(0, 0, 0), (1, 0, 0), (0, 1, 0), (1, 1, 0), (0, 0, 1), (1, 0, 1), (0, 1, 1), (1, 1, 1)]
        assert [int(_morton_key(*c, grid)) for c in first8] == list(range(8))
        kk = k.reshape(16, 16, 16)
        for j in (1, 2, 3):
            e = 1 << j
            block = kk[e:2 * e, 0:e, e:2 * e].ravel()
            assert block.max() - block.min() == e ** 3 - 1 and block.min() % e ** 3 == 0
    ks = want[perm]
    cs, ce = o.read_state("CELL_START"), o.read_state("CELL_END")
    for c in np.unique(ks)[::17]:
        assert (cs[c], ce[c]) == (np.searchsorted(ks, c), np.searchsorted(ks, c, side="right"))


def test_T15_order_is_fixed_once_particles_exist():
    o, _ = _setup((8, 8, 8), 0)
    with pytest.raises(axo.OracleError):
        o.set_key_order(1)
