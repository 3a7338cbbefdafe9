"""The sharded step loop (paper_1405_3331_b200/sharded.py) over two `gloo` processes on the CPU.

The loop is host logic and drives any object with the boundary's call names; here it drives the ORACLE binding in two
processes (sources split by index parity), with the integer all-reduce of the per-cone sums between P3 and P4.  What
must hold, and is checked against the unsharded oracle in the parent: cone positions, headings, states and polylines
are bit-identical on both ranks; the union of the two particle shards is the unsharded particle set (same ids, same
positions bit for bit); the id counter advances as in the unsharded run.
"""
import os
import socket
import sys

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

STEPS = 6


def host_exchange(sim):
    """The exchange step of the sharded loop for a binding whose sums live on the host (the oracle): read -> all-reduce
    (gloo) -> load.  Test harness only: the product's exchange is sharded.nccl_exchange on the device buffer."""
    def run():
        c = torch.from_numpy(sim.read_state("CONE_COUNTS").astype(np.int64))
        m = torch.from_numpy(sim.read_state("CONE_MOMENT").astype(np.int64))
        if c.numel() == 0:
            return
        # frozen cones keep stale sums on every rank; they are not read by P4, only kept consistent here
        dist.all_reduce(c, op=dist.ReduceOp.SUM)
        dist.all_reduce(m, op=dist.ReduceOp.SUM)
        sim.load_sense(c.numpy(), m.numpy())
    return run


def _workload():
    from paper_1405_3331_b200 import workloads as W
    w = W.small(seed=21, grid=(20, 18, 14), n_cones=40, n_sources=5, rate=60)
    w.speed = 0.4
    return w


def _oracle(w, sensing=0):
    from oracle import axo
    from paper_1405_3331_b200 import workloads as W
    o = axo.Oracle(w.grid, w.D, w.emission, w.radius, w.speed, w.noise, w.seed)
    o.set_sensing(sensing)
    return W.apply(o, w)


def _state(o):
    out = {k: o.read_state(k).copy() for k in ("CONE_POS", "CONE_HEADING", "CONE_STATE", "POLY_LEN", "POLYLINE",
                                                "PART_ID", "PART_X", "PART_Y", "PART_Z", "PART_SPECIES")}
    out["counters"] = o.counters()
    return out


def _worker(rank, world, port, q, sensing):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        from paper_1405_3331_b200 import sharded
        w = _workload()
        o = _oracle(w, sensing)
        stepper = sharded.ShardedStepper(o, rank, world, host_exchange)
        stepper.step(STEPS)
        st = _state(o)
        q.put((rank, {k: (v if isinstance(v, dict) else v.tolist()) for k, v in st.items()}))
        dist.barrier()      # no rank tears the group down while the other is still inside a collective
    finally:
        dist.destroy_process_group()


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    port = s.getsockname()[1]
    s.close()
    return port


@pytest.mark.timeout(300)
@pytest.mark.parametrize("sensing", [0, 2])   # per-cell rule; per-particle weighted rule (integer sums as well, A-26)
def test_two_ranks_equal_the_unsharded_run(sensing):
    w = _workload()
    ref = _oracle(w, sensing)
    ref.step(STEPS)
    want = _state(ref)

    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q, sensing)) for r in range(2)]
    for p in procs:
        p.start()
    got = dict(q.get(timeout=240) for _ in range(2))
    for p in procs:
        p.join(60)
        assert p.exitcode == 0

    for r in (0, 1):
        g = got[r]
        for k in ("CONE_STATE", "POLY_LEN"):
            assert np.array_equal(np.array(g[k], dtype=want[k].dtype), want[k]), (r, k)
        for k in ("CONE_POS", "CONE_HEADING", "POLYLINE"):
            a = np.array(g[k], dtype=np.float32)
            assert np.array_equal(a.view(np.uint32), want[k].view(np.uint32)), (r, k)
        assert g["counters"]["step"] == want["counters"]["step"]
        assert g["counters"]["next_id"] == want["counters"]["next_id"]
    # the shards partition the particle set
    ids = np.concatenate([np.array(got[r]["PART_ID"], dtype=np.uint32) for r in (0, 1)])
    assert len(ids) == len(want["PART_ID"]) and len(np.unique(ids)) == len(ids)
    order_w = np.argsort(want["PART_ID"])
    order_g = np.argsort(ids)
    assert np.array_equal(ids[order_g], want["PART_ID"][order_w])
    for k in ("PART_X", "PART_Y", "PART_Z"):
        a = np.concatenate([np.array(got[r][k], dtype=np.float32) for r in (0, 1)])
        assert np.array_equal(a[order_g].view(np.uint32), want[k][order_w].view(np.uint32)), k
    sp = np.concatenate([np.array(got[r]["PART_SPECIES"], dtype=np.uint8) for r in (0, 1)])
    assert np.array_equal(sp[order_g], want["PART_SPECIES"][order_w])
    assert got[0]["counters"]["emitted"] + got[1]["counters"]["emitted"] == want["counters"]["emitted"]


def test_owned_sources_partition():
    from paper_1405_3331_b200 import sharded
    for world in (1, 2, 3, 8):
        seen = sorted(s for r in range(world) for s in sharded.owned_sources(13, r, world))
        assert seen == list(range(13))


def test_weak_scaled_workload_gives_every_rank_one_configs_worth_of_sources():
    """bench.py --scaling weak: `world` times the sources (same species / polarity / rate pattern, new seeded positions
    inside the 4-cell margin), cones and grid unchanged, so that sharding by source leaves every rank with the source
    count -- hence the particle count -- of the 1-GPU config."""
    from paper_1405_3331_b200 import sharded, workloads as W
    base = W.c3()
    for world in (1, 2, 8):
        w = W.weak_scaled(W.c3(), world)
        assert len(w.sources) == world * len(base.sources) and w.grid == base.grid
        assert np.array_equal(w.neurons, base.neurons) and w.max_particles == base.max_particles
        assert w.sources[::world] == base.sources                                        # rank 0 owns the config's own
        for r in range(world):
            own = [w.sources[s] for s in sharded.owned_sources(len(w.sources), r, world)]
            assert len(own) == len(base.sources)
            assert sum(s[5] for s in own) == base.emitted_per_step
            assert sorted(s[3] for s in own) == sorted(s[3] for s in base.sources)      # same species mix per rank
        for s in w.sources:
            assert all(4.0 <= s[a] <= w.grid[a] - 4.0 for a in range(3))
        pol = {}
        for s in w.sources:
            assert pol.setdefault(s[3], s[4]) == s[4]                                    # one polarity per species
