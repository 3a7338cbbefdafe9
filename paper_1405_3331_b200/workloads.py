"""Seeded synthetic inputs C1..C5 (BASELINE.json `configs`, restated in DESIGN.md §4).

This module serves BOTH the CUDA path and the CPU oracle (tests, bench) and therefore holds none of the method's
arithmetic: it only draws input positions with numpy's `default_rng(seed)` and lists parameters.  The paper's own
workloads (100-5000 neurons on a sphere, "arbitrary" particle systems) publish no particle
counts; C1..C5 stand in for them.
"""
from __future__ import annotations

from dataclasses import dataclass, field

import numpy as np


@dataclass
class Workload:
    name: str
    grid: tuple            # (nx, ny, nz) unit cells
    D: float               # cell^2 / step
    emission: int          # default particles / step / source
    radius: float          # sensing radius, cells
    speed: float           # cells / step
    noise: float           # rad
    seed: int              # Philox seed
    neurons: np.ndarray    # (C, 3) float32 initial cone positions; headings default to +z (A-20)
    sources: list          # [(x, y, z, species, polarity, rate)]
    nominal_live: int      # particle count the config names
    timed_steps: int       # steps the config times
    prerun_steps: int      # real steps to the steady state (5 slowest-mode time constants), 0 = start empty
    max_particles: int = 0
    max_segments: int = 0
    notes: str = ""
    extra: dict = field(default_factory=dict)

    @property
    def cells(self):
        return int(self.grid[0]) * int(self.grid[1]) * int(self.grid[2])

    @property
    def emitted_per_step(self):
        return int(sum(s[5] for s in self.sources))


def _uniform_sources(rng, n, grid, margin, lo_z=None, hi_z=None):
    nx, ny, nz = grid
    x = rng.uniform(margin, nx - margin, n)
    y = rng.uniform(margin, ny - margin, n)
    z = rng.uniform(margin if lo_z is None else lo_z, (nz - margin) if hi_z is None else hi_z, n)
    return np.stack([x, y, z], 1).astype(np.float32)


def c1():
    """32^3, 8 cones on z=0.5, one source at (16,16,31) emitting 8/step, 200 steps from empty."""
    rng = np.random.default_rng(1001)
    xy = rng.uniform(0.0, 32.0, (8, 2))
    neurons = np.concatenate([xy, np.full((8, 1), 0.5)], 1).astype(np.float32)
    return Workload("C1", (32, 32, 32), 0.5, 8, 2.0, 0.25, 0.1, 1, neurons, [(16.0, 16.0, 31.0, 0, 1, 8)],
                    nominal_live=1500, timed_steps=200, prerun_steps=0, max_particles=1 << 14, max_segments=256,
                    notes="source is 1 sigma from an absorbing wall: steady n_live ~ 200, not 1.5k (DESIGN.md §4)")


def c2():
    """128^3, 1024 cones on z=0.5, 4 attractive sources in the top quarter, 256/step each, ~1M live (nominal)."""
    rng = np.random.default_rng(1002)
    xy = rng.uniform(0.0, 128.0, (1024, 2))
    neurons = np.concatenate([xy, np.full((1024, 1), 0.5)], 1).astype(np.float32)
    src = _uniform_sources(rng, 4, (128, 128, 128), 4.0, lo_z=96.0, hi_z=124.0)
    sources = [(float(p[0]), float(p[1]), float(p[2]), 0, 1, 256) for p in src]
    return Workload("C2", (128, 128, 128), 0.5, 256, 2.0, 0.25, 0.1, 2, neurons, sources, nominal_live=1_000_000,
                    timed_steps=1000, prerun_steps=5500, max_particles=3 << 20, max_segments=1200)


def c3(rate=350):
    """256^3, 16384 cones in the slab z<2, 12 attractive (species 0) + 4 repulsive (species 1) sources, ~16M live.
    rate: calibrated so that the steady state holds the ~16M particles the config names (226/step, the survey's
    estimate from mean exit times, settles at 10.4M on the GPU; the count is linear in the rate)."""
    rng = np.random.default_rng(1003)
    neurons = np.stack([rng.uniform(0.0, 256.0, 16384), rng.uniform(0.0, 256.0, 16384),
                        rng.uniform(0.0, 2.0, 16384)], 1).astype(np.float32)
    src = _uniform_sources(rng, 16, (256, 256, 256), 4.0)
    sources = [(float(p[0]), float(p[1]), float(p[2]), 0 if i < 12 else 1, 1 if i < 12 else -1, rate)
               for i, p in enumerate(src)]
    return Workload("C3", (256, 256, 256), 0.5, rate, 2.0, 0.25, 0.1, 3, neurons, sources, nominal_live=16_000_000,
                    timed_steps=500, prerun_steps=22000, max_particles=24_000_000, max_segments=1200)


def c4(rate=100):
    """512^3, 100k cones in 32 Gaussian clusters on z<8, 64 sources in 8 Gaussian blobs, two species, D=1, R=3."""
    rng = np.random.default_rng(1004)
    centres = np.stack([rng.uniform(16, 496, 32), rng.uniform(16, 496, 32), rng.uniform(0, 8, 32)], 1)
    which = rng.integers(0, 32, 100_000)
    p = centres[which] + rng.normal(0.0, 4.0, (100_000, 3))
    p[:, 0] = np.clip(p[:, 0], 0.0, 511.99)
    p[:, 1] = np.clip(p[:, 1], 0.0, 511.99)
    p[:, 2] = np.clip(p[:, 2], 0.0, 7.99)
    neurons = p.astype(np.float32)
    blob = _uniform_sources(rng, 8, (512, 512, 512), 40.0)
    sources = []
    for i in range(64):
        q = blob[i % 8] + rng.normal(0.0, 8.0, 3)
        q = np.clip(q, 4.0, 507.0)
        sp = i % 2
        sources.append((float(q[0]), float(q[1]), float(q[2]), sp, 1 if sp == 0 else -1, rate))
    return Workload("C4", (512, 512, 512), 1.0, rate, 3.0, 0.5, 0.05, 4, neurons, sources, nominal_live=64_000_000,
                    timed_steps=200, prerun_steps=45000, max_particles=120_000_000, max_segments=400)


def c5(rate=110):
    """1024x1024x256, 1M cones uniform on z<4, 256 sources, two species, ~256M live (bandwidth stress)."""
    rng = np.random.default_rng(1005)
    n = 1_000_000
    neurons = np.stack([rng.uniform(0.0, 1024.0, n), rng.uniform(0.0, 1024.0, n), rng.uniform(0.0, 4.0, n)],
                       1).astype(np.float32)
    src = _uniform_sources(rng, 256, (1024, 1024, 256), 4.0)
    sources = [(float(p[0]), float(p[1]), float(p[2]), i % 2, 1 if i % 2 == 0 else -1, rate)
               for i, p in enumerate(src)]
    return Workload("C5", (1024, 1024, 256), 0.5, rate, 2.0, 0.25, 0.1, 5, neurons, sources,
                    nominal_live=256_000_000, timed_steps=100, prerun_steps=60000, max_particles=300_000_000,
                    max_segments=200)


def small(seed=7, grid=(24, 20, 16), n_cones=24, n_sources=3, rate=40, two_species=True, radius=2.0):
    """A ragged little case for parity tests: non-cubic grid, sources of both polarities, cones anywhere."""
    rng = np.random.default_rng(seed)
    nx, ny, nz = grid
    neurons = np.stack([rng.uniform(0, nx, n_cones), rng.uniform(0, ny, n_cones), rng.uniform(0, nz, n_cones)],
                       1).astype(np.float32)
    src = _uniform_sources(rng, n_sources, grid, 2.0)
    sources = []
    for i, p in enumerate(src):
        sp = (i % 2) if two_species else 0
        sources.append((float(p[0]), float(p[1]), float(p[2]), sp, 1 if sp == 0 else -1, rate + i))
    return Workload("small", grid, 0.5, rate, radius, 0.25, 0.1, seed, neurons, sources, nominal_live=0,
                    timed_steps=0, prerun_steps=0, max_particles=1 << 16, max_segments=128)


def random_particles(seed, n, grid, n_species=2, clustered=True):
    """n particle rows inside the grid (for load_particles): a uniform background plus dense Gaussian clumps, so that
    some cells hold hundreds of particles and most hold none or one (the value structure of DESIGN.md §4)."""
    rng = np.random.default_rng(seed)
    nx, ny, nz = grid
    n_clump = n // 3 if clustered else 0
    bg = np.stack([rng.uniform(0, nx, n - n_clump), rng.uniform(0, ny, n - n_clump), rng.uniform(0, nz, n - n_clump)], 1)
    if n_clump:
        centres = np.stack([rng.uniform(0, nx, 4), rng.uniform(0, ny, 4), rng.uniform(0, nz, 4)], 1)
        cl = centres[rng.integers(0, 4, n_clump)] + rng.normal(0, 0.7, (n_clump, 3))
        p = np.concatenate([bg, cl], 0)
    else:
        p = bg
    p = p.astype(np.float32)
    hi = np.array([np.nextafter(np.float32(nx), np.float32(0)), np.nextafter(np.float32(ny), np.float32(0)),
                   np.nextafter(np.float32(nz), np.float32(0))], dtype=np.float32)
    p = np.clip(p, np.float32(0), hi)
    perm = rng.permutation(n)
    p = p[perm]
    species = rng.integers(0, n_species, n).astype(np.uint8)
    ids = rng.permutation(n).astype(np.uint32)
    return p[:, 0].copy(), p[:, 1].copy(), p[:, 2].copy(), species, ids


def weak_scaled(w: Workload, world: int) -> Workload:
    """The same config with `world` times the sources (hence particles): new sources of the same species / polarity / rate
    pattern at fresh seeded positions (4-cell margin), so that under sharding by source every rank owns one config's worth
    of particles while the cones and the grid stay those of `w` -- the weak-scaling input of `bench.py --scaling weak`."""
    if world <= 1:
        return w
    rng = np.random.default_rng(7000 + w.seed)
    copies = [list(w.sources)]
    for _ in range(world - 1):
        pos = _uniform_sources(rng, len(w.sources), w.grid, 4.0)
        copies.append([(float(p[0]), float(p[1]), float(p[2]), s[3], s[4], s[5]) for p, s in zip(pos, w.sources)])
    # rank r owns the sources with index % world == r (axg_set_shard): interleave, so that rank r owns exactly copy r
    w.sources = [copies[r][i] for i in range(len(copies[0])) for r in range(world)]
    w.nominal_live *= world
    w.notes += " weak-scaled x%d" % world
    return w


BY_NAME = {"C1": c1, "C2": c2, "C3": c3, "C4": c4, "C5": c5}


def apply(sim, w: Workload, place=True):
    """Drive any object with the boundary's call names (CUDA binding or oracle binding)."""
    if w.max_particles or w.max_segments:
        sim.set_capacity(w.max_particles or (1 << 20), w.max_segments or 1024)
    for s in w.sources:
        sim.add_source(*s)
    if place and len(w.neurons):
        sim.place_neurons(w.neurons, None)
    return sim


def synthetic_population(w: Workload, n, seed):
    """n particle rows shaped like the steady state of `w` WITHOUT running the method (input for CPU timing samples,
    bench.py `cpu_baseline` / `--impl reference`): per source a cloud whose width is drawn log-uniformly between one
    cell and the box size (dense within a few cells of the source, ~uniform far away), clipped by rejection to the
    box.  Species = the source's.  Ids 0..n-1 in a seeded random order."""
    rng = np.random.default_rng(seed)
    nx, ny, nz = w.grid
    src = np.array([[s[0], s[1], s[2]] for s in w.sources], dtype=np.float64)
    sp_of = np.array([s[3] for s in w.sources], dtype=np.uint8)
    out_p, out_s = [], []
    need = n
    while need > 0:
        m = int(need * 1.6) + 64
        which = rng.integers(0, len(src), m)
        width = np.exp(rng.uniform(0.0, np.log(max(nx, ny, nz) / 2.0), m))
        p = src[which] + rng.normal(0.0, 1.0, (m, 3)) * width[:, None]
        ok = (p[:, 0] >= 0) & (p[:, 0] < nx - 1e-3) & (p[:, 1] >= 0) & (p[:, 1] < ny - 1e-3) & (p[:, 2] >= 0) & \
             (p[:, 2] < nz - 1e-3)
        p, s = p[ok][:need], sp_of[which[ok]][:need]
        out_p.append(p.astype(np.float32))
        out_s.append(s)
        need -= len(p)
    p = np.concatenate(out_p, 0)
    species = np.concatenate(out_s, 0)
    ids = rng.permutation(n).astype(np.uint32)
    return p[:, 0].copy(), p[:, 1].copy(), p[:, 2].copy(), species, ids


def prerun(make_sim, w: Workload, coarse=16, relax=100, progress=None):
    """Bring a fresh simulation of `w` to its steady state with the library itself (DESIGN.md §4 "reaching the
    steady state"): a second context WITHOUT cones runs prerun_steps/coarse steps with D' = coarse*D and
    rate' = coarse*rate (the continuous steady state depends on rate/D only), its particle array is handed to the
    real context through read_state -> load_particles, and `relax` real steps wash out the coarse wall layer.
    `make_sim(D, emission)` returns an object with the boundary's call names.  coarse <= 1: plain pre-run.
    Returns the simulation, with neurons placed and the step counter at 0."""
    if w.prerun_steps <= 0:
        return apply(make_sim(w.D, w.emission), w)
    if coarse <= 1:
        pre = apply(make_sim(w.D, w.emission), w, place=False)
        pre.step(w.prerun_steps)
        cols = [pre.read_state("PART_" + k).copy() for k in ("X", "Y", "Z", "SPECIES", "ID")]
        next_id = pre.counters()["next_id"]
        pre.close()
        relax = 0
    else:
        pre = make_sim(w.D * coarse, w.emission * coarse)
        pre.set_capacity(w.max_particles or (1 << 20), 1)
        for s in w.sources:
            pre.add_source(s[0], s[1], s[2], s[3], s[4], s[5] * coarse)
        cap = w.max_particles or (1 << 20)
        e_coarse = sum(s[5] for s in w.sources) * coarse
        todo = max(1, w.prerun_steps // coarse)
        while todo > 0:
            # the boundary refuses a call whose host-side bound n_live + k * E could overflow the capacity
            n_live = pre.counters()["n_live"]
            k = int(min(todo, 256, (cap - n_live) // max(e_coarse, 1)))
            if k < 1:       # the capacity is reached before the steady state: hand over what there is
                break
            pre.step(k)
            todo -= k
            if progress:
                progress(n_live)
        cols = [pre.read_state("PART_" + k).copy() for k in ("X", "Y", "Z", "SPECIES", "ID")]
        next_id = pre.counters()["next_id"]
        pre.close()
    if relax:                # a cone-less context with the real D washes out the coarse wall layer
        mid = make_sim(w.D, w.emission)
        apply(mid, w, place=False)
        mid.load_particles(*cols, next_id=next_id, step=0)
        mid.step(relax)
        cols = [mid.read_state("PART_" + k).copy() for k in ("X", "Y", "Z", "SPECIES", "ID")]
        next_id = mid.counters()["next_id"]
        mid.close()
    sim = make_sim(w.D, w.emission)
    apply(sim, w)            # neurons are placed before the first step (AXG_ESTATE afterwards)
    sim.load_particles(*cols, next_id=next_id, step=0)
    return sim
