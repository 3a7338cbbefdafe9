#!/usr/bin/env python
"""bench.py -- particle-steps/s of the whole axon-guidance step (P1..P5) on the synthetic configs of BASELINE.json.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload C3] [--impl ours|reference]

One "step" = one pass of the whole hot path (diffuse+absorb+emit+compact+key, radix sort, reorder + cell ranges,
sense, advance, append) over the live particle population of the workload.  Default workload: C3 (256^3 grid,
16 384 cones, 16 sources of two species, ~16M live particles), the configuration north_star quotes its target on.

Prints ONE JSON line (rank 0).  `value` is measured with every input resident in HBM; `e2e` goes through the C-ABI
with host buffers (pinned) and has the host<->device copies inside the timed region; `roofline` is the dominant
kernel (algorithmic bytes / CUDA-event time / measured copy bandwidth); `cpu_baseline` is the oracle, as it stands,
on the box's host cores over a bounded sample.  DESIGN.md §7 states every byte count used here.

N > 1 (torchrun): the workload is sharded BY SOURCE: every rank owns sources s % N == rank and all
their particles, senses all cones over its own particles, and one integer all-reduce (NCCL) of the per-cone sums per
step makes the cone update bit-identical to the 1-GPU run.  Total work is fixed => "scaling": "strong".

`--impl reference`: this tier has no reference program; the arm times the CPU oracle (oracle/) on host cores over a
bounded sample of the same workload (rank 0 only).
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import tempfile
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "particle-steps/s of diffuse+bin+sense step"
UNIT = "particle-steps/s"
HBM_FALLBACK_GBS = 6650.0     # /opt/skills/guides/B200_PROFILING.md "FALLBACK"
NOMINAL_GBS = 8000.0          # north_star's "~8 TB/s"
# dram__bytes_read.sum + dram__bytes_write.sum per launch of the dominant kernel, from the `ncu --set full` capture
# summarised in profiles/ (a capture is not repeatable inside a timed run, so it is a recorded number).
TRAFFIC_NCU = {   # (workload, kernel) -> bytes per launch; profiles/r02_summary.md (radix kernels: r01_summary.md)
    ("C3", "k_diffuse_chunked"): 754.8e6, ("C3", "k_diffuse"): 578.9e6, ("C3", "k_settle"): 654.7e6,
    ("C3", "k_place"): 247.1e6, ("C3", "k_cell_scan2"): 175.0e6, ("C3", "k_sort_pass"): 203.7e6,
    ("C3", "k_reorder"): 740.8e6,
    ("C4", "k_diffuse_chunked"): 3718.3e6, ("C4", "k_settle"): 2855.0e6, ("C4", "k_place"): 1255.4e6,
    ("C4", "k_cell_scan2"): 2088.0e6,
}
# the same capture summed over the kernels of one step (count binning: P1 + scan + place + settle + sense + advance)
STEP_TRAFFIC_NCU = {("C3", "count"): 1836.0e6, ("C4", "count"): 9920.0e6}


def log(*a):
    print(*a, file=sys.stderr, flush=True)


def measured_peak():
    try:
        with open(os.path.join(ROOT, "MEASURED_PEAKS.json")) as f:
            return float(json.load(f)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs, torch copy read+write)"
    except Exception:
        return HBM_FALLBACK_GBS, "fallback (B200_PROFILING.md)"


# ---------------------------------------------------------------------------------------------------------------
# algorithmic bytes: what the method must move per particle and per step
# ---------------------------------------------------------------------------------------------------------------
def key_passes(cells):
    """digit passes of the radix sort: 8-bit digits, 9-bit where that saves a pass (axg_api.cu digit_bits_for)"""
    bits = 1
    while bits < 32 and (1 << bits) < cells:
        bits += 1
    return min((bits + 7) // 8, (bits + 8) // 9)


def bytes_model(w, n_live, n_active_cones, n_stencil, count_mode):
    """Algorithmic bytes of ONE step at n_live particles.  `step` is SURVEY.md §8(d)'s figure for the
    METHOD (K1 38 + sort 12 + 16 (passes - 1) + reorder 42 per particle, 8 B per cell of cell-range upkeep, the cone
    bytes) and does not depend on how P2 is computed; the per-kernel entries are what each kernel of the chosen
    binning mode must move itself."""
    passes = key_passes(w.cells)
    two_species = len({s[3] for s in w.sources}) > 1
    per_cone = n_stencil * 8 + 90 + 12 + (n_stencil * 1 if two_species else 0)
    sense = float(per_cone) * n_active_cones
    step = (38.0 + 12.0 + 16.0 * (passes - 1) + 42.0) * n_live + 8.0 * w.cells + sense
    if count_mode:
        k = {"diffuse": (37.0 + 8.0) * n_live,    # 17 read + record 16 + key 4, + the 4 B counting atomic on cnt[key] and
                                                   # the 4 B arrival rank it returns (the species byte rides in its top bits)
             "scan": 12.0 * (w.cells + 1),         # read cnt, write cell_lo, re-zero cnt
             "place": 16.0 * n_live,               # key 4 + arrival rank | species 4 + cell start 4 + slot 4
             "settle": 45.0 * n_live,              # slot 4 + record 16 + cell_lo 8 + SoA 17 (keys / perm: derived on read)
             "sense": sense}
        launches = {"diffuse": 1, "scan": 1, "place": 1, "settle": 1, "sense": 1}
        # SURVEY.md §8(d) bytes of the phases these kernels stand for: K1 38; sort (12 + 16 (passes - 1)) split over scan
        # and place (which together replace the digit passes); reorder + cell ranges 42 B + 8 B per cell
        sort_b = (12.0 + 16.0 * (passes - 1)) * n_live
        survey = {"diffuse": 38.0 * n_live, "scan": 8.0 * w.cells, "place": sort_b, "settle": 42.0 * n_live, "sense": sense}
    else:
        k = {"diffuse": 38.0 * n_live,
             "sort": (12.0 + 16.0 * (passes - 1)) * n_live,   # pass 0: 4 read + 8 write; later passes 8 + 8
             "reorder": 42.0 * n_live + 4.0 * w.cells,        # perm 4 + key 4 + gather 17 + write 17; 4 B / cell
             "sense": sense}
        launches = {"diffuse": 1, "sort": passes, "reorder": 1, "sense": 1}
        survey = {"diffuse": 38.0 * n_live, "sort": (12.0 + 16.0 * (passes - 1)) * n_live,
                  "reorder": 42.0 * n_live + 8.0 * w.cells, "sense": sense}
    return step, k, launches, survey


class ClockSampler:
    """SM clock and throttle reasons sampled DURING the run (B200_PROFILING.md clocks line): a thread that polls NVML
    every millisecond from before the warm-up to after the last measured phase (ctypes calls release the GIL, so it
    runs while axg_step blocks).  `mark()` brackets the timed region; the record reports the samples that fell inside
    it and, separately, all samples under load.  Falls back to an `nvidia-smi -lms` subprocess without pynvml."""

    REASONS = ((0x8, "hw_slowdown"), (0x40, "hw_thermal_slowdown"), (0x20, "sw_thermal_slowdown"), (0x4, "sw_power_cap"))

    def __init__(self, index):
        import threading
        self.samples = []      # (t, sm_mhz, reasons bitmask, power_w)
        self.t0 = self.t1 = None
        self.max_mhz = None
        self._stop = threading.Event()
        self._thread = None
        try:
            import pynvml
            pynvml.nvmlInit()
            idx = index
            vis = os.environ.get("CUDA_VISIBLE_DEVICES")
            if vis:
                try:
                    idx = int(vis.split(",")[index])
                except (ValueError, IndexError):
                    idx = index
            h = pynvml.nvmlDeviceGetHandleByIndex(idx)
            self.max_mhz = float(pynvml.nvmlDeviceGetMaxClockInfo(h, pynvml.NVML_CLOCK_SM))
            reasons = getattr(pynvml, "nvmlDeviceGetCurrentClocksEventReasons", None) or \
                pynvml.nvmlDeviceGetCurrentClocksThrottleReasons

            def poll():
                while not self._stop.is_set():
                    try:
                        self.samples.append((time.time(), float(pynvml.nvmlDeviceGetClockInfo(h, pynvml.NVML_CLOCK_SM)),
                                             int(reasons(h)), pynvml.nvmlDeviceGetPowerUsage(h) / 1000.0))
                    except Exception:
                        pass
                    self._stop.wait(0.001)
            self._thread = threading.Thread(target=poll, daemon=True)
            self._thread.start()
        except Exception as e:    # no NVML binding: the recipe's nvidia-smi line, 20 ms period
            log("[bench] pynvml unavailable (%s): nvidia-smi sampler" % e)
            self._smi(index)

    def _smi(self, index):
        self.f = tempfile.NamedTemporaryFile("w+", suffix=".csv", delete=False)
        try:
            self.p = subprocess.Popen(["nvidia-smi", "-i", str(index), "--query-gpu=timestamp,clocks.sm,clocks.max.sm,"
                                       "power.draw,clocks_event_reasons.hw_slowdown,"
                                       "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
                                       "clocks_event_reasons.sw_power_cap", "--format=csv,noheader,nounits", "-lms", "20"],
                                      stdout=self.f, stderr=subprocess.DEVNULL)
        except Exception:
            self.p = None

    def mark(self, begin):
        if begin:
            self.t0 = time.time()
        else:
            self.t1 = time.time()

    def stop(self):
        import datetime
        self._stop.set()
        if self._thread is not None:
            self._thread.join(timeout=2)
        elif getattr(self, "p", None) is not None:
            self.p.terminate()
            try:
                self.p.wait(timeout=5)
            except Exception:
                self.p.kill()
            self.f.flush()
            self.f.seek(0)
            for line in self.f:
                c = [x.strip() for x in line.split(",")]
                if len(c) < 8:
                    continue
                try:
                    t = datetime.datetime.strptime(c[0], "%Y/%m/%d %H:%M:%S.%f").timestamp()
                    mask = sum(bit for (bit, _), v in zip(self.REASONS, c[4:8]) if v == "Active")
                    self.samples.append((t, float(c[1]), mask, float(c[3])))
                    self.max_mhz = float(c[2])
                except ValueError:
                    continue
            self.f.close()
            try:
                os.unlink(self.f.name)
            except OSError:
                pass
        out = {"sm_mhz": None, "sm_max_mhz": self.max_mhz, "reasons": [], "samples": 0}
        if not self.samples:
            return out
        inside = [x for x in self.samples if self.t0 is not None and self.t1 is not None and self.t0 <= x[0] <= self.t1]
        busy = [x for x in self.samples if x[3] > 0.5 * max(y[3] for y in self.samples)] or self.samples
        use = inside or busy
        mask = 0
        for x in use:
            mask |= x[2]
        out.update({"sm_mhz": float(np.median([x[1] for x in use])), "samples": len(inside),
                    "samples_under_load": len(busy), "sm_mhz_under_load": float(np.median([x[1] for x in busy])),
                    "reasons": [nm for bit, nm in self.REASONS if mask & bit],
                    "power_w_max": float(max(x[3] for x in self.samples)),
                    "how": "NVML polled every ms in a thread; sm_mhz / reasons = the samples inside the timed region "
                           "(all samples under load if none fell inside)"})
        return out


# ---------------------------------------------------------------------------------------------------------------
# the oracle on host cores (cpu_baseline leg and --impl reference arm): the only places bench.py runs oracle/
# ---------------------------------------------------------------------------------------------------------------
def time_oracle(w, n_sample, steps, warmup, seed=4242, want_n_end=False):
    """Particle-steps/s of the CPU oracle (single thread, as it stands) on `w` with a synthetic steady-state-shaped
    population of n_sample particles (workloads.synthetic_population).  Returns (value, seconds, particle_steps)."""
    from oracle import axo
    from paper_1405_3331_b200 import workloads as W
    o = axo.Oracle(w.grid, w.D, w.emission, w.radius, w.speed, w.noise, w.seed)
    o.set_capacity(n_sample + (steps + warmup + 2) * w.emitted_per_step + 64, steps + warmup + 4)
    for s in w.sources:
        o.add_source(*s)
    if len(w.neurons):
        o.place_neurons(w.neurons, None)
    o.load_particles(*W.synthetic_population(w, n_sample, seed), next_id=n_sample, step=0)
    if warmup:
        o.step(warmup)
    psteps, secs = 0, 0.0
    for _ in range(steps):
        n_in = o.counters()["n_live"]
        t0 = time.perf_counter()
        o.step(1)
        secs += time.perf_counter() - t0
        psteps += n_in
    n_end = o.counters()["n_live"]
    o.close()
    if want_n_end:
        return psteps / max(secs, 1e-12), secs, psteps, n_end
    return psteps / max(secs, 1e-12), secs, psteps


def oracle_sample_size(w, budget_s, steps):
    """Particles per step so that `steps` oracle steps take about budget_s: t(n) = a + b n from two short probes
    (a = the per-step fixed cost: clearing cellStart / cellEnd of the whole grid, the cones)."""
    n0, n1 = 50_000, 200_000
    _, t0, _ = time_oracle(w, n0, 1, 0)
    _, t1, _ = time_oracle(w, n1, 1, 0)
    b = max((t1 - t0) / (n1 - n0), 1e-9)
    a = max(t0 - b * n0, 0.0)
    n = int((budget_s / max(steps, 1) - a) / b)
    return max(20_000, min(n, w.nominal_live or n))


def run_reference(args, w):
    """--impl reference: the oracle, timed on host cores; each step a bounded sample of the workload."""
    budget = float(os.environ.get("AXG_REFERENCE_BUDGET_S", "60"))
    n = oracle_sample_size(w, budget, args.steps + args.warmup)
    value, secs, psteps, n_end = time_oracle(w, n, args.steps, args.warmup, want_n_end=True)
    sample = "%d of the workload's ~%d particles (synthetic steady-state-shaped population), all %d cones, %d steps" % (
        n, w.nominal_live, len(w.neurons), args.steps)
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": 1e3 * secs / max(args.steps, 1), "higher_is_better": True,
        "scaling": "strong" if args.gpus > 1 else "weak", "vs_baseline": None, "dtype": "f32+u32 (oracle: f64 Box-Muller)",
        "data": "synthetic", "config": {"workload": w.name, "grid": list(w.grid), "cones": int(len(w.neurons)),
                                        "sources": len(w.sources), "n_live_start": n, "n_live_end": n_end,
                                        "sample_particles": n},
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": 1, "kind": "oracle", "sample": sample},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line), flush=True)


# ---------------------------------------------------------------------------------------------------------------
# the CUDA path
# ---------------------------------------------------------------------------------------------------------------
def pinned(n, dtype):
    import torch
    tdt = {np.float32: torch.float32, np.uint8: torch.uint8, np.uint32: torch.int32, np.uint64: torch.int64,
           np.int64: torch.int64}[dtype]
    return torch.empty(max(int(n), 1), dtype=tdt, pin_memory=True).numpy().view(dtype)[: int(n)]


def run_ours(args, w):
    import torch
    import torch.distributed as dist
    from paper_1405_3331_b200 import axg, sharded, workloads as W

    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the library has no CPU fallback")
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    axg.lib()   # raises if libaxg.so is missing: no fallback

    K, Wm = args.steps, args.warmup
    e2e_steps = max(1, min(K, args.e2e_steps))
    w.max_segments = 2 * Wm + 4 * K + e2e_steps + 16     # warm-up + timed + per-kernel pass, twice (radix record), + e2e
    seed = w.seed

    bin_req = {"auto": axg.BIN_AUTO, "radix": axg.BIN_RADIX, "count": axg.BIN_COUNT}[args.binning]

    def make_sim(D, emission):
        sim_ = axg.Axg(w.grid, D, emission, w.radius, w.speed, w.noise, seed)
        if args.key_order != "linear":
            sim_.set_key_order(axg.KEY_BRICK if args.key_order == "brick" else axg.KEY_MORTON)
        sim_.set_binning(bin_req)
        if world > 1:
            sim_.set_shard(rank, world)   # every rank pre-runs its own shard: particle sets of sources never interact
        return sim_

    t0 = time.time()
    sim = W.prerun(make_sim, w, coarse=args.coarse)
    if args.steering == "snr":
        sim.set_steering(axg.STEER_SNR, 8.0, np.pi / 30)
    if args.sensing != "cell":
        sim.set_sensing(axg.SENSE_PARTICLE if args.sensing == "particle" else axg.SENSE_PARTICLE_WEIGHTED)
    if world > 1 or args.force_sharded_loop:
        step = sharded.ShardedStepper(sim, rank, world, sharded.nccl_exchange).step
    else:
        step = sim.step
    count_mode = sim.get_binning() == axg.BIN_COUNT     # what AXG_BIN_AUTO resolved to, asked of the library
    c0 = sim.counters()
    log("[bench] rank %d: %s steady state in %.1f s: n_live=%d" % (rank, w.name, time.time() - t0, c0["n_live"]))

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    def timed(fn):
        ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        barrier()
        ev0.record()
        fn()
        ev1.record()
        barrier()
        ms = ev0.elapsed_time(ev1)
        if world > 1:
            t = torch.tensor([ms], device="cuda", dtype=torch.float64)
            dist.all_reduce(t, op=dist.ReduceOp.MAX)
            ms = float(t.item())
        return ms

    def total(v):
        if world > 1:
            t = torch.tensor([float(v)], device="cuda", dtype=torch.float64)
            dist.all_reduce(t, op=dist.ReduceOp.SUM)
            return float(t.item())
        return float(v)

    # ---- warm-up, then the timed region: exactly K steps, inputs resident in HBM ------------------------------
    clocks = ClockSampler(local)    # from before the warm-up to after the last measured phase
    step(Wm)
    n_start = sim.counters()["n_live"]
    torch.cuda.profiler.start()     # `ncu --profile-from-start off` captures the timed region only
    clocks.mark(True)
    ms = timed(lambda: step(K))
    clocks.mark(False)
    torch.cuda.profiler.stop()
    st = sim.last_step_stats()
    psteps = total(st["particle_steps"])
    launches = int(st["launches"])
    value = psteps / (ms * 1e-3)
    cnt = sim.counters()
    n_end = cnt["n_live"]

    # ---- per-kernel CUDA-event times over K more steps (same launch configuration; events between kernels) ----
    ktimes, roof = None, None
    if world == 1 and not args.force_sharded_loop:     # (the sharded loop enqueues phases itself: no per-kernel events)
        sim.profile_next_step(True)
        step(K)
        ktimes = sim.kernel_times()
        st2 = sim.last_step_stats()
        n_avg = st2["particle_steps"] / K
        active = sim.counters()["active"]
    # ---- the path north_star spells out (onesweep radix passes + reorder), timed on the same state, same K ---------
    radix_rec = None
    if world == 1 and count_mode and not args.no_radix_record and not args.force_sharded_loop:
        sim.set_binning(axg.BIN_RADIX)
        step(Wm)
        ms_r = timed(lambda: step(K))
        ps_r = sim.last_step_stats()["particle_steps"]
        sim.profile_next_step(True)
        step(K)
        kt_r = sim.kernel_times()
        sort_ms = kt_r["sort"] / K
        radix_rec = {"ms_per_step": ms_r / K, "particle_steps_per_s": ps_r / (ms_r * 1e-3),
                     "sort_ms_per_step": sort_ms, "passes": key_passes(w.cells),
                     "sort_keys_per_s": (sim.last_step_stats()["particle_steps"] / K) / max(sort_ms * 1e-3, 1e-12),
                     "kernels_ms_per_step": {k: round(v / K, 5) for k, v in kt_r.items() if v > 0},
                     "what": "axg_set_binning(AXG_BIN_RADIX): k_diffuse (chained compaction), one k_sort_pass per 8-bit "
                             "digit, k_reorder; same state, same K, bit-identical results"}
        sim.set_binning(bin_req)
    clock_rec = clocks.stop()

    # ---- roofline of the dominant kernel: algorithmic bytes per launch / CUDA-event time -------
    peak, peak_src = measured_peak()
    r2 = int(np.floor(w.radius * w.radius))
    R = int(np.floor(w.radius))
    n_stencil = sum(1 for dz in range(-R, R + 1) for dy in range(-R, R + 1) for dx in range(-R, R + 1)
                    if dx * dx + dy * dy + dz * dz <= r2)
    extra = {}
    if ktimes is not None:
        step_bytes, bm, launches_of, survey = bytes_model(w, n_avg, active, n_stencil, count_mode)
        per_step_ms = {k: v / K for k, v in ktimes.items()}
        kernel_name = {"diffuse": "k_diffuse_chunked" if count_mode else "k_diffuse", "sort": "k_sort_pass", "reorder": "k_reorder", "sense": "k_sense",
                       "scan": "k_cell_scan2", "place": "k_place", "settle": "k_settle"}
        dom = max(bm.keys(), key=lambda k: per_step_ms[k])
        per_launch_ms = per_step_ms[dom] / launches_of[dom]
        own_bytes = bm[dom] / launches_of[dom]
        # `achieved` / `frac` follow SURVEY.md §8(d): the METHOD's bytes for this phase (P1: 17 read + 17 written + 4 key
        # = 38 B per particle, whatever this kernel's own layout moves); `frac_own_bytes` uses what the kernel itself
        # must move (P1 of count binning writes a 16 B record + an 8 B {key, arrival rank} word and issues
        # one 4 B counting atomic = 45 B)
        per_launch_bytes = survey[dom] / launches_of[dom]
        achieved = per_launch_bytes / (per_launch_ms * 1e-3) / 1e9
        roof = {"bound": "hbm", "kernel": kernel_name[dom], "achieved": achieved, "peak": peak, "unit": "GB/s",
                "frac": achieved / peak, "traffic": TRAFFIC_NCU.get((w.name, kernel_name[dom])),
                "peak_source": peak_src, "launches_per_step": launches_of[dom],
                "algorithmic_bytes_per_launch": per_launch_bytes, "ms_per_launch": per_launch_ms,
                "bytes_convention": "SURVEY.md 8(d) per-phase bytes of the method",
                "frac_own_bytes": own_bytes / (per_launch_ms * 1e-3) / 1e9 / peak, "own_bytes_per_launch": own_bytes,
                "share_of_step": per_step_ms[dom] / max(sum(per_step_ms.values()), 1e-12)}
        step_ms = ms / K
        step_gbs = step_bytes / (step_ms * 1e-3) / 1e9
        moved = sum(bm.values())     # what the kernels of the benchmarked binning mode must move themselves
        dram = STEP_TRAFFIC_NCU.get((w.name, "count" if count_mode else "radix"))
        extra["roofline_step"] = {
            "achieved": step_gbs, "unit": "GB/s", "frac_of_measured_copy": step_gbs / peak,
            "frac_of_nominal_8TBs": step_gbs / NOMINAL_GBS,
            "algorithmic_bytes_per_particle": step_bytes / max(n_avg, 1),
            "bytes_convention": "SURVEY.md 8(d): bytes of the METHOD (K1 38 + 3-pass sort 44 + reorder 42 B per particle "
                                "+ 8 B per cell + cones), whatever the binning mode moves",
            "own_bytes_per_particle": moved / max(n_avg, 1),
            "frac_own_bytes_of_measured_copy": moved / (step_ms * 1e-3) / 1e9 / peak,
            "frac_own_bytes_of_nominal_8TBs": moved / (step_ms * 1e-3) / 1e9 / NOMINAL_GBS,
            "dram_bytes_per_step_ncu": dram,
            "frac_dram_of_measured_copy": None if dram is None else dram / (step_ms * 1e-3) / 1e9 / peak,
            "frac_dram_of_nominal_8TBs": None if dram is None else dram / (step_ms * 1e-3) / 1e9 / NOMINAL_GBS,
            "dram_note": "dram__bytes_read+write summed over one step's kernels in the committed ncu capture (profiles/); "
                         "below the algorithmic bytes where the 126 MB L2 holds the per-cell arrays"}
        extra["materialised"] = (
            "count binning: the sorted SoA and the prefix array cell_lo are written every step; KEYS_SORTED / PERM and "
            "cellStart / cellEnd are derived on read (axg_read_state), bit-identical to the radix path that stores them"
            if count_mode else "radix binning: sorted keys, permutation, sorted SoA and cell_lo are written every step")
        extra["kernels_ms_per_step"] = {k: round(v, 5) for k, v in per_step_ms.items() if v > 0}
        extra["kernels_gbs"] = {k: bm[k] / (per_step_ms[k] * 1e-3) / 1e9 for k in bm if per_step_ms[k] > 0}
        extra["cone_steps_per_s"] = active / (step_ms * 1e-3)
        extra["binning"] = "count" if count_mode else "radix"
        if radix_rec:
            extra["radix"] = radix_rec

    # ---- e2e: the same job through the C-ABI with HOST buffers; every host<->device copy inside the timed region --
    # upload of the particle SoA + cone state from pinned host memory, then e2e_steps x [axg_step(1), read back cone
    # positions + states + counters], then download of the particle SoA (what a caller who keeps the state on the
    # host between jobs does).  Bytes are counted from the arrays copied.
    names = ("X", "Y", "Z", "SPECIES", "ID")
    dts = (np.float32, np.float32, np.float32, np.uint8, np.uint32)
    n_now = sim.counters()["n_live"]
    host_cols = [pinned(n_now, d) for d in dts]
    for nm, hc in zip(names, host_cols):
        sim.read_state("PART_" + nm, out=hc)
    cone_pos = pinned(len(w.neurons) * 3, np.float32)
    cone_hd = pinned(len(w.neurons) * 3, np.float32)
    cone_state = pinned(len(w.neurons), np.uint8)
    poly_len = pinned(len(w.neurons), np.uint32)
    cdict = sim.counters()
    if len(w.neurons):
        sim.read_state("CONE_POS", out=cone_pos)
        sim.read_state("CONE_HEADING", out=cone_hd)
        sim.read_state("CONE_STATE", out=cone_state)
        sim.read_state("POLY_LEN", out=poly_len)
    out_cols = [pinned(n_now + (e2e_steps + 1) * w.emitted_per_step + 64, d) for d in dts]
    counters_host = pinned(16, np.uint64)
    h2d = d2h = 0
    e2e_psteps = 0

    def e2e_job():
        nonlocal h2d, d2h, e2e_psteps
        sim.load_particles(*host_cols, next_id=cdict["next_id"], step=cdict["step"])
        h2d += sum(c.nbytes for c in host_cols)
        if len(w.neurons):
            sim.load_cones(cone_pos, cone_hd, cone_state, poly_len)
            h2d += cone_pos.nbytes + cone_hd.nbytes + cone_state.nbytes + poly_len.nbytes
        for _ in range(e2e_steps):
            step(1)
            e2e_psteps += sim.last_step_stats()["particle_steps"]
            if len(w.neurons):
                sim.read_state("CONE_POS", out=cone_pos)
                sim.read_state("CONE_STATE", out=cone_state)
                d2h += cone_pos.nbytes + cone_state.nbytes
            sim.read_state("COUNTERS", out=counters_host)
            d2h += counters_host.nbytes
        for nm, oc in zip(names, out_cols):
            d2h += sim.read_state("PART_" + nm, out=oc).nbytes

    e2e_ms = timed(e2e_job)
    e2e_value = total(e2e_psteps) / (e2e_ms * 1e-3)
    e2e = {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": h2d / e2e_steps, "d2h_bytes_per_step": d2h / e2e_steps,
           "steps": e2e_steps, "ms_per_step": e2e_ms / e2e_steps,
           "what": "load_particles+load_cones from pinned host SoA, %d x [axg_step(1), read cone pos/state + counters], "
                   "read back the particle SoA; all inside the timed region" % e2e_steps}

    # ---- cpu_baseline: the oracle as it stands, on this box's host cores, bounded sample (rank 0, N = 1 only) ------
    cpu = None
    if world == 1 and not args.no_cpu_baseline:
        budget = float(os.environ.get("AXG_CPU_BASELINE_BUDGET_S", "15"))
        cpu_steps = 3
        n_cpu = oracle_sample_size(w, budget, cpu_steps)
        v, secs, ps = time_oracle(w, n_cpu, cpu_steps, 0)
        cpu = {"value": v, "unit": UNIT, "cores": 1, "kind": "oracle", "host_cores_on_box": os.cpu_count(),
               "sample": "%d steps of %s with %d of its ~%d particles (synthetic steady-state-shaped population, all "
                         "%d cones, grid sensing), %.1f s" % (cpu_steps, w.name, n_cpu, w.nominal_live,
                                                              len(w.neurons), secs)}

    if rank == 0:
        line = {
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": K, "warmup": Wm,
            "ms_per_step": ms / K, "higher_is_better": True,
            "scaling": args.scaling if world > 1 else "weak",
            "vs_baseline": None, "dtype": "f32+u32", "data": "synthetic",
            "config": {"workload": w.name, "grid": list(w.grid), "cones": int(len(w.neurons)),
                       "sources": len(w.sources), "n_live_start": int(n_start), "n_live_end": int(n_end),
                       "l2": "inputs larger than L2 (particle SoA + sort buffers = %.0f MB per step)" % (
                           (2 * 17 + 20) * n_end / 1e6),
                       "parallelism": "shard-by-source x%d + int all-reduce" % world if world > 1 else "1 GPU",
                       "prerun": "coarse-time x%d + 100 relax steps" % args.coarse, "steering": args.steering,
                       "sensing": args.sensing, "key_order": args.key_order},
            "clocks": clock_rec, "e2e": e2e, "gpu_launches": launches, "roofline": roof, "cpu_baseline": cpu,
            "cones": {k: cnt[k] for k in ("active", "arrived", "exited")},
        }
        line.update(extra)
        print(json.dumps(line), flush=True)
    sim.close()
    if world > 1:
        dist.destroy_process_group()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=200)
    ap.add_argument("--warmup", type=int, default=20)
    ap.add_argument("--workload", default=os.environ.get("AXG_WORKLOAD", "C3"))
    ap.add_argument("--impl", default="ours", choices=("ours", "reference"))
    ap.add_argument("--coarse", type=int, default=16, help="coarse-time factor of the steady-state pre-run")
    ap.add_argument("--e2e-steps", type=int, default=20)
    ap.add_argument("--binning", default="auto", choices=("auto", "radix", "count"))
    ap.add_argument("--steering", default="vector", choices=("vector", "snr"),
                    help="P4 rule: north_star's vector addition, or the paper's fixed turn by the sign of N(SNR, 1)")
    ap.add_argument("--key-order", default="linear", choices=("linear", "brick", "morton"),
                    help="cell key: north_star's linear id, bricks of 8 x 4 x 4 cells, or the Z-order curve (axg_set_key_order)")
    ap.add_argument("--sensing", default="cell", choices=("cell", "particle", "weighted"),
                    help="P3 rule: north_star's per-cell sums, or the per-particle rule of the paper's section 5.3")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--scaling", default="strong", choices=("strong", "weak"),
                    help="N > 1: shard the fixed workload (strong), or give every rank one config's worth of sources (weak)")
    ap.add_argument("--force-sharded-loop", action="store_true",
                    help="run the multi-GPU step loop (sharded.ShardedStepper) also at N = 1, to time it against axg_step")
    ap.add_argument("--no-radix-record", action="store_true",
                    help="skip the `radix` sub-record (the same K steps under AXG_BIN_RADIX)")
    args = ap.parse_args()
    from paper_1405_3331_b200 import workloads as W
    w = W.BY_NAME[args.workload]()
    world = int(os.environ.get("WORLD_SIZE", "1"))
    if args.scaling == "weak" and world > 1:
        # per-rank work fixed: `world` times the sources; max_particles is a PER-RANK capacity, so it stays
        w = W.weak_scaled(w, world)
    if args.impl == "reference":
        if int(os.environ.get("RANK", "0")) == 0:
            run_reference(args, w)
        return
    run_ours(args, w)


if __name__ == "__main__":
    main()
