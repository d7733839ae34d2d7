#!/usr/bin/env python
"""bench.py — particle-steps/s of the GLISSE hot path on B200 (BASELINE.json metric), one JSON line.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload 1m_x4|c2|c3|c4|c5]
                    [--impl glisse|reference] [--no-extras] [--ablations]

A "step" is one pass of the whole hot path over one chunk: the planet-history kernel writes
CHUNK = 1,024 integrator steps of planet positions (one chunk ahead, on its own stream), the
particle kernel advances every active particle through those 1,024 steps (as eight chained launches
of 128 steps), and the survivor compaction runs.
Default workload: BASELINE.json north_star's target, 1,048,576 particles x 4 planets; the
BASELINE.json configs[1..4] (c2, c3, c4, c5) are measured in the same run and reported under
"workloads", each with its own roofline figures.

value   = particle-steps actually integrated (sum over steps of the active count) per second, state
          resident in HBM, device time from CUDA events on the launching stream, max over ranks.
e2e     = the same metric through the C ABI with HOST buffers: every step does glisse_create (H2D of
          the particle state from pinned memory), glisse_advance(1,024), glisse_read (D2H) and
          glisse_destroy, wall clock.
roofline= FP64-ALU bound.  `achieved` / `frac` use the ALGORITHMIC flops per particle-step (SURVEY.md
          §8(d): 410 at N_p = 4, the defined step with the two Newton updates its convergence needs) x
          particle-steps per chunk / the particle kernel's time per chunk, against the nominal FP64 FMA
          rate (148 SMs x 64 lanes x 2 x 1.965 GHz).  `executed_frac` is the same with the flops the
          kernel really issues, taken from THAT workload's ncu counters (profiles/, named in the line):
          it is the hardware utilisation; `frac` is the useful-work rate.
cpu_baseline            the oracle as it stands, one thread, bounded sample of the same workload.
cpu_baseline_all_cores  T independent copies of it over disjoint slices on all host cores.
--impl reference times the oracle (oracle/, plain single-threaded C++) on a bounded sample.
--ablations runs the measurement ablations of SURVEY.md §8(d) instead and prints them as one JSON line.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import tempfile
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

from paper_2011_03484_b200 import inputs  # noqa: E402

CHUNK = 1024                     # BASELINE.json configs[1]: "planet-history chunk K = 1024 steps"
METRIC = "particle-steps/sec (fp64, 1 B200)"
UNIT = "particle-steps/s"
L2_FLUSH_BYTES = 256 << 20       # > 126 MB L2

# ALGORITHMIC fp64 flops per particle-step (DFMA = 2, DADD/DMUL = 1; compares, MUFU seeds and
# integer work = 0): SURVEY.md §8(d)'s figure for the method as the paper defines it with the two
# Newton updates its convergence needs on these workloads — ~410 at N_p = 4, +25 per further planet
# (DESIGN.md §7 restates the count).  The roofline's `achieved` uses this figure.
ALGO_FLOPS_NP4 = 410.0
FLOPS_PER_PLANET = 25.0
# EXECUTED flops per particle-step of the particle kernel and its DRAM traffic per launch, per workload,
# from that workload's own ncu capture (2 DFMA + DMUL + DADD thread-instructions / thread-steps;
# dram__bytes_read.sum + dram__bytes_write.sum): (flops, bytes per launch, profile it was read from).
#   flops per thread-step = (2 DFMA + DMUL + DADD of a launch) / (grid x 32 threads x 128 steps of the launch):
#   1m_x4 3.594e10 / (31670 x 32 x 128), c2 4.497e9 / (3961 x ...), c3 9.291e9 / (8192 x ...),
#   c4 4.973e10 / (32492 x ...), c5 1.385e11 / (116554 x ...) (iteration binning on: the default there)
NCU = {
    "1m_x4": (277.1, 5.51e7, "profiles/r02b_particle_kernel_1m_x4.md"),
    "c2": (277.2, 6.68e6, "profiles/r02b_particle_kernel_c2.md"),
    "c3": (276.9, 1.37e7, "profiles/r02b_particle_kernel_c3.md"),
    "c4": (373.6, 5.54e7, "profiles/r02b_particle_kernel_c4.md"),
    "c5": (290.2, 3.36e8, "profiles/r02b_particle_kernel_c5.md"),
}
# FP64 peak: ncu reports sm__sass_thread_inst_executed_op_dfma_pred_on.sum.peak_sustained = 64 per SM
# per cycle; x 148 SMs x 2 flops x 1.965 GHz (clocks.max.sm of B200_PROFILING.md)
FP64_NOMINAL_TFLOPS = 148 * 64 * 2 * 1.965e9 / 1e12


def algo_flops(n_planets: int) -> float:
    return ALGO_FLOPS_NP4 + FLOPS_PER_PLANET * (n_planets - 4)


WORKLOADS = {
    "1m_x4": ("north_star target: 1,048,576 particles x 4 planets (4 giants, a~U[20,28], dt=180 d, K=1024)",
              lambda n: inputs.one_m_four_planets(n or 1_048_576)),
    "c2": ("BASELINE.json configs[1]: 4 giants, 131,072 particles a~U[20,28], dt=180 d, K=1024", lambda n: inputs.config(2, n)),
    "c3": ("BASELINE.json configs[2]: 4 giants, 262,144 particles a~U[53,65], e<0.4", lambda n: inputs.config(3, n)),
    "c4": ("BASELINE.json configs[3]: 8 planets, 1,048,576 particles, dt=4 d", lambda n: inputs.config(4, n)),
    "c5": ("BASELINE.json configs[4]: 4 giants, 4,194,304 planet-crossing particles", lambda n: inputs.config(5, n)),
}


def make_workload(name: str, world: int = 1, rank: int = 0):
    """The workload of one rank.  Weak scaling: world x N particles are drawn from the same seeded
    distribution and rank r takes its contiguous slice (particles never interact, PAPER.md:27, 35:
    planets replicated, particles partitioned, no exchange)."""
    desc, fn = WORKLOADS[name]
    w = fn(None)
    if world > 1:
        n = w.n_particles
        big = fn(n * world)
        lo, hi = inputs.shard_range(n * world, rank, world)
        import dataclasses
        w = dataclasses.replace(big, pos=np.ascontiguousarray(big.pos[:, lo:hi]),
                                vel=np.ascontiguousarray(big.vel[:, lo:hi]))
    return desc, w


def reduce_over_ranks(local_ms: float, local_units: float, dist=None):
    """Whole-job figures: time = max over ranks, units = sum over ranks (no data-path collective;
    these two scalars are the only thing exchanged)."""
    if dist is None or not dist.is_initialized() or dist.get_world_size() == 1:
        return local_ms, local_units
    import torch
    dev = "cuda" if dist.get_backend() == "nccl" else "cpu"
    t = torch.tensor([local_ms], dtype=torch.float64, device=dev)
    u = torch.tensor([local_units], dtype=torch.float64, device=dev)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    dist.all_reduce(u, op=dist.ReduceOp.SUM)
    return float(t.item()), float(u.item())


def _rank_entry(rank: int, world: int, port: int, fn, argv):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), LOCAL_RANK=str(rank),
                      WORLD_SIZE=str(world))
    fn(argv)


def launch_ranks(world: int, fn, argv, port: int | None = None):
    """`python bench.py --gpus N` without torchrun: start the N ranks here (one process per GPU, spawn),
    each with RANK / LOCAL_RANK / WORLD_SIZE / MASTER_* set as torchrun would; `fn(argv)` is the rank's
    main.  Returns when every rank has exited; raises if one failed."""
    import torch.multiprocessing as mp
    port = port or (29500 + os.getpid() % 2000)
    mp.spawn(_rank_entry, args=(world, port, fn, argv), nprocs=world, join=True)


class ClockSampler:
    """Samples SM clock and throttle reasons through NVML during the timed region."""

    def __init__(self, index: int):
        self.samples, self.reasons, self.max_mhz = [], set(), None
        self._stop = threading.Event()
        self._thread = None
        try:
            import pynvml
            pynvml.nvmlInit()
            self._nv = pynvml
            self._h = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.max_mhz = pynvml.nvmlDeviceGetMaxClockInfo(self._h, pynvml.NVML_CLOCK_SM)
        except Exception:
            self._nv = None

    def _run(self):
        nv = self._nv
        names = {"hw_slowdown": nv.nvmlClocksThrottleReasonHwSlowdown,
                 "hw_thermal_slowdown": nv.nvmlClocksThrottleReasonHwThermalSlowdown,
                 "sw_thermal_slowdown": nv.nvmlClocksThrottleReasonSwThermalSlowdown,
                 "sw_power_cap": nv.nvmlClocksThrottleReasonSwPowerCap}
        while not self._stop.is_set():
            try:
                self.samples.append(nv.nvmlDeviceGetClockInfo(self._h, nv.NVML_CLOCK_SM))
                mask = nv.nvmlDeviceGetCurrentClocksThrottleReasons(self._h)
                for k, bit in names.items():
                    if mask & bit:
                        self.reasons.add(k)
            except Exception:
                pass
            self._stop.wait(0.02)

    def __enter__(self):
        if self._nv is not None:
            self._thread = threading.Thread(target=self._run, daemon=True)
            self._thread.start()
        return self

    def __exit__(self, *exc):
        self._stop.set()
        if self._thread:
            self._thread.join()

    def summary(self):
        return {"sm_mhz": float(np.median(self.samples)) if self.samples else None,
                "sm_max_mhz": self.max_mhz, "reasons": sorted(self.reasons), "samples": len(self.samples)}


def _visible_index(local_rank: int) -> int:
    vis = os.environ.get("CUDA_VISIBLE_DEVICES")
    if vis:
        try:
            return int(vis.split(",")[local_rank])
        except Exception:
            return local_rank
    return local_rank


def time_resident(binding, torch, w, steps, warmup, device, flush, chunks_per_step=1, **simkw):
    """`steps` timed steps of `chunks_per_step` chunks each with the state resident in HBM (L2 flushed
    between timed steps when `flush` is given); returns per-rank totals."""
    stream = torch.cuda.Stream(device=device)
    simkw.setdefault("chunk_steps", CHUNK)
    simkw.setdefault("resync_chunks", 1)
    K = simkw["chunk_steps"]
    sim = binding.GlisseSim.from_workload(w, device=device.index, stream=stream.cuda_stream, **simkw)
    with torch.cuda.stream(stream):
        for _ in range(warmup):
            sim.advance(K * chunks_per_step)
        sim.sync()
        sim.particle_kernel_time()
        ps0, l0 = sim.particle_steps(), sim.launch_count()
        ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(steps)]
        torch.cuda.synchronize(device)
        for a, b in ev:
            if flush is not None:
                flush.zero_()            # L2 flush between timed iterations (not timed)
            a.record(stream)
            sim.advance(K * chunks_per_step)
            b.record(stream)
        torch.cuda.synchronize(device)
        sim.sync()
    ms = sum(a.elapsed_time(b) for a, b in ev)
    kms, kruns = sim.particle_kernel_time()
    ps1, l1 = sim.particle_steps(), sim.launch_count()
    active = sim.active_count()
    sim.close()
    return dict(ms=ms, psteps=ps1 - ps0, launches=l1 - l0, kernel_ms=kms, kernel_runs=kruns, active=active)


def roofline_of(name: str, n_planets: int, res: dict, peak_probe: float) -> dict:
    """Roofline record of the particle kernel from one time_resident result.  The launches of a chunk
    overlap by design (launch chaining), so the kernel is timed per chunk: one pair of CUDA events
    around the chunk's launches on the launching stream (glisse_particle_kernel_time)."""
    fl = algo_flops(n_planets)
    ex, traffic, prof = NCU.get(name, (None, None, None))
    runs = max(res["kernel_runs"], 1)
    k_ms = res["kernel_ms"] / runs
    achieved = fl * (res["psteps"] / runs) / (k_ms * 1e-3) / 1e12
    r = {"bound": "alu", "achieved": achieved, "peak": FP64_NOMINAL_TFLOPS, "unit": "TFLOP/s",
         "frac": achieved / FP64_NOMINAL_TFLOPS, "traffic": traffic,
         "kernel": "particle_kernel (8 chained launches of 128 steps per chunk, timed together)",
         "kernel_ms_per_chunk": k_ms, "kernel_share_of_step": res["kernel_ms"] / res["ms"],
         "flops_per_particle_step": fl,
         "flops_source": "algorithmic: SURVEY.md 8(d) / DESIGN.md 7 count of the defined step with 2 Newton updates",
         "peak_source": "nominal FP64 FMA rate: 148 SMs x 64 DFMA lanes (ncu peak_sustained) x 2 x 1.965 GHz; "
                        "MEASURED_PEAKS.json has no FP64 figure",
         "probe_tflops": peak_probe / 1e12, "frac_of_probe": achieved / (peak_probe / 1e12),
         "probe": "glisse_fp64_peak_probe: register-resident DFMA chains timed in this run"}
    if ex is not None:
        r.update({"executed_flops_per_particle_step": ex, "executed_tflops": achieved * ex / fl,
                  "executed_frac": achieved * ex / fl / FP64_NOMINAL_TFLOPS, "executed_source": prof,
                  "traffic_source": prof})
    return r


def time_e2e(binding, torch, w, steps, warmup, device):
    """The same chunk through the C ABI with HOST buffers: glisse_run = create (H2D) + advance + read (D2H) +
    destroy, pipelined by the library over slices of the particles (automatic part count)."""
    n = w.n_particles
    pos = torch.from_numpy(w.pos).pin_memory()
    vel = torch.from_numpy(w.vel).pin_memory()
    out = (torch.empty((3, n), dtype=torch.float64).pin_memory(), torch.empty((3, n), dtype=torch.float64).pin_memory(),
           torch.empty(n, dtype=torch.int32).pin_memory(), torch.empty(n, dtype=torch.int64).pin_memory())
    out_np = tuple(t.numpy() for t in out)
    import dataclasses
    wp = dataclasses.replace(w, pos=pos.numpy(), vel=vel.numpy())
    total, psteps = 0.0, 0
    for it in range(warmup + steps):
        torch.cuda.synchronize(device)
        t0 = time.perf_counter()
        _, _, flag, rstep, ps = binding.run(wp, CHUNK, 0, out=out_np, chunk_steps=CHUNK, resync_chunks=1,
                                            device=device.index)
        t1 = time.perf_counter()
        if it >= warmup:
            total += t1 - t0
            # particle-steps of this round trip, rebuilt from what was read back (the result of the step)
            rebuilt = int(np.where(rstep < 0, CHUNK, rstep + ((flag == 3) | (flag == 4))).sum())
            assert rebuilt == ps, (rebuilt, ps)
            psteps += rebuilt
    h2d = 6 * 8 * n + int(w.gm_planet.nbytes + w.planet_pos.nbytes + w.planet_vel.nbytes + w.planet_rcrit.nbytes)
    d2h = (6 * 8 + 4 + 8) * n
    return dict(seconds=total, psteps=psteps, h2d=h2d, d2h=d2h)


# ---- the oracle on the host cores ---------------------------------------------------------------------
def oracle_rate(w, n_particles, n_steps):
    """The oracle as it stands, single-threaded, on the first n_particles of the workload."""
    import oracle
    ws = w.subset(min(n_particles, w.n_particles))
    S = oracle.OracleSim.from_workload(ws)
    t0 = time.perf_counter()
    S.advance(n_steps)
    dt = time.perf_counter() - t0
    ps = S.particle_steps()
    S.close()
    return ps / dt, dt, ps


def _oracle_worker(path: str, lo: int, hi: int, n_steps: int):
    """One of the T copies: the oracle on particles [lo, hi) of the sample stored at `path`."""
    import oracle
    d = np.load(path)
    S = oracle.OracleSim(float(d["gm_star"]), d["gm_planet"], d["planet_pos"], d["planet_vel"], d["planet_rcrit"],
                         np.ascontiguousarray(d["pos"][:, lo:hi]), np.ascontiguousarray(d["vel"][:, lo:hi]),
                         float(d["dt"]), r_min=float(d["r_min"]), r_max=float(d["r_max"]))
    t0 = time.perf_counter()
    S.advance(n_steps)
    dt = time.perf_counter() - t0
    print(json.dumps({"ps": S.particle_steps(), "seconds": dt}))


def oracle_rate_all_cores(w, per_core_particles, n_steps):
    """T independent copies of the oracle over disjoint slices of the workload's first T x m particles,
    one process per host core (particles are independent, so this is what an embarrassingly parallel
    run of the same program does).  Rate = total particle-steps / the slowest copy's time."""
    import oracle
    oracle.build()
    cores = len(os.sched_getaffinity(0)) if hasattr(os, "sched_getaffinity") else (os.cpu_count() or 1)
    m = per_core_particles
    T = max(1, min(cores, w.n_particles // m))
    ws = w.subset(T * m)
    with tempfile.TemporaryDirectory() as td:
        path = os.path.join(td, "sample.npz")
        np.savez(path, gm_star=ws.gm_star, gm_planet=ws.gm_planet, planet_pos=ws.planet_pos, planet_vel=ws.planet_vel,
                 planet_rcrit=ws.planet_rcrit, pos=ws.pos, vel=ws.vel, dt=ws.dt, r_min=ws.r_min, r_max=ws.r_max)
        procs = [subprocess.Popen([sys.executable, os.path.abspath(__file__), "--oracle-worker", path, str(i * m),
                                   str((i + 1) * m), str(n_steps)], stdout=subprocess.PIPE, text=True, cwd=ROOT)
                 for i in range(T)]
        outs = [json.loads(p.communicate()[0].strip().splitlines()[-1]) for p in procs]
    ps = sum(o["ps"] for o in outs)
    slowest = max(o["seconds"] for o in outs)
    model = ""
    try:
        for line in open("/proc/cpuinfo"):
            if line.startswith("model name"):
                model = line.split(":", 1)[1].strip()
                break
    except OSError:
        pass
    return ps / slowest, slowest, ps, T, model


def run_reference(args):
    """--impl reference: the oracle on the host cores, same config/metric, bounded sample per step."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    desc, w = make_workload(args.workload)
    sample_n = 4096
    import oracle
    ws = w.subset(sample_n)
    S = oracle.OracleSim.from_workload(ws)
    for _ in range(args.warmup):
        S.advance(CHUNK)
    ps0 = S.particle_steps()
    t0 = time.perf_counter()
    for _ in range(args.steps):
        S.advance(CHUNK)
    dt = time.perf_counter() - t0
    ps = S.particle_steps() - ps0
    S.close()
    value = ps / dt
    sample = f"first {sample_n} particles of the workload x {CHUNK} integrator steps per bench step, 1 thread"
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * dt / args.steps,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": desc, "n_particles": w.n_particles, "n_planets": w.n_planets, "chunk_steps": CHUNK,
                   "dt_days": w.dt, "sampled_particles": sample_n},
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": 1, "kind": "oracle", "sample": sample},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }))


# ---- measurement ablations --------------------------------------------------------
def run_ablations(binding, torch, device, flush):
    """K sweep (the paper's Fig. 3), resync on / off on config 5,
    the definition's fixed-count Newton path against the fast solver, launch-chain segment length,
    iteration binning on config 5, periodic output overhead, streamed host planet log."""
    out = {}
    _, c2 = make_workload("c2")

    def rate(w, steps=6, warmup=3, fl=flush, **kw):
        r = time_resident(binding, torch, w, steps, warmup, device, fl, **kw)
        return {"value": r["psteps"] / (r["ms"] * 1e-3), "ms_per_step": r["ms"] / steps,
                "kernel_ms_per_chunk": r["kernel_ms"] / max(r["kernel_runs"], 1), "active_end": r["active"]}

    # K sweep at N = 131,072: a timed step is 1,024 integrator steps in chunks of K (1,024 / K launches
    # of the whole path), so the rows are directly comparable
    out["chunk_size_K"] = {}
    for K in (1, 8, 32, 128, 1024):
        out["chunk_size_K"][str(K)] = rate(c2, steps=3 if K < 8 else 5, chunk_steps=K, chunks_per_step=CHUNK // K)
    # launch chaining: segment length at K = 1024 (0 = one launch per chunk, the round-1 schedule)
    out["segment_steps"] = {}
    for name in ("c2", "1m_x4"):
        _, w = make_workload(name)
        out["segment_steps"][name] = {str(sg): rate(w, segment_steps=sg) for sg in (0, 512, 256, 128, 64)}
    # the same without the L2 flush and 16 chunks per timed step (a long glisse_advance)
    out["long_advance_16_chunks_no_flush"] = {}
    for name in ("c2", "1m_x4"):
        _, w = make_workload(name)
        out["long_advance_16_chunks_no_flush"][name] = {
            str(sg): rate(w, steps=2, warmup=1, fl=None, chunks_per_step=16, segment_steps=sg) for sg in (0, 128)}
    # fixed-count Newton of the definition (kepler_iters = 4 switches the fast solver off) vs the fast solver
    out["kepler_solver"] = {"fast_solver_iters5": rate(c2), "definition_newton_iters4": rate(c2, kepler_iters=4)}
    # config 5: resync on / off, binning on / off, after 8 warm-up chunks (about 20 % removed)
    _, c5 = make_workload("c5")
    out["config5"] = {
        "resync_every_chunk": rate(c5, steps=4, warmup=8, bin_iterations=0),
        "resync_off": rate(c5, steps=4, warmup=8, resync_chunks=0, bin_iterations=0),
        "resync_every_chunk_binned": rate(c5, steps=4, warmup=8, bin_iterations=1),
    }
    # a quiet population with a few planet-crossing bodies mixed in: without the ordering every warp that
    # holds one of them pays for it at every step
    import dataclasses
    _, w1 = make_workload("1m_x4")
    rng = np.random.default_rng(5)
    pick = rng.uniform(size=w1.pos.shape[1])
    out["mixed_population_1m_x4"] = {}
    for frac in (0.0, 0.01, 0.03):
        pos, vel = w1.pos.copy(), w1.vel.copy()
        m = pick < frac
        pos[:, m], vel[:, m] = c5.pos[:, :pos.shape[1]][:, m], c5.vel[:, :pos.shape[1]][:, m]
        wm = dataclasses.replace(w1, pos=pos, vel=vel)
        out["mixed_population_1m_x4"][f"{frac:.2f}"] = {
            "particle_id_order": rate(wm, steps=4, warmup=3, bin_iterations=0)["value"],
            "ordered_by_hardness": rate(wm, steps=4, warmup=3, bin_iterations=1)["value"]}
    # the drift-kick-drift splitting (BASELINE.json's wording; two half drifts per step) against kick-drift-kick
    out["scheme_1m_x4"] = {"kdk": rate(w1, steps=4, warmup=3)["value"], "dkd": rate(w1, steps=4, warmup=3, scheme="dkd")["value"]}
    # mean fast-solver iterations per warp-step with and without binning (instrumented kernel)
    for binned in (0, 1):
        sim = binding.GlisseSim.from_workload(c5, chunk_steps=CHUNK, bin_iterations=binned, device=device.index)
        sim.advance(8 * CHUNK)
        sim.solver_stats_enable(True)
        sim.advance(CHUNK)
        calls, iters, slow = sim.solver_stats()
        sim.close()
        out["config5"]["binned" if binned else "unbinned"] = {
            "mean_fast_iters_per_warp_step": iters / calls, "slow_path_fraction": slow / calls, "warp_steps": calls}
    # periodic output: elements snapshot into a pinned ring + resonance sample after EVERY chunk
    n = c2.n_particles
    ring = (torch.empty((4, 6, n), dtype=torch.float64).pin_memory(), torch.empty((4, n), dtype=torch.int32).pin_memory(),
            torch.empty((4, n), dtype=torch.int64).pin_memory(), torch.empty(4, dtype=torch.int64).pin_memory())
    for label, kw in (("off", {}), ("snapshot_every_chunk", dict(snapshot_chunks=1)),
                      ("resonance_every_chunk", dict(resonance_chunks=1)),
                      ("snapshot_and_resonance_every_chunk", dict(snapshot_chunks=1, resonance_chunks=1))):
        stream = torch.cuda.Stream(device=device)
        sim = binding.GlisseSim.from_workload(c2, chunk_steps=CHUNK, device=device.index, stream=stream.cuda_stream, **kw)
        if "snapshot_chunks" in kw:
            sim.snapshot_ring("elements", 4, *(t.numpy() for t in ring))
        if "resonance_chunks" in kw:
            sim.resonance_begin(3, 3, 1, np.deg2rad(10.0))
        with torch.cuda.stream(stream):
            sim.advance(3 * CHUNK)
            sim.sync()
            a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            ps0 = sim.particle_steps()
            a.record(stream)
            sim.advance(16 * CHUNK)
            b.record(stream)
            sim.sync()
            sim.snapshot_wait()
        ms = a.elapsed_time(b)
        out.setdefault("periodic_output_c2_16_chunks", {})[label] = {
            "value": (sim.particle_steps() - ps0) / (ms * 1e-3), "ms_per_chunk": ms / 16}
        sim.close()
    # particle-count sweep (BASELINE.json configs[4]: "Also sweep particle count over 2^10 to 2^22"): config
    # 5's planet-crossing distribution, compaction every chunk, wall clock per chunk after 2 warm-up chunks
    out["particle_count_sweep_config5"] = {}
    for lg in range(10, 23):
        n = 1 << lg
        wn = inputs.config(5, n)
        sim = binding.GlisseSim.from_workload(wn, chunk_steps=CHUNK, resync_chunks=1, device=device.index)
        sim.advance(2 * CHUNK)
        sim.sync()
        sim.particle_kernel_time()
        ps0 = sim.particle_steps()
        chunks = 8 if lg < 21 else 4
        t0 = time.perf_counter()
        sim.advance(chunks * CHUNK)
        sim.sync()
        dt = time.perf_counter() - t0
        kms, kruns = sim.particle_kernel_time()
        out["particle_count_sweep_config5"][str(n)] = {
            "value": (sim.particle_steps() - ps0) / dt, "ms_per_chunk": 1e3 * dt / chunks,
            "kernel_ms_per_chunk": kms / max(kruns, 1), "active_fraction_end": sim.active_count() / n}
        sim.close()
        del wn
    # external planet history streamed from pinned host memory, 10^5 steps at N = 131,072, vs the
    # internal planet clock over the same steps
    steps = 100_000
    sim = binding.GlisseSim.from_workload(c2, chunk_steps=CHUNK, device=device.index)
    log = torch.from_numpy(sim.planet_log(steps)).pin_memory()
    for label in ("internal_planets", "host_log_streamed"):
        t0 = time.perf_counter()
        if label == "internal_planets":
            sim.advance(steps)
        else:
            sim.advance_with_log(steps, log.numpy())
        ps = sim.particle_steps()
        dt = time.perf_counter() - t0
        out.setdefault("external_log_1e5_steps_c2", {})[label] = {"value": ps / dt, "seconds": dt}
        sim.close()
        if label == "internal_planets":
            sim = binding.GlisseSim.from_workload(c2, chunk_steps=CHUNK, device=device.index)
    return out


def run_full_configs(binding, device):
    """BASELINE.json's five configurations AS STATED — every particle, every step (10^4, 10^5, 10^5, 2 x 10^4,
    5 x 10^4), K = 1,024, compaction every chunk — in one glisse_advance each: wall time, particle-steps
    (sum over steps of the active count), how many particles each removal flag took, surviving fraction."""
    out = {}
    for c in (1, 2, 3, 4, 5):
        w = inputs.config(c)
        t0 = time.perf_counter()
        sim = binding.GlisseSim.from_workload(w, chunk_steps=CHUNK, resync_chunks=1, device=device.index)
        t1 = time.perf_counter()
        sim.advance(w.steps)
        sim.sync()
        t2 = time.perf_counter()
        _, _, flag, rstep = sim.read()
        ps = sim.particle_steps()
        sim.close()
        n = int(flag.shape[0])
        flags = {str(int(k)): int(v) for k, v in zip(*np.unique(flag, return_counts=True))}
        out[f"c{c}"] = {"n_particles": n, "n_planets": w.n_planets, "steps": int(w.steps), "dt_days": float(w.dt),
                        "create_s": t1 - t0, "advance_s": t2 - t1, "particle_steps": int(ps),
                        "value": ps / (t2 - t1), "nominal_particle_steps": n * int(w.steps),
                        "surviving_fraction": float((flag == 0).mean()), "flags": flags,
                        "median_removal_step": float(np.median(rstep[flag != 0])) if (flag != 0).any() else None}
    return out


def rank_main(argv):
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="glisse", choices=["glisse", "reference"])
    ap.add_argument("--workload", default="1m_x4", choices=sorted(WORKLOADS))
    ap.add_argument("--no-extras", action="store_true",
                    help="skip e2e, the other workloads, the long-advance line and the cpu baselines")
    ap.add_argument("--ablations", action="store_true", help="run the SURVEY.md 8(d) ablations instead")
    ap.add_argument("--full-configs", action="store_true",
                    help="run BASELINE.json's five configurations as stated (all particles, all steps) instead")
    args = ap.parse_args(argv)
    if args.warmup < 3:
        args.warmup = 3
    if args.impl == "reference":
        run_reference(args)
        return

    import torch
    from paper_2011_03484_b200 import binding
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the hot path has no CPU fallback")
    rank = int(os.environ.get("RANK", "0"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    dist = None
    device = torch.device("cuda", local_rank)
    torch.cuda.set_device(device)
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=device)
    binding.lib()

    if args.full_configs:
        if rank == 0:
            print(json.dumps({"full_configs": run_full_configs(binding, device)}))
        if dist is not None:
            dist.destroy_process_group()
        return
    flush = torch.empty(L2_FLUSH_BYTES, dtype=torch.uint8, device=device)
    if args.ablations:
        if rank == 0:
            print(json.dumps({"ablations": run_ablations(binding, torch, device, flush)}))
        if dist is not None:
            dist.destroy_process_group()
        return

    desc, w = make_workload(args.workload, world, rank)
    peak = binding.fp64_peak_probe(device.index, 200.0)      # FP64 FMA rate of this GPU, FLOP/s

    if dist is not None:
        dist.barrier()
    torch.cuda.synchronize(device)
    with ClockSampler(_visible_index(local_rank)) as clk:
        res = time_resident(binding, torch, w, args.steps, args.warmup, device, flush)
    if dist is not None:
        dist.barrier()
    torch.cuda.synchronize(device)
    ms, psteps = reduce_over_ranks(res["ms"], res["psteps"], dist)
    value = psteps / (ms * 1e-3)

    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": ms / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f64", "data": "synthetic",
        "config": {"workload": desc, "n_particles_per_gpu": w.n_particles, "n_planets": w.n_planets,
                   "chunk_steps": CHUNK, "dt_days": w.dt, "resync_chunks": 1, "segment_steps": 128,
                   "step": "one chunk of 1,024 integrator steps: planet-history + particle kernel (8 chained "
                           "launches of 128 steps) + compaction",
                   "l2": "flushed between timed steps (256 MiB write, untimed)",
                   "parallelism": "particles sharded across ranks, planets replicated, no collectives"},
        "nominal_particle_steps_per_s": w.n_particles * world * CHUNK * args.steps / (ms * 1e-3),
        "active_fraction_end": res["active"] / w.n_particles,
        "gpu_launches": res["launches"],
        "roofline": roofline_of(args.workload, w.n_planets, res, peak),
        "clocks": clk.summary(),
    }

    if not args.no_extras:
        e = time_e2e(binding, torch, w, max(3, min(args.steps, 10)), 5, device)
        if dist is not None:
            dist.barrier()
        e_s, e_ps = reduce_over_ranks(e["seconds"] * 1e3, e["psteps"], dist)
        line["e2e"] = {"value": e_ps / (e_s * 1e-3), "unit": UNIT, "h2d_bytes_per_step": e["h2d"],
                       "d2h_bytes_per_step": e["d2h"],
                       "what": "per step, all inside the timed region: one glisse_run call = glisse_create from "
                               "pinned host arrays + glisse_advance(1024) + glisse_read to pinned host arrays + "
                               "glisse_destroy, pipelined by the library over slices of the particles (parts of "
                               "2^17, at most 8: uploads and downloads of the other parts behind the kernels), "
                               "wall clock"}
        if rank == 0 and world == 1:
            # a long glisse_advance: 16 chunks per timed step, no L2 flush in between (the library's
            # natural use; the per-chunk figure above drains the device before every timed chunk)
            rl = time_resident(binding, torch, w, 2, 1, device, None, chunks_per_step=16)
            line["long_advance"] = {"value": rl["psteps"] / (rl["ms"] * 1e-3), "unit": UNIT,
                                    "ms_per_chunk": rl["ms"] / 32, "what": "2 timed glisse_advance(16 x 1024) calls, "
                                    "no L2 flush between chunks, same workload"}
            # the BASELINE.json configs, same run, same method, fewer steps
            others = {}
            for name in ("c2", "c3", "c4", "c5"):
                if name == args.workload:
                    continue
                d_, wo = make_workload(name)
                n_steps = max(3, args.steps // 4)
                ro = time_resident(binding, torch, wo, n_steps, 3, device, flush)
                rf = roofline_of(name, wo.n_planets, ro, peak)
                others[name] = {"workload": d_, "value": ro["psteps"] / (ro["ms"] * 1e-3), "unit": UNIT,
                                "ms_per_step": ro["ms"] / n_steps, "steps": n_steps,
                                "kernel_ms_per_chunk": rf["kernel_ms_per_chunk"],
                                "active_fraction_end": ro["active"] / wo.n_particles,
                                "roofline": {k: rf[k] for k in ("achieved", "frac", "executed_frac", "executed_source",
                                                                "flops_per_particle_step",
                                                                "executed_flops_per_particle_step") if k in rf}}
                if name == "c2":   # the paper-sized workload end to end as well (one wave: the costliest case)
                    ec = time_e2e(binding, torch, wo, 5, 5, device)
                    others[name]["e2e"] = {"value": ec["psteps"] / ec["seconds"], "unit": UNIT,
                                           "h2d_bytes_per_step": ec["h2d"], "d2h_bytes_per_step": ec["d2h"]}
                del wo
            line["workloads"] = others
            rate, secs, ps = oracle_rate(w, 16384, 3000)
            line["cpu_baseline"] = {"value": rate, "unit": UNIT, "cores": 1, "kind": "oracle",
                                    "sample": f"first 16,384 particles x 3,000 steps of the same workload "
                                              f"({ps:.3g} particle-steps in {secs:.1f} s), single thread"}
            rate, secs, ps, T, model = oracle_rate_all_cores(w, 2048, 3000)
            line["cpu_baseline_all_cores"] = {
                "value": rate, "unit": UNIT, "cores": T, "kind": "oracle", "cpu": model,
                "sample": f"{T} independent copies of the oracle, one process per host core, each on its own "
                          f"2,048 particles of the workload's first {T * 2048:,} x 3,000 steps "
                          f"({ps:.3g} particle-steps, slowest copy {secs:.1f} s)"}
    if rank == 0:
        print(json.dumps(line))
    if dist is not None:
        dist.destroy_process_group()


def main():
    argv = sys.argv[1:]
    if argv and argv[0] == "--oracle-worker":
        _oracle_worker(argv[1], int(argv[2]), int(argv[3]), int(argv[4]))
        return
    ap = argparse.ArgumentParser(add_help=False)
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--impl", default="glisse")
    known, _ = ap.parse_known_args(argv)
    if known.gpus > 1 and "WORLD_SIZE" not in os.environ and known.impl != "reference":
        launch_ranks(known.gpus, rank_main, argv)    # one process per GPU, as torchrun would start them
        return
    rank_main(argv)


if __name__ == "__main__":
    main()
