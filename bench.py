#!/usr/bin/env python
"""bench.py — particle-steps/s of the GLISSE hot path on B200 (BASELINE.json metric), one JSON line.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload c2|1m_x4|c3|c4|c5] [--impl glisse|reference]

A "step" is one pass of the whole hot path over one chunk: the planet-history kernel writes
CHUNK = 1,024 integrator steps of planet positions (one chunk ahead, on its own stream), the
particle kernel advances every active particle through those 1,024 steps, and the survivor
compaction runs.  Default workload: BASELINE.json
configs[1] (4 giants, 131,072 particles, dt = 180 d, K = 1,024); the north_star target workload
(1M particles x 4 planets) is measured in the same run and reported under "target_1m_x4".

value   = particle-steps actually integrated (sum over steps of the active count) per second, state
          resident in HBM, device time from CUDA events on the launching stream, max over ranks.
e2e     = the same metric through the C ABI with HOST buffers: every step does glisse_create (H2D of
          the particle state from pinned memory), glisse_advance(1,024), glisse_read (D2H), destroy.
roofline= FP64-ALU bound: algorithmic flops per particle-step (410 at N_p = 4) x
          particle-steps per launch / mean particle-kernel duration, against the nominal FP64 FMA
          rate (148 SMs x 64 lanes x 2 x 1.965 GHz); the flops the kernel actually executes (ncu
          counters) and the library's measured DFMA probe are reported beside it.
--impl reference times the oracle (oracle/, plain single-threaded C++) on a bounded sample.
"""
from __future__ import annotations

import argparse
import json
import os
import sys
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
# dram__bytes_read.sum + dram__bytes_write.sum per particle-kernel launch, from the ncu --set full
# captures under profiles/ (the kernel is ALU-bound; this only shows that state traffic is negligible)
TRAFFIC_BYTES_PER_LAUNCH = {"c2": 6.9e6, "1m_x4": 5.6e7, "c4": 5.7e7}

# ALGORITHMIC fp64 flops per particle-step (DFMA = 2, DADD/DMUL = 1; compares, MUFU seeds and
# integer work = 0): SURVEY.md §8(d)'s figure for the method as the paper defines it with the two
# Newton updates its convergence needs on these workloads — ~410 at N_p = 4, +25 per further planet
# (DESIGN.md §7 restates the count).  The roofline's `achieved` uses this figure.
ALGO_FLOPS_NP4 = 410.0
# EXECUTED flops per particle-step of the current particle kernel, from its ncu instruction counters
# (profiles/*_particle_kernel_*.md, "Derived per launch"): the quartic solver and the merged
# gm/d^3 do the same step in fewer operations.  Reported beside the algorithmic figure.
EXEC_FLOPS_NP4 = 282.0
FLOPS_PER_PLANET = 25.0
# FP64 peak: ncu reports sm__sass_thread_inst_executed_op_dfma_pred_on.sum.peak_sustained = 64 per SM
# per cycle; x 148 SMs x 2 flops x 1.965 GHz (clocks.max.sm of B200_PROFILING.md)
FP64_NOMINAL_TFLOPS = 148 * 64 * 2 * 1.965e9 / 1e12


def flops_per_pstep(n_planets: int, executed: bool = False) -> float:
    return (EXEC_FLOPS_NP4 if executed else ALGO_FLOPS_NP4) + FLOPS_PER_PLANET * (n_planets - 4)

WORKLOADS = {
    "c2": ("BASELINE.json configs[1]: 4 giants, 131,072 particles a~U[20,28], dt=180 d, K=1024", lambda n: inputs.config(2, n)),
    "1m_x4": ("north_star target: 4 giants, 1,048,576 particles a~U[20,28], dt=180 d, K=1024",
              lambda n: inputs.one_m_four_planets(n or 1_048_576)),
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


def time_resident(binding, torch, w, steps, warmup, device, flush):
    """K timed chunks with the state resident in HBM; returns per-rank totals."""
    stream = torch.cuda.Stream(device=device)
    sim = binding.GlisseSim.from_workload(w, chunk_steps=CHUNK, resync_chunks=1, device=device.index,
                                          stream=stream.cuda_stream)
    with torch.cuda.stream(stream):
        for _ in range(warmup):
            sim.advance(CHUNK)
        sim.sync()
        sim.particle_kernel_time()
        ps0, l0 = sim.particle_steps(), sim.launch_count()
        ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(steps)]
        torch.cuda.synchronize(device)
        for a, b in ev:
            flush.zero_()            # L2 flush between timed iterations (not timed)
            a.record(stream)
            sim.advance(CHUNK)
            b.record(stream)
        torch.cuda.synchronize(device)
        sim.sync()
    ms = sum(a.elapsed_time(b) for a, b in ev)
    kms, klaunches = sim.particle_kernel_time()
    ps1, l1 = sim.particle_steps(), sim.launch_count()
    active = sim.active_count()
    sim.close()
    return dict(ms=ms, psteps=ps1 - ps0, launches=l1 - l0, kernel_ms=kms, kernel_launches=klaunches, active=active)


def time_e2e(binding, torch, w, steps, warmup, device):
    """The same chunk through the C ABI with HOST buffers: create (H2D) + advance + read (D2H)."""
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
        sim = binding.GlisseSim.from_workload(wp, chunk_steps=CHUNK, resync_chunks=1, device=device.index)
        sim.advance(CHUNK)
        _, _, _, rstep = sim.read(out_np)
        t1 = time.perf_counter()
        ps = sim.particle_steps()
        sim.close()
        if it >= warmup:
            total += t1 - t0
            psteps += ps
    h2d = 6 * 8 * n + int(w.gm_planet.nbytes + w.planet_pos.nbytes + w.planet_vel.nbytes + w.planet_rcrit.nbytes)
    d2h = (6 * 8 + 4 + 8) * n
    return dict(seconds=total, psteps=psteps, h2d=h2d, d2h=d2h)


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


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="glisse", choices=["glisse", "reference"])
    ap.add_argument("--workload", default="c2", choices=sorted(WORKLOADS))
    ap.add_argument("--no-extras", action="store_true", help="skip e2e, cpu_baseline and the 1M x 4 target line")
    args = ap.parse_args()
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

    desc, w = make_workload(args.workload, world, rank)
    flush = torch.empty(L2_FLUSH_BYTES, dtype=torch.uint8, device=device)
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

    # roofline of the dominant kernel (rank 0's launches)
    fl = flops_per_pstep(w.n_planets)
    k_ms = res["kernel_ms"] / max(res["kernel_launches"], 1)
    achieved = fl * (res["psteps"] / max(res["kernel_launches"], 1)) / (k_ms * 1e-3) / 1e12
    roofline = {"bound": "alu", "achieved": achieved, "peak": FP64_NOMINAL_TFLOPS, "unit": "TFLOP/s",
                "frac": achieved / FP64_NOMINAL_TFLOPS, "traffic": TRAFFIC_BYTES_PER_LAUNCH.get(args.workload),
                "kernel": "particle_kernel", "kernel_ms_per_launch": k_ms,
                "kernel_share_of_step": res["kernel_ms"] / res["ms"],
                "flops_per_particle_step": fl,
                "flops_source": "algorithmic: SURVEY.md 8(d) / DESIGN.md 7 count of the defined step with 2 Newton updates",
                "executed_flops_per_particle_step": flops_per_pstep(w.n_planets, executed=True),
                "executed_tflops": achieved * flops_per_pstep(w.n_planets, executed=True) / fl,
                "executed_frac": achieved * flops_per_pstep(w.n_planets, executed=True) / fl / FP64_NOMINAL_TFLOPS,
                "peak_source": "nominal FP64 FMA rate: 148 SMs x 64 DFMA lanes (ncu peak_sustained) x 2 x "
                               "1.965 GHz; MEASURED_PEAKS.json has no FP64 figure",
                "probe_tflops": peak / 1e12, "frac_of_probe": achieved / (peak / 1e12),
                "probe": "glisse_fp64_peak_probe: register-resident DFMA chains timed in this run"}

    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": ms / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f64", "data": "synthetic",
        "config": {"workload": desc, "n_particles_per_gpu": w.n_particles, "n_planets": w.n_planets,
                   "chunk_steps": CHUNK, "dt_days": w.dt, "resync_chunks": 1,
                   "step": "one chunk of 1,024 integrator steps: planet-history + particle kernel + compaction",
                   "l2": "flushed between timed steps (256 MiB write, untimed)",
                   "parallelism": "particles sharded across ranks, planets replicated, no collectives"},
        "nominal_particle_steps_per_s": w.n_particles * world * CHUNK * args.steps / (ms * 1e-3),
        "active_fraction_end": res["active"] / w.n_particles,
        "gpu_launches": res["launches"],
        "roofline": roofline,
        "clocks": clk.summary(),
    }

    if not args.no_extras:
        e = time_e2e(binding, torch, w, max(3, min(args.steps, 10)), 3, device)
        if dist is not None:
            dist.barrier()
        e_s, e_ps = reduce_over_ranks(e["seconds"] * 1e3, e["psteps"], dist)
        line["e2e"] = {"value": e_ps / (e_s * 1e-3), "unit": UNIT, "h2d_bytes_per_step": e["h2d"],
                       "d2h_bytes_per_step": e["d2h"],
                       "what": "per step: glisse_create from pinned host arrays + glisse_advance(1024) + "
                               "glisse_read to pinned host arrays + destroy, wall clock"}
        if rank == 0 and world == 1:
            if args.workload != "1m_x4":
                _, wt = make_workload("1m_x4")
                rt = time_resident(binding, torch, wt, max(3, args.steps // 4), 3, device, flush)
                kt = rt["kernel_ms"] / max(rt["kernel_launches"], 1)
                at = flops_per_pstep(4) * (rt["psteps"] / max(rt["kernel_launches"], 1)) / (kt * 1e-3) / 1e12
                line["target_1m_x4"] = {"value": rt["psteps"] / (rt["ms"] * 1e-3), "unit": UNIT,
                                        "ms_per_step": rt["ms"] / max(3, args.steps // 4),
                                        "roofline_frac": at / FP64_NOMINAL_TFLOPS, "achieved_tflops": at,
                                        "executed_frac": at * EXEC_FLOPS_NP4 / ALGO_FLOPS_NP4 / FP64_NOMINAL_TFLOPS,
                                        "frac_of_probe": at / (peak / 1e12),
                                        "workload": WORKLOADS["1m_x4"][0]}
            rate, secs, ps = oracle_rate(w, 16384, 3000)
            line["cpu_baseline"] = {"value": rate, "unit": UNIT, "cores": 1, "kind": "oracle",
                                    "sample": f"first 16,384 particles x 3,000 steps of the same workload "
                                              f"({ps:.3g} particle-steps in {secs:.1f} s), single thread"}
    if rank == 0:
        print(json.dumps(line))
    if dist is not None:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
