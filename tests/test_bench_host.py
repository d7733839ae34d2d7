"""Host-side logic of bench.py's multi-GPU path, on CPU: world_size-2 gloo processes shard the
particles (no data-path collective) and reduce time (max) and units (sum)."""
import os
import sys

import numpy as np
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def _worker(rank, world, port, q):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    import bench
    from paper_2011_03484_b200 import inputs
    dist.init_process_group("gloo", rank=rank, world_size=world)
    bench.WORKLOADS["tiny"] = ("tiny", lambda n: inputs.config(1, n))
    _, w = bench.make_workload("tiny", world, rank)
    ms, units = bench.reduce_over_ranks(10.0 + 5.0 * rank, float(w.n_particles), dist)
    q.put((rank, ms, units, w.n_particles, w.pos[:, :2].tolist(), w.planet_pos.tolist()))
    dist.barrier()
    dist.destroy_process_group()


def test_two_rank_sharding_and_reduction():
    world, port = 2, 29000 + os.getpid() % 2000
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_worker, args=(r, world, port, q)) for r in range(world)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=120) for _ in range(world))
    for p in procs:
        p.join(60)
        assert p.exitcode == 0
    from paper_2011_03484_b200 import inputs
    big = inputs.config(1, 2048)
    for rank, ms, units, n, head, planets in res:
        assert ms == 15.0                      # max over ranks
        assert units == 2048.0 and n == 1024   # weak scaling: every rank holds a full-size batch
        lo, _ = inputs.shard_range(2048, rank, world)
        assert np.array_equal(np.array(head), big.pos[:, lo:lo + 2])   # disjoint contiguous slices
        assert np.array_equal(np.array(planets), big.planet_pos)        # planets replicated


def _gloo_rank(argv):
    """Stand-in for bench.rank_main on a box without GPUs: what a rank does minus the kernels."""
    import bench
    from paper_2011_03484_b200 import inputs
    rank, world = int(os.environ["RANK"]), int(os.environ["WORLD_SIZE"])
    assert int(os.environ["LOCAL_RANK"]) == rank and os.environ["MASTER_ADDR"] == "127.0.0.1"
    dist.init_process_group("gloo", rank=rank, world_size=world)
    bench.WORKLOADS["tiny"] = ("tiny", lambda n: inputs.config(1, n))
    _, w = bench.make_workload("tiny", world, rank)
    ms, units = bench.reduce_over_ranks(2.0 + rank, float(w.n_particles), dist)
    with open(os.path.join(argv[0], f"rank{rank}.txt"), "w") as fh:
        fh.write(f"{world} {ms} {units}")
    dist.barrier()
    dist.destroy_process_group()


def test_gpus_flag_starts_the_ranks_itself(tmp_path):
    """`python bench.py --gpus N` without torchrun: bench.launch_ranks starts one process per GPU with
    the torchrun environment; here with gloo at world size 2 and a CPU stand-in for the rank body."""
    import bench
    bench.launch_ranks(2, _gloo_rank, [str(tmp_path)], port=31000 + os.getpid() % 2000)
    got = sorted(open(tmp_path / f"rank{r}.txt").read() for r in range(2))
    assert got == ["2 3.0 2048.0", "2 3.0 2048.0"]      # both ranks see max time and summed units


def test_single_process_reduction_is_identity():
    import bench
    assert bench.reduce_over_ranks(3.5, 7.0, None) == (3.5, 7.0)


def test_reference_arm_prints_contract_line():
    import json
    import subprocess
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--steps", "1",
                          "--warmup", "3"], capture_output=True, text=True, check=True, cwd=ROOT).stdout
    line = json.loads(out.strip().splitlines()[-1])
    assert line["impl"] == "reference" and line["unit"] == "particle-steps/s" and line["value"] > 1e5
    assert line["cpu_baseline"]["kind"] == "oracle" and line["e2e"]["h2d_bytes_per_step"] == 0
