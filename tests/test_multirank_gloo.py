"""The N > 1 path of bench.py on CPU: two gloo ranks (the factorisation does not
shard, `--gpus N` runs N independent replicas; there is no data-path collective, only the timing
reduction).  Covers the replica seeding, the max-over-ranks step time, the whole-job value, and the
reference arm's rank-0-only output under torchrun."""
import json
import os
import subprocess
import sys

import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)


def _worker(rank, world, port, out):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    import bench
    from krr_inputs import CONFIGS, genotypes, scaled_config
    cfg = scaled_config(CONFIGS["C1"], nb=32, n=64, p=64)
    mine = bench.replica_config(cfg, rank)
    G = genotypes(mine.seed, mine.n, mine.p, mine.genotype)
    # every rank sees every rank's genotype checksum: replicas must differ
    sums = [torch.zeros(1, dtype=torch.int64) for _ in range(world)]
    dist.all_gather(sums, G.to(torch.int64).sum().reshape(1))
    ms_local = 10.0 + 5.0 * rank                       # rank 1 is the slow one
    ms = bench.max_over_ranks(ms_local, world, "cpu")
    out.put((rank, mine.seed, [int(x) for x in sums], ms, bench.whole_job_value(cfg.n, world, ms)))
    dist.barrier()
    dist.destroy_process_group()


def test_replicas_and_max_over_ranks_world2():
    ctx = mp.get_context("spawn")
    out = ctx.Queue()
    port = 29500 + (os.getpid() % 2000)
    procs = [ctx.Process(target=_worker, args=(r, 2, port, out)) for r in range(2)]
    for p in procs:
        p.start()
    res = sorted(out.get(timeout=120) for _ in range(2))
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    (r0, seed0, sums0, ms0, v0), (r1, seed1, sums1, ms1, v1) = res
    assert (r0, r1) == (0, 1) and seed1 == seed0 + 1000
    assert sums0 == sums1 and sums0[0] != sums0[1]     # independent replicas, seen consistently
    assert ms0 == ms1 == 15.0                          # the slowest rank sets the step time
    assert v0 == v1 == 2 * (64 ** 3 / 3.0) / 15e-3 / 1e12


def test_whole_job_value_is_identity_at_world1():
    import bench
    assert bench.max_over_ranks(7.5, 1, "cpu") == 7.5
    assert abs(bench.whole_job_value(65536, 1, 250.0) - 65536 ** 3 / 3.0 / 0.25 / 1e12) < 1e-9


def test_reference_arm_under_torchrun_prints_one_line_from_rank0():
    port = 31500 + (os.getpid() % 2000)
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "2", "--master-addr",
           "127.0.0.1", "--master-port", str(port), os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2",
           "--steps", "1", "--warmup", "0", "--config", "C1", "--sample-tiles", "2"]
    env = dict(os.environ, OMP_NUM_THREADS="2", CUDA_VISIBLE_DEVICES="")
    res = subprocess.run(cmd, capture_output=True, text=True, timeout=600, env=env, cwd=ROOT)
    assert res.returncode == 0, res.stderr[-2000:]
    lines = [ln for ln in res.stdout.splitlines() if ln.startswith("{")]
    assert len(lines) == 1
    d = json.loads(lines[0])
    assert d["impl"] == "reference" and d["n_gpus"] == 2 and d["cpu_baseline"]["kind"] == "oracle"
    assert d["e2e"]["h2d_bytes_per_step"] == 0 and d["value"] > 0
