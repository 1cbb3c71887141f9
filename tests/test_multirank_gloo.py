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


# ---- NEXT-3: the multi-GPU schedule of the factorisation (krr_dist_schedule, host logic) executed symbolically by two
# gloo ranks: every message is a real collective (tile ids travel), every compute task checks that the tiles it reads are
# present on its rank when it is issued.
def _dist_worker(rank, world, port, NT, nb, out):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    import numpy as np
    import paper_2409_01712_b200 as krr
    rng = np.random.default_rng(4)
    h_map = krr.uniform_map(NT, krr.FP32)
    for i in range(NT):
        for j in range(i):
            h_map[i, j] = int(rng.integers(0, 3))                      # a mosaic: message sizes differ per tile
    sched = krr.dist_schedule(NT, nb, h_map, world, rank)
    owner = lambda i: i % world
    have, have_m, produced, recv_bytes = set(), set(), [], 0
    tile_bytes = lambda i, j: nb * nb * {0: 4, 1: 2, 2: 1}[int(h_map[i, j])]
    for t in sched:
        k = t["k"]
        mine_below = [i for i in range(k + 1, NT) if owner(i) == rank]
        if t["op"] == "newest":
            assert t["nrows"] == len(mine_below) and (k, k - 1) in have
            assert all((i, k - 1) in have for i in mine_below)
        elif t["op"] == "older":                                        # O(k): terms s < k-1 of column k
            rows = [i for i in range(k, NT) if owner(i) == rank]
            assert t["nrows"] == len(rows)
            for s in range(k - 1):
                assert (k, s) in have, (rank, k, s)
                assert all((i, s) in have for i in rows if i > k)
        elif t["op"] == "chain":
            assert owner(k) == rank and all((k, s) in have for s in range(k))
        elif t["op"] == "trsm":
            assert k in have_m and t["nrows"] == len(mine_below)
            for i in mine_below:
                have.add((i, k)); produced.append((i, k))
        elif t["op"] == "bcast_m":
            buf = torch.tensor([k if rank == t["root"] else -1])
            assert t["root"] == owner(k)
            dist.broadcast(buf, src=t["root"])
            assert int(buf) == k
            have_m.add(k); recv_bytes += t["bytes"] * 0
        elif t["op"] == "bcast_next":
            assert t["root"] == owner(k + 1) and t["bytes"] == tile_bytes(k + 1, k)
            if rank == t["root"]:
                assert (k + 1, k) in have
            buf = torch.tensor([k + 1, k] if rank == t["root"] else [-1, -1])
            dist.broadcast(buf, src=t["root"])
            have.add((int(buf[0]), int(buf[1]))); recv_bytes += t["bytes"]
        elif t["op"] == "allgather":
            mine = [(i, k) for i in range(k + 2, NT) if owner(i) == rank]
            assert t["nrows"] == len(mine) and all(x in have for x in mine)
            gathered = [None] * world
            dist.all_gather_object(gathered, mine)
            got = [x for part in gathered for x in part]
            assert sum(tile_bytes(i, j) for (i, j) in got) == t["bytes"]
            have.update(tuple(x) for x in got); recv_bytes += t["bytes"]
    out.put((rank, sorted(produced), len(have), recv_bytes, [t["op"] for t in sched].count("chain")))
    dist.barrier()
    dist.destroy_process_group()


def test_multigpu_schedule_world2_covers_the_factor_and_respects_dependences():
    from paper_2409_01712_b200 import build
    build.build()
    NT, nb, world = 9, 128, 2
    ctx = mp.get_context("spawn")
    out = ctx.Queue()
    port = 33500 + (os.getpid() % 2000)
    procs = [ctx.Process(target=_dist_worker, args=(r, world, port, NT, nb, out)) for r in range(world)]
    for p in procs:
        p.start()
    res = sorted(out.get(timeout=180) for _ in range(world))
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    all_tiles = sorted((i, j) for i in range(NT) for j in range(i))
    produced = sorted(x for r in res for x in r[1])
    assert produced == all_tiles                                         # every off-diagonal tile exactly once, by its row's owner
    for rank, prod, nhave, recv, nchain in res:
        assert all(i % world == rank for (i, j) in prod)
        assert nhave == len(all_tiles)                                   # every rank ends with the whole factor's images
        assert nchain == len([k for k in range(NT) if k % world == rank])
    # with one rank the schedule degenerates to the single-GPU sequence: no tile ever crosses a link but is "received" from itself
    import paper_2409_01712_b200 as krr
    single = krr.dist_schedule(NT, nb, krr.uniform_map(NT, krr.FP16), 1, 0)
    ops = [t["op"] for t in single]
    assert ops.count("chain") == NT and ops.count("trsm") == NT - 1 and ops.count("newest") == NT - 2 and ops.count("older") == NT - 2
    order = [(t["op"], t["k"]) for t in single if t["op"] in ("newest", "older", "chain", "trsm")]
    assert order[:6] == [("chain", 0), ("trsm", 0), ("newest", 1), ("older", 2), ("chain", 1), ("trsm", 1)]
