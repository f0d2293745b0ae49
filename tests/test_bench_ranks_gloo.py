"""The N > 1 path of bench.py is "replicas only": no data-path collective, one seeded
replica per rank, timing = MAX over ranks, value = whole-job aggregate.  This covers that rank logic with
world_size 2 on CPU (gloo); no kernel runs here."""
import json
import os
import subprocess
import sys

import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _worker(rank, world, port, out):
    os.environ.update(RANK=str(rank), WORLD_SIZE=str(world), LOCAL_RANK=str(rank), MASTER_ADDR="127.0.0.1",
                      MASTER_PORT=str(port))
    sys.path.insert(0, ROOT)
    import bench
    r, w, dist = bench._dist_setup(world, backend="gloo")
    try:
        bench._barrier(dist)
        slowest = bench._max_over_ranks(10.0 + 5.0 * r, dist)          # rank 1 is slower
        seed = bench.replica_seed(1003, r)
        out.put((r, w, slowest, seed, bench.whole_job_rate(1000, 4, w, slowest)))
    finally:
        dist.destroy_process_group()


def test_two_ranks_take_the_max_time_and_aggregate_the_whole_job():
    ctx = mp.get_context("spawn")
    out = ctx.Queue()
    port = 29500 + os.getpid() % 2000
    procs = [ctx.Process(target=_worker, args=(r, 2, port, out)) for r in range(2)]
    for p in procs:
        p.start()
    got = sorted(out.get(timeout=120) for _ in procs)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    assert [g[0] for g in got] == [0, 1] and all(g[1] == 2 for g in got)
    assert all(g[2] == 15.0 for g in got)                               # MAX over ranks on both ranks
    assert [g[3] for g in got] == [1003, 1004]                          # distinct seeded replicas
    # 2 ranks x 4 steps x 1000^2 interactions in 15 ms
    assert all(abs(g[4] - 2 * 4 * 1e6 / 15e-3 / 1e9) < 1e-12 for g in got)


def test_reference_arm_runs_on_rank_zero_only():
    env = dict(os.environ, RANK="1", WORLD_SIZE="2", LOCAL_RANK="1", MASTER_ADDR="127.0.0.1", MASTER_PORT="29999")
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2",
                        "--steps", "1", "--warmup", "0", "--config", "0"], env=env, capture_output=True, text=True,
                       timeout=300)
    assert r.returncode == 0 and r.stdout.strip() == ""
    env["RANK"] = "0"
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2",
                        "--steps", "1", "--warmup", "0", "--config", "0"], env=env, capture_output=True, text=True,
                       timeout=300)
    assert r.returncode == 0
    line = json.loads(r.stdout.strip().splitlines()[-1])
    assert line["impl"] == "reference" and line["n_gpus"] == 2 and line["value"] > 0
    assert line["e2e"]["h2d_bytes_per_step"] == 0 and line["cpu_baseline"]["kind"] == "oracle"
