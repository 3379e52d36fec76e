"""The N>1 path of bench.py on CPU (-m "not gpu"): world_size-2 gloo processes exercise the rank plumbing the GPU
run uses with nccl -- barrier, max-over-ranks timing, whole-job value of N independent replicas -- and the
reference arm's "rank 0 alone runs" rule.  The path itself has no data-path collective."""
import json
import os
import socket
import subprocess
import sys

import pytest
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def _worker(rank, world, port, q):
    os.environ.update(RANK=str(rank), WORLD_SIZE=str(world), LOCAL_RANK=str(rank), MASTER_ADDR="127.0.0.1",
                      MASTER_PORT=str(port))
    sys.path.insert(0, ROOT)
    import bench
    r = bench.Ranks(backend="gloo")
    r.barrier()
    local_seconds = 0.010 * (rank + 1)            # rank 1 is the slow one
    mx = r.max(local_seconds)
    total = r.sum(1.0)
    val = bench.whole_job_value(1000.0, r.world, mx)
    r.barrier()
    r.close()
    q.put((rank, mx, total, val))


def test_world_size_2_gloo_max_over_ranks():
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    out = sorted(q.get(timeout=120) for _ in procs)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    for rank, mx, total, val in out:
        assert mx == pytest.approx(0.020)          # the MAX over ranks, on every rank
        assert total == 2.0
        assert val == pytest.approx(2 * 1000.0 / 0.020)   # replicas: units of all ranks / slowest rank's time


def test_reference_arm_runs_on_rank0_only():
    env = dict(os.environ, RANK="1", WORLD_SIZE="2", LOCAL_RANK="1", MASTER_ADDR="127.0.0.1",
               MASTER_PORT=str(_free_port()))
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2",
                        "--steps", "1", "--warmup", "0", "--workload", "c1"], env=env, capture_output=True, text=True,
                       timeout=300)
    assert r.returncode == 0 and r.stdout.strip() == ""
    env["RANK"] = env["LOCAL_RANK"] = "0"
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2",
                        "--steps", "1", "--warmup", "0", "--workload", "c1"], env=env, capture_output=True, text=True,
                       timeout=300)
    assert r.returncode == 0, r.stderr
    line = json.loads(r.stdout.strip().splitlines()[-1])
    assert line["impl"] == "reference" and line["cpu_baseline"]["kind"] == "oracle"
    assert line["e2e"]["h2d_bytes_per_step"] == 0 and line["value"] > 0


def test_roofline_model_matches_survey_table():
    sys.path.insert(0, ROOT)
    import bench
    import lqcd_inputs as li
    c5 = li.CONFIGS["c5"]
    m = bench.model(c5)
    assert m["wilson_clover"]["bytes"] == 768 * c5.volume            # 768 B / site
    assert bench.model(c5, links12=True)["wilson_clover"]["bytes"] == 672 * c5.volume
    assert m["wilson_clover"]["flops"] == 1872 * c5.volume
    assert m["coarse_mult"]["bytes"] == 295936 * c5.cvolume          # 9 N^2 8 + 2 N 8, N = 64
    assert m["restrict"]["bytes"] == 3168 * c5.volume + 512 * c5.cvolume
    m64 = bench.model(c5, real_bytes=8)                              # fp64 variants: twice the bytes, same flops
    for k in bench.STEP_ORDER:
        assert m64[k]["bytes"] == 2 * m[k]["bytes"] and m64[k]["flops"] == m[k]["flops"]


def test_default_rank_grid_splits_t_z_y_first():
    """bench.py --sharded: the x direction (one 16-byte vector per 128-byte line on its faces) is split last."""
    sys.path.insert(0, ROOT)
    import bench
    assert bench.default_rank_grid(1) == (1, 1, 1, 1)
    assert bench.default_rank_grid(2) == (1, 1, 1, 2)
    assert bench.default_rank_grid(4) == (1, 1, 2, 2)
    assert bench.default_rank_grid(8) == (1, 2, 2, 2)
    assert bench.default_rank_grid(16) == (2, 2, 2, 2)
    assert bench.default_rank_grid(6) == (1, 1, 1, 6)
    for n in (1, 2, 3, 4, 6, 8, 12, 16):
        g = bench.default_rank_grid(n)
        assert g[0] * g[1] * g[2] * g[3] == n
