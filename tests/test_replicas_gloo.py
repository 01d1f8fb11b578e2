"""N > 1 path of bench.py on CPU: two gloo ranks, the barrier and the max-over-ranks timing that
turn per-replica times into the whole-job MLUPS."""
import os
import socket

import pytest
import torch.multiprocessing as mp


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def _worker(rank, world, port, out):
    os.environ.update(RANK=str(rank), WORLD_SIZE=str(world), LOCAL_RANK=str(rank),
                      MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    from paper_2308_16597_b200 import replicas
    assert replicas.rank_info() == (rank, world, rank)
    assert replicas.init("gloo") == world
    replicas.barrier()
    ms = [10.0, 12.5][rank]                      # rank 1 is the slow one
    ms_max = replicas.max_over_ranks(ms)
    out[rank] = (ms_max, replicas.whole_job_mlups(1000 * 1000, 50, ms_max, world))
    replicas.barrier()
    replicas.shutdown()


def test_two_gloo_ranks_report_the_slowest_time_and_the_whole_job_rate():
    world, port = 2, _free_port()
    with mp.Manager() as m:
        out = m.dict()
        mp.spawn(_worker, args=(world, port, out), nprocs=world, join=True)
        res = dict(out)
    assert res[0] == res[1]
    ms_max, mlups = res[0]
    assert ms_max == 12.5
    # 2 replicas x 1e6 nodes x 50 steps in 12.5 ms = 8000 MLUPS
    assert mlups == pytest.approx(8000.0)


def test_single_process_needs_no_group():
    from paper_2308_16597_b200 import replicas
    for k in ("RANK", "WORLD_SIZE", "LOCAL_RANK"):
        os.environ.pop(k, None)
    assert replicas.rank_info() == (0, 1, 0)
    assert replicas.init("gloo") == 1
    assert replicas.max_over_ranks(3.25) == 3.25
    assert replicas.whole_job_mlups(16_000_000, 2000, 1316.0, 1) == pytest.approx(24316.1, rel=1e-4)


def test_reference_arm_prints_one_json_line():
    """bench.py --impl reference: the oracle on a bounded sample, one JSON line with the contract's
    keys (runs here on CPU; on the GPU box the driver launches it the same way)."""
    import json
    import subprocess
    import sys
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    env = {k: v for k, v in os.environ.items() if k not in ("RANK", "WORLD_SIZE", "LOCAL_RANK")}
    r = subprocess.run([sys.executable, os.path.join(root, "bench.py"), "--impl", "reference",
                        "--steps", "2", "--warmup", "1", "--config", "0"],
                       capture_output=True, text=True, timeout=240, env=env)
    assert r.returncode == 0, r.stderr[-500:]
    lines = [l for l in r.stdout.splitlines() if l.strip()]
    assert len(lines) == 1
    d = json.loads(lines[0])
    assert d["impl"] == "reference" and d["unit"] == "MLUPS" and d["value"] > 0
    assert d["cpu_baseline"]["kind"] == "oracle" and d["cpu_baseline"]["value"] == d["value"]
    assert d["e2e"]["h2d_bytes_per_step"] == 0 and d["e2e"]["d2h_bytes_per_step"] == 0
