"""Host logic of bench.py on CPU: the N > 1 protocol ("replicas only": independent lattices, no
data-path collective; barrier, max over ranks, whole-job rate) with world_size 2 over gloo, and
the reference arm's JSON line."""
import json
import os
import socket
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def _worker(rank, world, port, out_dir):
    import torch
    import torch.distributed as dist
    sys.path.insert(0, ROOT)
    import bench
    dist.init_process_group("gloo", init_method="tcp://127.0.0.1:%d" % port, rank=rank, world_size=world)
    local_ms = 100.0 + 50.0 * rank                     # rank 1 is the slow one
    dist.barrier()
    ms_max = bench.max_over_ranks(local_ms, world, "cpu")
    value = bench.whole_job_rate(world, 64 ** 3, 10, 3, ms_max)
    json.dump({"rank": rank, "seed": bench.rank_seed(rank), "ms_max": ms_max, "value": value},
              open(os.path.join(out_dir, "r%d.json" % rank), "w"))
    dist.barrier()
    dist.destroy_process_group()


def test_two_rank_protocol_over_gloo(tmp_path):
    import torch.multiprocessing as mp
    port = _free_port()
    mp.spawn(_worker, args=(2, port, str(tmp_path)), nprocs=2, join=True)
    r = [json.load(open(tmp_path / ("r%d.json" % i))) for i in range(2)]
    assert [x["seed"] for x in r] == [4, 5]            # distinct lattices, config 5's seed on rank 0
    assert r[0]["ms_max"] == r[1]["ms_max"] == 150.0   # max over ranks, same on every rank
    want = 2 * 64 ** 3 * 10 * 3 / (150.0 * 1e6)        # both ranks' work over the slowest rank's time
    assert r[0]["value"] == pytest.approx(want) and r[1]["value"] == pytest.approx(want)


def test_single_rank_needs_no_process_group():
    sys.path.insert(0, ROOT)
    import bench
    assert bench.max_over_ranks(12.5, 1, "cpu") == 12.5
    assert bench.whole_job_rate(1, 2048 ** 3, 1000, 1, 418.0) == pytest.approx(2048 ** 3 * 1000 / 418.0e6)


def test_reference_arm_line():
    """bench.py --impl reference times the oracle on host cores and prints the contract's line."""
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference",
                          "--steps", "1", "--warmup", "1", "--ref-L", "64"],
                         capture_output=True, text=True, timeout=600)
    assert out.returncode == 0, out.stderr
    line = json.loads(out.stdout.strip().splitlines()[-1])
    assert line["impl"] == "reference" and line["metric"] == "site_updates_per_ns"
    assert line["value"] > 0 and line["cpu_baseline"]["kind"] == "oracle" and line["cpu_baseline"]["cores"] >= 1
    assert line["e2e"]["h2d_bytes_per_step"] == 0 and line["e2e"]["value"] == line["value"]
    assert line["higher_is_better"] is True and line["vs_baseline"] is None


def test_reference_arm_other_ranks_exit_quietly():
    env = dict(os.environ, RANK="1", WORLD_SIZE="2")
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference"],
                         capture_output=True, text=True, timeout=120, env=env)
    assert out.returncode == 0 and out.stdout.strip() == ""
