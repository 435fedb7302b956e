"""The N > 1 path of bench.py on CPU (gloo, world_size 2): the path does not shard ("replicas only"),
so the only cross-rank step is the MAX over ranks of the device time, and the whole-job value is
world x lines / that time.  The reference arm must print on rank 0 only."""
import json
import os
import socket
import subprocess
import sys

import pytest

torch = pytest.importorskip("torch")
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, q):
    import torch.distributed as dist
    sys.path.insert(0, ROOT)
    import bench
    dist.init_process_group("gloo", init_method=f"tcp://127.0.0.1:{port}", rank=rank, world_size=world)
    local_ms = 100.0 + 50.0 * rank                     # rank 1 is the slow one
    total = bench.max_over_ranks(local_ms, dist, "cpu")
    dist.barrier()
    q.put((rank, total, bench.replicas_value(1000, 5, world, total)))
    dist.destroy_process_group()


def test_max_over_ranks_and_value_gloo_world2():
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    got = sorted(q.get(timeout=120) for _ in procs)
    for p in procs:
        p.join(60)
        assert p.exitcode == 0
    for rank, total, value in got:
        assert total == 150.0                           # the max, on every rank
        assert value == pytest.approx(2 * 1000 * 5 / 0.150)


def test_single_rank_needs_no_process_group():
    sys.path.insert(0, ROOT)
    import bench
    assert bench.max_over_ranks(12.5) == 12.5
    assert bench.replicas_value(10, 2, 1, 1000.0) == 20.0


def test_reference_arm_prints_on_rank0_only():
    """`bench.py --impl reference` under a 2-rank launch: rank 1 exits 0 without output; rank 0 prints one JSON
    line with impl = reference (tiny workload so the CPU suite stays fast)."""
    base = [sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2", "--steps", "1",
            "--warmup", "0", "--config", "1", "--n-lines", "2000"]
    outs = []
    for rank in (0, 1):
        env = dict(os.environ, RANK=str(rank), LOCAL_RANK=str(rank), WORLD_SIZE="2", CUDA_VISIBLE_DEVICES="",
                   OMP_NUM_THREADS="2")
        r = subprocess.run(base, env=env, capture_output=True, text=True, timeout=600)
        assert r.returncode == 0, r.stderr[-2000:]
        outs.append(r.stdout.strip())
    assert outs[1] == ""
    line = json.loads(outs[0].splitlines()[-1])
    assert line["impl"] == "reference" and line["n_gpus"] == 2 and line["value"] > 0
    assert line["e2e"]["h2d_bytes_per_step"] == 0 and line["cpu_baseline"]["kind"] == "oracle"
