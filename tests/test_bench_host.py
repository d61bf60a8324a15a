"""Host-side logic of bench.py that needs no GPU: the N > 1 aggregation (world_size-2 gloo run on
CPU) and the `--impl reference` arm (rank 0 prints the JSON line, other ranks exit 0 silently)."""
import json
import os
import subprocess
import sys
from pathlib import Path

import pytest

ROOT = Path(__file__).resolve().parents[1]


def _worker(rank, world, port, q):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    sys.path.insert(0, str(ROOT))
    import torch.distributed as dist
    import bench
    dist.init_process_group("gloo", rank=rank, world_size=world)
    ms = bench.max_over_ranks(1.5 + rank, "cpu")          # rank 0: 1.5 ms, rank 1: 2.5 ms
    q.put((rank, ms, bench.job_throughput(world, 1000, 10, ms)))
    dist.barrier()
    dist.destroy_process_group()


def test_replica_aggregation_world_size_2_gloo():
    import torch.multiprocessing as mp
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = 29500 + os.getpid() % 2000
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    out = sorted(q.get(timeout=120) for _ in range(2))
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    # both ranks agree on the slowest rank's time; value counts the cells of BOTH replicas
    assert [o[1] for o in out] == [2.5, 2.5]
    assert out[0][2] == pytest.approx(2 * 1000 * 10 / 2.5e-3)


def test_single_process_needs_no_process_group():
    sys.path.insert(0, str(ROOT))
    import bench
    assert bench.max_over_ranks(3.25, "cpu") == 3.25
    assert bench.job_throughput(1, 4, 5, 2.0) == pytest.approx(10000.0)


def _run_reference(rank):
    env = dict(os.environ, RANK=str(rank), WORLD_SIZE="2")
    return subprocess.run([sys.executable, str(ROOT / "bench.py"), "--impl", "reference", "--gpus", "2",
                           "--ref-n", "32", "--steps", "2", "--warmup", "1"],
                          capture_output=True, text=True, env=env, timeout=300)


def test_reference_arm_contract():
    r0, r1 = _run_reference(0), _run_reference(1)
    assert r0.returncode == 0 and r1.returncode == 0
    assert r1.stdout.strip() == ""                         # other ranks exit 0 without work
    line = json.loads(r0.stdout.strip().splitlines()[-1])
    assert line["impl"] == "reference" and line["unit"] == "cell-updates/s" and line["value"] > 0
    assert line["cpu_baseline"]["kind"] == "oracle" and line["cpu_baseline"]["cores"] >= 1
    assert line["e2e"] == {"value": line["value"], "unit": line["unit"],
                           "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}
    assert line["vs_baseline"] is None and line["higher_is_better"] is True
