"""Host logic of bench.py that needs no GPU: the reference arm's JSON line, and the N > 1 plumbing (workload
hand-over from rank 0, max-over-ranks timing, whole-job aggregation) on a world_size-2 gloo group."""
import json
import os
import subprocess
import sys

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_reference_arm_prints_one_json_line():
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--config", "1",
                          "--steps", "3", "--warmup", "1"], capture_output=True, text=True, check=True).stdout
    lines = [l for l in out.splitlines() if l.strip()]
    assert len(lines) == 1
    d = json.loads(lines[0])
    assert d["impl"] == "reference" and d["metric"] == "cell_updates_per_s" and d["unit"] == "cell-updates/s"
    assert d["value"] > 0 and d["higher_is_better"] is True and d["dtype"] == "f64" and d["vs_baseline"] is None
    assert d["cpu_baseline"]["kind"] == "oracle" and d["cpu_baseline"]["cores"] == 1
    assert d["e2e"] == {"value": d["value"], "unit": d["unit"], "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}
    assert d["config"]["n_cells"] == 4000 and d["steps"] == 3 and d["warmup"] == 1


def test_reference_arm_other_ranks_exit_without_work():
    env = dict(os.environ, RANK="1", LOCAL_RANK="1", WORLD_SIZE="2")
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--config", "1",
                        "--gpus", "2", "--steps", "2", "--warmup", "1"], capture_output=True, text=True, env=env)
    assert r.returncode == 0 and r.stdout.strip() == ""


def _worker(rank, world, port, q):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    sys.path.insert(0, ROOT)
    import torch
    import torch.distributed as dist
    import bench
    dist.init_process_group("gloo", rank=rank, world_size=world)
    w = bench.load_workload(1, 0.25, rank, world, dist.barrier)            # rank 0 generates, rank 1 reads its file
    ms = bench.max_over_ranks(10.0 + 5.0 * rank, world, torch.device("cpu"))
    q.put((rank, w.n_cells, float(np.sum(w.h)), int(w.edge_cell.sum()), ms,
           bench.aggregate_value(w.n_cells, 100, 2, world, ms * 1e-3)))
    dist.destroy_process_group()


def test_two_rank_replicas_gloo():
    import torch.multiprocessing as mp
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = 29500 + os.getpid() % 2000
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=180) for _ in procs)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    (r0, n0, h0, e0, ms0, v0), (r1, n1, h1, e1, ms1, v1) = res
    assert (n0, h0, e0) == (n1, h1, e1) and n0 == 250                       # both ranks hold the same workload
    assert ms0 == ms1 == 15.0                                                # max over ranks
    assert v0 == v1 == pytest.approx(2 * 250 * 100 * 2 / 15e-3)              # whole-job aggregate
