"""Host-side logic of bench.py that only matters with more than one rank (replicas only),
run on CPU with the gloo backend, world_size 2: max-over-ranks timing, the whole-job aggregate, and that only
rank 0 of `--impl reference` does any work."""
import json
import os
import socket
import subprocess
import sys

import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, out):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    import bench
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        my_ms = 10.0 + 5.0 * rank                            # rank 1 is the slow one
        total = bench.max_over_ranks(my_ms)
        val = bench.whole_job_value(npts=1000, n_sweeps=9, steps=4, world=world, total_ms=total)
        with open(os.path.join(out, f"r{rank}.json"), "w") as fh:
            json.dump({"total": total, "value": val}, fh)
    finally:
        dist.destroy_process_group()


def test_max_over_ranks_and_aggregate_gloo_world2(tmp_path):
    port = _free_port()
    mp.spawn(_worker, args=(2, port, str(tmp_path)), nprocs=2, join=True)
    r = [json.load(open(tmp_path / f"r{k}.json")) for k in range(2)]
    assert r[0]["total"] == r[1]["total"] == 15.0            # the max, on every rank
    want = 2 * 9 * 1000 * 4 / 15.0e-3 / 1e9
    assert abs(r[0]["value"] - want) < 1e-12 * want and r[0]["value"] == r[1]["value"]


def test_single_process_is_identity():
    import bench
    assert bench.max_over_ranks(3.5) == 3.5
    assert bench.whole_job_value(10, 9, 1, 1, 1.0) == 9 * 10 / 1e-3 / 1e9


def test_reference_arm_other_ranks_exit_without_work():
    env = dict(os.environ, RANK="1", WORLD_SIZE="2", LOCAL_RANK="1")
    p = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2",
                        "--steps", "1", "--warmup", "0"], capture_output=True, text=True, env=env, timeout=120)
    assert p.returncode == 0 and p.stdout.strip() == ""


def test_traffic_row_and_its_source_stamp():
    """roofline.traffic comes from profiles/traffic.csv; the file's stamp (sha256 of the per-sweep kernels' source at
    capture time) decides traffic_stale.  The stamp line must not be mistaken for a data row."""
    import bench
    val, src, stale = bench.read_traffic("C5")
    assert val is not None and 5.7e10 < val < 5.9e10          # ~16 B/point x 48^3 x 32^3
    assert "not measured in this run" in src
    assert stale in (True, False)                             # a stamp is on record
    assert len(bench.sweep_source_sha()) == 64
    none, why, st = bench.read_traffic("no-such-workload")
    assert none is None and st is None and "no ncu capture" in why
