"""Host-side logic of bench.py for N > 1 (replicas only), on CPU with gloo."""
import json
import os
import socket
import subprocess
import sys

import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, out):
    import bench
    dist.init_process_group("gloo", init_method=f"tcp://127.0.0.1:{port}", rank=rank, world_size=world)
    ms, e2e = bench.max_over_ranks([10.0 + 5.0 * rank, 100.0 - rank], world)
    out[rank] = (ms, e2e, bench.job_throughput(1000, 7, world, ms))
    dist.destroy_process_group()


def test_max_over_ranks_and_whole_job_value_world2():
    world, port = 2, _free_port()
    with mp.Manager() as mgr:
        out = mgr.dict()
        mp.spawn(_worker, args=(world, port, out), nprocs=world, join=True)
        res = dict(out)
    for rank in range(world):
        ms, e2e, value = res[rank]
        assert ms == 15.0 and e2e == 100.0                      # slowest rank decides
        assert value == 1000 * 7 * 2 / 15e-3                    # whole-job aggregate


def test_reference_arm_under_torchrun_prints_one_line():
    """--impl reference with 2 ranks: rank 0 alone runs the oracle and prints; rank 1 exits 0."""
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "2",
           "--master-addr", "127.0.0.1", "--master-port", str(_free_port()),
           os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2", "--steps", "3",
           "--warmup", "3", "--workload", "config1"]
    r = subprocess.run(cmd, capture_output=True, text=True, timeout=600, cwd=ROOT)
    assert r.returncode == 0, r.stderr[-2000:]
    lines = [json.loads(x) for x in r.stdout.splitlines() if x.startswith("{")]
    assert len(lines) == 1
    d = lines[0]
    assert d["impl"] == "reference" and d["n_gpus"] == 2 and d["vs_baseline"] is None
    assert d["cpu_baseline"]["kind"] == "oracle" and d["cpu_baseline"]["value"] == d["value"] > 0
    assert d["e2e"] == {"value": d["value"], "unit": d["unit"], "h2d_bytes_per_step": 0,
                        "d2h_bytes_per_step": 0}
    assert d["config"]["workload"] == "config1" and d["dtype"] == "f64"


def test_roofline_record_is_reproducible_from_its_own_fields():
    """roofline.frac = (156 B x cells of active tiles + 64 B x cells of all-dry tiles) / time / peak:
    it can be recomputed by hand from the line, and skipping work (a low active share) lowers the
    bytes it is credited with instead of inflating the fraction."""
    import bench
    tiles = {"tile_cells": 192}
    n, ms, peak = 13_005_000, 0.2, 6547.5
    r = bench.roofline_record(n, ms, 0.063, 0.07, 9.0e8, tiles, peak, "test")
    algo = (156.0 * 0.063 + 64.0 * (1 - 0.063)) * n
    assert r["achieved"] == algo / (ms * 1e-3) / 1e9 and r["frac"] == r["achieved"] / peak
    assert r["frac"] < 1.0 < r["frac_fixed_156"]            # the round-1 headline (1.53) was this one
    assert r["traffic"] == 9.0e8 and r["frac_traffic"] == 9.0e8 / (ms * 1e-3) / 1e9 / peak
    full = bench.roofline_record(n, ms, 1.0, 1.0, 9.0e8, tiles, peak, "test")
    assert full["frac"] == full["frac_fixed_156"]
