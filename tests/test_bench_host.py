"""Host logic of bench.py: the replicas-only N > 1 aggregation (world_size 2 over gloo, on CPU), the clock-sample
parser and the reference arm's JSON line.  No GPU needed."""
import json
import os
import subprocess
import sys

import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)
import bench  # noqa: E402


def _worker(rank, world, port, out):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    my_ms = 10.0 + 5.0 * rank                       # rank 1 is the slow replica
    tot = bench.max_over_ranks(my_ms, world, torch.device("cpu"))
    val = bench.aggregate_value(1000, world, tot)
    dist.barrier()
    if rank == 0:
        json.dump({"tot": tot, "val": val}, open(out, "w"))
    dist.destroy_process_group()


def test_max_over_ranks_gloo_world2(tmp_path):
    out = str(tmp_path / "r.json")
    port = 29500 + os.getpid() % 2000
    mp.spawn(_worker, args=(2, port, out), nprocs=2, join=True)
    r = json.load(open(out))
    assert r["tot"] == 15.0                                        # the max, not the mean or rank 0's own time
    assert abs(r["val"] - 2 * 1000 / 15e-3 / 1e9) < 1e-12          # both replicas' pairs over the slowest one's time


def test_single_rank_passthrough():
    assert bench.max_over_ranks(3.5, 1, torch.device("cpu")) == 3.5


def test_clock_sampler_parsing():
    s = bench.ClockSampler(0)
    s.proc = object()                                # pretend nvidia-smi ran; feed rows directly
    s.rows = [(100.0, "1965, 1965, 400.1, Not Active, Not Active, Not Active, Not Active"),
              (100.1, "1800, 1965, 950.0, Not Active, Not Active, Not Active, Active"),
              (100.2, "1785, 1965, 990.0, Not Active, Not Active, Not Active, Active")]

    class P:                                          # minimal stand-in for the Popen handle
        def terminate(self): pass
        def wait(self, timeout=None): pass
        def kill(self): pass
    s.proc = P()
    c = s.stop(99.9, 100.3)
    assert c["sm_mhz"] == 1800.0 and c["sm_max_mhz"] == 1965.0 and c["reasons"] == ["sw_power_cap"]


def test_reference_arm_line():
    """--impl reference prints ONE JSON line with the contract's keys (oracle on the host cores, bounded sample)."""
    p = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--steps", "1",
                        "--warmup", "0", "--ref-seconds", "0.5"], capture_output=True, text=True, timeout=300)
    assert p.returncode == 0, p.stderr
    lines = [l for l in p.stdout.splitlines() if l.startswith("{")]
    assert len(lines) == 1
    d = json.loads(lines[0])
    assert d["impl"] == "reference" and d["unit"] == bench.UNIT and d["value"] > 0 and d["higher_is_better"] is True
    assert d["cpu_baseline"]["kind"] == "oracle" and d["cpu_baseline"]["cores"] >= 1
    assert d["e2e"] == {"value": d["value"], "unit": d["unit"], "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}
    assert d["config"]["workload"].startswith("cfg4")
