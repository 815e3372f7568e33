"""N>1 path of bench.py on CPU (replicas only, no data-path collective).

World-size-2 `gloo` runs launched exactly as the driver launches bench.py (torch.distributed.run, 127.0.0.1):
  * the rank helpers (max over ranks, whole-job aggregate) under a real process group,
  * the reference arm: rank 0 alone runs and prints ONE JSON line, the other rank exits 0 without work.
The GPU arm itself needs a device and is covered by the -m gpu tests and the driver's bench run.
"""
import json
import os
import socket
import subprocess
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

WORKER = r"""
import json, os, sys
sys.path.insert(0, os.environ["FAR_ROOT"])
import torch.distributed as dist
import bench
dist.init_process_group("gloo")
rank, world = dist.get_rank(), dist.get_world_size()
# rank r "measured" (r + 1) * 10 ms for 4 steps: the job time is the slowest rank's
total_ms = bench.max_over_ranks((rank + 1) * 10.0, dist, "cpu")
value = bench.aggregate_value(world, 4, total_ms)
dist.barrier()
with open(os.path.join(os.environ["FAR_OUT"], f"rank{rank}.json"), "w") as f:
    json.dump({"rank": rank, "world": world, "total_ms": total_ms, "value": value}, f)
dist.destroy_process_group()
"""


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _torchrun(args, env=None, timeout=300):
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "2",
           "--master-addr", "127.0.0.1", "--master-port", str(_free_port())] + args
    e = dict(os.environ)
    e.update(env or {})
    return subprocess.run(cmd, cwd=ROOT, env=e, capture_output=True, text=True, timeout=timeout)


def test_max_over_ranks_and_aggregate_world2_gloo(tmp_path):
    script = tmp_path / "worker.py"
    script.write_text(WORKER)
    r = _torchrun([str(script)], env={"FAR_ROOT": ROOT, "FAR_OUT": str(tmp_path)})
    assert r.returncode == 0, r.stderr[-2000:]
    outs = [json.load(open(tmp_path / f"rank{i}.json")) for i in range(2)]
    for o in outs:
        assert o["world"] == 2
        assert o["total_ms"] == 20.0                 # max over ranks, not this rank's own 10 / 20
        assert abs(o["value"] - 2 * 4 / 0.020) < 1e-9  # replicas: both ranks' frames over the slowest rank's time


def test_single_process_helpers_are_identity():
    sys.path.insert(0, ROOT)
    import bench
    assert bench.max_over_ranks(3.5, None, "cpu") == 3.5
    assert bench.aggregate_value(1, 10, 5.0) == 2000.0


def test_reference_arm_under_torchrun_prints_one_line_from_rank0():
    r = _torchrun(["bench.py", "--impl", "reference", "--workload", "c1", "--gpus", "2", "--steps", "2", "--warmup", "1"])
    assert r.returncode == 0, r.stderr[-2000:]
    lines = [l for l in r.stdout.splitlines() if l.startswith("{")]
    assert len(lines) == 1, r.stdout
    d = json.loads(lines[0])
    assert d["impl"] == "reference" and d["n_gpus"] == 2 and d["steps"] == 2 and d["warmup"] == 1
    assert d["unit"] == "registrations/s" and d["higher_is_better"] is True and d["value"] > 0
    assert d["cpu_baseline"]["kind"] == "oracle" and d["cpu_baseline"]["value"] == d["value"]
    assert d["e2e"] == {"value": d["value"], "unit": d["unit"], "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}
