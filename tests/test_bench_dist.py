"""The N>1 path of bench.py on CPU (gloo, world_size 2): replicas only, no data-path collective — the process group carries the
barrier and the reduction value = sum of units over ranks / max over ranks of the time."""
import os
import socket
import subprocess
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

WORKER = """
import os, sys, json
sys.path.insert(0, %r)
import bench
rank, world, local = bench.dist_setup(2)
bench.barrier(world)
ms, units = [(10.0, 100.0), (20.0, 300.0)][rank]
value, tot_ms, tot_units = bench.aggregate(world, ms, units)
bench.barrier(world)
if rank == 0:
    print(json.dumps(dict(value=value, ms=tot_ms, units=tot_units, world=world)))
import torch.distributed as dist
dist.destroy_process_group()
"""


def test_two_rank_aggregation_over_gloo(tmp_path):
    import json
    script = tmp_path / "worker.py"
    script.write_text(WORKER % ROOT)
    s = socket.socket(); s.bind(("127.0.0.1", 0)); port = s.getsockname()[1]; s.close()
    env = dict(os.environ, CUDA_VISIBLE_DEVICES="")
    out = subprocess.run([sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "2", "--master-addr", "127.0.0.1",
                          "--master-port", str(port), str(script)], capture_output=True, text=True, env=env, timeout=300)
    assert out.returncode == 0, out.stderr[-2000:]
    line = [l for l in out.stdout.splitlines() if l.startswith("{")][-1]
    r = json.loads(line)
    assert r["world"] == 2 and r["ms"] == 20.0 and r["units"] == 400.0
    assert abs(r["value"] - 400.0 / 0.020) < 1e-6


def test_single_process_aggregate_is_identity():
    sys.path.insert(0, ROOT)
    import bench
    v, ms, units = bench.aggregate(1, 5.0, 50.0)
    assert (v, ms, units) == (50.0 / 0.005, 5.0, 50.0)
