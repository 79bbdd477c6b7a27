"""N > 1 path of bench.py on CPU: world_size 2 over gloo (rank logic only; the GPU work is per-replica and has no
data-path collective -- DESIGN.md section 8)."""
import json
import os
import socket
import subprocess
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

WORKER = r"""
import os, sys, json
sys.path.insert(0, sys.argv[1])
import torch, torch.distributed as dist
import bench
dist.init_process_group("gloo")
rank, world = dist.get_rank(), dist.get_world_size()
ms_local = 10.0 + 5.0 * rank                      # rank 1 is the slow replica
ms = bench.max_over_ranks(ms_local, dist, "cpu")
val = bench.aggregate_value(64 ** 3, 7, world, ms)
dist.barrier()
with open(os.path.join(sys.argv[2], "rank%d.json" % rank), "w") as f:   # a file per rank: two ranks' stdout lines can interleave
    json.dump({"rank": rank, "ms": ms, "value": val}, f)
dist.destroy_process_group()
"""


def free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def torchrun2(args, **kw):
    """world_size-2 launch on 127.0.0.1; a second try on another port if the probed one was taken in between."""
    for attempt in range(3):
        cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "2", "--master-addr", "127.0.0.1",
               "--master-port", str(free_port())] + args
        r = subprocess.run(cmd, capture_output=True, text=True, **kw)
        if r.returncode == 0 or "in use" not in r.stderr:
            break
    return r


def test_max_over_ranks_and_aggregate_world2(tmp_path):
    script = tmp_path / "worker.py"
    script.write_text(WORKER)
    r = torchrun2([str(script), ROOT, str(tmp_path)], timeout=300)
    assert r.returncode == 0, r.stderr[-2000:]
    rows = [json.loads((tmp_path / ("rank%d.json" % k)).read_text()) for k in range(2)]
    assert sorted(x["rank"] for x in rows) == [0, 1]
    for x in rows:
        assert x["ms"] == 15.0                                    # max over ranks, on every rank
        assert abs(x["value"] - 2 * 64 ** 3 * 7 / 15.0e-3) < 1e-3


def test_reference_arm_prints_on_rank0_only():
    r = torchrun2([os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2", "--steps", "20", "--warmup", "1"],
                  timeout=600, cwd=ROOT)
    assert r.returncode == 0, r.stderr[-2000:]
    lines = [json.loads(l) for l in r.stdout.splitlines() if l.startswith("{")]
    assert len(lines) == 1
    d = lines[0]
    assert d["impl"] == "reference" and d["cpu_baseline"]["kind"] == "oracle" and d["value"] > 0
    assert d["e2e"]["h2d_bytes_per_step"] == 0 and d["n_gpus"] == 2 and d["unit"] == "cell-updates/s"
