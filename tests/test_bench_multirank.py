"""N > 1 path of bench.py on CPU: world_size-2 gloo run of the rank aggregation (max time, summed
units) and of the reference arm's rank gating (rank 0 prints one JSON line, other ranks exit 0)."""
import json
import os
import subprocess
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

_WORKER = r"""
import os, sys, json
sys.path.insert(0, {root!r})
import torch.distributed as dist
import bench
dist.init_process_group("gloo")
rank = dist.get_rank(); world = dist.get_world_size()
ms = bench.aggregate_max(10.0 + 5.0 * rank, world)       # rank 1 is the slow one
units = bench.aggregate_sum(1000.0 * (rank + 1), world)
sys.stdout.write(json.dumps({{"rank": rank, "ms": ms, "units": units}}) + "\n")   # one write: ranks share the pipe
sys.stdout.flush()
dist.barrier()
dist.destroy_process_group()
"""


def _free_port() -> int:
    import socket
    with socket.socket() as s:      # a fixed port collides with a run that has just ended (TIME_WAIT)
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _torchrun(args, timeout=300):
    env = dict(os.environ, MASTER_ADDR="127.0.0.1", OMP_NUM_THREADS="1")
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node=2",
           "--master-addr", "127.0.0.1", "--master-port", str(_free_port())] + args
    return subprocess.run(cmd, capture_output=True, text=True, timeout=timeout, env=env, cwd=ROOT)


def _json_objects(text):
    """Every JSON object in the output, even if two ranks' lines ran together on the shared pipe."""
    dec, out, i = json.JSONDecoder(), [], 0
    while True:
        i = text.find("{", i)
        if i < 0:
            return out
        try:
            obj, end = dec.raw_decode(text, i)
            out.append(obj)
            i = end
        except json.JSONDecodeError:
            i += 1


def test_aggregation_world_size_2_gloo(tmp_path):
    script = tmp_path / "worker.py"
    script.write_text(_WORKER.format(root=ROOT))
    r = _torchrun([str(script)])
    assert r.returncode == 0, r.stderr[-2000:]
    rows = _json_objects(r.stdout)
    assert len(rows) == 2
    for row in rows:
        assert row["ms"] == 15.0           # max over ranks
        assert row["units"] == 3000.0      # whole-job units


def test_reference_arm_prints_one_line_under_torchrun():
    r = _torchrun([os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2", "--steps", "3",
                   "--warmup", "3"])
    assert r.returncode == 0, r.stderr[-2000:]
    rows = _json_objects(r.stdout)
    assert len(rows) == 1
    line = rows[0]
    assert line["impl"] == "reference" and line["n_gpus"] == 2 and line["unit"] == "atom-steps/s"
    assert line["cpu_baseline"]["kind"] == "oracle" and line["e2e"]["h2d_bytes_per_step"] == 0
    assert line["value"] > 0
