"""N > 1 path of bench.py on CPU: world_size-2 gloo (the path does not shard -- "replicas only", DESIGN.md section 6 --
so the only cross-rank step is the max-over-ranks of the locally measured time; there is no collective on the data path)."""
import os
import socket
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

WORKER = r"""
import json, os, sys
sys.path.insert(0, {root!r})
import torch.distributed as dist
import bench
dist.init_process_group("gloo")
rank, world = dist.get_rank(), dist.get_world_size()
local = 2.0 if rank == 0 else 3.5            # rank 1 is the slow replica
t = bench.max_over_ranks(local, world, "cpu")
v = bench.job_value(1 << 20, 1000, 4, world, t)
print(json.dumps({{"rank": rank, "t": t, "v": v}}), flush=True)
dist.destroy_process_group()
"""


def _free_port() -> int:
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def test_max_over_ranks_single_process_is_identity():
    sys.path.insert(0, ROOT)
    import bench
    assert bench.max_over_ranks(1.25, 1) == 1.25
    assert bench.job_value(1 << 10, 100, 2, 1, 0.5) == pytest.approx((1 << 10) * 100 * 2 / 0.5 / 1e9)


def test_world_size_2_gloo_takes_slowest_rank_and_counts_all_replicas(tmp_path):
    script = tmp_path / "worker.py"
    script.write_text(WORKER.format(root=ROOT))
    port = _free_port()
    procs = []
    for rank in range(2):
        env = dict(os.environ, RANK=str(rank), LOCAL_RANK=str(rank), WORLD_SIZE="2", MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
        procs.append(subprocess.Popen([sys.executable, str(script)], env=env, stdout=subprocess.PIPE, stderr=subprocess.PIPE, text=True))
    outs = []
    for p in procs:
        out, err = p.communicate(timeout=120)
        assert p.returncode == 0, err
        outs.append(out.strip().splitlines()[-1])
    import json
    rows = sorted((json.loads(o) for o in outs), key=lambda r: r["rank"])
    for r in rows:
        assert r["t"] == 3.5                                          # both ranks see the slowest replica's time
        assert r["v"] == pytest.approx(2 * (1 << 20) * 1000 * 4 / 3.5 / 1e9)   # 2 replicas' units / max time


def test_reference_arm_runs_on_rank0_only(tmp_path):
    """`bench.py --impl reference` under torchrun: rank 0 alone prints the line, the other ranks exit 0 without work."""
    env = dict(os.environ, RANK="1", LOCAL_RANK="1", WORLD_SIZE="2", MASTER_ADDR="127.0.0.1", MASTER_PORT=str(_free_port()))
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2", "--steps", "1", "--warmup", "0"],
                       env=env, capture_output=True, text=True, timeout=120)
    assert r.returncode == 0 and r.stdout.strip() == ""
