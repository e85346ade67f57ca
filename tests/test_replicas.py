"""The N > 1 path (replicas only), on the CPU with world_size-2 gloo."""
from __future__ import annotations

import os
import socket
import subprocess
import sys

import pytest

from paper_1004_0014_b200 import replicas

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

_WORKER = r"""
import os, sys, json
sys.path.insert(0, sys.argv[1])
from paper_1004_0014_b200 import replicas
rank, local_rank, world = replicas.env_rank_world()
dist = replicas.init_process_group("gloo")
assert dist is not None and dist.get_world_size() == world == 2
ids = replicas.frame_block(rank, world, 5, 358, 360)
replicas.barrier(dist)
mx = replicas.max_over_ranks(dist, 10.0 + rank)
sm = replicas.sum_over_ranks(dist, 100 * (rank + 1))
replicas.barrier(dist)
print(json.dumps({"rank": rank, "ids": ids, "max": mx, "sum": sm}), flush=True)
dist.destroy_process_group()
"""


def _free_port() -> int:
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def test_frame_blocks_are_contiguous_disjoint_and_wrap():
    blocks = [replicas.frame_block(r, 4, 6, 350, 360) for r in range(4)]
    flat = [i for b in blocks for i in b]
    assert flat == [(350 + i) % 360 for i in range(24)]
    assert len(set(flat)) == 24
    assert replicas.frame_block(0, 1, 3, 60, 360) == [60, 61, 62]
    with pytest.raises(ValueError):
        replicas.frame_block(2, 2, 3, 0, 360)


def test_single_process_needs_no_process_group():
    env = {k: v for k, v in os.environ.items() if k not in ("RANK", "WORLD_SIZE", "LOCAL_RANK")}
    out = subprocess.run([sys.executable, "-c",
                          "import sys; sys.path.insert(0, sys.argv[1]);"
                          "from paper_1004_0014_b200 import replicas as r;"
                          "d = r.init_process_group('gloo'); assert d is None; r.barrier(d);"
                          "assert r.max_over_ranks(d, 3.5) == 3.5 and r.sum_over_ranks(d, 7) == 7.0; print('ok')",
                          ROOT], env=env, capture_output=True, text=True, timeout=120)
    assert out.returncode == 0 and "ok" in out.stdout, out.stderr


def test_two_replicas_over_gloo():
    import json
    port = _free_port()
    procs = []
    for rank in range(2):
        env = dict(os.environ, RANK=str(rank), LOCAL_RANK=str(rank), WORLD_SIZE="2", MASTER_ADDR="127.0.0.1",
                   MASTER_PORT=str(port))
        procs.append(subprocess.Popen([sys.executable, "-c", _WORKER, ROOT], env=env, stdout=subprocess.PIPE,
                                      stderr=subprocess.PIPE, text=True))
    res = {}
    for p in procs:
        out, err = p.communicate(timeout=180)
        assert p.returncode == 0, err
        d = json.loads(out.strip().splitlines()[-1])
        res[d["rank"]] = d
    assert res[0]["ids"] == [358, 359, 0, 1, 2] and res[1]["ids"] == [3, 4, 5, 6, 7]
    for r in (0, 1):
        assert res[r]["max"] == 11.0 and res[r]["sum"] == 300.0
