"""The N > 1 path of bench.py is "replicas only": its host logic -- per-rank key and
seed, barrier, max-over-ranks of the time, whole-job aggregate, rank-0-only output -- run here with two
processes over the gloo backend on CPU."""
import json
import os
import socket
import subprocess
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

WORKER = r"""
import json, os, sys
sys.path.insert(0, %(root)r)
from paper_2602_23067_b200 import replicas
rank, local, world = replicas.rank_env()
assert replicas.init("gloo") == 2 and world == 2
key = replicas.replica_key(bytes(range(32)), rank)
replicas.barrier()
my_ms = 10.0 + 5.0 * rank                      # rank 1 is the slow one
slowest = replicas.max_over_ranks(my_ms)
agg = replicas.aggregate_gbs(1 << 30, 4, slowest, world)
replicas.barrier()
if rank == 0:
    print(json.dumps({"slowest": slowest, "agg": agg, "key0": key.hex(), "seed": replicas.replica_seed(1005, rank)}))
else:
    assert key != bytes(range(32)) and key == bytes(b ^ 1 for b in range(32))
    assert replicas.replica_seed(1005, rank) == 1006
replicas.finish()
"""


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    port = s.getsockname()[1]
    s.close()
    return port


def test_two_rank_replicas_over_gloo(tmp_path):
    script = tmp_path / "worker.py"
    script.write_text(WORKER % {"root": ROOT})
    port = _free_port()
    procs = []
    for rank in range(2):
        env = dict(os.environ, RANK=str(rank), LOCAL_RANK=str(rank), WORLD_SIZE="2",
                   MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
        procs.append(subprocess.Popen([sys.executable, str(script)], env=env, stdout=subprocess.PIPE,
                                      stderr=subprocess.PIPE, text=True))
    outs = [p.communicate(timeout=240) for p in procs]
    for p, (out, err) in zip(procs, outs):
        assert p.returncode == 0, err[-2000:]
    assert outs[1][0].strip() == ""                       # only rank 0 prints
    line = json.loads(outs[0][0].strip().splitlines()[-1])
    assert line["slowest"] == 15.0                        # the max over ranks, not rank 0's own 10 ms
    assert abs(line["agg"] - 2 * 4 * (1 << 30) / 15e-3 / 1e9) < 1e-6
    assert line["key0"] == bytes(range(32)).hex() and line["seed"] == 1005


def test_single_process_defaults():
    sys.path.insert(0, ROOT)
    from paper_2602_23067_b200 import replicas
    for k in ("RANK", "LOCAL_RANK", "WORLD_SIZE"):
        assert k not in os.environ or os.environ[k] in ("0", "1")
    assert replicas.max_over_ranks(3.5) == 3.5
    assert replicas.replica_key(b"\x01\x02", 0) == b"\x01\x02"
    assert replicas.aggregate_gbs(10 ** 9, 2, 1000.0, 1) == 2.0
