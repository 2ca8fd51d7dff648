"""Multi-GPU host logic (replicas only) on CPU: world_size-2 gloo process group.

The data path has no collective; what N > 1 adds is bookkeeping -- which independent batches a rank owns, the
max-over-ranks step time, the whole-job unit count and the concatenation of per-sample integer observables --
and that bookkeeping is what runs here, in two real processes over gloo on 127.0.0.1.
"""
import os
import socket
import subprocess
import sys

import numpy as np
import pytest

from paper_1411_5512_b200 import replicas
from paper_1411_5512_b200 import workloads as wl

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

WORKER = r"""
import json, os, sys
sys.path.insert(0, %(root)r)
import numpy as np
from paper_1411_5512_b200 import replicas, workloads as wl
rank, local_rank, ws = replicas.init(backend="gloo")
items = sorted(k for k in wl.CONFIGS if k.startswith("cfg5"))
mine = replicas.shard(items, rank, ws)
seed = replicas.replica_seed(wl.CONFIGS["cfg4"].seed, rank)
replicas.barrier()
t_max = replicas.max_over_ranks(1.5 + rank)           # rank 1 is the slow one
units, t2 = replicas.aggregate_throughput(1000.0 * (rank + 1), 0.25 * (rank + 1))
obs = np.arange(64, dtype=np.int64) + 1000 * rank     # stands for a per-sample observable
allobs = replicas.gather_lanes(obs)
replicas.barrier()
print("RESULT " + json.dumps({"rank": rank, "ws": ws, "mine": mine, "seed": seed, "t_max": t_max, "units": units,
                              "t2": t2, "obs": allobs.tolist()}))
"""


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    port = s.getsockname()[1]
    s.close()
    return port


def test_shard_is_a_partition():
    items = list(range(13))
    for ws in (1, 2, 3, 8):
        parts = [replicas.shard(items, r, ws) for r in range(ws)]
        assert sorted(x for p in parts for x in p) == items
        assert max(len(p) for p in parts) - min(len(p) for p in parts) <= 1
    with pytest.raises(ValueError):
        replicas.shard(items, 2, 2)


def test_single_process_is_the_identity():
    assert replicas.world() == (0, 0, 1) or "RANK" in os.environ
    assert replicas.max_over_ranks(2.5) == 2.5
    assert replicas.sum_over_ranks(3.0) == 3.0
    a = np.arange(64, dtype=np.int64)
    assert np.array_equal(replicas.gather_lanes(a), a[None])
    assert replicas.replica_seed(wl.seed_for(4), 3) == wl.seed_for(4, 3)


def test_two_ranks_over_gloo(tmp_path):
    port = _free_port()
    script = tmp_path / "worker.py"
    script.write_text(WORKER % {"root": ROOT})
    procs = []
    for rank in range(2):
        env = dict(os.environ, RANK=str(rank), LOCAL_RANK=str(rank), WORLD_SIZE="2", MASTER_ADDR="127.0.0.1",
                   MASTER_PORT=str(port), OMP_NUM_THREADS="1")
        procs.append(subprocess.Popen([sys.executable, str(script)], env=env, stdout=subprocess.PIPE,
                                      stderr=subprocess.PIPE, text=True))
    outs = []
    for p in procs:
        out, err = p.communicate(timeout=240)
        assert p.returncode == 0, err[-2000:]
        outs.append(out)
    import json
    res = [json.loads(next(l for l in o.splitlines() if l.startswith("RESULT "))[7:]) for o in outs]
    res.sort(key=lambda r: r["rank"])
    items = sorted(k for k in wl.CONFIGS if k.startswith("cfg5"))
    assert sorted(res[0]["mine"] + res[1]["mine"]) == items and not set(res[0]["mine"]) & set(res[1]["mine"])
    assert res[0]["seed"] + 1 == res[1]["seed"]
    for r in res:
        assert r["ws"] == 2
        assert r["t_max"] == 2.5                    # the slowest rank's time, on every rank
        assert r["units"] == 3000.0 and r["t2"] == 0.5
        got = np.array(r["obs"])
        assert got.shape == (2, 64)
        assert np.array_equal(got[0], np.arange(64)) and np.array_equal(got[1], np.arange(64) + 1000)


def test_bench_reference_arm_other_ranks_exit_quietly():
    """Under torchrun only rank 0 runs the oracle; the other ranks exit 0 without output."""
    env = dict(os.environ, RANK="1", LOCAL_RANK="1", WORLD_SIZE="2", MASTER_ADDR="127.0.0.1", MASTER_PORT="1")
    p = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2",
                        "--steps", "1", "--warmup", "1"], env=env, capture_output=True, text=True, timeout=120)
    assert p.returncode == 0 and p.stdout.strip() == ""


def test_bench_reference_arm_prints_the_contract_line():
    import json
    p = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--config", "cfg2",
                        "--steps", "2", "--warmup", "1"], capture_output=True, text=True, timeout=300)
    assert p.returncode == 0, p.stderr[-2000:]
    d = json.loads(p.stdout.strip().splitlines()[-1])
    assert d["impl"] == "reference" and d["unit"] == "ps/attempt" and d["higher_is_better"] is False
    assert d["cpu_baseline"]["kind"] == "oracle" and d["cpu_baseline"]["cores"] >= 1
    assert d["e2e"]["h2d_bytes_per_step"] == 0 and d["e2e"]["value"] == d["value"] > 0
    assert d["config"]["workload"].startswith("BASELINE.json configs[1]")
