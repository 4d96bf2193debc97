"""The N>1 path of bench.py is "replicas only": independent solves, with a barrier and a
max/sum over ranks for timing.  Covered here with world_size 2 on the gloo backend (CPU)."""
import os
import socket
import subprocess
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

WORKER = r"""
import json, os, sys
sys.path.insert(0, os.environ["PS_ROOT"])
from paper_2104_01636_b200 import replicas, workload
r = replicas.init(backend="gloo")
w = workload.make_config(1, seed_offset=replicas.seed_offset(r))
replicas.barrier(r)
value, units, secs = replicas.aggregate_throughput(r, float(w.cells * (r.rank + 1)), 1.0 + r.rank)
mx = replicas.reduce_scalars(r, [float(r.rank)], "max")[0]
print(json.dumps({"rank": r.rank, "world": r.world, "seed": w.seed, "value": value,
                  "units": units, "secs": secs, "max": mx, "rhs0": float(w.rhs.flat[0])}))
replicas.finalize(r)
"""


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def test_two_replicas_gloo(tmp_path):
    import json
    script = tmp_path / "worker.py"
    script.write_text(WORKER)
    port = _free_port()
    procs = []
    for rank in range(2):
        env = dict(os.environ, RANK=str(rank), LOCAL_RANK=str(rank), WORLD_SIZE="2",
                   MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), PS_ROOT=ROOT)
        procs.append(subprocess.Popen([sys.executable, str(script)], env=env,
                                      stdout=subprocess.PIPE, stderr=subprocess.PIPE, text=True))
    outs = []
    for p in procs:
        out, err = p.communicate(timeout=180)
        assert p.returncode == 0, err
        outs.append(json.loads(out.strip().splitlines()[-1]))
    outs.sort(key=lambda o: o["rank"])
    cells = 32 * 32 * 64
    assert [o["world"] for o in outs] == [2, 2]
    assert outs[0]["seed"] + 1000 == outs[1]["seed"]            # distinct workloads per replica
    assert outs[0]["rhs0"] != outs[1]["rhs0"]
    for o in outs:                                              # sum of units / max of time
        assert o["units"] == cells * 3.0 and o["secs"] == 2.0 and o["value"] == cells * 1.5
        assert o["max"] == 1.0


def test_single_process_identity():
    from paper_2104_01636_b200 import replicas
    env = {k: os.environ.pop(k) for k in ("WORLD_SIZE", "RANK", "LOCAL_RANK") if k in os.environ}
    try:
        r = replicas.init()
        assert r.world == 1 and r.backend is None
        assert replicas.reduce_scalars(r, [1.0, 2.0], "max") == [1.0, 2.0]
        assert replicas.aggregate_throughput(r, 10.0, 2.0) == (5.0, 10.0, 2.0)
        replicas.barrier(r)
    finally:
        os.environ.update(env)
