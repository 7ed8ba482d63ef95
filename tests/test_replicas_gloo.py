"""The N > 1 path of bench.py on CPU: world_size-2 gloo process group, one process per (pretend) GPU.  The overlap path
does not shard (replicas only), so what is covered is the plumbing every rank runs: rank discovery from
the torchrun environment, per-rank right-hand sides, barrier + MAX-over-ranks timing and the whole-job rate."""
import os
import socket
import subprocess
import sys
import textwrap

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

WORKER = textwrap.dedent("""
    import json, os, sys
    sys.path.insert(0, %r)
    import numpy as np
    import torch.distributed as dist
    from paper_1510_06897_b200 import inputs, replicas
    rank, local, world = replicas.world()
    dist.init_process_group("gloo")
    assert dist.get_rank() == rank and dist.get_world_size() == world == 2
    dist.barrier()
    psi = inputs.gaussian_spinor((2, 2, 2, 2), 7 + 1000 * replicas.rhs_seed_offset(rank))
    ms_local = 10.0 * (rank + 1)              # rank 1 is the slow one
    rate, ms = replicas.aggregate_rate(3.0, ms_local, world, dist, "cpu")
    dist.barrier()
    print(json.dumps({"rank": rank, "local": local, "rate": rate, "ms": ms, "psi0": [psi.ravel()[0].real, psi.ravel()[0].imag]}))
    dist.destroy_process_group()
""") % ROOT


def free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def test_two_rank_gloo_replicas(tmp_path):
    script = tmp_path / "worker.py"
    script.write_text(WORKER)
    port = free_port()
    procs = []
    for r in range(2):
        env = dict(os.environ, RANK=str(r), LOCAL_RANK=str(r), WORLD_SIZE="2", MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
        procs.append(subprocess.Popen([sys.executable, str(script)], env=env, stdout=subprocess.PIPE, stderr=subprocess.PIPE, text=True))
    outs = []
    for p in procs:
        o, e = p.communicate(timeout=240)
        assert p.returncode == 0, e[-2000:]
        outs.append(__import__("json").loads(o.strip().splitlines()[-1]))
    outs.sort(key=lambda d: d["rank"])
    assert [d["rank"] for d in outs] == [0, 1] and [d["local"] for d in outs] == [0, 1]
    # the job took the slowest rank's time; both ranks agree on it and on the whole-job rate
    assert outs[0]["ms"] == outs[1]["ms"] == 20.0
    assert outs[0]["rate"] == outs[1]["rate"] == 2 * 3.0 / 20e-3
    # independent right-hand sides per replica
    assert outs[0]["psi0"] != outs[1]["psi0"]


def test_single_process_defaults(monkeypatch):
    from paper_1510_06897_b200 import replicas
    for k in ("RANK", "LOCAL_RANK", "WORLD_SIZE"):
        monkeypatch.delenv(k, raising=False)
    assert replicas.world() == (0, 0, 1)
    assert replicas.aggregate_rate(5.0, 250.0, 1) == (20.0, 250.0)
    assert replicas.rhs_seed_offset(0) == 0
