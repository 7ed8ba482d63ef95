"""One process per GPU wiring of the t-split lattice (ovl_slab_*: CUDA IPC halo buffers, interprocess events, shared-memory
round counters), exercised as TWO PROCESSES THAT SHARE ONE GPU -- the only multi-process configuration a one-GPU box
offers.  No kernel waits on another process (ordering is by events and host-side counters), so sharing a GPU is safe."""
import os
import socket
import subprocess
import sys

import pytest

pytestmark = pytest.mark.gpu
ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_two_processes_one_gpu_ipc_split():
    with socket.socket() as sk:
        sk.bind(("127.0.0.1", 0))
        port = sk.getsockname()[1]
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node=2", "--master-addr", "127.0.0.1",
           "--master-port", str(port), os.path.join(ROOT, "tests", "split_ipc_worker.py")]
    res = subprocess.run(cmd, capture_output=True, text=True, timeout=420, cwd=ROOT)
    assert res.returncode == 0, res.stdout[-3000:] + res.stderr[-3000:]
    assert "IPC_SPLIT_OK 2 ranks" in res.stdout, res.stdout[-3000:] + res.stderr[-3000:]
