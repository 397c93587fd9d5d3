"""NEXT-4 host logic on CPU (gloo): slab split, neighbour map, the halo exchange pairing and the max-reduction
of DistComm with world_size 2 and 3 — the same code path NCCL runs on GPUs."""
import os
import socket
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_split_and_neighbours():
    from paper_2509_08971_b200 import sharded
    assert sharded.split_z(37, 3) == [(0, 13), (13, 25), (25, 37)]
    assert sharded.split_z(896, 8)[-1] == (784, 896)
    assert sharded.neighbours(0, 4, True) == (3, 1) and sharded.neighbours(0, 4, False) == (None, 1)
    assert sharded.neighbours(3, 4, True) == (2, 0) and sharded.neighbours(3, 4, False) == (2, None)
    assert sharded.neighbours(0, 1, True) == (0, 0) and sharded.neighbours(0, 1, False) == (None, None)


_WORKER = r"""
import sys
sys.path.insert(0, %r)
import torch, torch.distributed as dist
from paper_2509_08971_b200 import sharded
rank, world, port = int(sys.argv[1]), int(sys.argv[2]), sys.argv[3]
dist.init_process_group("gloo", init_method="tcp://127.0.0.1:" + port, rank=rank, world_size=world)
for periodic in (True, False):
    comm = sharded.DistComm(periodic)
    lo, hi = sharded.neighbours(rank, world, periodic)
    assert (comm.lo, comm.hi) == (lo, hi)
    send_low = torch.full((6,), 10.0 * rank + 1.0, dtype=torch.float64)     # my lowest planes
    send_high = torch.full((6,), 10.0 * rank + 2.0, dtype=torch.float64)    # my highest planes
    recv_low = torch.full((6,), -1.0, dtype=torch.float64)
    recv_high = torch.full((6,), -1.0, dtype=torch.float64)
    comm.exchange(send_low, send_high, recv_low, recv_high)
    # my low ghosts hold the lower neighbour's highest planes, my high ghosts the upper neighbour's lowest
    assert torch.all(recv_low == (10.0 * lo + 2.0 if lo is not None else -1.0)), (rank, periodic, recv_low)
    assert torch.all(recv_high == (10.0 * hi + 1.0 if hi is not None else -1.0)), (rank, periodic, recv_high)
    lam = torch.tensor([1.0 + rank], dtype=torch.float64)
    comm.allreduce_max(lam)
    assert lam.item() == float(world)
dist.barrier()
dist.destroy_process_group()
print("ok", rank)
"""


@pytest.mark.parametrize("world", [2, 3])
def test_halo_exchange_and_max_reduction_gloo(tmp_path, world):
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    port = s.getsockname()[1]
    s.close()
    script = tmp_path / "worker.py"
    script.write_text(_WORKER % ROOT)
    procs = [subprocess.Popen([sys.executable, str(script), str(r), str(world), str(port)], stdout=subprocess.PIPE,
                              stderr=subprocess.STDOUT, text=True) for r in range(world)]
    outs = [p.communicate(timeout=300)[0] for p in procs]
    for r, (p, o) in enumerate(zip(procs, outs)):
        assert p.returncode == 0 and ("ok %d" % r) in o, o


def test_bench_shard_reaches_the_communicator_setup_on_cpu():
    """`bench.py --shard --gpus 2` launched the way the driver launches it (torchrun, one process per rank): on this
    GPU-less box the arguments parse, both ranks bring the communicator up (gloo), build the z-slab neighbour map,
    and only then stop because there is no CUDA device (exit code 3, no CPU fallback)."""
    import torch
    if torch.cuda.is_available():
        pytest.skip("needs a box without a GPU")
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    port = s.getsockname()[1]
    s.close()
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "2", "--master-addr", "127.0.0.1",
           "--master-port", str(port), os.path.join(ROOT, "bench.py"), "--gpus", "2", "--shard", "--steps", "1", "--warmup", "0"]
    out = subprocess.run(cmd, capture_output=True, text=True, timeout=600)
    text = out.stdout + out.stderr
    assert out.returncode != 0
    for r, nb, slab in ((0, (1, 1), (0, 448)), (1, (0, 0), (448, 896))):
        assert ("communicator up: world 2, backend gloo, rank %d, z-slab neighbours %s, slab %s of nz=896" % (r, nb, slab)) in text, text[-2000:]
    assert "no CPU fallback" in text
