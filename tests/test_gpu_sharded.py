"""NEXT-4: z-slab sharding, all ranks emulated in one process on one GPU (phases in lockstep, no kernel waits
on another rank).  A sharded run must reproduce the single-domain run BIT FOR BIT: every cell sees the same
stencil values and the same dt (lambda is max-reduced exactly)."""
import os
import socket
import subprocess
import sys

import numpy as np
import pytest

from paper_2509_08971_b200 import hard, sharded
from paper_2509_08971_b200 import workloads as wl

pytestmark = pytest.mark.gpu


@pytest.mark.parametrize("scheme", [0, 1])
@pytest.mark.parametrize("world", [2, 3])
@pytest.mark.parametrize("bc", [wl.BC_PERIODIC, wl.BC_OUTFLOW, wl.BC_REFLECT])
def test_sharded_equals_single_domain_bitwise(scheme, world, bc):
    n = (40, 33, 37)
    sp = (0.1, 0.07, 0.13)
    st = wl.random_state(n, seed=90 + world)
    h = hard.Hard(*n, 1.4, bc, scheme=scheme, spacing=sp)
    h.set_state(*st)
    h.step(0.4, 5)
    ref = h.get_state()
    dt_ref = h.max_dt()
    h.close()
    grp = sharded.LocalGroup(n, 1.4, bc, world, scheme=scheme, spacing=sp)
    grp.set_state(st)
    grp.step(0.4, 5)
    out = grp.get_state()
    for f in range(5):
        assert np.array_equal(out[f], ref[f])
    assert grp.max_dt() == dt_ref
    assert [s.k1 - s.k0 for s in grp.slabs] == [b - a for a, b in sharded.split_z(n[2], world)]
    grp.close()


def test_sharded_turbulence_matches_oracle():
    import oracle
    w = wl.turbulence(32, nsteps=10)
    o = oracle.Oracle(*w.n, w.gamma, w.bc, spacing=w.spacing)
    o.set_state(*w.state)
    o.step(w.cfl, 10)
    ref = o.get_state()
    grp = sharded.LocalGroup(w.n, w.gamma, w.bc, 4, spacing=w.spacing)
    grp.set_state(w.state)
    grp.step(w.cfl, 10)
    out = grp.get_state()
    for a, b in zip(out, ref):
        assert np.abs(a - b).max() <= 1e-9 * np.abs(b).max()
    grp.close()
    o.close()


# ---------------------------------------------------------------- the real classes, real processes
_RANK = r"""
import sys
sys.path.insert(0, %r)
import numpy as np, torch, torch.distributed as dist
from paper_2509_08971_b200 import hard, sharded
from paper_2509_08971_b200 import workloads as wl
rank, world, port, out = int(sys.argv[1]), int(sys.argv[2]), sys.argv[3], sys.argv[4]
torch.cuda.set_device(0)                                   # every rank shares the one GPU
dist.init_process_group("gloo", init_method="tcp://127.0.0.1:" + port, rank=rank, world_size=world)
n, sp = (40, 33, 37), (0.1, 0.07, 0.13)
res = {}
for scheme in (0, 1):
    for bc in (wl.BC_PERIODIC, wl.BC_OUTFLOW):
        st = wl.random_state(n, seed=90 + world)
        sh = sharded.ShardedHard(n, 1.4, bc, scheme=scheme, spacing=sp)
        assert type(sh.comm) is sharded.HostStagedComm and sh.comm.world == world
        sh.set_state(st)
        sh.step(0.4, 5)
        fields = sh.get_state()
        res["f_%%d_%%d" %% (scheme, bc)] = np.stack(fields)
        res["dt_%%d_%%d" %% (scheme, bc)] = np.array([sh.max_dt(), sh.slab.k0, sh.slab.k1])
        sh.close()
np.savez(out + ".%%d.npz" %% rank, **res)
dist.barrier()
dist.destroy_process_group()
print("ok", rank)
"""


@pytest.mark.parametrize("world", [2, 3])
def test_sharded_hard_class_with_real_processes_on_one_gpu(tmp_path, world):
    """`ShardedHard` + `DistComm`'s pairing code driven by `world` real processes (gloo, halos staged through pinned
    host memory by `HostStagedComm`, all ranks time-sharing the one GPU; no kernel waits on another rank): five steps
    must equal the single-domain run bit for bit, dt included — periodic and outflow, both schemes."""
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    port = s.getsockname()[1]
    s.close()
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    script = tmp_path / "rank.py"
    script.write_text(_RANK % root)
    out = str(tmp_path / "res")
    procs = [subprocess.Popen([sys.executable, str(script), str(r), str(world), str(port), out], stdout=subprocess.PIPE,
                              stderr=subprocess.STDOUT, text=True) for r in range(world)]
    outs = [p.communicate(timeout=900)[0] for p in procs]
    for r, (p, o) in enumerate(zip(procs, outs)):
        assert p.returncode == 0 and ("ok %d" % r) in o, o
    parts = [np.load(out + ".%d.npz" % r) for r in range(world)]
    n, sp = (40, 33, 37), (0.1, 0.07, 0.13)
    for scheme in (0, 1):
        for bc in (wl.BC_PERIODIC, wl.BC_OUTFLOW):
            st = wl.random_state(n, seed=90 + world)
            h = hard.Hard(*n, 1.4, bc, scheme=scheme, spacing=sp)
            h.set_state(*st)
            h.step(0.4, 5)
            ref, dt_ref = h.get_state(), h.max_dt()
            h.close()
            key = "_%d_%d" % (scheme, bc)
            got = np.concatenate([p["f" + key] for p in parts], axis=1)        # (field, z, y, x): slabs stacked along z
            for f in range(5):
                assert np.array_equal(got[f], ref[f]), (scheme, bc, f)
            assert all(p["dt" + key][0] == dt_ref for p in parts)
            assert [(int(p["dt" + key][1]), int(p["dt" + key][2])) for p in parts] == sharded.split_z(n[2], world)
