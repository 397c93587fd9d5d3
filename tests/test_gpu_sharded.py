"""NEXT-4: z-slab sharding, all ranks emulated in one process on one GPU (phases in lockstep, no kernel waits
on another rank).  A sharded run must reproduce the single-domain run BIT FOR BIT: every cell sees the same
stencil values and the same dt (lambda is max-reduced exactly)."""
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
