"""NEXT-2: reflecting walls (G17) and the non-radiative Kelvin-Helmholtz workload
(G18).  Pins of the oracle's reflecting ghost fill: a closed box is the mirror-periodic
doubled domain bit for bit; walls conserve mass and energy and hold a gas at rest exactly."""
import math

import numpy as np
import pytest

import oracle
from paper_2509_08971_b200 import workloads as wl


def _run(state, n, bc, scheme, sp, nsteps, cfl=0.4, gamma=1.4):
    o = oracle.Oracle(*n, gamma, bc, scheme=scheme, spacing=sp)
    o.set_state(*state)
    o.step(cfl, nsteps)
    out = o.get_state()
    o.close()
    return out


def _mirror_extend(state, axis):
    """Append the mirror image along spatial `axis` (momentum component `axis` negated)."""
    ax_np = 2 - axis
    out = []
    for f, a in enumerate(state):
        m = np.flip(a, ax_np)
        if f == 1 + axis:
            m = -m
        out.append(np.ascontiguousarray(np.concatenate([a, m], axis=ax_np)))
    return out


@pytest.mark.parametrize("scheme", [0, 1])
def test_reflecting_box_equals_mirror_periodic_domain_bitwise(scheme):
    n = (9, 7, 8)
    sp = (0.1, 0.07, 0.13)
    st = wl.random_state(n, seed=31)
    out = _run(st, n, wl.BC_REFLECT, scheme, sp, nsteps=4)
    big = st
    for axis in range(3):
        big = _mirror_extend(big, axis)
    n2 = tuple(2 * x for x in n)
    out2 = _run(big, n2, wl.BC_PERIODIC, scheme, sp, nsteps=4)
    for f in range(5):
        assert np.array_equal(out2[f][:n[2], :n[1], :n[0]], out[f])
    assert any(not np.array_equal(out[f], st[f]) for f in range(5))


@pytest.mark.parametrize("scheme", [0, 1])
def test_reflecting_walls_conserve_mass_energy_and_hold_gas_at_rest(scheme):
    n = (10, 8, 1)
    st = wl.random_state(n, seed=32)
    out = _run(st, n, wl.BC_REFLECT, scheme, (0.1, 0.1, 1.0), nsteps=10)
    for f in (0, 4):
        ref = math.fsum(st[f].ravel().tolist())
        assert abs(math.fsum(out[f].ravel().tolist()) - ref) <= 1e-13 * abs(ref)
    g = 1.4
    rest = [np.full((1, 8, 10), v) for v in (1.2, 0.0, 0.0, 0.0, 0.7 / (g - 1))]
    out = _run(rest, n, wl.BC_REFLECT, scheme, (0.1, 0.1, 1.0), nsteps=5)
    for f in range(5):
        assert np.array_equal(out[f], rest[f])


@pytest.mark.parametrize("scheme", [0, 1])
def test_kelvin_helmholtz_workload(scheme):
    """two layers rho = 1 / 2.5, v_x = +-0.5; conservation on the periodic box and growth of
    the transverse kinetic energy seeded by the perturbation (the instability develops)."""
    w = wl.kelvin_helmholtz(64, nsteps=1200)
    rho0 = w.state[0]
    assert set(np.unique(rho0)) == {1.0, 2.5}
    assert float(np.mean(rho0 == 2.5)) == 0.5                 # layer |y| <= 0.25 is half the box
    u0 = w.state[1] / rho0
    assert np.all(u0[rho0 == 2.5] == -0.5) and np.all(u0[rho0 == 1.0] == 0.5)
    out = _run(w.state, w.n, w.bc, scheme, w.spacing, nsteps=1200, cfl=w.cfl, gamma=w.gamma)     # t ~ 3.1
    for f in (0, 1, 2, 4):
        ref = math.fsum(w.state[f].ravel().tolist())
        scale = math.fsum(np.abs(w.state[f]).ravel().tolist())
        assert abs(math.fsum(out[f].ravel().tolist()) - ref) <= 1e-13 * scale
    assert np.all(out[3] == 0.0)
    ke_y0 = float(np.sum(w.state[2] ** 2 / rho0))
    ke_y1 = float(np.sum(out[2] ** 2 / out[0]))
    assert ke_y1 > 20.0 * ke_y0            # measured: x2000 (A), x100 (B, more diffusive) at 64^2
