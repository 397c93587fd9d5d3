"""NEXT-3: the pointwise radiative heating / cooling source q = c kappa rho (E_rad - a T^4)
(eq.6; d_t e = q, d_t E_rad = -q, eq.4), operator-split after the advection step
(P:66), backward Euler (reading G20).  Pins: the paper's heating and cooling cases against an
ODE solver, the equilibrium temperature, exact energy conservation, a one-step independent root."""
import numpy as np
import pytest
from scipy.integrate import solve_ivp
from scipy.optimize import brentq

import oracle
from paper_2509_08971_b200 import workloads as wl

# cgs constants and the parameters of P:211
C_LIGHT, A_RAD, K_B, M_P = 2.99792458e10, 7.5657e-15, 1.380649e-16, 1.67262192e-24
GAMMA, RHO, MU, KAPPA, T_RAD0 = 5.0 / 3.0, 1e-7, 0.6, 0.4, 3.4e6
CV = K_B / ((GAMMA - 1.0) * MU * M_P)              # T = e / (rho cv)


def _setup(T0, n=(4, 1, 1), vel=(0.0, 0.0, 0.0)):
    e0 = RHO * CV * T0
    shape = n[::-1]
    E = e0 + 0.5 * RHO * sum(v * v for v in vel)
    st = [np.full(shape, x) for x in (RHO, RHO * vel[0], RHO * vel[1], RHO * vel[2], E)]
    o = oracle.Oracle(*n, GAMMA, wl.BC_PERIODIC, scheme=0, spacing=(1.0, 1.0, 1.0), radiation=True)
    o.set_source(KAPPA, C_LIGHT, A_RAD, CV)
    o.set_state(*st)
    o.set_rad_energy(np.full(shape, A_RAD * T_RAD0 ** 4))
    return o, e0, A_RAD * T_RAD0 ** 4


def _e_of(o, vel=(0.0, 0.0, 0.0)):
    s = o.get_state()
    return float(s[4].ravel()[0] - 0.5 * RHO * sum(v * v for v in vel))


def _rhs(t, y, etot):
    return [C_LIGHT * KAPPA * RHO * (etot - y[0] - A_RAD * (y[0] / (RHO * CV)) ** 4)]


@pytest.mark.parametrize("T0", [11.0, 1.1e9])          # heating and cooling cases
def test_heating_cooling_against_ode_solver_first_order(T0):
    t_end = 2e-7 if T0 < 1e6 else 2e-10               # a few e-folding times of each case
    ref = None
    errs = []
    for nsteps in (100, 200, 400, 800):
        o, e0, er0 = _setup(T0)
        if ref is None:
            sol = solve_ivp(_rhs, (0.0, t_end), [e0], args=(e0 + er0,), method="Radau", rtol=1e-12, atol=1e-6 * e0)
            ref = sol.y[0, -1]
        o.step_dt(t_end / nsteps, nsteps)
        e = _e_of(o)
        er = float(o.get_rad_energy().ravel()[0])
        assert abs((e + er) - (e0 + er0)) <= 4e-16 * nsteps * (e0 + er0)       # e + E_rad conserved
        errs.append(abs(e - ref) / abs(ref))
        o.close()
    assert errs[0] < 0.05 and errs[-1] < errs[0] / 6          # converges ...
    ratios = np.array(errs[:-1]) / np.array(errs[1:])
    assert np.all(ratios > 1.7) and 1.8 < ratios[-1] < 2.2    # ... at first order (backward Euler)


@pytest.mark.parametrize("T0", [11.0, 1.1e9])
def test_equilibrium_temperature(T0):
    """'the fluid eventually equilibrates to the radiation temperature': a T^4 + rho cv T = E_tot."""
    o, e0, er0 = _setup(T0)
    o.step_dt(1e-5, 40)
    T = _e_of(o) / (RHO * CV)
    Teq = brentq(lambda x: A_RAD * x ** 4 + RHO * CV * x - (e0 + er0), 1.0, 1e10, xtol=1e-6, rtol=1e-15)
    assert abs(T - Teq) <= 1e-9 * Teq
    assert abs(Teq - T_RAD0) <= 0.01 * T_RAD0          # radiation dominated: E_rad stays nearly constant
    o.close()


def test_one_backward_euler_step_is_the_root_of_its_equation():
    vel = (3.0e5, -1.0e5, 2.0e5)
    o, e0, er0 = _setup(2.0e5, vel=vel)
    dt = 3e-8
    o.step_dt(dt, 1)
    beta = dt * C_LIGHT * KAPPA * RHO
    g = lambda x: (x - e0) - beta * ((e0 + er0 - x) - A_RAD * (x / (RHO * CV)) ** 4)
    root = brentq(g, 0.0, e0 + er0, xtol=1e-300, rtol=1e-15)
    assert abs(_e_of(o, vel) - root) <= 1e-13 * root
    s = o.get_state()
    for f, v in zip((0, 1, 2, 3), (RHO, RHO * vel[0], RHO * vel[1], RHO * vel[2])):
        assert np.all(s[f] == v)                        # density and momenta untouched
    o.close()


def test_zero_opacity_is_a_no_op():
    n = (6, 5, 4)
    st = wl.random_state(n, seed=51)
    er = 1.0 + np.random.default_rng(1).random(n[::-1])
    outs = []
    for kappa in (None, 0.0):
        o = oracle.Oracle(*n, 1.4, wl.BC_PERIODIC, scheme=1, spacing=(0.1, 0.1, 0.1), radiation=True)
        if kappa is not None:
            o.set_source(kappa, 1.0, 1.0, 1.0)
        o.set_state(*st)
        o.set_rad_energy(er)
        o.step(0.4, 3)
        outs.append(o.get_state() + [o.get_rad_energy()])
        o.close()
    for a, b in zip(*outs):
        assert np.abs(a - b).max() <= 1e-13 * np.abs(a).max()      # (E - ke) + ke rounds once per step
