"""GPU parity (run on the B200 box, -m gpu): CUDA path through the C-ABI vs the oracle, element by
element on the same seeded inputs.  Tolerances are BASELINE.json north_star's: relative L-infinity
1e-12 per field after one step, 1e-9 after 100 steps, dt 1e-14 relative on an identical state."""
import numpy as np
import pytest

from paper_2509_08971_b200 import hard
from paper_2509_08971_b200 import workloads as wl

from _parity import field_errors, run_both

pytestmark = pytest.mark.gpu

TOL_1 = 1e-12
TOL_100 = 1e-9
TOL_DT = 1e-14
SCHEMES = [hard.SCHEME_WENO5Z_HLL, hard.SCHEME_MUSCL_HLLC]
VARIANTS = [hard.VARIANT_FUSED, hard.VARIANT_PERDIR]


def _check(w, scheme, variant, nsteps, tol, **kw):
    g, o, dts, ts, dte = run_both(w, scheme, variant, nsteps=nsteps, **kw)
    assert abs(dts[0] - dts[1]) <= TOL_DT * dts[1], "dt after set_state"
    errs = field_errors(g, o)
    assert max(errs) <= tol, "field errors %s" % (errs,)
    assert abs(ts[0] - ts[1]) <= max(tol, 1e-13) * abs(ts[1])
    assert abs(dte[0] - dte[1]) <= max(10 * tol, 1e-12) * dte[1]
    assert any(np.abs(a - b).max() > 0 for a, b in zip(o, w.state)), "oracle did not move"
    return errs


def _random_workload(n, bc, seed, spacing):
    return wl.Workload("rand", n, 1.4, bc, spacing, 0.4, nsteps=1, state=wl.random_state(n, seed))


@pytest.mark.parametrize("scheme", SCHEMES)
@pytest.mark.parametrize("variant", VARIANTS)
@pytest.mark.parametrize("n,bc", [((37, 21, 19), wl.BC_PERIODIC), ((16, 16, 16), wl.BC_OUTFLOW),
                                  ((50, 33, 1), wl.BC_PERIODIC), ((1, 40, 35), wl.BC_OUTFLOW),
                                  ((131, 1, 1), wl.BC_PERIODIC), ((3, 3, 3), wl.BC_PERIODIC)])
def test_one_step_random_state(scheme, variant, n, bc):
    """several tiles, ragged tails in every direction, inactive directions, the minimum size"""
    w = _random_workload(n, bc, seed=100 + sum(n), spacing=(0.1, 0.07, 0.13))
    _check(w, scheme, variant, 1, TOL_1)


@pytest.mark.parametrize("scheme", SCHEMES)
@pytest.mark.parametrize("bc", [wl.BC_PERIODIC, wl.BC_OUTFLOW])
def test_supersonic_random_state(scheme, bc):
    """Mach 0..2.5 in every direction and both senses (smooth modes + noise): the clamped (one-sided) branches of HLL / HLLC — SL >= 0 and
    SR <= 0 — on most faces, subsonic ones in between."""
    n = (37, 21, 19)
    z, y, x = np.meshgrid((np.arange(n[2]) + 0.5) / n[2], (np.arange(n[1]) + 0.5) / n[1], (np.arange(n[0]) + 0.5) / n[0],
                          indexing="ij")
    rng = np.random.default_rng(314)
    rho = 1.0 + 0.2 * np.sin(2 * np.pi * (x - z)) + 0.05 * (rng.random(x.shape) - 0.5)
    prs = 1.0 + 0.2 * np.cos(2 * np.pi * (y + z)) + 0.05 * (rng.random(x.shape) - 0.5)
    vel = [3.0 * np.sin(2 * np.pi * (x + y)), 3.0 * np.cos(2 * np.pi * (y - z)), 3.0 * np.sin(2 * np.pi * (z + x) + 1.0)]
    E = prs / 0.4 + 0.5 * rho * (vel[0] ** 2 + vel[1] ** 2 + vel[2] ** 2)
    w = wl.Workload("supersonic", n, 1.4, bc, (0.1, 0.07, 0.13), 0.4, nsteps=5,
                    state=[rho, rho * vel[0], rho * vel[1], rho * vel[2], E])
    _check(w, scheme, hard.VARIANT_FUSED, 1, TOL_1)
    _check(w, scheme, hard.VARIANT_FUSED, 5, TOL_100)


def test_positivity_fallback_is_taken_in_3d_and_matches():
    """Scheme A on a field with density and pressure spikes in all three directions: the oracle reports fallbacks
    (G4), the kernel's branch-free version of it gives the same step."""
    import oracle
    n = (30, 20, 18)
    rng = np.random.default_rng(9)
    shp = n[::-1]
    rho = np.where(rng.random(shp) < 0.08, 0.01, 1.0) * (1.0 + 0.2 * rng.random(shp))
    rho = np.where(rng.random(shp) < 0.04, 5.0, rho)
    prs = np.where(rng.random(shp) < 0.08, 0.02, 1.0) * (1.0 + 0.2 * rng.random(shp))
    vel = [0.4 * (rng.random(shp) - 0.5) for _ in range(3)]
    E = prs / 0.4 + 0.5 * rho * (vel[0] ** 2 + vel[1] ** 2 + vel[2] ** 2)
    st = [rho, rho * vel[0], rho * vel[1], rho * vel[2], E]
    o = oracle.Oracle(*n, 1.4, wl.BC_PERIODIC, scheme=hard.SCHEME_WENO5Z_HLL, spacing=(0.1, 0.07, 0.13))
    o.set_state(*st)
    o.rhs()
    assert o.fallbacks() > 200, o.fallbacks()
    o.close()
    w = wl.Workload("spikes", n, 1.4, wl.BC_PERIODIC, (0.1, 0.07, 0.13), 0.2, nsteps=1, state=st)
    _check(w, hard.SCHEME_WENO5Z_HLL, hard.VARIANT_FUSED, 1, TOL_1)
    _check(w, hard.SCHEME_WENO5Z_HLL, hard.VARIANT_PERDIR, 1, TOL_1)


@pytest.mark.parametrize("scheme", SCHEMES)
@pytest.mark.parametrize("variant", VARIANTS)
def test_sod_c0(scheme, variant):
    w = wl.sod(1000)
    _check(w, scheme, variant, 1, TOL_1)
    _check(w, scheme, variant, 100, TOL_100)


@pytest.mark.parametrize("scheme", SCHEMES)
def test_leblanc_c1(scheme):
    w = wl.leblanc(4096)
    _check(w, scheme, hard.VARIANT_FUSED, 1, TOL_1)
    _check(w, scheme, hard.VARIANT_FUSED, 100, TOL_100)


@pytest.mark.parametrize("scheme", SCHEMES)
@pytest.mark.parametrize("variant", VARIANTS)
def test_sedov_small(scheme, variant):
    w = wl.sedov(32)
    _check(w, scheme, variant, 1, TOL_1)
    _check(w, scheme, variant, 30, TOL_100)


@pytest.mark.parametrize("scheme", SCHEMES)
def test_turbulence_small_100_steps(scheme):
    w = wl.turbulence(40, nsteps=100)
    _check(w, scheme, hard.VARIANT_FUSED, 1, TOL_1)
    _check(w, scheme, hard.VARIANT_FUSED, 100, TOL_100)


@pytest.mark.parametrize("scheme", SCHEMES)
def test_fixed_dt_and_run_to(scheme):
    w = wl.sod(200, t_end=0.05)
    _check(w, scheme, hard.VARIANT_FUSED, 7, TOL_100, dt=1e-4)
    h = hard.Hard(*w.n, w.gamma, w.bc, scheme=scheme, spacing=w.spacing)
    h.set_state(*w.state)
    n = h.run_to(w.t_end, w.cfl)
    t, steps = h.time()
    assert steps == n and abs(t - w.t_end) <= 1e-12 * w.t_end
    h.close()


def test_errors_and_status():
    with pytest.raises(hard.HardError):
        hard.Hard(0, 1, 1, 1.4, 0)
    with pytest.raises(hard.HardError):
        hard.Hard(2, 1, 1, 1.4, 0)
    h = hard.Hard(8, 8, 8, 1.4, 0)
    with pytest.raises(hard.HardError) as e:
        h.step(0.4, 1)
    assert e.value.code == hard.ERR_NOSTATE
    st = wl.random_state((8, 8, 8), 3)
    st[0][0, 0, 0] = -1.0
    with pytest.raises(hard.HardError) as e:
        h.set_state(*st)
    assert e.value.code == hard.ERR_NONPHYSICAL
    h.close()


def test_device_pointers_and_uniform_state():
    import torch
    n = (24, 20, 18)
    g = 1.4
    vals = (1.3, 1.3 * 0.37, 1.3 * -0.21, 1.3 * 0.11, 0.9 / 0.4 + 0.5 * 1.3 * (0.37 ** 2 + 0.21 ** 2 + 0.11 ** 2))
    st = [torch.full(n[::-1], v, dtype=torch.float64, device="cuda") for v in vals]
    for scheme in SCHEMES:
        h = hard.Hard(*n, g, wl.BC_PERIODIC, scheme=scheme)
        h.set_state(*st)
        h.step(0.4, 5)
        out = [torch.empty_like(a) for a in st]
        h.get_state(out)
        for a, b in zip(out, st):
            assert torch.equal(a, b)        # uniform state preserved exactly
        h.close()


# ---------------------------------------------------------------- NEXT-2: reflecting walls, Kelvin-Helmholtz
@pytest.mark.parametrize("scheme", SCHEMES)
@pytest.mark.parametrize("variant", VARIANTS)
@pytest.mark.parametrize("n", [(37, 21, 19), (45, 30, 1), (131, 1, 1)])
def test_reflecting_walls(scheme, variant, n):
    w = _random_workload(n, wl.BC_REFLECT, seed=7 + sum(n), spacing=(0.1, 0.07, 0.13))
    _check(w, scheme, variant, 1, TOL_1)
    _check(w, scheme, variant, 25, TOL_100)


@pytest.mark.parametrize("scheme", SCHEMES)
def test_kelvin_helmholtz_2d(scheme):
    w = wl.kelvin_helmholtz(256, nsteps=100)
    _check(w, scheme, hard.VARIANT_FUSED, 1, TOL_1)
    _check(w, scheme, hard.VARIANT_FUSED, 100, TOL_100)


# ---------------------------------------------------------------- NEXT-1: advected radiation energy density
def _check_rad(w, er, scheme, variant, nsteps, tol):
    import oracle
    st = [np.ascontiguousarray(a, dtype=np.float64) for a in w.state]
    o = oracle.Oracle(*w.n, w.gamma, w.bc, scheme=scheme, spacing=w.spacing, radiation=True)
    o.set_state(*st)
    o.set_rad_energy(er)
    h = hard.Hard(*w.n, w.gamma, w.bc, scheme=scheme, variant=variant, spacing=w.spacing, radiation=True)
    h.set_state(*st)
    h.set_rad_energy(np.ascontiguousarray(er))
    assert abs(h.max_dt() - o.max_dt()) <= TOL_DT * o.max_dt()
    o.step(w.cfl, nsteps)
    h.step(w.cfl, nsteps)
    errs = field_errors(h.get_state() + [h.get_rad_energy()], o.get_state() + [o.get_rad_energy()])
    assert max(errs) <= tol, errs
    assert np.abs(o.get_rad_energy() - er).max() > 0
    h.close()
    o.close()


@pytest.mark.parametrize("scheme", SCHEMES)
@pytest.mark.parametrize("variant", VARIANTS)
@pytest.mark.parametrize("n,bc", [((37, 21, 19), wl.BC_PERIODIC), ((45, 30, 1), wl.BC_REFLECT), ((131, 1, 1), wl.BC_OUTFLOW)])
def test_radiation_energy_advection(scheme, variant, n, bc):
    w = _random_workload(n, bc, seed=11 + sum(n), spacing=(0.1, 0.07, 0.13))
    er = 1.0 + 0.5 * np.random.default_rng(5).random(n[::-1])
    _check_rad(w, er, scheme, variant, 1, TOL_1)
    _check_rad(w, er, scheme, variant, 25, TOL_100)


@pytest.mark.parametrize("scheme", SCHEMES)
def test_radiation_energy_turbulence_100_steps(scheme):
    w = wl.turbulence(40, nsteps=100)
    er = 1.0 + 0.3 * np.sin(2 * np.pi * np.arange(40) / 40.0)[None, None, :] * np.ones((40, 40, 40))
    _check_rad(w, er, scheme, hard.VARIANT_FUSED, 100, TOL_100)


@pytest.mark.parametrize("scheme", SCHEMES)
def test_radiation_energy_in_cgs_magnitudes(scheme):
    """Physical-unit data: a stellar-interior-like state in cgs, rho ~ 1e2 g/cm^3, p ~ 1e17 erg/cm^3,
    v ~ 1e7 cm/s, non-uniform E_rad ~ 1e14..1e15 erg/cm^3, cells of 1e9 cm.  The division-free WENO-Z weights are
    cubic in the smoothness indicators (data^6 ~ 1e100 here): no overflow, same parity bars."""
    n = (37, 21, 19)
    rng = np.random.default_rng(21)
    shp = n[::-1]
    rho = 1e2 * (1.0 + 0.3 * rng.random(shp))
    vel = [1e7 * (rng.random(shp) - 0.5) for _ in range(3)]
    prs = 1e17 * (1.0 + 0.5 * rng.random(shp))
    gamma = 5.0 / 3.0
    E = prs / (gamma - 1.0) + 0.5 * rho * (vel[0] ** 2 + vel[1] ** 2 + vel[2] ** 2)
    w = wl.Workload("cgs", n, gamma, wl.BC_PERIODIC, (1e9, 0.7e9, 1.3e9), 0.4, nsteps=10,
                    state=[rho, rho * vel[0], rho * vel[1], rho * vel[2], E])
    er = 1e14 * (1.0 + 9.0 * rng.random(shp))
    _check_rad(w, er, scheme, hard.VARIANT_FUSED, 1, TOL_1)
    _check_rad(w, er, scheme, hard.VARIANT_FUSED, 10, TOL_100)


# ---------------------------------------------------------------- NEXT-3: radiative heating / cooling source
def _check_source(w, er, params, scheme, variant, nsteps, tol, dt=None):
    import oracle
    st = [np.ascontiguousarray(a, dtype=np.float64) for a in w.state]
    o = oracle.Oracle(*w.n, w.gamma, w.bc, scheme=scheme, spacing=w.spacing, radiation=True)
    o.set_source(*params)
    o.set_state(*st)
    o.set_rad_energy(er)
    h = hard.Hard(*w.n, w.gamma, w.bc, scheme=scheme, variant=variant, spacing=w.spacing, radiation=True)
    h.set_source(*params)
    h.set_state(*st)
    h.set_rad_energy(np.ascontiguousarray(er))
    if dt is None:
        o.step(w.cfl, nsteps)
        h.step(w.cfl, nsteps)
    else:
        o.step_dt(dt, nsteps)
        h.step_dt(dt, nsteps)
    errs = field_errors(h.get_state() + [h.get_rad_energy()], o.get_state() + [o.get_rad_energy()])
    assert max(errs) <= tol, errs
    assert abs(h.max_dt() - o.max_dt()) <= max(10 * tol, 1e-12) * o.max_dt()
    assert abs(h.time()[0] - o.time()[0]) <= 1e-12 * o.time()[0]
    assert np.abs(o.get_rad_energy() - er).max() > 0
    h.close()
    o.close()


@pytest.mark.parametrize("scheme", SCHEMES)
@pytest.mark.parametrize("variant", VARIANTS)
def test_source_on_random_state(scheme, variant):
    n = (37, 21, 19)
    w = _random_workload(n, wl.BC_PERIODIC, seed=77, spacing=(0.1, 0.07, 0.13))
    er = 1.0 + 0.5 * np.random.default_rng(6).random(n[::-1])
    params = (0.7, 3.0, 0.5, 1.2)                  # kappa, c, a, cv in code units
    _check_source(w, er, params, scheme, variant, 1, TOL_1)
    _check_source(w, er, params, scheme, variant, 25, TOL_100)


@pytest.mark.parametrize("T0", [11.0, 1.1e9])
def test_paper_heating_cooling_cases(T0):
    """P:209-211 in cgs units: rho = 1e-7, mu = 0.6, kappa = 0.4, T_rad = 3.4e6 K, gas at 11 K / 1.1e9 K."""
    c_light, a_rad, k_b, m_p = 2.99792458e10, 7.5657e-15, 1.380649e-16, 1.67262192e-24
    gamma, rho, cv = 5.0 / 3.0, 1e-7, 1.380649e-16 / ((5.0 / 3.0 - 1.0) * 0.6 * 1.67262192e-24)
    n = (20, 18, 1)
    e0 = rho * cv * T0
    z = np.zeros(n[::-1])
    w = wl.Workload("heat", n, gamma, wl.BC_PERIODIC, (1.0, 1.0, 1.0), 0.4, nsteps=20,
                    state=[z + rho, z.copy(), z.copy(), z.copy(), z + e0])
    er = z + a_rad * 3.4e6 ** 4
    t_end = 2e-7 if T0 < 1e6 else 2e-10
    _check_source(w, er, (0.4, c_light, a_rad, cv), hard.SCHEME_WENO5Z_HLL, hard.VARIANT_FUSED, 20, TOL_100, dt=t_end / 20)
