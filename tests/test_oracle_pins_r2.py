"""Independent pins for three parts of the oracle that only the oracle itself used to vouch for (CPU only):

  1. fill_ghosts, outflow (G10; ghost entities P:64): ghost = the NEAREST interior cell;
  2. the positivity fallback of scheme A (G4): ALL five variables become piecewise constant in a cell
     whose reconstructed rho or p is <= 0;
  3. the WENO5-Z smoothness indicators / weights ("[18]", G1), from their integral definition.

Every expected value is derived from the mathematics (scalar upwind advection, the textbook HLL flux,
numpy.polynomial on the candidate parabolas), never from the oracle's own lines.  Each test fails under the
matching mutation of oracle/hard_oracle.cpp (second-nearest cell as outflow ghost; fallback that keeps the
reconstructed velocities; 13/12 -> 1 in beta).
"""
import numpy as np
import pytest

import oracle
import _weno_def as wd

G = 1.4


# ------------------------------------------------------------------------------------------------- helpers
def _axis_shape(n, axis):
    """(nx, ny, nz) with n cells along `axis` (0 = x) and 1 elsewhere."""
    nn = [1, 1, 1]
    nn[axis] = n
    return tuple(nn)


def _as3d(a, axis):
    """1-D array along `axis` -> (nz, ny, nx) array."""
    sh = [1, 1, 1]
    sh[2 - axis] = a.size
    return np.asarray(a, dtype=np.float64).reshape(sh)


def _cons(rho, vel, p):
    rho = np.asarray(rho, dtype=np.float64)
    vel = [np.broadcast_to(np.asarray(v, dtype=np.float64), rho.shape) for v in vel]
    p = np.broadcast_to(np.asarray(p, dtype=np.float64), rho.shape)
    E = p / (G - 1) + 0.5 * rho * (vel[0] ** 2 + vel[1] ** 2 + vel[2] ** 2)
    return [rho, rho * vel[0], rho * vel[1], rho * vel[2], E]


# ================================================================================ 1. outflow ghost fill (G10)
# With uniform velocity u and pressure p the Euler equations reduce to scalar advection of rho, and the
# scheme reduces with them whenever the Riemann flux is the upwind one:
#   scheme B: HLLC resolves a contact exactly (S* = u, pbar = p => the upwind side's physical flux);
#   scheme A: HLL with SL >= 0 (or SR <= 0) returns the upwind side's physical flux — supersonic flow.
# Then rho^{n+1} follows the scalar MUSCL-minmod / WENO5-Z upwind scheme with Heun's method, and u, p stay
# uniform.  The scalar scheme is written here on an explicitly extended array whose ghosts are, by the
# definition of zero-gradient outflow, copies of the nearest interior cell.
def _face_plus(q, i, scheme):
    """value at the i+1/2 face of cell i of the extended array q (left-biased)"""
    if scheme == 0:
        return wd.wenoz(q[i - 2], q[i - 1], q[i], q[i + 1], q[i + 2])
    a, b = q[i] - q[i - 1], q[i + 1] - q[i]
    s = min(a, b) if (a > 0 and b > 0) else max(a, b) if (a < 0 and b < 0) else 0.0
    return q[i] + 0.5 * s


def _face_minus(q, i, scheme):
    """value at the i-1/2 face of cell i (right-biased): the mirror image"""
    if scheme == 0:
        return wd.wenoz(q[i + 2], q[i + 1], q[i], q[i - 1], q[i - 2])
    a, b = q[i] - q[i - 1], q[i + 1] - q[i]
    s = min(a, b) if (a > 0 and b > 0) else max(a, b) if (a < 0 and b < 0) else 0.0
    return q[i] - 0.5 * s


def _scalar_heun_outflow(rho, u, dt, dx, scheme):
    g = 3 if scheme == 0 else 2
    n = rho.size

    def Lop(r):
        q = np.concatenate([[r[0]] * g, r, [r[-1]] * g])        # zero-gradient: nearest interior cell
        f = np.empty(n + 1)                                     # f[i] = flux through face i-1/2
        for i in range(n + 1):
            left, right = i - 1 + g, i + g                      # extended indices of the two cells
            f[i] = u * (_face_plus(q, left, scheme) if u > 0 else _face_minus(q, right, scheme))
        return -(f[1:] - f[:-1]) / dx

    r1 = rho + dt * Lop(rho)
    return 0.5 * rho + 0.5 * (r1 + dt * Lop(r1))


RAMP = np.array([1.0, 1.3, 1.1, 1.6, 1.2, 1.9, 1.5, 2.2])       # slopes of both signs; also a plain ramp below


@pytest.mark.parametrize("axis", [0, 1, 2])
@pytest.mark.parametrize("scheme,u", [(1, 0.5), (1, -0.5), (0, 3.0), (0, -3.0)])
@pytest.mark.parametrize("profile", [RAMP, 1.0 + 0.1 * np.arange(8)])
def test_outflow_ghosts_are_the_nearest_interior_cell(scheme, u, axis, profile):
    n, dx, dt, p0 = profile.size, 0.125, 0.01, 1.0
    vel = [0.0, 0.0, 0.0]
    vel[axis] = u
    o = oracle.Oracle(*_axis_shape(n, axis), G, oracle.BC_OUTFLOW, scheme=scheme,
                      spacing=tuple(dx if a == axis else 1.0 for a in range(3)))
    o.set_state(*[_as3d(a, axis) for a in _cons(profile, vel, p0)])
    o.step_dt(dt, 1)
    out = [a.ravel() for a in o.get_state()]
    rho = _scalar_heun_outflow(profile, u, dt, dx, scheme)
    assert np.abs(rho - profile).max() > 1e-3                   # the step moved the profile
    assert np.abs(rho[0] - profile[0]) + np.abs(rho[-1] - profile[-1]) > 1e-4 or scheme == 1
    exp = _cons(rho, vel, p0)
    for f in range(5):
        assert np.abs(out[f] - exp[f]).max() <= 1e-13 * max(1.0, np.abs(exp[f]).max()), f


@pytest.mark.parametrize("scheme,u", [(1, 0.5), (0, 3.0)])
def test_pulse_leaves_through_the_outflow_face(scheme, u):
    # a density pulse carried by a uniform stream (u, p uniform: a pure contact) leaves through the high-x
    # face; nothing comes back, nothing wraps around: the box returns to the background to 1e-12
    n, dx = 64, 1.0 / 64
    x = (np.arange(n) + 0.5) * dx
    rho0 = 1.0 + 0.8 * np.exp(-((x - 0.6) / 0.08) ** 2)
    o = oracle.Oracle(n, 1, 1, G, oracle.BC_OUTFLOW, scheme=scheme, spacing=(dx, 1.0, 1.0))
    o.set_state(*[_as3d(a, 0) for a in _cons(rho0, [u, 0.0, 0.0], 1.0)])
    mass0 = o.get_state()[0].sum() * dx
    t_end = 3.0 / abs(u)                                        # three box lengths of travel
    nsteps = o.run_to(t_end, 0.4)
    assert nsteps > 100
    rho, mx, my, mz, E = [a.ravel() for a in o.get_state()]
    assert mass0 > 1.1
    assert abs(rho.sum() * dx - 1.0) <= 1e-12                   # mass in the box = background
    assert np.abs(rho - 1.0).max() <= 1e-12
    assert np.abs(mx - u).max() <= 1e-12
    assert np.abs(E - (1.0 / (G - 1) + 0.5 * u * u)).max() <= 1e-11


# ================================================================================ 2. positivity fallback (G4)
def _hll_textbook(WL, WR):
    """HLL flux (x normal) with Davis' bounds, written out: states (rho, u, v, w, p)."""
    def UF(W):
        rho, u, v, w, p = W
        E = p / (G - 1) + 0.5 * rho * (u * u + v * v + w * w)
        return (np.array([rho, rho * u, rho * v, rho * w, E]),
                np.array([rho * u, rho * u * u + p, rho * u * v, rho * u * w, (E + p) * u]))
    UL, FL = UF(WL)
    UR, FR = UF(WR)
    cL, cR = np.sqrt(G * WL[4] / WL[0]), np.sqrt(G * WR[4] / WR[0])
    SL, SR = min(WL[1] - cL, WR[1] - cR), max(WL[1] + cL, WR[1] + cR)
    assert SL < 0.0 < SR                                        # the subsonic branch is the one under test
    return (SR * FL - SL * FR + SL * SR * (UR - UL)) / (SR - SL)


def _fallback_data():
    n = 20
    i = np.arange(n)
    rho = np.ones(n)
    rho[7:13] = [0.01, 0.01, 4.98, 0.45, 0.03, 0.1]             # spikes: WENO undershoots below zero
    var = (i >= 5) & (i <= 14)
    u = np.where(var, 0.3 + 0.2 * np.sin(1.3 * i), 0.3)
    v = np.where(var, 0.1 * np.cos(0.7 * i), 0.0)
    w = np.where(var, -0.2 * np.sin(0.4 * i + 1.0), 0.0)
    p = np.where(var, 1.0 + 0.3 * np.cos(0.9 * i), 1.0)
    return rho, u, v, w, p


def _rot(vec3, axis):
    """components (normal, t1, t2) -> (x, y, z) for a normal along `axis` (cyclic order)"""
    out = [None] * 3
    out[axis], out[(axis + 1) % 3], out[(axis + 2) % 3] = vec3
    return out


@pytest.mark.parametrize("axis", [0, 1, 2])
def test_fallback_makes_all_five_variables_piecewise_constant(axis):
    rho, u, v, w, p = _fallback_data()
    n, dx = rho.size, 0.05
    W = np.stack([rho, u, v, w, p])                             # (normal, t1, t2) velocity order

    # which cells fall back, from the definition: a reconstructed rho or p <= 0 at either face
    def pm(q):
        pl = wd.wenoz(np.roll(q, 2), np.roll(q, 1), q, np.roll(q, -1), np.roll(q, -2))
        mi = wd.wenoz(np.roll(q, -2), np.roll(q, -1), q, np.roll(q, 1), np.roll(q, 2))
        return pl, mi
    PL, MI = zip(*[pm(q) for q in W])
    bad = (PL[0] <= 0) | (MI[0] <= 0) | (PL[4] <= 0) | (MI[4] <= 0)
    assert list(np.nonzero(bad)[0]) == [7, 8, 11, 12]           # two pairs of adjacent cells
    assert min(np.abs(PL[0][bad]).min(), np.abs(MI[0][bad]).min()) > 0.02   # clearly, not marginally

    o = oracle.Oracle(*_axis_shape(n, axis), G, oracle.BC_PERIODIC, scheme=0,
                      spacing=tuple(dx if a == axis else 1.0 for a in range(3)))
    o.set_state(*[_as3d(a, axis) for a in _cons(rho, _rot([u, v, w], axis), p)])
    L = [a.ravel() for a in o.rhs()]
    assert o.fallbacks() == 4
    Ln = np.stack([L[0], L[1 + axis], L[1 + (axis + 1) % 3], L[1 + (axis + 2) % 3], L[4]])   # (n, t1, t2) order

    # single face fluxes by telescoping from the uniform region: face -1/2 (between cells n-1 and 0) has both
    # stencils inside the uniform run 15..19, 0..4, so its flux is the physical flux of the background state
    rho0, u0, p0 = 1.0, 0.3, 1.0
    E0 = p0 / (G - 1) + 0.5 * rho0 * u0 * u0
    F0 = np.array([rho0 * u0, rho0 * u0 * u0 + p0, 0.0, 0.0, (E0 + p0) * u0])
    face = lambda i: F0 - dx * Ln[:, :i + 1].sum(axis=1)        # flux through face i+1/2

    # (a) between two fallen-back cells: first-order Godunov-HLL flux of the two CELL AVERAGES
    for i in (7, 11):
        exp = _hll_textbook(W[:, i], W[:, i + 1])
        assert np.abs(face(i) - exp).max() <= 1e-12 * np.abs(exp).max(), i
    # with numbers: face 7+1/2 separates two cells of density 0.01 — mass flux 0.01*u7... written out
    WL, WR = W[:, 7], W[:, 8]
    assert WL[0] == 0.01 and WR[0] == 0.01 and abs(WL[1] - WR[1]) > 0.1      # u varies across the face
    # (b) fallen-back cell next to a regular one: cell average on one side, WENO value on the other
    exp = _hll_textbook(W[:, 8], np.array([MI[k][9] for k in range(5)]))
    assert np.abs(face(8) - exp).max() <= 1e-12 * np.abs(exp).max()
    exp = _hll_textbook(np.array([PL[k][6] for k in range(5)]), W[:, 7])
    assert np.abs(face(6) - exp).max() <= 1e-12 * np.abs(exp).max()
    # (c) the telescoped sum closes: after the last varying cell the flux is the background flux again
    assert np.abs(face(n - 1) - F0).max() <= 1e-12


# ================================================================================ 3. WENO5-Z from its definition (G1)
def test_definition_reproduces_the_published_tables():
    # sanity of the helper itself: the derived numbers are the familiar rational tables
    assert np.allclose(wd.D, [0.1, 0.6, 0.3], rtol=0, atol=1e-14)
    assert np.allclose(6 * wd.Q, [[2, -7, 11], [-1, 5, 2], [2, 5, -1]], rtol=0, atol=1e-13)
    # beta_1 = 13/12 (b - 2c + d)^2 + 1/4 (b - d)^2 as a quadratic form
    b1 = 13 / 12 * np.outer([1, -2, 1], [1, -2, 1]) + 0.25 * np.outer([1, 0, -1], [1, 0, -1])
    assert np.allclose(wd.M[1], b1, rtol=0, atol=1e-13)


def test_wenoz_equals_the_definition_on_random_data():
    rng = np.random.default_rng(11)
    worst = 0.0
    for _ in range(2000):
        q = rng.standard_normal(5) * 10.0 ** rng.integers(-3, 3)
        ref = float(wd.wenoz(*q))
        worst = max(worst, abs(oracle.wenoz(*q) - ref) / np.abs(q).max())
    assert worst <= 1e-13


def test_wenoz_single_weight_probes_isolate_each_beta():
    # data for which two of the three parabolas are straight lines through flat data (beta = 0 exactly) and
    # the third is not: the weights then collapse onto... the smooth candidates; comparing against the
    # definition on such one-sided data exercises each beta_k separately.
    for q in ([0.0, 0.0, 0.0, 0.0, 1.0], [1.0, 0.0, 0.0, 0.0, 0.0], [0.0, 0.0, 0.0, 1.0, 2.5], [2.5, 1.0, 0.0, 0.0, 0.0],
              [0.3, 0.3, 0.3, 1.0, -2.0], [1.0, 2.0, 3.0, 4.0, 7.5]):
        be = wd.betas(*q)
        assert min(be) <= 1e-30 or max(be) > 0
        assert oracle.wenoz(*q) == pytest.approx(float(wd.wenoz(*q)), rel=1e-13, abs=1e-15)
    # and a value that depends on the 13/12 : 1/4 ratio at first order: one rough, two comparable stencils
    q = [1.0, 1.2, 1.1, 1.5, 0.2]
    be = wd.betas(*q)
    assert be[0] == pytest.approx(13 / 12 * (1.0 - 2.4 + 1.1) ** 2 + 0.25 * (1.0 - 4.8 + 3.3) ** 2, rel=1e-12)
    assert oracle.wenoz(*q) == pytest.approx(float(wd.wenoz(*q)), rel=1e-13)


# --- round-2 mutation sweep (39 mutants of oracle/hard_oracle.cpp): three survived the suite; their pins:
def _pressure_spike_data():
    """rho smooth and well away from zero, PRESSURE with the spikes: WENO undershoots p, never rho"""
    n = 20
    i = np.arange(n)
    var = (i >= 5) & (i <= 14)
    p = np.ones(n)
    p[7:13] = [0.01, 0.01, 4.98, 0.45, 0.03, 0.1]
    rho = np.where(var, 1.0 + 0.3 * np.cos(0.9 * i), 1.0)
    u = np.where(var, 0.03 + 0.02 * np.sin(1.3 * i), 0.03)       # slow: subsonic even where p = 0.01
    v = np.where(var, 0.1 * np.cos(0.7 * i), 0.0)
    w = np.where(var, -0.2 * np.sin(0.4 * i + 1.0), 0.0)
    return rho, u, v, w, p


def _pm(q):
    pl = wd.wenoz(np.roll(q, 2), np.roll(q, 1), q, np.roll(q, -1), np.roll(q, -2))
    mi = wd.wenoz(np.roll(q, -2), np.roll(q, -1), q, np.roll(q, 1), np.roll(q, 2))
    return pl, mi


def test_fallback_is_triggered_by_the_pressure_alone():
    """G4: 'a reconstructed rho OR p <= 0'.  (mutant: only rho tested)"""
    rho, u, v, w, p = _pressure_spike_data()
    n, dx = rho.size, 0.05
    W = np.stack([rho, u, v, w, p])
    PL, MI = zip(*[_pm(q) for q in W])
    assert PL[0].min() > 0.5 and MI[0].min() > 0.5                 # rho never triggers
    bad = (PL[4] <= 0) | (MI[4] <= 0)
    assert list(np.nonzero(bad)[0]) == [7, 8, 11, 12]
    o = oracle.Oracle(n, 1, 1, G, oracle.BC_PERIODIC, scheme=0, spacing=(dx, 1.0, 1.0))
    o.set_state(*[_as3d(a, 0) for a in _cons(rho, [u, v, w], p)])
    L = np.stack([a.ravel() for a in o.rhs()])
    assert o.fallbacks() == 4
    rho0, u0, p0 = 1.0, 0.03, 1.0
    E0 = p0 / (G - 1) + 0.5 * rho0 * u0 * u0
    F0 = np.array([rho0 * u0, rho0 * u0 * u0 + p0, 0.0, 0.0, (E0 + p0) * u0])
    face = lambda i: F0 - dx * L[:, :i + 1].sum(axis=1)
    for i in (7, 11):                                              # between two fallen-back cells: cell averages
        exp = _hll_textbook(W[:, i], W[:, i + 1])
        assert np.abs(face(i) - exp).max() <= 1e-12 * np.abs(exp).max(), i


def test_fallback_takes_the_radiation_energy_along():
    """G19: E_rad 'follows the positivity fallback but does not trigger it'.  Between two fallen-back cells the
    Rusanov flux is that of the two CELL values of E_rad (typed out); and E_rad <= 0 reconstructions alone trigger
    nothing.  (mutant: E_rad keeps its WENO values in a fallen-back cell)"""
    rho, u, v, w, p = _fallback_data()
    n, dx = rho.size, 0.05
    i = np.arange(n)
    er = np.where((i >= 5) & (i <= 14), 2.0 + np.sin(1.1 * i), 2.0)
    o = oracle.Oracle(n, 1, 1, G, oracle.BC_PERIODIC, scheme=0, spacing=(dx, 1.0, 1.0), radiation=True)
    o.set_state(*[_as3d(a, 0) for a in _cons(rho, [u, v, w], p)])
    o.set_rad_energy(_as3d(er, 0))
    L5 = o.rhs(nf=6)[5].ravel()
    assert o.fallbacks() == 4
    face = lambda k: 2.0 * 0.3 - dx * L5[:k + 1].sum()             # face -1/2 lies in the uniform run: F = E u
    for k in (7, 11):
        cL, cR = np.sqrt(G * p[k] / rho[k]), np.sqrt(G * p[k + 1] / rho[k + 1])
        alpha = max(abs(u[k]) + cL, abs(u[k + 1]) + cR)
        exp = 0.5 * (er[k] * u[k] + er[k + 1] * u[k + 1]) - 0.5 * alpha * (er[k + 1] - er[k])
        assert abs(face(k) - exp) <= 1e-12 * abs(exp), k
    # spikes in E_rad alone (hydro smooth): WENO undershoots E_rad below zero, and nothing falls back
    er2 = np.ones(n)
    er2[7:13] = [0.01, 0.01, 4.98, 0.45, 0.03, 0.1]
    pl, mi = _pm(er2)
    assert min(pl.min(), mi.min()) < 0.0
    o2 = oracle.Oracle(n, 1, 1, G, oracle.BC_PERIODIC, scheme=0, spacing=(dx, 1.0, 1.0), radiation=True)
    o2.set_state(*[_as3d(a, 0) for a in _cons(np.ones(n), [0.3 + 0 * er2, 0 * er2, 0 * er2], np.ones(n))])
    o2.set_rad_energy(_as3d(er2, 0))
    o2.rhs(nf=6)
    assert o2.fallbacks() == 0


def test_next_dt_is_evaluated_after_the_source_update():
    """G20: lambda (hence the next dt) belongs to the state the step RETURNS, i.e. after the source has changed the
    pressure.  (mutant: max wavespeed taken before apply_source)"""
    n = (12, 1, 1)
    z = np.zeros(n[::-1])
    gam, rho, cv = 5.0 / 3.0, 1.0, 1.5
    o = oracle.Oracle(*n, gam, oracle.BC_PERIODIC, scheme=0, spacing=(0.1, 1.0, 1.0), radiation=True)
    o.set_source(5.0, 3.0, 0.5, cv)                                 # kappa, c, a, cv: strong heating by the radiation
    o.set_state(z + rho, z.copy(), z.copy(), z.copy(), z + 0.3)
    o.set_rad_energy(z + 4.0)
    dt0 = o.max_dt()
    o.step_dt(0.05, 1)
    E = o.get_state()[4].ravel()
    assert E.min() > 0.5                                            # the gas has been heated a lot
    p = (gam - 1.0) * E[0]                                          # gas at rest
    assert abs(o.max_dt() - 0.1 / np.sqrt(gam * p / rho)) <= 1e-14 * o.max_dt()
    assert o.max_dt() < 0.8 * dt0


def test_negative_pressure_is_reported_as_non_physical():
    """G4: 'a non-physical state is an error' — rho > 0 but p <= 0 (E below the kinetic energy).  (mutant: only rho)"""
    z = np.zeros((1, 1, 8))
    o = oracle.Oracle(8, 1, 1, G, oracle.BC_PERIODIC, scheme=1, spacing=(0.1, 1.0, 1.0))
    E = z + 2.5
    E[0, 0, 3] = 0.4                                               # kinetic energy there is 0.5: p < 0
    with pytest.raises(oracle.OracleError):
        o.set_state(z + 1.0, z + 1.0, z.copy(), z.copy(), E)


def test_set_state_zeroes_the_radiation_energy_and_set_spacing_reevaluates_lambda():
    """API contract shared with include/hard.h: hard_set_state zeroes E_rad; hard_set_spacing re-evaluates lambda."""
    z = np.zeros((1, 1, 8))
    o = oracle.Oracle(8, 1, 1, G, oracle.BC_PERIODIC, scheme=0, spacing=(0.1, 1.0, 1.0), radiation=True)
    st = [z + 1.0, z + 0.5, z.copy(), z.copy(), z + 2.5]
    o.set_state(*st)
    o.set_rad_energy(z + 7.0)
    assert o.get_rad_energy().min() == 7.0
    o.set_state(*st)
    assert not o.get_rad_energy().any()
    dt1 = o.max_dt()
    o._chk(o.L.oracle_set_spacing(o.h, 0.05, 1.0, 1.0), "set_spacing")
    assert abs(o.max_dt() - 0.5 * dt1) <= 1e-15 * dt1
