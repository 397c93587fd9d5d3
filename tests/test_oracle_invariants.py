"""Invariant pins of the oracle's stepper (BASELINE.json north_star): conservation to 1e-13, exact
uniform-state preservation, bit-for-bit mirror / axis-permutation symmetry, 1-D == replicated 3-D
pencil, the CFL formula by hand, and an independent whole-array (np.roll) restatement of one full
Heun step on a 4x4x4 periodic grid."""
import math

import numpy as np
import pytest

import oracle
import _weno_def as wd
from paper_2509_08971_b200 import workloads as wl

SCHEMES = [0, 1]


def _run(state, n, gamma, bc, scheme, spacing, cfl=0.4, nsteps=1, dt=None):
    o = oracle.Oracle(*n, gamma, bc, scheme=scheme, spacing=spacing)
    o.set_state(*state)
    if dt is None:
        o.step(cfl, nsteps)
    else:
        o.step_dt(dt, nsteps)
    out = o.get_state()
    o.close()
    return out


def _fsum(a):
    return math.fsum(a.ravel().tolist())


@pytest.mark.parametrize("scheme", SCHEMES)
def test_conservation_periodic(scheme):
    n = (12, 10, 8)
    st = wl.random_state(n, seed=11)
    out = _run(st, n, 1.4, wl.BC_PERIODIC, scheme, (0.1, 0.12, 0.09), nsteps=10)
    for f in range(5):
        ref = _fsum(st[f])
        scale = _fsum(np.abs(st[f]))
        assert abs(_fsum(out[f]) - ref) <= 1e-13 * scale
    assert any(not np.array_equal(out[f], st[f]) for f in range(5))


@pytest.mark.parametrize("scheme", SCHEMES)
@pytest.mark.parametrize("bc", [wl.BC_PERIODIC, wl.BC_OUTFLOW])
def test_uniform_state_preserved_exactly(scheme, bc):
    n = (9, 7, 8)
    g = 1.4
    rho, u, v, w, p = 1.3, 0.37, -0.21, 0.11, 0.9
    E = p / (g - 1) + 0.5 * rho * (u * u + v * v + w * w)
    st = [np.full(n[::-1], x) for x in (rho, rho * u, rho * v, rho * w, E)]
    out = _run(st, n, g, bc, scheme, (0.1, 0.1, 0.1), nsteps=5)
    for f in range(5):
        assert np.array_equal(out[f], st[f])


@pytest.mark.parametrize("scheme", SCHEMES)
@pytest.mark.parametrize("axis", [0, 1, 2])
def test_mirror_symmetry_bitwise(scheme, axis):
    n = (10, 8, 9)
    sp = (0.1, 0.07, 0.13)
    st = wl.random_state(n, seed=5)
    out = _run(st, n, 1.4, wl.BC_OUTFLOW, scheme, sp, nsteps=3)
    ax_np = 2 - axis                       # arrays are (z, y, x)
    stm = [np.flip(a, ax_np).copy() for a in st]
    stm[1 + axis] = -stm[1 + axis]
    outm = _run(stm, n, 1.4, wl.BC_OUTFLOW, scheme, sp, nsteps=3)
    back = [np.flip(a, ax_np) for a in outm]
    back[1 + axis] = -back[1 + axis]
    for f in range(5):
        assert np.array_equal(back[f], out[f])


@pytest.mark.parametrize("scheme", SCHEMES)
@pytest.mark.parametrize("perm", [(1, 0, 2), (2, 1, 0), (1, 2, 0)])
def test_axis_permutation_bitwise(scheme, perm):
    # new axis a carries old axis perm[a]
    n = (8, 9, 10)
    sp = (0.1, 0.07, 0.13)
    st = wl.random_state(n, seed=6)
    out = _run(st, n, 1.4, wl.BC_PERIODIC, scheme, sp, nsteps=3)
    # numpy axes are (z,y,x) = spatial (2,1,0): transpose so that new spatial axis a = old perm[a]
    tp = tuple(2 - perm[2 - m] for m in range(3))
    n2 = tuple(n[perm[a]] for a in range(3))
    sp2 = tuple(sp[perm[a]] for a in range(3))

    def permute(fields):
        res = [np.ascontiguousarray(np.transpose(a, tp)) for a in fields]
        mom = [res[1 + perm[a]] for a in range(3)]
        return [res[0], mom[0], mom[1], mom[2], res[4]]
    out2 = _run(permute(st), n2, 1.4, wl.BC_PERIODIC, scheme, sp2, nsteps=3)
    ref = permute(out)
    for f in range(5):
        assert np.array_equal(out2[f], ref[f])


@pytest.mark.parametrize("scheme", SCHEMES)
def test_1d_equals_replicated_3d_pencil(scheme):
    w = wl.sod(64)
    o1 = _run(w.state, w.n, w.gamma, w.bc, scheme, w.spacing, nsteps=20)
    st3 = [np.broadcast_to(a, (4, 5, 64)).copy() for a in w.state]
    o3 = _run(st3, (64, 5, 4), w.gamma, w.bc, scheme, (w.spacing[0], 0.3, 0.2), nsteps=20)
    for f in range(5):
        assert np.array_equal(o3[f], np.broadcast_to(o1[f], (4, 5, 64)))


def test_cfl_formula_by_hand():
    # uniform state: lambda = max_d (|u_d| + c)/Delta_d  (G6)
    g = 1.4
    rho, vel, p = 2.0, (0.3, -0.8, 0.1), 1.5
    E = p / (g - 1) + 0.5 * rho * sum(x * x for x in vel)
    n = (6, 5, 4)
    sp = (0.2, 0.25, 0.1)
    st = [np.full(n[::-1], x) for x in (rho, rho * vel[0], rho * vel[1], rho * vel[2], E)]
    o = oracle.Oracle(*n, g, wl.BC_PERIODIC, scheme=0, spacing=sp)
    o.set_state(*st)
    c = math.sqrt(g * p / rho)
    lam = max((abs(vel[d]) + c) / sp[d] for d in range(3))
    assert o.max_dt() == pytest.approx(1.0 / lam, rel=1e-15)
    # 1-D: inactive directions do not enter (G11)
    o1 = oracle.Oracle(6, 1, 1, g, wl.BC_PERIODIC, scheme=0, spacing=(0.2, 1e-9, 1e-9))
    o1.set_state(*[a[:1, :1, :] for a in st])
    assert o1.max_dt() == pytest.approx(0.2 / (abs(vel[0]) + c), rel=1e-15)


def test_sedov_initial_dt_and_energy():
    # G13: 32 hot cells, initial 1/lambda = dx / sqrt(gamma * (gamma-1) * e_hot)
    w = wl.sedov(32)
    assert w.meta["nhot"] == 32
    dx = w.spacing[0]
    assert _fsum(w.state[4]) * dx ** 3 == pytest.approx(1.0 + (8.0 - 32 * dx ** 3) * 2.5e-5, rel=1e-12)
    o = oracle.Oracle(*w.n, w.gamma, w.bc, scheme=1, spacing=w.spacing)
    o.set_state(*w.state)
    e_hot = 1.0 / (32 * dx ** 3)
    assert o.max_dt() == pytest.approx(dx / math.sqrt(1.4 * 0.4 * e_hot), rel=1e-14)


# ---------------------------------------------------------------- independent whole-array restatement
def _np_step(st, g, sp, dt, scheme):
    """One Heun step on a fully periodic grid written with np.roll on whole arrays (no pencils, no
    ghosts, no index arithmetic) — structure independent of the oracle's loops."""
    def prim(U):
        rho = U[0]
        vel = [U[1 + a] / rho for a in range(3)]
        p = (g - 1) * (U[4] - 0.5 * (U[1] * vel[0] + U[2] * vel[1] + U[3] * vel[2]))
        return [rho, vel[0], vel[1], vel[2], p]

    # WENO5-Z from its integral definition (tests/_weno_def.py: parabolas, smoothness integrals and ideal
    # weights derived with numpy.polynomial, pinned against the oracle in tests/test_oracle_pins_r2.py)
    wz = wd.wenoz

    def L(U):
        W = prim(U)
        out = [np.zeros_like(U[0]) for _ in range(5)]
        for d in range(3):
            ax = 2 - d
            sh = lambda a, s: np.roll(a, -s, axis=ax)      # value at i+s
            if scheme == 0:
                plus = [wz(sh(q, -2), sh(q, -1), q, sh(q, 1), sh(q, 2)) for q in W]
                minus = [wz(sh(q, 2), sh(q, 1), q, sh(q, -1), sh(q, -2)) for q in W]
                bad = (plus[0] <= 0) | (plus[4] <= 0) | (minus[0] <= 0) | (minus[4] <= 0)
                plus = [np.where(bad, q, x) for q, x in zip(W, plus)]
                minus = [np.where(bad, q, x) for q, x in zip(W, minus)]
            else:
                plus, minus = [], []
                for q in W:
                    a, b = q - sh(q, -1), sh(q, 1) - q
                    s = np.where((a > 0) & (b > 0), np.minimum(a, b), np.where((a < 0) & (b < 0), np.maximum(a, b), 0.0))
                    plus.append(q + 0.5 * s)
                    minus.append(q - 0.5 * s)
            WL = plus                                       # left of face i+1/2
            WR = [sh(q, 1) for q in minus]                  # right of face i+1/2

            def consflux(Wk):
                rho, vel, p = Wk[0], Wk[1:4], Wk[4]
                E = p / (g - 1) + 0.5 * rho * (vel[0] ** 2 + vel[1] ** 2 + vel[2] ** 2)
                Uc = [rho, rho * vel[0], rho * vel[1], rho * vel[2], E]
                Fc = [rho * vel[d], rho * vel[0] * vel[d], rho * vel[1] * vel[d], rho * vel[2] * vel[d], (E + p) * vel[d]]
                Fc[1 + d] = Fc[1 + d] + p
                return Uc, Fc
            UL, FL = consflux(WL)
            UR, FR = consflux(WR)
            cL, cR = np.sqrt(g * WL[4] / WL[0]), np.sqrt(g * WR[4] / WR[0])
            SL = np.minimum(WL[1 + d] - cL, WR[1 + d] - cR)
            SR = np.maximum(WL[1 + d] + cL, WR[1 + d] + cR)
            F = []
            if scheme == 0:
                for m in range(5):
                    hll = (SR * FL[m] - SL * FR[m] + SL * SR * (UR[m] - UL[m])) / (SR - SL)
                    F.append(np.where(SL >= 0, FL[m], np.where(SR <= 0, FR[m], hll)))
            else:
                A = WL[0] * (SL - WL[1 + d])
                B = WR[0] * (SR - WR[1 + d])
                Ss = (WR[4] - WL[4] + A * WL[1 + d] - B * WR[1 + d]) / (A - B)
                # classical star-state form F_K + S_K (U*_K - U_K)
                for m in range(5):
                    res = []
                    for (Wk, Uk, Fk, Sk, Ak) in ((WL, UL, FL, SL, A), (WR, UR, FR, SR, B)):
                        fac = Ak / (Sk - Ss)
                        if m == 0:
                            us = fac
                        elif m == 1 + d:
                            us = fac * Ss
                        elif m == 4:
                            us = fac * (Uk[4] / Wk[0] + (Ss - Wk[1 + d]) * (Ss + Wk[4] / Ak))
                        else:
                            us = fac * Wk[m]
                        res.append(Fk[m] + Sk * (us - Uk[m]))
                    star = np.where(Ss >= 0, res[0], res[1])
                    F.append(np.where(SL >= 0, FL[m], np.where(SR <= 0, FR[m], star)))
            for m in range(5):
                out[m] -= (F[m] - sh(F[m], -1)) / sp[d]
        return out
    U = [a.copy() for a in st]
    L1 = L(U)
    U1 = [U[m] + dt * L1[m] for m in range(5)]
    L2 = L(U1)
    return [0.5 * U[m] + 0.5 * (U1[m] + dt * L2[m]) for m in range(5)]


@pytest.mark.parametrize("scheme", SCHEMES)
@pytest.mark.parametrize("n", [(4, 4, 4), (7, 5, 6)])
def test_bruteforce_whole_array_step(scheme, n):
    g = 1.4
    sp = (0.25, 0.2, 0.3)
    st = wl.random_state(n, seed=21, amp=0.6)
    dt = 0.02
    ref = _np_step(st, g, sp, dt, scheme)
    out = _run(st, n, g, wl.BC_PERIODIC, scheme, sp, dt=dt)
    for f in range(5):
        scale = np.abs(ref[f]).max()
        assert np.abs(out[f] - ref[f]).max() <= 2e-14 * scale
        assert np.abs(out[f] - st[f]).max() > 1e-4 * scale      # the step did something
