"""Pins for the one constant of the oracle's WENO5-Z that round 2's mutation sweep could not see: eps.

P:151 says "WENO5-Z [18]" and no more; reading G1 takes eps = 1e-40 (power 1).  With data of ordinary
magnitude eps is invisible (beta_k >> eps), which is why eps = 1e-20 used to pass every test.  Three things the
definition itself fixes, none of which retypes oracle code:

1. Closed form.  On the stencil (s, 0, 0, 0, 0): beta_0 = 13/12 s^2 + 1/4 s^2 = 4/3 s^2, beta_1 = beta_2 = 0,
   tau = 4/3 s^2, q_0 = s/3, q_1 = q_2 = 0, alpha_0 = 0.1 (1 + 1), alpha_1 + alpha_2 = 0.9 (1 + tau/eps), so
       wenoz = (s/15) / (0.2 + 0.9 (1 + 4 s^2 / (3 eps))) = eps / (18 s) * (1 + O(eps / s^2)).
   Mirror stencil (0, 0, 0, 0, s): beta_2 = 4/3 s^2, q_2 = -s/6, alpha_2 = 0.3 * 2, alpha_0 + alpha_1 = 0.7 (1 + tau/eps):
       wenoz = -(s/10) / (0.6 + 0.7 (1 + 4 s^2 / (3 eps))) = -3 eps / (28 s) * (1 + O(eps / s^2)).
   The value is proportional to eps: it measures it.
2. Degree-1 homogeneity.  For eps -> 0 WENO-Z commutes with scaling the data; with eps = 1e-40 it does so to
   rounding for data down to 1e-12 (beta ~ 1e-24 >> eps), with eps = 1e-20 it does not.
3. The other side.  For data so small that beta << eps (scale 1e-25: beta ~ 1e-50) the non-linear weights are
   switched off, alpha_k = d_k (1 + O(1e-10)), and the result is the linear fifth-order value (ideal weights
   derived in tests/_weno_def.py from the quartic through the five cell averages).  An eps far below 1e-40
   (1e-60, 0) fails this.
"""
import numpy as np
import pytest

import oracle
import _weno_def as wd

EPS_G1 = 1e-40          # DESIGN.md reading G1

JUMPS = [(1.0, 1.0, 1.0, 0.0, 0.0), (0.0, 0.0, 1.0, 1.0, 1.0), (1.0, 1.0, 1.0, 1.0, 0.0), (0.0, 1.0, 1.0, 1.0, 1.0),
         (1.0, 2.0, 4.0, -1.0, 0.5), (0.3, 0.3, 0.3, 1.0, -2.0)]


def _random_stencils(n, seed):
    rng = np.random.default_rng(seed)
    return [tuple(rng.standard_normal(5)) for _ in range(n)]


@pytest.mark.parametrize("s", [1.0, 1e-6, 1e3, 0.37])
def test_value_on_a_one_cell_spike_measures_eps(s):
    exact_left = (s / 15.0) / (0.2 + 0.9 * (1.0 + 4.0 * s * s / (3.0 * EPS_G1)))
    exact_right = -(s / 10.0) / (0.6 + 0.7 * (1.0 + 4.0 * s * s / (3.0 * EPS_G1)))
    assert exact_left == pytest.approx(EPS_G1 / (18.0 * s), rel=1e-12)
    assert exact_right == pytest.approx(-3.0 * EPS_G1 / (28.0 * s), rel=1e-12)
    assert oracle.wenoz(s, 0.0, 0.0, 0.0, 0.0) == pytest.approx(exact_left, rel=1e-12, abs=0.0)
    assert oracle.wenoz(0.0, 0.0, 0.0, 0.0, s) == pytest.approx(exact_right, rel=1e-12, abs=0.0)


def test_the_spike_value_tells_neighbouring_eps_apart():
    # the pin has teeth: the definition evaluated with another eps gives another value, far outside the tolerance
    for wrong in (1e-20, 1e-30, 1e-36, 0.9e-40, 1.1e-40, 1e-50):
        v = float(wd.wenoz(1.0, 0.0, 0.0, 0.0, 0.0, eps=wrong))
        assert abs(v - oracle.wenoz(1.0, 0.0, 0.0, 0.0, 0.0)) > 0.05 * abs(v)
    assert float(wd.wenoz(1.0, 0.0, 0.0, 0.0, 0.0, eps=EPS_G1)) == pytest.approx(oracle.wenoz(1.0, 0.0, 0.0, 0.0, 0.0), rel=1e-12)


@pytest.mark.parametrize("s", [1e-12, 1e-8, 1e-3, 1e8, 1e12])
def test_homogeneous_of_degree_one_down_to_small_data(s):
    for q in JUMPS + _random_stencils(200, 5):
        base = oracle.wenoz(*q)
        scaled = oracle.wenoz(*[s * x for x in q])
        assert scaled == pytest.approx(s * base, rel=1e-13, abs=1e-13 * s * max(abs(x) for x in q))
    # the same property separates eps = 1e-20 (and 1e-30 at the smallest scale) from 1e-40 in the definition
    if s == 1e-12:
        q = JUMPS[0]
        good = float(wd.wenoz(*[s * x for x in q], eps=EPS_G1)) / s
        bad20 = float(wd.wenoz(*[s * x for x in q], eps=1e-20)) / s
        assert abs(good - float(wd.wenoz(*q, eps=EPS_G1))) < 1e-13 and abs(bad20 - good) > 1e-3


def test_equals_the_definition_at_every_data_scale():
    # round 2 compared at scales 1e-3 .. 1e3 only, where eps cannot be seen; 1e-18 .. 1e3 here (beta down to 1e-36)
    rng = np.random.default_rng(12)
    for _ in range(4000):
        q = rng.standard_normal(5) * 10.0 ** rng.integers(-18, 4)
        if rng.random() < 0.3:
            q[rng.integers(0, 5)] = 0.0
        ref = float(wd.wenoz(*q, eps=EPS_G1))
        assert oracle.wenoz(*q) == pytest.approx(ref, rel=2e-13, abs=2e-13 * np.abs(q).max())
    # on the same kind of data the definition with eps = 1e-30 differs visibly at the small scales
    q = np.array(JUMPS[0]) * 1e-15
    assert abs(float(wd.wenoz(*q, eps=1e-30)) - float(wd.wenoz(*q, eps=EPS_G1))) > 1e-3 * 1e-15


def test_far_below_eps_the_weights_are_the_ideal_ones():
    lin = np.zeros(5)                                    # ideal-weight combination of the three candidates
    for k in range(3):
        lin[k:k + 3] += wd.D[k] * wd.Q[k]
    s = 1e-25
    for q in JUMPS + _random_stencils(50, 6):
        want = s * float(lin @ np.array(q))
        assert oracle.wenoz(*[s * x for x in q]) == pytest.approx(want, rel=1e-8, abs=1e-8 * s * max(abs(x) for x in q))
    # while at ordinary scale the same stencils are far from the linear value (the test above is not vacuous)
    q = JUMPS[0]
    assert abs(oracle.wenoz(*q) - float(lin @ np.array(q))) > 0.1
