"""The five BASELINE.json configs run to completion on the GPU (-m gpu) and checked against what the mathematics
fixes: exact Riemann solutions (C0, C1), the Sedov-Taylor shock radius (C2), conservation on the periodic boxes
(C3, C4).  The oracle cannot do the long ones in reasonable time (C2: ~300 steps of 128^3); these tests hold the
CUDA path itself to the analytic pins the oracle is held to."""
import math

import numpy as np
import pytest

import oracle
from oracle import exact
from paper_2509_08971_b200 import hard
from paper_2509_08971_b200 import workloads as wl

from _parity import field_errors

pytestmark = pytest.mark.gpu


def _gpu_run_to(w, scheme):
    h = hard.Hard(*w.n, w.gamma, w.bc, scheme=scheme, spacing=w.spacing)
    h.set_state(*w.state)
    n = h.run_to(w.t_end, w.cfl)
    out = h.get_state()
    t, steps = h.time()
    h.close()
    assert steps == n and abs(t - w.t_end) <= 1e-12 * w.t_end
    return out, n


@pytest.mark.parametrize("scheme,bound", [(0, 6e-4), (1, 1.5e-3)])
def test_c0_sod_full_run(scheme, bound):
    w = wl.sod(1000)
    out, n = _gpu_run_to(w, scheme)
    m = w.meta
    l1 = exact.riemann_l1_density(out[0].ravel(), m["x_lo"], w.spacing[0], m["x0"], w.t_end, m["left"], m["right"], w.gamma)
    assert l1 <= bound
    # the whole ~1100-step run stays on the oracle's trajectory
    o = oracle.Oracle(*w.n, w.gamma, w.bc, scheme=scheme, spacing=w.spacing)
    o.set_state(*w.state)
    assert o.run_to(w.t_end, w.cfl) == n
    assert max(field_errors(out, o.get_state())) <= 1e-9
    o.close()


def test_paper_sod_bound_on_gpu():
    """P:215 on the CUDA path: scheme A, dx = 2^-10, t = 0.0669, CFL 0.3: L1 < 5e-4."""
    w = wl.sod(1024, 0.0669, 0.3)
    out, _ = _gpu_run_to(w, 0)
    m = w.meta
    assert exact.riemann_l1_density(out[0].ravel(), 0.0, w.spacing[0], 0.5, 0.0669, m["left"], m["right"], 1.4) < 5e-4


@pytest.mark.parametrize("scheme", [0, 1])
def test_c1_leblanc_full_run(scheme):
    w = wl.leblanc(4096)
    out, n = _gpu_run_to(w, scheme)
    assert n > 9000 and out[0].min() > 0
    g = w.gamma
    ws = exact.riemann_waves(1.0, 0.0, (g - 1) * 0.1, 1e-3, 0.0, (g - 1) * 1e-10, g)
    x_shock = 3.0 + 6.0 * ws["shock_R"]
    xc = (np.arange(4096) + 0.5) * w.spacing[0]
    shock = xc[np.where(out[0].ravel() > 0.5 * (ws["rho_star_R"] + 1e-3))[0].max()]
    assert abs(shock - x_shock) <= 0.005 * x_shock
    m = w.meta
    l1 = exact.riemann_l1_density(out[0].ravel(), 0.0, w.spacing[0], 3.0, 6.0, m["left"], m["right"], g)
    assert l1 <= (2.0e-3 if scheme == 0 else 3.0e-3)


@pytest.mark.parametrize("scheme", [0, 1])
def test_c2_sedov_full_run(scheme):
    w = wl.sedov(128)
    out, n = _gpu_run_to(w, scheme)
    rho = out[0]
    dx = w.spacing[0]
    xc = -1.0 + (np.arange(128) + 0.5) * dx
    Z, Y, X = np.meshgrid(xc, xc, xc, indexing="ij")
    r = np.sqrt(X * X + Y * Y + Z * Z).ravel()
    nb = 64
    idx = np.minimum((r / dx).astype(int), nb - 1)
    prof = np.bincount(idx, weights=rho.ravel(), minlength=nb) / np.maximum(np.bincount(idx, minlength=nb), 1)
    ipk = int(np.argmax(prof))
    half = 0.5 * (prof[ipk] + 1.0)
    i = next(i for i in range(ipk, nb - 1) if prof[i] >= half > prof[i + 1])
    R_num = (i + 0.5) * dx + (prof[i] - half) / (prof[i] - prof[i + 1]) * dx
    assert abs(R_num - exact.sedov_radius(w.t_end, 1.0, 1.0, w.gamma)) <= 2.0 * dx
    E0 = math.fsum(w.state[4].ravel().tolist())
    assert abs(math.fsum(out[4].ravel().tolist()) - E0) <= 1e-11 * E0          # nothing has left the box
    for ax in range(3):                                                        # symmetric to rounding
        assert np.abs(rho - np.flip(rho, ax)).max() <= 1e-9 * rho.max()
    assert np.abs(rho - rho.transpose(2, 1, 0)).max() <= 1e-9 * rho.max()
    assert 150 < n < 600


@pytest.mark.parametrize("n,nsteps", [(512, 20), (896, 10)])
def test_c3_c4_conservation_full_size(n, nsteps):
    import torch
    w = wl.turbulence(n, nsteps=nsteps, device="cuda")
    before = [float(a.sum(dtype=torch.float64)) for a in w.state]
    scale = [float(a.abs().sum(dtype=torch.float64)) for a in w.state]
    h = hard.Hard(*w.n, w.gamma, w.bc, spacing=w.spacing)
    h.set_state(*w.state)
    h.step(w.cfl, nsteps)
    out = [torch.empty_like(a) for a in w.state]
    h.get_state(out)
    h.close()
    for f in range(5):
        assert abs(float(out[f].sum(dtype=torch.float64)) - before[f]) <= 1e-11 * scale[f]
        assert float((out[f] - w.state[f]).abs().max()) > 0
    assert float(out[0].min()) > 0.1
