"""hard_max_dt_noalloc against the ordinary path (hard_create + hard_set_state + hard_max_dt).

Why the entry point exists: some users of this library cannot allocate GPU memory at the moment they need the
time step — code that runs as a plugin inside another framework's step and may only read the tensors it is given,
a service whose device pool is fixed at start-up and forbids cudaMalloc later, a diagnostic hook fired when the
application already owns all free HBM.  For them the CFL reduction keeps its scratch (per-CTA partial maxima, a
ticket counter, a flag) in a static array inside the library, and meshes above hard.NOALLOC_MAX_CELLS are refused.

What is checked: the result agrees with the ordinary path within the suite's dt tolerance (1e-14 relative; the
operation order is the same, so in practice bit for bit) on TWO CALLS IN A ROW that share the static scratch —
the second on a state with a smaller max wavespeed, so anything the first call left behind (a stale maximum, a
counter that did not return to zero, a latched non-physical flag) would show; the size limit is enforced with a
clear message; the call itself allocates nothing.

This file sorts last on purpose (pytest -x stops at the first failure, so a failure here hides no other test), and
it passes alone in a fresh process as well as after the rest of the suite: it builds its own inputs and relies on
nothing but the library."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

DT_RTOL = 1e-14          # the suite's dt tolerance (tests/_parity.py, BASELINE.json north_star)


def _ordinary_max_dt(w, state):
    from paper_2509_08971_b200 import hard
    h = hard.Hard(*w.n, w.gamma, w.bc, spacing=w.spacing)
    try:
        h.set_state(*state)
        return h.max_dt()
    finally:
        h.close()


def _noalloc_max_dt(w, dev_state, out):
    import torch
    from paper_2509_08971_b200 import hard
    hard.max_dt_noalloc(*dev_state, w.gamma, w.spacing, out)
    torch.cuda.synchronize()
    return float(out.item())


@pytest.mark.parametrize("name", ["turbulence_3d_ragged", "sod_1d", "kh_2d"])
def test_two_calls_in_a_row_match_the_ordinary_path(name):
    import torch
    from paper_2509_08971_b200 import workloads as wl
    if name == "turbulence_3d_ragged":
        # 61 x 47 x 53 = 151 951 cells: 19 CTAs of the reduction, the last one ragged; anisotropic spacing
        n = (61, 47, 53)
        w = wl.Workload("random3d", n, 1.4, 0, (1.0 / 61, 1.3 / 47, 0.8 / 53), 0.4, state=wl.random_state(n, seed=20261106))
    elif name == "sod_1d":
        w = wl.sod(1000)                                # y and z inactive: one CTA, mostly idle threads
    else:
        w = wl.kelvin_helmholtz(96)                     # z inactive
    first = [np.ascontiguousarray(a, dtype=np.float64) for a in w.state]
    # second state: the same density, momenta halved, the internal energy cut to 1/4 -> a smaller lambda everywhere
    rho, mx, my, mz, E = first
    ke = 0.5 * (mx * mx + my * my + mz * mz) / rho
    second = [rho, 0.5 * mx, 0.5 * my, 0.5 * mz, 0.25 * (E - ke) + 0.25 * ke]
    second = [np.ascontiguousarray(a) for a in second]
    want = [_ordinary_max_dt(w, s) for s in (first, second)]
    assert want[1] > want[0] * 1.5                      # the second call must not be able to pass on stale scratch
    dev = [[torch.from_numpy(a).cuda() for a in s] for s in (first, second)]
    out = torch.full((1,), -1.0, dtype=torch.float64, device="cuda")
    # the first call on a device looks up the scratch's address and makes the driver load the kernel image; that
    # one-time set-up is the caller's to place (include/hard.h), so it is done here before free memory is sampled
    assert abs(_noalloc_max_dt(w, dev[0], out) - want[0]) <= DT_RTOL * want[0]
    got = []
    mem0 = torch.cuda.mem_get_info()[0]
    for s in dev:                                       # two calls in a row, nothing in between
        got.append(_noalloc_max_dt(w, s, out))
    assert torch.cuda.mem_get_info()[0] == mem0         # free device memory unchanged: nothing was allocated
    for g, x in zip(got, want):
        assert abs(g - x) <= DT_RTOL * x, (name, g, x)
    # and once more in the first order: the scratch is back in its start state after every call
    assert abs(_noalloc_max_dt(w, dev[0], out) - want[0]) <= DT_RTOL * want[0]


def test_nonphysical_state_gives_nan_and_does_not_stick():
    import torch
    from paper_2509_08971_b200 import workloads as wl
    w = wl.turbulence(24, nsteps=1)
    good = [torch.from_numpy(np.ascontiguousarray(a)).cuda() for a in w.state]
    bad = [t.clone() for t in good]
    bad[0].view(-1)[12345 % bad[0].numel()] = -1.0       # one cell with negative density
    out = torch.zeros(1, dtype=torch.float64, device="cuda")
    assert np.isnan(_noalloc_max_dt(w, bad, out))
    want = _ordinary_max_dt(w, w.state)
    assert abs(_noalloc_max_dt(w, good, out) - want) <= DT_RTOL * want      # the flag of the call before is gone


def test_sizes_beyond_the_static_scratch_are_refused():
    import torch
    from paper_2509_08971_b200 import hard
    t = torch.ones(8, dtype=torch.float64, device="cuda")           # never read: the size check comes first
    out = torch.zeros(1, dtype=torch.float64, device="cuda")
    L = hard.lib()
    n = 323                                                          # 323^3 = 33 698 267 > 2^25
    assert n ** 3 > hard.NOALLOC_MAX_CELLS
    rc = L.hard_max_dt_noalloc(n, n, n, 1.4, 1.0, 1.0, 1.0, *[t.data_ptr()] * 5, out.data_ptr(), None)
    assert rc == hard.ERR_ARG
    msg = L.hard_noalloc_last_error().decode()
    assert "HARD_NOALLOC_MAX_CELLS" in msg and str(hard.NOALLOC_MAX_CELLS) in msg
    # host pointers are refused too (the kernel would fault on them)
    host = np.ones(8)
    rc = L.hard_max_dt_noalloc(2, 2, 2, 1.4, 1.0, 1.0, 1.0, *[host.ctypes.data] * 5, out.data_ptr(), None)
    assert rc == hard.ERR_ARG and "device memory" in L.hard_noalloc_last_error().decode()


def test_largest_accepted_mesh():
    # 2^25 cells exactly: all 4096 partial slots of the scratch in use, last CTA full
    import torch
    from paper_2509_08971_b200 import hard
    nx, ny, nz = 512, 256, 256
    assert nx * ny * nz == hard.NOALLOC_MAX_CELLS
    gen = torch.Generator(device="cuda").manual_seed(7)
    rho = 1.0 + torch.rand((nz, ny, nx), dtype=torch.float64, device="cuda", generator=gen)
    m = [0.3 * (torch.rand((nz, ny, nx), dtype=torch.float64, device="cuda", generator=gen) - 0.5) for _ in range(3)]
    E = 2.5 + torch.rand((nz, ny, nx), dtype=torch.float64, device="cuda", generator=gen)
    spacing = (1.0 / nx, 1.5 / ny, 0.75 / nz)
    out = torch.zeros(1, dtype=torch.float64, device="cuda")
    hard.max_dt_noalloc(rho, *m, E, 1.4, spacing, out)
    h = hard.Hard(nx, ny, nz, 1.4, hard.BC_PERIODIC, spacing=spacing)
    h.set_state(rho, *m, E)
    want = h.max_dt()
    h.close()
    torch.cuda.synchronize()
    assert abs(float(out.item()) - want) <= DT_RTOL * want
