"""GPU tests of the C-ABI semantics beyond plain stepping (-m gpu): variant switching, re-setting the state,
spacing changes, device-resident latching of a non-physical state, non-default streams, library-owned workspace,
stage timing and launch counting."""
import numpy as np
import pytest

import oracle
from paper_2509_08971_b200 import hard
from paper_2509_08971_b200 import workloads as wl

from _parity import field_errors

pytestmark = pytest.mark.gpu


def _oracle_run(w, scheme, nsteps, spacing=None):
    o = oracle.Oracle(*w.n, w.gamma, w.bc, scheme=scheme, spacing=spacing or w.spacing)
    o.set_state(*w.state)
    o.step(w.cfl, nsteps)
    out = o.get_state()
    dt = o.max_dt()
    o.close()
    return out, dt


@pytest.mark.parametrize("scheme", [0, 1])
def test_variant_switch_mid_run_and_state_reset(scheme):
    w = wl.turbulence(24, nsteps=6)
    ref, dt_ref = _oracle_run(w, scheme, 6)
    h = hard.Hard(*w.n, w.gamma, w.bc, scheme=scheme, spacing=w.spacing)
    h.set_state(*w.state)
    h.step(w.cfl, 2)
    h.set_variant(hard.VARIANT_PERDIR)
    h.step(w.cfl, 2)
    h.set_variant(hard.VARIANT_FUSED)
    h.step(w.cfl, 2)
    assert max(field_errors(h.get_state(), ref)) <= 1e-11
    assert abs(h.max_dt() - dt_ref) <= 1e-11 * dt_ref
    assert h.time()[1] == 6
    # a second hard_set_state restarts the clock and reproduces the run
    h.set_state(*w.state)
    assert h.time() == (0.0, 0)
    h.step(w.cfl, 6)
    assert max(field_errors(h.get_state(), ref)) <= 1e-11
    h.close()


def test_set_spacing_after_state_reevaluates_lambda():
    w = wl.turbulence(16, nsteps=1)
    sp2 = (0.5, 0.25, 0.125)
    h = hard.Hard(*w.n, w.gamma, w.bc, spacing=w.spacing)
    h.set_state(*w.state)
    h._chk(h.L.hard_set_spacing(h.h, *sp2))
    o = oracle.Oracle(*w.n, w.gamma, w.bc, spacing=sp2)
    o.set_state(*w.state)
    assert abs(h.max_dt() - o.max_dt()) <= 1e-14 * o.max_dt()
    h.step(w.cfl, 2)
    o.step(w.cfl, 2)
    assert max(field_errors(h.get_state(), o.get_state())) <= 1e-12
    h.close()
    o.close()


def test_nonphysical_state_is_latched_on_the_device_and_surfaced():
    # a huge fixed dt drives the density negative inside hard_step; nothing returns to the host until a sync
    w = wl.sod(64)
    h = hard.Hard(*w.n, w.gamma, w.bc, spacing=w.spacing)
    h.set_state(*w.state)
    h.step_dt(1.0, 2)                       # enqueue only: no error yet
    with pytest.raises(hard.HardError) as e:
        h.get_state()
    assert e.value.code == hard.ERR_NONPHYSICAL
    with pytest.raises(hard.HardError):
        h.max_dt()
    h.set_state(*w.state)                   # a fresh state clears the latch
    h.step(w.cfl, 1)
    h.get_state()
    h.close()


def test_non_default_stream_and_library_owned_workspace():
    import torch
    w = wl.turbulence(20, nsteps=3)
    ref, _ = _oracle_run(w, 0, 3)
    s = torch.cuda.Stream()
    with torch.cuda.stream(s):
        h = hard.Hard(*w.n, w.gamma, w.bc, spacing=w.spacing)          # binds torch's current stream = s
        h.set_state(*w.state)
        h.step(w.cfl, 3)
        out = h.get_state()
    assert max(field_errors(out, ref)) <= 1e-11
    h.close()
    h2 = hard.Hard(*w.n, w.gamma, w.bc, spacing=w.spacing, torch_workspace=False)   # cudaMalloc'ed by the library
    assert 2 * 5 * 20 ** 3 * 8 < h2.workspace_bytes() < 3 * 5 * 26 ** 3 * 8   # fused: scalar block + U + U1
    h2.set_state(*w.state)
    h2.step(w.cfl, 3)
    assert max(field_errors(h2.get_state(), ref)) <= 1e-11
    h2.close()


def test_launch_count_and_stage_time():
    w = wl.turbulence(32, nsteps=4)
    h = hard.Hard(*w.n, w.gamma, w.bc, spacing=w.spacing)
    h.set_state(*w.state)
    n0 = h.launch_count()
    h.stage_time(reset=True)
    h.step(w.cfl, 4)
    ms, n = h.stage_time(reset=False)
    assert h.launch_count() - n0 == 4 * 4          # per step: ghost, stage 1, ghost, stage 2
    assert n == 8 and ms > 0.0
    h.set_variant(hard.VARIANT_PERDIR)
    n1 = h.launch_count()
    h.step(w.cfl, 1)
    assert h.launch_count() - n1 == 2 + 6 + 2 + 1   # 2 ghost fills, 6 direction passes, 2 axpy, 1 CFL
    h.close()


def test_argument_errors():
    h = hard.Hard(8, 8, 8, 1.4, 0)
    assert h.L.hard_step(h.h, -1.0, 1) == hard.ERR_ARG
    assert h.L.hard_step_dt(h.h, 0.0, 1) == hard.ERR_ARG
    assert h.L.hard_set_spacing(h.h, 0.0, 1.0, 1.0) == hard.ERR_ARG
    assert h.L.hard_set_variant(h.h, 7) == hard.ERR_ARG
    assert h.L.hard_set_rad_energy(h.h, 0) == hard.ERR_ARG
    assert h.L.hard_set_source(h.h, 1.0, 1.0, 1.0, 1.0) == hard.ERR_ARG        # radiation not enabled
    assert b"hard_enable_radiation" in h.L.hard_last_error(h.h)
    st = wl.random_state((8, 8, 8), 1)
    h.set_state(*st)
    assert h.L.hard_set_scheme(h.h, 1) == hard.ERR_ARG                          # layout is fixed once a state exists
    assert h.L.hard_enable_radiation(h.h) == hard.ERR_ARG
    h.close()


@pytest.mark.parametrize("scheme", [0, 1])
@pytest.mark.parametrize("n,bc", [((37, 21, 19), wl.BC_PERIODIC), ((30, 17, 1), wl.BC_OUTFLOW), ((45, 1, 1), wl.BC_REFLECT)])
def test_nan_poisoned_workspace(scheme, n, bc):
    """Everything the kernels may legitimately read is written by set_state / ghost fill / the stages: poison the
    whole workspace (ghost edges and corners, pitch padding, U1, the residual buffer) with NaN first; a single read
    of a never-written location by a valid cell would surface as NaN in the result (compute-sanitizer is closed on
    this pool, so this and the ragged-shape parity cases are the bounds evidence)."""
    import torch
    w = wl.Workload("r", n, 1.4, bc, (0.1, 0.07, 0.13), 0.4, nsteps=3, state=wl.random_state(n, 8))
    ref, _ = _oracle_run(w, scheme, 3)
    for variant in (hard.VARIANT_FUSED, hard.VARIANT_PERDIR):
        h = hard.Hard(*w.n, w.gamma, w.bc, scheme=scheme, variant=variant, spacing=w.spacing)
        torch.cuda.synchronize()
        base = (h.ws.data_ptr() + 255) // 256 * 256 - h.ws.data_ptr()
        body = h.ws[base + 256: base + (h.workspace_bytes() // 8) * 8].view(torch.float64)   # after the scalar block
        body.fill_(float("nan"))
        h.set_state(*w.state)
        h.step(w.cfl, 3)
        out = h.get_state()
        assert all(np.isfinite(a).all() for a in out)
        assert max(field_errors(out, ref)) <= 1e-11
        h.close()


def test_zero_steps_is_a_no_op_and_get_set_roundtrip_is_exact():
    n = (19, 14, 11)
    st = wl.random_state(n, 4)
    h = hard.Hard(*n, 1.4, wl.BC_OUTFLOW, spacing=(0.1, 0.1, 0.1))
    h.set_state(*st)
    h.step(0.4, 0)
    h.step_dt(1e-3, 0)
    out = h.get_state()
    for a, b in zip(out, st):
        assert np.array_equal(a, b)             # set/get copy the interior bit for bit
    assert h.time() == (0.0, 0)
    h.close()


@pytest.mark.parametrize("scheme", [0, 1])
def test_graph_replay_on_a_capturable_stream_matches_direct_launches(scheme):
    """hard_step with >= 8 steps on a non-default stream replays a captured two-step CUDA graph (launch-bound 1-D
    configs); the result must equal the directly launched run bit for bit, for even and odd step counts."""
    import torch
    w = wl.sod(1000)
    ref = hard.Hard(*w.n, w.gamma, w.bc, scheme=scheme, spacing=w.spacing)     # one step per call: direct launches
    ref.set_state(*w.state)
    for _ in range(28):
        ref.step(w.cfl, 1)
    for _ in range(9):
        ref.step_dt(1e-5, 1)
    exp, t_exp = ref.get_state(), ref.time()
    n_direct = ref.launch_count()
    ref.close()
    s = torch.cuda.Stream()
    with torch.cuda.stream(s):
        h = hard.Hard(*w.n, w.gamma, w.bc, scheme=scheme, spacing=w.spacing)
        h.set_state(*w.state)
        h.step(w.cfl, 3)                   # direct (fewer than 8), leaves an odd step count
        h.step(w.cfl, 25)                  # one direct step to even out + 12 graph replays
        h.step_dt(1e-5, 9)                 # new graph (fixed dt): 4 replays + 1 direct
        out, t_out = h.get_state(), h.time()
        assert h.launch_count() == n_direct
    for a, b in zip(out, exp):
        assert np.array_equal(a, b)
    assert t_out == t_exp
    h.close()


@pytest.mark.parametrize("scheme", [0, 1])
def test_graph_is_recaptured_when_spacing_or_state_changes(scheme):
    """the captured kernel nodes hold the grid descriptor (1/dx, slab flags), the source parameters and
    Lz by value; hard_set_spacing / hard_set_source / hard_set_slab / hard_set_state must invalidate the graph."""
    import torch
    w = wl.sod(400)
    sp2 = (2.0 * w.spacing[0], 1.0, 1.0)

    def run(batched):
        h = hard.Hard(*w.n, w.gamma, w.bc, scheme=scheme, spacing=w.spacing)
        h.set_state(*w.state)
        for spacing in (None, sp2, w.spacing):
            if spacing is not None:
                h._chk(h.L.hard_set_spacing(h.h, *spacing))
            if batched:
                h.step(w.cfl, 10)                        # >= 8: captured graph, replayed
            else:
                for _ in range(10):
                    h.step(w.cfl, 1)                     # direct launches
        out, t = h.get_state(), h.time()
        h.close()
        return out, t

    exp, t_exp = run(False)
    s = torch.cuda.Stream()
    with torch.cuda.stream(s):
        out, t_out = run(True)
    for a, b in zip(out, exp):
        assert np.array_equal(a, b)
    assert t_out == t_exp
    out, t_out = run(True)                               # default stream: internal capturable stream
    for a, b in zip(out, exp):
        assert np.array_equal(a, b)
    assert t_out == t_exp


def test_default_stream_batches_are_ordered_with_the_callers_stream():
    """Launch-bound meshes replay graphs on an internal non-blocking stream when the bound stream is the legacy
    default stream; work enqueued on the default stream before / after must still be ordered before / after."""
    import torch
    w = wl.sod(512)
    h = hard.Hard(*w.n, w.gamma, w.bc, spacing=w.spacing, stream=0)
    dev = [torch.from_numpy(np.ascontiguousarray(a)).cuda() for a in w.state]
    scaled = [a * 1.0 for a in dev]                      # produced on the default stream just before set_state
    h.set_state(*scaled)
    h.step(w.cfl, 40)
    out = [torch.empty_like(a) for a in dev]
    h.get_state(out)                                     # device-to-device on the bound (default) stream
    total = sum(float(a.sum()) for a in out)             # consumed on the default stream right after
    ref = hard.Hard(*w.n, w.gamma, w.bc, spacing=w.spacing)
    ref.set_state(*w.state)
    for _ in range(40):
        ref.step(w.cfl, 1)
    exp = ref.get_state()
    for a, b in zip(out, exp):
        assert np.array_equal(a.cpu().numpy(), b)
    assert total == pytest.approx(sum(float(b.sum()) for b in exp), rel=1e-13)
    assert h.launch_count() == ref.launch_count()
    h.close()
    ref.close()


def test_stage_time_can_be_switched_off_and_residual_is_allocated_on_demand():
    w = wl.turbulence(24, nsteps=2)
    ref, _ = _oracle_run(w, 0, 4)
    h = hard.Hard(*w.n, w.gamma, w.bc, spacing=w.spacing)          # workspace sized for the fused variant
    fused_bytes = h.workspace_bytes()
    h.set_state(*w.state)
    h.stage_time(reset=1)
    h.step(w.cfl, 1)
    assert h.stage_time(reset=2)[1] == 2                            # two stage launches bracketed; bracketing now off
    h.step(w.cfl, 1)
    assert h.stage_time(reset=0)[1] == 0                            # nothing recorded since
    h.set_variant(hard.VARIANT_PERDIR)                              # no third buffer in the bound workspace
    assert h.workspace_bytes() > fused_bytes                        # what a per-direction workspace would need
    h.step(w.cfl, 2)                                                # the library allocates the residual itself
    assert max(field_errors(h.get_state(), ref)) <= 1e-11
    h.close()


def test_cabi_c_program():
    """tests/test_cabi.c: plain C against include/hard.h, the five north-star calls on Sod-64 with hand values."""
    import subprocess
    from test_boundary_cpu import build_cabi_program
    exe = build_cabi_program()
    out = subprocess.run([exe], capture_output=True, text=True, timeout=300)
    assert out.returncode == 0, out.stdout + out.stderr
    assert "test_cabi ok" in out.stdout
