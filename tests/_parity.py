"""Shared helpers of the GPU parity tests: run the CUDA path (through the C-ABI binding) and the
oracle on the same seeded inputs and compare per field with the norm of DESIGN.md G15."""
import numpy as np

import oracle
from paper_2509_08971_b200 import hard

FIELDS = ("rho", "mx", "my", "mz", "E")


def field_errors(gpu, orc):
    """max |gpu - orc| / max |orc| per field; a field that is identically zero in the oracle must be
    identically zero on the GPU (reported as 0.0, else inf)."""
    errs = []
    for a, b in zip(gpu, orc):
        scale = np.abs(b).max()
        if scale == 0.0:
            errs.append(0.0 if not np.any(a) else np.inf)
        else:
            errs.append(float(np.abs(a - b).max() / scale))
    return errs


def pointwise_errors(gpu, orc):
    """max over cells of |gpu - orc| / |orc| for the strictly positive fields rho and E (fields 0 and 4): the cell-by-cell
    relative error, which the field norm above cannot see where a field spans many decades."""
    out = []
    for f in (0, 4):
        a, b = gpu[f], orc[f]
        assert np.all(b > 0)
        out.append(float((np.abs(a - b) / b).max()))
    return out


def run_both(w, scheme, variant=hard.VARIANT_FUSED, nsteps=1, cfl=None, dt=None, state=None):
    """Returns (gpu_fields, oracle_fields, (gpu_dt0, orc_dt0), (gpu_t, orc_t))."""
    cfl = w.cfl if cfl is None else cfl
    st = [np.ascontiguousarray(a, dtype=np.float64) for a in (w.state if state is None else state)]
    o = oracle.Oracle(*w.n, w.gamma, w.bc, scheme=scheme, spacing=w.spacing)
    o.set_state(*st)
    h = hard.Hard(*w.n, w.gamma, w.bc, scheme=scheme, variant=variant, spacing=w.spacing)
    h.set_state(*st)
    dts = (h.max_dt(), o.max_dt())
    if dt is None:
        o.step(cfl, nsteps)
        h.step(cfl, nsteps)
    else:
        o.step_dt(dt, nsteps)
        h.step_dt(dt, nsteps)
    out_h = h.get_state()
    out_o = o.get_state()
    ts = (h.time()[0], o.time()[0])
    dts_end = (h.max_dt(), o.max_dt())
    h.close()
    o.close()
    return out_h, out_o, dts, ts, dts_end
