"""Thin Python binding of the C-ABI in include/hard.h (same names, argument marshalling only).

PyTorch is used for device memory (the workspace tensor lent through hard_bind_workspace, state
tensors) and streams; every step of the hot path runs in the CUDA kernels of csrc/.  There is no CPU
fallback: loading fails loudly when the extension is missing, hard_create fails without a B200.
"""
from __future__ import annotations

import ctypes
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libhard_b200.so")
PROBE_LIB_PATH = os.path.join(_HERE, "libhard_probe.so")     # include/hard_probe.h: measurement utility, not the product ABI

OK, ERR_ARG, ERR_CUDA, ERR_NOMEM, ERR_NOSTATE, ERR_NONPHYSICAL = 0, -1, -2, -3, -4, -5
BC_PERIODIC, BC_OUTFLOW, BC_REFLECT = 0, 1, 2
SCHEME_WENO5Z_HLL, SCHEME_MUSCL_HLLC = 0, 1
VARIANT_FUSED, VARIANT_PERDIR = 0, 1

EXPORTS = ["hard_create", "hard_set_state", "hard_step", "hard_get_state", "hard_max_dt", "hard_destroy",
           "hard_set_spacing", "hard_set_scheme", "hard_set_variant", "hard_set_stream", "hard_workspace_bytes",
           "hard_bind_workspace", "hard_step_dt", "hard_get_time", "hard_last_error", "hard_launch_count",
           "hard_stage_time", "hard_enable_radiation", "hard_set_rad_energy",
           "hard_get_rad_energy", "hard_set_source", "hard_set_slab", "hard_halo_doubles", "hard_halo_pack",
           "hard_halo_unpack", "hard_substep", "hard_lambda_ptr", "hard_max_dt_noalloc", "hard_noalloc_last_error"]
NOALLOC_MAX_CELLS = 1 << 25          # HARD_NOALLOC_MAX_CELLS of include/hard.h

_lib = None


def lib():
    """Load libhard_b200.so (built in-tree by paper_2509_08971_b200.build / __graft_entry__.build)."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        try:                                   # compile it (nvcc, sm_100a); this is a build step, not a fallback
            from . import build as _build
            _build.build()
        except Exception as ex:
            raise RuntimeError("libhard_b200.so is not built and could not be compiled (%s): run "
                               "`python -m paper_2509_08971_b200.build` (there is no CPU fallback)" % ex)
    L = ctypes.CDLL(LIB_PATH)
    vp, dp, c_int, c_dbl = ctypes.c_void_p, ctypes.c_void_p, ctypes.c_int, ctypes.c_double
    L.hard_create.restype = vp
    L.hard_create.argtypes = [c_int, c_int, c_int, c_dbl, c_int]
    L.hard_set_state.argtypes = [vp] + [dp] * 5
    L.hard_get_state.argtypes = [vp] + [dp] * 5
    L.hard_step.argtypes = [vp, c_dbl, c_int]
    L.hard_step_dt.argtypes = [vp, c_dbl, c_int]
    L.hard_max_dt.argtypes = [vp, ctypes.POINTER(c_dbl)]
    L.hard_destroy.argtypes = [vp]
    L.hard_set_spacing.argtypes = [vp, c_dbl, c_dbl, c_dbl]
    L.hard_set_scheme.argtypes = [vp, c_int]
    L.hard_set_variant.argtypes = [vp, c_int]
    L.hard_set_stream.argtypes = [vp, vp]
    L.hard_workspace_bytes.restype = ctypes.c_size_t
    L.hard_workspace_bytes.argtypes = [vp]
    L.hard_bind_workspace.argtypes = [vp, vp, ctypes.c_size_t]
    L.hard_get_time.argtypes = [vp, ctypes.POINTER(c_dbl), ctypes.POINTER(ctypes.c_longlong)]
    L.hard_last_error.restype = ctypes.c_char_p
    L.hard_last_error.argtypes = [vp]
    L.hard_launch_count.restype = ctypes.c_longlong
    L.hard_launch_count.argtypes = [vp]
    L.hard_stage_time.argtypes = [vp, c_int, ctypes.POINTER(c_dbl), ctypes.POINTER(ctypes.c_longlong)]
    L.hard_enable_radiation.argtypes = [vp]
    L.hard_set_rad_energy.argtypes = [vp, dp]
    L.hard_get_rad_energy.argtypes = [vp, dp]
    L.hard_set_source.argtypes = [vp, c_dbl, c_dbl, c_dbl, c_dbl]
    L.hard_set_slab.argtypes = [vp, c_int, c_int]
    L.hard_halo_doubles.restype = ctypes.c_size_t
    L.hard_halo_doubles.argtypes = [vp]
    L.hard_halo_pack.argtypes = [vp, c_int, c_int, dp]
    L.hard_halo_unpack.argtypes = [vp, c_int, c_int, dp]
    L.hard_substep.argtypes = [vp, c_dbl, c_dbl, c_int]
    L.hard_lambda_ptr.argtypes = [vp, c_int, ctypes.POINTER(ctypes.c_void_p)]
    L.hard_max_dt_noalloc.argtypes = [c_int, c_int, c_int, c_dbl, c_dbl, c_dbl, c_dbl] + [dp] * 6 + [vp]
    L.hard_noalloc_last_error.restype = ctypes.c_char_p
    L.hard_noalloc_last_error.argtypes = []
    _lib = L
    return L


_probe = None


def probe_fp64_peak():
    """fp64 vector peak of the current device, TFLOP/s (measurement utility, libhard_probe.so)."""
    global _probe
    if _probe is None:
        if not os.path.exists(PROBE_LIB_PATH):
            from . import build as _build
            _build.build()
        _probe = ctypes.CDLL(PROBE_LIB_PATH)
        _probe.hard_probe_fp64_peak.argtypes = [ctypes.POINTER(ctypes.c_double), ctypes.POINTER(ctypes.c_double)]
    v = ctypes.c_double()
    rc = _probe.hard_probe_fp64_peak(ctypes.byref(v), None)
    if rc != OK:
        raise HardError(rc, "hard_probe_fp64_peak")
    return v.value


class HardError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__("hard error %d: %s" % (code, msg))
        self.code = code


def _ptr(a):
    """Raw address of a numpy array (host) or torch tensor (host or device), float64 contiguous."""
    if isinstance(a, np.ndarray):
        assert a.dtype == np.float64 and a.flags["C_CONTIGUOUS"]
        return a.ctypes.data
    assert a.dtype.is_floating_point and a.element_size() == 8 and a.is_contiguous()
    return a.data_ptr()


def max_dt_noalloc(rho, mx, my, mz, E, gamma, spacing, out, stream=None):
    """hard_max_dt_noalloc: 1 / lambda_max of five device fields of shape (nz, ny, nx) into the one-element device
    tensor `out`, without any device allocation (the reduction's scratch is a static array inside the library).

    For callers that may not allocate on the GPU when they need dt (code running inside another framework's step,
    fixed memory pools, hooks fired when no HBM is free) — see include/hard.h for the limit (NOALLOC_MAX_CELLS
    cells), the first-call set-up and the rule that overlapping calls race.  Marshalling only: this function creates
    no tensor; the call is asynchronous on `stream` (default: torch's current stream), so synchronise before reading
    `out`, which holds NaN if the state is non-physical."""
    L = lib()
    nz, ny, nx = rho.shape
    for a in (rho, mx, my, mz, E):
        assert tuple(a.shape) == (nz, ny, nx) and a.is_cuda
    assert out.is_cuda and out.numel() >= 1
    if stream is None:
        import torch
        stream = torch.cuda.current_stream().cuda_stream
    rc = L.hard_max_dt_noalloc(nx, ny, nz, float(gamma), *map(float, spacing), *[_ptr(a) for a in (rho, mx, my, mz, E)],
                               _ptr(out), stream)
    if rc != OK:
        raise HardError(rc, L.hard_noalloc_last_error().decode())


class Hard:
    """One simulation (hard_ctx).  Fields are (nz, ny, nx) float64, conserved (rho, mx, my, mz, E)."""

    def __init__(self, nx, ny, nz, gamma, bc, scheme=SCHEME_WENO5Z_HLL, variant=VARIANT_FUSED, spacing=None,
                 torch_workspace=True, stream=None, radiation=False):
        self.L = lib()
        self.n = (nx, ny, nz)
        self.shape = (nz, ny, nx)
        self.h = self.L.hard_create(nx, ny, nz, float(gamma), int(bc))
        if not self.h:
            raise HardError(ERR_CUDA, self.L.hard_last_error(None).decode())
        self._chk(self.L.hard_set_scheme(self.h, scheme))
        self._chk(self.L.hard_set_variant(self.h, variant))
        if radiation:
            self._chk(self.L.hard_enable_radiation(self.h))
        if spacing is not None:
            self._chk(self.L.hard_set_spacing(self.h, *map(float, spacing)))
        self.ws = None
        if torch_workspace:
            import torch
            nbytes = self.L.hard_workspace_bytes(self.h)
            self.ws = torch.empty(nbytes + 256, dtype=torch.uint8, device="cuda")
            base = (self.ws.data_ptr() + 255) // 256 * 256
            self._chk(self.L.hard_bind_workspace(self.h, base, nbytes))
            if stream is None:
                stream = torch.cuda.current_stream().cuda_stream
        if stream:
            self._chk(self.L.hard_set_stream(self.h, stream))

    def _chk(self, rc):
        if rc != OK:
            raise HardError(rc, self.L.hard_last_error(self.h).decode())

    def close(self):
        if getattr(self, "h", None):
            self.L.hard_destroy(self.h)
            self.h = None
            self.ws = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    # ---- the five north-star calls
    def set_state(self, rho, mx, my, mz, E):
        self._chk(self.L.hard_set_state(self.h, *[_ptr(a) for a in (rho, mx, my, mz, E)]))

    def step(self, cfl, nsteps=1):
        self._chk(self.L.hard_step(self.h, float(cfl), int(nsteps)))

    def get_state(self, out=None):
        if out is None:
            out = [np.empty(self.shape, dtype=np.float64) for _ in range(5)]
        self._chk(self.L.hard_get_state(self.h, *[_ptr(a) for a in out]))
        return out

    def max_dt(self):
        v = ctypes.c_double()
        self._chk(self.L.hard_max_dt(self.h, ctypes.byref(v)))
        return v.value

    # ---- extensions
    # ---- NEXT-4: z-slab sharding primitives (see sharded.py)
    def set_slab(self, lower, upper):
        self._chk(self.L.hard_set_slab(self.h, int(lower), int(upper)))

    def halo_doubles(self):
        return int(self.L.hard_halo_doubles(self.h))

    def halo_pack(self, buffer, side, buf):
        self._chk(self.L.hard_halo_pack(self.h, buffer, side, _ptr(buf)))

    def halo_unpack(self, buffer, side, buf):
        self._chk(self.L.hard_halo_unpack(self.h, buffer, side, _ptr(buf)))

    def substep(self, phase, cfl=0.0, dt=0.0):
        self._chk(self.L.hard_substep(self.h, float(cfl), float(dt), int(phase)))

    def lambda_ptr(self, nxt):
        p = ctypes.c_void_p()
        self._chk(self.L.hard_lambda_ptr(self.h, int(nxt), ctypes.byref(p)))
        return p.value

    def set_source(self, kappa, c_light, a_rad, cv):
        self._chk(self.L.hard_set_source(self.h, float(kappa), float(c_light), float(a_rad), float(cv)))

    def set_rad_energy(self, er):
        self._chk(self.L.hard_set_rad_energy(self.h, _ptr(er)))

    def get_rad_energy(self, out=None):
        if out is None:
            out = np.empty(self.shape, dtype=np.float64)
        self._chk(self.L.hard_get_rad_energy(self.h, _ptr(out)))
        return out

    def set_variant(self, variant):
        self._chk(self.L.hard_set_variant(self.h, variant))

    def step_dt(self, dt, nsteps=1):
        self._chk(self.L.hard_step_dt(self.h, float(dt), int(nsteps)))

    def time(self):
        t, n = ctypes.c_double(), ctypes.c_longlong()
        self._chk(self.L.hard_get_time(self.h, ctypes.byref(t), ctypes.byref(n)))
        return t.value, n.value

    def launch_count(self):
        return int(self.L.hard_launch_count(self.h))

    def stage_time(self, reset=True):
        ms, n = ctypes.c_double(), ctypes.c_longlong()
        self._chk(self.L.hard_stage_time(self.h, int(reset), ctypes.byref(ms), ctypes.byref(n)))
        return ms.value, n.value

    def workspace_bytes(self):
        return int(self.L.hard_workspace_bytes(self.h))

    def run_to(self, t_end, cfl, max_steps=10 ** 7):
        """Harness loop: hard_step(cfl, .) while t < t_end, last step clamped to land on t_end.

        Far from t_end the steps are enqueued in batches (one host synchronisation per batch instead of two per
        step; on launch-bound meshes the batch replays a CUDA graph): a batch covers at most a quarter of the
        remaining time at the current dt and at most 256 steps, so it cannot reach t_end unless dt quadruples within
        256 steps — checked (an overshoot raises; 256 keeps the graph-replay benefit, one sync per 256 steps).
        The dt sequence is the same as stepping one by one: dt_n = cfl / lambda(U^n) is evaluated on the device."""
        n = 0
        while n < max_steps:
            t, _ = self.time()
            if t >= t_end:
                break
            dt = cfl * self.max_dt()
            if t + dt >= t_end:
                self.step_dt(t_end - t, 1)
                n += 1
                break
            batch = min(int(0.25 * (t_end - t) / dt), max_steps - n, 256)
            if batch >= 8:
                self.step(cfl, batch)
                n += batch
                t2, _ = self.time()
                if t2 >= t_end:
                    raise HardError(ERR_ARG, "run_to: a batch of steps overshot t_end (dt grew more than fourfold)")
            else:
                self.step(cfl, 1)
                n += 1
        return n
