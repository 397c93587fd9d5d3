/* hard.h — C-ABI boundary of hard-b200: the explicit finite-volume update of the compressible Euler
 * equations on a uniform Cartesian mesh, the hot path of HARD (arxiv 2509.08971), on one B200.
 *
 * Citations: P:NNN = PAPER.md line NNN; Gn = DESIGN.md reading n; BJ = BASELINE.json north_star.
 *
 * What a simulation computes (eq.1-3, hydro rows, S = 0):
 *   U = (rho, mx, my, mz, E) cell-centred conserved densities (E = e + rho v^2/2, eq.2),
 *   ideal gas p = (gamma-1) e.  One step is Heun's method (Table 2):
 *     U1      = U^n + dt L(U^n)
 *     U^{n+1} = 1/2 U^n + 1/2 (U1 + dt L(U1))
 *   with L(U)_i = - sum_d (F*_{i+1/2} - F*_{i-1/2})_d / Delta_d (eq.15), F* an approximate
 *   Riemann flux of face values reconstructed from cell-centred primitives, ghost cells
 *   filled before each stage, and dt = cfl / lambda, lambda = max over cells and active
 *   directions of (|u_d| + c_s)/Delta_d (G6), evaluated on U^n.
 *
 * Layout of every state pointer: nx*ny*nz contiguous doubles, index i + nx*(j + ny*k), x fastest,
 * interior cells only (ghost layers are internal).  A pointer may address HOST or DEVICE memory
 * (resolved with cudaPointerGetAttributes).  The caller keeps ownership of every pointer it passes;
 * set/get copy.  The library owns its state buffers unless hard_bind_workspace lent it memory.
 *
 * Errors: every int call returns HARD_OK or a negative code; nothing throws or aborts across the
 * ABI; hard_last_error gives text.  hard_step* only enqueue work on the bound stream and return;
 * hard_max_dt, hard_get_state and hard_get_time synchronise that stream and surface a latched
 * HARD_ERR_NONPHYSICAL (non-finite value, rho <= 0 or p <= 0 seen by the CFL pass).
 * A handle is not thread-safe; distinct handles are independent.  There is no CPU fallback: every
 * call fails with HARD_ERR_CUDA when no sm_100 device is usable.
 */
#ifndef HARD_B200_HARD_H
#define HARD_B200_HARD_H

#include <stddef.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct hard_ctx hard_ctx; /* opaque, one per simulation */

enum { HARD_OK = 0, HARD_ERR_ARG = -1, HARD_ERR_CUDA = -2, HARD_ERR_NOMEM = -3, HARD_ERR_NOSTATE = -4,
       HARD_ERR_NONPHYSICAL = -5 };
enum { HARD_BC_PERIODIC = 0, HARD_BC_OUTFLOW = 1,    /* applied on all faces of active dimensions (G10) */
       HARD_BC_REFLECT = 2 };                        /* reflecting wall: mirror image, normal momentum negated (G17) */
enum { HARD_SCHEME_WENO5Z_HLL = 0,   /* the paper's scheme, P:151 (default)                       */
       HARD_SCHEME_MUSCL_HLLC = 1 }; /* BJ fallback: MUSCL-minmod + HLLC                          */
enum { HARD_VARIANT_FUSED = 0,       /* one kernel per RK stage (BJ "fused RK stage")             */
       HARD_VARIANT_PERDIR = 1 };    /* one kernel per direction + axpy + CFL (BJ comparison)     */

/* ---- the five calls BASELINE.json north_star names ------------------------------------------- */

/* Create a simulation on an nx x ny x nz mesh.  A direction with n = 1 is inactive: no
 * ghosts, no flux, not in the CFL maximum (G11); an active direction needs n >= 3.  gamma > 1.
 * Spacing defaults to 1/nx, 1/ny, 1/nz.  Uses the current CUDA device.  NULL on failure (text via
 * hard_last_error(NULL)). */
hard_ctx* hard_create(int nx, int ny, int nz, double gamma, int bc);

/* Copy five conserved fields (host or device pointers, layout above) into the state, reset t = 0,
 * fill ghosts and evaluate lambda.  Returns HARD_ERR_NONPHYSICAL if the state is not admissible. */
int hard_set_state(hard_ctx*, const double* rho, const double* mx, const double* my, const double* mz,
                   const double* E);

/* Enqueue nsteps Heun steps, each with dt_n = cfl / lambda(U^n) evaluated on the device (no host
 * round trip inside).  cfl > 0, nsteps >= 0. */
int hard_step(hard_ctx*, double cfl, int nsteps);

/* Synchronise and copy the five interior fields out (host or device pointers). */
int hard_get_state(hard_ctx*, double* rho, double* mx, double* my, double* mz, double* E);

/* Synchronise; *dt_out = 1 / lambda_max of the current state (so cfl * *dt_out is the next dt). */
int hard_max_dt(hard_ctx*, double* dt_out);

/* ---- extensions the configs cannot be run without ------------------------------------------- */

int hard_destroy(hard_ctx*);

/* Cell sizes (> 0).  Re-evaluates lambda if a state is present. */
int hard_set_spacing(hard_ctx*, double dx, double dy, double dz);

/* HARD_SCHEME_*; only before hard_set_state (ghost width 3 vs 2 changes the padded layout) and
 * before hard_bind_workspace. */
int hard_set_scheme(hard_ctx*, int scheme);

/* NEXT-1: carry the radiation energy density E_rad as a sixth advected field,
 * d_t E_rad + d_j(E_rad v^j) = 0 (eq.2 fourth row; advection part of P:141 eq.14), reconstructed like the
 * other variables, local Lax-Friedrichs (Rusanov) flux with alpha = max(|u_n| + c_s) (G19).  Sources and
 * diffusion stay out of scope.  Only before hard_set_state / hard_bind_workspace (the layout grows to six fields). */
int hard_enable_radiation(hard_ctx*);

/* Copy E_rad in / out (host or device pointer, nx*ny*nz doubles, same layout as the other fields).
 * hard_set_state zeroes E_rad; call hard_set_rad_energy after it.  hard_get_rad_energy synchronises. */
int hard_set_rad_energy(hard_ctx*, const double* e_rad);
int hard_get_rad_energy(hard_ctx*, double* e_rad);

/* NEXT-3: after every Heun step apply the pointwise radiative heating / cooling source of the
 * paper's operator split: q = c kappa rho (E_rad - a T^4) (eq.6), d_t e = q, d_t E_rad = -q
 * (eq.4), T = e / (rho cv) for the ideal gas, backward Euler over the step's dt (G20); e + E_rad is
 * conserved exactly.  Needs hard_enable_radiation.  kappa >= 0, the other parameters > 0 (any unit system). */
int hard_set_source(hard_ctx*, double kappa, double c_light, double a_rad, double cv);

/* ---- NEXT-4 (SURVEY §8(e),(f)): z-slab sharding over several GPUs, one hard_ctx per rank -------------------
 * Each rank creates its context with its own nz (>= g planes) and tells which z faces border a neighbour rank
 * (their ghost planes are then filled by the halo exchange instead of the boundary condition).  A step is driven
 * phase by phase so that the caller can exchange halos in between (paper_2509_08971_b200/sharded.py does it with
 * NCCL send/recv and one all-reduce(MAX) of lambda per step, all stream-ordered, no host synchronisation):
 *   exchange halos of buffer 0; GHOST_U; STAGE1; exchange halos of buffer 1; GHOST_U1; STAGE2;
 *   all-reduce(MAX) the double at hard_lambda_ptr(next = 1); END.
 * After hard_set_state the double at hard_lambda_ptr(next = 0) must be all-reduced likewise. */
enum { HARD_PHASE_GHOST_U = 0, HARD_PHASE_STAGE1 = 1, HARD_PHASE_GHOST_U1 = 2, HARD_PHASE_STAGE2 = 3, HARD_PHASE_END = 4 };
int hard_set_slab(hard_ctx*, int lower_neighbor, int upper_neighbor);
/* Doubles in one halo buffer: g * nx * ny * fields, laid out [field][plane][y][x]. */
size_t hard_halo_doubles(const hard_ctx*);
/* buffer: 0 = U, 1 = U1.  pack: side 0 / 1 = the g lowest / highest interior planes (for the lower / upper
 * neighbour).  unpack: side 0 / 1 = into the low / high ghost planes.  dev_buf is device memory. */
int hard_halo_pack(hard_ctx*, int buffer, int side, double* dev_buf);
int hard_halo_unpack(hard_ctx*, int buffer, int side, const double* dev_buf);
/* One phase of a step (HARD_PHASE_*); dt > 0 fixes the step, else dt = cfl / lambda.  Fused variant only. */
int hard_substep(hard_ctx*, double cfl, double dt, int phase);
/* Device address of lambda_max of the current state (next = 0) or of the state the running step produces
 * (next = 1), as a non-negative double, for an in-place all-reduce(MAX) across ranks. */
int hard_lambda_ptr(hard_ctx*, int next, double** dev_ptr);

/* HARD_VARIANT_*; may be switched at any time between steps (same state buffers). */
int hard_set_variant(hard_ctx*, int variant);

/* cudaStream_t to enqueue on (e.g. torch.cuda.current_stream().cuda_stream); default stream 0.  On launch-bound
 * meshes (<= 2^21 cells) hard_step* with >= 8 steps replays a CUDA graph of two steps; the legacy default stream
 * cannot be captured, so there the library runs those steps on an internal non-blocking stream, ordered after the
 * work already enqueued on the bound stream and before whatever is enqueued on it next (events, no host sync). */
int hard_set_stream(hard_ctx*, void* cuda_stream);

/* Bytes of device memory the simulation needs for the variant selected NOW: a 256-B scalar block + two state
 * buffers (U, U1) for HARD_VARIANT_FUSED, + one more (the residual) for HARD_VARIANT_PERDIR — select the variant
 * before asking.  If HARD_VARIANT_PERDIR is selected later on a workspace that lacks the third buffer, the library
 * cudaMalloc's the residual itself on the first per-direction step (HARD_ERR_NOMEM if that fails). */
size_t hard_workspace_bytes(const hard_ctx*);

/* Lend the library `bytes` >= hard_workspace_bytes() of device memory aligned to 256 B (e.g. a torch
 * tensor); the caller keeps it alive until hard_destroy.  Without this call the first
 * hard_set_state cudaMalloc's the workspace. */
int hard_bind_workspace(hard_ctx*, void* dev, size_t bytes);

/* nsteps Heun steps with a fixed dt (end-time clamp; light-cone sub-box parity). */
int hard_step_dt(hard_ctx*, double dt, int nsteps);

/* Synchronise; simulation time and number of steps taken since hard_set_state. */
int hard_get_time(hard_ctx*, double* t, long long* steps_done);

/* Text of the last error of this handle (NULL handle: of the last failed hard_create on this thread). */
const char* hard_last_error(const hard_ctx*);

/* Number of kernels this handle has launched since creation (bench.py's gpu_launches). */
long long hard_launch_count(const hard_ctx*);

/* Bracket the stage kernels with CUDA events on the bound stream: after hard_step returns and the
 * stream is synchronised, *ms is the summed device time and *launches the number of stage-kernel
 * launches (fused variant: the fused stage kernel; per-direction variant: all flux/axpy kernels)
 * since the last call with reset != 0.  reset = 1 (re)starts the bracketing, reset = 2 stops it (no more events
 * recorded), reset = 0 only reads.  While it is on, hard_step* does not replay CUDA graphs.  Used by bench.py for
 * the roofline of the dominant kernel. */
int hard_stage_time(hard_ctx*, int reset, double* ms, long long* launches);

/* ---- one entry point for callers that must not allocate device memory -------------------------------------
 * Everything above needs a workspace that somebody allocates: the library with cudaMalloc, or the caller before
 * hard_bind_workspace.  A caller that can do neither when it needs the time step — a plugin running inside another
 * framework's step that may only read the tensors it is handed, a process whose device pool was sized at start-up
 * and whose policy forbids cudaMalloc afterwards, a diagnostic hook fired while the application owns all free HBM —
 * uses this call instead.  It is the CFL reduction of row a7 (G6) on five caller-held fields:
 *   *dt_out = 1 / max over cells and active directions of (|u_d| + c_s) / Delta_d,
 * bit-equal to hard_set_state + hard_max_dt on the same fields and spacing (same operation order), and NaN if any
 * cell is non-physical (non-finite, rho <= 0 or p <= 0).  A direction with n = 1 is inactive, as in hard_create.
 *
 * Pointers: rho, mx, my, mz, E and dt_out are DEVICE pointers on the current CUDA device (layout at the top of this
 * file; dt_out addresses one double); the caller owns them.  The call only enqueues a 256-byte memset and one
 * kernel on cuda_stream (NULL = default stream) and returns; read *dt_out after synchronising that stream.
 * It calls no cudaMalloc, cudaFree or allocating library routine.  Its scratch (one partial maximum per 8192 cells,
 * a ticket counter, a flag: 33 024 bytes) is a static __device__ array inside the library, resident on every GPU
 * that loads the library until the process exits.  Hence the size limit: nx*ny*nz <= HARD_NOALLOC_MAX_CELLS
 * (2^25 = 33 554 432 cells, e.g. 322^3; every 1-D config and the 128^3 Sedov mesh fit); larger meshes are rejected
 * with HARD_ERR_ARG and a message naming the limit.
 * First call on a device: it looks up the device address of that array (cudaGetSymbolAddress, once per device, with
 * that device current); make this first call outside any stream capture.
 * Sharing: all calls on a device use the same array.  The call clears the counter and the flag before each launch,
 * so back-to-back calls on one stream are independent; calls whose kernels can overlap on the GPU (unordered
 * streams, several host threads) race on the array and must be ordered by the caller.
 * Errors: HARD_OK, HARD_ERR_ARG (bad size / null / host pointer / over the limit) or HARD_ERR_CUDA; text from
 * hard_noalloc_last_error() (thread-local, valid until this thread's next hard_max_dt_noalloc). */
#define HARD_NOALLOC_MAX_CELLS (1LL << 25)
int hard_max_dt_noalloc(int nx, int ny, int nz, double gamma, double dx, double dy, double dz, const double* rho,
                        const double* mx, const double* my, const double* mz, const double* E, double* dt_out,
                        void* cuda_stream);
const char* hard_noalloc_last_error(void);

/* ---- environment variables read by the library (tuning / debugging; none is needed for normal use) -------
 *   HARD_LZ=<n>            planes per z-chunk of the fused stage kernel (default: a cost model, choose_Lz)
 *   HARD_NO_GRAPH=1        never replay CUDA graphs in hard_step* (launch-bound 1-D meshes then cost more per step)
 *   HARD_DEBUG_SYNC=1      (read at hard_create) synchronise and check for errors after every kernel launch
 *   HARD_GENERIC_STAGE=1   3-D meshes use the generic stage kernel instead of the 3-D specialisation (A/B timing)
 * The fp64-peak probe bench.py uses for its roofline lives in its own library: include/hard_probe.h. */

#ifdef __cplusplus
}
#endif
#endif /* HARD_B200_HARD_H */
