// hard_api.cu — host side of the C-ABI declared in include/hard.h: handle, padded SoA layout in HBM,
// tensor maps, launch sequencing of one Heun step (Table 2), set/get copies, errors.
// No CPU fallback: every entry point fails with HARD_ERR_CUDA when CUDA is unusable.
#include <cuda.h>
#include <cuda_runtime.h>

#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <string>
#include <vector>

#include "../../include/hard.h"
#include "hard_kernels.cuh"

using namespace hard;

namespace {

thread_local std::string g_create_error;

typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*,
                                  const cuuint64_t*, const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave,
                                  CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

size_t align_up(size_t x, size_t a) { return (x + a - 1) / a * a; }

}  // namespace

struct hard_ctx {
  GridDesc g;
  int scheme = HARD_SCHEME_WENO5Z_HLL, variant = HARD_VARIANT_FUSED;
  int zskip = 0;                    // NEXT-4: z ghost faces that a neighbour rank fills (hard_set_slab)
  bool src_on = false;              // NEXT-3: heating/cooling source after every step (hard_set_source)
  SourceParams src{};
  int nf = 5;                       // 6 with the advected radiation energy density (hard_enable_radiation)
  cudaStream_t stream = 0;
  void* ws = nullptr;
  size_t ws_bytes = 0;
  bool ws_owned = false;
  DevScalars* sc = nullptr;
  double *U = nullptr, *U1 = nullptr, *Rres = nullptr;
  bool rres_owned = false;          // residual of the per-direction variant cudaMalloc'ed by the library
  cudaStream_t own_stream = nullptr;   // internal capturable stream for graph replay when the bound stream is the legacy default
  cudaEvent_t ev_in = nullptr, ev_out = nullptr;
  CUtensorMap tmU, tmU1;
  bool maps_ready = false;
  bool have_state = false;
  long long steps_enq = 0;          // host-side parity of the lambda ping-pong
  long long launches = 0;
  int Lz = 0;
  int sm_count = 148;
  int device = 0;                   // the CUDA device the context was created on
  std::string err;
  bool profiling = false;
  bool debug_sync = false;            // HARD_DEBUG_SYNC=1: synchronise and check after every launch
  // CUDA graph of two consecutive steps (even + odd lambda slot), replayed by hard_step* on capturable streams
  cudaGraphExec_t gexec = nullptr;
  double g_cfl = 0.0, g_dt = 0.0;
  int g_sig = -1;                   // variant / source / stream signature the graph was captured for
  long long g_gen = -1, gen = 0;    // generation of everything the captured nodes bake in by value (grid, spacing, source, slab, Lz)
  cudaStream_t g_stream = nullptr;
  bool graphs_ok = true;            // cleared when the bound stream cannot be captured (legacy default stream)
  std::vector<cudaEvent_t> ev;      // start/stop pairs around stage kernels
  size_t ev_used = 0;
};

namespace {

// Entry points run on the context's device whatever the caller's current device is.
struct DeviceGuard {
  int prev = -1;
  explicit DeviceGuard(const hard_ctx* c) {
    if (c && cudaGetDevice(&prev) == cudaSuccess && prev != c->device) cudaSetDevice(c->device); else prev = -1;
  }
  ~DeviceGuard() { if (prev >= 0) cudaSetDevice(prev); }
};

int fail(hard_ctx* c, int code, const std::string& msg) {
  if (c) c->err = msg;
  return code;
}
int cuda_fail(hard_ctx* c, cudaError_t e, const char* where) {
  return fail(c, HARD_ERR_CUDA, std::string(where) + ": " + cudaGetErrorString(e));
}
int after_launch(hard_ctx* c, const char* name);
#define CK(call)                                                  \
  do {                                                            \
    cudaError_t e__ = (call);                                     \
    if (e__ != cudaSuccess) return cuda_fail(c, e__, #call);      \
  } while (0)

int after_launch(hard_ctx* c, const char* name) {
  c->launches++;
  cudaError_t e = cudaGetLastError();
  if (e == cudaSuccess && c->debug_sync) e = cudaStreamSynchronize(c->stream);
  if (e != cudaSuccess) return cuda_fail(c, e, name);
  return HARD_OK;
}

void compute_layout(hard_ctx* c) {
  GridDesc& g = c->g;
  g.g = (c->scheme == HARD_SCHEME_WENO5Z_HLL) ? 3 : 2;
  g.nf = c->nf;
  g.zskip = c->zskip;
  for (int a = 0; a < 3; ++a) g.act[a] = g.n[a] > 1;
  // x: ghost width g on the left, so that a tile's TMA box (which starts g cells left of the 14-cell tile)
  // starts at padded x-coordinate 14 * tile, an EVEN coordinate: the innermost start coordinate of an fp64
  // box must be 16-byte aligned (measured: an odd start raises "illegal instruction" on sm_100a).
  // Row pitch: a multiple of 16 doubles (TMA strides must be multiples of 16 B; rows start on 128-B lines).
  g.off[0] = g.g;   // also when x is inactive (the columns stay zero and are never read by a valid cell)
  g.off[1] = g.act[1] ? g.g : 0;
  g.off[2] = g.act[2] ? g.g : 0;
  g.P[0] = (int)align_up((size_t)g.off[0] + g.n[0] + (g.act[0] ? g.g : 0), 16);
  g.P[1] = g.n[1] + 2 * g.off[1];
  g.P[2] = g.n[2] + 2 * g.off[2];
  g.pitch = g.P[0];
  g.plane = g.pitch * g.P[1];
  g.fstride = (long long)align_up((size_t)(g.plane * g.P[2]), 32);
}

size_t state_bytes(const hard_ctx* c) { return (size_t)c->nf * c->g.fstride * sizeof(double); }

void carve(hard_ctx* c) {
  char* p = (char*)c->ws;
  c->sc = (DevScalars*)p;
  p += 256;
  const size_t sb = align_up(state_bytes(c), 256);
  c->U = (double*)p;  p += sb;
  c->U1 = (double*)p; p += sb;
  if (!c->rres_owned) c->Rres = (c->ws_bytes >= 256 + 3 * sb) ? (double*)p : nullptr;   // else allocated on first use
}

int make_map(hard_ctx* c, CUtensorMap* m, double* base) {
  static EncodeTiledFn fn = nullptr;
  if (!fn) {
    void* p = nullptr;
    cudaDriverEntryPointQueryResult q;
    cudaError_t e = cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &q);
    if (e != cudaSuccess || q != cudaDriverEntryPointSuccess || !p)
      return fail(c, HARD_ERR_CUDA, "cuTensorMapEncodeTiled entry point unavailable");
    fn = (EncodeTiledFn)p;
  }
  const GridDesc& g = c->g;
  const int BXh = 14 + 2 * g.g, BYh = 16 + 2 * g.g;          // StageCfg<S>::BX, BY
  cuuint64_t dims[4] = { (cuuint64_t)g.P[0], (cuuint64_t)g.P[1], (cuuint64_t)g.P[2], (cuuint64_t)g.nf };
  cuuint64_t strides[3] = { (cuuint64_t)g.pitch * 8, (cuuint64_t)g.plane * 8, (cuuint64_t)g.fstride * 8 };
  cuuint32_t box[4] = { (cuuint32_t)BXh, (cuuint32_t)BYh, 1, (cuuint32_t)g.nf };
  cuuint32_t es[4] = { 1, 1, 1, 1 };
  CUresult r = fn(m, CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 4, base, dims, strides, box, es, CU_TENSOR_MAP_INTERLEAVE_NONE,
                  CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_128B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
  if (r != CUDA_SUCCESS) {
    char buf[96];
    snprintf(buf, sizeof buf, "cuTensorMapEncodeTiled failed with CUresult %d", (int)r);
    return fail(c, HARD_ERR_CUDA, buf);
  }
  return HARD_OK;
}

int choose_Lz(const hard_ctx* c) {
  const GridDesc& g = c->g;
  const long long tiles = (long long)((g.n[0] + 13) / 14) * ((g.n[1] + 15) / 16);
  const int nz = g.n[2];
  if (!g.act[2]) return 1;
  if (const char* e = getenv("HARD_LZ")) {                   // tuning override (planes per z-chunk)
    const int v = atoi(e);
    if (v >= 1) return v < nz ? v : nz;
  }
  // cost model (planes of work on the critical path): (waves + 1) * (chunk length + lead-in), where
  // waves = CTAs / (2 CTAs per SM * SMs) and the +1 is the measured tail of unequal CTA progress
  // (512^3: one 512-plane chunk per tile = exactly 4 waves ran 15 % slower than 64-plane chunks).
  const double lead = 2.0 + 0.5 * (2 * (g.g - 1) + 1);      // z-only iterations + prologue loads, in plane units
  const double ctas_per_sm = (c->nf == 6 && c->scheme == HARD_SCHEME_WENO5Z_HLL) ? 1.0 : 2.0;
  double best = 1e300;
  int bestc = 1;
  for (int ch = 1; ch <= (nz + 15) / 16; ++ch) {
    const int lz = (nz + ch - 1) / ch;
    const long long ctas = tiles * ((nz + lz - 1) / lz);
    const double waves = (double)ctas / (ctas_per_sm * c->sm_count);
    const double cost = (waves + 1.0) * (lz + lead);
    if (cost < best * 0.999) { best = cost; bestc = ch; }
  }
  return (nz + bestc - 1) / bestc;
}

int ensure_ready(hard_ctx* c) {
  if (!c->ws) {
    const size_t need = hard_workspace_bytes(c);
    cudaError_t e = cudaMalloc(&c->ws, need);
    if (e != cudaSuccess) { c->ws = nullptr; return fail(c, HARD_ERR_NOMEM, std::string("cudaMalloc: ") + cudaGetErrorString(e)); }
    c->ws_bytes = need;
    c->ws_owned = true;
    CK(cudaMemsetAsync(c->ws, 0, need, c->stream));
    carve(c);
  }
  if (!c->maps_ready) {
    int rc = make_map(c, &c->tmU, c->U);
    if (rc) return rc;
    rc = make_map(c, &c->tmU1, c->U1);
    if (rc) return rc;
#define HARD_SET_SMEM(S, NF) \
  CK(cudaFuncSetAttribute(stage_kernel<S, NF>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)StageCfg<S, NF>::SMEM)); \
  CK(cudaFuncSetAttribute(stage3d_kernel<S, NF, MODE_STAGE1>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)StageCfg<S, NF>::SMEM3D)); \
  CK(cudaFuncSetAttribute(stage3d_kernel<S, NF, MODE_STAGE2>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)StageCfg<S, NF>::SMEM3D));
    HARD_SET_SMEM(SCHEME_A, 5) HARD_SET_SMEM(SCHEME_B, 5) HARD_SET_SMEM(SCHEME_A, 6) HARD_SET_SMEM(SCHEME_B, 6)
#undef HARD_SET_SMEM
    c->Lz = choose_Lz(c);
    c->maps_ready = true;
  }
  return HARD_OK;
}

int small_grid(const hard_ctx* c, long long work) {
  long long b = (work + 255) / 256;
  const long long cap = (long long)c->sm_count * 8;
  if (b > cap) b = cap;
  if (b < 1) b = 1;
  return (int)b;
}

int launch_ghost(hard_ctx* c, double* U, int advance, double cfl, double dt_fixed) {
  const GridDesc& g = c->g;
  long long work = 0;
  if (g.act[0]) work += 2LL * g.g * g.n[1] * g.n[2];
  if (g.act[1]) work += 2LL * g.g * g.n[0] * g.n[2];
  if (g.act[2]) work += 2LL * g.g * g.n[0] * g.n[1];
  ghost_fill_kernel<<<small_grid(c, work), 256, 0, c->stream>>>(U, g, c->sc, advance, (int)(c->steps_enq & 1), cfl, dt_fixed);
  return after_launch(c, "ghost_fill_kernel");
}

int launch_cfl(hard_ctx* c, const double* U, int slot) {
  const long long N = (long long)c->g.n[0] * c->g.n[1] * c->g.n[2];
  cfl_kernel<<<small_grid(c, N), 256, 0, c->stream>>>(U, c->g, c->sc, slot);
  return after_launch(c, "cfl_kernel");
}

int prof_begin(hard_ctx* c) {
  if (!c->profiling) return HARD_OK;
  if (c->ev_used + 2 > c->ev.size()) {
    for (int i = 0; i < 2; ++i) {
      cudaEvent_t e;
      CK(cudaEventCreate(&e));
      c->ev.push_back(e);
    }
  }
  CK(cudaEventRecord(c->ev[c->ev_used], c->stream));
  return HARD_OK;
}
int prof_end(hard_ctx* c) {
  if (!c->profiling) return HARD_OK;
  CK(cudaEventRecord(c->ev[c->ev_used + 1], c->stream));
  c->ev_used += 2;
  return HARD_OK;
}

int launch_stage(hard_ctx* c, const CUtensorMap& tm, const double* Usrc, const double* Uaux, double* Uout, int mode,
                 int dirmask, int first, double cfl, double dt_fixed) {
  const GridDesc& g = c->g;
  StageArgs a;
  a.mode = mode; a.dirmask = dirmask; a.first = first; a.cur = (int)(c->steps_enq & 1);
  a.cfl = cfl; a.dt_fixed = dt_fixed;
  a.skip_cfl = c->src_on ? 1 : 0;
  const bool zact = g.act[2] && (dirmask & 4);
  a.Lz = zact ? c->Lz : (g.n[2] + ((g.n[2] + 63) / 64) - 1) / ((g.n[2] + 63) / 64);   // z inactive: chunks of <= 64 planes
  dim3 grid((g.n[0] + 13) / 14, (g.n[1] + 15) / 16, (g.n[2] + a.Lz - 1) / a.Lz);
  int rc = prof_begin(c);
  if (rc) return rc;
  // 3-D meshes with all fluxes in one launch take the specialised kernel (hard_stage3d.cuh)
  static const bool generic_only = getenv("HARD_GENERIC_STAGE") != nullptr;
  const bool spec3d = !generic_only && g.act[0] && g.act[1] && g.act[2] && dirmask == 7 && (mode == MODE_STAGE1 || mode == MODE_STAGE2);
#define HARD_LAUNCH(S, NF) \
  do { \
    if (spec3d && mode == MODE_STAGE1) stage3d_kernel<S, NF, MODE_STAGE1><<<grid, 256, StageCfg<S, NF>::SMEM3D, c->stream>>>(tm, Usrc, Uaux, Uout, g, c->sc, a); \
    else if (spec3d) stage3d_kernel<S, NF, MODE_STAGE2><<<grid, 256, StageCfg<S, NF>::SMEM3D, c->stream>>>(tm, Usrc, Uaux, Uout, g, c->sc, a); \
    else stage_kernel<S, NF><<<grid, 256, StageCfg<S, NF>::SMEM, c->stream>>>(tm, Usrc, Uaux, Uout, g, c->sc, a); \
  } while (0)
  if (c->scheme == HARD_SCHEME_WENO5Z_HLL) { if (c->nf == 6) HARD_LAUNCH(SCHEME_A, 6); else HARD_LAUNCH(SCHEME_A, 5); }
  else                                     { if (c->nf == 6) HARD_LAUNCH(SCHEME_B, 6); else HARD_LAUNCH(SCHEME_B, 5); }
#undef HARD_LAUNCH
  if ((rc = after_launch(c, "stage_kernel"))) return rc;
  return prof_end(c);
}

int launch_source(hard_ctx* c, double cfl, double dt_fixed) {
  const long long N = (long long)c->g.n[0] * c->g.n[1] * c->g.n[2];
  source_kernel<<<small_grid(c, N), 256, 0, c->stream>>>(c->U, c->g, c->sc, c->src, (int)(c->steps_enq & 1), cfl, dt_fixed);
  return after_launch(c, "source_kernel");
}

int launch_axpy(hard_ctx* c, int stage2, double cfl, double dt_fixed) {
  const long long N = (long long)c->g.n[0] * c->g.n[1] * c->g.n[2];
  int rc = prof_begin(c);
  if (rc) return rc;
  axpy_kernel<<<small_grid(c, N), 256, 0, c->stream>>>(c->U, c->U1, c->Rres, stage2 ? c->U : c->U1, c->g, c->sc, stage2,
                                                        (int)(c->steps_enq & 1), cfl, dt_fixed);
  if ((rc = after_launch(c, "axpy_kernel"))) return rc;
  return prof_end(c);
}

// L(Usrc) into the residual array, one launch per active direction (variant a8)
int perdir_residual(hard_ctx* c, const CUtensorMap& tm, const double* Usrc, double cfl, double dt_fixed) {
  if (!c->Rres) {                                          // workspace sized for the fused variant: own residual
    void* r = nullptr;
    cudaError_t e = cudaMalloc(&r, state_bytes(c));
    if (e != cudaSuccess) return fail(c, HARD_ERR_NOMEM, std::string("cudaMalloc (per-direction residual): ") + cudaGetErrorString(e));
    c->Rres = (double*)r;
    c->rres_owned = true;
    CK(cudaMemsetAsync(r, 0, state_bytes(c), c->stream));   // ghost layers of the residual are never written: defined from the start
  }
  int first = 1;
  for (int d = 0; d < 3; ++d) {
    if (!c->g.act[d]) continue;
    int rc = launch_stage(c, tm, Usrc, c->Rres, c->Rres, MODE_RESID, 1 << d, first, cfl, dt_fixed);
    if (rc) return rc;
    first = 0;
  }
  return HARD_OK;
}

int enqueue_one_step(hard_ctx* c, double cfl, double dt_fixed) {
  int rc;
  if ((rc = launch_ghost(c, c->U, 1, cfl, dt_fixed))) return rc;
  if (c->variant == HARD_VARIANT_FUSED) {
    if ((rc = launch_stage(c, c->tmU, c->U, nullptr, c->U1, MODE_STAGE1, 7, 0, cfl, dt_fixed))) return rc;
    if ((rc = launch_ghost(c, c->U1, 0, cfl, dt_fixed))) return rc;
    if ((rc = launch_stage(c, c->tmU1, c->U1, c->U, c->U, MODE_STAGE2, 7, 0, cfl, dt_fixed))) return rc;
    if (c->src_on && (rc = launch_source(c, cfl, dt_fixed))) return rc;
  } else {
    if ((rc = perdir_residual(c, c->tmU, c->U, cfl, dt_fixed))) return rc;
    if ((rc = launch_axpy(c, 0, cfl, dt_fixed))) return rc;
    if ((rc = launch_ghost(c, c->U1, 0, cfl, dt_fixed))) return rc;
    if ((rc = perdir_residual(c, c->tmU1, c->U1, cfl, dt_fixed))) return rc;
    if ((rc = launch_axpy(c, 1, cfl, dt_fixed))) return rc;
    if (c->src_on) { if ((rc = launch_source(c, cfl, dt_fixed))) return rc; }
    else if ((rc = launch_cfl(c, c->U, (int)((c->steps_enq & 1) ^ 1)))) return rc;
  }
  c->steps_enq++;
  return HARD_OK;
}

// Launch-bound meshes (the 1-D configs: ~10^3 cells, ~10^4 steps): replay a captured graph of two steps.  dt and
// lambda live on the device, so the graph needs no host value; the pair covers both lambda ping-pong slots.
// Only on capturable streams (not the legacy default stream), never while stage timing is on.
bool ensure_graph(hard_ctx* c, double cfl, double dt_fixed) {
  static const bool disabled = getenv("HARD_NO_GRAPH") != nullptr;
  if (disabled || !c->graphs_ok || c->profiling || c->debug_sync || (c->steps_enq & 1)) return false;
  const int sig = c->variant * 4 + (c->src_on ? 2 : 0) + 1;
  if (c->gexec && c->g_cfl == cfl && c->g_dt == dt_fixed && c->g_sig == sig && c->g_stream == c->stream && c->g_gen == c->gen) return true;
  if (c->gexec) { cudaGraphExecDestroy(c->gexec); c->gexec = nullptr; }
  if (cudaStreamBeginCapture(c->stream, cudaStreamCaptureModeThreadLocal) != cudaSuccess) {
    cudaGetLastError();
    c->graphs_ok = false;
    return false;
  }
  const long long enq0 = c->steps_enq, l0 = c->launches;
  int rc = enqueue_one_step(c, cfl, dt_fixed);
  if (!rc) rc = enqueue_one_step(c, cfl, dt_fixed);
  c->steps_enq = enq0;                                   // nothing ran: capture only
  c->launches = l0;
  cudaGraph_t graph = nullptr;
  cudaError_t e = cudaStreamEndCapture(c->stream, &graph);
  if (rc || e != cudaSuccess || !graph) { cudaGetLastError(); c->graphs_ok = false; if (graph) cudaGraphDestroy(graph); return false; }
  e = cudaGraphInstantiate(&c->gexec, graph, 0);
  cudaGraphDestroy(graph);
  if (e != cudaSuccess) { cudaGetLastError(); c->gexec = nullptr; c->graphs_ok = false; return false; }
  c->g_cfl = cfl; c->g_dt = dt_fixed; c->g_sig = sig; c->g_stream = c->stream; c->g_gen = c->gen;
  return true;
}

int do_steps(hard_ctx* c, double cfl, double dt_fixed, int nsteps) {
  if (!c->have_state) return fail(c, HARD_ERR_NOSTATE, "no state: call hard_set_state first");
  int rc = ensure_ready(c);
  if (rc) return rc;
  int left = nsteps;
  const long long cells = (long long)c->g.n[0] * c->g.n[1] * c->g.n[2];
  const bool want_graph = left >= 8 && c->variant == HARD_VARIANT_FUSED && c->graphs_ok && !c->profiling && !c->debug_sync;
  // The legacy default stream cannot be captured: launch-bound meshes borrow an internal non-blocking stream,
  // ordered after the bound stream's earlier work and before its later work by two events.
  cudaStream_t user = c->stream;
  bool borrowed = false;
  if (want_graph && user == 0 && cells <= (1LL << 21)) {
    if (!c->own_stream) {
      if (cudaStreamCreateWithFlags(&c->own_stream, cudaStreamNonBlocking) != cudaSuccess ||
          cudaEventCreateWithFlags(&c->ev_in, cudaEventDisableTiming) != cudaSuccess ||
          cudaEventCreateWithFlags(&c->ev_out, cudaEventDisableTiming) != cudaSuccess) {
        cudaGetLastError();
        c->own_stream = nullptr;
      }
    }
    if (c->own_stream) {
      CK(cudaEventRecord(c->ev_in, user));
      CK(cudaStreamWaitEvent(c->own_stream, c->ev_in, 0));
      c->stream = c->own_stream;
      borrowed = true;
    }
  }
  auto give_back = [&](int code) {
    if (borrowed) {
      c->stream = user;
      if (cudaEventRecord(c->ev_out, c->own_stream) != cudaSuccess || cudaStreamWaitEvent(user, c->ev_out, 0) != cudaSuccess)
        return code ? code : cuda_fail(c, cudaGetLastError(), "internal stream hand-back");
    }
    return code;
  };
  if (want_graph && c->stream != 0) {
    if (c->steps_enq & 1) {                              // the captured pair starts on an even step
      if ((rc = enqueue_one_step(c, cfl, dt_fixed))) return give_back(rc);
      --left;
    }
    if (ensure_graph(c, cfl, dt_fixed)) {
      const long long per_pair = 8 + (c->src_on ? 2 : 0);
      while (left >= 2) {
        cudaError_t e = cudaGraphLaunch(c->gexec, c->stream);
        if (e != cudaSuccess) return give_back(cuda_fail(c, e, "cudaGraphLaunch"));
        c->steps_enq += 2;
        c->launches += per_pair;
        left -= 2;
      }
    }
  }
  for (; left > 0; --left)
    if ((rc = enqueue_one_step(c, cfl, dt_fixed))) return give_back(rc);
  return give_back(HARD_OK);
}

int sync_status(hard_ctx* c, DevScalars* host) {
  CK(cudaMemcpyAsync(host, c->sc, sizeof(DevScalars), cudaMemcpyDeviceToHost, c->stream));
  CK(cudaStreamSynchronize(c->stream));
  if (host->status & 1) return fail(c, HARD_ERR_NONPHYSICAL, "non-physical state (non-finite, rho <= 0 or p <= 0)");
  return HARD_OK;
}

int copy_field(hard_ctx* c, double* dev_field, const double* user, bool to_device) {
  const GridDesc& g = c->g;
  cudaMemcpy3DParms p;
  memset(&p, 0, sizeof p);
  cudaPitchedPtr up = make_cudaPitchedPtr((void*)user, (size_t)g.n[0] * 8, (size_t)g.n[0], (size_t)g.n[1]);
  cudaPitchedPtr dp = make_cudaPitchedPtr((void*)dev_field, (size_t)g.pitch * 8, (size_t)g.pitch, (size_t)g.P[1]);
  cudaPos dpos = make_cudaPos((size_t)g.off[0] * 8, (size_t)g.off[1], (size_t)g.off[2]);
  if (to_device) { p.srcPtr = up; p.dstPtr = dp; p.dstPos = dpos; }
  else           { p.srcPtr = dp; p.srcPos = dpos; p.dstPtr = up; }
  p.extent = make_cudaExtent((size_t)g.n[0] * 8, (size_t)g.n[1], (size_t)g.n[2]);
  p.kind = cudaMemcpyDefault;
  CK(cudaMemcpy3DAsync(&p, c->stream));
  return HARD_OK;
}

}  // namespace

// ================================================================================ C ABI (include/hard.h)
extern "C" {

hard_ctx* hard_create(int nx, int ny, int nz, double gamma, int bc) {
  g_create_error.clear();
  if (nx < 1 || ny < 1 || nz < 1 || !(gamma > 1.0) || (bc != HARD_BC_PERIODIC && bc != HARD_BC_OUTFLOW && bc != HARD_BC_REFLECT)) {
    g_create_error = "hard_create: bad argument";
    return nullptr;
  }
  const int n[3] = { nx, ny, nz };
  int nact = 0;
  for (int a = 0; a < 3; ++a) {
    if (n[a] > 1 && n[a] < 3) { g_create_error = "hard_create: an active direction needs n >= 3"; return nullptr; }
    nact += n[a] > 1;
  }
  if (!nact) { g_create_error = "hard_create: at least one direction must have n > 1"; return nullptr; }
  int dev = 0;
  cudaDeviceProp prop;
  cudaError_t e = cudaGetDevice(&dev);
  if (e == cudaSuccess) e = cudaGetDeviceProperties(&prop, dev);
  if (e != cudaSuccess) {
    g_create_error = std::string("hard_create: no usable CUDA device (") + cudaGetErrorString(e) + "); there is no CPU fallback";
    return nullptr;
  }
  // The library holds one cubin (sm_100a, no PTX): ask the runtime whether THIS device can run it instead of
  // guessing from the compute capability (an sm_103 / sm_12x part would pass "major >= 10" and fail at the first launch).
  cudaFuncAttributes fa;
  if (prop.major != 10 || prop.minor != 0 || cudaFuncGetAttributes(&fa, cfl_kernel) != cudaSuccess) {
    cudaGetLastError();
    char buf[160];
    snprintf(buf, sizeof buf, "hard_create: kernels are built for sm_100a only (device %d is sm_%d%d); there is no CPU fallback",
             dev, prop.major, prop.minor);
    g_create_error = buf;
    return nullptr;
  }
  hard_ctx* c = new hard_ctx();
  memset(&c->g, 0, sizeof c->g);
  for (int a = 0; a < 3; ++a) { c->g.n[a] = n[a]; c->g.inv_d[a] = (double)n[a]; }
  c->g.gamma = gamma;
  c->g.bc = bc;
  c->sm_count = prop.multiProcessorCount;
  c->device = dev;
  { const char* d = getenv("HARD_DEBUG_SYNC"); c->debug_sync = d && d[0] == '1'; }
  compute_layout(c);
  return c;
}

int hard_destroy(hard_ctx* c) {
  DeviceGuard dg__(c);
  if (!c) return HARD_ERR_ARG;
  cudaStreamSynchronize(c->stream);
  for (cudaEvent_t e : c->ev) cudaEventDestroy(e);
  if (c->gexec) cudaGraphExecDestroy(c->gexec);
  if (c->own_stream) { cudaStreamSynchronize(c->own_stream); cudaStreamDestroy(c->own_stream); }
  if (c->ev_in) cudaEventDestroy(c->ev_in);
  if (c->ev_out) cudaEventDestroy(c->ev_out);
  if (c->rres_owned && c->Rres) cudaFree(c->Rres);
  if (c->ws_owned && c->ws) cudaFree(c->ws);
  delete c;
  return HARD_OK;
}

const char* hard_last_error(const hard_ctx* c) { return c ? c->err.c_str() : g_create_error.c_str(); }

long long hard_launch_count(const hard_ctx* c) { return c ? c->launches : -1; }

int hard_set_spacing(hard_ctx* c, double dx, double dy, double dz) {
  DeviceGuard dg__(c);
  if (!c || !(dx > 0.0 && dy > 0.0 && dz > 0.0)) return fail(c, HARD_ERR_ARG, "hard_set_spacing: spacings must be > 0");
  c->g.inv_d[0] = 1.0 / dx; c->g.inv_d[1] = 1.0 / dy; c->g.inv_d[2] = 1.0 / dz;
  c->gen++;                                              // a captured graph holds the old spacing by value
  if (c->have_state) {
    const int slot = (int)(c->steps_enq & 1);
    CK(cudaMemsetAsync(&c->sc->lam_bits[slot], 0, sizeof(unsigned long long), c->stream));
    return launch_cfl(c, c->U, slot);
  }
  return HARD_OK;
}

int hard_set_scheme(hard_ctx* c, int scheme) {
  if (!c || (scheme != HARD_SCHEME_WENO5Z_HLL && scheme != HARD_SCHEME_MUSCL_HLLC))
    return fail(c, HARD_ERR_ARG, "hard_set_scheme: unknown scheme");
  if (c->have_state || c->ws) return fail(c, HARD_ERR_ARG, "hard_set_scheme: only before hard_set_state / hard_bind_workspace");
  c->scheme = scheme;
  compute_layout(c);
  return HARD_OK;
}

int hard_enable_radiation(hard_ctx* c) {
  if (!c) return HARD_ERR_ARG;
  if (c->have_state || c->ws) return fail(c, HARD_ERR_ARG, "hard_enable_radiation: only before hard_set_state / hard_bind_workspace");
  c->nf = 6;
  compute_layout(c);
  return HARD_OK;
}

int hard_set_rad_energy(hard_ctx* c, const double* er) {
  DeviceGuard dg__(c);
  if (!c || !er) return fail(c, HARD_ERR_ARG, "hard_set_rad_energy: null pointer");
  if (c->nf != 6) return fail(c, HARD_ERR_ARG, "hard_set_rad_energy: call hard_enable_radiation first");
  if (!c->have_state) return fail(c, HARD_ERR_NOSTATE, "no state: call hard_set_state first");
  return copy_field(c, c->U + 5 * c->g.fstride, er, true);
}

int hard_get_rad_energy(hard_ctx* c, double* er) {
  DeviceGuard dg__(c);
  if (!c || !er) return fail(c, HARD_ERR_ARG, "hard_get_rad_energy: null pointer");
  if (c->nf != 6) return fail(c, HARD_ERR_ARG, "hard_get_rad_energy: call hard_enable_radiation first");
  if (!c->have_state) return fail(c, HARD_ERR_NOSTATE, "no state");
  int rc = copy_field(c, c->U + 5 * c->g.fstride, er, false);
  if (rc) return rc;
  DevScalars h;
  return sync_status(c, &h);
}

int hard_set_source(hard_ctx* c, double kappa, double c_light, double a_rad, double cv) {
  if (!c) return HARD_ERR_ARG;
  if (c->nf != 6) return fail(c, HARD_ERR_ARG, "hard_set_source: call hard_enable_radiation first");
  if (!(kappa >= 0.0 && c_light > 0.0 && a_rad > 0.0 && cv > 0.0)) return fail(c, HARD_ERR_ARG, "hard_set_source: bad parameter");
  c->src_on = true;
  c->gen++;
  c->src.kappa = kappa; c->src.c_light = c_light; c->src.a_rad = a_rad; c->src.cv = cv;
  return HARD_OK;
}

int hard_set_slab(hard_ctx* c, int lower_neighbor, int upper_neighbor) {
  if (!c) return HARD_ERR_ARG;
  if (!c->g.act[2]) return fail(c, HARD_ERR_ARG, "hard_set_slab: the z direction is inactive");
  c->zskip = (lower_neighbor ? 1 : 0) | (upper_neighbor ? 2 : 0);
  c->g.zskip = c->zskip;
  c->gen++;
  return HARD_OK;
}

size_t hard_halo_doubles(const hard_ctx* c) {
  return c ? (size_t)c->g.g * c->g.n[0] * c->g.n[1] * c->nf : 0;
}

static int halo_copy(hard_ctx* c, int buffer, int side, double* buf, int unpack) {
  DeviceGuard dg__(c);
  if (!c || !buf || (buffer != 0 && buffer != 1) || (side != 0 && side != 1)) return fail(c, HARD_ERR_ARG, "hard_halo_*: bad argument");
  if (!c->have_state) return fail(c, HARD_ERR_NOSTATE, "no state");
  if (!c->g.act[2] || c->g.n[2] < c->g.g) return fail(c, HARD_ERR_ARG, "hard_halo_*: a slab needs at least g z-planes");
  const long long total = (long long)hard_halo_doubles(c);
  halo_copy_kernel<<<small_grid(c, total), 256, 0, c->stream>>>(buffer ? c->U1 : c->U, buf, c->g, side, unpack);
  return after_launch(c, "halo_copy_kernel");
}
int hard_halo_pack(hard_ctx* c, int buffer, int side, double* dev_buf) { return halo_copy(c, buffer, side, dev_buf, 0); }
int hard_halo_unpack(hard_ctx* c, int buffer, int side, const double* dev_buf) {
  return halo_copy(c, buffer, side, const_cast<double*>(dev_buf), 1);
}

int hard_substep(hard_ctx* c, double cfl, double dt, int phase) {
  DeviceGuard dg__(c);
  if (!c || !((dt > 0.0) || (cfl > 0.0))) return fail(c, HARD_ERR_ARG, "hard_substep: cfl > 0 or dt > 0 required");
  if (!c->have_state) return fail(c, HARD_ERR_NOSTATE, "no state: call hard_set_state first");
  if (c->variant != HARD_VARIANT_FUSED) return fail(c, HARD_ERR_ARG, "hard_substep: fused variant only");
  int rc = ensure_ready(c);
  if (rc) return rc;
  const double dtf = dt > 0.0 ? dt : 0.0, cf = dt > 0.0 ? 1.0 : cfl;
  switch (phase) {
    case HARD_PHASE_GHOST_U:  return launch_ghost(c, c->U, 1, cf, dtf);
    case HARD_PHASE_STAGE1:   return launch_stage(c, c->tmU, c->U, nullptr, c->U1, MODE_STAGE1, 7, 0, cf, dtf);
    case HARD_PHASE_GHOST_U1: return launch_ghost(c, c->U1, 0, cf, dtf);
    case HARD_PHASE_STAGE2:
      if ((rc = launch_stage(c, c->tmU1, c->U1, c->U, c->U, MODE_STAGE2, 7, 0, cf, dtf))) return rc;
      return c->src_on ? launch_source(c, cf, dtf) : HARD_OK;
    case HARD_PHASE_END:      c->steps_enq++; return HARD_OK;
    default: return fail(c, HARD_ERR_ARG, "hard_substep: unknown phase");
  }
}

int hard_lambda_ptr(hard_ctx* c, int next, double** dev_ptr) {
  DeviceGuard dg__(c);
  if (!c || !dev_ptr) return HARD_ERR_ARG;
  int rc = ensure_ready(c);
  if (rc) return rc;
  *dev_ptr = reinterpret_cast<double*>(&c->sc->lam_bits[(c->steps_enq & 1) ^ (next ? 1 : 0)]);
  return HARD_OK;
}

int hard_set_variant(hard_ctx* c, int variant) {
  if (!c || (variant != HARD_VARIANT_FUSED && variant != HARD_VARIANT_PERDIR))
    return fail(c, HARD_ERR_ARG, "hard_set_variant: unknown variant");
  c->variant = variant;
  return HARD_OK;
}

int hard_set_stream(hard_ctx* c, void* s) {
  DeviceGuard dg__(c);
  if (!c) return HARD_ERR_ARG;
  CK(cudaStreamSynchronize(c->stream));
  c->stream = (cudaStream_t)s;
  return HARD_OK;
}

size_t hard_workspace_bytes(const hard_ctx* c) {
  if (!c) return 0;
  return 256 + (c->variant == HARD_VARIANT_PERDIR ? 3 : 2) * align_up(state_bytes(c), 256);
}

int hard_bind_workspace(hard_ctx* c, void* dev, size_t bytes) {
  DeviceGuard dg__(c);
  if (!c || !dev) return fail(c, HARD_ERR_ARG, "hard_bind_workspace: null");
  if (c->ws) return fail(c, HARD_ERR_ARG, "hard_bind_workspace: a workspace is already bound");
  if (bytes < hard_workspace_bytes(c) || ((uintptr_t)dev & 255)) return fail(c, HARD_ERR_ARG, "hard_bind_workspace: too small or not 256-B aligned");
  cudaPointerAttributes at;
  CK(cudaPointerGetAttributes(&at, dev));
  if (at.type != cudaMemoryTypeDevice) return fail(c, HARD_ERR_ARG, "hard_bind_workspace: not device memory");
  c->ws = dev;
  c->ws_bytes = bytes;
  c->ws_owned = false;
  // zero everything carve() may hand out: also the residual of the per-direction variant when the lent buffer is
  // large enough for it although the fused variant is selected now
  const size_t with_resid = 256 + 3 * align_up(state_bytes(c), 256);
  CK(cudaMemsetAsync(c->ws, 0, bytes >= with_resid ? with_resid : hard_workspace_bytes(c), c->stream));
  carve(c);
  return HARD_OK;
}

int hard_set_state(hard_ctx* c, const double* rho, const double* mx, const double* my, const double* mz, const double* E) {
  DeviceGuard dg__(c);
  if (!c || !rho || !mx || !my || !mz || !E) return fail(c, HARD_ERR_ARG, "hard_set_state: null pointer");
  int rc = ensure_ready(c);
  if (rc) return rc;
  const double* src[5] = { rho, mx, my, mz, E };
  for (int f = 0; f < 5; ++f)
    if ((rc = copy_field(c, c->U + f * c->g.fstride, src[f], true))) return rc;
  if (c->nf == 6) CK(cudaMemsetAsync(c->U + 5 * c->g.fstride, 0, (size_t)c->g.fstride * sizeof(double), c->stream));
  CK(cudaMemsetAsync(c->sc, 0, sizeof(DevScalars), c->stream));
  c->steps_enq = 0;                                      // even: a captured two-step graph stays valid (it bakes in no state value)
  c->have_state = true;
  c->err.clear();
  if ((rc = launch_cfl(c, c->U, 0))) return rc;
  DevScalars h;
  return sync_status(c, &h);
}

int hard_get_state(hard_ctx* c, double* rho, double* mx, double* my, double* mz, double* E) {
  DeviceGuard dg__(c);
  if (!c || !rho || !mx || !my || !mz || !E) return fail(c, HARD_ERR_ARG, "hard_get_state: null pointer");
  if (!c->have_state) return fail(c, HARD_ERR_NOSTATE, "no state");
  double* dst[5] = { rho, mx, my, mz, E };
  int rc;
  for (int f = 0; f < 5; ++f)
    if ((rc = copy_field(c, c->U + f * c->g.fstride, dst[f], false))) return rc;
  DevScalars h;
  return sync_status(c, &h);
}

int hard_step(hard_ctx* c, double cfl, int nsteps) {
  DeviceGuard dg__(c);
  if (!c || !(cfl > 0.0) || nsteps < 0) return fail(c, HARD_ERR_ARG, "hard_step: cfl > 0 and nsteps >= 0 required");
  return do_steps(c, cfl, 0.0, nsteps);
}

int hard_step_dt(hard_ctx* c, double dt, int nsteps) {
  DeviceGuard dg__(c);
  if (!c || !(dt > 0.0) || nsteps < 0) return fail(c, HARD_ERR_ARG, "hard_step_dt: dt > 0 and nsteps >= 0 required");
  return do_steps(c, 1.0, dt, nsteps);
}

int hard_max_dt(hard_ctx* c, double* dt_out) {
  DeviceGuard dg__(c);
  if (!c || !dt_out) return fail(c, HARD_ERR_ARG, "hard_max_dt: null");
  if (!c->have_state) return fail(c, HARD_ERR_NOSTATE, "no state");
  DevScalars h;
  int rc = sync_status(c, &h);
  double lam;
  memcpy(&lam, &h.lam_bits[c->steps_enq & 1], sizeof lam);
  *dt_out = 1.0 / lam;
  return rc;
}

int hard_get_time(hard_ctx* c, double* t, long long* steps_done) {
  DeviceGuard dg__(c);
  if (!c) return HARD_ERR_ARG;
  if (!c->have_state) return fail(c, HARD_ERR_NOSTATE, "no state");
  DevScalars h;
  int rc = sync_status(c, &h);
  if (t) *t = h.t;
  if (steps_done) *steps_done = h.steps;
  return rc;
}

int hard_stage_time(hard_ctx* c, int reset, double* ms, long long* launches) {
  DeviceGuard dg__(c);
  if (!c) return HARD_ERR_ARG;
  CK(cudaStreamSynchronize(c->stream));
  double tot = 0.0;
  for (size_t i = 0; i + 1 < c->ev_used; i += 2) {
    float f = 0.f;
    CK(cudaEventElapsedTime(&f, c->ev[i], c->ev[i + 1]));
    tot += f;
  }
  if (ms) *ms = tot;
  if (launches) *launches = (long long)(c->ev_used / 2);
  if (reset) { c->ev_used = 0; c->profiling = (reset == 1); }
  return HARD_OK;
}

}  // extern "C"
