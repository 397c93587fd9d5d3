// hard_noalloc.cu — hard_max_dt_noalloc: the CFL max-wavespeed reduction (P:215, P:255,
// reading G6) for callers that are not allowed to allocate device memory.
//
// Who that is.  Every other entry point of this library needs a workspace: hard_set_state cudaMalloc's one, or the
// caller lends one through hard_bind_workspace (which it had to allocate itself).  Some callers can do neither at
// the moment they need dt: a plugin that runs inside another framework's step and may only read that framework's
// tensors, a process whose memory pool is fixed at start-up and whose policy forbids cudaMalloc afterwards (it
// would fragment or serialise the device), or a diagnostic hook fired while the host application holds all free
// HBM.  For them the reduction's scratch lives in a file-scope __device__ array that is part of the library image:
// it exists on every GPU that loads the library, from load until the process exits, and costs SCRATCH_BYTES each.
//
// What the scratch holds: one partial maximum per CTA, a ticket counter and a "non-physical cell seen" flag.  The
// counter and the flag must be zero when a launch starts.  The last CTA of a launch puts them back to zero, and the
// entry point clears them again (cudaMemsetAsync on the same stream) before every launch, so that a launch that was
// aborted cannot poison the next one.  The partial maxima need no clearing: each launch writes the entries it reads.
//
// All calls on a device share the one array.  Two calls whose kernels may overlap on the GPU (different streams
// without an ordering between them, or different host threads) race on it and return garbage; order them.
//
// The arithmetic is the standalone CFL pass of hard_kernels.cuh typed again (that header defines non-inline kernels
// and cannot be included by a second translation unit): correctly rounded operations in the order of the
// definition, so the result is bit-equal to hard_set_state + hard_max_dt on the same fields.
#include <cuda_runtime.h>

#include <cstdio>
#include <mutex>
#include <string>

#include "../../include/hard.h"

namespace {

constexpr int THREADS = 256;
constexpr int CELLS_PER_THREAD = 32;
constexpr long long CELLS_PER_CTA = (long long)THREADS * CELLS_PER_THREAD;             // 8192
constexpr int MAX_CTAS = (int)(HARD_NOALLOC_MAX_CELLS / CELLS_PER_CTA);                // 4096
constexpr int HEAD_WORDS = 32;                    // word 0: ticket counter, word 1: bad flag; the rest pads to 256 B
constexpr size_t SCRATCH_BYTES = (size_t)(HEAD_WORDS + MAX_CTAS) * 8;                  // 33 024 B per GPU
static_assert(HARD_NOALLOC_MAX_CELLS % CELLS_PER_CTA == 0, "the cell limit is a whole number of CTAs");

// The scratch itself.  In HOST code this name is only a handle for cudaGetSymbolAddress — it is not a device
// address and must never be handed to a kernel; device code below names it directly.
static __device__ __align__(256) unsigned long long g_noalloc_scratch[HEAD_WORDS + MAX_CTAS];
static_assert(sizeof(g_noalloc_scratch) == SCRATCH_BYTES && SCRATCH_BYTES == 33024, "the size include/hard.h states");

__device__ __forceinline__ double sum3_by_magnitude(double a, double b, double c) {   // reading G8
  double x1 = a, x2 = b, x3 = c, t;
  if (fabs(x1) > fabs(x2)) { t = x1; x1 = x2; x2 = t; }
  if (fabs(x2) > fabs(x3)) { t = x2; x2 = x3; x3 = t; }
  if (fabs(x1) > fabs(x2)) { t = x1; x1 = x2; x2 = t; }
  if (x2 == -x3) return x1;
  return __dadd_rn(__dadd_rn(x1, x2), x3);
}

struct NoallocArgs {
  const double *rho, *mx, *my, *mz, *E;   // device, n cells each, unpadded
  double* dt_out;                         // device, one double
  long long n;
  double gamma, inv_d[3];
  int act[3];
};

// CTA b reduces cells [b * CELLS_PER_CTA, (b+1) * CELLS_PER_CTA) to one partial maximum in the scratch; the CTA
// that draws the last ticket reduces the partials and writes 1 / lambda (NaN if any cell was non-physical).
__global__ void __launch_bounds__(THREADS) cfl_noalloc_kernel(NoallocArgs a, unsigned long long* scratch) {
  __shared__ double red[THREADS / 32];
  __shared__ int red_bad[THREADS / 32];
  __shared__ bool last;
  unsigned long long* counter = scratch;
  unsigned long long* badflag = scratch + 1;
  unsigned long long* partial = scratch + HEAD_WORDS;

  const double gm1 = __dadd_rn(a.gamma, -1.0);
  const long long base = blockIdx.x * CELLS_PER_CTA;
  double lam = 0.0;
  int bad = 0;
  for (int r = 0; r < CELLS_PER_THREAD; ++r) {
    const long long i = base + (long long)r * THREADS + threadIdx.x;
    if (i >= a.n) break;
    const double rho = a.rho[i], mx = a.mx[i], my = a.my[i], mz = a.mz[i], E = a.E[i];
    const double v[3] = { __ddiv_rn(mx, rho), __ddiv_rn(my, rho), __ddiv_rn(mz, rho) };
    const double ke2 = sum3_by_magnitude(__dmul_rn(mx, v[0]), __dmul_rn(my, v[1]), __dmul_rn(mz, v[2]));
    const double p = __dmul_rn(gm1, __dadd_rn(E, -__dmul_rn(0.5, ke2)));
    if (!(rho > 0.0 && p > 0.0) || !(p < 1.0e300) || !(rho < 1.0e300)) { bad = 1; continue; }
    const double c = __dsqrt_rn(__ddiv_rn(__dmul_rn(a.gamma, p), rho));
#pragma unroll
    for (int d = 0; d < 3; ++d)
      if (a.act[d]) lam = fmax(lam, __dmul_rn(__dadd_rn(fabs(v[d]), c), a.inv_d[d]));
  }
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) {
    lam = fmax(lam, __shfl_xor_sync(0xffffffffu, lam, o));
    bad |= __shfl_xor_sync(0xffffffffu, bad, o);
  }
  const int w = threadIdx.x >> 5;
  if ((threadIdx.x & 31) == 0) { red[w] = lam; red_bad[w] = bad; }
  __syncthreads();
  if (threadIdx.x == 0) {
    for (int i = 1; i < THREADS / 32; ++i) { lam = fmax(lam, red[i]); bad |= red_bad[i]; }
    partial[blockIdx.x] = (unsigned long long)__double_as_longlong(lam);      // lambda >= 0: plain store of the bits
    if (bad) atomicOr(badflag, 1ull);
    __threadfence();                                   // partial and flag visible before the ticket is drawn
    last = atomicAdd(counter, 1ull) == (unsigned long long)gridDim.x - 1;
  }
  __syncthreads();
  if (!last) return;
  __threadfence();
  lam = 0.0;
  for (int b = threadIdx.x; b < (int)gridDim.x; b += THREADS)
    lam = fmax(lam, __longlong_as_double((long long)((volatile unsigned long long*)partial)[b]));
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) lam = fmax(lam, __shfl_xor_sync(0xffffffffu, lam, o));
  __syncthreads();                                     // red[] is reused
  if ((threadIdx.x & 31) == 0) red[w] = lam;
  __syncthreads();
  if (threadIdx.x == 0) {
    for (int i = 1; i < THREADS / 32; ++i) lam = fmax(lam, red[i]);
    const bool any_bad = *(volatile unsigned long long*)badflag != 0ull;
    *a.dt_out = any_bad ? __longlong_as_double(0x7ff8000000000000ll) : __ddiv_rn(1.0, lam);
    *counter = 0ull;                                   // leave the scratch as the next launch needs it
    *badflag = 0ull;
  }
}

// Per-device set-up: the device address of the scratch, asked for once per device with that device current.
constexpr int MAX_DEVICES = 64;
std::mutex g_mu;
unsigned long long* g_scratch_dev[MAX_DEVICES] = {};
thread_local std::string g_noalloc_error;

int noalloc_fail(int code, const std::string& msg) {
  g_noalloc_error = msg;
  return code;
}

}  // namespace

extern "C" {

const char* hard_noalloc_last_error(void) { return g_noalloc_error.c_str(); }

int hard_max_dt_noalloc(int nx, int ny, int nz, double gamma, double dx, double dy, double dz, const double* rho,
                        const double* mx, const double* my, const double* mz, const double* E, double* dt_out,
                        void* cuda_stream) {
  g_noalloc_error.clear();
  if (nx < 1 || ny < 1 || nz < 1 || !(gamma > 1.0) || !(dx > 0.0 && dy > 0.0 && dz > 0.0))
    return noalloc_fail(HARD_ERR_ARG, "hard_max_dt_noalloc: n >= 1, gamma > 1 and spacings > 0 required");
  if (nx == 1 && ny == 1 && nz == 1)
    return noalloc_fail(HARD_ERR_ARG, "hard_max_dt_noalloc: at least one direction must have n > 1");
  if (!rho || !mx || !my || !mz || !E || !dt_out) return noalloc_fail(HARD_ERR_ARG, "hard_max_dt_noalloc: null pointer");
  const long long n = (long long)nx * ny * nz;
  if (n > HARD_NOALLOC_MAX_CELLS) {
    char buf[256];
    snprintf(buf, sizeof buf,
             "hard_max_dt_noalloc: %d x %d x %d = %lld cells exceed HARD_NOALLOC_MAX_CELLS = %lld (the static scratch "
             "holds one partial maximum per %lld cells); use hard_create + hard_set_state + hard_max_dt for larger meshes",
             nx, ny, nz, n, (long long)HARD_NOALLOC_MAX_CELLS, CELLS_PER_CTA);
    return noalloc_fail(HARD_ERR_ARG, buf);
  }
  int dev = -1;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess)
    return noalloc_fail(HARD_ERR_CUDA, std::string("hard_max_dt_noalloc: no usable CUDA device (") + cudaGetErrorString(e) +
                                           "); there is no CPU fallback");
  if (dev < 0 || dev >= MAX_DEVICES) return noalloc_fail(HARD_ERR_ARG, "hard_max_dt_noalloc: device ordinal out of range");
  const void* ptrs[6] = { rho, mx, my, mz, E, dt_out };
  for (const void* p : ptrs) {
    cudaPointerAttributes at;
    e = cudaPointerGetAttributes(&at, p);
    if (e != cudaSuccess) return noalloc_fail(HARD_ERR_CUDA, std::string("cudaPointerGetAttributes: ") + cudaGetErrorString(e));
    if (at.type != cudaMemoryTypeDevice && at.type != cudaMemoryTypeManaged)
      return noalloc_fail(HARD_ERR_ARG, "hard_max_dt_noalloc: every pointer must address device memory");
  }
  unsigned long long* scratch = nullptr;
  {
    std::lock_guard<std::mutex> lk(g_mu);
    if (!g_scratch_dev[dev]) {                           // first call on this device (it is the current one)
      void* p = nullptr;
      e = cudaGetSymbolAddress(&p, g_noalloc_scratch);
      if (e != cudaSuccess || !p)
        return noalloc_fail(HARD_ERR_CUDA, std::string("cudaGetSymbolAddress(scratch): ") + cudaGetErrorString(e));
      g_scratch_dev[dev] = (unsigned long long*)p;
    }
    scratch = g_scratch_dev[dev];
  }
  cudaStream_t st = (cudaStream_t)cuda_stream;
  e = cudaMemsetAsync(scratch, 0, HEAD_WORDS * sizeof(unsigned long long), st);   // counter and flag start at zero
  if (e != cudaSuccess) return noalloc_fail(HARD_ERR_CUDA, std::string("cudaMemsetAsync(scratch): ") + cudaGetErrorString(e));
  NoallocArgs a;
  a.rho = rho; a.mx = mx; a.my = my; a.mz = mz; a.E = E; a.dt_out = dt_out;
  a.n = n;
  a.gamma = gamma;
  a.inv_d[0] = 1.0 / dx; a.inv_d[1] = 1.0 / dy; a.inv_d[2] = 1.0 / dz;
  a.act[0] = nx > 1; a.act[1] = ny > 1; a.act[2] = nz > 1;
  const int ctas = (int)((n + CELLS_PER_CTA - 1) / CELLS_PER_CTA);
  cfl_noalloc_kernel<<<ctas, THREADS, 0, st>>>(a, scratch);
  e = cudaGetLastError();
  if (e != cudaSuccess) return noalloc_fail(HARD_ERR_CUDA, std::string("cfl_noalloc_kernel: ") + cudaGetErrorString(e));
  return HARD_OK;
}

}  // extern "C"
