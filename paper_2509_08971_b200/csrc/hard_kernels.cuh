// hard_kernels.cuh — CUDA kernels of the hot path for sm_100a:
//   ghost_fill_kernel    a1  ghost-cell fill (periodic / outflow / reflecting), all faces, one launch
//   stage_kernel<S, NF>  a2..a6 (+a7 fused in stage 2): TMA-staged 14x16 x-y tile marched along z;
//                        NF = 6 carries the advected radiation energy density (NEXT-1, Rusanov flux)
//   cfl_kernel           a7  standalone max-wavespeed reduction (set_state, per-direction variant)
//   axpy_kernel          a6  RK combination of the per-direction variant (a8)
//   source_kernel        NEXT-3  pointwise heating / cooling source (backward Euler) + the step's CFL reduction
//   halo_copy_kernel     NEXT-4  pack / unpack z-slab halo planes for the exchange between ranks
// The stage kernel also serves the per-direction comparison variant (a8): dirmask selects one
// direction and MODE_RESID read-modify-writes a residual array instead of applying the RK update.
#pragma once
#include <cuda.h>
#include <cuda_runtime.h>
#include <stdint.h>

#include "hard_device.cuh"

namespace hard {

struct GridDesc {
  int n[3];                 // interior cells
  int off[3];               // padded coordinate of interior cell 0 (>= ghost width; 0 if inactive)
  int act[3];               // n > 1
  int P[3];                 // padded extents: P[0] = row pitch (doubles), P[1], P[2]
  long long pitch, plane, fstride;   // doubles: row, z-plane, field
  double inv_d[3];
  double gamma;
  int bc;                   // 0 periodic, 1 outflow, 2 reflecting
  int g;                    // ghost width of the scheme
  int nf;                   // fields per state: 5, or 6 with the advected radiation energy density (NEXT-1)
  int zskip;                // NEXT-4 z-slab sharding: bit 0 / 1 = low / high z ghosts come from a neighbour rank
};

// Device-resident scalars: nothing returns to the host inside hard_step.
struct DevScalars {
  unsigned long long lam_bits[2];   // ping-pong max wavespeed (bit pattern of a non-negative double)
  double t, dt_last;
  long long steps;
  int status;                       // bit 0: non-physical state seen
  int pad;
};

enum { MODE_STAGE1 = 0, MODE_STAGE2 = 1, MODE_RESID = 2 };

struct StageArgs {
  int mode;
  int dirmask;      // bit d: take direction d's fluxes (fused: 7)
  int first;        // MODE_RESID: overwrite instead of accumulate
  int Lz;           // planes per z-chunk
  int cur;          // lam_bits[cur] is lambda(U^n); stage 2 accumulates into lam_bits[cur^1]
  double cfl, dt_fixed;   // dt = dt_fixed > 0 ? dt_fixed : cfl / lambda
  int skip_cfl;           // stage 2: leave the max-wavespeed reduction to the source kernel (NEXT-3)
};

__device__ __forceinline__ double step_dt(const DevScalars* sc, int cur, double cfl, double dt_fixed) {
  if (dt_fixed > 0.0) return dt_fixed;
  return __ddiv_rn(cfl, __longlong_as_double((long long)sc->lam_bits[cur]));
}

__device__ __forceinline__ long long cell_addr(const GridDesc& g, int i, int j, int k) {
  return (long long)(i + g.off[0]) + g.pitch * (long long)(j + g.off[1]) + g.plane * (long long)(k + g.off[2]);
}

// ------------------------------------------------------------------------------------------- a1
// One thread per ghost cell (all five fields).  Index space: [x faces | y faces | z faces]; x-face
// threads are laid out layer-fastest, y/z-face threads x-fastest (coalesced).  Thread 0 also
// advances the device clock when `advance` (first fill of a step) and clears the lambda slot the
// step will reduce into.
__global__ void ghost_fill_kernel(double* __restrict__ U, GridDesc g, DevScalars* sc, int advance, int cur,
                                  double cfl, double dt_fixed) {
  if (advance && blockIdx.x == 0 && threadIdx.x == 0) {
    const double dt = step_dt(sc, cur, cfl, dt_fixed);
    sc->lam_bits[cur ^ 1] = 0ull;
    sc->t += dt;
    sc->dt_last = dt;
    sc->steps += 1;
  }
  const int G = g.g;
  const long long nx = g.n[0], ny = g.n[1], nz = g.n[2];
  const long long cx = g.act[0] ? 2LL * G * ny * nz : 0;
  const long long cy = g.act[1] ? 2LL * G * nx * nz : 0;
  const long long cz = g.act[2] ? 2LL * G * nx * ny : 0;
  const long long total = cx + cy + cz;
  for (long long idx = blockIdx.x * (long long)blockDim.x + threadIdx.x; idx < total;
       idx += (long long)gridDim.x * blockDim.x) {
    int d, m, c[3];
    if (idx < cx) {
      d = 0; m = (int)(idx % (2 * G));
      long long r = idx / (2 * G);
      c[1] = (int)(r % ny); c[2] = (int)(r / ny);
    } else if (idx < cx + cy) {
      long long r = idx - cx;
      d = 1; c[0] = (int)(r % nx); r /= nx;
      m = (int)(r % (2 * G)); c[2] = (int)(r / (2 * G));
    } else {
      long long r = idx - cx - cy;
      d = 2; c[0] = (int)(r % nx); r /= nx;
      c[1] = (int)(r % ny); m = (int)(r / ny);
    }
    const int n = g.n[d];
    if (d == 2 && ((m < G) ? (g.zskip & 1) : (g.zskip & 2))) continue;   // filled by the halo exchange
    int dst, src;
    if (m < G) {                                    // low side, layer m+1
      dst = -(m + 1);
      src = (g.bc == 0) ? n - (m + 1) : (g.bc == 2) ? m : 0;
    } else {                                        // high side, layer m-G+1
      const int l = m - G;
      dst = n + l;
      src = (g.bc == 0) ? l : (g.bc == 2) ? n - 1 - l : n - 1;
    }
    c[d] = dst; const long long pd = cell_addr(g, c[0], c[1], c[2]);
    c[d] = src; const long long ps = cell_addr(g, c[0], c[1], c[2]);
    for (int f = 0; f < g.nf; ++f) {
      const double v = U[f * g.fstride + ps];
      U[f * g.fstride + pd] = (g.bc == 2 && f == 1 + d) ? -v : v;   // reflecting wall: mirror image
    }
  }
}

// ------------------------------------------------------------------------------------------- a7
__device__ __forceinline__ double sum3_sorted(double a, double b, double c) {
  // magnitude-ordered three-term sum (G8) so that lambda after set_state is bit-equal to
  // the definition evaluated in any axis order.
  double x1 = a, x2 = b, x3 = c, t;
  if (fabs(x1) > fabs(x2)) { t = x1; x1 = x2; x2 = t; }
  if (fabs(x2) > fabs(x3)) { t = x2; x2 = x3; x3 = t; }
  if (fabs(x1) > fabs(x2)) { t = x1; x1 = x2; x2 = t; }
  if (x2 == -x3) return x1;
  return __dadd_rn(__dadd_rn(x1, x2), x3);
}

__device__ __forceinline__ void block_max_to_slot(double lam, int bad, DevScalars* sc, int slot, double* red) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) {
    lam = fmax(lam, __shfl_xor_sync(0xffffffffu, lam, o));
    bad |= __shfl_xor_sync(0xffffffffu, bad, o);
  }
  const int w = threadIdx.x >> 5, nw = (blockDim.x + 31) >> 5;
  if ((threadIdx.x & 31) == 0) { red[w] = lam; red[32 + w] = (double)bad; }
  __syncthreads();
  if (threadIdx.x == 0) {
    for (int i = 1; i < nw; ++i) { lam = fmax(lam, red[i]); bad |= (red[32 + i] != 0.0); }
    // lambda >= 0: the IEEE bit pattern is order-preserving as an unsigned integer; max is exact
    // and order-independent, so dt is reproducible run to run.
    atomicMax(&sc->lam_bits[slot], (unsigned long long)__double_as_longlong(lam));
    if (bad) atomicOr(&sc->status, 1);
  }
}

// Standalone CFL pass, correctly rounded operations in the order of the definition (G6, G9).
__global__ void cfl_kernel(const double* __restrict__ U, GridDesc g, DevScalars* sc, int slot) {
  __shared__ double red[64];
  const long long N = (long long)g.n[0] * g.n[1] * g.n[2];
  double lam = 0.0;
  int bad = 0;
  const double gm1 = __dadd_rn(g.gamma, -1.0);
  for (long long idx = blockIdx.x * (long long)blockDim.x + threadIdx.x; idx < N;
       idx += (long long)gridDim.x * blockDim.x) {
    const int i = (int)(idx % g.n[0]);
    const long long r = idx / g.n[0];
    const int j = (int)(r % g.n[1]), k = (int)(r / g.n[1]);
    const long long p = cell_addr(g, i, j, k);
    const double rho = U[p], mx = U[g.fstride + p], my = U[2 * g.fstride + p], mz = U[3 * g.fstride + p],
                 E = U[4 * g.fstride + p];
    const double v[3] = { __ddiv_rn(mx, rho), __ddiv_rn(my, rho), __ddiv_rn(mz, rho) };
    const double ke2 = sum3_sorted(__dmul_rn(mx, v[0]), __dmul_rn(my, v[1]), __dmul_rn(mz, v[2]));
    const double pr = __dmul_rn(gm1, __dadd_rn(E, -__dmul_rn(0.5, ke2)));
    if (!(rho > 0.0 && pr > 0.0) || !(pr < 1.0e300) || !(rho < 1.0e300)) { bad = 1; continue; }
    const double c = __dsqrt_rn(__ddiv_rn(__dmul_rn(g.gamma, pr), rho));
#pragma unroll
    for (int a = 0; a < 3; ++a)
      if (g.act[a]) lam = fmax(lam, __dmul_rn(__dadd_rn(fabs(v[a]), c), g.inv_d[a]));
  }
  block_max_to_slot(lam, bad, sc, slot, red);
}

// ------------------------------------------------------------------------------------------- a6 (per-direction variant)
// stage 1: U1 = U + dt R;   stage 2: U = 1/2 U + 1/2 (U1 + dt R).   Interior cells only.
__global__ void axpy_kernel(const double* __restrict__ Un, const double* __restrict__ U1, const double* __restrict__ R,
                            double* __restrict__ out, GridDesc g, const DevScalars* sc, int stage2, int cur,
                            double cfl, double dt_fixed) {
  const double dt = step_dt(sc, cur, cfl, dt_fixed);
  const long long N = (long long)g.n[0] * g.n[1] * g.n[2];
  for (long long idx = blockIdx.x * (long long)blockDim.x + threadIdx.x; idx < N;
       idx += (long long)gridDim.x * blockDim.x) {
    const int i = (int)(idx % g.n[0]);
    const long long r = idx / g.n[0];
    const int j = (int)(r % g.n[1]), k = (int)(r / g.n[1]);
    const long long p = cell_addr(g, i, j, k);
    for (int f = 0; f < g.nf; ++f) {
      const long long q = f * g.fstride + p;
      if (!stage2) out[q] = fma(dt, R[q], Un[q]);
      else out[q] = 0.5 * Un[q] + 0.5 * fma(dt, R[q], U1[q]);
    }
  }
}

// ------------------------------------------------------------------------------------------- NEXT-4: z-slab halos
// Pack the g lowest / highest interior z-planes of all fields into a contiguous buffer [nf][g][ny][nx]
// (to be sent to the lower / upper neighbour rank), or unpack such a buffer into the low / high z ghost
// planes.  side: 0 = low, 1 = high.  Interior x-y only: the stencils never read edges or corners.
__global__ void halo_copy_kernel(double* __restrict__ U, double* __restrict__ buf, GridDesc g, int side, int unpack) {
  const int G = g.g;
  const long long plane = (long long)g.n[0] * g.n[1], per_field = plane * G, total = per_field * g.nf;
  for (long long idx = blockIdx.x * (long long)blockDim.x + threadIdx.x; idx < total;
       idx += (long long)gridDim.x * blockDim.x) {
    const int f = (int)(idx / per_field);
    long long r = idx - f * per_field;
    const int m = (int)(r / plane);
    r -= m * plane;
    const int j = (int)(r / g.n[0]), i = (int)(r - (long long)j * g.n[0]);
    int k;
    if (!unpack) k = side ? g.n[2] - G + m : m;              // interior planes to send
    else         k = side ? g.n[2] + m : m - G;              // ghost planes to fill
    const long long p = f * g.fstride + cell_addr(g, i, j, k);
    if (unpack) U[p] = buf[idx]; else buf[idx] = U[p];
  }
}

// ------------------------------------------------------------------------------------------- NEXT-3: source update
// Pointwise radiative heating / cooling (eq.6; d_t e = q, d_t E_rad = -q, eq.4), operator-split
// after the advection step, backward Euler over dt (G20): the new internal energy density x solves
// g(x) = x - e - dt c kappa rho (E_tot - x - a (x/(rho c_v))^4) = 0 on [0, E_tot] (g increasing): Newton,
// bisecting when an iterate leaves the bracket.  e + E_rad is conserved exactly.  HBM-bound (6 fields read,
// 2 written: 64 B per cell).  It also carries the step's max-wavespeed reduction (a7), since the source
// changes the pressure.
struct SourceParams { double kappa, c_light, a_rad, cv; };

__global__ void source_kernel(double* __restrict__ U, GridDesc g, DevScalars* sc, SourceParams sp, int cur, double cfl,
                              double dt_fixed) {
  __shared__ double red[64];
  const double dt = step_dt(sc, cur, cfl, dt_fixed);
  const long long N = (long long)g.n[0] * g.n[1] * g.n[2];
  const double gm1 = g.gamma - 1.0;
  const bool act3[3] = { g.act[0] != 0, g.act[1] != 0, g.act[2] != 0 };
  double lam = 0.0;
  int bad = 0;
  for (long long idx = blockIdx.x * (long long)blockDim.x + threadIdx.x; idx < N;
       idx += (long long)gridDim.x * blockDim.x) {
    const int i = (int)(idx % g.n[0]);
    const long long r = idx / g.n[0];
    const int j = (int)(r % g.n[1]), k = (int)(r / g.n[1]);
    const long long p = cell_addr(g, i, j, k);
    double Uc[5];
#pragma unroll
    for (int f = 0; f < 5; ++f) Uc[f] = U[f * g.fstride + p];
    const double Er = U[5 * g.fstride + p];
    const double rho = Uc[0];
    const double ke = 0.5 * (Uc[1] * Uc[1] + Uc[2] * Uc[2] + Uc[3] * Uc[3]) * fast_rcp(rho);
    const double e = Uc[4] - ke, Etot = e + Er;
    const double beta = dt * sp.c_light * sp.kappa * rho, rcv = rho * sp.cv, inv_rcv = fast_rcp(rcv);
    double lo = 0.0, hi = Etot, x = e < 0.0 ? 0.0 : (e > Etot ? Etot : e);
    for (int it = 0; it < 200; ++it) {
      const double T = x * inv_rcv, T2 = T * T, T4 = T2 * T2;
      const double gx = (x - e) - beta * ((Etot - x) - sp.a_rad * T4);
      if (gx > 0.0) hi = x; else lo = x;
      const double dg = 1.0 + beta * (1.0 + 4.0 * sp.a_rad * T2 * T * inv_rcv);
      double xn = fma(-gx, fast_rcp(dg), x);                   // dg >= 1: normal
      if (fabs(xn - x) <= 1e-15 * fabs(xn)) { x = xn; break; }  // converged (also onto a bracket end)
      if (!(xn >= lo && xn <= hi)) xn = 0.5 * (lo + hi);       // Newton left the bracket: bisect
      x = xn;
    }
    Uc[4] = x + ke;
    U[4 * g.fstride + p] = Uc[4];
    U[5 * g.fstride + p] = Etot - x;
    const double l = cell_lambda(Uc, g.gamma, gm1, g.inv_d, act3);
    if (l < 0.0 || !(Etot - x >= 0.0)) bad = 1; else lam = fmax(lam, l);
  }
  block_max_to_slot(lam, bad, sc, cur ^ 1, red);
}

// ------------------------------------------------------------------------------------------- TMA / mbarrier PTX
__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void mbar_init(uint32_t bar, uint32_t count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint32_t bar, uint32_t bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t parity) {
  asm volatile(
      "{\n"
      ".reg .pred p;\n"
      "HARD_WAIT:\n"
      "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
      "@p bra HARD_DONE;\n"
      "bra HARD_WAIT;\n"
      "HARD_DONE:\n"
      "}\n" ::"r"(bar), "r"(parity) : "memory");
}
__device__ __forceinline__ void fence_proxy_async() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }
__device__ __forceinline__ void fence_mbar_init() { asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory"); }

// 4-D tiled TMA load (x, y, z, field) of one x-y box of one z-plane, all five fields.
__device__ __forceinline__ void tma_load_4d(uint32_t dst, const CUtensorMap* map, uint32_t bar, int cx, int cy, int cz,
                                            int cf) {
  asm volatile(
      "cp.async.bulk.tensor.4d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3, %4, %5}], [%6];"
      ::"r"(dst), "l"((unsigned long long)map), "r"(cx), "r"(cy), "r"(cz), "r"(cf), "r"(bar) : "memory");
}

// ------------------------------------------------------------------------------------------- a2..a7 fused stage
// One CTA = a 14 x 16 (x, y) tile of cells marched along z; 256 threads laid out 16 x 16:
//   x: thread (tx, ty) reconstructs cell ix = tx-1 (-1..14) of row ty; the minus value of the right
//      neighbour and the flux of the left face travel by warp shuffles inside the 16-lane row
//      segment: no shared-memory exchange, no barrier.  Threads tx = 1..14 own cells 0..13.
//   y: 14 x 18 = 252 items (cells iy = -1..16) through shared memory (minus values, then fluxes).
//   z: each owner thread marches its own column: the plus value and the flux of the previous plane
//      stay in registers; the z stencil is read from a ring of primitive planes in shared memory.
// Every face flux and every cell reconstruction inside a tile is computed once; 224 of 256 lanes do
// useful work in every phase.  The ring holds conserved planes loaded by TMA (4-D box: x, y, one z
// plane, all NF fields) and converted to primitives in place (a2).  NF = 6 adds the radiation energy
// density (NEXT-1): reconstructed like the other variables, Rusanov flux, untouched by the conversion.
template <int S, int NF = 5>
struct StageCfg {
  static constexpr int G = SchemeTraits<S>::G, R = SchemeTraits<S>::R;
  static constexpr int TX = 14, TY = 16, NT = 256;
  static constexpr int BX = TX + 2 * G, BY = TY + 2 * G;      // TMA box
  static constexpr int VS = BX * BY;                          // doubles per field per plane slot
  static constexpr int SLOT = (NF * VS + 15) / 16 * 16;       // slot stride, multiple of 128 B
  // z window of 2R+1 planes.  R >= 2: the oldest plane is not the x/y plane, it is released after the
  // z reconstruction and its slot takes the next plane (no spare slot); otherwise one spare slot.
  static constexpr int NS = (R >= 2) ? 2 * R + 1 : 2 * R + 2;
  static constexpr int NYI = TX * (TY + 2);                   // y reconstruction items
  static constexpr uint32_t BOX_BYTES = (uint32_t)NF * VS * 8u;
  static constexpr size_t SMEM = (size_t)NS * SLOT * 8 + 2ull * NF * NYI * 8 + NS * 8 + 64 * 8;
  // stage3d_kernel, scheme B: y items in thread order (hard_stage3d.cuh), exchange arrays of TY+2 rows of pitch BX
  static constexpr bool YT = (R < 2);
  static constexpr int NYX = YT ? (TY + 2) * BX : NYI;
  static constexpr size_t SMEM3D = (size_t)NS * SLOT * 8 + 2ull * NF * NYX * 8 + NS * 8 + 64 * 8;
  // resident CTAs per SM: 2, except WENO with six fields (130 KB of shared memory)
  static constexpr int CTAS = (SMEM > 113 * 1024 || SMEM3D > 113 * 1024) ? 1 : 2;
};

// Both face values of all five primitives of one cell along one direction; o[s] = ring offset of
// field 0 at stencil position s - R.  Scheme A applies the positivity fallback (G4): if a reconstructed rho
// or p is <= 0, all variables of the cell become piecewise constant.  No branch: rho and p are reconstructed
// first and fall back by selects; the other variables add their WENO increments with the factor 0 instead of
// 1/6.  "<= 0" is taken on the high words (sign set, or zero): exact for every value but a positive denormal,
// which no admissible state reconstructs.
template <int S, int NF>
__device__ __forceinline__ void recon_item(const double* __restrict__ ring, const int* o, double* pl, double* mi) {
  constexpr int VS = StageCfg<S, NF>::VS;
  if (S == SCHEME_A) {
    double c[NF], wp[NF], wm[NF];
    constexpr int order[6] = { 0, 4, 1, 2, 3, 5 };       // rho and p first: they decide the fallback
    // rho and p get their face values at once; if any of the four is <= 0 they fall back to the cell value by
    // selects (integer pipe), and the other variables take the factor 0 instead of 1/6 in their one DFMA
    int hmin = 0x7fffffff;
    double f6 = 1.0 / 6.0;
#pragma unroll
    for (int q = 0; q < NF; ++q) {
      const int v = order[q];
      c[v] = ring[o[2] + v * VS];
      wenoz_incr(ring[o[0] + v * VS], ring[o[1] + v * VS], c[v], ring[o[3] + v * VS], ring[o[4] + v * VS], wp[v], wm[v]);
      if (q < 2) {
        pl[v] = fma(wp[v], 1.0 / 6.0, c[v]);
        mi[v] = fma(wm[v], 1.0 / 6.0, c[v]);
        hmin = min(hmin, min(__double2hiint(pl[v]), __double2hiint(mi[v])));
      }
      if (q == 1) {
        const bool fb = hmin <= 0;
        f6 = fb ? 0.0 : 1.0 / 6.0;
        pl[0] = fb ? c[0] : pl[0]; mi[0] = fb ? c[0] : mi[0];
        pl[4] = fb ? c[4] : pl[4]; mi[4] = fb ? c[4] : mi[4];
      }
      if (q >= 2) { pl[v] = fma(wp[v], f6, c[v]); mi[v] = fma(wm[v], f6, c[v]); }
    }
  } else {
#pragma unroll
    for (int v = 0; v < NF; ++v)
      minmod_pair(ring[o[0] + v * VS], ring[o[1] + v * VS], ring[o[2] + v * VS], pl[v], mi[v]);
  }
}

// Flux through a face with normal along direction D from (rho,u,v,w,p) face states; result in
// (rho, mx, my, mz, E) order.
template <int S, int D, int NF>
__device__ __forceinline__ void face_flux(const double* L, const double* Rr, double gamma, double inv_gm1, double* F) {
  constexpr int n = 1 + D, t1 = 1 + (D + 1) % 3, t2 = 1 + (D + 2) % 3;
  const double WL[5] = { L[0], L[n], L[t1], L[t2], L[4] };
  const double WR[5] = { Rr[0], Rr[n], Rr[t1], Rr[t2], Rr[4] };
  double f[5], alpha;
  riemann_flux<S>(WL, WR, gamma, inv_gm1, f, alpha);
  F[0] = f[0]; F[n] = f[1]; F[t1] = f[2]; F[t2] = f[3]; F[4] = f[4];
  // NEXT-1 (G19): Rusanov flux of the advected radiation energy density, alpha = max(|u_n| + c_s)
  if (NF == 6) F[5] = 0.5 * (L[5] * WL[1] + Rr[5] * WR[1]) - 0.5 * alpha * (Rr[5] - L[5]);
}

template <int S, int NF>
__global__ void __launch_bounds__(256, (StageCfg<S, NF>::CTAS))
stage_kernel(const __grid_constant__ CUtensorMap tmap, const double* __restrict__ Usrc, const double* Uaux,
             double* Uout, GridDesc g, DevScalars* sc, StageArgs a) {
  using C = StageCfg<S, NF>;
  constexpr int G = C::G, R = C::R, TX = C::TX, TY = C::TY, BX = C::BX, VS = C::VS, SLOT = C::SLOT, NS = C::NS,
                NYI = C::NYI;
  extern __shared__ __align__(1024) unsigned char smem_raw[];
  double* ring = reinterpret_cast<double*>(smem_raw);   // dynamic smem base is 1024-B aligned (TMA needs 128)
  double* RMy = ring + NS * SLOT;      // y minus values, item-indexed [v][item]
  double* Fy = RMy + NF * NYI;         // y face fluxes: item's upper face
  unsigned long long* bars = reinterpret_cast<unsigned long long*>(Fy + NF * NYI);
  double* red = reinterpret_cast<double*>(bars + NS);

  const int tid = threadIdx.x, tx = tid & 15, ty = tid >> 4;
  const int i0 = blockIdx.x * TX, j0 = blockIdx.y * TY, k0 = blockIdx.z * a.Lz;
  const int kend = min(g.n[2], k0 + a.Lz);
  const bool ax = g.act[0] && (a.dirmask & 1), ay = g.act[1] && (a.dirmask & 2), az = g.act[2] && (a.dirmask & 4);
  const int rows = min(TY, g.n[1] - j0), cols = min(TX, g.n[0] - i0);
  const bool mine = tx >= 1 && tx <= cols && ty < rows;          // thread tx owns cell ix = tx - 1
  const bool yitem = ay && tid < TX * (rows + 2), yface = ay && tid < TX * (rows + 1);
  const int y_c = tid / TX, y_ix = tid - y_c * TX;               // y item: cell (y_ix, y_c - 1)
  const double gamma = g.gamma, gm1 = gamma - 1.0, inv_gm1 = 1.0 / gm1;
  const double dt = step_dt(sc, a.cur, a.cfl, a.dt_fixed);
  const double idx = g.inv_d[0], idy = g.inv_d[1], idz = g.inv_d[2];

  // z window of iteration kk: planes [kk + ld - rz, kk + ld + rz]; with z active the z stencil runs
  // one plane ahead so that both z faces of plane kk are known when its x/y fluxes are.
  const int ld = az ? 1 : 0, rz = az ? R : 0;
  const int kfirst = az ? k0 - 2 : k0;
  const int zb = kfirst + ld - rz;                     // first plane ever loaded; ring slot = (z - zb) % NS
  const int cx = g.off[0] + i0 - G, cy = g.off[1] + j0 - G;      // cx = i0: even, so 16-byte aligned

  if (tid == 0) {
    for (int s = 0; s < NS; ++s) mbar_init(smem_u32(&bars[s]), 1);
    fence_mbar_init();
  }
  __syncthreads();

  auto issue = [&](int z) {                            // one thread
    const int q = z - zb, slot = q % NS;
    const uint32_t bar = smem_u32(&bars[slot]);
    mbar_expect_tx(bar, C::BOX_BYTES);
    tma_load_4d(smem_u32(ring + slot * SLOT), &tmap, bar, cx, cy, g.off[2] + z, 0);
  };
  auto convert_cell = [&](double* sl, int c) {
    double U[5], W[5];
#pragma unroll
    for (int v = 0; v < 5; ++v) U[v] = sl[v * VS + c];
    cons_to_prim(U, gm1, W);
#pragma unroll
    for (int v = 1; v < 5; ++v) sl[v * VS + c] = W[v];
  };
  // all threads: wait for the plane, conserved -> primitive in place (a2).  Each thread converts first the cell
  // of ITS OWN column (the only cell of the new plane that the next z reconstruction reads, and only this
  // thread reads it), then a share of the halo ring, which nobody reads before the plane becomes the x/y
  // plane several barriers later: no block-wide barrier is needed after the conversion when z is active.
  auto wait_convert = [&](int z) {
    const int q = z - zb, slot = q % NS;
    mbar_wait(smem_u32(&bars[slot]), (uint32_t)((q / NS) & 1));
    double* sl = ring + slot * SLOT;
    convert_cell(sl, (ty + G) * BX + (tx - 1 + G));
    constexpr int NTB = 2 * G * BX, NCOL = BX - 16, NREM = NTB + NCOL * TY;
    for (int r = tid; r < NREM; r += C::NT) {
      int row, col;
      if (r < NTB) {
        row = r / BX; col = r - row * BX;
        row = row < G ? row : row + TY;
      } else {
        const int qq = r - NTB, rm = qq / NCOL, cc = qq - rm * NCOL;
        row = G + rm; col = cc < G - 1 ? cc : cc + 16;
      }
      convert_cell(sl, row * BX + col);
    }
  };

  if (tid == 0)
    for (int z = zb; z <= zb + 2 * rz; ++z) issue(z);
  for (int z = zb; z <= zb + 2 * rz; ++z) wait_convert(z);
  __syncthreads();

  double zplus[NF] = {}, Fzold[NF] = {};
  double lam_loc = 0.0;
  int bad = 0;
  const bool act3[3] = { g.act[0] != 0, g.act[1] != 0, g.act[2] != 0 };

  for (int kk = kfirst; kk < kend; ++kk) {
    const bool doxy = kk >= k0;
    const int znext = kk + 1 + ld + rz;
    const bool more = kk + 1 < kend;
    // the slot of the next plane still holds the oldest plane of this window (no spare slot): it is
    // released by the barrier after the z reconstruction
    const bool late = (znext - NS) >= (kk + ld - rz);
    if (more && !late && tid == 0) { fence_proxy_async(); issue(znext); }
    const int slot_c = ((kk - zb) % NS) * SLOT;        // plane kk (x/y stencils)
    double Lacc[NF] = {};                             // L(U) of the owned cell, accumulated in registers (a5)

    // ---- z: reconstruct plane kk+1 (own column), flux through face kk+1/2 with the carried plus value
    if (az) {
      int o[2 * R + 1];
      const int cell = (ty + G) * BX + (tx - 1 + G);
#pragma unroll
      for (int s = -R; s <= R; ++s) o[s + R] = ((kk + 1 + s - zb) % NS) * SLOT + cell;
      double pl[NF], mi[NF];
      recon_item<S, NF>(ring, o, pl, mi);
      if (kk >= k0 - 1) {
        double F[NF];
        face_flux<S, 2, NF>(zplus, mi, gamma, inv_gm1, F);
#pragma unroll
        for (int v = 0; v < NF; ++v) { Lacc[v] = (Fzold[v] - F[v]) * idz; Fzold[v] = F[v]; }
      }
#pragma unroll
      for (int v = 0; v < NF; ++v) zplus[v] = pl[v];
    }
    // ---- y: reconstruct the 14 x (rows+2) items of plane kk; minus values to shared memory
    double plY[NF] = {};
    if (doxy && yitem) {
      int o[2 * R + 1];
      const int cell = slot_c + (y_c - 1 + G) * BX + (y_ix + G);
#pragma unroll
      for (int s = -R; s <= R; ++s) o[s + R] = cell + s * BX;
      double mi[NF];
      recon_item<S, NF>(ring, o, plY, mi);
#pragma unroll
      for (int v = 0; v < NF; ++v) RMy[v * NYI + tid] = mi[v];
    }
    __syncthreads();                                                             // barrier 1
    if (more && late && tid == 0) { fence_proxy_async(); issue(znext); }

    // own-cell conserved values for the RK combination, consumed after barrier 2.  Scheme A issues the
    // loads here; scheme B after the x phase (measured: holding 10-20 registers through the x phase
    // costs B 4 %, while the later issue costs A 2 %).
    double uc[NF] = {}, ua[NF] = {};
    long long pc = 0;
    auto load_own = [&]() {
      if (doxy && mine) {
        pc = cell_addr(g, i0 + tx - 1, j0 + ty, kk);
        if (a.mode != MODE_RESID) {
#pragma unroll
          for (int v = 0; v < NF; ++v) uc[v] = Usrc[v * g.fstride + pc];
        }
        if (a.mode == MODE_STAGE2 || (a.mode == MODE_RESID && !a.first)) {
#pragma unroll
          for (int v = 0; v < NF; ++v) ua[v] = Uaux[v * g.fstride + pc];
        }
      }
    };
    if (S == SCHEME_A) load_own();
    // ---- x: reconstruct cell tx-1 of row ty; neighbours by shuffles inside the 16-lane row segment
    if (doxy && ax) {
      double pl[NF], mi[NF], mr[NF], F[NF];
#pragma unroll
      for (int v = 0; v < NF; ++v) pl[v] = mi[v] = (v == 0 || v == 4) ? 1.0 : 0.0;
      if (ty < rows) {
        int o[2 * R + 1];
        const int cell = slot_c + (ty + G) * BX + (tx - 1 + G);
#pragma unroll
        for (int s = -R; s <= R; ++s) o[s + R] = cell + s;
        recon_item<S, NF>(ring, o, pl, mi);
      }
#pragma unroll
      for (int v = 0; v < NF; ++v) mr[v] = __shfl_down_sync(0xffffffffu, mi[v], 1, 16);   // minus of cell tx
      face_flux<S, 0, NF>(pl, mr, gamma, inv_gm1, F);                                        // face right of cell tx-1
#pragma unroll
      for (int v = 0; v < NF; ++v) {
        const double Fl = __shfl_up_sync(0xffffffffu, F[v], 1, 16);                      // face left of cell tx-1
        Lacc[v] -= (F[v] - Fl) * idx;
      }
    }
    if (S != SCHEME_A) load_own();
    // ---- y fluxes: face above item (between item and item + TX)
    if (doxy && yface) {
      double mr[NF], F[NF];
#pragma unroll
      for (int v = 0; v < NF; ++v) mr[v] = RMy[v * NYI + tid + TX];
      face_flux<S, 1, NF>(plY, mr, gamma, inv_gm1, F);
#pragma unroll
      for (int v = 0; v < NF; ++v) Fy[v * NYI + tid] = F[v];
    }
    __syncthreads();                                                             // barrier 2

    // ---- a5 + a6 (+ a7): finish the divergence, RK combination, store
    if (doxy && mine) {
      double out[NF];
      const int yi = ty * TX + (tx - 1);               // item of cell (tx-1, ty-1): its upper face is our lower face
#pragma unroll
      for (int v = 0; v < NF; ++v) {
        double L = Lacc[v];
        if (ay) L -= (Fy[v * NYI + yi + TX] - Fy[v * NYI + yi]) * idy;
        if (a.mode == MODE_STAGE1) out[v] = fma(dt, L, uc[v]);
        else if (a.mode == MODE_STAGE2) out[v] = 0.5 * ua[v] + 0.5 * fma(dt, L, uc[v]);
        else out[v] = a.first ? L : ua[v] + L;
        Uout[v * g.fstride + pc] = out[v];
      }
      if (a.mode == MODE_STAGE2 && !a.skip_cfl) {
        const double l = cell_lambda(out, gamma, gm1, g.inv_d, act3);
        if (l < 0.0) bad = 1; else lam_loc = dmax(lam_loc, l);
      }
    }
    if (more) wait_convert(znext);
    // z inactive: the plane just converted is the next iteration's x/y plane, read by other threads at once
    if (!az) __syncthreads();                                                    // barrier 3 (2-D / 1-D / x,y passes)
  }
  if (a.mode == MODE_STAGE2 && !a.skip_cfl) block_max_to_slot(lam_loc, bad, sc, a.cur ^ 1, red);
}

#include "hard_stage3d.cuh"

}  // namespace hard
