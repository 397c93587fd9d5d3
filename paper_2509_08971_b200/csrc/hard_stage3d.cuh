// hard_stage3d.cuh — the fused RK stage (a2..a7) specialised for the 3-D case: all three directions
// active, all fluxes in one launch, the stage (1 or 2) a template parameter.  Same tiling, ring and thread
// mapping as the generic stage_kernel (hard_kernels.cuh), which keeps serving 1-D / 2-D meshes and the
// per-direction variant.  What the specialisation buys (measured):
//  * straight-line code between the synchronisation points of a plane (no activity / mode tests, no ragged-tile
//    branches: out-of-range lanes recompute a valid item and only the stores are predicated), so ptxas
//    interleaves the serial Riemann chains with the reconstruction next to them;
//  * loop-carried z state updated in place (no register copies at the back edge); two peeled lead-in planes;
//  * split-phase barriers on mbarriers (arrive after producing, wait before consuming) wherever independent work
//    lies in between: scheme B around the x phase and the plane conversion, scheme A around the x phase;
//  * own-cell loads for the RK combination pinned early (volatile asm) so a whole phase covers their latency.
//  * scheme B: y items in thread order with the 28 items of rows -1 and TY placed on the lanes whose spare banks they
//    fall on, exchange arrays with the ring's pitch: every shared-memory load is bank-conflict-free (see `celly`).
// Included by hard_kernels.cuh inside namespace hard.
#pragma once

__device__ __forceinline__ double ldg_pinned(const double* p) {
  double v;
  asm volatile("ld.global.f64 %0, [%1];" : "=d"(v) : "l"(p));
  return v;
}

// Split-phase CTA barrier on an mbarrier (8 arrivals: one elected lane per warp): arrive after producing,
// wait just before consuming, with independent work in between, so that no warp idles for the slowest one.
__device__ __forceinline__ void warp_arrive(uint32_t bar) {
  __syncwarp();
  if ((threadIdx.x & 31) == 0) asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(bar) : "memory");
}

template <int S, int NF, int MODE>
__global__ void __launch_bounds__(256, (StageCfg<S, NF>::CTAS))
stage3d_kernel(const __grid_constant__ CUtensorMap tmap, const double* __restrict__ Usrc, const double* Uaux,
               double* Uout, GridDesc g, DevScalars* sc, StageArgs a) {
  using C = StageCfg<S, NF>;
  constexpr int G = C::G, R = C::R, TX = C::TX, TY = C::TY, BX = C::BX, VS = C::VS, SLOT = C::SLOT, NS = C::NS,
                NYI = C::NYI;
  constexpr bool LATE = (R >= 2);          // no spare ring slot: the next plane is requested after the z reconstruction
  // phase order after the y reconstruction: y fluxes then x (frees the y plus values before the x phase; LATE needs
  // the full barrier 1 anyway), or x then y fluxes (barrier 1 split-phase around the x phase)
  constexpr bool YFIRST = LATE;
  static_assert(YFIRST || !LATE, "the late ring request needs the full barrier of the y-first order");
  extern __shared__ __align__(1024) unsigned char smem_raw[];
  double* ring = reinterpret_cast<double*>(smem_raw);
  constexpr bool YT = C::YT;           // y items in thread order (scheme B), see below
  constexpr int NYX = C::NYX;          // doubles per field of a y exchange array
  double* RMy = ring + NS * SLOT;      // y minus values [v][slot of the item]
  double* Fy = RMy + NF * NYX;         // y face fluxes: item's upper face
  unsigned long long* bars = reinterpret_cast<unsigned long long*>(Fy + NF * NYX);
  double* red = reinterpret_cast<double*>(bars + NS);

  const int tid = threadIdx.x, tx = tid & 15, ty = tid >> 4;
  const int i0 = blockIdx.x * TX, j0 = blockIdx.y * TY, k0 = blockIdx.z * a.Lz;
  const int kend = min(g.n[2], k0 + a.Lz);
  const int rows = min(TY, g.n[1] - j0), cols = min(TX, g.n[0] - i0);
  const bool mine = tx >= 1 && tx <= cols && ty < rows;          // thread tx owns cell ix = tx - 1
  // y items: cells (y_ix, y_c - 1), y_c = 0..TY+1; the last four threads repeat item NYI-1 (nothing stored)
  const int yit = min(tid, NYI - 1), y_c = yit / TX, y_ix = yit - y_c * TX;
  const double gamma = g.gamma, gm1 = gamma - 1.0, inv_gm1 = 1.0 / gm1;
  const double dt = step_dt(sc, a.cur, a.cfl, a.dt_fixed);
  const double idx = g.inv_d[0], idy = g.inv_d[1], idz = g.inv_d[2];
  const int zb = k0 - R - 1;                                     // first plane loaded; ring slot of plane z = (z - zb) % NS
  const int cx = g.off[0] + i0 - G, cy = g.off[1] + j0 - G;      // cx = i0: even, so 16-byte aligned
  const int cellz = (ty + G) * BX + (tx - 1 + G);                // own column (also the x item of this thread)
  // Scheme A: the 252 items in linear order, item = cell (y_ix, y_c - 1); exchange slot = item index.  A half-warp
  // then straddles ring rows (pitch 20): two-way bank conflicts on part of the y reads (with pitch 20
  // no conflict-free placement exists next to 2 CTAs/SM).
  // Scheme B (YT): items in THREAD ORDER.  Lane tx = 1..14 of row ty takes its own cell (tx-1, ty): a half-warp reads
  // 14 consecutive doubles of one ring row.  The 28 items of rows -1 and TY go to the lanes tx = 0 / 15, each to
  // the half-warp whose two spare banks (ring pitch 18: banks 2ty+5 and 2ty+4 mod 16, counted in doubles) are exactly
  // the banks of that item: lane 0 takes (row -1, col 2ty+1) for ty <= 6, (row TY, col 13) for ty = 7, (row TY, col
  // 2ty-17) for ty = 9..14; lane 15 takes (row -1, col 2ty), (row TY, col 12), (row TY, col 2ty-18).  Stencil, field
  // and slot offsets shift every lane's bank alike, so all y ring reads are conflict-free.  The four lanes left over
  // (ty = 8, 15) repeat their neighbour's cell (same address: a broadcast).  The exchange arrays mirror the ring's
  // geometry — slot of item (col, row) = (row + 1) * BX + col + 1 — so the same bank matching holds there: a
  // half-warp reads the 14 slots of the row above plus, for its two row -1 items, two slots of row 0 that fall on
  // its spare banks.
  static_assert(!YT || (BX == 18 && TX == 14 && TY == 16 && G == 2), "the bank matching of the extra y items is worked out for ring pitch 18");
  int e_row = 0, e_col = 0;
  bool e_item = false;
  if (YT && (tx == 0 || tx == 15)) {
    const int odd = (tx == 0) ? 1 : 0;
    if (ty <= 6)                  { e_item = true; e_row = -1; e_col = 2 * ty + odd; }
    else if (ty == 7)             { e_item = true; e_row = TY; e_col = 12 + odd; }
    else if (ty >= 9 && ty <= 14) { e_item = true; e_row = TY; e_col = 2 * ty - 18 + odd; }
    else                          { e_row = ty; e_col = (tx == 0) ? 0 : TX - 1; }
  }
  const bool xl = YT && (tx == 0 || tx == 15);
  const int celly = !YT ? (y_c - 1 + G) * BX + (y_ix + G) : xl ? (e_row + G) * BX + (e_col + G) : cellz;
  const int ys_own = !YT ? tid : (ty + 1) * BX + tx;                         // where every lane stores (edge slots: unused)
  const int ys_x = (e_row + 1) * BX + e_col + 1;                             // slot of an extra item
  const int ys_up = !YT ? min(tid + TX, NYI - 1) : (xl && e_item && e_row < 0) ? ys_x + BX : ys_own + BX;   // item above
  const bool ystore = YT || tid < NYI;
  const bool xstore_rm = YT && e_item && e_row == TY, xstore_fy = YT && e_item && e_row == -1;

  // red[62], red[63] (unused by the final reduction) hold the two split-phase barriers of the plane loop
  const uint32_t barY = smem_u32(&red[62]), barF = smem_u32(&red[63]);
  if (tid == 0) {
    for (int s = 0; s < NS; ++s) mbar_init(smem_u32(&bars[s]), 1);
    mbar_init(barY, 8);
    mbar_init(barF, 8);
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
  // wait for the plane, conserved -> primitive in place (a2): own column first (see stage_kernel), then a share of the halo
  auto wait_convert = [&](int z) {
    const int q = z - zb, slot = q % NS;
    mbar_wait(smem_u32(&bars[slot]), (uint32_t)((q / NS) & 1));
    double* sl = ring + slot * SLOT;
    convert_cell(sl, cellz);
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
    for (int z = zb; z <= zb + 2 * R; ++z) issue(z);
  for (int z = zb; z <= zb + 2 * R; ++z) wait_convert(z);
  __syncthreads();

  // loop-carried z state of the own column: plus value of the last reconstructed plane, and the flux through
  // the last face already multiplied by 1/dz
  double zplus[NF], Cz[NF];
#pragma unroll
  for (int v = 0; v < NF; ++v) { zplus[v] = (v == 0 || v == 4) ? 1.0 : 0.0; Cz[v] = 0.0; }
  double lam_loc = 0.0;
  int bad = 0;
  const bool act3[3] = { true, true, true };

  // z: reconstruct plane kk+1 (own column), flux through face kk+1/2 with the carried plus value.
  // p = ring slot of plane kk.  Lz = -(F(kk+1/2) - F(kk-1/2)) / dz.
  auto zphase = [&](int p, double* Lz) {
    int o[2 * R + 1];
#pragma unroll
    for (int s = -R; s <= R; ++s) {
      int sl = p + 1 + s;                               // in [1 - R, NS + R]
      sl = sl < 0 ? sl + NS : (sl >= NS ? sl - NS : sl);
      o[s + R] = sl * SLOT + cellz;
    }
    double pl[NF], mi[NF], F[NF];
    recon_item<S, NF>(ring, o, pl, mi);
    face_flux<S, 2, NF>(zplus, mi, gamma, inv_gm1, F);
#pragma unroll
    for (int v = 0; v < NF; ++v) {
      const double Cn = __dmul_rn(F[v], idz);           // rounded product, never contracted: equal fluxes cancel
      Lz[v] = Cz[v] - Cn;                               // exactly (a uniform state is preserved bit for bit)
      Cz[v] = Cn;
      zplus[v] = pl[v];
    }
  };

  int p = R - 1;                                        // slot of plane kk = k0 - 2
  // ---- two lead-in planes: z only
  for (int kk = k0 - 2; kk < k0; ++kk) {
    const int znext = kk + 2 + R;
    if (!LATE && tid == 0) { fence_proxy_async(); issue(znext); }
    double Lz[NF];
    zphase(p, Lz);
    __syncthreads();
    if (LATE && tid == 0) { fence_proxy_async(); issue(znext); }
    wait_convert(znext);
    p = (p + 1 == NS) ? 0 : p + 1;
  }

  uint32_t ph = 0;                                      // phase parity of the split-phase barriers
  for (int kk = k0; kk < kend; ++kk) {
    const int znext = kk + 2 + R;
    const bool more = kk + 1 < kend;
    if (!LATE && more && tid == 0) { fence_proxy_async(); issue(znext); }
    const int slot_c = p * SLOT;                        // plane kk (x/y stencils)
    double Lacc[NF];
    zphase(p, Lacc);
    // own-cell conserved values for the RK combination (consumed in the epilogue), requested early so that a whole
    // phase covers their latency; volatile asm keeps ptxas from sinking them to the point of use.
    double uc[NF], ua[NF];
    const long long pc = cell_addr(g, i0 + tx - 1, j0 + ty, kk);
    auto load_uc = [&]() {
      if (mine) {
#pragma unroll
        for (int v = 0; v < NF; ++v) uc[v] = ldg_pinned(Usrc + v * g.fstride + pc);
      }
    };
    auto load_ua = [&]() {
      if (MODE == MODE_STAGE2 && mine) {
#pragma unroll
        for (int v = 0; v < NF; ++v) ua[v] = ldg_pinned(Uaux + v * g.fstride + pc);
      }
    };
    // ---- y: reconstruct the 14 x 18 items of plane kk; minus values to shared memory
    double plY[NF];
    {
      int o[2 * R + 1];
#pragma unroll
      for (int s = -R; s <= R; ++s) o[s + R] = slot_c + celly + s * BX;
      double mi[NF];
      recon_item<S, NF>(ring, o, plY, mi);
      if (ystore) {
#pragma unroll
        for (int v = 0; v < NF; ++v) RMy[v * NYX + ys_own] = mi[v];
      }
      if (xstore_rm) {                                 // a second store: the extra lanes' items of row TY
#pragma unroll
        for (int v = 0; v < NF; ++v) RMy[v * NYX + ys_x] = mi[v];
      }
    }
    // barrier 1 (RMy written -> read).  YFIRST: a full barrier, the y fluxes follow at once.  Otherwise split-phase:
    // arrive here, wait before the y fluxes, with the x phase in between.
    if (YFIRST) {
      __syncthreads();
      if (LATE && more && tid == 0) { fence_proxy_async(); issue(znext); }   // every warp is past its z reconstruction
    } else {
      warp_arrive(barY);
    }
    // ---- x: reconstruct cell tx-1 of row ty; neighbours by shuffles inside the 16-lane row segment
    auto xphase = [&]() {
      double pl[NF], mi[NF], mr[NF], F[NF];
      int o[2 * R + 1];
#pragma unroll
      for (int s = -R; s <= R; ++s) o[s + R] = slot_c + cellz + s;
      recon_item<S, NF>(ring, o, pl, mi);
#pragma unroll
      for (int v = 0; v < NF; ++v) mr[v] = __shfl_down_sync(0xffffffffu, mi[v], 1, 16);   // minus of cell tx
      face_flux<S, 0, NF>(pl, mr, gamma, inv_gm1, F);                                        // face right of cell tx-1
#pragma unroll
      for (int v = 0; v < NF; ++v) {
        const double Fl = __shfl_up_sync(0xffffffffu, F[v], 1, 16);                      // face left of cell tx-1
        Lacc[v] = fma(Fl - F[v], idx, Lacc[v]);
      }
    };
    // ---- y fluxes: face above item (between item and item + TX); the top row's result is not used
    auto yflux = [&]() {
      double mr[NF], F[NF];
#pragma unroll
      for (int v = 0; v < NF; ++v) mr[v] = RMy[v * NYX + ys_up];
      face_flux<S, 1, NF>(plY, mr, gamma, inv_gm1, F);
      if (ystore) {
#pragma unroll
        for (int v = 0; v < NF; ++v) Fy[v * NYX + ys_own] = F[v];
      }
      if (xstore_fy) {                                 // a second store: the extra lanes' faces below row 0
#pragma unroll
        for (int v = 0; v < NF; ++v) Fy[v * NYX + ys_x] = F[v];
      }
    };
    // barrier 2 (Fy written -> read) is split-phase in both orders
    if (YFIRST) {
      load_uc();                                       // measured: both requests here, or both after the y fluxes, cost 3-4 %
      yflux();
      warp_arrive(barF);
      load_ua();
      xphase();
      if (more) wait_convert(znext);                   // independent of Fy
    } else {
      load_uc();
      load_ua();
      xphase();
      mbar_wait(barY, ph);
      yflux();
      warp_arrive(barF);
      if (more) wait_convert(znext);                   // independent of Fy: covers the other warps' arrival
    }
    mbar_wait(barF, ph);
    ph ^= 1u;

    // ---- a5 + a6 (+ a7): finish the divergence, RK combination, store
    if (mine) {
      double out[NF];
      // slot of the item of cell (tx-1, ty-1): its upper face is our lower face; the next row's slot is our own item
      const int yi = YT ? ty * BX + tx : ty * TX + (tx - 1), yj = YT ? yi + BX : yi + TX;
#pragma unroll
      for (int v = 0; v < NF; ++v) {
        const double L = fma(Fy[v * NYX + yi] - Fy[v * NYX + yj], idy, Lacc[v]);
        if (MODE == MODE_STAGE1) out[v] = fma(dt, L, uc[v]);
        else out[v] = 0.5 * ua[v] + 0.5 * fma(dt, L, uc[v]);
        Uout[v * g.fstride + pc] = out[v];
      }
      if (MODE == MODE_STAGE2 && !a.skip_cfl) {
        const double l = cell_lambda(out, gamma, gm1, g.inv_d, act3);
        if (l < 0.0) bad = 1; else lam_loc = dmax(lam_loc, l);
      }
    }
    p = (p + 1 == NS) ? 0 : p + 1;
  }
  if (MODE == MODE_STAGE2 && !a.skip_cfl) block_max_to_slot(lam_loc, bad, sc, a.cur ^ 1, red);
}
