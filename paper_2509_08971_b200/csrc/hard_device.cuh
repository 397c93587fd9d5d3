// hard_device.cuh — device arithmetic of the hot path (sm_100a): conserved->primitive with the
// ideal-gas EOS, limited face reconstruction, approximate Riemann fluxes.  Written from PAPER.md
// (eq.2-3) and the DESIGN.md readings; shares nothing with oracle/.
//
// Precision: everything is fp64.  Unlike the oracle (correctly rounded ops in a fixed order, no FMA
// contraction) this code lets nvcc contract to DFMA and regroups sums; DESIGN.md "Tolerance"
// derives why that stays inside 1e-12 (one step) / 1e-9 (100 steps).
#pragma once
#include <cuda_runtime.h>

namespace hard {

constexpr int SCHEME_A = 0;   // WENO5-Z + HLL
constexpr int SCHEME_B = 1;   // MUSCL-minmod + HLLC (BASELINE.json north_star fallback)

template <int S> struct SchemeTraits;
template <> struct SchemeTraits<SCHEME_A> { static constexpr int G = 3, R = 2; };
template <> struct SchemeTraits<SCHEME_B> { static constexpr int G = 2, R = 1; };

// 1/x for normal, finite x: MUFU.RCP64H seed (about 20 good bits) + two Newton steps (4 DFMA), error
// about 1 ulp; no special-case handling (the IEEE division sequence costs about 10 fp64-pipe
// instructions).  Callers pass quantities that are normal by construction.
__device__ __forceinline__ double fast_rcp(double x) {
  double y;
  asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(x));
  double e = fma(-x, y, 1.0);
  y = fma(y, e, y);
  e = fma(-x, y, 1.0);
  return fma(y, e, y);
}

// 1/sqrt(x) for normal, finite x > 0: MUFU.RSQ64H seed + two Newton steps (7 fp64-pipe instructions,
// about 1 ulp), no special-case handling.
__device__ __forceinline__ double fast_rsqrt(double x) {
  double y;
  asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(x));
  const double h = 0.5 * x;
  double e = fma(-h, y * y, 0.5);
  y = fma(y, e, y);
  e = fma(-h, y * y, 0.5);
  return fma(y, e, y);
}

// a2 (eq.2): (rho, mx, my, mz, E) -> (rho, u, v, w, p).
__device__ __forceinline__ void cons_to_prim(const double U[5], double gm1, double W[5]) {
  const double inv = fast_rcp(U[0]);
  W[0] = U[0];
  W[1] = U[1] * inv;
  W[2] = U[2] * inv;
  W[3] = U[3] * inv;
  W[4] = gm1 * (U[4] - 0.5 * (U[1] * W[1] + U[2] * W[2] + U[3] * W[3]));
}

// a3, scheme A (Borges et al. [18]; G1: eps = 1e-40, power 1, d = (1/10, 6/10, 3/10)).
// Both face values of cell i from q[i-2..i+2] = (a,b,c,d,e): plus at i+1/2, minus at i-1/2.  The
// minus value is the same function on the mirrored stencil, so the smoothness indicators are shared
// (beta0' = beta2, beta1' = beta1, beta2' = beta0).  Algebraically identical to the definition, but
// arranged for the fp64 pipe:
//  * everything in terms of the four differences d1..d4 (candidates minus c are 2-term forms);
//  * beta scaled by 12/13 (beta' = s^2 + 3/13 t^2, eps' = 12/13 eps): tau/(beta+eps) is unchanged;
//  * weights d_k (1 + tau/B_k) multiplied through by B0 B1 B2: d_k (B_k + tau) prod_{j!=k} B_j, which
//    needs no division; ONE reciprocal 1/(sp*sm) normalises both sides.
//    Range: B in [9e-41, ~1e17] for admissible data of the configs, so products of three B's and the
//    square of their sum stay within [1e-241, 1e110]: no overflow / underflow in fp64.
__device__ __forceinline__ void wenoz_pair(double a, double b, double c, double d, double e, double& plus,
                                           double& minus) {
  const double eps = (12.0 / 13.0) * 1e-40, k3 = 3.0 / 13.0;
  const double d1 = b - a, d2 = c - b, d3 = d - c, d4 = e - d;
  const double s0 = d2 - d1, s1 = d3 - d2, s2 = d4 - d3;
  const double t0 = fma(3.0, d2, -d1), t1 = d2 + d3, t2 = fma(-3.0, d3, d4);
  const double B0 = fma(s0, s0, fma(k3 * t0, t0, eps));
  const double B1 = fma(s1, s1, fma(k3 * t1, t1, eps));
  const double B2 = fma(s2, s2, fma(k3 * t2, t2, eps));
  const double tau = fabs(B0 - B2);
  const double P12 = B1 * B2, P02 = B0 * B2, P01 = B0 * B1;
  const double T0 = B0 + tau, T1 = B1 + tau, T2 = B2 + tau;
  const double a0 = (0.1 * T0) * P12, a1 = (0.6 * T1) * P02;                // plus weights (unnormalised)
  const double m0 = (0.1 * T2) * P01;                                       // minus weights; m1 = a1
  const double a2 = 3.0 * m0, m2 = 3.0 * a0;                                // 0.3 T2 P01 and 0.3 T0 P12
  const double sp = (a0 + a1) + a2, sm = (m0 + a1) + m2;
  // 6 (q_k - c) for the plus side and 6 (p_k - c) for the minus side
  const double q0 = fma(5.0, d2, -2.0 * d1), q1 = fma(2.0, d3, d2), q2 = fma(4.0, d3, -d4);
  const double p0 = fma(-5.0, d3, 2.0 * d4), p1 = -fma(2.0, d2, d3), p2 = fma(-4.0, d2, d1);
  const double np = fma(a2, q2, fma(a1, q1, a0 * q0));
  const double nm = fma(m2, p2, fma(a1, p1, m0 * p0));
  const double inv6 = (1.0 / 6.0) * fast_rcp(sp * sm);
  plus = fma(np, inv6 * sm, c);
  minus = fma(nm, inv6 * sp, c);
}

// a3, scheme B: MUSCL with the minmod limiter.  Branch-free: the slope is min(|x|,|y|) with the sign
// of x when x and y have the same sign (test on the sign bits, integer pipe) and 0 otherwise —
// the same value as the sign-test definition for all finite inputs (x or y = 0 gives 0).
__device__ __forceinline__ void minmod_pair(double b, double c, double d, double& plus, double& minus) {
  const double x = c - b, y = d - c;
  const double m = fmin(fabs(x), fabs(y));
  const int hx = __double2hiint(x), hy = __double2hiint(y);
  const int hm = ((hx ^ hy) < 0) ? 0 : (__double2hiint(m) | (hx & 0x80000000));
  const int lm = ((hx ^ hy) < 0) ? 0 : __double2loint(m);
  const double s = __hiloint2double(hm, lm);
  plus = fma(0.5, s, c);
  minus = fma(-0.5, s, c);
}

// a4 (G2 Davis bounds; G5 inclusive tie-breaks).  WL/WR = (rho, un, ut1, ut2, p) already
// rotated so that component 1 is the face normal.  F in the same rotated (rho, n, t1, t2, E) order;
// alpha returns the largest signal speed max(|u_n| + c_s) of the two sides.
template <int S>
__device__ __forceinline__ void riemann_flux(const double WL[5], const double WR[5], double gamma, double inv_gm1,
                                             double F[5], double& alpha) {
  // c = sqrt(gamma p / rho) = gamma p * rsqrt(gamma p rho): no division
  const double gpL = gamma * WL[4], gpR = gamma * WR[4];
  const double cL = gpL * fast_rsqrt(gpL * WL[0]);
  const double cR = gpR * fast_rsqrt(gpR * WR[0]);
  const double SL = fmin(WL[1] - cL, WR[1] - cR);
  const double SR = fmax(WL[1] + cL, WR[1] + cR);
  alpha = fmax(SR, -SL);                                 // = max(|u_n| + c_s) over the two sides (Rusanov, NEXT-1)
  if (S == SCHEME_A) {                                   // HLL needs both sides' U and F
    const double EL = WL[4] * inv_gm1 + 0.5 * WL[0] * (WL[1] * WL[1] + (WL[2] * WL[2] + WL[3] * WL[3]));
    const double ER = WR[4] * inv_gm1 + 0.5 * WR[0] * (WR[1] * WR[1] + (WR[2] * WR[2] + WR[3] * WR[3]));
    const double UL[5] = { WL[0], WL[0] * WL[1], WL[0] * WL[2], WL[0] * WL[3], EL };
    const double UR[5] = { WR[0], WR[0] * WR[1], WR[0] * WR[2], WR[0] * WR[3], ER };
    const double FL[5] = { UL[1], UL[1] * WL[1] + WL[4], UL[1] * WL[2], UL[1] * WL[3], (EL + WL[4]) * WL[1] };
    const double FR[5] = { UR[1], UR[1] * WR[1] + WR[4], UR[1] * WR[2], UR[1] * WR[3], (ER + WR[4]) * WR[1] };
    if (SL >= 0.0) {
#pragma unroll
      for (int m = 0; m < 5; ++m) F[m] = FL[m];
      return;
    }
    if (SR <= 0.0) {
#pragma unroll
      for (int m = 0; m < 5; ++m) F[m] = FR[m];
      return;
    }
    const double inv = fast_rcp(SR - SL);
    const double ss = SL * SR;
#pragma unroll
    for (int m = 0; m < 5; ++m) F[m] = ((SR * FL[m] - SL * FR[m]) + ss * (UR[m] - UL[m])) * inv;
  } else {
    // HLLC, averaged-pressure form (G5).  Only the upwind side's U and F enter the result: side L if
    // SL >= 0 or (SR > 0 and S* > 0), else side R; the supersonic cases return that side's F.
    const double A = WL[0] * (SL - WL[1]);
    const double B = WR[0] * (SR - WR[1]);
    const double Ss = ((WR[4] - WL[4]) + (A * WL[1] - B * WR[1])) * fast_rcp(A - B);
    const double pbar = 0.5 * ((WL[4] + WR[4]) + (A * (Ss - WL[1]) + B * (Ss - WR[1])));
    const bool supL = SL >= 0.0, supR = !supL && SR <= 0.0;
    const bool left = supL || (!supR && Ss > 0.0);
    double W[5];
#pragma unroll
    for (int m = 0; m < 5; ++m) W[m] = left ? WL[m] : WR[m];
    const double SK = left ? SL : SR;
    const double E = W[4] * inv_gm1 + 0.5 * W[0] * (W[1] * W[1] + (W[2] * W[2] + W[3] * W[3]));
    const double UK[5] = { W[0], W[0] * W[1], W[0] * W[2], W[0] * W[3], E };
    const double FK[5] = { UK[1], UK[1] * W[1] + W[4], UK[1] * W[2], UK[1] * W[3], (E + W[4]) * W[1] };
    // Branch-free tail: S* = 0 needs no special case here (the formula gives (0, pbar, 0, 0, 0) exactly:
    // every term carries the factor S* except SK pbar / SK), and the supersonic cases select F_K.
    const bool sup = supL || supR;
    const double inv = fast_rcp(SK - Ss);
    const double sp = SK * pbar;
#pragma unroll
    for (int m = 0; m < 5; ++m) {
      double t = Ss * (SK * UK[m] - FK[m]);
      if (m == 1) t += sp;
      if (m == 4) t = fma(sp, Ss, t);
      F[m] = sup ? FK[m] : t * inv;
    }
  }
}

// a7 building block for the fused epilogue: local max wavespeed of one conserved state; returns a
// negative value if the state is not admissible (non-finite, rho <= 0 or p <= 0).
__device__ __forceinline__ double cell_lambda(const double U[5], double gamma, double gm1, const double inv_d[3],
                                              const bool act[3]) {
  double W[5];
  cons_to_prim(U, gm1, W);
  if (!(W[0] > 0.0 && W[4] > 0.0) || !(W[4] < 1.0e300)) return -1.0;
  const double c = sqrt(gamma * W[4] / W[0]);
  double lam = 0.0;
#pragma unroll
  for (int a = 0; a < 3; ++a)
    if (act[a]) lam = fmax(lam, (fabs(W[1 + a]) + c) * inv_d[a]);
  return lam;
}

}  // namespace hard
