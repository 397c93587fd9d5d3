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

// min / max of two finite doubles without the NaN bookkeeping of fmin / fmax (one DSETP + two selects
// instead of DSETP.MIN + select + NaN fix-up + moves); callers pass finite values by construction.
__device__ __forceinline__ double dmin(double a, double b) { return a < b ? a : b; }
__device__ __forceinline__ double dmax(double a, double b) { return a > b ? a : b; }

// 1/x for normal, finite x: MUFU.RCP64H seed y (it reads only the upper 32 bits of x: relative error
// e = 1 - x y below 2^-19) refined with the third-order step y (1 + e + e^2): 3 DFMA, remainder e^3 < 2^-57,
// about 1 ulp; no special-case handling (the IEEE division sequence costs about 10 fp64-pipe
// instructions).  Callers pass quantities that are normal by construction.
__device__ __forceinline__ double fast_rcp(double x) {
  double y;
  asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(x));
  const double e = fma(-x, y, 1.0);
  return fma(y, fma(e, e, e), y);
}

// 1/sqrt(x) for normal, finite x > 0: MUFU.RSQ64H seed y, e = 1 - x y^2 (below 2^-18), third-order step
// y (1 + e/2 + 3 e^2/8): 5 fp64-pipe instructions, remainder 5/16 e^3 < 2^-55, about 1 ulp.
__device__ __forceinline__ double fast_rsqrt(double x) {
  double y;
  asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(x));
  const double e = fma(-x, y * y, 1.0);
  return fma(y * e, fma(0.375, e, 0.5), y);
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
//  * everything in terms of the four differences d1..d4 and their differences s_k (which the betas need anyway);
//  * beta scaled by 12/13 (beta' = s^2 + 3/13 t^2, eps' = 12/13 eps): tau/(beta+eps) is unchanged;
//  * weights d_k (1 + tau/B_k) multiplied through by 10 B0 B1 B2: X_k = (B_k + tau) prod_{j!=k} B_j with the
//    integer multipliers (1, 6, 3), which needs no division; one reciprocal per face normalises.
//    Range: the X are cubic in B, so data up to about 1e51 in magnitude neither overflow nor (B >= 9e-41)
//    underflow.
//  * returned: the increments 6 (plus - c) and 6 (minus - c); the caller adds c back with the factor 1/6 — or
//    with the factor 0 where the positivity fallback (G4) applies, which costs nothing.
__device__ __forceinline__ void wenoz_incr(double a, double b, double c, double d, double e, double& wp, double& wm) {
  const double eps = (12.0 / 13.0) * 1e-40, k3 = 3.0 / 13.0;
  const double d1 = b - a, d2 = c - b, d3 = d - c, d4 = e - d;
  const double s0 = d2 - d1, s1 = d3 - d2, s2 = d4 - d3;
  const double t0 = fma(3.0, d2, -d1), t1 = d2 + d3, t2 = fma(-3.0, d3, d4);
  const double B0 = fma(s0, s0, fma(k3 * t0, t0, eps));
  const double B1 = fma(s1, s1, fma(k3 * t1, t1, eps));
  const double B2 = fma(s2, s2, fma(k3 * t2, t2, eps));
  const double tau = fabs(B0 - B2);
  // X_k = (B_k + tau) prod_{j != k} B_j = P + tau M_k with M_k = prod_{j != k} B_j, P = B0 B1 B2: 4 DMUL + 3 DFMA
  const double M0 = B1 * B2, M1 = B0 * B2, M2 = B0 * B1, P = B0 * M0;
  const double X0 = fma(tau, M0, P), X1 = fma(tau, M1, P), X2 = fma(tau, M2, P);
  // 6 (q_k - c), 6 (p_k - c): the candidates' increments.  Relative to the MIDDLE candidate they are second differences
  // the betas already hold: q0 - q1 = 2 (s0 - s1), q2 - q1 = s1 - s2, p0 - p1 = -2 (s1 - s2), p2 - p1 = -(s0 - s1), so with
  // the weights (X0, 6 X1, 3 X2) of the plus face and (3 X0, 6 X1, X2) of the minus face, e0 = s0 - s1, e2 = s1 - s2:
  //   6 (plus  - c) = q1 + (2 X0 e0 + 3 X2 e2) / (X0 + 6 X1 + 3 X2),
  //   6 (minus - c) = p1 - (3 X0 e0 + 2 X2 e2) / (3 X0 + 6 X1 + X2).
  // Numerators and denominators are taken divided by 3 (the quotients do not change): one DFMA for each numerator on
  // the two shared products, two for each denominator.
  const double q1 = fma(2.0, d3, d2), p1 = -fma(2.0, d2, d3);
  const double A0 = X0 * (s0 - s1), A2 = X2 * (s1 - s2);
  const double np = fma(2.0 / 3.0, A0, A2), nm = fma(2.0 / 3.0, A2, A0);
  const double sp = fma(1.0 / 3.0, X0, fma(2.0, X1, X2)), sm = fma(1.0 / 3.0, X2, fma(2.0, X1, X0));
  wp = fma(np, fast_rcp(sp), q1);
  wm = fma(-nm, fast_rcp(sm), p1);
}

// a3, scheme B: MUSCL with the minmod limiter.  Branch-free: the slope is the argument of smaller
// magnitude when x and y have the same sign (test on the sign bits, integer pipe) and 0 otherwise —
// the same value as the sign-test definition for all finite inputs (x or y = 0 gives 0).  The zero
// case is folded into the factor 1/2 (its high word is selected, the low word is zero either way).
__device__ __forceinline__ void minmod_pair(double b, double c, double d, double& plus, double& minus) {
  const double x = c - b, y = d - c;
  const double s = fabs(x) < fabs(y) ? x : y;
  const int hh = ((__double2hiint(x) ^ __double2hiint(y)) < 0) ? 0 : 0x3fe00000;       // 0.0 or 0.5
  const double h = __hiloint2double(hh, 0);
  plus = fma(h, s, c);
  minus = fma(-h, s, c);
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
  const double SL = dmin(WL[1] - cL, WR[1] - cR);
  const double SR = dmax(WL[1] + cL, WR[1] + cR);
  alpha = dmax(SR, -SL);                                 // = max(|u_n| + c_s) over the two sides (Rusanov, NEXT-1)
  if (S == SCHEME_A) {
    // HLL: F = (SR+ F_L - SL- F_R + SL- SR+ (U_R - U_L)) / (SR+ - SL-) = wl G_L - wr G_R with G_L = F_L - SL- U_L,
    // G_R = F_R - SR+ U_R, wl = SR+ / (SR+ - SL-), wr = SL- / (SR+ - SL-), and SL- = min(SL, 0), SR+ = max(SR, 0):
    // branch-free, F_L when SL >= 0 and F_R when SR <= 0 (G5's inclusive tie-breaks, to rounding); c > 0 keeps
    // SR+ - SL- > 0.  With k = rho (u_n - S): G = (k, k u_n + p, k u_t1, k u_t2, E (u_n - S) + p u_n) — the
    // conserved vector and the physical flux are never formed.
    // energy row: E (u_n - S) + p u_n with E = rho |v|^2 / 2 + p / (gamma - 1)  =  (k / 2) |v|^2 + p ((u_n - S) / (gamma - 1) + u_n).
    // The weights are multiplied into k and p once (a = w k, w p), so that the five rows are short FMA chains on the two
    // sides' primitives: 58 fp64 instructions per face.
    const double SLm = dmin(SL, 0.0), SRp = dmax(SR, 0.0);
    const double dL = WL[1] - SLm, dR = WR[1] - SRp;
    const double inv = fast_rcp(SRp - SLm);
    const double wl = SRp * inv, wr = SLm * inv;
    const double aL = wl * (WL[0] * dL), aR = wr * (WR[0] * dR);
    const double pl = wl * WL[4], pr = wr * WR[4];
    const double v2L = fma(WL[1], WL[1], fma(WL[2], WL[2], WL[3] * WL[3]));
    const double v2R = fma(WR[1], WR[1], fma(WR[2], WR[2], WR[3] * WR[3]));
    const double hL = fma(dL, inv_gm1, WL[1]), hR = fma(dR, inv_gm1, WR[1]);
    F[0] = aL - aR;
    F[1] = fma(aL, WL[1], fma(-aR, WR[1], pl - pr));
    F[2] = fma(aL, WL[2], -aR * WR[2]);
    F[3] = fma(aL, WL[3], -aR * WR[3]);
    F[4] = fma(0.5 * aL, v2L, fma(-0.5 * aR, v2R, fma(pl, hL, -pr * hR)));
  } else {
    // HLLC, averaged-pressure form (G5).  Only the upwind side's U and F enter the result: side L if
    // SL >= 0 or (SR > 0 and S* > 0), else side R; the supersonic cases return that side's F.
    const double A = WL[0] * (SL - WL[1]);
    const double B = WR[0] * (SR - WR[1]);
    const double Ss = ((WR[4] - WL[4]) + fma(A, WL[1], -B * WR[1])) * fast_rcp(A - B);
    const double pbar = 0.5 * ((WL[4] + WR[4]) + fma(A, Ss - WL[1], B * (Ss - WR[1])));
    // S* lies strictly between SL and SR, so SL >= 0 implies S* > 0 and SR <= 0 implies S* < 0: "left" covers the
    // supersonic cases too.  With G = F_K - S U_K = (k, k u_n + p, k u_t1, k u_t2, (k/2)|v|^2 + p ((u_n - S)/(gamma-1) + u_n)),
    // k = rho (u_n - S) (neither U_K nor F_K is formed), the star flux F_K + S_K (U*_K - U_K) with
    // U*_K = (pbar D* - G) / (S_K - S*), D* = (0, 1, 0, 0, S*), is (1 - g) G + g pbar D*, g = S_K / (S_K - S*).
    // S clamped to zero on the supersonic side makes G = F_K and g = 0: no branch, no select on the result.
    // h = 1 - g = -S* / (S_K - S*) is formed directly and g as 1 - h, so that a stationary contact (S* = +-0) gives
    // h = 0 and g = 1 EXACTLY and the flux is (0, pbar, 0, 0, 0) to the last bit, as in the oracle's tie-break (G5).
    const bool left = Ss > 0.0;
    double W[5];
#pragma unroll
    for (int m = 0; m < 5; ++m) W[m] = left ? WL[m] : WR[m];
    const double SK = left ? SL : SR;
    const bool sub = left ? (SK < 0.0) : (SK > 0.0);
    const double SKc = sub ? SK : 0.0;
    const double d = W[1] - SKc, k = W[0] * d;
    const double v2 = fma(W[1], W[1], fma(W[2], W[2], W[3] * W[3]));
    const double G4 = fma(0.5 * k, v2, W[4] * fma(d, inv_gm1, W[1]));
    const double h = sub ? -Ss * fast_rcp(SK - Ss) : 1.0, g = 1.0 - h, gp = g * pbar;
    F[0] = h * k;
    F[1] = fma(h, fma(k, W[1], W[4]), gp);
    F[2] = h * (k * W[2]);
    F[3] = h * (k * W[3]);
    F[4] = fma(h, G4, gp * Ss);
  }
}

// a7 building block for the fused epilogue: local max wavespeed of one conserved state; returns a
// negative value if the state is not admissible (non-finite, rho <= 0 or p <= 0).  The next step's dt
// inherits the state's rounding differences anyway (G9: compared at 1e-9), so this uses the fast
// reciprocal / rsqrt forms; the standalone cfl_kernel keeps the correctly rounded definition.
__device__ __forceinline__ double cell_lambda(const double U[5], double gamma, double gm1, const double inv_d[3],
                                              const bool act[3]) {
  double W[5];
  cons_to_prim(U, gm1, W);
  if (!(W[0] > 0.0 && W[4] > 0.0) || !(W[4] < 1.0e300)) return -1.0;
  const double gp = gamma * W[4];
  const double c = gp * fast_rsqrt(gp * W[0]);
  double lam = 0.0;
#pragma unroll
  for (int a = 0; a < 3; ++a)
    if (act[a]) lam = dmax(lam, (fabs(W[1 + a]) + c) * inv_d[a]);
  return lam;
}

}  // namespace hard
