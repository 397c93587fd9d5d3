// ORACLE — TEST INFRASTRUCTURE, NOT THE PRODUCT.
//
// Plain, slow, single-threaded fp64 C++ restatement of the explicit finite-volume update of the
// compressible Euler equations that PAPER.md describes (arxiv 2509.08971, "HARD"), written from the
// paper before any CUDA kernel and sharing no code with paper_2509_08971_b200/csrc.
// Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may load
// it.  Build:  g++ -O2 -std=c++17 -ffp-contract=off -fPIC -shared   (no fast-math, no -march=native:
// every operation is a correctly rounded IEEE double operation in the order written here, which is
// what makes the mirror / axis-permutation invariants hold bit for bit).
//
// What follows which passage (P:NNN = /root/reference/PAPER.md line; Gn = DESIGN.md reading n):
//   evolved variables U = [rho, rho v^i, e + rho v^2/2]           P:93  eq.2 (hydro rows; S = 0)
//   fluxes F^j = [rho v^j, rho v^i v^j + p delta_ij, (E+p) v^j]   P:97  eq.3
//   ideal-gas closure p = (gamma-1) e, c_s = sqrt(gamma p / rho)
//   uniform Cartesian mesh, cell-centred variables
//   flux-difference form (F*_{i+1/2} - F*_{i-1/2}) / dx           P:149 eq.15
//   WENO5-Z reconstruction "for all variables" + HLL flux         P:151            (scheme 0, "A")
//   MUSCL-minmod + HLLC                                           BASELINE.json north_star fallback
//                                                                                  (scheme 1, "B")
//   Heun's method, tableau 0 | 1 1 | 1/2 1/2                      P:151-160 Table 2
//   dt from the CFL condition                                     P:215, P:255     (formula: G6)
//   ghost entities of the N-array topology                        P:64             (BCs: G10, G17)
//   radiation energy density advected with the fluid, Rusanov    P:93 eq.2 (4th row), eq.14 LHS,
//   (local Lax-Friedrichs) flux                                   P:151            (NEXT-1; G19)
//   radiative heating q = c kappa rho (E_rad - a T^4), operator   P:66, eq.4,6
//   split after the advection step, backward Euler, root by bisection             (NEXT-3; G20)
// Every place where the paper is silent is a DESIGN.md reading (G1..G13) and is marked below.
//
// Pins (tests/test_oracle_*.py, all -m "not gpu"): exact Sod / LeBlanc Riemann solutions and L1
// convergence, the paper's printed Sod bound, Sedov-Taylor shock radius, acoustic-wave
// order, conservation to 1e-13, exact uniform-state preservation, bit-for-bit mirror
// and axis-permutation symmetry, 1-D == replicated 3-D pencil, polynomial exactness of the WENO
// candidate stencils, flux consistency F*(W,W) = F(W), stationary contact under HLLC, a whole-array
// restatement of a full step, and (tests/test_oracle_pins_r2.py, each failing under the matching mutation
// of this file): wenoz against WENO5-Z rebuilt from its integral definition with numpy.polynomial;
// outflow ghosts against the scalar upwind scheme that uniform-(u,p) flow reduces to; the G4 fallback
// against textbook HLL fluxes of cell averages read off L(U) by telescoping; and
// (tests/test_oracle_eps_pin.py, round 3) the WENO-Z eps through the closed-form value eps/(18 s) on a one-cell spike,
// degree-1 homogeneity down to data of 1e-12 and the linear-weight limit below eps.  No function here is
// "parity unpinned" under the mutation sweeps run so far (DESIGN.md sections 2-3).

#include <algorithm>
#include <cmath>
#include <cstddef>
#include <cstdlib>
#include <cstring>
#include <vector>

namespace {

enum { ORC_OK = 0, ORC_ERR_ARG = -1, ORC_ERR_NOSTATE = -4, ORC_ERR_NONPHYSICAL = -5 };
enum { BC_PERIODIC = 0, BC_OUTFLOW = 1, BC_REFLECT = 2 };
enum { SCHEME_A = 0, SCHEME_B = 1 };

// G8: permutation-symmetric, sign-odd three-term sum.  Order by magnitude, add the two smallest
// first; if the two largest cancel exactly, the result is the smallest term.
double sum3sym(double a, double b, double c) {
  double x1 = a, x2 = b, x3 = c, t;
  if (std::fabs(x1) > std::fabs(x2)) { t = x1; x1 = x2; x2 = t; }
  if (std::fabs(x2) > std::fabs(x3)) { t = x2; x2 = x3; x3 = t; }
  if (std::fabs(x1) > std::fabs(x2)) { t = x1; x1 = x2; x2 = t; }
  if (x2 == -x3) return x1;
  return (x1 + x2) + x3;
}

struct Prim { double rho, v[3], p; };          // primitive state (rho, u, v, w, p)        G3
struct Cons { double q[6]; };                  // (rho, mx, my, mz, E [, E_rad])

// a2: conserved -> primitive with the ideal-gas EOS.
Prim cons_to_prim(const double U[5], double gamma) {
  Prim W;
  W.rho = U[0];
  W.v[0] = U[1] / U[0];
  W.v[1] = U[2] / U[0];
  W.v[2] = U[3] / U[0];
  double ke2 = sum3sym(U[1] * W.v[0], U[2] * W.v[1], U[3] * W.v[2]);
  W.p = (gamma - 1.0) * (U[4] - 0.5 * ke2);
  return W;
}

// WENO5-Z of Borges et al. (ref. [18]); value at the i+1/2 face from cell averages
// (a,b,c,d,e) = q[i-2..i+2].  G1: eps = 1e-40, power 1, linear weights (1/10, 6/10, 3/10),
// Jiang-Shu smoothness indicators.
double wenoz(double a, double b, double c, double d, double e) {
  const double eps = 1e-40;
  double s0 = (a - 2.0 * b) + c, t0 = (a - 4.0 * b) + 3.0 * c;
  double s1 = (b - 2.0 * c) + d, t1 = b - d;
  double s2 = (c - 2.0 * d) + e, t2 = (3.0 * c - 4.0 * d) + e;
  double b0 = (13.0 / 12.0) * (s0 * s0) + 0.25 * (t0 * t0);
  double b1 = (13.0 / 12.0) * (s1 * s1) + 0.25 * (t1 * t1);
  double b2 = (13.0 / 12.0) * (s2 * s2) + 0.25 * (t2 * t2);
  double tau = std::fabs(b0 - b2);
  double al0 = 0.1 * (1.0 + tau / (b0 + eps));
  double al1 = 0.6 * (1.0 + tau / (b1 + eps));
  double al2 = 0.3 * (1.0 + tau / (b2 + eps));
  double q0 = ((2.0 * a - 7.0 * b) + 11.0 * c) / 6.0;
  double q1 = ((-b + 5.0 * c) + 2.0 * d) / 6.0;
  double q2 = ((2.0 * c + 5.0 * d) - e) / 6.0;
  return ((al0 * q0 + al1 * q1) + al2 * q2) / ((al0 + al1) + al2);
}

// MUSCL slope with the minmod limiter (north_star fallback scheme); sign tests, no product.
double minmod(double a, double b) {
  if (a > 0.0 && b > 0.0) return a < b ? a : b;
  if (a < 0.0 && b < 0.0) return a > b ? a : b;
  return 0.0;
}

// a3: face values of one variable in one cell: plus at i+1/2, minus at i-1/2, from the 5-point
// window w[0..4] = q[i-2..i+2] (scheme B only uses w[1..3]).
void reconstruct(int scheme, const double w[5], double* plus, double* minus) {
  if (scheme == SCHEME_A) {
    *plus = wenoz(w[0], w[1], w[2], w[3], w[4]);
    *minus = wenoz(w[4], w[3], w[2], w[1], w[0]);      // the same function on the mirrored stencil
  } else {
    double s = minmod(w[2] - w[1], w[3] - w[2]);
    *plus = w[2] + 0.5 * s;
    *minus = w[2] - 0.5 * s;
  }
}

// a4: approximate Riemann flux through a face with normal along `dir`; WL/WR are the primitive
// states left/right of the face.  Davis wave-speed bounds (G2); inclusive tie-breaks (G5).
// F is returned in (rho, mx, my, mz, E) order.
void riemann(int scheme, const Prim& WL, const Prim& WR, int dir, double gamma, double F[5]) {
  const int n = dir, t1 = (dir + 1) % 3, t2 = (dir + 2) % 3;
  const Prim* W[2] = { &WL, &WR };
  double un[2], c[2], UK[2][5], FK[2][5];      // per side, in (rho, n, t1, t2, E) order
  for (int K = 0; K < 2; ++K) {
    const Prim& w = *W[K];
    un[K] = w.v[n];
    c[K] = std::sqrt(gamma * w.p / w.rho);
    double E = w.p / (gamma - 1.0) + 0.5 * w.rho * (un[K] * un[K] + (w.v[t1] * w.v[t1] + w.v[t2] * w.v[t2]));
    UK[K][0] = w.rho;
    UK[K][1] = w.rho * un[K];
    UK[K][2] = w.rho * w.v[t1];
    UK[K][3] = w.rho * w.v[t2];
    UK[K][4] = E;
    FK[K][0] = w.rho * un[K];
    FK[K][1] = w.rho * un[K] * un[K] + w.p;
    FK[K][2] = w.rho * un[K] * w.v[t1];
    FK[K][3] = w.rho * un[K] * w.v[t2];
    FK[K][4] = (E + w.p) * un[K];
  }
  double SL = std::fmin(un[0] - c[0], un[1] - c[1]);
  double SR = std::fmax(un[0] + c[0], un[1] + c[1]);
  double Fl[5];                                  // local (rho, n, t1, t2, E) order
  if (SL >= 0.0) {
    for (int m = 0; m < 5; ++m) Fl[m] = FK[0][m];
  } else if (SR <= 0.0) {
    for (int m = 0; m < 5; ++m) Fl[m] = FK[1][m];
  } else if (scheme == SCHEME_A) {               // HLL (ref. [19])
    for (int m = 0; m < 5; ++m)
      Fl[m] = ((SR * FK[0][m] - SL * FK[1][m]) + SL * SR * (UK[1][m] - UK[0][m])) / (SR - SL);
  } else {                                       // HLLC, Toro's averaged-pressure form (G5)
    double A = WL.rho * (SL - un[0]);
    double B = WR.rho * (SR - un[1]);
    double Ss = ((WR.p - WL.p) + (A * un[0] - B * un[1])) / (A - B);
    double pbar = 0.5 * ((WL.p + WR.p) + (A * (Ss - un[0]) + B * (Ss - un[1])));
    if (Ss == 0.0) {
      Fl[0] = 0.0; Fl[1] = pbar; Fl[2] = 0.0; Fl[3] = 0.0; Fl[4] = 0.0;
    } else {
      int K = (Ss > 0.0) ? 0 : 1;
      double SK = (K == 0) ? SL : SR;
      const double D[5] = { 0.0, 1.0, 0.0, 0.0, Ss };
      for (int m = 0; m < 5; ++m)
        Fl[m] = (Ss * (SK * UK[K][m] - FK[K][m]) + SK * pbar * D[m]) / (SK - Ss);
    }
  }
  F[0] = Fl[0];
  F[1 + n] = Fl[1];
  F[1 + t1] = Fl[2];
  F[1 + t2] = Fl[3];
  F[4] = Fl[4];
}

// NEXT-1 (G19): local Lax-Friedrichs (Rusanov) flux of the advected radiation energy density
// (advection part of P:141 eq.14: d_t E + d_j(E v^j) = 0).  EL/ER and the primitive states are
// the reconstructed face values; alpha = max(|u_n| + c_s) over the two sides.
double rusanov(double EL, double ER, const Prim& WL, const Prim& WR, int dir, double gamma) {
  double unL = WL.v[dir], unR = WR.v[dir];
  double cL = std::sqrt(gamma * WL.p / WL.rho), cR = std::sqrt(gamma * WR.p / WR.rho);
  double alpha = std::fmax(std::fabs(unL) + cL, std::fabs(unR) + cR);
  return 0.5 * (EL * unL + ER * unR) - 0.5 * alpha * (ER - EL);
}

struct Ctx {
  int n[3];                 // interior cells per direction
  int gh[3];                // ghost width per direction (g if n>1, else 0: G11)
  long P[3];                // padded extents
  int g;                    // 3 for scheme A, 2 for scheme B
  int scheme, bc;
  double gamma, d[3];
  int nf;                   // 5, or 6 with the advected radiation energy density (NEXT-1)
  std::vector<double> U[6], U1[6];
  int src_on;               // NEXT-3: radiative heating/cooling source after each advection step
  double src_kappa, src_c, src_a, src_cv;
  double lambda, t;
  long long steps;
  long long fallbacks;      // G4 positivity fallbacks taken so far
  int have_state, status, check;
  bool active(int a) const { return n[a] > 1; }
  long idx(int i, int j, int k) const {          // interior coordinates; ghosts are negative / >= n
    return (long)(i + gh[0]) + P[0] * ((long)(j + gh[1]) + P[1] * (long)(k + gh[2]));
  }
  long ncell() const { return (long)n[0] * n[1] * n[2]; }
};

void layout(Ctx* c) {
  c->g = (c->scheme == SCHEME_A) ? 3 : 2;
  for (int a = 0; a < 3; ++a) {
    c->gh[a] = c->active(a) ? c->g : 0;
    c->P[a] = c->n[a] + 2 * c->gh[a];
  }
  size_t tot = (size_t)c->P[0] * c->P[1] * c->P[2];
  for (int f = 0; f < 6; ++f) { c->U[f].assign(f < c->nf ? tot : 0, 0.0); c->U1[f].assign(f < c->nf ? tot : 0, 0.0); }
  c->have_state = 0;
}

// a1: ghost-cell fill (P:64 ghost entities; G10).  Faces only: the stencils are one-dimensional.
void fill_ghosts(const Ctx* c, std::vector<double> V[6]) {
  for (int a = 0; a < 3; ++a) {
    if (!c->active(a)) continue;
    const int b1 = (a + 1) % 3, b2 = (a + 2) % 3;
    int ijk[3];
    for (int f = 0; f < c->nf; ++f)
      for (int q2 = 0; q2 < c->n[b2]; ++q2)
        for (int q1 = 0; q1 < c->n[b1]; ++q1)
          for (int m = 1; m <= c->g; ++m) {
            ijk[b1] = q1; ijk[b2] = q2;
            int lo_src, hi_src;
            if (c->bc == BC_PERIODIC)     { lo_src = c->n[a] - m; hi_src = m - 1; }
            else if (c->bc == BC_REFLECT) { lo_src = m - 1;       hi_src = c->n[a] - m; }   // mirror image (G17)
            else                          { lo_src = 0;           hi_src = c->n[a] - 1; }
            ijk[a] = lo_src;  long s_lo = c->idx(ijk[0], ijk[1], ijk[2]);
            ijk[a] = -m;      long d_lo = c->idx(ijk[0], ijk[1], ijk[2]);
            ijk[a] = hi_src;  long s_hi = c->idx(ijk[0], ijk[1], ijk[2]);
            ijk[a] = c->n[a] - 1 + m; long d_hi = c->idx(ijk[0], ijk[1], ijk[2]);
            // reflecting wall: the ghost state is the mirror image, i.e. the normal momentum changes sign
            const double sgn = (c->bc == BC_REFLECT && f == 1 + a) ? -1.0 : 1.0;
            V[f][d_lo] = sgn * V[f][s_lo];
            V[f][d_hi] = sgn * V[f][s_hi];
          }
  }
}

// a7: max wavespeed over interior cells (G6).  Returns lambda; flags non-physical cells.
double maxwavespeed(Ctx* c, const std::vector<double> V[6]) {
  double lam = 0.0;
  for (int k = 0; k < c->n[2]; ++k)
    for (int j = 0; j < c->n[1]; ++j)
      for (int i = 0; i < c->n[0]; ++i) {
        long p = c->idx(i, j, k);
        double u5[5] = { V[0][p], V[1][p], V[2][p], V[3][p], V[4][p] };
        Prim W = cons_to_prim(u5, c->gamma);
        if (!(W.rho > 0.0 && W.p > 0.0)) { c->status = ORC_ERR_NONPHYSICAL; continue; }
        double cs = std::sqrt(c->gamma * W.p / W.rho);
        for (int a = 0; a < 3; ++a) {
          if (!c->active(a)) continue;
          double l = (std::fabs(W.v[a]) + cs) / c->d[a];
          if (l > lam) lam = l;
        }
      }
  return lam;
}

// L(U) (eq.15): dF[a][f][cell] = (F*_{+1/2} - F*_{-1/2}) / Delta_a, per direction, then
// L = -sum3sym over directions.  Lout[f] is indexed over interior cells i + nx (j + ny k).
void rhs(Ctx* c, const std::vector<double> V[6], std::vector<double> Lout[6]) {
  const long N = c->ncell();
  const int nf = c->nf;
  std::vector<double> dF[3][6];
  for (int a = 0; a < 3; ++a)
    for (int f = 0; f < nf; ++f) dF[a][f].assign(N, 0.0);
  const int r = c->g - 1;                                    // reconstruction stencil radius
  for (int a = 0; a < 3; ++a) {
    if (!c->active(a)) continue;
    const int b1 = (a + 1) % 3, b2 = (a + 2) % 3;
    const int na = c->n[a], g = c->g;
    std::vector<Prim> W(na + 2 * g), Wp(na + 2 * g), Wm(na + 2 * g);   // index s = i + g
    std::vector<double> Er(na + 2 * g), Erp(na + 2 * g), Erm(na + 2 * g);  // radiation energy density (nf = 6)
    std::vector<Cons> Fs(na + 1);                                      // face i+1/2 at slot i+1
    int ijk[3];
    for (int q2 = 0; q2 < c->n[b2]; ++q2)
      for (int q1 = 0; q1 < c->n[b1]; ++q1) {
        ijk[b1] = q1; ijk[b2] = q2;
        for (int i = -g; i < na + g; ++i) {                            // a2
          ijk[a] = i;
          long p = c->idx(ijk[0], ijk[1], ijk[2]);
          double u5[5] = { V[0][p], V[1][p], V[2][p], V[3][p], V[4][p] };
          W[i + g] = cons_to_prim(u5, c->gamma);
          if (nf == 6) Er[i + g] = V[5][p];
        }
        for (int i = -1; i <= na; ++i) {                               // a3
          double w[5], pl[5], mi[5];
          for (int v = 0; v < 5; ++v) {
            for (int s = -2; s <= 2; ++s) {
              int ii = i + s;
              if (s < -r || s > r) { w[s + 2] = 0.0; continue; }       // not read by scheme B
              const Prim& q = W[ii + g];
              w[s + 2] = (v == 0) ? q.rho : (v == 4) ? q.p : q.v[v - 1];
            }
            reconstruct(c->scheme, w, &pl[v], &mi[v]);
          }
          double epl = 0.0, emi = 0.0;
          if (nf == 6) {                                               // "WENO5-Z for all variables"
            for (int s = -2; s <= 2; ++s) w[s + 2] = (s < -r || s > r) ? 0.0 : Er[i + s + g];
            reconstruct(c->scheme, w, &epl, &emi);
          }
          if (c->scheme == SCHEME_A && (pl[0] <= 0.0 || pl[4] <= 0.0 || mi[0] <= 0.0 || mi[4] <= 0.0)) {
            const Prim& q = W[i + g];                                  // G4: piecewise constant
            pl[0] = mi[0] = q.rho; pl[4] = mi[4] = q.p;
            for (int m = 0; m < 3; ++m) pl[1 + m] = mi[1 + m] = q.v[m];
            if (nf == 6) epl = emi = Er[i + g];                        // G19: the fallback takes E_rad along
            c->fallbacks++;
          }
          Erp[i + g] = epl; Erm[i + g] = emi;
          Prim& P = Wp[i + g]; Prim& M = Wm[i + g];
          P.rho = pl[0]; P.p = pl[4]; M.rho = mi[0]; M.p = mi[4];
          for (int m = 0; m < 3; ++m) { P.v[m] = pl[1 + m]; M.v[m] = mi[1 + m]; }
        }
        for (int i = -1; i < na; ++i) {                                // a4: face between i, i+1
          riemann(c->scheme, Wp[i + g], Wm[i + 1 + g], a, c->gamma, Fs[i + 1].q);
          if (nf == 6) Fs[i + 1].q[5] = rusanov(Erp[i + g], Erm[i + 1 + g], Wp[i + g], Wm[i + 1 + g], a, c->gamma);
        }
        for (int i = 0; i < na; ++i) {                                 // a5
          ijk[a] = i;
          long cell = (long)ijk[0] + (long)c->n[0] * ((long)ijk[1] + (long)c->n[1] * ijk[2]);
          for (int f = 0; f < nf; ++f) dF[a][f][cell] = (Fs[i + 1].q[f] - Fs[i].q[f]) / c->d[a];
        }
      }
  }
  for (int f = 0; f < nf; ++f) {
    Lout[f].resize(N);
    for (long p = 0; p < N; ++p) Lout[f][p] = -sum3sym(dF[0][f][p], dF[1][f][p], dF[2][f][p]);
  }
}

// NEXT-3 (G20): the pointwise source update of the paper's operator split ("advection, diffusion, source
// updates") restricted to the heating rate q = c kappa rho (E_rad - a T^4) (eq.6; force and
// diffusion out of scope): d_t e = q, d_t E_rad = -q (eq.4), T = e / (rho c_v) (ideal gas).  Backward
// Euler over dt conserves e + E_rad exactly: the new internal energy density x is the root of
//   g(x) = x - e - dt c kappa rho (E_tot - x - a (x/(rho c_v))^4)
// on [0, E_tot], where g is increasing with g(0) <= 0 <= g(E_tot).  The oracle finds it the plainest way:
// bisection until the bracket is two adjacent doubles (no Newton step, no tolerance), then the end with the
// smaller |g|.  How the CUDA path iterates is its own business; parity compares the root.
void apply_source(Ctx* c, double dt) {
  for (int k = 0; k < c->n[2]; ++k)
    for (int j = 0; j < c->n[1]; ++j)
      for (int i = 0; i < c->n[0]; ++i) {
        long p = c->idx(i, j, k);
        double rho = c->U[0][p];
        double ke = 0.5 * sum3sym(c->U[1][p] * c->U[1][p], c->U[2][p] * c->U[2][p], c->U[3][p] * c->U[3][p]) / rho;
        double e = c->U[4][p] - ke, Er = c->U[5][p];
        double Etot = e + Er;
        double beta = dt * c->src_c * c->src_kappa * rho;
        double rcv = rho * c->src_cv;
        auto g = [&](double x) {
          double T = x / rcv, T2 = T * T;
          return (x - e) - beta * ((Etot - x) - c->src_a * (T2 * T2));
        };
        double lo = 0.0, hi = Etot;
        for (int it = 0; it < 4000; ++it) {                      // 1075 halvings reach any double from [0, hi]
          double mid = lo + 0.5 * (hi - lo);
          if (!(mid > lo && mid < hi)) break;                    // lo and hi are adjacent doubles
          if (g(mid) > 0.0) hi = mid; else lo = mid;
        }
        double x = (std::fabs(g(lo)) <= std::fabs(g(hi))) ? lo : hi;
        c->U[4][p] = x + ke;
        c->U[5][p] = Etot - x;
      }
}

// One Heun / SSP-RK2 step with a given dt (Table 2; Shu-Osher form, G7).
void step_dt(Ctx* c, double dt) {
  std::vector<double> L[6];
  fill_ghosts(c, c->U);
  rhs(c, c->U, L);
  for (int k = 0; k < c->n[2]; ++k)
    for (int j = 0; j < c->n[1]; ++j)
      for (int i = 0; i < c->n[0]; ++i) {
        long p = c->idx(i, j, k), q = (long)i + (long)c->n[0] * ((long)j + (long)c->n[1] * k);
        for (int f = 0; f < c->nf; ++f) c->U1[f][p] = c->U[f][p] + dt * L[f][q];
      }
  fill_ghosts(c, c->U1);
  rhs(c, c->U1, L);
  for (int k = 0; k < c->n[2]; ++k)
    for (int j = 0; j < c->n[1]; ++j)
      for (int i = 0; i < c->n[0]; ++i) {
        long p = c->idx(i, j, k), q = (long)i + (long)c->n[0] * ((long)j + (long)c->n[1] * k);
        for (int f = 0; f < c->nf; ++f)
          c->U[f][p] = 0.5 * c->U[f][p] + 0.5 * (c->U1[f][p] + dt * L[f][q]);
      }
  if (c->src_on) apply_source(c, dt);
  if (c->check) c->lambda = maxwavespeed(c, c->U);
  c->t += dt;
  c->steps += 1;
}

}  // namespace

extern "C" {

void* oracle_create(int nx, int ny, int nz, double gamma, int bc) {
  if (nx < 1 || ny < 1 || nz < 1 || !(gamma > 1.0) || (bc != BC_PERIODIC && bc != BC_OUTFLOW && bc != BC_REFLECT)) return nullptr;
  Ctx* c = new Ctx();
  c->n[0] = nx; c->n[1] = ny; c->n[2] = nz;
  c->gamma = gamma; c->bc = bc; c->scheme = SCHEME_A; c->nf = 5; c->src_on = 0;
  c->d[0] = 1.0 / nx; c->d[1] = 1.0 / ny; c->d[2] = 1.0 / nz;
  c->lambda = 0.0; c->t = 0.0; c->steps = 0; c->fallbacks = 0;
  c->status = ORC_OK; c->check = 1;
  for (int a = 0; a < 3; ++a) if (c->active(a) && c->n[a] < 3) { delete c; return nullptr; }
  layout(c);
  return c;
}

int oracle_destroy(void* h) { delete (Ctx*)h; return ORC_OK; }

int oracle_set_spacing(void* h, double dx, double dy, double dz) {
  Ctx* c = (Ctx*)h;
  if (!c || !(dx > 0.0 && dy > 0.0 && dz > 0.0)) return ORC_ERR_ARG;
  c->d[0] = dx; c->d[1] = dy; c->d[2] = dz;
  if (c->have_state && c->check) c->lambda = maxwavespeed(c, c->U);
  return ORC_OK;
}

// NEXT-1: switch the advected radiation energy density on (6 fields); only before oracle_set_state.
int oracle_enable_radiation(void* h) {
  Ctx* c = (Ctx*)h;
  if (!c || c->have_state) return ORC_ERR_ARG;
  c->nf = 6;
  layout(c);
  return ORC_OK;
}

// Interior copy of E_rad, layout as the other fields; after oracle_set_state (which zeroes E_rad).
int oracle_set_rad_energy(void* h, const double* er) {
  Ctx* c = (Ctx*)h;
  if (!c || !er || c->nf != 6) return ORC_ERR_ARG;
  if (!c->have_state) return ORC_ERR_NOSTATE;
  for (int k = 0; k < c->n[2]; ++k)
    for (int j = 0; j < c->n[1]; ++j)
      for (int i = 0; i < c->n[0]; ++i)
        c->U[5][c->idx(i, j, k)] = er[(long)i + (long)c->n[0] * ((long)j + (long)c->n[1] * k)];
  return ORC_OK;
}

int oracle_get_rad_energy(void* h, double* er) {
  Ctx* c = (Ctx*)h;
  if (!c || !er || c->nf != 6) return ORC_ERR_ARG;
  if (!c->have_state) return ORC_ERR_NOSTATE;
  for (int k = 0; k < c->n[2]; ++k)
    for (int j = 0; j < c->n[1]; ++j)
      for (int i = 0; i < c->n[0]; ++i)
        er[(long)i + (long)c->n[0] * ((long)j + (long)c->n[1] * k)] = c->U[5][c->idx(i, j, k)];
  return c->status;
}

// NEXT-3: heating/cooling source after every step; needs oracle_enable_radiation.  cv: T = e / (rho cv).
int oracle_set_source(void* h, double kappa, double c_light, double a_rad, double cv) {
  Ctx* c = (Ctx*)h;
  if (!c || c->nf != 6 || !(kappa >= 0.0 && c_light > 0.0 && a_rad > 0.0 && cv > 0.0)) return ORC_ERR_ARG;
  c->src_on = 1; c->src_kappa = kappa; c->src_c = c_light; c->src_a = a_rad; c->src_cv = cv;
  return ORC_OK;
}

int oracle_set_scheme(void* h, int scheme) {
  Ctx* c = (Ctx*)h;
  if (!c || (scheme != SCHEME_A && scheme != SCHEME_B) || c->have_state) return ORC_ERR_ARG;
  c->scheme = scheme;
  layout(c);
  return ORC_OK;
}

// check = 0: light-cone sub-box mode: no non-physical
// test and no lambda; only step_dt is allowed.
int oracle_set_check(void* h, int on) {
  Ctx* c = (Ctx*)h;
  if (!c) return ORC_ERR_ARG;
  c->check = on ? 1 : 0;
  return ORC_OK;
}

int oracle_set_state(void* h, const double* rho, const double* mx, const double* my, const double* mz,
                     const double* E) {
  Ctx* c = (Ctx*)h;
  if (!c || !rho || !mx || !my || !mz || !E) return ORC_ERR_ARG;
  const double* src[5] = { rho, mx, my, mz, E };
  for (int f = 0; f < 5; ++f)
    for (int k = 0; k < c->n[2]; ++k)
      for (int j = 0; j < c->n[1]; ++j)
        for (int i = 0; i < c->n[0]; ++i)
          c->U[f][c->idx(i, j, k)] = src[f][(long)i + (long)c->n[0] * ((long)j + (long)c->n[1] * k)];
  if (c->nf == 6) std::fill(c->U[5].begin(), c->U[5].end(), 0.0);
  c->have_state = 1;
  c->status = ORC_OK;
  c->t = 0.0; c->steps = 0; c->fallbacks = 0;
  if (c->check) c->lambda = maxwavespeed(c, c->U);
  return c->status;
}

int oracle_get_state(void* h, double* rho, double* mx, double* my, double* mz, double* E) {
  Ctx* c = (Ctx*)h;
  if (!c || !rho || !mx || !my || !mz || !E) return ORC_ERR_ARG;
  if (!c->have_state) return ORC_ERR_NOSTATE;
  double* dst[5] = { rho, mx, my, mz, E };
  for (int f = 0; f < 5; ++f)
    for (int k = 0; k < c->n[2]; ++k)
      for (int j = 0; j < c->n[1]; ++j)
        for (int i = 0; i < c->n[0]; ++i)
          dst[f][(long)i + (long)c->n[0] * ((long)j + (long)c->n[1] * k)] = c->U[f][c->idx(i, j, k)];
  return c->status;
}

int oracle_step(void* h, double cfl, int nsteps) {     // dt_n = cfl / lambda(U^n), every step (G6, G7)
  Ctx* c = (Ctx*)h;
  if (!c || !(cfl > 0.0) || nsteps < 0 || !c->check) return ORC_ERR_ARG;
  if (!c->have_state) return ORC_ERR_NOSTATE;
  for (int s = 0; s < nsteps; ++s) {
    if (c->status != ORC_OK) return c->status;
    step_dt(c, cfl / c->lambda);
  }
  return c->status;
}

int oracle_step_dt(void* h, double dt, int nsteps) {
  Ctx* c = (Ctx*)h;
  if (!c || !(dt > 0.0) || nsteps < 0) return ORC_ERR_ARG;
  if (!c->have_state) return ORC_ERR_NOSTATE;
  for (int s = 0; s < nsteps; ++s) {
    if (c->status != ORC_OK) return c->status;
    step_dt(c, dt);
  }
  return c->status;
}

int oracle_max_dt(void* h, double* dt_out) {           // 1 / lambda_max of the current state
  Ctx* c = (Ctx*)h;
  if (!c || !dt_out || !c->check) return ORC_ERR_ARG;
  if (!c->have_state) return ORC_ERR_NOSTATE;
  *dt_out = 1.0 / c->lambda;
  return c->status;
}

int oracle_get_time(void* h, double* t, long long* steps_done) {
  Ctx* c = (Ctx*)h;
  if (!c) return ORC_ERR_ARG;
  if (t) *t = c->t;
  if (steps_done) *steps_done = c->steps;
  return ORC_OK;
}

long long oracle_fallback_count(void* h) { return h ? ((Ctx*)h)->fallbacks : -1; }

// L(U) of the current state (eq.15), ghosts filled first; out holds nf arrays of nx*ny*nz doubles,
// field-major.  Observability for the pins (tests read single face fluxes off it by telescoping).
int oracle_rhs(void* h, double* out) {
  Ctx* c = (Ctx*)h;
  if (!c || !out) return ORC_ERR_ARG;
  if (!c->have_state) return ORC_ERR_NOSTATE;
  std::vector<double> L[6];
  fill_ghosts(c, c->U);
  rhs(c, c->U, L);
  for (int f = 0; f < c->nf; ++f) std::copy(L[f].begin(), L[f].end(), out + (size_t)f * c->ncell());
  return ORC_OK;
}

// Building blocks exposed so that tests can pin them one by one.
double oracle_sum3sym(double a, double b, double c) { return sum3sym(a, b, c); }
double oracle_wenoz(double a, double b, double c, double d, double e) { return wenoz(a, b, c, d, e); }
double oracle_minmod(double a, double b) { return minmod(a, b); }
void oracle_cons_to_prim(const double U[5], double gamma, double W[5]) {
  Prim p = cons_to_prim(U, gamma);
  W[0] = p.rho; W[1] = p.v[0]; W[2] = p.v[1]; W[3] = p.v[2]; W[4] = p.p;
}
// WL, WR = (rho, u, v, w, p); F = (rho, mx, my, mz, E) flux through a face with normal `dir`.
void oracle_riemann(int scheme, const double WL[5], const double WR[5], int dir, double gamma, double F[5]) {
  Prim L, R;
  L.rho = WL[0]; L.v[0] = WL[1]; L.v[1] = WL[2]; L.v[2] = WL[3]; L.p = WL[4];
  R.rho = WR[0]; R.v[0] = WR[1]; R.v[1] = WR[2]; R.v[2] = WR[3]; R.p = WR[4];
  riemann(scheme, L, R, dir, gamma, F);
}

// NEXT-1: WL, WR = (rho, u, v, w, p) face states; returns the Rusanov flux of E_rad.
double oracle_rusanov(double EL, double ER, const double WL[5], const double WR[5], int dir, double gamma) {
  Prim L, R;
  L.rho = WL[0]; L.v[0] = WL[1]; L.v[1] = WL[2]; L.v[2] = WL[3]; L.p = WL[4];
  R.rho = WR[0]; R.v[0] = WR[1]; R.v[1] = WR[2]; R.v[2] = WR[3]; R.p = WR[4];
  return rusanov(EL, ER, L, R, dir, gamma);
}

}  // extern "C"
