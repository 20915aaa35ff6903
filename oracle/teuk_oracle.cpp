// teuk_oracle.cpp -- CPU ORACLE.  TEST INFRASTRUCTURE ONLY.
//
// A plain, slow, obviously-correct FP64 implementation of the hot path of the time-domain
// Teukolsky solver of arXiv:1206.0270 (McKennon, Forrester, Khanna): the two-step
// Lax-Wendroff iteration of PAPER.md:90-100 (Eq. 3, Eq. 4) for the first-order system
// u = {Phi, Pi} obtained from the Teukolsky master equation
// (Eq. 1), after the m-mode split Psi = e^{im phi~} r^3 Phi (Eq. 2), with
// second-order centred theta differences, parity pole conditions and radial
// edge conditions, a Gaussian-smeared point source and a
// waveform tap at a fixed r* (PAPER.md:161).
//
// Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference leg may
// build, load or call this file.  It shares no code with paper_1206_0270_b200/csrc and neither
// imports the other.  One loop nest per stage, full-size arrays for the half-step values and
// for the coefficient fields D, S, each coefficient computed point by point
// from the closed forms below.  No blocking, fusion or reordering; OpenMP only splits the
// outermost r* loop of each stage.  Compile WITHOUT -ffast-math.
//
// The paper defers D and S to its ref. [8]; the closed forms here are the
// exact reduction of Eq. (1) listed in SURVEY.md section 8(c) C.1-C.3.  They are pinned by
// tests/test_oracle_pins.py against a computer-algebra substitution into Eq. (1) (pin P1),
// by second-order self-convergence (P2), by the Schwarzschild and Kerr l=m=2 quasinormal
// frequencies (P3, P3b), by the (m, theta) reflection invariant (P4), a = 0 realness (P5),
// linearity (P6), the unit norm of the deposit (P7), the edge rows' closed forms (P8), for the
// discrete-delta deposits the paper's step-function construction in exact rationals and the moment /
// interpolation conditions (P9), the waveform tap with an off-node observer against the interpolated weighted sum of
// the state and a closed form on a field linear in x (P10), and the derivative profiles of the multi-term deposit
// against exact-rational Lagrange derivatives, moment conditions and mpmath derivatives of the printed Gaussian
// (P12).  (P11 pins the seeded input generator that both sides share.)  The paper prints no field
// values: beyond those pins the numbers this file produces are "parity unpinned" by the paper; no function of this
// file is without a pin of its own.
//
// Readings of silent/ambiguous passages are the A1-A12 of SURVEY.md 8(c), restated in DESIGN.md.

#include <cmath>
#include <complex>
#include <cstdint>
#include <cstdlib>
#include <cstring>
#include <vector>

namespace {

typedef std::complex<double> cplx;
const cplx I1(0.0, 1.0);
const double PI = 3.14159265358979323846264338327950288;

// ---------------------------------------------------------------------------------------------
// C.1 Kerr quantities (textbook; Delta is defined at PAPER.md:78).
// ---------------------------------------------------------------------------------------------
struct Kerr {
  double M, a, rp, rm, cp, cm;  // r+-, tortoise constants c+- = 2 M r+- / (r+ - r-)
  Kerr(double M_, double a_) : M(M_), a(a_) {
    const double root = std::sqrt(M * M - a * a);
    rp = M + root;
    rm = M - root;
    cp = 2.0 * M * rp / (rp - rm);
    cm = (a == 0.0) ? 0.0 : 2.0 * M * rm / (rp - rm);
  }
};

// Radial point: r, delta = r - r+, Delta = delta (delta + r+ - r-)   (SURVEY.md 8(c) A3:
// Delta must never be formed from r^2 - 2Mr + a^2 near the horizon).
struct RPoint {
  double r, delta, Delta;
};

// f(y) = x(r+ + e^y) - x_target with y = ln(r - r+);  x(r) = r + c+ ln((r-r+)/2M) - c- ln((r-r-)/2M).
double tortoise_residual(const Kerr& k, double y, double x) {
  const double d = std::exp(y);
  double f = k.rp + d + k.cp * (y - std::log(2.0 * k.M)) - x;
  if (k.a != 0.0) f -= k.cm * std::log((d + k.rp - k.rm) / (2.0 * k.M));
  return f;
}

// Invert the tortoise map by bracketed Newton on y (f is strictly increasing in y).
RPoint r_of_rstar(const Kerr& k, double x) {
  double y = (x < 2.0 * k.rp) ? (x - k.rp) / k.cp + std::log(2.0 * k.M) : std::log(x);
  double lo = y, hi = y;
  while (tortoise_residual(k, lo, x) > 0.0) lo -= 1.0 + std::fabs(lo) * 0.5;
  while (tortoise_residual(k, hi, x) < 0.0) hi += 1.0 + std::fabs(hi) * 0.5;
  for (int it = 0; it < 200; ++it) {
    const double d = std::exp(y);
    const double f = tortoise_residual(k, y, x);
    if (f > 0.0) hi = y; else lo = y;
    double fp = d + k.cp;
    if (k.a != 0.0) fp -= k.cm * d / (d + k.rp - k.rm);
    double yn = y - f / fp;
    if (!(yn > lo && yn < hi)) yn = 0.5 * (lo + hi);
    const double dy = yn - y;
    y = yn;
    if (std::fabs(dy) <= 4e-16 * (1.0 + std::fabs(y))) break;
  }
  RPoint p;
  p.delta = std::exp(y);
  p.r = k.rp + p.delta;
  p.Delta = p.delta * (p.delta + k.rp - k.rm);
  return p;
}

// ---------------------------------------------------------------------------------------------
// C.2 / C.3 coefficients of
//   Phi_t = -b Phi_x + Pi
//   Pi_t  = +b Pi_x + kappa Phi_x + alpha Pi + gamma Phi + cL (Phi_thth + cot(th) Phi_th) + T
// i.e. the paper's u_t + D u_x = S with D = [[b,0],[-kappa,-b]],
// S = (Pi, alpha Pi + gamma Phi + cL L_theta Phi + T), for s = -2.
// ---------------------------------------------------------------------------------------------
struct Coef {
  double b, bx, cL;
  cplx kappa, alpha, gamma, beta;
};

Coef coefficients(const Kerr& k, int m, const RPoint& p, double theta) {
  const double M = k.M, a = k.a, r = p.r, Delta = p.Delta;
  const double sn = std::sin(theta), cs = std::cos(theta);
  const double R2 = r * r + a * a;
  const double Sig2 = R2 * R2 - a * a * Delta * sn * sn;
  Coef c;
  c.b = R2 / std::sqrt(Sig2);
  c.cL = Delta / Sig2;
  c.alpha = cplx(4.0 * (r * Delta - M * (r * r - a * a)),
                 -4.0 * M * a * m * r + 4.0 * a * Delta * cs) / Sig2;
  c.beta = cplx(2.0 * Delta * (4.0 * r * r + 3.0 * a * a) / r - 4.0 * (r - M) * R2,
                2.0 * m * a * R2) / Sig2;
  const double mc = m - 2.0 * cs;
  c.gamma = cplx(-Delta * (mc * mc / (sn * sn) + 2.0 + 6.0 * M / r - 6.0 * a * a / (r * r)),
                 -2.0 * a * m * (r + 2.0 * M - 3.0 * a * a / r)) / Sig2;
  const double b3 = c.b * c.b * c.b;
  const double dbdr = 2.0 * r * c.b / R2
                      - b3 * (4.0 * r * R2 - 2.0 * a * a * (r - M) * sn * sn) / (2.0 * R2 * R2);
  c.bx = Delta / R2 * dbdr;
  c.kappa = c.beta - c.alpha * c.b - c.b * c.bx;
  return c;
}

// g(y; sigma) = exp(-y^2 / (2 sigma^2)) / (sigma sqrt(2 pi))      (C.6)
double gauss(double y, double sigma) {
  return std::exp(-y * y / (2.0 * sigma * sigma)) / (sigma * std::sqrt(2.0 * PI));
}

// Discrete delta ("define a step function on a discrete numerical grid and then apply the
// finite-difference derivative operation on the discrete step-function").  On a grid of spacing h with the
// particle at x_p = x_k + gamma h, 0 <= gamma < 1, the discrete step is H_{i+1/2} = 0 (i < k), 1 - gamma
// (i = k), 1 (i > k) -- the cell averages of the step, i.e. the first difference of the sampled ramp
// max(x - x_p, 0) -- and its difference (H_{i+1/2} - H_{i-1/2})/h is (1 - gamma)/h at x_k, gamma/h at x_{k+1},
// 0 elsewhere: the hat function below evaluated at y = x_i - x_p.  (reading A13.)
double delta_linear(double y, double h) {
  const double s = std::fabs(y) / h;
  return (s < 1.0) ? (1.0 - s) / h : 0.0;
}

// "Refined version" (details in its refs [3, 4], not in the container; reading A13): the
// four-point delta whose weights are the cubic Lagrange interpolation weights at x_p divided by h, so that
// sum_i d_i f(x_i) h = f(x_p) for every cubic f.  As a function of y = x_i - x_p, s = |y|/h:
//   s < 1 : (1 - s)(1 + s)(2 - s)/2 ;   1 <= s < 2 : (1 - s)(2 - s)(3 - s)/6 ;   else 0.
double delta_cubic(double y, double h) {
  const double s = std::fabs(y) / h;
  if (s < 1.0) return (1.0 - s) * (1.0 + s) * (2.0 - s) / 2.0 / h;
  if (s < 2.0) return (1.0 - s) * (2.0 - s) * (3.0 - s) / 6.0 / h;
  return 0.0;
}

// ---------------------------------------------------------------------------------------------
// f2 (SURVEY.md 8(f); PAPER.md:80 "T is ... constructed from the energy-momentum tensor", :145-151): the physical
// s = -2 source is a sum of terms proportional to the delta function AND ITS FIRST AND SECOND DERIVATIVES in r
// and theta with long coefficients that are not printed in the paper (its refs [7], [3]) and are NOT in this
// file.  What is here is the deposit mechanism for such a sum: rank-1 terms
//     A_t(t) * P^(a_t)(x - x_p; w_r) * P^(b_t)(theta - theta_p; w_theta),   a_t, b_t in {0, 1, 2},
// where P^(k)(y) is the k-th derivative with respect to y of the deposit profile P (the Gaussian g, or a
// discrete delta), so that sum_i P^(k)(x_i - x_p) f(x_i) h  ->  (-1)^k f^(k)(x_p): the action of delta^(k).
// (reading A14.)
// ---------------------------------------------------------------------------------------------

// k-th y-derivative of g(y; sigma) = exp(-y^2/(2 sigma^2))/(sigma sqrt(2 pi)):
//   g' = -(y/sigma^2) g,   g'' = (y^2/sigma^4 - 1/sigma^2) g.
double gauss_deriv(int order, double y, double sigma) {
  const double g = gauss(y, sigma);
  if (order == 0) return g;
  const double s2 = sigma * sigma;
  if (order == 1) return -(y / s2) * g;
  return (y * y / (s2 * s2) - 1.0 / s2) * g;
}

// Derivatives of the discrete deltas.  The weights of delta_linear / delta_cubic are L_i(x_p)/h, L_i the
// Lagrange basis polynomials of the stencil around x_p = x_k + gamma h, 0 <= gamma < 1 (two points k, k+1; four
// points k-1 .. k+2).  delta' and delta'' act as -f'(x_p) and +f''(x_p), so their weights are -L_i'(x_p)/h and
// L_i''(x_p)/h: the y-derivatives of the same piecewise polynomials, piece chosen by the stencil position of the
// point: y = x_i - x_p lies in (-2h,-h], (-h,0], (0,h], (h,2h] for i = k-1, k, k+1, k+2.  (The pieces join
// continuously but with kinks, so the half-open ends matter for the derivatives and only for them.)
// Two points carry no second derivative (L_i'' = 0): order 2 needs the four-point rule.
double delta_linear_deriv(int order, double y, double h) {
  if (order == 0) return delta_linear(y, h);
  if (order == 1) {
    if (y > -h && y <= 0.0) return 1.0 / (h * h);
    if (y > 0.0 && y <= h) return -1.0 / (h * h);
  }
  return 0.0;
}

double delta_cubic_deriv(int order, double y, double h) {
  if (order == 0) return delta_cubic(y, h);
  const double s = std::fabs(y) / h;
  const double sg = (y > 0.0) ? 1.0 : -1.0;           // d|y|/dy on the piece the point belongs to
  const bool inner = (y <= 0.0) ? (s < 1.0) : (s <= 1.0);
  const bool outer = !inner && ((y <= 0.0) ? (s < 2.0) : (s <= 2.0));
  if (order == 1) {
    if (inner) return sg * (-1.0 - 4.0 * s + 3.0 * s * s) / 2.0 / (h * h);     // d/ds (2 - s - 2s^2 + s^3)/2
    if (outer) return sg * (-11.0 + 12.0 * s - 3.0 * s * s) / 6.0 / (h * h);   // d/ds (6 - 11s + 6s^2 - s^3)/6
    return 0.0;
  }
  if (inner) return (3.0 * s - 2.0) / (h * h * h);
  if (outer) return (2.0 - s) / (h * h * h);
  return 0.0;
}

double profile_deriv(int kind, int order, double y, double width) {
  if (kind == 1) return delta_linear_deriv(order, y, width);
  if (kind == 2) return delta_cubic_deriv(order, y, width);
  return gauss_deriv(order, y, width);
}

}  // namespace

namespace {

struct Observer {
  double x_obs;
  int i0;
  double f;
  std::vector<double> weights;               // [n_theta]
  std::vector<double> t;                     // [n_rec]
  std::vector<cplx> w;                       // [n_rec][n_modes]
};

struct Oracle {
  Kerr kerr;
  int n_modes, n_r, n_theta, outer_bc;       // outer_bc: 0 = OUTGOING, 1 = DIRICHLET (A6)
  std::vector<int> m;
  double x_min, x_max, dx, dth, dt;
  int64_t step;                              // completed iterations n; t = n dt
  std::vector<double> x, xh, theta;          // x_i, x_{i+1/2}, theta_j
  // fields, [mode][i][j]
  std::vector<cplx> Phi, Pi, PhiN, PiN;      // level n and n+1, n_r rows
  std::vector<cplx> Phih, Pih;               // half-step values, n_r-1 rows (row i <-> x_{i+1/2})
  // coefficient fields, full size ("matrices D and S"), nodes and half points
  std::vector<Coef> cn, ch;                  // [mode][i][j], [mode][i+1/2][j]
  std::vector<double> Ap, Am;                // C.4: A+-_j = 1/dth^2 +- cot(th_j)/(2 dth)
  // source (C.6)
  bool has_source;
  int64_t n_samples;
  std::vector<double> xp, thp;               // [n_samples]
  std::vector<cplx> amp;                     // [mode][n_samples]
  double sigma_r, sigma_th;
  int W;
  int source_kind;                           // 0 Gaussian (C.6), 1 two-point, 2 four-point discrete delta (f3)
  // f2: when n_terms > 0 the deposited source is the sum of these rank-1 terms INSTEAD of the monopole `amp`
  int n_terms;
  std::vector<int> term_or, term_oth;        // [n_terms] derivative order of the profile in r* and in theta
  std::vector<cplx> term_amp;                // [term][mode][n_samples]
  std::vector<Observer> obs;

  Oracle(double a, double M) : kerr(M, a) {}
  size_t idx(int k, int i, int j) const { return ((size_t)k * n_r + i) * n_theta + j; }
  size_t idh(int k, int i, int j) const { return ((size_t)k * (n_r - 1) + i) * n_theta + j; }
};

// C.4 with the ghosts of PAPER.md:104 (reading A5): f_{-1} = P f_0, f_{N} = P f_{N-1}, P = (-1)^m.
// `row` points at n_theta values of one r* row.
inline cplx L_theta(const Oracle& o, const cplx* row, int j, double P) {
  const cplx fm = (j == 0) ? P * row[0] : row[j - 1];
  const cplx fp = (j == o.n_theta - 1) ? P * row[o.n_theta - 1] : row[j + 1];
  return o.Ap[j] * fp + o.Am[j] * fm - (2.0 / (o.dth * o.dth)) * row[j];
}

// C.6: T(t, x, theta) for mode k at orbit sample ks; `half` selects the half-point stage.
// Zero outside the (2W+1)^2 window around (i_p, j_p); the window is clipped at the grid edges.
inline cplx source_term(const Oracle& o, int k, int64_t ks, bool half, int i, int j) {
  if (!o.has_source) return cplx(0.0, 0.0);
  const double xp = o.xp[ks], thp = o.thp[ks];
  const double v = (xp - o.x_min) / o.dx;
  const int ip = half ? (int)std::floor(v - 0.5 + 0.5) : (int)std::floor(v + 0.5);
  const int jp = (int)std::floor(thp / o.dth - 0.5 + 0.5);
  // discrete deltas: the window is their support (nearest point +-1 or +-2), widths are the grid spacings
  const int W = (o.source_kind == 0) ? o.W : o.source_kind;
  if (std::abs(i - ip) > W || std::abs(j - jp) > W) return cplx(0.0, 0.0);
  const double xx = half ? o.xh[i] : o.x[i];
  if (o.n_terms > 0) {                       // f2: sum of rank-1 terms with derivative profiles
    const double wr = (o.source_kind == 0) ? o.sigma_r : o.dx, wth = (o.source_kind == 0) ? o.sigma_th : o.dth;
    cplx T(0.0, 0.0);
    for (int t = 0; t < o.n_terms; ++t) {
      const cplx At = o.term_amp[((size_t)t * o.n_modes + k) * o.n_samples + ks];
      T += At * profile_deriv(o.source_kind, o.term_or[t], xx - xp, wr) *
           profile_deriv(o.source_kind, o.term_oth[t], o.theta[j] - thp, wth);
    }
    return T;
  }
  const cplx A = o.amp[(size_t)k * o.n_samples + ks];
  if (o.source_kind == 1) return A * delta_linear(xx - xp, o.dx) * delta_linear(o.theta[j] - thp, o.dth);
  if (o.source_kind == 2) return A * delta_cubic(xx - xp, o.dx) * delta_cubic(o.theta[j] - thp, o.dth);
  return A * gauss(xx - xp, o.sigma_r) * gauss(o.theta[j] - thp, o.sigma_th);
}

// One iteration (C.5): half step Eq. (3), full step Eq. (4), radial edges, then the tap (C.7).
void iterate(Oracle& o) {
  const int nr = o.n_r, nth = o.n_theta;
  const double dt = o.dt, dx = o.dx;
  const int64_t ks_half = 2 * o.step, ks_full = 2 * o.step + 1;
  for (int k = 0; k < o.n_modes; ++k) {
    const double P = (o.m[k] % 2 == 0) ? 1.0 : -1.0;
    // ---- half step, Eq. (3): i = 0 .. n_r-2 -------------------------------------------------
#pragma omp parallel for schedule(static)
    for (int i = 0; i < nr - 1; ++i) {
      std::vector<cplx> Phibar((size_t)nth);
      for (int j = 0; j < nth; ++j) Phibar[j] = 0.5 * (o.Phi[o.idx(k, i, j)] + o.Phi[o.idx(k, i + 1, j)]);
      for (int j = 0; j < nth; ++j) {
        const Coef& c = o.ch[o.idh(k, i, j)];
        const cplx Pibar = 0.5 * (o.Pi[o.idx(k, i, j)] + o.Pi[o.idx(k, i + 1, j)]);
        const cplx dPhi = (o.Phi[o.idx(k, i + 1, j)] - o.Phi[o.idx(k, i, j)]) / dx;
        const cplx dPi = (o.Pi[o.idx(k, i + 1, j)] - o.Pi[o.idx(k, i, j)]) / dx;
        const cplx T = source_term(o, k, ks_half, true, i, j);
        o.Phih[o.idh(k, i, j)] = Phibar[j] + 0.5 * dt * (-c.b * dPhi + Pibar);
        o.Pih[o.idh(k, i, j)] =
            Pibar + 0.5 * dt * (c.b * dPi + c.kappa * dPhi + c.alpha * Pibar + c.gamma * Phibar[j] +
                                c.cL * L_theta(o, Phibar.data(), j, P) + T);
      }
    }
    // ---- full step, Eq. (4): i = 1 .. n_r-2 -------------------------------------------------
#pragma omp parallel for schedule(static)
    for (int i = 1; i < nr - 1; ++i) {
      std::vector<cplx> Phit((size_t)nth);
      for (int j = 0; j < nth; ++j) Phit[j] = 0.5 * (o.Phih[o.idh(k, i, j)] + o.Phih[o.idh(k, i - 1, j)]);
      for (int j = 0; j < nth; ++j) {
        const Coef& c = o.cn[o.idx(k, i, j)];
        const cplx Pit = 0.5 * (o.Pih[o.idh(k, i, j)] + o.Pih[o.idh(k, i - 1, j)]);
        const cplx dPhi = (o.Phih[o.idh(k, i, j)] - o.Phih[o.idh(k, i - 1, j)]) / dx;
        const cplx dPi = (o.Pih[o.idh(k, i, j)] - o.Pih[o.idh(k, i - 1, j)]) / dx;
        const cplx T = source_term(o, k, ks_full, false, i, j);
        o.PhiN[o.idx(k, i, j)] = o.Phi[o.idx(k, i, j)] + dt * (-c.b * dPhi + Pit);
        o.PiN[o.idx(k, i, j)] =
            o.Pi[o.idx(k, i, j)] + dt * (c.b * dPi + c.kappa * dPhi + c.alpha * Pit + c.gamma * Phit[j] +
                                         c.cL * L_theta(o, Phit.data(), j, P) + T);
      }
    }
    // ---- radial edges (outer edge reading A6) ---------------------------------
    for (int j = 0; j < nth; ++j) {
      o.PhiN[o.idx(k, 0, j)] = 0.0;
      o.PiN[o.idx(k, 0, j)] = 0.0;
      if (o.outer_bc == 0) {
        const double b = o.cn[o.idx(k, nr - 1, j)].b;
        o.PiN[o.idx(k, nr - 1, j)] = 0.0;
        o.PhiN[o.idx(k, nr - 1, j)] =
            o.Phi[o.idx(k, nr - 1, j)] -
            dt * b * (o.Phi[o.idx(k, nr - 1, j)] - o.Phi[o.idx(k, nr - 2, j)]) / dx;
      } else {
        o.PhiN[o.idx(k, nr - 1, j)] = 0.0;
        o.PiN[o.idx(k, nr - 1, j)] = 0.0;
      }
    }
  }
  o.Phi.swap(o.PhiN);
  o.Pi.swap(o.PiN);
  o.step += 1;
  // ---- C.7 waveform tap: linear interpolation in x of Phi^{n} at x_obs, weighted theta sum ---
  for (size_t q = 0; q < o.obs.size(); ++q) {
    Observer& ob = o.obs[q];
    ob.t.push_back((double)o.step * dt);
    for (int k = 0; k < o.n_modes; ++k) {
      cplx w(0.0, 0.0);
      for (int j = 0; j < nth; ++j) {
        const cplx line = (1.0 - ob.f) * o.Phi[o.idx(k, ob.i0, j)] + ob.f * o.Phi[o.idx(k, ob.i0 + 1, j)];
        w += ob.weights[j] * line;
      }
      ob.w.push_back(w);
    }
  }
}

}  // namespace

// ---------------------------------------------------------------------------------------------
// C interface (ctypes).  Prefix orc_ : nothing here has the product's teuk_ names.
// ---------------------------------------------------------------------------------------------
extern "C" {

// r, r - r+, Delta at tortoise coordinate x.
void orc_r_of_rstar(double M, double a, double x, double* r, double* delta, double* Delta) {
  Kerr k(M, a);
  RPoint p = r_of_rstar(k, x);
  *r = p.r;
  *delta = p.delta;
  *Delta = p.Delta;
}

// out[13] = b, b_x, cL, Re/Im kappa, Re/Im alpha, Re/Im gamma, Re/Im beta, r, Delta at (x, theta).
void orc_coefficients(double M, double a, int m, double x, double theta, double* out) {
  Kerr k(M, a);
  RPoint p = r_of_rstar(k, x);
  Coef c = coefficients(k, m, p, theta);
  out[0] = c.b; out[1] = c.bx; out[2] = c.cL;
  out[3] = c.kappa.real(); out[4] = c.kappa.imag();
  out[5] = c.alpha.real(); out[6] = c.alpha.imag();
  out[7] = c.gamma.real(); out[8] = c.gamma.imag();
  out[9] = c.beta.real(); out[10] = c.beta.imag();
  out[11] = p.r; out[12] = p.Delta;
}

double orc_gauss(double y, double sigma) { return gauss(y, sigma); }
double orc_delta(int32_t kind, double y, double h) { return kind == 2 ? delta_cubic(y, h) : delta_linear(y, h); }

void* orc_create(double a, double M, const int32_t* m, int32_t n_modes, double rs_min, double rs_max,
                 int32_t n_r, int32_t n_theta, double dt, int32_t outer_bc) {
  if (!(std::fabs(a) < M) || n_modes < 1 || n_r < 4 || n_theta < 4 || !(dt > 0.0) || !(rs_max > rs_min))
    return nullptr;
  Oracle* o = new Oracle(a, M);
  o->n_modes = n_modes; o->n_r = n_r; o->n_theta = n_theta; o->outer_bc = outer_bc;
  o->m.assign(m, m + n_modes);
  o->x_min = rs_min; o->x_max = rs_max;
  o->dx = (rs_max - rs_min) / (n_r - 1);
  o->dth = PI / n_theta;
  o->dt = dt;
  o->step = 0;
  o->has_source = false; o->n_samples = 0; o->W = 0; o->sigma_r = o->sigma_th = 1.0; o->source_kind = 0;
  o->n_terms = 0;
  o->x.resize(n_r); o->xh.resize(n_r - 1); o->theta.resize(n_theta);
  for (int i = 0; i < n_r; ++i) o->x[i] = rs_min + i * o->dx;
  for (int i = 0; i < n_r - 1; ++i) o->xh[i] = o->x[i] + 0.5 * o->dx;
  for (int j = 0; j < n_theta; ++j) o->theta[j] = (j + 0.5) * o->dth;
  o->Ap.resize(n_theta); o->Am.resize(n_theta);
  for (int j = 0; j < n_theta; ++j) {
    const double cot = std::cos(o->theta[j]) / std::sin(o->theta[j]);
    o->Ap[j] = 1.0 / (o->dth * o->dth) + cot / (2.0 * o->dth);
    o->Am[j] = 1.0 / (o->dth * o->dth) - cot / (2.0 * o->dth);
  }
  const size_t nn = (size_t)n_modes * n_r * n_theta, nh = (size_t)n_modes * (n_r - 1) * n_theta;
  o->Phi.assign(nn, cplx(0, 0)); o->Pi.assign(nn, cplx(0, 0));
  o->PhiN.assign(nn, cplx(0, 0)); o->PiN.assign(nn, cplx(0, 0));
  o->Phih.assign(nh, cplx(0, 0)); o->Pih.assign(nh, cplx(0, 0));
  o->cn.resize(nn); o->ch.resize(nh);
  std::vector<RPoint> rn(n_r), rh(n_r - 1);
#pragma omp parallel for schedule(static)
  for (int i = 0; i < n_r; ++i) {
    rn[i] = r_of_rstar(o->kerr, o->x[i]);
    if (i < n_r - 1) rh[i] = r_of_rstar(o->kerr, o->xh[i]);
  }
  for (int k = 0; k < n_modes; ++k) {
#pragma omp parallel for schedule(static)
    for (int i = 0; i < n_r; ++i)
      for (int j = 0; j < n_theta; ++j) {
        o->cn[o->idx(k, i, j)] = coefficients(o->kerr, o->m[k], rn[i], o->theta[j]);
        if (i < n_r - 1) o->ch[o->idh(k, i, j)] = coefficients(o->kerr, o->m[k], rh[i], o->theta[j]);
      }
  }
  return o;
}

void orc_destroy(void* h) { delete (Oracle*)h; }

// Each array [n_modes][n_r][n_theta], theta fastest; NULL = zeros.  Resets t and the step count.
void orc_set_initial(void* h, const double* phi_re, const double* phi_im, const double* pi_re,
                     const double* pi_im) {
  Oracle* o = (Oracle*)h;
  const size_t nn = o->Phi.size();
  for (size_t q = 0; q < nn; ++q) {
    o->Phi[q] = cplx(phi_re ? phi_re[q] : 0.0, phi_im ? phi_im[q] : 0.0);
    o->Pi[q] = cplx(pi_re ? pi_re[q] : 0.0, pi_im ? pi_im[q] : 0.0);
  }
  o->step = 0;
  for (size_t q = 0; q < o->obs.size(); ++q) { o->obs[q].t.clear(); o->obs[q].w.clear(); }
}

// Sample k of the trajectory is at t = k dt/2.  n_samples = 0 removes the source.
void orc_set_source(void* h, int64_t n_samples, const double* rs_p, const double* theta_p,
                    const double* amp_re, const double* amp_im, double sigma_r, double sigma_theta,
                    int32_t half_window) {
  Oracle* o = (Oracle*)h;
  o->has_source = n_samples > 0;
  o->n_samples = n_samples;
  o->n_terms = 0;                            // a new trajectory starts with the monopole term only
  if (!o->has_source) return;
  o->xp.assign(rs_p, rs_p + n_samples);
  o->thp.assign(theta_p, theta_p + n_samples);
  o->amp.resize((size_t)o->n_modes * n_samples);
  for (size_t q = 0; q < o->amp.size(); ++q) o->amp[q] = cplx(amp_re[q], amp_im[q]);
  o->sigma_r = sigma_r; o->sigma_th = sigma_theta; o->W = half_window;
}

// 0 = Gaussian of C.6 (default), 1 = two-point, 2 = four-point discrete delta (f3).
void orc_set_source_kind(void* h, int32_t kind) { ((Oracle*)h)->source_kind = kind; }

// f2: replace the monopole by n_terms rank-1 terms (orders 0..2 per axis; amplitudes [term][mode][n_samples] on the
// trajectory installed by orc_set_source).  n_terms = 0 goes back to the monopole.  Returns 0, or -1 on a bad order.
int32_t orc_set_source_terms(void* h, int32_t n_terms, const int32_t* order_r, const int32_t* order_theta,
                             const double* amp_re, const double* amp_im) {
  Oracle* o = (Oracle*)h;
  if (n_terms < 0 || (n_terms > 0 && !o->has_source)) return -1;
  for (int t = 0; t < n_terms; ++t)
    if (order_r[t] < 0 || order_r[t] > 2 || order_theta[t] < 0 || order_theta[t] > 2) return -1;
  o->n_terms = n_terms;
  o->term_or.assign(order_r, order_r + n_terms);
  o->term_oth.assign(order_theta, order_theta + n_terms);
  const size_t n = (size_t)n_terms * o->n_modes * o->n_samples;
  o->term_amp.resize(n);
  for (size_t q = 0; q < n; ++q) o->term_amp[q] = cplx(amp_re[q], amp_im[q]);
  return 0;
}

double orc_profile_deriv(int32_t kind, int32_t order, double y, double width) { return profile_deriv(kind, order, y, width); }

// Returns the observer index, or -1 if x_obs is outside [x_0, x_{n_r-1}).  weights NULL = all ones.
int32_t orc_add_observer(void* h, double rs_obs, const double* weights) {
  Oracle* o = (Oracle*)h;
  Observer ob;
  ob.x_obs = rs_obs;
  const double v = (rs_obs - o->x_min) / o->dx;
  ob.i0 = (int)std::floor(v);
  if (ob.i0 < 0 || ob.i0 > o->n_r - 2) return -1;
  ob.f = v - ob.i0;
  ob.weights.assign(o->n_theta, 1.0);
  if (weights) ob.weights.assign(weights, weights + o->n_theta);
  o->obs.push_back(ob);
  return (int32_t)o->obs.size() - 1;
}

// Returns 0, or -1 if the trajectory table is too short for n more iterations.
int32_t orc_step(void* h, int64_t n) {
  Oracle* o = (Oracle*)h;
  if (o->has_source && 2 * (o->step + n) + 1 > o->n_samples + 1) return -1;
  for (int64_t q = 0; q < n; ++q) iterate(*o);
  return 0;
}

void orc_get_state(void* h, double* phi_re, double* phi_im, double* pi_re, double* pi_im) {
  Oracle* o = (Oracle*)h;
  const size_t nn = o->Phi.size();
  for (size_t q = 0; q < nn; ++q) {
    phi_re[q] = o->Phi[q].real(); phi_im[q] = o->Phi[q].imag();
    pi_re[q] = o->Pi[q].real(); pi_im[q] = o->Pi[q].imag();
  }
}

// Half-step fields of the LAST iteration, [n_modes][n_r-1][n_theta] (for stage-level checks).
void orc_get_half(void* h, double* phih_re, double* phih_im, double* pih_re, double* pih_im) {
  Oracle* o = (Oracle*)h;
  for (size_t q = 0; q < o->Phih.size(); ++q) {
    phih_re[q] = o->Phih[q].real(); phih_im[q] = o->Phih[q].imag();
    pih_re[q] = o->Pih[q].real(); pih_im[q] = o->Pih[q].imag();
  }
}

int64_t orc_step_count(void* h) { return ((Oracle*)h)->step; }

// Copies the whole recorded series of observer `obs`: t[n], w_re/w_im [n][n_modes].  Returns n.
int64_t orc_get_waveform(void* h, int32_t obs, double* t, double* w_re, double* w_im, int64_t capacity) {
  Oracle* o = (Oracle*)h;
  const Observer& ob = o->obs[obs];
  const int64_t n = (int64_t)ob.t.size();
  if (!t) return n;
  const int64_t c = n < capacity ? n : capacity;
  for (int64_t q = 0; q < c; ++q) {
    t[q] = ob.t[q];
    for (int k = 0; k < o->n_modes; ++k) {
      w_re[q * o->n_modes + k] = ob.w[q * o->n_modes + k].real();
      w_im[q * o->n_modes + k] = ob.w[q * o->n_modes + k].imag();
    }
  }
  return c;
}

// Source term T for mode k at orbit sample ks on the node (half = 0) or half-point (half = 1) grid,
// into re/im [rows][n_theta] (rows = n_r or n_r - 1).  For pin P7.
void orc_source_field(void* h, int32_t k, int64_t ks, int32_t half, double* re, double* im) {
  Oracle* o = (Oracle*)h;
  const int rows = half ? o->n_r - 1 : o->n_r;
  for (int i = 0; i < rows; ++i)
    for (int j = 0; j < o->n_theta; ++j) {
      const cplx T = source_term(*o, k, ks, half != 0, i, j);
      re[(size_t)i * o->n_theta + j] = T.real();
      im[(size_t)i * o->n_theta + j] = T.imag();
    }
}

}  // extern "C"
