// teuk_tables.cu -- setup kernels (run once per teuk_create, off the hot loop): the separable
// factors of the coefficient matrices D and S of PAPER.md:102, derived from the Teukolsky
// equation PAPER.md:68-76 (Eq. 1) with Psi = e^{im phi~} r^3 Phi and s = -2.
// DESIGN.md section "Coefficients" gives the algebra; the product never calls the CPU checker of the tests.
#include <cuda_runtime.h>
#include <math.h>

#include "teuk_internal.h"

namespace {

struct KerrDev {
  double M, a, rp, rm, cp, cm, h;  // h = r+ - r-
};

__device__ inline KerrDev make_kerr(double M, double a) {
  KerrDev k;
  k.M = M;
  k.a = a;
  const double root = sqrt(M * M - a * a);
  k.rp = M + root;
  k.rm = M - root;
  k.h = k.rp - k.rm;
  k.cp = 2.0 * M * k.rp / k.h;
  k.cm = (a == 0.0) ? 0.0 : 2.0 * M * k.rm / k.h;
  return k;
}

// g(y) = x(r+ + e^y) - x, the tortoise map written in y = ln(r - r+) so that the horizon side
// (r - r+ ~ 1e-19) keeps full relative accuracy (reading A3).
__device__ inline double tort_res(const KerrDev& k, double y, double x, double* slope) {
  const double d = exp(y);
  double g = k.rp + d + k.cp * (y - log(2.0 * k.M)) - x;
  double s = d + k.cp;
  if (k.cm != 0.0) {
    g -= k.cm * log((d + k.h) / (2.0 * k.M));
    s -= k.cm * d / (d + k.h);
  }
  *slope = s;
  return g;
}

// Safeguarded Newton: g is strictly increasing in y, so a sign bracket always exists.
__device__ double solve_log_delta(const KerrDev& k, double x) {
  double y = (x < 2.0 * k.rp) ? (x - k.rp) / k.cp + log(2.0 * k.M) : log(x);
  double s;
  double ylo = y, yhi = y;
  for (int q = 0; q < 64 && tort_res(k, ylo, x, &s) > 0.0; ++q) ylo -= 1.0 + 0.5 * fabs(ylo);
  for (int q = 0; q < 64 && tort_res(k, yhi, x, &s) < 0.0; ++q) yhi += 1.0 + 0.5 * fabs(yhi);
  for (int it = 0; it < 100; ++it) {
    const double g = tort_res(k, y, x, &s);
    if (g > 0.0) yhi = y; else ylo = y;
    double yn = y - g / s;
    if (!(yn > ylo && yn < yhi)) yn = 0.5 * (ylo + yhi);
    const double step = fabs(yn - y);
    y = yn;
    if (step <= 4e-16 * (1.0 + fabs(y))) break;
  }
  return y;
}

}  // namespace

// One thread per radial location p (p = 2i: node x_i, p = 2i+1: half point x_i + dx/2).
__global__ void teuk_rtab_kernel(double* __restrict__ rtab, const int* __restrict__ mvals, int n_modes,
                                 int n_r, double rs_min, double dx, double M, double a) {
  const int n_loc = 2 * n_r - 1;
  const int p = blockIdx.x * blockDim.x + threadIdx.x;
  if (p >= n_loc) return;
  const KerrDev k = make_kerr(M, a);
  // same rounding sequence as the grid definition: x_i = rs_min + i*dx, x_{i+1/2} = x_i + dx/2
  double x = __dadd_rn(rs_min, __dmul_rn((double)(p >> 1), dx));
  if (p & 1) x = __dadd_rn(x, __dmul_rn(0.5, dx));
  const double y = solve_log_delta(k, x);
  const double delta = exp(y);
  const double r = k.rp + delta;
  const double Delta = delta * (delta + k.h);
  const double R2 = r * r + a * a;
  const double iR4 = 1.0 / (R2 * R2);
  const double eps = a * a * Delta * iR4;
  const double X3 = a * a * Delta * ((r - M) - 2.0 * r * Delta / R2) * iR4 / R2;
  const double bre = (2.0 * Delta * (4.0 * r * r + 3.0 * a * a) / r - 4.0 * (r - M) * R2) * iR4;
  const double a0 = 4.0 * (r * Delta - M * (r * r - a * a)) * iR4;
  const double a2 = 4.0 * a * Delta * iR4;
  const double gr = 2.0 + 6.0 * M / r - 6.0 * a * a / (r * r);
  const double cl = Delta * iR4;
  const double s2dx = 2.0 / dx;
  for (int q = 0; q < n_modes; ++q) {
    const double m = (double)mvals[q];
    double* rec = rtab + ((size_t)q * n_loc + p) * RT_N;
    rec[RT_EPS] = eps;
    rec[RT_X32] = s2dx * X3;
    rec[RT_BRE] = s2dx * bre;
    rec[RT_BIM] = s2dx * (2.0 * m * a / R2);
    rec[RT_A0] = a0;
    rec[RT_A1] = -4.0 * M * a * m * r * iR4;
    rec[RT_A2] = a2;
    rec[RT_G1] = -2.0 * a * m * (r + 2.0 * M - 3.0 * a * a / r) * iR4;
    rec[RT_GR] = gr;
    rec[RT_CL] = cl;
  }
}

// One thread per (mode, j).
__global__ void teuk_ttab_kernel(double* __restrict__ ttab, const int* __restrict__ mvals, int n_modes,
                                 int n_theta, double dth) {
  const int t = blockIdx.x * blockDim.x + threadIdx.x;
  if (t >= n_modes * n_theta) return;
  const int q = t / n_theta, j = t - q * n_theta;
  const int mi = mvals[q];
  const double m = (double)mi;
  const double P = (mi & 1) ? -1.0 : 1.0;
  const double th = __dmul_rn((double)j + 0.5, dth);
  double sn, cs;
  sincos(th, &sn, &cs);
  const double cot = cs / sn;
  const double idth2 = 1.0 / (dth * dth);
  double ap = idth2 + cot / (2.0 * dth);
  double am = idth2 - cot / (2.0 * dth);
  const double mc = m - 2.0 * cs;
  double d0 = -2.0 * idth2 - mc * mc / (sn * sn);
  if (j == 0) { d0 += P * am; am = 0.0; }                 // f_{-1} = P f_0
  if (j == n_theta - 1) { d0 += P * ap; ap = 0.0; }       // f_{N}  = P f_{N-1}
  double* base = ttab + (size_t)q * TT_N * n_theta;
  base[TT_S2 * n_theta + j] = sn * sn;
  base[TT_COS * n_theta + j] = cs;
  base[TT_AP * n_theta + j] = ap;
  base[TT_AM * n_theta + j] = am;
  base[TT_D0 * n_theta + j] = d0;
}

// coef_mode 1: eight full 2D coefficient planes per location, i.e. the paper's stored "matrices D and S"
// (PAPER.md:102), assembled once from the 1D tables and then STREAMED by the step kernel instead of being
// rebuilt.  Layout [mode][p][8][n_theta]; planes (prescaled so the kernel needs no assembly at all):
//   0: (2/dx) b   1,2: (2/dx) Re/Im kappa   3,4: Re/Im alpha   5: -cL Gr (r-part of Re gamma; the theta
//   part rides on the D0 table together with the pole ghosts)   6: Im gamma   7: cL.
__global__ void teuk_coef2d_kernel(double* __restrict__ c2d, const double* __restrict__ rtab,
                                   const double* __restrict__ ttab, int n_modes, int n_r, int n_theta,
                                   double dx) {
  const int n_loc = 2 * n_r - 1;
  const size_t t = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  const size_t total = (size_t)n_modes * n_loc * n_theta;
  if (t >= total) return;
  const int j = (int)(t % n_theta);
  const size_t qp = t / n_theta;  // q * n_loc + p
  const int q = (int)(qp / n_loc);
  const double* rec = rtab + qp * RT_N;
  const double* tb = ttab + (size_t)q * TT_N * n_theta;
  const double s2 = tb[TT_S2 * n_theta + j], cs = tb[TT_COS * n_theta + j];
  const double b = rsqrt(1.0 - rec[RT_EPS] * s2);
  const double Q = b * b;
  const double b2d = b * (2.0 / dx);
  const double are = Q * rec[RT_A0], aim = Q * (rec[RT_A1] + rec[RT_A2] * cs);
  double* out = c2d + (qp * 8) * n_theta + j;
  const size_t st = (size_t)n_theta;
  out[0 * st] = b2d;
  out[1 * st] = Q * rec[RT_BRE] - are * b2d - Q * Q * s2 * rec[RT_X32];  // (2/dx)(Re beta - Re alpha b - b b_x)
  out[2 * st] = Q * rec[RT_BIM] - aim * b2d;                             // (2/dx)(Im beta - Im alpha b)
  out[3 * st] = are;
  out[4 * st] = aim;
  out[5 * st] = -Q * rec[RT_CL] * rec[RT_GR];
  out[6 * st] = Q * rec[RT_G1];
  out[7 * st] = Q * rec[RT_CL];
}

cudaError_t teuk_launch_coef2d(double* c2d, const double* rtab, const double* ttab, int n_modes, int n_r,
                               int n_theta, double dx, cudaStream_t st) {
  const size_t total = (size_t)n_modes * (2 * (size_t)n_r - 1) * n_theta;
  teuk_coef2d_kernel<<<(unsigned)((total + 255) / 256), 256, 0, st>>>(c2d, rtab, ttab, n_modes, n_r, n_theta, dx);
  return cudaGetLastError();
}

// ---- host-side launcher (called from teuk_api.cu) --------------------------------------------
cudaError_t teuk_launch_tables(double* rtab, double* ttab, const int* d_m, int n_modes, int n_r, int n_theta,
                               double rs_min, double dx, double dth, double M, double a, cudaStream_t st) {
  const int n_loc = 2 * n_r - 1;
  teuk_rtab_kernel<<<(n_loc + 127) / 128, 128, 0, st>>>(rtab, d_m, n_modes, n_r, rs_min, dx, M, a);
  cudaError_t e = cudaGetLastError();
  if (e != cudaSuccess) return e;
  const int nt = n_modes * n_theta;
  teuk_ttab_kernel<<<(nt + 127) / 128, 128, 0, st>>>(ttab, d_m, n_modes, n_theta, dth);
  return cudaGetLastError();
}
