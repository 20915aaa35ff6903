// teuk_internal.h -- device data layout and kernel parameter blocks of libteuk.so (sm_100a).
// Product code: shares nothing with the test checker.
//
// HBM layout:
//   state U[2] (ping-pong), each [n_modes][n_r][4][n_theta] FP64, theta fastest; the 4 components
//     of one r* row (Phi_R, Phi_I, Pi_R, Pi_I) are contiguous, so one marching
//     iteration of a warp reads one contiguous 32*n_theta-byte row and writes one.
//   rtab [n_modes][2 n_r - 1][RT_N] FP64: separable r-dependent factors of the coefficient
//     matrices D, S at location p = 2i (node x_i) and p = 2i+1 (half point).
//   ttab [n_modes][TT_N][n_theta] FP64: theta-dependent factors with the pole-parity ghosts
//      folded in.
#ifndef TEUK_INTERNAL_H_
#define TEUK_INTERNAL_H_

#include <stdint.h>

// r-table record (all divided by R2^2 = (r^2+a^2)^2 where the closed form has 1/Sigma^2;
// Q = b^2 = R2^2/Sigma^2 = 1/(1 - eps sin^2 theta) is applied per point):
enum {
  RT_EPS = 0,   // eps = a^2 Delta / R2^2
  RT_X32 = 1,   // (2/dx) * X3,  b b_x = Q^2 sin^2(theta) X3,  X3 = Delta[a^2 (r-M) - 2 r eps R2]/R2^3
  RT_BRE = 2,   // (2/dx) * Re beta^ = (2/dx) [2 Delta (4r^2+3a^2)/r - 4 (r-M) R2] / R2^2
  RT_BIM = 3,   // (2/dx) * Im beta^ = (2/dx) 2 m a / R2
  RT_A0 = 4,    // Re alpha^ = 4 (r Delta - M (r^2 - a^2)) / R2^2
  RT_A1 = 5,    // Im alpha^ = A1 + A2 cos(theta),  A1 = -4 M a m r / R2^2
  RT_A2 = 6,    //                                   A2 = 4 a Delta / R2^2
  RT_G1 = 7,    // Im gamma^ = -2 a m (r + 2M - 3a^2/r) / R2^2
  RT_GR = 8,    // Gr = 2 + 6M/r - 6a^2/r^2   (Re gamma^ = -cL^ (Gtheta + Gr))
  RT_CL = 9,    // cL^ = Delta / R2^2
  RT_N = 10
};

// theta-table rows
enum {
  TT_S2 = 0,    // sin^2 theta_j
  TT_COS = 1,   // cos theta_j
  TT_AP = 2,    // A+_j = 1/dth^2 + cot/(2 dth)   (0 at j = n_theta-1: ghost folded into TT_D0)
  TT_AM = 3,    // A-_j = 1/dth^2 - cot/(2 dth)   (0 at j = 0)
  TT_D0 = 4,    // -2/dth^2 - (m - 2 cos)^2/sin^2 (+ P A-_0 at j=0, + P A+_{N-1} at j=N-1), P=(-1)^m
  TT_N = 5
};

#define TEUK_MAX_OBS 8
#define TEUK_MAX_TERMS 12
#define TEUK_MAX_MODES 64

struct ObsDev {
  int i0;                 // floor((x_obs - x_min)/dx)
  double f;               // (x_obs - x_min)/dx - i0
  const double* weights;  // [n_theta] device
  double* ring;           // [ring_cap][n_modes][2] device
};

struct StepParams {
  const double* uin;
  double* uout;
  const double* rtab;
  const double* ttab;
  const double* coef2d;   // coef_mode 1: [n_modes][2 n_r - 1][8][n_theta] streamed coefficient planes
  int coef_mode;
  int n_r, n_theta, n_modes;
  int n_slabs, slab_q, slab_rem;   // marching kernels: slabs per mode; rows per slab = slab_q (+ 1 for the first slab_rem)
  int n_seg, seg_payload; // theta segments (register kernel, n_theta > 128): count and payload columns each
  int pdl;                // host side only: launch teuk_step_kernel as a programmatic dependent of the previous launch
  int variant;            // 0 = register-resident kernel, 1 = shared-memory-resident kernel, 2 = resident (on-chip) kernel
  int outer_bc;
  double dt, dx, rs_min, dth;
  // source
  int has_source, W;
  int source_kind;        // 0 Gaussian (sigma_r, sigma_th), 1 / 2 two- / four-point discrete delta (widths dx, dth)
  long long n_samples;
  const double *xp, *thp, *amp_re, *amp_im;   // amplitudes [n_modes][n_samples] ([n_terms][n_modes][n_samples] if n_terms > 0)
  double sigma_r, sigma_th;
  // f2, teuk_set_source_terms: n_terms > 0 = sum of rank-1 terms with derivative order 0..2 of the profile in r*
  // and in theta (kernels instantiated with TERMS = true); 0 = the single term of the trajectory table
  int n_terms;
  signed char term_or[TEUK_MAX_TERMS], term_oth[TEUK_MAX_TERMS];
  // iteration index of the INPUT state: n = *d_base + k
  const long long* d_base;
  int k;
  // waveform tap of the input state (sample n, slot (n-1) % ring_cap)
  int tap_enable, tap_enable2, n_obs;   // tap_enable2: level n+1 inside a temporal-blocking launch
  long long ring_cap;
  int* nonfinite;
  // resident kernel ("kernel" = 2, teuk_resident.cu): iterations per launch, rows of r* per block, tag of the
  // input level in the block-to-block exchange buffer `ll` ([n_modes][blocks][2 sides][2 parities] rows of
  // 16-byte {value.lo, tag, value.hi, tag} elements)
  int n_iter, res_rows, res_cache;   // res_cache: time-independent coefficients kept in shared memory
  unsigned tag0;
  void* ll;
  ObsDev obs[TEUK_MAX_OBS];
};

#endif
