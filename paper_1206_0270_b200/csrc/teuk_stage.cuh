// teuk_stage.cuh -- device code shared by the step kernels of libteuk.so (teuk_step.cu: marching kernels,
// teuk_resident.cu: resident kernel): register rows, the Lax-Wendroff stage (Eq. 3-4) in the
// scaled variables of DESIGN.md "Stage arithmetic", the source deposit, the waveform tap
// and the TMA / mbarrier helpers.  Every kernel calls the SAME lw_stage / add_source / tap, which
// is what makes their fields bit-identical.  Product code: shares nothing with the test checker.
#ifndef TEUK_STAGE_CUH_
#define TEUK_STAGE_CUH_

#include <cuda_runtime.h>
#include <math.h>
#include <stdint.h>

#include "teuk_internal.h"

namespace {

constexpr unsigned FULL = 0xffffffffu;

// The n_r - 2 interior rows are dealt to the n_slabs slabs as evenly as possible: the first slab_rem slabs get
// slab_q + 1 rows, the others slab_q (so that n_slabs = a whole number of waves of warps leaves no ragged tail).
__device__ __forceinline__ int slab_first_row(const StepParams& p, int slab) {
  return 1 + slab * p.slab_q + min(slab, p.slab_rem);
}

template <int V>
struct Row {
  double c[4][V];  // Phi_R, Phi_I, Pi_R, Pi_I for this lane's V columns
};

#ifndef TEUK_MIN_BLOCKS
#define TEUK_MIN_BLOCKS 2   // resident blocks for V = 1, 4 (V = 2 always asks for 3); 3 with V = 4 spills: 29 GPts/s
#endif
#ifndef TEUK_V2_BLOCKS
#define TEUK_V2_BLOCKS 3     // resident blocks of the marching kernel for V = 2 (160 registers, no spills); 4 (128 registers,
                             // 228 B of spill stores): configs 3 / 4 at 62 / 74 instead of 67 / 78 GPts/s
#endif
#ifndef TEUK_FAST_RSQRT
#define TEUK_FAST_RSQRT 1   // own MUFU.RSQ64H + one third-order step instead of CUDA's rsqrt(): +6 GPts/s
#endif
#ifndef TEUK_SLOTS
#define TEUK_SLOTS 2    // TMA landing slots per warp (register kernel): rows i+2 .. i+TEUK_SLOTS+1 in flight (3, 4: no gain)
#endif
#ifndef TEUK_GROUP
#define TEUK_GROUP 2    // columns processed "vertically" together inside a stage (ILP)
#endif

// theta-dependent factors of this lane's V columns (rows of teuk_internal.h TT_*)
template <int V>
struct ThetaVals {
  double s2[V], cs[V], ap[V], am[V], d0[V];
};

template <int V>
struct ThetaTab {
  ThetaVals<V> vals;
  __device__ __forceinline__ void get(ThetaVals<V>& t) const { t = vals; }
};

// theta tables read from a block-shared copy [TT_N][n_theta_pad] under lane mapping MAP 1: the two-column
// piece of lane l starts at column q*64 + 2l, so a warp-wide 16-byte load is bank-conflict free.
template <int V>
struct ThetaTabShared {
  const double* base;   // shared memory, row stride `stride` doubles, zero padded to 32*V columns
  int stride, lane;
  __device__ __forceinline__ void get(ThetaVals<V>& t) const {
    double* dst[TT_N] = {t.s2, t.cs, t.ap, t.am, t.d0};
#pragma unroll
    for (int k = 0; k < TT_N; ++k) {
      if (V == 1) {
        dst[k][0] = base[k * stride + lane];
      } else {
#pragma unroll
        for (int q = 0; q < V / 2; ++q) {
          const double2 w = *reinterpret_cast<const double2*>(base + k * stride + q * 64 + 2 * lane);
          dst[k][2 * q] = w.x;
          dst[k][2 * q + 1] = w.y;
        }
      }
    }
  }
};

// 1/sqrt(x) for x in (0.9, 1]: MUFU.RSQ64H seed (rel. error < 2^-20) + one third-order step
// y <- y + y e (1/2 + 3/8 e), e = 1 - x y^2  (error ~ e^3): no range checks, no branch.
__device__ __forceinline__ double rsqrt_near_one(double x);
__device__ __forceinline__ double rsqrt_near_one_arg(double x) { return rsqrt_near_one(x); }
__device__ __forceinline__ double rsqrt_near_one(double x) {
#if TEUK_FAST_RSQRT
  double y;
  asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(x));
  const double e = fma(-x * y, y, 1.0);
  return fma(y * e, fma(0.375, e, 0.5), y);
#else
  return rsqrt(x);
#endif
}

// ---- global <-> register rows ---------------------------------------------------------------
__device__ __forceinline__ void ld256(const double* p, double& a, double& b, double& c, double& d) {
  asm volatile("ld.global.L1::no_allocate.v4.f64 {%0,%1,%2,%3}, [%4];"
               : "=d"(a), "=d"(b), "=d"(c), "=d"(d) : "l"(p));
}
__device__ __forceinline__ void st256(double* p, double a, double b, double c, double d) {
  asm volatile("st.global.v4.f64 [%0], {%1,%2,%3,%4};" ::"l"(p), "d"(a), "d"(b), "d"(c), "d"(d) : "memory");
}

// VEC: n_theta % V == 0, so a lane's chunk is either fully valid (aligned vector access) or absent.
template <int V, bool VEC>
__device__ __forceinline__ void load_row(Row<V>& u, const double* __restrict__ row, int nth, int j0) {
#pragma unroll
  for (int c = 0; c < 4; ++c) {
    const double* p = row + (size_t)c * nth + j0;
    if (VEC) {
      if ((unsigned)j0 < (unsigned)nth) {
        if (V == 1) {
          u.c[c][0] = __ldcs(p);
        } else if (V % 4 == 0) {
#pragma unroll
          for (int v = 0; v < V; v += 4) ld256(p + v, u.c[c][v], u.c[c][v + 1], u.c[c][v + 2], u.c[c][v + 3]);
        } else {
#pragma unroll
          for (int v = 0; v < V; v += 2) {
            const double2 t = __ldcs(reinterpret_cast<const double2*>(p + v));
            u.c[c][v] = t.x;
            u.c[c][v + 1] = t.y;
          }
        }
      } else {
#pragma unroll
        for (int v = 0; v < V; ++v) u.c[c][v] = 0.0;
      }
    } else {
#pragma unroll
      for (int v = 0; v < V; ++v) u.c[c][v] = ((unsigned)(j0 + v) < (unsigned)nth) ? __ldcs(p + v) : 0.0;
    }
  }
}

// Columns outside [pay_lo, pay_hi) (halo columns of a theta segment, idle lanes) are not stored.
template <int V, bool VEC>
__device__ __forceinline__ void store_row(const Row<V>& u, double* __restrict__ row, int nth, int j0, int pay_lo,
                                          int pay_hi) {
#pragma unroll
  for (int c = 0; c < 4; ++c) {
    double* p = row + (size_t)c * nth + j0;
    if (VEC) {
      if (j0 >= pay_lo && j0 < pay_hi) {
        if (V == 1) {
          __stcs(p, u.c[c][0]);
        } else if (V % 4 == 0) {
#pragma unroll
          for (int v = 0; v < V; v += 4) st256(p + v, u.c[c][v], u.c[c][v + 1], u.c[c][v + 2], u.c[c][v + 3]);
        } else {
#pragma unroll
          for (int v = 0; v < V; v += 2) __stcs(reinterpret_cast<double2*>(p + v), make_double2(u.c[c][v], u.c[c][v + 1]));
        }
      }
    } else {
#pragma unroll
      for (int v = 0; v < V; ++v)
        if (j0 + v >= pay_lo && j0 + v < pay_hi) __stcs(p + v, u.c[c][v]);
    }
  }
}

// ---- lane <-> column mappings ------------------------------------------------------------------
// MAP 0 (register-resident kernel): lane owns V contiguous columns j = lane*V + v.
// MAP 1 (shared-memory-resident kernel): lane owns V/2 two-column pieces, j = (v/2)*64 + 2*lane + (v&1)
//        (V = 1: j = lane), so a warp-wide 16-byte access touches 512 contiguous bytes: shared-memory
//        reads are bank-conflict free and global stores are fully coalesced.
template <int V, int MAP>
__device__ __forceinline__ int col_of(int lane, int v) {
  if (MAP == 0 || V == 1) return lane * V + v;
  return (v >> 1) * 64 + 2 * lane + (v & 1);
}

// theta-neighbours of f[v] across lanes: lf[v] = f at column-1, rt[v] = f at column+1 (values beyond
// the poles are garbage-but-finite: their coefficients are zero, see teuk_ttab_kernel).
template <int V, int MAP>
__device__ __forceinline__ void theta_neighbours(const double (&f)[V], double (&lf)[V], double (&rt)[V], int lane) {
  if (MAP == 0 || V == 1) {
    const double l = __shfl_up_sync(FULL, f[V - 1], 1), r = __shfl_down_sync(FULL, f[0], 1);
#pragma unroll
    for (int v = 0; v < V; ++v) {
      lf[v] = (v > 0) ? f[v > 0 ? v - 1 : 0] : l;
      rt[v] = (v < V - 1) ? f[v < V - 1 ? v + 1 : 0] : r;
    }
  } else {
    constexpr int NP = V / 2;
#pragma unroll
    for (int q = 0; q < NP; ++q) {
      // right neighbour of (q, lane, 1): (q, lane+1, 0), or (q+1, 0, 0) for lane 31
      const double send_r = (lane == 0 && q + 1 < NP) ? f[2 * (q + 1 < NP ? q + 1 : q)] : f[2 * q];
      // left neighbour of (q, lane, 0): (q, lane-1, 1), or (q-1, 31, 1) for lane 0
      const double send_l = (lane == 31 && q > 0) ? f[2 * (q > 0 ? q - 1 : 0) + 1] : f[2 * q + 1];
      const double r = __shfl_sync(FULL, send_r, (lane + 1) & 31);
      const double l = __shfl_sync(FULL, send_l, (lane + 31) & 31);
      lf[2 * q] = l;
      lf[2 * q + 1] = f[2 * q];
      rt[2 * q] = f[2 * q + 1];
      rt[2 * q + 1] = r;
    }
  }
}

// ---- one Lax-Wendroff stage at one radial location ------------------------------------------
// HALF: A = u^n_i, B = u^n_{i+1}, out = 2 u^{n+1/2}_{i+1/2}             (Eq. 3, tau = dt/2)
// else: A = H_{i-1/2}, B = H_{i+1/2} (doubled), out = u^{n+1}_i, base = u^n_i   (Eq. 4, tau = dt/4)
// The stage comes in two pieces so that a kernel whose rows span several warps can exchange the boundary columns
// of S_Phi between them (teuk_wide.cu): lw_stage_sums (S_Phi = A_Phi + B_Phi), then the theta-neighbours, then
// lw_stage_body (everything else).  lw_stage = the three in a row, within one warp.
template <int V>
__device__ __forceinline__ void lw_stage_sums(const Row<V>& A, const Row<V>& B, double (&sfr)[V], double (&sfi)[V]) {
#pragma unroll
  for (int v = 0; v < V; ++v) {
    sfr[v] = A.c[0][v] + B.c[0][v];
    sfi[v] = A.c[1][v] + B.c[1][v];
  }
}

template <int V, bool HALF, class TT>
__device__ __forceinline__ void lw_stage_body(const Row<V>& A, const Row<V>& B, const Row<V>& base,
                                              const double* __restrict__ rec, const TT& tht, double tau,
                                              double two_over_dx, Row<V>& out, const double (&sfr)[V],
                                              const double (&sfi)[V], const double (&nlr)[V], const double (&nrr)[V],
                                              const double (&nli)[V], const double (&nri)[V]);

template <int V, bool HALF, int MAP = 0, class TT = ThetaTab<V>>
__device__ __forceinline__ void lw_stage(const Row<V>& A, const Row<V>& B, const Row<V>& base,
                                         const double* __restrict__ rec, const TT& tht,
                                         double tau, double two_over_dx, Row<V>& out, int lane = 0) {
  double sfr[V], sfi[V];
  lw_stage_sums<V>(A, B, sfr, sfi);
  // theta-neighbours across lanes (pole ghosts are folded into ap/am/d0; see teuk_ttab_kernel)
  double nlr[V], nrr[V], nli[V], nri[V];
  theta_neighbours<V, MAP>(sfr, nlr, nrr, lane);
  theta_neighbours<V, MAP>(sfi, nli, nri, lane);
  lw_stage_body<V, HALF, TT>(A, B, base, rec, tht, tau, two_over_dx, out, sfr, sfi, nlr, nrr, nli, nri);
}

template <int V, bool HALF, class TT>
__device__ __forceinline__ void lw_stage_body(const Row<V>& A, const Row<V>& B, const Row<V>& base,
                                              const double* __restrict__ rec, const TT& tht, double tau,
                                              double two_over_dx, Row<V>& out, const double (&sfr)[V],
                                              const double (&sfi)[V], const double (&nlr)[V], const double (&nrr)[V],
                                              const double (&nli)[V], const double (&nri)[V]) {
  ThetaVals<V> th;
  tht.get(th);
  const double2 r01 = *reinterpret_cast<const double2*>(rec + 0);
  const double2 r23 = *reinterpret_cast<const double2*>(rec + 2);
  const double2 r45 = *reinterpret_cast<const double2*>(rec + 4);
  const double2 r67 = *reinterpret_cast<const double2*>(rec + 6);
  const double2 r89 = *reinterpret_cast<const double2*>(rec + 8);
  const double eps = r01.x, x32 = r01.y, bre2 = r23.x, bim2 = r23.y;
  const double a0 = r45.x, a1 = r45.y, a2 = r67.x, g1 = r67.y, gr = r89.x, cl = r89.y;
  // The V columns are processed in groups of G: inside a group every operation is written for all
  // G columns back to back, so consecutive FP64 instructions are independent (DFMA latency is 8
  // cycles at one issue per 2 cycles: a lone dependent chain leaves the pipe 3/4 idle).
  constexpr int G = (TEUK_GROUP < V) ? TEUK_GROUP : V;
#pragma unroll
  for (int v0 = 0; v0 < V; v0 += G) {
    double dfr[G], dfi[G], spr[G], spi[G], dpr[G], dpi[G], b[G], Q[G], b2d[G], aim[G], diag[G], bre[G];
    double e2r[G], e2i[G], ltr[G], lti[G], br[G], bi[G];
#define FORG _Pragma("unroll") for (int g = 0; g < G; ++g)
    FORG b[g] = fma(-eps, th.s2[v0 + g], 1.0);
    FORG b[g] = rsqrt_near_one_arg(b[g]);
    FORG { dfr[g] = B.c[0][v0 + g] - A.c[0][v0 + g]; dfi[g] = B.c[1][v0 + g] - A.c[1][v0 + g]; }
    FORG { spr[g] = A.c[2][v0 + g] + B.c[2][v0 + g]; spi[g] = A.c[3][v0 + g] + B.c[3][v0 + g]; }
    FORG { dpr[g] = B.c[2][v0 + g] - A.c[2][v0 + g]; dpi[g] = B.c[3][v0 + g] - A.c[3][v0 + g]; }
    FORG { aim[g] = fma(a2, th.cs[v0 + g], a1); diag[g] = th.d0[v0 + g] - gr; }
    FORG { Q[g] = b[g] * b[g]; b2d[g] = b[g] * two_over_dx; }
    FORG bre[g] = fma(-Q[g], th.s2[v0 + g] * x32, bre2);
    // E2 = 2 (Pi - b dPhi/dx)
    FORG { e2r[g] = fma(-b2d[g], dfr[g], spr[g]); e2i[g] = fma(-b2d[g], dfi[g], spi[g]); }
    FORG {
      out.c[0][v0 + g] = fma(tau, e2r[g], HALF ? sfr[v0 + g] : base.c[0][v0 + g]);
      out.c[1][v0 + g] = fma(tau, e2i[g], HALF ? sfi[v0 + g] : base.c[1][v0 + g]);
    }
    // L'_theta S_Phi
    FORG { ltr[g] = diag[g] * sfr[v0 + g]; lti[g] = diag[g] * sfi[v0 + g]; }
    FORG { ltr[g] = fma(th.am[v0 + g], nlr[v0 + g], ltr[g]); lti[g] = fma(th.am[v0 + g], nli[v0 + g], lti[g]); }
    FORG { ltr[g] = fma(th.ap[v0 + g], nrr[v0 + g], ltr[g]); lti[g] = fma(th.ap[v0 + g], nri[v0 + g], lti[g]); }
    // bracket B (same order of operations for every G: results do not depend on the grouping)
    FORG { br[g] = bre[g] * dfr[g]; bi[g] = bre[g] * dfi[g]; }
    FORG { br[g] = fma(-bim2, dfi[g], br[g]); bi[g] = fma(bim2, dfr[g], bi[g]); }
    FORG { br[g] = fma(a0, e2r[g], br[g]); bi[g] = fma(a0, e2i[g], bi[g]); }
    FORG { br[g] = fma(-aim[g], e2i[g], br[g]); bi[g] = fma(aim[g], e2r[g], bi[g]); }
    FORG { br[g] = fma(cl, ltr[g], br[g]); bi[g] = fma(cl, lti[g], bi[g]); }
    FORG { br[g] = fma(-g1, sfi[v0 + g], br[g]); bi[g] = fma(g1, sfr[v0 + g], bi[g]); }
    FORG { br[g] = fma(b2d[g], dpr[g], Q[g] * br[g]); bi[g] = fma(b2d[g], dpi[g], Q[g] * bi[g]); }
    FORG {
      out.c[2][v0 + g] = fma(tau, br[g], HALF ? spr[g] : base.c[2][v0 + g]);
      out.c[3][v0 + g] = fma(tau, bi[g], HALF ? spi[g] : base.c[3][v0 + g]);
    }
#undef FORG
  }
}

// The time-independent part of lw_stage for one location and this lane's V columns: b2d = (2/dx) b, Q = b^2 and
// Re beta^' = Re beta^ - Q s^2 X3, by the SAME operations in the same order as lw_stage, so that a kernel which
// keeps them (the resident kernel caches them in shared memory) reproduces lw_stage bit for bit.
template <int V>
__device__ __forceinline__ void lw_stage_coefficients(const double* __restrict__ rec, const ThetaVals<V>& th,
                                                      double two_over_dx, double (&b2d)[V], double (&Q)[V],
                                                      double (&bre)[V]) {
  const double eps = rec[RT_EPS], x32 = rec[RT_X32], bre2 = rec[RT_BRE];
#pragma unroll
  for (int v = 0; v < V; ++v) {
    double b = fma(-eps, th.s2[v], 1.0);
    b = rsqrt_near_one_arg(b);
    Q[v] = b * b;
    b2d[v] = b * two_over_dx;
    bre[v] = fma(-Q[v], th.s2[v] * x32, bre2);
  }
}

// lw_stage with b2d, Q, Re beta^' given (see lw_stage_coefficients): 12 of the 49 FP64 instructions per point
// and the rsqrt chain at the head of the stage are gone; everything else is lw_stage, operation for operation.
template <int V, bool HALF>
__device__ __forceinline__ void lw_stage_cached(const Row<V>& A, const Row<V>& B, const Row<V>& base,
                                                const double* __restrict__ rec, const ThetaTab<V>& tht,
                                                const double (&b2d)[V], const double (&Q)[V], const double (&bre)[V],
                                                double tau, Row<V>& out) {
  ThetaVals<V> th;
  tht.get(th);
  const double2 r23 = *reinterpret_cast<const double2*>(rec + 2);
  const double2 r45 = *reinterpret_cast<const double2*>(rec + 4);
  const double2 r67 = *reinterpret_cast<const double2*>(rec + 6);
  const double2 r89 = *reinterpret_cast<const double2*>(rec + 8);
  const double bim2 = r23.y;
  const double a0 = r45.x, a1 = r45.y, a2 = r67.x, g1 = r67.y, gr = r89.x, cl = r89.y;
  double sfr[V], sfi[V];
#pragma unroll
  for (int v = 0; v < V; ++v) {
    sfr[v] = A.c[0][v] + B.c[0][v];
    sfi[v] = A.c[1][v] + B.c[1][v];
  }
  double nlr[V], nrr[V], nli[V], nri[V];
  theta_neighbours<V, 0>(sfr, nlr, nrr, 0);
  theta_neighbours<V, 0>(sfi, nli, nri, 0);
  constexpr int G = (TEUK_GROUP < V) ? TEUK_GROUP : V;
#pragma unroll
  for (int v0 = 0; v0 < V; v0 += G) {
    double dfr[G], dfi[G], spr[G], spi[G], dpr[G], dpi[G], aim[G], diag[G];
    double e2r[G], e2i[G], ltr[G], lti[G], br[G], bi[G];
#define FORG _Pragma("unroll") for (int g = 0; g < G; ++g)
    FORG { dfr[g] = B.c[0][v0 + g] - A.c[0][v0 + g]; dfi[g] = B.c[1][v0 + g] - A.c[1][v0 + g]; }
    FORG { spr[g] = A.c[2][v0 + g] + B.c[2][v0 + g]; spi[g] = A.c[3][v0 + g] + B.c[3][v0 + g]; }
    FORG { dpr[g] = B.c[2][v0 + g] - A.c[2][v0 + g]; dpi[g] = B.c[3][v0 + g] - A.c[3][v0 + g]; }
    FORG { aim[g] = fma(a2, th.cs[v0 + g], a1); diag[g] = th.d0[v0 + g] - gr; }
    FORG { e2r[g] = fma(-b2d[v0 + g], dfr[g], spr[g]); e2i[g] = fma(-b2d[v0 + g], dfi[g], spi[g]); }
    FORG {
      out.c[0][v0 + g] = fma(tau, e2r[g], HALF ? sfr[v0 + g] : base.c[0][v0 + g]);
      out.c[1][v0 + g] = fma(tau, e2i[g], HALF ? sfi[v0 + g] : base.c[1][v0 + g]);
    }
    FORG { ltr[g] = diag[g] * sfr[v0 + g]; lti[g] = diag[g] * sfi[v0 + g]; }
    FORG { ltr[g] = fma(th.am[v0 + g], nlr[v0 + g], ltr[g]); lti[g] = fma(th.am[v0 + g], nli[v0 + g], lti[g]); }
    FORG { ltr[g] = fma(th.ap[v0 + g], nrr[v0 + g], ltr[g]); lti[g] = fma(th.ap[v0 + g], nri[v0 + g], lti[g]); }
    FORG { br[g] = bre[v0 + g] * dfr[g]; bi[g] = bre[v0 + g] * dfi[g]; }
    FORG { br[g] = fma(-bim2, dfi[g], br[g]); bi[g] = fma(bim2, dfr[g], bi[g]); }
    FORG { br[g] = fma(a0, e2r[g], br[g]); bi[g] = fma(a0, e2i[g], bi[g]); }
    FORG { br[g] = fma(-aim[g], e2i[g], br[g]); bi[g] = fma(aim[g], e2r[g], bi[g]); }
    FORG { br[g] = fma(cl, ltr[g], br[g]); bi[g] = fma(cl, lti[g], bi[g]); }
    FORG { br[g] = fma(-g1, sfi[v0 + g], br[g]); bi[g] = fma(g1, sfr[v0 + g], bi[g]); }
    FORG { br[g] = fma(b2d[v0 + g], dpr[g], Q[v0 + g] * br[g]); bi[g] = fma(b2d[v0 + g], dpi[g], Q[v0 + g] * bi[g]); }
    FORG {
      out.c[2][v0 + g] = fma(tau, br[g], HALF ? spr[g] : base.c[2][v0 + g]);
      out.c[3][v0 + g] = fma(tau, bi[g], HALF ? spi[g] : base.c[3][v0 + g]);
    }
#undef FORG
  }
}

// ---- coef_mode 1: the same stage with the eight 2D coefficient planes STREAMED from HBM ----------
// (comparison arm for the bytes-vs-flops choice: +128 B per point per iteration, -26 FP64 instructions).
// `loc` points at this location's [8][n_theta] planes (see teuk_coef2d_kernel); textbook form
// R = b dPi + kappa dPhi + alpha Pi + gamma Phi + cL L_theta Phi in the scaled variables S, D.
template <int V, bool HALF, bool VEC>
__device__ __forceinline__ void lw_stage_planes(const Row<V>& A, const Row<V>& B, const Row<V>& base,
                                                const double* __restrict__ loc, const ThetaTab<V>& tht, double tau,
                                                Row<V>& out, int nth, int j0) {
  ThetaVals<V> th;
  tht.get(th);
  double cf[8][V];
#pragma unroll
  for (int k = 0; k < 8; ++k) {
    const double* q = loc + (size_t)k * nth + j0;
    if (VEC && j0 < nth) {
      if (V == 1) {
        cf[k][0] = __ldcs(q);
      } else if (V % 4 == 0) {
#pragma unroll
        for (int v = 0; v < V; v += 4) ld256(q + v, cf[k][v], cf[k][v + 1], cf[k][v + 2], cf[k][v + 3]);
      } else {
#pragma unroll
        for (int v = 0; v < V; v += 2) {
          const double2 t = __ldcs(reinterpret_cast<const double2*>(q + v));
          cf[k][v] = t.x;
          cf[k][v + 1] = t.y;
        }
      }
    } else {
#pragma unroll
      for (int v = 0; v < V; ++v) cf[k][v] = (j0 + v < nth) ? __ldcs(q + v) : 0.0;
    }
  }
  double sfr[V], sfi[V];
#pragma unroll
  for (int v = 0; v < V; ++v) {
    sfr[v] = A.c[0][v] + B.c[0][v];
    sfi[v] = A.c[1][v] + B.c[1][v];
  }
  double nlr[V], nrr[V], nli[V], nri[V];
  theta_neighbours<V, 0>(sfr, nlr, nrr, 0);
  theta_neighbours<V, 0>(sfi, nli, nri, 0);
#pragma unroll
  for (int v = 0; v < V; ++v) {
    const double dfr = B.c[0][v] - A.c[0][v], dfi = B.c[1][v] - A.c[1][v];
    const double spr = A.c[2][v] + B.c[2][v], spi = A.c[3][v] + B.c[3][v];
    const double dpr = B.c[2][v] - A.c[2][v], dpi = B.c[3][v] - A.c[3][v];
    const double b2d = cf[0][v], kre = cf[1][v], kim = cf[2][v], are = cf[3][v], aim = cf[4][v];
    const double gre = cf[5][v], gim = cf[6][v], cl = cf[7][v];
    const double e2r = fma(-b2d, dfr, spr), e2i = fma(-b2d, dfi, spi);
    out.c[0][v] = fma(tau, e2r, HALF ? sfr[v] : base.c[0][v]);
    out.c[1][v] = fma(tau, e2i, HALF ? sfi[v] : base.c[1][v]);
    const double ltr = fma(th.ap[v], nrr[v], fma(th.am[v], nlr[v], th.d0[v] * sfr[v]));
    const double lti = fma(th.ap[v], nri[v], fma(th.am[v], nli[v], th.d0[v] * sfi[v]));
    double br = kre * dfr;
    br = fma(-kim, dfi, br);
    br = fma(are, spr, br);
    br = fma(-aim, spi, br);
    br = fma(cl, ltr, br);
    br = fma(gre, sfr[v], br);
    br = fma(-gim, sfi[v], br);
    br = fma(b2d, dpr, br);
    double bi = kre * dfi;
    bi = fma(kim, dfr, bi);
    bi = fma(are, spi, bi);
    bi = fma(aim, spr, bi);
    bi = fma(cl, lti, bi);
    bi = fma(gre, sfi[v], bi);
    bi = fma(gim, sfr[v], bi);
    bi = fma(b2d, dpi, bi);
    out.c[2][v] = fma(tau, br, HALF ? spr : base.c[2][v]);
    out.c[3][v] = fma(tau, bi, HALF ? spi : base.c[3][v]);
  }
}

// g(y; sigma) = exp(-y^2/(2 sigma^2)) / (sigma sqrt(2 pi))
__device__ __forceinline__ double gauss_dev(double y, double sigma) {
  return exp(-y * y / (2.0 * sigma * sigma)) / (sigma * sqrt(2.0 * 3.14159265358979323846264338327950288));
}

// Deposit profile along one axis at offset y from the particle.  kind 0: the Gaussian above, width = sigma.
// kind 1 / 2: two-point / four-point discrete delta on a grid of spacing `width`:
// the interpolation weight of the grid point at distance s = |y|/width, over the spacing.
__device__ __forceinline__ double deposit_profile(int kind, double y, double width) {
  if (kind == 0) return gauss_dev(y, width);
  const double s = fabs(y) / width;
  if (kind == 1) return s < 1.0 ? (1.0 - s) / width : 0.0;
  if (s < 1.0) return (1.0 - s) * (1.0 + s) * (2.0 - s) / 2.0 / width;
  if (s < 2.0) return (1.0 - s) * (2.0 - s) * (3.0 - s) / 6.0 / width;
  return 0.0;
}

}  // namespace

namespace {

// Source bookkeeping of one stage for one warp: window test and the theta Gaussian per column.
template <int V>
struct StageSource {
  bool on;          // the window of this stage intersects this slab
  int ip;           // centre row index (nodes: i, half points: i + 1/2 -> i)
  double xp, are, aim;
  double gth[V];    // g(theta_j - theta_p) inside |j - jp| <= W, else 0
};

template <int V, int MAP = 0>
__device__ __forceinline__ void setup_source(StageSource<V>& s, const StepParams& p, int mode, long long ks,
                                             bool half, int row_lo, int row_hi, int lane, int col0 = 0) {
  s.on = false;
  if (!p.has_source) return;
  const double xp = p.xp[ks], thp = p.thp[ks];
  // identical rounding decisions to the definition: i_p = round((x_p - x_min)/dx [- 1/2]),
  // j_p = round(theta_p/dtheta - 1/2), round(z) = floor(z + 1/2); division and adds only.
  const double v = __ddiv_rn(__dsub_rn(xp, p.rs_min), p.dx);
  const int ip = half ? (int)floor(__dadd_rn(__dsub_rn(v, 0.5), 0.5)) : (int)floor(__dadd_rn(v, 0.5));
  const int jp = (int)floor(__dadd_rn(__dsub_rn(__ddiv_rn(thp, p.dth), 0.5), 0.5));
  if (ip + p.W < row_lo || ip - p.W > row_hi) return;
  s.on = true;
  s.ip = ip;
  s.xp = xp;
  s.are = p.amp_re[(size_t)mode * p.n_samples + ks];
  s.aim = p.amp_im[(size_t)mode * p.n_samples + ks];
#pragma unroll
  for (int q = 0; q < V; ++q) {
    const int j = col0 + col_of<V, MAP>(lane, q);
    const double th = __dmul_rn((double)j + 0.5, p.dth);
    s.gth[q] = ((unsigned)j < (unsigned)p.n_theta && abs(j - jp) <= p.W) ? deposit_profile(p.source_kind, th - thp, p.sigma_th) : 0.0;
  }
}

// out.Pi += dt * A' g(x - x_p) g(theta - theta_p) on row `i` of this stage's grid.
template <int V>
__device__ __forceinline__ void add_source(Row<V>& out, const StageSource<V>& s, const StepParams& p, int i,
                                           bool half) {
  if (!s.on || abs(i - s.ip) > p.W) return;
  double x = __dadd_rn(p.rs_min, __dmul_rn((double)i, p.dx));
  if (half) x = __dadd_rn(x, __dmul_rn(0.5, p.dx));
  const double g = p.dt * deposit_profile(p.source_kind, x - s.xp, p.sigma_r);
#pragma unroll
  for (int q = 0; q < V; ++q) {
    const double gg = g * s.gth[q];
    out.c[2][q] = fma(s.are, gg, out.c[2][q]);
    out.c[3][q] = fma(s.aim, gg, out.c[3][q]);
  }
}

// ---- f2: sums of rank-1 deposit terms with derivative profiles (teuk_set_source_terms) ----------------------
// The physical s = -2 source (PAPER.md:80 "constructed from the energy-momentum tensor", :145-151) is a sum of
// terms in the delta function and its first and second derivatives in r and theta; its coefficients are the
// caller's (they are not printed in the paper and not in this library), the deposit is ours:
//     dt * sum_t A_t P^(a_t)(x - x_p; w_r) P^(b_t)(theta - theta_p; w_theta),   a_t, b_t in {0, 1, 2},
// P^(k) = k-th derivative of the deposit profile with respect to its argument.  Gaussian: g' = -(y/s^2) g,
// g'' = (y^2/s^4 - 1/s^2) g.  Discrete deltas: the weights are L_i(x_p)/h with L_i the Lagrange polynomials of the
// stencil around x_p = x_k + gamma h (two points k, k+1; four points k-1 .. k+2), so delta^(n) has the weights
// (-1)^n L_i^(n)(x_p)/h = the y-derivatives of the same piecewise polynomials, the piece chosen by where the point
// sits in the stencil: y in (-2h,-h], (-h,0], (0,h], (h,2h] for i = k-1 .. k+2 (the pieces join with kinks, so the
// half-open ends matter here).  Kernels instantiated with TERMS = true use TermSource below; the default kernels
// (TERMS = false) contain none of this code.
struct Profile3 {
  double d[3];
};
__device__ __forceinline__ Profile3 deposit_profile3(int kind, double y, double width) {
  Profile3 r;
  r.d[0] = deposit_profile(kind, y, width);
  r.d[1] = 0.0;
  r.d[2] = 0.0;
  if (kind == 0) {
    const double s2 = width * width;
    r.d[1] = -(y / s2) * r.d[0];
    r.d[2] = (y * y / (s2 * s2) - 1.0 / s2) * r.d[0];
    return r;
  }
  const double h = width, s = fabs(y) / h;
  if (kind == 1) {                                  // two points carry no second derivative
    if (y > -h && y <= 0.0) r.d[1] = 1.0 / (h * h);
    if (y > 0.0 && y <= h) r.d[1] = -1.0 / (h * h);
    return r;
  }
  const double sg = (y > 0.0) ? 1.0 : -1.0;
  const bool inner = (y <= 0.0) ? (s < 1.0) : (s <= 1.0);
  const bool outer = !inner && ((y <= 0.0) ? (s < 2.0) : (s <= 2.0));
  if (inner) {
    r.d[1] = sg * (-1.0 - 4.0 * s + 3.0 * s * s) / 2.0 / (h * h);
    r.d[2] = (3.0 * s - 2.0) / (h * h * h);
  } else if (outer) {
    r.d[1] = sg * (-11.0 + 12.0 * s - 3.0 * s * s) / 6.0 / (h * h);
    r.d[2] = (2.0 - s) / (h * h * h);
  }
  return r;
}
__device__ __forceinline__ double pick3(const Profile3& r, int order) {
  return order == 0 ? r.d[0] : (order == 1 ? r.d[1] : r.d[2]);
}

// Window bookkeeping of one stage for the multi-term deposit.  The theta profiles (three derivative orders per
// column) do not depend on the row: a marching kernel gives every warp a table in shared memory (`tab`,
// [3][V][32] doubles, this lane's entries at [(k V + q) 32 + lane]) that setup_source fills once per stage, so a row
// of the window costs one radial profile and a short loop over the terms (round 2, first version: the profiles were
// rebuilt per row and column, exp and divisions included, and the one warp whose slab meets the window made the
// whole launch 3.5 times longer).  tab = nullptr (the resident kernel: one task = one row): built on the spot.
template <int V>
struct TermSource {
  bool on;
  int ip, jp, mode, lane, col0;
  long long ks;
  double xp, thp;
  double* tab;
};

template <int V, int MAP = 0>
__device__ __forceinline__ void setup_source(TermSource<V>& s, const StepParams& p, int mode, long long ks,
                                             bool half, int row_lo, int row_hi, int lane, int col0 = 0) {
  s.on = false;
  if (!p.has_source) return;
  const double xp = p.xp[ks], thp = p.thp[ks];
  const double v = __ddiv_rn(__dsub_rn(xp, p.rs_min), p.dx);       // same rounding decisions as the plain deposit
  const int ip = half ? (int)floor(__dadd_rn(__dsub_rn(v, 0.5), 0.5)) : (int)floor(__dadd_rn(v, 0.5));
  const int jp = (int)floor(__dadd_rn(__dsub_rn(__ddiv_rn(thp, p.dth), 0.5), 0.5));
  if (ip + p.W < row_lo || ip - p.W > row_hi) return;
  s.on = true;
  s.ip = ip;
  s.jp = jp;
  s.mode = mode;
  s.lane = lane;
  s.col0 = col0;
  s.ks = ks;
  s.xp = xp;
  s.thp = thp;
  if (s.tab) {
    for (int q = 0; q < V; ++q) {
      const int j = col0 + lane * V + q;                             // lane <-> column mapping MAP 0
      Profile3 pt;
      pt.d[0] = pt.d[1] = pt.d[2] = 0.0;
      if ((unsigned)j < (unsigned)p.n_theta && abs(j - jp) <= p.W)
        pt = deposit_profile3(p.source_kind, __dmul_rn((double)j + 0.5, p.dth) - thp, p.sigma_th);
#pragma unroll
      for (int k = 0; k < 3; ++k) s.tab[(k * V + q) * 32 + lane] = pt.d[k];
    }
  }
}

template <int V>
__device__ __forceinline__ void add_source(Row<V>& out, const TermSource<V>& s, const StepParams& p, int i,
                                           bool half) {
  if (!s.on || abs(i - s.ip) > p.W) return;
  double x = __dadd_rn(p.rs_min, __dmul_rn((double)i, p.dx));
  if (half) x = __dadd_rn(x, __dmul_rn(0.5, p.dx));
  const Profile3 pr = deposit_profile3(p.source_kind, x - s.xp, p.sigma_r);
  Profile3 pt[V];
  if (!s.tab) {
#pragma unroll
    for (int q = 0; q < V; ++q) {
      const int j = s.col0 + s.lane * V + q;
      pt[q].d[0] = pt[q].d[1] = pt[q].d[2] = 0.0;
      if ((unsigned)j < (unsigned)p.n_theta && abs(j - s.jp) <= p.W)
        pt[q] = deposit_profile3(p.source_kind, __dmul_rn((double)j + 0.5, p.dth) - s.thp, p.sigma_th);
    }
  }
  for (int t = 0; t < p.n_terms; ++t) {
    const size_t ia = ((size_t)t * p.n_modes + s.mode) * p.n_samples + s.ks;
    const double are = p.amp_re[ia], aim = p.amp_im[ia];
    const double gr = p.dt * pick3(pr, p.term_or[t]);
    const int kth = p.term_oth[t];
#pragma unroll
    for (int q = 0; q < V; ++q) {
      const double gg = gr * (s.tab ? s.tab[(kth * V + q) * 32 + s.lane] : pick3(pt[q], kth));
      out.c[2][q] = fma(are, gg, out.c[2][q]);
      out.c[3][q] = fma(aim, gg, out.c[3][q]);
    }
  }
}

// The same with the radial profile values given (marching kernels: built once per 16-row chunk, one row per lane,
// and fetched by shuffle) and the theta profiles in the table: all that is left per row is the loop over the terms.
template <int V>
__device__ __forceinline__ void add_source_row(Row<V>& out, const TermSource<V>& s, const StepParams& p,
                                               const Profile3& pr) {
  for (int t = 0; t < p.n_terms; ++t) {
    const size_t ia = ((size_t)t * p.n_modes + s.mode) * p.n_samples + s.ks;
    const double are = p.amp_re[ia], aim = p.amp_im[ia];
    const double gr = p.dt * pick3(pr, p.term_or[t]);
    const int kth = p.term_oth[t];
#pragma unroll
    for (int q = 0; q < V; ++q) {
      const double gg = gr * s.tab[(kth * V + q) * 32 + s.lane];
      out.c[2][q] = fma(are, gg, out.c[2][q]);
      out.c[3][q] = fma(aim, gg, out.c[3][q]);
    }
  }
}
template <int V>
__device__ __forceinline__ void add_source_row(Row<V>&, const StageSource<V>&, const StepParams&, const Profile3&) {}

// Shared-memory doubles of one warp's theta-profile tables (two stages) in a TERMS instantiation of a marching kernel
template <int V>
struct TermTab {
  static constexpr int PER_STAGE = 3 * V * 32;
};

// StageSource (one term, the profile itself: the configs' deposit) or TermSource (teuk_set_source_terms)
template <int V, bool TERMS>
struct SourceSel {
  typedef StageSource<V> type;
};
template <int V>
struct SourceSel<V, true> {
  typedef TermSource<V> type;
};

// Waveform tap of the INPUT state (sample n): w = sum_j W_j [(1-f) Phi_{i0,j} + f Phi_{i0+1,j}], in two pieces:
// tap_partial = this lane's columns (cheap, needs the rows), tap_finish = the warp reduction and the ring store
// (latency: ten shuffles and a global store; needs two doubles).  A kernel whose tasks sit on a critical path
// (teuk_resident.cu) runs tap_finish after it has handed its row over.  tap = both, for every observer of cell i.
template <int V, int MAP = 0>
__device__ __forceinline__ void tap_partial(const Row<V>& lo, const Row<V>& hi, const StepParams& p, int q, int lane,
                                            double& wr, double& wi) {
  const double f = p.obs[q].f;
  wr = 0.0;
  wi = 0.0;
#pragma unroll
  for (int v = 0; v < V; ++v) {
    const int j = col_of<V, MAP>(lane, v);
    const double wt = (j < p.n_theta) ? __ldg(p.obs[q].weights + j) : 0.0;
    wr = fma(wt, fma(f, hi.c[0][v], (1.0 - f) * lo.c[0][v]), wr);
    wi = fma(wt, fma(f, hi.c[1][v], (1.0 - f) * lo.c[1][v]), wi);
  }
}
__device__ __forceinline__ void tap_finish(const StepParams& p, int q, int mode, long long n, int lane, double wr,
                                           double wi) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) {
    wr += __shfl_xor_sync(FULL, wr, o);
    wi += __shfl_xor_sync(FULL, wi, o);
  }
  if (lane == 0) {
    const long long slot = (n - 1) % p.ring_cap;
    double* dst = p.obs[q].ring + ((size_t)slot * p.n_modes + mode) * 2;
    dst[0] = wr;
    dst[1] = wi;
    if (!isfinite(wr) || !isfinite(wi)) *p.nonfinite = 1;
  }
}
template <int V, int MAP = 0>
__device__ __forceinline__ void tap(const Row<V>& lo, const Row<V>& hi, const StepParams& p, int i, int mode,
                                    long long n, int lane) {
  for (int q = 0; q < p.n_obs; ++q) {
    if (p.obs[q].i0 != i) continue;
    double wr, wi;
    tap_partial<V, MAP>(lo, hi, p, q, lane, wr, wi);
    tap_finish(p, q, mode, n, lane, wr, wi);
  }
}

}  // namespace

// ---- TMA bulk-copy row prefetch (cp.async.bulk + mbarrier; SASS: UBLKCP) ------------------------
// One lane of each warp asks the TMA engine for the whole next r* row (4 components x n_theta
// doubles, contiguous in HBM) into the warp's shared-memory landing slot; the warp keeps computing
// and picks the row up from shared memory 1.5 marching iterations later.  No registers are tied
// up by loads in flight.
static __device__ __forceinline__ unsigned smem_u32(const void* p) { return (unsigned)__cvta_generic_to_shared(p); }

static __device__ __forceinline__ void mbar_init(unsigned long long* bar, unsigned count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
}
static __device__ __forceinline__ void tma_load_row(void* dst, const void* src, unsigned bytes, unsigned long long* bar) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
  asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
               ::"r"(smem_u32(dst)), "l"(src), "r"(bytes), "r"(smem_u32(bar)) : "memory");
}
// same operations on precomputed 32-bit shared addresses (keeps the address conversion out of the hot loop)
static __device__ __forceinline__ void tma_load_row_u32(unsigned dst, const void* src, unsigned bytes, unsigned bar) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
  asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
               ::"r"(dst), "l"(src), "r"(bytes), "r"(bar) : "memory");
}
// Bounded spin: try_wait suspends the warp for a hardware time slice per attempt, so 2^22 failed attempts
// are seconds, far beyond any HBM latency; a row that never arrives (a faulted TMA copy) then becomes a
// reported CUDA error (trap -> sticky TEUK_ECUDA) instead of a hung GPU.
static __device__ __forceinline__ void mbar_wait_u32(unsigned bar, unsigned parity) {
  unsigned ok, tries = 0;
  do {
    asm volatile("{ .reg .pred p; mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2; selp.u32 %0, 1, 0, p; }"
                 : "=r"(ok) : "r"(bar), "r"(parity) : "memory");
    if (!ok && ++tries > (1u << 22)) asm volatile("trap;");
  } while (!ok);
}
static __device__ __forceinline__ void mbar_wait(unsigned long long* bar, unsigned parity) {
  mbar_wait_u32(smem_u32(bar), parity);
}

// r-table staging: the 2*RT_CH records (node + half point) of the next RT_CH marching iterations
// are copied global -> shared with cp.async while the current chunk is being consumed, so the
// warp-uniform coefficient loads are short LDS broadcasts instead of exposed L2 round trips.
constexpr int RT_CH = 16;
constexpr int RT_CHUNK_DOUBLES = RT_CH * 2 * RT_N;

static __device__ __forceinline__ void stage_rtab_chunk(double* sbuf, const double* __restrict__ rtab, int p_begin,
                                                 int n_loc, int lane) {
  const size_t g0 = (size_t)p_begin * RT_N, gend = (size_t)n_loc * RT_N;
#pragma unroll
  for (int q = lane; q < RT_CHUNK_DOUBLES / 2; q += 32) {
    if (g0 + 2 * q < gend) {
      const unsigned saddr = (unsigned)__cvta_generic_to_shared(sbuf + 2 * q);
      asm volatile("cp.async.ca.shared.global [%0], [%1], 16;" ::"r"(saddr), "l"(rtab + g0 + 2 * q) : "memory");
    }
  }
  asm volatile("cp.async.commit_group;" ::: "memory");
}

// shared-memory row (same [comp][n_theta] layout as HBM) -> registers
template <int V>
__device__ __forceinline__ void lds_row(Row<V>& u, const double* srow, int comp_stride, int col, bool valid) {
#pragma unroll
  for (int c = 0; c < 4; ++c) {
    if (valid) {
      const double* q = srow + c * comp_stride + col;
      if (V == 1) {
        u.c[c][0] = q[0];
      } else {
#pragma unroll
        for (int v = 0; v < V; v += 2) {
          const double2 t = *reinterpret_cast<const double2*>(q + v);
          u.c[c][v] = t.x;
          u.c[c][v + 1] = t.y;
        }
      }
    } else {
#pragma unroll
      for (int v = 0; v < V; ++v) u.c[c][v] = 0.0;
    }
  }
}

// registers -> shared-memory row ([comp][nth] layout)
namespace {
template <int V>
__device__ __forceinline__ void sts_row(const Row<V>& u, double* srow, int nth, int j0) {
#pragma unroll
  for (int c = 0; c < 4; ++c) {
    if (j0 < nth) {
      double* q = srow + c * nth + j0;
      if (V == 1) {
        q[0] = u.c[c][0];
      } else {
#pragma unroll
        for (int v = 0; v < V; v += 2) *reinterpret_cast<double2*>(q + v) = make_double2(u.c[c][v], u.c[c][v + 1]);
      }
    }
  }
}
}  // namespace

#endif
