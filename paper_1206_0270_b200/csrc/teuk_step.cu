// teuk_step.cu -- the hot path: one two-step Lax-Wendroff iteration (Eq. 3-4)
// of u = {Phi, Pi} per launch, all modes, fused with the pole ghosts and radial edges
// (PAPER.md:104), the Gaussian source deposit and the waveform tap
// (PAPER.md:161).  Hand-written for sm_100a; no tensor cores (a stencil, not a contraction).
//
// Mapping: theta is the fastest index and one WARP spans the whole theta
// range, each lane owning V = ceil(n_theta/32) contiguous columns, so the theta-neighbours of
// the centred differences are register neighbours or one warp shuffle.  Each warp
// MARCHES along r* over a slab of rows, keeping u^n_i, u^n_{i+1} and the half-step values
// u^{n+1/2}_{i-1/2} (Eq. 3) in registers: every row of u^n is read from HBM once (plus one halo
// row per slab end) and every row of u^{n+1} is written once = 64 B per point per iteration, the
// algorithmic minimum.  Half-step values never touch memory.  The coefficient matrices D, S
// are rebuilt per point from 1D tables: the only genuinely 2D factor is
// Q = b^2 = 1/(1 - eps(r) sin^2 theta), one FP64 rsqrt.
//
// Scaled variables (exact algebra): with inputs A, B on two
// neighbouring rows, S = A + B, D = B - A, E2 = S_Pi - (2b/dx) D_Phi (twice the Phi right-hand
// side), and the half step stores H = 2 u^{n+1/2}:
//   half:  H_Phi = S_Phi + (dt/2) E2           H_Pi = S_Pi + (dt/2) [ (2b/dx) D_Pi + Q B ] + dt T
//   full:  Phi' = Phi + (dt/4) E2(H)           Pi'  = Pi  + (dt/4) [ (2b/dx) D_Pi + Q B ](H) + dt T
//   B = (2 beta^'/dx) D_Phi + alpha^ E2 + cL^ L'_theta S_Phi + i G1 S_Phi,
// which uses kappa dPhi + alpha Pi = Q[(beta^ - Q s2 X3) dPhi + alpha^ (Pi - b dPhi)].
#include <cuda_runtime.h>
#include <math.h>
#include <stdint.h>

#include "teuk_internal.h"

namespace {

constexpr unsigned FULL = 0xffffffffu;

template <int V>
struct Row {
  double c[4][V];  // Phi_R, Phi_I, Pi_R, Pi_I for this lane's V columns
};

#ifndef TEUK_TT_SMEM
#define TEUK_TT_SMEM 0   // theta tables: 0 = registers (measured faster), 1 = shared memory (16-byte pieces)
#endif
#ifndef TEUK_MIN_BLOCKS
#define TEUK_MIN_BLOCKS 2
#endif
#ifndef TEUK_FAST_RSQRT
#define TEUK_FAST_RSQRT 1
#endif
#ifndef TEUK_UNROLL2
#define TEUK_UNROLL2 1
#endif
#ifndef TEUK_PHASED
#define TEUK_PHASED 1   // compute the V reciprocal square roots of a stage up front (independent chains)
#endif

// theta-dependent factors of this lane's V columns (rows of teuk_internal.h TT_*)
template <int V>
struct ThetaVals {
  double s2[V], cs[V], ap[V], am[V], d0[V];
};

#if TEUK_TT_SMEM
// Block-shared copy, laid out so that a warp-wide 16-byte load touches 512 contiguous bytes:
// double index ((tbl * NP + piece) * 32 + lane) * PW + (v % PW), PW = min(V,2), NP = V / PW.
template <int V>
struct ThetaTab {
  const double* base;   // shared memory
  int lane;
  __device__ __forceinline__ void get(ThetaVals<V>& t) const {
    constexpr int PW = V >= 2 ? 2 : 1, NP = V / PW;
    double* dst[TT_N] = {t.s2, t.cs, t.ap, t.am, t.d0};
#pragma unroll
    for (int k = 0; k < TT_N; ++k)
#pragma unroll
      for (int q = 0; q < NP; ++q) {
        const double* src = base + ((k * NP + q) * 32 + lane) * PW;
        if (PW == 2) {
          const double2 w = *reinterpret_cast<const double2*>(src);
          dst[k][2 * q] = w.x;
          dst[k][2 * q + 1] = w.y;
        } else {
          dst[k][q] = src[0];
        }
      }
  }
};
#else
template <int V>
struct ThetaTab {
  ThetaVals<V> vals;
  __device__ __forceinline__ void get(ThetaVals<V>& t) const { t = vals; }
};
#endif

// 1/sqrt(x) for x in (0.9, 1]: MUFU.RSQ64H seed (rel. error < 2^-20) + one third-order step
// y <- y + y e (1/2 + 3/8 e), e = 1 - x y^2  (error ~ e^3): no range checks, no branch.
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
      if (j0 < nth) {
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
      for (int v = 0; v < V; ++v) u.c[c][v] = (j0 + v < nth) ? __ldcs(p + v) : 0.0;
    }
  }
}

template <int V, bool VEC>
__device__ __forceinline__ void store_row(const Row<V>& u, double* __restrict__ row, int nth, int j0) {
#pragma unroll
  for (int c = 0; c < 4; ++c) {
    double* p = row + (size_t)c * nth + j0;
    if (VEC) {
      if (j0 < nth) {
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
        if (j0 + v < nth) __stcs(p + v, u.c[c][v]);
    }
  }
}

// ---- one Lax-Wendroff stage at one radial location ------------------------------------------
// HALF: A = u^n_i, B = u^n_{i+1}, out = 2 u^{n+1/2}_{i+1/2}             (Eq. 3, tau = dt/2)
// else: A = H_{i-1/2}, B = H_{i+1/2} (doubled), out = u^{n+1}_i, base = u^n_i   (Eq. 4, tau = dt/4)
template <int V, bool HALF>
__device__ __forceinline__ void lw_stage(const Row<V>& A, const Row<V>& B, const Row<V>& base,
                                         const double* __restrict__ rec, const ThetaTab<V>& tht,
                                         double tau, double two_over_dx, Row<V>& out) {
  ThetaVals<V> th;
  tht.get(th);
  const double2 r01 = *reinterpret_cast<const double2*>(rec + 0);
  const double2 r23 = *reinterpret_cast<const double2*>(rec + 2);
  const double2 r45 = *reinterpret_cast<const double2*>(rec + 4);
  const double2 r67 = *reinterpret_cast<const double2*>(rec + 6);
  const double2 r89 = *reinterpret_cast<const double2*>(rec + 8);
  const double eps = r01.x, x32 = r01.y, bre2 = r23.x, bim2 = r23.y;
  const double a0 = r45.x, a1 = r45.y, a2 = r67.x, g1 = r67.y, gr = r89.x, cl = r89.y;

  double sfr[V], sfi[V];
#pragma unroll
  for (int v = 0; v < V; ++v) {
    sfr[v] = A.c[0][v] + B.c[0][v];
    sfi[v] = A.c[1][v] + B.c[1][v];
  }
  // theta-neighbours across lanes (pole ghosts are folded into ap/am/d0; see teuk_ttab_kernel)
  const double left_r = __shfl_up_sync(FULL, sfr[V - 1], 1), left_i = __shfl_up_sync(FULL, sfi[V - 1], 1);
  const double right_r = __shfl_down_sync(FULL, sfr[0], 1), right_i = __shfl_down_sync(FULL, sfi[0], 1);
#if TEUK_PHASED
  double bv[V];
#pragma unroll
  for (int v = 0; v < V; ++v) bv[v] = rsqrt_near_one(fma(-eps, th.s2[v], 1.0));
#endif
#pragma unroll
  for (int v = 0; v < V; ++v) {
    const double dfr = B.c[0][v] - A.c[0][v], dfi = B.c[1][v] - A.c[1][v];
    const double spr = A.c[2][v] + B.c[2][v], spi = A.c[3][v] + B.c[3][v];
    const double dpr = B.c[2][v] - A.c[2][v], dpi = B.c[3][v] - A.c[3][v];
    const double fmr = (v > 0) ? sfr[v > 0 ? v - 1 : 0] : left_r, fmi = (v > 0) ? sfi[v > 0 ? v - 1 : 0] : left_i;
    const double fpr = (v < V - 1) ? sfr[v < V - 1 ? v + 1 : 0] : right_r;
    const double fpi = (v < V - 1) ? sfi[v < V - 1 ? v + 1 : 0] : right_i;
    // coefficients at (r, theta_j)
#if TEUK_PHASED
    const double b = bv[v];
#else
    const double b = rsqrt_near_one(fma(-eps, th.s2[v], 1.0));
#endif
    const double Q = b * b;
    const double b2d = b * two_over_dx;
    const double aim = fma(a2, th.cs[v], a1);
    const double diag = th.d0[v] - gr;
    const double bre = fma(-Q, th.s2[v] * x32, bre2);
    // E2 = 2 (Pi - b dPhi/dx)
    const double e2r = fma(-b2d, dfr, spr), e2i = fma(-b2d, dfi, spi);
    out.c[0][v] = fma(tau, e2r, HALF ? sfr[v] : base.c[0][v]);
    out.c[1][v] = fma(tau, e2i, HALF ? sfi[v] : base.c[1][v]);
    // L'_theta S_Phi
    const double ltr = fma(th.ap[v], fpr, fma(th.am[v], fmr, diag * sfr[v]));
    const double lti = fma(th.ap[v], fpi, fma(th.am[v], fmi, diag * sfi[v]));
    // bracket B
    double br = bre * dfr;
    br = fma(-bim2, dfi, br);
    br = fma(a0, e2r, br);
    br = fma(-aim, e2i, br);
    br = fma(cl, ltr, br);
    br = fma(-g1, sfi[v], br);
    double bi = bre * dfi;
    bi = fma(bim2, dfr, bi);
    bi = fma(a0, e2i, bi);
    bi = fma(aim, e2r, bi);
    bi = fma(cl, lti, bi);
    bi = fma(g1, sfr[v], bi);
    const double tr = fma(b2d, dpr, Q * br), ti = fma(b2d, dpi, Q * bi);
    out.c[2][v] = fma(tau, tr, HALF ? spr : base.c[2][v]);
    out.c[3][v] = fma(tau, ti, HALF ? spi : base.c[3][v]);
  }
}

// g(y; sigma) = exp(-y^2/(2 sigma^2)) / (sigma sqrt(2 pi))
__device__ __forceinline__ double gauss_dev(double y, double sigma) {
  return exp(-y * y / (2.0 * sigma * sigma)) / (sigma * sqrt(2.0 * 3.14159265358979323846264338327950288));
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

template <int V>
__device__ __forceinline__ void setup_source(StageSource<V>& s, const StepParams& p, int mode, long long ks,
                                             bool half, int row_lo, int row_hi, int j0) {
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
    const int j = j0 + q;
    const double th = __dmul_rn((double)j + 0.5, p.dth);
    s.gth[q] = (j < p.n_theta && abs(j - jp) <= p.W) ? gauss_dev(th - thp, p.sigma_th) : 0.0;
  }
}

// out.Pi += dt * A' g(x - x_p) g(theta - theta_p) on row `i` of this stage's grid.
template <int V>
__device__ __forceinline__ void add_source(Row<V>& out, const StageSource<V>& s, const StepParams& p, int i,
                                           bool half) {
  if (!s.on || abs(i - s.ip) > p.W) return;
  double x = __dadd_rn(p.rs_min, __dmul_rn((double)i, p.dx));
  if (half) x = __dadd_rn(x, __dmul_rn(0.5, p.dx));
  const double g = p.dt * gauss_dev(x - s.xp, p.sigma_r);
#pragma unroll
  for (int q = 0; q < V; ++q) {
    const double gg = g * s.gth[q];
    out.c[2][q] = fma(s.are, gg, out.c[2][q]);
    out.c[3][q] = fma(s.aim, gg, out.c[3][q]);
  }
}

// Waveform tap of the INPUT state (sample n): w = sum_j W_j [(1-f) Phi_{i0,j} + f Phi_{i0+1,j}].
template <int V>
__device__ __forceinline__ void tap(const Row<V>& lo, const Row<V>& hi, const StepParams& p, int i, int mode,
                                    long long n, int j0, int lane) {
  for (int q = 0; q < p.n_obs; ++q) {
    if (p.obs[q].i0 != i) continue;
    const double f = p.obs[q].f;
    double wr = 0.0, wi = 0.0;
#pragma unroll
    for (int v = 0; v < V; ++v) {
      const double wt = (j0 + v < p.n_theta) ? __ldg(p.obs[q].weights + j0 + v) : 0.0;
      wr = fma(wt, fma(f, hi.c[0][v], (1.0 - f) * lo.c[0][v]), wr);
      wi = fma(wt, fma(f, hi.c[1][v], (1.0 - f) * lo.c[1][v]), wi);
    }
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
}

}  // namespace

// ---- TMA bulk-copy row prefetch (cp.async.bulk + mbarrier; SASS: UBLKCP) ------------------------
// One lane of each warp asks the TMA engine for the whole next r* row (4 components x n_theta
// doubles, contiguous in HBM) into the warp's shared-memory landing slot; the warp keeps computing
// and picks the row up from shared memory 1.5 marching iterations later.  No registers are tied
// up by loads in flight.
__device__ __forceinline__ unsigned smem_u32(const void* p) { return (unsigned)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void mbar_init(unsigned long long* bar, unsigned count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void tma_load_row(void* dst, const void* src, unsigned bytes, unsigned long long* bar) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
  asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
               ::"r"(smem_u32(dst)), "l"(src), "r"(bytes), "r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void mbar_wait(unsigned long long* bar, unsigned parity) {
  unsigned ok;
  do {
    asm volatile("{ .reg .pred p; mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2; selp.u32 %0, 1, 0, p; }"
                 : "=r"(ok) : "r"(smem_u32(bar)), "r"(parity) : "memory");
  } while (!ok);
}

// shared-memory row (same [comp][n_theta] layout as HBM) -> registers
template <int V>
__device__ __forceinline__ void lds_row(Row<V>& u, const double* srow, int nth, int j0) {
#pragma unroll
  for (int c = 0; c < 4; ++c) {
    if (j0 < nth) {
      const double* q = srow + c * nth + j0;
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

// r-table staging: the 2*RT_CH records (node + half point) of the next RT_CH marching iterations
// are copied global -> shared with cp.async while the current chunk is being consumed, so the
// warp-uniform coefficient loads are short LDS broadcasts instead of exposed L2 round trips.
constexpr int RT_CH = 16;
constexpr int RT_CHUNK_DOUBLES = RT_CH * 2 * RT_N;

__device__ __forceinline__ void stage_rtab_chunk(double* sbuf, const double* __restrict__ rtab, int p_begin,
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

template <int V, bool VEC>
__global__ void __launch_bounds__(128, TEUK_MIN_BLOCKS) teuk_step_kernel(const __grid_constant__ StepParams p) {
  const int lane = threadIdx.x & 31;
  const int slab = blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5);
  const int mode = blockIdx.y;
  const int nth = p.n_theta, nr = p.n_r;
#if TEUK_TT_SMEM
  __shared__ __align__(16) double s_tt[TT_N * 32 * V];
  {
    constexpr int PW = V >= 2 ? 2 : 1, NP = V / PW;
    const double* tb = p.ttab + (size_t)mode * TT_N * nth;
    for (int t = threadIdx.x; t < TT_N * 32 * V; t += blockDim.x) {
      const int k = t / (32 * V), r = t - k * 32 * V;      // table, position inside the table
      const int q = r / (32 * PW), l = (r / PW) % 32, w = r % PW;
      const int j = l * V + q * PW + w;                    // column owned by lane l
      s_tt[t] = (j < nth) ? tb[k * nth + j] : 0.0;
      (void)NP;
    }
    __syncthreads();
  }
#endif
  if (slab >= p.n_slabs) return;
  const int r0 = 1 + slab * p.slab_rows;             // first interior node of this slab
  const int r1 = min(r0 + p.slab_rows, nr - 1);      // one past the last
  const int j0 = lane * V;
  const size_t row_stride = (size_t)4 * nth;
  const double* __restrict__ uin = p.uin + (size_t)mode * nr * row_stride;
  double* __restrict__ uout = p.uout + (size_t)mode * nr * row_stride;
  const double* __restrict__ rtab = p.rtab + (size_t)mode * (2 * nr - 1) * RT_N;
  const long long n = *p.d_base + p.k;               // index of the input time level
  __shared__ __align__(16) double s_rt[4][2][RT_CHUNK_DOUBLES];
  __shared__ __align__(8) unsigned long long s_bar[4][2];
  extern __shared__ __align__(128) unsigned char s_dyn[];   // VEC: [warp][2 slots][4 n_theta] doubles
  const int wib = threadIdx.x >> 5;
  double* const rt_buf = &s_rt[wib][0][0];
  stage_rtab_chunk(rt_buf, rtab, 2 * r0, 2 * nr - 1, lane);
  const unsigned row_bytes = (unsigned)(row_stride * sizeof(double));
  double* const slot0 = reinterpret_cast<double*>(s_dyn) + (size_t)wib * 2 * row_stride;
  unsigned long long* const bars = &s_bar[wib][0];
  if (VEC) {
    if (lane == 0) {
      mbar_init(&bars[0], 1);
      mbar_init(&bars[1], 1);
      asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
      asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
      // row q lands in slot q & 1; rows r0+2 and (mid-iteration r0) r0+3 are the first uses
      if (r0 + 2 <= r1)
        tma_load_row(slot0 + (size_t)((r0 + 2) & 1) * row_stride, uin + (size_t)(r0 + 2) * row_stride, row_bytes,
                     &bars[(r0 + 2) & 1]);
    }
    __syncwarp();
  }

  ThetaTab<V> th;
#if TEUK_TT_SMEM
  th.base = s_tt;
  th.lane = lane;
#else
  {
    const double* tb = p.ttab + (size_t)mode * TT_N * nth;
#pragma unroll
    for (int v = 0; v < V; ++v) {
      const bool ok = j0 + v < nth;
      th.vals.s2[v] = ok ? tb[TT_S2 * nth + j0 + v] : 0.0;
      th.vals.cs[v] = ok ? tb[TT_COS * nth + j0 + v] : 0.0;
      th.vals.ap[v] = ok ? tb[TT_AP * nth + j0 + v] : 0.0;
      th.vals.am[v] = ok ? tb[TT_AM * nth + j0 + v] : 0.0;
      th.vals.d0[v] = ok ? tb[TT_D0 * nth + j0 + v] : 0.0;
    }
  }
#endif
  StageSource<V> src_h, src_f;   // half stage: sample 2n at half points; full stage: 2n+1 at nodes
  setup_source<V>(src_h, p, mode, 2 * n, true, r0 - 1, r1 - 1, j0);
  setup_source<V>(src_f, p, mode, 2 * n + 1, false, r0, r1 - 1, j0);
  const bool do_tap = p.tap_enable && p.n_obs > 0 && n >= 1;
  const double tau_h = 0.5 * p.dt, tau_f = 0.25 * p.dt, tdx = 2.0 / p.dx;

  Row<V> ua, ub, uc, hp, hn, out;
  load_row<V, VEC>(ua, uin + (size_t)(r0 - 1) * row_stride, nth, j0);
  load_row<V, VEC>(ub, uin + (size_t)r0 * row_stride, nth, j0);
  load_row<V, VEC>(uc, uin + (size_t)(r0 + 1) * row_stride, nth, j0);
  if (do_tap && r0 == 1) tap<V>(ua, ub, p, 0, mode, n, j0, lane);
  lw_stage<V, true>(ua, ub, ua, rtab + (size_t)(2 * (r0 - 1) + 1) * RT_N, th, tau_h, tdx, hp);
  add_source<V>(hp, src_h, p, r0 - 1, true);

  const double* rt_cur = rt_buf;
  // One marching iteration at node i.  On entry A = u^n_i, B = u^n_{i+1}, Hp = 2 u^{n+1/2}_{i-1/2};
  // on exit Hn = 2 u^{n+1/2}_{i+1/2} and A = u^n_{i+2}.  The caller alternates the roles of
  // (A, B) and (Hp, Hn), so no register rotation is needed.
  auto march = [&](const int i, Row<V>& A, Row<V>& B, Row<V>& Hp, Row<V>& Hn) {
    if (!VEC) {  // scalar fallback: prefetch row i+2 with plain loads
      if (i + 2 <= r1) load_row<V, VEC>(ua, uin + (size_t)(i + 2) * row_stride, nth, j0);
    }
    const int o = (i - r0) & (RT_CH - 1);
    if (o == 0) {  // chunk boundary (warp-uniform): current chunk has landed, start the next one
      asm volatile("cp.async.wait_group 0;" ::: "memory");
      __syncwarp();
      const int c = (i - r0) / RT_CH;
      rt_cur = rt_buf + (c & 1) * RT_CHUNK_DOUBLES;
      if (i + RT_CH < r1)
        stage_rtab_chunk(rt_buf + ((c + 1) & 1) * RT_CHUNK_DOUBLES, rtab, 2 * (i + RT_CH), 2 * nr - 1, lane);
    }
    if (do_tap) tap<V>(A, B, p, i, mode, n, j0, lane);
    lw_stage<V, true>(A, B, A, rt_cur + (2 * o + 1) * RT_N, th, tau_h, tdx, Hn);
    add_source<V>(Hn, src_h, p, i, true);
    if (VEC) {
      // B (row i+1, read from slot (i+1)&1 at the end of the last iteration) has been consumed by
      // every lane: its slot may now receive row i+3.
      __syncwarp();
      if (lane == 0 && i + 3 <= r1)
        tma_load_row(slot0 + (size_t)((i + 3) & 1) * row_stride, uin + (size_t)(i + 3) * row_stride, row_bytes,
                     &bars[(i + 3) & 1]);
    }
    lw_stage<V, false>(Hp, Hn, A, rt_cur + (2 * o) * RT_N, th, tau_f, tdx, out);
    add_source<V>(out, src_f, p, i, false);
    store_row<V, VEC>(out, uout + (size_t)i * row_stride, nth, j0);
    if (VEC) {
      if (i + 2 <= r1) {
        mbar_wait(&bars[(i + 2) & 1], (unsigned)(((i + 2) - (r0 + 2)) >> 1) & 1u);
        lds_row<V>(A, slot0 + (size_t)((i + 2) & 1) * row_stride, nth, j0);
      }
    } else {
      A = ua;
    }
  };
  {
    int i = r0;
#if TEUK_UNROLL2
    for (; i + 1 < r1; i += 2) {
      march(i, ub, uc, hp, hn);
      march(i + 1, uc, ub, hn, hp);
    }
    if (i < r1) march(i, ub, uc, hp, hn);
#else
    for (; i < r1; ++i) {
      march(i, ub, uc, hp, hn);
      hp = hn;
      Row<V> t = ub; ub = uc; uc = t;
    }
#endif
  }

  // radial edges (outer edge: DESIGN.md reading A6)
  if (r0 == 1) {
#pragma unroll
    for (int c = 0; c < 4; ++c)
#pragma unroll
      for (int v = 0; v < V; ++v) out.c[c][v] = 0.0;
    store_row<V, VEC>(out, uout, nth, j0);
  }
  if (r1 == nr - 1) {
    load_row<V, VEC>(ub, uin + (size_t)(nr - 1) * row_stride, nth, j0);
    load_row<V, VEC>(ua, uin + (size_t)(nr - 2) * row_stride, nth, j0);
    const double eps = __ldg(rtab + (size_t)(2 * (nr - 1)) * RT_N + RT_EPS);
    ThetaVals<V> tv;
    th.get(tv);
#pragma unroll
    for (int v = 0; v < V; ++v) {
      if (p.outer_bc == 0) {
        const double b = rsqrt_near_one(fma(-eps, tv.s2[v], 1.0));
        out.c[0][v] = ub.c[0][v] - p.dt * b * (ub.c[0][v] - ua.c[0][v]) / p.dx;
        out.c[1][v] = ub.c[1][v] - p.dt * b * (ub.c[1][v] - ua.c[1][v]) / p.dx;
      } else {
        out.c[0][v] = 0.0;
        out.c[1][v] = 0.0;
      }
      out.c[2][v] = 0.0;
      out.c[3][v] = 0.0;
    }
    store_row<V, VEC>(out, uout + (size_t)(nr - 1) * row_stride, nth, j0);
  }
}

// Tap of the CURRENT state at the end of a teuk_step call (the in-kernel tap records the input
// level of each iteration, so the last level needs one tiny launch).  One warp per (mode, observer).
__global__ void teuk_flush_tap_kernel(const __grid_constant__ StepParams p) {
  const int lane = threadIdx.x & 31;
  const int mode = blockIdx.x, q = blockIdx.y;
  const long long n = *p.d_base + p.k;
  if (n < 1) return;
  const int nth = p.n_theta;
  const double* lo = p.uin + ((size_t)mode * p.n_r + p.obs[q].i0) * 4 * nth;
  const double* hi = lo + (size_t)4 * nth;
  const double f = p.obs[q].f;
  double wr = 0.0, wi = 0.0;
  // same lane -> column ownership and summation order as the in-kernel tap (bitwise identical)
  const int vreq = (nth + 31) / 32;
  const int V = vreq <= 1 ? 1 : (vreq <= 2 ? 2 : (vreq <= 4 ? 4 : 8));
  for (int v = 0; v < V; ++v) {
    const int j = lane * V + v;
    if (j >= nth) break;
    const double wt = p.obs[q].weights[j];
    wr = fma(wt, fma(f, hi[j], (1.0 - f) * lo[j]), wr);
    wi = fma(wt, fma(f, hi[nth + j], (1.0 - f) * lo[nth + j]), wi);
  }
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

// d_base += inc (one thread; ends a CUDA-graph batch so that replays see the right time level).
__global__ void teuk_bump_kernel(long long* d_base, long long inc) { *d_base += inc; }
__global__ void teuk_set_base_kernel(long long* d_base, long long v) { *d_base = v; }

// Boundary layout [comp][mode][i][j] (one array per component, may be NULL) <-> internal
// [mode][i][comp][j].  `planes` are 4 device pointers.
struct Planes {
  double* c[4];
};
__global__ void teuk_pack_kernel(double* __restrict__ u, Planes src, size_t n_rows, int nth) {
  const size_t t = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (t >= n_rows * nth) return;
  const size_t row = t / nth;
  const int j = (int)(t - row * nth);
#pragma unroll
  for (int c = 0; c < 4; ++c) u[(row * 4 + c) * nth + j] = src.c[c] ? src.c[c][t] : 0.0;
}
__global__ void teuk_unpack_kernel(const double* __restrict__ u, Planes dst, size_t n_rows, int nth) {
  const size_t t = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (t >= n_rows * nth) return;
  const size_t row = t / nth;
  const int j = (int)(t - row * nth);
#pragma unroll
  for (int c = 0; c < 4; ++c)
    if (dst.c[c]) dst.c[c][t] = u[(row * 4 + c) * nth + j];
}

// ---- host-side launchers (called from teuk_api.cu) -------------------------------------------
template <int V>
static cudaError_t launch_v(const StepParams& p, cudaStream_t st) {
  const int warps_per_block = 4;
  dim3 grid((p.n_slabs + warps_per_block - 1) / warps_per_block, p.n_modes), block(32 * warps_per_block);
  if (p.n_theta % V == 0) {
    const size_t dyn = (size_t)warps_per_block * 2 * 4 * p.n_theta * sizeof(double);
    static bool attr_set = false;   // per instantiation
    if (!attr_set) {
      cudaError_t e = cudaFuncSetAttribute(teuk_step_kernel<V, true>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                           (int)((size_t)warps_per_block * 2 * 4 * 32 * V * sizeof(double)));
      if (e != cudaSuccess) return e;
      attr_set = true;
    }
    teuk_step_kernel<V, true><<<grid, block, dyn, st>>>(p);
  } else {
    teuk_step_kernel<V, false><<<grid, block, 0, st>>>(p);
  }
  return cudaGetLastError();
}

cudaError_t teuk_launch_step(const StepParams& p, cudaStream_t st) {
  const int v = (p.n_theta + 31) / 32;
  if (v <= 1) return launch_v<1>(p, st);
  if (v <= 2) return launch_v<2>(p, st);
  if (v <= 4) return launch_v<4>(p, st);
  return launch_v<8>(p, st);
}

cudaError_t teuk_launch_flush_tap(const StepParams& p, cudaStream_t st) {
  if (p.n_obs == 0) return cudaSuccess;
  teuk_flush_tap_kernel<<<dim3(p.n_modes, p.n_obs), 32, 0, st>>>(p);
  return cudaGetLastError();
}

cudaError_t teuk_launch_bump(long long* d_base, long long inc, cudaStream_t st) {
  teuk_bump_kernel<<<1, 1, 0, st>>>(d_base, inc);
  return cudaGetLastError();
}

cudaError_t teuk_launch_set_base(long long* d_base, long long v, cudaStream_t st) {
  teuk_set_base_kernel<<<1, 1, 0, st>>>(d_base, v);
  return cudaGetLastError();
}

cudaError_t teuk_launch_pack(double* u, double* const src[4], size_t n_rows, int nth, cudaStream_t st) {
  Planes pl;
  for (int c = 0; c < 4; ++c) pl.c[c] = src[c];
  const size_t n = n_rows * nth;
  teuk_pack_kernel<<<(unsigned)((n + 255) / 256), 256, 0, st>>>(u, pl, n_rows, nth);
  return cudaGetLastError();
}

cudaError_t teuk_launch_unpack(const double* u, double* const dst[4], size_t n_rows, int nth, cudaStream_t st) {
  Planes pl;
  for (int c = 0; c < 4; ++c) pl.c[c] = dst[c];
  const size_t n = n_rows * nth;
  teuk_unpack_kernel<<<(unsigned)((n + 255) / 256), 256, 0, st>>>(u, pl, n_rows, nth);
  return cudaGetLastError();
}
