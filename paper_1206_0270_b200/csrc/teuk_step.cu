// teuk_step.cu -- the hot path: one two-step Lax-Wendroff iteration (Eq. 3-4)
// of u = {Phi, Pi} per launch, all modes, fused with the pole ghosts and radial edges
// (PAPER.md:104), the Gaussian source deposit and the waveform tap
// (PAPER.md:161).  Hand-written for sm_100a; no tensor cores (a stencil, not a contraction).
//
// Mapping: theta is the fastest index and one WARP spans the whole theta
// range (n_theta <= 128; wider grids are cut into theta segments with a redundant halo, SEG), each
// lane owning V = 1, 2 or 4 contiguous columns, so the theta-neighbours of the centred
// differences are register neighbours or one warp shuffle.  Each warp
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
//
// Loop structure of teuk_step_kernel (round 2): an outer loop over chunks of RT_CH = 16 rows does everything that
// is rare or per-chunk (r-table chunk hand-over, the radial deposit profile of the chunk's rows -- one exp per lane,
// kept in a register and fetched by shuffle --, the waveform tap of observers in the chunk), and the inner loop is
// the marching iteration proper, instantiated twice with the roles of the row / half-row registers swapped (no
// register rotation): two stages, one TMA issue, one row store.  With the cold code (exp and division slow paths
// of the deposit, the tap) inlined three times INSIDE the marching loop, as in round 1, the V = 2 kernel spent 16 %
// of its stall samples waiting for instructions and ran 566 instructions per warp-row for 257 FP64 ones: config 3
// 64 -> 89 GPts/s, config 4 72 -> 81-87 with this structure, bit-identical results (profiles/r2_bench.md).
//
// Kernels in this file: teuk_step_kernel (register-resident marching kernel, the default; template flags
// VEC = vector/TMA path, CM = coefficients rebuilt / streamed planes, SEG = theta segments, FULLW =
// n_theta == 32 V compile-time, TERMS = multi-term deposit), teuk_step_smem_kernel (same arithmetic, state in shared memory; bitwise
// cross-check), teuk_flush_tap_kernel, pack/unpack and counter kernels.  The compile-time knobs below
// record what was measured on config 5 (profiles/r1_step_kernel_full.md); the defaults are the winners.
#include <cuda_runtime.h>
#include <math.h>
#include <stdint.h>

#include "teuk_internal.h"

#include "teuk_stage.cuh"

// SEG: the theta range is split into gridDim.z segments of p.seg_payload columns (n_theta > 32 V, e.g. the
// paper's 32000 x 304 grid).  A warp then owns a window of 32 V columns: its payload plus a
// 4-column halo on each side, recomputed redundantly (the stencil reaches 2 columns per iteration), so no
// exchange between warps is needed; only payload columns are stored.
// FULLW: n_theta == 32 V exactly (all five BASELINE.json configs): n_theta becomes a compile-time constant,
// every lane is valid, and all per-lane bounds predicates fold away.
// Resident blocks per SM: V = 2 fits 160 registers without spills -> 3 blocks (12 warps; measured +5-9 %);
// V = 4 needs all 255 registers -> 2 blocks; V = 1 lands at ~120 registers -> 4 blocks either way.
// Measured and rejected for V = 4 (config 5, same box, base 88.6-92.0 GPts/s): 9 warps per SM (96-thread
// blocks, __maxnreg__(224): 388 B of spill stores) 69.6; bracket B accumulated in two partial sums
// (shorter dependent chains, more spills) 89.1.
// TERMS: the deposit is a sum of rank-1 terms with derivative profiles (teuk_set_source_terms)
// instead of the single term of the trajectory table; a separate instantiation, so that the default kernel's code
// and register allocation do not change with it.
template <int V, bool VEC, int CM, bool SEG, bool FULLW, bool TERMS = false>
__global__ void __launch_bounds__(128, (V == 2 ? TEUK_V2_BLOCKS : TEUK_MIN_BLOCKS)) teuk_step_kernel(const __grid_constant__ StepParams p) {
  const int lane = threadIdx.x & 31;
  // warp index broadcast from lane 0: tells the compiler that everything derived from it (slab bounds, loop
  // trip count, the early exit) is warp-uniform, so the warp stays provably converged: no BRA.DIV guards
  // around the shuffles, uniform-datapath address arithmetic, larger basic blocks to schedule.
  const int wib_u = __shfl_sync(FULL, (int)(threadIdx.x >> 5), 0);
  const int slab = blockIdx.x * (blockDim.x >> 5) + wib_u;
  const int mode = blockIdx.y;
  const int nth = FULLW ? 32 * V : p.n_theta, nr = p.n_r;
  if (slab >= p.n_slabs) return;
  const int r0 = slab_first_row(p, slab);            // first interior node of this slab
  const int r1 = slab_first_row(p, slab + 1);        // one past the last
  const int c_lo = SEG ? (int)blockIdx.z * p.seg_payload - 4 : 0;            // first column of the window
  const int pay_lo = SEG ? (int)blockIdx.z * p.seg_payload : 0;
  const int pay_hi = SEG ? min(pay_lo + p.seg_payload, nth) : nth;
  const int j0 = c_lo + lane * V;                    // may be negative or >= nth in a segment's halo
  const int slot_cs = SEG ? 32 * V : nth;            // component stride inside a landing slot
  const size_t row_stride = (size_t)4 * nth;
  const double* __restrict__ uin = p.uin + (size_t)mode * nr * row_stride;
  double* __restrict__ uout = p.uout + (size_t)mode * nr * row_stride;
  const double* __restrict__ rtab = p.rtab + (size_t)mode * (2 * nr - 1) * RT_N;
  __shared__ __align__(16) double s_rt[4][2][RT_CHUNK_DOUBLES];
  constexpr int NS = TEUK_SLOTS;
  __shared__ __align__(8) unsigned long long s_bar[4][NS];
  extern __shared__ __align__(128) unsigned char s_dyn[];   // VEC: [warp][TEUK_SLOTS][4 n_theta] doubles
  const int wib = wib_u;
  double* const rt_buf = &s_rt[wib][0][0];
  stage_rtab_chunk(rt_buf, rtab, 2 * r0, 2 * nr - 1, lane);
  const unsigned row_bytes = (unsigned)(row_stride * sizeof(double));
  const size_t slot_doubles = (size_t)4 * slot_cs;
  double* const slot0 = reinterpret_cast<double*>(s_dyn) + (size_t)wib * NS * slot_doubles;
  unsigned long long* const bars = &s_bar[wib][0];
  // One TMA bulk copy per row (whole row), or four (one per component) for a theta segment's window.
  const int g_lo = max(c_lo, 0), g_hi = min(c_lo + 32 * V, nth);
  const unsigned slot0_u32 = smem_u32(slot0), bars_u32 = smem_u32(bars);
  auto issue_row = [&](int q) {
    double* dst = slot0 + (size_t)(q % NS) * slot_doubles;
    const double* src = uin + (size_t)q * row_stride;
    if (!SEG) {
      tma_load_row_u32(slot0_u32 + (unsigned)((q % NS) * slot_doubles * sizeof(double)), src, row_bytes,
                       bars_u32 + 8u * (unsigned)(q % NS));
    } else {
      const unsigned bytes = (unsigned)((g_hi - g_lo) * sizeof(double));
      asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(&bars[q % NS])), "r"(4u * bytes) : "memory");
#pragma unroll
      for (int c = 0; c < 4; ++c)
        asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                     ::"r"(smem_u32(dst + c * slot_cs + (g_lo - c_lo))), "l"(src + (size_t)c * nth + g_lo), "r"(bytes),
                     "r"(smem_u32(&bars[q % NS])) : "memory");
    }
  };
  const long long n = *p.d_base + p.k;               // index of the input time level (step kernels never write it)
  if (VEC && lane == 0) {
#pragma unroll
    for (int q = 0; q < NS; ++q) mbar_init(&bars[q], 1);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
  }

  ThetaTab<V> th;
  {
    const double* tb = p.ttab + (size_t)mode * TT_N * nth;
#pragma unroll
    for (int v = 0; v < V; ++v) {
      const bool ok = (unsigned)(j0 + v) < (unsigned)nth;
      th.vals.s2[v] = ok ? tb[TT_S2 * nth + j0 + v] : 0.0;
      th.vals.cs[v] = ok ? tb[TT_COS * nth + j0 + v] : 0.0;
      th.vals.ap[v] = ok ? tb[TT_AP * nth + j0 + v] : 0.0;
      th.vals.am[v] = ok ? tb[TT_AM * nth + j0 + v] : 0.0;
      th.vals.d0[v] = ok ? tb[TT_D0 * nth + j0 + v] : 0.0;
    }
  }
  typename SourceSel<V, TERMS>::type src_h, src_f;   // half stage: sample 2n at half points; full stage: 2n+1 at nodes
  __shared__ double s_tp[TERMS ? 4 * 2 * TermTab<V>::PER_STAGE : 1];   // theta-profile tables of the multi-term deposit
  if constexpr (TERMS) {
    src_h.tab = &s_tp[(wib_u * 2 + 0) * TermTab<V>::PER_STAGE];
    src_f.tab = &s_tp[(wib_u * 2 + 1) * TermTab<V>::PER_STAGE];
  }
  setup_source<V>(src_h, p, mode, 2 * n, true, r0 - 1, r1 - 1, lane, c_lo);
  setup_source<V>(src_f, p, mode, 2 * n + 1, false, r0, r1 - 1, lane, c_lo);
  bool do_tap = !SEG && p.tap_enable && p.n_obs > 0 && n >= 1;   // segments: separate tap kernel
  if (do_tap) {  // only the warp whose slab holds an observer's rows i0, i0+1 ever taps
    bool mine = false;
    for (int q = 0; q < p.n_obs; ++q) mine = mine || (p.obs[q].i0 >= r0 - 1 && p.obs[q].i0 < r1);
    do_tap = mine;
  }
  const bool any_src = __any_sync(FULL, src_h.on || src_f.on);   // vote result: provably warp-uniform
  const double tau_h = 0.5 * p.dt, tau_f = 0.25 * p.dt, tdx = 2.0 / p.dx;

  // Programmatic dependent launch: when the host launched this grid with the stream-serialisation attribute
  // (iterations 2..32 of a CUDA-graph batch), everything above -- index arithmetic, the first r-table chunk, the
  // theta tables, the source window and deposit profile, none of which a step kernel writes -- ran while the
  // previous iteration was still finishing.  From here on the previous iteration's output (our input) is read and
  // its input (our output) overwritten: wait for it, and let the next iteration's grid start its own prologue as
  // soon as SM slots free up.  (Without the attribute both instructions do nothing.)
  asm volatile("griddepcontrol.wait;" ::: "memory");
  asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
  if (VEC) {
    if (lane == 0) {
      // row q lands in slot q % NS; rows r0+2 .. r0+NS go out now, row i+NS+1 in the middle of iteration i
#pragma unroll
      for (int q = 2; q <= NS; ++q)
        if (r0 + q <= r1) issue_row(r0 + q);
    }
    __syncwarp();
  }

  Row<V> ua, ub, uc, hp, hn, out;
  load_row<V, VEC>(ua, uin + (size_t)(r0 - 1) * row_stride, nth, j0);
  load_row<V, VEC>(ub, uin + (size_t)r0 * row_stride, nth, j0);
  load_row<V, VEC>(uc, uin + (size_t)(r0 + 1) * row_stride, nth, j0);
  if (do_tap && r0 == 1) tap<V>(ua, ub, p, 0, mode, n, lane);
  const double* __restrict__ planes = nullptr;   // coef_mode 1: [2 nr - 1][8][nth] of this mode
  if (CM == 1) planes = p.coef2d + (size_t)mode * (2 * nr - 1) * 8 * nth;
  const size_t loc_stride = (size_t)8 * nth;
  if (CM == 1)
    lw_stage_planes<V, true, VEC>(ua, ub, ua, planes + (size_t)(2 * (r0 - 1) + 1) * loc_stride, th, tau_h, hp, nth, j0);
  else
    lw_stage<V, true>(ua, ub, ua, rtab + (size_t)(2 * (r0 - 1) + 1) * RT_N, th, tau_h, tdx, hp);
  add_source<V>(hp, src_h, p, r0 - 1, true);

  const double* rt_cur = rt_buf;
  // Work that is rare or happens once per RT_CH rows is kept OUT of the marching iteration, in chunk_begin: the
  // r-table chunk hand-over, the radial deposit profile of the chunk's rows (one exp per lane: lanes 0-15 hold
  // dt * P(x_{i+1/2} - x_p) of the half stage for rows cb .. cb+15, lanes 16-31 dt * P(x_i - x_p) of the full stage;
  // the marching iteration fetches its row's value with one shuffle), and the waveform tap of observers whose cell
  // starts in the chunk (read from the input level in global memory: same values as the register rows, same
  // summation order).  The marching iteration is then two stages, one TMA issue, one store and nothing else: a
  // short hot loop without cold branches in it.
  double gprof = 0.0, gprof1 = 0.0, gprof2 = 0.0;
  auto chunk_begin = [&](const int cb) {
    asm volatile("cp.async.wait_group 0;" ::: "memory");
    __syncwarp();
    const int c = (cb - r0) / RT_CH;
    rt_cur = rt_buf + (c & 1) * RT_CHUNK_DOUBLES;
    if (cb + RT_CH < r1)
      stage_rtab_chunk(rt_buf + ((c + 1) & 1) * RT_CHUNK_DOUBLES, rtab, 2 * (cb + RT_CH), 2 * nr - 1, lane);
    if (!TERMS && any_src) {
      const bool hf = lane < 16;
      const int i = cb + (lane & 15);
      const bool on = hf ? src_h.on : src_f.on;
      const int ip = hf ? src_h.ip : src_f.ip;
      double g = 0.0;
      if (on && i < r1 && abs(i - ip) <= p.W) {
        double x = __dadd_rn(p.rs_min, __dmul_rn((double)i, p.dx));
        if (hf) x = __dadd_rn(x, __dmul_rn(0.5, p.dx));
        g = p.dt * deposit_profile(p.source_kind, x - (hf ? src_h.xp : src_f.xp), p.sigma_r);
      }
      gprof = g;
    }
    if (TERMS && any_src) {    // multi-term deposit: the three radial profile values of this lane's row (0 outside the window)
      const bool hf = lane < 16;
      const int i = cb + (lane & 15);
      const bool on = hf ? src_h.on : src_f.on;
      const int ip = hf ? src_h.ip : src_f.ip;
      Profile3 g3;
      g3.d[0] = g3.d[1] = g3.d[2] = 0.0;
      if (on && i < r1 && abs(i - ip) <= p.W) {
        double x = __dadd_rn(p.rs_min, __dmul_rn((double)i, p.dx));
        if (hf) x = __dadd_rn(x, __dmul_rn(0.5, p.dx));
        g3 = deposit_profile3(p.source_kind, x - (hf ? src_h.xp : src_f.xp), p.sigma_r);
      }
      gprof = g3.d[0];
      gprof1 = g3.d[1];
      gprof2 = g3.d[2];
    }
    if (do_tap) {
      for (int q = 0; q < p.n_obs; ++q) {
        const int i0 = p.obs[q].i0;
        if (i0 < cb || i0 >= min(cb + RT_CH, r1)) continue;
        const double* lo = uin + (size_t)i0 * row_stride;
        const double* hi = lo + row_stride;
        const double f = p.obs[q].f;
        double wr = 0.0, wi = 0.0;
#pragma unroll
        for (int v = 0; v < V; ++v) {
          const int j = lane * V + v;
          const bool ok = j < p.n_theta;
          const double wt = ok ? __ldg(p.obs[q].weights + j) : 0.0;
          const double lr = ok ? lo[j] : 0.0, li = ok ? lo[nth + j] : 0.0;
          const double hr = ok ? hi[j] : 0.0, hi_i = ok ? hi[nth + j] : 0.0;
          wr = fma(wt, fma(f, hr, (1.0 - f) * lr), wr);
          wi = fma(wt, fma(f, hi_i, (1.0 - f) * li), wi);
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
  };
  // dt * T on this lane's columns of row i: g = the row's radial profile value (0 outside the window)
  auto deposit = [&](Row<V>& o_, const typename SourceSel<V, TERMS>::type& s_, const double g) {
    if constexpr (!TERMS) {
      if (g != 0.0) {
#pragma unroll
        for (int q = 0; q < V; ++q) {
          const double gg = g * s_.gth[q];
          o_.c[2][q] = fma(s_.are, gg, o_.c[2][q]);
          o_.c[3][q] = fma(s_.aim, gg, o_.c[3][q]);
        }
      }
    }
  };
  // One marching iteration at node i.  On entry A = u^n_i, B = u^n_{i+1}, Hp = 2 u^{n+1/2}_{i-1/2};
  // on exit Hn = 2 u^{n+1/2}_{i+1/2} and A = u^n_{i+2}.  The caller alternates the roles of
  // (A, B) and (Hp, Hn), so no register rotation is needed.
  auto march = [&](const int i, Row<V>& A, Row<V>& B, Row<V>& Hp, Row<V>& Hn) {
    if (!VEC) {  // scalar fallback: prefetch row i+2 with plain loads
      if (i + 2 <= r1) load_row<V, VEC>(ua, uin + (size_t)(i + 2) * row_stride, nth, j0);
    }
    const int o = (i - r0) & (RT_CH - 1);
    if (CM == 1) {
      // pull the next iteration's two coefficient rows (2 x 8 planes) towards L2 while this one computes
      if (i + 1 < r1) {
        const char* nxt = reinterpret_cast<const char*>(planes + (size_t)(2 * (i + 1)) * loc_stride);
        for (unsigned off = lane * 128u; off < 2u * (unsigned)loc_stride * 8u; off += 32u * 128u)
          asm volatile("prefetch.global.L2 [%0];" ::"l"(nxt + off));
      }
      lw_stage_planes<V, true, VEC>(A, B, A, planes + (size_t)(2 * i + 1) * loc_stride, th, tau_h, Hn, nth, j0);
    } else {
      lw_stage<V, true>(A, B, A, rt_cur + (2 * o + 1) * RT_N, th, tau_h, tdx, Hn);
    }
    if (any_src) {
      if constexpr (TERMS) {
        Profile3 pr;
        pr.d[0] = __shfl_sync(FULL, gprof, o);
        pr.d[1] = __shfl_sync(FULL, gprof1, o);
        pr.d[2] = __shfl_sync(FULL, gprof2, o);
        if (pr.d[0] != 0.0 || pr.d[1] != 0.0 || pr.d[2] != 0.0) add_source_row<V>(Hn, src_h, p, pr);
      }
      else deposit(Hn, src_h, __shfl_sync(FULL, gprof, o));
    }
    if (VEC) {
      // B (row i+1, copied out of slot (i+1) % NS at the end of the last iteration) has been consumed by
      // every lane: its slot may now receive row i+NS+1.
      __syncwarp();
      if (lane == 0 && i + NS + 1 <= r1) issue_row(i + NS + 1);
    }
    if (CM == 1)
      lw_stage_planes<V, false, VEC>(Hp, Hn, A, planes + (size_t)(2 * i) * loc_stride, th, tau_f, out, nth, j0);
    else
      lw_stage<V, false>(Hp, Hn, A, rt_cur + (2 * o) * RT_N, th, tau_f, tdx, out);
    if (any_src) {
      if constexpr (TERMS) {
        Profile3 pr;
        pr.d[0] = __shfl_sync(FULL, gprof, 16 + o);
        pr.d[1] = __shfl_sync(FULL, gprof1, 16 + o);
        pr.d[2] = __shfl_sync(FULL, gprof2, 16 + o);
        if (pr.d[0] != 0.0 || pr.d[1] != 0.0 || pr.d[2] != 0.0) add_source_row<V>(out, src_f, p, pr);
      }
      else deposit(out, src_f, __shfl_sync(FULL, gprof, 16 + o));
    }
    store_row<V, VEC>(out, uout + (size_t)i * row_stride, nth, j0, pay_lo, pay_hi);
    if (VEC) {
      if (i + 2 <= r1) {
        mbar_wait_u32(bars_u32 + 8u * (unsigned)((i + 2) % NS), (unsigned)((i - r0) / NS) & 1u);
        lds_row<V>(A, slot0 + (size_t)((i + 2) % NS) * slot_doubles, slot_cs, lane * V, (unsigned)j0 < (unsigned)nth);
      }
    } else {
      A = ua;
    }
  };
  static_assert(RT_CH == 16, "chunk_begin keeps one chunk's deposit profile in the two halves of a warp");
  for (int cb = r0; cb < r1; cb += RT_CH) {
    chunk_begin(cb);
    const int ce = min(cb + RT_CH, r1);
    int i = cb;
#pragma unroll 1
    for (; i + 1 < ce; i += 2) {
      march(i, ub, uc, hp, hn);
      march(i + 1, uc, ub, hn, hp);
    }
    if (i < ce) march(i, ub, uc, hp, hn);     // odd row count: only the last chunk can have one
  }

  // radial edges (outer edge: DESIGN.md reading A6)
  if (r0 == 1) {
#pragma unroll
    for (int c = 0; c < 4; ++c)
#pragma unroll
      for (int v = 0; v < V; ++v) out.c[c][v] = 0.0;
    store_row<V, VEC>(out, uout, nth, j0, pay_lo, pay_hi);
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
    store_row<V, VEC>(out, uout + (size_t)(nr - 1) * row_stride, nth, j0, pay_lo, pay_hi);
  }
}

// ================================================================================================
// Shared-memory-resident variant (variant 1).  Same arithmetic per point as teuk_step_kernel (the
// two produce bitwise identical fields), different residency: only u^n_i lives in registers across
// iterations; u^n_{i+1} is read from its TMA landing slot where it is used, and the half-step row
// 2u^{n+1/2}_{i-1/2} lives in a per-warp shared-memory slot.  That brings the kernel under 168
// registers, i.e. 12 instead of 8 warps per SM, which is what the fixed-latency `wait` stalls of the
// register-resident kernel ask for (profiles/r1_step_kernel_full.md).  Lane <-> column mapping MAP 1.
namespace {

template <int V, bool EVEN>
__device__ __forceinline__ void piece_load(Row<V>& u, const double* row, int nth, int lane) {
#pragma unroll
  for (int c = 0; c < 4; ++c) {
    if (V == 1) {
      u.c[c][0] = (lane < nth) ? row[c * nth + lane] : 0.0;
    } else {
#pragma unroll
      for (int q = 0; q < V / 2; ++q) {
        const int j = q * 64 + 2 * lane;
        if (EVEN) {
          double2 t = make_double2(0.0, 0.0);
          if (j < nth) t = *reinterpret_cast<const double2*>(row + c * nth + j);
          u.c[c][2 * q] = t.x;
          u.c[c][2 * q + 1] = t.y;
        } else {
          u.c[c][2 * q] = (j < nth) ? row[c * nth + j] : 0.0;
          u.c[c][2 * q + 1] = (j + 1 < nth) ? row[c * nth + j + 1] : 0.0;
        }
      }
    }
  }
}

template <int V, bool EVEN>
__device__ __forceinline__ void piece_store_global(const Row<V>& u, double* __restrict__ row, int nth, int lane) {
#pragma unroll
  for (int c = 0; c < 4; ++c) {
    if (V == 1) {
      if (lane < nth) __stcs(row + c * nth + lane, u.c[c][0]);
    } else {
#pragma unroll
      for (int q = 0; q < V / 2; ++q) {
        const int j = q * 64 + 2 * lane;
        if (EVEN) {
          if (j < nth) __stcs(reinterpret_cast<double2*>(row + c * nth + j), make_double2(u.c[c][2 * q], u.c[c][2 * q + 1]));
        } else {
          if (j < nth) __stcs(row + c * nth + j, u.c[c][2 * q]);
          if (j + 1 < nth) __stcs(row + c * nth + j + 1, u.c[c][2 * q + 1]);
        }
      }
    }
  }
}

// private half-row slot: [comp][piece][lane] 16-byte entries (V = 1: [comp][lane] doubles)
template <int V>
__device__ __forceinline__ void hslot_store(const Row<V>& h, double* slot, int lane) {
#pragma unroll
  for (int c = 0; c < 4; ++c) {
    if (V == 1) {
      slot[c * 32 + lane] = h.c[c][0];
    } else {
#pragma unroll
      for (int q = 0; q < V / 2; ++q)
        *reinterpret_cast<double2*>(slot + ((c * (V / 2) + q) * 32 + lane) * 2) = make_double2(h.c[c][2 * q], h.c[c][2 * q + 1]);
    }
  }
}
template <int V>
__device__ __forceinline__ void hslot_load(Row<V>& h, const double* slot, int lane) {
#pragma unroll
  for (int c = 0; c < 4; ++c) {
    if (V == 1) {
      h.c[c][0] = slot[c * 32 + lane];
    } else {
#pragma unroll
      for (int q = 0; q < V / 2; ++q) {
        const double2 t = *reinterpret_cast<const double2*>(slot + ((c * (V / 2) + q) * 32 + lane) * 2);
        h.c[c][2 * q] = t.x;
        h.c[c][2 * q + 1] = t.y;
      }
    }
  }
}

}  // namespace

#ifndef TEUK_SMEM_MIN_BLOCKS
#define TEUK_SMEM_MIN_BLOCKS 3
#endif
#ifndef TEUK_SMEM_TT
#define TEUK_SMEM_TT 0   // 1: theta tables of the shared-memory-resident kernel in shared memory too (no gain measured)
#endif

template <int V, bool EVEN>
__global__ void __launch_bounds__(128, TEUK_SMEM_MIN_BLOCKS) teuk_step_smem_kernel(const __grid_constant__ StepParams p) {
  const int lane = threadIdx.x & 31;
  const int wib = __shfl_sync(FULL, (int)(threadIdx.x >> 5), 0);   // provably warp-uniform (see teuk_step_kernel)
  const int slab = blockIdx.x * (blockDim.x >> 5) + wib;
  const int mode = blockIdx.y;
  const int nth = p.n_theta, nr = p.n_r;
#if TEUK_SMEM_TT
  __shared__ __align__(16) double s_tt[TT_N * 32 * V];
  for (int t = threadIdx.x; t < TT_N * 32 * V; t += blockDim.x) {
    const int k = t / (32 * V), j = t - k * 32 * V;
    s_tt[t] = (j < nth) ? p.ttab[((size_t)mode * TT_N + k) * nth + j] : 0.0;
  }
  __syncthreads();
#endif
  if (slab >= p.n_slabs) return;
  const int r0 = slab_first_row(p, slab);
  const int r1 = slab_first_row(p, slab + 1);
  const size_t row_stride = (size_t)4 * nth;
  const double* __restrict__ uin = p.uin + (size_t)mode * nr * row_stride;
  double* __restrict__ uout = p.uout + (size_t)mode * nr * row_stride;
  const double* __restrict__ rtab = p.rtab + (size_t)mode * (2 * nr - 1) * RT_N;
  const long long n = *p.d_base + p.k;

  __shared__ __align__(16) double s_rt[4][2][RT_CHUNK_DOUBLES];
  __shared__ __align__(8) unsigned long long s_bar[4][2];
  extern __shared__ __align__(128) unsigned char s_dyn[];  // per warp: 2 row slots + 1 half-row slot
  const size_t warp_doubles = 2 * row_stride + (size_t)4 * 32 * V;
  double* const slot0 = reinterpret_cast<double*>(s_dyn) + (size_t)wib * warp_doubles;
  double* const hslot = slot0 + 2 * row_stride;
  double* const rt_buf = &s_rt[wib][0][0];
  unsigned long long* const bars = &s_bar[wib][0];
  const unsigned row_bytes = (unsigned)(row_stride * sizeof(double));
  // row q uses slot q & 1; its k-th use of the slot has mbarrier parity k & 1
  auto slot_of = [&](int q) { return slot0 + (size_t)(q & 1) * row_stride; };
  auto issue = [&](int q) { tma_load_row(slot_of(q), uin + (size_t)q * row_stride, row_bytes, &bars[q & 1]); };
  auto wait_row = [&](int q) { mbar_wait(&bars[q & 1], (unsigned)((q - (r0 - 1)) >> 1) & 1u); };

  if (lane == 0) {
    mbar_init(&bars[0], 1);
    mbar_init(&bars[1], 1);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
    issue(r0 - 1);
    issue(r0);
  }
  __syncwarp();
  stage_rtab_chunk(rt_buf, rtab, 2 * r0, 2 * nr - 1, lane);

#if TEUK_SMEM_TT
  ThetaTabShared<V> th;
  th.base = s_tt;
  th.stride = 32 * V;
  th.lane = lane;
  typedef ThetaTabShared<V> TTab;
#else
  ThetaTab<V> th;
  {
    const double* tb = p.ttab + (size_t)mode * TT_N * nth;
#pragma unroll
    for (int v = 0; v < V; ++v) {
      const int j = col_of<V, 1>(lane, v);
      const bool ok = j < nth;
      th.vals.s2[v] = ok ? tb[TT_S2 * nth + j] : 0.0;
      th.vals.cs[v] = ok ? tb[TT_COS * nth + j] : 0.0;
      th.vals.ap[v] = ok ? tb[TT_AP * nth + j] : 0.0;
      th.vals.am[v] = ok ? tb[TT_AM * nth + j] : 0.0;
      th.vals.d0[v] = ok ? tb[TT_D0 * nth + j] : 0.0;
    }
  }
  typedef ThetaTab<V> TTab;
#endif
  StageSource<V> src_h, src_f;
  setup_source<V, 1>(src_h, p, mode, 2 * n, true, r0 - 1, r1 - 1, lane);
  setup_source<V, 1>(src_f, p, mode, 2 * n + 1, false, r0, r1 - 1, lane);
  const bool do_tap = p.tap_enable && p.n_obs > 0 && n >= 1;
  const double tau_h = 0.5 * p.dt, tau_f = 0.25 * p.dt, tdx = 2.0 / p.dx;

  Row<V> A, out;
  {  // prologue: half step at (r0-1)+1/2
    Row<V> B, H;
    wait_row(r0 - 1);
    wait_row(r0);
    piece_load<V, EVEN>(A, slot_of(r0 - 1), nth, lane);
    piece_load<V, EVEN>(B, slot_of(r0), nth, lane);
    if (do_tap && r0 == 1) tap<V, 1>(A, B, p, 0, mode, n, lane);
    lw_stage<V, true, 1, TTab>(A, B, A, rtab + (size_t)(2 * (r0 - 1) + 1) * RT_N, th, tau_h, tdx, H, lane);
    add_source<V>(H, src_h, p, r0 - 1, true);
    hslot_store<V>(H, hslot, lane);
    A = B;
    __syncwarp();
    if (lane == 0) issue(r0 + 1);   // into the slot of row r0-1, read by every lane above
    wait_row(r0 + 1);
  }

  const double* rt_cur = rt_buf;
  for (int i = r0; i < r1; ++i) {
    // A = u^n_i (registers); u^n_{i+1} has landed in slot (i+1)&1; hslot = 2 u^{n+1/2}_{i-1/2}
    __syncwarp();
    if (lane == 0 && i + 2 <= r1) issue(i + 2);   // slot i&1: row i was copied into A by every lane
    const int o = (i - r0) & (RT_CH - 1);
    if (o == 0) {
      asm volatile("cp.async.wait_group 0;" ::: "memory");
      __syncwarp();
      const int c = (i - r0) / RT_CH;
      rt_cur = rt_buf + (c & 1) * RT_CHUNK_DOUBLES;
      if (i + RT_CH < r1)
        stage_rtab_chunk(rt_buf + ((c + 1) & 1) * RT_CHUNK_DOUBLES, rtab, 2 * (i + RT_CH), 2 * nr - 1, lane);
    }
    Row<V> Hn;
    {
      Row<V> B;
      piece_load<V, EVEN>(B, slot_of(i + 1), nth, lane);
      if (do_tap) tap<V, 1>(A, B, p, i, mode, n, lane);
      lw_stage<V, true, 1, TTab>(A, B, A, rt_cur + (2 * o + 1) * RT_N, th, tau_h, tdx, Hn, lane);
      add_source<V>(Hn, src_h, p, i, true);
    }
    {
      Row<V> Hp;
      hslot_load<V>(Hp, hslot, lane);
      lw_stage<V, false, 1, TTab>(Hp, Hn, A, rt_cur + (2 * o) * RT_N, th, tau_f, tdx, out, lane);
      add_source<V>(out, src_f, p, i, false);
    }
    piece_store_global<V, EVEN>(out, uout + (size_t)i * row_stride, nth, lane);
    hslot_store<V>(Hn, hslot, lane);
    piece_load<V, EVEN>(A, slot_of(i + 1), nth, lane);   // u^n_{i+1} becomes the register row
    if (i + 2 <= r1) wait_row(i + 2);
  }

  if (r0 == 1) {
#pragma unroll
    for (int c = 0; c < 4; ++c)
#pragma unroll
      for (int v = 0; v < V; ++v) out.c[c][v] = 0.0;
    piece_store_global<V, EVEN>(out, uout, nth, lane);
  }
  if (r1 == nr - 1) {
    Row<V> L, K;
    piece_load<V, EVEN>(L, uin + (size_t)(nr - 1) * row_stride, nth, lane);
    piece_load<V, EVEN>(K, uin + (size_t)(nr - 2) * row_stride, nth, lane);
    const double eps = __ldg(rtab + (size_t)(2 * (nr - 1)) * RT_N + RT_EPS);
    ThetaVals<V> tv;
    th.get(tv);
#pragma unroll
    for (int v = 0; v < V; ++v) {
      if (p.outer_bc == 0) {
        const double b = rsqrt_near_one(fma(-eps, tv.s2[v], 1.0));
        out.c[0][v] = L.c[0][v] - p.dt * b * (L.c[0][v] - K.c[0][v]) / p.dx;
        out.c[1][v] = L.c[1][v] - p.dt * b * (L.c[1][v] - K.c[1][v]) / p.dx;
      } else {
        out.c[0][v] = 0.0;
        out.c[1][v] = 0.0;
      }
      out.c[2][v] = 0.0;
      out.c[3][v] = 0.0;
    }
    piece_store_global<V, EVEN>(out, uout + (size_t)(nr - 1) * row_stride, nth, lane);
  }
}

// ================================================================================================
// Temporal blocking, k = 2 ("temporal_block" = 2): two iterations per HBM round trip.
// Every slab is worked on by a PAIR of warps of the same block.  The producer warp is the marching
// kernel above for time level n -> n+1 on the slab's rows plus one halo row on each side, except that
// it never stores to HBM: each finished row of level n+1 goes into a small shared-memory ring.  The
// consumer warp marches over the same slab one level up (n+1 -> n+2), taking its input rows from the
// ring instead of from TMA landing slots, and stores level n+2.  Level n+1 never touches HBM: 32 B per
// point per iteration instead of 64.  Ring slots are handed over with a full/empty mbarrier pair per
// slot (count 1: lane 0 arrives after __syncwarp).  Same stage arithmetic (lw_stage), same results bit
// for bit as two k = 1 launches.
namespace {

#ifndef TEUK_TB_RING
#define TEUK_TB_RING 4
#endif
constexpr int TB_RING = TEUK_TB_RING;

__device__ __forceinline__ void mbar_arrive_u32(unsigned bar) {
  asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(bar) : "memory");
}

struct Tb2Shared {
  double* rt_buf;              // this warp's r-table chunk buffers
  double* slot0;               // producer: TMA landing slots of this pair
  double* ring;                // level n+1 rows, TB_RING slots of 4 n_theta doubles
  unsigned tma_u32, full_u32, empty_u32;   // shared addresses of the barrier arrays of this pair
};

// ROLE 0: producer (reads level n from HBM, pushes level n+1 rows r0-1 .. r1 into the ring)
// ROLE 1: consumer (pops them, stores level n+2 rows r0 .. r1-1, plus the grid-edge rows)
template <int V, bool FULLW, int ROLE>
__device__ __forceinline__ void tb2_warp(const StepParams& p, const Tb2Shared& sh, int lane, int mode, int r0, int r1) {
  const int nth = FULLW ? 32 * V : p.n_theta, nr = p.n_r;
  const int j0 = lane * V;
  const bool lane_ok = j0 < nth;
  const size_t row_stride = (size_t)4 * nth;
  const double* __restrict__ uin = p.uin + (size_t)mode * nr * row_stride;
  double* __restrict__ uout = p.uout + (size_t)mode * nr * row_stride;
  const double* __restrict__ rtab = p.rtab + (size_t)mode * (2 * nr - 1) * RT_N;
  const long long n = *p.d_base + p.k + ROLE;                 // time level this warp reads
  const int m0 = ROLE == 0 ? max(r0 - 1, 1) : r0;             // interior nodes [m0, m1) this warp updates
  const int m1 = ROLE == 0 ? min(r1 + 1, nr - 1) : r1;
  constexpr int NS = TEUK_SLOTS;
  const unsigned row_bytes = (unsigned)(row_stride * sizeof(double));
  const unsigned slot0_u32 = smem_u32(sh.slot0);
  auto issue_row = [&](int q) {
    tma_load_row_u32(slot0_u32 + (unsigned)((q % NS) * row_stride * sizeof(double)), uin + (size_t)q * row_stride,
                     row_bytes, sh.tma_u32 + 8u * (unsigned)(q % NS));
  };
  auto push = [&](const Row<V>& r, int q) {                   // row q of level n+1
    const int seq = q - (r0 - 1), s = seq % TB_RING;
    if (seq >= TB_RING) mbar_wait_u32(sh.empty_u32 + 8u * s, (unsigned)(seq / TB_RING - 1) & 1u);
    sts_row<V>(r, sh.ring + (size_t)s * row_stride, nth, j0);
    __syncwarp();
    if (lane == 0) mbar_arrive_u32(sh.full_u32 + 8u * s);
  };
  auto pop = [&](Row<V>& r, int q) {
    const int seq = q - (r0 - 1), s = seq % TB_RING;
    mbar_wait_u32(sh.full_u32 + 8u * s, (unsigned)(seq / TB_RING) & 1u);
    lds_row<V>(r, sh.ring + (size_t)s * row_stride, nth, j0, lane_ok);
    __syncwarp();
    if (lane == 0) mbar_arrive_u32(sh.empty_u32 + 8u * s);
  };

  stage_rtab_chunk(sh.rt_buf, rtab, 2 * m0, 2 * nr - 1, lane);
  if (ROLE == 0) {
    if (lane == 0) {
#pragma unroll
      for (int q = 2; q <= NS; ++q)
        if (m0 + q <= m1) issue_row(m0 + q);
    }
    __syncwarp();
  }
  ThetaTab<V> th;
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
  StageSource<V> src_h, src_f;
  setup_source<V>(src_h, p, mode, 2 * n, true, m0 - 1, m1 - 1, lane, 0);
  setup_source<V>(src_f, p, mode, 2 * n + 1, false, m0, m1 - 1, lane, 0);
  bool do_tap = (ROLE == 0 ? p.tap_enable : p.tap_enable2) && p.n_obs > 0 && n >= 1;
  if (do_tap) {
    bool mine = false;
    for (int q = 0; q < p.n_obs; ++q) mine = mine || (p.obs[q].i0 >= r0 - 1 && p.obs[q].i0 < r1);
    do_tap = mine;
  }
  const bool any_src = __any_sync(FULL, src_h.on || src_f.on);
  const double tau_h = 0.5 * p.dt, tau_f = 0.25 * p.dt, tdx = 2.0 / p.dx;

  Row<V> ua, ub, uc, hp, hn, out;
  if (ROLE == 0) {
    if (r0 - 1 == 0) {                                        // grid edge row 0 of level n+1: zeros
#pragma unroll
      for (int c = 0; c < 4; ++c)
#pragma unroll
        for (int v = 0; v < V; ++v) out.c[c][v] = 0.0;
      push(out, 0);
    }
    load_row<V, true>(ua, uin + (size_t)(m0 - 1) * row_stride, nth, j0);
    load_row<V, true>(ub, uin + (size_t)m0 * row_stride, nth, j0);
    load_row<V, true>(uc, uin + (size_t)(m0 + 1) * row_stride, nth, j0);
  } else {
    pop(ua, r0 - 1);
    pop(ub, r0);
    pop(uc, r0 + 1);
  }
  if (do_tap && r0 == 1) tap<V>(ua, ub, p, 0, mode, n, lane);     // both roles hold rows 0, 1 here when r0 == 1
  lw_stage<V, true>(ua, ub, ua, rtab + (size_t)(2 * (m0 - 1) + 1) * RT_N, th, tau_h, tdx, hp);
  add_source<V>(hp, src_h, p, m0 - 1, true);

  const double* rt_cur = sh.rt_buf;
  auto march = [&](const int i, Row<V>& A, Row<V>& B, Row<V>& Hp, Row<V>& Hn) {
    const int o = (i - m0) & (RT_CH - 1);
    if (o == 0) {
      asm volatile("cp.async.wait_group 0;" ::: "memory");
      __syncwarp();
      const int c = (i - m0) / RT_CH;
      rt_cur = sh.rt_buf + (c & 1) * RT_CHUNK_DOUBLES;
      if (i + RT_CH < m1)
        stage_rtab_chunk(sh.rt_buf + ((c + 1) & 1) * RT_CHUNK_DOUBLES, rtab, 2 * (i + RT_CH), 2 * nr - 1, lane);
    }
    if (do_tap && i >= r0 && i < r1) tap<V>(A, B, p, i, mode, n, lane);   // halo iterations belong to neighbours
    lw_stage<V, true>(A, B, A, rt_cur + (2 * o + 1) * RT_N, th, tau_h, tdx, Hn);
    if (any_src) add_source<V>(Hn, src_h, p, i, true);
    if (ROLE == 0) {
      __syncwarp();
      if (lane == 0 && i + NS + 1 <= m1) issue_row(i + NS + 1);
    }
    lw_stage<V, false>(Hp, Hn, A, rt_cur + (2 * o) * RT_N, th, tau_f, tdx, out);
    if (any_src) add_source<V>(out, src_f, p, i, false);
    if (ROLE == 0) {
      push(out, i);
      if (i + 2 <= m1) {
        mbar_wait_u32(sh.tma_u32 + 8u * (unsigned)((i + 2) % NS), (unsigned)((i - m0) / NS) & 1u);
        lds_row<V>(A, sh.slot0 + (size_t)((i + 2) % NS) * row_stride, nth, j0, lane_ok);
      }
    } else {
      store_row<V, true>(out, uout + (size_t)i * row_stride, nth, j0, 0, nth);
      if (i + 2 <= m1) pop(A, i + 2);
    }
  };
  bool tail = false;
  {
    int i = m0;
    for (; i + 1 < m1; i += 2) {
      march(i, ub, uc, hp, hn);
      march(i + 1, uc, ub, hn, hp);
    }
    if (i < m1) {
      march(i, ub, uc, hp, hn);
      tail = true;
    }
  }
  // After the loop the last call's (A, B) hold input rows m1-1 and m1: (ub, uc) if the tail ran, else (uc, ub).

  if (ROLE == 1 && r0 == 1) {
#pragma unroll
    for (int c = 0; c < 4; ++c)
#pragma unroll
      for (int v = 0; v < V; ++v) out.c[c][v] = 0.0;
    store_row<V, true>(out, uout, nth, j0, 0, nth);
  }
  if (r1 == nr - 1) {                                         // outer grid edge at this warp's output level
    if (ROLE == 0) {
      load_row<V, true>(ub, uin + (size_t)(nr - 1) * row_stride, nth, j0);
      load_row<V, true>(ua, uin + (size_t)(nr - 2) * row_stride, nth, j0);
    } else if (tail) {
      ua = ub;                                                // row nr-2 of level n+1
      ub = uc;                                                // row nr-1
    } else {
      ua = uc;
    }
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
    if (ROLE == 0) push(out, nr - 1);
    else store_row<V, true>(out, uout + (size_t)(nr - 1) * row_stride, nth, j0, 0, nth);
  }
}

}  // namespace

template <int V, bool FULLW>
__global__ void __launch_bounds__(128, (V == 2 ? 3 : TEUK_MIN_BLOCKS)) teuk_step_tb2_kernel(const __grid_constant__ StepParams p) {
  const int lane = threadIdx.x & 31;
  const int wib = __shfl_sync(FULL, (int)(threadIdx.x >> 5), 0);   // provably warp-uniform
  const int pair = wib >> 1, role = wib & 1;
  const int slab = blockIdx.x * 2 + pair;
  const int mode = blockIdx.y;
  const int nth = FULLW ? 32 * V : p.n_theta;
  constexpr int NS = TEUK_SLOTS;
  __shared__ __align__(16) double s_rt[4][2][RT_CHUNK_DOUBLES];
  __shared__ __align__(8) unsigned long long s_tma[2][NS], s_full[2][TB_RING], s_empty[2][TB_RING];
  extern __shared__ __align__(128) unsigned char s_dyn[];   // [pair][NS landing slots + TB_RING ring slots][4 n_theta]
  if (role == 0 && lane == 0) {
#pragma unroll
    for (int q = 0; q < NS; ++q) mbar_init(&s_tma[pair][q], 1);
#pragma unroll
    for (int q = 0; q < TB_RING; ++q) {
      mbar_init(&s_full[pair][q], 1);
      mbar_init(&s_empty[pair][q], 1);
    }
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
  }
  __syncthreads();                                          // barriers are initialised for both warps of a pair
  if (slab >= p.n_slabs) return;                            // both warps of the pair leave together
  const int r0 = slab_first_row(p, slab);
  const int r1 = slab_first_row(p, slab + 1);
  const size_t row_doubles = (size_t)4 * nth;
  Tb2Shared sh;
  sh.rt_buf = &s_rt[wib][0][0];
  sh.slot0 = reinterpret_cast<double*>(s_dyn) + (size_t)pair * (NS + TB_RING) * row_doubles;
  sh.ring = sh.slot0 + (size_t)NS * row_doubles;
  sh.tma_u32 = smem_u32(&s_tma[pair][0]);
  sh.full_u32 = smem_u32(&s_full[pair][0]);
  sh.empty_u32 = smem_u32(&s_empty[pair][0]);
  if (role == 0) tb2_warp<V, FULLW, 0>(p, sh, lane, mode, r0, r1);
  else tb2_warp<V, FULLW, 1>(p, sh, lane, mode, r0, r1);
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
  const int n_it = p.n_seg > 1 ? (nth + 31) / 32 : V;
  for (int v = 0; v < n_it; ++v) {
    const int j = p.n_seg > 1 ? v * 32 + lane
                              : ((p.variant == 1 && V > 1) ? (v >> 1) * 64 + 2 * lane + (v & 1) : lane * V + v);
    if (j >= nth) continue;
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
  dim3 grid((p.n_slabs + warps_per_block - 1) / warps_per_block, p.n_modes, p.n_seg), block(32 * warps_per_block);
  const bool vec = p.n_theta % V == 0;
  const int dyn_max = (int)((size_t)warps_per_block * TEUK_SLOTS * 4 * 32 * V * sizeof(double));
  const size_t dyn = vec ? (size_t)dyn_max : 0;
#define TEUK_LAUNCH(VECF, CMF, SEGF, FWF) TEUK_LAUNCH_T(VECF, CMF, SEGF, FWF, false)
#define TEUK_LAUNCH_T(VECF, CMF, SEGF, FWF, TF)                                                                  \
  do {                                                                                                       \
    static bool attr_set[64] = {false};   /* per device: function attributes belong to a context */         \
    int dev_ = 0;                                                                                            \
    cudaGetDevice(&dev_);                                                                                    \
    if (!attr_set[dev_ & 63]) {                                                                              \
      cudaError_t e = cudaFuncSetAttribute(teuk_step_kernel<V, VECF, CMF, SEGF, FWF, TF>,                    \
                                           cudaFuncAttributeMaxDynamicSharedMemorySize, dyn_max);            \
      if (e != cudaSuccess) return e;                                                                        \
      attr_set[dev_ & 63] = true;                                                                            \
    }                                                                                                        \
    if (p.pdl) {                                                                                             \
      cudaLaunchAttribute at_[1];                                                                            \
      at_[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;                                        \
      at_[0].val.programmaticStreamSerializationAllowed = 1;                                                 \
      cudaLaunchConfig_t lc_ = {};                                                                           \
      lc_.gridDim = grid; lc_.blockDim = block; lc_.dynamicSmemBytes = dyn; lc_.stream = st;                 \
      lc_.attrs = at_; lc_.numAttrs = 1;                                                                     \
      cudaError_t e = cudaLaunchKernelEx(&lc_, teuk_step_kernel<V, VECF, CMF, SEGF, FWF, TF>, p);            \
      if (e != cudaSuccess) return e;                                                                        \
    } else                                                                                                   \
    teuk_step_kernel<V, VECF, CMF, SEGF, FWF, TF><<<grid, block, dyn, st>>>(p);                              \
  } while (0)
  const bool fullw = p.n_theta == 32 * V;
  if (p.n_terms > 0) {              // multi-term deposit: coef_mode 0 only (checked by teuk_set_source_terms)
    if (p.n_seg > 1) {
      if (vec) TEUK_LAUNCH_T(true, 0, true, false, true); else TEUK_LAUNCH_T(false, 0, true, false, true);
    } else {
      if (fullw) TEUK_LAUNCH_T(true, 0, false, true, true);
      else if (vec) TEUK_LAUNCH_T(true, 0, false, false, true);
      else TEUK_LAUNCH_T(false, 0, false, false, true);
    }
  } else if (p.n_seg > 1) {
    if (vec) TEUK_LAUNCH(true, 0, true, false); else TEUK_LAUNCH(false, 0, true, false);
  } else if (p.coef_mode == 1) {
    if (fullw) TEUK_LAUNCH(true, 1, false, true);
    else if (vec) TEUK_LAUNCH(true, 1, false, false);
    else TEUK_LAUNCH(false, 1, false, false);
  } else {
    if (fullw) TEUK_LAUNCH(true, 0, false, true);
    else if (vec) TEUK_LAUNCH(true, 0, false, false);
    else TEUK_LAUNCH(false, 0, false, false);
  }
#undef TEUK_LAUNCH
#undef TEUK_LAUNCH_T
  return cudaGetLastError();
}

template <int V>
static cudaError_t launch_smem_v(const StepParams& p, cudaStream_t st) {
  const int warps_per_block = 4;
  dim3 grid((p.n_slabs + warps_per_block - 1) / warps_per_block, p.n_modes), block(32 * warps_per_block);
  const size_t dyn = (size_t)warps_per_block * (2 * 4 * (size_t)p.n_theta + 4 * 32 * V) * sizeof(double);
  const int dyn_max = (int)((size_t)warps_per_block * (2 * 4 * 32 * V + 4 * 32 * V) * sizeof(double));
  if (p.n_theta % 2 == 0 || V == 1) {
    static bool attr_set[64] = {false};   // per device
    int dev_ = 0;
    cudaGetDevice(&dev_);
    if (!attr_set[dev_ & 63]) {
      cudaError_t e = cudaFuncSetAttribute(teuk_step_smem_kernel<V, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, dyn_max);
      if (e != cudaSuccess) return e;
      attr_set[dev_ & 63] = true;
    }
    teuk_step_smem_kernel<V, true><<<grid, block, dyn, st>>>(p);
  } else {
    static bool attr_set[64] = {false};   // per device
    int dev_ = 0;
    cudaGetDevice(&dev_);
    if (!attr_set[dev_ & 63]) {
      cudaError_t e = cudaFuncSetAttribute(teuk_step_smem_kernel<V, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, dyn_max);
      if (e != cudaSuccess) return e;
      attr_set[dev_ & 63] = true;
    }
    teuk_step_smem_kernel<V, false><<<grid, block, dyn, st>>>(p);
  }
  return cudaGetLastError();
}

cudaError_t teuk_launch_step(const StepParams& p, cudaStream_t st) {
  const int v = (p.n_theta + 31) / 32;
  if (p.variant == 1) {
    if (v <= 1) return launch_smem_v<1>(p, st);
    if (v <= 2) return launch_smem_v<2>(p, st);
    if (v <= 4) return launch_smem_v<4>(p, st);
    return launch_smem_v<8>(p, st);
  }
  if (v <= 1) return launch_v<1>(p, st);
  if (v <= 2) return launch_v<2>(p, st);
  return launch_v<4>(p, st);   // n_theta > 128: theta segments of <= 120 payload columns (p.n_seg > 1)
}

template <int V>
static cudaError_t launch_tb2_v(const StepParams& p, cudaStream_t st) {
  dim3 grid((p.n_slabs + 1) / 2, p.n_modes), block(128);
  const size_t dyn = (size_t)2 * (TEUK_SLOTS + TB_RING) * 4 * p.n_theta * sizeof(double);
  const int dyn_max = (int)((size_t)2 * (TEUK_SLOTS + TB_RING) * 4 * 32 * V * sizeof(double));
  int dev_ = 0;
  cudaGetDevice(&dev_);
  if (p.n_theta == 32 * V) {
    static bool attr_set[64] = {false};
    if (!attr_set[dev_ & 63]) {
      cudaError_t e = cudaFuncSetAttribute(teuk_step_tb2_kernel<V, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, dyn_max);
      if (e != cudaSuccess) return e;
      attr_set[dev_ & 63] = true;
    }
    teuk_step_tb2_kernel<V, true><<<grid, block, dyn, st>>>(p);
  } else {
    static bool attr_set[64] = {false};
    if (!attr_set[dev_ & 63]) {
      cudaError_t e = cudaFuncSetAttribute(teuk_step_tb2_kernel<V, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, dyn_max);
      if (e != cudaSuccess) return e;
      attr_set[dev_ & 63] = true;
    }
    teuk_step_tb2_kernel<V, false><<<grid, block, dyn, st>>>(p);
  }
  return cudaGetLastError();
}

// Two iterations per launch (temporal blocking); needs n_theta % V == 0, one theta segment, coef_mode 0.
cudaError_t teuk_launch_step_tb2(const StepParams& p, cudaStream_t st) {
  const int v = (p.n_theta + 31) / 32;
  if (v <= 1) return launch_tb2_v<1>(p, st);
  if (v <= 2) return launch_tb2_v<2>(p, st);
  return launch_tb2_v<4>(p, st);
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
