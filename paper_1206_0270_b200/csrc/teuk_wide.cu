// teuk_wide.cu -- the marching step kernel for rows WIDER than one warp's best width: a GROUP of NWR warps shares
// one r* row (Eq. 3-4; same iteration, same stage arithmetic as teuk_step.cu: lw_stage_sums /
// lw_stage_body of teuk_stage.cuh, so fields are bit-identical).
//
// Why.  One warp per row with V = 4 columns per lane (teuk_step_kernel<4,...>, n_theta = 128) needs all 255
// registers and leaves 8 warps per SM: the FP64 pipe is busy 52 % of the time and the fixed-latency `wait` stall is
// the largest bucket (profiles/r2_step_kernel_before_chunk.md).  With V = 2 the same code needs 162 registers and
// runs 12 warps per SM.  Here every lane owns V = 2 columns and warp w of a group owns columns 64 w .. 64 w + 63;
// the only data the warps of a group exchange are the two boundary columns of S_Phi per stage (the theta stencil
// of PAPER.md:102 reaches one column), through shared memory behind one named barrier per stage.  The same barrier
// orders the hand-over of the TMA landing slots, which are per GROUP: one bulk copy per row, whatever the width.
// Rows wider than 128 columns -- the paper's own grid has 304 -- no longer need theta segments with
// recomputed halos (79 % useful lanes): 5 warps cover 320 columns (95 %).
//
// NWR = ceil(n_theta / 64) = 2 .. 5 (n_theta even, 66 .. 320); groups per block: 2 for NWR = 2, else 1.
#include <cuda_runtime.h>
#include <math.h>
#include <stdint.h>

#include <type_traits>

#include "teuk_internal.h"

#include "teuk_stage.cuh"

namespace {

template <int NWR>
struct WideShape {
  static constexpr int GPB = NWR == 2 ? 2 : 1;                                  // groups (slabs) per block
  static constexpr int WARPS = NWR * GPB;
  static constexpr int BLOCKS = NWR == 2 ? 3 : (NWR == 3 ? 4 : (NWR == 4 ? 3 : 2));   // resident blocks per SM (<= 168 / 204 registers)
};

__device__ __forceinline__ void group_barrier(int id, int threads) {
  asm volatile("bar.sync %0, %1;" ::"r"(id), "r"(threads) : "memory");
}

}  // namespace

// TERMS: the multi-term deposit of teuk_set_source_terms (a separate instantiation, as in teuk_step_kernel).
template <int NWR, bool TERMS = false>
__global__ void __launch_bounds__(32 * WideShape<NWR>::WARPS, WideShape<NWR>::BLOCKS)
teuk_step_wide_kernel(const __grid_constant__ StepParams p) {
  constexpr int V = 2, GPB = WideShape<NWR>::GPB, WARPS = WideShape<NWR>::WARPS, NS = TEUK_SLOTS;
  const int lane = threadIdx.x & 31;
  const int wib = __shfl_sync(FULL, (int)(threadIdx.x >> 5), 0);    // provably warp-uniform (see teuk_step_kernel)
  const int grp = wib / NWR, w = wib - grp * NWR;                   // group in the block, warp in the group
  const int slab = blockIdx.x * GPB + grp;
  const int mode = blockIdx.y;
  const int nth = p.n_theta, nr = p.n_r;
  __shared__ __align__(16) double s_rt[WARPS][2][RT_CHUNK_DOUBLES];
  __shared__ __align__(8) unsigned long long s_bar[GPB][NS];
  __shared__ __align__(16) double s_x[GPB][2][NWR][2][2];           // [parity][warp][left / right column][re, im]
  extern __shared__ __align__(128) unsigned char s_dyn[];           // [GPB][NS][4 n_theta] doubles: TMA landing slots
  if (w == 0 && lane == 0) {
#pragma unroll
    for (int q = 0; q < NS; ++q) mbar_init(&s_bar[grp][q], 1);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
  }
  __syncthreads();                                                   // barriers initialised for every warp of the group
  if (slab >= p.n_slabs) return;                                     // the whole group leaves together
  const int bar_id = 1 + grp;                                        // named barrier of this group (0 = __syncthreads)
  const int r0 = slab_first_row(p, slab);
  const int r1 = slab_first_row(p, slab + 1);
  const int j0 = w * 64 + lane * V;                                  // this lane's two columns (n_theta is even)
  const bool lane_ok = j0 < nth;
  const size_t row_stride = (size_t)4 * nth;
  const double* __restrict__ uin = p.uin + (size_t)mode * nr * row_stride;
  double* __restrict__ uout = p.uout + (size_t)mode * nr * row_stride;
  const double* __restrict__ rtab = p.rtab + (size_t)mode * (2 * nr - 1) * RT_N;
  double* const rt_buf = &s_rt[wib][0][0];
  stage_rtab_chunk(rt_buf, rtab, 2 * r0, 2 * nr - 1, lane);
  const unsigned row_bytes = (unsigned)(row_stride * sizeof(double));
  double* const slot0 = reinterpret_cast<double*>(s_dyn) + (size_t)grp * NS * row_stride;
  const unsigned slot0_u32 = smem_u32(slot0), bars_u32 = smem_u32(&s_bar[grp][0]);
  auto issue_row = [&](int q) {                                      // row q lands in slot q % NS of the group
    tma_load_row_u32(slot0_u32 + (unsigned)((q % NS) * row_stride * sizeof(double)), uin + (size_t)q * row_stride,
                     row_bytes, bars_u32 + 8u * (unsigned)(q % NS));
  };
  const long long n = *p.d_base + p.k;                               // index of the input time level

  ThetaTab<V> th;
  {
    const double* tb = p.ttab + (size_t)mode * TT_N * nth;
#pragma unroll
    for (int v = 0; v < V; ++v) {
      th.vals.s2[v] = lane_ok ? tb[TT_S2 * nth + j0 + v] : 0.0;
      th.vals.cs[v] = lane_ok ? tb[TT_COS * nth + j0 + v] : 0.0;
      th.vals.ap[v] = lane_ok ? tb[TT_AP * nth + j0 + v] : 0.0;
      th.vals.am[v] = lane_ok ? tb[TT_AM * nth + j0 + v] : 0.0;
      th.vals.d0[v] = lane_ok ? tb[TT_D0 * nth + j0 + v] : 0.0;
    }
  }
  typename SourceSel<V, TERMS>::type src_h, src_f;   // half stage: sample 2n at the half points; full stage: 2n+1 at the nodes
  __shared__ double s_tp[TERMS ? WARPS * 2 * TermTab<V>::PER_STAGE : 1];   // theta-profile tables of the multi-term deposit
  if constexpr (TERMS) {
    src_h.tab = &s_tp[(wib * 2 + 0) * TermTab<V>::PER_STAGE];
    src_f.tab = &s_tp[(wib * 2 + 1) * TermTab<V>::PER_STAGE];
  }
  setup_source<V>(src_h, p, mode, 2 * n, true, r0 - 1, r1 - 1, lane, w * 64);
  setup_source<V>(src_f, p, mode, 2 * n + 1, false, r0, r1 - 1, lane, w * 64);
  bool do_tap = w == 0 && p.tap_enable && p.n_obs > 0 && n >= 1;     // warp 0 of the group taps the whole row
  if (do_tap) {
    bool mine = false;
    for (int q = 0; q < p.n_obs; ++q) mine = mine || (p.obs[q].i0 >= r0 - 1 && p.obs[q].i0 < r1);
    do_tap = mine;
  }
  const bool any_src = __any_sync(FULL, src_h.on || src_f.on);
  const double tau_h = 0.5 * p.dt, tau_f = 0.25 * p.dt, tdx = 2.0 / p.dx;

  // Waveform tap of row pair (i0, i0 + 1) of the INPUT level, read from global memory by one warp, with the lane <->
  // column ownership and summation order of teuk_flush_tap_kernel (so chunking of teuk_step calls stays invisible).
  auto tap_row = [&](int q) {
    const int i0 = p.obs[q].i0;
    const double* lo = uin + (size_t)i0 * row_stride;
    const double* hi = lo + row_stride;
    const double f = p.obs[q].f;
    double wr = 0.0, wi = 0.0;
    const int vreq = (nth + 31) / 32;
    const int VV = vreq <= 1 ? 1 : (vreq <= 2 ? 2 : (vreq <= 4 ? 4 : 8));
    const int n_it = p.n_seg > 1 ? (nth + 31) / 32 : VV;
    for (int v = 0; v < n_it; ++v) {
      const int j = p.n_seg > 1 ? v * 32 + lane : lane * VV + v;
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
  };

  // Programmatic dependent launch: everything above reads nothing a step kernel writes (see teuk_step_kernel).
  asm volatile("griddepcontrol.wait;" ::: "memory");
  asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
  if (w == 0 && lane == 0) {
#pragma unroll
    for (int q = 2; q <= NS; ++q)
      if (r0 + q <= r1) issue_row(r0 + q);
  }

  // One stage across the group: S_Phi, exchange of its boundary columns, then the rest of the stage.  The barrier is
  // also what orders the landing slots: when a warp has passed the barrier of the half stage of iteration i, every
  // warp of the group has finished iteration i - 1, including its copy of row i + 1 out of slot (i + 1) % NS.
  int xpar = 0;
  auto stage = [&](auto half_tag, const Row<V>& A, const Row<V>& B, const Row<V>& base, const double* rec, double tau,
                   Row<V>& o_) {
    constexpr bool HALF = decltype(half_tag)::value;
    double sfr[V], sfi[V];
    lw_stage_sums<V>(A, B, sfr, sfi);
    double* xs = &s_x[grp][xpar][0][0][0];
    if (lane == 0) *reinterpret_cast<double2*>(xs + (w * 2 + 0) * 2) = make_double2(sfr[0], sfi[0]);
    if (lane == 31) *reinterpret_cast<double2*>(xs + (w * 2 + 1) * 2) = make_double2(sfr[V - 1], sfi[V - 1]);
    group_barrier(bar_id, 32 * NWR);
    double nlr[V], nrr[V], nli[V], nri[V];
    theta_neighbours<V, 0>(sfr, nlr, nrr, lane);
    theta_neighbours<V, 0>(sfi, nli, nri, lane);
    if (lane == 0 && w > 0) {                        // left neighbour of this warp's first column
      const double2 t = *reinterpret_cast<const double2*>(xs + ((w - 1) * 2 + 1) * 2);
      nlr[0] = t.x;
      nli[0] = t.y;
    }
    if (lane == 31 && w < NWR - 1) {                 // right neighbour of its last column
      const double2 t = *reinterpret_cast<const double2*>(xs + ((w + 1) * 2 + 0) * 2);
      nrr[V - 1] = t.x;
      nri[V - 1] = t.y;
    }
    xpar ^= 1;   // two buffers suffice: the next-but-one stage's writes come after the next stage's barrier
    lw_stage_body<V, HALF, ThetaTab<V>>(A, B, base, rec, th, tau, tdx, o_, sfr, sfi, nlr, nrr, nli, nri);
  };

  Row<V> ua, ub, uc, hp, hn, out;
  load_row<V, true>(ua, uin + (size_t)(r0 - 1) * row_stride, nth, j0);
  load_row<V, true>(ub, uin + (size_t)r0 * row_stride, nth, j0);
  load_row<V, true>(uc, uin + (size_t)(r0 + 1) * row_stride, nth, j0);
  if (do_tap && r0 == 1)
    for (int q = 0; q < p.n_obs; ++q)
      if (p.obs[q].i0 == 0) tap_row(q);
  stage(std::true_type(), ua, ub, ua, rtab + (size_t)(2 * (r0 - 1) + 1) * RT_N, tau_h, hp);
  add_source<V>(hp, src_h, p, r0 - 1, true);

  const double* rt_cur = rt_buf;
  double gprof = 0.0, gprof1 = 0.0, gprof2 = 0.0;
  // Per-chunk work, outside the marching iteration (see teuk_step_kernel): r-table hand-over, the radial deposit
  // profile of the chunk's rows (lanes 0-15: half stage, lanes 16-31: full stage), taps of observers in the chunk.
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
    if (do_tap)
      for (int q = 0; q < p.n_obs; ++q)
        if (p.obs[q].i0 >= cb && p.obs[q].i0 < min(cb + RT_CH, r1)) tap_row(q);
  };
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
  // One marching iteration at node i.  On entry A = u^n_i, B = u^n_{i+1}, Hp = 2 u^{n+1/2}_{i-1/2}; on exit
  // Hn = 2 u^{n+1/2}_{i+1/2} and A = u^n_{i+2}.
  auto march = [&](const int i, Row<V>& A, Row<V>& B, Row<V>& Hp, Row<V>& Hn) {
    const int o = (i - r0) & (RT_CH - 1);
    stage(std::true_type(), A, B, A, rt_cur + (2 * o + 1) * RT_N, tau_h, Hn);
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
    // every warp of the group is past the barrier of this half stage: slot (i + 1) % NS has been copied out by all
    if (w == 0 && lane == 0 && i + NS + 1 <= r1) issue_row(i + NS + 1);
    stage(std::false_type(), Hp, Hn, A, rt_cur + (2 * o) * RT_N, tau_f, out);
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
    store_row<V, true>(out, uout + (size_t)i * row_stride, nth, j0, 0, nth);
    if (i + 2 <= r1) {
      mbar_wait_u32(bars_u32 + 8u * (unsigned)((i + 2) % NS), (unsigned)((i - r0) / NS) & 1u);
      lds_row<V>(A, slot0 + (size_t)((i + 2) % NS) * row_stride, nth, j0, lane_ok);
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
    store_row<V, true>(out, uout, nth, j0, 0, nth);
  }
  if (r1 == nr - 1) {
    load_row<V, true>(ub, uin + (size_t)(nr - 1) * row_stride, nth, j0);
    load_row<V, true>(ua, uin + (size_t)(nr - 2) * row_stride, nth, j0);
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
    store_row<V, true>(out, uout + (size_t)(nr - 1) * row_stride, nth, j0, 0, nth);
  }
}

// ---- host-side launcher (called from teuk_api.cu) ------------------------------------------------------------
template <int NWR, bool TERMS>
static cudaError_t launch_wide(const StepParams& p, cudaStream_t st) {
  constexpr int GPB = WideShape<NWR>::GPB, WARPS = WideShape<NWR>::WARPS;
  dim3 grid((p.n_slabs + GPB - 1) / GPB, p.n_modes), block(32 * WARPS);
  const size_t dyn = (size_t)GPB * TEUK_SLOTS * 4 * p.n_theta * sizeof(double);
  const int dyn_max = (int)((size_t)GPB * TEUK_SLOTS * 4 * 64 * NWR * sizeof(double));
  static bool attr_set[64] = {false};   // per device
  int dev_ = 0;
  cudaGetDevice(&dev_);
  if (!attr_set[dev_ & 63]) {
    cudaError_t e = cudaFuncSetAttribute(teuk_step_wide_kernel<NWR, TERMS>, cudaFuncAttributeMaxDynamicSharedMemorySize, dyn_max);
    if (e != cudaSuccess) return e;
    attr_set[dev_ & 63] = true;
  }
  if (p.pdl) {
    cudaLaunchAttribute at_[1];
    at_[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    at_[0].val.programmaticStreamSerializationAllowed = 1;
    cudaLaunchConfig_t lc_ = {};
    lc_.gridDim = grid; lc_.blockDim = block; lc_.dynamicSmemBytes = dyn; lc_.stream = st;
    lc_.attrs = at_; lc_.numAttrs = 1;
    cudaError_t e = cudaLaunchKernelEx(&lc_, teuk_step_wide_kernel<NWR, TERMS>, p);
    if (e != cudaSuccess) return e;
  } else {
    teuk_step_wide_kernel<NWR, TERMS><<<grid, block, dyn, st>>>(p);
  }
  return cudaGetLastError();
}

// n_theta even, 66 .. 320; coef_mode 0 (the caller checks: teuk_wide_applies).
bool teuk_wide_applies(int n_theta) { return n_theta % 2 == 0 && n_theta > 64 && n_theta <= 320; }

// slabs that are in flight at once on one SM (for the launch-shape measurement)
int teuk_wide_groups_per_sm(int n_theta) {
  const int nwr = (n_theta + 63) / 64;
  return nwr == 2 ? 6 : (nwr == 3 ? 4 : (nwr == 4 ? 3 : 2));
}

cudaError_t teuk_launch_step_wide(const StepParams& p, cudaStream_t st) {
  const bool terms = p.n_terms > 0;
  switch ((p.n_theta + 63) / 64) {
    case 2: return terms ? launch_wide<2, true>(p, st) : launch_wide<2, false>(p, st);
    case 3: return terms ? launch_wide<3, true>(p, st) : launch_wide<3, false>(p, st);
    case 4: return terms ? launch_wide<4, true>(p, st) : launch_wide<4, false>(p, st);
    case 5: return terms ? launch_wide<5, true>(p, st) : launch_wide<5, false>(p, st);
    default: return cudaErrorInvalidValue;
  }
}
