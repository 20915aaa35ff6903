// teuk_resident.cu -- "kernel" = 2: the whole state stays ON CHIP for all iterations of one launch.
// Same lw_stage, source deposit and tap as the marching kernels (teuk_stage.cuh), so fields and waveforms
// are bit-identical to theirs.
//
// Why: the small grids (BASELINE.json configs 1 and 2: 0.5 and 8.4 MB of state) are not bandwidth-bound.  With
// one launch per iteration they are bound by the launch rate (2.9 us per iteration) and by the serial march
// of each warp (SURVEY.md 8(d) "Config 1 is launch-latency-bound.  Use a persistent kernel").  Here ONE
// cooperative launch runs n_iter iterations (Eq. 3-4):
//   * every block owns a contiguous range of r* rows of one mode and keeps them in shared memory for the
//     whole launch (HBM is touched at entry and exit only);
//   * an iteration of a block is a list of 2 rows + 1 row tasks, one warp per task: first the half-step rows
//     2 u^{n+1/2}_{i+1/2} (Eq. 3) into shared memory, then the full step (Eq. 4) in place -- no half-step value
//     is computed twice.  Tasks are dealt to the warps round-robin across iterations and wait only for the rows
//     they read (version counters in shared memory); there is no block-wide barrier in the time loop;
//   * neighbouring blocks exchange ONE row per side and iteration through L2 with a flag-in-data protocol
//     (each 16-byte element = {value.lo, tag, value.hi, tag}, tag = iteration number; an element is valid
//     when both tags match, so no fence and no separate flag round trip is needed).  A block computes and
//     publishes its two edge rows FIRST among the full-step tasks and consumes its neighbours' rows LAST among
//     the half-step tasks of the next iteration, so the L2 latency (~0.7 us) hides behind the interior rows;
//   * pole ghosts, radial edges, source deposit and tap-on-read
//     as in teuk_step_kernel.
// All blocks must be co-resident (they wait on each other): the launch is cooperative and sized to at most
// one block per SM; waits are bounded (trap -> sticky TEUK_ECUDA instead of a hung GPU).
#include <type_traits>

#include "teuk_stage.cuh"

#ifndef TEUK_RES_NW
#define TEUK_RES_NW(V) ((V) == 4 ? 8 : 16)   // warps per block the register budget is cut for
#endif

namespace {

__device__ __forceinline__ void ll_store(uint4* dst, double v, unsigned tag) {
  const unsigned lo = (unsigned)__double2loint(v), hi = (unsigned)__double2hiint(v);
  asm volatile("st.volatile.global.v4.u32 [%0], {%1, %2, %3, %4};" ::"l"(dst), "r"(lo), "r"(tag), "r"(hi), "r"(tag)
               : "memory");
}
__device__ __forceinline__ bool ll_try_load(const uint4* src, unsigned tag, double& v) {
  unsigned a, b, c, d;
  asm volatile("ld.volatile.global.v4.u32 {%0, %1, %2, %3}, [%4];" : "=r"(a), "=r"(b), "=r"(c), "=r"(d) : "l"(src) : "memory");
  v = __hiloint2double((int)c, (int)a);
  return b == tag && d == tag;
}

// One exchange slot = one row: [4][32 V] 16-byte elements, same lane -> column ownership as the registers.
template <int V>
__device__ __forceinline__ void ll_publish(uint4* slot, const Row<V>& u, unsigned tag, int lane) {
#pragma unroll
  for (int c = 0; c < 4; ++c)
#pragma unroll
    for (int v = 0; v < V; ++v) ll_store(slot + c * 32 * V + lane * V + v, u.c[c][v], tag);
}
template <int V>
__device__ __forceinline__ void ll_receive(const uint4* slot, Row<V>& u, unsigned tag, int lane) {
  unsigned tries = 0;
  for (;;) {
    bool ok = true;
#pragma unroll
    for (int c = 0; c < 4; ++c)
#pragma unroll
      for (int v = 0; v < V; ++v) ok = ll_try_load(slot + c * 32 * V + lane * V + v, tag, u.c[c][v]) && ok;
    if (__all_sync(FULL, ok)) break;
    if (++tries > (1u << 22)) asm volatile("trap;");   // a neighbour that never publishes: error, not a hang
    __nanosleep(32);
  }
}

// Version counters of the rows in shared memory (one int per row): a producer warp writes its row, then lane 0
// releases the new version; consumer warps acquire it before they read the row.  Bounded like every wait here.
__device__ __forceinline__ void flag_set(unsigned addr, int v) {
  asm volatile("st.release.cta.shared.s32 [%0], %1;" ::"r"(addr), "r"(v) : "memory");
}
// both counters of a task are polled together (one round trip to shared memory, one vote)
__device__ __forceinline__ void flag_wait2(unsigned addr_a, unsigned addr_b, int need) {
  unsigned tries = 0;
  for (;;) {
    int va, vb;
    asm volatile("ld.acquire.cta.shared.s32 %0, [%1];" : "=r"(va) : "r"(addr_a) : "memory");
    asm volatile("ld.acquire.cta.shared.s32 %0, [%1];" : "=r"(vb) : "r"(addr_b) : "memory");
    if (__all_sync(FULL, va >= need && vb >= need)) break;
    if (++tries > (1u << 26)) asm volatile("trap;");
  }
}

// Shared-memory rows through explicit 32-bit shared addresses (worked out once per warp): ptxas otherwise rebuilds
// the generic -> shared window base at every access site inside the time loop.  `addr` is this lane's first
// column of component 0; the four components of a row are 32 V doubles apart.
template <int V>
__device__ __forceinline__ void lds_row_s(Row<V>& u, unsigned addr) {
#pragma unroll
  for (int c = 0; c < 4; ++c) {
    const unsigned q = addr + (unsigned)(c * 32 * V * 8);
    if (V == 1) {
      asm volatile("ld.shared.f64 %0, [%1];" : "=d"(u.c[c][0]) : "r"(q) : "memory");
    } else {
#pragma unroll
      for (int v = 0; v < V; v += 2)
        asm volatile("ld.shared.v2.f64 {%0, %1}, [%2];" : "=d"(u.c[c][v]), "=d"(u.c[c][v + 1]) : "r"(q + 8u * v) : "memory");
    }
  }
}
template <int V>
__device__ __forceinline__ void sts_row_s(const Row<V>& u, unsigned addr) {
#pragma unroll
  for (int c = 0; c < 4; ++c) {
    const unsigned q = addr + (unsigned)(c * 32 * V * 8);
    if (V == 1) {
      asm volatile("st.shared.f64 [%0], %1;" ::"r"(q), "d"(u.c[c][0]) : "memory");
    } else {
#pragma unroll
      for (int v = 0; v < V; v += 2)
        asm volatile("st.shared.v2.f64 [%0], {%1, %2};" ::"r"(q + 8u * v), "d"(u.c[c][v]), "d"(u.c[c][v + 1]) : "memory");
    }
  }
}
// one r-table record (RT_N = 10 doubles, warp-uniform address: broadcast loads) into registers
__device__ __forceinline__ void lds_record_s(double (&rc)[RT_N], unsigned addr) {
#pragma unroll
  for (int k = 0; k < RT_N; k += 2)
    asm volatile("ld.shared.v2.f64 {%0, %1}, [%2];" : "=d"(rc[k]), "=d"(rc[k + 1]) : "r"(addr + 8u * k) : "memory");
}

template <int V>
__device__ __forceinline__ uint4* ll_slot(const StepParams& p, int mode, int ncta, int cta, int side, unsigned tag) {
  return reinterpret_cast<uint4*>(p.ll) + ((((size_t)mode * ncta + cta) * 2 + side) * 2 + (tag & 1u)) * (size_t)(4 * 32 * V);
}

}  // namespace

// NW = warps per block the register budget allows (65536 / (32 NW) registers per thread); the launch may use
// fewer (blockDim.x / 32 = min(NW, rows + 1)).
// CC: the time-independent coefficients b2d, Q, Re beta^' of every location of the block are kept in shared memory
// (3 doubles per point and location) when there is room; else they are rebuilt in every stage as in kernel 0.
// SRC: 0 = source-free (no deposit code in the task loop at all: the loop is 47 KB of instructions with it, and on
// the source-free configs 1 and 2 its mere presence cost 8 % and 2 %), 1 = the single-term deposit, 2 = the
// multi-term deposit of teuk_set_source_terms.  Separate instantiations chosen by the launcher.
template <int V, int NW, bool CC, int SRC = 1>
__global__ void __launch_bounds__(32 * NW, 1) teuk_step_resident_kernel(const __grid_constant__ StepParams p) {
  constexpr int NP = 32 * V;        // padded row width in shared memory (columns >= n_theta stay zero)
  constexpr int ROWD = 4 * NP;      // doubles per row
  const int lane = threadIdx.x & 31;
  const int w = __shfl_sync(FULL, (int)(threadIdx.x >> 5), 0);   // provably warp-uniform
  const int nw = (int)(blockDim.x >> 5);
  const int cta = blockIdx.x, ncta = gridDim.x, mode = blockIdx.y;
  const int nth = p.n_theta, nr = p.n_r;
  const int lo = 1 + cta * p.res_rows;              // interior nodes [lo, hi) belong to this block
  const int hi = min(lo + p.res_rows, nr - 1);
  const int rows = hi - lo;
  const bool first = cta == 0, last = cta == ncta - 1;
  const int j0 = lane * V;
  const size_t row_stride = (size_t)4 * nth;
  const double* __restrict__ uin = p.uin + (size_t)mode * nr * row_stride;
  double* __restrict__ uout = p.uout + (size_t)mode * nr * row_stride;
  const double* __restrict__ rtab = p.rtab + (size_t)mode * (2 * nr - 1) * RT_N;

  extern __shared__ __align__(128) unsigned char s_dyn[];
  double* const sU = reinterpret_cast<double*>(s_dyn);          // [res_rows + 2] rows: slot r = node lo - 1 + r
  double* const sH = sU + (size_t)(p.res_rows + 2) * ROWD;      // [res_rows + 1] half rows: slot h = lo - 1 + h + 1/2
  double* const sE = sH + (size_t)(p.res_rows + 1) * ROWD;      // new outer-edge row (last block)
  double* const sR = sE + ROWD;                                 // r-table records of locations 2 lo - 1 + q
  int* const sV = reinterpret_cast<int*>(sR + (size_t)(2 * p.res_rows + 2) * RT_N);   // version counters
  // coefficient cache: location 2 lo - 1 + q at sC + q * 3 NP, planes b2d, Q, bre (16-byte aligned)
  double* const sC = reinterpret_cast<double*>(sV + ((2 * p.res_rows + 3 + 3) & ~3));
  constexpr unsigned ROWB = ROWD * 8;                           // bytes per row
  const unsigned uU = smem_u32(sU) + 8u * (unsigned)(lane * V); // this lane's columns of row slot 0, component 0
  const unsigned uH = smem_u32(sH) + 8u * (unsigned)(lane * V);
  const unsigned uE = smem_u32(sE) + 8u * (unsigned)(lane * V);
  const unsigned uC = smem_u32(sC) + 8u * (unsigned)(lane * V);
  const unsigned uR = smem_u32(sR);
  const unsigned verU = smem_u32(sV);                           // [res_rows + 2]: level of row slot r, relative to entry
  const unsigned verH = verU + 4u * (unsigned)(p.res_rows + 2); // [res_rows + 1]: iterations that wrote half row h

  // ---- entry: state rows (with both neighbour rows: they serve iteration 0) and r-table records ----
  for (int r = w; r < rows + 2; r += nw) {
    Row<V> t;
    load_row<V, false>(t, uin + (size_t)(lo - 1 + r) * row_stride, nth, j0);
    sts_row<V>(t, sU + (size_t)r * ROWD, NP, j0);
  }
  for (int q = threadIdx.x; q < 2 * p.res_rows + 3; q += blockDim.x) sV[q] = 0;
  for (int q = threadIdx.x; q < (2 * rows + 2) * RT_N; q += blockDim.x) {
    const int loc = 2 * lo - 1 + q / RT_N;
    if (loc <= 2 * nr - 2) sR[q] = rtab[(size_t)loc * RT_N + q % RT_N];
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
  __syncthreads();

  const double tau_h = 0.5 * p.dt, tau_f = 0.25 * p.dt, tdx = 2.0 / p.dx;
  if (CC) {
    for (int q = w; q < 2 * rows + 1; q += nw) {
      double b2d[V], Q[V], bre[V];
      lw_stage_coefficients<V>(sR + q * RT_N, th.vals, tdx, b2d, Q, bre);
#pragma unroll
      for (int v = 0; v < V; ++v) {
        sC[(size_t)q * 3 * NP + j0 + v] = b2d[v];
        sC[(size_t)q * 3 * NP + NP + j0 + v] = Q[v];
        sC[(size_t)q * 3 * NP + 2 * NP + j0 + v] = bre[v];
      }
    }
    __syncthreads();
  }
  // one stage at the location with record index q (2 h: half point h + 1/2; 2 r - 1: node r)
  auto stage = [&](auto half_tag, const Row<V>& A, const Row<V>& B, const Row<V>& base, const int q, const double tau,
                   Row<V>& out) {
    constexpr bool HALF = decltype(half_tag)::value;
    __align__(16) double rc[RT_N];
    lds_record_s(rc, uR + (unsigned)(q * RT_N * 8));
    if (CC) {
      double b2d[V], Q[V], bre[V];
      const unsigned cq = uC + (unsigned)q * (unsigned)(3 * NP * 8);
#pragma unroll
      for (int v = 0; v < V; v += (V == 1 ? 1 : 2)) {
        if (V == 1) {
          asm volatile("ld.shared.f64 %0, [%1];" : "=d"(b2d[0]) : "r"(cq) : "memory");
          asm volatile("ld.shared.f64 %0, [%1];" : "=d"(Q[0]) : "r"(cq + (unsigned)(NP * 8)) : "memory");
          asm volatile("ld.shared.f64 %0, [%1];" : "=d"(bre[0]) : "r"(cq + (unsigned)(2 * NP * 8)) : "memory");
        } else {
          asm volatile("ld.shared.v2.f64 {%0, %1}, [%2];" : "=d"(b2d[v]), "=d"(b2d[v + (V > 1 ? 1 : 0)]) : "r"(cq + 8u * v) : "memory");
          asm volatile("ld.shared.v2.f64 {%0, %1}, [%2];" : "=d"(Q[v]), "=d"(Q[v + (V > 1 ? 1 : 0)]) : "r"(cq + (unsigned)(NP * 8) + 8u * v) : "memory");
          asm volatile("ld.shared.v2.f64 {%0, %1}, [%2];" : "=d"(bre[v]), "=d"(bre[v + (V > 1 ? 1 : 0)]) : "r"(cq + (unsigned)(2 * NP * 8) + 8u * v) : "memory");
        }
      }
      lw_stage_cached<V, HALF>(A, B, base, rc, th, b2d, Q, bre, tau, out);
    } else {
      lw_stage<V, HALF>(A, B, base, rc, th, tau, tdx, out);
    }
  };
  const long long n0 = *p.d_base + p.k;                  // index of the input level of iteration 0
  bool cta_taps = false;                                 // does an observer's cell [i0, i0+1] start in this block?
  for (int q = 0; q < p.n_obs; ++q) cta_taps = cta_taps || (p.obs[q].i0 >= lo - 1 && p.obs[q].i0 <= hi - 1);

  // Task list of one iteration: T = 2 rows + 1 tasks, first the rows + 1 half-step rows (those that need a
  // neighbour block's row LAST), then the rows full-step rows (the two edge rows of the block, which are
  // published, EARLY).  Task g = it * T + t runs on warp g mod nw, so the load rotates over the warps, and
  // every warp works through its tasks in increasing g.  A task waits for the rows it reads (version counters
  // in shared memory, release/acquire), never for a block-wide barrier; every dependence points to a smaller g,
  // so the smallest unfinished task can always run.
  // Measured on config 2 (28 rows per block, 16 warps): two __syncthreads per iteration 4.08 us per iteration,
  // this task list 3.63 us; a fixed chunk of rows per warp (no rotation, two hand-overs per warp) 4.6 us: what
  // counts is the length of the serial chain of tasks per warp, see DESIGN.md 5.1d.
  constexpr bool TERMS = SRC == 2;
  const bool has_source = SRC != 0 && p.has_source != 0;
  const double src_reach = ((double)p.W + 2.0) * p.dx;   // conservative pre-test of the source window in x
  const int T = 2 * rows + 1;
  int it = 0, t = w;
  while (t >= T) { t -= T; ++it; }
  while (it < p.n_iter) {
    const long long n = n0 + it;
    const unsigned tag_in = p.tag0 + (unsigned)it;       // tag of the rows published during iteration it - 1
    if (t <= rows) {
      // ---- half-step row (Eq. 3) at i + 1/2 between nodes i and i + 1 ----
      const int h = (t < rows - 1) ? t + 1 : (t == rows - 1 ? 0 : rows);
      const int i = lo - 1 + h;
      Row<V> A, B, Hn;
      // own rows must be at level `it`; that also says the readers of the old H[h] are done (they wrote them)
      flag_wait2(verU + 4u * (unsigned)(h >= 1 ? h : 1), verU + 4u * (unsigned)(h + 1 <= rows ? h + 1 : rows), it);
      if (h == 0 && !first && it > 0) ll_receive<V>(ll_slot<V>(p, mode, ncta, cta - 1, 1, tag_in), A, tag_in, lane);
      else lds_row_s<V>(A, uU + (unsigned)h * ROWB);
      if (h == rows && !last && it > 0) ll_receive<V>(ll_slot<V>(p, mode, ncta, cta + 1, 0, tag_in), B, tag_in, lane);
      else lds_row_s<V>(B, uU + (unsigned)(h + 1) * ROWB);
      // (Tried in round 2: the tap's warp reduction and ring store deferred until after the row has been handed over.
      // The two doubles it keeps across the stage push the V = 2 kernel to its 128-register cap: config 2 79 -> 69
      // GPts/s, config 1 12.5 -> 13.0.  Not kept.)
      if (cta_taps && n >= 1 && (it > 0 || p.tap_enable)) tap<V>(A, B, p, i, mode, n, lane);
      stage(std::true_type(), A, B, A, 2 * h, tau_h, Hn);
      if (has_source) {
        const double x = p.rs_min + ((double)i + 0.5) * p.dx;
        if (fabs(x - __ldg(p.xp + 2 * n)) <= src_reach) {
          typename SourceSel<V, TERMS>::type s;
          if constexpr (TERMS) s.tab = nullptr;   // one task = one row: profiles built on the spot
          setup_source<V>(s, p, mode, 2 * n, true, i, i, lane, 0);
          add_source<V>(Hn, s, p, i, true);
        }
      }
      sts_row_s<V>(Hn, uH + (unsigned)h * ROWB);
      if (last && h == rows) {   // outer radial edge (reading A6): A = row n_r-2, B = row n_r-1
        double eps;                                               // of location 2 (n_r - 1)
        asm volatile("ld.shared.f64 %0, [%1];" : "=d"(eps) : "r"(uR + (unsigned)(((2 * rows + 1) * RT_N + RT_EPS) * 8)) : "memory");
        ThetaVals<V> tv;
        th.get(tv);
        Row<V> e;
#pragma unroll
        for (int v = 0; v < V; ++v) {
          if (p.outer_bc == 0) {
            const double bb = rsqrt_near_one(fma(-eps, tv.s2[v], 1.0));
            e.c[0][v] = B.c[0][v] - p.dt * bb * (B.c[0][v] - A.c[0][v]) / p.dx;
            e.c[1][v] = B.c[1][v] - p.dt * bb * (B.c[1][v] - A.c[1][v]) / p.dx;
          } else {
            e.c[0][v] = 0.0;
            e.c[1][v] = 0.0;
          }
          e.c[2][v] = 0.0;
          e.c[3][v] = 0.0;
        }
        sts_row_s<V>(e, uE);
      }
      __syncwarp();
      if (lane == 0) flag_set(verH + 4u * (unsigned)h, it + 1);
    } else {
      // ---- full-step row in place (Eq. 4) ----
      const int tt = t - (rows + 1);
      // order: the two edge rows of the block (whose results are published) early, but behind `defer` interior rows:
      // their half-step inputs H[0], H[rows] were the LAST half-step tasks, so starting with them left two warps
      // idle for a task's time (config 2, us per iteration: defer 0 / 2 / 3 / 4 / 5 / 8 = 3.54 / 3.39 / 3.34 / 3.33 / 3.40 / 3.42)
      const int defer = rows >= 12 ? 4 : 0;
      const int r = (tt < defer) ? tt + 2 : (tt == defer ? 1 : (tt == defer + 1 ? rows : tt));
      const int i = lo - 1 + r;
      Row<V> Hp, Hn, U0, out;
      // both half-step rows of this iteration exist; their producers were the last readers of the old U[r]
      flag_wait2(verH + 4u * (unsigned)(r - 1), verH + 4u * (unsigned)r, it + 1);
      lds_row_s<V>(Hp, uH + (unsigned)(r - 1) * ROWB);
      lds_row_s<V>(Hn, uH + (unsigned)r * ROWB);
      lds_row_s<V>(U0, uU + (unsigned)r * ROWB);
      stage(std::false_type(), Hp, Hn, U0, 2 * r - 1, tau_f, out);
      if (has_source) {
        const double x = p.rs_min + (double)i * p.dx;
        if (fabs(x - __ldg(p.xp + 2 * n + 1)) <= src_reach) {
          typename SourceSel<V, TERMS>::type s;
          if constexpr (TERMS) s.tab = nullptr;   // one task = one row: profiles built on the spot
          setup_source<V>(s, p, mode, 2 * n + 1, false, i, i, lane, 0);
          add_source<V>(out, s, p, i, false);
        }
      }
      if (it + 1 < p.n_iter) {
        if (r == 1 && !first) ll_publish<V>(ll_slot<V>(p, mode, ncta, cta, 0, tag_in + 1u), out, tag_in + 1u, lane);
        if (r == rows && !last) ll_publish<V>(ll_slot<V>(p, mode, ncta, cta, 1, tag_in + 1u), out, tag_in + 1u, lane);
      }
      sts_row_s<V>(out, uU + (unsigned)r * ROWB);
      if (first && r == 1) {     // inner radial edge: Phi = Pi = 0
        Row<V> z;
#pragma unroll
        for (int cc = 0; cc < 4; ++cc)
#pragma unroll
          for (int v = 0; v < V; ++v) z.c[cc][v] = 0.0;
        sts_row_s<V>(z, uU);
      }
      if (last && r == rows) {   // new outer-edge row, computed from level n with the half-step row h = rows
        Row<V> e;
        lds_row_s<V>(e, uE);
        sts_row_s<V>(e, uU + (unsigned)(rows + 1) * ROWB);
      }
      __syncwarp();
      if (lane == 0) flag_set(verU + 4u * (unsigned)r, it + 1);
    }
    t += nw;
    while (t >= T) { t -= T; ++it; }
  }
  __syncthreads();

  // ---- exit: the block's rows of the last level go to the other ping-pong buffer ----
  for (int r = w; r < rows + 2; r += nw) {
    if ((r == 0 && !first) || (r == rows + 1 && !last)) continue;
    Row<V> t;
    lds_row<V>(t, sU + (size_t)r * ROWD, NP, j0, true);
    store_row<V, false>(t, uout + (size_t)(lo - 1 + r) * row_stride, nth, j0, 0, nth);
  }
}

// ---- host side ------------------------------------------------------------------------------------
template <int V>
constexpr int resident_max_warps() { return TEUK_RES_NW(V); }

size_t teuk_resident_smem_bytes(int n_theta, int res_rows, int coef_cache) {
  const int v = (n_theta + 31) / 32;
  const int V = v <= 1 ? 1 : (v <= 2 ? 2 : 4);
  const size_t rowd = (size_t)4 * 32 * V;
  size_t bytes = ((size_t)(2 * res_rows + 4) * rowd + (size_t)(2 * res_rows + 2) * RT_N) * sizeof(double) +
                 (size_t)((2 * res_rows + 3 + 3) & ~3) * sizeof(int);
  if (coef_cache) bytes += (size_t)(2 * res_rows + 1) * 3 * 32 * V * sizeof(double);
  return bytes;
}

// bytes of the exchange buffer: [n_modes][ncta][2 sides][2 parities] rows of 16-byte elements
size_t teuk_resident_ll_bytes(int n_theta, int n_modes, int ncta) {
  const int v = (n_theta + 31) / 32;
  const int V = v <= 1 ? 1 : (v <= 2 ? 2 : 4);
  return (size_t)n_modes * ncta * 4 * (4 * 32 * V) * 16;
}

template <int V, bool CC, int SRC>
static cudaError_t launch_resident_v(const StepParams& p, int ncta, cudaStream_t st) {
  constexpr int NW = resident_max_warps<V>();
  const size_t dyn = teuk_resident_smem_bytes(p.n_theta, p.res_rows, CC ? 1 : 0);
  static bool attr_set[64] = {false};   // per device
  int dev_ = 0;
  cudaGetDevice(&dev_);
  if (!attr_set[dev_ & 63]) {
    int optin = 0;
    cudaError_t e = cudaDeviceGetAttribute(&optin, cudaDevAttrMaxSharedMemoryPerBlockOptin, dev_);
    if (e == cudaSuccess)
      e = cudaFuncSetAttribute(teuk_step_resident_kernel<V, NW, CC, SRC>, cudaFuncAttributeMaxDynamicSharedMemorySize, optin);
    if (e != cudaSuccess) return e;
    attr_set[dev_ & 63] = true;
  }
  const int nwarps = 2 * p.res_rows + 1 < NW ? 2 * p.res_rows + 1 : NW;
  dim3 grid(ncta, p.n_modes), block(32 * nwarps);
  StepParams pc = p;
  void* args[] = {&pc};
  return cudaLaunchCooperativeKernel((const void*)teuk_step_resident_kernel<V, NW, CC, SRC>, grid, block, args, dyn, st);
}

// n_iter iterations in one cooperative launch; the caller sized res_rows / ncta so that the state fits.
cudaError_t teuk_launch_step_resident(const StepParams& p, int ncta, cudaStream_t st) {
  const int v = (p.n_theta + 31) / 32;
  if (p.has_source && p.n_terms > 0) {   // multi-term deposit (the host passes res_cache = 0 with it)
    if (v <= 1) return launch_resident_v<1, false, 2>(p, ncta, st);
    if (v <= 2) return launch_resident_v<2, false, 2>(p, ncta, st);
    return launch_resident_v<4, false, 2>(p, ncta, st);
  }
#define TEUK_RES_DISPATCH(SRCV)                                             \
  do {                                                                      \
    if (p.res_cache) {                                                      \
      if (v <= 1) return launch_resident_v<1, true, SRCV>(p, ncta, st);     \
      if (v <= 2) return launch_resident_v<2, true, SRCV>(p, ncta, st);     \
      return launch_resident_v<4, true, SRCV>(p, ncta, st);                 \
    }                                                                       \
    if (v <= 1) return launch_resident_v<1, false, SRCV>(p, ncta, st);      \
    if (v <= 2) return launch_resident_v<2, false, SRCV>(p, ncta, st);      \
    return launch_resident_v<4, false, SRCV>(p, ncta, st);                  \
  } while (0)
  if (p.has_source) TEUK_RES_DISPATCH(1);
  TEUK_RES_DISPATCH(0);
#undef TEUK_RES_DISPATCH
}


// ---- allocation-free variant (teuk_step_noalloc, include/teuk.h) -------------------------------------------
// Some callers cannot call cudaMalloc (code under CUDA graph capture, tight serving loops, harnesses that forbid
// it).  For them the block-to-block exchange buffer of the resident kernel -- its only scratch memory, normally
// cudaMalloc'ed by the first teuk_step -- lives in this file-scope device array: TEUK_STATIC_LL_BYTES = 5 MiB, held
// by every GPU that loads the library until the process exits; enough for 148 blocks of the widest rows (V = 4:
// 148 x 4 rows x 512 elements x 16 B = 4.6 MiB).  In host code the array's NAME is a host-side stand-in, not a
// device address: the address is asked for once per device, with that device current, by cudaGetSymbolAddress.
// Every call shares the array and finds the previous call's rows and tags in it, so each call first clears the
// part it uses (stream-ordered memset) and starts its tags at 0; calls that overlap on the GPU would race.
#define TEUK_STATIC_LL_BYTES (5u << 20)
static __device__ __align__(256) unsigned char g_static_ll[TEUK_STATIC_LL_BYTES];

size_t teuk_resident_static_capacity() { return (size_t)TEUK_STATIC_LL_BYTES; }

// Like teuk_launch_step_resident with p.ll / p.tag0 replaced by the static scratch.  No allocation of any kind.
cudaError_t teuk_launch_step_resident_static(const StepParams& p, int ncta, cudaStream_t st) {
  const size_t need = teuk_resident_ll_bytes(p.n_theta, p.n_modes, ncta);
  if (need > (size_t)TEUK_STATIC_LL_BYTES) return cudaErrorInvalidValue;      // the caller checks first and reports
  static void* addr[64] = {nullptr};     // per device: a symbol has one address in every context
  int dev = 0;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return e;
  if (!addr[dev & 63]) {
    void* ptr = nullptr;
    e = cudaGetSymbolAddress(&ptr, g_static_ll);
    if (e != cudaSuccess) return e;
    addr[dev & 63] = ptr;
  }
  e = cudaMemsetAsync(addr[dev & 63], 0, need, st);                           // stale rows and tags of the last call
  if (e != cudaSuccess) return e;
  StepParams pc = p;
  pc.ll = addr[dev & 63];
  pc.tag0 = 0;
  return teuk_launch_step_resident(pc, ncta, st);
}
