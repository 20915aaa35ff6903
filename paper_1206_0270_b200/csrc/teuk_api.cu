// teuk_api.cu -- the C ABI of include/teuk.h: argument checks, device memory, stream/graph
// plumbing, ring-buffer drains.  Every arithmetic step of the path runs in the kernels of
// teuk_step.cu / teuk_tables.cu; there is no CPU fallback.
#include <cuda_runtime.h>
#include <math.h>
#include <stdint.h>
#include <stdio.h>
#include <string.h>

#include <new>
#include <vector>

#include "../../include/teuk.h"
#include "teuk_internal.h"

// kernels / launchers defined in the other translation units
cudaError_t teuk_launch_tables(double* rtab, double* ttab, const int* d_m, int n_modes, int n_r, int n_theta,
                               double rs_min, double dx, double dth, double M, double a, cudaStream_t st);
cudaError_t teuk_launch_coef2d(double* c2d, const double* rtab, const double* ttab, int n_modes, int n_r,
                               int n_theta, double dx, cudaStream_t st);
cudaError_t teuk_launch_step(const StepParams& p, cudaStream_t st);
cudaError_t teuk_launch_step_tb2(const StepParams& p, cudaStream_t st);
cudaError_t teuk_launch_step_wide(const StepParams& p, cudaStream_t st);
bool teuk_wide_applies(int n_theta);
int teuk_wide_groups_per_sm(int n_theta);
cudaError_t teuk_launch_step_resident(const StepParams& p, int ncta, cudaStream_t st);
size_t teuk_resident_smem_bytes(int n_theta, int res_rows, int coef_cache);
size_t teuk_resident_ll_bytes(int n_theta, int n_modes, int ncta);
cudaError_t teuk_launch_step_resident_static(const StepParams& p, int ncta, cudaStream_t st);
size_t teuk_resident_static_capacity();
cudaError_t teuk_launch_flush_tap(const StepParams& p, cudaStream_t st);
cudaError_t teuk_launch_bump(long long* d_base, long long inc, cudaStream_t st);
cudaError_t teuk_launch_set_base(long long* d_base, long long v, cudaStream_t st);
cudaError_t teuk_launch_pack(double* u, double* const src[4], size_t n_rows, int nth, cudaStream_t st);
cudaError_t teuk_launch_unpack(const double* u, double* const dst[4], size_t n_rows, int nth, cudaStream_t st);
double teuk_fp64_rate(int kind, cudaError_t* err);

namespace {

const double kPi = 3.14159265358979323846264338327950288;
const long long kRingCap = 1 << 15;  // samples per observer held on the device between drains
const int kGraphBatch = 32;          // iterations per CUDA-graph replay (even)

char g_create_error[256] = "no error";

struct HostChunk {      // drained samples of one observer: pinned, [count][n_modes][2]
  double* data;
  long long first;      // sample index (1-based iteration number) of data[0]
  long long count;
};

struct ObsHost {
  double rs_obs;
  int i0;
  double f;
  double* d_weights;
  double* d_ring;
  std::vector<HostChunk> chunks;
  long long read_cursor;  // next sample index to hand to the caller (1-based)
};

}  // namespace

struct teuk_solver {
  // problem
  double a, M, dt, dx, dth, rs_min, rs_max;
  int n_r, n_theta, n_modes;
  int m[TEUK_MAX_MODES];
  // options
  int outer_bc, coef_mode, slab_rows_opt, use_graph, variant, autotune;
  int tuned_rows;        // slabs per mode chosen by the one-time autotune (0 = not tuned yet)
  int temporal_block;    // 1 = one iteration per launch, 2 = two (warp pairs, level n+1 stays on chip)
  int wide_opt;          // "wide" option: -1 automatic, 0 = one warp per row / theta segment, 1 = a group of warps per row
  int tuned_rows2;       // autotuned slabs per mode of the temporal-blocking kernel
  int force_slabs;       // autotune in progress: slabs per mode of the candidate being timed
  // resident kernel ("kernel" = 2): rows per block, blocks per mode, exchange buffer and its running tag
  int kernel_opt;        // "kernel" option: -1 = automatic (resident kernel when the state fits on chip, else kernel 0)
  int use_pdl;           // "pdl" option: programmatic dependent launch inside CUDA-graph batches
  int res_cache_opt;     // "resident_cache" option: keep the time-independent coefficients on chip when they fit
  int res_failed;        // automatic choice: a cooperative launch was refused once, stay with kernel 0
  int res_rows, res_ncta, smem_optin;
  void* d_ll;
  unsigned ll_tag;
  // device
  int device, n_sms;
  cudaStream_t own_stream, stream, copy_stream;
  cudaEvent_t ev_compute, ev_copy;
  double* d_u[2];
  int cur;               // d_u[cur] holds the current time level
  double *d_rtab, *d_ttab, *d_coef2d;
  int* d_m;
  long long* d_base;     // device copy of the iteration index baseline
  long long base_on_device;
  int* d_nonfinite;
  // source
  int has_source, W, source_kind;
  long long n_samples;
  double *d_xp, *d_thp, *d_amp_re, *d_amp_im;
  double sigma_r, sigma_th;
  // rank-1 deposit terms installed by teuk_set_source_terms (0 = the single term of the trajectory table)
  int n_terms;
  signed char term_or[TEUK_MAX_TERMS], term_oth[TEUK_MAX_TERMS];
  double *d_term_re, *d_term_im;   // [n_terms][n_modes][n_samples]
  // time
  long long step;        // iterations done since set_initial
  long long recorded;    // samples recorded on the device (== step when observers exist)
  long long drained;     // samples already copied to host chunks
  // observers
  int n_obs;
  ObsHost obs[TEUK_MAX_OBS];
  // graph
  cudaGraphExec_t graph_exec[2];  // one per ping-pong parity of `cur`
  cudaGraphExec_t graph_exec_tb2[2];
  // stats / errors
  long long launches;
  int sticky;            // sticky CUDA failure
  char err[256];
};

namespace {

int fail(teuk_solver* s, int code, const char* msg) {
  if (s) {
    snprintf(s->err, sizeof(s->err), "%s", msg);
  } else {
    snprintf(g_create_error, sizeof(g_create_error), "%s", msg);
  }
  return code;
}

int cuda_fail(teuk_solver* s, cudaError_t e, const char* where) {
  char buf[256];
  snprintf(buf, sizeof(buf), "CUDA error in %s: %s", where, cudaGetErrorString(e));
  if (s) s->sticky = 1;
  return fail(s, e == cudaErrorMemoryAllocation ? TEUK_ENOMEM : TEUK_ECUDA, buf);
}

#define CK(call, where)                                   \
  do {                                                    \
    cudaError_t e_ = (call);                              \
    if (e_ != cudaSuccess) return cuda_fail(s, e_, where); \
  } while (0)

// Every entry point runs on the solver's own device and leaves the caller's current device as it found it
// (several solvers on different GPUs may be driven from one thread).
struct DeviceGuard {
  int prev;
  bool switched;
  explicit DeviceGuard(const teuk_solver* s) : prev(-1), switched(false) {
    if (cudaGetDevice(&prev) == cudaSuccess && prev != s->device) switched = cudaSetDevice(s->device) == cudaSuccess;
  }
  ~DeviceGuard() {
    if (switched) cudaSetDevice(prev);
  }
  DeviceGuard(const DeviceGuard&) = delete;
  DeviceGuard& operator=(const DeviceGuard&) = delete;
};

size_t state_doubles(const teuk_solver* s) { return (size_t)s->n_modes * s->n_r * 4 * s->n_theta; }

void drop_graph(teuk_solver* s) {
  for (int q = 0; q < 2; ++q) {
    if (s->graph_exec[q]) {
      cudaGraphExecDestroy(s->graph_exec[q]);
      s->graph_exec[q] = nullptr;
    }
    if (s->graph_exec_tb2[q]) {
      cudaGraphExecDestroy(s->graph_exec_tb2[q]);
      s->graph_exec_tb2[q] = nullptr;
    }
  }
}

// theta segments of the register kernel: one warp spans up to 128 columns; wider grids are cut into
// segments of <= 120 payload columns (+ 4 halo columns on each side inside the warp's 128-column window).
int n_segments(const teuk_solver* s) {
  if (s->variant == 1 || s->n_theta <= 128) return 1;
  return (s->n_theta + 119) / 120;
}

// The wide kernel (teuk_wide.cu: a group of ceil(n_theta / 64) warps per row, V = 2 columns per lane) replaces the
// one-warp-per-row kernel and the theta segments when it applies and is asked for (or chosen by default).
// Automatic choice (measured, profiles/r2_bench.md): for n_theta <= 128 one warp per row with V = 4 is faster (config 5:
// 86.5 vs 81.0 GPts/s: the group kernel issues 833 instead of 535 instructions per row and pays two barriers);
// for wider rows the group kernel beats the theta segments with their recomputed halo columns (32000 x 304: 68.0 vs 65.1).
bool wide_active(const teuk_solver* s) {
  if (s->wide_opt == 0 || (s->wide_opt < 0 && s->n_theta <= 128)) return false;
  return s->variant == 0 && s->coef_mode == 0 && s->temporal_block == 1 && teuk_wide_applies(s->n_theta);
}
// slabs per row: theta segments of the one-warp-per-row kernel; the wide kernel marches whole rows
int seg_factor(const teuk_solver* s) { return wide_active(s) ? 1 : n_segments(s); }
cudaError_t launch_step_any(const teuk_solver* s, const StepParams& p, cudaStream_t st) {
  return wide_active(s) ? teuk_launch_step_wide(p, st) : teuk_launch_step(p, st);
}

// Heuristic slab length (rows of r* marched by one warp): two waves of the warps that fit on the chip.
// It seeds the autotune below and is used as is when autotuning is switched off.
int resident_warps(const teuk_solver* s) {
  const int sms = s->n_sms > 0 ? s->n_sms : 148;
  const int v = (s->n_theta + 31) / 32;
  if (wide_active(s)) return sms * teuk_wide_groups_per_sm(s->n_theta);      // slabs in flight = groups of warps
  return sms * (s->variant == 1 ? 12 : (v <= 1 ? 16 : (v == 2 ? 12 : 8)));   // occupancies of the kernels
}

// Temporal blocking is available for the register kernel with rebuilt coefficients, one theta segment and
// whole vector chunks per lane (n_theta a multiple of V).
bool tb2_possible(const teuk_solver* s) {
  const int v = (s->n_theta + 31) / 32;
  const int vsel = v <= 1 ? 1 : (v <= 2 ? 2 : 4);
  return s->variant == 0 && s->coef_mode == 0 && n_segments(s) == 1 && s->n_theta % vsel == 0;
}
bool tb2_active(const teuk_solver* s) { return s->temporal_block == 2 && tb2_possible(s); }

// Resident kernel (teuk_resident.cu): at most one block per SM, every mode split over the same number of
// blocks, each block's rows (state + half-step rows) in shared memory.  Returns false if that does not fit.
bool resident_plan(const teuk_solver* s, int* res_rows, int* ncta) {
  if (s->n_theta > 128 || s->coef_mode != 0 || s->n_modes > s->n_sms) return false;
  const int interior = s->n_r - 2;
  int per_mode = s->n_sms / s->n_modes;
  if (per_mode > interior) per_mode = interior;
  const int rows = (interior + per_mode - 1) / per_mode;
  if (teuk_resident_smem_bytes(s->n_theta, rows, 0) > (size_t)s->smem_optin) return false;
  *res_rows = rows;
  *ncta = (interior + rows - 1) / rows;
  return true;
}

// Which kernel runs the next iterations: the resident one if asked for, or, by default, whenever it applies
// (results are bit-identical; an explicit slab length, coef_mode 1 or temporal_block 2 address kernel 0).
bool resident_active(const teuk_solver* s, int* res_rows, int* ncta) {
  if (s->kernel_opt != 2) {
    if (s->kernel_opt != -1 || s->res_failed || s->temporal_block != 1 || s->slab_rows_opt > 0) return false;
  }
  return resident_plan(s, res_rows, ncta);
}

int rows_for_waves(const teuk_solver* s, double waves, int tb = 1) {
  const long long interior = s->n_r - 2;
  const double target = waves * resident_warps(s) / tb;   // tb = 2: a slab occupies a pair of warps
  long long rows = (long long)((interior * s->n_modes * seg_factor(s) + target - 1) / target);
  if (rows < 1) rows = 1;
  if (rows > interior) rows = interior;
  return (int)rows;
}

int auto_slab_rows(const teuk_solver* s, int tb = 1) { return rows_for_waves(s, 2.0, tb); }

int slabs_for_rows(const teuk_solver* s, long long rows) {
  const long long interior = s->n_r - 2;
  if (rows < 1) rows = 1;
  if (rows > interior) rows = interior;
  return (int)((interior + rows - 1) / rows);
}

// Slabs per mode of the marching kernels: the candidate under measurement, an explicit "slab_rows", the measured
// optimum, or the two-wave heuristic.  The rows are then dealt evenly to that many slabs.
int slabs_in_use(const teuk_solver* s, int tb = 1) {
  if (s->force_slabs > 0) return s->force_slabs;
  if (s->slab_rows_opt > 0) return slabs_for_rows(s, s->slab_rows_opt);
  const int tuned = tb == 2 ? s->tuned_rows2 : s->tuned_rows;
  return tuned > 0 ? tuned : slabs_for_rows(s, auto_slab_rows(s, tb));
}

void fill_params(const teuk_solver* s, StepParams* p, int in_buf, int k, int tap_enable, int tb = 1) {
  memset(p, 0, sizeof(*p));
  p->uin = s->d_u[in_buf];
  p->uout = s->d_u[in_buf ^ 1];
  p->rtab = s->d_rtab;
  p->ttab = s->d_ttab;
  p->coef2d = s->d_coef2d;
  p->coef_mode = s->coef_mode;
  p->n_r = s->n_r;
  p->n_theta = s->n_theta;
  p->n_modes = s->n_modes;
  p->n_slabs = slabs_in_use(s, tb);
  p->slab_q = (s->n_r - 2) / p->n_slabs;
  p->slab_rem = (s->n_r - 2) % p->n_slabs;
  p->n_seg = n_segments(s);
  p->seg_payload = p->n_seg > 1 ? ((s->n_theta + p->n_seg - 1) / p->n_seg + 3) / 4 * 4 : s->n_theta;
  p->outer_bc = s->outer_bc;
  p->variant = s->variant;
  p->dt = s->dt;
  p->dx = s->dx;
  p->rs_min = s->rs_min;
  p->dth = s->dth;
  p->has_source = s->has_source;
  p->source_kind = s->source_kind;
  p->W = s->source_kind ? s->source_kind : s->W;           // discrete deltas: the window is their support
  p->n_samples = s->n_samples;
  p->xp = s->d_xp;
  p->thp = s->d_thp;
  p->amp_re = s->d_amp_re;
  p->amp_im = s->d_amp_im;
  if (s->n_terms > 0) {
    p->n_terms = s->n_terms;
    for (int t = 0; t < s->n_terms; ++t) { p->term_or[t] = s->term_or[t]; p->term_oth[t] = s->term_oth[t]; }
    p->amp_re = s->d_term_re;
    p->amp_im = s->d_term_im;
  }
  p->sigma_r = s->source_kind ? s->dx : s->sigma_r;       // ... and their widths are the grid spacings
  p->sigma_th = s->source_kind ? s->dth : s->sigma_th;
  p->d_base = s->d_base;
  p->k = k;
  p->tap_enable = tap_enable;
  p->tap_enable2 = 1;
  p->n_obs = s->n_obs;
  p->ring_cap = kRingCap;
  p->nonfinite = s->d_nonfinite;
  for (int q = 0; q < s->n_obs; ++q) {
    p->obs[q].i0 = s->obs[q].i0;
    p->obs[q].f = s->obs[q].f;
    p->obs[q].weights = s->obs[q].d_weights;
    p->obs[q].ring = s->obs[q].d_ring;
  }
}

}  // namespace

namespace {

void free_chunks(ObsHost* o) {
  for (size_t q = 0; q < o->chunks.size(); ++q) cudaFreeHost(o->chunks[q].data);
  o->chunks.clear();
}

void reset_series(teuk_solver* s) {
  for (int q = 0; q < s->n_obs; ++q) {
    free_chunks(&s->obs[q]);
    s->obs[q].read_cursor = 1;
  }
  s->recorded = 0;
  s->drained = 0;
}

// Enqueue copies of the samples drained+1 .. recorded from the device rings into new pinned
// host chunks on the copy stream; the compute stream then waits for the copies (no host sync).
int drain_rings(teuk_solver* s) {
  const long long count = s->recorded - s->drained;
  if (count <= 0 || s->n_obs == 0) {
    s->drained = s->recorded;
    return TEUK_OK;
  }
  CK(cudaEventRecord(s->ev_compute, s->stream), "drain: event record");
  CK(cudaStreamWaitEvent(s->copy_stream, s->ev_compute, 0), "drain: wait compute");
  const size_t rec_bytes = (size_t)s->n_modes * 2 * sizeof(double);
  for (int q = 0; q < s->n_obs; ++q) {
    HostChunk ch;
    ch.first = s->drained + 1;
    ch.count = count;
    ch.data = nullptr;
    CK(cudaMallocHost((void**)&ch.data, (size_t)count * rec_bytes), "drain: pinned alloc");
    const long long slot0 = s->drained % kRingCap;  // slot of sample drained+1
    const long long first_part = (slot0 + count <= kRingCap) ? count : kRingCap - slot0;
    CK(cudaMemcpyAsync(ch.data, (char*)s->obs[q].d_ring + (size_t)slot0 * rec_bytes,
                       (size_t)first_part * rec_bytes, cudaMemcpyDeviceToHost, s->copy_stream),
       "drain: copy");
    if (first_part < count)
      CK(cudaMemcpyAsync((char*)ch.data + (size_t)first_part * rec_bytes, s->obs[q].d_ring,
                         (size_t)(count - first_part) * rec_bytes, cudaMemcpyDeviceToHost, s->copy_stream),
         "drain: copy wrap");
    s->obs[q].chunks.push_back(ch);
  }
  CK(cudaEventRecord(s->ev_copy, s->copy_stream), "drain: event record copy");
  CK(cudaStreamWaitEvent(s->stream, s->ev_copy, 0), "drain: wait copy");
  s->drained = s->recorded;
  return TEUK_OK;
}

int tune_if_needed(teuk_solver* s);

int build_tables(teuk_solver* s) {
  CK(teuk_launch_tables(s->d_rtab, s->d_ttab, s->d_m, s->n_modes, s->n_r, s->n_theta, s->rs_min, s->dx,
                        s->dth, s->M, s->a, s->stream),
     "table kernels");
  s->launches += 2;
  return TEUK_OK;
}

}  // namespace

extern "C" {

const char* teuk_last_error(const teuk_solver* s) { return s ? s->err : g_create_error; }

void teuk_destroy(teuk_solver* s) {
  if (!s) return;
  DeviceGuard guard(s);
  if (s->stream) cudaStreamSynchronize(s->stream);
  if (s->copy_stream) cudaStreamSynchronize(s->copy_stream);
  drop_graph(s);
  for (int q = 0; q < s->n_obs; ++q) {
    free_chunks(&s->obs[q]);
    cudaFree(s->obs[q].d_weights);
    cudaFree(s->obs[q].d_ring);
  }
  cudaFree(s->d_u[0]);
  cudaFree(s->d_u[1]);
  cudaFree(s->d_rtab);
  cudaFree(s->d_ttab);
  cudaFree(s->d_coef2d);
  cudaFree(s->d_m);
  cudaFree(s->d_base);
  cudaFree(s->d_nonfinite);
  cudaFree(s->d_ll);
  cudaFree(s->d_xp);
  cudaFree(s->d_thp);
  cudaFree(s->d_amp_re);
  cudaFree(s->d_amp_im);
  cudaFree(s->d_term_re);
  cudaFree(s->d_term_im);
  if (s->ev_compute) cudaEventDestroy(s->ev_compute);
  if (s->ev_copy) cudaEventDestroy(s->ev_copy);
  if (s->own_stream) cudaStreamDestroy(s->own_stream);
  if (s->copy_stream) cudaStreamDestroy(s->copy_stream);
  delete s;
}

int teuk_select_device(int32_t device) {
  int ndev = 0;
  if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev < 1) {
    cudaGetLastError();
    return fail(nullptr, TEUK_ECUDA, "teuk_select_device: no CUDA device (this library has no CPU fallback)");
  }
  if (device < 0 || device >= ndev) return fail(nullptr, TEUK_EINVAL, "teuk_select_device: no such device");
  if (cudaSetDevice(device) != cudaSuccess) {
    cudaGetLastError();
    return fail(nullptr, TEUK_ECUDA, "teuk_select_device: cudaSetDevice failed");
  }
  return TEUK_OK;
}

int teuk_measure_fp64(int32_t kind, double* lane_ops_per_s) {
  if (!lane_ops_per_s || kind < 0 || kind > 3) return fail(nullptr, TEUK_EINVAL, "teuk_measure_fp64: kind must be 0..3, output not NULL");
  int ndev = 0;
  if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev < 1) {
    cudaGetLastError();
    return fail(nullptr, TEUK_ECUDA, "teuk_measure_fp64: no CUDA device (this library has no CPU fallback)");
  }
  cudaError_t e = cudaSuccess;
  const double r = teuk_fp64_rate(kind, &e);
  if (e != cudaSuccess) return cuda_fail(nullptr, e, "teuk_measure_fp64");
  *lane_ops_per_s = r;
  return TEUK_OK;
}

int teuk_create(teuk_solver** out, double a, double M, const int32_t* m, int32_t n_modes,
                const teuk_grid* grid, double dt) {
  if (!out) return fail(nullptr, TEUK_EINVAL, "teuk_create: out is NULL");
  *out = nullptr;
  if (!m || !grid) return fail(nullptr, TEUK_EINVAL, "teuk_create: m or grid is NULL");
  if (!(M > 0.0) || !(fabs(a) < M)) return fail(nullptr, TEUK_EINVAL, "teuk_create: need M > 0 and |a| < M");
  if (n_modes < 1 || n_modes > TEUK_MAX_MODES) return fail(nullptr, TEUK_EINVAL, "teuk_create: n_modes must be 1..64");
  if (grid->n_r < 4 || grid->n_theta < 4 || grid->n_theta > 4096)
    return fail(nullptr, TEUK_EINVAL, "teuk_create: need n_r >= 4 and 4 <= n_theta <= 4096");
  if (!(grid->rs_max > grid->rs_min) || !(dt > 0.0) || !isfinite(dt) || !isfinite(grid->rs_min) ||
      !isfinite(grid->rs_max))
    return fail(nullptr, TEUK_EINVAL, "teuk_create: need rs_max > rs_min and dt > 0");
  int dev = 0, ndev = 0;
  if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev < 1) {
    cudaGetLastError();
    return fail(nullptr, TEUK_ECUDA, "teuk_create: no CUDA device (this library has no CPU fallback)");
  }
  if (cudaGetDevice(&dev) != cudaSuccess) return fail(nullptr, TEUK_ECUDA, "teuk_create: cudaGetDevice failed");
  teuk_solver* s = new (std::nothrow) teuk_solver();
  if (!s) return fail(nullptr, TEUK_ENOMEM, "teuk_create: host allocation failed");
  s->a = a; s->M = M; s->dt = dt;
  s->rs_min = grid->rs_min; s->rs_max = grid->rs_max;
  s->n_r = grid->n_r; s->n_theta = grid->n_theta; s->n_modes = n_modes;
  s->dx = (grid->rs_max - grid->rs_min) / (grid->n_r - 1);
  s->dth = kPi / grid->n_theta;
  for (int q = 0; q < n_modes; ++q) s->m[q] = m[q];
  s->outer_bc = 0; s->coef_mode = 0; s->slab_rows_opt = 0; s->use_graph = 1; s->autotune = 1; s->tuned_rows = 0; s->temporal_block = 1; s->tuned_rows2 = 0;
  s->kernel_opt = -1;
  s->wide_opt = -1;
  s->res_cache_opt = 1;
  s->use_pdl = 1;
  s->device = dev;
  if (cudaDeviceGetAttribute(&s->n_sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess) s->n_sms = 148;
  if (cudaDeviceGetAttribute(&s->smem_optin, cudaDevAttrMaxSharedMemoryPerBlockOptin, dev) != cudaSuccess) s->smem_optin = 0;
  snprintf(s->err, sizeof(s->err), "no error");
  int rc = TEUK_OK;
  do {
    const size_t nst = state_doubles(s) * sizeof(double);
    const size_t n_loc = (size_t)(2 * s->n_r - 1);
#define CKC(call, where) { cudaError_t e_ = (call); if (e_ != cudaSuccess) { rc = cuda_fail(s, e_, where); break; } }
    CKC(cudaStreamCreateWithFlags(&s->own_stream, cudaStreamNonBlocking), "stream create");
    CKC(cudaStreamCreateWithFlags(&s->copy_stream, cudaStreamNonBlocking), "stream create");
    s->stream = s->own_stream;
    CKC(cudaEventCreateWithFlags(&s->ev_compute, cudaEventDisableTiming), "event create");
    CKC(cudaEventCreateWithFlags(&s->ev_copy, cudaEventDisableTiming), "event create");
    CKC(cudaMalloc((void**)&s->d_u[0], nst), "state alloc");
    CKC(cudaMalloc((void**)&s->d_u[1], nst), "state alloc");
    CKC(cudaMalloc((void**)&s->d_rtab, (size_t)n_modes * n_loc * RT_N * sizeof(double)), "rtab alloc");
    CKC(cudaMalloc((void**)&s->d_ttab, (size_t)n_modes * TT_N * s->n_theta * sizeof(double)), "ttab alloc");
    CKC(cudaMalloc((void**)&s->d_m, n_modes * sizeof(int)), "m alloc");
    CKC(cudaMalloc((void**)&s->d_base, sizeof(long long)), "counter alloc");
    CKC(cudaMalloc((void**)&s->d_nonfinite, sizeof(int)), "flag alloc");
    CKC(cudaMemcpyAsync(s->d_m, s->m, n_modes * sizeof(int), cudaMemcpyHostToDevice, s->stream), "m copy");
    CKC(cudaMemsetAsync(s->d_u[0], 0, nst, s->stream), "state zero");
    CKC(cudaMemsetAsync(s->d_u[1], 0, nst, s->stream), "state zero");
    CKC(cudaMemsetAsync(s->d_base, 0, sizeof(long long), s->stream), "counter zero");
    CKC(cudaMemsetAsync(s->d_nonfinite, 0, sizeof(int), s->stream), "flag zero");
#undef CKC
    rc = build_tables(s);
    if (rc != TEUK_OK) break;
    cudaError_t e = cudaStreamSynchronize(s->stream);
    if (e != cudaSuccess) { rc = cuda_fail(s, e, "teuk_create sync"); break; }
    rc = tune_if_needed(s);     // launch shape of the marching kernel, measured once on the zeroed state
    if (rc != TEUK_OK) break;
  } while (0);
  if (rc != TEUK_OK) {
    snprintf(g_create_error, sizeof(g_create_error), "%s", s->err);
    teuk_destroy(s);
    return rc;
  }
  *out = s;
  return TEUK_OK;
}

int teuk_sync(teuk_solver* s) {
  if (!s) return TEUK_EINVAL;
  DeviceGuard guard(s);
  if (s->sticky) return TEUK_ECUDA;
  CK(cudaStreamSynchronize(s->stream), "teuk_sync");
  CK(cudaStreamSynchronize(s->copy_stream), "teuk_sync");
  return TEUK_OK;
}

int teuk_set_initial(teuk_solver* s, const double* phi_re, const double* phi_im, const double* pi_re,
                     const double* pi_im, int32_t ptr_is_device) {
  if (!s) return TEUK_EINVAL;
  DeviceGuard guard(s);
  if (s->sticky) return TEUK_ECUDA;
  const double* src[4] = {phi_re, phi_im, pi_re, pi_im};
  const size_t n_pts = (size_t)s->n_modes * s->n_r * s->n_theta;
  double* planes[4];
  double* scratch = s->d_u[s->cur ^ 1];
  for (int c = 0; c < 4; ++c) {
    planes[c] = nullptr;
    if (!src[c]) continue;
    if (ptr_is_device) {
      planes[c] = const_cast<double*>(src[c]);
    } else {
      planes[c] = scratch + (size_t)c * n_pts;
      CK(cudaMemcpyAsync(planes[c], src[c], n_pts * sizeof(double), cudaMemcpyHostToDevice, s->stream),
         "set_initial: H2D");
    }
  }
  CK(teuk_launch_pack(s->d_u[s->cur], planes, (size_t)s->n_modes * s->n_r, s->n_theta, s->stream),
     "set_initial: pack");
  CK(teuk_launch_set_base(s->d_base, 0, s->stream), "set_initial: counter");
  CK(cudaMemsetAsync(s->d_nonfinite, 0, sizeof(int), s->stream), "set_initial: flag");
  s->launches += 2;
  s->base_on_device = 0;
  s->step = 0;
  // series restart; pending copies of the old series must land before their buffers are freed
  CK(cudaStreamSynchronize(s->copy_stream), "set_initial: copy stream");
  reset_series(s);
  if (!ptr_is_device) CK(cudaStreamSynchronize(s->stream), "set_initial: sync");  // host arrays may be reused
  return TEUK_OK;
}

int teuk_set_source(teuk_solver* s, const teuk_orbit* orbit) {
  if (!s) return TEUK_EINVAL;
  DeviceGuard guard(s);
  if (s->sticky) return TEUK_ECUDA;
  if (orbit) {
    if (orbit->n_samples < 2 || !orbit->rs_p || !orbit->theta_p || !orbit->amp_re || !orbit->amp_im)
      return fail(s, TEUK_EINVAL, "teuk_set_source: NULL table or n_samples < 2");
    if (!(orbit->sigma_r > 0.0) || !(orbit->sigma_theta > 0.0) || orbit->half_window < 0 ||
        orbit->half_window > 4096)
      return fail(s, TEUK_EINVAL, "teuk_set_source: need sigma > 0 and 0 <= half_window <= 4096");
  }
  CK(cudaStreamSynchronize(s->stream), "set_source: sync");  // old tables may still be in use
  drop_graph(s);
  cudaFree(s->d_xp); cudaFree(s->d_thp); cudaFree(s->d_amp_re); cudaFree(s->d_amp_im);
  cudaFree(s->d_term_re); cudaFree(s->d_term_im);
  s->d_xp = s->d_thp = s->d_amp_re = s->d_amp_im = s->d_term_re = s->d_term_im = nullptr;
  s->n_terms = 0;                                           // a new trajectory starts with its single term
  s->has_source = 0;
  s->n_samples = 0;
  if (!orbit) return TEUK_OK;
  const size_t ns = (size_t)orbit->n_samples;
  CK(cudaMalloc((void**)&s->d_xp, ns * sizeof(double)), "set_source: alloc");
  CK(cudaMalloc((void**)&s->d_thp, ns * sizeof(double)), "set_source: alloc");
  CK(cudaMalloc((void**)&s->d_amp_re, ns * s->n_modes * sizeof(double)), "set_source: alloc");
  CK(cudaMalloc((void**)&s->d_amp_im, ns * s->n_modes * sizeof(double)), "set_source: alloc");
  CK(cudaMemcpyAsync(s->d_xp, orbit->rs_p, ns * sizeof(double), cudaMemcpyHostToDevice, s->stream), "set_source: H2D");
  CK(cudaMemcpyAsync(s->d_thp, orbit->theta_p, ns * sizeof(double), cudaMemcpyHostToDevice, s->stream), "set_source: H2D");
  CK(cudaMemcpyAsync(s->d_amp_re, orbit->amp_re, ns * s->n_modes * sizeof(double), cudaMemcpyHostToDevice, s->stream), "set_source: H2D");
  CK(cudaMemcpyAsync(s->d_amp_im, orbit->amp_im, ns * s->n_modes * sizeof(double), cudaMemcpyHostToDevice, s->stream), "set_source: H2D");
  CK(cudaStreamSynchronize(s->stream), "set_source: sync");  // caller may free its arrays on return
  s->has_source = 1;
  s->n_samples = orbit->n_samples;
  s->sigma_r = orbit->sigma_r;
  s->sigma_th = orbit->sigma_theta;
  s->W = orbit->half_window;
  return TEUK_OK;
}

int teuk_set_source_terms(teuk_solver* s, int32_t n_terms, const int32_t* order_r, const int32_t* order_theta,
                          const double* amp_re, const double* amp_im) {
  if (!s) return TEUK_EINVAL;
  DeviceGuard guard(s);
  if (s->sticky) return TEUK_ECUDA;
  if (n_terms < 0 || n_terms > TEUK_MAX_TERMS) return fail(s, TEUK_EINVAL, "teuk_set_source_terms: n_terms must be 0..12");
  if (n_terms > 0 && !s->has_source)
    return fail(s, TEUK_EINVAL, "teuk_set_source_terms: install the trajectory with teuk_set_source first");
  if (n_terms > 0 && (!order_r || !order_theta || !amp_re || !amp_im))
    return fail(s, TEUK_EINVAL, "teuk_set_source_terms: NULL array");
  if (n_terms > 0 && (s->variant == 1 || s->temporal_block == 2 || s->coef_mode != 0))
    return fail(s, TEUK_EINVAL, "teuk_set_source_terms: needs kernel -1, 0 or 2, temporal_block 1 and coef_mode 0");
  for (int t = 0; t < n_terms; ++t)
    if (order_r[t] < 0 || order_r[t] > 2 || order_theta[t] < 0 || order_theta[t] > 2)
      return fail(s, TEUK_EINVAL, "teuk_set_source_terms: derivative orders must be 0, 1 or 2");
  CK(cudaStreamSynchronize(s->stream), "set_source_terms: sync");   // the old tables may still be in use
  drop_graph(s);
  cudaFree(s->d_term_re); cudaFree(s->d_term_im);
  s->d_term_re = s->d_term_im = nullptr;
  const bool had_terms = s->n_terms > 0;
  s->n_terms = 0;
  if (n_terms == 0) {
    if (had_terms) { s->tuned_rows = 0; return tune_if_needed(s); }
    return TEUK_OK;
  }
  const size_t n = (size_t)n_terms * s->n_modes * (size_t)s->n_samples;
  CK(cudaMalloc((void**)&s->d_term_re, n * sizeof(double)), "set_source_terms: alloc");
  CK(cudaMalloc((void**)&s->d_term_im, n * sizeof(double)), "set_source_terms: alloc");
  CK(cudaMemcpyAsync(s->d_term_re, amp_re, n * sizeof(double), cudaMemcpyHostToDevice, s->stream), "set_source_terms: H2D");
  CK(cudaMemcpyAsync(s->d_term_im, amp_im, n * sizeof(double), cudaMemcpyHostToDevice, s->stream), "set_source_terms: H2D");
  CK(cudaStreamSynchronize(s->stream), "set_source_terms: sync");   // the caller may free its arrays on return
  for (int t = 0; t < n_terms; ++t) {
    s->term_or[t] = (signed char)order_r[t];
    s->term_oth[t] = (signed char)order_theta[t];
  }
  s->n_terms = n_terms;
  s->tuned_rows = 0;               // another kernel instantiation runs from now on: measure its launch shape
  return tune_if_needed(s);
}

}  // extern "C"

namespace {

// Capture kGraphBatch tapping iterations + the counter bump for the current ping-pong parity
// (tb = 2: kGraphBatch / 2 temporal-blocking launches of two iterations each).
int build_graph(teuk_solver* s, int tb) {
  cudaGraph_t graph = nullptr;
  CK(cudaStreamBeginCapture(s->own_stream, cudaStreamCaptureModeThreadLocal), "graph: begin capture");
  cudaError_t e = cudaSuccess;
  const bool sep_tap = seg_factor(s) > 1 && s->n_obs > 0;   // theta segments: the tap is its own small kernel
  if (tb == 2) {
    for (int j = 0; j < kGraphBatch / 2 && e == cudaSuccess; ++j) {
      StepParams p;
      fill_params(s, &p, s->cur ^ (j & 1), 2 * j, 1, 2);
      e = teuk_launch_step_tb2(p, s->own_stream);
    }
  } else {
    for (int k = 0; k < kGraphBatch && e == cudaSuccess; ++k) {
      StepParams p;
      fill_params(s, &p, s->cur ^ (k & 1), k, sep_tap ? 0 : 1);
      // iterations 2..32 of the batch follow another step kernel directly: their prologue may overlap its tail
      p.pdl = (s->use_pdl && k > 0 && !sep_tap && s->variant == 0) ? 1 : 0;
      e = launch_step_any(s, p, s->own_stream);
      if (sep_tap && e == cudaSuccess) {
        fill_params(s, &p, s->cur ^ ((k + 1) & 1), k + 1, 1);
        e = teuk_launch_flush_tap(p, s->own_stream);
      }
    }
  }
  if (e == cudaSuccess) e = teuk_launch_bump(s->d_base, kGraphBatch, s->own_stream);
  cudaError_t e2 = cudaStreamEndCapture(s->own_stream, &graph);
  if (e != cudaSuccess) { if (graph) cudaGraphDestroy(graph); return cuda_fail(s, e, "graph: capture launch"); }
  CK(e2, "graph: end capture");
  e = cudaGraphInstantiate(tb == 2 ? &s->graph_exec_tb2[s->cur] : &s->graph_exec[s->cur], graph, 0);
  cudaGraphDestroy(graph);
  CK(e, "graph: instantiate");
  return TEUK_OK;
}

// One-time measurement of the slab length: the march of a slab is serial, so the
// best length depends on grid size, mode count and wave quantisation.  Candidates are timed with the real
// kernel reading the current level and writing the idle ping-pong buffer (tap off): the state, the
// iteration counter and the recorded series are untouched, and results do not depend on the slab length.
int tune_slab_rows(teuk_solver* s, int tb) {
  const double waves[] = {0.95, 1.9, 2.0, 2.9, 3.9, 5.8};
  int cand[64];
  int nc = 0;
  const int interior = s->n_r - 2;
  auto add = [&](long long n) {                        // candidate: n slabs per mode
    if (n < 1) n = 1;
    if (n > interior) n = interior;
    for (int q = 0; q < nc; ++q)
      if (cand[q] == (int)n) return;
    if (nc < 64) cand[nc++] = (int)n;
  };
  const int base = auto_slab_rows(s, tb);
  if (base <= 24) {
    const int small[] = {1, 2, 3, 4, 5, 6, 7, 8, 10, 12, 14, 16, 20, 24};   // small grids: wave quantisation is coarse
    for (int r : small) add(slabs_for_rows(s, r));
  } else {
    for (double w : waves) {
      const int r = rows_for_waves(s, w, tb);
      add(slabs_for_rows(s, r));
      add(slabs_for_rows(s, r + (r + 9) / 10));        // and its +-10 % neighbours
      add(slabs_for_rows(s, r - (r + 9) / 10));
    }
  }
  // whole numbers of waves: k times the warps that are resident at once, shared by the modes and theta segments
  const long long per_wave = (long long)resident_warps(s) / tb / ((long long)s->n_modes * seg_factor(s));
  for (int k = 1; k <= 6; ++k) add(k * per_wave);
  cudaEvent_t e0, e1;
  CK(cudaEventCreate(&e0), "autotune: event");
  CK(cudaEventCreate(&e1), "autotune: event");
  float best = 1e30f;
  int best_slabs = slabs_for_rows(s, base);
  for (int q = 0; q < nc; ++q) {
    s->force_slabs = cand[q];
    StepParams p;
    fill_params(s, &p, s->cur, (int)(s->step - s->base_on_device), 0, tb);
    p.tap_enable2 = 0;
    p.has_source = 0;      // trial launches read nothing but the state and the tables (no trajectory sample, no observer)
    p.n_obs = 0;
    // launched like iterations 2..32 of a graph batch (programmatic dependent launch), so that what is timed is
    // the back-to-back rate of production and not the gap between two plain launches
    p.pdl = (tb == 1 && s->use_pdl && s->variant == 0 && seg_factor(s) == 1) ? 1 : 0;
    auto launch = [&]() { return tb == 2 ? teuk_launch_step_tb2(p, s->stream) : launch_step_any(s, p, s->stream); };
    cudaError_t e = launch();                                      // warm-up
    float ms = 0.f;
    int reps = 3;
    for (int pass = 0; pass < 3 && e == cudaSuccess; ++pass) {   // short kernels: time at least ~1 ms of launches
      e = cudaEventRecord(e0, s->stream);
      for (int r = 0; r < reps && e == cudaSuccess; ++r) e = launch();
      if (e == cudaSuccess) e = cudaEventRecord(e1, s->stream);
      if (e == cudaSuccess) e = cudaEventSynchronize(e1);
      if (e == cudaSuccess) e = cudaEventElapsedTime(&ms, e0, e1);
      s->launches += reps;
      const float total = ms;
      ms /= reps;
      if (total > 1.0f || pass == 2) break;
      reps *= 8;
    }
    if (e == cudaSuccess) {   // once more at the final repetition count: the smaller of the two (clock ramps, stragglers)
      float ms2 = 0.f;
      e = cudaEventRecord(e0, s->stream);
      for (int r = 0; r < reps && e == cudaSuccess; ++r) e = launch();
      if (e == cudaSuccess) e = cudaEventRecord(e1, s->stream);
      if (e == cudaSuccess) e = cudaEventSynchronize(e1);
      if (e == cudaSuccess) e = cudaEventElapsedTime(&ms2, e0, e1);
      s->launches += reps;
      if (e == cudaSuccess && ms2 / reps < ms) ms = ms2 / reps;
    }
    s->launches += 1;
    if (e != cudaSuccess) {
      s->force_slabs = 0;
      cudaEventDestroy(e0);
      cudaEventDestroy(e1);
      return cuda_fail(s, e, "autotune");
    }
    if (ms < best) { best = ms; best_slabs = cand[q]; }
  }
  s->force_slabs = 0;
  if (tb == 2) s->tuned_rows2 = best_slabs; else s->tuned_rows = best_slabs;
  cudaEventDestroy(e0);
  cudaEventDestroy(e1);
  return TEUK_OK;
}

// Measure the launch shape of the marching kernels the solver would run now, if it has not been measured yet.
// Called from teuk_create and teuk_set_option (both wait for the stream anyway), never from teuk_step.
int tune_if_needed(teuk_solver* s) {
  int rr_ = 0, nc_ = 0;
  if (!s->autotune || s->slab_rows_opt != 0 || resident_active(s, &rr_, &nc_)) return TEUK_OK;
  if (s->tuned_rows == 0) {
    const int rc = tune_slab_rows(s, 1);
    if (rc != TEUK_OK) return rc;
    drop_graph(s);
  }
  if (tb2_active(s) && s->tuned_rows2 == 0) {
    const int rc = tune_slab_rows(s, 2);
    if (rc != TEUK_OK) return rc;
    drop_graph(s);
  }
  return TEUK_OK;
}

// Run c >= 1 iterations whose samples fit in the ring.
int run_chunk(teuk_solver* s, long long c) {
  long long left = c;
  int first = 1;
  const bool tb2 = tb2_active(s);
  if (resident_active(s, &s->res_rows, &s->res_ncta)) {   // all c iterations in one cooperative launch, state on chip in between
    if (!s->d_ll) {
      const size_t bytes = teuk_resident_ll_bytes(s->n_theta, s->n_modes, s->res_ncta);
      CK(cudaMalloc(&s->d_ll, bytes), "resident: exchange buffer alloc");
      CK(cudaMemsetAsync(s->d_ll, 0, bytes, s->stream), "resident: exchange buffer zero");
      s->ll_tag = 0;
    }
    while (left > 0) {
      const long long k = s->step - s->base_on_device;
      if (k < 0 || k > (1LL << 30)) {
        CK(teuk_launch_set_base(s->d_base, s->step, s->stream), "step: counter");
        s->base_on_device = s->step;
        s->launches += 1;
      }
      const long long m = left < (1LL << 30) ? left : (1LL << 30);
      if ((unsigned long long)s->ll_tag + (unsigned long long)m >= 0xfffffff0ull) {   // tags would wrap: start over
        CK(cudaMemsetAsync(s->d_ll, 0, teuk_resident_ll_bytes(s->n_theta, s->n_modes, s->res_ncta), s->stream),
           "resident: exchange buffer zero");
        s->ll_tag = 0;
      }
      StepParams p;
      fill_params(s, &p, s->cur, (int)(s->step - s->base_on_device), 0);   // level s->step was tapped by the last flush
      p.n_iter = (int)m;
      p.res_rows = s->res_rows;
      p.res_cache = s->res_cache_opt && s->n_terms == 0 &&
                    teuk_resident_smem_bytes(s->n_theta, s->res_rows, 1) <= (size_t)s->smem_optin;
      p.tag0 = s->ll_tag;
      p.ll = s->d_ll;
      const cudaError_t el = teuk_launch_step_resident(p, s->res_ncta, s->stream);
      if (el != cudaSuccess && s->kernel_opt == -1 &&
          (el == cudaErrorCooperativeLaunchTooLarge || el == cudaErrorNotSupported || el == cudaErrorLaunchOutOfResources)) {
        cudaGetLastError();        // the automatic choice does not apply on this device: kernel 0 from now on
        s->res_failed = 1;
        break;
      }
      CK(el, "step: resident launch");
      s->ll_tag += (unsigned)m;
      s->launches += 1;
      s->cur ^= 1;
      s->step += m;
      left -= m;
    }
  }
  while (left > 0) {
    const bool graph_ok = s->use_graph && !first && left >= kGraphBatch;
    if (graph_ok) {
      cudaGraphExec_t* ge = tb2 ? &s->graph_exec_tb2[s->cur] : &s->graph_exec[s->cur];
      if (!*ge) {
        const int rc = build_graph(s, tb2 ? 2 : 1);
        if (rc != TEUK_OK) return rc;
      }
      if (s->base_on_device != s->step) {
        CK(teuk_launch_set_base(s->d_base, s->step, s->stream), "step: counter");
        s->base_on_device = s->step;
        s->launches += 1;
      }
      CK(cudaGraphLaunch(*ge, s->stream), "step: graph launch");
      s->base_on_device += kGraphBatch;
      s->step += kGraphBatch;
      s->launches += (tb2 ? kGraphBatch / 2 : kGraphBatch * (seg_factor(s) > 1 && s->n_obs > 0 ? 2 : 1)) + 1;
      left -= kGraphBatch;
      continue;
    }
    const long long k = s->step - s->base_on_device;
    if (k < 0 || k > (1LL << 30)) {
      CK(teuk_launch_set_base(s->d_base, s->step, s->stream), "step: counter");
      s->base_on_device = s->step;
      s->launches += 1;
    }
    if (tb2 && left >= 2) {   // two iterations, level n+1 stays on chip
      StepParams p;
      fill_params(s, &p, s->cur, (int)(s->step - s->base_on_device), first ? 0 : 1, 2);
      CK(teuk_launch_step_tb2(p, s->stream), "step: temporal-blocking launch");
      s->launches += 1;
      s->cur ^= 1;
      s->step += 2;
      left -= 2;
      first = 0;
      continue;
    }
    const bool sep_tap = seg_factor(s) > 1 && s->n_obs > 0;
    StepParams p;
    fill_params(s, &p, s->cur, (int)(s->step - s->base_on_device), (first || sep_tap) ? 0 : 1);
    CK(launch_step_any(s, p, s->stream), "step: launch");
    s->launches += 1;
    s->cur ^= 1;
    s->step += 1;
    left -= 1;
    first = 0;
    if (sep_tap && left > 0) {   // the level just produced (the last one is tapped below)
      fill_params(s, &p, s->cur, (int)(s->step - s->base_on_device), 1);
      CK(teuk_launch_flush_tap(p, s->stream), "step: tap");
      s->launches += 1;
    }
  }
  if (s->n_obs > 0) {
    StepParams p;
    fill_params(s, &p, s->cur, (int)(s->step - s->base_on_device), 1);
    CK(teuk_launch_flush_tap(p, s->stream), "step: flush tap");
    s->launches += 1;
    s->recorded = s->step;
  }
  return TEUK_OK;
}

}  // namespace

extern "C" {

int teuk_step(teuk_solver* s, int64_t n) {
  if (!s) return TEUK_EINVAL;
  DeviceGuard guard(s);
  if (s->sticky) return TEUK_ECUDA;
  if (n < 0) return fail(s, TEUK_EINVAL, "teuk_step: n < 0");
  if (s->has_source && 2 * (s->step + n) > s->n_samples)
    return fail(s, TEUK_EINVAL, "teuk_step: trajectory table too short for n more iterations");
  long long remaining = n;
  while (remaining > 0) {
    long long room = remaining;
    if (s->n_obs > 0) {
      room = kRingCap - (s->recorded - s->drained);
      if (room <= 0) {
        const int rc = drain_rings(s);
        if (rc != TEUK_OK) return rc;
        continue;
      }
    }
    const long long c = remaining < room ? remaining : room;
    const int rc = run_chunk(s, c);
    if (rc != TEUK_OK) return rc;
    remaining -= c;
  }
  return TEUK_OK;
}

// Allocation-free variant of set_initial(device) + step(n) + get_state(device) on the resident kernel, with the
// exchange scratch in a static device array (teuk_resident.cu).  Calls no cudaMalloc / cudaFree / cudaMallocHost /
// cudaFreeHost and waits for nothing: three kernels, one memset and at most one counter kernel are enqueued.
int teuk_step_noalloc(teuk_solver* s, const double* const in_dev[4], int64_t n0, int64_t n, double* const out_dev[4]) {
  if (!s) return TEUK_EINVAL;
  DeviceGuard guard(s);
  if (s->sticky) return TEUK_ECUDA;
  if (!in_dev || !out_dev) return fail(s, TEUK_EINVAL, "teuk_step_noalloc: in_dev / out_dev is NULL");
  if (n < 1 || n > (1LL << 30) || n0 < 0) return fail(s, TEUK_EINVAL, "teuk_step_noalloc: need n0 >= 0 and 1 <= n <= 2^30");
  if (s->n_obs > 0) return fail(s, TEUK_EINVAL, "teuk_step_noalloc: not available with armed observers (their drains allocate)");
  if (s->variant == 1 || s->temporal_block != 1 || s->coef_mode != 0)
    return fail(s, TEUK_EINVAL, "teuk_step_noalloc: needs kernel -1, 0 or 2, temporal_block 1, coef_mode 0");
  int rows = 0, ncta = 0;
  if (!resident_plan(s, &rows, &ncta))
    return fail(s, TEUK_EINVAL, "teuk_step_noalloc: the state does not fit on chip (resident kernel: n_theta <= 128 and about n_modes*n_r*n_theta <= 5e5 points)");
  const size_t need = teuk_resident_ll_bytes(s->n_theta, s->n_modes, ncta);
  if (need > teuk_resident_static_capacity()) {
    char buf[200];
    snprintf(buf, sizeof(buf), "teuk_step_noalloc: exchange scratch of %zu bytes exceeds the static maximum of %zu bytes",
             need, teuk_resident_static_capacity());
    return fail(s, TEUK_EINVAL, buf);
  }
  if (s->has_source && 2 * (n0 + n) > s->n_samples)
    return fail(s, TEUK_EINVAL, "teuk_step_noalloc: trajectory table too short for n0 + n iterations");
  double* planes[4];
  for (int c = 0; c < 4; ++c) planes[c] = const_cast<double*>(in_dev[c]);
  CK(teuk_launch_pack(s->d_u[s->cur], planes, (size_t)s->n_modes * s->n_r, s->n_theta, s->stream), "step_noalloc: pack");
  s->launches += 1;
  const long long k = n0 - s->base_on_device;
  if (k < 0 || k > (1LL << 30)) {
    CK(teuk_launch_set_base(s->d_base, n0, s->stream), "step_noalloc: counter");
    s->base_on_device = n0;
    s->launches += 1;
  }
  StepParams p;                        // (captured graphs of kernel 0 stay valid: they address the buffers by parity)
  fill_params(s, &p, s->cur, (int)(n0 - s->base_on_device), 0);
  p.n_iter = (int)n;
  p.res_rows = rows;
  p.res_cache = s->res_cache_opt && s->n_terms == 0 &&
                teuk_resident_smem_bytes(s->n_theta, rows, 1) <= (size_t)s->smem_optin;
  CK(teuk_launch_step_resident_static(p, ncta, s->stream), "step_noalloc: resident launch");
  s->launches += 1;
  s->cur ^= 1;
  s->step = n0 + n;
  for (int c = 0; c < 4; ++c) planes[c] = out_dev[c];
  CK(teuk_launch_unpack(s->d_u[s->cur], planes, (size_t)s->n_modes * s->n_r, s->n_theta, s->stream), "step_noalloc: unpack");
  s->launches += 1;
  return TEUK_OK;
}

int teuk_extract(teuk_solver* s, double rs_obs, const double* weights, double* t_out, double* w_re,
                 double* w_im, int64_t capacity, int64_t* n_written) {
  if (!s) return TEUK_EINVAL;
  DeviceGuard guard(s);
  if (s->sticky) return TEUK_ECUDA;
  if (n_written) *n_written = 0;
  int q = -1;
  for (int k = 0; k < s->n_obs; ++k)
    if (s->obs[k].rs_obs == rs_obs) q = k;
  if (q < 0) {  // arm a new observer
    if (s->n_obs >= TEUK_MAX_OBS) return fail(s, TEUK_EINVAL, "teuk_extract: too many observers");
    if (s->step != 0) return fail(s, TEUK_EINVAL, "teuk_extract: arm observers before stepping (after teuk_set_initial)");
    const double v = (rs_obs - s->rs_min) / s->dx;
    const int i0 = (int)floor(v);
    if (!(v >= 0.0) || i0 > s->n_r - 2) return fail(s, TEUK_EINVAL, "teuk_extract: rs_obs outside [x_0, x_{n_r-1})");
    CK(cudaStreamSynchronize(s->stream), "extract: sync");
    drop_graph(s);
    ObsHost* o = &s->obs[s->n_obs];
    o->rs_obs = rs_obs;
    o->i0 = i0;
    o->f = v - i0;
    o->read_cursor = 1;
    o->d_weights = nullptr;
    o->d_ring = nullptr;
    std::vector<double> w((size_t)s->n_theta, 1.0);
    if (weights) memcpy(w.data(), weights, (size_t)s->n_theta * sizeof(double));
    CK(cudaMalloc((void**)&o->d_weights, (size_t)s->n_theta * sizeof(double)), "extract: alloc");
    CK(cudaMalloc((void**)&o->d_ring, (size_t)kRingCap * s->n_modes * 2 * sizeof(double)), "extract: alloc");
    // on the solver's stream (the legacy default stream is not ordered against it), then wait: `w` is local
    CK(cudaMemcpyAsync(o->d_weights, w.data(), (size_t)s->n_theta * sizeof(double), cudaMemcpyHostToDevice, s->stream), "extract: H2D");
    CK(cudaMemsetAsync(o->d_ring, 0, (size_t)kRingCap * s->n_modes * 2 * sizeof(double), s->stream), "extract: zero");
    CK(cudaStreamSynchronize(s->stream), "extract: sync");
    s->n_obs += 1;
    return TEUK_OK;
  }
  if (capacity < 0 || (capacity > 0 && (!t_out || !w_re || !w_im)) || !n_written)
    return fail(s, TEUK_EINVAL, "teuk_extract: NULL output or negative capacity");
  int rc = drain_rings(s);
  if (rc != TEUK_OK) return rc;
  CK(cudaStreamSynchronize(s->copy_stream), "extract: sync copies");
  CK(cudaStreamSynchronize(s->stream), "extract: sync");
  int nonfinite = 0;
  CK(cudaMemcpyAsync(&nonfinite, s->d_nonfinite, sizeof(int), cudaMemcpyDeviceToHost, s->stream), "extract: flag");
  CK(cudaStreamSynchronize(s->stream), "extract: flag sync");
  ObsHost* o = &s->obs[q];
  int64_t written = 0;
  size_t ci = 0;
  while (written < capacity && ci < o->chunks.size()) {
    HostChunk& ch = o->chunks[ci];
    const long long end = ch.first + ch.count;  // one past the last sample of this chunk
    if (o->read_cursor >= end) { ++ci; continue; }
    const long long off = o->read_cursor - ch.first;
    for (int k = 0; k < s->n_modes; ++k) {
      w_re[written * s->n_modes + k] = ch.data[((size_t)off * s->n_modes + k) * 2 + 0];
      w_im[written * s->n_modes + k] = ch.data[((size_t)off * s->n_modes + k) * 2 + 1];
    }
    t_out[written] = (double)o->read_cursor * s->dt;
    o->read_cursor += 1;
    written += 1;
  }
  // release fully consumed chunks
  while (!o->chunks.empty() && o->read_cursor >= o->chunks.front().first + o->chunks.front().count) {
    cudaFreeHost(o->chunks.front().data);
    o->chunks.erase(o->chunks.begin());
  }
  *n_written = written;
  if (nonfinite) return fail(s, TEUK_ENONFINITE, "teuk_extract: a tapped sample was NaN/Inf");
  return TEUK_OK;
}

int teuk_get_state(teuk_solver* s, double* phi_re, double* phi_im, double* pi_re, double* pi_im,
                   int32_t ptr_is_device) {
  if (!s) return TEUK_EINVAL;
  DeviceGuard guard(s);
  if (s->sticky) return TEUK_ECUDA;
  double* dst[4] = {phi_re, phi_im, pi_re, pi_im};
  const size_t n_pts = (size_t)s->n_modes * s->n_r * s->n_theta;
  double* planes[4];
  double* scratch = s->d_u[s->cur ^ 1];
  for (int c = 0; c < 4; ++c) planes[c] = dst[c] ? (ptr_is_device ? dst[c] : scratch + (size_t)c * n_pts) : nullptr;
  CK(teuk_launch_unpack(s->d_u[s->cur], planes, (size_t)s->n_modes * s->n_r, s->n_theta, s->stream),
     "get_state: unpack");
  s->launches += 1;
  if (!ptr_is_device) {
    for (int c = 0; c < 4; ++c)
      if (dst[c])
        CK(cudaMemcpyAsync(dst[c], planes[c], n_pts * sizeof(double), cudaMemcpyDeviceToHost, s->stream),
           "get_state: D2H");
    CK(cudaStreamSynchronize(s->stream), "get_state: sync");
  }
  return TEUK_OK;
}

int teuk_set_option(teuk_solver* s, const char* key, int64_t value) {
  if (!s || !key) return TEUK_EINVAL;
  DeviceGuard guard(s);
  if (s->sticky) return TEUK_ECUDA;
  CK(cudaStreamSynchronize(s->stream), "set_option: sync");
  if (!strcmp(key, "outer_bc")) {
    if (value != 0 && value != 1) return fail(s, TEUK_EINVAL, "outer_bc must be 0 or 1");
    s->outer_bc = (int)value;
  } else if (!strcmp(key, "source_kind")) {
    if (value < 0 || value > 2) return fail(s, TEUK_EINVAL, "source_kind must be 0 (Gaussian), 1 or 2 (discrete delta)");
    s->source_kind = (int)value;
  } else if (!strcmp(key, "stream")) {
    s->stream = value ? (cudaStream_t)(uintptr_t)value : s->own_stream;
  } else if (!strcmp(key, "coef_mode")) {
    if (value != 0 && value != 1) return fail(s, TEUK_EINVAL, "coef_mode must be 0 or 1");
    if (value == 1 && s->variant != 0) return fail(s, TEUK_EINVAL, "coef_mode 1 needs kernel 0");
    if (value == 1 && s->n_terms > 0) return fail(s, TEUK_EINVAL, "coef_mode 1 is not available with teuk_set_source_terms");
    if (value == 1 && n_segments(s) > 1) return fail(s, TEUK_EINVAL, "coef_mode 1 needs n_theta <= 128");
    if (value == 1 && s->temporal_block == 2) return fail(s, TEUK_EINVAL, "coef_mode 1 needs temporal_block 1");
    if (value == 1 && !s->d_coef2d) {
      const size_t bytes = (size_t)s->n_modes * (2 * (size_t)s->n_r - 1) * 8 * s->n_theta * sizeof(double);
      CK(cudaMalloc((void**)&s->d_coef2d, bytes), "coef_mode: alloc of the 2D coefficient planes");
      CK(teuk_launch_coef2d(s->d_coef2d, s->d_rtab, s->d_ttab, s->n_modes, s->n_r, s->n_theta, s->dx, s->stream),
         "coef_mode: plane kernel");
      s->launches += 1;
    }
    s->coef_mode = (int)value;
  } else if (!strcmp(key, "slab_rows")) {
    if (value < 0 || value > (1 << 30)) return fail(s, TEUK_EINVAL, "slab_rows out of range");
    s->slab_rows_opt = (int)value;
  } else if (!strcmp(key, "graph")) {
    s->use_graph = value ? 1 : 0;
  } else if (!strcmp(key, "wide")) {
    if (value < -1 || value > 1) return fail(s, TEUK_EINVAL, "wide must be -1 (automatic), 0 or 1");
    if (value == 1 && !teuk_wide_applies(s->n_theta))
      return fail(s, TEUK_EINVAL, "wide 1 needs an even n_theta between 66 and 320");
    s->wide_opt = (int)value;
  } else if (!strcmp(key, "pdl")) {
    s->use_pdl = value ? 1 : 0;
  } else if (!strcmp(key, "resident_cache")) {
    s->res_cache_opt = value ? 1 : 0;
  } else if (!strcmp(key, "autotune")) {
    s->autotune = value ? 1 : 0;
  } else if (!strcmp(key, "temporal_block")) {
    if (value != 1 && value != 2) return fail(s, TEUK_EINVAL, "temporal_block must be 1 or 2");
    if (value == 2 && s->n_terms > 0) return fail(s, TEUK_EINVAL, "temporal_block 2 is not available with teuk_set_source_terms");
    s->temporal_block = (int)value;
    if (value == 2 && (!tb2_possible(s) || s->kernel_opt == 2)) {
      s->temporal_block = 1;
      return fail(s, TEUK_EINVAL, "temporal_block 2 needs kernel 0, coef_mode 0, n_theta <= 128 and a multiple of its lane width (1, 2 or 4)");
    }
  } else if (!strcmp(key, "kernel")) {
    if (value < -1 || value > 2)
      return fail(s, TEUK_EINVAL, "kernel must be -1 (automatic), 0 (register-resident), 1 (shared-memory-resident) or 2 (resident, whole state on chip)");
    if (value > 0 && s->coef_mode != 0) return fail(s, TEUK_EINVAL, "kernels 1 and 2 need coef_mode 0");
    if (value == 1 && s->n_terms > 0) return fail(s, TEUK_EINVAL, "kernel 1 is not available with teuk_set_source_terms");
    if (value == 2) {
      if (s->temporal_block == 2) return fail(s, TEUK_EINVAL, "kernel 2 needs temporal_block 1");
      if (!resident_plan(s, &s->res_rows, &s->res_ncta))
        return fail(s, TEUK_EINVAL, "kernel 2 needs n_theta <= 128 and a state that fits in the shared memory of one block per SM");
    }
    if (value == 1 && s->n_theta > 256) return fail(s, TEUK_EINVAL, "kernel 1 needs n_theta <= 256");
    if (value == 1 && s->temporal_block == 2) return fail(s, TEUK_EINVAL, "kernel 1 needs temporal_block 1");
    s->kernel_opt = (int)value;
    s->variant = value < 0 ? 0 : (int)value;
  } else {
    return fail(s, TEUK_EINVAL, "teuk_set_option: unknown key");
  }
  drop_graph(s);
  // options that change the launch shape of the marching kernels: measure it again, here, so that teuk_step
  // never has to wait for the device
  if (!strcmp(key, "kernel") || !strcmp(key, "coef_mode") || !strcmp(key, "temporal_block") || !strcmp(key, "wide") ||
      !strcmp(key, "slab_rows") || !strcmp(key, "autotune")) {
    s->tuned_rows = 0;
    s->tuned_rows2 = 0;
    return tune_if_needed(s);
  }
  return TEUK_OK;
}

int teuk_get_stat(const teuk_solver* s, const char* key, int64_t* value) {
  if (!s || !key || !value) return TEUK_EINVAL;
  if (!strcmp(key, "steps")) *value = s->step;
  else if (!strcmp(key, "launches")) *value = s->launches;
  else if (!strcmp(key, "n_pts")) *value = (int64_t)s->n_modes * s->n_r * s->n_theta;
  else if (!strcmp(key, "state_bytes")) *value = (int64_t)(state_doubles(s) * sizeof(double));
  else if (!strcmp(key, "kernel") || !strcmp(key, "resident_rows") || !strcmp(key, "resident_blocks")) {
    int rr = 0, nc = 0;
    const bool res = resident_active(s, &rr, &nc);
    if (!strcmp(key, "kernel")) *value = res ? 2 : s->variant;
    else if (!strcmp(key, "resident_rows")) *value = res ? rr : 0;
    else *value = res ? (int64_t)nc * s->n_modes : 0;
  }
  else if (!strcmp(key, "wide")) {
    int rr = 0, nc = 0;
    *value = (!resident_active(s, &rr, &nc) && wide_active(s)) ? 1 : 0;
  }
  else if (!strcmp(key, "slabs")) *value = slabs_in_use(s, tb2_active(s) ? 2 : 1);
  else if (!strcmp(key, "slab_rows")) {                 // longest slab in use
    const int n = slabs_in_use(s, tb2_active(s) ? 2 : 1);
    *value = (s->n_r - 2 + n - 1) / n;
  }
  else return TEUK_EINVAL;
  return TEUK_OK;
}

}  // extern "C"
