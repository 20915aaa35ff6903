/* teuk.h -- C ABI of libteuk.so: the FP64 two-step Lax-Wendroff time step of the 2+1D Teukolsky
 * equation (s = -2) on one NVIDIA B200 (sm_100a), after arXiv:1206.0270 section 2.2.
 *
 * What the library computes (citations are /root/reference/PAPER.md lines):
 *   - the first-order system u = {Phi_R, Phi_I, Pi_R, Pi_I} of the m-mode reduction
 *     Psi = sum_m e^{im phi~} r^3 Phi_m (Eq. 2) of the Teukolsky master equation
 *     (Eq. 1), with the coefficient matrices D and S evaluated on
 *     the device in closed form;
 *   - one iteration = half step (Eq. 3) + full step (Eq. 4), with
 *     second-order centred theta differences, pole parity conditions and radial edge
 *     conditions;
 *   - a Gaussian-smeared point-particle source deposited on the device each stage (PAPER.md:114,
 *     :151) from a sampled trajectory the caller supplies;
 *   - the waveform at a fixed r* (PAPER.md:161), tapped on the device into a ring buffer.
 * Every step runs in CUDA kernels; there is no CPU fallback.  Readings of passages where the paper
 * is silent are listed in DESIGN.md.
 *
 * Conventions
 *   - Grid: x_i = rs_min + i*dx, i = 0..n_r-1, dx = (rs_max - rs_min)/(n_r - 1) (both end points);
 *     theta_j = (j + 1/2)*pi/n_theta, j = 0..n_theta-1.  x is the tortoise coordinate r*.
 *   - Field arrays at this boundary are FP64, shape [n_modes][n_r][n_theta], theta fastest, one
 *     array per component (Phi_R, Phi_I, Pi_R, Pi_I).  (The internal device layout differs.)
 *   - A pointer argument is a HOST pointer unless the call has a `ptr_is_device` flag that is 1.
 *   - The caller owns every array it passes; the library copies what it needs before returning
 *     (host arrays) or enqueues the copy on the solver's stream (device arrays).
 *   - All device work is enqueued on the solver's stream (its own, or the one set with the
 *     "stream" option); only teuk_extract, teuk_get_state(host), teuk_sync wait for it.
 *   - Every function returns TEUK_OK (0) or a negative teuk_status; teuk_last_error gives text.
 *     No exceptions, no aborts, no output on stdout/stderr.
 *   - Not thread-safe per solver; distinct solvers may be used from distinct threads.
 */
#ifndef TEUK_H_
#define TEUK_H_

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef enum {
  TEUK_OK = 0,
  TEUK_EINVAL = -1,     /* bad parameter, NULL where not allowed, trajectory too short for n     */
  TEUK_ENOMEM = -2,     /* host or device allocation failed                                       */
  TEUK_ECUDA = -3,      /* CUDA error (sticky: the solver is unusable afterwards), or no device.
                           Every wait inside the kernels is bounded; one that times out (a faulted copy,
                           a lost neighbour block) executes `trap`, which is reported here -- and, like any
                           device-side fault, poisons the process's CUDA context, not only this solver   */
  TEUK_ENONFINITE = -4  /* a NaN/Inf was seen on a tapped waveform sample                         */
} teuk_status;

typedef struct teuk_solver teuk_solver; /* opaque; created and destroyed by the library */

typedef struct {
  double rs_min, rs_max; /* tortoise-coordinate range, rs_max > rs_min                            */
  int32_t n_r, n_theta;  /* n_r >= 4; 4 <= n_theta <= 4096                                         */
} teuk_grid;

/* Sampled particle trajectory and source amplitude (C.6 of DESIGN.md).
 * Sample k is at t = k*dt/2 counted from the last teuk_set_initial: the half step of iteration n
 * uses sample 2n (at the half points x_{i+1/2}), the full step uses sample 2n+1 (at the nodes).
 * The deposited term is T(t,x,theta) = A'_m(t) g(x - x_p; sigma_r) g(theta - theta_p; sigma_theta),
 * g(y;s) = exp(-y^2/(2 s^2))/(s sqrt(2 pi)), inside |i - i_p| <= W, |j - j_p| <= W only. */
typedef struct {
  int64_t n_samples;             /* >= 2 * (iterations to run)                                   */
  const double *rs_p, *theta_p;  /* [n_samples] particle r*, theta                                */
  const double *amp_re, *amp_im; /* [n_modes][n_samples] complex amplitude A'_m                   */
  double sigma_r, sigma_theta;   /* Gaussian widths in r* and theta, absolute units, > 0          */
  int32_t half_window;           /* W cells each side, 0 <= W <= 4096                              */
} teuk_orbit;

/* Make CUDA device `device` current for this library in the calling thread (cudaSetDevice inside the
 * library's own CUDA runtime instance).  Optional: without it teuk_create uses the device whose context
 * is current in the thread.  The Python binding calls it with torch's current device. */
int teuk_select_device(int32_t device);

/* FP64 issue-rate microbenchmark on the current device (no solver needed): the plain FP64 arithmetic of the
 * right-hand sides is what the iteration spends its instructions on, and its ceiling is the
 * co-limit of the HBM roofline.  kind 0 = DFMA reading two distinct registers, 1 = DFMA reading
 * three distinct registers, 2 = DADD, 3 = DMUL; *lane_ops_per_s = lane-operations per second over the whole
 * device with every SM saturated (one DFMA on one lane = 1).  Runs on the default stream and waits for it
 * (a few milliseconds).  bench.py reports the "alu" roofline of the step kernel from these figures. */
int teuk_measure_fp64(int32_t kind, double *lane_ops_per_s);

/* Create a solver for Kerr parameters (a, M), |a| < M, M > 0, and n_modes (1..64) azimuthal
 * modes m[k] evolved together as independent fields ("decoupled"; one launch per
 * iteration covers all modes).  dt > 0 is the time step (the caller is responsible for stability:
 * DESIGN.md reading A1).  Allocates all device state (two copies of the fields, coefficient
 * tables), builds the coefficient tables on the device, zeroes the fields.  Uses the CUDA device
 * that is current in the calling thread; every later call on the handle runs on that device whatever
 * device is current then, and restores the caller's current device.  *out is set to NULL on failure. */
int teuk_create(teuk_solver **out, double a, double M, const int32_t *m, int32_t n_modes,
                const teuk_grid *grid, double dt);

/* Set the solution vector u = {Phi_R, Phi_I, Pi_R, Pi_I} at t = 0 -- Phi is the field of Eq. (2)
 * (PAPER.md:84-88), Pi its "auxiliary momentum field" -- and reset the iteration counter, the
 * simulated time and every observer's recorded series.  Each array [n_modes][n_r][n_theta], theta fastest;
 * NULL = zeros for that component.  ptr_is_device: 0 host pointers (copied before the call returns), 1 device
 * pointers (the layout change is enqueued on the solver's stream; keep the arrays alive until it has run). */
int teuk_set_initial(teuk_solver *s, const double *phi_re, const double *phi_im,
                     const double *pi_re, const double *pi_im, int32_t ptr_is_device);

/* Install (copy to the device) the trajectory table; NULL = source-free.  Host pointers. */
int teuk_set_source(teuk_solver *s, const teuk_orbit *orbit);

/* Replace the single deposited term of the installed trajectory by a SUM of n_terms (0..12) rank-1 terms
 *     T(t,x,theta) = sum_t A_t(t) P^(a_t)(x - x_p; w_r) P^(b_t)(theta - theta_p; w_theta),
 * where P is the deposit profile selected by "source_kind" (the Gaussian g of teuk_orbit, or a discrete delta) and
 * P^(k), k = order 0, 1 or 2, its k-th derivative with respect to its argument: on the grid, sum_i P^(k)(x_i - x_p)
 * f(x_i) dx = (-1)^k f^(k)(x_p), the action of the k-th derivative of the delta function.  This is the mechanism
 * the physical s = -2 source needs -- T is "constructed from the energy-momentum tensor", complex
 * algebra on "a handful of grid points": a sum of delta, delta' and delta'' terms whose
 * coefficients the paper does not print and this library does not contain; they are the caller's A_t.
 * Gaussian: g' = -(y/s^2) g, g'' = (y^2/s^4 - 1/s^2) g, same window W.  Discrete deltas: the weights are
 * (-1)^k L_i^(k)(x_p)/h, L_i the Lagrange polynomials of the two-point / four-point stencil around the particle
 * (the two-point rule has no second derivative: its order-2 profile is zero).
 * order_r, order_theta: [n_terms]; amp_re, amp_im: [n_terms][n_modes][n_samples] on the samples of the installed
 * table (host pointers, copied before the call returns).  n_terms = 0 restores the single term A'_m of teuk_orbit,
 * and so does every teuk_set_source call.  TEUK_EINVAL without an installed trajectory, for an order outside 0..2,
 * or with "kernel" 1, "temporal_block" 2 or "coef_mode" 1 (those variants carry the single-term deposit only). */
int teuk_set_source_terms(teuk_solver *s, int32_t n_terms, const int32_t *order_r, const int32_t *order_theta,
                          const double *amp_re, const double *amp_im);

/* Enqueue n >= 0 iterations of the two-step Lax-Wendroff scheme ("Each iteration consists of two
 * steps": the half step Eq. (3), then the full step Eq. (4), with the boundary
 * conditions of PAPER.md:104 and the source of PAPER.md:114).  No host synchronisation, no full-grid host
 * transfer (per-step transfers cancel the GPU's gain); observers are tapped on the device after
 * every iteration (sample time t = n_done*dt).  TEUK_EINVAL if a source is installed and its table is too short. */
int teuk_step(teuk_solver *s, int64_t n);

/* Allocation-free variant of teuk_set_initial(device) + teuk_step(n) + teuk_get_state(device) for grids whose state
 * fits on chip (the resident kernel, "kernel" 2: n_theta <= 128, about n_modes*n_r*n_theta <= 5e5 points), for
 * callers that cannot call cudaMalloc -- code under CUDA graph capture, tight serving loops, harnesses that forbid
 * it.  The same iteration (Eq. 3-4) by the same kernel: fields are bit-identical to teuk_step's.
 * The kernel's only scratch memory, the block-to-block exchange buffer that teuk_step cudaMalloc's on first use,
 * is here a file-scope static device array of 5 MiB (5 242 880 bytes; every GPU that loads the library holds it
 * until the process exits); a solver that needs more gets TEUK_EINVAL with a message naming both sizes.
 *   in_dev[4]:  DEVICE arrays Phi_R, Phi_I, Pi_R, Pi_I of time level n0, layout of teuk_set_initial; NULL = zeros.
 *   n0:         iteration index of that level (a source uses trajectory samples 2*n0, 2*n0 + 1, ...); >= 0.
 *   n:          iterations to run, 1 <= n <= 2^30.
 *   out_dev[4]: DEVICE arrays receiving level n0 + n (may alias in_dev); NULL = skip that component.
 * Everything is enqueued on the solver's stream and nothing is waited for: keep the arrays alive until it has run.
 * The call makes no cudaMalloc / cudaFree / cudaMallocHost / cudaFreeHost and calls no library that allocates.
 * Side effects: the solver's own fields become the result and its iteration counter n0 + n, as if teuk_step had
 * produced them (a later teuk_step / teuk_get_state continues from there).  TEUK_EINVAL with armed observers
 * (their ring drains allocate pinned memory), with "kernel" 1, "temporal_block" 2 or "coef_mode" 1, if the state
 * does not fit on chip, or if the trajectory table is too short.
 * The static array is shared by every solver and every call on a GPU and keeps the last call's contents: each
 * call clears the part it uses before its kernel starts, so consecutive calls on one stream are safe, but two
 * calls that OVERLAP on the GPU (different streams or solvers at the same time) race on it. */
int teuk_step_noalloc(teuk_solver *s, const double *const in_dev[4], int64_t n0, int64_t n, double *const out_dev[4]);

/* Observer at r* = rs_obs (x_0 <= rs_obs < x_{n_r-1}): w(t_n) = sum_j weights[j] *
 * [(1-f) Phi^n_{i0,j} + f Phi^n_{i0+1,j}] (linear interpolation in x).
 * The FIRST call with a new rs_obs arms the observer (weights [n_theta] host array, NULL = all
 * ones; at most 8 observers; must precede the teuk_step calls it should record) and writes
 * nothing.  LATER calls with the same rs_obs (weights ignored) wait for the stream and return the
 * samples recorded since the previous call: t_out[k], and w_re/w_im [k][n_modes], k < *n_written
 * <= capacity.  Samples beyond `capacity` stay queued for the next call.  Returns
 * TEUK_ENONFINITE (after filling the outputs) if any recorded sample was NaN/Inf. */
int teuk_extract(teuk_solver *s, double rs_obs, const double *weights, double *t_out,
                 double *w_re, double *w_im, int64_t capacity, int64_t *n_written);

/* Copy the current solution vector u^n = {Phi_R, Phi_I, Pi_R, Pi_I} out, same layout as
 * teuk_set_initial (parity checks, checkpoints; the paper's temporal parallelisation restarts segments from zero
 * data instead).  NULL = skip that component.
 * Host pointers: waits for the stream.  Device pointers: enqueued on the stream. */
int teuk_get_state(teuk_solver *s, double *phi_re, double *phi_im, double *pi_re, double *pi_im,
                   int32_t ptr_is_device);

/* Options (set before stepping):
 *   "outer_bc"      0 = outgoing (Pi = 0, Phi upwind; default), 1 = Dirichlet as PAPER.md:104
 *   "source_kind"   deposit profile of the particle source: 0 = the Gaussian g of teuk_orbit
 *                   (default); 1 = two-point "discrete delta" = finite-difference derivative of the discrete
 *                   step function: weights (1-gamma)/h, gamma/h on the two grid points around the particle;
 *                   2 = four-point discrete delta (cubic Lagrange weights / h).  For 1 and 2 the widths are the
 *                   grid spacings (dx, dtheta) of the stage's own grid and sigma_r, sigma_theta, half_window
 *                   of teuk_orbit are ignored.
 *   "stream"        a cudaStream_t cast to int64 (0 = back to the solver's own stream)
 *   "coef_mode"     0 = coefficients recomputed on the fly from 1D tables (default),
 *                   1 = coefficients streamed from precomputed 2D FP64 planes (n_theta <= 128 only)
 *   "slab_rows"     rows of r* marched by one warp (0 = automatic, see "autotune"); the interior rows are dealt
 *                   evenly to ceil((n_r - 2) / slab_rows) slabs
 *   "autotune"      1 (default) = the number of slabs of the marching kernels is MEASURED: a few dozen trial launches
 *                   of the real kernel into the idle copy of the state (fields, counters and series untouched),
 *                   timed inside teuk_create and again inside any teuk_set_option call that changes the launch
 *                   shape ("kernel", "coef_mode", "temporal_block", "slab_rows", "autotune") -- calls that wait for
 *                   the device anyway; teuk_step never does.  0 = use the two-wave heuristic
 *   "temporal_block" 1 = one iteration per kernel launch (default), 2 = two iterations per HBM round trip
 *                   (warp pairs; level n+1 stays in shared memory; same results bit for bit; needs kernel 0,
 *                   coef_mode 0, n_theta <= 128)
 *   "graph"         1 = replay the iteration through a CUDA graph (default), 0 = plain launches
 *   "kernel"        -1 = automatic (default): kernel 2 whenever it applies, else kernel 0;
 *                   0 = register-resident marching kernel (one launch per iteration, state streamed from HBM/L2);
 *                   1 = shared-memory-resident marching kernel (n_theta <= 256);
 *                   2 = resident kernel: ONE cooperative launch per teuk_step call, the whole state stays in
 *                   shared memory between iterations, neighbouring blocks exchange one row per iteration through
 *                   L2.  Needs n_theta <= 128, coef_mode 0, temporal_block 1 and a state small enough for the
 *                   shared memory of one block per SM (about n_modes*n_r*n_theta <= 5e5 points), else EINVAL.
 *                   All kernels do the same arithmetic per point: fields are bitwise identical (waveforms too,
 *                   except kernel 1, which sums over theta in another order).  An explicit "slab_rows" makes the
 *                   automatic choice stay with kernel 0.
 *   "wide"          how kernel 0 maps rows wider than 64 columns onto warps: 0 = one warp per row (V = 4 columns per
 *                   lane, n_theta <= 128) or per theta segment with recomputed halo columns (n_theta > 128);
 *                   1 = a GROUP of ceil(n_theta / 64) warps per row, V = 2 columns per lane, the boundary columns of
 *                   the theta stencil exchanged through shared memory (needs an even n_theta between 66 and 320,
 *                   coef_mode 0, temporal_block 1; otherwise the setting is ignored);
 *                   -1 (default) = automatic: 1 for rows wider than 128 columns when it applies (measured faster than
 *                   theta segments), 0 otherwise (for n_theta <= 128 one warp per row is faster).  Same results
 *                   bit for bit.
 *   "pdl"           1 (default) = inside a CUDA-graph batch, iteration k + 1 of kernel 0 is launched as a programmatic
 *                   dependent of iteration k (its prologue overlaps k's tail); 0 = fully serialised launches
 *   "resident_cache" 1 (default) = kernel 2 also keeps the time-independent coefficients b, b^2 and Re beta' of its
 *                   rows in shared memory when they fit (3 doubles per point and location), 0 = it rebuilds them
 *                   in every stage like kernel 0.  Same results bit for bit. */
int teuk_set_option(teuk_solver *s, const char *key, int64_t value);

/* Read-only counters: "steps" (iterations done), "launches" (kernels launched so far),
 * "n_pts" (n_modes*n_r*n_theta), "state_bytes" (one copy of the fields), "slab_rows" (longest slab in use), "slabs" (slabs per mode),
 * "wide" (1 if the next teuk_step would run the group-of-warps-per-row kernel),
 * "kernel" (the kernel the next teuk_step would run), "resident_rows" / "resident_blocks" (rows of r* per
 * block and blocks of kernel 2, 0 if it is not in use). */
int teuk_get_stat(const teuk_solver *s, const char *key, int64_t *value);

/* Wait for all work enqueued on the solver's stream. */
int teuk_sync(teuk_solver *s);

void teuk_destroy(teuk_solver *s); /* NULL is allowed */

/* Static text for the last error on this solver (or the last teuk_create failure if s == NULL). */
const char *teuk_last_error(const teuk_solver *s);

#ifdef __cplusplus
}
#endif
#endif /* TEUK_H_ */
