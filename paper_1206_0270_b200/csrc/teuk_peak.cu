// teuk_peak.cu -- FP64 issue-rate microbenchmark behind teuk_measure_fp64 (include/teuk.h).
//
// The Lax-Wendroff stage ("computing the right-hand-sides ... take most of the application's
// overall runtime") is plain FP64 arithmetic on the CUDA cores; its ceiling on this chip is not in
// MEASURED_PEAKS.json, so the library measures it: blocks of 256 threads, several per SM, every thread running ILP
// independent dependent chains of one instruction kind for `iters` rounds.  Kinds:
//   0  DFMA, accumulator + ONE more distinct register (x = fma(x, c, x) style: two register-file operands)
//   1  DFMA with THREE distinct register operands          (x = fma(c_k, y_k, x))
//   2  DADD  (x = x + c)            3  DMUL  (x = x * c)
// Result: lane-operations per second over the whole device (one DFMA on one lane = 1).  bench.py turns the
// figures into the "alu" roofline of the step kernel from its SASS instruction mix.
#include <cuda_runtime.h>
#include <stdint.h>

namespace {

constexpr int PEAK_ILP = 8;

template <int KIND>
__global__ void __launch_bounds__(256) teuk_fp64_peak_kernel(double* out, int iters, double seed) {
  double x[PEAK_ILP], y[PEAK_ILP], c[PEAK_ILP];
#pragma unroll
  for (int k = 0; k < PEAK_ILP; ++k) {
    x[k] = seed + 1e-3 * (threadIdx.x + k);
    y[k] = 1.0 + 1e-9 * (threadIdx.x * 3 + k);      // distinct registers per chain
    c[k] = 1e-9 * (k + 1) + seed * 1e-12;
  }
  for (int it = 0; it < iters; ++it) {
#pragma unroll
    for (int r = 0; r < 8; ++r) {
#pragma unroll
      for (int k = 0; k < PEAK_ILP; ++k) {
        if (KIND == 0) x[k] = fma(x[k], c[0], x[k]);            // registers: x_k, c_0 (shared by all chains)
        else if (KIND == 1) x[k] = fma(c[k], y[k], x[k]);       // registers: c_k, y_k, x_k
        else if (KIND == 2) x[k] = x[k] + c[k];
        else x[k] = x[k] * y[k];
      }
    }
  }
  double s = 0.0;
#pragma unroll
  for (int k = 0; k < PEAK_ILP; ++k) s += x[k];
  if (s == 123.456) out[blockIdx.x * blockDim.x + threadIdx.x] = s;   // keeps the chains alive, never true in practice
}

template <int KIND>
cudaError_t run_kind(double* d_out, int blocks, int iters, cudaStream_t st, float* ms) {
  cudaEvent_t e0, e1;
  cudaError_t e = cudaEventCreate(&e0);
  if (e != cudaSuccess) return e;
  e = cudaEventCreate(&e1);
  if (e != cudaSuccess) { cudaEventDestroy(e0); return e; }
  teuk_fp64_peak_kernel<KIND><<<blocks, 256, 0, st>>>(d_out, iters / 8, 1.0);   // warm-up
  float best = 1e30f;
  for (int rep = 0; rep < 3 && e == cudaSuccess; ++rep) {
    cudaEventRecord(e0, st);
    teuk_fp64_peak_kernel<KIND><<<blocks, 256, 0, st>>>(d_out, iters, 1.0);
    cudaEventRecord(e1, st);
    e = cudaEventSynchronize(e1);
    float t = 0.f;
    if (e == cudaSuccess) e = cudaEventElapsedTime(&t, e0, e1);
    if (t < best) best = t;
  }
  cudaEventDestroy(e0);
  cudaEventDestroy(e1);
  if (e == cudaSuccess) e = cudaGetLastError();
  *ms = best;
  return e;
}

}  // namespace

// lane-operations per second of instruction kind `kind` over the whole current device; < 0 on error.
double teuk_fp64_rate(int kind, cudaError_t* err) {
  int dev = 0, sms = 0;
  *err = cudaGetDevice(&dev);
  if (*err == cudaSuccess) *err = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
  if (*err != cudaSuccess) return -1.0;
  const int blocks = sms * 4;          // 32 warps per SM x ILP 8: far beyond what the pipe needs to saturate
  const int iters = 4096;
  double* d_out = nullptr;
  *err = cudaMalloc((void**)&d_out, (size_t)blocks * 256 * sizeof(double));
  if (*err != cudaSuccess) return -1.0;
  float ms = 0.f;
  switch (kind) {
    case 0: *err = run_kind<0>(d_out, blocks, iters, 0, &ms); break;
    case 1: *err = run_kind<1>(d_out, blocks, iters, 0, &ms); break;
    case 2: *err = run_kind<2>(d_out, blocks, iters, 0, &ms); break;
    default: *err = run_kind<3>(d_out, blocks, iters, 0, &ms); break;
  }
  cudaFree(d_out);
  if (*err != cudaSuccess) return -1.0;
  const double ops = (double)blocks * 256.0 * PEAK_ILP * 8.0 * iters;
  return ops / (ms * 1e-3);
}
