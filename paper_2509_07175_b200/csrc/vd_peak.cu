// vd_peak.cu -- the denominator of the "alu" roofline ("no FP64 figure is in MEASURED_PEAKS.json --
// measure it"): a chain of dependent fused multiply-adds per thread, eight independent chains, enough warps to
// keep the FP64 pipe of every SM busy.  Not part of the hot path; bench.py calls it once, outside the timed region.
#include "vd_internal.h"

namespace vd {

constexpr int kPeakChains = 8;

__global__ void __launch_bounds__(256) k_fp64_fma_chain(double* __restrict__ out, int iters, double a, double b) {
  double x[kPeakChains];
#pragma unroll
  for (int k = 0; k < kPeakChains; ++k) x[k] = (double)(threadIdx.x + k) * 1e-3;
  for (int it = 0; it < iters; ++it) {
#pragma unroll
    for (int k = 0; k < kPeakChains; ++k) x[k] = fma(x[k], a, b);
  }
  double s = 0.0;
#pragma unroll
  for (int k = 0; k < kPeakChains; ++k) s += x[k];
  if (s == 123.456) out[0] = s;   // never true for the constants used; keeps the chains alive
}

}  // namespace vd

using namespace vd;

extern "C" vd_status vd_dfma_peak(void* cuda_stream, double* tflops_out, double* ms_out) {
  if (!tflops_out) return VD_E_ARG;
  int ndev = 0;
  if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev < 1) { cudaGetLastError(); return VD_E_CUDA; }
  cudaStream_t st = (cudaStream_t)cuda_stream;
  int dev = 0, sms = 0;
  cudaGetDevice(&dev);
  cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
  double* out = nullptr;
  if (cudaMalloc(&out, sizeof(double)) != cudaSuccess) { cudaGetLastError(); return VD_E_NOMEM; }
  cudaEvent_t e0, e1;
  cudaEventCreate(&e0);
  cudaEventCreate(&e1);
  const int blocks = sms * 8, threads = 256, iters = 1 << 15;
  float best = 1e30f;
  for (int rep = 0; rep < 4; ++rep) {   // the first repetition warms up
    cudaEventRecord(e0, st);
    VD_LAUNCH(k_fp64_fma_chain, blocks, threads, 0, st)(out, iters, 0.999999, 1e-9);
    cudaEventRecord(e1, st);
    if (cudaEventSynchronize(e1) != cudaSuccess) break;
    float ms = 0.f;
    cudaEventElapsedTime(&ms, e0, e1);
    if (rep > 0 && ms < best) best = ms;
  }
  const cudaError_t err = cudaGetLastError();
  cudaEventDestroy(e0);
  cudaEventDestroy(e1);
  cudaFree(out);
  if (err != cudaSuccess || best > 1e29f) return VD_E_CUDA;
  const double flop = 2.0 * (double)blocks * threads * kPeakChains * (double)iters;
  *tflops_out = flop / (best * 1e-3) / 1e12;
  if (ms_out) *ms_out = best;
  return VD_OK;
}
