// peak.cu -- measured FMA peak of the device's plain fp64 / fp32 pipes, the denominator of the "alu" rooflines
// (MEASURED_PEAKS.json holds no FP64/FP32 figure, the build measures one).
// Every thread runs CHAINS independent dependent-FMA chains; 2 flop per FMA; the grid fills every SM to its thread limit.
#include <cuda_runtime.h>

#include "../../include/lbm.h"

namespace {

constexpr int CHAINS = 8;
constexpr int INNER = 4096;

template <typename T>
__global__ void __launch_bounds__(256) fma_peak_kernel(T* out, T a, T b) {
  T x[CHAINS];
#pragma unroll
  for (int k = 0; k < CHAINS; ++k) x[k] = T(threadIdx.x + k) * T(1e-3);
  for (int it = 0; it < INNER; ++it) {
#pragma unroll
    for (int k = 0; k < CHAINS; ++k) x[k] = fma(x[k], a, b);
  }
  T s = T(0);
#pragma unroll
  for (int k = 0; k < CHAINS; ++k) s += x[k];
  if (s == T(-1)) out[0] = s;     // never true for these operands: keeps the chains alive
}

template <typename T>
int measure(double seconds, double* tflops, double* sm_mhz_hint) {
  int dev = 0, sms = 0, tpsm = 0;
  if (cudaGetDevice(&dev) != cudaSuccess) return LBM_ECUDA;
  cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
  cudaDeviceGetAttribute(&tpsm, cudaDevAttrMaxThreadsPerMultiProcessor, dev);
  const int block = 256, grid = sms * (tpsm / block) * 4;
  T* d = nullptr;
  if (cudaMalloc(&d, sizeof(T)) != cudaSuccess) return LBM_ECUDA;
  cudaEvent_t e0, e1;
  cudaEventCreate(&e0);
  cudaEventCreate(&e1);
  fma_peak_kernel<T><<<grid, block>>>(d, T(0.999), T(1e-4));   // warm-up
  cudaDeviceSynchronize();
  double best = 0.0, total_ms = 0.0;
  const double flop = 2.0 * CHAINS * INNER * (double)grid * block;
  while (total_ms < seconds * 1e3) {
    cudaEventRecord(e0);
    fma_peak_kernel<T><<<grid, block>>>(d, T(0.999), T(1e-4));
    cudaEventRecord(e1);
    if (cudaEventSynchronize(e1) != cudaSuccess) { cudaFree(d); return LBM_ECUDA; }
    float ms = 0.f;
    cudaEventElapsedTime(&ms, e0, e1);
    total_ms += ms;
    const double tf = flop / (ms * 1e-3) / 1e12;
    if (tf > best) best = tf;
  }
  *tflops = best;
  if (sm_mhz_hint) *sm_mhz_hint = best * 1e12 / (2.0 * sms) / 1e6;   // FMA lanes per SM x MHz
  cudaEventDestroy(e0);
  cudaEventDestroy(e1);
  cudaFree(d);
  return LBM_OK;
}

}  // namespace

extern "C" int lbm_measure_fma_peak(int precision, double seconds, double* tflops, double* lanes_mhz_per_sm) {
  if (!tflops || !(seconds >= 0.0)) return LBM_EINVAL;
  int ndev = 0;
  if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev < 1) return LBM_ECUDA;
  if (precision == 64) return measure<double>(seconds, tflops, lanes_mhz_per_sm);
  if (precision == 32) return measure<float>(seconds, tflops, lanes_mhz_per_sm);
  return LBM_EINVAL;
}
