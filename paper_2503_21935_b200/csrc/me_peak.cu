// me_peak.cu -- register-resident FMA-chain microbenchmark: the measured FP64 / FP32 FMA peak that the
// roofline fractions of bench.py are quoted against (MEASURED_PEAKS.json has no FMA figure).
#include <cuda_runtime.h>

#include "../../include/me_b200.h"

namespace {

template <typename T, int ILP>
__global__ void __launch_bounds__(256) fma_chain(T* out, int iters, T a, T b) {
  T x[ILP];
#pragma unroll
  for (int i = 0; i < ILP; i++) x[i] = T(threadIdx.x + i) * T(1e-3);
  for (int it = 0; it < iters; it++) {
#pragma unroll
    for (int r = 0; r < 16; r++) {
#pragma unroll
      for (int i = 0; i < ILP; i++) x[i] = x[i] * a + b;
    }
  }
  T s = T(0);
#pragma unroll
  for (int i = 0; i < ILP; i++) s += x[i];
  if (s == T(123.456)) out[0] = s;  // never true: keeps the chain alive
}

template <typename T>
int run(double* tflops, double* ms_out) {
  int dev = 0, sms = 0;
  cudaError_t e = cudaGetDevice(&dev);
  if (e == cudaSuccess) e = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
  if (e != cudaSuccess) return ME_ERR_CUDA;
  T* d = nullptr;
  if (cudaMalloc(&d, sizeof(T)) != cudaSuccess) return ME_ERR_NOMEM;
  constexpr int ILP = 8;
  const int blocks = sms * 8, threads = 256, iters = 4096;
  cudaEvent_t t0, t1;
  cudaEventCreate(&t0);
  cudaEventCreate(&t1);
  fma_chain<T, ILP><<<blocks, threads>>>(d, iters / 8, T(0.999), T(1e-4));  // warm-up
  double best = 1e30;
  for (int rep = 0; rep < 5; rep++) {
    cudaEventRecord(t0);
    fma_chain<T, ILP><<<blocks, threads>>>(d, iters, T(0.999), T(1e-4));
    cudaEventRecord(t1);
    if ((e = cudaEventSynchronize(t1)) != cudaSuccess) break;
    float ms = 0;
    cudaEventElapsedTime(&ms, t0, t1);
    if (ms < best) best = ms;
  }
  cudaEventDestroy(t0);
  cudaEventDestroy(t1);
  cudaFree(d);
  if (e != cudaSuccess) return ME_ERR_CUDA;
  const double flops = 2.0 * double(blocks) * threads * double(iters) * 16 * ILP;
  *tflops = flops / (best * 1e-3) * 1e-12;
  if (ms_out) *ms_out = best;
  return ME_OK;
}

}  // namespace

extern "C" int me_fma_peak(int precision, int device, double* tflops) {
  if (!tflops || (precision != ME_FP64 && precision != ME_FP32)) return ME_ERR_ARG;
  int prev = -1;
  if (cudaGetDevice(&prev) != cudaSuccess || cudaSetDevice(device) != cudaSuccess) return ME_ERR_CUDA;
  const int rc = precision == ME_FP64 ? run<double>(tflops, nullptr) : run<float>(tflops, nullptr);
  if (prev != device) cudaSetDevice(prev);  // leave the caller's current device as it was
  return rc;
}
