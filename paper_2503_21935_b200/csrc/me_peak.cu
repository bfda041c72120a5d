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

// Tensor-pipe counterparts (the colour contraction of the lane-group pipeline): register-resident chains of
// mma.sync m8n8k4 f64 (SASS DMMA) and m16n8k8 tf32 (SASS HMMA.1688.F32.TF32), 8 independent accumulators per warp.
template <int KIND>
__global__ void __launch_bounds__(256) mma_chain(double* out, int iters, double seed) {
  constexpr int ILP = 8;
  double d0[ILP], d1[ILP];
  float f[ILP][4];
#pragma unroll
  for (int i = 0; i < ILP; i++) { d0[i] = d1[i] = seed * (threadIdx.x + i); f[i][0] = f[i][1] = f[i][2] = f[i][3] = (float)d0[i]; }
  const double a = seed, b = 0.5 * seed;
  const unsigned ua = __float_as_uint((float)a), ub = __float_as_uint((float)b);
  for (int it = 0; it < iters; it++) {
#pragma unroll
    for (int r = 0; r < 8; r++) {
#pragma unroll
      for (int i = 0; i < ILP; i++) {
        if (KIND == 0)
          asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};" : "+d"(d0[i]), "+d"(d1[i]) : "d"(a), "d"(b));
        else
          asm volatile("mma.sync.aligned.m16n8k8.row.col.f32.tf32.tf32.f32 {%0,%1,%2,%3}, {%4,%5,%6,%7}, {%8,%9}, {%0,%1,%2,%3};"
                       : "+f"(f[i][0]), "+f"(f[i][1]), "+f"(f[i][2]), "+f"(f[i][3]) : "r"(ua), "r"(ua), "r"(ub), "r"(ub), "r"(ua), "r"(ub));
      }
    }
  }
  double s = 0.0;
#pragma unroll
  for (int i = 0; i < ILP; i++) s += d0[i] + d1[i] + f[i][0] + f[i][1] + f[i][2] + f[i][3];
  if (s == 123.456) out[0] = s;
}

template <int KIND>
int run_mma(double* tflops) {
  int dev = 0, sms = 0;
  cudaError_t e = cudaGetDevice(&dev);
  if (e == cudaSuccess) e = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
  if (e != cudaSuccess) return ME_ERR_CUDA;
  double* d = nullptr;
  if (cudaMalloc(&d, sizeof(double)) != cudaSuccess) return ME_ERR_NOMEM;
  const int blocks = sms * 8, threads = 256, iters = (KIND == 0) ? 512 : 4096;
  cudaEvent_t t0, t1;
  cudaEventCreate(&t0);
  cudaEventCreate(&t1);
  mma_chain<KIND><<<blocks, threads>>>(d, iters / 8, 1e-3);
  double best = 1e30;
  for (int rep = 0; rep < 5; rep++) {
    cudaEventRecord(t0);
    mma_chain<KIND><<<blocks, threads>>>(d, iters, 1e-3);
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
  const double per_mma = (KIND == 0) ? 2.0 * 8 * 8 * 4 : 2.0 * 16 * 8 * 8;   // FLOPs of one warp-wide MMA
  *tflops = per_mma * double(blocks) * (threads / 32) * double(iters) * 8 * 8 / (best * 1e-3) * 1e-12;
  return ME_OK;
}

}  // namespace

extern "C" int me_mma_peak(int kind, int device, double* tflops) {
  if (!tflops || (kind != 0 && kind != 1)) return ME_ERR_ARG;
  int prev = -1;
  if (cudaGetDevice(&prev) != cudaSuccess || cudaSetDevice(device) != cudaSuccess) return ME_ERR_CUDA;
  const int rc = kind == 0 ? run_mma<0>(tflops) : run_mma<1>(tflops);
  if (prev != device) cudaSetDevice(prev);
  return rc;
}

extern "C" int me_fma_peak(int precision, int device, double* tflops) {
  if (!tflops || (precision != ME_FP64 && precision != ME_FP32)) return ME_ERR_ARG;
  int prev = -1;
  if (cudaGetDevice(&prev) != cudaSuccess || cudaSetDevice(device) != cudaSuccess) return ME_ERR_CUDA;
  const int rc = precision == ME_FP64 ? run<double>(tflops, nullptr) : run<float>(tflops, nullptr);
  if (prev != device) cudaSetDevice(prev);  // leave the caller's current device as it was
  return rc;
}
