// microbench.cu -- FFMA / DFMA peak of the CUDA cores, the roofline denominator of the pair and
// convolution kernels (MEASURED_PEAKS.json has only HBM and tensor numbers).
#include <cuda_runtime.h>

#include "../../include/msm.h"

namespace {

template <typename T>
__global__ void __launch_bounds__(256) k_fma_chain(T* out, int iters, T a, T b) {
  T x[16];
#pragma unroll
  for (int i = 0; i < 16; ++i) x[i] = (T)(threadIdx.x + i) * (T)1e-3;
  for (int it = 0; it < iters; ++it) {
#pragma unroll
    for (int r = 0; r < 8; ++r)
#pragma unroll
      for (int i = 0; i < 16; ++i) x[i] = fma(x[i], a, b);
  }
  T s = 0;
#pragma unroll
  for (int i = 0; i < 16; ++i) s += x[i];
  out[blockIdx.x * blockDim.x + threadIdx.x] = s;
}

// packed pairs: fma.rn.f32x2 (SASS FFMA2) does two fp32 multiply-adds per instruction and lane
__global__ void __launch_bounds__(256) k_fma2_chain(float* out, int iters, float a, float b) {
  unsigned long long x[8];
#pragma unroll
  for (int i = 0; i < 8; ++i) {
    const float2 v = make_float2((threadIdx.x + i) * 1e-3f, (threadIdx.x + i) * 2e-3f);
    x[i] = *reinterpret_cast<const unsigned long long*>(&v);
  }
  const float2 av = make_float2(a, a), bv = make_float2(b, b);
  const unsigned long long aa = *reinterpret_cast<const unsigned long long*>(&av);
  const unsigned long long bb = *reinterpret_cast<const unsigned long long*>(&bv);
  for (int it = 0; it < iters; ++it) {
#pragma unroll
    for (int r = 0; r < 8; ++r)
#pragma unroll
      for (int i = 0; i < 8; ++i) asm volatile("fma.rn.f32x2 %0, %0, %1, %2;" : "+l"(x[i]) : "l"(aa), "l"(bb));
  }
  float s = 0;
#pragma unroll
  for (int i = 0; i < 8; ++i) {
    const float2 v = *reinterpret_cast<const float2*>(&x[i]);
    s += v.x + v.y;
  }
  out[blockIdx.x * blockDim.x + threadIdx.x] = s;
}

template <typename T> msm_status_t measure(double* tflops, bool packed = false) {
  int sms = 0, dev = 0;
  cudaGetDevice(&dev);
  cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
  const int blocks = sms * 8, threads = 256, iters = 4096;
  T* out = nullptr;
  if (cudaMalloc(&out, (size_t)blocks * threads * sizeof(T)) != cudaSuccess) return MSM_ERR_NOMEM;
  cudaEvent_t e0, e1;
  cudaEventCreate(&e0); cudaEventCreate(&e1);
  double best = 0.0;
  for (int rep = 0; rep < 5; ++rep) {
    cudaEventRecord(e0);
    if (packed) k_fma2_chain<<<blocks, threads>>>((float*)out, iters, 0.999f, 1e-4f);
    else k_fma_chain<T><<<blocks, threads>>>(out, iters, (T)0.999, (T)1e-4);
    cudaEventRecord(e1);
    if (cudaEventSynchronize(e1) != cudaSuccess) { cudaFree(out); return MSM_ERR_CUDA; }
    float ms = 0;
    cudaEventElapsedTime(&ms, e0, e1);
    const double flops = 2.0 * 16 * 8 * (double)iters * blocks * threads;
    if (rep > 0) best = best > flops / (ms * 1e-3) * 1e-12 ? best : flops / (ms * 1e-3) * 1e-12;
  }
  cudaEventDestroy(e0); cudaEventDestroy(e1);
  cudaFree(out);
  *tflops = best;
  return cudaGetLastError() == cudaSuccess ? MSM_OK : MSM_ERR_CUDA;
}

}  // namespace

extern "C" msm_status_t msm_measure_fma_peak(int device, int kind, double* tflops) {
  if (!tflops || kind < 0 || kind > 2) return MSM_ERR_INVALID_ARG;
  int prev = -1;
  if (cudaGetDevice(&prev) != cudaSuccess) prev = -1;
  if (cudaSetDevice(device) != cudaSuccess) return MSM_ERR_CUDA;
  const msm_status_t s = kind == 2 ? measure<float>(tflops, true) : (kind == 0 ? measure<float>(tflops) : measure<double>(tflops));
  if (prev >= 0) cudaSetDevice(prev);
  return s;
}
