// device_common.cuh -- shared device-side types and helpers of libmsm_b200 (sm_100a).
#pragma once
#include <cuda_runtime.h>

#include <cstdint>

namespace msm {

template <typename T> struct Vec4;
template <> struct Vec4<float> { using type = float4; };
template <> struct Vec4<double> { using type = double4; };

template <typename T> __device__ __forceinline__ typename Vec4<T>::type make_vec4(T x, T y, T z, T w);
template <> __device__ __forceinline__ float4 make_vec4<float>(float x, float y, float z, float w) {
  return make_float4(x, y, z, w);
}
template <> __device__ __forceinline__ double4 make_vec4<double>(double x, double y, double z, double w) {
  return make_double4(x, y, z, w);
}

// read-only 4-vector loads (fp64: two 16-byte loads)
__device__ __forceinline__ float4 ldg4(const float4* p) { return __ldg(p); }
__device__ __forceinline__ double4 ldg4(const double4* p) {
  const double2 a = __ldg(reinterpret_cast<const double2*>(p));
  const double2 b = __ldg(reinterpret_cast<const double2*>(p) + 1);
  return make_double4(a.x, a.y, b.x, b.y);
}

template <typename T> __device__ __forceinline__ T rsqrt_t(T x);
template <> __device__ __forceinline__ float rsqrt_t<float>(float x) { return rsqrtf(x); }
template <> __device__ __forceinline__ double rsqrt_t<double>(double x) { return 1.0 / sqrt(x); }

// 16-byte asynchronous copy global -> shared (LDGSTS, bypasses L1)
__device__ __forceinline__ void cp_async16(void* smem, const void* gmem, int n) {   // n = 16, or 0: zero fill
  const unsigned s = (unsigned)__cvta_generic_to_shared(smem);
  asm volatile("cp.async.cg.shared.global [%0], [%1], 16, %2;" ::"r"(s), "l"(gmem), "r"(n) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
template <int N> __device__ __forceinline__ void cp_async_wait() { asm volatile("cp.async.wait_group %0;" ::"n"(N) : "memory"); }

__device__ __forceinline__ int imod(int i, int m) {
  int r = i % m;
  return r < 0 ? r + m : r;
}

// B-spline piece polynomials, passed to kernels by value (lives in the constant bank)
template <typename T, int P> struct SplineTab {
  T c[P][P];   // weight of node offset j (row j + P/2 - 1): sum_k c[.][k] t^k
  T d[P][P];   // derivative w.r.t. t (degree P-2; last column 0)
};

template <typename T, int P>
__device__ __forceinline__ void spline_weights(const SplineTab<T, P>& tab, T t, T (&w)[P]) {
#pragma unroll
  for (int j = 0; j < P; ++j) {
    T acc = tab.c[j][P - 1];
#pragma unroll
    for (int k = P - 2; k >= 0; --k) acc = fma(acc, t, tab.c[j][k]);
    w[j] = acc;
  }
}

template <typename T, int P>
__device__ __forceinline__ void spline_dweights(const SplineTab<T, P>& tab, T t, T (&dw)[P]) {
#pragma unroll
  for (int j = 0; j < P; ++j) {
    T acc = tab.d[j][P - 2];
#pragma unroll
    for (int k = P - 3; k >= 0; --k) acc = fma(acc, t, tab.d[j][k]);
    dw[j] = acc;
  }
}

// one spline weight for a run-time node offset (row jrow), used by the gather anterpolation
template <typename T, int P>
__device__ __forceinline__ T spline_weight_row(const SplineTab<T, P>& tab, int jrow, T t) {
  T acc = tab.c[jrow][P - 1];
#pragma unroll
  for (int k = P - 2; k >= 0; --k) acc = fma(acc, t, tab.c[jrow][k]);
  return acc;
}

// geometry of the particle <-> cell maps, by value
struct BinGeom {
  double box[3];
  int periodic[3];
  // pair cells; along x every cell is cut into 2^sxs sub-bins (the sort key), so that a cell row
  // is ordered by x finely enough for the pair kernel's windows
  int nc[3];
  double cell_edge[3];
  int sxs;
  // level-1 grid cells (one per grid interval)
  int ng[3];        // number of grid cells per axis
  double h1[3];
};

// fixed-order block reduction in double: result valid in thread 0
template <int BLOCK>
__device__ __forceinline__ double block_reduce_sum(double v, double* smem /* BLOCK/32 doubles */) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_down_sync(0xffffffffu, v, o);
  const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
  __syncthreads();
  if (lane == 0) smem[wid] = v;
  __syncthreads();
  double r = 0.0;
  if (threadIdx.x == 0)
    for (int i = 0; i < BLOCK / 32; ++i) r += smem[i];
  return r;
}

}  // namespace msm
