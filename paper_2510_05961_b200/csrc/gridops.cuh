// gridops.cuh -- S4 restriction (Eq. 19 line 1, separable, one axis at a time; the
// prolongation is in gridops_fused.cuh), and the omega' pre-filter that writes the haloed (padded)
// copy of a level's grid charge which the stencil convolution reads (Eq. 20's omega' factors moved
// from the stencil to the grid charge: K * q = s * (omega' (x) omega' (x) omega' * q)).
//
// One thread per output element; x is the fastest index in every array, so each warp reads and
// writes contiguous runs (the grids at config sizes are L2-resident).
#pragma once
#include "device_common.cuh"

namespace msm {

constexpr int kMaxAxisTaps = 2 * 32 + 1;

template <typename T> struct AxisTaps {
  int n;                  // number of taps, offsets -(n/2) .. n/2
  T c[kMaxAxisTaps];
};

struct AxisDims {
  int in[3], out[3];      // array dims (x, y, z)
  int axis;
  int periodic;
};

__device__ __forceinline__ size_t lin(const int d[3], int x, int y, int z) {
  return ((size_t)z * d[1] + y) * d[0] + x;
}

// Launch shape of the separable kernels: one thread per output element, consecutive threads along
// x (coalesced across rows); arrays hold fewer than 2^31 elements, so the index maths is 32-bit.
constexpr int kAxisThreads = 256;
inline unsigned axis_grid(const AxisDims& d) {
  const size_t total = (size_t)d.out[0] * d.out[1] * d.out[2];
  return (unsigned)((total + kAxisThreads - 1) / kAxisThreads);
}
inline unsigned axis_block() { return kAxisThreads; }

// coordinates of this thread's output element, its linear index, and the working-axis stride
struct AxisPos {
  int c[3];
  bool valid;
  size_t t;        // linear index in the output array
  size_t base;     // offset of the input line's element 0 (working-axis coordinate 0)
  size_t stride;   // input stride along the working axis
};
template <int AXIS> __device__ __forceinline__ AxisPos axis_pos(const AxisDims& d) {
  AxisPos p;
  const unsigned t = blockIdx.x * kAxisThreads + threadIdx.x;
  const unsigned total = (unsigned)d.out[0] * (unsigned)d.out[1] * (unsigned)d.out[2];
  p.valid = t < total;
  p.t = t;
  const unsigned r = t / (unsigned)d.out[0];
  p.c[0] = (int)(t - r * (unsigned)d.out[0]);
  p.c[2] = (int)(r / (unsigned)d.out[1]);
  p.c[1] = (int)(r - (unsigned)p.c[2] * (unsigned)d.out[1]);
  // the working axis is a compile-time constant: no dynamically indexed local arrays
  p.base = lin(d.in, AXIS == 0 ? 0 : p.c[0], AXIS == 1 ? 0 : p.c[1], AXIS == 2 ? 0 : p.c[2]);
  p.stride = AXIS == 0 ? 1 : (AXIS == 1 ? (size_t)d.in[0] : (size_t)d.in[0] * d.in[1]);
  return p;
}

// out[o] = sum_k w[k] in_logical[o - H - k]: omega' filter that also lays down the halo.
// Logical input index i: periodic -> in[i mod M]; open -> in[i] inside [0, M), else 0.
// One thread per output; the wrapped index is carried along the taps (one modulo per thread).
template <typename T, int AXIS>
__global__ void k_pad_filter(AxisDims d, int H, AxisTaps<T> w, const T* __restrict__ in, T* __restrict__ out) {
  const AxisPos p = axis_pos<AXIS>(d);
  if (!p.valid) return;
  const size_t t = p.t;
  const int g = p.c[AXIS] - H, M = d.in[AXIS], hw = w.n / 2;
  const T* line = in + p.base;
  T acc = 0;
  if (d.periodic) {
    int i = imod(g + hw, M);                       // tap k = -hw reads logical index g + hw
    for (int k = 0; k < w.n; ++k) {
      acc = fma(w.c[k], line[(size_t)i * p.stride], acc);
      if (--i < 0) i += M;
    }
  } else {
    const int klo = max(0, g + hw - (M - 1)), khi = min(w.n - 1, g + hw);   // 0 <= g + hw - k < M
    for (int k = klo; k <= khi; ++k) acc = fma(w.c[k], line[(size_t)(g + hw - k) * p.stride], acc);
  }
  out[t] = acc;
}

// The same filter with the tap count NT known at compile time: one thread computes RUN consecutive
// outputs along the working axis from NT + RUN - 1 loaded inputs (each input is read once per
// thread instead of NT times by NT threads), taps as immediates/constant operands.
constexpr int kFilterRun = 4;
template <typename T, int AXIS, int NT>
__global__ void __launch_bounds__(kAxisThreads)
k_pad_filter_run(AxisDims d, int H, AxisTaps<T> w, const T* __restrict__ in, T* __restrict__ out) {
  constexpr int RUN = kFilterRun, HW = NT / 2;
  // thread grid: the output dims with the working axis divided by RUN
  const unsigned na = ((unsigned)d.out[AXIS] + RUN - 1) / RUN;
  const unsigned g0 = AXIS == 0 ? na : (unsigned)d.out[0], g1 = AXIS == 1 ? na : (unsigned)d.out[1],
                 g2 = AXIS == 2 ? na : (unsigned)d.out[2];
  const unsigned t = blockIdx.x * kAxisThreads + threadIdx.x;
  if (t >= g0 * g1 * g2) return;
  const unsigned r = t / g0;
  int c[3] = {(int)(t - r * g0), 0, (int)(r / g1)};
  c[1] = (int)(r - (unsigned)c[2] * g1);
  const int o0 = c[AXIS] * RUN;                      // first output of this thread along the axis
  const int M = d.in[AXIS];
  const size_t istride = AXIS == 0 ? 1 : (AXIS == 1 ? (size_t)d.in[0] : (size_t)d.in[0] * d.in[1]);
  const size_t ostride = AXIS == 0 ? 1 : (AXIS == 1 ? (size_t)d.out[0] : (size_t)d.out[0] * d.out[1]);
  const T* line = in + lin(d.in, AXIS == 0 ? 0 : c[0], AXIS == 1 ? 0 : c[1], AXIS == 2 ? 0 : c[2]);
  T* oline = out + lin(d.out, AXIS == 0 ? 0 : c[0], AXIS == 1 ? 0 : c[1], AXIS == 2 ? 0 : c[2]);
  // inputs: logical indices g = o0 - H - HW ... o0 - H + HW + RUN - 1
  T v[NT + RUN - 1];
  int i = o0 - H - HW;
  if (d.periodic) {
    i = imod(i, M);
#pragma unroll
    for (int j = 0; j < NT + RUN - 1; ++j) {
      v[j] = line[(size_t)i * istride];
      if (++i >= M) i -= M;
    }
  } else {
#pragma unroll
    for (int j = 0; j < NT + RUN - 1; ++j, ++i) v[j] = (i >= 0 && i < M) ? line[(size_t)i * istride] : (T)0;
  }
  // output o0 + q reads logical o0 + q - H - k', k' = -HW..HW: v[q + HW - k'] with tap w.c[k' + HW]
#pragma unroll
  for (int q = 0; q < RUN; ++q) {
    if (o0 + q >= d.out[AXIS]) break;
    T acc = 0;
#pragma unroll
    for (int k = 0; k < NT; ++k) acc = fma(w.c[k], v[q + NT - 1 - k], acc);
    oline[(size_t)(o0 + q) * ostride] = acc;
  }
}
inline unsigned filter_run_grid(const AxisDims& d) {
  size_t total = 1;
  for (int k = 0; k < 3; ++k) total *= k == d.axis ? (size_t)(d.out[k] + kFilterRun - 1) / kFilterRun : (size_t)d.out[k];
  return (unsigned)((total + kAxisThreads - 1) / kAxisThreads);
}

// out[m] = sum_n J_n in[2(m + lo_out) + n - lo_in]   (restriction along one axis)
template <typename T, int AXIS>
__global__ void k_restrict_axis(AxisDims d, int lo_in, int lo_out, AxisTaps<T> J, const T* __restrict__ in,
                                T* __restrict__ out) {
  const AxisPos p = axis_pos<AXIS>(d);
  if (!p.valid) return;
  const size_t t = p.t;
  const int m = p.c[AXIS], M = d.in[AXIS], hw = J.n / 2;
  const T* line = in + p.base;
  if (d.periodic && M == 1) { out[t] = line[0]; return; }
  T acc = 0;
  const int i0 = 2 * (m + lo_out) - hw - lo_in;    // tap n = -hw
  if (d.periodic) {
    int i = imod(i0, M);
    for (int k = 0; k < J.n; ++k) {
      acc = fma(J.c[k], line[(size_t)i * p.stride], acc);
      if (++i >= M) i -= M;
    }
  } else {
    const int klo = max(0, -i0), khi = min(J.n - 1, M - 1 - i0);
    for (int k = klo; k <= khi; ++k) acc = fma(J.c[k], line[(size_t)(i0 + k) * p.stride], acc);
  }
  out[t] = acc;
}

// Restriction with the mask length NJ = p + 1 known at compile time: one thread computes RUN
// consecutive coarse outputs along the working axis from 2 RUN + NJ - 2 loaded fine values.
template <typename T, int AXIS, int NJ>
__global__ void __launch_bounds__(kAxisThreads)
k_restrict_axis_run(AxisDims d, int lo_in, int lo_out, AxisTaps<T> J, const T* __restrict__ in, T* __restrict__ out) {
  constexpr int RUN = kFilterRun, HW = NJ / 2, NV = 2 * RUN + NJ - 2;
  const unsigned na = ((unsigned)d.out[AXIS] + RUN - 1) / RUN;
  const unsigned g0 = AXIS == 0 ? na : (unsigned)d.out[0], g1 = AXIS == 1 ? na : (unsigned)d.out[1],
                 g2 = AXIS == 2 ? na : (unsigned)d.out[2];
  const unsigned t = blockIdx.x * kAxisThreads + threadIdx.x;
  if (t >= g0 * g1 * g2) return;
  const unsigned r = t / g0;
  int c[3] = {(int)(t - r * g0), 0, (int)(r / g1)};
  c[1] = (int)(r - (unsigned)c[2] * g1);
  const int m0 = c[AXIS] * RUN;
  const int M = d.in[AXIS];
  const size_t istride = AXIS == 0 ? 1 : (AXIS == 1 ? (size_t)d.in[0] : (size_t)d.in[0] * d.in[1]);
  const size_t ostride = AXIS == 0 ? 1 : (AXIS == 1 ? (size_t)d.out[0] : (size_t)d.out[0] * d.out[1]);
  const T* line = in + lin(d.in, AXIS == 0 ? 0 : c[0], AXIS == 1 ? 0 : c[1], AXIS == 2 ? 0 : c[2]);
  T* oline = out + lin(d.out, AXIS == 0 ? 0 : c[0], AXIS == 1 ? 0 : c[1], AXIS == 2 ? 0 : c[2]);
  T v[NV];
  int i = 2 * (m0 + lo_out) - HW - lo_in;            // fine array index of tap -HW of output m0
  if (d.periodic) {
    i = imod(i, M);
#pragma unroll
    for (int j = 0; j < NV; ++j) {
      v[j] = line[(size_t)i * istride];
      if (++i >= M) i -= M;
    }
  } else {
#pragma unroll
    for (int j = 0; j < NV; ++j, ++i) v[j] = (i >= 0 && i < M) ? line[(size_t)i * istride] : (T)0;
  }
#pragma unroll
  for (int q = 0; q < RUN; ++q) {
    if (m0 + q >= d.out[AXIS]) break;
    T acc = 0;
#pragma unroll
    for (int k = 0; k < NJ; ++k) acc = fma(J.c[k], v[2 * q + k], acc);
    oline[(size_t)(m0 + q) * ostride] = acc;
  }
}

// S6: dense top-level operator e = T q, one warp per row; with VIRIAL also the six quadratic forms
// q_r (TD_k q)_r per row (summed later in fixed order).
template <typename T, bool VIRIAL>
__global__ void __launch_bounds__(128)
k_top_dense(int G, const T* __restrict__ Tm, const T* __restrict__ TD, const T* __restrict__ q,
            T* __restrict__ e, double* __restrict__ wrow) {
  const int row = blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5);
  const int lane = threadIdx.x & 31;
  if (row >= G) return;
  constexpr int NK = VIRIAL ? 7 : 1;
  double acc[NK];
#pragma unroll
  for (int k = 0; k < NK; ++k) acc[k] = 0.0;
  for (int col = lane; col < G; col += 32) {
    const double qc = (double)q[col];
    acc[0] += (double)Tm[(size_t)row * G + col] * qc;
    if (VIRIAL) {
#pragma unroll
      for (int k = 0; k < 6; ++k) acc[k + 1] += (double)TD[((size_t)k * G + row) * G + col] * qc;
    }
  }
#pragma unroll
  for (int k = 0; k < NK; ++k)
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) acc[k] += __shfl_down_sync(0xffffffffu, acc[k], o);
  if (lane == 0) {
    e[row] = (T)acc[0];
    if (VIRIAL) {
      const double qr = (double)q[row];
#pragma unroll
      for (int k = 0; k < 6; ++k) wrow[(size_t)row * 6 + k] = -0.5 * qr * acc[k + 1];
    }
  }
}

}  // namespace msm
