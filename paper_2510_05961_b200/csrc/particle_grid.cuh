// particle_grid.cuh -- S3 anterpolation (Eq. 9; Alg. 1) as a scatter-free gather,
// and S8 fused interpolation of potential and gradient (Eq. 16-18).
#pragma once
#include "device_common.cuh"

namespace msm {

struct GridGeom {
  int M[3];         // level-1 grid points per axis
  int lo[3];        // node index of array position 0
  int ng[3];        // grid cells per axis (particle cell index i0 in [0, ng))
  int periodic[3];
};

// 2^lg lanes per level-1 grid point m (16 for a plan on its own, 1 inside a batch, where the other
// systems fill the GPU): q~_m = sum_i q_i phi_m(r_i), gathered from the particles of the p^3 grid
// cells whose support contains m. Lane s of a node's group takes the cell rows (jz, jy) with index
// s (mod 2^lg) and walks their p cells along x (ascending cell index, particles inside a cell in
// ascending original index); the partial sums are added in a fixed shuffle tree -> no atomics,
// bit-reproducible. (One thread per node walks p^3 cells one after the other, two dependent global
// loads each: 43 us for 3000 particles on a 16^3 grid, 11 us with 16 lanes.)
template <typename T, int P>
__global__ void __launch_bounds__(128)
k_anterpolate(GridGeom g, SplineTab<T, P> tab, const int* __restrict__ gstart,
              const typename Vec4<T>::type* __restrict__ grec, T* __restrict__ Q, int lg) {
  constexpr int HP = P / 2;
  const int total = g.M[0] * g.M[1] * g.M[2];
  const int G = 1 << lg;
  const int sub = threadIdx.x & (G - 1);
  const int m = (int)((blockIdx.x * blockDim.x + threadIdx.x) >> lg);
  const bool live = m < total;                       // (whole groups: every lane reaches the shuffles)
  const int mc = live ? m : 0;
  const int mx = mc % g.M[0], my = (mc / g.M[0]) % g.M[1], mz = mc / (g.M[0] * g.M[1]);
  const int nx = mx + g.lo[0], ny = my + g.lo[1], nz = mz + g.lo[2];   // node indices
  T acc = 0;
  // node n = i0 + j, j = -HP+1..HP  ->  cell i0 = n - j, spline row j + HP - 1
#pragma unroll 1
  for (int row = sub; row < P * P; row += G) {
    const int jz = row / P - HP + 1, jy = row % P - HP + 1;
    int cz = nz - jz, cy = ny - jy;
    if (g.periodic[2]) cz = imod(cz, g.ng[2]);
    else if (cz < 0 || cz >= g.ng[2]) continue;
    if (g.periodic[1]) cy = imod(cy, g.ng[1]);
    else if (cy < 0 || cy >= g.ng[1]) continue;
    if (!live) continue;
    const int rowbase = (cz * g.ng[1] + cy) * g.ng[0];
#pragma unroll
    for (int jx = HP; jx >= -HP + 1; --jx) {         // ascending cell index
      int cx = nx - jx;
      if (g.periodic[0]) cx = imod(cx, g.ng[0]);
      else if (cx < 0 || cx >= g.ng[0]) continue;
      const int s = gstart[rowbase + cx], e = gstart[rowbase + cx + 1];
      for (int k = s; k < e; ++k) {
        const auto r = ldg4(grec + k);
        const T wx = spline_weight_row<T, P>(tab, jx + HP - 1, r.x);
        const T wy = spline_weight_row<T, P>(tab, jy + HP - 1, r.y);
        const T wz = spline_weight_row<T, P>(tab, jz + HP - 1, r.z);
        acc = fma(r.w, wx * wy * wz, acc);
      }
    }
  }
  for (int o = G >> 1; o > 0; o >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, o);
  if (live && sub == 0) Q[m] = acc;
}

// One thread per particle (grid-cell order): V_i^lr = sum_m e_m phi_m(r_i), grad = sum_m e_m grad
// phi_m(r_i); final outputs in caller order:
//   potential_i = V_i^sr + V_i^lr - q_i gamma(0)/a        (self term, Eq. 5, reading K2)
//   F_i         = F_i^sr - q_i grad                        (Eq. 17)
// and the block's share of U = 1/2 sum_i q_i potential_i (fp64, fixed order).
template <typename T, int P>
__global__ void __launch_bounds__(128)
k_interpolate(int n, int nsplit, size_t part_stride, GridGeom g, SplineTab<T, P> tab, T inv_h0, T inv_h1, T inv_h2,
              T self_coef,
              const typename Vec4<T>::type* __restrict__ grec, const int* __restrict__ gcell_sorted,
              const int* __restrict__ gorder, const T* __restrict__ E, const T* __restrict__ Fsr,
              const T* __restrict__ Vsr, T* __restrict__ F_out, T* __restrict__ V_out,
              double* __restrict__ epart) {
  constexpr int HP = P / 2;
  __shared__ double red[4];
  const int k = blockIdx.x * blockDim.x + threadIdx.x;
  double e_i = 0.0;
  if (k < n) {
    const auto r = ldg4(grec + k);
    int c = gcell_sorted[k];
    const int cx = c % g.ng[0]; c /= g.ng[0];
    const int cy = c % g.ng[1], cz = c / g.ng[1];
    T wx[P], wy[P], wz[P], dx[P], dy[P], dz[P];
    spline_weights<T, P>(tab, r.x, wx); spline_dweights<T, P>(tab, r.x, dx);
    spline_weights<T, P>(tab, r.y, wy); spline_dweights<T, P>(tab, r.y, dy);
    spline_weights<T, P>(tab, r.z, wz); spline_dweights<T, P>(tab, r.z, dz);
    int ix[P], iy[P], iz[P];
#pragma unroll
    for (int j = 0; j < P; ++j) {
      const int o = j - HP + 1;           // node = i0 + o
      ix[j] = g.periodic[0] ? imod(cx + o, g.M[0]) : cx + o - g.lo[0];
      iy[j] = g.periodic[1] ? imod(cy + o, g.M[1]) : cy + o - g.lo[1];
      iz[j] = g.periodic[2] ? imod(cz + o, g.M[2]) : cz + o - g.lo[2];
    }
    T v = 0, gx = 0, gy = 0, gz = 0;
#pragma unroll
    for (int a = 0; a < P; ++a) {
      T vz = 0, gxz = 0, gyz = 0;
#pragma unroll
      for (int b = 0; b < P; ++b) {
        const T* row = E + ((size_t)iz[a] * g.M[1] + iy[b]) * g.M[0];
        T rw = 0, rd = 0;
#pragma unroll
        for (int cc = 0; cc < P; ++cc) {
          const T e = __ldg(row + ix[cc]);
          rw = fma(e, wx[cc], rw);
          rd = fma(e, dx[cc], rd);
        }
        vz = fma(wy[b], rw, vz);
        gxz = fma(wy[b], rd, gxz);
        gyz = fma(dy[b], rw, gyz);
      }
      v = fma(wz[a], vz, v);
      gx = fma(wz[a], gxz, gx);
      gy = fma(wz[a], gyz, gy);
      gz = fma(dz[a], vz, gz);
    }
    const int orig = gorder[k];
    const T q = r.w;
    // short-range partials of the pair kernel's splits, added in split order
    T vs = Vsr[orig], fsx = Fsr[3 * (size_t)orig + 0], fsy = Fsr[3 * (size_t)orig + 1], fsz = Fsr[3 * (size_t)orig + 2];
    for (int s = 1; s < nsplit; ++s) {
      vs += Vsr[s * part_stride + orig];
      const T* Fp = Fsr + s * 3 * part_stride;
      fsx += Fp[3 * (size_t)orig + 0]; fsy += Fp[3 * (size_t)orig + 1]; fsz += Fp[3 * (size_t)orig + 2];
    }
    const T pot = vs + v - q * self_coef;
    if (V_out) V_out[orig] = pot;
    if (F_out) {
      F_out[3 * (size_t)orig + 0] = fsx - q * gx * inv_h0;
      F_out[3 * (size_t)orig + 1] = fsy - q * gy * inv_h1;
      F_out[3 * (size_t)orig + 2] = fsz - q * gz * inv_h2;
    }
    e_i = 0.5 * (double)q * (double)pot;
  }
  const double s = block_reduce_sum<128>(e_i, red);
  if (threadIdx.x == 0) epart[blockIdx.x] = s;
}

}  // namespace msm
