// gridops_fused.cuh -- S7 prolongation + accumulate (Eq. 19 line 2; Eq. 13) as ONE
// kernel per level: the three one-axis passes of the separable operator run inside shared
// memory on a tile, so E^l is read and written once (HBM-bound stage: read G_l / 8 + G_l, write
// G_l). A block owns 32 x 8 x 8 fine points, stages the (T/2 + p/2 + 1)^3-shaped coarse region that
// reaches them (periodic wrap or zeros outside an open grid), expands x, y, z and accumulates.
// (A restriction fused the same way measured slower than the three one-axis kernels of gridops.cuh
// -- its tile has to stage 14 fine values per coarse output -- and was not kept.)
#pragma once
#include "gridops.cuh"

namespace msm {

struct Grid3 {
  int M[3];    // array dims (x, y, z)
  int lo[3];   // node index of array position 0
};

constexpr int kPTX = 32, kPTY = 8, kPTZ = 8;   // prolongation tile (fine points)

// shared-memory elements of the kernel for spline order p
inline size_t prolong3_smem_elems(int p) {
  const size_t rx = kPTX / 2 + p / 2 + 1, ry = kPTY / 2 + p / 2 + 1, rz = kPTZ / 2 + p / 2 + 1;
  return rx * ry * rz + (size_t)kPTX * ry * rz + (size_t)kPTX * kPTY * rz;
}

__device__ __forceinline__ int floor_div2(int v) { return v >> 1; }            // arithmetic shift: floor
__device__ __forceinline__ int ceil_div2(int v) { return -((-v) >> 1); }

// E_fine[i] += sum_{nx,ny,nz} J J J e_coarse[m], 2 m + n = i on every axis (exact transpose)
template <typename T>
__global__ void __launch_bounds__(256)
k_prolong3(Grid3 f, Grid3 c, int per_x, int per_y, int per_z, AxisTaps<T> J, const T* __restrict__ ec,
           T* __restrict__ E) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  const int hp = J.n / 2;
  const int per[3] = {per_x, per_y, per_z};
  const int i0[3] = {(int)blockIdx.x * kPTX, (int)blockIdx.y * kPTY, (int)blockIdx.z * kPTZ};
  int c0[3], RL[3], n0[3];
#pragma unroll
  for (int a = 0; a < 3; ++a) {
    n0[a] = i0[a] + f.lo[a];                                    // first fine node of the tile
    c0[a] = ceil_div2(n0[a] - hp);                              // first coarse node that reaches it
    RL[a] = (a == 0 ? kPTX : a == 1 ? kPTY : kPTZ) / 2 + hp + 1;
  }
  T* A = reinterpret_cast<T*>(smem_raw);             // [RLz][RLy][RLx] coarse
  T* B = A + RL[0] * RL[1] * RL[2];                  // [RLz][RLy][TX]
  T* C = B + kPTX * RL[1] * RL[2];                 // [RLz][TY][TX]
  const int tid = threadIdx.x;
  const int nA = RL[0] * RL[1] * RL[2];
  for (int e = tid; e < nA; e += 256) {
    const int rx = e % RL[0], r2 = e / RL[0];
    const int ry = r2 % RL[1], rz = r2 / RL[1];
    int ix = c0[0] + rx - c.lo[0], iy = c0[1] + ry - c.lo[1], iz = c0[2] + rz - c.lo[2];
    bool ok = true;
    if (per[0]) ix = imod(ix, c.M[0]); else ok &= ix >= 0 && ix < c.M[0];
    if (per[1]) iy = imod(iy, c.M[1]); else ok &= iy >= 0 && iy < c.M[1];
    if (per[2]) iz = imod(iz, c.M[2]); else ok &= iz >= 0 && iz < c.M[2];
    A[e] = ok ? ec[((size_t)iz * c.M[1] + iy) * c.M[0] + ix] : (T)0;
  }
  __syncthreads();
  // one axis: fine node i takes taps n = n_first, n_first + 2, ... <= hp with (i - n) even, coarse
  // node (i - n) / 2 descending by one per tap
  // x: B[z][y][fx]
  const int nB = kPTX * RL[1] * RL[2];
  for (int e = tid; e < nB; e += 256) {
    const int fx = e % kPTX, zy = e / kPTX;
    const int i = n0[0] + fx;
    const int nf = -hp + ((i + hp) & 1);
    int m = floor_div2(i - nf) - c0[0];
    const T* a = A + zy * RL[0];
    T s = 0;
    for (int n = nf; n <= hp; n += 2, --m)
      if (m >= 0 && m < RL[0]) s = fma(J.c[n + hp], a[m], s);
    B[e] = s;
  }
  __syncthreads();
  // y: C[z][fy][fx]
  const int nC = kPTX * kPTY * RL[2];
  for (int e = tid; e < nC; e += 256) {
    const int fx = e % kPTX, r2 = e / kPTX;
    const int fy = r2 % kPTY, z = r2 / kPTY;
    const int i = n0[1] + fy;
    const int nf = -hp + ((i + hp) & 1);
    int m = floor_div2(i - nf) - c0[1];
    const T* b = B + (size_t)z * RL[1] * kPTX + fx;
    T s = 0;
    for (int n = nf; n <= hp; n += 2, --m)
      if (m >= 0 && m < RL[1]) s = fma(J.c[n + hp], b[m * kPTX], s);
    C[e] = s;
  }
  __syncthreads();
  // z and accumulate
  const int nO = kPTX * kPTY * kPTZ;
  for (int e = tid; e < nO; e += 256) {
    const int fx = e % kPTX, r2 = e / kPTX;
    const int fy = r2 % kPTY, fz = r2 / kPTY;
    const int ox = i0[0] + fx, oy = i0[1] + fy, oz = i0[2] + fz;
    if (ox >= f.M[0] || oy >= f.M[1] || oz >= f.M[2]) continue;
    const int i = n0[2] + fz;
    const int nf = -hp + ((i + hp) & 1);
    int m = floor_div2(i - nf) - c0[2];
    const T* cc = C + fy * kPTX + fx;
    T s = 0;
    for (int n = nf; n <= hp; n += 2, --m)
      if (m >= 0 && m < RL[2]) s = fma(J.c[n + hp], cc[(size_t)m * kPTY * kPTX], s);
    E[((size_t)oz * f.M[1] + oy) * f.M[0] + ox] += s;
  }
}

}  // namespace msm
