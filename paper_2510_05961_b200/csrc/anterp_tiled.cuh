// anterp_tiled.cuh -- S3 anterpolation (Eq. 9; Alg. 1) with warp-private shared-
// memory grids reduced in a fixed order: scatter-free in global memory, no atomics, deterministic.
//
// A tile is a box of AT^3 level-1 grid cells owned by ONE warp. The warp walks the tile's particles
// in the canonical sorted order (cell by cell, ascending original index inside a cell) and adds
// each particle's p^3 contributions q_i phi_m(r_i) to its private (AT+p-1)^3 node grid in shared
// memory: lane t handles nodes t, t+32, ... of the p^3 block, so one particle's targets are all
// distinct, and particles are processed one after the other, so every node sees its additions in a
// fixed order. The 3p one-dimensional weights are evaluated once per particle (lane k < 3p
// evaluates weight k) and handed round by shuffles. The tile grids go to a scratch array; a second
// kernel sums, for every node, the (at most 27, typically 1-8) tiles that cover it in a fixed
// order. Used when every periodic axis has at least AT + p - 1 nodes (each node then appears at
// most once in a tile's grid); smaller grids use the gather kernel of particle_grid.cuh.
#pragma once
#include "particle_grid.cuh"

namespace msm {

constexpr int kAT = 8;   // tile edge in grid cells

struct AnterpTiles {
  int nt[3];       // tiles per axis
  int D;           // AT + p - 1: tile grid edge in nodes
};

template <typename T, int P>
__global__ void __launch_bounds__(32)
k_anterp_tiles(GridGeom g, AnterpTiles at, SplineTab<T, P> tab, const int* __restrict__ gstart,
               const typename Vec4<T>::type* __restrict__ grec, const int* __restrict__ gcell_sorted,
               T* __restrict__ scratch) {
  using V4 = typename Vec4<T>::type;
  extern __shared__ __align__(16) unsigned char smem_raw[];
  T* tg = reinterpret_cast<T*>(smem_raw);          // D^3 node grid
  T* coef = tg + at.D * at.D * at.D;               // P x P spline piece coefficients
  constexpr int NT = (P * P * P + 31) / 32;        // nodes per lane
  const int lane = threadIdx.x;
  const int D = at.D, D3 = D * D * D;
  int tl = blockIdx.x;
  const int tx = tl % at.nt[0]; tl /= at.nt[0];
  const int ty = tl % at.nt[1], tz = tl / at.nt[1];
  const int C0[3] = {tx * kAT, ty * kAT, tz * kAT};
  for (int i = lane; i < D3; i += 32) tg[i] = 0;
  for (int i = lane; i < P * P; i += 32) coef[i] = tab.c[i / P][i % P];
  // static node offsets of this lane inside a particle's p^3 block, and the lanes that hold its weights
  int noff[NT], lx[NT], ly[NT], lz[NT];
#pragma unroll
  for (int s = 0; s < NT; ++s) {
    const int t = min(lane + 32 * s, P * P * P - 1);
    const int jx = t % P, jy = (t / P) % P, jz = t / (P * P);
    noff[s] = (jz * D + jy) * D + jx;
    lx[s] = jx; ly[s] = P + jy; lz[s] = 2 * P + jz;
  }
  __syncwarp();
  const int czn = min(kAT, g.ng[2] - C0[2]), cyn = min(kAT, g.ng[1] - C0[1]), cxn = min(kAT, g.ng[0] - C0[0]);
  for (int cz = 0; cz < czn; ++cz)
    for (int cy = 0; cy < cyn; ++cy) {
      const int rowbase = ((C0[2] + cz) * g.ng[1] + (C0[1] + cy)) * g.ng[0];
      const int ks = gstart[rowbase + C0[0]], ke = gstart[rowbase + C0[0] + cxn];
      const int rowoff = (cz * D + cy) * D - C0[0];
      for (int k0 = ks; k0 < ke; k0 += 32) {
        // coalesced load of up to 32 particles, then one after the other through shuffles
        V4 r = make_vec4<T>(0, 0, 0, 0);
        int cx = 0;
        if (k0 + lane < ke) { r = ldg4(grec + k0 + lane); cx = gcell_sorted[k0 + lane] - rowbase; }
        const int cnt = min(32, ke - k0);
        // weight (axis a = lane / P, node offset j = lane % P) of MY particle's coordinate... is per
        // particle, so it is evaluated inside the loop from the broadcast fractions
        for (int i = 0; i < cnt; ++i) {
          const T fx = __shfl_sync(0xffffffffu, r.x, i), fy = __shfl_sync(0xffffffffu, r.y, i);
          const T fz = __shfl_sync(0xffffffffu, r.z, i), q = __shfl_sync(0xffffffffu, r.w, i);
          const int base = rowoff + __shfl_sync(0xffffffffu, cx, i);
          const int a = lane / P, j = lane - a * P;
          const T f = a == 0 ? fx : (a == 1 ? fy : fz);
          T w = 0;
          if (lane < 3 * P) {
            const T* c = coef + j * P;
            w = c[P - 1];
#pragma unroll
            for (int k = P - 2; k >= 0; --k) w = fma(w, f, c[k]);
            if (a == 2) w *= q;
          }
#pragma unroll
          for (int s = 0; s < NT; ++s) {
            const T wx = __shfl_sync(0xffffffffu, w, lx[s]);
            const T wy = __shfl_sync(0xffffffffu, w, ly[s]);
            const T wz = __shfl_sync(0xffffffffu, w, lz[s]);
            if (lane + 32 * s < P * P * P) {
              T* dst = tg + base + noff[s];
              *dst = fma(wz * wy, wx, *dst);
            }
          }
          __syncwarp();
        }
      }
    }
  T* out = scratch + (size_t)blockIdx.x * D3;
  for (int i = lane; i < D3; i += 32) out[i] = tg[i];
}

// Q[m] = sum over the tiles whose grid covers node m, tiles in ascending (z, y, x) visiting order
template <typename T, int P>
__global__ void __launch_bounds__(128)
k_anterp_combine(GridGeom g, AnterpTiles at, const T* __restrict__ scratch, T* __restrict__ Q) {
  constexpr int HP = P / 2;
  const int total = g.M[0] * g.M[1] * g.M[2];
  const int m = blockIdx.x * blockDim.x + threadIdx.x;
  if (m >= total) return;
  const int mi[3] = {m % g.M[0], (m / g.M[0]) % g.M[1], m / (g.M[0] * g.M[1])};
  const int D = at.D;
  // per axis: up to 3 (tile, local node index) candidates
  int tix[3][3], lix[3][3], cnt[3];
#pragma unroll
  for (int ax = 0; ax < 3; ++ax) {
    const int n = mi[ax] + g.lo[ax];                 // node index
    cnt[ax] = 0;
    int prev = -1;
#pragma unroll 1
    for (int i = 0; i < P; ++i) {                    // cells n - HP .. n + HP - 1 touch node n
      int c = n - HP + i;
      if (g.periodic[ax]) c = imod(c, g.ng[ax]);
      else if (c < 0 || c >= g.ng[ax]) continue;
      const int t = c / kAT;
      if (t == prev) continue;
      prev = t;
      // local index of node n in tile t's grid, whose first node is kAT * t - HP + 1
      int ln = n - (kAT * t - HP + 1);
      if (g.periodic[ax]) ln = imod(ln, g.M[ax]);
      if (cnt[ax] < 3 && ln >= 0 && ln < D) {
        bool dup = false;
        for (int k = 0; k < cnt[ax]; ++k) dup |= tix[ax][k] == t;
        if (!dup) { tix[ax][cnt[ax]] = t; lix[ax][cnt[ax]] = ln; ++cnt[ax]; }
      }
    }
  }
  T acc = 0;
  for (int a = 0; a < cnt[2]; ++a)
    for (int b = 0; b < cnt[1]; ++b)
      for (int c = 0; c < cnt[0]; ++c) {
        const size_t tile = ((size_t)tix[2][a] * at.nt[1] + tix[1][b]) * at.nt[0] + tix[0][c];
        acc += scratch[tile * D * D * D + ((size_t)lix[2][a] * D + lix[1][b]) * D + lix[0][c]];
      }
  Q[m] = acc;
}

}  // namespace msm
