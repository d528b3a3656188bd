// anterp_tiled.cuh -- S3 anterpolation (Eq. 9; Alg. 1) with warp-private shared-
// memory grids reduced in a fixed order: scatter-free in global memory, no atomics, deterministic.
//
// A tile is a box of T[0] x T[1] x T[2] level-1 grid cells owned by ONE warp. The warp walks the tile's particles
// in the canonical sorted order (cell by cell, ascending original index inside a cell) and adds
// each particle's p^3 contributions q_i phi_m(r_i) to its private (T+p-1)^3 node grid in shared
// memory: lane t handles nodes t, t+32, ... of the p^3 block, so one particle's targets are all
// distinct, and particles are processed one after the other, so every node sees its additions in a
// fixed order. Every lane evaluates the weights of its own nodes from spline pieces it holds in
// registers or takes as constant operands (no shuffles: the shared-memory/shuffle pipe is the
// bottleneck of this kernel): for p = 4 a lane owns nodes t and t + 32 of the 64, for p >= 6 it owns
// (jx, jy) pairs and walks jz. The batch of particle records is broadcast from shared memory. Grids
// with few tiles give every tile several warps (each takes every split-th row of cells and writes
// its own scratch grid). The tile grids go to a scratch array; a second
// kernel sums, for every node, the (at most 8) tiles that cover it in a fixed order. Used when
// every periodic axis has at least T + p - 1 nodes (each node then appears at
// most once in a tile's grid); smaller grids use the gather kernel of particle_grid.cuh.
#pragma once
#include "particle_grid.cuh"

namespace msm {

constexpr int kMaxAnterpRows = 64;   // T[1] * T[2]

struct AnterpTiles {
  int T[3];        // tile edge in grid cells per axis (each >= p - 1), a power of two
  int tshift[3];   // log2(T)
  int nt[3];       // tiles per axis
  int D[3];        // T + p - 1: tile grid edge in nodes
  int split;       // warps per tile: warp s takes the cell rows r = s (mod split), own scratch grid
};

// dynamic shared memory of k_anterp_tiles: node grid (padded so that the int arrays
// and the 32-byte records that follow stay aligned), row tables, batch staging
template <typename T, int P> inline size_t anterp_smem_bytes(int D3) {
  const size_t grid_elems = ((size_t)D3 + P * P + 7) / 8 * 8;
  return grid_elems * sizeof(T) + (2 * kMaxAnterpRows + 2 + 32 + 6) * sizeof(int) + 32 * 4 * sizeof(T);
}

template <typename T, int P>
__global__ void __launch_bounds__(32)
k_anterp_tiles(GridGeom g, AnterpTiles at, SplineTab<T, P> tab, const int* __restrict__ gstart,
               const typename Vec4<T>::type* __restrict__ grec, const int* __restrict__ gcell_sorted,
               T* __restrict__ scratch) {
  using V4 = typename Vec4<T>::type;
  extern __shared__ __align__(16) unsigned char smem_raw[];
  T* tg = reinterpret_cast<T*>(smem_raw);          // D^3 node grid
  const int D3 = at.D[0] * at.D[1] * at.D[2], Dx = at.D[0], Dy = at.D[1];
  constexpr int NT = (P * P * P + 31) / 32;        // nodes per lane
  const int lane = threadIdx.x;
  const int sub = blockIdx.x % at.split;
  int tl = blockIdx.x / at.split;
  const int tx = tl % at.nt[0]; tl /= at.nt[0];
  const int ty = tl % at.nt[1], tz = tl / at.nt[1];
  const int C0[3] = {tx * at.T[0], ty * at.T[1], tz * at.T[2]};
  for (int i = lane; i < D3; i += 32) tg[i] = 0;
  // static node offsets of this lane inside a particle's p^3 block, and the lanes that hold its weights
  int noff[NT];
#pragma unroll
  for (int s = 0; s < NT; ++s) {
    const int t = min(lane + 32 * s, P * P * P - 1);
    const int jx = t % P, jy = (t / P) % P, jz = t / (P * P);
    noff[s] = (jz * Dy + jy) * Dx + jx;
  }
  constexpr bool kRegRows = (32 % P) == 0 && P * P <= 32;
  constexpr int NP = (P * P + 31) / 32;              // (jx, jy) pairs per lane in the other path
  T pxr[kRegRows ? 1 : NP][P], pyr[kRegRows ? 1 : NP][P];
  int poff[NP];
  if (!kRegRows) {
#pragma unroll
    for (int s2 = 0; s2 < NP; ++s2) {
      const int t = min(lane + 32 * s2, P * P - 1);
      const int jx = t % P, jy = t / P;
      poff[s2] = jy * Dx + jx;
#pragma unroll
      for (int k = 0; k < P; ++k) { pxr[s2][k] = tab.c[jx][k]; pyr[s2][k] = tab.c[jy][k]; }
    }
  }
  T cxr[P], cyr[P], czr[kRegRows ? NT : 1][P];       // spline pieces of this lane's rows
  if (kRegRows) {
    const int jx = lane % P, jy = (lane / P) % P;
#pragma unroll
    for (int k = 0; k < P; ++k) { cxr[k] = tab.c[jx][k]; cyr[k] = tab.c[jy][k]; }
#pragma unroll
    for (int s2 = 0; s2 < NT; ++s2) {
      const int jz = min((lane + 32 * s2) / (P * P), P - 1);
#pragma unroll
      for (int k = 0; k < P; ++k) czr[s2][k] = tab.c[jz][k];
    }
  }
  __syncwarp();
  const int czn = min(at.T[2], g.ng[2] - C0[2]), cyn = min(at.T[1], g.ng[1] - C0[1]),
            cxn = min(at.T[0], g.ng[0] - C0[0]);
  // the tile's particles are one contiguous run per (cz, cy) row of cells: fetch all row bounds at
  // once and walk the concatenation of the runs (row-major, so the canonical order is kept)
  const int nrows_all = czn * cyn;
  const int nrows = (nrows_all - sub + at.split - 1) / at.split;      // rows sub, sub + split, ...
  int* rks = reinterpret_cast<int*>(tg + (D3 + P * P + 7) / 8 * 8);   // first particle of row r
  int* roff = rks + kMaxAnterpRows;                  // particles before row r; roff[nrows] = total
  int* sbase = roff + kMaxAnterpRows + 2;            // node offset of each particle of the batch
  V4* srec = reinterpret_cast<V4*>(sbase + 32 + 6);  // the batch's records (offset is a multiple of 32 B)
  for (int r = lane; r < nrows; r += 32) {
    const int ra = sub + r * at.split;
    const int cz = ra / cyn, cy = ra - cz * cyn;
    const int rowbase = ((C0[2] + cz) * g.ng[1] + (C0[1] + cy)) * g.ng[0];
    const int ks = gstart[rowbase + C0[0]], ke = gstart[rowbase + C0[0] + cxn];
    rks[r] = ks;
    roff[r + 1] = ke - ks;
  }
  __syncwarp();
  if (lane == 0) {
    roff[0] = 0;
    for (int r = 0; r < nrows; ++r) roff[r + 1] += roff[r];
  }
  __syncwarp();
  const int total = roff[nrows];
  for (int k0 = 0; k0 < total; k0 += 32) {
    // coalesced (per row) load of up to 32 particles, then one after the other through shuffles
    V4 r = make_vec4<T>(0, 0, 0, 0);
    int mybase = 0;
    const int flat = k0 + lane;
    if (flat < total) {
      int lo = 0, hi = nrows - 1;                     // last row with roff[row] <= flat
      while (lo < hi) {
        const int mid = (lo + hi + 1) >> 1;
        if (roff[mid] <= flat) lo = mid; else hi = mid - 1;
      }
      const int ra = sub + lo * at.split;
      const int cz = ra / cyn, cy = ra - cz * cyn;
      const int rowbase = ((C0[2] + cz) * g.ng[1] + (C0[1] + cy)) * g.ng[0];
      const int k = rks[lo] + (flat - roff[lo]);
      r = ldg4(grec + k);
      mybase = (cz * Dy + cy) * Dx - C0[0] + (gcell_sorted[k] - rowbase);
    }
    const int cnt = min(32, total - k0);
    srec[lane] = r;
    sbase[lane] = mybase;
    __syncwarp();
    for (int i = 0; i < cnt; ++i) {
      const V4 pr = srec[i];                          // broadcast
      const int base = sbase[i];
      if (kRegRows) {
        T wx = cxr[P - 1], wy = cyr[P - 1];
#pragma unroll
        for (int k = P - 2; k >= 0; --k) { wx = fma(wx, pr.x, cxr[k]); wy = fma(wy, pr.y, cyr[k]); }
        const T wxy = wx * wy * pr.w;
#pragma unroll
        for (int s2 = 0; s2 < NT; ++s2) {
          T wz = czr[s2][P - 1];
#pragma unroll
          for (int k = P - 2; k >= 0; --k) wz = fma(wz, pr.z, czr[s2][k]);
          if (lane + 32 * s2 < P * P * P) {
            T* dst = tg + base + noff[s2];
            *dst = fma(wz, wxy, *dst);
          }
        }
      } else {
        // lanes own (jx, jy) pairs (pair t = lane + 32 s) and walk jz; the z weights use the spline
        // pieces straight from the kernel parameters (compile-time rows: constant operands), the x
        // and y weights the pieces of the lane's own rows in registers -- no shuffles
        T wz[P];
#pragma unroll
        for (int j = 0; j < P; ++j) {
          T w = tab.c[j][P - 1];
#pragma unroll
          for (int k = P - 2; k >= 0; --k) w = fma(w, pr.z, tab.c[j][k]);
          wz[j] = w * pr.w;
        }
#pragma unroll
        for (int s2 = 0; s2 < NP; ++s2) {
          T wx = pxr[s2][P - 1], wy = pyr[s2][P - 1];
#pragma unroll
          for (int k = P - 2; k >= 0; --k) { wx = fma(wx, pr.x, pxr[s2][k]); wy = fma(wy, pr.y, pyr[s2][k]); }
          const T wxy = wx * wy;
          if (lane + 32 * s2 < P * P) {
            T* dst = tg + base + poff[s2];
#pragma unroll
            for (int j = 0; j < P; ++j) dst[j * Dx * Dy] = fma(wz[j], wxy, dst[j * Dx * Dy]);
          }
        }
      }
      __syncwarp();
    }
  }
  T* out = scratch + (size_t)blockIdx.x * D3;
  for (int i = lane; i < D3; i += 32) out[i] = tg[i];
}

// Q[m] = sum over the tiles whose grid covers node m (at most two per axis), in a fixed order.
// Threads are laid out in 3-D (32 nodes in x, 4 in y per block, blockIdx.z = z) and the tile edges
// are powers of two, so a node's tiles and local indices cost shifts instead of the ten integer
// divisions per node of the linear layout (49 M warp instructions for 2 M nodes at N = 10^6).
template <typename T, int P, bool SPLIT>
__global__ void __launch_bounds__(128)
k_anterp_combine(GridGeom g, AnterpTiles at, const T* __restrict__ scratch, T* __restrict__ Q) {
  constexpr int HP = P / 2;
  const int mi[3] = {(int)(blockIdx.x * 32 + threadIdx.x), (int)(blockIdx.y * 4 + threadIdx.y), (int)blockIdx.z};
  if (mi[0] >= g.M[0] || mi[1] >= g.M[1]) return;
  int tix[3][2], lix[3][2], cnt[3];
#pragma unroll
  for (int ax = 0; ax < 3; ++ax) {
    const int n = mi[ax] + g.lo[ax];                 // node index; cells n - HP .. n + HP - 1 touch it
    int c0 = n - HP, c1 = n + HP - 1;
    if (g.periodic[ax]) {                            // -HP <= c0, c1 < M + HP and M >= D > P
      if (c0 < 0) c0 += g.ng[ax];
      if (c1 >= g.ng[ax]) c1 -= g.ng[ax];
    } else {
      c0 = max(c0, 0); c1 = min(c1, g.ng[ax] - 1);
    }
    const int t0 = c0 >> at.tshift[ax], t1 = c1 >> at.tshift[ax];
    // local index of node n in tile t's grid, whose first node is T * t - HP + 1
    int l0 = n - ((t0 << at.tshift[ax]) - HP + 1), l1 = n - ((t1 << at.tshift[ax]) - HP + 1);
    if (g.periodic[ax]) {
      if (l0 < 0) l0 += g.M[ax]; else if (l0 >= g.M[ax]) l0 -= g.M[ax];
      if (l1 < 0) l1 += g.M[ax]; else if (l1 >= g.M[ax]) l1 -= g.M[ax];
    }
    tix[ax][0] = t0; lix[ax][0] = l0;
    tix[ax][1] = t1; lix[ax][1] = l1;
    cnt[ax] = t1 != t0 ? 2 : 1;
  }
  const unsigned D3 = (unsigned)(at.D[0] * at.D[1] * at.D[2]);
  T acc = 0;
  for (int a = 0; a < cnt[2]; ++a)
    for (int b = 0; b < cnt[1]; ++b)
      for (int c = 0; c < cnt[0]; ++c) {
        const unsigned tile = ((unsigned)tix[2][a] * at.nt[1] + tix[1][b]) * at.nt[0] + tix[0][c];
        const unsigned off = ((unsigned)lix[2][a] * at.D[1] + lix[1][b]) * at.D[0] + lix[0][c];
        if (SPLIT) {
          for (int sb = 0; sb < at.split; ++sb) acc += scratch[(size_t)(tile * at.split + sb) * D3 + off];
        } else {
          acc += scratch[(size_t)tile * D3 + off];
        }
      }
  Q[((size_t)mi[2] * g.M[1] + mi[1]) * g.M[0] + mi[0]] = acc;
}

}  // namespace msm
