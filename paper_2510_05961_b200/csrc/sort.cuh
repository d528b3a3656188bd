// sort.cuh -- S1: binning and counting sort of the particles, once by short-range cell and once
// by level-1 grid cell (replaces the paper's neighbour list; its construction is inside our
// timing). Within a cell particles are ordered by original index, so every later per-cell sum has
// a fixed order (run-to-run deterministic results).
#pragma once
#include "device_common.cuh"

namespace msm {

// wrapped / clamped coordinate and its integer cell, in fp64 on both precisions
__device__ __forceinline__ double wrap_coord(double x, double L, int periodic) {
  if (periodic) {
    x -= L * floor(x / L);
    if (x >= L) x = 0.0;
  }
  return x;
}

// pass 1: cell ids + histograms (+ input validation)
template <typename T>
__global__ void k_bin(int n, const T* __restrict__ pos, BinGeom g, int* __restrict__ pcell,
                      int* __restrict__ gcell, int* __restrict__ phist, int* __restrict__ ghist,
                      int* __restrict__ pslot, int* __restrict__ gslot, int* __restrict__ flag) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  int pc[3], gc[3], sub = 0;
  bool bad = false;
#pragma unroll
  for (int ax = 0; ax < 3; ++ax) {
    double x = (double)pos[3 * (size_t)i + ax];
    if (!isfinite(x)) { bad = true; x = 0.0; }
    if (!g.periodic[ax] && (x < 0.0 || x > g.box[ax])) { bad = true; x = fmin(fmax(x, 0.0), g.box[ax]); }
    x = wrap_coord(x, g.box[ax], g.periodic[ax]);
    int c = (int)floor(x / g.cell_edge[ax]);
    pc[ax] = min(max(c, 0), g.nc[ax] - 1);
    if (ax == 0) {   // sub-bin of the cell along x
      const int nsub = 1 << g.sxs;
      const int sb = (int)floor((x - pc[0] * g.cell_edge[0]) * (double)nsub / g.cell_edge[0]);
      sub = min(max(sb, 0), nsub - 1);
    }
    int k = (int)floor(x / g.h1[ax]);
    gc[ax] = min(max(k, 0), g.ng[ax] - 1);
  }
  if (bad) atomicOr(flag, 1);
  const int pci = (pc[2] * g.nc[1] + pc[1]) * (g.nc[0] << g.sxs) + (pc[0] << g.sxs) + sub;
  const int gci = (gc[2] * g.ng[1] + gc[1]) * g.ng[0] + gc[0];
  pcell[i] = pci;
  gcell[i] = gci;
  pslot[i] = atomicAdd(&phist[pci], 1);   // arrival rank inside the cell (any order: k_sort_cells fixes it)
  gslot[i] = atomicAdd(&ghist[gci], 1);
}

// exclusive scan, three kernels: per-block scan of 4096-element tiles, scan of the tile totals,
// add-back. data[m] must be writable (the total is written there).
constexpr int kScanThreads = 1024;
constexpr int kScanPerThread = 4;
constexpr int kScanTile = kScanThreads * kScanPerThread;

__global__ void k_scan_tiles(int m, const int* __restrict__ in, int* __restrict__ out,
                             int* __restrict__ totals) {
  __shared__ int wsum[32];
  const int base = blockIdx.x * kScanTile + threadIdx.x * kScanPerThread;
  int v[kScanPerThread], s = 0;
#pragma unroll
  for (int k = 0; k < kScanPerThread; ++k) {
    v[k] = (base + k < m) ? in[base + k] : 0;
    s += v[k];
  }
  const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
  int inc = s;
#pragma unroll
  for (int o = 1; o < 32; o <<= 1) {
    const int t = __shfl_up_sync(0xffffffffu, inc, o);
    if (lane >= o) inc += t;
  }
  if (lane == 31) wsum[wid] = inc;
  __syncthreads();
  if (wid == 0) {
    int t = wsum[lane];
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
      const int u = __shfl_up_sync(0xffffffffu, t, o);
      if (lane >= o) t += u;
    }
    wsum[lane] = t;
  }
  __syncthreads();
  int excl = inc - s + (wid > 0 ? wsum[wid - 1] : 0);
#pragma unroll
  for (int k = 0; k < kScanPerThread; ++k) {
    if (base + k < m) out[base + k] = excl;
    excl += v[k];
  }
  if (threadIdx.x == kScanThreads - 1) totals[blockIdx.x] = excl;
}

__global__ void k_scan_totals(int nt, int* __restrict__ totals) {  // one block, nt <= 1024*? loop
  __shared__ int carry_s;
  __shared__ int wsum[32];
  if (threadIdx.x == 0) carry_s = 0;
  __syncthreads();
  for (int base = 0; base < nt; base += kScanThreads) {
    const int i = base + threadIdx.x;
    const int v = i < nt ? totals[i] : 0;
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    int inc = v;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
      const int t = __shfl_up_sync(0xffffffffu, inc, o);
      if (lane >= o) inc += t;
    }
    if (lane == 31) wsum[wid] = inc;
    __syncthreads();
    if (wid == 0) {
      int t = wsum[lane];
#pragma unroll
      for (int o = 1; o < 32; o <<= 1) {
        const int u = __shfl_up_sync(0xffffffffu, t, o);
        if (lane >= o) t += u;
      }
      wsum[lane] = t;
    }
    __syncthreads();
    const int carry = carry_s;
    const int excl = carry + inc - v + (wid > 0 ? wsum[wid - 1] : 0);
    if (i < nt) totals[i] = excl;
    __syncthreads();
    if (threadIdx.x == kScanThreads - 1) carry_s = excl + v;
    __syncthreads();
  }
}

// Both exclusive scans of a small system in ONE launch: block 0 scans the pair bins, block 1 the
// grid cells, tile after tile with a running carry (used while each array has at most
// kScanSerialMax elements; a small system is bound by its launch count, not by this loop).
constexpr int kScanSerialMax = 16 * kScanTile;
__global__ void __launch_bounds__(kScanThreads)
k_scan_serial2(int m0, const int* __restrict__ in0, int* __restrict__ out0, int m1, const int* __restrict__ in1,
               int* __restrict__ out1, int n_total) {
  __shared__ int wsum[32];
  __shared__ int carry_s;
  const int m = blockIdx.x == 0 ? m0 : m1;
  const int* __restrict__ in = blockIdx.x == 0 ? in0 : in1;
  int* __restrict__ out = blockIdx.x == 0 ? out0 : out1;
  const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
  if (threadIdx.x == 0) carry_s = 0;
  __syncthreads();
  for (int t0 = 0; t0 < m; t0 += kScanTile) {
    const int base = t0 + threadIdx.x * kScanPerThread;
    int v[kScanPerThread], s = 0;
#pragma unroll
    for (int k = 0; k < kScanPerThread; ++k) {
      v[k] = (base + k < m) ? in[base + k] : 0;
      s += v[k];
    }
    int inc = s;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
      const int t = __shfl_up_sync(0xffffffffu, inc, o);
      if (lane >= o) inc += t;
    }
    if (lane == 31) wsum[wid] = inc;
    __syncthreads();
    if (wid == 0) {
      int t = wsum[lane];
#pragma unroll
      for (int o = 1; o < 32; o <<= 1) {
        const int u = __shfl_up_sync(0xffffffffu, t, o);
        if (lane >= o) t += u;
      }
      wsum[lane] = t;
    }
    __syncthreads();
    int excl = carry_s + inc - s + (wid > 0 ? wsum[wid - 1] : 0);
#pragma unroll
    for (int k = 0; k < kScanPerThread; ++k) {
      if (base + k < m) out[base + k] = excl;
      excl += v[k];
    }
    __syncthreads();
    if (threadIdx.x == kScanThreads - 1) carry_s = excl;
    __syncthreads();
  }
  if (threadIdx.x == 0) out[m] = n_total;
}

__global__ void k_scan_add(int m, int* __restrict__ out, const int* __restrict__ totals, int n_total) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i < m) out[i] += totals[i / kScanTile];
  if (i == 0) out[m] = n_total;
}

// pass 2: scatter original indices into their cell's segment (slot = arrival rank from pass 1)
__global__ void k_scatter(int n, const int* __restrict__ pcell, const int* __restrict__ gcell,
                          const int* __restrict__ pstart, const int* __restrict__ gstart,
                          const int* __restrict__ pslot, const int* __restrict__ gslot, int* __restrict__ porder,
                          int* __restrict__ gorder) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  porder[pstart[pcell[i]] + pslot[i]] = i;
  gorder[gstart[gcell[i]] + gslot[i]] = i;
}

// pass 3: canonical order inside each cell (ascending original index). One thread per cell with an
// insertion sort for the usual few particles per cell; a cell with more than kSortWarpMin particles
// (clustered input: the single thread would do O(k^2) dependent global loads and stores) is then
// rank-sorted by its whole warp through `tmp` (the arrival slots of pass 2, dead by now): every
// element counts the smaller ones (the indices are distinct) and goes to that position.
// (blockIdx.y = 0: the pair bins, 1: the grid cells)
constexpr int kSortWarpMin = 24;
__global__ void k_sort_cells(int ncell0, const int* __restrict__ start0, int* __restrict__ order0, int* __restrict__ tmp0,
                             int ncell1, const int* __restrict__ start1, int* __restrict__ order1, int* __restrict__ tmp1) {
  const int ncell = blockIdx.y == 0 ? ncell0 : ncell1;
  const int* __restrict__ start = blockIdx.y == 0 ? start0 : start1;
  int* __restrict__ order = blockIdx.y == 0 ? order0 : order1;
  int* __restrict__ tmp = blockIdx.y == 0 ? tmp0 : tmp1;
  const int c = blockIdx.x * blockDim.x + threadIdx.x;
  const int lane = threadIdx.x & 31;
  int s = 0, e = 0;
  if (c < ncell) { s = start[c]; e = start[c + 1]; }
  if (e - s <= kSortWarpMin) {
    for (int i = s + 1; i < e; ++i) {
      const int v = order[i];
      int j = i - 1;
      while (j >= s && order[j] > v) { order[j + 1] = order[j]; --j; }
      order[j + 1] = v;
    }
  }
  unsigned big = __ballot_sync(0xffffffffu, e - s > kSortWarpMin);
  while (big) {
    const int L = __ffs(big) - 1;
    big &= big - 1;
    const int bs = __shfl_sync(0xffffffffu, s, L), be = __shfl_sync(0xffffffffu, e, L);
    for (int i = bs + lane; i < be; i += 32) {
      const int v = order[i];
      int rank = 0;
      for (int j = bs; j < be; ++j) rank += order[j] < v;
      tmp[bs + rank] = v;
    }
    __syncwarp();
    for (int i = bs + lane; i < be; i += 32) order[i] = tmp[i];
    __syncwarp();
  }
}

// pass 4: sorted records. Pair order: cell-relative coordinates + charge (fp32-safe: magnitudes
// stay below one cell edge). Grid order: fractions t in [0,1] of the particle's grid cell + charge.
template <typename T>
__global__ void k_build_records(int n, const T* __restrict__ pos, const T* __restrict__ q, BinGeom g,
                                const int* __restrict__ porder, const int* __restrict__ pcell,
                                const int* __restrict__ gorder, const int* __restrict__ gcell,
                                typename Vec4<T>::type* __restrict__ prec,
                                typename Vec4<T>::type* __restrict__ grec, int* __restrict__ gcell_sorted,
                                int* __restrict__ pbinx) {
  const int k = blockIdx.x * blockDim.x + threadIdx.x;
  if (k >= n) return;
  {
    const int i = porder[k];
    int c = pcell[i];
    const int nbx = g.nc[0] << g.sxs;
    const int bx = c % nbx; c /= nbx;                  // sub-bin along x
    const int cx = bx >> g.sxs;
    const int cy = c % g.nc[1], cz = c / g.nc[1];
    const int cc[3] = {cx, cy, cz};
    T r[3];
#pragma unroll
    for (int ax = 0; ax < 3; ++ax) {
      double x = (double)pos[3 * (size_t)i + ax];
      if (!isfinite(x)) x = 0.0;
      if (!g.periodic[ax]) x = fmin(fmax(x, 0.0), g.box[ax]);
      x = wrap_coord(x, g.box[ax], g.periodic[ax]);
      r[ax] = (T)(x - cc[ax] * g.cell_edge[ax]);
    }
    prec[k] = make_vec4<T>(r[0], r[1], r[2], q[i]);
    pbinx[k] = bx;
  }
  {
    const int i = gorder[k];
    const int cid = gcell[i];
    int c = cid;
    const int cx = c % g.ng[0]; c /= g.ng[0];
    const int cy = c % g.ng[1], cz = c / g.ng[1];
    const int cc[3] = {cx, cy, cz};
    T t[3];
#pragma unroll
    for (int ax = 0; ax < 3; ++ax) {
      double x = (double)pos[3 * (size_t)i + ax];
      if (!isfinite(x)) x = 0.0;
      if (!g.periodic[ax]) x = fmin(fmax(x, 0.0), g.box[ax]);
      x = wrap_coord(x, g.box[ax], g.periodic[ax]);
      t[ax] = (T)(x / g.h1[ax] - (double)cc[ax]);
    }
    grec[k] = make_vec4<T>(t[0], t[1], t[2], q[i]);
    gcell_sorted[k] = cid;
  }
}

}  // namespace msm
