// gridops_stream.cuh -- S4 restriction and S7 prolongation (Eq. 19; mask J of P:122-125
// Eq. 13) for grids that do not fit the L2: each kernel applies the three one-axis passes of the
// separable operator in ONE sweep, so that the fine grid crosses HBM once (restriction:
// read G_l, write G_l / 8; prolongation: read G_l / 8 + G_l, write G_l) instead of once per axis.
//
// A block owns a column of the grid in x-y and marches along z:
//  * x is done in registers on 16-byte chunks (the neighbours' values come by warp shuffle, resp.
//    by a few extra loads of the small coarse array),
//  * y goes through one shared-memory plane,
//  * z is a rolling window of register accumulators (a fine plane feeds <= p/2 + 1 coarse planes).
// Loads of the next plane pair are issued before the current one is processed.
//
// Requirements (checked by the host, which otherwise uses the one-axis kernels of gridops.cuh and
// k_prolong3): x periodic with lo = 0 and M_x a multiple of the chunk; y and z periodic or open.
#pragma once
#include "gridops.cuh"
#include "gridops_fused.cuh"

namespace msm {

constexpr int kStreamThreads = 256;

template <typename T> struct VecT;
template <> struct VecT<float> { using type = float4; static constexpr int VE = 4; };
template <> struct VecT<double> { using type = double2; static constexpr int VE = 2; };

__device__ __forceinline__ void unpack(const float4& v, float (&a)[4]) { a[0] = v.x; a[1] = v.y; a[2] = v.z; a[3] = v.w; }
__device__ __forceinline__ void unpack(const double2& v, double (&a)[2]) { a[0] = v.x; a[1] = v.y; }
__device__ __forceinline__ float4 pack_vec(float4*, const float* a) { return make_float4(a[0], a[1], a[2], a[3]); }
__device__ __forceinline__ double2 pack_vec(double2*, const double* a) { return make_double2(a[0], a[1]); }
__device__ __forceinline__ float4 zero_vec(float4*) { return make_float4(0.f, 0.f, 0.f, 0.f); }
__device__ __forceinline__ double2 zero_vec(double2*) { return make_double2(0.0, 0.0); }

struct StreamGeom {
  Grid3 f, c;        // fine and coarse arrays (dims, node index of element 0)
  int per_y, per_z;
  int ntx;           // tiles along x
  int zseg;          // restriction: coarse planes per block; prolongation: fine plane pairs per block
};

// Offsets of the coarse planes that one pair of fine planes (nodes 2a, 2a + 1) exchanges with:
// even node 2a and tap n = 2j <-> coarse a - j, |2j| <= HW; odd node 2a + 1 and tap n = 2j + 1 <->
// coarse a - j, |2j + 1| <= HW. Window of offsets [kOffMin, kOffMax].
template <int HW> struct PairWindow {
  static constexpr int JE = HW / 2, JOLO = -((HW + 1) / 2), JOHI = (HW - 1) / 2;
  static constexpr int OFFMIN = -(JE > JOHI ? JE : JOHI), OFFMAX = (JE > -JOLO ? JE : -JOLO);
  static constexpr int KA = OFFMAX - OFFMIN + 1;
  // tap index (into J.c, offset HW) of window slot d for the even / odd plane, or -1
  __host__ __device__ static constexpr int even_tap(int d) { return (d + OFFMIN >= -JE && d + OFFMIN <= JE) ? HW - 2 * (d + OFFMIN) : -1; }
  __host__ __device__ static constexpr int odd_tap(int d) {
    return (-(d + OFFMIN) >= JOLO && -(d + OFFMIN) <= JOHI) ? HW - 2 * (d + OFFMIN) + 1 : -1;
  }
};

__host__ __device__ constexpr int cfloor_div(int o, int v) { return o >= 0 ? o / v : -((-o + v - 1) / v); }

// array index of node `node` on an axis (periodic wrap, or -1 outside an open array)
__device__ __forceinline__ int axis_index(int node, int lo, int M, int periodic) {
  const int i = node - lo;
  if (periodic) return imod(i, M);
  return (i >= 0 && i < M) ? i : -1;
}

// ---------------------------------------------------------------------------------------------
// Restriction: out[m] = sum_n J J J in[2 m + n]
// Tile: CX = (32 - 2 HC) VE / 2 coarse x (a warp row of 32 chunks, HC halo chunks each side),
// CY coarse y; gridDim = (x tiles * y tiles, z segments).
template <typename T, int NJ, int CY>
__global__ void __launch_bounds__(kStreamThreads)
k_restrict_stream(StreamGeom g, AxisTaps<T> J, const T* __restrict__ in, T* __restrict__ out) {
  using V = typename VecT<T>::type;
  using W = PairWindow<NJ / 2>;
  constexpr int VE = VecT<T>::VE, HW = NJ / 2, HC = (HW + VE - 1) / VE;
  constexpr int CPL = VE / 2;                    // coarse outputs per chunk
  constexpr int CX = (32 - 2 * HC) * CPL;
  constexpr int CXP = 32 * CPL;                  // row length in shared memory
  constexpr int NG = kStreamThreads / CXP;       // thread groups along y
  constexpr int CYT = CY / NG;                   // coarse y per thread
  constexpr int NR = 2 * CY + 2 * HW - 1;        // fine rows of one plane
  constexpr int NOPS = (2 * NR + 7) / 8;         // rows per warp and plane pair
  constexpr int KA = W::KA;
  static_assert(CY % NG == 0, "tile shape");
  __shared__ __align__(16) T X[2][NR][CXP];

  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int tx = blockIdx.x % g.ntx, ty = blockIdx.x / g.ntx;
  const int cx0 = tx * CX, cy0 = ty * CY;
  const int cz0 = blockIdx.y * g.zseg, nz = min(g.zseg, g.c.M[2] - cz0);
  const int ncx = min(CX, g.c.M[0] - cx0);
  const size_t fplane = (size_t)g.f.M[0] * g.f.M[1];

  // this lane's chunk: fine offsets xo .. xo + VE - 1 from 2 cx0
  const int xo = (lane - HC) * VE;
  const bool xneed = xo <= 2 * (ncx - 1) + HW && xo + VE - 1 >= -HW;
  const int fx = imod(2 * cx0 + xo, g.f.M[0]);
  int rowoff[NOPS];
#pragma unroll
  for (int i = 0; i < NOPS; ++i) {
    const int r = warp + 8 * i, row = r >= NR ? r - NR : r;
    const int fy = axis_index(2 * (cy0 + g.c.lo[1]) - HW + row, g.f.lo[1], g.f.M[1], g.per_y);
    rowoff[i] = (r < 2 * NR && xneed && fy >= 0) ? fy * g.f.M[0] + fx : -1;
  }
  auto load_pair = [&](int k, V (&buf)[NOPS]) {
    const int e = 2 * (cz0 + g.c.lo[2] + k);
    const int fe = axis_index(e, g.f.lo[2], g.f.M[2], g.per_z), fo = axis_index(e + 1, g.f.lo[2], g.f.M[2], g.per_z);
#pragma unroll
    for (int i = 0; i < NOPS; ++i) {
      const int fz = (warp + 8 * i >= NR) ? fo : fe;
      buf[i] = (rowoff[i] >= 0 && fz >= 0) ? __ldg(reinterpret_cast<const V*>(in + (size_t)fz * fplane + rowoff[i]))
                                           : zero_vec((V*)nullptr);
    }
  };

  const int cxl = tid % CXP, grp = tid / CXP;
  T acc[CYT][KA];
#pragma unroll
  for (int q = 0; q < CYT; ++q)
#pragma unroll
    for (int d = 0; d < KA; ++d) acc[q][d] = 0;

  const int kfirst = -W::OFFMAX, klast = nz - 1 - W::OFFMIN;
  V cur[NOPS], nxt[NOPS];
  load_pair(kfirst, cur);
  for (int k = kfirst; k <= klast; ++k) {
    if (k < klast) load_pair(k + 1, nxt);
    // x: every lane restricts its chunk; the window comes from the neighbouring lanes
#pragma unroll
    for (int i = 0; i < NOPS; ++i) {
      const int r = warp + 8 * i;
      if (r < 2 * NR) {
        T v[VE];
        unpack(cur[i], v);
        T w[VE - 1 + 2 * HW];                      // fine offsets -HW .. VE - 2 + HW of the chunk
#pragma unroll
        for (int o = -HW; o <= VE - 2 + HW; ++o) {
          const int d = cfloor_div(o, VE), e = o - d * VE;
          w[o + HW] = d == 0 ? v[e] : __shfl_sync(0xffffffffu, v[e], lane + d);
        }
        if (lane >= HC && lane < 32 - HC) {
          T* dst = &X[r >= NR][r >= NR ? r - NR : r][(lane - HC) * CPL];
#pragma unroll
          for (int q = 0; q < CPL; ++q) {
            T s = 0;
#pragma unroll
            for (int n = 0; n < NJ; ++n) s = fma(J.c[n], w[2 * q + n], s);
            dst[q] = s;
          }
        }
      }
    }
    __syncthreads();
    // y from shared memory, z into the rolling accumulators
    if (cxl < ncx) {
      T yv[2][CYT];
#pragma unroll
      for (int pl = 0; pl < 2; ++pl) {
        T rows[2 * CYT + 2 * HW - 1];
#pragma unroll
        for (int j = 0; j < 2 * CYT + 2 * HW - 1; ++j) rows[j] = X[pl][2 * grp * CYT + j][cxl];
#pragma unroll
        for (int q = 0; q < CYT; ++q) {
          T s = 0;
#pragma unroll
          for (int n = 0; n < NJ; ++n) s = fma(J.c[n], rows[2 * q + n], s);
          yv[pl][q] = s;
        }
      }
      const int cz = k + W::OFFMIN;
#pragma unroll
      for (int q = 0; q < CYT; ++q) {
#pragma unroll
        for (int d = 0; d < KA; ++d) {
          if (W::even_tap(d) >= 0) acc[q][d] = fma(J.c[W::even_tap(d) >= 0 ? W::even_tap(d) : 0], yv[0][q], acc[q][d]);
          if (W::odd_tap(d) >= 0) acc[q][d] = fma(J.c[W::odd_tap(d) >= 0 ? W::odd_tap(d) : 0], yv[1][q], acc[q][d]);
        }
        const int cy = cy0 + grp * CYT + q;
        if (cz >= 0 && cy < g.c.M[1])
          out[((size_t)(cz0 + cz) * g.c.M[1] + cy) * g.c.M[0] + cx0 + cxl] = acc[q][0];
#pragma unroll
        for (int d = 0; d + 1 < KA; ++d) acc[q][d] = acc[q][d + 1];
        acc[q][KA - 1] = 0;
      }
    }
    __syncthreads();
#pragma unroll
    for (int i = 0; i < NOPS; ++i) cur[i] = nxt[i];
  }
}

template <typename T, int NJ> constexpr int restrict_stream_cx() {
  return (32 - 2 * ((NJ / 2 + VecT<T>::VE - 1) / VecT<T>::VE)) * VecT<T>::VE / 2;
}

// ---------------------------------------------------------------------------------------------
// Prolongation + accumulate: E[i] += sum_m J J J ec[m], 2 m + n = i on every axis.
// Tile: 64 VE fine x (a warp row of 32 coarse chunks; the coarse neighbours of a chunk are loaded
// directly -- the coarse array is 1/8 of the traffic), 8 fine y (4 node pairs); the block marches
// over the coarse planes, keeps the x-y-prolonged planes of the window in registers and emits one
// pair of fine planes (nodes 2a, 2a + 1) per step. In the y/z phase a thread owns one 16-byte
// vector of fine x and one node pair in y: four vector loads and stores of E per step.
template <typename T, int NJ>
__global__ void __launch_bounds__(kStreamThreads, sizeof(T) == 4 ? 3 : 2)
k_prolong_stream(StreamGeom g, AxisTaps<T> J, const T* __restrict__ ec, T* __restrict__ E) {
  using V = typename VecT<T>::type;
  using W = PairWindow<NJ / 2>;
  constexpr int VE = VecT<T>::VE;
  constexpr int KA = W::KA, OFFMIN = W::OFFMIN, OFFMAX = W::OFFMAX;
  constexpr int FXP = 64 * VE;                   // fine x per tile
  constexpr int BY = kStreamThreads / 64;        // y node pairs per tile (one per thread group)
  constexpr int NRC = BY + KA - 1;               // coarse rows per plane
  static_assert(NRC <= 8, "one row per warp");
  __shared__ __align__(16) T XP[NRC][FXP];

  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int tx = blockIdx.x % g.ntx, ty = blockIdx.x / g.ntx;
  // x: coarse chunk of this lane (coarse array index = coarse node, lo = 0, periodic)
  const int mcx = g.c.M[0];
  const int c0 = tx * 32 * VE + lane * VE;
  const bool xact = c0 < mcx;
  // y: node pairs b0 .. b0 + BY - 1 (fine nodes 2b, 2b + 1); the first pair holds the array's first node
  const int b0 = (g.f.lo[1] >> 1) + ty * BY;
  // z: node pairs a0 .. a0 + na - 1
  const int alast = (g.f.lo[2] + g.f.M[2] - 1) >> 1;
  const int a0 = (g.f.lo[2] >> 1) + blockIdx.y * g.zseg, na = min(g.zseg, alast - a0 + 1);
  const size_t cplane = (size_t)g.c.M[0] * g.c.M[1], fplane = (size_t)g.f.M[0] * g.f.M[1];

  // coarse row of this warp: node b0 + OFFMIN + warp
  const int crow = warp < NRC ? axis_index(b0 + OFFMIN + warp, g.c.lo[1], g.c.M[1], g.per_y) : -1;
  // coarse x offsets OFFMIN .. VE - 1 + OFFMAX around the chunk, wrapped
  int cxi[VE + KA - 1];
#pragma unroll
  for (int j = 0; j < VE + KA - 1; ++j) cxi[j] = imod(c0 + OFFMIN + j, mcx);

  // the thread's fine points in the y/z phase: x vector xg, node pair yg
  const int xg = tid & 63, yg = tid >> 6;
  const int fx = tx * FXP + xg * VE;
  const bool pact = fx < g.f.M[0];
  int rowoff[2];                                 // offset of (fine y, fx) inside a plane, or -1
#pragma unroll
  for (int s = 0; s < 2; ++s) {
    const int i = 2 * (b0 + yg) + s - g.f.lo[1];
    rowoff[s] = (pact && i >= 0 && i < g.f.M[1]) ? i * g.f.M[0] + fx : -1;
  }

  T Pw[KA][2][VE];
#pragma unroll
  for (int d = 0; d < KA; ++d)
#pragma unroll
    for (int s = 0; s < 2; ++s)
#pragma unroll
      for (int e = 0; e < VE; ++e) Pw[d][s][e] = 0;

  auto load_row = [&](int m, T (&buf)[VE + KA - 1]) {     // coarse plane node m, this warp's row
    const int cz = axis_index(m, g.c.lo[2], g.c.M[2], g.per_z);
    const bool ok = cz >= 0 && crow >= 0 && xact;
    const T* row = ec + (size_t)(ok ? cz : 0) * cplane + (size_t)(ok ? crow : 0) * mcx;
#pragma unroll
    for (int j = 0; j < VE + KA - 1; ++j) buf[j] = ok ? __ldg(row + cxi[j]) : (T)0;
  };

  // planes m = a0 + OFFMIN .. a0 + na - 1 + OFFMAX; after plane a + OFFMAX the pair a is complete
  const int mfirst = a0 + OFFMIN, mlast = a0 + na - 1 + OFFMAX;
  T cur[VE + KA - 1], nxt[VE + KA - 1];
  load_row(mfirst, cur);
  for (int m = mfirst; m <= mlast; ++m) {
    if (m < mlast) load_row(m + 1, nxt);
    const int a = m - OFFMAX;                            // pair emitted in this step (if >= a0)
    // prefetch the fine values of that pair
    V eold[2][2];
    T* eptr[2][2];
#pragma unroll
    for (int sz = 0; sz < 2; ++sz) {
      const int i = 2 * a + sz - g.f.lo[2];
      const bool zok = a >= a0 && i >= 0 && i < g.f.M[2];
#pragma unroll
      for (int sy = 0; sy < 2; ++sy) {
        eptr[sz][sy] = (zok && rowoff[sy] >= 0) ? E + (size_t)i * fplane + rowoff[sy] : nullptr;
        eold[sz][sy] = eptr[sz][sy] ? *reinterpret_cast<const V*>(eptr[sz][sy]) : zero_vec((V*)nullptr);
      }
    }
    // x: fine 2 c + s <- sum over window slots of the coarse values around c
    if (warp < NRC) {
      T fine[2 * VE];
#pragma unroll
      for (int e = 0; e < VE; ++e) {
        T se = 0, so = 0;
#pragma unroll
        for (int d = 0; d < KA; ++d) {
          if (W::even_tap(d) >= 0) se = fma(J.c[W::even_tap(d) >= 0 ? W::even_tap(d) : 0], cur[e + d], se);
          if (W::odd_tap(d) >= 0) so = fma(J.c[W::odd_tap(d) >= 0 ? W::odd_tap(d) : 0], cur[e + d], so);
        }
        fine[2 * e] = se; fine[2 * e + 1] = so;
      }
      V* dst = reinterpret_cast<V*>(&XP[warp][lane * 2 * VE]);
      dst[0] = pack_vec((V*)nullptr, &fine[0]);
      dst[1] = pack_vec((V*)nullptr, &fine[VE]);
    }
    __syncthreads();
    // y: fine y (pair yg, parity s) <- rows yg + d; the result is the newest plane of the window
    {
      T rows[KA][VE];
#pragma unroll
      for (int d = 0; d < KA; ++d) unpack(*reinterpret_cast<const V*>(&XP[yg + d][xg * VE]), rows[d]);
#pragma unroll
      for (int s = 0; s < 2; ++s)
#pragma unroll
        for (int e = 0; e < VE; ++e) {
          T v = 0;
#pragma unroll
          for (int d = 0; d < KA; ++d) {
            const int tap = s ? W::odd_tap(d) : W::even_tap(d);
            if (tap >= 0) v = fma(J.c[tap >= 0 ? tap : 0], rows[d][e], v);
          }
          Pw[KA - 1][s][e] = v;
        }
    }
    // z: emit the pair a
#pragma unroll
    for (int sz = 0; sz < 2; ++sz)
#pragma unroll
      for (int sy = 0; sy < 2; ++sy) {
        if (eptr[sz][sy]) {
          T o[VE];
          unpack(eold[sz][sy], o);
#pragma unroll
          for (int e = 0; e < VE; ++e) {
            T v = 0;
#pragma unroll
            for (int d = 0; d < KA; ++d) {
              const int tap = sz ? W::odd_tap(d) : W::even_tap(d);
              if (tap >= 0) v = fma(J.c[tap >= 0 ? tap : 0], Pw[d][sy][e], v);
            }
            o[e] += v;
          }
          *reinterpret_cast<V*>(eptr[sz][sy]) = pack_vec((V*)nullptr, o);
        }
      }
#pragma unroll
    for (int d = 0; d + 1 < KA; ++d)
#pragma unroll
      for (int s = 0; s < 2; ++s)
#pragma unroll
        for (int e = 0; e < VE; ++e) Pw[d][s][e] = Pw[d + 1][s][e];
    __syncthreads();
#pragma unroll
    for (int j = 0; j < VE + KA - 1; ++j) cur[j] = nxt[j];
  }
}

}  // namespace msm
