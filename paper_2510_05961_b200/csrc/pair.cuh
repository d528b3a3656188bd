// pair.cuh -- S2: short-range pair sum of k_0(r) = 1/r - gamma(r/a)/a over a cell list
// (Eq. 5 first term; Eq. 21 l = 0), with forces and the pair virial.
//
// Cells have edge >= a/2, so the neighbourhood is 5x5x5 cells. An i-tile is up to 32 consecutive
// sorted particles of one x-row of cells (lane = particle i); for each of the 25 neighbouring
// rows the j-particles of cells [cx_first-2, cx_last+2] are contiguous in the sorted order and
// are staged through shared memory 32 at a time, in a frame relative to the tile's first cell
// (cell-relative coordinates keep fp32 differences accurate). -k_0'(r)/r = 1/r^3 + (2/a^3) g'(s),
// s = r^2/a^2 - 1, so one rsqrt per pair inside the cutoff is the only special function.
#pragma once
#include "device_common.cuh"

namespace msm {

template <typename T> struct PairParams {
  int nc[3];
  int periodic[3];
  int omin[3], omax[3];   // neighbour cell offsets per axis (y, z use these; x: +-2 around the tile)
  int minimg[3];          // periodic axis with fewer than 5 cells: explicit minimum image
  T edge[3];
  T box[3], inv_box[3];
  T a2, inv_a, inv_a2, two_inv_a3;
  T c[8];                 // binom(-1/2, k)
  int p;
};

constexpr int kPairWarps = 4;

template <typename T, int P, bool VIRIAL>
__global__ void __launch_bounds__(kPairWarps * 32)
k_pair(PairParams<T> prm, const int* __restrict__ pstart, const typename Vec4<T>::type* __restrict__ prec,
       const int* __restrict__ pcellx, const int* __restrict__ porder, T* __restrict__ Fsr,
       T* __restrict__ Vsr, double* __restrict__ wpart) {
  using V4 = typename Vec4<T>::type;
  __shared__ V4 sj[kPairWarps][32];
  __shared__ double red[kPairWarps];
  const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
  const int row = blockIdx.x;                       // (cy, cz)
  const int cy = row % prm.nc[1], cz = row / prm.nc[1];
  const int ncx = prm.nc[0];
  const int row_s = pstart[row * ncx], row_e = pstart[(row + 1) * ncx];
  const int ntile = (row_e - row_s + 31) >> 5;
  double W[6] = {0, 0, 0, 0, 0, 0};

  for (int tile = wid; tile < ntile; tile += kPairWarps) {
    const int ki = row_s + tile * 32 + lane;
    const bool iv = ki < row_e;
    V4 ri = make_vec4<T>(0, 0, 0, 0);
    int cxi = 0;
    if (iv) { ri = ldg4(prec + ki); cxi = pcellx[ki]; }
    const int last = min(31, row_e - 1 - (row_s + tile * 32));
    const int cxf = __shfl_sync(0xffffffffu, cxi, 0), cxl = __shfl_sync(0xffffffffu, cxi, last);
    const T xi = ri.x + (T)(cxi - cxf) * prm.edge[0], yi = ri.y, zi = ri.z;
    // x-range of neighbour cells in unwrapped cell coordinates
    int xa = cxf - 2, xb = cxl + 2;
    bool mix = prm.minimg[0] != 0;
    if (!prm.periodic[0]) { xa = max(xa, 0); xb = min(xb, ncx - 1); }
    else if (xb - xa + 1 > ncx) { xa = 0; xb = ncx - 1; mix = true; }   // every cell once + min. image
    T ax = 0, ay = 0, az = 0, av = 0;
    T w0 = 0, w1 = 0, w2 = 0, w3 = 0, w4 = 0, w5 = 0;

    for (int dz = prm.omin[2]; dz <= prm.omax[2]; ++dz) {
      int czj = cz + dz;
      if (prm.periodic[2]) czj = imod(czj, prm.nc[2]);
      else if (czj < 0 || czj >= prm.nc[2]) continue;
      for (int dy = prm.omin[1]; dy <= prm.omax[1]; ++dy) {
        int cyj = cy + dy;
        if (prm.periodic[1]) cyj = imod(cyj, prm.nc[1]);
        else if (cyj < 0 || cyj >= prm.nc[1]) continue;
        const int rowbase = (czj * prm.nc[1] + cyj) * ncx;
        const T yoff = (T)dy * prm.edge[1], zoff = (T)dz * prm.edge[2];
        // up to three contiguous segments: wrapped-left, main, wrapped-right
        for (int seg = 0; seg < 3; ++seg) {
          int ca, cb, shift;   // stored cell range and unwrapped = stored + shift
          if (seg == 0) { if (xa >= 0) continue; ca = xa + ncx; cb = min(xb, -1) + ncx; shift = -ncx; }
          else if (seg == 1) { ca = max(xa, 0); cb = min(xb, ncx - 1); shift = 0; if (ca > cb) continue; }
          else { if (xb < ncx) continue; ca = max(xa, ncx) - ncx; cb = xb - ncx; shift = ncx; }
          const int js = pstart[rowbase + ca], je = pstart[rowbase + cb + 1];
          for (int j0 = js; j0 < je; j0 += 32) {
            const int kj = j0 + lane;
            V4 rj = make_vec4<T>((T)1e30, 0, 0, 0);
            if (kj < je) {
              rj = ldg4(prec + kj);
              rj.x += (T)(pcellx[kj] + shift - cxf) * prm.edge[0];
              rj.y += yoff;
              rj.z += zoff;
            }
            __syncwarp();
            sj[wid][lane] = rj;
            __syncwarp();
            const int cnt = min(32, je - j0);
            for (int kk = 0; kk < cnt; ++kk) {
              const V4 pj = sj[wid][kk];
              T dx = xi - pj.x, dy_ = yi - pj.y, dz_ = zi - pj.z;
              if (mix) dx -= prm.box[0] * rint(dx * prm.inv_box[0]);
              if (prm.minimg[1]) dy_ -= prm.box[1] * rint(dy_ * prm.inv_box[1]);
              if (prm.minimg[2]) dz_ -= prm.box[2] * rint(dz_ * prm.inv_box[2]);
              const T r2 = fma(dx, dx, fma(dy_, dy_, dz_ * dz_));
              if (r2 < prm.a2 && (j0 + kk) != ki && iv) {
                const T rinv = rsqrt_t<T>(r2);
                const T s = fma(r2, prm.inv_a2, (T)-1);
                T g = prm.c[P - 1], dg = (T)(P - 1) * prm.c[P - 1];
#pragma unroll
                for (int k = P - 2; k >= 0; --k) g = fma(g, s, prm.c[k]);
#pragma unroll
                for (int k = P - 2; k >= 1; --k) dg = fma(dg, s, (T)k * prm.c[k]);
                const T qj = pj.w;
                av = fma(qj, rinv - g * prm.inv_a, av);
                const T fs = qj * fma(prm.two_inv_a3, dg, rinv * rinv * rinv);
                ax = fma(fs, dx, ax); ay = fma(fs, dy_, ay); az = fma(fs, dz_, az);
                if (VIRIAL) {
                  const T fx = fs * dx, fy = fs * dy_, fz = fs * dz_;
                  w0 = fma(fx, dx, w0); w1 = fma(fy, dy_, w1); w2 = fma(fz, dz_, w2);
                  w3 = fma(fx, dy_, w3); w4 = fma(fx, dz_, w4); w5 = fma(fy, dz_, w5);
                }
              }
            }
          }
        }
      }
    }
    if (iv) {
      const int orig = porder[ki];
      const T qi = ri.w;
      Fsr[3 * (size_t)orig + 0] = qi * ax;
      Fsr[3 * (size_t)orig + 1] = qi * ay;
      Fsr[3 * (size_t)orig + 2] = qi * az;
      Vsr[orig] = av;
      if (VIRIAL) {
        const double hq = 0.5 * (double)qi;   // every pair is visited from both ends
        W[0] += hq * (double)w0; W[1] += hq * (double)w1; W[2] += hq * (double)w2;
        W[3] += hq * (double)w3; W[4] += hq * (double)w4; W[5] += hq * (double)w5;
      }
    }
  }
  if (VIRIAL) {
#pragma unroll
    for (int k = 0; k < 6; ++k) {
      const double r = block_reduce_sum<kPairWarps * 32>(W[k], red);
      if (threadIdx.x == 0) wpart[(size_t)blockIdx.x * 6 + k] = r;
    }
  }
}

}  // namespace msm
