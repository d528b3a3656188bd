// pair.cuh -- S2: short-range pair sum of k_0(r) = 1/r - gamma(r/a)/a over a cell list
// (Eq. 5 first term; Eq. 21 l = 0), with forces and the pair virial.
//
// Cells have edge >= a/2, so the neighbourhood is 5x5x5 cells. An i-tile is up to 32 consecutive
// sorted particles of one x-row of cells (lane = particle i); for each of the 25 neighbouring
// rows the j-particles of cells [cx_first-2, cx_last+2] are contiguous in the sorted order and
// are staged through shared memory kPairBatch at a time, in a frame relative to the tile's first
// cell (cell-relative coordinates keep fp32 differences accurate).
//
// Only 17-27 % of the candidates are inside the cutoff, and a warp that branches per candidate
// pays the full interaction whenever ANY lane hits. So the candidates of consecutive neighbour
// rows are gathered into batches and each batch is processed in two phases:
//   scan  -- every lane tests every candidate (broadcast shared loads, 3 subtractions, 3 multiply-
//            adds, one compare, in fp32 on both precisions, two candidates per packed f32x2
//            instruction) and appends the index of
//            each hit to its private list in shared memory; in fp64 mode the fp32 test uses a
//            widened cutoff and the exact test is repeated in the drain;
//   drain -- round r evaluates, on every lane that has one, the r-th hit of its list in full
//            precision. Rounds = the largest hit count of any lane in the batch, so the expensive
//            path runs at 60-70 % lane utilisation instead of ~20 %, with ~6 instructions of
//            bookkeeping per round.
// Small systems have too few tiles to fill the GPU: the dz planes of the neighbourhood are then
// dealt to up to kPairMaxSplit blocks (blockIdx.z) whose partial sums k_interpolate adds in order.
// Every lane visits its hits in ascending candidate order, so the sums have a fixed order
// (deterministic). -k_0'(r)/r = 1/r^3 + (2/a^3) g'(s), s = r^2/a^2 - 1: one rsqrt per pair is the
// only special function.
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
  float a2_scan;          // cutoff^2 of the fp32 scan (widened by rounding slack in fp64 mode)
  T c[8];                 // binom(-1/2, k)
  int p;
  int nsplit;             // the dz planes of the neighbourhood are dealt to nsplit blocks (blockIdx.z)
  size_t part_stride;     // elements between the per-split partial outputs (capacity)
};

constexpr int kPairWarps = 1;
constexpr int kPairMaxSplit = 5;

// Shared-memory staging of one warp. The fp32 records are interleaved in pairs of candidates,
// (x0 x1 | y0 y1 | z0 z1 | q0 q1), so that the scan tests two candidates per packed instruction:
// candidate k sits at float offset pair_slot(k) + {0, 2, 4, 6}.
__device__ __forceinline__ int pair_slot(int k) { return (k >> 1) * 8 + (k & 1); }
template <typename T> struct PairStage;
template <> struct PairStage<float> {
  static constexpr int kBatch = 160;          // candidates per batch (multiple of 32)
  __align__(16) float f[kBatch * 4];          // scan and drain read the same records
  unsigned char list[kBatch * 32];            // hit r of lane l at [r * 32 + l]
  __device__ __forceinline__ void put(int k, float4 r) {
    float* q = f + pair_slot(k);
    q[0] = r.x; q[2] = r.y; q[4] = r.z; q[6] = r.w;
  }
  __device__ __forceinline__ float4 full(int k) const {
    const float* q = f + pair_slot(k);
    return make_float4(q[0], q[2], q[4], q[6]);
  }
};
template <> struct PairStage<double> {
  static constexpr int kBatch = 96;
  __align__(16) float f[kBatch * 4];          // fp32 copy for the scan
  double4 d[kBatch];                          // full precision for the drain
  unsigned char list[kBatch * 32];
  __device__ __forceinline__ void put(int k, double4 r) {
    d[k] = r;
    float* q = f + pair_slot(k);
    q[0] = (float)r.x; q[2] = (float)r.y; q[4] = (float)r.z;
  }
  __device__ __forceinline__ double4 full(int k) const { return d[k]; }
};

__device__ __forceinline__ float rsqrt_fast(float x) {
  float y;
  asm("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
  return y;
}
// fp64: fp32 hardware seed (relative error 2^-22.9) + two Newton steps y <- y (3/2 - x/2 y^2), each of
// which squares the error: ~1e-13, then below the fp64 rounding unit. x is a squared distance inside
// the cutoff (far from the fp32 range limits).
__device__ __forceinline__ double rsqrt_fast(double x) {
  double y = (double)rsqrt_fast((float)x);
  const double hx = 0.5 * x;
  y = y * fma(-hx, y * y, 1.5);
  y = y * fma(-hx, y * y, 1.5);
  return y;
}

template <typename T, int P, bool VIRIAL, bool MI>
__global__ void __launch_bounds__(kPairWarps * 32)
k_pair(PairParams<T> prm, const int* __restrict__ pstart, const typename Vec4<T>::type* __restrict__ prec,
       const int* __restrict__ pcellx, const int* __restrict__ porder, T* __restrict__ Fsr,
       T* __restrict__ Vsr, double* __restrict__ wpart) {
  using V4 = typename Vec4<T>::type;
  constexpr int B = PairStage<T>::kBatch;
  __shared__ PairStage<T> stage[kPairWarps];
  const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
  PairStage<T>& sj = stage[wid];
  const int row = blockIdx.x;                       // (cy, cz); blockIdx.y strides over the row's tiles
  const int cy = row % prm.nc[1], cz = row / prm.nc[1];
  const int ncx = prm.nc[0];
  const int row_s = pstart[row * ncx], row_e = pstart[(row + 1) * ncx];
  const int ntile = (row_e - row_s + 31) >> 5;
  const bool mix = MI && prm.minimg[0] != 0, miy = MI && prm.minimg[1] != 0, miz = MI && prm.minimg[2] != 0;
  // a (sub-)tile may span at most span_max cells so that its +-2 neighbourhood never overlaps itself
  const int span_max = prm.periodic[0] && !mix ? max(ncx - 5, 0) : (1 << 30);
  const T a2 = prm.a2, inv_a = prm.inv_a, inv_a2 = prm.inv_a2, two_inv_a3 = prm.two_inv_a3;
  const float a2_scan = prm.a2_scan;
  T cf[P], cd[P];                                   // g(s) = sum cf[k] s^k, g'(s) = sum cd[k] s^(k-1)
#pragma unroll
  for (int k = 0; k < P; ++k) { cf[k] = prm.c[k]; cd[k] = (T)k * prm.c[k]; }
  double W[6] = {0, 0, 0, 0, 0, 0};

  for (int tile = blockIdx.y * kPairWarps + wid; tile < ntile; tile += kPairWarps * gridDim.y) {
    const int ki = row_s + tile * 32 + lane;
    const bool inrow = ki < row_e;
    V4 ri = make_vec4<T>(0, 0, 0, 0);
    int cxi = 0;
    if (inrow) { ri = ldg4(prec + ki); cxi = pcellx[ki]; }
    const int last = min(31, row_e - 1 - (row_s + tile * 32));
   // sub-tiles: consecutive lanes whose cells span at most span_max (one pass unless the row is sparse)
   for (int first = 0; first <= last;) {
    const int cxf = __shfl_sync(0xffffffffu, cxi, first);
    const unsigned fits = __ballot_sync(0xffffffffu, inrow && lane >= first && cxi - cxf <= span_max);
    const int sub_last = 31 - __clz((int)fits);            // cells ascend with the lane
    const bool iv = lane >= first && lane <= sub_last;
    const int cxl = __shfl_sync(0xffffffffu, cxi, sub_last);
    first = sub_last + 1;
    const T xi = ri.x + (T)(cxi - cxf) * prm.edge[0], yi = ri.y, zi = ri.z;
    // fp32 copy for the scan; an idle lane sits far away and never hits
    const float xs = iv ? (float)xi : 3e30f, ys = (float)yi, zs = (float)zi;
    // x-range of neighbour cells in unwrapped cell coordinates
    int xa = cxf - 2, xb = cxl + 2;
    if (!prm.periodic[0]) { xa = max(xa, 0); xb = min(xb, ncx - 1); }
    else if (mix) { xa = 0; xb = ncx - 1; }                 // fewer than 5 cells: each once + min. image
    constexpr bool anymi = MI;
    T ax = 0, ay = 0, az = 0, av = 0;
    T w0 = 0, w1 = 0, w2 = 0, w3 = 0, w4 = 0, w5 = 0;
    // fp32 drains two hits per lane and round with packed f32x2 arithmetic (FADD2/FMUL2/FFMA2: two
    // results per instruction and lane, half the issue slots); the halves are added at the end
    constexpr bool kPacked = sizeof(T) == 4 && !MI;
    float2 ax2 = {0.f, 0.f}, ay2 = {0.f, 0.f}, az2 = {0.f, 0.f}, av2 = {0.f, 0.f};
    float2 u0 = {0.f, 0.f}, u1 = {0.f, 0.f}, u2 = {0.f, 0.f}, u3 = {0.f, 0.f}, u4 = {0.f, 0.f}, u5 = {0.f, 0.f};
    int fill = 0;          // candidates staged in the current batch
    int selfpos = -1;      // stage index of the lane's own particle, if it is in the batch

    // ---- scan + drain of the staged batch
    auto process = [&]() {
      const int nw = (fill + 31) >> 5;
      for (int k = fill + lane; k < nw * 32; k += 32) sj.put(k, make_vec4<T>((T)1e30, 0, 0, 0));   // pads: far away
      __syncwarp();
      unsigned char* const lp = sj.list + lane;
      unsigned char* le = lp;                                 // end of this lane's hit list (stride 32)
      for (int w = 0; w < nw; ++w) {
        const float* fw = sj.f + w * 128;                     // 16 candidate pairs of 8 floats
        const int ib = w * 32;
        if (!anymi) {
          // two candidates per packed instruction (FADD2 / FMUL2 / FFMA2); same roundings as scalar
#pragma unroll
          for (int m = 0; m < 16; ++m) {
            const float4 xy = *reinterpret_cast<const float4*>(fw + m * 8);        // x0 x1 y0 y1
            const float2 zz = *reinterpret_cast<const float2*>(fw + m * 8 + 4);    // z0 z1
            const float2 dx = __fadd2_rn(make_float2(xs, xs), make_float2(-xy.x, -xy.y));
            const float2 dy_ = __fadd2_rn(make_float2(ys, ys), make_float2(-xy.z, -xy.w));
            const float2 dz_ = __fadd2_rn(make_float2(zs, zs), make_float2(-zz.x, -zz.y));
            const float2 r2 = __ffma2_rn(dx, dx, __ffma2_rn(dy_, dy_, __fmul2_rn(dz_, dz_)));
            if (r2.x < a2_scan) { *le = (unsigned char)(ib + 2 * m); le += 32; }
            if (r2.y < a2_scan) { *le = (unsigned char)(ib + 2 * m + 1); le += 32; }
          }
        } else {
#pragma unroll 4
          for (int kk = 0; kk < 32; ++kk) {
            const float* pq = fw + pair_slot(kk);
            const float4 pj = make_float4(pq[0], pq[2], pq[4], 0.f);
            float dx = xs - pj.x, dy_ = ys - pj.y, dz_ = zs - pj.z;
            if (mix) dx -= (float)prm.box[0] * rintf(dx * (float)prm.inv_box[0]);
            if (miy) dy_ -= (float)prm.box[1] * rintf(dy_ * (float)prm.inv_box[1]);
            if (miz) dz_ -= (float)prm.box[2] * rintf(dz_ * (float)prm.inv_box[2]);
            const float r2 = fmaf(dx, dx, fmaf(dy_, dy_, dz_ * dz_));
            if (r2 < a2_scan) { *le = (unsigned char)(ib + kk); le += 32; }
          }
        }
      }
      const int n = (int)(le - lp) >> 5;                      // hits of this lane
      int nmax = n;
#pragma unroll
      for (int o = 16; o > 0; o >>= 1) nmax = max(nmax, __shfl_xor_sync(0xffffffffu, nmax, o));
      if constexpr (kPacked) {
        const float* sf = reinterpret_cast<const float*>(sj.f);
        const float xf = (float)xi, yf = (float)yi, zf = (float)zi;
        for (int r = 0; r < nmax; r += 2) {
          if (r < n) {
            // hits r and r + 1 of this lane; a missing second hit repeats the first with charge 0,
            // the particle itself gets charge 0 and a harmless distance
            const bool two = r + 1 < n;
            const int ia = lp[r * 32], ib = two ? lp[(r + 1) * 32] : ia;
            const float* pa = sf + pair_slot(ia);
            const float* pb = sf + pair_slot(ib);
            const float2 xj = make_float2(pa[0], pb[0]), yj = make_float2(pa[2], pb[2]), zj = make_float2(pa[4], pb[4]);
            const float2 qj = make_float2(ia != selfpos ? pa[6] : 0.f, (two && ib != selfpos) ? pb[6] : 0.f);
            const float2 dx = __fadd2_rn(make_float2(xf, xf), make_float2(-xj.x, -xj.y));
            const float2 dy_ = __fadd2_rn(make_float2(yf, yf), make_float2(-yj.x, -yj.y));
            const float2 dz_ = __fadd2_rn(make_float2(zf, zf), make_float2(-zj.x, -zj.y));
            float2 r2 = __ffma2_rn(dx, dx, __ffma2_rn(dy_, dy_, __fmul2_rn(dz_, dz_)));
            r2.x = fmaxf(r2.x, 1e-20f); r2.y = fmaxf(r2.y, 1e-20f);       // only the self pair is this close
            const float2 rinv = make_float2(rsqrt_fast(r2.x), rsqrt_fast(r2.y));
            const float2 sv = __ffma2_rn(r2, make_float2((float)inv_a2, (float)inv_a2), make_float2(-1.f, -1.f));
            float2 g = make_float2((float)cf[P - 1], (float)cf[P - 1]), dg = make_float2((float)cd[P - 1], (float)cd[P - 1]);
#pragma unroll
            for (int k = P - 2; k >= 0; --k) g = __ffma2_rn(g, sv, make_float2((float)cf[k], (float)cf[k]));
#pragma unroll
            for (int k = P - 2; k >= 1; --k) dg = __ffma2_rn(dg, sv, make_float2((float)cd[k], (float)cd[k]));
            const float nia = -(float)inv_a, t3 = (float)two_inv_a3;
            av2 = __ffma2_rn(qj, __ffma2_rn(g, make_float2(nia, nia), rinv), av2);
            const float2 rinv3 = __fmul2_rn(__fmul2_rn(rinv, rinv), rinv);
            const float2 fs = __fmul2_rn(qj, __ffma2_rn(make_float2(t3, t3), dg, rinv3));
            ax2 = __ffma2_rn(fs, dx, ax2); ay2 = __ffma2_rn(fs, dy_, ay2); az2 = __ffma2_rn(fs, dz_, az2);
            if (VIRIAL) {
              const float2 fx = __fmul2_rn(fs, dx), fy = __fmul2_rn(fs, dy_), fz = __fmul2_rn(fs, dz_);
              u0 = __ffma2_rn(fx, dx, u0); u1 = __ffma2_rn(fy, dy_, u1); u2 = __ffma2_rn(fz, dz_, u2);
              u3 = __ffma2_rn(fx, dy_, u3); u4 = __ffma2_rn(fx, dz_, u4); u5 = __ffma2_rn(fy, dz_, u5);
            }
          }
        }
      } else {
      for (int r = 0; r < nmax; ++r) {
        if (r < n) {
          const int idx = lp[r * 32];
          if (idx != selfpos) {                               // the particle itself, dropped by index
            const V4 pj = sj.full(idx);
            T dx = xi - pj.x, dy_ = yi - pj.y, dz_ = zi - pj.z;
            if (anymi) {
              if (mix) dx -= prm.box[0] * rint(dx * prm.inv_box[0]);
              if (miy) dy_ -= prm.box[1] * rint(dy_ * prm.inv_box[1]);
              if (miz) dz_ -= prm.box[2] * rint(dz_ * prm.inv_box[2]);
            }
            const T r2 = fma(dx, dx, fma(dy_, dy_, dz_ * dz_));
            if (sizeof(T) == 4 || r2 < a2) {                  // fp32: the scan was already exact
              const T rinv = rsqrt_fast(r2);
              const T s = fma(r2, inv_a2, (T)-1);
              T g = cf[P - 1], dg = cd[P - 1];
#pragma unroll
              for (int k = P - 2; k >= 0; --k) g = fma(g, s, cf[k]);
#pragma unroll
              for (int k = P - 2; k >= 1; --k) dg = fma(dg, s, cd[k]);
              const T qj = pj.w;
              av = fma(qj, fma(-g, inv_a, rinv), av);
              const T fs = qj * fma(two_inv_a3, dg, rinv * rinv * rinv);
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
      __syncwarp();
      fill = 0;
      selfpos = -1;
    };

    for (int dz = prm.omin[2] + (int)blockIdx.z; dz <= prm.omax[2]; dz += prm.nsplit) {
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
          for (int j = js; j < je;) {
            // stage as many candidates of this segment as fit, in the tile's frame
            const int take = min(je - j, B - fill);
            for (int t = lane; t < take; t += 32) {
              const int kj = j + t;
              V4 rj = ldg4(prec + kj);
              rj.x += (T)(pcellx[kj] + shift - cxf) * prm.edge[0];
              rj.y += yoff;
              rj.z += zoff;
              sj.put(fill + t, rj);
            }
            if (ki >= j && ki < j + take) selfpos = fill + (ki - j);
            fill += take;
            j += take;
            if (fill == B) process();
          }
        }
      }
    }
    if (fill > 0) process();
    if (kPacked) {
      ax += (T)(ax2.x + ax2.y); ay += (T)(ay2.x + ay2.y); az += (T)(az2.x + az2.y); av += (T)(av2.x + av2.y);
      w0 += (T)(u0.x + u0.y); w1 += (T)(u1.x + u1.y); w2 += (T)(u2.x + u2.y);
      w3 += (T)(u3.x + u3.y); w4 += (T)(u4.x + u4.y); w5 += (T)(u5.x + u5.y);
    }

    if (iv) {
      const int orig = porder[ki];
      const T qi = ri.w;
      T* Fp = Fsr + (size_t)blockIdx.z * 3 * prm.part_stride;   // partial of this split
      Fp[3 * (size_t)orig + 0] = qi * ax;
      Fp[3 * (size_t)orig + 1] = qi * ay;
      Fp[3 * (size_t)orig + 2] = qi * az;
      Vsr[(size_t)blockIdx.z * prm.part_stride + orig] = av;
      if (VIRIAL) {
        const double hq = 0.5 * (double)qi;   // every pair is visited from both ends
        W[0] += hq * (double)w0; W[1] += hq * (double)w1; W[2] += hq * (double)w2;
        W[3] += hq * (double)w3; W[4] += hq * (double)w4; W[5] += hq * (double)w5;
      }
    }
   }
  }
  if (VIRIAL) {   // one partial per warp, fixed shuffle order; no block barrier (warps finish at different times)
#pragma unroll
    for (int k = 0; k < 6; ++k) {
      double v = W[k];
#pragma unroll
      for (int o = 16; o > 0; o >>= 1) v += __shfl_down_sync(0xffffffffu, v, o);
      if (lane == 0)
        wpart[((((size_t)blockIdx.z * gridDim.y + blockIdx.y) * gridDim.x + blockIdx.x) * kPairWarps + wid) * 6 + k] = v;
    }
  }
}

}  // namespace msm
