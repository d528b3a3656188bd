// pair.cuh -- S2: short-range pair sum of k_0(r) = 1/r - gamma(r/a)/a over a cell list
// (Eq. 5 first term; Eq. 21 l = 0), with forces and the pair virial.
//
// Cells have edge >= a/2, so the neighbourhood of a cell is 5 x 5 x 5 cells. The particles are
// sorted by cell, x fastest, so the neighbours of a particle in one of the 25 neighbouring cell
// rows (dy, dz) are ONE contiguous range of the sorted order (two when the x window wraps).
//
// Work unit = one warp = a CLUSTER of 8 consecutive sorted particles of one cell row, laid out as
// 8 i-particles x 4 j-phases: lane = 8 * jq + il owns particle il and every fourth PAIR of
// candidates. A 32-particle tile (round 1) is as long as the cutoff itself, so its lanes scanned a
// 7-cell x-range for a 5-cell need; a cluster of 8 is ~0.7 cells long, its window is 5-6 cells, and
// each lane now walks only a quarter of it. The candidates of all 25 rows are staged through
// shared memory in the cluster's frame (coordinates relative to the cluster's first cell: fp32
// differences stay accurate), flattened into one list, so that every step of the inner loop is a
// full 8 i x 8 j block of pairs with no ragged row ends.
//
// fp32: every staged candidate is evaluated in full with packed f32x2 arithmetic (FADD2 / FMUL2 /
//   FFMA2: two pairs per instruction and lane) and masked by the cutoff test -- no hit lists, no
//   divergence, no shared-memory traffic beyond two broadcast 16-byte loads per step. Only 25-30 %
//   of the candidates are inside the cutoff, but filtering them costs as many issue slots as the
//   interaction itself in packed fp32 (round 1's scan + drain kernel spent 71 % of its time in the
//   shared-memory pipe on list bookkeeping).
// fp64: DFMA runs at half the FP32 rate and the interaction needs ~45 of them, so here filtering
//   pays: a packed fp32 scan (slightly widened cutoff) appends each lane's hits to its private
//   list in shared memory, and the drain evaluates only those in fp64 (exact cutoff test repeated).
// The virial is accumulated over HALF the neighbourhood: rows above the cluster's own row with
// weight 1, the own row with weight 1/2 (both ends visit it), rows below not at all -- every
// unordered pair exactly once.
// Small systems have too few clusters to fill the GPU: the dz planes of the neighbourhood are then
// dealt to up to kPairMaxSplit blocks (blockIdx.z) whose partial sums k_interpolate adds in order.
// Every lane visits its candidates in a fixed order and the four phases of a particle are added
// in a fixed order, so the sums are run-to-run deterministic.
// -k_0'(r)/r = 1/r^3 + (2/a^3) g'(s), s = r^2/a^2 - 1: one rsqrt per pair is the only special
// function.
#pragma once
#include <type_traits>

#include "device_common.cuh"

namespace msm {

template <typename T> struct PairParams {
  int nc[3];
  int periodic[3];
  int omin[3], omax[3];   // neighbour cell offsets per axis (y, z use these; x: +-2 around the cluster)
  int minimg[3];          // periodic axis with fewer than 5 cells: explicit minimum image
  T edge[3];
  T box[3], inv_box[3];
  T a, a2, inv_a, inv_a2, two_inv_a3;
  float a2_scan;          // cutoff^2 of the fp32 scan (widened by rounding slack in fp64 mode)
  T c[8];                 // binom(-1/2, k)
  int p;
  int nsplit;             // the dz planes of the neighbourhood are dealt to nsplit blocks (blockIdx.z)
  size_t part_stride;     // elements between the per-split partial outputs (capacity)
};

constexpr int kPairWarpsMax = 4;
// independent warps (clusters) per block: fp64 stages 14 KB per warp (48 KB static limit)
template <typename T> struct PairWarps { static constexpr int value = sizeof(T) == 4 ? 4 : 2; };
constexpr int kPairCluster = 8;     // i-particles per warp
constexpr int kPairMaxSplit = 5;
constexpr int kPairSpanCap = 2;     // a cluster pass spans at most this many cells beyond its first

// Shared-memory staging of one warp. fp32 records are interleaved in pairs of candidates,
// (x0 x1 | y0 y1 | z0 z1 | q0 q1), so that a lane's pair is two 16-byte loads feeding packed
// instructions without any register shuffling: candidate k sits at float offset
// pair_slot(k) + {0, 2, 4, 6}.
__device__ __forceinline__ int pair_slot(int k) { return (k >> 1) * 8 + (k & 1); }
template <typename T> struct PairStage;
template <> struct PairStage<float> {
  static constexpr int kCap = 512;            // candidates per chunk (multiple of 8)
  __align__(16) float f[kCap * 4];
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
  static constexpr int kCap = 256;
  __align__(16) float f[kCap * 4];            // fp32 copy for the scan (q slots unused)
  double4 d[kCap];                            // full precision for the drain
  unsigned char list[kCap * 8];               // hit r of lane l at [r * 32 + l]; a lane scans kCap / 4 candidates
  __device__ __forceinline__ void put(int k, double4 r) {
    d[k] = r;
    float* q = f + pair_slot(k);
    q[0] = (float)r.x; q[2] = (float)r.y; q[4] = (float)r.z; q[6] = 0.f;
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

// accumulators of one lane: force factor sums, potential, virial (xx yy zz xy xz yz)
template <typename T> struct PairAcc {
  T ax = 0, ay = 0, az = 0, av = 0;
  T w[6] = {0, 0, 0, 0, 0, 0};
};
struct PairAcc2 {   // fp32 packed: two partial sums per quantity
  float2 ax = {0.f, 0.f}, ay = {0.f, 0.f}, az = {0.f, 0.f}, av = {0.f, 0.f};
  float2 w[6] = {{0.f, 0.f}, {0.f, 0.f}, {0.f, 0.f}, {0.f, 0.f}, {0.f, 0.f}, {0.f, 0.f}};
};

// one full interaction in precision T (scalar path: fp64 drain, minimum-image instances)
template <typename T, int P, bool VIR>
__device__ __forceinline__ void pair_interact(PairAcc<T>& A, T dx, T dy, T dz, T r2, T qj, T inv_a, T inv_a2,
                                              T two_inv_a3, const T (&cf)[P], const T (&cd)[P]) {
  const T rinv = rsqrt_fast(r2);
  const T s = fma(r2, inv_a2, (T)-1);
  T g = cf[P - 1], dg = cd[P - 1];
#pragma unroll
  for (int k = P - 2; k >= 0; --k) g = fma(g, s, cf[k]);
#pragma unroll
  for (int k = P - 2; k >= 1; --k) dg = fma(dg, s, cd[k]);
  A.av = fma(qj, fma(-g, inv_a, rinv), A.av);
  const T fs = qj * fma(two_inv_a3, dg, rinv * rinv * rinv);
  A.ax = fma(fs, dx, A.ax); A.ay = fma(fs, dy, A.ay); A.az = fma(fs, dz, A.az);
  if (VIR) {
    const T fx = fs * dx, fy = fs * dy, fz = fs * dz;
    A.w[0] = fma(fx, dx, A.w[0]); A.w[1] = fma(fy, dy, A.w[1]); A.w[2] = fma(fz, dz, A.w[2]);
    A.w[3] = fma(fx, dy, A.w[3]); A.w[4] = fma(fx, dz, A.w[4]); A.w[5] = fma(fy, dz, A.w[5]);
  }
}

template <typename T, int P, bool VIRIAL, bool MI>
__global__ void __launch_bounds__(PairWarps<T>::value * 32, sizeof(T) == 4 ? 6 : 1)
k_pair(PairParams<T> prm, const int* __restrict__ pstart, const typename Vec4<T>::type* __restrict__ prec,
       const int* __restrict__ pcellx, const int* __restrict__ porder, T* __restrict__ Fsr,
       T* __restrict__ Vsr, double* __restrict__ wpart) {
  using V4 = typename Vec4<T>::type;
  constexpr int CAP = PairStage<T>::kCap;
  constexpr int kPairWarps = PairWarps<T>::value;
  constexpr bool kPacked = sizeof(T) == 4 && !MI;     // fp32: brute force with packed arithmetic
  constexpr bool kLists = sizeof(T) == 8 && !MI;      // fp64: fp32 scan + hit lists + fp64 drain
  __shared__ PairStage<T> stage[kPairWarps];
  const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
  const int il = lane & 7, jq = lane >> 3;
  PairStage<T>& sj = stage[wid];
  const int row = blockIdx.x;                       // (cy, cz); blockIdx.y strides over the row's clusters
  const int cy = row % prm.nc[1], cz = row / prm.nc[1];
  const int ncx = prm.nc[0];
  const int row_s = pstart[row * ncx], row_e = pstart[(row + 1) * ncx];
  const int ntile = (row_e - row_s + kPairCluster - 1) / kPairCluster;
  const bool mix = MI && prm.minimg[0] != 0, miy = MI && prm.minimg[1] != 0, miz = MI && prm.minimg[2] != 0;
  // a cluster pass may span at most span_max cells beyond its first one, so that its +-2
  // neighbourhood never overlaps itself on a periodic axis and the window stays short
  const int span_max = prm.periodic[0] && !mix ? max(min(ncx - 5, kPairSpanCap), 0) : kPairSpanCap;
  const T a2 = prm.a2, inv_a = prm.inv_a, inv_a2 = prm.inv_a2, two_inv_a3 = prm.two_inv_a3;
  const float a2_scan = prm.a2_scan;
  T cf[P], cd[P];                                   // g(s) = sum cf[k] s^k, g'(s) = sum cd[k] s^(k-1)
#pragma unroll
  for (int k = 0; k < P; ++k) { cf[k] = prm.c[k]; cd[k] = (T)k * prm.c[k]; }
  double W[6] = {0, 0, 0, 0, 0, 0};

  // the neighbour rows of this block in class order: lane r describes row r.
  //   class 1 (r = 0): the cluster's own row, virial weight 1/2;  class 2: rows above (dz > 0, or
  //   dz = 0 and dy > 0), weight 1;  class 3: rows below, no virial. Minimum-image instances (fewer
  //   than 5 cells on a periodic axis: offsets alias) put every row into class 1.
  const int ny_off = prm.omax[1] - prm.omin[1] + 1, nz_off = prm.omax[2] - prm.omin[2] + 1;
  const int nrows = ny_off * nz_off;                // <= 25
  int my_dy = 0, my_dz = 0, my_class = 0, my_rowbase = 0;   // class 0: row absent
  if (lane < nrows) {
    if (MI) {
      my_dy = prm.omin[1] + lane % ny_off; my_dz = prm.omin[2] + lane / ny_off;
      my_class = 1;
    } else {                                        // offsets -2 .. 2 on both axes
      if (lane == 0) { my_dy = 0; my_dz = 0; my_class = 1; }
      else {
        const int u = (lane - 1) % 12, neg = (lane - 1) / 12;   // upper rows: (dz 0: dy 1, 2), (dz 1, 2: dy -2 .. 2)
        if (u < 2) { my_dy = u + 1; my_dz = 0; }
        else { my_dy = (u - 2) % 5 - 2; my_dz = (u - 2) / 5 + 1; }
        if (neg) { my_dy = -my_dy; my_dz = -my_dz; }
        my_class = neg ? 3 : 2;
      }
    }
    if ((my_dz - prm.omin[2]) % prm.nsplit != (int)blockIdx.z) my_class = 0;
    int cyj = cy + my_dy, czj = cz + my_dz;
    if (prm.periodic[1]) cyj = imod(cyj, prm.nc[1]); else if (cyj < 0 || cyj >= prm.nc[1]) my_class = 0;
    if (prm.periodic[2]) czj = imod(czj, prm.nc[2]); else if (czj < 0 || czj >= prm.nc[2]) my_class = 0;
    my_rowbase = (czj * prm.nc[1] + cyj) * ncx;
  }

  for (int tile = blockIdx.y * kPairWarps + wid; tile < ntile; tile += kPairWarps * gridDim.y) {
    const int k0 = row_s + tile * kPairCluster;     // first sorted particle of the cluster
    const int ki = k0 + il;
    const bool inrow = ki < row_e;
    V4 ri = make_vec4<T>(0, 0, 0, 0);
    int cxi = 0;
    if (inrow) { ri = ldg4(prec + ki); cxi = pcellx[ki]; }
    const int last = min(kPairCluster - 1, row_e - 1 - k0);
   // passes: consecutive particles whose cells span at most span_max (one pass unless the row is sparse)
   for (int first = 0; first <= last;) {
    const int cxf = __shfl_sync(0xffffffffu, cxi, first);
    const unsigned fits = __ballot_sync(0xffffffffu, inrow && il >= first && cxi - cxf <= span_max) & 0xffu;
    const int sub_last = 31 - __clz((int)fits);            // cells ascend with il
    const bool iv = il >= first && il <= sub_last;
    const int cxl = __shfl_sync(0xffffffffu, cxi, sub_last);
    first = sub_last + 1;
    const T xi = ri.x + (T)(cxi - cxf) * prm.edge[0], yi = ri.y, zi = ri.z;
    // x-range of neighbour cells in unwrapped cell coordinates
    int xa = cxf - 2, xb = cxl + 2;
    if (!prm.periodic[0]) { xa = max(xa, 0); xb = min(xb, ncx - 1); }
    else if (mix) { xa = 0; xb = ncx - 1; }                 // fewer than 5 cells: each once + min. image
    // this lane's row: up to two contiguous segments of the sorted order (main, wrapped)
    int sA = 0, lA = 0, sB = 0, lB = 0, shB = 0;
    if (my_class != 0) {
      const int ca = max(xa, 0), cb = min(xb, ncx - 1);
      if (ca <= cb) { sA = pstart[my_rowbase + ca]; lA = pstart[my_rowbase + cb + 1] - sA; }
      if (xa < 0) { sB = pstart[my_rowbase + xa + ncx]; lB = pstart[my_rowbase + ncx] - sB; shB = -ncx; }
      else if (xb >= ncx) { sB = pstart[my_rowbase]; lB = pstart[my_rowbase + xb - ncx + 1] - sB; shB = ncx; }
    }
    // The candidates of all rows form ONE flat list (row after row, class after class); each class
    // region is padded to a multiple of 8 so that a step of 8 candidates never straddles two classes.
    const int len = lA + lB;
    int incl = len;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
      const int t = __shfl_up_sync(0xffffffffu, incl, o);
      if (lane >= o) incl += t;
    }
    int r1e = 0, b1 = 1 << 30, r2e = 0, b2 = 1 << 30;       // raw and padded ends of the class 1 / 2 regions
    if (!MI) {
      r1e = __shfl_sync(0xffffffffu, incl, 0);
      b1 = (r1e + 7) & ~7;
      r2e = __shfl_sync(0xffffffffu, incl, 12) + (b1 - r1e);
      b2 = (r2e + 7) & ~7;
    }
    const int off = incl - len + (!MI && lane >= 1 ? b1 - r1e : 0) + (!MI && lane >= 13 ? b2 - r2e : 0);
    const int r3e = __shfl_sync(0xffffffffu, incl, 31) + (MI ? 0 : (b1 - r1e) + (b2 - r2e));
    const int total = (r3e + 7) & ~7;
    // flat position of the lane's own particle (in the cluster's own row), -1 if that row is absent
    int selfpos = -1;
    {
      const int r0 = MI ? (-prm.omin[1]) + (-prm.omin[2]) * ny_off : 0;
      const int a0 = __shfl_sync(0xffffffffu, sA, r0), la0 = __shfl_sync(0xffffffffu, lA, r0);
      const int b0 = __shfl_sync(0xffffffffu, sB, r0), lb0 = __shfl_sync(0xffffffffu, lB, r0);
      const int o0 = __shfl_sync(0xffffffffu, off, r0);
      if (ki >= a0 && ki < a0 + la0) selfpos = o0 + ki - a0;
      else if (ki >= b0 && ki < b0 + lb0) selfpos = o0 + la0 + ki - b0;
    }

    PairAcc<T> A;                       // scalar accumulators (fp64, minimum image)
    PairAcc2 A2;                        // packed accumulators (fp32)
    // an idle lane sits 64 cutoffs to the left, the pads 64 cutoffs to the right: neither ever
    // hits, and the softening polynomial of such a distance stays finite in fp32
    const T far = (T)64 * prm.a;
    const float xs = iv ? (float)xi : -(float)far, ys = (float)yi, zs = (float)zi;
    const int grp = lane >> 3;

    for (int base = 0; base < total; base += CAP) {
      const int hi = min(base + CAP, total);
      // ---- pads of the three class regions
      {
        const int gs = grp == 0 ? r1e : grp == 1 ? r2e : r3e, ge = grp == 0 ? b1 : grp == 1 ? b2 : total;
        const int pos = gs + il;
        if (grp < 3 && (!MI || grp == 2) && pos < ge && pos >= base && pos < hi)
          sj.put(pos - base, make_vec4<T>(far, 0, 0, 0));
      }
      // ---- stage: four rows at a time, eight lanes per row, into the cluster's frame
      for (int rr = 0; rr < nrows; rr += 4) {
        const int r = rr + grp;
        const int o = __shfl_sync(0xffffffffu, off, r), la = __shfl_sync(0xffffffffu, lA, r);
        const int lb = __shfl_sync(0xffffffffu, lB, r), sa = __shfl_sync(0xffffffffu, sA, r);
        const int sb = __shfl_sync(0xffffffffu, sB, r), sh = __shfl_sync(0xffffffffu, shB, r);
        const T yoff = (T)__shfl_sync(0xffffffffu, my_dy, r) * prm.edge[1];
        const T zoff = (T)__shfl_sync(0xffffffffu, my_dz, r) * prm.edge[2];
        const int t1 = min(la + lb, hi - o);
        // four elements per lane and batch: all eight loads of a batch are issued before the first
        // store, so a batch costs one global-memory latency instead of four
#pragma unroll 1
        for (int tb = max(0, base - o) + il; tb < t1; tb += 32) {
          V4 rj[4];
          int cj[4];
#pragma unroll
          for (int k = 0; k < 4; ++k) {
            const int t = tb + 8 * k;
            const bool inA = t < la;
            const int src = t < t1 ? (inA ? sa + t : sb + (t - la)) : 0;
            rj[k] = ldg4(prec + src);
            cj[k] = pcellx[src] + (inA ? 0 : sh) - cxf;
          }
#pragma unroll
          for (int k = 0; k < 4; ++k) {
            const int t = tb + 8 * k;
            if (t < t1) {
              rj[k].x += (T)cj[k] * prm.edge[0];
              rj[k].y += yoff;
              rj[k].z += zoff;
              sj.put(o + t - base, rj[k]);
            }
          }
        }
      }
      __syncwarp();

      // ---- candidates [lo, hi2) of the flat list (multiples of 8) against the 8 particles
      auto run = [&](int lo, int hi2, auto virc) {
        constexpr bool VIR = decltype(virc)::value;
        const int nsteps = (hi2 - lo) >> 3;
        if constexpr (kPacked) {
          const float ia2 = (float)inv_a2, nia = -(float)inv_a, t3 = (float)two_inv_a3;
          const float2 xi2 = make_float2(xs, xs), yi2 = make_float2(ys, ys), zi2 = make_float2(zs, zs);
          const float* fp = sj.f + (lo - base) * 4 + jq * 8;
          int jdx = lo + 2 * jq - selfpos;                  // candidate index minus the lane's own
#pragma unroll 2
          for (int s = 0; s < nsteps; ++s) {
            const float4 xy = *reinterpret_cast<const float4*>(fp);         // x0 x1 y0 y1
            const float4 zq = *reinterpret_cast<const float4*>(fp + 4);     // z0 z1 q0 q1
            const float2 dx = __fadd2_rn(xi2, make_float2(-xy.x, -xy.y));
            const float2 dy = __fadd2_rn(yi2, make_float2(-xy.z, -xy.w));
            const float2 dz = __fadd2_rn(zi2, make_float2(-zq.x, -zq.y));
            // + 1e-20: no effect on a real pair; keeps the masked self pair finite
            const float2 r2 = __ffma2_rn(dx, dx, __ffma2_rn(dy, dy, __ffma2_rn(dz, dz, make_float2(1e-20f, 1e-20f))));
            const float2 qj = make_float2((r2.x < a2_scan && jdx != 0) ? zq.z : 0.f,
                                          (r2.y < a2_scan && jdx != -1) ? zq.w : 0.f);
            const float2 rinv = make_float2(rsqrt_fast(r2.x), rsqrt_fast(r2.y));
            const float2 sv = __ffma2_rn(r2, make_float2(ia2, ia2), make_float2(-1.f, -1.f));
            float2 g = make_float2((float)cf[P - 1], (float)cf[P - 1]), dg = make_float2((float)cd[P - 1], (float)cd[P - 1]);
#pragma unroll
            for (int k = P - 2; k >= 0; --k) g = __ffma2_rn(g, sv, make_float2((float)cf[k], (float)cf[k]));
#pragma unroll
            for (int k = P - 2; k >= 1; --k) dg = __ffma2_rn(dg, sv, make_float2((float)cd[k], (float)cd[k]));
            A2.av = __ffma2_rn(qj, __ffma2_rn(g, make_float2(nia, nia), rinv), A2.av);
            const float2 rinv3 = __fmul2_rn(__fmul2_rn(rinv, rinv), rinv);
            const float2 fs = __fmul2_rn(qj, __ffma2_rn(make_float2(t3, t3), dg, rinv3));
            A2.ax = __ffma2_rn(fs, dx, A2.ax); A2.ay = __ffma2_rn(fs, dy, A2.ay); A2.az = __ffma2_rn(fs, dz, A2.az);
            if (VIR) {
              const float2 fx = __fmul2_rn(fs, dx), fy = __fmul2_rn(fs, dy), fz = __fmul2_rn(fs, dz);
              A2.w[0] = __ffma2_rn(fx, dx, A2.w[0]); A2.w[1] = __ffma2_rn(fy, dy, A2.w[1]); A2.w[2] = __ffma2_rn(fz, dz, A2.w[2]);
              A2.w[3] = __ffma2_rn(fx, dy, A2.w[3]); A2.w[4] = __ffma2_rn(fx, dz, A2.w[4]); A2.w[5] = __ffma2_rn(fy, dz, A2.w[5]);
            }
            fp += 32;
            jdx += 8;
          }
        } else if constexpr (kLists) {
          // scan: packed fp32 distance test of this lane's candidate pairs, hits appended to its list
          unsigned char* const lp = sj.list + lane;
          unsigned char* le = lp;
          {
            const float2 xi2 = make_float2(xs, xs), yi2 = make_float2(ys, ys), zi2 = make_float2(zs, zs);
            const float* fp = sj.f + (lo - base) * 4 + jq * 8;
            int idx = lo - base + 2 * jq;                   // index inside the chunk
            const int selfl = selfpos - base;
            for (int s = 0; s < nsteps; ++s) {
              const float4 xy = *reinterpret_cast<const float4*>(fp);
              const float2 zz = *reinterpret_cast<const float2*>(fp + 4);
              const float2 dx = __fadd2_rn(xi2, make_float2(-xy.x, -xy.y));
              const float2 dy = __fadd2_rn(yi2, make_float2(-xy.z, -xy.w));
              const float2 dz = __fadd2_rn(zi2, make_float2(-zz.x, -zz.y));
              const float2 r2 = __ffma2_rn(dx, dx, __ffma2_rn(dy, dy, __fmul2_rn(dz, dz)));
              if (r2.x < a2_scan && idx != selfl) { *le = (unsigned char)idx; le += 32; }
              if (r2.y < a2_scan && idx + 1 != selfl) { *le = (unsigned char)(idx + 1); le += 32; }
              fp += 32;
              idx += 8;
            }
          }
          const int n = (int)(le - lp) >> 5;                    // hits of this lane
          int nmax = n;
#pragma unroll
          for (int o = 16; o > 0; o >>= 1) nmax = max(nmax, __shfl_xor_sync(0xffffffffu, nmax, o));
          __syncwarp();
          // drain: hit r of every lane that has one, in full precision (exact cutoff test)
          for (int r = 0; r < nmax; ++r) {
            if (r < n) {
              const V4 pj = sj.full(lp[r * 32]);
              const T dx = xi - pj.x, dy = yi - pj.y, dz = zi - pj.z;
              const T r2 = fma(dx, dx, fma(dy, dy, dz * dz));
              if (r2 < a2) pair_interact<T, P, VIR>(A, dx, dy, dz, r2, pj.w, inv_a, inv_a2, two_inv_a3, cf, cd);
            }
          }
          __syncwarp();
        } else {
          // minimum-image instances (tiny periodic boxes): plain loop in precision T
          for (int s = 0; s < nsteps; ++s) {
#pragma unroll
            for (int h = 0; h < 2; ++h) {
              const int pos = lo + s * 8 + 2 * jq + h;
              const V4 pj = sj.full(pos - base);
              T dx = xi - pj.x, dy = yi - pj.y, dz = zi - pj.z;
              if (mix) dx -= prm.box[0] * rint(dx * prm.inv_box[0]);
              if (miy) dy -= prm.box[1] * rint(dy * prm.inv_box[1]);
              if (miz) dz -= prm.box[2] * rint(dz * prm.inv_box[2]);
              const T r2 = fma(dx, dx, fma(dy, dy, dz * dz));
              if (iv && pos < r3e && pos != selfpos && r2 < a2)
                pair_interact<T, P, VIR>(A, dx, dy, dz, r2, pj.w, inv_a, inv_a2, two_inv_a3, cf, cd);
            }
          }
        }
      };
      if (VIRIAL) {
        const int e1 = min(max(b1, base), hi), e2 = min(max(b2, base), hi);
        run(base, e1, std::true_type());
        if (!MI && b1 > base && b1 <= hi) {               // the own row is done: both ends visit its pairs
          if constexpr (kPacked) {
#pragma unroll
            for (int k = 0; k < 6; ++k) { A2.w[k].x *= 0.5f; A2.w[k].y *= 0.5f; }
          } else {
#pragma unroll
            for (int k = 0; k < 6; ++k) A.w[k] *= (T)0.5;
          }
        }
        run(e1, e2, std::true_type());
        run(e2, hi, std::false_type());
      } else {
        run(base, hi, std::false_type());
      }
      __syncwarp();
    }
    if (MI && VIRIAL) {                                   // every row in class 1: both ends visit every pair
#pragma unroll
      for (int k = 0; k < 6; ++k) A.w[k] *= (T)0.5;
    }
    if constexpr (kPacked) {
      A.ax = A2.ax.x + A2.ax.y; A.ay = A2.ay.x + A2.ay.y; A.az = A2.az.x + A2.az.y; A.av = A2.av.x + A2.av.y;
#pragma unroll
      for (int k = 0; k < 6; ++k) A.w[k] = A2.w[k].x + A2.w[k].y;
    }
    // the four phases of a particle, in a fixed order
    A.ax += __shfl_xor_sync(0xffffffffu, A.ax, 8); A.ay += __shfl_xor_sync(0xffffffffu, A.ay, 8);
    A.az += __shfl_xor_sync(0xffffffffu, A.az, 8); A.av += __shfl_xor_sync(0xffffffffu, A.av, 8);
    A.ax += __shfl_xor_sync(0xffffffffu, A.ax, 16); A.ay += __shfl_xor_sync(0xffffffffu, A.ay, 16);
    A.az += __shfl_xor_sync(0xffffffffu, A.az, 16); A.av += __shfl_xor_sync(0xffffffffu, A.av, 16);

    const T qi = ri.w;
    if (iv && jq == 0) {
      const int orig = porder[ki];
      T* Fp = Fsr + (size_t)blockIdx.z * 3 * prm.part_stride;   // partial of this split
      Fp[3 * (size_t)orig + 0] = qi * A.ax;
      Fp[3 * (size_t)orig + 1] = qi * A.ay;
      Fp[3 * (size_t)orig + 2] = qi * A.az;
      Vsr[(size_t)blockIdx.z * prm.part_stride + orig] = A.av;
    }
    if (VIRIAL && iv) {
      const double dq = (double)qi;      // every unordered pair is counted once (see the row classes)
#pragma unroll
      for (int k = 0; k < 6; ++k) W[k] += dq * (double)A.w[k];
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
