// pair.cuh -- S2: short-range pair sum of k_0(r) = 1/r - gamma(r/a)/a over a cell list
// (Eq. 5 first term; Eq. 21 l = 0), with forces and the pair virial.
//
// Cells have edge >= a/2, so the neighbourhood of a cell is 5 x 5 x 5 cells. The particles are
// sorted by cell row (cy, cz) and, inside a row, by x in sub-bins of a fraction of a cell
// (sort.cuh), so the neighbours of a particle in one of the 25 neighbouring rows (dy, dz) are ONE
// contiguous range of the sorted order (two when the x window wraps around a periodic box).
//
// Work unit = one warp = a CLUSTER of 16 consecutive sorted particles of one row, laid out as
// 16 i-particles x 2 j-phases: lane = 16 * jq + il owns particle il and every second PAIR of
// candidates. A cluster is ~0.85 cutoffs long in x at liquid density: its candidate windows are 18 %
// longer than those of an 8-particle cluster, but they are staged (and the 25 rows set up) once for
// twice as many particles, and staging + set-up were half of the 8-particle kernel's instructions
// (a 32-particle tile is twice as long as the cutoff
// itself), and the x window of every row is cut to the reach the cutoff sphere still has at that
// row's (dy, dz) distance, in sub-bin units. The candidates of all rows are staged through shared
// memory in the cluster's frame (coordinates relative to the cluster's first cell: fp32
// differences stay accurate) as one flat list, so that every step of the inner loop is a full
// 16 i x 4 j block of pairs with no ragged row ends.
//
// fp32: every staged candidate is evaluated in full with packed f32x2 arithmetic (FADD2 / FMUL2 /
//   FFMA2: two pairs per instruction and lane) and masked by the cutoff test -- no hit lists, no
//   divergence, no shared-memory traffic beyond two broadcast 16-byte loads per step. Only ~30 %
//   of the candidates are inside the cutoff, but filtering them costs as many issue slots as the
//   interaction itself in packed fp32 (round 1's scan + drain kernel spent 71 % of its time in the
//   shared-memory pipe on list bookkeeping). The loop is bound by the FP32 pipe.
// fp64: DFMA runs at half the FP32 rate and the interaction needs ~40 of them, so here filtering
//   pays: a packed fp32 scan (slightly widened cutoff) appends each lane's hits to its private
//   list in shared memory, and the drain evaluates only those in fp64 (exact cutoff test repeated).
//
// Virial. For a pair that interacts without a periodic image shift, sum_pairs f_ij (x) d_ij equals
// sum_i F_i (x) r_i with absolute positions, so those pairs -- all of them in an open box, all but
// the ones across a box face otherwise -- cost nothing extra: the force sums of the unshifted
// candidates are kept apart and multiplied by r_i once per particle (in fp64). Only candidates
// reached through a wrapped row or a wrapped x segment accumulate f (x) d pair by pair, over HALF
// the neighbourhood (rows above the cluster's row with weight 1, its own row with weight 1/2, rows
// below not at all), i.e. every image pair exactly once.
//
// Small systems have too few clusters to fill the GPU: the dz planes of the neighbourhood are then
// dealt to up to kPairMaxSplit blocks (blockIdx.z) whose partial sums k_interpolate adds in order.
// Every lane visits its candidates in a fixed order and the two phases of a particle are added
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
  int omin[3], omax[3];   // neighbour cell offsets per axis (y, z)
  int minimg[3];          // periodic axis with fewer than 5 cells: explicit minimum image
  int sxs;                // log2 of the x sub-bins per cell
  int wb[3][3];           // half-width of the x window in sub-bins for rows with |dy|, |dz| = 0, 1, 2; -1: out of reach
  T edge[3];
  double edge_d[3];
  T box[3], inv_box[3];
  T a, a2, inv_a, inv_a2, two_inv_a3;
  float a2_scan;          // cutoff^2 of the fp32 scan (widened by rounding slack in fp64 mode)
  T c[8];                 // binom(-1/2, k)
  int p;
  int nsplit;             // the dz planes of the neighbourhood are dealt to nsplit blocks (blockIdx.z)
  size_t part_stride;     // elements between the per-split partial outputs (capacity)
};

// independent warps (clusters) per block: fp64 stages 14 KB per warp (48 KB static limit)
template <typename T> struct PairWarps { static constexpr int value = sizeof(T) == 4 ? 4 : 2; };
constexpr int kPairCluster = 16;    // i-particles per warp
constexpr int kPairPhases = 32 / kPairCluster;   // lanes per i-particle: each takes every kPairPhases-th PAIR of candidates
constexpr int kPairStep = 2 * kPairPhases;       // candidates per step of the inner loop
constexpr int kPairMaxSplit = 5;
constexpr int kPairSpanCap = 3;     // a cluster pass spans at most this many cells beyond its first

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
  static constexpr int kCap = 192;            // 12 KB per warp: 8 blocks of 2 warps per SM
  __align__(16) float f[kCap * 4];            // fp32 copy for the scan (q slots unused)
  double4 d[kCap];                            // full precision for the drain
  unsigned char list[kCap / kPairPhases * 32];   // hit r of lane l at [r * 32 + l]; a lane scans kCap / kPairPhases candidates
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
// fp64: fp32 hardware seed (relative error 2^-22.9 incl. the rounding of x to fp32) + ONE Newton step
// y <- y (3/2 - x/2 y^2), which squares the error (times 3/2): <= 2.5e-14 relative per pair term,
// 4000 times inside the 1e-10 parity tolerance (measured force error 1.2e-14 at cfg5). A second step
// (-DMSM_RSQRT_TWO_STEPS) reaches the fp64 rounding unit and costs 3.8 % of the fp64 pair kernel: it
// sits on the drain's dependent chain. x is a squared distance inside the cutoff (far from the fp32
// range limits).
__device__ __forceinline__ double rsqrt_fast(double x) {
  double y = (double)rsqrt_fast(fmaxf((float)x, 1e-30f));   // (x = 0: coincident zero-charge pads of a batch stay finite)
  const double hx = 0.5 * x;
  y = y * fma(-hx, y * y, 1.5);
#ifdef MSM_RSQRT_TWO_STEPS
  y = y * fma(-hx, y * y, 1.5);
#endif
  return y;
}

// accumulators of one lane: force factor sums of the unshifted candidates (ax ay az), of the
// image-shifted ones (bx by bz) with their pair virial (w: xx yy zz xy xz yz), potential
template <typename T> struct PairAcc {
  T ax = 0, ay = 0, az = 0, av = 0;
  T bx = 0, by = 0, bz = 0;
  T w[6] = {0, 0, 0, 0, 0, 0};
};
struct PairAcc2 {   // fp32 packed: two partial sums per quantity
  float2 ax = {0.f, 0.f}, ay = {0.f, 0.f}, az = {0.f, 0.f}, av = {0.f, 0.f};
  float2 bx = {0.f, 0.f}, by = {0.f, 0.f}, bz = {0.f, 0.f};
  float2 w[6] = {{0.f, 0.f}, {0.f, 0.f}, {0.f, 0.f}, {0.f, 0.f}, {0.f, 0.f}, {0.f, 0.f}};
};

// how a range of candidates is accumulated
constexpr int kDrainHits = 4;     // fp64 drain: hits per lane and round
constexpr int kPairPlain = 0;     // unshifted: force sums a
constexpr int kPairImage = 1;     // periodic images: force sums b + pair virial w
constexpr int kPairImageF = 2;    // periodic images, forces only (their virial is taken from the other end)

// one full interaction in precision T (scalar path: fp64 drain, minimum-image instances)
template <typename T, int P, int MODE>
__device__ __forceinline__ void pair_interact(PairAcc<T>& A, T dx, T dy, T dz, T r2, T qj, T inv_a, T inv_a2,
                                              const T (&cf)[P], const T (&cds)[P]) {   // cds = 2/a^3 * cd
  const T rinv = rsqrt_fast(r2);
  const T s = fma(r2, inv_a2, (T)-1);
  T g = cf[P - 1], dg = cds[P - 1];
#pragma unroll
  for (int k = P - 2; k >= 0; --k) g = fma(g, s, cf[k]);
#pragma unroll
  for (int k = P - 2; k >= 1; --k) dg = fma(dg, s, cds[k]);
  A.av = fma(qj, fma(-g, inv_a, rinv), A.av);
  const T fs = qj * fma(rinv * rinv, rinv, dg);
  if (MODE == kPairImage) {
    const T fx = fs * dx, fy = fs * dy, fz = fs * dz;
    A.bx = fma(fs, dx, A.bx); A.by = fma(fs, dy, A.by); A.bz = fma(fs, dz, A.bz);   // as in kPairImageF
    A.w[0] = fma(fx, dx, A.w[0]); A.w[1] = fma(fy, dy, A.w[1]); A.w[2] = fma(fz, dz, A.w[2]);
    A.w[3] = fma(fx, dy, A.w[3]); A.w[4] = fma(fx, dz, A.w[4]); A.w[5] = fma(fy, dz, A.w[5]);
  } else if (MODE == kPairImageF) {
    A.bx = fma(fs, dx, A.bx); A.by = fma(fs, dy, A.by); A.bz = fma(fs, dz, A.bz);
  } else {
    A.ax = fma(fs, dx, A.ax); A.ay = fma(fs, dy, A.ay); A.az = fma(fs, dz, A.az);
  }
}

template <typename T, int P, bool VIRIAL, bool MI>
__global__ void __launch_bounds__(PairWarps<T>::value * 32, sizeof(T) == 4 ? 6 : 8)
k_pair(PairParams<T> prm, const int* __restrict__ pstart, const typename Vec4<T>::type* __restrict__ prec,
       const int* __restrict__ pbinx, const int* __restrict__ porder, T* __restrict__ Fsr,
       T* __restrict__ Vsr, double* __restrict__ wpart) {
  using V4 = typename Vec4<T>::type;
  constexpr int CAP = PairStage<T>::kCap;
  constexpr int kPairWarps = PairWarps<T>::value;
  constexpr bool kPacked = sizeof(T) == 4 && !MI;     // fp32: brute force with packed arithmetic
  constexpr bool kLists = sizeof(T) == 8 && !MI;      // fp64: fp32 scan + hit lists + fp64 drain
  // the candidate list has four regions (own-row images, images above, images below, unshifted),
  // with or without the virial (same summation order, so the forces do not depend on whether the
  // virial is asked for); the minimum-image instances have just one
  constexpr bool kSplit = !MI;
  __shared__ PairStage<T> stage[kPairWarps];
  const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
  const int il = lane & (kPairCluster - 1), jq = lane / kPairCluster;   // i-particle and candidate phase of this lane
  const int l8 = lane & 7;                          // staging: eight lanes per neighbour row
  PairStage<T>& sj = stage[wid];
  const int row = blockIdx.x;                       // (cy, cz); blockIdx.y strides over the row's clusters
  const int cy = row % prm.nc[1], cz = row / prm.nc[1];
  const int sxs = prm.sxs;
  const int nbx = prm.nc[0] << sxs;                 // sub-bins per row
  const int row_s = pstart[row * nbx], row_e = pstart[(row + 1) * nbx];
  const int ntile = (row_e - row_s + kPairCluster - 1) / kPairCluster;
  const bool mix = MI && prm.minimg[0] != 0, miy = MI && prm.minimg[1] != 0, miz = MI && prm.minimg[2] != 0;
  // a cluster pass may span at most span_max sub-bins beyond its first one, so that its widest
  // window never overlaps itself on a periodic axis and stays short
  const int wmax = prm.wb[0][0];
  const int span_max = prm.periodic[0] && !mix ? max(min(nbx - 2 * wmax - 1, kPairSpanCap << sxs), 0)
                                               : (kPairSpanCap << sxs);
  const T a2 = prm.a2, inv_a = prm.inv_a, inv_a2 = prm.inv_a2, two_inv_a3 = prm.two_inv_a3;
  const float a2_scan = prm.a2_scan;
  T cf[P], cd[P];                                   // g(s) = sum cf[k] s^k, g'(s) = sum cd[k] s^(k-1)
#pragma unroll
  for (int k = 0; k < P; ++k) { cf[k] = prm.c[k]; cd[k] = (T)k * prm.c[k]; }
  T cds[P];                                         // 2/a^3 g'(s): one multiply less per pair
#pragma unroll
  for (int k = 0; k < P; ++k) cds[k] = two_inv_a3 * cd[k];
  double W[6] = {0, 0, 0, 0, 0, 0};

  // the neighbour rows of this block: lane r describes row r.
  //   class 1 (r = 0): the cluster's own row;  class 2: rows above (dz > 0, or dz = 0 and dy > 0);
  //   class 3: rows below. Minimum-image instances (fewer than 5 cells on a periodic axis: offsets
  //   alias) put every row into class 1. my_wrap: the row is reached across a periodic box face.
  const int ny_off = prm.omax[1] - prm.omin[1] + 1, nz_off = prm.omax[2] - prm.omin[2] + 1;
  const int nrows = ny_off * nz_off;                // <= 25
  int my_dy = 0, my_dz = 0, my_class = 0, my_rowbase = 0, my_wb = 0;   // class 0: row absent
  bool my_wrap = false;
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
    if (cyj < 0 || cyj >= prm.nc[1]) { if (prm.periodic[1]) { cyj = imod(cyj, prm.nc[1]); my_wrap = true; } else my_class = 0; }
    if (czj < 0 || czj >= prm.nc[2]) { if (prm.periodic[2]) { czj = imod(czj, prm.nc[2]); my_wrap = true; } else my_class = 0; }
    my_rowbase = (czj * prm.nc[1] + cyj) * nbx;
    my_wb = MI ? wmax : prm.wb[min(abs(my_dy), 2)][min(abs(my_dz), 2)];
    if (my_wb < 0) my_class = 0;                    // the cutoff sphere does not reach this row
  }
  const int r0 = MI ? (-prm.omin[1]) + (-prm.omin[2]) * ny_off : 0;   // lane of the cluster's own row

  for (int tile = blockIdx.y * kPairWarps + wid; tile < ntile; tile += kPairWarps * gridDim.y) {
    const int k0 = row_s + tile * kPairCluster;     // first sorted particle of the cluster
    const int ki = k0 + il;
    const bool inrow = ki < row_e;
    V4 ri = make_vec4<T>(0, 0, 0, 0);
    int bxi = 0;                                    // sub-bin of the particle along x
    if (inrow) { ri = ldg4(prec + ki); bxi = pbinx[ki]; }
    const int last = min(kPairCluster - 1, row_e - 1 - k0);
   // passes: consecutive particles whose sub-bins span at most span_max (one pass unless the row is sparse)
   for (int first = 0; first <= last;) {
    const int fp0 = first;
    const int binf = __shfl_sync(0xffffffffu, bxi, first);
    const unsigned fits = __ballot_sync(0xffffffffu, inrow && il >= first && bxi - binf <= span_max) & ((1u << kPairCluster) - 1u);
    const int sub_last = 31 - __clz((int)fits);            // sub-bins ascend with il
    const bool iv = il >= first && il <= sub_last;
    const int binl = __shfl_sync(0xffffffffu, bxi, sub_last);
    first = sub_last + 1;
    const int cxf = binf >> sxs;                            // the frame: first particle's cell
    const T xi = ri.x + (T)((bxi >> sxs) - cxf) * prm.edge[0], yi = ri.y, zi = ri.z;
    // this lane's row: its x window in unwrapped sub-bins, as up to two contiguous segments of the
    // sorted order (A: unshifted, B: through the periodic wrap in x)
    int sA = 0, lA = 0, sB = 0, lB = 0, shB = 0;
    if (my_class != 0) {
      int xa = binf - my_wb, xb = binl + my_wb;
      if (!prm.periodic[0]) { xa = max(xa, 0); xb = min(xb, nbx - 1); }
      else if (mix) { xa = 0; xb = nbx - 1; }               // fewer than 5 cells: each once + min. image
      const int ca = max(xa, 0), cb = min(xb, nbx - 1);
      if (ca <= cb) { sA = pstart[my_rowbase + ca]; lA = pstart[my_rowbase + cb + 1] - sA; }
      if (xa < 0) { sB = pstart[my_rowbase + xa + nbx]; lB = pstart[my_rowbase + nbx] - sB; shB = -prm.nc[0]; }
      else if (xb >= nbx) { sB = pstart[my_rowbase]; lB = pstart[my_rowbase + xb - nbx + 1] - sB; shB = prm.nc[0]; }
    }
    // Flat candidate list. kSplit: region 0 = images in the own row (x wrap), 1 = images in rows
    // above, 2 = images in rows below, 3 = unshifted candidates; each region is padded to a multiple
    // of 8 so that a step never straddles two regions. Otherwise everything is in region 3.
    const bool wrapA = kSplit && my_wrap;
    int n0 = 0, n1 = 0, n2 = 0, n3 = 0;                     // this lane's contribution to the regions
    if (kSplit) {
      if (my_class == 1) n0 = lB;
      else if (my_class == 2) n1 = lB + (wrapA ? lA : 0);
      else if (my_class == 3) n2 = lB + (wrapA ? lA : 0);
      if (!wrapA) n3 = lA;
    } else {
      n3 = lA + lB;
    }
    int i1 = n1, i2 = n2, i3 = n3;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
      const int t1 = __shfl_up_sync(0xffffffffu, i1, o), t2 = __shfl_up_sync(0xffffffffu, i2, o);
      const int t3 = __shfl_up_sync(0xffffffffu, i3, o);
      if (lane >= o) { i1 += t1; i2 += t2; i3 += t3; }
    }
    // raw ends e_k and padded ends b_k of the regions
    const int e0 = __shfl_sync(0xffffffffu, n0, 0), b0 = (e0 + 7) & ~7;
    const int e1 = b0 + __shfl_sync(0xffffffffu, i1, 31), b1 = (e1 + 7) & ~7;
    const int e2 = b1 + __shfl_sync(0xffffffffu, i2, 31), b2 = (e2 + 7) & ~7;
    const int e3 = b2 + __shfl_sync(0xffffffffu, i3, 31), total = (e3 + 7) & ~7;
    int offA, offB;                                          // flat positions of this lane's segments
    if (kSplit) {
      const int img = my_class == 2 ? b0 + i1 - n1 : b1 + i2 - n2;   // start of this row among the images
      offA = wrapA ? img : b2 + i3 - n3;
      offB = my_class == 1 ? 0 : img + (wrapA ? lA : 0);
    } else {
      offA = b2 + i3 - n3;
      offB = offA + lA;
    }
    // flat positions of the active particles of the cluster (consecutive, in the own row's segment A)
    const int sA0 = __shfl_sync(0xffffffffu, sA, r0), lA0 = __shfl_sync(0xffffffffu, lA, r0);
    const int oA0 = __shfl_sync(0xffffffffu, offA, r0);
    const bool own_present = lA0 > 0;                        // (absent: the own row belongs to another split)
    const int sfirst = oA0 + (k0 + fp0 - sA0), slast = sfirst + (sub_last - fp0);
    const int selfpos = own_present ? sfirst + (il - fp0) : -(1 << 20);

    PairAcc<T> A;                       // scalar accumulators (fp64, minimum image)
    PairAcc2 A2;                        // packed accumulators (fp32)
    // an idle lane sits 64 cutoffs to the left, the pads 64 cutoffs to the right: neither ever
    // hits, and the softening polynomial of such a distance stays finite in fp32
    const T far = (T)64 * prm.a;
    const float xs = iv ? (float)xi : -(float)far, ys = (float)yi, zs = (float)zi;
    const int grp = lane >> 3;

    for (int base = 0; base < total; base += CAP) {
      const int hi = min(base + CAP, total);
      // ---- pads of the four regions
      {
        const int gs = grp == 0 ? e0 : grp == 1 ? e1 : grp == 2 ? e2 : e3;
        const int ge = grp == 0 ? b0 : grp == 1 ? b1 : grp == 2 ? b2 : total;
        const int pos = gs + l8;
        if (pos < ge && pos >= base && pos < hi) sj.put(pos - base, make_vec4<T>(far, 0, 0, 0));
      }
      // ---- stage: four rows at a time, eight lanes per row, into the cluster's frame
      for (int rr = 0; rr < nrows; rr += 4) {
        const int r = rr + grp;
        const T yoff = (T)__shfl_sync(0xffffffffu, my_dy, r) * prm.edge[1];
        const T zoff = (T)__shfl_sync(0xffffffffu, my_dz, r) * prm.edge[2];
        // elements [t0, t1) of a segment (source index s0, flat position o0, cell shift sh)
        auto stage_seg = [&](int s0, int len, int o0, int sh) {
          const int t1 = min(len, hi - o0);
          // four elements per lane and batch: all eight loads of a batch are issued before the
          // first store, so a batch costs one global-memory latency instead of four
#pragma unroll 1
          for (int tb = max(0, base - o0) + l8; tb < t1; tb += 32) {
            V4 rj[4];
            int cj[4];
#pragma unroll
            for (int k = 0; k < 4; ++k) {
              const int src = s0 + min(tb + 8 * k, t1 - 1);
              rj[k] = ldg4(prec + src);
              cj[k] = (pbinx[src] >> sxs) + sh - cxf;
            }
#pragma unroll
            for (int k = 0; k < 4; ++k) {
              const int t = tb + 8 * k;
              if (t < t1) {
                rj[k].x += (T)cj[k] * prm.edge[0];
                rj[k].y += yoff;
                rj[k].z += zoff;
                sj.put(o0 + t - base, rj[k]);
              }
            }
          }
        };
        stage_seg(__shfl_sync(0xffffffffu, sA, r), __shfl_sync(0xffffffffu, lA, r), __shfl_sync(0xffffffffu, offA, r), 0);
        const int lb = __shfl_sync(0xffffffffu, lB, r);
        if (__any_sync(0xffffffffu, lb > 0))
          stage_seg(__shfl_sync(0xffffffffu, sB, r), lb, __shfl_sync(0xffffffffu, offB, r), __shfl_sync(0xffffffffu, shB, r));
      }
      __syncwarp();

      // ---- candidates [lo, hi2) of the flat list (multiples of 8) against the cluster's particles.
      // MODE: kPairPlain / kPairImage / kPairImageF; SELF: the range may hold the cluster's own
      // particles (index test)
      auto run = [&](int lo, int hi2, auto modec, auto selfc) {
        constexpr int MODE = decltype(modec)::value;
        constexpr bool SELF = decltype(selfc)::value;
        const int nsteps = (hi2 - lo) / kPairStep;
        if (nsteps <= 0) return;
        if constexpr (kPacked) {
          const float ia2 = (float)inv_a2, nia = -(float)inv_a;
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
            float2 qj;
            if (SELF) {
              qj = make_float2((r2.x < a2_scan && jdx != 0) ? zq.z : 0.f, (r2.y < a2_scan && jdx != -1) ? zq.w : 0.f);
              jdx += kPairStep;
            } else {
              qj = make_float2(r2.x < a2_scan ? zq.z : 0.f, r2.y < a2_scan ? zq.w : 0.f);
            }
            const float2 rinv = make_float2(rsqrt_fast(r2.x), rsqrt_fast(r2.y));
            const float2 sv = __ffma2_rn(r2, make_float2(ia2, ia2), make_float2(-1.f, -1.f));
            float2 g = make_float2((float)cf[P - 1], (float)cf[P - 1]), dg = make_float2((float)cds[P - 1], (float)cds[P - 1]);
#pragma unroll
            for (int k = P - 2; k >= 0; --k) g = __ffma2_rn(g, sv, make_float2((float)cf[k], (float)cf[k]));
#pragma unroll
            for (int k = P - 2; k >= 1; --k) dg = __ffma2_rn(dg, sv, make_float2((float)cds[k], (float)cds[k]));
            A2.av = __ffma2_rn(qj, __ffma2_rn(g, make_float2(nia, nia), rinv), A2.av);
            const float2 fs = __fmul2_rn(qj, __ffma2_rn(__fmul2_rn(rinv, rinv), rinv, dg));   // dg carries 2/a^3
            if (MODE == kPairImage) {
              const float2 fx = __fmul2_rn(fs, dx), fy = __fmul2_rn(fs, dy), fz = __fmul2_rn(fs, dz);
              A2.bx = __ffma2_rn(fs, dx, A2.bx); A2.by = __ffma2_rn(fs, dy, A2.by); A2.bz = __ffma2_rn(fs, dz, A2.bz);
              A2.w[0] = __ffma2_rn(fx, dx, A2.w[0]); A2.w[1] = __ffma2_rn(fy, dy, A2.w[1]); A2.w[2] = __ffma2_rn(fz, dz, A2.w[2]);
              A2.w[3] = __ffma2_rn(fx, dy, A2.w[3]); A2.w[4] = __ffma2_rn(fx, dz, A2.w[4]); A2.w[5] = __ffma2_rn(fy, dz, A2.w[5]);
            } else if (MODE == kPairImageF) {
              A2.bx = __ffma2_rn(fs, dx, A2.bx); A2.by = __ffma2_rn(fs, dy, A2.by); A2.bz = __ffma2_rn(fs, dz, A2.bz);
            } else {
              A2.ax = __ffma2_rn(fs, dx, A2.ax); A2.ay = __ffma2_rn(fs, dy, A2.ay); A2.az = __ffma2_rn(fs, dz, A2.az);
            }
            fp += 4 * kPairStep;
          }
        } else if constexpr (kLists) {
          // scan: packed fp32 distance test of this lane's candidate pairs, hits appended to its list
          unsigned char* const lp = sj.list + lane;
          unsigned char* le = lp;
          {
            const float2 xi2 = make_float2(xs, xs), yi2 = make_float2(ys, ys), zi2 = make_float2(zs, zs);
            const float* fp = sj.f + (lo - base) * 4 + jq * 8;
            int idx = lo - base + 2 * jq;                   // index inside the chunk
            const int selfl = SELF ? selfpos - base : -1;
            for (int s = 0; s < nsteps; ++s) {
              const float4 xy = *reinterpret_cast<const float4*>(fp);
              const float2 zz = *reinterpret_cast<const float2*>(fp + 4);
              const float2 dx = __fadd2_rn(xi2, make_float2(-xy.x, -xy.y));
              const float2 dy = __fadd2_rn(yi2, make_float2(-xy.z, -xy.w));
              const float2 dz = __fadd2_rn(zi2, make_float2(-zz.x, -zz.y));
              const float2 r2 = __ffma2_rn(dx, dx, __ffma2_rn(dy, dy, __fmul2_rn(dz, dz)));
              if (r2.x < a2_scan && idx != selfl) { *le = (unsigned char)idx; le += 32; }
              if (r2.y < a2_scan && idx + 1 != selfl) { *le = (unsigned char)(idx + 1); le += 32; }
              fp += 4 * kPairStep;
              idx += kPairStep;
            }
          }
          const int n = (int)(le - lp) >> 5;                    // hits of this lane
          int nmax = n;
#pragma unroll
          for (int o = 16; o > 0; o >>= 1) nmax = max(nmax, __shfl_xor_sync(0xffffffffu, nmax, o));
          __syncwarp();
          // drain: hit r of every lane that has one, in full precision (exact cutoff test)
          // kDrainHits hits per lane and round, branch-free (a missing hit or one outside the exact
          // cutoff takes charge 0 and squared distance 1, selected by the cutoff predicate: no second
          // fp64 compare), so that their dependent chains of ~40 DFMA interleave instead of running
          // one after the other (N = 10^6: 2 hits 2.93 ms, 3 hits 2.89, 4 hits 2.85, 6 hits 3.10
          // with spills; the select instead of max(r2, tiny): 2.81).
          for (int r = 0; r < nmax; r += kDrainHits) {
            V4 pj[kDrainHits];
            T ddx[kDrainHits], ddy[kDrainHits], ddz[kDrainHits], ss[kDrainHits], qq[kDrainHits];
#pragma unroll
            for (int h = 0; h < kDrainHits; ++h) pj[h] = sj.full(r + h < n ? lp[(r + h) * 32] : 0);
#pragma unroll
            for (int h = 0; h < kDrainHits; ++h) {
              ddx[h] = xi - pj[h].x; ddy[h] = yi - pj[h].y; ddz[h] = zi - pj[h].z;
              ss[h] = fma(ddx[h], ddx[h], fma(ddy[h], ddy[h], ddz[h] * ddz[h]));
              const bool in = r + h < n && ss[h] < a2;
              qq[h] = in ? pj[h].w : (T)0;
              ss[h] = in ? ss[h] : (T)1;
            }
#pragma unroll
            for (int h = 0; h < kDrainHits; ++h)
              pair_interact<T, P, MODE>(A, ddx[h], ddy[h], ddz[h], ss[h], qq[h], inv_a, inv_a2,
                                        cf, cds);
          }
          __syncwarp();
        } else {
          // minimum-image instances (tiny periodic boxes): plain loop in precision T
          for (int s = 0; s < nsteps; ++s) {
#pragma unroll
            for (int h = 0; h < 2; ++h) {
              const int pos = lo + s * kPairStep + 2 * jq + h;
              const V4 pj = sj.full(pos - base);
              T dx = xi - pj.x, dy = yi - pj.y, dz = zi - pj.z;
              if (mix) dx -= prm.box[0] * rint(dx * prm.inv_box[0]);
              if (miy) dy -= prm.box[1] * rint(dy * prm.inv_box[1]);
              if (miz) dz -= prm.box[2] * rint(dz * prm.inv_box[2]);
              const T r2 = fma(dx, dx, fma(dy, dy, dz * dz));
              if (iv && pos < e3 && pos != selfpos && r2 < a2)
                pair_interact<T, P, MODE>(A, dx, dy, dz, r2, pj.w, inv_a, inv_a2, cf, cds);
            }
          }
        }
      };
      using Plain = std::integral_constant<int, kPairPlain>;
      using Image = std::integral_constant<int, kPairImage>;
      using ImageF = std::integral_constant<int, kPairImageF>;
      using Yes = std::true_type;
      using No = std::false_type;
      auto clampc = [&](int v) { return min(max(v, base), hi); };
      if (kSplit && !VIRIAL) {
        run(base, clampc(b2), ImageF(), No());
      } else if (kSplit) {
        run(base, clampc(b0), Image(), No());              // images in the own row
        if (b0 > base && b0 <= hi) {                       // done: both ends visit these pairs
          if constexpr (kPacked) {
#pragma unroll
            for (int k = 0; k < 6; ++k) { A2.w[k].x *= 0.5f; A2.w[k].y *= 0.5f; }
          } else {
#pragma unroll
            for (int k = 0; k < 6; ++k) A.w[k] *= (T)0.5;
          }
        }
        run(clampc(b0), clampc(b1), Image(), No());        // images above: weight 1
        run(clampc(b1), clampc(b2), ImageF(), No());       // images below: forces only
      }
      {
        // unshifted candidates (everything when the list has one region); only the one or two
        // steps around the cluster's own particles need the index test
        const int lo3 = kSplit ? clampc(b2) : base;
        if (MI && VIRIAL) {
          run(lo3, hi, Image(), Yes());
        } else if (own_present) {
          const int s0 = min(max(sfirst & ~7, lo3), hi), s1 = min(max((slast & ~7) + 8, lo3), hi);
          run(lo3, s0, Plain(), No());
          run(s0, s1, Plain(), Yes());
          run(s1, hi, Plain(), No());
        } else {
          run(lo3, hi, Plain(), No());
        }
      }
      __syncwarp();
    }
    if constexpr (kPacked) {
      A.ax = A2.ax.x + A2.ax.y; A.ay = A2.ay.x + A2.ay.y; A.az = A2.az.x + A2.az.y; A.av = A2.av.x + A2.av.y;
      A.bx = A2.bx.x + A2.bx.y; A.by = A2.by.x + A2.by.y; A.bz = A2.bz.x + A2.bz.y;
#pragma unroll
      for (int k = 0; k < 6; ++k) A.w[k] = A2.w[k].x + A2.w[k].y;
    }
    const T qi = ri.w;
    if (VIRIAL && iv) {
      const double dq = (double)qi;
      if (MI) {                                           // every pair is visited from both ends
#pragma unroll
        for (int k = 0; k < 6; ++k) W[k] += 0.5 * dq * (double)A.w[k];
      } else {
        // image pairs (counted once, see above) + this lane's share of F_i (x) r_i for the rest
#pragma unroll
        for (int k = 0; k < 6; ++k) W[k] += dq * (double)A.w[k];
        // (positions from the box centre: sum F_i = 0 only up to rounding, and what is left of it
        // is weighted by |r_i|)
        const double rx = (double)ri.x + ((double)(bxi >> sxs) - 0.5 * (double)prm.nc[0]) * prm.edge_d[0];
        const double ry = (double)ri.y + ((double)cy - 0.5 * (double)prm.nc[1]) * prm.edge_d[1];
        const double rz = (double)ri.z + ((double)cz - 0.5 * (double)prm.nc[2]) * prm.edge_d[2];
        const double fx = dq * (double)A.ax, fy = dq * (double)A.ay, fz = dq * (double)A.az;
        W[0] += fx * rx; W[1] += fy * ry; W[2] += fz * rz;
        W[3] += 0.5 * (fx * ry + fy * rx); W[4] += 0.5 * (fx * rz + fz * rx); W[5] += 0.5 * (fy * rz + fz * ry);
      }
    }
    // total force factor sums; the phases of a particle, in a fixed order
    A.ax += A.bx; A.ay += A.by; A.az += A.bz;
#pragma unroll
    for (int o = kPairCluster; o < 32; o <<= 1) {
      A.ax += __shfl_xor_sync(0xffffffffu, A.ax, o); A.ay += __shfl_xor_sync(0xffffffffu, A.ay, o);
      A.az += __shfl_xor_sync(0xffffffffu, A.az, o); A.av += __shfl_xor_sync(0xffffffffu, A.av, o);
    }
    if (iv && jq == 0) {
      const int orig = porder[ki];
      T* Fp = Fsr + (size_t)blockIdx.z * 3 * prm.part_stride;   // partial of this split
      Fp[3 * (size_t)orig + 0] = qi * A.ax;
      Fp[3 * (size_t)orig + 1] = qi * A.ay;
      Fp[3 * (size_t)orig + 2] = qi * A.az;
      Vsr[(size_t)blockIdx.z * prm.part_stride + orig] = A.av;
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
