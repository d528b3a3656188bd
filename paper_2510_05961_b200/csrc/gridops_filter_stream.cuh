// gridops_filter_stream.cuh -- the omega' pre-filter of S5 (Eq. 20: K^l = omega' (x) omega'
// (x) omega' * s_l; the omega' factors are applied to the grid charge, see gridops.cuh) in ONE sweep:
// the grid charge crosses HBM once (read G_l, write the haloed copy) instead of once per axis.
//
//   pad[oz][oy][ox] = sum_{kx,ky,kz} w[kx] w[ky] w[kz] Q_logical[ox - Hx - kx][oy - Hy - ky][oz - Hz - kz]
//
// (logical index: wrapped on a periodic axis, zero outside an open one). The output is cut into
// columns of 16 output chunks (16 bytes each) x 32 output rows and segments of planes; a block
// marches along z through one segment of one column (gridDim = (columns, segments): the blocks
// resident at one time work on neighbouring columns at about the same z, so the halo re-reads hit
// the L2):
//  * the raw plane (tile + halo) goes global -> shared memory by cp.async two planes ahead (zero
//    fill outside an open axis; no registers held across the step),
//  * y: a thread filters 4 rows of one chunk column, shared -> shared (double buffered, so the y
//    pass of plane s + 1 and the x/z pass of plane s share one barrier interval),
//  * x: a thread filters its output chunk from 1 + 2 HC neighbouring chunks of its row,
//  * z: scatter form -- the x-y-filtered value is added to the NT output planes it feeds, held in a
//    register ring (slot = plane mod NT; a switch over plane mod NT makes every slot a fixed
//    register); the plane that just received its last contribution is stored.
// fp32: the y and z passes use packed fma.rn.f32x2 (SASS FFMA2, two results per instruction) on the
// two halves of a 16-byte chunk, the tap pair (w, w) coming straight from the constant bank.
// Requirements (checked by the host, which otherwise uses k_pad_filter_run): M_x and P_x multiples
// of the chunk, H_x a multiple of the chunk, NT in {11, 13, 15}.
#pragma once
#include "gridops_stream.cuh"

namespace msm {

struct FilterGeom {
  int M[3];          // grid dims (input)
  int P[3];          // padded dims (output)
  int H[3];          // output index o <-> logical node o - H
  int per[3];
  int ntx;           // columns along x (gridDim.x = columns in all)
  int zseg;          // output planes per block (gridDim.y segments)
};
struct FilterTaps2 {      // tap pairs of the packed fp32 passes
  float2 c[15];           // (w[n], w[n])
  float2 x[16];           // (w[k - 1], w[k]), zero outside the mask
};

constexpr int kFilterTXC = 16;     // output chunks per tile row
constexpr int kFilterCYY = 4;      // rows per thread in the y pass

template <typename T, int NT, int TY> constexpr size_t filter_stream_smem() {   // TY = output rows per tile
  constexpr int VE = VecT<T>::VE, HW = NT / 2, HC = (HW + VE - 1) / VE;
  return (size_t)(2 * (TY + 2 * HW) + 2 * TY) * (kFilterTXC + 2 * HC) * VE * sizeof(T);
}

__device__ __forceinline__ unsigned long long f2_pack(float a, float b) {
  unsigned long long r;
  asm("mov.b64 %0, {%1, %2};" : "=l"(r) : "f"(a), "f"(b));
  return r;
}
__device__ __forceinline__ unsigned long long f2_pack(float2 a) { return f2_pack(a.x, a.y); }
__device__ __forceinline__ float2 f2_unpack(unsigned long long v) {
  float2 r;
  asm("mov.b64 {%0, %1}, %2;" : "=f"(r.x), "=f"(r.y) : "l"(v));
  return r;
}
__device__ __forceinline__ void f2_fma(unsigned long long& acc, unsigned long long a, unsigned long long b) {
  asm("fma.rn.f32x2 %0, %1, %2, %0;" : "+l"(acc) : "l"(a), "l"(b));
}

// Accumulator of one chunk: VE scalars (fp64) or two packed pairs (fp32)
template <typename T> struct ChunkAcc;
template <> struct ChunkAcc<double> {
  double v[2];
  __device__ __forceinline__ void zero() { v[0] = v[1] = 0.0; }
  __device__ __forceinline__ void fma_tap(const AxisTaps<double>& w, const FilterTaps2&, int n, const ChunkAcc& r) {
    v[0] = fma(w.c[n], r.v[0], v[0]); v[1] = fma(w.c[n], r.v[1], v[1]);
  }
  __device__ __forceinline__ void load(const double* p) { const double2 t = *reinterpret_cast<const double2*>(p); v[0] = t.x; v[1] = t.y; }
  __device__ __forceinline__ void store(double* p) const { *reinterpret_cast<double2*>(p) = make_double2(v[0], v[1]); }
  // x pass: outputs (2 H, 2 H + 1) of the chunk += (w[n], w[n + 1]) r
  template <int H, int NT> __device__ __forceinline__ void fma_x(const AxisTaps<double>& w, const FilterTaps2&, int n, double r) {
    if (n >= 0 && n < NT) v[0] = fma(w.c[n], r, v[0]);
    if (n + 1 >= 0 && n + 1 < NT) v[1] = fma(w.c[n + 1], r, v[1]);
  }
};
template <> struct ChunkAcc<float> {
  unsigned long long v[2];
  __device__ __forceinline__ void zero() { v[0] = v[1] = 0ull; }
  __device__ __forceinline__ void fma_tap(const AxisTaps<float>&, const FilterTaps2& w2, int n, const ChunkAcc& r) {
    const unsigned long long wp = f2_pack(w2.c[n]);
    f2_fma(v[0], wp, r.v[0]); f2_fma(v[1], wp, r.v[1]);
  }
  __device__ __forceinline__ void load(const float* p) {
    const float4 t = *reinterpret_cast<const float4*>(p);
    v[0] = f2_pack(t.x, t.y); v[1] = f2_pack(t.z, t.w);
  }
  __device__ __forceinline__ void store(float* p) const {
    const float2 a = f2_unpack(v[0]), b = f2_unpack(v[1]);
    *reinterpret_cast<float4*>(p) = make_float4(a.x, a.y, b.x, b.y);
  }
  // x pass: outputs (2 H, 2 H + 1) of the chunk += (w[n], w[n + 1]) r (r as broadcast operand)
  template <int H, int NT> __device__ __forceinline__ void fma_x(const AxisTaps<float>&, const FilterTaps2& w2, int n, float r) {
    if (n >= -1 && n < NT) f2_fma(v[H], f2_pack(w2.x[n + 1]), f2_pack(r, r));
  }
};

// z pass of one plane whose index is SS mod NT: add to the ring, store and clear the finished slot
template <int SS, typename T, int NT, int RY>
__device__ __forceinline__ void filter_zstep(ChunkAcc<T> (&acc)[NT][RY], const ChunkAcc<T> (&v)[RY], const AxisTaps<T>& w,
                                             const FilterTaps2& w2, T* const (&optr)[RY], const bool (&emit)[RY]) {
#pragma unroll
  for (int q = 0; q < RY; ++q) {
#pragma unroll
    for (int n = 0; n < NT; ++n) acc[(SS + n) % NT][q].fma_tap(w, w2, n, v[q]);
    if (emit[q]) acc[SS % NT][q].store(optr[q]);
    acc[SS % NT][q].zero();
  }
}

template <typename T, int NT, int MINB, int TY>
__global__ void __launch_bounds__(kStreamThreads, MINB)
k_pad_filter_stream(FilterGeom g, AxisTaps<T> w, FilterTaps2 w2, const T* __restrict__ in, T* __restrict__ out) {
  using V = typename VecT<T>::type;
  using CA = ChunkAcc<T>;
  constexpr int VE = VecT<T>::VE, HW = NT / 2, HC = (HW + VE - 1) / VE;
  constexpr int TXC = kFilterTXC, CYY = kFilterCYY;
  constexpr int RC = TXC + 2 * HC;               // raw chunks per row
  constexpr int RW = RC * VE;                    // raw row length
  constexpr int NR = TY + 2 * HW;                // raw rows
  constexpr int NLD = (RC * NR + kStreamThreads - 1) / kStreamThreads;
  constexpr int RY = TXC * TY / kStreamThreads;   // output rows per thread in the x/z pass
  static_assert(TXC * TY == kStreamThreads * RY && RY >= 1, "tile shape");
  static_assert(RC * (TY / CYY) <= kStreamThreads, "one y-pass item per thread");
  static_assert(NT <= 15, "switch over the ring slots");
  extern __shared__ __align__(16) unsigned char filter_smem[];
  T* const RAW = reinterpret_cast<T*>(filter_smem);            // [2][NR][RW]
  T* const YF = RAW + 2 * NR * RW;                             // [2][TY][RW]

  const int tid = threadIdx.x;
  const size_t iplane = (size_t)g.M[0] * g.M[1], oplane = (size_t)g.P[0] * g.P[1];
  const int tx = blockIdx.x % g.ntx, ty = blockIdx.x / g.ntx;
  const int xc0 = tx * TXC, oy0 = ty * TY;
  const int oz0 = blockIdx.y * g.zseg, nz = min(g.zseg, g.P[2] - oz0);
  const int S = nz + 2 * HW;                     // steps: raw planes oz0 - Hz - HW + s

  // this thread's raw chunks: element offset inside a plane and copy size (0: zero fill)
  unsigned roff[NLD];
  int rsz[NLD];
#pragma unroll
  for (int n = 0; n < NLD; ++n) {
    const int i = tid + kStreamThreads * n;
    const int r = i / RC, c = i - r * RC;
    int gx = VE * (xc0 + c - HC) - g.H[0], gy = oy0 - g.H[1] - HW + r;
    bool ok = i < RC * NR;
    if (g.per[0]) gx = imod(gx, g.M[0]); else ok = ok && gx >= 0 && gx < g.M[0];
    if (g.per[1]) gy = imod(gy, g.M[1]); else ok = ok && gy >= 0 && gy < g.M[1];
    roff[n] = ok ? (unsigned)(gy * g.M[0] + gx) : 0u;
    rsz[n] = ok ? 16 : 0;
  }
  int gz_next = oz0 - g.H[2] - HW;               // logical plane of the next fetch
  if (g.per[2]) gz_next = imod(gz_next, g.M[2]);
  auto fetch = [&](int s) {                      // raw plane of step s into RAW[s & 1]; always commits a group
    if (s < S) {
      const bool zok = gz_next >= 0 && gz_next < g.M[2];
      const T* base = zok ? in + (size_t)gz_next * iplane : in;
      T* dst = RAW + (s & 1) * NR * RW + tid * VE;
#pragma unroll
      for (int n = 0; n < NLD; ++n)
        if (tid + kStreamThreads * n < RC * NR) cp_async16(dst + kStreamThreads * n * VE, base + roff[n], zok ? rsz[n] : 0);
      if (++gz_next == g.M[2] && g.per[2]) gz_next = 0;
    }
    cp_async_commit();
  };
  // y pass item: chunk column ycol, rows CYY * yq .. + CYY - 1:
  // YF[s & 1][q][c] = sum_n w[n] RAW[s & 1][q + NT - 1 - n][c]
  const int ycol = tid % RC, yq = tid / RC;
  const bool yact = yq < TY / CYY;
  auto ypass = [&](int s) {
    if (!yact) return;
    const T* raw = RAW + (s & 1) * NR * RW + CYY * yq * RW + ycol * VE;
    CA o[CYY];
#pragma unroll
    for (int q = 0; q < CYY; ++q) o[q].zero();
#pragma unroll
    for (int j = 0; j < CYY + NT - 1; ++j) {
      CA r;
      r.load(raw + j * RW);
#pragma unroll
      for (int q = 0; q < CYY; ++q) {
        const int n = q + NT - 1 - j;
        if (n >= 0 && n < NT) o[q].fma_tap(w, w2, n, r);
      }
    }
    T* yf = YF + (s & 1) * TY * RW + CYY * yq * RW + ycol * VE;
#pragma unroll
    for (int q = 0; q < CYY; ++q) o[q].store(yf + q * RW);
  };

  // x/z pass item: output chunk xc, rows RY * xr, RY * xr + 1
  const int xc = tid % TXC, xr = tid / TXC;
  const bool xact = VE * (xc0 + xc) < g.P[0];
  unsigned ooff[RY];                             // offset of the thread's chunks inside an output plane
  bool oval[RY];
#pragma unroll
  for (int q = 0; q < RY; ++q) {
    const int oy = oy0 + RY * xr + q;
    oval[q] = xact && oy < g.P[1];
    ooff[q] = oval[q] ? (unsigned)(oy * g.P[0] + VE * (xc0 + xc)) : 0u;
  }
  T* obase = out + (size_t)oz0 * oplane;         // the plane that completes next
  CA acc[NT][RY];
#pragma unroll
  for (int d = 0; d < NT; ++d)
#pragma unroll
    for (int q = 0; q < RY; ++q) acc[d][q].zero();

  fetch(0);
  fetch(1);
  cp_async_wait<1>();
  __syncthreads();
  ypass(0);
  int ss = 0;                                    // s mod NT
  for (int s = 0; s < S; ++s) {
    cp_async_wait<0>();                          // raw plane s + 1 has landed
    __syncthreads();                             // ... for everyone; YF[s & 1] is complete
    fetch(s + 2);
    if (s + 1 < S) ypass(s + 1);
    // x: v[e] = sum_n w[n] row[VE xc + e + VE HC + HW - n]
    CA v[RY];
#pragma unroll
    for (int q = 0; q < RY; ++q) {
      const T* row = YF + (s & 1) * TY * RW + (RY * xr + q) * RW + xc * VE;
      v[q].zero();
#pragma unroll
      for (int c = 0; c < 2 * HC + 1; ++c) {
        if (VE * (c + 1) - 1 >= VE * HC - HW && VE * c <= VE - 1 + VE * HC + HW) {   // chunk holds needed values
          T r[VE];
          unpack(*reinterpret_cast<const V*>(row + c * VE), r);
#pragma unroll
          for (int i = 0; i < VE; ++i) {
            // output e takes tap n = e + VE HC + HW - (VE c + i)
            v[q].template fma_x<0, NT>(w, w2, VE * HC + HW - (VE * c + i), r[i]);
            if constexpr (VE == 4) v[q].template fma_x<1, NT>(w, w2, 2 + VE * HC + HW - (VE * c + i), r[i]);
          }
        }
      }
    }
    // z: into the ring; from step 2 HW on a plane is complete
    const bool zdone = s >= 2 * HW;
    T* st[RY];
    bool emit[RY];
#pragma unroll
    for (int q = 0; q < RY; ++q) { st[q] = obase + ooff[q]; emit[q] = zdone && oval[q]; }
    switch (ss) {
#define MSM_ZCASE(K) case K: if constexpr (K < NT) filter_zstep<K, T, NT, RY>(acc, v, w, w2, st, emit); break;
      MSM_ZCASE(0) MSM_ZCASE(1) MSM_ZCASE(2) MSM_ZCASE(3) MSM_ZCASE(4) MSM_ZCASE(5) MSM_ZCASE(6) MSM_ZCASE(7)
      MSM_ZCASE(8) MSM_ZCASE(9) MSM_ZCASE(10) MSM_ZCASE(11) MSM_ZCASE(12) MSM_ZCASE(13) MSM_ZCASE(14)
#undef MSM_ZCASE
    }
    if (++ss == NT) ss = 0;
    if (zdone) obase += oplane;
  }
}

}  // namespace msm
