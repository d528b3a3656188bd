// conv.cuh -- S5: per-level grid<->grid convolution with the truncated stencil of k_l
// (Eq. 11; stencil P:268 Eq. 20), FP-pipe bound, and the grid part of the virial (reading V).
//
// Formulation. K^l = omega'(x)omega'(x)omega' * s_l (Eq. 20) and convolution is associative, so
// e^l = s_l * qpad with qpad = omega'-filtered, haloed grid charge (gridops.cuh). s_l is non-zero
// only inside the cutoff ellipsoid (3-5x fewer taps than the folded K^l) and is even in n, so
// e_m = sum_n s(n) qpad[m + n]. The halo holds periodic images (as many wraps as the stencil
// needs) or zeros (open axes), so the kernels have no boundary logic.
//
// Work unit = one warp = one block: output tile x in [X, X+XT), y = Y + lane, z in [Z, Z+ZT) and a
// SLICE of the input z-planes. Each thread keeps XT*ZT accumulators in registers; the warp streams
// its input planes through shared memory; one plane feeds all ZT output planes (tap row
// dz = z_in - z_out), so a 16-byte shared-memory window load is amortised over up to 4*XT*ZT FMAs
// and every tap quad (one 16-byte broadcast load from the L1-resident table) feeds 4*XT FMAs.
// Stencil rows are stored as runs of 4-tap chunks covering only the ellipsoid; chunk tests are
// warp-uniform (no divergence). ONE launch covers every tiled level: a block finds its level from
// the unit ranges in the descriptor table, so the coarse levels (too small to fill 148 SMs on their
// own) run beside the finest one. Slicing the input planes gives the scheduler units of similar,
// small size; slice partials go to a scratch array and are summed in slice order by k_sum_slices
// (deterministic).
//
// MODE_VIRIAL computes the strain derivative of the level's energy: with the correlation
// C(n) = sum_m Q_m qpad[m + n] (even in n), W_ab ~ sum_n g(n) n_a n_b C(n), g = k_l'(r)/r. Only
// the half space n > 0 (lexicographic in z, y, x) is visited, with weight 2; per tap and output it
// costs one FMA (c_t = sum_i q_i win[i + t]) plus three per tap for the x-moments.
#pragma once
#include "device_common.cuh"

namespace msm {

constexpr int kMaxConvLevels = 16;
constexpr int kMaxConvSlices = 71;
constexpr int kMaxRowSlices = 6;     // small jobs: units per plane slice (by stencil rows)

struct ConvLevel {
  int M[3];        // output grid dims
  int P[3];        // padded input dims
  int R[3];        // stencil half-widths (y, z used as halo; x halo is X0)
  int X0;          // x halo, multiple of 4, >= R[0]
  int tiles[3];    // output tiles per axis
  int pitch;       // shared-memory row pitch in elements
  int ny;          // 2 R[1] + 1
  int nslices;     // potential kernel: slices of the 2 R[2] + ZT input planes
  int vslices;     // virial kernel: slices of the R[2] + ZT input planes with dz >= 0
  int ysl, vysl;   // small jobs: each plane slice is dealt to this many units by stencil rows (dy); nslices / vslices count them all
  unsigned char pb[kMaxConvSlices + 1];   // slice s covers input planes [pb[s], pb[s+1]) (balanced by taps)
  unsigned char vb[kMaxConvSlices + 1];
  int unit0, vunit0;          // first unit of this level in the potential / virial launch
  const int4* rows;           // (tap chunk offset, first chunk, last chunk, -) per (dz, dy)
  const int4* vrows;          // same for the half-space virial taps
  const void* staps;          // s_l in 4-tap chunks
  const int4* rows2;          // fp32 packed path: per (d, dy), d = -R[2] .. R[2]+1, rows d and d-1 merged
  const void* taps2;          // per chunk 8 floats: (s_d[t], s_{d-1}[t]) for the chunk's 4 taps
  int n_rows2, n_taps2q;      // entries of rows2; float4 quads of taps2 including the guard chunk in front
  int sunit0;                 // first unit of this level in the shared-table launch (multiple of kConvSW)
  const int4* elist;          // fp32 list-driven path: byte offsets of (window j * pitch + 4 c in the lane's rows, chunk of pair 0, of pair 1 in taps2)
  const int* ehead;           // [2 R[2] + 4][kConvListTypes + 1]: list bounds per input plane offset d0 = zr
  const void* vtaps;          // per chunk: 4 x 2g, 4 x 2g dx, 4 x 2g dx^2
  const int4* vrows2;         // fp32 packed virial: half-space rows d and d - 1 merged, d = 0 .. R[2]+1
  const void* vtaps2;         // per chunk 24 floats: for 2g, 2g dx, 2g dx^2: 4 taps x (row d, row d - 1)
  const int4* dlist;          // fp64 list-driven potential kernel: entry = 2 x int4 byte offsets (window, taps of planes 0 .. 3, -, -, -)
  const int* dhead;           // [2 R[2] + 4][kConvListTypes + 1]
  int n_stapsq, dsunit0;      // 16-byte quads of staps; first unit of this level in the fp64 list launch
  const int4* vlist;          // list-driven virial: byte offsets (window, chunk of pair 0, of pair 1 in vtaps2), dy as float bits
  const int* vhead;           // [R[2] + 4][kConvListTypes + 1]: list bounds per input plane offset zr
  int n_vtaps2q, vsunit0;     // float4 quads of vtaps2; first unit of this level in the list-driven virial launch
  const void* pad;            // omega'-filtered haloed grid charge
  const void* Q;              // grid charge (virial)
  void* out;                  // E^l if nslices == 1, else scratch [slice][z][y][x]
  double* wpart;              // virial partials, 6 per unit
};

constexpr int kConvListTypes = 7;   // both full | pair 0 full | pair 1 full | pair 0 lower, upper half | pair 1 lower, upper half
constexpr int kConvDW = 12;   // warps (units) per block of the fp64 list-driven potential kernel (one block per SM)
constexpr int kConvVW = 16;   // warps (units) per block of the list-driven virial kernel (one block per SM)
constexpr int kConvSW = 8;    // warps (units) per block of the shared-table convolution kernel

struct ConvTable {
  int nlev;
  int total_units, total_vunits, total_sunits, total_vsunits, total_dsunits;
  ConvLevel lev[kMaxConvLevels];
};

template <typename T> struct SmemVec;
template <> struct SmemVec<float> {
  static __device__ __forceinline__ void load4(const float* p, float (&v)[4]) {
    const float4 t = *reinterpret_cast<const float4*>(p);
    v[0] = t.x; v[1] = t.y; v[2] = t.z; v[3] = t.w;
  }
  static __device__ __forceinline__ void ldg(const float* p, float (&v)[4]) {
    const float4 t = __ldg(reinterpret_cast<const float4*>(p));
    v[0] = t.x; v[1] = t.y; v[2] = t.z; v[3] = t.w;
  }
  // streaming load that does not allocate in L1 (the L1 is kept for the tap tables)
  static __device__ __forceinline__ void ldcg(const float* p, float (&v)[4]) {
    const float4 t = __ldcg(reinterpret_cast<const float4*>(p));
    v[0] = t.x; v[1] = t.y; v[2] = t.z; v[3] = t.w;
  }
};
template <> struct SmemVec<double> {
  static __device__ __forceinline__ void load4(const double* p, double (&v)[4]) {
    const double2 a = *reinterpret_cast<const double2*>(p);
    const double2 b = *reinterpret_cast<const double2*>(p + 2);
    v[0] = a.x; v[1] = a.y; v[2] = b.x; v[3] = b.y;
  }
  static __device__ __forceinline__ void ldg(const double* p, double (&v)[4]) {
    const double2 a = __ldg(reinterpret_cast<const double2*>(p));
    const double2 b = __ldg(reinterpret_cast<const double2*>(p + 2));
    v[0] = a.x; v[1] = a.y; v[2] = b.x; v[3] = b.y;
  }
  static __device__ __forceinline__ void ldcg(const double* p, double (&v)[4]) {
    const double2 a = __ldcg(reinterpret_cast<const double2*>(p));
    const double2 b = __ldcg(reinterpret_cast<const double2*>(p + 2));
    v[0] = a.x; v[1] = a.y; v[2] = b.x; v[3] = b.y;
  }
};

// stage padded plane pz: rows Y .. Y+nrow-1, x X .. X+WX-1 (padded indices) into shared memory
template <typename T>
__device__ __forceinline__ void stage_plane(const ConvLevel& g, const T* __restrict__ qpad, T* plane, int pz,
                                            int X, int Y, int nrow, int WX, int lane) {
  const T* src = qpad + ((size_t)pz * g.P[1] + Y) * g.P[0] + X;
  const int vper = WX / 4, nvec = nrow * vper;
  __syncwarp();
  // asynchronous 16-byte copies: every load of the plane is in flight at once, no registers
  for (int v = lane; v < nvec; v += 32) {
    const int r = v / vper, cx = (v - r * vper) * 4;
    const T* s = src + (size_t)r * g.P[0] + cx;
    T* dst = plane + r * g.pitch + cx;
#pragma unroll
    for (int h = 0; h < (int)(4 * sizeof(T) / 16); ++h)
      cp_async16(reinterpret_cast<unsigned char*>(dst) + 16 * h, reinterpret_cast<const unsigned char*>(s) + 16 * h, 16);
  }
  cp_async_commit();
  cp_async_wait<0>();
  __syncwarp();
}

// The same plane through the bulk-copy engine (TMA, SASS UBLKCP): one cp.async.bulk per row of
// WX * 4 bytes (a multiple of 16, like every row's source and destination address), completion
// counted in bytes on the warp's own mbarrier. Two instructions per lane and plane instead of
// ~18 LDGSTS with their index arithmetic. `phase` is the barrier's parity, flipped per plane.
__device__ __forceinline__ void mbar_init(unsigned mbar) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], 1;" :: "r"(mbar) : "memory");
  asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
}
__device__ __forceinline__ void stage_plane_bulk(const ConvLevel& g, const float* __restrict__ qpad, unsigned plane_s,
                                                 unsigned mbar, unsigned& phase, int pz, int X, int Y, int nrow, int WX,
                                                 int lane) {
  const float* src = qpad + ((size_t)pz * g.P[1] + Y) * g.P[0] + X;
  __syncwarp();                                         // every lane is done reading the previous plane
  if (lane == 0)
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" :: "r"(mbar), "r"((unsigned)(nrow * WX * 4)) : "memory");
  __syncwarp();
  for (int r = lane; r < nrow; r += 32)
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                 :: "r"(plane_s + (unsigned)(r * g.pitch * 4)), "l"(src + (size_t)r * g.P[0]), "r"((unsigned)(WX * 4)), "r"(mbar)
                 : "memory");
  unsigned done;
  do {
    asm volatile("{\n .reg .pred p;\n mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n selp.u32 %0, 1, 0, p;\n}"
                 : "=r"(done) : "r"(mbar), "r"(phase) : "memory");
  } while (!done);
  phase ^= 1u;
}

struct ConvUnit {
  int lev, X, Y, Z, slice, local;
};

// input planes [p0, p1) and stencil rows [j0, j1) of slice `slice` (plane slices fastest)
struct SliceRange { int p0, p1, pstep, j0, j1; };   // planes p0, p0 + pstep, .. < p1
template <bool VIRIAL>
__device__ __forceinline__ SliceRange slice_range(const ConvLevel& g, int slice) {
  const int ysl = VIRIAL ? g.vysl : g.ysl;
  const int ps = (VIRIAL ? g.vslices : g.nslices) / ysl;
  const int s = slice % ps, y = slice / ps;
  SliceRange r;
  if (VIRIAL) {
    // the virial kernels deal the planes round-robin (equal taps and plane counts per slice)
    r.p0 = s; r.p1 = g.R[2] + 4; r.pstep = ps;
  } else {
    r.p0 = g.pb[s]; r.p1 = g.pb[s + 1]; r.pstep = 1;
  }
  r.j0 = y * g.ny / ysl;
  r.j1 = (y + 1) * g.ny / ysl;
  return r;
}

template <bool VIRIAL, int XT, int ZT>
__device__ __forceinline__ ConvUnit decode_unit(const ConvTable& tab, int u) {
  ConvUnit cu;
  int l = 0;
#pragma unroll 1
  for (int k = 1; k < tab.nlev; ++k)
    if (u >= (VIRIAL ? tab.lev[k].vunit0 : tab.lev[k].unit0)) l = k;
  const ConvLevel& g = tab.lev[l];
  int r = u - (VIRIAL ? g.vunit0 : g.unit0);
  cu.lev = l;
  cu.local = r;
  const int ns = VIRIAL ? g.vslices : g.nslices;
  cu.slice = r % ns; r /= ns;
  cu.X = (r % g.tiles[0]) * XT; r /= g.tiles[0];
  cu.Y = (r % g.tiles[1]) * 32;
  cu.Z = (r / g.tiles[1]) * ZT;
  return cu;
}

// Layout of a one-warp unit's shared memory in the generic (fp64) kernels: the input plane, then
// the row entries of the ZT stencil layers the plane feeds, then two buffers for the taps of one
// stencil row (all ZT layers). The table entries are copied with cp.async -- the next row's taps
// while the current row is computed -- so that no FMA waits for a global load and no registers
// are held for the prefetch.
struct ConvSmemLayout {
  int rows_off;      // byte offset of int4 srows[ZT][ny_max]
  int taps_off;      // byte offset of the two tap buffers
  int tapbuf;        // elements per tap buffer = ZT * tapk
  int tapk;          // elements per layer and buffer
};

// row entries of layers dz(k), k < ZT, of one plane; invalid layers are marked empty
template <int ZT, typename F>
__device__ __forceinline__ void stage_rows(int4* srows, const int4* __restrict__ rows, int ny, int lane, F layer_row0) {
  for (int i = lane; i < ZT * ny; i += 32) {
    const int k = i / ny, j = i - k * ny;
    const int r0 = layer_row0(k);                      // first entry of the layer in `rows`, or -1
    if (r0 >= 0) cp_async16(srows + i, rows + r0 + j, 16);
    else srows[i] = make_int4(0, 1, 0, 0);
  }
}

// taps of stencil row j (all layers) into buffer `buf`: EPC elements per chunk
template <typename T, int ZT, int EPC>
__device__ __forceinline__ void issue_row_taps(const int4* srows, int ny, int j, const T* __restrict__ taps, T* buf,
                                               int tapk, int lane) {
  constexpr int PPC = EPC * (int)sizeof(T) / 16;       // 16-byte pieces per chunk
#pragma unroll
  for (int k = 0; k < ZT; ++k) {
    const int4 e = srows[k * ny + j];
    const int np = (e.z - e.y + 1) * PPC;
    const unsigned char* src = reinterpret_cast<const unsigned char*>(taps + (size_t)e.x * EPC);
    unsigned char* dst = reinterpret_cast<unsigned char*>(buf + k * tapk);
    for (int q = lane; q < np; q += 32) cp_async16(dst + 16 * q, src + 16 * q, 16);
  }
  cp_async_commit();
}

// ---------------------------------------------------------------------------------- potential
template <typename T, int XT, int ZT>
__global__ void __launch_bounds__(32, sizeof(T) == 4 ? 16 : 12)
k_conv(const ConvTable* __restrict__ tabp, ConvSmemLayout sl) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  T* plane = reinterpret_cast<T*>(smem_raw);
  int4* srows = reinterpret_cast<int4*>(smem_raw + sl.rows_off);
  T* stap = reinterpret_cast<T*>(smem_raw + sl.taps_off);
  const ConvTable& tab = *tabp;
  const int lane = threadIdx.x;
  const ConvUnit cu = decode_unit<false, XT, ZT>(tab, blockIdx.x);
  const ConvLevel& g = tab.lev[cu.lev];
  const int X = cu.X, Y = cu.Y, Z = cu.Z;
  const int Ry = g.R[1], Rz = g.R[2];
  const int nrow = 32 + 2 * Ry;
  const int WX = XT + 2 * g.X0 + 4;
  const int ny = g.ny;
  const int4* __restrict__ rows = g.rows;
  const T* __restrict__ staps = reinterpret_cast<const T*>(g.staps);
  const T* __restrict__ qpad = reinterpret_cast<const T*>(g.pad);

  T acc[ZT][XT];
#pragma unroll
  for (int k = 0; k < ZT; ++k)
#pragma unroll
    for (int i = 0; i < XT; ++i) acc[k][i] = 0;

  const SliceRange sr = slice_range<false>(g, cu.slice);
  const int p0 = sr.p0, p1 = sr.p1;
  for (int pz = p0; pz < p1; ++pz) {
    const int zr = pz - Rz;              // input plane z = Z + zr
    stage_rows<ZT>(srows, rows, ny, lane, [&](int k) {
      const int dz = zr - k;
      return dz >= -Rz && dz <= Rz ? (dz + Rz) * ny : -1;
    });
    stage_plane<T>(g, qpad, plane, Z + pz, X, Y, nrow, WX, lane);     // commits and waits (the row entries too)
    issue_row_taps<T, ZT, 4>(srows, ny, sr.j0, staps, stap + (sr.j0 & 1) * sl.tapbuf, sl.tapk, lane);
    for (int dy = sr.j0 - Ry; dy < sr.j1 - Ry; ++dy) {
      const int j = dy + Ry;
      cp_async_wait<0>();                                  // this row's taps have landed
      __syncwarp();
      if (j + 1 < sr.j1) issue_row_taps<T, ZT, 4>(srows, ny, j + 1, staps, stap + ((j + 1) & 1) * sl.tapbuf, sl.tapk, lane);
      const T* tapb = stap + (j & 1) * sl.tapbuf;
      int4 re[ZT];
      int cl = 1 << 30, ch = -1;
#pragma unroll
      for (int k = 0; k < ZT; ++k) {
        re[k] = srows[k * ny + j];
        if (re[k].y <= re[k].z) { cl = min(cl, re[k].y); ch = max(ch, re[k].z); }
      }
      const T* srow = plane + (lane + dy + Ry) * g.pitch;
      for (int c = cl; c <= ch; ++c) {
        T win[XT + 4];
#pragma unroll
        for (int jj = 0; jj < XT + 4; jj += 4) {
          T t[4];
          SmemVec<T>::load4(srow + 4 * c + jj, t);
          win[jj] = t[0]; win[jj + 1] = t[1]; win[jj + 2] = t[2]; win[jj + 3] = t[3];
        }
        // all tap quads of this chunk are read before the first FMA (inactive rows read their
        // layer's first quad and do not use it)
        T tp[ZT][4];
        bool on[ZT];
#pragma unroll
        for (int k = 0; k < ZT; ++k) {
          on[k] = c >= re[k].y && c <= re[k].z;
          SmemVec<T>::load4(tapb + k * sl.tapk + (on[k] ? (c - re[k].y) * 4 : 0), tp[k]);
        }
#pragma unroll
        for (int k = 0; k < ZT; ++k) {
          if (on[k]) {
#pragma unroll
            for (int t = 0; t < 4; ++t)
#pragma unroll
              for (int i = 0; i < XT; ++i) acc[k][i] = fma(tp[k][t], win[i + t], acc[k][i]);
          }
        }
      }
      __syncwarp();                                        // the buffer is free for row dy + 2
    }
  }
  // outputs (slice partial or the final value)
  const int y = Y + lane;
  if (y < g.M[1]) {
    T* out = reinterpret_cast<T*>(g.out) + (size_t)cu.slice * g.M[0] * g.M[1] * g.M[2];
#pragma unroll
    for (int k = 0; k < ZT; ++k) {
      const int z = Z + k;
      if (z < g.M[2]) {
        T* dst = out + ((size_t)z * g.M[1] + y) * g.M[0] + X;
#pragma unroll
        for (int i = 0; i < XT; ++i)
          if (X + i < g.M[0]) dst[i] = acc[k][i];
      }
    }
  }
}

// ------------------------------------------------------------- potential, fp32 with packed FMAs
// Blackwell's fma.rn.f32x2 (SASS FFMA2) does two fp32 multiply-adds per instruction and lane at the
// same flop rate as FFMA, i.e. with half the issue slots -- and this kernel is bound by instruction
// issue (71 % of its instructions are FMAs). The pair is taken along z: the accumulators of output
// planes (2kp, 2kp+1) form one 64-bit register pair, the window value is the scalar (broadcast)
// operand, and the taps of the two stencil rows dz = d and d - 1 that feed those planes from one
// input plane are stored interleaved (taps2), so one FFMA2 replaces two FFMAs with no extra moves.
__device__ __forceinline__ unsigned long long pack2(float lo, float hi) {
  unsigned long long r;
  asm("mov.b64 %0, {%1, %2};" : "=l"(r) : "f"(lo), "f"(hi));
  return r;
}
__device__ __forceinline__ void unpack2(unsigned long long v, float& lo, float& hi) {
  asm("mov.b64 {%0, %1}, %2;" : "=f"(lo), "=f"(hi) : "l"(v));
}
// acc += s * pair (s broadcast to both halves; ptxas folds the duplicate into a scalar operand)
__device__ __forceinline__ void ffma2_bcast(unsigned long long& acc, float s, unsigned long long pair) {
  asm("fma.rn.f32x2 %0, %1, %2, %0;" : "+l"(acc) : "l"(pack2(s, s)), "l"(pair));
}

// One unit of the packed convolution. SM: the level's whole row and tap tables are in the block's
// shared memory; otherwise the warp stages the entries it needs row by row (see below).
template <int XT, bool SM>
__device__ __forceinline__ void conv_f2_unit(const ConvLevel& g, const ConvUnit& cu, const int4* rows2,
                                             const float4* taps2, float* plane, int lane,
                                             int4* wrows = nullptr, float* stap = nullptr,
                                             ConvSmemLayout sl = ConvSmemLayout()) {
  // SM: rows2 / taps2 are the block's shared-memory copies of the level's whole tables. Otherwise
  // (one-warp blocks, small jobs) they are the global tables: the warp copies the row entries of its
  // two merged layers to `wrows` with the plane and the taps of stencil row dy + 1 into one of the
  // two buffers of `stap` (cp.async) while row dy is computed.
  constexpr int ZP = 2;                               // two pairs of output planes
  const int X = cu.X, Y = cu.Y, Z = cu.Z;
  const int Ry = g.R[1], Rz = g.R[2];
  const int nrow = 32 + 2 * Ry;
  const int WX = XT + 2 * g.X0 + 4;
  const int ny = g.ny;
  const float* __restrict__ qpad = reinterpret_cast<const float*>(g.pad);

  unsigned long long acc[ZP][XT];                     // (plane 2kp, plane 2kp + 1) of output x + i
#pragma unroll
  for (int k = 0; k < ZP; ++k)
#pragma unroll
    for (int i = 0; i < XT; ++i) acc[k][i] = 0ull;

  const SliceRange sr = slice_range<false>(g, cu.slice);
  const int p0 = sr.p0, p1 = sr.p1;
  for (int pz = p0; pz < p1; ++pz) {
    const int zr = pz - Rz;                           // input plane z = Z + zr
    if (!SM)
      stage_rows<ZP>(wrows, rows2, ny, lane, [&](int k) {
        const int d = zr - 2 * k;
        return d >= -Rz && d <= Rz + 1 ? (d + Rz) * ny : -1;
      });
    stage_plane<float>(g, qpad, plane, Z + pz, X, Y, nrow, WX, lane);     // commits and waits
    if (!SM)
      issue_row_taps<float, ZP, 8>(wrows, ny, sr.j0, reinterpret_cast<const float*>(taps2), stap + (sr.j0 & 1) * sl.tapbuf, sl.tapk,
                                   lane);
    for (int dy = sr.j0 - Ry; dy < sr.j1 - Ry; ++dy) {
      const int jr = dy + Ry;
      const float* tapb = nullptr;
      if (!SM) {
        cp_async_wait<0>();                           // this row's taps have landed
        __syncwarp();
        if (jr + 1 < sr.j1)
          issue_row_taps<float, ZP, 8>(wrows, ny, jr + 1, reinterpret_cast<const float*>(taps2),
                                       stap + ((jr + 1) & 1) * sl.tapbuf, sl.tapk, lane);
        tapb = stap + (jr & 1) * sl.tapbuf;
      }
      int4 re[ZP];
      int cl = 1 << 30, ch = -1;
#pragma unroll
      for (int k = 0; k < ZP; ++k) {
        const int d = zr - 2 * k;                     // planes (2k, 2k+1) take stencil rows (d, d - 1)
        if (!SM) re[k] = wrows[k * ny + jr];
        else if (d >= -Rz && d <= Rz + 1) re[k] = rows2[(d + Rz) * ny + (dy + Ry)];
        else re[k] = make_int4(0, 0, -1, 0);          // empty
        if (re[k].y <= re[k].z) { cl = min(cl, re[k].y); ch = max(ch, re[k].z); }
      }
      const float* srow = plane + (lane + dy + Ry) * g.pitch;
      for (int c = cl; c <= ch; ++c) {
        float win[XT + 4];
#pragma unroll
        for (int j = 0; j < XT + 4; j += 4) {
          const float4 t = *reinterpret_cast<const float4*>(srow + 4 * c + j);
          win[j] = t.x; win[j + 1] = t.y; win[j + 2] = t.z; win[j + 3] = t.w;
        }
        float4 tq[ZP][2];
        bool on[ZP];
#pragma unroll
        for (int k = 0; k < ZP; ++k) {
          on[k] = c >= re[k].y && c <= re[k].z;
          // unconditional address (clamped into the row; an empty row reads the guard chunk in front
          // of the table), so the loads are not tied to the branch below
          const float4* tp = SM ? taps2 + (re[k].x + min(max(c, re[k].y), re[k].z) - re[k].y) * 2
                                : reinterpret_cast<const float4*>(tapb + k * sl.tapk + (on[k] ? (c - re[k].y) * 8 : 0));
          tq[k][0] = tp[0];
          tq[k][1] = tp[1];
        }
#pragma unroll
        for (int k = 0; k < ZP; ++k) {
          if (on[k]) {
            // the row's taps start / end inside a chunk: its empty 2-tap half is skipped
            // (re.w = first | last << 16 half-chunk that holds a tap; warp-uniform)
            const bool lo = 2 * c >= (re[k].w & 0xffff), hi = 2 * c + 1 <= (re[k].w >> 16);
            if (lo) {
              const unsigned long long t0 = pack2(tq[k][0].x, tq[k][0].y), t1 = pack2(tq[k][0].z, tq[k][0].w);
#pragma unroll
              for (int i = 0; i < XT; ++i) {
                ffma2_bcast(acc[k][i], win[i], t0);
                ffma2_bcast(acc[k][i], win[i + 1], t1);
              }
            }
            if (hi) {
              const unsigned long long t2 = pack2(tq[k][1].x, tq[k][1].y), t3 = pack2(tq[k][1].z, tq[k][1].w);
#pragma unroll
              for (int i = 0; i < XT; ++i) {
                ffma2_bcast(acc[k][i], win[i + 2], t2);
                ffma2_bcast(acc[k][i], win[i + 3], t3);
              }
            }
          }
        }
      }
    }
  }
  // outputs (slice partial or the final value)
  const int y = Y + lane;
  if (y < g.M[1]) {
    float* out = reinterpret_cast<float*>(g.out) + (size_t)cu.slice * g.M[0] * g.M[1] * g.M[2];
#pragma unroll
    for (int k = 0; k < ZP; ++k) {
      float* d0 = out + ((size_t)(Z + 2 * k) * g.M[1] + y) * g.M[0] + X;
      float* d1 = d0 + (size_t)g.M[1] * g.M[0];
      const bool z0 = Z + 2 * k < g.M[2], z1 = Z + 2 * k + 1 < g.M[2];
#pragma unroll
      for (int i = 0; i < XT; ++i) {
        float lo, hi;
        unpack2(acc[k][i], lo, hi);
        if (X + i < g.M[0]) {
          if (z0) d0[i] = lo;
          if (z1) d1[i] = hi;
        }
      }
    }
  }
}


template <int XT>
__global__ void __launch_bounds__(32, 16)
k_conv_f2(const ConvTable* __restrict__ tabp, ConvSmemLayout sl) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  const ConvTable& tab = *tabp;
  const ConvUnit cu = decode_unit<false, XT, 4>(tab, blockIdx.x);
  const ConvLevel& g = tab.lev[cu.lev];
  conv_f2_unit<XT, false>(g, cu, g.rows2, reinterpret_cast<const float4*>(g.taps2),
                          reinterpret_cast<float*>(smem_raw), threadIdx.x,
                          reinterpret_cast<int4*>(smem_raw + sl.rows_off), reinterpret_cast<float*>(smem_raw + sl.taps_off), sl);
}

// The same with the level's row and tap tables copied into shared memory once per block of kConvSW
// warps (one unit each, all of one level): a tap quad then costs a fixed-latency shared load instead
// of a global load that misses the L1 half of the time (30 % of the warp time of k_conv_f2).
template <int XT>
__global__ void __launch_bounds__(32 * kConvSW, 2)
k_conv_f2s(const ConvTable* __restrict__ tabp, int plane_bytes) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  const ConvTable& tab = *tabp;
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  int l = 0;
#pragma unroll 1
  for (int k = 1; k < tab.nlev; ++k)
    if ((int)blockIdx.x * kConvSW >= tab.lev[k].sunit0) l = k;
  const ConvLevel& g = tab.lev[l];
  float4* staps = reinterpret_cast<float4*>(smem_raw);
  int4* srows = reinterpret_cast<int4*>(staps + g.n_taps2q);
  float* planes = reinterpret_cast<float*>(srows + g.n_rows2);
  const float4* gt = reinterpret_cast<const float4*>(g.taps2) - 2;          // from the guard chunk on
  for (int i = threadIdx.x; i < g.n_taps2q; i += 32 * kConvSW) staps[i] = __ldg(gt + i);
  for (int i = threadIdx.x; i < g.n_rows2; i += 32 * kConvSW) srows[i] = __ldg(g.rows2 + i);
  __syncthreads();
  int r = (int)blockIdx.x * kConvSW + warp - g.sunit0;
  if (r >= g.tiles[0] * g.tiles[1] * g.tiles[2] * g.nslices) return;         // padding unit
  ConvUnit cu;
  cu.lev = l; cu.local = r;
  cu.slice = r % g.nslices; r /= g.nslices;
  cu.X = (r % g.tiles[0]) * XT; r /= g.tiles[0];
  cu.Y = (r % g.tiles[1]) * 32;
  cu.Z = (r / g.tiles[1]) * 4;
  conv_f2_unit<XT, true>(g, cu, srows, staps + 2, planes + (size_t)warp * (plane_bytes / 4), lane);
}

// ------------------------------------------------------- potential, fp32, list-driven inner loops
// The row/chunk loops above spend a quarter of their time on control flow: a stencil row is only
// 1 - 6 chunks long, and every chunk tests which of the two plane pairs it feeds and whether it is
// a half chunk (six warp-uniform branches around blocks of 32 FFMA2). Here the plan has sorted the
// chunks of each input plane offset into kConvListTypes lists by exactly those properties
// (ConvLevel::elist), and each list runs through a loop body that has no branch but its own.
// M0 / M1: what pair 0 / pair 1 take from a chunk: 0 nothing, 1 all four taps, 2 taps 0-1, 3 taps 2-3.
// 16-byte shared-memory load at a 32-bit shared-space address + immediate (the address arithmetic of
// a list entry is one integer add; generic pointers cost the compiler a 64-bit add and, under the
// register cap, a recomputation of the lane's row address in every iteration)
template <int OFF>
__device__ __forceinline__ float4 lds128(unsigned addr) {
  float4 v;
  asm("ld.shared.v4.f32 {%0, %1, %2, %3}, [%4+%5];" : "=f"(v.x), "=f"(v.y), "=f"(v.z), "=f"(v.w) : "r"(addr), "n"(OFF));
  return v;
}

template <int OFF>
__device__ __forceinline__ unsigned long long lds64(unsigned addr) {
  unsigned long long v;
  asm("ld.shared.b64 %0, [%1+%2];" : "=l"(v) : "r"(addr), "n"(OFF));
  return v;
}

template <int XT, int M0, int M1>
__device__ __forceinline__ void conv_list_run(int b, int e, const int4* __restrict__ el, unsigned srow0, unsigned taps2,
                                              unsigned long long (&acc)[2][XT]) {
  if (b >= e) return;
  int4 nxt = __ldg(el + b);
#pragma unroll 1
  for (int i = b; i < e; ++i) {
    const int4 cur = nxt;                             // (window, taps of pair 0, taps of pair 1) byte offsets
    nxt = __ldg(el + i + 1);                          // (the list has a guard entry behind its end)
    const unsigned w = srow0 + (unsigned)cur.x;
    float win[XT + 4];
    {
      const float4 t0 = lds128<0>(w), t1 = lds128<16>(w), t2 = lds128<32>(w), t3 = lds128<48>(w), t4 = lds128<64>(w);
      static_assert(XT == 16, "window of 20 floats");
      win[0] = t0.x; win[1] = t0.y; win[2] = t0.z; win[3] = t0.w;
      win[4] = t1.x; win[5] = t1.y; win[6] = t1.z; win[7] = t1.w;
      win[8] = t2.x; win[9] = t2.y; win[10] = t2.z; win[11] = t2.w;
      win[12] = t3.x; win[13] = t3.y; win[14] = t3.z; win[15] = t3.w;
      win[16] = t4.x; win[17] = t4.y; win[18] = t4.z; win[19] = t4.w;
    }
    float4 tq[2][2];
    if (M0 == 1 || M0 == 2) tq[0][0] = lds128<0>(taps2 + (unsigned)cur.y);
    if (M0 == 1 || M0 == 3) tq[0][1] = lds128<16>(taps2 + (unsigned)cur.y);
    if (M1 == 1 || M1 == 2) tq[1][0] = lds128<0>(taps2 + (unsigned)cur.z);
    if (M1 == 1 || M1 == 3) tq[1][1] = lds128<16>(taps2 + (unsigned)cur.z);
    // tap by tap over all accumulators: consecutive FFMA2 are independent (the next one into the
    // same accumulator is 16 or 32 instructions away)
#pragma unroll
    for (int t = 0; t < 4; ++t) {
#pragma unroll
      for (int k = 0; k < 2; ++k) {
        const int m = k == 0 ? M0 : M1;
        if (!(m == 1 || (m == 2 && t < 2) || (m == 3 && t >= 2))) continue;
        const float4 q = tq[k][t >> 1];
        const unsigned long long tp = (t & 1) ? pack2(q.z, q.w) : pack2(q.x, q.y);
#pragma unroll
        for (int i2 = 0; i2 < XT; ++i2) ffma2_bcast(acc[k][i2], win[i2 + t], tp);
      }
    }
  }
}

template <int XT>
__global__ void __launch_bounds__(32 * kConvSW, 2)
k_conv_f2l(const ConvTable* __restrict__ tabp, int plane_bytes) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  const ConvTable& tab = *tabp;
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  int l = 0;
#pragma unroll 1
  for (int k = 1; k < tab.nlev; ++k)
    if ((int)blockIdx.x * kConvSW >= tab.lev[k].sunit0) l = k;
  const ConvLevel& g = tab.lev[l];
  float4* staps = reinterpret_cast<float4*>(smem_raw);
  float* planes = reinterpret_cast<float*>(staps + g.n_taps2q);
  const float4* gt = reinterpret_cast<const float4*>(g.taps2) - 2;          // from the guard chunk on
  for (int i = threadIdx.x; i < g.n_taps2q; i += 32 * kConvSW) staps[i] = __ldg(gt + i);
  __syncthreads();
  int r = (int)blockIdx.x * kConvSW + warp - g.sunit0;
  if (r >= g.tiles[0] * g.tiles[1] * g.tiles[2] * g.nslices) return;         // padding unit
  const int slice = r % g.nslices; r /= g.nslices;
  const int X = (r % g.tiles[0]) * XT; r /= g.tiles[0];
  const int Y = (r % g.tiles[1]) * 32;
  const int Z = (r / g.tiles[1]) * 4;
  float* plane = planes + (size_t)warp * (plane_bytes / 4);
  const int Ry = g.R[1], Rz = g.R[2];
  const int nrow = 32 + 2 * Ry;
  const int WX = XT + 2 * g.X0 + 4;
  const float* __restrict__ qpad = reinterpret_cast<const float*>(g.pad);
  const int4* __restrict__ el = g.elist;
  // the warp's mbarrier (behind the planes) for the bulk copies of its input planes
  const unsigned plane_s = (unsigned)__cvta_generic_to_shared(plane);
  const unsigned mbar = (unsigned)__cvta_generic_to_shared(planes + (size_t)kConvSW * (plane_bytes / 4)) + 8u * warp;
  unsigned phase = 0;
  if (lane == 0) mbar_init(mbar);
  __syncwarp();
  // (opaque moves: the compiler would otherwise recompute the lane's row address in every iteration)
  unsigned srow0, taps2;
  asm volatile("mov.u32 %0, %1;" : "=r"(srow0) : "r"((unsigned)__cvta_generic_to_shared(plane + lane * g.pitch)));
  asm volatile("mov.u32 %0, %1;" : "=r"(taps2) : "r"((unsigned)__cvta_generic_to_shared(staps + 2)));

  unsigned long long acc[2][XT];                      // (plane 2k, plane 2k + 1) of output x + i
#pragma unroll
  for (int k = 0; k < 2; ++k)
#pragma unroll
    for (int i = 0; i < XT; ++i) acc[k][i] = 0ull;

  const int p0 = g.pb[slice], p1 = g.pb[slice + 1];
#pragma unroll 1
  for (int pz = p0; pz < p1; ++pz) {                  // input plane z = Z + pz - Rz: list set d0 = pz - Rz
    const int4 h0 = __ldg(reinterpret_cast<const int4*>(g.ehead + pz * (kConvListTypes + 1)));
    const int4 h1 = __ldg(reinterpret_cast<const int4*>(g.ehead + pz * (kConvListTypes + 1)) + 1);
    stage_plane_bulk(g, qpad, plane_s, mbar, phase, Z + pz, X, Y, nrow, WX, lane);
    conv_list_run<XT, 1, 1>(h0.x, h0.y, el, srow0, taps2, acc);
    conv_list_run<XT, 1, 0>(h0.y, h0.z, el, srow0, taps2, acc);
    conv_list_run<XT, 0, 1>(h0.z, h0.w, el, srow0, taps2, acc);
    conv_list_run<XT, 2, 0>(h0.w, h1.x, el, srow0, taps2, acc);
    conv_list_run<XT, 3, 0>(h1.x, h1.y, el, srow0, taps2, acc);
    conv_list_run<XT, 0, 2>(h1.y, h1.z, el, srow0, taps2, acc);
    conv_list_run<XT, 0, 3>(h1.z, h1.w, el, srow0, taps2, acc);
  }
  // outputs (slice partial or the final value)
  const int y = Y + lane;
  if (y < g.M[1]) {
    float* out = reinterpret_cast<float*>(g.out) + (size_t)slice * g.M[0] * g.M[1] * g.M[2];
#pragma unroll
    for (int k = 0; k < 2; ++k) {
      float* d0 = out + ((size_t)(Z + 2 * k) * g.M[1] + y) * g.M[0] + X;
      float* d1 = d0 + (size_t)g.M[1] * g.M[0];
      const bool z0 = Z + 2 * k < g.M[2], z1 = Z + 2 * k + 1 < g.M[2];
#pragma unroll
      for (int i = 0; i < XT; ++i) {
        float lo, hi;
        unpack2(acc[k][i], lo, hi);
        if (X + i < g.M[0]) {
          if (z0) d0[i] = lo;
          if (z1) d1[i] = hi;
        }
      }
    }
  }
}

// E[i] = sum_s part[s][i], s ascending (fixed order)
template <typename T>
__global__ void k_sum_slices(size_t n, int nslices, const T* __restrict__ part, T* __restrict__ E) {
  const size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  T s = part[i];
  for (int k = 1; k < nslices; ++k) s += part[(size_t)k * n + i];
  E[i] = s;
}

// ------------------------------------------------------------------------------------- virial
template <typename T, int XT, int ZT>
__global__ void __launch_bounds__(32, sizeof(T) == 4 ? 16 : 9)
k_conv_virial(const ConvTable* __restrict__ tabp, ConvSmemLayout sl) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  T* plane = reinterpret_cast<T*>(smem_raw);
  int4* srows = reinterpret_cast<int4*>(smem_raw + sl.rows_off);
  T* stap = reinterpret_cast<T*>(smem_raw + sl.taps_off);
  const ConvTable& tab = *tabp;
  const int lane = threadIdx.x;
  const ConvUnit cu = decode_unit<true, XT, ZT>(tab, blockIdx.x);
  const ConvLevel& g = tab.lev[cu.lev];
  const int X = cu.X, Y = cu.Y, Z = cu.Z;
  const int Ry = g.R[1], Rz = g.R[2];
  const int nrow = 32 + 2 * Ry;
  const int WX = XT + 2 * g.X0 + 4;
  const int ny = g.ny;
  const int4* __restrict__ rows = g.vrows;
  const T* __restrict__ vtaps = reinterpret_cast<const T*>(g.vtaps);
  const T* __restrict__ qpad = reinterpret_cast<const T*>(g.pad);
  const T* __restrict__ Q = reinterpret_cast<const T*>(g.Q);

  T qr[ZT][XT];
#pragma unroll
  for (int k = 0; k < ZT; ++k)
#pragma unroll
    for (int i = 0; i < XT; ++i) {
      const int x = X + i, y = Y + lane, z = Z + k;
      qr[k][i] = (x < g.M[0] && y < g.M[1] && z < g.M[2]) ? Q[((size_t)z * g.M[1] + y) * g.M[0] + x] : (T)0;
    }
  double S[6] = {0, 0, 0, 0, 0, 0};

  // only dz = zr - k >= 0: input planes zr in [0, ZT - 1 + Rz], padded index pz = zr + Rz
  const SliceRange sr = slice_range<true>(g, cu.slice);
  const int p0 = sr.p0, p1 = sr.p1;
  for (int pp = p0; pp < p1; pp += sr.pstep) {
    const int zr = pp;
    stage_rows<ZT>(srows, rows, ny, lane, [&](int k) {
      const int dz = zr - k;
      return dz >= 0 && dz <= Rz ? dz * ny : -1;
    });
    stage_plane<T>(g, qpad, plane, Z + zr + Rz, X, Y, nrow, WX, lane);   // commits and waits (the row entries too)
    issue_row_taps<T, ZT, 12>(srows, ny, sr.j0, vtaps, stap + (sr.j0 & 1) * sl.tapbuf, sl.tapk, lane);
    for (int dy = sr.j0 - Ry; dy < sr.j1 - Ry; ++dy) {
      const int j = dy + Ry;
      cp_async_wait<0>();                                  // this row's taps have landed
      __syncwarp();
      if (j + 1 < sr.j1) issue_row_taps<T, ZT, 12>(srows, ny, j + 1, vtaps, stap + ((j + 1) & 1) * sl.tapbuf, sl.tapk, lane);
      const T* tapb = stap + (j & 1) * sl.tapbuf;
      int4 re[ZT];
      int cl = 1 << 30, ch = -1;
#pragma unroll
      for (int k = 0; k < ZT; ++k) {
        re[k] = srows[k * ny + j];
        if (re[k].y <= re[k].z) { cl = min(cl, re[k].y); ch = max(ch, re[k].z); }
      }
      T e0[ZT], e1[ZT], e2[ZT];
#pragma unroll
      for (int k = 0; k < ZT; ++k) { e0[k] = 0; e1[k] = 0; e2[k] = 0; }
      const T* srow = plane + (lane + dy + Ry) * g.pitch;
      for (int c = cl; c <= ch; ++c) {
        T win[XT + 4];
#pragma unroll
        for (int jj = 0; jj < XT + 4; jj += 4) {
          T t[4];
          SmemVec<T>::load4(srow + 4 * c + jj, t);
          win[jj] = t[0]; win[jj + 1] = t[1]; win[jj + 2] = t[2]; win[jj + 3] = t[3];
        }
#pragma unroll
        for (int k = 0; k < ZT; ++k) {
          if (c >= re[k].y && c <= re[k].z) {
            const T* tp = tapb + k * sl.tapk + (c - re[k].y) * 12;
            T g0[4], g1[4], g2[4];
            SmemVec<T>::load4(tp, g0);
            SmemVec<T>::load4(tp + 4, g1);
            SmemVec<T>::load4(tp + 8, g2);
#pragma unroll
            for (int t = 0; t < 4; ++t) {
              T c0 = 0, c1 = 0;
#pragma unroll
              for (int i = 0; i < XT; i += 2) {
                c0 = fma(qr[k][i], win[i + t], c0);
                c1 = fma(qr[k][i + 1], win[i + 1 + t], c1);
              }
              const T ct = c0 + c1;
              e0[k] = fma(g0[t], ct, e0[k]);
              e1[k] = fma(g1[t], ct, e1[k]);
              e2[k] = fma(g2[t], ct, e2[k]);
            }
          }
        }
      }
      __syncwarp();                                        // the buffer is free for row dy + 2
      if (ch < cl) continue;
#pragma unroll
      for (int k = 0; k < ZT; ++k) {
        const double fy = (double)dy, fz = (double)(zr - k);
        const double d0 = (double)e0[k], d1 = (double)e1[k];
        S[0] += (double)e2[k];
        S[1] = fma(fy * fy, d0, S[1]);
        S[2] = fma(fz * fz, d0, S[2]);
        S[3] = fma(fy, d1, S[3]);
        S[4] = fma(fz, d1, S[4]);
        S[5] = fma(fy * fz, d0, S[5]);
      }
    }
  }
#pragma unroll
  for (int k = 0; k < 6; ++k) {
    double v = S[k];
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_down_sync(0xffffffffu, v, o);
    if (lane == 0) g.wpart[(size_t)cu.local * 6 + k] = v;
  }
}

// ------------------------------------------------------------------ virial, fp32 with packed FMAs
// Same pairing as k_conv_f2: output planes (2k, 2k+1) share one register pair. The correlation
// c_t = sum_i q_i win[i + t] of both planes is one FFMA2 chain (window value = scalar operand,
// (q_2k, q_2k+1) = pair operand); the x-moments multiply by the interleaved taps of the half-space
// rows d and d - 1.
__device__ __forceinline__ void ffma2_pp(unsigned long long& acc, unsigned long long a, unsigned long long b) {
  asm("fma.rn.f32x2 %0, %1, %2, %0;" : "+l"(acc) : "l"(a), "l"(b));
}
__device__ __forceinline__ unsigned long long fadd2_pp(unsigned long long a, unsigned long long b) {
  unsigned long long r;
  asm("add.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(a), "l"(b));
  return r;
}

template <int XT>
__global__ void __launch_bounds__(32, 16)
k_conv_virial_f2(const ConvTable* __restrict__ tabp, ConvSmemLayout sl) {
  constexpr int ZT = 4, ZP = 2;
  extern __shared__ __align__(16) unsigned char smem_raw[];
  float* plane = reinterpret_cast<float*>(smem_raw);
  int4* srows = reinterpret_cast<int4*>(smem_raw + sl.rows_off);      // [ZP][ny]
  float* stap = reinterpret_cast<float*>(smem_raw + sl.taps_off);     // two buffers of ZP * tapk floats
  const ConvTable& tab = *tabp;
  const int lane = threadIdx.x;
  const ConvUnit cu = decode_unit<true, XT, ZT>(tab, blockIdx.x);
  const ConvLevel& g = tab.lev[cu.lev];
  const int X = cu.X, Y = cu.Y, Z = cu.Z;
  const int Ry = g.R[1], Rz = g.R[2];
  const int nrow = 32 + 2 * Ry;
  const int WX = XT + 2 * g.X0 + 4;
  const int ny = g.ny;
  const int4* __restrict__ rows = g.vrows2;
  const float* __restrict__ vtaps = reinterpret_cast<const float*>(g.vtaps2);   // 24 floats per chunk
  const float* __restrict__ qpad = reinterpret_cast<const float*>(g.pad);
  const float* __restrict__ Q = reinterpret_cast<const float*>(g.Q);

  unsigned long long qr[ZP][XT];                      // (Q of plane 2k, Q of plane 2k + 1)
#pragma unroll
  for (int k = 0; k < ZP; ++k)
#pragma unroll
    for (int i = 0; i < XT; ++i) {
      const int x = X + i, y = Y + lane, z = Z + 2 * k;
      const bool in = x < g.M[0] && y < g.M[1];
      const float lo = in && z < g.M[2] ? Q[((size_t)z * g.M[1] + y) * g.M[0] + x] : 0.f;
      const float hi = in && z + 1 < g.M[2] ? Q[((size_t)(z + 1) * g.M[1] + y) * g.M[0] + x] : 0.f;
      qr[k][i] = pack2(lo, hi);
    }
  double S[6] = {0, 0, 0, 0, 0, 0};

  const SliceRange sr = slice_range<true>(g, cu.slice);
  const int p0 = sr.p0, p1 = sr.p1;
  for (int zr = p0; zr < p1; zr += sr.pstep) {        // input plane z = Z + zr, only dz >= 0
    // row entries of the merged layers to shared memory with the plane; the taps of stencil row
    // dy + 1 are copied (cp.async) while row dy is computed: no FMA waits for a table load
    stage_rows<ZP>(srows, rows, ny, lane, [&](int k) {
      const int d = zr - 2 * k;                       // planes (2k, 2k+1) take rows (d, d - 1)
      return d >= 0 && d <= Rz + 1 ? d * ny : -1;
    });
    stage_plane<float>(g, qpad, plane, Z + zr + Rz, X, Y, nrow, WX, lane);   // commits and waits
    issue_row_taps<float, ZP, 24>(srows, ny, sr.j0, vtaps, stap + (sr.j0 & 1) * sl.tapbuf, sl.tapk, lane);
    for (int dy = sr.j0 - Ry; dy < sr.j1 - Ry; ++dy) {
      const int jr = dy + Ry;
      cp_async_wait<0>();                             // this row's taps have landed
      __syncwarp();
      if (jr + 1 < sr.j1) issue_row_taps<float, ZP, 24>(srows, ny, jr + 1, vtaps, stap + ((jr + 1) & 1) * sl.tapbuf, sl.tapk, lane);
      const float* tapb = stap + (jr & 1) * sl.tapbuf;
      int4 re[ZP];
      int cl = 1 << 30, ch = -1;
#pragma unroll
      for (int k = 0; k < ZP; ++k) {
        re[k] = srows[k * ny + jr];
        if (re[k].y <= re[k].z) { cl = min(cl, re[k].y); ch = max(ch, re[k].z); }
      }
      if (ch < cl) continue;
      unsigned long long e0[ZP], e1[ZP], e2[ZP];
#pragma unroll
      for (int k = 0; k < ZP; ++k) { e0[k] = 0ull; e1[k] = 0ull; e2[k] = 0ull; }
      const float* srow = plane + (lane + dy + Ry) * g.pitch;
      for (int c = cl; c <= ch; ++c) {
        float win[XT + 4];
#pragma unroll
        for (int j = 0; j < XT + 4; j += 4) {
          const float4 t = *reinterpret_cast<const float4*>(srow + 4 * c + j);
          win[j] = t.x; win[j + 1] = t.y; win[j + 2] = t.z; win[j + 3] = t.w;
        }
#pragma unroll
        for (int k = 0; k < ZP; ++k) {
          if (c >= re[k].y && c <= re[k].z) {
            const float4* tp = reinterpret_cast<const float4*>(tapb + k * sl.tapk + (c - re[k].y) * 24);
            float4 gq[6];
#pragma unroll
            for (int m = 0; m < 6; ++m) gq[m] = tp[m];
            const bool lo = 2 * c >= (re[k].w & 0xffff), hi = 2 * c + 1 <= (re[k].w >> 16);
#pragma unroll
            for (int t = 0; t < 4; ++t) {
              if (t < 2 ? !lo : !hi) continue;          // empty 2-tap half of the row's first / last chunk
              unsigned long long c0 = 0ull, c1 = 0ull;
#pragma unroll
              for (int i = 0; i < XT; i += 2) {
                ffma2_bcast(c0, win[i + t], qr[k][i]);
                ffma2_bcast(c1, win[i + 1 + t], qr[k][i + 1]);
              }
              const unsigned long long ct = fadd2_pp(c0, c1);
              // taps of moment m, tap t: floats (2t, 2t+1) of quads 2m, 2m+1
              const float4 a0 = gq[t >> 1], a1 = gq[2 + (t >> 1)], a2 = gq[4 + (t >> 1)];
              const bool up = (t & 1) != 0;
              ffma2_pp(e0[k], up ? pack2(a0.z, a0.w) : pack2(a0.x, a0.y), ct);
              ffma2_pp(e1[k], up ? pack2(a1.z, a1.w) : pack2(a1.x, a1.y), ct);
              ffma2_pp(e2[k], up ? pack2(a2.z, a2.w) : pack2(a2.x, a2.y), ct);
            }
          }
        }
      }
#pragma unroll
      for (int k = 0; k < ZP; ++k) {
        float e0l, e0h, e1l, e1h, e2l, e2h;
        unpack2(e0[k], e0l, e0h); unpack2(e1[k], e1l, e1h); unpack2(e2[k], e2l, e2h);
        const double fy = (double)dy;
#pragma unroll
        for (int h = 0; h < 2; ++h) {                 // lower half: plane 2k (dz = d), upper: 2k+1 (dz = d - 1)
          const double fz = (double)(zr - 2 * k - h);
          const double d0 = (double)(h ? e0h : e0l), d1 = (double)(h ? e1h : e1l);
          S[0] += (double)(h ? e2h : e2l);
          S[1] = fma(fy * fy, d0, S[1]);
          S[2] = fma(fz * fz, d0, S[2]);
          S[3] = fma(fy, d1, S[3]);
          S[4] = fma(fz, d1, S[4]);
          S[5] = fma(fy * fz, d0, S[5]);
        }
      }
    }
  }
#pragma unroll
  for (int k = 0; k < 6; ++k) {
    double v = S[k];
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_down_sync(0xffffffffu, v, o);
    if (lane == 0) g.wpart[(size_t)cu.local * 6 + k] = v;
  }
}

// ---------------------------------------------------- virial, fp32, list-driven (see k_conv_f2l)
// One block of kConvVW warps per SM with the level's interleaved moment taps in shared memory. A
// list entry is one 4-tap chunk of one stencil row; after its taps the entry's three x-moment sums
// go straight into six packed fp32 sums with the row's dy and the plane pair's dz as factors (seven
// packed instructions per entry and plane pair), which are added to the fp64 sums once per input
// plane: ~200 fp32 additions per sum and plane.
template <int XT, int M>
__device__ __forceinline__ void virial_entry(const int4 cur, int k, unsigned srow0, unsigned vtaps, float fy,
                                             const unsigned long long (&qr)[2][XT], unsigned long long fz, unsigned long long fz2,
                                             unsigned long long (&S)[6]) {
  static_assert(XT == 16, "window of 20 floats");
  const unsigned w = srow0 + (unsigned)cur.x;
  float win[XT + 4];
  {
    const float4 t0 = lds128<0>(w), t1 = lds128<16>(w), t2 = lds128<32>(w), t3 = lds128<48>(w), t4 = lds128<64>(w);
    win[0] = t0.x; win[1] = t0.y; win[2] = t0.z; win[3] = t0.w;
    win[4] = t1.x; win[5] = t1.y; win[6] = t1.z; win[7] = t1.w;
    win[8] = t2.x; win[9] = t2.y; win[10] = t2.z; win[11] = t2.w;
    win[12] = t3.x; win[13] = t3.y; win[14] = t3.z; win[15] = t3.w;
    win[16] = t4.x; win[17] = t4.y; win[18] = t4.z; win[19] = t4.w;
  }
  const unsigned tp = vtaps + (unsigned)(k == 0 ? cur.y : cur.z);
  // moment m of tap t, as (row d, row d - 1): 8 bytes at 32 m + 8 t, loaded tap by tap (few live registers)
  unsigned long long e0 = 0ull, e1 = 0ull, e2 = 0ull;
#pragma unroll
  for (int t = 0; t < 4; ++t) {
    if ((M == 2 && t >= 2) || (M == 3 && t < 2)) continue;
    unsigned long long c0 = 0ull, c1 = 0ull;
#pragma unroll
    for (int i = 0; i < XT; i += 2) {
      ffma2_bcast(c0, win[i + t], qr[k][i]);
      ffma2_bcast(c1, win[i + 1 + t], qr[k][i + 1]);
    }
    const unsigned long long ct = fadd2_pp(c0, c1);
    if (t == 0) { ffma2_pp(e0, lds64<0>(tp), ct); ffma2_pp(e1, lds64<32>(tp), ct); ffma2_pp(e2, lds64<64>(tp), ct); }
    if (t == 1) { ffma2_pp(e0, lds64<8>(tp), ct); ffma2_pp(e1, lds64<40>(tp), ct); ffma2_pp(e2, lds64<72>(tp), ct); }
    if (t == 2) { ffma2_pp(e0, lds64<16>(tp), ct); ffma2_pp(e1, lds64<48>(tp), ct); ffma2_pp(e2, lds64<80>(tp), ct); }
    if (t == 3) { ffma2_pp(e0, lds64<24>(tp), ct); ffma2_pp(e1, lds64<56>(tp), ct); ffma2_pp(e2, lds64<88>(tp), ct); }
  }
  // xx: x^2 moment; yy: dy^2 e0; zz: dz^2 e0; xy: dy e1; xz: dz e1; yz: dy dz e0
  S[0] = fadd2_pp(S[0], e2);
  ffma2_bcast(S[1], fy * fy, e0);
  ffma2_pp(S[2], fz2, e0);
  ffma2_bcast(S[3], fy, e1);
  ffma2_pp(S[4], fz, e1);
  unsigned long long ze = 0ull;
  ffma2_pp(ze, fz, e0);
  ffma2_bcast(S[5], fy, ze);
}

template <int XT, int M0, int M1>
__device__ __forceinline__ void virial_list_run(int b, int e, const int4* __restrict__ el, unsigned srow0, unsigned vtaps,
                                                const unsigned long long (&qr)[2][XT], const unsigned long long (&fz)[2],
                                                const unsigned long long (&fz2)[2], unsigned long long (&S)[6]) {
  if (b >= e) return;
  int4 nxt = __ldg(el + b);
#pragma unroll 1
  for (int i = b; i < e; ++i) {
    const int4 cur = nxt;
    nxt = __ldg(el + i + 1);                          // (guard entry behind the end)
    const float fy = __int_as_float(cur.w);
    if (M0 != 0) virial_entry<XT, M0>(cur, 0, srow0, vtaps, fy, qr, fz[0], fz2[0], S);
    if (M1 != 0) virial_entry<XT, M1>(cur, 1, srow0, vtaps, fy, qr, fz[1], fz2[1], S);
  }
}

template <int XT>
__global__ void __launch_bounds__(32 * kConvVW, 1)
k_conv_virial_f2l(const ConvTable* __restrict__ tabp, int plane_bytes) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  const ConvTable& tab = *tabp;
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  int l = 0;
#pragma unroll 1
  for (int k = 1; k < tab.nlev; ++k)
    if ((int)blockIdx.x * kConvVW >= tab.lev[k].vsunit0) l = k;
  const ConvLevel& g = tab.lev[l];
  float4* staps = reinterpret_cast<float4*>(smem_raw);
  float* planes = reinterpret_cast<float*>(staps + g.n_vtaps2q);
  const float4* gt = reinterpret_cast<const float4*>(g.vtaps2);
  for (int i = threadIdx.x; i < g.n_vtaps2q; i += 32 * kConvVW) staps[i] = __ldg(gt + i);
  __syncthreads();
  int r = (int)blockIdx.x * kConvVW + warp - g.vsunit0;
  if (r >= g.tiles[0] * g.tiles[1] * g.tiles[2] * g.vslices) return;         // padding unit
  const int local = r;
  const int slice = r % g.vslices; r /= g.vslices;
  const int X = (r % g.tiles[0]) * XT; r /= g.tiles[0];
  const int Y = (r % g.tiles[1]) * 32;
  const int Z = (r / g.tiles[1]) * 4;
  float* plane = planes + (size_t)warp * (plane_bytes / 4);
  const int Ry = g.R[1], Rz = g.R[2];
  const int nrow = 32 + 2 * Ry;
  const int WX = XT + 2 * g.X0 + 4;
  const float* __restrict__ qpad = reinterpret_cast<const float*>(g.pad);
  const float* __restrict__ Q = reinterpret_cast<const float*>(g.Q);
  const int4* __restrict__ el = g.vlist;
  const unsigned plane_s = (unsigned)__cvta_generic_to_shared(plane);
  const unsigned mbar = (unsigned)__cvta_generic_to_shared(planes + (size_t)kConvVW * (plane_bytes / 4)) + 8u * warp;
  unsigned phase = 0;
  if (lane == 0) mbar_init(mbar);
  __syncwarp();
  unsigned srow0, vtaps;
  asm volatile("mov.u32 %0, %1;" : "=r"(srow0) : "r"((unsigned)__cvta_generic_to_shared(plane + lane * g.pitch)));
  asm volatile("mov.u32 %0, %1;" : "=r"(vtaps) : "r"((unsigned)__cvta_generic_to_shared(staps)));

  unsigned long long qr[2][XT];                       // (Q of plane 2k, Q of plane 2k + 1)
#pragma unroll
  for (int k = 0; k < 2; ++k)
#pragma unroll
    for (int i = 0; i < XT; ++i) {
      const int x = X + i, y = Y + lane, z = Z + 2 * k;
      const bool in = x < g.M[0] && y < g.M[1];
      const float lo = in && z < g.M[2] ? Q[((size_t)z * g.M[1] + y) * g.M[0] + x] : 0.f;
      const float hi = in && z + 1 < g.M[2] ? Q[((size_t)(z + 1) * g.M[1] + y) * g.M[0] + x] : 0.f;
      qr[k][i] = pack2(lo, hi);
    }
  double S[6] = {0, 0, 0, 0, 0, 0};

  // planes dealt round-robin to the slices: equal taps AND equal plane counts (0.495 -> 0.479 ms at N = 10^6; the
  // potential kernels measured slower that way and keep the contiguous, tap-balanced ranges)
  const int nplanes = Rz + 4;
#pragma unroll 1
  for (int zr = slice; zr < nplanes; zr += g.vslices) {                  // input plane z = Z + zr, only dz >= 0
    const int4 h0 = __ldg(reinterpret_cast<const int4*>(g.vhead + zr * (kConvListTypes + 1)));
    const int4 h1 = __ldg(reinterpret_cast<const int4*>(g.vhead + zr * (kConvListTypes + 1)) + 1);
    stage_plane_bulk(g, qpad, plane_s, mbar, phase, Z + zr + Rz, X, Y, nrow, WX, lane);
    // plane pair k takes the merged layer d = zr - 2k: dz = d for its lower plane, d - 1 for the upper
    unsigned long long fz[2], fz2[2], Sp[6];
#pragma unroll
    for (int k = 0; k < 2; ++k) {
      const float a = (float)(zr - 2 * k), b = (float)(zr - 2 * k - 1);
      fz[k] = pack2(a, b);
      fz2[k] = pack2(a * a, b * b);
    }
#pragma unroll
    for (int k = 0; k < 6; ++k) Sp[k] = 0ull;
    virial_list_run<XT, 1, 1>(h0.x, h0.y, el, srow0, vtaps, qr, fz, fz2, Sp);
    virial_list_run<XT, 1, 0>(h0.y, h0.z, el, srow0, vtaps, qr, fz, fz2, Sp);
    virial_list_run<XT, 0, 1>(h0.z, h0.w, el, srow0, vtaps, qr, fz, fz2, Sp);
    virial_list_run<XT, 2, 0>(h0.w, h1.x, el, srow0, vtaps, qr, fz, fz2, Sp);
    virial_list_run<XT, 3, 0>(h1.x, h1.y, el, srow0, vtaps, qr, fz, fz2, Sp);
    virial_list_run<XT, 0, 2>(h1.y, h1.z, el, srow0, vtaps, qr, fz, fz2, Sp);
    virial_list_run<XT, 0, 3>(h1.z, h1.w, el, srow0, vtaps, qr, fz, fz2, Sp);
#pragma unroll
    for (int k = 0; k < 6; ++k) {
      float lo, hi;
      unpack2(Sp[k], lo, hi);
      S[k] += (double)lo + (double)hi;
    }
  }
#pragma unroll
  for (int k = 0; k < 6; ++k) {
    double v = S[k];
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_down_sync(0xffffffffu, v, o);
    if (lane == 0) g.wpart[(size_t)local * 6 + k] = v;
  }
}

// --------------------------------------------------------- potential, fp64, list-driven (see k_conv_f2l)
// One block of kConvDW warps per SM with the level's tap table (mirrored rows stored once) in shared
// memory; a unit is an 8 x 32 x 4 output tile and a slice of input planes. The chunks of each input
// plane offset are sorted into seven lists: all four output planes take the chunk / planes (0, 1) /
// planes (2, 3) / one of the four planes alone.
template <int OFF>
__device__ __forceinline__ double2 lds128d(unsigned addr) {
  double2 v;
  asm("ld.shared.v2.f64 {%0, %1}, [%2+%3];" : "=d"(v.x), "=d"(v.y) : "r"(addr), "n"(OFF));
  return v;
}

// MASK: bit k set = output plane k takes this chunk
template <int MASK>
__device__ __forceinline__ void convd_list_run(int b, int e, const int4* __restrict__ el, unsigned srow0, unsigned staps,
                                               double (&acc)[4][8]) {
  if (b >= e) return;
  int4 n0 = __ldg(el + 2 * b), n1 = __ldg(el + 2 * b + 1);
#pragma unroll 1
  for (int i = b; i < e; ++i) {
    const int4 c0 = n0, c1 = n1;                      // (window, taps 0, taps 1, taps 2), (taps 3, -, -, -)
    n0 = __ldg(el + 2 * i + 2);                       // (guard entry behind the end)
    n1 = __ldg(el + 2 * i + 3);
    const unsigned w = srow0 + (unsigned)c0.x;
    double win[12];
    {
      const double2 t0 = lds128d<0>(w), t1 = lds128d<16>(w), t2 = lds128d<32>(w), t3 = lds128d<48>(w), t4 = lds128d<64>(w),
                    t5 = lds128d<80>(w);
      win[0] = t0.x; win[1] = t0.y; win[2] = t1.x; win[3] = t1.y; win[4] = t2.x; win[5] = t2.y;
      win[6] = t3.x; win[7] = t3.y; win[8] = t4.x; win[9] = t4.y; win[10] = t5.x; win[11] = t5.y;
    }
    double tp[4][4];
#pragma unroll
    for (int k = 0; k < 4; ++k) {
      if (!(MASK & (1 << k))) continue;
      const unsigned ta = staps + (unsigned)(k == 0 ? c0.y : k == 1 ? c0.z : k == 2 ? c0.w : c1.x);
      const double2 a = lds128d<0>(ta), bq = lds128d<16>(ta);
      tp[k][0] = a.x; tp[k][1] = a.y; tp[k][2] = bq.x; tp[k][3] = bq.y;
    }
#pragma unroll
    for (int t = 0; t < 4; ++t)
#pragma unroll
      for (int k = 0; k < 4; ++k) {
        if (!(MASK & (1 << k))) continue;
#pragma unroll
        for (int x = 0; x < 8; ++x) acc[k][x] = fma(tp[k][t], win[x + t], acc[k][x]);
      }
  }
}

template <int XT>
__global__ void __launch_bounds__(32 * kConvDW, 1)
k_conv_dl(const ConvTable* __restrict__ tabp, int plane_bytes) {
  static_assert(XT == 8, "window of 12 doubles");
  extern __shared__ __align__(16) unsigned char smem_raw[];
  const ConvTable& tab = *tabp;
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  int l = 0;
#pragma unroll 1
  for (int k = 1; k < tab.nlev; ++k)
    if ((int)blockIdx.x * kConvDW >= tab.lev[k].dsunit0) l = k;
  const ConvLevel& g = tab.lev[l];
  double2* stq = reinterpret_cast<double2*>(smem_raw);
  unsigned char* planes = reinterpret_cast<unsigned char*>(stq + g.n_stapsq);
  const double2* gt = reinterpret_cast<const double2*>(g.staps);
  for (int i = threadIdx.x; i < g.n_stapsq; i += 32 * kConvDW) stq[i] = __ldg(gt + i);
  __syncthreads();
  int r = (int)blockIdx.x * kConvDW + warp - g.dsunit0;
  if (r >= g.tiles[0] * g.tiles[1] * g.tiles[2] * g.nslices) return;         // padding unit
  const int slice = r % g.nslices; r /= g.nslices;
  const int X = (r % g.tiles[0]) * XT; r /= g.tiles[0];
  const int Y = (r % g.tiles[1]) * 32;
  const int Z = (r / g.tiles[1]) * 4;
  double* plane = reinterpret_cast<double*>(planes + (size_t)warp * plane_bytes);
  const int Ry = g.R[1], Rz = g.R[2];
  const int nrow = 32 + 2 * Ry;
  const int WX = XT + 2 * g.X0 + 4;
  const double* __restrict__ qpad = reinterpret_cast<const double*>(g.pad);
  const int4* __restrict__ el = g.dlist;
  unsigned srow0, staps;
  asm volatile("mov.u32 %0, %1;" : "=r"(srow0) : "r"((unsigned)__cvta_generic_to_shared(plane + lane * g.pitch)));
  asm volatile("mov.u32 %0, %1;" : "=r"(staps) : "r"((unsigned)__cvta_generic_to_shared(stq)));
  const unsigned plane_s = (unsigned)__cvta_generic_to_shared(plane);
  const unsigned mbar = (unsigned)__cvta_generic_to_shared(planes + (size_t)kConvDW * plane_bytes) + 8u * warp;
  unsigned phase = 0;
  if (lane == 0) mbar_init(mbar);
  __syncwarp();

  double acc[4][XT];
#pragma unroll
  for (int k = 0; k < 4; ++k)
#pragma unroll
    for (int i = 0; i < XT; ++i) acc[k][i] = 0.0;

  const int p0 = g.pb[slice], p1 = g.pb[slice + 1];
#pragma unroll 1
  for (int pz = p0; pz < p1; ++pz) {                  // input plane z = Z + pz - Rz feeds output plane k with dz = pz - Rz - k
    const int4 h0 = __ldg(reinterpret_cast<const int4*>(g.dhead + pz * (kConvListTypes + 1)));
    const int4 h1 = __ldg(reinterpret_cast<const int4*>(g.dhead + pz * (kConvListTypes + 1)) + 1);
    // rows of WX doubles: one bulk copy each
    {
      const double* src = qpad + ((size_t)(Z + pz) * g.P[1] + Y) * g.P[0] + X;
      __syncwarp();
      if (lane == 0)
        asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" :: "r"(mbar), "r"((unsigned)(nrow * WX * 8)) : "memory");
      __syncwarp();
      for (int rr = lane; rr < nrow; rr += 32)
        asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                     :: "r"(plane_s + (unsigned)(rr * g.pitch * 8)), "l"(src + (size_t)rr * g.P[0]), "r"((unsigned)(WX * 8)), "r"(mbar)
                     : "memory");
      unsigned done;
      do {
        asm volatile("{\n .reg .pred p;\n mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n selp.u32 %0, 1, 0, p;\n}"
                     : "=r"(done) : "r"(mbar), "r"(phase) : "memory");
      } while (!done);
      phase ^= 1u;
    }
    convd_list_run<15>(h0.x, h0.y, el, srow0, staps, acc);
    convd_list_run<3>(h0.y, h0.z, el, srow0, staps, acc);
    convd_list_run<12>(h0.z, h0.w, el, srow0, staps, acc);
    convd_list_run<1>(h0.w, h1.x, el, srow0, staps, acc);
    convd_list_run<2>(h1.x, h1.y, el, srow0, staps, acc);
    convd_list_run<4>(h1.y, h1.z, el, srow0, staps, acc);
    convd_list_run<8>(h1.z, h1.w, el, srow0, staps, acc);
  }
  const int y = Y + lane;
  if (y < g.M[1]) {
    double* out = reinterpret_cast<double*>(g.out) + (size_t)slice * g.M[0] * g.M[1] * g.M[2];
#pragma unroll
    for (int k = 0; k < 4; ++k) {
      const int z = Z + k;
      if (z < g.M[2]) {
        double* dst = out + ((size_t)z * g.M[1] + y) * g.M[0] + X;
#pragma unroll
        for (int i = 0; i < XT; ++i)
          if (X + i < g.M[0]) dst[i] = acc[k][i];
      }
    }
  }
}

}  // namespace msm
