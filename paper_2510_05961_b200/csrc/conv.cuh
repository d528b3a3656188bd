// conv.cuh -- S5: per-level grid<->grid convolution with the truncated stencil of k_l
// (Eq. 11; stencil P:268 Eq. 20), FP-pipe bound.
//
// Formulation. K^l = omega'(x)omega'(x)omega' * s_l (Eq. 20) and convolution is associative, so
// e^l = s_l * qpad with qpad = omega'-filtered, haloed grid charge (k_pad_filter). s_l is non-zero
// only inside the cutoff ellipsoid (3-5x fewer taps than the folded K^l) and is even in n, so
// e_m = sum_n s(n) qpad[m + n]. The halo holds periodic images (as many wraps as the stencil
// needs) or zeros (open axes), so the kernel has no boundary logic.
//
// Work unit = one warp: outputs x in [X, X+XT), y = Y + lane, z in [Z, Z+ZT); each thread keeps
// XT*ZT accumulators in registers. The warp streams input z-planes through shared memory; one
// plane feeds all ZT output planes (tap row dz = z_in - z_out), so a 16-byte shared-memory window
// load is amortised over up to 4*XT*ZT FMAs, and every tap quad (one 16-byte broadcast load from
// the L1-resident table) feeds 4*XT FMAs. Rows of the stencil are stored as runs of 4-tap chunks
// covering only the ellipsoid; chunk tests are warp-uniform, so there is no divergence.
//
// VIRIAL adds the strain derivative of the level's energy (reading V): with c_t = sum_i q_i
// qpad[i + n_t] over the thread's outputs, S_ab += g(n_t) n_a n_b c_t, g = k_l'(r)/r; the host
// scales by -1/2 h_a h_b. Costs one more FMA per tap and output.
#pragma once
#include "device_common.cuh"

namespace msm {

struct ConvGeom {
  int M[3];        // output grid dims
  int P[3];        // padded input dims
  int R[3];        // stencil half-widths (y, z used as halo; x halo is X0)
  int X0;          // x halo, multiple of 4, >= R[0]
  int tiles[3];    // units per axis
  int pitch;       // shared-memory row pitch in elements
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
};

template <typename T, int XT, int ZT, bool VIRIAL>
__global__ void __launch_bounds__(32)
k_conv(ConvGeom g, const int4* __restrict__ rows, const T* __restrict__ staps, const T* __restrict__ gtaps,
       const T* __restrict__ qpad, const T* __restrict__ Q, T* __restrict__ E, double* __restrict__ wpart) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  T* plane = reinterpret_cast<T*>(smem_raw);
  const int lane = threadIdx.x;
  int u = blockIdx.x;
  const int tx = u % g.tiles[0]; u /= g.tiles[0];
  const int ty = u % g.tiles[1], tz = u / g.tiles[1];
  const int X = tx * XT, Y = ty * 32, Z = tz * ZT;
  const int Ry = g.R[1], Rz = g.R[2];
  const int nrow = 32 + 2 * Ry;
  const int WX = XT + 2 * g.X0 + 4;
  const int ny = 2 * Ry + 1;

  T acc[ZT][XT];
#pragma unroll
  for (int k = 0; k < ZT; ++k)
#pragma unroll
    for (int i = 0; i < XT; ++i) acc[k][i] = 0;
  T qr[VIRIAL ? ZT : 1][VIRIAL ? XT : 1];
  double S[6] = {0, 0, 0, 0, 0, 0};
  if (VIRIAL) {
#pragma unroll
    for (int k = 0; k < ZT; ++k)
#pragma unroll
      for (int i = 0; i < XT; ++i) {
        const int x = X + i, y = Y + lane, z = Z + k;
        qr[k][i] = (x < g.M[0] && y < g.M[1] && z < g.M[2]) ? Q[((size_t)z * g.M[1] + y) * g.M[0] + x] : (T)0;
      }
  }

  for (int zr = -Rz; zr <= ZT - 1 + Rz; ++zr) {
    // stage input plane z = Z + zr (padded index + Rz): rows Y .. Y+nrow-1, x X .. X+WX-1 (padded)
    {
      const T* src = qpad + ((size_t)(Z + zr + Rz) * g.P[1] + Y) * g.P[0] + X;
      const int vper = WX / 4, nvec = nrow * vper;
      __syncwarp();
      for (int v = lane; v < nvec; v += 32) {
        const int r = v / vper, cx = (v - r * vper) * 4;
        T t[4];
        SmemVec<T>::ldg(src + (size_t)r * g.P[0] + cx, t);
        T* dst = plane + r * g.pitch + cx;
        dst[0] = t[0]; dst[1] = t[1]; dst[2] = t[2]; dst[3] = t[3];
      }
      __syncwarp();
    }
    for (int dy = -Ry; dy <= Ry; ++dy) {
      int4 re[ZT];
      int cl = 1 << 30, ch = -1;
#pragma unroll
      for (int k = 0; k < ZT; ++k) {
        const int dz = zr - k;
        if (dz >= -Rz && dz <= Rz) {
          re[k] = __ldg(rows + (dz + Rz) * ny + (dy + Ry));
        } else {
          re[k] = make_int4(0, 1, 0, 0);   // empty
        }
        if (re[k].y <= re[k].z) { cl = min(cl, re[k].y); ch = max(ch, re[k].z); }
      }
      const T* srow = plane + (lane + dy + Ry) * g.pitch;
      for (int c = cl; c <= ch; ++c) {
        T win[XT + 4];
#pragma unroll
        for (int j = 0; j < XT + 4; j += 4) {
          T t[4];
          SmemVec<T>::load4(srow + 4 * c + j, t);
          win[j] = t[0]; win[j + 1] = t[1]; win[j + 2] = t[2]; win[j + 3] = t[3];
        }
#pragma unroll
        for (int k = 0; k < ZT; ++k) {
          if (c >= re[k].y && c <= re[k].z) {
            const int toff = (re[k].x + c - re[k].y) * 4;
            T tp[4];
            SmemVec<T>::ldg(staps + toff, tp);
#pragma unroll
            for (int t = 0; t < 4; ++t)
#pragma unroll
              for (int i = 0; i < XT; ++i) acc[k][i] = fma(tp[t], win[i + t], acc[k][i]);
            if (VIRIAL) {
              T gp[4];
              SmemVec<T>::ldg(gtaps + toff, gp);
              const T fdx = (T)(4 * c - g.X0);
              T e0 = 0, e1 = 0, e2 = 0;
#pragma unroll
              for (int t = 0; t < 4; ++t) {
                T c0 = 0, c1 = 0;
#pragma unroll
                for (int i = 0; i < XT; i += 2) {
                  c0 = fma(qr[k][i], win[i + t], c0);
                  c1 = fma(qr[k][i + 1], win[i + 1 + t], c1);
                }
                const T gc = gp[t] * (c0 + c1), d = fdx + (T)t;
                e0 += gc;
                e1 = fma(d, gc, e1);
                e2 = fma(d * d, gc, e2);
              }
              const double fy = (double)dy, fz = (double)(zr - k);
              const double d0 = (double)e0, d1 = (double)e1;
              S[0] += (double)e2;
              S[1] = fma(fy * fy, d0, S[1]);
              S[2] = fma(fz * fz, d0, S[2]);
              S[3] = fma(fy, d1, S[3]);
              S[4] = fma(fz, d1, S[4]);
              S[5] = fma(fy * fz, d0, S[5]);
            }
          }
        }
      }
    }
  }
  // outputs
  {
    const int y = Y + lane;
    if (y < g.M[1]) {
#pragma unroll
      for (int k = 0; k < ZT; ++k) {
        const int z = Z + k;
        if (z < g.M[2]) {
          T* dst = E + ((size_t)z * g.M[1] + y) * g.M[0] + X;
#pragma unroll
          for (int i = 0; i < XT; ++i)
            if (X + i < g.M[0]) dst[i] = acc[k][i];
        }
      }
    }
  }
  if (VIRIAL) {
#pragma unroll
    for (int k = 0; k < 6; ++k) {
      double v = S[k];
#pragma unroll
      for (int o = 16; o > 0; o >>= 1) v += __shfl_down_sync(0xffffffffu, v, o);
      if (lane == 0) wpart[(size_t)blockIdx.x * 6 + k] = v;
    }
  }
}

}  // namespace msm
