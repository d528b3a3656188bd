// plan_top.cpp -- sampled stencils of the tiled levels and the dense top-level operator
// (host, fp64). See plan_math.hpp.
#include <algorithm>
#include <cstring>

#include "plan_math.hpp"

namespace msm {

// s(n) = k_l(|h o n|), g(n) = k_l'(r)/r inside the cutoff ellipsoid |h o n| < 2^l a (Eq. 20
// samples; the omega' factors are applied to the grid charge instead, which is the same sum).
SampledStencil sample_level_stencil(const Hierarchy& H, const Splitting& S, int l, const double* hstruct) {
  SampledStencil st;
  const Level& lv = H.lev[l];
  const double A = std::ldexp(S.a, l);
  for (int ax = 0; ax < 3; ++ax) {
    const double hs = hstruct ? hstruct[ax] : lv.h[ax];
    int R = (int)std::floor(A / hs);
    while (R > 0 && R * hs >= A) --R;
    st.R[ax] = R;
  }
  const size_t n = (size_t)(2 * st.R[0] + 1) * (2 * st.R[1] + 1) * (2 * st.R[2] + 1);
  st.s.assign(n, 0.0);
  st.g.assign(n, 0.0);
  st.taps = 0;
  size_t idx = 0;
  for (int dz = -st.R[2]; dz <= st.R[2]; ++dz)
    for (int dy = -st.R[1]; dy <= st.R[1]; ++dy)
      for (int dx = -st.R[0]; dx <= st.R[0]; ++dx, ++idx) {
        const double x = dx * lv.h[0], y = dy * lv.h[1], z = dz * lv.h[2];
        const double r = std::sqrt(x * x + y * y + z * z);
        if (r >= A) continue;
        st.s[idx] = S.k(l, r);
        st.g[idx] = (r > 0.0) ? S.dk(l, r) / r : 0.0;
        ++st.taps;
      }
  return st;
}

namespace {

struct Box3 {  // dense box [-R, R]^3, x fastest
  int R[3];
  std::vector<double> v;
  size_t idx(int dx, int dy, int dz) const {
    return ((size_t)(dz + R[2]) * (2 * R[1] + 1) + (dy + R[1])) * (2 * R[0] + 1) + (dx + R[0]);
  }
};

// slab top level (reading T3): plane average of k_L over the periodic plane, divergent constant
// dropped; P(x) = int_0^x t gamma(t) dt.
double slab_P(const Splitting& S, double x) {
  const double s1 = x * x - 1.0;
  double pw = s1, sgn = -1.0, acc = 0.0;
  for (int k = 0; k < S.p; ++k) {
    acc += S.c[k] * (pw - sgn) / (2.0 * (k + 1));
    pw *= s1;
    sgn = -sgn;
  }
  return acc;
}

// kind 0: the kernel; 1..6: its strain derivative, components xx yy zz xy xz yz
double sample_value(const Hierarchy& H, const Splitting& S, int l, int kind, const double r[3]) {
  static const int AB[7][2] = {{0, 0}, {0, 0}, {1, 1}, {2, 2}, {0, 1}, {0, 2}, {1, 2}};
  if (l == H.L && H.top == kTopSlab) {
    const int oz = H.open_axis;
    double area = 1.0;
    for (int ax = 0; ax < 3; ++ax)
      if (ax != oz) area *= H.prm.box[ax];
    const double A = std::ldexp(S.a, H.L - 1), z = std::fabs(r[oz]), rho = z / A;
    const double pi = 3.14159265358979323846;
    const double sL = -(2.0 * pi / area) * A * (slab_P(S, std::min(rho, 1.0)) + std::max(rho - 1.0, 0.0));
    if (kind == 0) return sL;
    if (kind > 3) return 0.0;
    if (kind - 1 != oz) return -sL;                       // area scales with the periodic strain
    return -(2.0 * pi / area) * z * z * S.k(l, z);
  }
  const double rr = std::sqrt(r[0] * r[0] + r[1] * r[1] + r[2] * r[2]);
  if (kind == 0) return S.k(l, rr);
  if (rr == 0.0) return 0.0;
  return S.dk(l, rr) * r[AB[kind][0]] * r[AB[kind][1]] / rr;
}

// K = omega' (x) omega' (x) omega' * samples (Eq. 20), for offsets |d| <= Kr
Box3 full_stencil(const Hierarchy& H, const Splitting& S, const std::vector<double>& omega, int l,
                  int kind, const int Kr[3], const int wax[3]) {
  int n0[3], dims[3];
  for (int ax = 0; ax < 3; ++ax) { n0[ax] = Kr[ax] + wax[ax]; dims[ax] = 2 * n0[ax] + 1; }
  std::vector<double> cur((size_t)dims[0] * dims[1] * dims[2]);
  const Level& lv = H.lev[l];
  size_t i = 0;
  for (int z = -n0[2]; z <= n0[2]; ++z)
    for (int y = -n0[1]; y <= n0[1]; ++y)
      for (int x = -n0[0]; x <= n0[0]; ++x, ++i) {
        const double r[3] = {x * lv.h[0], y * lv.h[1], z * lv.h[2]};
        cur[i] = sample_value(H, S, l, kind, r);
      }
  const int w = (int)(omega.size() / 2);
  for (int ax = 0; ax < 3; ++ax) {
    if (wax[ax] == 0) continue;
    int nd[3] = {dims[0], dims[1], dims[2]};
    nd[ax] = 2 * Kr[ax] + 1;
    std::vector<double> nxt((size_t)nd[0] * nd[1] * nd[2]);
    const size_t stride = ax == 0 ? 1 : (ax == 1 ? (size_t)dims[0] : (size_t)dims[0] * dims[1]);
    for (int z = 0; z < nd[2]; ++z)
      for (int y = 0; y < nd[1]; ++y)
        for (int x = 0; x < nd[0]; ++x) {
          // output position o along ax maps to input positions o + wax - k, k = -w..w
          const size_t base = ((size_t)z * dims[1] + y) * dims[0] + x;  // same coords in `cur`
          double acc = 0.0;
          for (int k = -w; k <= w; ++k) acc += omega[k + w] * cur[base + (size_t)(wax[ax] - k) * stride];
          nxt[((size_t)z * nd[1] + y) * nd[0] + x] = acc;
        }
    cur.swap(nxt);
    dims[ax] = nd[ax];
  }
  Box3 b;
  for (int ax = 0; ax < 3; ++ax) b.R[ax] = Kr[ax];
  b.v.swap(cur);
  return b;
}

// dense G x G matrix of "convolve with K on the level-l grid" (Eq. 11): periodic axes wrap
// (all images inside the stencil), open axes see zero outside the grid
std::vector<double> dense_convolution(const Hierarchy& H, int l, const Box3& K) {
  const Level& lv = H.lev[l];
  int F[3], off[3];  // folded extents per axis
  for (int ax = 0; ax < 3; ++ax) {
    if (H.prm.periodic[ax]) { F[ax] = lv.M[ax]; off[ax] = 0; }
    else { F[ax] = 2 * lv.M[ax] - 1; off[ax] = lv.M[ax] - 1; }
  }
  std::vector<double> fold((size_t)F[0] * F[1] * F[2], 0.0);
  auto fidx = [&](int ax, int d) -> int {
    if (H.prm.periodic[ax]) { int r = d % lv.M[ax]; return r < 0 ? r + lv.M[ax] : r; }
    return (d < -off[ax] || d > off[ax]) ? -1 : d + off[ax];
  };
  for (int dz = -K.R[2]; dz <= K.R[2]; ++dz) {
    const int fz = fidx(2, dz); if (fz < 0) continue;
    for (int dy = -K.R[1]; dy <= K.R[1]; ++dy) {
      const int fy = fidx(1, dy); if (fy < 0) continue;
      for (int dx = -K.R[0]; dx <= K.R[0]; ++dx) {
        const int fx = fidx(0, dx); if (fx < 0) continue;
        fold[((size_t)fz * F[1] + fy) * F[0] + fx] += K.v[K.idx(dx, dy, dz)];
      }
    }
  }
  const int G = (int)lv.points();
  std::vector<double> C((size_t)G * G);
  for (int m = 0; m < G; ++m) {
    const int mx = m % lv.M[0], my = (m / lv.M[0]) % lv.M[1], mz = m / (lv.M[0] * lv.M[1]);
    for (int n = 0; n < G; ++n) {
      const int nx = n % lv.M[0], ny = (n / lv.M[0]) % lv.M[1], nz = n / (lv.M[0] * lv.M[1]);
      const int fx = fidx(0, mx - nx), fy = fidx(1, my - ny), fz = fidx(2, mz - nz);
      C[(size_t)m * G + n] = fold[((size_t)fz * F[1] + fy) * F[0] + fx];
    }
  }
  return C;
}

// dense restriction matrix (G_{l+1} x G_l), Kronecker product of the one-axis maps (Eq. 19)
std::vector<double> dense_restriction(const Hierarchy& H, const std::vector<double>& J, int l) {
  const Level &f = H.lev[l], &c = H.lev[l + 1];
  std::vector<double> r1[3];
  for (int ax = 0; ax < 3; ++ax) {
    r1[ax].assign((size_t)c.M[ax] * f.M[ax], 0.0);
    if (H.prm.periodic[ax] && f.M[ax] == 1) { r1[ax][0] = 1.0; continue; }
    for (int m = 0; m < c.M[ax]; ++m)
      for (int n = -H.hp; n <= H.hp; ++n) {
        int g;
        if (H.prm.periodic[ax]) { g = (2 * m + n) % f.M[ax]; if (g < 0) g += f.M[ax]; }
        else { g = 2 * (m + c.lo[ax]) + n - f.lo[ax]; if (g < 0 || g >= f.M[ax]) continue; }
        r1[ax][(size_t)m * f.M[ax] + g] += J[n + H.hp];
      }
  }
  const int Gc = (int)c.points(), Gf = (int)f.points();
  std::vector<double> R((size_t)Gc * Gf);
  for (int m = 0; m < Gc; ++m) {
    const int mx = m % c.M[0], my = (m / c.M[0]) % c.M[1], mz = m / (c.M[0] * c.M[1]);
    for (int n = 0; n < Gf; ++n) {
      const int nx = n % f.M[0], ny = (n / f.M[0]) % f.M[1], nz = n / (f.M[0] * f.M[1]);
      R[(size_t)m * Gf + n] = r1[0][(size_t)mx * f.M[0] + nx] * r1[1][(size_t)my * f.M[1] + ny] *
                              r1[2][(size_t)mz * f.M[2] + nz];
    }
  }
  return R;
}

// out (Gf x Gf) += R^T (Gf x Gc) * T (Gc x Gc) * R (Gc x Gf)
void add_rt_t_r(std::vector<double>& out, const std::vector<double>& R, const std::vector<double>& T,
                int Gc, int Gf) {
  std::vector<double> TR((size_t)Gc * Gf, 0.0);
  for (int i = 0; i < Gc; ++i)
    for (int k = 0; k < Gc; ++k) {
      const double t = T[(size_t)i * Gc + k];
      if (t == 0.0) continue;
      const double* rk = &R[(size_t)k * Gf];
      double* o = &TR[(size_t)i * Gf];
      for (int j = 0; j < Gf; ++j) o[j] += t * rk[j];
    }
  for (int k = 0; k < Gc; ++k)
    for (int i = 0; i < Gf; ++i) {
      const double r = R[(size_t)k * Gf + i];
      if (r == 0.0) continue;
      const double* tk = &TR[(size_t)k * Gf];
      double* o = &out[(size_t)i * Gf];
      for (int j = 0; j < Gf; ++j) o[j] += r * tk[j];
    }
}

}  // namespace

TopOperator build_top_operator(const Hierarchy& H, const Splitting& S, const std::vector<double>& omega,
                               const std::vector<double>& J, int n_t, bool with_virial) {
  const int nk = with_virial ? 7 : 1;
  std::vector<double> T[7];  // running operator of the level above
  int Gabove = 0;
  for (int l = H.L; l >= n_t; --l) {
    const Level& lv = H.lev[l];
    const int G = (int)lv.points();
    std::vector<double> cur[7];
    const bool zero_level = (l == H.L && H.top == kTopPeriodic);  // reading T2
    int Kr[3], wax[3] = {H.w, H.w, H.w};
    for (int ax = 0; ax < 3; ++ax) {
      if (l < H.L) Kr[ax] = (int)std::floor(std::ldexp(S.a, l) / lv.h[ax]) + H.w;
      else if (H.top == kTopSlab && ax != H.open_axis) { Kr[ax] = 0; wax[ax] = 0; }
      else Kr[ax] = lv.M[ax] - 1;  // untruncated k_L over the whole grid (reading T1 / T3)
    }
    for (int k = 0; k < nk; ++k) {
      if (zero_level) cur[k].assign((size_t)G * G, 0.0);
      else cur[k] = dense_convolution(H, l, full_stencil(H, S, omega, l, k, Kr, wax));
    }
    if (l < H.L) {
      const std::vector<double> R = dense_restriction(H, J, l);
      for (int k = 0; k < nk; ++k) add_rt_t_r(cur[k], R, T[k], Gabove, G);
    }
    for (int k = 0; k < nk; ++k) T[k].swap(cur[k]);
    Gabove = G;
  }
  TopOperator op;
  op.G = Gabove;
  op.T.swap(T[0]);
  if (with_virial)
    for (int k = 0; k < 6; ++k) op.TD[k].swap(T[k + 1]);
  return op;
}

}  // namespace msm
