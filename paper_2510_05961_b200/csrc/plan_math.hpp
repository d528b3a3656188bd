// plan_math.hpp -- host-side (fp64) mathematics of an MSM plan: grid hierarchy, splitting kernels,
// B-spline piece polynomials, two-scale mask, quasi-interpolation sequence, sampled stencils and
// the dense top-level operator. Product code: shares nothing with oracle/.
//
// Citations: P:<line> = PAPER.md line; readings (K1, G1, ...) are listed in DESIGN.md.
#pragma once
#include <cmath>
#include <cstdint>
#include <vector>

namespace msm {

constexpr int kMaxLevels = 32;
constexpr int kMaxP = 8;

struct Params {
  double box[3];
  int periodic[3];
  double h, a;
  int p, levels, mu;
};

struct Level {
  int M[3];      // points per axis
  int lo[3];     // node index of the first point (0 on periodic axes)
  double h[3];   // spacing
  size_t points() const { return (size_t)M[0] * M[1] * M[2]; }
};

enum TopKind { kTopOpen = 1, kTopPeriodic = 2, kTopSlab = 3 };

// Softened splitting of 1/r (Eq. 21).
struct Splitting {
  int p;
  double a;
  int L;
  double c[kMaxP];  // binom(-1/2, k)
  Splitting(int p_, double a_, int L_);
  double g(double s) const;        // gamma(rho) for rho <= 1 as polynomial in s = rho^2 - 1
  double dg(double s) const;       // d g / d s
  double gamma(double rho) const;
  double dgamma(double rho) const; // d gamma / d rho
  double k(int l, double r) const;   // k_l(r), 1 <= l <= L
  double dk(int l, double r) const;  // k_l'(r)
  double gamma0() const { return gamma(0.0); }
};

// Piece polynomials of the central B-spline of order p: weight of node offset j (j = -p/2+1..p/2)
// for a particle at fraction t in [0,1) of its cell is sum_k coef[j + p/2 - 1][k] t^k.
struct SplinePieces {
  int p;
  double coef[kMaxP][kMaxP];
  double dcoef[kMaxP][kMaxP];  // derivative w.r.t. t (degree p-2)
  explicit SplinePieces(int p);
  double value_at_integer(int n) const;  // Phi(n)
};

std::vector<double> two_scale_mask(int p);              // J_n, n = -p/2..p/2 (reading J1)
std::vector<double> quasi_interp_sequence(int p, int mu);  // omega'_n, n = -w..w (reading Q)

struct Hierarchy {
  Params prm;
  int hp, L, n_per, w;
  TopKind top;
  int open_axis;  // slab only
  std::vector<Level> lev;  // index 1..L (0 unused)
  int status;              // 0 ok; 2 unsupported; 3 invalid; 4 cutoff too large
  explicit Hierarchy(const Params& prm);
};

// Sampled stencil of one tiled level: values s(n) = k_l(|h o n|) and g(n) = k_l'(r)/r inside the
// cutoff ellipsoid, as a dense box [-R, R] per axis (x fastest), zero outside.
struct SampledStencil {
  int R[3];
  std::vector<double> s, g;
  int taps;  // non-zero count of s
  double at(const std::vector<double>& v, int dx, int dy, int dz) const {
    return v[((size_t)(dz + R[2]) * (2 * R[1] + 1) + (dy + R[1])) * (2 * R[0] + 1) + (dx + R[0])];
  }
};
// hstruct (optional): spacings that size the box [-R, R] (a plan that reserves room for a smaller
// cell, msm_plan_set_box); the values are always sampled at the level's actual spacings.
SampledStencil sample_level_stencil(const Hierarchy& H, const Splitting& S, int l, const double* hstruct = nullptr);

// Dense operators of the top grid (level n_t): e = T q completes the hierarchy from level n_t up
// to level L (convolution at each level, restriction up, prolongation down; Eq. 13),
// and TD[k] are the same with every stencil replaced by its strain derivative (component k of
// xx yy zz xy xz yz), so that the top part of the virial is -1/2 q^T TD[k] q (reading V).
struct TopOperator {
  int G;
  std::vector<double> T;
  std::vector<double> TD[6];
};
TopOperator build_top_operator(const Hierarchy& H, const Splitting& S, const std::vector<double>& omega,
                               const std::vector<double>& J, int n_t, bool with_virial);

}  // namespace msm
