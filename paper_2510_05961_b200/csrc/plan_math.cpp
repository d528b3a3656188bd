// plan_math.cpp -- host-side fp64 mathematics of an MSM plan (see plan_math.hpp).
#include "plan_math.hpp"

#include <algorithm>
#include <cstring>

namespace msm {

// ------------------------------------------------------------------ splitting (Eq. 21)

Splitting::Splitting(int p_, double a_, int L_) : p(p_), a(a_), L(L_) {
  // Taylor coefficients of s^(-1/2) about s = 1: binom(-1/2, k)
  double v = 1.0;
  for (int k = 0; k < kMaxP; ++k) {
    c[k] = v;
    v *= (-0.5 - k) / (k + 1.0);
  }
}

double Splitting::g(double s) const {  // Horner in s = rho^2 - 1
  double acc = c[p - 1];
  for (int k = p - 2; k >= 0; --k) acc = acc * s + c[k];
  return acc;
}

double Splitting::dg(double s) const {
  double acc = (p - 1) * c[p - 1];
  for (int k = p - 2; k >= 1; --k) acc = acc * s + k * c[k];
  return acc;
}

double Splitting::gamma(double rho) const { return rho >= 1.0 ? 1.0 / rho : g(rho * rho - 1.0); }

double Splitting::dgamma(double rho) const {
  return rho >= 1.0 ? -1.0 / (rho * rho) : 2.0 * rho * dg(rho * rho - 1.0);
}

// k_l for 1 <= l <= L; the first gamma of the middle case takes r / (2^(l-1) a) (reading K1)
double Splitting::k(int l, double r) const {
  const double A0 = std::ldexp(a, l - 1), A1 = std::ldexp(a, l);
  if (l == L) return gamma(r / A0) / A0;
  if (r >= A1) return 0.0;  // r_cut^(l) = 2^l a (Eq. 3)
  return gamma(r / A0) / A0 - gamma(r / A1) / A1;
}

double Splitting::dk(int l, double r) const {
  const double A0 = std::ldexp(a, l - 1), A1 = std::ldexp(a, l);
  if (l == L) return dgamma(r / A0) / (A0 * A0);
  if (r >= A1) return 0.0;
  return dgamma(r / A0) / (A0 * A0) - dgamma(r / A1) / (A1 * A1);
}

// ------------------------------------------------------------------ B-spline pieces

SplinePieces::SplinePieces(int p_) : p(p_) {
  // piece[i] of Q_k on [i, i+1) as a polynomial in the local variable t = x - i;
  // Cox-de Boor: Q_k(x) = [x Q_{k-1}(x) + (k - x) Q_{k-1}(x-1)] / (k-1), carried out on coefficients
  std::vector<std::vector<double>> prev(1, std::vector<double>(1, 1.0));  // Q_1: one piece, 1
  for (int k = 2; k <= p; ++k) {
    std::vector<std::vector<double>> cur(k, std::vector<double>(k, 0.0));
    for (int i = 0; i < k; ++i) {
      for (int d = 0; d < k - 1; ++d) {
        const double ai = (i <= k - 2) ? prev[i][d] : 0.0;       // Q_{k-1} piece i
        const double am = (i >= 1) ? prev[i - 1][d] : 0.0;       // Q_{k-1}(x-1): piece i-1
        // (i + t) * ai t^d + (k - i - t) * am t^d
        cur[i][d] += (i * ai + (k - i) * am) / (k - 1);
        cur[i][d + 1] += (ai - am) / (k - 1);
      }
    }
    prev.swap(cur);
  }
  std::memset(coef, 0, sizeof(coef));
  std::memset(dcoef, 0, sizeof(dcoef));
  const int hp = p / 2;
  for (int j = -hp + 1; j <= hp; ++j) {
    // Phi(t - j) = Q_p(t + hp - j): piece hp - j
    const std::vector<double>& pc = prev[hp - j];
    for (int d = 0; d < p; ++d) coef[j + hp - 1][d] = pc[d];
    for (int d = 1; d < p; ++d) dcoef[j + hp - 1][d - 1] = d * pc[d];
  }
}

double SplinePieces::value_at_integer(int n) const {
  // Phi(n) = weight of node offset j = -n at t = 0
  const int hp = p / 2, j = -n;
  if (j < -hp + 1 || j > hp) return 0.0;
  return coef[j + hp - 1][0];
}

// ------------------------------------------------------------------ two-scale mask (reading J1)

std::vector<double> two_scale_mask(int p) {
  std::vector<double> J(p + 1);
  double b = 1.0;  // binom(p, k)
  for (int k = 0; k <= p; ++k) {
    J[k] = std::ldexp(b, 1 - p);
    b = b * (p - k) / (k + 1.0);
  }
  return J;
}

// ------------------------------------------------------------------ omega' (reading Q)

static double binom(int n, int k) {
  double b = 1.0;
  for (int j = 1; j <= k; ++j) b = b * (n - k + j) / j;
  return b;
}

std::vector<double> quasi_interp_sequence(int p, int mu) {
  const int hp = p / 2, w = hp - 1 + mu;
  SplinePieces sp(p);
  // symbol of the sampled spline in powers of t = delta^2 = z - 2 + 1/z
  std::vector<double> b(hp), A(hp);
  for (int n = 0; n < hp; ++n) b[n] = sp.value_at_integer(n);
  for (int k = hp - 1; k >= 0; --k) {
    A[k] = b[k];
    for (int n = 0; n <= k; ++n) b[n] -= A[k] * (((k - n) & 1) ? -1.0 : 1.0) * binom(2 * k, k + n);
  }
  // series of 1 / A(t)^2 up to t^w
  std::vector<double> A2(2 * hp - 1, 0.0), cs(w + 1, 0.0);
  for (int i = 0; i < hp; ++i)
    for (int j = 0; j < hp; ++j) A2[i + j] += A[i] * A[j];
  for (int k = 0; k <= w; ++k) {
    double s = (k == 0) ? 1.0 : 0.0;
    for (int j = 1; j <= k && j < (int)A2.size(); ++j) s -= A2[j] * cs[k - j];
    cs[k] = s / A2[0];
  }
  std::vector<double> om(2 * w + 1);
  for (int n = 0; n <= w; ++n) {
    double s = 0.0;
    for (int k = n; k <= w; ++k) s += cs[k] * (((k - n) & 1) ? -1.0 : 1.0) * binom(2 * k, k + n);
    om[w + n] = om[w - n] = s;
  }
  return om;
}

// ------------------------------------------------------------------ grid hierarchy (G1-G4)

Hierarchy::Hierarchy(const Params& P) : prm(P), hp(P.p / 2), L(0), n_per(0), w(0), top(kTopOpen),
                                        open_axis(-1), status(0) {
  if (P.p < 4 || P.p > kMaxP || (P.p & 1) || !(P.h > 0) || !(P.a > 0) || P.levels < 1 || P.mu < 0) {
    status = 3;
    return;
  }
  for (int ax = 0; ax < 3; ++ax) {
    if (!(P.box[ax] > 0)) { status = 3; return; }
    if (P.periodic[ax] && P.a > 0.5 * P.box[ax]) { status = 4; return; }
    n_per += P.periodic[ax] ? 1 : 0;
  }
  w = hp - 1 + P.mu;
  if (n_per == 1) { status = 2; return; }  // reading T4
  top = n_per == 0 ? kTopOpen : (n_per == 3 ? kTopPeriodic : kTopSlab);
  Level l1;
  int maxM = 1;
  for (int ax = 0; ax < 3; ++ax) {
    if (P.periodic[ax]) {
      int e = (int)std::lround(std::log2(P.box[ax] / P.h));  // reading G1
      if (e < 0) e = 0;
      l1.M[ax] = 1 << e;
      l1.lo[ax] = 0;
      l1.h[ax] = P.box[ax] / l1.M[ax];
      maxM = std::max(maxM, l1.M[ax]);
    } else {
      open_axis = ax;
      l1.lo[ax] = -(hp - 1);  // reading G2
      const int hi = (int)std::floor(P.box[ax] / P.h) + hp;
      l1.M[ax] = hi - l1.lo[ax] + 1;
      l1.h[ax] = P.h;
    }
  }
  // reading B3: periodic axes may start from different grid counts; an axis that has reached one
  // point keeps it (spacing = box edge) while the others go on halving
  if (n_per == 0) L = P.levels;
  else { L = 1; while ((1 << (L - 1)) < maxM) ++L; }  // until one point per periodic axis
  if (L > kMaxLevels) { status = 3; return; }
  lev.resize(L + 1);
  lev[1] = l1;
  for (int l = 1; l < L; ++l) {
    for (int ax = 0; ax < 3; ++ax) {
      const Level& f = lev[l];
      Level& c = lev[l + 1];
      if (P.periodic[ax]) {
        c.M[ax] = std::max(f.M[ax] / 2, 1);
        c.lo[ax] = 0;
        c.h[ax] = P.box[ax] / c.M[ax];
      } else {  // reading G3
        const int fhi = f.lo[ax] + f.M[ax] - 1;
        c.lo[ax] = (int)std::ceil(0.5 * (f.lo[ax] - hp));
        const int chi = (int)std::floor(0.5 * (fhi + hp));
        c.M[ax] = chi - c.lo[ax] + 1;
        c.h[ax] = 2.0 * f.h[ax];
      }
    }
  }
}

}  // namespace msm
