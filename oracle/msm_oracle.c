/* oracle/msm_oracle.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * A plain, slow, fp64 CPU implementation of the multilevel summation method with B-spline
 * interpolation (arxiv 2510.05961, "msmJAX"), written from the paper's text (PAPER.md, cited
 * as P:<line>) and the readings listed in DESIGN.md (K1, K2, G1-G4, J1, Q, T1-T4, V, B1-B3).
 * It follows the algorithm step by step in the paper's order and notation; there is no tiling,
 * fusion or reordering. It shares no code with the CUDA path (paper_2510_05961_b200/csrc) and
 * neither includes the other. Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
 * --impl reference legs may use it.
 *
 * OpenMP appears only on loops over independent outputs (each output is still the plain sum of
 * its definition, accumulated serially in lexicographic order).
 *
 * What pins it (tests/test_oracle_*.py): telescoping of Eq. 21, closed forms of gamma and of the
 * B-splines, partition of unity, the two-scale relation, <Iq,e> = <q,I^T e>, polynomial
 * reproduction of the quasi-interpolant, restricted charge == anterpolation on the coarse grid,
 * forces/potentials/virial == finite differences of the energy, convergence to the O(N^2) direct
 * Coulomb sum, the rock-salt Madelung constant, and a brute-force image sum for a small slab.
 * "parity unpinned": msmJAX's own numerical identity (its exact omega', its open-axis grid
 * extents, its slab treatment) -- neither its code nor printed intermediate values are available.
 */
#include <math.h>
#include <stdlib.h>
#include <string.h>
#include <stdio.h>

#define MSMO_MAXLEV 40
#define MSMO_MAXP 8
#define MSMO_MAXW 64

typedef struct {
  double box[3];
  int periodic[3];
  double h;      /* target finest spacing */
  double a;      /* level-zero cutoff r_cut^(0) */
  int p;         /* B-spline order (even) */
  int levels;    /* used only when no axis is periodic (reading G4) */
  int mu;        /* extra quasi-interpolation terms (reading Q) */
  int pad;       /* test knob for reading G3's pin: extra nodes added on both sides of every open
                    axis at every level (0 = the minimal extents of G2/G3); no output may depend
                    on it beyond round-off */
} msmo_params;

typedef struct {
  msmo_params prm;
  int hp, L, w, nper;
  int top_kind;                    /* 1 = T1 open, 2 = T2 periodic, 3 = T3 slab */
  int open_axis;                   /* for T3 */
  int lo[MSMO_MAXLEV + 1][3], hi[MSMO_MAXLEV + 1][3], M[MSMO_MAXLEV + 1][3];
  double hl[MSMO_MAXLEV + 1][3];
  double J[MSMO_MAXP + 1];         /* J_n at index n + hp */
  double omega[2 * MSMO_MAXW + 1]; /* omega'_n at index n + w */
  double *K[MSMO_MAXLEV + 1];      /* K^l, box of half-widths Kr */
  double *D[MSMO_MAXLEV + 1][6];   /* strain derivatives of K^l: xx yy zz xy xz yz */
  int Kr[MSMO_MAXLEV + 1][3];
  double *Q[MSMO_MAXLEV + 1], *E[MSMO_MAXLEV + 1];
  int have_D;
} msmo_ctx;

/* ------------------------------------------------------------------ softening and splitting */

/* c_k = binom(-1/2, k): Taylor coefficients of s^(-1/2) about s = 1. */
static double binom_mhalf(int k) {
  double c = 1.0;
  for (int j = 1; j <= k; ++j) c *= (-0.5 - (double)(j - 1)) / (double)j;
  return c;
}

/* gamma(rho): 1/rho for rho >= 1; for rho <= 1 the degree-(p-1) Taylor polynomial of s^(-1/2)
 * about s = 1 with s = rho^2. */
double msmo_gamma(int p, double rho) {
  if (rho >= 1.0) return 1.0 / rho;
  double s1 = rho * rho - 1.0, pw = 1.0, g = 0.0;
  for (int k = 0; k < p; ++k) { g += binom_mhalf(k) * pw; pw *= s1; }
  return g;
}

/* d gamma / d rho */
double msmo_dgamma(int p, double rho) {
  if (rho >= 1.0) return -1.0 / (rho * rho);
  double s1 = rho * rho - 1.0, pw = 1.0, g = 0.0;
  for (int k = 1; k < p; ++k) { g += binom_mhalf(k) * (double)k * pw; pw *= s1; }
  return g * 2.0 * rho;
}

/* k_l(r), Eq. 21 with reading K1 (argument of the first gamma of the middle case is
 * r / (2^(l-1) a)). l = 0..L. r > 0 for l = 0. */
double msmo_kernel(int p, double a, int L, int l, double r) {
  if (l == 0) return (r < a) ? 1.0 / r - msmo_gamma(p, r / a) / a : 0.0;
  double A0 = ldexp(a, l - 1), A1 = ldexp(a, l);
  if (l == L) return msmo_gamma(p, r / A0) / A0;
  if (r >= A1) return 0.0;                       /* finite range r_cut^(l) = 2^l a (Eq. 3) */
  return msmo_gamma(p, r / A0) / A0 - msmo_gamma(p, r / A1) / A1;
}

/* d k_l / d r */
double msmo_dkernel(int p, double a, int L, int l, double r) {
  if (l == 0) return (r < a) ? -1.0 / (r * r) - msmo_dgamma(p, r / a) / (a * a) : 0.0;
  double A0 = ldexp(a, l - 1), A1 = ldexp(a, l);
  if (l == L) return msmo_dgamma(p, r / A0) / (A0 * A0);
  if (r >= A1) return 0.0;
  return msmo_dgamma(p, r / A0) / (A0 * A0) - msmo_dgamma(p, r / A1) / (A1 * A1);
}

/* ------------------------------------------------------------------ B-splines */

/* Q_k(x): cardinal B-spline of order k on knots 0..k, Cox-de Boor recursion:
 * Q_1 = 1 on [0,1); Q_k(x) = [x Q_{k-1}(x) + (k-x) Q_{k-1}(x-1)] / (k-1). */
static double bspline_Q(int k, double x) {
  if (k == 1) return (x >= 0.0 && x < 1.0) ? 1.0 : 0.0;
  if (x <= 0.0 || x >= (double)k) return 0.0;
  return (x * bspline_Q(k - 1, x) + ((double)k - x) * bspline_Q(k - 1, x - 1.0)) / (double)(k - 1);
}

/* central B-spline Phi_p(u) = Q_p(u + p/2), support [-p/2, p/2] */
double msmo_bspline(int p, double u) { return bspline_Q(p, u + 0.5 * p); }

/* Phi_p'(u) = Phi_{p-1}(u + 1/2) - Phi_{p-1}(u - 1/2) */
double msmo_dbspline(int p, double u) {
  return bspline_Q(p - 1, u + 0.5 * p) - bspline_Q(p - 1, u + 0.5 * p - 1.0);
}

/* J_n = 2^(1-p) binom(p, n + p/2), |n| <= p/2 (reading J1): Phi(u/2) = sum_n J_n Phi(u - n). */
void msmo_two_scale(int p, double *J) {
  int hp = p / 2;
  for (int n = -hp; n <= hp; ++n) {
    double b = 1.0;
    int k = n + hp;
    for (int j = 1; j <= k; ++j) b = b * (double)(p - k + j) / (double)j;
    J[n + hp] = ldexp(b, 1 - p);
  }
}

/* omega'_n, |n| <= w = p/2 - 1 + mu (reading Q): the symmetric sequence whose symbol is the power
 * series of 1 / Phihat(t)^2 in t = delta^2 (second central difference), truncated after
 * t^(p/2-1+mu); Phihat(t) = symbol of the sampled spline Phi(n). out[n + w]. returns w. */
int msmo_omega(int p, int mu, double *out) {
  int hp = p / 2, w = hp - 1 + mu;
  /* sampled spline b_n = Phi(n), |n| <= hp-1, as a polynomial in t: b(z) = sum_k a_k t^k with
   * t^k = (z - 2 + 1/z)^k whose z^n coefficient is (-1)^(k-n) binom(2k, k+n). */
  double b[MSMO_MAXP], acoef[MSMO_MAXP];
  for (int n = 0; n <= hp - 1; ++n) b[n] = msmo_bspline(p, (double)n);
  for (int k = hp - 1; k >= 0; --k) {
    acoef[k] = b[k];                        /* leading coefficient of t^k at z^k is +1 */
    for (int n = 0; n <= k; ++n) {
      double c = 1.0;                       /* binom(2k, k+n) */
      for (int j = 1; j <= k + n; ++j) c = c * (double)(2 * k - (k + n) + j) / (double)j;
      b[n] -= acoef[k] * (((k - n) & 1) ? -c : c);
    }
  }
  /* d = a*a (polynomial), then c = 1/d as a power series up to order w */
  double d[2 * MSMO_MAXP + 2];
  for (int i = 0; i <= 2 * (hp - 1); ++i) d[i] = 0.0;
  for (int i = 0; i <= hp - 1; ++i)
    for (int j = 0; j <= hp - 1; ++j) d[i + j] += acoef[i] * acoef[j];
  double c[MSMO_MAXW + 1];
  for (int k = 0; k <= w; ++k) {
    double s = (k == 0) ? 1.0 : 0.0;
    for (int j = 1; j <= k && j <= 2 * (hp - 1); ++j) s -= d[j] * c[k - j];
    c[k] = s / d[0];
  }
  for (int n = -w; n <= w; ++n) {
    int an = n < 0 ? -n : n;
    double s = 0.0;
    for (int k = an; k <= w; ++k) {
      double bc = 1.0;
      for (int j = 1; j <= k + an; ++j) bc = bc * (double)(2 * k - (k + an) + j) / (double)j;
      s += c[k] * (((k - an) & 1) ? -bc : bc);
    }
    out[n + w] = s;
  }
  return w;
}

/* ------------------------------------------------------------------ geometry (O1) */

static int imod(int i, int m) { int r = i % m; return r < 0 ? r + m : r; }
static int iceil_div2(int v) { return (int)ceil(0.5 * (double)v); }
static int ifloor_div2(int v) { return (int)floor(0.5 * (double)v); }

static int setup_geometry(msmo_ctx *c) {
  const msmo_params *P = &c->prm;
  int hp = c->hp;
  c->nper = P->periodic[0] + P->periodic[1] + P->periodic[2];
  int maxM = 1;
  for (int ax = 0; ax < 3; ++ax) {
    if (P->periodic[ax]) {
      int e = (int)lround(log2(P->box[ax] / P->h));        /* reading G1 */
      if (e < 0) e = 0;
      int m = 1 << e;
      c->M[1][ax] = m; c->lo[1][ax] = 0; c->hi[1][ax] = m - 1;
      c->hl[1][ax] = P->box[ax] / (double)m;
      if (m > maxM) maxM = m;
    } else {
      c->lo[1][ax] = -(hp - 1) - P->pad;                    /* reading G2 (+ the G3 pin's padding) */
      c->hi[1][ax] = (int)floor(P->box[ax] / P->h) + hp + P->pad;
      c->M[1][ax] = c->hi[1][ax] - c->lo[1][ax] + 1;
      c->hl[1][ax] = P->h;
    }
  }
  if (c->nper == 0) c->L = P->levels;                       /* reading G4 */
  else { c->L = 1; while ((1 << (c->L - 1)) < maxM) c->L++; } /* L = log2(maxM) + 1 */
  if (c->L < 1 || c->L > MSMO_MAXLEV) return 1;
  for (int l = 1; l < c->L; ++l)
    for (int ax = 0; ax < 3; ++ax) {
      if (P->periodic[ax]) {
        int m = c->M[l][ax] / 2; if (m < 1) m = 1;
        c->M[l + 1][ax] = m; c->lo[l + 1][ax] = 0; c->hi[l + 1][ax] = m - 1;
        c->hl[l + 1][ax] = P->box[ax] / (double)m;          /* reading B3 */
      } else {
        c->lo[l + 1][ax] = iceil_div2(c->lo[l][ax] - hp) - P->pad;   /* reading G3 */
        c->hi[l + 1][ax] = ifloor_div2(c->hi[l][ax] + hp) + P->pad;
        c->M[l + 1][ax] = c->hi[l + 1][ax] - c->lo[l + 1][ax] + 1;
        c->hl[l + 1][ax] = 2.0 * c->hl[l][ax];
      }
    }
  if (c->nper == 0) c->top_kind = 1;
  else if (c->nper == 3) c->top_kind = 2;
  else if (c->nper == 2) { c->top_kind = 3; for (int ax = 0; ax < 3; ++ax) if (!P->periodic[ax]) c->open_axis = ax; }
  else return 2;                                            /* reading T4: unsupported */
  return 0;
}

/* ------------------------------------------------------------------ stencils (O7, O9, O12) */

typedef double (*sample_fn)(const msmo_ctx *c, int l, int kind, const double r[3]);

/* kind 0: k_l(|r|); kinds 1..6: k_l'(|r|) r_a r_b / |r| for (a,b) = xx yy zz xy xz yz */
static const int AB[7][2] = {{0, 0}, {0, 0}, {1, 1}, {2, 2}, {0, 1}, {0, 2}, {1, 2}};

static double sample_radial(const msmo_ctx *c, int l, int kind, const double r[3]) {
  double rr = sqrt(r[0] * r[0] + r[1] * r[1] + r[2] * r[2]);
  if (kind == 0) return msmo_kernel(c->prm.p, c->prm.a, c->L, l, rr);
  if (rr == 0.0) return 0.0;
  return msmo_dkernel(c->prm.p, c->prm.a, c->L, l, rr) * r[AB[kind][0]] * r[AB[kind][1]] / rr;
}

/* P(x) = int_0^x t gamma(t) dt for x <= 1 (reading T3), from the c_k:
 * t gamma(t) = sum_k c_k t (t^2-1)^k -> integral = sum_k c_k [(x^2-1)^(k+1) - (-1)^(k+1)] / (2(k+1)) */
static double slab_P(int p, double x) {
  double s1 = x * x - 1.0, pw = s1, sgn = -1.0, acc = 0.0;
  for (int k = 0; k < p; ++k) {
    acc += binom_mhalf(k) * (pw - sgn) / (2.0 * (double)(k + 1));
    pw *= s1; sgn = -sgn;
  }
  return acc;
}

/* slab top level (reading T3): plane-averaged k_L along the open axis; r has only the open
 * component non-zero. kind 0: s_L; strain derivatives: periodic diagonal -s_L, open diagonal
 * -(2 pi / (Lx Ly)) z^2 k_L(|z|), off-diagonal 0. */
static double sample_slab(const msmo_ctx *c, int l, int kind, const double r[3]) {
  int oz = c->open_axis;
  double area = 1.0;
  for (int ax = 0; ax < 3; ++ax) if (ax != oz) area *= c->prm.box[ax];
  double A = ldexp(c->prm.a, c->L - 1);
  double z = fabs(r[oz]), rho = z / A;
  double sL = -(2.0 * M_PI / area) * A * (slab_P(c->prm.p, rho < 1.0 ? rho : 1.0) + (rho > 1.0 ? rho - 1.0 : 0.0));
  if (kind == 0) return sL;
  if (kind > 3) return 0.0;
  if (kind - 1 != oz) return -sL;
  return -(2.0 * M_PI / area) * z * z * msmo_kernel(c->prm.p, c->prm.a, c->L, l, z);
}

/* K[d] = sum_n w'[dx-nx] w'[dy-ny] w'[dz-nz] f(h o n) for |d_ax| <= Kr_ax (Eq. 20), one
 * coordinate direction at a time; f sampled on |n_ax| <= Kr_ax + w_ax ("valid" convolution). */
static double *build_stencil(const msmo_ctx *c, int l, int kind, sample_fn fn, const int Kr[3],
                             const int wax[3]) {
  int S[3], n0[3];
  for (int ax = 0; ax < 3; ++ax) { n0[ax] = Kr[ax] + wax[ax]; S[ax] = 2 * n0[ax] + 1; }
  size_t tot = (size_t)S[0] * S[1] * S[2];
  double *cur = (double *)malloc(tot * sizeof(double));
  for (int z = 0; z < S[2]; ++z) for (int y = 0; y < S[1]; ++y) for (int x = 0; x < S[0]; ++x) {
    double r[3] = {(x - n0[0]) * c->hl[l][0], (y - n0[1]) * c->hl[l][1], (z - n0[2]) * c->hl[l][2]};
    cur[((size_t)z * S[1] + y) * S[0] + x] = fn(c, l, kind, r);
  }
  int dims[3] = {S[0], S[1], S[2]};
  for (int ax = 0; ax < 3; ++ax) {
    if (wax[ax] == 0) continue;
    int nd[3] = {dims[0], dims[1], dims[2]};
    nd[ax] = 2 * Kr[ax] + 1;
    double *nxt = (double *)calloc((size_t)nd[0] * nd[1] * nd[2], sizeof(double));
    int wv = wax[ax];
    for (int z = 0; z < nd[2]; ++z) for (int y = 0; y < nd[1]; ++y) for (int x = 0; x < nd[0]; ++x) {
      int o[3] = {x, y, z};
      double acc = 0.0;
      for (int k = -wv; k <= wv; ++k) {      /* out[d] = sum_k w'[k] in[d - k]; in index shifted by wv */
        int i[3] = {x, y, z};
        i[ax] = o[ax] - k + wv;
        acc += c->omega[k + c->w] * cur[((size_t)i[2] * dims[1] + i[1]) * dims[0] + i[0]];
      }
      nxt[((size_t)z * nd[1] + y) * nd[0] + x] = acc;
    }
    free(cur); cur = nxt; dims[ax] = nd[ax];
  }
  return cur;
}

static void setup_stencils(msmo_ctx *c, int with_D) {
  int Lk = (c->top_kind == 2) ? c->L - 1 : c->L;    /* T2: single-point top level contributes 0 */
  for (int l = 1; l <= Lk; ++l) {
    int wax[3] = {c->w, c->w, c->w};
    sample_fn fn = sample_radial;
    if (l < c->L) {
      double A = ldexp(c->prm.a, l);
      for (int ax = 0; ax < 3; ++ax) c->Kr[l][ax] = (int)floor(A / c->hl[l][ax]) + c->w;
    } else if (c->top_kind == 1) {
      for (int ax = 0; ax < 3; ++ax) c->Kr[l][ax] = c->M[l][ax] - 1;   /* T1: all pairs */
    } else {                                                          /* T3 */
      fn = sample_slab;
      for (int ax = 0; ax < 3; ++ax) {
        if (ax == c->open_axis) c->Kr[l][ax] = c->M[l][ax] - 1;
        else { c->Kr[l][ax] = 0; wax[ax] = 0; }
      }
    }
    if (!c->K[l]) c->K[l] = build_stencil(c, l, 0, fn, c->Kr[l], wax);
    if (with_D && !c->D[l][0])
      for (int k = 0; k < 6; ++k) c->D[l][k] = build_stencil(c, l, k + 1, fn, c->Kr[l], wax);
  }
  if (with_D) c->have_D = 1;
}

/* ------------------------------------------------------------------ create / destroy / info */

msmo_ctx *msmo_create(const msmo_params *prm, int *status) {
  msmo_ctx *c = (msmo_ctx *)calloc(1, sizeof(msmo_ctx));
  c->prm = *prm;
  int st = 0;
  if (prm->p < 2 || prm->p > MSMO_MAXP || (prm->p & 1) || prm->h <= 0 || prm->a <= 0 || prm->mu < 0 || prm->pad < 0) st = 3;
  for (int ax = 0; ax < 3 && !st; ++ax) {
    if (prm->box[ax] <= 0) st = 3;
    if (prm->periodic[ax] && prm->a > 0.5 * prm->box[ax]) st = 4;   /* minimum image */
  }
  if (!st) {
    c->hp = prm->p / 2;
    msmo_two_scale(prm->p, c->J);
    c->w = msmo_omega(prm->p, prm->mu, c->omega);
    st = setup_geometry(c);
  }
  if (!st) {
    for (int l = 1; l <= c->L; ++l) {
      size_t g = (size_t)c->M[l][0] * c->M[l][1] * c->M[l][2];
      c->Q[l] = (double *)calloc(g, sizeof(double));
      c->E[l] = (double *)calloc(g, sizeof(double));
    }
    setup_stencils(c, 0);
  }
  if (status) *status = st;
  if (st) { free(c); return NULL; }
  return c;
}

void msmo_destroy(msmo_ctx *c) {
  if (!c) return;
  for (int l = 0; l <= MSMO_MAXLEV; ++l) {
    free(c->K[l]); free(c->Q[l]); free(c->E[l]);
    for (int k = 0; k < 6; ++k) free(c->D[l][k]);
  }
  free(c);
}

int msmo_num_levels(const msmo_ctx *c) { return c->L; }
int msmo_omega_halfwidth(const msmo_ctx *c) { return c->w; }
void msmo_copy_omega(const msmo_ctx *c, double *out) { memcpy(out, c->omega, (2 * c->w + 1) * sizeof(double)); }

void msmo_level_info(const msmo_ctx *c, int l, int *M, int *lo, double *h, int *Kr) {
  for (int ax = 0; ax < 3; ++ax) { M[ax] = c->M[l][ax]; lo[ax] = c->lo[l][ax]; h[ax] = c->hl[l][ax]; Kr[ax] = c->K[l] ? c->Kr[l][ax] : -1; }
}

/* kind 0 = Q^l, 1 = E^l (after the last evaluate) */
void msmo_copy_grid(const msmo_ctx *c, int l, int kind, double *out) {
  size_t g = (size_t)c->M[l][0] * c->M[l][1] * c->M[l][2];
  memcpy(out, kind == 0 ? c->Q[l] : c->E[l], g * sizeof(double));
}

/* kind 0 = K^l, 1..6 = D^l components (built on demand) */
int msmo_copy_stencil(msmo_ctx *c, int l, int kind, double *out) {
  if (kind > 0 && !c->have_D) setup_stencils(c, 1);
  const double *src = kind == 0 ? c->K[l] : c->D[l][kind - 1];
  if (!src) return 1;
  size_t g = (size_t)(2 * c->Kr[l][0] + 1) * (2 * c->Kr[l][1] + 1) * (2 * c->Kr[l][2] + 1);
  memcpy(out, src, g * sizeof(double));
  return 0;
}

/* ------------------------------------------------------------------ particle <-> grid (O4, O5, O11) */

static double wrap_coord(double x, double L) { double y = x - L * floor(x / L); if (y >= L) y = 0.0; return y; }

/* nodes and weights of one particle on one axis (Eq. 15): i0 = floor(x/h), t = x/h - i0,
 * nodes i0 + j, j = -hp+1..hp, weights Phi(t - j), derivative Phi'(t - j) / h. */
static void axis_weights(const msmo_ctx *c, int ax, double x, int *idx, double *wv, double *dw) {
  int p = c->prm.p, hp = c->hp;
  double h = c->hl[1][ax];
  if (c->prm.periodic[ax]) x = wrap_coord(x, c->prm.box[ax]);
  double s = x / h;
  int i0 = (int)floor(s);
  double t = s - (double)i0;
  for (int j = -hp + 1; j <= hp; ++j) {
    int n = i0 + j;
    idx[j + hp - 1] = c->prm.periodic[ax] ? imod(n, c->M[1][ax]) : n - c->lo[1][ax];
    wv[j + hp - 1] = msmo_bspline(p, t - (double)j);
    if (dw) dw[j + hp - 1] = msmo_dbspline(p, t - (double)j) / h;
  }
}

/* Algorithm 1: q~1_m += q_i phi_m(r_i), outer loop particles, inner loop nearby points */
void msmo_anterpolate(msmo_ctx *c, int n, const double *pos, const double *q) {
  int p = c->prm.p;
  const int *M = c->M[1];
  memset(c->Q[1], 0, (size_t)M[0] * M[1] * M[2] * sizeof(double));
  for (int i = 0; i < n; ++i) {
    int ix[MSMO_MAXP], iy[MSMO_MAXP], iz[MSMO_MAXP];
    double wx[MSMO_MAXP], wy[MSMO_MAXP], wz[MSMO_MAXP];
    axis_weights(c, 0, pos[3 * i + 0], ix, wx, NULL);
    axis_weights(c, 1, pos[3 * i + 1], iy, wy, NULL);
    axis_weights(c, 2, pos[3 * i + 2], iz, wz, NULL);
    for (int kz = 0; kz < p; ++kz) for (int ky = 0; ky < p; ++ky) for (int kx = 0; kx < p; ++kx)
      c->Q[1][((size_t)iz[kz] * M[1] + iy[ky]) * M[0] + ix[kx]] += q[i] * (wx[kx] * wy[ky] * wz[kz]);
  }
}

/* Eq. 16-18: V_i += sum_m e_m phi_m(r_i);  F_i -= q_i sum_m e_m grad phi_m(r_i) */
void msmo_interpolate(const msmo_ctx *c, int n, const double *pos, const double *q, double *F, double *V) {
  int p = c->prm.p;
  const int *M = c->M[1];
  const double *E = c->E[1];
#pragma omp parallel for schedule(static)
  for (int i = 0; i < n; ++i) {
    int ix[MSMO_MAXP], iy[MSMO_MAXP], iz[MSMO_MAXP];
    double wx[MSMO_MAXP], wy[MSMO_MAXP], wz[MSMO_MAXP], dx[MSMO_MAXP], dy[MSMO_MAXP], dz[MSMO_MAXP];
    axis_weights(c, 0, pos[3 * i + 0], ix, wx, dx);
    axis_weights(c, 1, pos[3 * i + 1], iy, wy, dy);
    axis_weights(c, 2, pos[3 * i + 2], iz, wz, dz);
    double v = 0, gx = 0, gy = 0, gz = 0;
    for (int kz = 0; kz < p; ++kz) for (int ky = 0; ky < p; ++ky) for (int kx = 0; kx < p; ++kx) {
      double e = E[((size_t)iz[kz] * M[1] + iy[ky]) * M[0] + ix[kx]];
      v += e * (wx[kx] * wy[ky] * wz[kz]);
      gx += e * (dx[kx] * wy[ky] * wz[kz]);
      gy += e * (wx[kx] * dy[ky] * wz[kz]);
      gz += e * (wx[kx] * wy[ky] * dz[kz]);
    }
    V[i] += v;
    F[3 * i + 0] -= q[i] * gx; F[3 * i + 1] -= q[i] * gy; F[3 * i + 2] -= q[i] * gz;
  }
}

/* ------------------------------------------------------------------ grid <-> grid (O6, O8, O10) */

/* one-axis restriction (Eq. 19 line 1): out[m] = sum_{n=-hp..hp} J_n in[2m+n] */
static double *restrict_axis(const msmo_ctx *c, const double *in, const int din[3], int ax,
                             int per, int lo_in, int lo_out, int m_out, int dout[3]) {
  int hp = c->hp;
  dout[0] = din[0]; dout[1] = din[1]; dout[2] = din[2]; dout[ax] = m_out;
  double *out = (double *)calloc((size_t)dout[0] * dout[1] * dout[2], sizeof(double));
  if (per && din[ax] == 1) { memcpy(out, in, (size_t)din[0] * din[1] * din[2] * sizeof(double)); return out; }
  for (int z = 0; z < dout[2]; ++z) for (int y = 0; y < dout[1]; ++y) for (int x = 0; x < dout[0]; ++x) {
    int o[3] = {x, y, z};
    double acc = 0.0;
    for (int n = -hp; n <= hp; ++n) {
      int i[3] = {x, y, z};
      if (per) i[ax] = imod(2 * o[ax] + n, din[ax]);
      else {
        int g = 2 * (o[ax] + lo_out) + n - lo_in;     /* array position of node 2m+n */
        if (g < 0 || g >= din[ax]) continue;
        i[ax] = g;
      }
      acc += c->J[n + hp] * in[((size_t)i[2] * din[1] + i[1]) * din[0] + i[0]];
    }
    out[((size_t)z * dout[1] + y) * dout[0] + x] = acc;
  }
  return out;
}

/* one-axis prolongation (Eq. 19 line 2): out[2m+n] += J_n in[m]  (exact transpose) */
static double *prolong_axis(const msmo_ctx *c, const double *in, const int din[3], int ax,
                            int per, int lo_in, int lo_out, int m_out, int dout[3]) {
  int hp = c->hp;
  dout[0] = din[0]; dout[1] = din[1]; dout[2] = din[2]; dout[ax] = m_out;
  double *out = (double *)calloc((size_t)dout[0] * dout[1] * dout[2], sizeof(double));
  if (per && m_out == 1) { memcpy(out, in, (size_t)din[0] * din[1] * din[2] * sizeof(double)); return out; }
  for (int z = 0; z < din[2]; ++z) for (int y = 0; y < din[1]; ++y) for (int x = 0; x < din[0]; ++x) {
    int i[3] = {x, y, z};
    double v = in[((size_t)z * din[1] + y) * din[0] + x];
    for (int n = -hp; n <= hp; ++n) {
      int o[3] = {x, y, z};
      if (per) o[ax] = imod(2 * i[ax] + n, m_out);
      else {
        int g = 2 * (i[ax] + lo_in) + n - lo_out;
        if (g < 0 || g >= m_out) continue;
        o[ax] = g;
      }
      out[((size_t)o[2] * dout[1] + o[1]) * dout[0] + o[0]] += c->J[n + hp] * v;
    }
  }
  return out;
}

/* Q^{l+1} = I Q^l, separable, x then y then z */
void msmo_restrict(msmo_ctx *c, int l) {
  int d0[3] = {c->M[l][0], c->M[l][1], c->M[l][2]}, d1[3], d2[3], d3[3];
  double *t1 = restrict_axis(c, c->Q[l], d0, 0, c->prm.periodic[0], c->lo[l][0], c->lo[l + 1][0], c->M[l + 1][0], d1);
  double *t2 = restrict_axis(c, t1, d1, 1, c->prm.periodic[1], c->lo[l][1], c->lo[l + 1][1], c->M[l + 1][1], d2);
  double *t3 = restrict_axis(c, t2, d2, 2, c->prm.periodic[2], c->lo[l][2], c->lo[l + 1][2], c->M[l + 1][2], d3);
  memcpy(c->Q[l + 1], t3, (size_t)d3[0] * d3[1] * d3[2] * sizeof(double));
  free(t1); free(t2); free(t3);
}

/* E^l += I^T E^{l+1} */
void msmo_prolong_add(msmo_ctx *c, int l) {
  int d0[3] = {c->M[l + 1][0], c->M[l + 1][1], c->M[l + 1][2]}, d1[3], d2[3], d3[3];
  double *t1 = prolong_axis(c, c->E[l + 1], d0, 2, c->prm.periodic[2], c->lo[l + 1][2], c->lo[l][2], c->M[l][2], d1);
  double *t2 = prolong_axis(c, t1, d1, 1, c->prm.periodic[1], c->lo[l + 1][1], c->lo[l][1], c->M[l][1], d2);
  double *t3 = prolong_axis(c, t2, d2, 0, c->prm.periodic[0], c->lo[l + 1][0], c->lo[l][0], c->M[l][0], d3);
  size_t g = (size_t)d3[0] * d3[1] * d3[2];
  for (size_t i = 0; i < g; ++i) c->E[l][i] += t3[i];
  free(t1); free(t2); free(t3);
}

/* (K q)_m = sum_d K_d q_{m-d} (Eq. 11). Periodic axes: index (m-d) mod M, as many wraps as
 * needed (the sum over periodic images inside the cutoff); open axes: q is zero outside the grid.
 * Writes out[m] for every grid point (or only accumulates the contraction if out == NULL);
 * returns sum_m q_m (K q)_m. */
static double convolve(const msmo_ctx *c, int l, const double *K, const double *q, double *out) {
  const int *M = c->M[l], *Kr = c->Kr[l];
  int S[3] = {2 * Kr[0] + 1, 2 * Kr[1] + 1, 2 * Kr[2] + 1};
  /* index tables: src[ax][m*S + (d+Kr)] = array position of node m-d, or -1 */
  int *tab[3];
  for (int ax = 0; ax < 3; ++ax) {
    tab[ax] = (int *)malloc((size_t)M[ax] * S[ax] * sizeof(int));
    for (int m = 0; m < M[ax]; ++m) for (int d = -Kr[ax]; d <= Kr[ax]; ++d) {
      int g = m - d;
      if (c->prm.periodic[ax]) g = imod(g, M[ax]);
      else if (g < 0 || g >= M[ax]) g = -1;
      tab[ax][m * S[ax] + d + Kr[ax]] = g;
    }
  }
  double total = 0.0;
#pragma omp parallel for collapse(2) schedule(static) reduction(+ : total)
  for (int mz = 0; mz < M[2]; ++mz) for (int my = 0; my < M[1]; ++my) {
    for (int mx = 0; mx < M[0]; ++mx) {
      double acc = 0.0;
      for (int dz = 0; dz < S[2]; ++dz) {
        int gz = tab[2][mz * S[2] + dz]; if (gz < 0) continue;
        for (int dy = 0; dy < S[1]; ++dy) {
          int gy = tab[1][my * S[1] + dy]; if (gy < 0) continue;
          const double *Krow = K + ((size_t)dz * S[1] + dy) * S[0];
          const double *qrow = q + ((size_t)gz * M[1] + gy) * M[0];
          const int *tx = tab[0] + mx * S[0];
          for (int dx = 0; dx < S[0]; ++dx) {
            int gx = tx[dx];
            if (gx >= 0) acc += Krow[dx] * qrow[gx];
          }
        }
      }
      size_t mi = ((size_t)mz * M[1] + my) * M[0] + mx;
      if (out) out[mi] = acc;
      total += q[mi] * acc;
    }
  }
  for (int ax = 0; ax < 3; ++ax) free(tab[ax]);
  return total;
}

/* test tap: out = K^l * q for an arbitrary grid function q on the level-l grid */
void msmo_apply_stencil(msmo_ctx *c, int l, int kind, const double *q, double *out) {
  if (kind > 0 && !c->have_D) setup_stencils(c, 1);
  convolve(c, l, kind == 0 ? c->K[l] : c->D[l][kind - 1], q, out);
}

/* ------------------------------------------------------------------ short range (O3) */

static void min_image(const msmo_ctx *c, double d[3]) {
  for (int ax = 0; ax < 3; ++ax)
    if (c->prm.periodic[ax]) d[ax] -= c->prm.box[ax] * floor(d[ax] / c->prm.box[ax] + 0.5);
}

static void pair_term(const msmo_ctx *c, const double *pos, const double *q, int i, int j,
                      double *Vi, double Fi[3], double W[6]) {
  double d[3] = {pos[3 * i] - pos[3 * j], pos[3 * i + 1] - pos[3 * j + 1], pos[3 * i + 2] - pos[3 * j + 2]};
  min_image(c, d);
  double r = sqrt(d[0] * d[0] + d[1] * d[1] + d[2] * d[2]);
  if (!(r < c->prm.a)) return;
  double k0 = msmo_kernel(c->prm.p, c->prm.a, c->L, 0, r);
  double dk = msmo_dkernel(c->prm.p, c->prm.a, c->L, 0, r);
  *Vi += q[j] * k0;
  double f = -q[i] * q[j] * dk / r;
  Fi[0] += f * d[0]; Fi[1] += f * d[1]; Fi[2] += f * d[2];
  if (W) {    /* half of the unordered-pair term, because every pair is visited from both ends */
    W[0] += 0.5 * f * d[0] * d[0]; W[1] += 0.5 * f * d[1] * d[1]; W[2] += 0.5 * f * d[2] * d[2];
    W[3] += 0.5 * f * d[0] * d[1]; W[4] += 0.5 * f * d[0] * d[2]; W[5] += 0.5 * f * d[1] * d[2];
  }
}

/* brute force over all j != i (minimum image on periodic axes) for the listed particles.
 * sel == NULL: all particles. Outputs are indexed like sel (or like the particles). */
void msmo_short_range_brute(const msmo_ctx *c, int n, const double *pos, const double *q,
                            int nsel, const int *sel, double *F, double *V, double *W) {
  double w0 = 0, w1 = 0, w2 = 0, w3 = 0, w4 = 0, w5 = 0;
  int cnt = sel ? nsel : n;
#pragma omp parallel for schedule(dynamic, 16) reduction(+ : w0, w1, w2, w3, w4, w5)
  for (int s = 0; s < cnt; ++s) {
    int i = sel ? sel[s] : s;
    double Vi = 0, Fi[3] = {0, 0, 0}, Wi[6] = {0, 0, 0, 0, 0, 0};
    for (int j = 0; j < n; ++j) if (j != i) pair_term(c, pos, q, i, j, &Vi, Fi, Wi);
    V[s] += Vi; F[3 * s] += Fi[0]; F[3 * s + 1] += Fi[1]; F[3 * s + 2] += Fi[2];
    w0 += Wi[0]; w1 += Wi[1]; w2 += Wi[2]; w3 += Wi[3]; w4 += Wi[4]; w5 += Wi[5];
  }
  if (W) { W[0] += w0; W[1] += w1; W[2] += w2; W[3] += w3; W[4] += w4; W[5] += w5; }
}

/* the same sum through a simple cell list (cell edge >= a, 3x3x3 neighbourhood) */
void msmo_short_range_cells(const msmo_ctx *c, int n, const double *pos, const double *q,
                            double *F, double *V, double *W) {
  int nc[3];
  double ce[3];
  for (int ax = 0; ax < 3; ++ax) {
    nc[ax] = (int)floor(c->prm.box[ax] / c->prm.a); if (nc[ax] < 1) nc[ax] = 1;
    ce[ax] = c->prm.box[ax] / nc[ax];
  }
  int ncell = nc[0] * nc[1] * nc[2];
  int *head = (int *)malloc((size_t)(ncell + 1) * sizeof(int)), *cell = (int *)malloc((size_t)n * sizeof(int));
  int *order = (int *)malloc((size_t)n * sizeof(int));
  memset(head, 0, (size_t)(ncell + 1) * sizeof(int));
  for (int i = 0; i < n; ++i) {
    int ci[3];
    for (int ax = 0; ax < 3; ++ax) {
      double x = pos[3 * i + ax];
      if (c->prm.periodic[ax]) x = wrap_coord(x, c->prm.box[ax]);
      int k = (int)floor(x / ce[ax]);
      if (k < 0) k = 0;
      if (k >= nc[ax]) k = nc[ax] - 1;
      ci[ax] = k;
    }
    cell[i] = (ci[2] * nc[1] + ci[1]) * nc[0] + ci[0];
    head[cell[i] + 1]++;
  }
  for (int k = 0; k < ncell; ++k) head[k + 1] += head[k];
  int *fill = (int *)calloc((size_t)ncell, sizeof(int));
  for (int i = 0; i < n; ++i) order[head[cell[i]] + fill[cell[i]]++] = i;
  free(fill);
  double w0 = 0, w1 = 0, w2 = 0, w3 = 0, w4 = 0, w5 = 0;
#pragma omp parallel for schedule(dynamic, 64) reduction(+ : w0, w1, w2, w3, w4, w5)
  for (int i = 0; i < n; ++i) {
    int ci = cell[i], cx = ci % nc[0], cy = (ci / nc[0]) % nc[1], cz = ci / (nc[0] * nc[1]);
    double Vi = 0, Fi[3] = {0, 0, 0}, Wi[6] = {0, 0, 0, 0, 0, 0};
    int seen[27], nseen = 0;
    for (int dz = -1; dz <= 1; ++dz) for (int dy = -1; dy <= 1; ++dy) for (int dx = -1; dx <= 1; ++dx) {
      int o[3] = {cx + dx, cy + dy, cz + dz}, ok = 1;
      for (int ax = 0; ax < 3; ++ax) {
        if (c->prm.periodic[ax]) o[ax] = imod(o[ax], nc[ax]);
        else if (o[ax] < 0 || o[ax] >= nc[ax]) ok = 0;
      }
      if (!ok) continue;
      int cj = (o[2] * nc[1] + o[1]) * nc[0] + o[0], dup = 0;
      for (int k = 0; k < nseen; ++k) if (seen[k] == cj) dup = 1;   /* few cells on a periodic axis */
      if (dup) continue;
      seen[nseen++] = cj;
      for (int k = head[cj]; k < head[cj + 1]; ++k) {
        int j = order[k];
        if (j != i) pair_term(c, pos, q, i, j, &Vi, Fi, Wi);
      }
    }
    V[i] += Vi; F[3 * i] += Fi[0]; F[3 * i + 1] += Fi[1]; F[3 * i + 2] += Fi[2];
    w0 += Wi[0]; w1 += Wi[1]; w2 += Wi[2]; w3 += Wi[3]; w4 += Wi[4]; w5 += Wi[5];
  }
  if (W) { W[0] += w0; W[1] += w1; W[2] += w2; W[3] += w3; W[4] += w4; W[5] += w5; }
  free(head); free(cell); free(order);
}

/* ------------------------------------------------------------------ grid pass and evaluate */

/* e^{1+} from q~^1 (Eq. 13): restrict up, convolve every level, prolongate down.
 * Returns in Wlr (if non-NULL) the grid part of the virial, -1/2 sum_l Q^l . (D^l * Q^l). */
void msmo_grid_pass(msmo_ctx *c, double *Wlr) {
  if (Wlr && !c->have_D) setup_stencils(c, 1);
  for (int l = 1; l < c->L; ++l) msmo_restrict(c, l);
  for (int l = 1; l <= c->L; ++l) {
    size_t g = (size_t)c->M[l][0] * c->M[l][1] * c->M[l][2];
    if (!c->K[l]) { memset(c->E[l], 0, g * sizeof(double)); continue; }     /* T2 top: zero */
    convolve(c, l, c->K[l], c->Q[l], c->E[l]);
    if (Wlr) for (int k = 0; k < 6; ++k) Wlr[k] -= 0.5 * convolve(c, l, c->D[l][k], c->Q[l], NULL);
  }
  for (int l = c->L - 1; l >= 1; --l) msmo_prolong_add(c, l);
}

/* One MSM evaluation. forces (n x 3), potentials (n) = dU/dq_i, energy, virial[6] = xx yy zz xy
 * xz yz of -dU/d eps. Any output may be NULL. Returns 0, or 5 if an open coordinate is outside
 * [0, box]. */
int msmo_evaluate(msmo_ctx *c, int n, const double *pos, const double *q, double *forces,
                  double *potentials, double *energy, double *virial) {
  for (int i = 0; i < n; ++i) for (int ax = 0; ax < 3; ++ax) {
    double x = pos[3 * i + ax];
    if (!isfinite(x) || (!c->prm.periodic[ax] && (x < 0.0 || x > c->prm.box[ax]))) return 5;
  }
  double *F = (double *)calloc((size_t)3 * n + 1, sizeof(double)), *V = (double *)calloc((size_t)n + 1, sizeof(double));
  double W[6] = {0, 0, 0, 0, 0, 0};
  /* U^0 (Eq. 5): pair sum of k_0 ... */
  if (n <= 4096) msmo_short_range_brute(c, n, pos, q, 0, NULL, F, V, virial ? W : NULL);
  else msmo_short_range_cells(c, n, pos, q, F, V, virial ? W : NULL);
  /* ... minus the self term: sum_{l>=1} k_l(0) = gamma(0)/a by telescoping (reading K2) */
  double kself = 0.0;
  for (int l = 1; l <= c->L; ++l) kself += msmo_kernel(c->prm.p, c->prm.a, c->L, l, 0.0);
  for (int i = 0; i < n; ++i) V[i] -= q[i] * kself;
  /* U^{1+} */
  msmo_anterpolate(c, n, pos, q);
  msmo_grid_pass(c, virial ? W : NULL);
  msmo_interpolate(c, n, pos, q, F, V);
  double U = 0.0;
  for (int i = 0; i < n; ++i) U += 0.5 * q[i] * V[i];
  if (forces) memcpy(forces, F, (size_t)3 * n * sizeof(double));
  if (potentials) memcpy(potentials, V, (size_t)n * sizeof(double));
  if (energy) *energy = U;
  if (virial) memcpy(virial, W, sizeof(W));
  free(F); free(V);
  return 0;
}

/* ------------------------------------------------------------------ exact references (pins) */

/* Eq. 1 with k = 1/r by direct summation: open axes as they are, periodic axes summed over the
 * image cells |n_ax| <= nimg (the i == j term is skipped only in the home cell). nimg = 0 and no
 * periodic axis = the plain O(N^2) sum. Also forces and potentials if non-NULL. */
double msmo_direct_sum(int n, const double *pos, const double *q, const double *box, const int *periodic,
                       int nimg, double *F, double *V) {
  int r0 = periodic[0] ? nimg : 0, r1 = periodic[1] ? nimg : 0, r2 = periodic[2] ? nimg : 0;
  double U = 0.0;
#pragma omp parallel for schedule(dynamic, 8) reduction(+ : U)
  for (int i = 0; i < n; ++i) {
    double Vi = 0, Fi[3] = {0, 0, 0};
    for (int j = 0; j < n; ++j)
      for (int a = -r0; a <= r0; ++a) for (int b = -r1; b <= r1; ++b) for (int cc = -r2; cc <= r2; ++cc) {
        if (i == j && a == 0 && b == 0 && cc == 0) continue;
        double d[3] = {pos[3 * i] - pos[3 * j] - a * box[0], pos[3 * i + 1] - pos[3 * j + 1] - b * box[1],
                       pos[3 * i + 2] - pos[3 * j + 2] - cc * box[2]};
        double r2v = d[0] * d[0] + d[1] * d[1] + d[2] * d[2], r = sqrt(r2v);
        Vi += q[j] / r;
        double f = q[i] * q[j] / (r2v * r);
        Fi[0] += f * d[0]; Fi[1] += f * d[1]; Fi[2] += f * d[2];
      }
    if (V) V[i] = Vi;
    if (F) { F[3 * i] = Fi[0]; F[3 * i + 1] = Fi[1]; F[3 * i + 2] = Fi[2]; }
    U += 0.5 * q[i] * Vi;
  }
  return U;
}

/* test tap: overwrite Q^l (kind 0) or E^l (kind 1) */
void msmo_set_grid(msmo_ctx *c, int l, int kind, const double *in) {
  size_t g = (size_t)c->M[l][0] * c->M[l][1] * c->M[l][2];
  memcpy(kind == 0 ? c->Q[l] : c->E[l], in, g * sizeof(double));
}
