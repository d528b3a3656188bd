"""Pins for the oracle's building blocks (gamma, splitting, B-splines, J, omega').

Each test checks the oracle against something the paper or mathematics fixes -- a closed form,
an identity, or a library routine -- never against a retyped copy of the oracle's own formula.
"""
from fractions import Fraction

import numpy as np
import pytest

import oracle


# ---------------------------------------------------------------- gamma / splitting

@pytest.mark.parametrize("p", [4, 6, 8])
def test_gamma_zero_closed_form(p, golden):
    num, den = golden["gamma_at_zero"][str(p)]
    assert oracle.gamma(p, 0.0) == pytest.approx(num / den, rel=1e-15)


def test_gamma_p4_expanded_polynomial():
    # Taylor polynomial of s^(-1/2) about s=1, degree 3, s=rho^2, expanded by hand:
    # 35/16 - 35 rho^2/16 + 21 rho^4/16 - 5 rho^6/16
    for rho in np.linspace(0, 1, 23):
        ref = 35 / 16 - 35 * rho**2 / 16 + 21 * rho**4 / 16 - 5 * rho**6 / 16
        assert oracle.gamma(4, rho) == pytest.approx(ref, rel=1e-14)


@pytest.mark.parametrize("p", [4, 6, 8])
def test_gamma_is_taylor_of_inverse_sqrt(p):
    # the polynomial must agree with s^(-1/2) to O((s-1)^p) near s=1
    for eps in (0.2, 0.1):
        rho = np.sqrt(1 - eps)
        err = abs(oracle.gamma(p, rho) - 1 / rho)
        assert err < 2.0 * eps**p
        assert err > 0.01 * eps**p      # and not to higher order (degree is exactly p-1)


@pytest.mark.parametrize("p", [4, 6])
def test_gamma_smooth_at_one_and_derivative(p):
    assert oracle.gamma(p, 1.0) == pytest.approx(1.0, abs=1e-15)
    assert oracle.dgamma(p, 1.0 - 1e-12) == pytest.approx(-1.0, abs=1e-9)
    assert oracle.dgamma(p, 1.0 + 1e-12) == pytest.approx(-1.0, abs=1e-9)
    for rho in (0.1, 0.5, 0.93, 1.7):
        d = 1e-6
        fd = (oracle.gamma(p, rho + d) - oracle.gamma(p, rho - d)) / (2 * d)
        assert oracle.dgamma(p, rho) == pytest.approx(fd, rel=1e-8)


@pytest.mark.parametrize("p,L", [(4, 1), (4, 3), (6, 5)])
def test_splitting_telescopes_to_coulomb(p, L):
    # P:48 Eq. 2 and P:76: sum_l k_l(r) = 1/r ("nothing more than rewriting")
    rng = np.random.default_rng(0)
    a = 3.7
    for r in rng.uniform(0.05, 40 * a, 200):
        s = sum(oracle.kernel(p, a, L, l, r) for l in range(L + 1))
        assert s == pytest.approx(1 / r, rel=2e-14)


def test_kernels_have_finite_range_and_are_continuous():
    p, a, L = 4, 2.0, 4
    assert oracle.kernel(p, a, L, 0, a * (1 - 1e-13)) == pytest.approx(0.0, abs=1e-12)
    assert oracle.kernel(p, a, L, 0, a) == 0.0
    for l in range(1, L):                                  # P:52 Eq. 3: r_cut^(l) = 2^l a
        A = a * 2**l
        assert oracle.kernel(p, a, L, l, A * 1.0000001) == 0.0
        assert abs(oracle.kernel(p, a, L, l, A * (1 - 1e-9))) < 1e-12
        assert abs(oracle.dkernel(p, a, L, l, A * (1 - 1e-9))) < 1e-10
    assert oracle.kernel(p, a, L, L, 1e6) == pytest.approx(1e-6, rel=1e-14)   # k_L keeps the tail
    for l in range(0, L + 1):
        for r in (0.3, 1.9, 5.0, 17.0):
            d = 1e-6 * r
            fd = (oracle.kernel(p, a, L, l, r + d) - oracle.kernel(p, a, L, l, r - d)) / (2 * d)
            assert oracle.dkernel(p, a, L, l, r) == pytest.approx(fd, rel=1e-7, abs=1e-12)


def test_self_term_telescopes():
    # sum_{l>=1} k_l(0) = gamma(0)/a (reading K2)
    p, a = 6, 4.0
    for L in (1, 2, 5):
        s = sum(oracle.kernel(p, a, L, l, 0.0) for l in range(1, L + 1))
        assert s == pytest.approx(oracle.gamma(p, 0.0) / a, rel=1e-14)


def test_intermediate_kernels_same_form():
    # k_l(r) = 2^-(l-1) k_1(r / 2^(l-1)) for 1 <= l <= L-1
    p, a, L = 4, 3.0, 5
    for l in (2, 3, 4):
        for r in (0.0, 1.0, 7.0, 20.0):
            assert oracle.kernel(p, a, L, l, r) == pytest.approx(
                oracle.kernel(p, a, L, 1, r / 2**(l - 1)) / 2**(l - 1), rel=1e-14, abs=1e-18)


# ---------------------------------------------------------------- B-splines

@pytest.mark.parametrize("p", [2, 4, 6, 8])
def test_bspline_partition_of_unity_and_derivative(p):
    for u in np.linspace(-0.5, 0.5, 17):
        n = np.arange(-p, p + 1)
        assert sum(oracle.bspline(p, u - k) for k in n) == pytest.approx(1.0, abs=1e-14)
        assert sum(oracle.dbspline(p, u - k) for k in n) == pytest.approx(0.0, abs=1e-13)
        # first moment: sum_n n Phi(u - n) = u (linear reproduction)
        assert sum(k * oracle.bspline(p, u - k) for k in n) == pytest.approx(u, abs=1e-13)


@pytest.mark.parametrize("p", [4, 6])
def test_bspline_integer_values(p, golden):
    vals = [Fraction(*v) for v in golden["bspline_at_integers"][str(p)]]
    hp = p // 2
    for n, v in zip(range(-hp + 1, hp), vals):
        assert oracle.bspline(p, n) == pytest.approx(float(v), rel=1e-14)
    assert oracle.bspline(p, hp) == 0.0 and oracle.bspline(p, -hp) == 0.0


def test_bspline_p4_closed_form():
    # cubic B-spline pieces for t in [0,1) at nodes i0-1, i0, i0+1, i0+2
    for t in np.linspace(0, 0.999, 31):
        ref = [(1 - t)**3 / 6, (3 * t**3 - 6 * t**2 + 4) / 6, (-3 * t**3 + 3 * t**2 + 3 * t + 1) / 6, t**3 / 6]
        got = [oracle.bspline(4, t - j) for j in (-1, 0, 1, 2)]
        assert got == pytest.approx(ref, abs=1e-15)


@pytest.mark.parametrize("p", [4, 6, 8])
def test_bspline_matches_scipy(p):
    from scipy.interpolate import BSpline
    b = BSpline.basis_element(np.arange(p + 1) - p / 2, extrapolate=False)
    for u in np.linspace(-p / 2 + 1e-9, p / 2 - 1e-9, 41):
        assert oracle.bspline(p, u) == pytest.approx(float(b(u)), abs=1e-14)
        assert oracle.dbspline(p, u) == pytest.approx(float(b.derivative()(u)), abs=1e-12)


@pytest.mark.parametrize("p", [4, 6, 8])
def test_two_scale_relation(p, golden):
    J = oracle.two_scale(p)
    hp = p // 2
    if str(p) in golden["two_scale"]:
        assert J * golden["two_scale"][f"{p}_den"] == pytest.approx(golden["two_scale"][str(p)], abs=1e-14)
    # Phi(u/2) = sum_n J_n Phi(u - n), pointwise
    for u in np.linspace(-p, p, 57):
        rhs = sum(J[n + hp] * oracle.bspline(p, u - n) for n in range(-hp, hp + 1))
        assert oracle.bspline(p, u / 2) == pytest.approx(rhs, abs=1e-14)
    assert J[0::2].sum() == pytest.approx(1.0, abs=1e-15)      # charge conservation
    assert J[1::2].sum() == pytest.approx(1.0, abs=1e-15)


# ---------------------------------------------------------------- omega' (reading Q)

@pytest.mark.parametrize("p,mu", [(4, 0), (4, 4), (6, 0), (6, 4), (8, 2)])
def test_omega_sum_and_symmetry(p, mu):
    w = oracle.omega(p, mu)
    assert len(w) == 2 * (p // 2 - 1 + mu) + 1
    assert w.sum() == pytest.approx(1.0, abs=1e-12)
    assert w == pytest.approx(w[::-1], abs=1e-15)


@pytest.mark.parametrize("p,mu", [(4, 0), (4, 4), (6, 0), (6, 3)])
def test_quasi_interpolant_reproduces_polynomials(p, mu):
    # for f(x - x') a polynomial of degree < p:
    #   sum_mn Phi(x - m) (omega' * f)_{m-n} Phi(x' - n) = f(x - x')   exactly
    w = oracle.omega(p, mu)
    hw = len(w) // 2
    rng = np.random.default_rng(1)
    for deg in range(p):
        f = lambda u: (0.3 + u)**deg
        for _ in range(3):
            x, xp = rng.uniform(-1, 1, 2)
            total = 0.0
            for m in range(-p, p + 1):
                pm = oracle.bspline(p, x - m)
                if pm == 0:
                    continue
                for n in range(-p, p + 1):
                    pn = oracle.bspline(p, xp - n)
                    if pn == 0:
                        continue
                    c = sum(w[k + hw] * f(m - n - k) for k in range(-hw, hw + 1))
                    total += pm * c * pn
            assert total == pytest.approx(f(x - xp), abs=1e-9 * max(1.0, abs(f(x - xp))))
    # and NOT degree p (the scheme has order exactly p)
    f = lambda u: u**p
    x, xp = 0.4, -0.3
    total = sum(oracle.bspline(p, x - m) * sum(w[k + hw] * f(m - n - k) for k in range(-hw, hw + 1)) *
                oracle.bspline(p, xp - n) for m in range(-p, p + 1) for n in range(-p, p + 1))
    assert abs(total - f(x - xp)) > 1e-4


@pytest.mark.parametrize("p", [4, 6])
def test_omega_converges_to_exact_interpolation(p):
    # mu -> infinity: omega' * Phi(n) * Phi(n) -> delta (coefficients of exact interpolation, omega*omega)
    hp = p // 2
    phi = np.array([oracle.bspline(p, n) for n in range(-hp + 1, hp)])
    errs = []
    for mu in (0, 4, 12, 40):
        w = oracle.omega(p, mu)
        d = np.convolve(np.convolve(w, phi), phi)
        d[len(d) // 2] -= 1.0
        errs.append(np.abs(d).max())
    assert errs[0] > errs[1] > errs[2] > errs[3]
    assert errs[3] < 1e-3      # geometric convergence: ratio 2/3 for p=4, 0.84 for p=6


def test_omega_known_shortest_sequences():
    # mu = 0, p = 4: (1 + t/6)^-2 = 1 - t/3 + O(t^2) with t = delta^2 = [1, -2, 1]
    #   -> [-1/3, 1 + 2/3, -1/3]
    assert oracle.omega(4, 0) == pytest.approx([-1 / 3, 5 / 3, -1 / 3], abs=1e-15)


@pytest.mark.parametrize("key,p,mu", [("p4_mu0", 4, 0), ("p6_mu0", 6, 0), ("p4_mu4", 4, 4), ("p6_mu4", 6, 4)])
def test_omega_exact_rationals(golden, key, p, mu):
    """Reading Q with mu > 0: polynomial reproduction only constrains the first p/2 series terms, so
    the extra mu terms are pinned by the exact rationals of SURVEY.md Appendix A (computed
    symbolically, independent of the oracle)."""
    from fractions import Fraction
    ref = [float(Fraction(a, b)) for a, b in golden["omega_prime"][key]]
    w = oracle.omega(p, mu)
    hw = len(w) // 2
    assert hw == p // 2 - 1 + mu == len(ref) - 1
    assert w[hw:] == pytest.approx(ref, rel=1e-13, abs=1e-16)
    assert w[:hw + 1][::-1] == pytest.approx(ref, rel=1e-13, abs=1e-16)


@pytest.mark.parametrize("p", [4, 6])
def test_omega_is_the_truncated_series_of_the_inverse_squared_symbol(golden, p):
    """The stored series coefficients c_k satisfy (sum_k c_k t^k) * Phi_hat(t)^2 = 1 + O(t^(w+1)) in exact
    rational arithmetic, with Phi_hat the symbol of the sampled spline in t = delta^2 built here from
    the textbook integer values of the B-spline; and omega'(mu) - omega'(mu-1) is exactly
    c_w (z - 2 + 1/z)^w, i.e. the alternating binomial row scaled by c_w."""
    from fractions import Fraction
    from math import comb
    cs = [Fraction(a, b) for a, b in golden["omega_prime"][f"series_p{p}"]]
    phi = [Fraction(a, b) for a, b in golden["bspline_at_integers"][str(p)]]      # Phi(-hp+1 .. hp-1)
    hp = p // 2
    # symbol in powers of t: Phi_hat(z) = sum_n Phi(n) z^n with z + 1/z = t + 2; Chebyshev-like recursion
    # z^n + z^-n = T_n(t): T_0 = 2, T_1 = t + 2, T_n = (t + 2) T_{n-1} - T_{n-2}
    def polymul(a, b):
        out = [Fraction(0)] * (len(a) + len(b) - 1)
        for i, x in enumerate(a):
            for j, y in enumerate(b):
                out[i + j] += x * y
        return out
    T = [[Fraction(2)], [Fraction(2), Fraction(1)]]
    for n in range(2, hp):
        nxt = polymul([Fraction(2), Fraction(1)], T[-1])
        prev = T[-2] + [Fraction(0)] * (len(nxt) - len(T[-2]))
        T.append([x - y for x, y in zip(nxt, prev)])
    sym = [Fraction(0)] * hp
    sym[0] += phi[hp - 1]
    for n in range(1, hp):
        for k, c in enumerate(T[n]):
            sym[k] += phi[hp - 1 + n] * c
    sq = polymul(sym, sym)
    prod = polymul(cs, sq)
    assert prod[0] == 1 and all(v == 0 for v in prod[1:len(cs)])
    for mu in range(1, len(cs) - hp + 1):
        w = hp - 1 + mu
        full = oracle.omega(p, mu).copy()
        full[1:-1] -= oracle.omega(p, mu - 1)
        row = np.array([float(cs[w]) * (-1) ** (w - abs(n)) * comb(2 * w, w + n) for n in range(-w, w + 1)])
        assert full == pytest.approx(row, rel=1e-12, abs=1e-15)
