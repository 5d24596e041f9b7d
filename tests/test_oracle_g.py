"""Pin P4: the oracle's triangle function g(a,b,c) and its derivatives against the paper's closed
forms evaluated in 50-digit arithmetic (mpmath), the confluent limits, and the defining integral.

  eq. 9   PAPER.md:162   f_T = sum_p e^{-i v_p.xi} / ((e_{p-}.xi)(e_{p+}.xi))      (reading R1: z_p = v_p)
  eq. 14  PAPER.md:194   g(s,t,u) with arguments v_p.xi and exponents e^{-i.}      (reading R3)
  eq. 15  PAPER.md:203   g(t,t,u)
  eq. 16  PAPER.md:208   g(u,u,u) = e^{-iu}/2
  eq. 11  PAPER.md:171   d f_T / d v_p with e_q.xi in the denominators             (reading R2)
"""
import itertools

import mpmath as mp
import numpy as np
import pytest

import oracle

mp.mp.dps = 60


def eq9_paper(a):
    """eq. 9 in the paper's own index notation: e_p = v_{p-} - v_{p+}."""
    a = [mp.mpf(x) for x in a]
    tot = mp.mpc(0)
    for p in range(3):
        pm, pp = (p - 1) % 3, (p + 1) % 3
        e_pm = a[(pm - 1) % 3] - a[(pm + 1) % 3]   # e_{p-} . xi
        e_pp = a[(pp - 1) % 3] - a[(pp + 1) % 3]   # e_{p+} . xi
        tot += mp.e ** (-1j * a[p]) / (e_pm * e_pp)
    return tot


def eq14(s, t, u):
    s, t, u = mp.mpf(s), mp.mpf(t), mp.mpf(u)
    E = lambda x: mp.e ** (-1j * x)
    return -E(s) / ((s - t) * (s - u)) - E(t) / ((t - u) * (t - s)) - E(u) / ((u - s) * (u - t))


def eq15(t, u):
    t, u = mp.mpf(t), mp.mpf(u)
    E = lambda x: mp.e ** (-1j * x)
    return 1j * E(t) / (t - u) + E(t) / (t - u) ** 2 - E(u) / (t - u) ** 2


def eq16(u):
    return mp.e ** (-1j * mp.mpf(u)) / 2


def eq11_R2(a, p):
    """eq. 11 with reading R2 (every v_q.xi in a denominator replaced by e_q.xi): d f_T / d a_p."""
    a = [mp.mpf(x) for x in a]
    pm, pp = (p - 1) % 3, (p + 1) % 3
    e = [a[(q - 1) % 3] - a[(q + 1) % 3] for q in range(3)]
    E = lambda x: mp.e ** (-1j * x)
    return (E(a[pp]) / (e[pm] ** 2 * e[p]) - E(a[pm]) / (e[p] * e[pp] ** 2)
            - 1j * E(a[p]) / (e[pm] * e[pp]) + E(a[p]) / (e[pm] ** 2 * e[pp]) - E(a[p]) / (e[pm] * e[pp] ** 2))


_GL_X, _GL_W = np.polynomial.legendre.leggauss(48)
_GL_X, _GL_W = 0.5 * (_GL_X + 1.0), 0.5 * _GL_W


def simplex_integral(a, b, c, weight=lambda t1, t2: 1.0):
    """The defining double integral over t1,t2>=0, t1+t2<=1 by a 48x48 Gauss-Legendre rule on the
    Duffy square (t1 = u, t2 = w(1-u), Jacobian 1-u); exact to rounding for |arguments| <~ 20."""
    u, w = np.meshgrid(_GL_X, _GL_X, indexing="ij")
    t1, t2 = u, w * (1.0 - u)
    f = weight(t1, t2) * np.exp(-1j * (a + t1 * (b - a) + t2 * (c - a))) * (1.0 - u)
    return complex(np.einsum("i,j,ij->", _GL_W, _GL_W, f))


def _c(z):
    return complex(z)


def test_g_matches_eq9_and_eq14_random():
    rng = np.random.default_rng(1)
    for scale in (0.7, 5.0, 60.0, 600.0):
        for _ in range(60):
            a, b, c = rng.uniform(-scale, scale, 3)
            ref9 = _c(eq9_paper((a, b, c)))
            ref14 = _c(eq14(a, b, c))
            got = oracle.g_fun(a, b, c)
            assert abs(ref9 - ref14) < 1e-30 * max(1, abs(ref9))
            assert abs(got - ref9) < 2e-14, (a, b, c, got, ref9)


def test_g_is_the_simplex_integral():
    rng = np.random.default_rng(2)
    for _ in range(8):
        a, b, c = rng.uniform(-6, 6, 3)
        assert abs(oracle.g_fun(a, b, c) - _c(simplex_integral(a, b, c))) < 1e-14
    # degenerate triples straight from the definition
    for a, b, c in [(1.3, 1.3, -2.0), (0.4, 0.4, 0.4), (0.0, 0.0, 0.0), (2.0, -1.0, 2.0)]:
        assert abs(oracle.g_fun(a, b, c) - _c(simplex_integral(a, b, c))) < 1e-14


def test_g_confluent_limits_eq15_eq16():
    rng = np.random.default_rng(3)
    for _ in range(50):
        t, u = rng.uniform(-20, 20, 2)
        ref = _c(eq15(t, u))
        for args in ((t, t, u), (u, t, t), (t, u, t)):
            assert abs(oracle.g_fun(*args) - ref) < 2e-14
        assert abs(oracle.g_fun(u, u, u) - _c(eq16(u))) < 1e-15
    assert oracle.g_fun(0, 0, 0) == pytest.approx(0.5, abs=1e-16)


@pytest.mark.parametrize("gap", [1e-1, 1e-2, 1e-4, 1e-7, 1e-10, 1e-13])
def test_g_near_degenerate_against_50_digit_eq9(gap):
    rng = np.random.default_rng(4)
    for _ in range(20):
        a = rng.uniform(-50, 50)
        far = a + rng.uniform(1, 9) * rng.choice([-1, 1])
        # two close, one far
        assert abs(oracle.g_fun(a, a + gap, far) - _c(eq14(a, a + gap, far))) < 2e-14
        # all three close
        b, c = a + gap, a - 0.37 * gap
        assert abs(oracle.g_fun(a, b, c) - _c(eq14(a, b, c))) < 2e-15
        # across the series/recursion switch of step O2 (cluster diameter 0.5)
        for d in (0.49999, 0.5, 0.50001):
            assert abs(oracle.g_fun(a, a + d, a + gap) - _c(eq14(a, a + d, a + gap))) < 2e-14


def test_g_symmetric_in_its_arguments():
    rng = np.random.default_rng(5)
    for _ in range(20):
        x = rng.uniform(-10, 10, 3)
        vals = [oracle.g_fun(*p) for p in itertools.permutations(x)]
        assert max(abs(v - vals[0]) for v in vals) < 1e-14


def test_g_grad_matches_eq11_R2_and_numerical_derivative():
    rng = np.random.default_rng(6)
    for scale in (1.0, 8.0, 100.0):
        for _ in range(25):
            x = rng.uniform(-scale, scale, 3)
            got = oracle.g_grad(*x)
            for p in range(3):
                ref = _c(eq11_R2(x, p))
                num = _c(mp.diff(lambda s: eq14(*[s if q == p else x[q] for q in range(3)]), mp.mpf(x[p])))
                assert abs(ref - num) < 1e-20 * max(1.0, abs(num))
                assert abs(got[p] - ref) < 5e-14, (x, p, got[p], ref)


def test_g_grad_degenerate_and_sum_identity():
    rng = np.random.default_rng(7)
    cases = [(0.0, 0.0, 0.0), (1.0, 1.0, 1.0), (2.5, 2.5, -1.0), (-3.0, 4.0, -3.0), (0.3, 0.3 + 1e-9, 5.0)]
    cases += [tuple(rng.uniform(-5, 5, 3)) for _ in range(20)]
    for x in cases:
        dg = oracle.g_grad(*x)
        g = oracle.g_fun(*x)
        # shifting all three arguments multiplies g by e^{-i s}:  sum_p dg/da_p = -i g      (pin P9)
        assert abs(dg.sum() + 1j * g) < 1e-14
        # derivative straight from the defining integral:  dg/da = -i int (1-t1-t2) e^{...}
        a, b, c = x
        ref = -1j * simplex_integral(a, b, c, weight=lambda t1, t2: 1.0 - t1 - t2)
        assert abs(dg[0] - ref) < 1e-14
    assert np.allclose(oracle.g_grad(0, 0, 0), -1j / 6, atol=1e-16)


def test_edge_sinc_form_equals_2A_g():
    """2D divergence theorem on the triangle: u_T = (i/|k_t|^2) sum_p (k.w_p) sinc(k.e_p/2) e^{-ik.c_p}."""
    rng = np.random.default_rng(8)
    for _ in range(30):
        v = rng.uniform(-1, 1, (3, 3))
        k = rng.uniform(-9, 9, 3)
        e = np.array([v[(p - 1) % 3] - v[(p + 1) % 3] for p in range(3)])
        m = np.cross(e[2], e[0])
        N = m / np.linalg.norm(m)
        kt2 = k @ k - (k @ N) ** 2
        tot = 0
        for p in range(3):
            w = np.cross(e[p], N)
            mid = 0.5 * (v[(p - 1) % 3] + v[(p + 1) % 3])
            tot += (k @ w) * np.sinc((k @ e[p]) / 2 / np.pi) * np.exp(-1j * (k @ mid))
        ref = 1j / kt2 * tot
        got = np.linalg.norm(m) * oracle.g_fun(k @ v[0], k @ v[1], k @ v[2])
        assert abs(got - ref) < 1e-12
