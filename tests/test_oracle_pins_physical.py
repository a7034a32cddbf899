"""Pins P15-P17 of the CPU oracle (none touches the CUDA path): the regimes round 1 left to GPU-vs-oracle
agreement alone.

  P15  the PHYSICAL region of the deformed class (A5): F changes sign on the cube, the branch of (F - i delta)^q and of
       Log F is fixed by the sign of f_im together with the direction of the deformation ("contour deformation",
       PAPER.md:422; BASELINE.json config 3 "mixed-sign coefficients plus a -i 1e-12 prescription").  Closed forms
       (tests/golden/make_closed_forms.py) for d = 1, F = a - x; a separable d = 2 variant with a non-trivial U; a
       genuinely two-dimensional F = a - x1 x2 against QUADPACK with algebraic end-point weights; and the mirror
       statement (f_im > 0, lambda < 0 gives the complex conjugate).  A wrong sign of f_im, the conjugate handed to
       Log, a wrong sign in z(x) or a dropped / transposed Jacobian entry fails one of them.
  P16  the zero-weight branch (reading Q4) and both diagnostics counters, with hand-counted non-zero values.
  P17  the Neumaier accumulator (A6) against the exactly rounded sum of the same terms, on a sum that a plain
       FP64 accumulation gets wrong.
"""
import cmath
import math
import os

import numpy as np
import pytest

from oracle import oracle as O
from paper_2305_19768_b200 import workloads as W


def _golden():
    out = {}
    path = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden", "closed_forms.txt")
    for ln in open(path):
        if ln.strip() and not ln.startswith("#"):
            k, v = ln.split()
            out[k] = float(v)
    return out


def _gc(G, name):
    return complex(G[name + "_re"], G[name + "_im"])


def _uf(dim, U, F, p, q, logc, first_order, n_orders, transform, lam, f_im, a=None):
    aa = np.zeros(8, np.int32)
    if a is not None:
        aa[:dim] = a
    return W.Sector(dim=dim, kind=W.KIND_UF, transform=transform, deformed=1, first_order=first_order,
                    n_orders=n_orders, a=aa, p=p, q=q,
                    U_coef=np.array([t[0] for t in U], float), U_exp=np.array([t[1] for t in U], np.uint8).reshape(len(U), dim),
                    F_coef=np.array([t[0] for t in F], float), F_exp=np.array([t[1] for t in F], np.uint8).reshape(len(F), dim),
                    lam=lam, f_im=f_im, logc=np.array(logc, float))


def physical_1d_sector(a, q, lam, f_im, transform=W.TRANSFORM_KOROBOV3, c0=1.0, c00=0.5, c10=7.0, c01=-2.0):
    """d = 1, U = 1, F = a - x: order 0 = c0 F^q, order 1 = F^q (c00 + c10 Log U + c01 Log F), Log U = 0."""
    return _uf(1, U=[(1.0, (0,))], F=[(a, (0,)), (-1.0, (1,))], p=0.0, q=q, logc=[c0, c00, c10, c01],
               first_order=0, n_orders=2, transform=transform, lam=lam, f_im=f_im)


def _within(res_row, exact, nsig=6.0, floor=1e-13):
    tol_re = nsig * res_row[2] + floor * abs(exact)
    tol_im = nsig * res_row[3] + floor * abs(exact)
    return abs(res_row[0] - exact.real) <= tol_re and abs(res_row[1] - exact.imag) <= tol_im


# ------------------------------------------------------------------------------- P15
@pytest.mark.parametrize("a,q", [(0.37, -0.5), (0.37, -1.3), (0.62, -0.5), (0.62, 0.75)])
@pytest.mark.parametrize("lam,transform", [(0.3, W.TRANSFORM_KOROBOV3), (1.0, W.TRANSFORM_KOROBOV3), (0.5, W.TRANSFORM_BAKER)])
def test_p15_physical_region_closed_form_1d(a, q, lam, transform):
    """int_0^1 (a - x - i0)^q dx and the same with Log(a - x - i0): F < 0 for x > a, so the result is complex and
    its imaginary part has the sign the -i delta prescription dictates (for q = -1/2: 2 sqrt(a) + 2 i sqrt(1 - a))."""
    G = _golden()
    I_pow, I_log = _gc(G, "phys1d_a%s_q%s_pow" % (a, q)), _gc(G, "phys1d_a%s_q%s_log" % (a, q))
    if q == -0.5:
        assert I_pow == pytest.approx(2 * math.sqrt(a) + 2j * math.sqrt(1 - a), rel=1e-11)   # stored at delta = 1e-12
    c0, c00, c01 = 1.0, 0.5, -2.0
    sec = O.OracleSector(physical_1d_sector(a, q, lam, -1e-12, transform, c0=c0, c00=c00, c01=c01))
    n = 100003 if transform == W.TRANSFORM_KOROBOV3 else 1000003
    shifts = np.random.default_rng(15).random((8, 1))
    _, res, diag = O.integrate(sec, n, np.array([1], np.uint64), shifts)
    assert diag[1] == 0                                   # Im F(z) = -lambda x (1 - x) - 1e-12 < 0 everywhere
    want0, want1 = c0 * I_pow, c00 * I_pow + c01 * I_log
    assert _within(res[0], want0), (res[0], want0)
    assert _within(res[1], want1), (res[1], want1)
    # the comparison is sharp: the error bars are far below the size of the imaginary part that a wrong branch flips
    assert 6.0 * max(res[0, 2], res[0, 3]) < 1e-5 * abs(want0.imag)


def test_p15_mirror_prescription_gives_the_complex_conjugate():
    """f_im = +1e-12 with the deformation turned the other way (lambda < 0) is the +i delta prescription: every
    per-shift sum is the complex conjugate of the -i delta one, bit for bit up to the last place, and the sign
    check now fails on every point (Im F > 0)."""
    a, q = 0.37, -0.5
    n, z = 10007, np.array([1], np.uint64)
    shifts = np.random.default_rng(16).random((4, 1))
    minus = O.OracleSector(physical_1d_sector(a, q, 0.5, -1e-12))
    plus = O.OracleSector(physical_1d_sector(a, q, -0.5, +1e-12))
    s_m, r_m, d_m = O.integrate(minus, n, z, shifts)
    s_p, r_p, d_p = O.integrate(plus, n, z, shifts)
    assert d_m[1] == 0 and d_p[1] == n * len(shifts) - d_p[0]
    assert np.allclose(s_p[:, :, 0], s_m[:, :, 0], rtol=1e-13, atol=0)
    assert np.allclose(s_p[:, :, 1], -s_m[:, :, 1], rtol=1e-13, atol=0)
    assert np.allclose(s_p[:, :, 2], s_m[:, :, 2], rtol=1e-13, atol=0)
    assert r_m[0, 1] > 1.0 and r_p[0, 1] < -1.0          # 2 sqrt(0.63) = 1.587 and its mirror image


def test_p15_wrong_direction_of_the_deformation_is_flagged_and_wrong():
    """lambda < 0 with the -i delta prescription pushes the contour across the cut side: Im F(z) > 0 on the
    interior points, which is what diag[1] exists to report, and the principal Log then returns the other branch."""
    a, q = 0.37, -0.5
    n, z = 10007, np.array([1], np.uint64)
    shifts = np.random.default_rng(17).random((4, 1))
    sec = O.OracleSector(physical_1d_sector(a, q, -0.5, -1e-12, W.TRANSFORM_BAKER))
    _, res, diag = O.integrate(sec, n, z, shifts)
    # Im F(z) = +0.5 x (1 - x) - 1e-12 >= 0 unless x (1 - x) < 2e-12: hand count over the baker points
    fails = 0
    for s in range(len(shifts)):
        for k in range(n):
            t = k / n + shifts[s, 0]
            t -= 1.0 if t >= 1.0 else 0.0
            x = 1.0 - abs(2.0 * t - 1.0)
            fails += 0.5 * x * (1.0 - x) >= 1e-12
    assert diag[1] == fails and fails >= n * len(shifts) - 4
    assert res[0, 1] < -1.0                               # conjugate branch: -2 sqrt(1 - a)


def test_p15_separable_2d_with_nontrivial_u():
    """d = 2: F = a - x1 (depends on x1 only), U = 1 + b x2 with power p: the integral factorises into the d = 1
    closed form times int (1 + b y)^p dy; the Jacobian matrix is diagonal with a trivial second row."""
    G = _golden()
    a, q, b, p_ = 0.37, -0.5, 0.8, -1.7
    exact = _gc(G, "phys1d_a0.37_q-0.5_pow") * G["sep_u_b0.8_p-1.7"]
    sec = O.OracleSector(_uf(2, U=[(1.0, (0, 0)), (b, (0, 1))], F=[(a, (0, 0)), (-1.0, (1, 0))], p=p_, q=q, logc=[1.0],
                             first_order=0, n_orders=1, transform=W.TRANSFORM_KOROBOV3, lam=0.7, f_im=-1e-12))
    n, z = 100003, np.array([1, 38117], np.uint64)
    shifts = np.random.default_rng(18).random((8, 2))
    _, res, diag = O.integrate(sec, n, z, shifts)
    assert diag[1] == 0
    assert _within(res[0], exact), (res[0], exact)
    assert 6.0 * max(res[0, 2], res[0, 3]) < 1e-5 * abs(exact.imag)


@pytest.mark.parametrize("q", [-0.5, 0.5])
def test_p15_two_dimensional_sign_change_against_quadpack(q):
    """d = 2, F = a - x1 x2: both derivatives and the off-diagonal Hessian entry are non-zero and F changes sign on
    the hyperbola x1 x2 = a.  With u = x1 x2 (density -log u on (0, 1]):
        I = int_0^a (a - u)^q (-log u) du + e^(-i pi q) int_a^1 (u - a)^q (-log u) du,
    both computed by QUADPACK's algebraic-weight rules (scipy.integrate.quad, weight='alg' / 'alg-loga').
    Im F(z) = -lambda x1 x2 ((1 - x1) x2 + (1 - x2) x1) < 0 inside the cube for every lambda > 0, so the contour is
    admissible and Cauchy's theorem applies."""
    from scipy import integrate as SI
    a, lam = 0.45, 0.8
    left, e1 = SI.quad(lambda u: -1.0, 0.0, a, weight="alg-loga", wvar=(0.0, q), epsabs=1e-13, epsrel=1e-13)
    right, e2 = SI.quad(lambda u: -math.log(u), a, 1.0, weight="alg", wvar=(q, 0.0), epsabs=1e-13, epsrel=1e-13)
    exact = left + cmath.exp(-1j * math.pi * q) * right
    assert e1 + e2 < 1e-11
    sec = O.OracleSector(_uf(2, U=[(1.0, (0, 0))], F=[(a, (0, 0)), (-1.0, (1, 1))], p=0.0, q=q, logc=[1.0],
                             first_order=0, n_orders=1, transform=W.TRANSFORM_KOROBOV3, lam=lam, f_im=-1e-12))
    n, z = 400009, np.array([1, 152471], np.uint64)
    shifts = np.random.default_rng(19).random((8, 2))
    _, res, diag = O.integrate(sec, n, z, shifts)
    assert diag[1] == 0
    assert _within(res[0], exact, floor=1e-10), (res[0], exact)
    assert 6.0 * max(res[0, 2], res[0, 3]) < 1e-3 * abs(exact.imag)


# ------------------------------------------------------------------------------- P16
def test_p16_zero_weight_points_contribute_zero_and_are_counted():
    """Reading Q4: a point whose Korobov weight is exactly 0 contributes 0 whatever the integrand does there and is
    counted in diag[0].  g = x^(-1/2) (U = 1, F = x, q = -1/2) is infinite at x = 0, so evaluating it there would
    give 0 * inf = NaN.  z = 4 is not a unit mod n = 12: r = 0 for k = 0, 3, 6, 9; the first shift row is 0.0
    (t = 0 at those four k), the second is not (no zero weight)."""
    n, z = 12, np.array([4], np.uint64)
    sec = O.OracleSector(W.Sector(dim=1, kind=W.KIND_UF, transform=W.TRANSFORM_KOROBOV3, deformed=0, first_order=0,
                                  n_orders=1, a=np.zeros(8, np.int32), p=0.0, q=-0.5,
                                  U_coef=np.ones(1), U_exp=np.zeros((1, 1), np.uint8),
                                  F_coef=np.ones(1), F_exp=np.ones((1, 1), np.uint8), logc=np.ones(1)))
    shifts = np.array([[0.0], [0.3125]])
    sums, diag = O.shift_sums(sec, n, z, shifts)
    assert diag[0] == 4 and diag[1] == 0
    assert np.all(np.isfinite(sums))
    for s, delta in enumerate([0.0, 0.3125]):
        want = 0.0
        for k in range(n):
            t = ((k * 4) % n) / n + delta
            t -= 1.0 if t >= 1.0 else 0.0
            w = 140.0 * t**3 * (1.0 - t) ** 3
            if w == 0.0:
                continue
            x = t**4 * (35.0 - 84.0 * t + 70.0 * t * t - 20.0 * t**3)
            want += w / math.sqrt(x)
        assert sums[s, 0, 0] == pytest.approx(want, rel=1e-13)
        assert sums[s, 0, 2] == pytest.approx(want, rel=1e-13)
    # one shift at a time: the counter is per call and adds over the shifts
    _, d0 = O.shift_sums(sec, n, z, shifts[:1])
    _, d1 = O.shift_sums(sec, n, z, shifts[1:])
    assert d0[0] == 4 and d1[0] == 0
    # a k-range that holds exactly one of the four
    _, dk = O.shift_sums(sec, n, z, shifts[:1], k0=1, k1=4)
    assert dk[0] == 1


def test_p16_zero_weight_in_one_of_two_dimensions_kills_the_point():
    """W is the product over the dimensions: t_2 = 0 alone makes W = 0 (C0's toy class, finite integrand)."""
    sec = O.OracleSector(W.Sector(dim=2, kind=W.KIND_TOY, transform=W.TRANSFORM_KOROBOV3,
                                  U_coef=np.array([0.5, -0.25, 0.75, 0.125]), U_exp=np.zeros((4, 2), np.uint8)))
    n, z = 7, np.array([3, 5], np.uint64)
    sums, diag = O.shift_sums(sec, n, z, np.array([[0.4375, 0.0]]))     # k = 0: t = (0.4375, 0)
    assert diag[0] == 1
    t, x, Wt, wg, _ = O.eval_point(sec, n, z, np.array([0.4375, 0.0]), 0)
    assert t[1] == 0.0 and Wt == 0.0 and wg[0] == 0.0


def test_p16_sign_check_counter_counts_exactly_the_points_with_im_f_nonnegative():
    """diag[1] counts Im F(z) >= 0.  (i) lambda = 0, f_im > 0: every point, n m.  (ii) lambda = 0, f_im = 0 on a
    real F: Im F = 0 counts (>=).  (iii) f_im < 0: none.  (iv) f_im = +c against a proper deformation of F = a - x:
    Im F = c - lambda x (1 - x) >= 0 exactly where x (1 - x) <= c / lambda -- counted by hand over the baker points."""
    n, z, m = 1009, np.array([1], np.uint64), 3
    shifts = np.random.default_rng(20).random((m, 1))
    count = lambda lam, f_im: O.integrate(O.OracleSector(physical_1d_sector(0.37, -0.5, lam, f_im, W.TRANSFORM_BAKER)),
                                          n, z, shifts)[2]
    assert tuple(count(0.0, +1e-12)) == (0, n * m)
    assert tuple(count(0.0, 0.0)) == (0, n * m)
    assert tuple(count(0.0, -1e-12)) == (0, 0)
    lam, c = 0.5, 0.05
    want = 0
    for s in range(m):
        for k in range(n):
            t = k / n + shifts[s, 0]
            t -= 1.0 if t >= 1.0 else 0.0
            x = 1.0 - abs(2.0 * t - 1.0)
            want += (x * (1.0 - x) <= c / lam)
    got = count(lam, c)
    assert 0 < want < n * m and abs(int(got[1]) - want) <= 2       # <= 2: points within rounding of the threshold


# ------------------------------------------------------------------------------- P17
def test_p17_neumaier_sum_equals_the_exactly_rounded_sum_where_a_plain_sum_fails():
    """A6: trigonometric terms of amplitude 1e8 that cancel to c0 per point on average (pin P5's class).  The sum
    of the n computed terms is compared with math.fsum of the very same per-point values (exactly rounded): the
    compensated accumulator agrees to an ulp, a plain left-to-right FP64 sum of the same values does not."""
    n, z = 65521, np.array([1, 17492, 0, 0, 0, 0, 0, 0], np.uint64)
    hs = [(1, 0), (0, 1), (3, -2), (5, 7)]
    amps = [1.0e8, -0.7e8, 0.4e8, 0.9e8]
    sector = W.Sector(dim=2, kind=W.KIND_TRIG, transform=W.TRANSFORM_NONE, logc=np.array([1.0]),
                      trig_h=np.array(hs, np.int32), trig_amp=np.array(amps), trig_phase=np.array([0.1, 0.7, 1.3, 2.9]))
    sec = O.OracleSector(sector)
    delta = np.array([[0.123456789, 0.987654321]])
    sums, _ = O.shift_sums(sec, n, z, delta)
    vals = [O.eval_point(sec, n, z, delta[0], k)[3][0].real for k in range(n)]
    exact = math.fsum(vals)
    exact_abs = math.fsum(abs(v) for v in vals)
    plain = 0.0
    for v in vals:
        plain += v
    ulp = math.ulp(abs(exact))
    assert abs(sums[0, 0, 0] - exact) <= 2 * ulp + 1e-30 * exact_abs
    assert abs(sums[0, 0, 2] - exact_abs) <= 2 * math.ulp(exact_abs)
    assert abs(plain - exact) > 1000 * ulp                        # the pin is sharp: a plain sum fails it
    assert exact_abs > 1e7 * abs(exact)                           # cancellation by more than seven digits
