"""Writes tests/golden/closed_forms.txt: exact values the CPU oracle is pinned to (tests/test_oracle_pins.py).

Pure mathematics only (Python ``math`` and exact ``fractions``): this script calls neither the oracle nor the
CUDA path.  The paper (arXiv:2305.19768) prints no numerical value on the hot path -- its only equations there
are Eq. (1)-(8), PAPER.md:215-288 -- so the stored values are closed forms of textbook integrals that the
method must reproduce (SURVEY.md 8(c).4 pins P3, P7, P8):

  korobov3_const_n<n>_d<delta>   rank-1 lattice rule with the Korobov r=3 transform applied to f = 1 in d = 1:
                                 Q = 1 - 70 B4(theta)/n^4 - 140 B6(theta)/n^6, theta = frac(n delta)
                                 (Euler-Maclaurin for the degree-6 weight 140 t^3 (1-t)^3; transform named at PAPER.md:707)
  bubble_eps0_m2_1.3_P2_2.7      eps^0 coefficient of the one-loop Euclidean massive bubble,
                                 -[log m^2 - 2 + beta log((beta+1)/(beta-1))], beta = sqrt(1 + 4 m^2/P^2)
  triangle_m2_1.3_P2_2.7         one-loop Euclidean triangle, log^2((beta+1)/(beta-1)) / (2 P^2)
  phys1d_a<a>_q<q>_pow_{re,im}   pin P15, the physical region (F changes sign; "contour deformation"; the
  phys1d_a<a>_q<q>_log_{re,im}   -i delta prescription of BASELINE.json config 3): for 0 < a < 1
                                   int_0^1 (a - x - i0)^q dx          = [a^(q+1) - w^(q+1)] / (q+1)
                                   int_0^1 (a - x - i0)^q Log(a - x - i0) dx = G(a) - G(w),
                                   G(v) = v^(q+1) (Log v / (q+1) - 1/(q+1)^2),
                                 with w = a - 1 - i0 = (1 - a) e^(-i pi), i.e. w^(q+1) = (1-a)^(q+1) e^(-i pi (q+1)) and
                                 Log w = log(1-a) - i pi.  For q = -1/2 the first is 2 sqrt(a) + 2 i sqrt(1-a).  The
                                 stored values keep the finite delta = 1e-12 (a -> a - i delta in the formulas).  For
                                 q <= -1 the real-axis integral diverges at x = a; the value is the analytic
                                 continuation, which is what the deformed contour computes.
  sep_u_b<b>_p<p>                int_0^1 (1 + b y)^p dy = ((1+b)^(p+1) - 1) / (b (p+1)): the U-factor of the separable
                                 d = 2 variant of P15

    python tests/golden/make_closed_forms.py
"""
import cmath
import math
import os
from fractions import Fraction


def korobov3_const(n: int, delta: str) -> float:
    th = (n * Fraction(delta)) % 1
    B4 = th**4 - 2 * th**3 + th**2 - Fraction(1, 30)
    B6 = th**6 - 3 * th**5 + Fraction(5, 2) * th**4 - Fraction(1, 2) * th**2 + Fraction(1, 42)
    return float(1 - 70 * B4 / Fraction(n)**4 - 140 * B6 / Fraction(n)**6)


def phys1d(a: float, q: float, delta: float = 1e-12):
    """(int (A - x)^q dx, int (A - x)^q Log(A - x) dx) over [0, 1] with A = a - i delta, by the antiderivatives in
    the docstring.  Im A < 0 keeps A - x in the lower half plane, where the principal branch (cmath) is the -i0 one:
    at delta = 1e-12 (BASELINE.json config 3's prescription) the values differ from the delta -> 0 limit by ~1e-12."""
    e = q + 1.0
    A = complex(a, -delta)
    G = lambda v: v ** e * (cmath.log(v) / e - 1.0 / (e * e))
    return (A ** e - (A - 1.0) ** e) / e, G(A) - G(A - 1.0)


def main():
    m2, P2 = 1.3, 2.7
    beta = math.sqrt(1.0 + 4.0 * m2 / P2)
    lines = ["# name value   (written by tests/golden/make_closed_forms.py; see its docstring for the citations)"]
    for n in (1, 2, 5, 7, 13):
        for delta in ("1/10", "37/100", "1/2", "93/100"):
            lines.append("korobov3_const_n%d_d%s %r" % (n, delta, korobov3_const(n, delta)))
    lines.append("bubble_eps0_m2_1.3_P2_2.7 %r" % (-(math.log(m2) - 2.0 + beta * math.log((beta + 1.0) / (beta - 1.0)))))
    lines.append("triangle_m2_1.3_P2_2.7 %r" % (math.log((beta + 1.0) / (beta - 1.0)) ** 2 / (2.0 * P2)))
    for a, q in ((0.37, -0.5), (0.37, -1.3), (0.62, -0.5), (0.62, 0.75)):
        v_pow, v_log = phys1d(a, q)
        for tag, v in (("pow", v_pow), ("log", v_log)):
            lines.append("phys1d_a%s_q%s_%s_re %r" % (a, q, tag, v.real))
            lines.append("phys1d_a%s_q%s_%s_im %r" % (a, q, tag, v.imag))
    for b, p_ in ((0.8, -1.7),):
        lines.append("sep_u_b%s_p%s %r" % (b, p_, ((1.0 + b) ** (p_ + 1.0) - 1.0) / (b * (p_ + 1.0))))
    with open(os.path.join(os.path.dirname(os.path.abspath(__file__)), "closed_forms.txt"), "w") as f:
        f.write("\n".join(lines) + "\n")


if __name__ == "__main__":
    main()
