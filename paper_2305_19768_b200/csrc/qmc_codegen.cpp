// =====================================================================================
// qmc_codegen.cpp -- "compiled from a seedable polynomial description" (north_star (3)).
//
// pySecDec generates one C++/CUDA function per sector integrand so that the compiler can
// optimise it.  This file does the same at qmc_plan time from the numeric
// description of include/qmc.h: it emits, per sector, a straight-line device function in
// which
//   - U, F, dF/dx_i and d2F/dx_i dx_k are sparse multivariate Horner forms (greedy: factor
//     out the variable shared by most monomials), coefficients as hex-float literals;
//   - real and complex arithmetic share one symbolic scalar layer that folds constants
//     (0, +-1, real coefficients, the real initial part of the deformation matrix), so the
//     real class and every real-valued sub-expression of the deformed class cost real ops;
//   - the d x d complex Jacobian determinant is an unrolled LU (no pivoting: the matrix is
//     I - i lambda B with B real);
//   - U^p F^q = exp(p log U + q log F) shares its logarithms with the log-polynomial orders.
// It also counts the FP64 operations it emitted and the algorithmic flops of the evaluation.
// =====================================================================================
#include "qmc_codegen.h"

#include <algorithm>
#include <array>
#include <cmath>
#include <cstdio>
#include <cstring>
#include <map>
#include <sstream>

namespace qmc {
namespace {

// FP64 instruction counts charged for the elementary functions of qmc_device.cuh (fma = 1)
constexpr double OPS_LOG = 8, OPS_EXP = 9, OPS_RCP = 4, OPS_ATAN2 = 16, OPS_SINCOS = 16, OPS_SQRT = 7;
// algorithmic flop constants.  SURVEY.md 8(d)'s cost model carries placeholders for the elementary
// functions (log 40, exp 36, atan2 60, sincos 70) "to be replaced by SASS counts of the build's own
// routines": these are the flops (fma = 2) of qmc_log / qmc_exp / qmc_atan2 / qmc_sincos in qmc_math.cuh.
constexpr double FL_LOG = 12, FL_EXP = 16, FL_ATAN2 = 27, FL_SINCOS = 30;

std::string lit(double v) {
    char buf[64];
    if (v == 0.0) return "0.0";
    std::snprintf(buf, sizeof buf, "%a", v);
    std::string s(buf);
    if (v < 0) s = "(" + s + ")";
    return s;
}

// ---- symbolic real scalar: a constant or a named temporary, with a free sign ------------
struct Sc {
    bool is_const = true;
    double c = 0.0;
    std::string name;
    bool neg = false;
    static Sc K(double v) { Sc s; s.is_const = true; s.c = v; return s; }
    static Sc V(const std::string& n) { Sc s; s.is_const = false; s.name = n; return s; }
    bool isK(double v) const { return is_const && c == v; }
};

struct Cx { Sc re, im; };

// A double whose low 32 mantissa bits are zero fits the 32-bit immediate field of DFMA / DMUL /
// DADD.  Any other literal would be materialised by two moves per use (UMOV / IMAD.MOV pairs:
// 40 % of the issue slots of the first version of these kernels), so it goes to the sector's
// __constant__ pool instead and is read as a constant-bank operand c[3][..] at no issue cost.
bool fits_immediate(double v) {
    uint64_t b;
    std::memcpy(&b, &v, sizeof b);
    return (b & 0xffffffffull) == 0;
}

class Emitter {
public:
    std::ostringstream os;
    double ops = 0;
    double eflops = 0;   // flops of the emitted code: fma = 2, add / mul = 1, calls = the flops of their routine
    int ntmp = 0;
    std::string pool_name = "qmc_kc";
    std::vector<double> pool;
    std::map<uint64_t, int> pool_index;
    std::string konst(double v) {
        if (fits_immediate(v)) return lit(v);
        uint64_t b;
        std::memcpy(&b, &v, sizeof b);
        auto it = pool_index.find(b);
        int idx;
        if (it == pool_index.end()) { idx = (int)pool.size(); pool.push_back(v); pool_index[b] = idx; }
        else idx = it->second;
        return pool_name + "[" + std::to_string(idx) + "]";
    }
    std::string str(const Sc& a) {
        if (a.is_const) return konst(a.c);
        return a.neg ? "(-" + a.name + ")" : a.name;
    }
    // hash-consing: an expression already emitted (same text = same operands, all temporaries are
    // single-assignment) is reused -- the gradient and Hessian Horner forms share many sub-polynomials
    std::map<std::string, std::string> seen;
    Sc emit(const std::string& expr, double cost = 1.0, double fl = 1.0) {
        auto it = seen.find(expr);
        if (it != seen.end()) return Sc::V(it->second);
        std::string n = "t" + std::to_string(ntmp++);
        seen[expr] = n;
        os << "        const double " << n << " = " << expr << ";\n";
        ops += cost;
        eflops += fl;
        return Sc::V(n);
    }
    Sc neg(Sc a) {
        if (a.is_const) return Sc::K(-a.c);
        a.neg = !a.neg;
        return a;
    }
    Sc add(const Sc& a, const Sc& b) {
        if (a.is_const && b.is_const) return Sc::K(a.c + b.c);
        if (a.isK(0.0)) return b;
        if (b.isK(0.0)) return a;
        if (!b.is_const && b.neg) { Sc bb = b; bb.neg = false; return emit(str(a) + " - " + str(bb)); }
        return emit(str(a) + " + " + str(b));
    }
    Sc sub(const Sc& a, const Sc& b) { return add(a, neg(b)); }
    Sc mul(const Sc& a, const Sc& b) {
        if (a.is_const && b.is_const) return Sc::K(a.c * b.c);
        if (a.isK(0.0) || b.isK(0.0)) return Sc::K(0.0);
        if (a.isK(1.0)) return b;
        if (b.isK(1.0)) return a;
        if (a.isK(-1.0)) return neg(b);
        if (b.isK(-1.0)) return neg(a);
        return emit(str(a) + " * " + str(b));
    }
    Sc fma(const Sc& a, const Sc& b, const Sc& c) {
        if (a.isK(0.0) || b.isK(0.0)) return c;
        if (a.is_const && b.is_const) return add(Sc::K(a.c * b.c), c);
        if (c.isK(0.0)) return mul(a, b);
        if (a.isK(1.0)) return add(b, c);
        if (b.isK(1.0)) return add(a, c);
        if (a.isK(-1.0)) return add(neg(b), c);
        if (b.isK(-1.0)) return add(neg(a), c);
        return emit("fma(" + str(a) + ", " + str(b) + ", " + str(c) + ")", 1.0, 2.0);
    }
    // complex
    Cx cK(double re, double im = 0.0) { return Cx{Sc::K(re), Sc::K(im)}; }
    Cx cneg(const Cx& a) { return Cx{neg(a.re), neg(a.im)}; }
    Cx cadd(const Cx& a, const Cx& b) { return Cx{add(a.re, b.re), add(a.im, b.im)}; }
    Cx cmul(const Cx& a, const Cx& b) {
        Sc re = fma(a.re, b.re, neg(mul(a.im, b.im)));
        Sc im = fma(a.re, b.im, mul(a.im, b.re));
        return Cx{re, im};
    }
    Cx cfma(const Cx& a, const Cx& b, const Cx& c) {
        Sc re = fma(a.re, b.re, fma(neg(a.im), b.im, c.re));
        Sc im = fma(a.re, b.im, fma(a.im, b.re, c.im));
        return Cx{re, im};
    }
    // a real-valued function call returning one double
    Sc call1(const char* fn, const Sc& a, double cost, double fl) { return emit(std::string(fn) + "(" + str(a) + ")", cost, fl); }
    // a call with two outputs
    Cx call2(const char* fn, const Sc& a, const Sc& b, double cost, double fl) {
        std::string n0 = "t" + std::to_string(ntmp++), n1 = "t" + std::to_string(ntmp++);
        os << "        double " << n0 << ", " << n1 << "; " << fn << "(" << str(a) << ", " << str(b) << ", " << n0
           << ", " << n1 << ");\n";
        ops += cost;
        eflops += fl;
        return Cx{Sc::V(n0), Sc::V(n1)};
    }
};

// ---- sparse polynomials -----------------------------------------------------------------
constexpr int MAXV = 8;
struct Term {
    double coef;
    std::array<uint8_t, MAXV> e;
};
typedef std::vector<Term> Poly;

Poly make_poly(const std::vector<double>& coef, const std::vector<uint8_t>& exps, int dim) {
    Poly p;
    for (size_t t = 0; t < coef.size(); ++t) {
        Term tm;
        tm.coef = coef[t];
        tm.e.fill(0);
        for (int i = 0; i < dim; ++i) tm.e[i] = exps[t * dim + i];
        p.push_back(tm);
    }
    return p;
}

Poly merged(const Poly& p) {
    std::map<std::array<uint8_t, MAXV>, double> acc;
    std::vector<std::array<uint8_t, MAXV>> order;
    for (const Term& t : p) {
        auto it = acc.find(t.e);
        if (it == acc.end()) { acc[t.e] = t.coef; order.push_back(t.e); }
        else it->second += t.coef;
    }
    Poly out;
    for (const auto& e : order)
        if (acc[e] != 0.0) out.push_back(Term{acc[e], e});
    return out;
}

Poly derivative(const Poly& p, int i) {
    Poly out;
    for (const Term& t : p) {
        if (t.e[i] == 0) continue;
        Term d = t;
        d.coef = t.coef * (double)t.e[i];
        d.e[i] = (uint8_t)(t.e[i] - 1);
        out.push_back(d);
    }
    return merged(out);
}

double poly_flops(const Poly& p) {  // monomial of degree g: g + 1 flops (coefficient multiply + add)
    double f = 0;
    for (const Term& t : p) {
        int g = 0;
        for (int i = 0; i < MAXV; ++i) g += t.e[i];
        f += g + 1;
    }
    return f;
}

// Greedy multivariate Horner: factor out the variable that occurs in most monomials.
Cx horner(Emitter& E, const Poly& p_in, const std::vector<Cx>& vars) {
    Poly p = merged(p_in);
    if (p.empty()) return E.cK(0.0);
    int nv = (int)vars.size();
    int best = -1, best_cnt = 0;
    for (int v = 0; v < nv; ++v) {
        int cnt = 0;
        for (const Term& t : p) cnt += t.e[v] > 0;
        if (cnt > best_cnt) { best_cnt = cnt; best = v; }
    }
    if (best < 0) return E.cK(p[0].coef);  // merged: a single constant term
    Poly A, B;
    for (const Term& t : p) {
        if (t.e[best] > 0) { Term a = t; a.e[best]--; A.push_back(a); }
        else B.push_back(t);
    }
    Cx b = horner(E, B, vars);
    Cx a = horner(E, A, vars);
    return E.cfma(vars[best], a, b);
}

Cx ipow(Emitter& E, const Cx& x, int e) {
    Cx r = E.cK(1.0);
    Cx base = x;
    while (e > 0) {
        if (e & 1) r = E.cmul(r, base);
        e >>= 1;
        if (e) base = E.cmul(base, base);
    }
    return r;
}

}  // namespace

SectorCode generate_sector(const SectorSpec& s, int case_id) {
    SectorCode out;
    const int d = s.dim;
    const bool toy = (s.kind == 1);
    const bool cplx = (!toy && s.deformed != 0);
    const int J = toy ? 1 : s.n_orders;
    out.cplx = cplx; out.J = J; out.D = d; out.TR = s.transform;

    bool regular = toy;     // d log g / dx bounded up to the prefactor: proved below for the real U/F class
    Emitter E;
    E.pool_name = "qmc_kc" + std::to_string(case_id);
    std::vector<Cx> x(d);
    for (int i = 0; i < d; ++i) x[i] = Cx{Sc::V("x[" + std::to_string(i) + "]"), Sc::K(0.0)};
    std::vector<Cx> g(J);
    Sc sign_flag = Sc::K(0.0);
    bool have_sign = false;
    double flops = 0;

    // lattice + shift + transform + weight (qmc_point): counted here, emitted in qmc_device.cuh
    double pre_ops = 0;
    const bool gen_korobov = s.transform >= 100;
    const int kr0 = gen_korobov ? (s.transform - 100) / 10 : 3, kr1 = gen_korobov ? (s.transform - 100) % 10 : 3;
    auto pow_muls = [](int e) { int m = 0; while (e > 1) { m += 1 + (e & 1); e >>= 1; } return m; };   // multiplications of x^e by squaring
    if (gen_korobov) {
        // t fma, t^(r0+1), Horner of degree r1, x = power * poly, t(1-t) or (t, 1-t), running product(s); weight at the end
        const int per_dim = 1 + pow_muls(kr0 + 1) + kr1 + 1 + (kr0 == kr1 ? 2 : 3);
        pre_ops = d * per_dim + pow_muls(kr0) + (kr0 == kr1 ? 1 : pow_muls(kr1) + 2);
        flops += d * (3 + 2 * (kr0 + kr1) + 4);
    } else if (s.transform == 1) { pre_ops = d * (2 + 6 + 2) + 3; flops += d * (3 + 14); }
    else if (s.transform == 2) { pre_ops = d * (2 + 2); flops += d * (3 + 3); }
    else { pre_ops = d * 2; flops += d * 3; }

    if (toy) {
        // prod_i (1 + c_i (x_i - 1/2) + d_i x_i^2) = prod_i ((1 - c_i/2) + x_i (c_i + d_i x_i))
        Sc prod = Sc::K(1.0);
        for (int i = 0; i < d; ++i) {
            const double c = s.U_coef[i], dd = s.U_coef[d + i];
            Sc inner = E.fma(Sc::K(dd), x[i].re, Sc::K(c));
            Sc f = E.fma(x[i].re, inner, Sc::K(1.0 - 0.5 * c));
            prod = E.mul(prod, f);
        }
        g[0] = Cx{prod, Sc::K(0.0)};
        flops += 5.0 * d + (d - 1);
    } else {
        Poly U = make_poly(s.U_coef, s.U_exp, d), F = make_poly(s.F_coef, s.F_exp, d);
        // which logarithms are needed
        bool needU = (s.p != 0.0), needF = (s.q != 0.0);
        {
            size_t idx = 0;
            for (int jj = 0; jj < J; ++jj) {
                int j = s.first_order + jj;
                for (int deg = 0; deg <= j; ++deg)
                    for (int beta = 0; beta <= deg; ++beta) {
                        int alpha = deg - beta;
                        double c = s.logc[idx++];
                        if (c != 0.0 && alpha > 0) needU = true;
                        if (c != 0.0 && beta > 0) needF = true;
                    }
            }
        }
        std::vector<Cx> pt = x;   // evaluation point: x (real class) or z (deformed)
        Cx jac = E.cK(1.0);
        if (cplx) {
            // gradient and Hessian of F at the real point x
            std::vector<Sc> G(d);
            std::vector<std::vector<Sc>> H(d, std::vector<Sc>(d));
            // Every use of the gradient and the Hessian below carries the factor -lambda (Im z_i and Im M_ik),
            // so it is folded into the coefficients of the derivative polynomials: G = -lambda dF/dx_i,
            // H = -lambda d2F/dx_i dx_k cost no multiplication at run time.
            auto scaled = [&](Poly p) { for (Term& t : p) t.coef *= -s.lambda; return p; };
            for (int i = 0; i < d; ++i) {
                Poly dF = derivative(F, i);
                flops += poly_flops(dF);
                G[i] = horner(E, scaled(dF), x).re;
                for (int k = i; k < d; ++k) {
                    Poly ddF = derivative(dF, k);
                    flops += poly_flops(ddF);
                    H[i][k] = horner(E, scaled(ddF), x).re;
                }
            }
            for (int i = 0; i < d; ++i)
                for (int k = 0; k < i; ++k) H[i][k] = H[k][i];
            // z_i = x_i - i lambda x_i (1 - x_i) G_i ;  M_ik = delta_ik - i lambda B_ik
            std::vector<Sc> xm(d), om2x(d);
            for (int i = 0; i < d; ++i) {
                xm[i] = E.fma(E.neg(x[i].re), x[i].re, x[i].re);          // x (1 - x)
                pt[i] = Cx{x[i].re, E.mul(xm[i], G[i])};                   // Im z_i = -lambda x (1 - x) dF/dx_i
                om2x[i] = E.fma(Sc::K(-2.0), x[i].re, Sc::K(1.0));         // 1 - 2 x
            }
            flops += 4.0 * d + 2.5 * d * d;
            if (d >= 6) {
                // det M through the SYMMETRIC similar matrix S = D^(-1/2) M D^(1/2), D = diag(x_i (1 - x_i)):
                //   S_ik = delta_ik (1 - i lambda (1 - 2 x_i) G_i) - i lambda s_i H_ik s_k,   s_i = sqrt(max(x_i (1 - x_i), 0)),
                // which needs no 1 / D_i.  A complex symmetric matrix is eliminated on its upper triangle alone
                // (L D L^T: sum k (k + 1) / 2 instead of sum k^2 complex updates, and half the live registers); it pays
                // from d = 6 on, where the d square roots cost less than the saved updates.  Pivots as in DESIGN.md Q16
                // (Hermitian part = 1).  x (1 - x) can round to -1e-16 at x = 1 + ulp: clamped, the row then decouples.
                std::vector<Sc> sq(d);
                for (int i = 0; i < d; ++i) sq[i] = E.call1("qmc_sqrt", E.call1("qmc_max0", xm[i], 1.0, 1.0), OPS_SQRT, 12.0);
                std::vector<std::vector<Cx>> S(d, std::vector<Cx>(d));
                for (int i = 0; i < d; ++i)
                    for (int k = i; k < d; ++k) {
                        Sc b = E.mul(E.mul(sq[i], H[i][k]), sq[k]);
                        if (i == k) b = E.fma(om2x[i], G[i], E.mul(xm[i], H[i][i]));
                        S[i][k] = Cx{Sc::K(i == k ? 1.0 : 0.0), b};
                    }
                for (int c = 0; c < d; ++c) {
                    jac = E.cmul(jac, S[c][c]);
                    if (c == d - 1) break;
                    const Cx& pv = S[c][c];
                    Sc den = E.fma(pv.re, pv.re, E.mul(pv.im, pv.im));
                    Sc rden = den.is_const ? Sc::K(1.0 / den.c) : E.call1("qmc_rcp", den, OPS_RCP, 8.0);
                    Cx inv{E.mul(pv.re, rden), E.neg(E.mul(pv.im, rden))};
                    for (int r = c + 1; r < d; ++r) {
                        Cx nf = E.cneg(E.cmul(S[c][r], inv));
                        for (int l = r; l < d; ++l) S[r][l] = E.cfma(nf, S[c][l], S[r][l]);
                    }
                }
            } else {
                std::vector<std::vector<Cx>> M(d, std::vector<Cx>(d));
                for (int i = 0; i < d; ++i)
                    for (int k = 0; k < d; ++k) {
                        Sc b = E.mul(xm[i], H[i][k]);
                        if (i == k) b = E.fma(om2x[i], G[i], b);
                        M[i][k] = Cx{Sc::K(i == k ? 1.0 : 0.0), b};             // Im M_ik, -lambda included
                    }
                // det M by unrolled LU
                for (int c = 0; c < d; ++c) {
                    jac = E.cmul(jac, M[c][c]);
                    if (c == d - 1) break;
                    const Cx& pv = M[c][c];
                    Sc den = E.fma(pv.re, pv.re, E.mul(pv.im, pv.im));
                    Sc rden = den.is_const ? Sc::K(1.0 / den.c) : E.call1("qmc_rcp", den, OPS_RCP, 8.0);
                    Cx inv{E.mul(pv.re, rden), E.neg(E.mul(pv.im, rden))};
                    for (int r = c + 1; r < d; ++r) {
                        Cx f = E.cmul(M[r][c], inv);
                        Cx nf = E.cneg(f);
                        for (int l = c + 1; l < d; ++l) M[r][l] = E.cfma(nf, M[c][l], M[r][l]);
                    }
                }
            }
            {
                double lu = 0;
                for (int k = 1; k < d; ++k) lu += 8.0 * k * k;
                flops += lu + 30.0 * d * (d - 1) / 2.0;
            }
        }
        // U and F at the evaluation point
        Cx Uv = E.cK(1.0), Fv = E.cK(1.0);
        if (needU) { Uv = horner(E, U, pt); flops += poly_flops(U) * (cplx ? 4 : 1); }
        if (needF) { Fv = horner(E, F, pt); flops += poly_flops(F) * (cplx ? 4 : 1); }
        Cx lU = E.cK(0.0), lF = E.cK(0.0);
        bool exp_bounded = false;
        if (cplx) {
            if (needF) {
                Fv.im = E.add(Fv.im, Sc::K(s.f_im));
                sign_flag = Fv.im; have_sign = true;
            }
            if (needU) {
                if (Uv.re.is_const && Uv.im.is_const) lU = E.cK(std::log(std::hypot(Uv.re.c, Uv.im.c)), std::atan2(Uv.im.c, Uv.re.c));
                else { lU = E.call2("QMC_CLOG", Uv.re, Uv.im, OPS_LOG + OPS_ATAN2 + 3, FL_LOG + FL_ATAN2 + 4); flops += FL_LOG + FL_ATAN2 + 3; }
            }
            if (needF) {
                if (Fv.re.is_const && Fv.im.is_const) lF = E.cK(std::log(std::hypot(Fv.re.c, Fv.im.c)), std::atan2(Fv.im.c, Fv.re.c));
                else { lF = E.call2("QMC_CLOG", Fv.re, Fv.im, OPS_LOG + OPS_ATAN2 + 3, FL_LOG + FL_ATAN2 + 4); flops += FL_LOG + FL_ATAN2 + 3; }
            }
        } else {
            // Range of a polynomial with non-negative coefficients and a positive constant term on the cube
            // 0 <= x_i <= 1 (+ 1 ulp from the transform): [c_0, sum c].  Where that proves the argument of the
            // logarithm positive and normal, and the exponent below bounded, the range guards of qmc_log /
            // qmc_exp are dead code and the unguarded versions are called (all of BASELINE.json C1 / C2).
            auto bounds = [&](const Poly& P, double& lo, double& hi) {
                lo = 0.0; hi = 0.0;
                for (const Term& t : P) {
                    if (!(t.coef >= 0.0)) return false;
                    bool constant = true;
                    for (int i = 0; i < d; ++i) constant = constant && t.e[i] == 0;
                    if (constant) lo += t.coef;
                    hi += t.coef;
                }
                hi *= 1.0 + 1e-9;
                return lo >= 1e-300 && hi <= 1e300;
            };
            double ulo = 1, uhi = 1, flo = 1, fhi = 1;
            const bool u_ok = bounds(U, ulo, uhi), f_ok = bounds(F, flo, fhi);
            if (needU) {
                if (Uv.re.is_const) lU = E.cK(std::log(Uv.re.c));
                else { lU = Cx{E.call1(u_ok ? "qmc_log_nocheck" : "qmc_log", Uv.re, OPS_LOG, FL_LOG), Sc::K(0.0)}; flops += FL_LOG; }
            }
            if (needF) {
                if (Fv.re.is_const) lF = E.cK(std::log(Fv.re.c));
                else { lF = Cx{E.call1(f_ok ? "qmc_log_nocheck" : "qmc_log", Fv.re, OPS_LOG, FL_LOG), Sc::K(0.0)}; flops += FL_LOG; }
            }
            regular = u_ok && f_ok;
            if (u_ok && f_ok) {
                const double lu = std::max(std::fabs(std::log(ulo)), std::fabs(std::log(uhi)));
                const double lf = std::max(std::fabs(std::log(flo)), std::fabs(std::log(fhi)));
                exp_bounded = std::fabs(s.p) * lu + std::fabs(s.q) * lf <= 600.0;
            }
        }
        // base = Jac * prod pt_i^{a_i} * exp(p lU + q lF)
        Cx arg{E.fma(Sc::K(s.p), lU.re, E.mul(Sc::K(s.q), lF.re)), E.fma(Sc::K(s.p), lU.im, E.mul(Sc::K(s.q), lF.im))};
        Cx ex = E.cK(1.0);
        if (arg.re.is_const && arg.im.is_const) {
            ex = E.cK(std::exp(arg.re.c) * std::cos(arg.im.c), std::exp(arg.re.c) * std::sin(arg.im.c));
        } else if (arg.im.isK(0.0)) {
            ex = Cx{E.call1(exp_bounded ? "qmc_exp_nocheck" : "qmc_exp", arg.re, OPS_EXP, FL_EXP), Sc::K(0.0)};
            flops += FL_EXP;
        } else {
            ex = E.call2("QMC_CEXP", arg.re, arg.im, OPS_EXP + OPS_SINCOS + 2, FL_EXP + FL_SINCOS + 2);
            flops += FL_EXP + FL_SINCOS + 2;
        }
        Cx mono = E.cK(1.0);
        for (int i = 0; i < d; ++i)
            if (s.a[i] > 0) mono = E.cmul(mono, ipow(E, pt[i], s.a[i]));
        Cx base = E.cmul(E.cmul(jac, mono), ex);
        // orders
        std::vector<Cx> lv = {lU, lF};
        size_t idx = 0;
        for (int jj = 0; jj < J; ++jj) {
            int j = s.first_order + jj;
            Poly L;
            for (int deg = 0; deg <= j; ++deg)
                for (int beta = 0; beta <= deg; ++beta) {
                    Term t; t.coef = s.logc[idx++]; t.e.fill(0);
                    t.e[0] = (uint8_t)(deg - beta); t.e[1] = (uint8_t)beta;
                    L.push_back(t);
                }
            g[jj] = E.cmul(base, horner(E, L, lv));
        }
        flops += cplx ? (30.0 * J + 20.0) : 20.0;
    }

    // accumulation: W g (1), S += (1), A += |.| (1) per real component; sqrt for the complex modulus
    double acc_ops = 0;
    if (cplx) acc_ops = J * (2 + 3 + 2 + OPS_SQRT); else acc_ops = J * 3;
    if (s.transform != 1 && !gen_korobov) acc_ops -= cplx ? 2 * J : J;
    if (s.transform == 1 && regular)                 // centred Korobov form: one FP64 instruction less per such dimension (same flops)
        for (int i = 0; i < d; ++i) if (toy || s.a[i] == 0) pre_ops -= 1;
    out.ops = E.ops + pre_ops + acc_ops;
    // flops of the code as emitted (what ncu's 2 DFMA + DMUL + DADD counts): a1/a2 per dimension
    // t = fma (2); korobov3: t^2, two Horner halves, their fma, t^4, x, s = fma, P *= s (12) + 3 for the weight;
    // baker: fma, 1 - |.| (3); accumulation per order: W g (1, korobov3 only), S += (1), A += |.| (1), and for the
    // complex class twice the products and sums plus the modulus (fma, mul, sqrt = 2 mul + 5 fma: 15)
    const bool any_korobov = s.transform == 1 || gen_korobov;
    double pre_fl = s.transform == 1 ? d * 14.0 + 3.0 : (s.transform == 2 ? d * 5.0 : d * 2.0);
    if (gen_korobov)   // fma = 2: t, Horner steps; mul = 1: powers, x, products; 1 - t or fma(-t, t, t)
        pre_fl = d * (2.0 + pow_muls(kr0 + 1) + 2.0 * kr1 + 1.0 + (kr0 == kr1 ? 3.0 : 3.0)) + pow_muls(kr0) + (kr0 == kr1 ? 1.0 : pow_muls(kr1) + 2.0);
    double acc_fl = cplx ? J * (3.0 + 15.0 + (any_korobov ? 2.0 : 0.0)) : J * (2.0 + (any_korobov ? 1.0 : 0.0));
    out.eflops = E.eflops + pre_fl + acc_fl;
    out.flops = flops + (cplx ? 7.0 * J : 3.0 * J);

    std::ostringstream os;
    // the result expressions may add pool entries: render them before the pool is written out
    std::vector<std::string> gre(J), gim(J);
    for (int jj = 0; jj < J; ++jj) { gre[jj] = E.str(g[jj].re); gim[jj] = E.str(g[jj].im); }
    const std::string sign_str = have_sign ? E.str(sign_flag) : std::string();
    if (!E.pool.empty()) {
        os << "__constant__ double " << E.pool_name << "[" << E.pool.size() << "] = {";
        for (size_t i = 0; i < E.pool.size(); ++i) os << (i ? ", " : "") << lit(E.pool[i]);
        os << "};\n";
    }
    out.n_const = (int)E.pool.size();
    os << "struct Sector_" << case_id << " {\n";
    os << "    static constexpr int D = " << d << ", TR = " << s.transform << ", J = " << J << ";\n";
    os << "    static constexpr bool CPLX = " << (cplx ? "true" : "false") << ";\n";
    // REGULAR: the integrand and d log g / dx_i (up to x_i^a_i) are bounded on the closed cube -- toy class, and U, F with
    // non-negative coefficients and a positive constant term; qmc_device.cuh then takes the centred Korobov form and
    // drops the select at zero-weight points
    os << "    static constexpr bool REGULAR = " << (regular ? "true" : "false") << ";\n";
    // CENTRED: dimensions that take the centred Korobov-3 form (qmc_device.cuh): regular sectors, dimensions without a
    // prefactor x_i^a_i (the toy class has none)
    unsigned centred = 0;
    if (regular && s.transform == 1)
        for (int i = 0; i < d; ++i) if (toy || s.a[i] == 0) centred |= 1u << i;
    os << "    static constexpr unsigned CENTRED = " << centred << "u;\n";
    os << "    static __device__ __forceinline__ double wscale() { return "
       << lit(s.transform == 1 ? std::pow(140.0, d) : (gen_korobov ? std::pow(std::tgamma(kr0 + kr1 + 2.0) / (std::tgamma(kr0 + 1.0) * std::tgamma(kr1 + 1.0)), d) : 1.0)) << "; }\n";
    os << "    static __device__ __forceinline__ int eval(const double (&x)[" << d << "], double (&g)["
       << (cplx ? 2 * J : J) << "]) {\n";
    if (cplx) os << "        int qmc_bad = 0;   // set by QMC_CLOG / QMC_CEXP when an argument leaves the fast range\n";
    os << E.os.str();
    for (int jj = 0; jj < J; ++jj) {
        if (cplx) {
            os << "        g[" << 2 * jj << "] = " << gre[jj] << ";\n";
            os << "        g[" << 2 * jj + 1 << "] = " << gim[jj] << ";\n";
        } else {
            os << "        g[" << jj << "] = " << gre[jj] << ";\n";
        }
    }
    const std::string bad_bits = cplx ? " | (qmc_bad << 1)" : "";
    if (have_sign) os << "        return ((" << sign_str << " >= 0.0) ? 1 : 0)" << bad_bits << ";\n";
    else os << "        return 0" << bad_bits << ";\n";
    os << "    }\n";
    if (cplx) {
        // The same evaluation with the range-guarded functions, out of line: the kernel calls it for a point
        // whose eval() came back with bit 1 set (an argument outside the fast range of log / exp / atan2 / sincos).
        std::string body = E.os.str();
        for (const char* pair : {"QMC_CLOG(", "QMC_CEXP("}) {
            const std::string from(pair), to = std::string(pair[4] == 'C' && pair[5] == 'L' ? "qmc_clog(" : "qmc_cexp(");
            for (size_t pos = 0; (pos = body.find(from, pos)) != std::string::npos; pos += to.size()) body.replace(pos, from.size(), to);
        }
        os << "    static __device__ __noinline__ int eval_checked(const double (&x)[" << d << "], double (&g)[" << 2 * J << "]) {\n";
        os << body;
        for (int jj = 0; jj < J; ++jj) {
            os << "        g[" << 2 * jj << "] = " << gre[jj] << ";\n";
            os << "        g[" << 2 * jj + 1 << "] = " << gim[jj] << ";\n";
        }
        if (have_sign) os << "        return (" << sign_str << " >= 0.0) ? 1 : 0;\n";
        else os << "        return 0;\n";
        os << "    }\n";
    }
    os << "};\n";
    out.text = os.str();
    return out;
}

}  // namespace qmc
