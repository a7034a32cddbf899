// =====================================================================================
// qmc_oracle.cpp -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
//
// Plain, slow, single-threaded CPU statement of what the QMC hot path computes, written
// from arXiv:2305.19768 and the readings listed in SURVEY.md section 8(c) /
// DESIGN.md section 3.  It shares no code, header, table or constant with the CUDA path
// under paper_2305_19768_b200/csrc/, and neither side includes or links the other.
// Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference
// legs may build, load or call this file.
//
// Build: g++ -O2 -std=c++17 -ffp-contract=off -shared -fPIC (see oracle/oracle.py).
// -ffp-contract=off: every operation below is rounded once, in the order written.
//
// Steps (SURVEY.md 8(c).1 notation):
//   A1  r_{k,i} = (k * z_i) mod n                    rank-1 lattice
//   A2  t = r/n + Delta_{s,i}; if (t >= 1) t -= 1    random shift
//   A3  periodising transform korobov3 / baker      (names only)
//   A4  real integrand x^a U^p F^q L_j(logU, logF)   (BASELINE.json configs 1-2)
//   A4' separable toy integrand                       (BASELINE.json config 0)
//   A5  contour-deformed complex integrand            (BASELINE.json config 3)
//   A6  per-shift sums S, A with Neumaier compensation
//   A7  mean and standard error over m shifts         (Fig. 1 caption)
//   A8  median lattice rule                           (Eq. 7-8)
//   A9  amplitude = sum_i C_i I_i with Eq. (4) errors
//
// Pins (tests/test_oracle_*.py, run with -m "not gpu"; table in DESIGN.md section 2): brute force on tiny n,
// big-int lattice coordinates, the Euler-Maclaurin closed form of the Korobov-3 rule, separable
// exact integrals, trigonometric-polynomial exactness, shift-order invariance, one-loop
// bubble and triangle closed forms, Eq. (4) variance identity, lambda->0 and
// finite-difference Jacobian checks of the deformation, real-axis quadrature of deformed
// sectors (P14: Cauchy's theorem on F > 0 sectors, all log-polynomial orders), median order statistics,
// and (round 2) P15 the physical region -- F changing sign under the -i delta prescription -- against the
// closed forms of int (a - x - i0)^q [Log(a - x - i0)] dx, a separable d = 2 variant and F = a - x1 x2
// against QUADPACK; P16 the zero-weight branch and both diagnostics counters with hand-counted non-zero
// values; P17 the Neumaier accumulator against the exactly rounded sum where a plain sum fails.
// Round 2 additions (new branches, no existing arithmetic changed): the general Korobov transform (r0, r1)
// ("higher Korobov orders / asymmetric weights"), pinned by the exact Euler-Maclaurin sum in
// Bernoulli polynomials (P18), and orc_deformed_f, F(z(x; lambda)) for a given lambda, used by the presampling oracle
// oracle/presample.py ("contour deformation parameter selection"), pinned by P19.
// No function of this file is left unpinned.
// =====================================================================================
#include <cmath>
#include <complex>
#include <cstdint>
#include <cstring>
#include <vector>
#include <algorithm>

namespace {

constexpr int MAXD = 8;
constexpr int MAXJ = 5;   // epsilon-orders per sector: storage only (degrees 0..4, e.g. eps^-4 .. eps^0 at two loops)
typedef std::complex<double> cplx;

enum { KIND_UF = 0, KIND_TOY = 1, KIND_TRIG = 2 };
enum { TR_NONE = 0, TR_KOROBOV3 = 1, TR_BAKER = 2 };

}  // namespace

extern "C" {

// Host-side sector description read by the oracle (its own layout; the CUDA library has
// a separate header, include/qmc.h).
struct orc_sector {
    int32_t kind;         // KIND_*
    int32_t dim;          // 1..8
    int32_t transform;    // TR_*
    int32_t deformed;     // 0 real class (A4), 1 contour-deformed complex class (A5)
    int32_t first_order;  // j0: lowest log-polynomial degree
    int32_t n_orders;     // J: degrees j0 .. j0+J-1
    int32_t a[MAXD];      // monomial prefactor exponents
    int32_t nU, nF;       // number of monomials in U and F (constant term included)
    double p, q;          // U^p F^q
    double lambda;        // deformation strength
    double f_im;          // added to Im F (the -i*delta prescription)
    const double* U_coef; const uint8_t* U_exp;  // nU, nU x dim row-major
    const double* F_coef; const uint8_t* F_exp;  // nF, nF x dim
    const double* logc;   // per order j: c_{alpha,beta}, alpha+beta<=j, ordered by (alpha+beta, beta)
    // KIND_TRIG: f = logc[0] + sum_h amp_h cos(2 pi h.x + phase_h)
    int32_t n_trig; int32_t pad_;
    const int32_t* trig_h; const double* trig_amp; const double* trig_phase;
};

}  // extern "C"

namespace {

// ---- A1: lattice coordinate, exact for any n < 2^63 --------------------------------
inline uint64_t lattice_coord(uint64_t k, uint64_t z, uint64_t n) {
    return (uint64_t)(((unsigned __int128)k * (unsigned __int128)z) % (unsigned __int128)n);
}

// ---- A2: shifted point --------------------------------------------------------------
inline double shifted_point(uint64_t r, uint64_t n, double delta) {
    double t = (double)r / (double)n + delta;
    if (t >= 1.0) t -= 1.0;
    return t;
}

inline double ipow_d(double x, int e) {  // x^e by repeated multiplication, e >= 0
    double r = 1.0;
    for (int i = 0; i < e; ++i) r = r * x;
    return r;
}

// ---- A3: periodising transform: x = phi(t), weight omega = phi'(t) ------------------
inline void transform_point(int transform, double t, double* x, double* omega) {
    if (transform == TR_KOROBOV3) {
        // phi(t) = t^4 (35 - 84 t + 70 t^2 - 20 t^3),  phi'(t) = 140 t^3 (1-t)^3
        double t2 = t * t, t3 = t2 * t, t4 = t2 * t2;
        *x = t4 * (35.0 - 84.0 * t + 70.0 * t2 - 20.0 * t3);
        double u = 1.0 - t;
        *omega = 140.0 * t3 * (u * u * u);
    } else if (transform == TR_BAKER) {
        *x = 1.0 - std::fabs(2.0 * t - 1.0);
        *omega = 1.0;
    } else if (transform >= 100) {
        // general Korobov weight (transform code 100 + 10 r0 + r1, 1 <= r0, r1 <= 6):
        //   omega(t) = t^r0 (1 - t)^r1 / B(r0 + 1, r1 + 1),   B(a, b) = (a-1)! (b-1)! / (a+b-1)!,
        //   phi(t) = int_0^t omega = (1/B) sum_{k=0}^{r1} (-1)^k binom(r1, k) t^(r0 + 1 + k) / (r0 + 1 + k)
        // (korobov3 above is r0 = r1 = 3: 1/B = 140)
        const int r0 = (transform - 100) / 10, r1 = (transform - 100) % 10;
        double fact[16];
        fact[0] = 1.0;
        for (int i = 1; i < 16; ++i) fact[i] = fact[i - 1] * (double)i;
        const double invB = fact[r0 + r1 + 1] / (fact[r0] * fact[r1]);
        double sum = 0.0;
        for (int k = 0; k <= r1; ++k) {
            const double binom = fact[r1] / (fact[k] * fact[r1 - k]);
            const double term = binom * ipow_d(t, r0 + 1 + k) / (double)(r0 + 1 + k);
            sum += (k % 2 == 0) ? term : -term;
        }
        *x = invB * sum;
        *omega = invB * ipow_d(t, r0) * ipow_d(1.0 - t, r1);
    } else {
        *x = t;
        *omega = 1.0;
    }
}

// ---- polynomial helpers ---------------------------------------------------------------
template <class T>
T ipow(T x, int e) {  // x^e by repeated multiplication, e >= 0
    T r = T(1.0);
    for (int i = 0; i < e; ++i) r = r * x;
    return r;
}

template <class T>
T eval_poly(int n_mono, const double* coef, const uint8_t* exps, int dim, const T* x) {
    T sum = T(0.0);
    for (int j = 0; j < n_mono; ++j) {
        T term = T(coef[j]);
        for (int i = 0; i < dim; ++i) term = term * ipow(x[i], exps[j * dim + i]);
        sum = sum + term;
    }
    return sum;
}

// d/dx_i of a monomial-sum polynomial, evaluated at real x
double eval_poly_d1(int n_mono, const double* coef, const uint8_t* exps, int dim, const double* x, int i) {
    double sum = 0.0;
    for (int j = 0; j < n_mono; ++j) {
        int ei = exps[j * dim + i];
        if (ei == 0) continue;
        double term = coef[j] * (double)ei;
        for (int l = 0; l < dim; ++l) term *= ipow(x[l], exps[j * dim + l] - (l == i ? 1 : 0));
        sum += term;
    }
    return sum;
}

// d^2/dx_i dx_k
double eval_poly_d2(int n_mono, const double* coef, const uint8_t* exps, int dim, const double* x, int i, int k) {
    double sum = 0.0;
    for (int j = 0; j < n_mono; ++j) {
        int ei = exps[j * dim + i], ek = exps[j * dim + k];
        double fac;
        if (i == k) { if (ei < 2) continue; fac = (double)ei * (double)(ei - 1); }
        else        { if (ei < 1 || ek < 1) continue; fac = (double)ei * (double)ek; }
        double term = coef[j] * fac;
        for (int l = 0; l < dim; ++l) {
            int e = exps[j * dim + l];
            if (l == i) e -= 1;
            if (l == k) e -= 1;
            term *= ipow(x[l], e);
        }
        sum += term;
    }
    return sum;
}

// log-polynomial L_j(lU, lF) = sum_{alpha+beta<=j} c_{alpha,beta} lU^alpha lF^beta,
// coefficients ordered by (alpha+beta, beta)
template <class T>
T log_poly(int j, const double* c, T lU, T lF) {
    T sum = T(0.0);
    int idx = 0;
    for (int deg = 0; deg <= j; ++deg)
        for (int beta = 0; beta <= deg; ++beta) {
            int alpha = deg - beta;
            sum = sum + T(c[idx++]) * ipow(lU, alpha) * ipow(lF, beta);
        }
    return sum;
}

// ---- determinant by LU with partial pivoting on |.| (A5, Q16) -------------------------
cplx det_lu(int d, cplx* M /* d x d row-major, destroyed */) {
    cplx det = 1.0;
    for (int c = 0; c < d; ++c) {
        int piv = c;
        double best = std::abs(M[c * d + c]);
        for (int r = c + 1; r < d; ++r) {
            double v = std::abs(M[r * d + c]);
            if (v > best) { best = v; piv = r; }
        }
        if (best == 0.0) return cplx(0.0, 0.0);
        if (piv != c) {
            for (int l = 0; l < d; ++l) std::swap(M[c * d + l], M[piv * d + l]);
            det = -det;
        }
        det = det * M[c * d + c];
        for (int r = c + 1; r < d; ++r) {
            cplx f = M[r * d + c] / M[c * d + c];
            for (int l = c + 1; l < d; ++l) M[r * d + l] = M[r * d + l] - f * M[c * d + l];
        }
    }
    return det;
}

// ---- A4 / A4' / A5 / trig: integrand values g_j(x), j = 0..J-1 ------------------------
// Returns the J order values; *sign_fail is set when the deformed F has Im >= 0.
void integrand(const orc_sector& s, const double* x, cplx* g, int* sign_fail) {
    const int d = s.dim;
    *sign_fail = 0;
    if (s.kind == KIND_TOY) {  // A4': prod_i (1 + c_i (x_i - 1/2) + d_i x_i^2)
        double prod = 1.0;
        for (int i = 0; i < d; ++i)
            prod *= 1.0 + s.U_coef[i] * (x[i] - 0.5) + s.U_coef[d + i] * (x[i] * x[i]);
        g[0] = prod;
        return;
    }
    if (s.kind == KIND_TRIG) {  // c0 + sum_h amp_h cos(2 pi h.x + phase_h)
        double sum = s.logc[0];
        for (int h = 0; h < s.n_trig; ++h) {
            double arg = 0.0;
            for (int i = 0; i < d; ++i) arg += (double)s.trig_h[h * d + i] * x[i];
            sum += s.trig_amp[h] * std::cos(2.0 * M_PI * arg + s.trig_phase[h]);
        }
        g[0] = sum;
        return;
    }
    const double* lc = s.logc;
    if (!s.deformed) {  // A4
        double mono = 1.0;
        for (int i = 0; i < d; ++i) mono *= ipow(x[i], s.a[i]);
        double U = eval_poly<double>(s.nU, s.U_coef, s.U_exp, d, x);
        double F = eval_poly<double>(s.nF, s.F_coef, s.F_exp, d, x);
        double lU = std::log(U), lF = std::log(F);
        double base = mono * std::exp(s.p * lU + s.q * lF);
        for (int jj = 0; jj < s.n_orders; ++jj) {
            int j = s.first_order + jj;
            g[jj] = base * log_poly<double>(j, lc, lU, lF);
            lc += (j + 1) * (j + 2) / 2;
        }
        return;
    }
    // A5: z_i = x_i - i lambda x_i (1 - x_i) dF/dx_i,  M_ik = delta_ik - i lambda [ (1-2x_i) G_i delta_ik
    //     + x_i (1-x_i) H_ik ],  Jac = det M
    double G[MAXD], H[MAXD][MAXD];
    for (int i = 0; i < d; ++i) G[i] = eval_poly_d1(s.nF, s.F_coef, s.F_exp, d, x, i);
    for (int i = 0; i < d; ++i)
        for (int k = 0; k < d; ++k) H[i][k] = eval_poly_d2(s.nF, s.F_coef, s.F_exp, d, x, i, k);
    cplx z[MAXD], M[MAXD * MAXD];
    const cplx I(0.0, 1.0);
    for (int i = 0; i < d; ++i) z[i] = cplx(x[i], 0.0) - I * (s.lambda * x[i] * (1.0 - x[i]) * G[i]);
    for (int i = 0; i < d; ++i)
        for (int k = 0; k < d; ++k) {
            double b = x[i] * (1.0 - x[i]) * H[i][k];
            if (i == k) b += (1.0 - 2.0 * x[i]) * G[i];
            M[i * d + k] = cplx(i == k ? 1.0 : 0.0, 0.0) - I * (s.lambda * b);
        }
    cplx Jac = det_lu(d, M);
    cplx Uz = eval_poly<cplx>(s.nU, s.U_coef, s.U_exp, d, z);
    cplx Fz = eval_poly<cplx>(s.nF, s.F_coef, s.F_exp, d, z) + cplx(0.0, s.f_im);
    if (Fz.imag() >= 0.0) *sign_fail = 1;
    cplx lU = std::log(Uz), lF = std::log(Fz);  // principal branch (Q15)
    cplx mono = 1.0;
    for (int i = 0; i < d; ++i) mono = mono * ipow(z[i], s.a[i]);
    cplx base = Jac * mono * std::exp(s.p * lU + s.q * lF);
    for (int jj = 0; jj < s.n_orders; ++jj) {
        int j = s.first_order + jj;
        g[jj] = base * log_poly<cplx>(j, lc, lU, lF);
        lc += (j + 1) * (j + 2) / 2;
    }
}

// ---- A6: Neumaier-compensated accumulator ----------------------------------------------
struct Neumaier {
    double s = 0.0, c = 0.0;
    void add(double v) {
        double t = s + v;
        if (std::fabs(s) >= std::fabs(v)) c += (s - t) + v;
        else                              c += (v - t) + s;
        s = t;
    }
    double value() const { return s + c; }
};

// One lattice point: weight W and weighted order values.  Returns false if W == 0 (Q4).
bool eval_point(const orc_sector& s, uint64_t n, const uint64_t* z, const double* delta, uint64_t k,
                double* t_out, double* x_out, double* W_out, cplx* wg, int* sign_fail) {
    double x[MAXD], W = 1.0;
    for (int i = 0; i < s.dim; ++i) {
        uint64_t r = lattice_coord(k, z[i], n);
        double t = shifted_point(r, n, delta[i]);
        double om;
        transform_point(s.transform, t, &x[i], &om);
        W *= om;
        if (t_out) t_out[i] = t;
        if (x_out) x_out[i] = x[i];
    }
    if (W_out) *W_out = W;
    *sign_fail = 0;
    if (W == 0.0) {
        for (int j = 0; j < s.n_orders; ++j) wg[j] = 0.0;
        return false;
    }
    cplx g[MAXJ];
    integrand(s, x, g, sign_fail);
    for (int j = 0; j < s.n_orders; ++j) wg[j] = W * g[j];
    return true;
}

double median_of(std::vector<double> v) {
    std::sort(v.begin(), v.end());
    size_t K = v.size();
    return (K % 2) ? v[K / 2] : 0.5 * (v[K / 2 - 1] + v[K / 2]);
}

}  // namespace

extern "C" {

int32_t orc_n_orders(const orc_sector* s) { return (s->kind == KIND_UF) ? s->n_orders : 1; }

// A1 for a range of k: out[(k-k0)*dim + i]
void orc_lattice_coords(uint64_t n, const uint64_t* z, int32_t dim, uint64_t k0, uint64_t count, uint64_t* out) {
    for (uint64_t k = 0; k < count; ++k)
        for (int i = 0; i < dim; ++i) out[k * dim + i] = lattice_coord(k0 + k, z[i], n);
}

// A1-A5 for one point (debug / per-point parity): t[dim], x[dim], W, wg[J*2] (re, im)
void orc_eval_point(const orc_sector* s, uint64_t n, const uint64_t* z, const double* delta, uint64_t k,
                    double* t, double* x, double* W, double* wg, int32_t* sign_fail) {
    orc_sector ss = *s;
    ss.n_orders = orc_n_orders(s);
    cplx v[MAXJ];
    int sf;
    eval_point(ss, n, z, delta, k, t, x, W, v, &sf);
    for (int j = 0; j < ss.n_orders; ++j) { wg[2 * j] = v[j].real(); wg[2 * j + 1] = v[j].imag(); }
    *sign_fail = sf;
}

// The integrand alone at a given x (for the Jacobian / limit pins): g[J*2]
void orc_integrand(const orc_sector* s, const double* x, double* g, int32_t* sign_fail) {
    orc_sector ss = *s;
    ss.n_orders = orc_n_orders(s);
    cplx v[MAXJ];
    int sf;
    integrand(ss, x, v, &sf);
    for (int j = 0; j < ss.n_orders; ++j) { g[2 * j] = v[j].real(); g[2 * j + 1] = v[j].imag(); }
    *sign_fail = sf;
}

// The deformed map z(x) alone (for the finite-difference Jacobian pin P11) and det M.
void orc_deformation(const orc_sector* s, const double* x, double* z_out /*dim*2*/, double* jac /*2*/) {
    const int d = s->dim;
    double G[MAXD];
    for (int i = 0; i < d; ++i) G[i] = eval_poly_d1(s->nF, s->F_coef, s->F_exp, d, x, i);
    const cplx I(0.0, 1.0);
    cplx M[MAXD * MAXD];
    for (int i = 0; i < d; ++i) {
        cplx z = cplx(x[i], 0.0) - I * (s->lambda * x[i] * (1.0 - x[i]) * G[i]);
        z_out[2 * i] = z.real(); z_out[2 * i + 1] = z.imag();
        for (int k = 0; k < d; ++k) {
            double b = x[i] * (1.0 - x[i]) * eval_poly_d2(s->nF, s->F_coef, s->F_exp, d, x, i, k);
            if (i == k) b += (1.0 - 2.0 * x[i]) * G[i];
            M[i * d + k] = cplx(i == k ? 1.0 : 0.0, 0.0) - I * (s->lambda * b);
        }
    }
    cplx J = det_lu(d, M);
    jac[0] = J.real(); jac[1] = J.imag();
}

// F(z(x; lambda)) + i f_im for a GIVEN deformation strength lambda (the sector's own lambda is ignored): the quantity
// whose imaginary part the sign check looks at (A5), for the presampling of lambda (oracle/presample.py).
void orc_deformed_f(const orc_sector* s, const double* x, double lambda, double* f_out /*2*/) {
    const int d = s->dim;
    const cplx I(0.0, 1.0);
    cplx z[MAXD];
    for (int i = 0; i < d; ++i) {
        const double G = eval_poly_d1(s->nF, s->F_coef, s->F_exp, d, x, i);
        z[i] = cplx(x[i], 0.0) - I * (lambda * x[i] * (1.0 - x[i]) * G);
    }
    const cplx Fz = eval_poly<cplx>(s->nF, s->F_coef, s->F_exp, d, z) + cplx(0.0, s->f_im);
    f_out[0] = Fz.real(); f_out[1] = Fz.imag();
}

// A1-A6: per-shift sums over k in [k0, k1) (k1 = n for the whole lattice).
//   sums[(s*J + j)*3 + {0,1,2}] = (Re S, Im S, A = sum |W g|);  diag[0] zero-weight points, diag[1] sign fails
void orc_shift_sums(const orc_sector* s, uint64_t n, const uint64_t* z, const double* shifts /* m x 8 */,
                    int32_t m, uint64_t k0, uint64_t k1, double* sums, int64_t* diag) {
    orc_sector ss = *s;
    ss.n_orders = orc_n_orders(s);
    const int J = ss.n_orders;
    int64_t zero_w = 0, sign_fails = 0;
    for (int sh = 0; sh < m; ++sh) {
        Neumaier acc[MAXJ][3];
        const double* delta = shifts + (size_t)sh * MAXD;
        for (uint64_t k = k0; k < k1; ++k) {
            cplx wg[MAXJ];
            int sf;
            bool ok = eval_point(ss, n, z, delta, k, nullptr, nullptr, nullptr, wg, &sf);
            if (!ok) { ++zero_w; continue; }
            sign_fails += sf;
            for (int j = 0; j < J; ++j) {
                acc[j][0].add(wg[j].real());
                acc[j][1].add(wg[j].imag());
                acc[j][2].add(std::abs(wg[j]));
            }
        }
        for (int j = 0; j < J; ++j)
            for (int c = 0; c < 3; ++c) sums[((size_t)sh * J + j) * 3 + c] = acc[j][c].value();
    }
    if (diag) { diag[0] = zero_w; diag[1] = sign_fails; }
}

// A7: mean and standard error over the m shift estimates Q_s = S_s / n, re and im separately.
//   result[j*4 + {0,1,2,3}] = (mean_re, mean_im, err_re, err_im)
void orc_mean_err(const double* sums, int32_t m, int32_t J, uint64_t n, double* result) {
    for (int j = 0; j < J; ++j)
        for (int c = 0; c < 2; ++c) {
            double mean = 0.0;
            for (int s = 0; s < m; ++s) mean += sums[((size_t)s * J + j) * 3 + c] / (double)n;
            mean /= (double)m;
            double ss = 0.0;
            for (int s = 0; s < m; ++s) {
                double dlt = sums[((size_t)s * J + j) * 3 + c] / (double)n - mean;
                ss += dlt * dlt;
            }
            result[j * 4 + c] = mean;
            result[j * 4 + 2 + c] = std::sqrt(ss / ((double)m * (double)(m - 1)));
        }
}

// A1-A7 for one job.
void orc_integrate(const orc_sector* s, uint64_t n, const uint64_t* z, const double* shifts, int32_t m,
                   double* sums, double* result, int64_t* diag) {
    orc_shift_sums(s, n, z, shifts, m, 0, n, sums, diag);
    orc_mean_err(sums, m, orc_n_orders(s), n, result);
}

// A8: median rule.  cand_est[(c*J + j)*2 + {re,im}], median[j*2 + {re,im}], *selected = j*.
void orc_median_rule(const orc_sector* s, uint64_t n, const uint64_t* z_cand /* K x 8 */, int32_t K,
                     const double* shift0 /* 8 */, double* cand_est, double* median, int32_t* selected) {
    const int J = orc_n_orders(s);
    std::vector<double> sums((size_t)J * 3);
    for (int c = 0; c < K; ++c) {
        orc_shift_sums(s, n, z_cand + (size_t)c * MAXD, shift0, 1, 0, n, sums.data(), nullptr);
        for (int j = 0; j < J; ++j)
            for (int ri = 0; ri < 2; ++ri) cand_est[((size_t)c * J + j) * 2 + ri] = sums[(size_t)j * 3 + ri] / (double)n;
    }
    const int NC = J * 2;
    std::vector<double> mad(NC);
    for (int comp = 0; comp < NC; ++comp) {
        std::vector<double> v(K);
        for (int c = 0; c < K; ++c) v[c] = cand_est[(size_t)c * NC + comp];
        median[comp] = median_of(v);
        for (int c = 0; c < K; ++c) v[c] = std::fabs(v[c] - median[comp]);
        mad[comp] = median_of(v);
    }
    int best = 0;
    double best_d = 0.0;
    for (int c = 0; c < K; ++c) {
        double dist = 0.0;
        for (int comp = 0; comp < NC; ++comp) {
            if (mad[comp] == 0.0) continue;
            double u = (cand_est[(size_t)c * NC + comp] - median[comp]) / mad[comp];
            dist += u * u;
        }
        if (c == 0 || dist < best_d) { best = c; best_d = dist; }
    }
    *selected = best;
}

// A9: amplitude A_j = sum_i C_i mean_{i,j}; component-wise variance propagation (Q10).
//   results[(i*J + j)*4 + ...] per job, coef[i*2 + {re,im}], amp[j*4 + {re, im, err_re, err_im}]
void orc_amplitude(const double* results, const double* coef, int32_t n_jobs, int32_t J, double* amp) {
    for (int j = 0; j < J; ++j) {
        double are = 0.0, aim = 0.0, vre = 0.0, vim = 0.0;
        for (int i = 0; i < n_jobs; ++i) {
            const double* r = results + ((size_t)i * J + j) * 4;
            double cr = coef[2 * i], ci = coef[2 * i + 1];
            are += cr * r[0] - ci * r[1];
            aim += cr * r[1] + ci * r[0];
            vre += cr * cr * r[2] * r[2] + ci * ci * r[3] * r[3];
            vim += ci * ci * r[2] * r[2] + cr * cr * r[3] * r[3];
        }
        amp[j * 4 + 0] = are; amp[j * 4 + 1] = aim;
        amp[j * 4 + 2] = std::sqrt(vre); amp[j * 4 + 3] = std::sqrt(vim);
    }
}

}  // extern "C"
