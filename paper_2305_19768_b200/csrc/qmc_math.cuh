// =====================================================================================
// qmc_math.cuh -- FP64 elementary functions of the integrand evaluator (step a3), written for
// an FP64-pipe-bound kernel on sm_100a.  Part of the NVRTC program of every plan module (after
// the generated tables qmc_tab_*, see qmc_mathtab.cpp); no header, only CUDA built-ins.
//
// The CUDA library versions cost 24-45 FP64 instructions each and carry their polynomial
// coefficients as 64-bit literals, which the compiler materialises with two UMOVs per use.
// Here every function is  table lookup (shared memory, LDS pipe) + short polynomial, with all
// coefficients in the constant bank:
//     qmc_log     11 FP64 instructions    |err| <= 1.0e-16 max(1, |log x|)   (measured, see
//     qmc_exp     10                      rel err <= 2.3e-16                  tests/test_math_host.py)
// Arguments outside the fast range (non-positive, subnormal, huge, NaN) take the CUDA library
// function through a branch that the workloads never execute.
//
// Tables (generated in long double by qmc_mathtab.cpp, copied to shared memory by
// qmc_math_init at kernel start):
//     qmc_tab_log[2 i], [2 i + 1]   i = 0..128:  c_i = fl(1 / (1 + i/128)),  L_i = -log(c_i) - (i > 53) log 2
//     qmc_tab_exp[j]                j = 0..127:  2^(j/128)
// =====================================================================================
#ifndef QMC_MATH_CUH_
#define QMC_MATH_CUH_

#define QMC_LOG_TAB 258
#define QMC_EXP_TAB 128

__shared__ double qmc_sh_log[QMC_LOG_TAB];
__shared__ double qmc_sh_exp[QMC_EXP_TAB];

// polynomial and reduction constants: a __constant__ array so that they are c[3][..] operands
__constant__ double qmc_mc[16] = {
    0x1.62e42fefa39efp-1,    //  0  ln2 hi
    0x1.abc9e3b39803fp-56,   //  1  ln2 lo
    -0.5,                    //  2  log1p: -1/2
    0x1.5555555555555p-2,    //  3  +1/3
    -0.25,                   //  4  -1/4
    0x1.999999999999ap-3,    //  5  +1/5
    -0x1.5555555555555p-3,   //  6  -1/6
    0x1.71547652b82fep+7,    //  7  128 / ln2
    -0x1.62e42fefa39efp-8,   //  8  -(ln2 / 128) hi
    -0x1.abc9e3b39803fp-63,  //  9  -(ln2 / 128) lo
    0.5,                     // 10  exp: 1/2
    0x1.5555555555555p-3,    // 11  1/6
    0x1.5555555555555p-5,    // 12  1/24
    0x1.1111111111111p-7,    // 13  1/120
    0x1.8p+52,               // 14  2^52 + 2^51: round-to-nearest-integer magic
    0.0};

__device__ __forceinline__ void qmc_math_init() {
    for (int i = threadIdx.x; i < QMC_LOG_TAB; i += blockDim.x) qmc_sh_log[i] = qmc_tab_log[i];
    for (int i = threadIdx.x; i < QMC_EXP_TAB; i += blockDim.x) qmc_sh_exp[i] = qmc_tab_exp[i];
    __syncthreads();
}

// the never-taken slow paths stay out of line so that the hot loop stays compact
__device__ __noinline__ double qmc_log_slow(double x) { return log(x); }
__device__ __noinline__ double qmc_exp_slow(double x) { return exp(x); }

// log x for positive normal x: x = 2^e m, m in [1, 2); i = round((m - 1) 128) picks c_i ~ 1/m, so
// r = m c_i - 1 is exact up to one rounding with |r| <= 2^-8, and
//     log x = e' log 2 + L_i + log1p(r),     log1p(r) = r - r^2/2 + r^3/3 - ... - r^6/6  (|r^7/7| < 2e-18)
// e' = e + (i > 53) keeps |L_i| <= log(2)/2 and makes L = 0, c = 1 or 1/2 around x = 1, so the
// result keeps full relative accuracy where log x -> 0.
__device__ __forceinline__ double qmc_log(double x) {
    const int hi = __double2hiint(x);
    if ((unsigned)(hi - 0x00100000) >= 0x7fe00000u - 0x00100000u) return qmc_log_slow(x);   // <= 0, subnormal, inf, nan
    const int idx = ((hi & 0x000fffff) + 0x1000) >> 13;                            // 0 .. 128
    const int e = (hi >> 20) - 1023 + (idx > 53 ? 1 : 0);
    const double m = __hiloint2double((hi & 0x000fffff) | 0x3ff00000, __double2loint(x));
    const double c = qmc_sh_log[2 * idx], L = qmc_sh_log[2 * idx + 1];
    const double r = fma(m, c, -1.0);
    const double ed = (double)e;
    double q = fma(r, qmc_mc[6], qmc_mc[5]);
    q = fma(r, q, qmc_mc[4]);
    q = fma(r, q, qmc_mc[3]);
    q = fma(r, q, qmc_mc[2]);
    const double r2 = r * r;
    const double base = fma(ed, qmc_mc[0], L);
    const double p = fma(r2, q, r);
    return fma(ed, qmc_mc[1], p) + base;
}

// exp a: k = round(a 128 / ln2), a = k ln2/128 + r with |r| <= ln2/256, so
//     exp a = 2^(k >> 7) T[k & 127] (1 + r + r^2/2 + r^3/6 + r^4/24 + r^5/120)   (|r^6/720| < 6e-19)
// The power of two is added to the exponent field; |a| <= 690 keeps the result normal.
__device__ __forceinline__ double qmc_exp(double a) {
    if (!(fabs(a) <= 690.0)) return qmc_exp_slow(a);
    const double t = fma(a, qmc_mc[7], qmc_mc[14]);
    const int k = __double2loint(t);
    const double kd = t - qmc_mc[14];
    double r = fma(kd, qmc_mc[8], a);
    r = fma(kd, qmc_mc[9], r);
    const double T = qmc_sh_exp[k & 127];
    double q = fma(r, qmc_mc[13], qmc_mc[12]);
    q = fma(r, q, qmc_mc[11]);
    q = fma(r, q, qmc_mc[10]);
    const double r2 = r * r;
    const double p = fma(r2, q, r);
    const double v = fma(T, p, T);
    return __hiloint2double(__double2hiint(v) + ((k >> 7) << 20), __double2loint(v));
}

#ifdef QMC_LIBDEVICE_MATH   // A/B measurement: the CUDA library versions (qmc_plan_opts.fast_math = 1)
#define qmc_log(x) log(x)
#define qmc_exp(x) exp(x)
#endif

__device__ __forceinline__ double qmc_rcp(double x) { return 1.0 / x; }
// principal complex logarithm
__device__ __forceinline__ void qmc_clog(double re, double im, double& lre, double& lim) {
    lre = 0.5 * qmc_log(fma(re, re, im * im));
    lim = atan2(im, re);
}
__device__ __forceinline__ void qmc_cexp(double are, double aim, double& ere, double& eim) {
    const double e = qmc_exp(are);
    double s, c;
    sincos(aim, &s, &c);
    ere = e * c;
    eim = e * s;
}

#endif  // QMC_MATH_CUH_
