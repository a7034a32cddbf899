// =====================================================================================
// qmc_math.cuh -- FP64 elementary functions of the integrand evaluator (step a3), written for
// an FP64-pipe-bound kernel on sm_100a.  Part of the NVRTC program of every plan module (after
// the generated tables qmc_tab_*, see qmc_mathtab.cpp); no header, only CUDA built-ins.
//
// The CUDA library versions cost 24-45 FP64 instructions each and carry their polynomial
// coefficients as 64-bit literals, which the compiler materialises with two UMOVs per use.
// Here every function is  table lookup (shared memory, LDS pipe) + short polynomial, with all
// coefficients in the constant bank:
//     qmc_log      8 FP64 instructions    (errors measured over 2e7 random arguments against long double:
//     qmc_exp      9                       see DESIGN.md section 5)
// The tables are checked by tests/test_library_host.py, the functions end to end by the per-point
// parity tests in tests/test_gpu_parity.py.
// Arguments outside the fast range (non-positive, subnormal, huge, NaN) take the CUDA library
// function through a branch that the workloads never execute.
//
// Tables (generated in long double by qmc_mathtab.cpp, copied to shared memory by
// qmc_math_init at kernel start):
//     qmc_tab_log[2 i], [2 i + 1]   i = 0..1024: c_i = fl(1 / (1 + i/1024)), L_i = -log(c_i) - (i > 424) log 2
//     qmc_tab_exp[j]                j = 0..255:  2^(j/256)
//     qmc_tab_trig[2 j], [2 j + 1]  j = 0..255:  cos(2 pi j / 256), sin(2 pi j / 256)   (modules with
//                                   deformed sectors only: QMC_HAVE_CPLX)
// Complex class:  qmc_sincos 16 FP64 instructions, qmc_atan2 16 (+ an FP32 atan2f for the table
// index), qmc_rcp 4, qmc_sqrt 7, against 45-50 / 45-50 / 9 / 12 for the CUDA library versions.
// =====================================================================================
#ifndef QMC_MATH_CUH_
#define QMC_MATH_CUH_

#define QMC_LOG_TAB 2050
#define QMC_EXP_TAB 256

#define QMC_TRIG_N 256

__shared__ double qmc_sh_log[QMC_LOG_TAB];
__shared__ double qmc_sh_exp[QMC_EXP_TAB];
#ifdef QMC_HAVE_CPLX
__shared__ double qmc_sh_trig[2 * QMC_TRIG_N];
#endif

// polynomial and reduction constants: a __constant__ array so that they are c[3][..] operands
__constant__ double qmc_mc[32] = {
    0x1.62e42fefa39efp-1,    //  0  ln2 hi
    0x1.abc9e3b39803fp-56,   //  1  ln2 lo
    -0.5,                    //  2  log1p: -1/2
    0x1.5555555555555p-2,    //  3  +1/3
    -0.25,                   //  4  -1/4
    0x1.999999999999ap-3,    //  5  +1/5
    -0x1.5555555555555p-3,   //  6  -1/6
    0x1.71547652b82fep+8,    //  7  256 / ln2
    -0x1.62e42fefa39efp-9,   //  8  -(ln2 / 256) hi
    -0x1.abc9e3b39803fp-64,  //  9  -(ln2 / 256) lo
    0.5,                     // 10  exp: 1/2
    0x1.5555555555555p-3,    // 11  1/6
    0x1.5555555555555p-5,    // 12  1/24
    0x1.1111111111111p-7,    // 13  1/120
    0x1.8p+52,               // 14  2^52 + 2^51: round-to-nearest-integer magic
    0.0,                     // 15
    0x1.45f306dc9c883p+5,    // 16  256 / (2 pi)
    -0x1.921fb54442d18p-6,   // 17  -(2 pi / 256) hi
    -0x1.1a62633145c07p-60,  // 18  -(2 pi / 256) lo
    -0x1.5555555555555p-3,   // 19  sin: -1/6
    0x1.1111111111111p-7,    // 20  1/120
    -0x1.a01a01a01a01ap-13,  // 21  -1/5040
    0x1.5555555555555p-5,    // 22  cos: 1/24   (-1/2 is [2])
    -0x1.6c16c16c16c17p-10,  // 23  -1/720
    -0x1.5555555555555p-2,   // 24  atan: -1/3
    0x1.999999999999ap-3,    // 25  1/5
    -0x1.2492492492492p-3,   // 26  -1/7
    0x1.921fb54442d18p-6,    // 27  (2 pi / 256) hi
    0x1.1a62633145c07p-60,   // 28  (2 pi / 256) lo
    0.0, 0.0, 0.0};

__device__ __forceinline__ void qmc_math_init() {
    for (int i = threadIdx.x; i < QMC_LOG_TAB; i += blockDim.x) qmc_sh_log[i] = qmc_tab_log[i];
    for (int i = threadIdx.x; i < QMC_EXP_TAB; i += blockDim.x) qmc_sh_exp[i] = qmc_tab_exp[i];
#ifdef QMC_HAVE_CPLX
    for (int i = threadIdx.x; i < 2 * QMC_TRIG_N; i += blockDim.x) qmc_sh_trig[i] = qmc_tab_trig[i];
#endif
    __syncthreads();
}

// Rare paths are counted per tile in shared memory and added to the call's counters by the kernel (read by
// qmc_plan_slow_path_counts; tests assert > 0 where a case forces the path and 0 on the BASELINE.json configs):
// qmc_sh_slow = calls of the out-of-line CUDA-library versions below (argument outside the fast range of a guarded
// function); the evaluations re-done by eval_checked() of the deformed class are counted at the call site.
__shared__ unsigned int qmc_sh_slow;
__device__ __forceinline__ void qmc_count_slow() { atomicAdd(&qmc_sh_slow, 1u); }

// the rarely-taken slow paths stay out of line so that the hot loop stays compact
__device__ __noinline__ double qmc_log_slow(double x) { qmc_count_slow(); return log(x); }
__device__ __noinline__ double qmc_exp_slow(double x) { qmc_count_slow(); return exp(x); }

// log x for positive normal x: x = 2^e m, m in [1, 2); i = round((m - 1) 1024) picks c_i ~ 1/m, so
// r = m c_i - 1 is exact up to one rounding with |r| <= 2^-11, and
//     log x = e' log 2 + L_i + log1p(r),     log1p(r) = r - r^2/2 + r^3/3 - r^4/4   (|r^5/5| < 6e-18)
// e' = e + (i > 424) keeps |L_i| <= log(2)/2 and makes L = 0, c = 1 or 1/2 around x = 1, so the
// result keeps its relative accuracy where log x -> 0 (to r^4/5 < 1.2e-14 of it).  log 2 enters as one double: its
// rounding error 2.3e-17 e' is below 0.3 ulp of the result for every exponent.  (Round 1 used 257 entries and one
// more term: the kernels are bound by their FP64 instruction count, a 16 KB table in shared memory costs nothing.)
__device__ __forceinline__ double qmc_log_nocheck(double x) {   // x positive and normal (proved by the caller)
    const int hi = __double2hiint(x);
    const int idx = ((hi & 0x000fffff) + 0x200) >> 10;                             // 0 .. 1024
    const int e = (hi >> 20) - 1023 + (idx > 424 ? 1 : 0);
    const double m = __hiloint2double((hi & 0x000fffff) | 0x3ff00000, __double2loint(x));
    const double c = qmc_sh_log[2 * idx], L = qmc_sh_log[2 * idx + 1];
    const double r = fma(m, c, -1.0);
    const double ed = (double)e;
    double q = fma(r, qmc_mc[4], qmc_mc[3]);
    q = fma(r, q, qmc_mc[2]);
    const double r2 = r * r;
    const double base = fma(ed, qmc_mc[0], L);
    const double p = fma(r2, q, r);
    return p + base;
}
__device__ __forceinline__ double qmc_log(double x) {
    const int hi = __double2hiint(x);
    if ((unsigned)(hi - 0x00100000) >= 0x7fe00000u - 0x00100000u) return qmc_log_slow(x);   // <= 0, subnormal, inf, nan
    return qmc_log_nocheck(x);
}

// exp a: k = round(a 256 / ln2), a = k ln2/256 + r with |r| <= ln2/512, so
//     exp a = 2^(k >> 8) T[k & 255] (1 + r + r^2/2 + r^3/6 + r^4/24)   (|r^5/120| < 4e-17)
// The power of two is added to the exponent field; |a| <= 690 keeps the result normal.
__device__ __forceinline__ double qmc_exp_nocheck(double a) {   // |a| <= 690 (proved by the caller)
    const double t = fma(a, qmc_mc[7], qmc_mc[14]);
    const int k = __double2loint(t);
    const double kd = t - qmc_mc[14];
    double r = fma(kd, qmc_mc[8], a);
    r = fma(kd, qmc_mc[9], r);
    const double T = qmc_sh_exp[k & 255];
    double q = fma(r, qmc_mc[12], qmc_mc[11]);
    q = fma(r, q, qmc_mc[10]);
    const double r2 = r * r;
    const double p = fma(r2, q, r);
    const double v = fma(T, p, T);
    return __hiloint2double(__double2hiint(v) + ((k >> 8) << 20), __double2loint(v));
}
__device__ __forceinline__ double qmc_exp(double a) {
    if (!(fabs(a) <= 690.0)) return qmc_exp_slow(a);
    return qmc_exp_nocheck(a);
}

#ifdef QMC_LIBDEVICE_MATH   // A/B measurement: the CUDA library versions (qmc_plan_opts.libdevice_math = 1)
#define qmc_log(x) log(x)
#define qmc_exp(x) exp(x)
#define qmc_log_nocheck(x) log(x)
#define qmc_exp_nocheck(x) exp(x)
#endif

// ------------------------------------------------------------------------------------ complex class
#ifdef QMC_HAVE_CPLX
#define QMC_SQRT(x) qmc_sqrt(x)
// Hardware seeds (MUFU.RCP64H / MUFU.RSQ64H, about 20 good bits); a host harness may predefine them.
#ifndef QMC_RCP_APPROX
__device__ __forceinline__ double qmc_rcp_approx(double x) {
    double y;
    asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(x));
    return y;
}
__device__ __forceinline__ double qmc_rsqrt_approx(double x) {
    double y;
    asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(x));
    return y;
}
#define QMC_RCP_APPROX(x) qmc_rcp_approx(x)
#define QMC_RSQRT_APPROX(x) qmc_rsqrt_approx(x)
#endif

#ifdef QMC_LIBDEVICE_MATH
__device__ __forceinline__ double qmc_rcp(double x) { return 1.0 / x; }
__device__ __forceinline__ double qmc_sqrt(double x) { return sqrt(x); }
__device__ __forceinline__ void qmc_sincos(double a, double& sn, double& cs) { sincos(a, &sn, &cs); }
__device__ __forceinline__ double qmc_atan2(double y, double x) { return atan2(y, x); }
#else
// 1/x for normal x (LU pivots |M_cc|^2 >= 1 here): two Newton steps on the hardware seed, ~1 ulp
__device__ __forceinline__ double qmc_rcp(double x) {
    double y = QMC_RCP_APPROX(x);
    double e = fma(-x, y, 1.0);
    y = fma(y, e, y);
    e = fma(-x, y, 1.0);
    return fma(y, e, y);
}
// sqrt x, x >= 0: coupled Newton iteration for (sqrt x, 1 / (2 sqrt x)) and one residual step, ~1 ulp.
// Zero and subnormal x give 0 (the seed would be infinite).
__device__ __forceinline__ double qmc_sqrt(double x) {
    const double y = QMC_RSQRT_APPROX(x);
    double g = x * y, h = 0.5 * y;
    const double r = fma(-g, h, 0.5);
    g = fma(g, r, g);
    h = fma(h, r, h);
    const double d = fma(-g, g, x);
    g = fma(d, h, g);
    return ((unsigned)__double2hiint(x) < 0x00100000u) ? 0.0 : g;   // a select, no branch (x is a sum of squares)
}
__device__ __forceinline__ double qmc_max0(double x) { return fmax(x, 0.0); }
__device__ __noinline__ void qmc_sincos_slow(double a, double* sn, double* cs) { qmc_count_slow(); sincos(a, sn, cs); }
__device__ __noinline__ double qmc_atan2_slow(double y, double x) { qmc_count_slow(); return atan2(y, x); }

// sin a, cos a: j = round(a 256 / 2 pi), r = a - j 2 pi/256 (two-term constant), |r| <= pi/256;
// sin r and cos r - 1 by their series to r^7 and r^6 (next terms < 2e-23), then the angle-sum
// formulas with (cos, sin)(2 pi j/256) from the table.  |a| <= 1e5 keeps the reduction exact.
__device__ __forceinline__ void qmc_sincos(double a, double& sn, double& cs) {
    if (!(fabs(a) <= 1.0e5)) { qmc_sincos_slow(a, &sn, &cs); return; }
    const double t = fma(a, qmc_mc[16], qmc_mc[14]);
    const int j = __double2loint(t) & (QMC_TRIG_N - 1);
    const double kd = t - qmc_mc[14];
    double r = fma(kd, qmc_mc[17], a);
    r = fma(kd, qmc_mc[18], r);
    const double C = qmc_sh_trig[2 * j], S = qmc_sh_trig[2 * j + 1];
    const double r2 = r * r;
    double ps = fma(r2, qmc_mc[21], qmc_mc[20]);
    ps = fma(r2, ps, qmc_mc[19]);
    double pc = fma(r2, qmc_mc[23], qmc_mc[22]);
    pc = fma(r2, pc, qmc_mc[2]);
    const double sr = fma(r * r2, ps, r);   // sin r
    const double cm = r2 * pc;              // cos r - 1
    sn = fma(C, sr, fma(S, cm, S));
    cs = fma(-S, sr, fma(C, cm, C));
}

// atan2(y, x), principal value: the FP32 atan2f (FP32 / ALU pipes, idle here) picks the table angle
// theta_j = 2 pi j/256 nearest the argument; (x, y) is rotated by -theta_j exactly in FP64 to (u, v)
// with u > 0 and |v/u| <= tan(pi/256 + 1e-6), and   atan2 = theta_j + atan(v/u),
// atan w = w - w^3/3 + w^5/5 - w^7/7 (next term < 8e-19).  The sign of a zero or tiny y survives the
// float conversion, so the branch cut on the negative real axis is the library's.
__device__ __forceinline__ double qmc_atan2(double y, double x) {
    const unsigned ex = ((unsigned)__double2hiint(x) >> 20) & 0x7ffu, ey = ((unsigned)__double2hiint(y) >> 20) & 0x7ffu;
    const unsigned em = ex > ey ? ex : ey;
    if (em - 924u > 200u) return qmc_atan2_slow(y, x);          // max(|x|, |y|) outside [2^-99, 2^101]
    const float th = atan2f((float)y, (float)x);
    const int j = __float2int_rn(th * 40.7436654315f);          // 256 / (2 pi); -128 .. 128
    const int idx = j & (QMC_TRIG_N - 1);
    const double C = qmc_sh_trig[2 * idx], S = qmc_sh_trig[2 * idx + 1];
    const double u = fma(x, C, y * S);
    const double v = fma(y, C, -(x * S));
    const double w = v * qmc_rcp(u);
    const double w2 = w * w;
    double p = fma(w2, qmc_mc[26], qmc_mc[25]);
    p = fma(w2, p, qmc_mc[24]);
    const double at = fma(w * w2, p, w);
    const double jd = (double)j;
    return fma(jd, qmc_mc[27], fma(jd, qmc_mc[28], at));
}
#endif

// ---- unguarded versions for the hot path of the deformed class ---------------------------------
// The range guards above are branches, and a branch ends a basic block: ptxas cannot schedule across
// it (omitting the provably dead guards of the real class gave +7 %).  The arguments of the deformed
// class cannot be bounded at code-generation time, so its generated eval() calls these versions, which
// compute the fast path unconditionally (every table index is masked, so nothing can fault) and OR a
// flag when an argument was outside the fast range; the kernel then re-evaluates that point with the
// guarded functions (eval_checked, out of line).  No workload here ever sets the flag.
__device__ __forceinline__ int qmc_bad_log(double x) {
    return ((unsigned)(__double2hiint(x) - 0x00100000) >= 0x7fe00000u - 0x00100000u) ? 1 : 0;
}
__device__ __forceinline__ int qmc_bad_abs(double a, int hi_limit) {   // |a| > limit, inf or nan (by the high word)
    return ((__double2hiint(a) & 0x7fffffff) >= hi_limit) ? 1 : 0;
}
// angle of (x, y) to ~1e-5 rad in FP32, branch-free: odd minimax polynomial of atan on [0, 1] and
// octant fix-ups by selects; only used to pick the table cell of qmc_atan2_nc
__device__ __forceinline__ float qmc_angle_f32(float y, float x) {
    const float ax = fabsf(x), ay = fabsf(y);
    const float mx = fmaxf(ax, ay), mn = fminf(ax, ay);
    const float q = __fdividef(mn, mx);
    const float q2 = q * q;
    float p = fmaf(q2, -0.01172120f, 0.05265332f);
    p = fmaf(q2, p, -0.11643287f);
    p = fmaf(q2, p, 0.19354346f);
    p = fmaf(q2, p, -0.33262347f);
    p = fmaf(q2, p, 0.99997726f);
    float a = q * p;
    a = (ay > ax) ? 1.57079637f - a : a;
    a = (__float_as_int(x) < 0) ? 3.14159274f - a : a;
    return (__float_as_int(y) < 0) ? -a : a;
}
__device__ __forceinline__ double qmc_atan2_nc(double y, double x, int& bad) {
    const unsigned ex = ((unsigned)__double2hiint(x) >> 20) & 0x7ffu, ey = ((unsigned)__double2hiint(y) >> 20) & 0x7ffu;
    const unsigned em = ex > ey ? ex : ey;
    bad |= (em - 924u > 200u) ? 1 : 0;
    const float th = qmc_angle_f32((float)y, (float)x);
    const int j = __float2int_rn(th * 40.7436654315f);
    const int idx = j & (QMC_TRIG_N - 1);
    const double C = qmc_sh_trig[2 * idx], S = qmc_sh_trig[2 * idx + 1];
    const double u = fma(x, C, y * S);
    const double v = fma(y, C, -(x * S));
    const double w = v * qmc_rcp(u);
    const double w2 = w * w;
    double p = fma(w2, qmc_mc[26], qmc_mc[25]);
    p = fma(w2, p, qmc_mc[24]);
    const double at = fma(w * w2, p, w);
    const double jd = (double)j;
    return fma(jd, qmc_mc[27], fma(jd, qmc_mc[28], at));
}
__device__ __forceinline__ void qmc_sincos_nc(double a, double& sn, double& cs, int& bad) {
    bad |= qmc_bad_abs(a, 0x40f86a01);                           // |a| > 1e5
    const double t = fma(a, qmc_mc[16], qmc_mc[14]);
    const int j = __double2loint(t) & (QMC_TRIG_N - 1);
    const double kd = t - qmc_mc[14];
    double r = fma(kd, qmc_mc[17], a);
    r = fma(kd, qmc_mc[18], r);
    const double C = qmc_sh_trig[2 * j], S = qmc_sh_trig[2 * j + 1];
    const double r2 = r * r;
    double ps = fma(r2, qmc_mc[21], qmc_mc[20]);
    ps = fma(r2, ps, qmc_mc[19]);
    double pc = fma(r2, qmc_mc[23], qmc_mc[22]);
    pc = fma(r2, pc, qmc_mc[2]);
    const double sr = fma(r * r2, ps, r);
    const double cm = r2 * pc;
    sn = fma(C, sr, fma(S, cm, S));
    cs = fma(-S, sr, fma(C, cm, C));
}
#ifdef QMC_LIBDEVICE_MATH
#define qmc_clog_nc(re, im, lre, lim, bad) qmc_clog(re, im, lre, lim)
#define qmc_cexp_nc(are, aim, ere, eim, bad) qmc_cexp(are, aim, ere, eim)
#else
__device__ __forceinline__ void qmc_clog_nc(double re, double im, double& lre, double& lim, int& bad) {
    const double m2 = fma(re, re, im * im);
    bad |= qmc_bad_log(m2);
    lre = 0.5 * qmc_log_nocheck(m2);
    lim = qmc_atan2_nc(im, re, bad);
}
__device__ __forceinline__ void qmc_cexp_nc(double are, double aim, double& ere, double& eim, int& bad) {
    bad |= qmc_bad_abs(are, 0x40859001);                         // |Re| > 690
    const double e = qmc_exp_nocheck(are);
    double s, c;
    qmc_sincos_nc(aim, s, c, bad);
    ere = e * c;
    eim = e * s;
}
#endif
// the generated hot-path eval() of the deformed class calls these with its local flag `qmc_bad`
#define QMC_CLOG(a, b, c, d) qmc_clog_nc(a, b, c, d, qmc_bad)
#define QMC_CEXP(a, b, c, d) qmc_cexp_nc(a, b, c, d, qmc_bad)

// principal complex logarithm (guarded version, used by eval_checked only).  re^2 + im^2 under- or overflows for
// |z| outside [1e-146, 1e146]: there both parts are scaled by a power of two first (exact) and the exponent is added
// back as e log 2, so that log|z| keeps full accuracy down to subnormal z.
__device__ __noinline__ double qmc_clog_re_scaled(double re, double im) {
    qmc_count_slow();
    const double big = fmax(fabs(re), fabs(im));
    if (!(big > 0.0) || !(big < 1.0 / 0.0)) return log(big);        // 0 -> -inf, inf -> inf, nan -> nan
    int e;
    (void)frexp(big, &e);
    const double a = ldexp(re, -e), b = ldexp(im, -e);
    return fma((double)e, qmc_mc[0], 0.5 * log(fma(a, a, b * b)));
}
__device__ __forceinline__ void qmc_clog(double re, double im, double& lre, double& lim) {
    const double m2 = fma(re, re, im * im);
    const int hi = __double2hiint(m2);
    if ((unsigned)(hi - 0x01000000) >= 0x7e000000u - 0x01000000u) lre = qmc_clog_re_scaled(re, im);   // m2 outside [7e-304, 8e298)
    else lre = 0.5 * qmc_log(m2);
    lim = qmc_atan2(im, re);
}
__device__ __forceinline__ void qmc_cexp(double are, double aim, double& ere, double& eim) {
    const double e = qmc_exp(are);
    double s, c;
    qmc_sincos(aim, s, c);
    ere = e * c;
    eim = e * s;
}
#endif  // QMC_HAVE_CPLX

#endif  // QMC_MATH_CUH_
