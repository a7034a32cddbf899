// =====================================================================================
// qmc_device.cuh -- hand-written sm_100a device code of the QMC hot path.
//
// This text is compiled twice: by nvcc into libqmc.so (the lattice debug kernel, so that the
// bit-exact coordinate check runs these very functions) and by NVRTC at qmc_plan time, where
// the generated per-sector integrand structs (qmc_codegen.cpp) are appended and the
// persistent kernel qmc_eval_kernel below is instantiated over them.  It therefore uses no
// header: only CUDA built-ins.  qmc_job_dev.h is prepended to it.
//
// Steps:
//   a1  qmc_lattice_start / qmc_lattice_next   r = (k z_i) mod n in exact 64-bit integers
//                                              (PAPER.md:102 rank-1 lattice; north_star (1))
//   a2  qmc_point                              shift + frac, Korobov-3 / baker transform and
//                                              weight (north_star (2))
//   a3  S::eval (generated)                    the sector integrand (north_star (3))
//   a4  qmc_block_reduce                       warp-shuffle + double-double block sum, one
//                                              (hi, lo) pair per tile and component
//                                              (north_star (4))
//   a6  qmc_eval_kernel                        persistent CTAs pulling (job, shift, k-range)
//                                              tiles from an atomic counter (north_star (6))
// =====================================================================================
#ifndef QMC_DEVICE_CUH_
#define QMC_DEVICE_CUH_

typedef unsigned int u32;
typedef unsigned long long u64;

#ifndef QMC_THREADS
#define QMC_THREADS 256
#endif
#ifndef QMC_MIN_CTAS
#define QMC_MIN_CTAS 1
#endif
#ifndef QMC_JOUT
#define QMC_JOUT 3
#endif
#define QMC_NCOMP (3 * QMC_JOUT)       // (Re S, Im S, A) per order slot
#define QMC_WARPS (QMC_THREADS / 32)

#define QMC_TR_NONE 0
#define QMC_TR_KOROBOV3 1
#define QMC_TR_BAKER 2
// internal: Korobov r = 3 evaluated about the centre, u = t - 1/2 (see QmcTransform<QMC_TR_KOROBOV3C>); chosen per
// dimension by the mask S::CENTRED of the generated sector
#define QMC_TR_KOROBOV3C 3

// ------------------------------------------------------------------------------------ a1
// (k z) mod n for k, z, n < 2^32: the 64-bit product is exact; Barrett reduction with
// barrett = floor((2^64-1)/n) under-estimates the quotient by at most 2.
__device__ __forceinline__ u32 qmc_lattice_start(u64 k, u32 z, u32 n, u64 barrett) {
    const u64 a = k * (u64)z;
    const u64 q = __umul64hi(a, barrett);
    u64 r = a - q * (u64)n;
    if (r >= (u64)n) r -= (u64)n;
    if (r >= (u64)n) r -= (u64)n;
    return (u32)r;
}
// r(k + stride) from r(k): step = (stride z) mod n, n_minus_step = n - step (no overflow in u32)
__device__ __forceinline__ u32 qmc_lattice_next(u32 r, u32 step, u32 n_minus_step) {
    return (r >= n_minus_step) ? r - n_minus_step : r + step;
}

// The same two steps for lattices with 2^32 <= n < 2^53 (the paper reaches n = 4.3e9 and ~7e10,
// PAPER.md:279, 300): k z no longer fits 64 bits, so the start is a double-and-add modular product
// over the bits of k (2 r and r + z stay below 2^54, no overflow), run once per thread and tile;
// the per-point increment is the same compare / select / add on 64-bit integers.
__device__ __forceinline__ u64 qmc_lattice_start(u64 k, u64 z, u64 n, u64 /*barrett unused*/) {
    u64 r = 0;
    const u64 zz = z % n;
    for (int b = 63 - __clzll((long long)(k | 1ull)); b >= 0; --b) {
        r += r;
        if (r >= n) r -= n;
        if ((k >> b) & 1ull) { r += zz; if (r >= n) r -= n; }
    }
    return r;
}
__device__ __forceinline__ u64 qmc_lattice_next(u64 r, u64 step, u64 n_minus_step) {
    return (r >= n_minus_step) ? r - n_minus_step : r + step;
}

// index type of the evaluation kernels: 32-bit unless the plan was made with wide_lattice
#ifdef QMC_WIDE
typedef u64 qmc_idx;
#else
typedef u32 qmc_idx;
#endif

// ------------------------------------------------------------------------------------ a2
// t = frac(r/n + delta) without a wrap in the loop: delta = (a + f)/n with a = floor(delta n) an
// integer and f in [0, 1), so   frac((r + a + f)/n) = ((r + a) mod n + f)/n.   The integer part a
// joins the lattice index (exact modular arithmetic, one modular add per tile and thread), and
// the loop takes t = fma(r', 1/n, c) with r' = (r + a) mod n and c = f/n in [0, 1/n): no compare,
// no select, and t < 1 by construction.  delta n is split exactly (fma residual) so that c
// carries the full precision of delta.
template <class IDX>
__device__ __forceinline__ void qmc_shift_split(IDX n, double delta, IDX& a_out, double& c_out) {
    const double nd = (double)n;
    const double p = delta * nd;
    const double e = fma(delta, nd, -p);      // delta n = p + e exactly
    double a = floor(p);
    double f = (p - a) + e;                   // p - a is exact
    if (f < 0.0) { a -= 1.0; f += 1.0; }
    else if (f >= 1.0) { a += 1.0; f -= 1.0; }
    if (f >= 1.0) f = 0x1.fffffffffffffp-1;   // f + 1 rounded up to 1
    if (a < 0.0) { a = 0.0; f = 0.0; }
    if (a >= nd) { a = nd - 1.0; f = 0x1.fffffffffffffp-1; }
    a_out = (IDX)a;
    c_out = f / nd;
}

// compile-time helpers of the general Korobov transform
__device__ __forceinline__ constexpr double qmc_cfact(int n) { return n <= 1 ? 1.0 : (double)n * qmc_cfact(n - 1); }
__device__ __forceinline__ constexpr double qmc_cbinom(int n, int k) { return qmc_cfact(n) / (qmc_cfact(k) * qmc_cfact(n - k)); }
template <int E>
__device__ __forceinline__ double qmc_ipow(double x) {   // x^E, E >= 0, by squaring, unrolled at compile time
    if constexpr (E == 0) return 1.0;
    else if constexpr (E == 1) return x;
    else if constexpr (E % 2 == 0) { const double h = qmc_ipow<E / 2>(x); return h * h; }
    else return x * qmc_ipow<E - 1>(x);
}

// Primary template: the general Korobov transform, TR = 100 + 10 r0 + r1 with 1 <= r0, r1 <= 6 (QMC_TRANSFORM_KOROBOV
// in qmc.h; "korobov3" is the default of this family):
//   omega(t) = t^r0 (1 - t)^r1 / B(r0+1, r1+1),   phi(t) = t^(r0+1) sum_{k=0}^{r1} a_k t^k,
//   a_k = (-1)^k binom(r1, k) / ((r0 + 1 + k) B),   1/B = (r0 + r1 + 1)! / (r0! r1!).
// P accumulates prod t_i (1 - t_i) for r0 = r1 (one multiply per dimension); for r0 != r1 the two products are kept
// apart in (P, P1) by apply2 / weight2.
template <int TR>
struct QmcTransform {
    static constexpr int R0 = (TR - 100) / 10, R1 = (TR - 100) % 10;
    static_assert(TR >= 111 && R0 >= 1 && R0 <= 6 && R1 >= 1 && R1 <= 6, "transform code");
    static constexpr bool SYM = (R0 == R1);
    static constexpr double INVB = qmc_cfact(R0 + R1 + 1) / (qmc_cfact(R0) * qmc_cfact(R1));
    template <int K>
    static __device__ __forceinline__ constexpr double coef() {
        return ((K % 2) ? -1.0 : 1.0) * qmc_cbinom(R1, K) * INVB / (double)(R0 + 1 + K);
    }
    template <int K>
    static __device__ __forceinline__ double horner(double t) {      // a_K + t (a_{K+1} + ...)
        if constexpr (K == R1) return coef<K>();
        else return fma(t, horner<K + 1>(t), coef<K>());
    }
    static __device__ __forceinline__ void apply2(double t, double& x, double& P, double& P1) {
        x = qmc_ipow<R0 + 1>(t) * horner<0>(t);
        if constexpr (SYM) P *= fma(-t, t, t);
        else { P *= t; P1 *= 1.0 - t; }
    }
    static __device__ __forceinline__ double weight2(double P, double P1, double scale) {   // scale = (1/B)^d
        if constexpr (SYM) return qmc_ipow<R0>(P) * scale;
        else return (qmc_ipow<R0>(P) * qmc_ipow<R1>(P1)) * scale;
    }
};
template <>
struct QmcTransform<QMC_TR_NONE> {
    static __device__ __forceinline__ void apply(double t, double& x, double& P) { x = t; }
    static __device__ __forceinline__ double weight(double P, double scale) { return 1.0; }
};
// Korobov r = 3: phi(t) = t^4 (35 - 84 t + 70 t^2 - 20 t^3), phi'(t) = 140 t^3 (1-t)^3.
// The product of the weights is 140^d (prod_i t_i (1 - t_i))^3: one multiply per dimension.
template <>
struct QmcTransform<QMC_TR_KOROBOV3> {
    static __device__ __forceinline__ void apply(double t, double& x, double& P) {
        const double t2 = t * t;
        const double a = fma(-84.0, t, 35.0);
        const double b = fma(-20.0, t, 70.0);
        const double poly = fma(b, t2, a);
        x = (t2 * t2) * poly;
        P *= fma(-t, t, t);   // t (1 - t) rounded once: no cancellation as t -> 1
    }
    static __device__ __forceinline__ double weight(double P, double scale) { return (P * P) * (P * scale); }
};
// The same map about the centre of the interval.  With u = t - 1/2 and w = u^2,
//     phi = 1/2 + u (35/16 - 35/4 w + 21 w^2 - 20 w^3)      (phi - 1/2 is odd in u: integrate 140 (1/4 - v^2)^3),
//     t (1 - t) = 1/4 - w,
// i.e. 8 FP64 instructions per dimension instead of 9 (the kernels are bound by their FP64 instruction count), and the
// shift offset absorbs the -1/2 so that u itself comes out of the one fma of qmc_point.  The price: x -> 0 is reached
// by cancellation, so x carries an ABSOLUTE error of ~1e-16 instead of a relative one.  That is harmless exactly when
// d log g / dx_i is bounded up to the prefactor x_i^a_i (then the error of W g is ~1e-16 W |g| like every other
// rounding).  The generator proves that for the toy class and for U, F with non-negative coefficients and a positive
// constant term (S::REGULAR), and there only for the dimensions WITHOUT a prefactor x_i^a_i (bit i of S::CENTRED): x_i
// then enters g through U and F alone, whose logarithmic derivatives are bounded, so even a sum that consists of a
// single point next to the boundary (n = 1) keeps its relative accuracy.  Every other dimension keeps the form above,
// whose x is relatively accurate down to 0.
template <>
struct QmcTransform<QMC_TR_KOROBOV3C> {
    static __device__ __forceinline__ void apply(double u, double& x, double& P) {
        const double w = u * u;
        double q = fma(-20.0, w, 21.0);
        q = fma(q, w, -8.75);
        q = fma(q, w, 2.1875);
        x = fma(u, q, 0.5);
        P *= fma(-u, u, 0.25);
    }
    static __device__ __forceinline__ double weight(double P, double scale) { return (P * P) * (P * scale); }
};
// baker (tent) map: x = 1 - |2 t - 1|, weight 1
template <>
struct QmcTransform<QMC_TR_BAKER> {
    static __device__ __forceinline__ void apply(double t, double& x, double& P) {
        x = 1.0 - fabs(fma(2.0, t, -1.0));
    }
    static __device__ __forceinline__ double weight(double P, double scale) { return 1.0; }
};

// The kernels are bound by the FP64 pipe, so the exact u32 -> double conversion goes to the conversion unit
// (I2F.F64.U32), not through a 2^52 + r DADD.
__device__ __forceinline__ double qmc_index_to_double(u32 r) { return (double)r; }
__device__ __forceinline__ double qmc_index_to_double(u64 r) { return (double)r; }   // exact below 2^53

// per-dimension choice of the Korobov r = 3 form: bit i of S::CENTRED set = dimension i uses the centred form
template <int TR>
__device__ __forceinline__ constexpr int qmc_tr_dim(unsigned centred_mask, int i) {
    return (TR == QMC_TR_KOROBOV3 && ((centred_mask >> i) & 1u)) ? QMC_TR_KOROBOV3C : TR;
}
// the additive constant of t = fma(r', 1/n, c): f/n, minus 1/2 for a dimension in the centred Korobov form
template <int TR>
__device__ __forceinline__ double qmc_shift_offset(double shift_c, unsigned centred_mask, int i) {
    return qmc_tr_dim<TR>(centred_mask, i) == QMC_TR_KOROBOV3C ? shift_c - 0.5 : shift_c;
}

// uniform interface over all transforms: the named ones use one running product
template <int TR>
__device__ __forceinline__ void qmc_tr_apply(double t, double& x, double& P, double& P1) {
    if constexpr (TR >= 100) QmcTransform<TR>::apply2(t, x, P, P1);
    else QmcTransform<TR>::apply(t, x, P);
}
template <int TR>
__device__ __forceinline__ double qmc_tr_weight(double P, double P1, double scale) {
    if constexpr (TR >= 100) return QmcTransform<TR>::weight2(P, P1, scale);
    else return QmcTransform<TR>::weight(P, scale);
}
// transforms whose weight can vanish (a point of weight exactly 0 contributes 0, reading Q4)
__device__ __forceinline__ constexpr bool qmc_is_korobov(int tr) { return tr == QMC_TR_KOROBOV3 || tr >= 100; }

// r: shifted lattice indices (r + a) mod n;  c: the fractional shift offsets f/n (qmc_shift_offset)
template <int D, int TR, unsigned CM, class IDX>
__device__ __forceinline__ void qmc_point(const IDX (&r)[D], const double (&c)[D], double inv_n, double wscale,
                                          double (&x)[D], double& W, double* t_out) {
    double P = 1.0, P1 = 1.0;
#pragma unroll
    for (int i = 0; i < D; ++i) {
        const double t = fma(qmc_index_to_double(r[i]), inv_n, c[i]);    // u = t - 1/2 in a centred dimension
        if (((CM >> i) & 1u) && TR == QMC_TR_KOROBOV3) {                 // resolved at compile time after unrolling
            if (t_out) t_out[i] = t + 0.5;
            qmc_tr_apply<QMC_TR_KOROBOV3C>(t, x[i], P, P1);
        } else {
            if (t_out) t_out[i] = t;
            qmc_tr_apply<TR>(t, x[i], P, P1);
        }
    }
    W = qmc_tr_weight<TR>(P, P1, wscale);
}

// modulus of a complex term for the sum of |W g| (the elementary functions are in qmc_math.cuh)
#ifndef QMC_SQRT
#define QMC_SQRT(x) sqrt(x)
#endif
__device__ __forceinline__ double qmc_cabs(double re, double im) { return QMC_SQRT(fma(re, re, im * im)); }

// ------------------------------------------------------------------------------------ a4
// Double-double sum over the block of N per-thread values: xor-butterfly of TwoSum inside each
// warp, then across the warps through shared memory.  Result (hi, lo) valid in thread 0.
__device__ __forceinline__ void qmc_two_sum_acc(double& hi, double& lo, double oh, double ol) {
    const double s = hi + oh;
    const double bb = s - hi;
    const double e = (hi - (s - bb)) + (oh - bb);
    hi = s;
    lo = (lo + ol) + e;
}

template <int N>
__device__ __forceinline__ void qmc_block_reduce(double (&hi)[N], double (&lo)[N], double* red /*QMC_WARPS*N*2*/) {
    const u32 lane = threadIdx.x & 31u, warp = threadIdx.x >> 5;
#pragma unroll
    for (int c = 0; c < N; ++c) {
#pragma unroll
        for (int off = 16; off >= 1; off >>= 1) {
            const double oh = __shfl_xor_sync(0xffffffffu, hi[c], off);
            const double ol = __shfl_xor_sync(0xffffffffu, lo[c], off);
            qmc_two_sum_acc(hi[c], lo[c], oh, ol);
        }
        if (lane == 0) {
            red[(warp * N + c) * 2 + 0] = hi[c];
            red[(warp * N + c) * 2 + 1] = lo[c];
        }
    }
    __syncthreads();
    if (warp == 0) {
#pragma unroll
        for (int c = 0; c < N; ++c) {
            double h = lane < QMC_WARPS ? red[(lane * N + c) * 2 + 0] : 0.0;
            double l = lane < QMC_WARPS ? red[(lane * N + c) * 2 + 1] : 0.0;
#pragma unroll
            for (int off = 16; off >= 1; off >>= 1) {
                const double oh = __shfl_xor_sync(0xffffffffu, h, off);
                const double ol = __shfl_xor_sync(0xffffffffu, l, off);
                qmc_two_sum_acc(h, l, oh, ol);
            }
            hi[c] = h;
            lo[c] = l;
        }
    }
}

// ------------------------------------------------------------------------------------ tiles
// Per-tile context staged in shared memory by warp 0 ("stages per-block z / Delta in shared
// memory", north_star (1)).
struct QmcTileCtx {
    u64 n, k0, k1, barrett;
    double inv_n;
    u32 sector_case, diag_slot;
    qmc_idx z[QMC_DEV_MAX_DIM], step[QMC_DEV_MAX_DIM], shift_a[QMC_DEV_MAX_DIM];   // a = floor(delta n)
    double shift_c[QMC_DEV_MAX_DIM];                                            // frac(delta n) / n
};

__device__ __forceinline__ void qmc_setup_tile(const QmcLaunchArgs& a, u32 tile, QmcTileCtx& ctx) {
    // warp 0: every lane finds the job (largest j with tile_base <= tile), lanes < 8 fill one dimension
    const u32 lane = threadIdx.x;
    int lo = 0, hi = a.n_jobs - 1;
    while (lo < hi) {
        const int mid = (lo + hi + 1) >> 1;
        if (a.jobs[mid].tile_base <= tile) lo = mid; else hi = mid - 1;
    }
    const QmcJobDev jb = a.jobs[lo];
    const u32 local = tile - jb.tile_base;
    const u32 shift = local / jb.tiles_per_shift;
    const u32 kt = local - shift * jb.tiles_per_shift;
    const u64 k0 = jb.k_begin + (u64)kt * jb.tile_points;
    u64 k1 = k0 + jb.tile_points;
    if (k1 > jb.k_end) k1 = jb.k_end;
    if (lane == 0) {
        ctx.n = jb.n; ctx.sector_case = jb.sector_case; ctx.k0 = k0; ctx.k1 = k1;
        ctx.diag_slot = jb.diag_slot; ctx.barrett = jb.barrett; ctx.inv_n = jb.inv_n;
    }
    if (lane < QMC_DEV_MAX_DIM) {
        u32 zrow = jb.z_row;
        if (jb.sel_index >= 0) zrow += (u32)a.selected[jb.sel_index];
        const qmc_idx z = (qmc_idx)a.z_table[(u64)zrow * QMC_DEV_MAX_DIM + lane];
        const double d = a.shifts[((u64)jb.shift_row + shift) * QMC_DEV_MAX_DIM + lane];
        ctx.z[lane] = z;
        ctx.step[lane] = qmc_lattice_start((u64)QMC_THREADS, z, (qmc_idx)jb.n, jb.barrett);
        qmc_shift_split((qmc_idx)jb.n, d, ctx.shift_a[lane], ctx.shift_c[lane]);
    }
}

// Adds one evaluated point to the thread's sums: S += W g_j, A += |W g_j| per order.
template <class S, int NA, int NG>
__device__ __forceinline__ void qmc_accumulate(double W, const double (&g)[NG], int sf, double (&acc)[NA],
                                               u32& zero_w, u32& sign_fail) {
    constexpr int J = S::J;
    if (qmc_is_korobov(S::TR)) {
        // a point of weight exactly 0 contributes 0 whatever the integrand does there
        // W >= 0 is a product of non-negative factors, so W == 0.0 iff all its bits are zero: an integer test,
        // off the FP64 pipe
        const bool zw = ((__double2hiint(W) | __double2loint(W)) == 0);
        zero_w += zw ? 1u : 0u;
        sign_fail += (!zw && sf) ? 1u : 0u;
#pragma unroll
        for (int j = 0; j < J; ++j) {
            if (S::CPLX) {
                const double wr = zw ? 0.0 : W * g[2 * j], wi = zw ? 0.0 : W * g[2 * j + 1];
                acc[3 * j] += wr; acc[3 * j + 1] += wi; acc[3 * j + 2] += qmc_cabs(wr, wi);
            } else {
                // a regular integrand is finite everywhere, so W g = 0 without a select when W = 0
                const double wg = (S::REGULAR || !zw) ? W * g[j] : 0.0;
                acc[2 * j] += wg; acc[2 * j + 1] += fabs(wg);
            }
        }
    } else {
        sign_fail += sf ? 1u : 0u;
#pragma unroll
        for (int j = 0; j < J; ++j) {
            if (S::CPLX) {
                acc[3 * j] += g[2 * j]; acc[3 * j + 1] += g[2 * j + 1];
                acc[3 * j + 2] += qmc_cabs(g[2 * j], g[2 * j + 1]);
            } else {
                acc[2 * j] += g[j]; acc[2 * j + 1] += fabs(g[j]);
            }
        }
    }
}

// One tile of one sector: every thread walks k = k0 + tid, k0 + tid + T, ... < k1 with the
// modular increment, accumulates W g_j per order, then the block sum goes to the tile's slot.
// QMC_PPT = P > 1 evaluates P consecutive points of the thread per loop iteration: P independent
// instruction streams for the FP64 pipe (at 4 warps per scheduler a single evaluation's dependency
// chains leave the pipe idle a third of the time); the order of the thread's additions is unchanged.
#ifndef QMC_PPT
#define QMC_PPT 1
#endif
// a4, thread level.  A thread adds its points in plain FP64, so the chain is kept short by construction: the kernel
// walks a tile in chunks of QMC_CHUNK points per thread (QMC_CHUNK x QMC_THREADS consecutive lattice indices), and
// after every chunk the block's double-double sum is folded into the tile's (hi, lo) pairs in shared memory.  The
// rounding error of a per-shift sum is therefore bounded by (QMC_CHUNK + 1) 2^-53 sum|W g| = 1.1e-13 A however long
// the tile is (north_star: 1e-11 A); everything above the thread level is double-double (2^-104).  The chunk costs one
// block reduction (~100-500 instructions per thread) per 1020 evaluations (150-1500 instructions each).
#define QMC_CHUNK 1020u
// One chunk [ks0, ks1) of the tile staged in ctx; tile_acc: QMC_NCOMP x (hi, lo) in shared memory, owned by thread 0.
template <class S>
__device__ __forceinline__ void qmc_tile_body(const QmcTileCtx& ctx, u64 ks0, u64 ks1, double* tile_acc,
                                              double* red, u32* diag_sh) {
    constexpr int D = S::D;
    constexpr int J = S::J;
    constexpr int NA = S::CPLX ? 3 * J : 2 * J;
    constexpr int NG = S::CPLX ? 2 * J : J;
    const u32 tid = threadIdx.x;
    const qmc_idx n = (qmc_idx)ctx.n;
    const double inv_n = ctx.inv_n;
    qmc_idx r[D], st[D], cm[D];
    double sc[D];
    const u64 first = ks0 + tid;
    const u32 cnt = first < ks1 ? (u32)((ks1 - first + (QMC_THREADS - 1)) / QMC_THREADS) : 0u;
#pragma unroll
    for (int i = 0; i < D; ++i) {
        st[i] = ctx.step[i];
        cm[i] = n - st[i];
        sc[i] = qmc_shift_offset<S::TR>(ctx.shift_c[i], S::CENTRED, i);
        const qmc_idx a = ctx.shift_a[i];
        r[i] = qmc_lattice_next(qmc_lattice_start(first, ctx.z[i], n, ctx.barrett), a, (qmc_idx)(n - a));
    }
    double acc[NA];
#pragma unroll
    for (int c = 0; c < NA; ++c) acc[c] = 0.0;
    u32 zero_w = 0, sign_fail = 0;

    u32 it = 0;
#if QMC_PPT > 1
#pragma unroll 1
    for (; it + QMC_PPT <= cnt; it += QMC_PPT) {
        double xs[QMC_PPT][D], Ws[QMC_PPT], gs[QMC_PPT][NG];
        int sfs[QMC_PPT];
#pragma unroll
        for (int p = 0; p < QMC_PPT; ++p) {
            qmc_point<D, S::TR, S::CENTRED, qmc_idx>(r, sc, inv_n, S::wscale(), xs[p], Ws[p], nullptr);
#pragma unroll
            for (int i = 0; i < D; ++i) r[i] = qmc_lattice_next(r[i], st[i], cm[i]);
        }
#pragma unroll
        for (int p = 0; p < QMC_PPT; ++p) sfs[p] = S::eval(xs[p], gs[p]);
        if constexpr (S::CPLX) {   // bit 1: an argument left the fast range of the unguarded functions (never seen in practice)
#pragma unroll
            for (int p = 0; p < QMC_PPT; ++p) if (sfs[p] & 2) { sfs[p] = S::eval_checked(xs[p], gs[p]); atomicAdd(&diag_sh[2], 1u); }
        }
#pragma unroll
        for (int p = 0; p < QMC_PPT; ++p) qmc_accumulate<S, NA, NG>(Ws[p], gs[p], sfs[p], acc, zero_w, sign_fail);
    }
#endif
#pragma unroll 1
    for (; it < cnt; ++it) {
        double x[D], W;
        qmc_point<D, S::TR, S::CENTRED, qmc_idx>(r, sc, inv_n, S::wscale(), x, W, nullptr);
#pragma unroll
        for (int i = 0; i < D; ++i) r[i] = qmc_lattice_next(r[i], st[i], cm[i]);
        double g[NG];
        int sf = S::eval(x, g);
        if constexpr (S::CPLX) { if (sf & 2) { sf = S::eval_checked(x, g); atomicAdd(&diag_sh[2], 1u); } }
        qmc_accumulate<S, NA, NG>(W, g, sf, acc, zero_w, sign_fail);
    }

    double lo[NA];
#pragma unroll
    for (int c = 0; c < NA; ++c) lo[c] = 0.0;
    qmc_block_reduce<NA>(acc, lo, red);
    // diagnostics: integer counters, exact whatever the order
    const u32 zw_w = __reduce_add_sync(0xffffffffu, zero_w);
    const u32 sf_w = __reduce_add_sync(0xffffffffu, sign_fail);
    if ((tid & 31u) == 0 && (zw_w | sf_w)) {
        if (zw_w) atomicAdd(&diag_sh[0], zw_w);
        if (sf_w) atomicAdd(&diag_sh[1], sf_w);
    }
    if (tid == 0) {
#pragma unroll
        for (int j = 0; j < J; ++j) {
            if (S::CPLX) {
#pragma unroll
                for (int c = 0; c < 3; ++c)
                    qmc_two_sum_acc(tile_acc[(3 * j + c) * 2], tile_acc[(3 * j + c) * 2 + 1], acc[3 * j + c], lo[3 * j + c]);
            } else {
                qmc_two_sum_acc(tile_acc[(3 * j + 0) * 2], tile_acc[(3 * j + 0) * 2 + 1], acc[2 * j], lo[2 * j]);
                qmc_two_sum_acc(tile_acc[(3 * j + 2) * 2], tile_acc[(3 * j + 2) * 2 + 1], acc[2 * j + 1], lo[2 * j + 1]);
            }
        }
    }
}

// single lattice points through the same a1-a3 code (per-point parity)
template <class S>
__device__ __forceinline__ void qmc_debug_point(qmc_idx n, u64 barrett, double inv_n, const u64* z, const double* delta,
                                                u64 k, double* out /* 2*8 + 1 + 2*QMC_JOUT */) {
    constexpr int D = S::D;
    constexpr int J = S::J;
    qmc_idx r[D];
    double sc[D], x[D], t[D], W;
#pragma unroll
    for (int i = 0; i < D; ++i) {
        qmc_idx a;
        qmc_shift_split(n, delta[i], a, sc[i]);
        sc[i] = qmc_shift_offset<S::TR>(sc[i], S::CENTRED, i);
        r[i] = qmc_lattice_next(qmc_lattice_start(k, (qmc_idx)z[i], n, barrett), a, (qmc_idx)(n - a));
    }
    qmc_point<D, S::TR, S::CENTRED, qmc_idx>(r, sc, inv_n, S::wscale(), x, W, t);
    double g[S::CPLX ? 2 * J : J];
    const int sf_dbg = S::eval(x, g);
    if constexpr (S::CPLX) { if (sf_dbg & 2) S::eval_checked(x, g); }
    for (int i = 0; i < 2 * QMC_DEV_MAX_DIM + 1 + 2 * QMC_JOUT; ++i) out[i] = 0.0;
#pragma unroll
    for (int i = 0; i < D; ++i) { out[i] = t[i]; out[QMC_DEV_MAX_DIM + i] = x[i]; }
    out[2 * QMC_DEV_MAX_DIM] = W;
    const bool zw = qmc_is_korobov(S::TR) && ((__double2hiint(W) | __double2loint(W)) == 0);
#pragma unroll
    for (int j = 0; j < J; ++j) {
        const double gr = S::CPLX ? g[2 * j] : g[j], gi = S::CPLX ? g[2 * j + 1] : 0.0;
        out[2 * QMC_DEV_MAX_DIM + 1 + 2 * j] = zw ? 0.0 : W * gr;
        out[2 * QMC_DEV_MAX_DIM + 2 + 2 * j] = zw ? 0.0 : W * gi;
    }
}

#endif  // QMC_DEVICE_CUH_
