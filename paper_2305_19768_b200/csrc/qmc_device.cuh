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

// exact u32 -> double without the conversion pipe: 2^52 + r has r in its low mantissa bits
__device__ __forceinline__ double qmc_u32_to_double(u32 r) {
    return __hiloint2double(0x43300000, (int)r) - 4503599627370496.0;
}

// ------------------------------------------------------------------------------------ a2
// t = frac(r/n + delta) is taken as fma(r, 1/n, delta) for r < thr and fma(r, 1/n, delta - 1)
// for r >= thr, where thr is the smallest r whose wrapped value is >= 0; t lies in [0, 1].
// The integer comparison keeps the wrap off the FP64 pipe.
__device__ __forceinline__ u32 qmc_wrap_threshold(u32 n, double inv_n, double delta) {
    const double dm1 = delta - 1.0;
    double est = ceil((1.0 - delta) * (double)n);
    u32 thr = est <= 0.0 ? 0u : (est >= (double)n ? n : (u32)est);
    while (thr > 0u && fma((double)(thr - 1u), inv_n, dm1) >= 0.0) --thr;
    while (thr < n && fma((double)thr, inv_n, dm1) < 0.0) ++thr;
    return thr;
}

template <int TR>
struct QmcTransform;
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
        P *= (t - t2);
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

template <int D, int TR>
__device__ __forceinline__ void qmc_point(const u32 (&r)[D], const u32 (&thr)[D], const double (&dl)[D],
                                          double inv_n, double wscale, double (&x)[D], double& W,
                                          double* t_out) {
    double P = 1.0;
#pragma unroll
    for (int i = 0; i < D; ++i) {
        const double rd = qmc_u32_to_double(r[i]);
        const double t = fma(rd, inv_n, (r[i] >= thr[i]) ? dl[i] - 1.0 : dl[i]);
        if (t_out) t_out[i] = t;
        QmcTransform<TR>::apply(t, x[i], P);
    }
    W = QmcTransform<TR>::weight(P, wscale);
}

// ------------------------------------------------------------------------------------ math
// FP64 elementary functions of the integrand.  Arguments are finite; U and F are positive in
// the real class.  QMC_LIBDEVICE_MATH selects the CUDA library versions (A/B measurement).
__device__ __forceinline__ double qmc_log(double x) { return log(x); }
__device__ __forceinline__ double qmc_exp(double x) { return exp(x); }
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
__device__ __forceinline__ double qmc_cabs(double re, double im) { return sqrt(fma(re, re, im * im)); }

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
    u32 n, sector_case, k0, k1, diag_slot, pad_;
    u64 barrett;
    double inv_n;
    u32 z[QMC_DEV_MAX_DIM], step[QMC_DEV_MAX_DIM], thr[QMC_DEV_MAX_DIM];
    double delta[QMC_DEV_MAX_DIM];
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
    const u64 k0 = (u64)kt * jb.tile_points;
    u64 k1 = k0 + jb.tile_points;
    if (k1 > jb.n) k1 = jb.n;
    if (lane == 0) {
        ctx.n = jb.n; ctx.sector_case = jb.sector_case; ctx.k0 = (u32)k0; ctx.k1 = (u32)k1;
        ctx.diag_slot = jb.diag_slot; ctx.barrett = jb.barrett; ctx.inv_n = jb.inv_n;
    }
    if (lane < QMC_DEV_MAX_DIM) {
        u32 zrow = jb.z_row;
        if (jb.sel_index >= 0) zrow += (u32)a.selected[jb.sel_index];
        const u32 z = a.z_table[(u64)zrow * QMC_DEV_MAX_DIM + lane];
        const double d = a.shifts[((u64)jb.shift_row + shift) * QMC_DEV_MAX_DIM + lane];
        ctx.z[lane] = z;
        ctx.step[lane] = qmc_lattice_start((u64)QMC_THREADS, z, jb.n, jb.barrett);
        ctx.thr[lane] = qmc_wrap_threshold(jb.n, jb.inv_n, d);
        ctx.delta[lane] = d;
    }
}

// One tile of one sector: every thread walks k = k0 + tid, k0 + tid + T, ... < k1 with the
// modular increment, accumulates W g_j per order, then the block sum goes to the tile's slot.
template <class S>
__device__ __forceinline__ void qmc_tile_body(const QmcTileCtx& ctx, const QmcLaunchArgs& a, u32 tile,
                                              double* red, u32* diag_sh) {
    constexpr int D = S::D;
    constexpr int J = S::J;
    constexpr int NA = S::CPLX ? 3 * J : 2 * J;
    const u32 tid = threadIdx.x;
    const u32 n = ctx.n;
    const double inv_n = ctx.inv_n;
    u32 r[D], st[D], cm[D], thr[D];
    double dl[D];
    const u64 first = (u64)ctx.k0 + tid;
    const u32 cnt = first < (u64)ctx.k1 ? (u32)(((u64)ctx.k1 - first + (QMC_THREADS - 1)) / QMC_THREADS) : 0u;
#pragma unroll
    for (int i = 0; i < D; ++i) {
        st[i] = ctx.step[i];
        cm[i] = n - st[i];
        thr[i] = ctx.thr[i];
        dl[i] = ctx.delta[i];
        r[i] = qmc_lattice_start(first, ctx.z[i], n, ctx.barrett);
    }
    double acc[NA];
#pragma unroll
    for (int c = 0; c < NA; ++c) acc[c] = 0.0;
    u32 zero_w = 0, sign_fail = 0;

#pragma unroll 1
    for (u32 it = 0; it < cnt; ++it) {
        double x[D], W;
        qmc_point<D, S::TR>(r, thr, dl, inv_n, S::wscale(), x, W, nullptr);
#pragma unroll
        for (int i = 0; i < D; ++i) r[i] = qmc_lattice_next(r[i], st[i], cm[i]);
        double g[S::CPLX ? 2 * J : J];
        const int sf = S::eval(x, g);
        if (S::TR == QMC_TR_KOROBOV3) {
            // a point of weight exactly 0 contributes 0 whatever the integrand does there
            const bool zw = (W == 0.0);
            zero_w += zw ? 1u : 0u;
            sign_fail += (!zw && sf) ? 1u : 0u;
#pragma unroll
            for (int j = 0; j < J; ++j) {
                if (S::CPLX) {
                    const double wr = zw ? 0.0 : W * g[2 * j], wi = zw ? 0.0 : W * g[2 * j + 1];
                    acc[3 * j] += wr; acc[3 * j + 1] += wi; acc[3 * j + 2] += qmc_cabs(wr, wi);
                } else {
                    const double wg = zw ? 0.0 : W * g[j];
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
        double* out = a.partials + (u64)tile * (QMC_NCOMP * 2);
#pragma unroll
        for (int c = 0; c < QMC_NCOMP * 2; ++c) out[c] = 0.0;
#pragma unroll
        for (int j = 0; j < J; ++j) {
            if (S::CPLX) {
#pragma unroll
                for (int c = 0; c < 3; ++c) {
                    out[(3 * j + c) * 2 + 0] = acc[3 * j + c];
                    out[(3 * j + c) * 2 + 1] = lo[3 * j + c];
                }
            } else {
                out[(3 * j + 0) * 2 + 0] = acc[2 * j];     out[(3 * j + 0) * 2 + 1] = lo[2 * j];
                out[(3 * j + 2) * 2 + 0] = acc[2 * j + 1]; out[(3 * j + 2) * 2 + 1] = lo[2 * j + 1];
            }
        }
    }
}

// single lattice points through the same a1-a3 code (per-point parity)
template <class S>
__device__ __forceinline__ void qmc_debug_point(u32 n, u64 barrett, double inv_n, const u32* z, const double* delta,
                                                u64 k, double* out /* 2*8 + 1 + 2*QMC_JOUT */) {
    constexpr int D = S::D;
    constexpr int J = S::J;
    u32 r[D], thr[D];
    double dl[D], x[D], t[D], W;
#pragma unroll
    for (int i = 0; i < D; ++i) {
        r[i] = qmc_lattice_start(k, z[i], n, barrett);
        thr[i] = qmc_wrap_threshold(n, inv_n, delta[i]);
        dl[i] = delta[i];
    }
    qmc_point<D, S::TR>(r, thr, dl, inv_n, S::wscale(), x, W, t);
    double g[S::CPLX ? 2 * J : J];
    S::eval(x, g);
    for (int i = 0; i < 2 * QMC_DEV_MAX_DIM + 1 + 2 * QMC_JOUT; ++i) out[i] = 0.0;
#pragma unroll
    for (int i = 0; i < D; ++i) { out[i] = t[i]; out[QMC_DEV_MAX_DIM + i] = x[i]; }
    out[2 * QMC_DEV_MAX_DIM] = W;
    const bool zw = (S::TR == QMC_TR_KOROBOV3) && (W == 0.0);
#pragma unroll
    for (int j = 0; j < J; ++j) {
        const double gr = S::CPLX ? g[2 * j] : g[j], gi = S::CPLX ? g[2 * j + 1] : 0.0;
        out[2 * QMC_DEV_MAX_DIM + 1 + 2 * j] = zw ? 0.0 : W * gr;
        out[2 * QMC_DEV_MAX_DIM + 2 + 2 * j] = zw ? 0.0 : W * gi;
    }
}

#endif  // QMC_DEVICE_CUH_
