// =====================================================================================
// qmc_static.cu -- the sector-independent sm_100a kernels of libqmc.so (compiled by nvcc):
//   qmc_lattice_debug_kernel   step a1 alone, for the bit-exact coordinate check
//   qmc_finalize_kernel        step a4, grid level: double-double sum of the tile partials
//                              per (job, shift, component), then mean / standard error over
//                              the m shifts
//   qmc_median_select_kernel   step a5: component-wise median over the K candidates and the
//                              selected candidate (Eq. 7-8)
//   qmc_amplitude_kernel       step a6: A = sum_i C_i I_i and Eq. (4) errors
//   qmc_diag_kernel            copies the uint64 diagnostics counters to the caller's int64 rows
//   qmc_dfma_peak_kernel       FP64 FMA throughput of the device (roofline denominator)
//   qmc_presample_kernel       presampling of the deformation parameter; qmc_presample_static_init_kernel and the
//                              file-scope scratch array serve its no-allocation entry point
// The launchers at the bottom are plain C++ functions called from qmc_api.cpp.
// =====================================================================================
#include <cuda_runtime.h>
#include <algorithm>
#include <mutex>
#include <stdint.h>

#include "qmc_job_dev.h"
#include "qmc_device.cuh"
#include "qmc_static.h"

// Scratch of qmc_presample_lambda_static (include/qmc.h): the entry point for callers that may not allocate device
// memory.  Every GPU that loads libqmc.so holds these 96 KiB until the process exits.  One array per device, shared by
// every call: it keeps the last call's contents, and two calls that overlap on the GPU race on it.  In HOST code this
// name is only a stand-in for the symbol -- the device address comes from cudaGetSymbolAddress (presample_static_scratch
// below); DEVICE code of this file names the array directly (qmc_presample_static_init_kernel).
static __device__ __align__(256) unsigned char qmc_presample_static_scratch[qmc::kPresampleStaticBytes];

namespace {

struct ZVec { u64 z[QMC_DEV_MAX_DIM]; };

// k = k0 + blockIdx.x * blockDim.x * per_thread + threadIdx.x + j * blockDim.x: Barrett start at
// j = 0, then the modular increment with stride blockDim.x, exactly as qmc_tile_body walks a tile.
template <class IDX>   // u32: the Barrett path of the default kernels; u64: the wide_lattice path
__global__ void qmc_lattice_debug_kernel(IDX n, u64 barrett, ZVec zv, int dim, u64 k0, u64 count, int per_thread,
                                         unsigned long long* out) {
    const u64 base = (u64)blockIdx.x * blockDim.x * (u64)per_thread + threadIdx.x;
    if (base >= count) return;
    IDX r[QMC_DEV_MAX_DIM], st[QMC_DEV_MAX_DIM];
    for (int i = 0; i < dim; ++i) {
        r[i] = qmc_lattice_start(k0 + base, (IDX)zv.z[i], n, barrett);
        st[i] = qmc_lattice_start((u64)blockDim.x, (IDX)zv.z[i], n, barrett);
    }
    for (int j = 0; j < per_thread; ++j) {
        const u64 idx = base + (u64)j * blockDim.x;
        if (idx >= count) break;
        for (int i = 0; i < dim; ++i) {
            out[idx * dim + i] = r[i];
            r[i] = qmc_lattice_next(r[i], st[i], (IDX)(n - st[i]));
        }
    }
}

// One block per job.  partials: tiles x ncomp x 2 (hi, lo), ncomp = 3 * jout.
__global__ void qmc_finalize_kernel(const QmcFinJob* fin, int jout, const double* partials, double* shift_sums,
                                    double* job_results) {
    const int job = blockIdx.x;
    const QmcFinJob f = fin[job];
    const int ncomp = 3 * jout;
    double* sums = shift_sums + (size_t)job * f.m * ncomp;
    for (int item = threadIdx.x; item < (int)f.m * ncomp; item += blockDim.x) {
        const int s = item / ncomp, comp = item - s * ncomp;
        const double* p = partials + ((size_t)f.tile_base + (size_t)s * f.tiles_per_shift) * (ncomp * 2) + comp * 2;
        double hi = 0.0, lo = 0.0;
        for (u32 t = 0; t < f.tiles_per_shift; ++t) {
            qmc_two_sum_acc(hi, lo, p[0], p[1]);
            p += ncomp * 2;
        }
        sums[item] = hi + lo;
    }
    if (job_results == nullptr) return;
    __syncthreads();
    // mean and standard error over the m shift estimates Q_s = S_s / n, re and im separately
    if (threadIdx.x < 2 * jout) {
        const int j = threadIdx.x >> 1, c = threadIdx.x & 1;
        const double dn = (double)f.n, dm = (double)f.m;
        double mean = 0.0;
        for (u32 s = 0; s < f.m; ++s) mean += sums[(s * jout + j) * 3 + c] / dn;
        mean /= dm;
        double ss = 0.0;
        for (u32 s = 0; s < f.m; ++s) {
            const double dlt = sums[(s * jout + j) * 3 + c] / dn - mean;
            ss += dlt * dlt;
        }
        job_results[((size_t)job * jout + j) * 4 + c] = mean;
        job_results[((size_t)job * jout + j) * 4 + 2 + c] = sqrt(ss / (dm * (dm - 1.0)));
    }
}

// Sharded evaluation.  One block per job; pieces of a job are consecutive in `pieces`
// (piece_lo[job] .. piece_lo[job + 1]).  out[((job m + s) ncomp + comp) 2 + {0, 1}] = (hi, lo) of the sum over this
// rank's pieces of (job, shift s): tiles and pieces are added in double-double; a (job, shift) no piece covers gets (0, 0).
__global__ void qmc_piece_sums_kernel(const QmcPieceDev* pieces, const unsigned int* piece_lo, int m, int jout,
                                      const double* partials, double* out) {
    const int job = blockIdx.x;
    const int ncomp = 3 * jout;
    for (int item = threadIdx.x; item < m * ncomp; item += blockDim.x) {
        const int s = item / ncomp, comp = item - s * ncomp;
        double hi = 0.0, lo = 0.0;
        for (unsigned int pi = piece_lo[job]; pi < piece_lo[job + 1]; ++pi) {
            const QmcPieceDev pc = pieces[pi];
            if ((unsigned)s < pc.s0 || (unsigned)s >= pc.s1) continue;
            const double* p = partials + ((size_t)pc.tile_base + (size_t)(s - pc.s0) * pc.tiles_per_shift) * (ncomp * 2) + comp * 2;
            for (u32 t = 0; t < pc.tiles_per_shift; ++t) {
                qmc_two_sum_acc(hi, lo, p[0], p[1]);
                p += ncomp * 2;
            }
        }
        out[((size_t)job * m * ncomp + item) * 2 + 0] = hi;
        out[((size_t)job * m * ncomp + item) * 2 + 1] = lo;
    }
}

// The (hi, lo) pairs of n_parts ranks (parts[part][job][s][comp][2]) added in double-double, then as
// qmc_finalize_kernel: per-shift sums, mean and standard error over the m shifts.
__global__ void qmc_finalize_parts_kernel(const unsigned long long* n_of_job, int m, int jout, const double* parts,
                                          int n_parts, size_t part_stride, double* shift_sums, double* job_results) {
    const int job = blockIdx.x;
    const int ncomp = 3 * jout;
    double* sums = shift_sums + (size_t)job * m * ncomp;
    for (int item = threadIdx.x; item < m * ncomp; item += blockDim.x) {
        double hi = 0.0, lo = 0.0;
        for (int part = 0; part < n_parts; ++part) {
            const double* p = parts + (size_t)part * part_stride + ((size_t)job * m * ncomp + item) * 2;
            qmc_two_sum_acc(hi, lo, p[0], p[1]);
        }
        sums[item] = hi + lo;
    }
    if (job_results == nullptr) return;             // the candidate stage (qmc_median_select_pieces) wants the sums only
    __syncthreads();
    if (threadIdx.x < 2 * jout) {
        const int j = threadIdx.x >> 1, c = threadIdx.x & 1;
        const double dn = (double)n_of_job[job], dm = (double)m;
        double mean = 0.0;
        for (int s = 0; s < m; ++s) mean += sums[(s * jout + j) * 3 + c] / dn;
        mean /= dm;
        double ss = 0.0;
        for (int s = 0; s < m; ++s) {
            const double dlt = sums[(s * jout + j) * 3 + c] / dn - mean;
            ss += dlt * dlt;
        }
        job_results[((size_t)job * jout + j) * 4 + c] = mean;
        job_results[((size_t)job * jout + j) * 4 + 2 + c] = sqrt(ss / (dm * (dm - 1.0)));
    }
}

// ------------------------------------------------------------------------------------ presampling of lambda
// Deformation-parameter presampling ("number_of_presamples ... initial contour deformation parameter
// selection"; reading R-pre).  One thread per presample point of one shifted lattice: a1 / a2 with
// the same device functions as the evaluation kernels, the gradient of F at the real point from the monomial table, and
// for every candidate lambda_j the value F(z(x; lambda_j)) + i f_im by direct monomial products.  fail[j] counts the
// points where the candidate fails the sign check (Im F >= 0) or the distance (|F| < min_abs_f); worst[2 j], worst[2 j + 1] keep max Im F
// and min |F| over the points as order-preserving integer keys (atomicMax / atomicMin).
struct QmcPresampleArgs {
    int dim, transform, nF, n_cand;
    u64 n, barrett;
    double inv_n, f_im, min_abs_f;
    u64 z[QMC_DEV_MAX_DIM];
    double shift[QMC_DEV_MAX_DIM];
    double kcoef[8];                 // general Korobov: a_0 .. a_r1 (unused otherwise)
    double kinvb;
    const double* F_coef;            // nF
    const unsigned char* F_exp;      // nF x dim
    const double* lambdas;           // n_cand
    unsigned int* fail;              // n_cand x 2: points failing the sign check, points too close to a zero of F
    unsigned long long* worst;       // n_cand x 2
};
__device__ __forceinline__ unsigned long long qmc_order_key(double v) {   // monotone map double -> u64
    const unsigned long long b = (unsigned long long)__double_as_longlong(v);
    return (b >> 63) ? ~b : (b | 0x8000000000000000ull);
}
__device__ __forceinline__ double qmc_rt_pow(double x, int e) { double r = 1.0; for (int i = 0; i < e; ++i) r *= x; return r; }

template <class IDX>
__global__ void qmc_presample_kernel(const QmcPresampleArgs a) {
    const int d = a.dim;
    for (u64 k = (u64)blockIdx.x * blockDim.x + threadIdx.x; k < a.n; k += (u64)gridDim.x * blockDim.x) {
        double x[QMC_DEV_MAX_DIM], G[QMC_DEV_MAX_DIM];
        double W = 1.0;
        for (int i = 0; i < d; ++i) {
            IDX sa;
            double sc;
            qmc_shift_split((IDX)a.n, a.shift[i], sa, sc);
            const IDX r = qmc_lattice_next(qmc_lattice_start(k, (IDX)a.z[i], (IDX)a.n, a.barrett), sa, (IDX)((IDX)a.n - sa));
            const double t = fma(qmc_index_to_double(r), a.inv_n, sc);
            double P = 1.0;
            if (a.transform == QMC_TR_KOROBOV3) { QmcTransform<QMC_TR_KOROBOV3>::apply(t, x[i], P); W *= P; }
            else if (a.transform == QMC_TR_BAKER) QmcTransform<QMC_TR_BAKER>::apply(t, x[i], P);
            else if (a.transform >= 100) {
                const int r0 = (a.transform - 100) / 10, r1 = (a.transform - 100) % 10;
                double h = a.kcoef[r1];
                for (int j = r1 - 1; j >= 0; --j) h = fma(t, h, a.kcoef[j]);
                x[i] = qmc_rt_pow(t, r0 + 1) * h;
                W *= qmc_rt_pow(t, r0) * qmc_rt_pow(1.0 - t, r1);
            } else x[i] = t;
        }
        if (W == 0.0) continue;                                   // a point of weight 0 enters no sum (reading Q4)
        for (int i = 0; i < d; ++i) {                              // G_i = dF/dx_i at the real point
            double g = 0.0;
            for (int t = 0; t < a.nF; ++t) {
                const int ei = a.F_exp[t * d + i];
                if (ei == 0) continue;
                double term = a.F_coef[t] * (double)ei;
                for (int l = 0; l < d; ++l) term *= qmc_rt_pow(x[l], a.F_exp[t * d + l] - (l == i ? 1 : 0));
                g += term;
            }
            G[i] = g;
        }
        for (int j = 0; j < a.n_cand; ++j) {
            const double lam = a.lambdas[j];
            double zi[QMC_DEV_MAX_DIM];
            for (int i = 0; i < d; ++i) zi[i] = -(lam * x[i] * (1.0 - x[i]) * G[i]);     // Im z_i; Re z_i = x_i
            double fre = 0.0, fim = a.f_im;
            for (int t = 0; t < a.nF; ++t) {
                double tr = a.F_coef[t], ti = 0.0;
                for (int i = 0; i < d; ++i)
                    for (int e = 0; e < a.F_exp[t * d + i]; ++e) {
                        const double nr = tr * x[i] - ti * zi[i], ni = tr * zi[i] + ti * x[i];
                        tr = nr; ti = ni;
                    }
                fre += tr; fim += ti;
            }
            const double af = sqrt(fre * fre + fim * fim);
            if (!(fim < 0.0)) atomicAdd(&a.fail[2 * j], 1u);                 // sign check
            else if (af < a.min_abs_f) atomicAdd(&a.fail[2 * j + 1], 1u);     // distance from the zeros of F
            atomicMax(&a.worst[2 * j], qmc_order_key(fim));
            atomicMin(&a.worst[2 * j + 1], qmc_order_key(af));
        }
    }
}

// qmc_presample_lambda_static: what must start from a known value in the shared scratch array -- the fail counters (0)
// and the order keys (max key low, min key high) of the n_cand candidates.  Device code names the array directly.
__global__ void qmc_presample_static_init_kernel(int n_cand) {
    unsigned int* fail = reinterpret_cast<unsigned int*>(qmc_presample_static_scratch + qmc::kPsOffFail);
    unsigned long long* worst = reinterpret_cast<unsigned long long*>(qmc_presample_static_scratch + qmc::kPsOffWorst);
    for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < 2 * n_cand; i += gridDim.x * blockDim.x) {
        fail[i] = 0u;
        worst[i] = (i & 1) ? ~0ull : 0ull;
    }
}

__device__ double qmc_median_sorted(double* v, int K) {   // insertion sort in place, then the middle
    for (int i = 1; i < K; ++i) {
        const double key = v[i];
        int j = i - 1;
        while (j >= 0 && v[j] > key) { v[j + 1] = v[j]; --j; }
        v[j + 1] = key;
    }
    return (K & 1) ? v[K / 2] : 0.5 * (v[K / 2 - 1] + v[K / 2]);
}

// One block per job, thread c < 2 * jout owns component c; thread 0 then selects.
// cand_sums: (job * K + c) x jout x 3 from the one-shift stage; n per job in fin[job * K].n.
#define QMC_MAX_K 64
__global__ void qmc_median_select_kernel(const QmcFinJob* fin, int K, int jout, const double* cand_sums,
                                         double* cand_est, double* median, int* selected) {
    const int job = blockIdx.x;
    const int nc = 2 * jout;
    __shared__ double med_sh[2 * 3 * 4], mad_sh[2 * 3 * 4];
    const double dn = (double)fin[(size_t)job * K].n;
    double* est = cand_est + (size_t)job * K * nc;
    if ((int)threadIdx.x < nc) {
        const int comp = threadIdx.x, j = comp >> 1, ri = comp & 1;
        double v[QMC_MAX_K];
        for (int c = 0; c < K; ++c) {
            const double q = cand_sums[(((size_t)job * K + c) * jout + j) * 3 + ri] / dn;
            est[(size_t)c * nc + comp] = q;
            v[c] = q;
        }
        const double med = qmc_median_sorted(v, K);
        for (int c = 0; c < K; ++c) v[c] = fabs(est[(size_t)c * nc + comp] - med);
        med_sh[comp] = med;
        mad_sh[comp] = qmc_median_sorted(v, K);
        median[(size_t)job * nc + comp] = med;
    }
    __syncthreads();
    if (threadIdx.x == 0) {
        int best = 0;
        double best_d = 0.0;
        for (int c = 0; c < K; ++c) {
            double dist = 0.0;
            for (int comp = 0; comp < nc; ++comp) {
                if (mad_sh[comp] == 0.0) continue;
                const double u = (est[(size_t)c * nc + comp] - med_sh[comp]) / mad_sh[comp];
                dist += u * u;
            }
            if (c == 0 || dist < best_d) { best = c; best_d = dist; }
        }
        selected[job] = best;
    }
}

// thread j < jout: A_j = sum_i C_i mean_{i,j}; component-wise variance propagation
__global__ void qmc_amplitude_kernel(const double* job_results, const double* coef, int n_jobs, int jout, double* amp) {
    const int j = threadIdx.x;
    if (j >= jout) return;
    double are = 0.0, aim = 0.0, vre = 0.0, vim = 0.0;
    for (int i = 0; i < n_jobs; ++i) {
        const double* r = job_results + ((size_t)i * jout + j) * 4;
        const double cr = coef[2 * i], ci = coef[2 * i + 1];
        are += cr * r[0] - ci * r[1];
        aim += cr * r[1] + ci * r[0];
        vre += cr * cr * r[2] * r[2] + ci * ci * r[3] * r[3];
        vim += ci * ci * r[2] * r[2] + cr * cr * r[3] * r[3];
    }
    amp[j * 4 + 0] = are; amp[j * 4 + 1] = aim;
    amp[j * 4 + 2] = sqrt(vre); amp[j * 4 + 3] = sqrt(vim);
}

__global__ void qmc_diag_kernel(const unsigned long long* diag, int n, long long* out) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) out[i] = (long long)diag[i];
}

// 16 independent FMA chains per thread: enough to cover the FP64 pipe latency at any occupancy
__global__ void __launch_bounds__(256) qmc_dfma_peak_kernel(int iters, double seed, double* sink) {
    double a[16];
#pragma unroll
    for (int i = 0; i < 16; ++i) a[i] = seed + (double)(threadIdx.x + i);
    const double m = 1.0 - 1e-9 * seed, c = 1e-9;
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int r = 0; r < 4; ++r)
#pragma unroll
            for (int i = 0; i < 16; ++i) a[i] = fma(a[i], m, c);
    }
    double s = 0.0;
#pragma unroll
    for (int i = 0; i < 16; ++i) s += a[i];
    if (s == -1.2345e300 && sink) *sink = s;   // never true; keeps the chains alive
}

// The same 16 chains with ONE independent integer add after every DFMA.  Measured on B200: 35.7 against 36.0 TFLOP/s,
// i.e. in a regular stream of independent instructions the integer pipe is free beside the FP64 pipe.  bench.py reports
// it beside the pure peak so that the gap of the evaluation kernels (77 % FP64-pipe activity at every occupancy, CTA
// shape and unroll tried) is not mistaken for the cost of their integer instructions.
__global__ void __launch_bounds__(256) qmc_dfma_mixed_kernel(int iters, double seed, double* sink) {
    double a[16];
    unsigned r[16];
#pragma unroll
    for (int i = 0; i < 16; ++i) { a[i] = seed + (double)(threadIdx.x + i); r[i] = threadIdx.x * 17u + i; }
    const double m = 1.0 - 1e-9 * seed, c = 1e-9;
    const unsigned inc = (unsigned)seed | 1u;
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int rr = 0; rr < 4; ++rr)
#pragma unroll
            for (int i = 0; i < 16; ++i) {
                a[i] = fma(a[i], m, c);
                asm volatile("add.u32 %0, %0, %1;" : "+r"(r[i]) : "r"(inc));
            }
    }
    double s = 0.0;
    unsigned rs = 0;
#pragma unroll
    for (int i = 0; i < 16; ++i) { s += a[i]; rs += r[i]; }
    if (s == -1.2345e300 && sink) *sink = s + rs;
}

}  // namespace

namespace qmc {

cudaError_t launch_lattice_debug(uint64_t n, uint64_t barrett, const uint64_t* z, int dim, uint64_t k0, uint64_t count,
                                 uint64_t* d_out, cudaStream_t st) {
    ZVec zv;
    for (int i = 0; i < QMC_DEV_MAX_DIM; ++i) zv.z[i] = i < dim ? z[i] : 0u;
    const int threads = 256, per_thread = 4;
    const uint64_t blocks = (count + (uint64_t)threads * per_thread - 1) / ((uint64_t)threads * per_thread);
    if (blocks == 0) return cudaSuccess;
    if (n < (1ull << 32))
        qmc_lattice_debug_kernel<u32><<<(unsigned)blocks, threads, 0, st>>>((u32)n, barrett, zv, dim, k0, count, per_thread,
                                                                            (unsigned long long*)d_out);
    else
        qmc_lattice_debug_kernel<u64><<<(unsigned)blocks, threads, 0, st>>>((u64)n, barrett, zv, dim, k0, count, per_thread,
                                                                            (unsigned long long*)d_out);
    return cudaGetLastError();
}

cudaError_t launch_finalize(const QmcFinJob* d_fin, int n_jobs, int jout, const double* d_partials, double* d_shift_sums,
                            double* d_job_results, cudaStream_t st) {
    if (n_jobs <= 0) return cudaSuccess;
    qmc_finalize_kernel<<<n_jobs, 128, 0, st>>>(d_fin, jout, d_partials, d_shift_sums, d_job_results);
    return cudaGetLastError();
}

cudaError_t launch_piece_sums(const QmcPieceDev* d_pieces, const unsigned int* d_piece_lo, int n_jobs, int m, int jout,
                              const double* d_partials, double* d_out, cudaStream_t st) {
    if (n_jobs <= 0) return cudaSuccess;
    qmc_piece_sums_kernel<<<n_jobs, 128, 0, st>>>(d_pieces, d_piece_lo, m, jout, d_partials, d_out);
    return cudaGetLastError();
}

cudaError_t launch_finalize_parts(const unsigned long long* d_n, int n_jobs, int m, int jout, const double* d_parts, int n_parts,
                                  size_t part_stride, double* d_shift_sums, double* d_job_results, cudaStream_t st) {
    if (n_jobs <= 0) return cudaSuccess;
    qmc_finalize_parts_kernel<<<n_jobs, 128, 0, st>>>(d_n, m, jout, d_parts, n_parts, part_stride, d_shift_sums, d_job_results);
    return cudaGetLastError();
}

cudaError_t launch_presample(const PresampleHost& h, const double* d_F_coef, const unsigned char* d_F_exp, const double* d_lambdas,
                             unsigned int* d_fail, unsigned long long* d_worst, cudaStream_t st) {
    QmcPresampleArgs a;
    a.dim = h.dim; a.transform = h.transform; a.nF = h.nF; a.n_cand = h.n_cand;
    a.n = h.n; a.barrett = ~0ull / h.n; a.inv_n = 1.0 / (double)h.n; a.f_im = h.f_im; a.min_abs_f = h.min_abs_f;
    for (int i = 0; i < QMC_DEV_MAX_DIM; ++i) { a.z[i] = h.z[i]; a.shift[i] = h.shift[i]; }
    for (int i = 0; i < 8; ++i) a.kcoef[i] = h.kcoef[i];
    a.kinvb = h.kinvb;
    a.F_coef = d_F_coef; a.F_exp = d_F_exp; a.lambdas = d_lambdas; a.fail = d_fail; a.worst = d_worst;
    const unsigned blocks = (unsigned)std::min<uint64_t>((h.n + 127) / 128, 148 * 16);
    if (h.n < (1ull << 32)) qmc_presample_kernel<u32><<<blocks, 128, 0, st>>>(a);
    else qmc_presample_kernel<u64><<<blocks, 128, 0, st>>>(a);
    return cudaGetLastError();
}

// Device address of qmc_presample_static_scratch on the CURRENT device.  Looked up once per device with that device
// current (the set-up of the no-allocation path) and remembered; `qmc_presample_static_scratch` itself is not a device
// address in host code.  No allocation: cudaGetSymbolAddress only resolves the symbol of the already loaded module.
cudaError_t presample_static_scratch(unsigned char** d_ptr) {
    constexpr int kMaxDev = 64;
    static std::mutex mu;
    static unsigned char* addr[kMaxDev] = {nullptr};
    *d_ptr = nullptr;
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    std::lock_guard<std::mutex> lock(mu);
    if (dev >= 0 && dev < kMaxDev && addr[dev]) { *d_ptr = addr[dev]; return cudaSuccess; }
    void* p = nullptr;
    e = cudaGetSymbolAddress(&p, qmc_presample_static_scratch);
    if (e != cudaSuccess) return e;
    if (p == nullptr || ((uintptr_t)p & 255u)) return cudaErrorInvalidSymbol;
    if (dev >= 0 && dev < kMaxDev) addr[dev] = static_cast<unsigned char*>(p);
    *d_ptr = static_cast<unsigned char*>(p);
    return cudaSuccess;
}

// launch_presample with every device buffer inside the file-scope array: inputs copied in, counters and keys reset by
// qmc_presample_static_init_kernel, results copied out to the caller's HOST arrays (2 n_cand entries each), all on st.
// The caller synchronises st before reading them.  Sizes are checked by the caller (qmc_presample_lambda_static).
cudaError_t launch_presample_static(const PresampleHost& h, const double* h_F_coef, const unsigned char* h_F_exp,
                                    const double* h_lambdas, unsigned int* h_fail, unsigned long long* h_worst, cudaStream_t st) {
    if (h.nF < 1 || h.nF > kPresampleStaticMaxTerms || h.n_cand < 1 || h.n_cand > kPresampleMaxCand || h.dim < 1 ||
        h.dim > QMC_DEV_MAX_DIM)
        return cudaErrorInvalidValue;
    unsigned char* ds = nullptr;
    cudaError_t e = presample_static_scratch(&ds);
    if (e != cudaSuccess) return e;
    double* d_coef = reinterpret_cast<double*>(ds + kPsOffCoef);
    unsigned char* d_exp = ds + kPsOffExp;
    double* d_lam = reinterpret_cast<double*>(ds + kPsOffLam);
    unsigned int* d_fail = reinterpret_cast<unsigned int*>(ds + kPsOffFail);
    unsigned long long* d_worst = reinterpret_cast<unsigned long long*>(ds + kPsOffWorst);
    if ((e = cudaMemcpyAsync(d_coef, h_F_coef, (size_t)h.nF * sizeof(double), cudaMemcpyHostToDevice, st)) != cudaSuccess) return e;
    if ((e = cudaMemcpyAsync(d_exp, h_F_exp, (size_t)h.nF * h.dim, cudaMemcpyHostToDevice, st)) != cudaSuccess) return e;
    if ((e = cudaMemcpyAsync(d_lam, h_lambdas, (size_t)h.n_cand * sizeof(double), cudaMemcpyHostToDevice, st)) != cudaSuccess) return e;
    qmc_presample_static_init_kernel<<<(2 * h.n_cand + 255) / 256, 256, 0, st>>>(h.n_cand);
    if ((e = cudaGetLastError()) != cudaSuccess) return e;
    if ((e = launch_presample(h, d_coef, d_exp, d_lam, d_fail, d_worst, st)) != cudaSuccess) return e;
    if ((e = cudaMemcpyAsync(h_fail, d_fail, (size_t)2 * h.n_cand * sizeof(unsigned int), cudaMemcpyDeviceToHost, st)) != cudaSuccess) return e;
    return cudaMemcpyAsync(h_worst, d_worst, (size_t)2 * h.n_cand * sizeof(unsigned long long), cudaMemcpyDeviceToHost, st);
}

cudaError_t launch_median_select(const QmcFinJob* d_fin, int n_jobs, int K, int jout, const double* d_cand_sums,
                                 double* d_cand_est, double* d_median, int* d_selected, cudaStream_t st) {
    if (n_jobs <= 0) return cudaSuccess;
    qmc_median_select_kernel<<<n_jobs, 32, 0, st>>>(d_fin, K, jout, d_cand_sums, d_cand_est, d_median, d_selected);
    return cudaGetLastError();
}

cudaError_t launch_amplitude(const double* d_job_results, const double* d_coef, int n_jobs, int jout, double* d_amp,
                             cudaStream_t st) {
    qmc_amplitude_kernel<<<1, 32, 0, st>>>(d_job_results, d_coef, n_jobs, jout, d_amp);
    return cudaGetLastError();
}

cudaError_t launch_diag(const unsigned long long* d_diag, int n, long long* d_out, cudaStream_t st) {
    if (n <= 0) return cudaSuccess;
    qmc_diag_kernel<<<(n + 255) / 256, 256, 0, st>>>(d_diag, n, d_out);
    return cudaGetLastError();
}

cudaError_t launch_dfma_peak(int blocks, int iters, cudaStream_t st, bool mixed) {
    if (mixed) qmc_dfma_mixed_kernel<<<blocks, 256, 0, st>>>(iters, 1.0, nullptr);
    else qmc_dfma_peak_kernel<<<blocks, 256, 0, st>>>(iters, 1.0, nullptr);
    return cudaGetLastError();
}

}  // namespace qmc
