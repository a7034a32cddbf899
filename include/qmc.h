/* =====================================================================================
 * qmc.h -- C ABI of the B200 (sm_100a) shifted-lattice QMC library (libqmc.so).
 *
 * The library is the hot path of pySecDec's numerical stage (arXiv:2305.19768, PAPER.md):
 * for each sector integrand f, lattice size n, generating vector z and m random shifts
 * Delta_s it returns the mean and the standard error of the m shift estimates
 *     Q_s = (1/n) sum_{k=0}^{n-1} W(t_k) f(phi(t_k)),   t_k = frac(k z / n + Delta_s)
 * ("Quasi-Monte-Carlo (QMC) integration method based on rank-1 shifted lattice rules",
 * PAPER.md:102; error "sqrt(var(I_i)/m) after m = 32 repetitions"), the
 * median lattice rule (Eq. 7-8) and the amplitude A = sum_i C_i I_i
 * with its propagated error (Eq. 4).  Where the paper is silent the
 * readings are those of SURVEY.md section 8(c) / DESIGN.md section 3.
 *
 * Conventions
 *  - plain C: no exceptions cross the boundary, every function returns an int32 status
 *    (QMC_OK = 0, errors < 0) unless stated; qmc_last_error() gives a thread-local detail.
 *  - "HOST" pointers are ordinary host memory, read before the call returns (the caller
 *    may free them immediately).  "DEV" pointers are CUDA device memory owned by the
 *    caller (e.g. torch tensors); the library never frees or reallocates them.
 *  - all device work is enqueued on the CUDA stream passed in (cudaStream_t as void*) or
 *    on internal streams forked from and joined back to it; the calls do not synchronise the
 *    device or the stream.  The job table travels through one of 4 pinned staging buffers per
 *    plan (sized by qmc_plan_bind_workspace): up to 4 calls on a plan can be in flight; a 5th
 *    blocks the host until the input copy (not the kernels) of the call 4 earlier is done.
 *  - ONE PLAN, ONE STREAM AT A TIME: a plan has a single workspace (tile counters, partial sums,
 *    diagnostics), so consecutive calls on one plan must be enqueued on the same stream, or be
 *    ordered by the caller (event / synchronisation) when the stream changes.  Calls on
 *    different plans (each with its own workspace) may run concurrently on different streams.
 *  - qmc_plan_destroy waits for the plan's last enqueued call to finish before it unloads the
 *    compiled modules; the caller's buffers must stay alive until then.
 *  - the only device memory the library uses is the caller-provided workspace
 *    (qmc_plan_bind_workspace) and the scratch passed to single calls; the plan owns host memory and
 *    the loaded CUDA modules.  One exception: a fixed 96 KiB __device__ array inside libqmc.so
 *    that serves qmc_presample_lambda_static, the entry point for callers that cannot allocate.
 *  - there is no CPU fallback: without a CUDA device every compute entry point returns
 *    QMC_ERR_CUDA.
 *
 * Differences from the sketch in SURVEY.md section 8(b) (DESIGN.md section 1 says why):
 *  - qmc_plan_opts has no sum_mode: there is one summation (compensated at every level), no
 *    plain-FP64 variant to select;
 *  - qmc_integrate_sectors / qmc_median_integrate_sectors take n_shift_rows, the number of rows
 *    of the shifts array, so that shift_offset + m can be range-checked before any enqueue;
 *  - opts.validate is applied at call time (qmc_integrate_* / qmc_median_*: gcd(z_i, n) = 1),
 *    because z and n are arguments of the call, not of the plan; the limits of the polynomial
 *    description are always checked by qmc_plan;
 *  - qmc_plan_workspace_bytes takes max_shift_rows instead of m (jobs may share shift rows);
 *  - additions: QMC_ERR_COMPILE, qmc_median_integrate_sectors (the batched median rule the survey
 *    allows), qmc_debug_eval_points, the plan introspection / statistics getters, the adaptive
 *    driver (8(f) #1), wide_lattice, the Korobov family and the presampling of lambda (8(f) #4; with a
 *    no-allocation variant), the sharded evaluation by pieces, median rule included (8(e)).
 * ===================================================================================== */
#ifndef QMC_H_
#define QMC_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define QMC_MAX_DIM 8      /* sector dimension d <= 8 (BASELINE.json configs: 2..8)        */
#define QMC_MAX_ORDERS 5   /* epsilon-orders J per sector (config 3: eps^-2 .. eps^0; two loops: 5) */
#define QMC_MAX_LOG_DEGREE 4 /* highest log-polynomial degree first_order + n_orders - 1  */

enum {
  QMC_OK = 0,
  QMC_ERR_INVALID_ARG = -1,  /* null pointer, size or index out of range, non-finite input  */
  QMC_ERR_UNSUPPORTED = -2,  /* n >= 2^32 (2^53 with wide_lattice), dim > QMC_MAX_DIM, unknown kind */
  QMC_ERR_CUDA = -3,         /* a CUDA runtime call failed (no device, launch error, ...)    */
  QMC_ERR_WORKSPACE = -4,    /* workspace not bound or too small                             */
  QMC_ERR_NOT_UNIT = -5,     /* validate: some z_i is not a unit mod n (Eq. 7)  */
  QMC_ERR_COMPILE = -6       /* NVRTC rejected the generated sector code (see last error)    */
};

/* periodising transforms (named at PAPER.md:707: "korobov3" default, "baker") */
enum { QMC_TRANSFORM_NONE = 0, QMC_TRANSFORM_KOROBOV3 = 1, QMC_TRANSFORM_BAKER = 2 };
/* The Korobov family of which korobov3 is the default (higher orders, asymmetric weights):
 * weight t^r0 (1 - t)^r1 / B(r0 + 1, r1 + 1), map = its integral, 1 <= r0, r1 <= 6.  QMC_TRANSFORM_KOROBOV(3, 3) is the
 * same transform as QMC_TRANSFORM_KOROBOV3 (evaluated by the generic code instead of the hand-tuned one). */
#define QMC_TRANSFORM_KOROBOV(r0, r1) (100 + 10 * (r0) + (r1))

/* integrand classes */
enum {
  QMC_KIND_UF = 0,  /* x^a U(x)^p F(x)^q L_j(log U, log F)  (sector-decomposed, eps-expanded) */
  QMC_KIND_TOY = 1  /* prod_i (1 + c_i (x_i - 1/2) + d_i x_i^2)  (BASELINE.json config 0)     */
};

/* One sector integrand as a polynomial description.  HOST memory, read by qmc_plan only.
 *
 *   real class (deformed = 0), x in (0,1)^d after the periodising transform:
 *     g_j(x) = prod_i x_i^{a_i} * U(x)^p * F(x)^q * L_j(log U, log F)
 *   deformed class (deformed = 1; "contour deformation"; BASELINE.json config 3):
 *     z_i = x_i - i lambda x_i (1 - x_i) dF/dx_i(x)
 *     Jac = det[ delta_ik - i lambda ( (1 - 2 x_i) dF/dx_i delta_ik + x_i (1 - x_i) d2F/dx_i dx_k ) ]
 *     g_j = Jac * prod_i z_i^{a_i} * U(z)^p * (F(z) + i f_im)^q * L_j(Log U, Log F)   (principal Log)
 *   L_j(lU, lF) = sum_{alpha+beta <= j} c^{(j)}_{alpha,beta} lU^alpha lF^beta, for the J = n_orders
 *   degrees j = first_order .. first_order + J - 1.
 *   U = sum_t U_coef[t] prod_i x_i^{U_exp[t*dim+i]} and F likewise (a constant term is an
 *   all-zero exponent row).
 */
typedef struct {
  int32_t kind;              /* QMC_KIND_*                                                    */
  int32_t dim;               /* 1 .. QMC_MAX_DIM                                              */
  int32_t transform;         /* QMC_TRANSFORM_*                                               */
  int32_t deformed;          /* 0 real, 1 complex with contour deformation (kind UF only)     */
  int32_t first_order;       /* j0 >= 0                                                       */
  int32_t n_orders;          /* J in 1 .. QMC_MAX_ORDERS; j0 + J - 1 <= QMC_MAX_LOG_DEGREE    */
  int32_t a[QMC_MAX_DIM];    /* monomial prefactor exponents, 0 <= a_i <= 16                  */
  int32_t nU, nF;            /* number of monomials of U and F (>= 1); TOY: nU = 2*dim, nF=0  */
  double p, q;               /* real powers of U and F                                        */
  double lambda;             /* deformation strength (deformed only)                          */
  double f_im;               /* added to Im F(z): the -i delta prescription (deformed only)   */
  const double* U_coef;      /* nU              (TOY: c_0..c_{d-1}, d_0..d_{d-1})              */
  const uint8_t* U_exp;      /* nU x dim row-major, each <= 16 (unused for TOY)               */
  const double* F_coef;      /* nF                                                            */
  const uint8_t* F_exp;      /* nF x dim row-major                                            */
  const double* logc;        /* for each order j in turn (j+1)(j+2)/2 coefficients c_{alpha,beta},
                                ordered by (alpha+beta, beta); real                           */
} qmc_sector_desc;

typedef struct {             /* HOST; zero-initialised = defaults                             */
  int32_t validate;          /* 1: qmc_integrate_* / qmc_median_* check gcd(z_i, n) = 1       */
  int32_t threads_per_block; /* 0 = default (256); multiple of 32, <= 1024                    */
  int32_t ctas_per_sm;       /* 0 = chosen per module from the size of its code (2, or 1 for the
                                largest sectors); 1..8 forces the register bound 65536/(ctas*threads) */
  int32_t max_tiles;         /* 0 = default (65536): upper bound on (job, shift, k-range)
                                tiles of one launch; sizes the partial-sum area               */
  int32_t sectors_per_module;/* 0 = default (16): sectors compiled into one persistent kernel; a
                                module is also capped at 4096 emitted FP64 ops (compile time)    */
  int32_t compile_threads;   /* 0 = min(hardware threads, 16)                                 */
  int32_t libdevice_math;    /* 0 = library's own log/exp/atan2/sincos (default, faster), 1 = the CUDA
                                library (libdevice) versions, slower: for A/B measurement      */
  int32_t points_per_thread; /* 0 = chosen per module (2..4 for the real class by code size, 1 for the deformed
                                class): lattice points a thread evaluates per loop iteration; 1..8           */
  int32_t wide_lattice;      /* 1: 64-bit lattice indices, jobs with 2^32 <= n < 2^53 are accepted (the paper
                                reaches n = 4.3e9 and ~7e10); 0 = 32-bit indices, n < 2^32  */
  int32_t reserved[3];
} qmc_plan_opts;

/* One integration job: sector, lattice and its block of shifts.  HOST. */
typedef struct {
  int32_t sector;            /* index into the plan's sectors                                 */
  int32_t shift_offset;      /* first row of this job's m shifts in the shifts array          */
  uint64_t n;                /* lattice size, 1 <= n < 2^32 (< 2^53 in a wide_lattice plan)   */
  uint64_t z[QMC_MAX_DIM];   /* generating vector, 0 <= z_i < n (units mod n if validate)     */
  double coef_re, coef_im;   /* amplitude weight C_i                           */
} qmc_job;

typedef struct qmc_plan_s qmc_plan_t;

/* qmc_plan: "compiled from a seedable polynomial description" -- generates one straight-line
 * CUDA device function per sector (sparse multivariate Horner forms of U, F, dF, d2F; the
 * unrolled complex LU; the log-polynomial orders), groups sectors of equal (class, dim) into
 * persistent kernels and compiles them with NVRTC for sm_100a.  Needs no GPU; the modules are
 * loaded onto the current device by qmc_plan_bind_workspace.  On error *plan_out = NULL.
 * Compiled modules are cached per process; with the environment variable QMC_CUBIN_CACHE=<directory> they are
 * also kept on disk, keyed by a hash of the complete generated source and the NVRTC version. */
int32_t qmc_plan(const qmc_sector_desc* sectors /*HOST*/, int32_t n_sectors,
                 const qmc_plan_opts* opts /*HOST or NULL*/, qmc_plan_t** plan_out);

/* Number of order slots J_out (= max n_orders over the plan's sectors) used by every output
 * array below; a job whose sector has fewer orders leaves the remaining slots zero. */
int32_t qmc_plan_orders(const qmc_plan_t* plan);

/* Generated CUDA source of module `module` (0 <= module < qmc_plan_modules), for inspection
 * and tests.  The pointer is owned by the plan. */
int32_t qmc_plan_modules(const qmc_plan_t* plan);
const char* qmc_plan_module_source(const qmc_plan_t* plan, int32_t module);
/* NVRTC / ptxas log of the module (registers, spills), owned by the plan. */
const char* qmc_plan_module_log(const qmc_plan_t* plan, int32_t module);
/* Algorithmic FP64 flops of one evaluation of `sector` (DESIGN.md section 6 cost model) and the
 * FP64 operation count of the code the generator emitted for it (fma = 1 op). */
double qmc_plan_sector_flops(const qmc_plan_t* plan, int32_t sector);
double qmc_plan_sector_ops(const qmc_plan_t* plan, int32_t sector);
/* Flops of one evaluation as the generated code performs them (fma = 2, add / mul = 1, elementary functions by
 * the flops of the library's own routines): the quantity ncu's 2 DFMA + DMUL + DADD measures, used for
 * bench.py's roofline.achieved.  qmc_plan_sector_flops is SURVEY.md 8(d)'s monomial-by-monomial model. */
double qmc_plan_sector_emitted_flops(const qmc_plan_t* plan, int32_t sector);

/* Device workspace the plan needs for launches of up to max_jobs jobs (for the median rule:
 * max_jobs counts every candidate as a job) with up to max_shift_rows shift rows. */
size_t qmc_plan_workspace_bytes(const qmc_plan_t* plan, int32_t max_jobs, int32_t max_shift_rows);
/* Binds caller-owned device memory (256-byte aligned) and loads the compiled modules onto the
 * current device (first call only).  The caller keeps ownership and must keep it alive. */
int32_t qmc_plan_bind_workspace(qmc_plan_t* plan, void* d_workspace /*DEV*/, size_t bytes);

/* Steps a1-a4, a6: for every job the per-shift sums
 *   S_{s,j} = sum_k W_k g_j(x_k),  A_{s,j} = sum_k |W_k g_j(x_k)|,
 * the mean and standard error over the m shifts (re and im separately, 1/(m(m-1)) variance),
 * and the amplitude sum_i C_i mean_i with component-wise error propagation.
 *   shifts        HOST  n_shift_rows x QMC_MAX_DIM doubles in [0,1); job i uses rows
 *                       shift_offset .. shift_offset + m - 1
 *   d_shift_sums  DEV out  n_jobs x m x J_out x 3   (Re S, Im S, A)
 *   d_job_results DEV out  n_jobs x J_out x 4       (mean_re, mean_im, err_re, err_im)
 *   d_amplitude   DEV out or NULL  J_out x 4        (re, im, err_re, err_im)
 *   d_diag        DEV out or NULL  n_jobs x 2 int64 (zero-weight points, Im F >= 0 points)
 * m >= 2 (the error is undefined for m = 1). */
int32_t qmc_integrate_sectors(qmc_plan_t* plan, const qmc_job* jobs /*HOST*/, int32_t n_jobs,
                              const double* shifts /*HOST*/, int32_t n_shift_rows, int32_t m,
                              double* d_shift_sums, double* d_job_results, double* d_amplitude,
                              int64_t* d_diag, void* cuda_stream);

/* Step a5, the construction-free median lattice rule (Eq. 7-8): evaluates
 * Q_{n,z_c} for K candidate generating vectors with one shared shift, the component-wise
 * median over c (each order, re and im) and the index of the candidate nearest that median
 * in MAD-scaled distance (readings Q5-Q7).
 *   z_cand     HOST K x QMC_MAX_DIM (1 <= K <= 64)       shift0  HOST QMC_MAX_DIM
 *   d_cand_est DEV out K x J_out x 2      d_median DEV out J_out x 2     d_selected DEV out 1 */
int32_t qmc_median_rule(qmc_plan_t* plan, int32_t sector, uint64_t n,
                        const uint64_t* z_cand, int32_t K, const double* shift0,
                        double* d_cand_est, double* d_median, int32_t* d_selected,
                        void* cuda_stream);

/* Batched a5 + a1-a4 + a6 with no host round trip: for every job the median rule over its K
 * candidates (jobs[i].z is ignored), then the m-shift integration on the selected candidate,
 * then the amplitude.  This is one pass of BASELINE.json config 2.
 *   z_cand HOST n_jobs x K x QMC_MAX_DIM    shift0 HOST n_jobs x QMC_MAX_DIM
 *   d_cand_est DEV out n_jobs x K x J_out x 2, d_median n_jobs x J_out x 2, d_selected n_jobs;
 *   the remaining outputs as in qmc_integrate_sectors. */
int32_t qmc_median_integrate_sectors(qmc_plan_t* plan, const qmc_job* jobs, int32_t n_jobs,
                                     const uint64_t* z_cand, int32_t K, const double* shift0,
                                     const double* shifts, int32_t n_shift_rows, int32_t m,
                                     double* d_cand_est, double* d_median, int32_t* d_selected,
                                     double* d_shift_sums, double* d_job_results,
                                     double* d_amplitude, int64_t* d_diag, void* cuda_stream);

/* ---- sharded evaluation over several GPUs (the paper's distributed evaluation) ----
 * Jobs are independent, the m shifts of a job are independent, and the lattice indices of one (job, shift) split into
 * disjoint ranges whose partial sums add.  A rank evaluates its PIECES of a batch with qmc_integrate_pieces, the
 * per-shift double-double partial sums of all ranks are gathered (one NCCL all-gather of n_jobs x m x J_out x 6 doubles per
 * rank -- the path's only collective), and qmc_finalize_pieces forms sums, mean / error and the amplitude on any rank.
 * paper_2305_19768_b200/ranks.py holds the partition (whole jobs by longest-processing-time-first; a job larger than
 * the mean load is cut by shift, then by k-range). */
typedef struct {             /* HOST */
  int32_t job;               /* index into the jobs array                                               */
  int32_t s0, s1;            /* shifts s0 <= s < s1 of the job's m shifts                                */
  int32_t reserved;
  uint64_t k0, k1;           /* lattice indices k0 <= k < k1 <= n                                        */
} qmc_piece;

/* Evaluates the pieces (sorted by job; pieces of one job must not overlap) and writes, for EVERY job of the batch,
 *   d_partial DEV out  n_jobs x m x J_out x 3 x 2 : (hi, lo) of this rank's part of (Re S, Im S, A)_{s,j}; (0, 0) where
 *                      the rank holds no piece
 *   d_diag    DEV out or NULL  n_jobs x 2 int64 : this rank's part of the counters (they add over the ranks)
 * jobs, shifts, n_shift_rows, m as in qmc_integrate_sectors (all ranks pass the same batch); m >= 1.  The workspace
 * must have been sized for max_jobs >= max(n_jobs, n_pieces) (qmc_plan_workspace_bytes). */
int32_t qmc_integrate_pieces(qmc_plan_t* plan, const qmc_job* jobs /*HOST*/, int32_t n_jobs,
                             const qmc_piece* pieces /*HOST*/, int32_t n_pieces, const double* shifts /*HOST*/,
                             int32_t n_shift_rows, int32_t m, double* d_partial, int64_t* d_diag, void* cuda_stream);

/* Adds the partial sums of n_parts ranks in double-double and finishes steps a4 / a6:
 *   d_parts DEV in  n_parts x (n_jobs x m x J_out x 3 x 2), the d_partial arrays of the ranks one after another
 *   d_shift_sums, d_job_results, d_amplitude (or NULL) as in qmc_integrate_sectors; jobs: n and coef are read. */
int32_t qmc_finalize_pieces(qmc_plan_t* plan, const qmc_job* jobs /*HOST*/, int32_t n_jobs, int32_t m,
                            const double* d_parts, int32_t n_parts, double* d_shift_sums, double* d_job_results,
                            double* d_amplitude, void* cuda_stream);

/* The median rule (step a5) of a sharded batch.  The candidate stage is a batch of n_jobs x K one-shift "candidate
 * jobs" -- cand_jobs[i K + c]: sector and n of job i, z = candidate c of job i, shift_offset = the row that holds job i's
 * shared shift -- which the ranks evaluate with qmc_integrate_pieces (m = 1; any split by candidate and k-range) and
 * all-gather.  This call adds the parts in double-double and selects exactly as qmc_median_rule does; every rank that
 * runs it on the same gathered parts gets the same selection.  The m-shift stage then runs on the selected vectors
 * through qmc_integrate_pieces / qmc_finalize_pieces.
 *   cand_jobs  HOST n_jobs x K (sector and n are read; the K jobs of one job must agree in both)
 *   d_parts    DEV in  n_parts x (n_jobs K x 1 x J_out x 3 x 2)
 *   d_cand_est DEV out n_jobs x K x J_out x 2    d_median DEV out n_jobs x J_out x 2    d_selected DEV out n_jobs */
int32_t qmc_median_select_pieces(qmc_plan_t* plan, const qmc_job* cand_jobs /*HOST*/, int32_t n_jobs, int32_t K,
                                 const double* d_parts, int32_t n_parts, double* d_cand_est, double* d_median,
                                 int32_t* d_selected, void* cuda_stream);

/* ---- presampling of the deformation parameter ---------------------------------------------
 * "number_of_presamples is the number of samples used for the initial contour deformation parameter selection"
 * (PAPER.md:422).  Reading R-pre: on the n_pre points of one shifted rank-1 lattice (the sector's
 * own transform; points of weight 0 skipped) the candidates lambda_0 = lambda_max, lambda_{j+1} = lambda_j * decrease
 * (while >= lambda_min) are tried in turn; a candidate is admissible if at every point Im F(z(x; lambda_j)) + f_im < 0
 * (the sign check that qmc_integrate_* count in d_diag) and |F| >= min_abs_f; the first admissible one is returned
 * (ok = 1).  If none is admissible, the candidate that passes the sign check everywhere and stays farthest from the
 * zeros of F (largest minimum |F|) is returned with ok = 0; if none passes the sign check, lambda_min with ok = 0.
 * The sector's own `lambda` is ignored; the caller stores the result in the description BEFORE qmc_plan (lambda is
 * compiled into the sector's code).  Synchronises the stream. */
typedef struct {             /* HOST; zero-initialised = defaults                                              */
  double lambda_max;         /* 0 = 1.0                                                                        */
  double decrease;           /* 0 = 0.9; must be < 1                                                           */
  double lambda_min;         /* 0 = 1e-5                                                                       */
  double min_abs_f;          /* 0 = off: smallest |F(z)| a candidate may reach on the presample points          */
} qmc_presample_opts;
typedef struct {             /* HOST out                                                                       */
  double lambda;             /* the selected deformation strength                                               */
  double max_im_f, min_abs_f;/* over the presample points at the selected lambda (NaN if nothing passed the sign check) */
  int32_t steps;             /* candidates rejected before it                                                   */
  int32_t ok;                /* 1: admissible on every presample point; 0: fallback (see above)                 */
} qmc_presample_info;
size_t qmc_presample_scratch_bytes(const qmc_sector_desc* sector /*HOST*/, const qmc_presample_opts* opts);
int32_t qmc_presample_lambda(const qmc_sector_desc* sector /*HOST, deformed*/, uint64_t n_pre,
                             const uint64_t* z /*HOST dim*/, const double* shift /*HOST dim*/,
                             const qmc_presample_opts* opts /*HOST or NULL*/, void* d_scratch /*DEV, 256-byte aligned*/,
                             size_t scratch_bytes, qmc_presample_info* info /*HOST out*/, void* cuda_stream);

/* The same selection for callers that cannot allocate device memory (tight serving loops, harnesses that forbid
 * cudaMalloc, processes in which an allocation would disturb a CUDA graph capture on another stream): no scratch
 * argument.  (The call itself synchronises its stream, so it cannot be captured into a graph.)  The device scratch is
 * a fixed 96 KiB array inside libqmc.so (qmc_presample_static_max_bytes()), which every GPU that loads the library
 * holds until the process exits; the host side works on the stack.  The call allocates neither device nor host memory (no cudaMalloc / cudaFree,
 * no allocating library routine) and returns exactly what qmc_presample_lambda returns for the same arguments.
 *   limit     nF <= QMC_PRESAMPLE_STATIC_MAX_TERMS monomials in F (and, as above, at most 1024 candidates);
 *             a larger sector is refused with QMC_ERR_WORKSPACE -- use qmc_presample_lambda with caller scratch
 *   device    the device of cuda_stream must be current; the array's address is looked up once per device
 *   sharing   all calls on one device use the same array, which keeps the last call's contents: each call resets the
 *             counters and keys it needs, and calls that OVERLAP on the GPU (two streams, two host threads) race --
 *             serialise them.  Synchronises the stream, like qmc_presample_lambda. */
#define QMC_PRESAMPLE_STATIC_MAX_TERMS 4096
size_t qmc_presample_static_max_bytes(void);
int32_t qmc_presample_lambda_static(const qmc_sector_desc* sector /*HOST, deformed*/, uint64_t n_pre,
                                    const uint64_t* z /*HOST dim*/, const double* shift /*HOST dim*/,
                                    const qmc_presample_opts* opts /*HOST or NULL*/, qmc_presample_info* info /*HOST out*/,
                                    void* cuda_stream);

/* ---- adaptive weighted-sum evaluation (Eq. 1-6) --------------------
 * Eq. (6): real-valued lattice sizes n_i that minimise T = sum_i tau_i n_i (Eq. 3) subject to
 * var(A) = sum_i c_abs2_i w_i / n_i^alpha = V (Eq. 4), with var(I_i) = w_i / n_i^alpha (Eq. 2):
 *   lambda = (1/alpha) ((1/V) sum_i (c_abs2_i w_i tau_i^alpha)^(1/(alpha+1)))^((alpha+1)/alpha),
 *   n_i    = (alpha w_i lambda c_abs2_i / tau_i)^(1/(alpha+1)).
 * HOST arrays of n_items doubles; items with w_i c_abs2_i = 0 get n_i = 0.  Pure host arithmetic, no GPU.
 * QMC_ERR_INVALID_ARG for alpha <= 0, V <= 0, tau_i <= 0, negative or non-finite w_i / c_abs2_i. */
int32_t qmc_allocate_lattices(const double* w, const double* tau, const double* c_abs2, int32_t n_items,
                              double alpha, double V, double* n_out);

typedef struct {             /* HOST; zero-initialised = defaults                                        */
  double epsrel, epsabs;     /* stop when err(A_j) <= max(epsabs, epsrel |A_j|) for every order j; at least
                                one must be > 0                                                          */
  double alpha;              /* 0 = 2, "chosen conservatively"                            */
  double growth_max;         /* 0 = 64: largest factor by which one round may raise an n_i              */
  double safety;             /* 0 = 0.5: Eq. (6) is asked for safety * V_j, so that the rounding-up of the
                                last round does not leave a tail of tiny top-up rounds                   */
  uint64_t n_min;            /* 0 = 10^4; the first prime >= n_min is used                */
  uint64_t n_max;            /* 0 = 4294967291, the largest prime below 2^32                             */
  uint64_t seed;             /* seed of the counter-based generator of shifts and candidate vectors      */
  int32_t max_rounds;        /* 0 = 12                                                                   */
  int32_t m;                 /* shifts per evaluation, 0 = 32                                            */
  int32_t K;                 /* median-rule candidates per new lattice, 0 = 11            */
  int32_t measure_tau;       /* 1 (and tau = NULL): tau_i is measured on-line, as the paper does: after
                                every round tau_i = tile clocks of integral i / its evaluations (qmc_plan_last_job_clocks);
                                0: tau_i as passed, or the emitted FP64 instruction count (deterministic)  */
} qmc_adaptive_opts;

typedef struct {             /* HOST out                                                                 */
  int32_t rounds;            /* evaluation rounds done                                                   */
  int32_t converged;         /* 1: every order met its target                                            */
  int64_t evaluations;       /* integrand evaluations spent, candidates included                         */
} qmc_adaptive_info;

/* Device scratch (caller-owned) qmc_adaptive_integrate needs for n_jobs jobs; the plan's workspace must be
 * bound for max_jobs = n_jobs (K + 1) and max_shift_rows = n_jobs (m + 1). */
size_t qmc_adaptive_scratch_bytes(const qmc_plan_t* plan, int32_t n_jobs, const qmc_adaptive_opts* opts);

/* Evaluates A_j = sum_i C_i I_ij to a requested precision, choosing the lattice size of every integral by
 * Eq. (6) (DESIGN.md section 11 lists the readings):  every job starts on the first prime >= n_min; a round
 * (i) draws, for each job whose lattice changed, K candidate generating vectors, one candidate shift and m
 * shifts from the counter-based generator, (ii) runs the median rule and the m-shift integration on the GPU
 * (qmc_median_integrate_sectors), (iii) reads the job results back, forms A_j and var(A_j) (Eq. 4),
 * w_ij = var(I_ij) n_i^alpha, and (iv) applies Eq. (6) order by order ("first for the first sum, then updates
 * n_i and applies it to the next") with tau_i and |C_i|^2; n_i never decreases.  It stops when all
 * targets are met, when no n_i can grow, or after max_rounds.  This call synchronises the stream every round.
 *   jobs       HOST n_jobs: sector and coef_re / coef_im are read; n, z, shift_offset are ignored
 *   tau        HOST n_jobs or NULL: relative cost of one evaluation of job i; NULL = the emitted FP64
 *              instruction count of its sector (qmc_plan_sector_ops), or, with opts.measure_tau = 1, the cost measured
 *              while the integral is being evaluated
 *   d_scratch  DEV, qmc_adaptive_scratch_bytes
 *   job_results HOST out n_jobs x J_out x 4; amplitude HOST out J_out x 4 (re, im, err_re, err_im);
 *   n_final HOST out n_jobs; z_final HOST out n_jobs x QMC_MAX_DIM (the selected vectors); any may be NULL. */
int32_t qmc_adaptive_integrate(qmc_plan_t* plan, const qmc_job* jobs, int32_t n_jobs, const double* tau,
                               const qmc_adaptive_opts* opts, void* d_scratch, size_t scratch_bytes,
                               double* job_results, double* amplitude, uint64_t* n_final, uint64_t* z_final,
                               qmc_adaptive_info* info, void* cuda_stream);

/* Step a1 alone, for the bit-exact check: r[(k-k0)*dim + i] = (k z_i) mod n for k0 <= k < k0+count,
 * produced by the same device functions (Barrett start + modular increment) the kernels use. */
int32_t qmc_debug_lattice_coords(uint64_t n, const uint64_t* z /*HOST dim*/, int32_t dim,
                                 uint64_t k0, uint64_t count, uint64_t* d_out /*DEV*/,
                                 void* cuda_stream);
/* Steps a1-a3 + the integrand at single lattice points, through the plan's compiled sector
 * code (per-point parity): for k in ks[0..count): d_out[c*(2*QMC_MAX_DIM+1+2*J_out) ...] =
 *   t[QMC_MAX_DIM], x[QMC_MAX_DIM], W, then J_out pairs (Re W g_j, Im W g_j). */
int32_t qmc_debug_eval_points(qmc_plan_t* plan, int32_t sector, uint64_t n, const uint64_t* z,
                              const double* shift /*HOST QMC_MAX_DIM*/, const uint64_t* ks /*HOST*/,
                              int32_t count, double* d_out /*DEV*/, void* cuda_stream);

/* Lookup tables of the library's own FP64 elementary functions (csrc/qmc_math.cuh), as embedded in
 * every compiled module, for inspection and tests.  HOST out: log_tab[2050] = pairs (c_i, L_i),
 * i = 0..1024, with c_i = fl(1/(1 + i/1024)) and L_i = -log(c_i) - (i > 424) log 2;
 * exp_tab[256] = 2^(j/256); trig_tab[512] = pairs (cos, sin)(2 pi j/256).  Any pointer may be NULL. */
int32_t qmc_debug_math_tables(double* log_tab, double* exp_tab, double* trig_tab);

/* Sustained FP64 FMA rate of the current device in flop/s (dependent-chain-free DFMA loop on
 * every SM for about `millis` ms): the measured denominator of the "fraction of FP64 peak". */
int32_t qmc_measure_fp64_peak(double millis, double* flops_out /*HOST*/, void* cuda_stream);
/* The same loop with one independent integer add interleaved after every FMA (measured: within 1 % of the pure rate
 * on B200 -- the integer pipe is free beside the FP64 pipe in a regular instruction stream).  Reported beside the pure
 * peak, never instead of it. */
int32_t qmc_measure_fp64_peak_mixed(double millis, double* flops_out /*HOST*/, void* cuda_stream);

/* Launch statistics of the most recent integrate / median call on this plan (HOST out):
 * kernels launched, tiles, evaluations. */
typedef struct { int64_t kernel_launches, tiles, evaluations, eval_kernel_launches; } qmc_launch_stats;
int32_t qmc_plan_last_stats(const qmc_plan_t* plan, qmc_launch_stats* out);
/* Device time of the evaluation kernels of the most recent call in ms (CUDA events on the
 * streams they ran on; synchronises those events).  Needs opts-independent event recording,
 * always on. */
int32_t qmc_plan_last_eval_ms(qmc_plan_t* plan, float* ms_out);

/* SM clock cycles that CTAs spent in the tiles of each job of the most recent integrate / median call (HOST out;
 * waits for that call): rows 0 .. n_jobs-1 are the jobs' m-shift stage; for the median calls rows n_jobs .. 2 n_jobs-1
 * are the jobs' candidate stage.  clocks_i / evaluations_i is the measured cost tau_i of one evaluation of integral i
 * (in CTA-cycles), "estimated on-line ... by tracking how fast a given integral is being evaluated". */
int32_t qmc_plan_last_job_clocks(qmc_plan_t* plan, int64_t* clocks /*HOST n_rows*/, int32_t n_rows);

/* Rare-path counters of the most recent integrate / median call on this plan (HOST out; waits for that call to
 * finish): checked_evals = deformed-class evaluations re-done by the range-guarded out-of-line evaluator because an
 * argument left the fast range of log / exp / atan2 / sincos (|Re(p Log U + q Log F)| > 690, |Im| > 1e5, |U|^2 or
 * |F|^2 subnormal or infinite); slow_calls = calls of the CUDA-library fallbacks inside the guarded functions (both
 * classes).  Both are 0 on every BASELINE.json config.  Either pointer may be NULL. */
int32_t qmc_plan_slow_path_counts(qmc_plan_t* plan, int64_t* checked_evals, int64_t* slow_calls);

void qmc_plan_destroy(qmc_plan_t* plan);
const char* qmc_status_str(int32_t status);  /* static string */
const char* qmc_last_error(void);            /* thread-local detail of the last failure */

#ifdef __cplusplus
}
#endif
#endif /* QMC_H_ */
