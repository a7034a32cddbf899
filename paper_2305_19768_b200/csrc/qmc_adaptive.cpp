// =====================================================================================
// qmc_adaptive.cpp -- adaptive weighted-sum evaluation (arXiv:2305.19768 section 2.1.3,
// PAPER.md:211-247, Eq. 1-6) on top of the library's own C ABI.
//
//   qmc_allocate_lattices     Eq. (6), closed form, host arithmetic
//   qmc_adaptive_integrate    the round loop: draw lattices and shifts -> median rule + m-shift
//                             integration on the GPU (qmc_median_integrate_sectors) -> read the
//                             job results back -> Eq. (4), Eq. (2) -> Eq. (6) -> next round
// Readings of what the paper leaves open are listed in DESIGN.md section 11 and in include/qmc.h.
// =====================================================================================
#include <cuda_runtime_api.h>

#include <algorithm>
#include <cmath>
#include <cstring>
#include <string>
#include <vector>

#include "qmc.h"

namespace qmc {
int32_t set_error(int32_t code, const std::string& msg);   // qmc_api.cpp: thread-local last error
}

namespace {

typedef unsigned __int128 u128;

// ---- counter-based generator (restated independently by the oracle, oracle/adaptive.py) ----------
uint64_t splitmix64(uint64_t x) {
    x += 0x9E3779B97F4A7C15ull;
    uint64_t z = x;
    z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9ull;
    z = (z ^ (z >> 27)) * 0x94D049BB133111EBull;
    return z ^ (z >> 31);
}
// one 64-bit draw per (seed, round, job, stream, counter); streams: 0 candidate vectors, 1 candidate shift, 2 shifts
uint64_t draw(uint64_t seed, uint64_t round, uint64_t job, uint64_t stream, uint64_t counter) {
    return splitmix64(splitmix64(splitmix64(splitmix64(seed ^ round) ^ job) ^ stream) ^ counter);
}
double draw_shift(uint64_t u) {   // (u >> 11) 2^-53 in [0, 1); a zero is replaced by 2^-53
    const uint64_t v = u >> 11;
    return (double)(v == 0 ? 1 : v) * 0x1.0p-53;
}

// ---- primes -------------------------------------------------------------------------------
uint64_t mulmod(uint64_t a, uint64_t b, uint64_t m) { return (uint64_t)((u128)a * b % m); }
uint64_t powmod(uint64_t a, uint64_t e, uint64_t m) {
    uint64_t r = 1;
    a %= m;
    while (e) { if (e & 1) r = mulmod(r, a, m); a = mulmod(a, a, m); e >>= 1; }
    return r;
}
bool is_prime(uint64_t n) {   // deterministic Miller-Rabin for 64-bit n (first 12 prime bases)
    if (n < 2) return false;
    const uint64_t bases[12] = {2, 3, 5, 7, 11, 13, 17, 19, 23, 29, 31, 37};
    for (uint64_t p : bases) if (n % p == 0) return n == p;
    uint64_t d = n - 1;
    int s = 0;
    while ((d & 1) == 0) { d >>= 1; ++s; }
    for (uint64_t a : bases) {
        uint64_t x = powmod(a, d, n);
        if (x == 1 || x == n - 1) continue;
        bool comp = true;
        for (int r = 1; r < s; ++r) { x = mulmod(x, x, n); if (x == n - 1) { comp = false; break; } }
        if (comp) return false;
    }
    return true;
}
uint64_t next_prime(uint64_t n) { if (n < 2) n = 2; while (!is_prime(n)) ++n; return n; }
uint64_t prev_prime(uint64_t n) { while (n > 2 && !is_prime(n)) --n; return n; }

int32_t allocate(const double* w, const double* tau, const double* c2, int n, double alpha, double V, double* out) {
    double s = 0.0;
    for (int i = 0; i < n; ++i) s += std::pow(c2[i] * w[i] * std::pow(tau[i], alpha), 1.0 / (alpha + 1.0));
    const double lam = (1.0 / alpha) * std::pow(s / V, (alpha + 1.0) / alpha);
    for (int i = 0; i < n; ++i) out[i] = std::pow(alpha * w[i] * lam * c2[i] / tau[i], 1.0 / (alpha + 1.0));
    return QMC_OK;
}

struct Resolved { double epsrel, epsabs, alpha, growth, safety; uint64_t n_min, n_max, seed; int rounds, m, K; };
Resolved resolve(const qmc_adaptive_opts* o) {
    qmc_adaptive_opts z;
    std::memset(&z, 0, sizeof z);
    if (o) z = *o;
    Resolved r;
    r.epsrel = z.epsrel; r.epsabs = z.epsabs;
    r.alpha = z.alpha > 0 ? z.alpha : 2.0;
    r.growth = z.growth_max > 1.0 ? z.growth_max : 64.0;
    r.safety = z.safety > 0 ? z.safety : 0.5;
    r.n_min = z.n_min ? z.n_min : 10000;
    r.n_max = z.n_max ? z.n_max : 4294967291ull;
    r.seed = z.seed;
    r.rounds = z.max_rounds > 0 ? z.max_rounds : 12;
    r.m = z.m > 0 ? z.m : 32;
    r.K = z.K > 0 ? z.K : 11;
    return r;
}

size_t align256(size_t v) { return (v + 255) / 256 * 256; }
struct Scratch { size_t cand_est, median, selected, sums, results, total; };
Scratch scratch_layout(int n_jobs, int J, int m, int K) {
    Scratch s;
    size_t off = 0;
    s.cand_est = off; off = align256(off + (size_t)n_jobs * K * J * 2 * sizeof(double));
    s.median = off;   off = align256(off + (size_t)n_jobs * J * 2 * sizeof(double));
    s.selected = off; off = align256(off + (size_t)n_jobs * sizeof(int32_t));
    s.sums = off;     off = align256(off + (size_t)n_jobs * m * J * 3 * sizeof(double));
    s.results = off;  off = align256(off + (size_t)n_jobs * J * 4 * sizeof(double));
    s.total = off;
    return s;
}

}  // namespace

extern "C" {

int32_t qmc_allocate_lattices(const double* w, const double* tau, const double* c_abs2, int32_t n_items, double alpha,
                              double V, double* n_out) {
    if (!w || !tau || !c_abs2 || !n_out || n_items < 1) return qmc::set_error(QMC_ERR_INVALID_ARG, "qmc_allocate_lattices: null or empty input");
    if (!(alpha > 0) || !(V > 0) || !std::isfinite(alpha) || !std::isfinite(V))
        return qmc::set_error(QMC_ERR_INVALID_ARG, "qmc_allocate_lattices: alpha and V must be positive and finite");
    for (int i = 0; i < n_items; ++i)
        if (!(tau[i] > 0) || !(w[i] >= 0) || !(c_abs2[i] >= 0) || !std::isfinite(tau[i]) || !std::isfinite(w[i]) || !std::isfinite(c_abs2[i]))
            return qmc::set_error(QMC_ERR_INVALID_ARG, "qmc_allocate_lattices: need tau > 0, w >= 0, |C|^2 >= 0, all finite");
    return allocate(w, tau, c_abs2, n_items, alpha, V, n_out);
}

size_t qmc_adaptive_scratch_bytes(const qmc_plan_t* plan, int32_t n_jobs, const qmc_adaptive_opts* opts) {
    if (!plan || n_jobs < 1) return 0;
    const Resolved o = resolve(opts);
    return scratch_layout(n_jobs, qmc_plan_orders(plan), o.m, o.K).total;
}

int32_t qmc_adaptive_integrate(qmc_plan_t* plan, const qmc_job* jobs, int32_t n_jobs, const double* tau_in,
                               const qmc_adaptive_opts* opts, void* d_scratch, size_t scratch_bytes, double* job_results,
                               double* amplitude, uint64_t* n_final, uint64_t* z_final, qmc_adaptive_info* info,
                               void* cuda_stream) {
    if (!plan || !jobs || n_jobs < 1) return qmc::set_error(QMC_ERR_INVALID_ARG, "qmc_adaptive_integrate: null or empty input");
    const Resolved o = resolve(opts);
    if (!(o.epsrel > 0) && !(o.epsabs > 0)) return qmc::set_error(QMC_ERR_INVALID_ARG, "qmc_adaptive_integrate: epsrel or epsabs must be > 0");
    if (o.m < 2 || o.n_min < 3 || o.n_max < o.n_min || o.n_max >= (1ull << 32))
        return qmc::set_error(QMC_ERR_INVALID_ARG, "qmc_adaptive_integrate: need m >= 2 and 3 <= n_min <= n_max < 2^32");
    const int J = qmc_plan_orders(plan), m = o.m, K = o.K;
    const Scratch S = scratch_layout(n_jobs, J, m, K);
    if (!d_scratch || scratch_bytes < S.total) return qmc::set_error(QMC_ERR_WORKSPACE, "qmc_adaptive_integrate: scratch too small");
    cudaStream_t stream = static_cast<cudaStream_t>(cuda_stream);
    char* ds = static_cast<char*>(d_scratch);

    const bool measure_tau = (!tau_in && opts && opts->measure_tau != 0);
    std::vector<double> tau(n_jobs), c2(n_jobs);
    for (int i = 0; i < n_jobs; ++i) {
        tau[i] = tau_in ? tau_in[i] : qmc_plan_sector_ops(plan, jobs[i].sector);
        if (!(tau[i] > 0) || !std::isfinite(tau[i])) return qmc::set_error(QMC_ERR_INVALID_ARG, "qmc_adaptive_integrate: tau must be positive");
        c2[i] = jobs[i].coef_re * jobs[i].coef_re + jobs[i].coef_im * jobs[i].coef_im;
    }
    const uint64_t n_hi = prev_prime(o.n_max);
    std::vector<uint64_t> n(n_jobs, std::min(next_prime(o.n_min), n_hi));
    std::vector<uint64_t> n_done(n_jobs, 0);                      // lattice of the latest result of every job
    std::vector<char> need(n_jobs, 1);
    std::vector<double> res((size_t)n_jobs * J * 4, 0.0);          // latest result of every job
    std::vector<uint64_t> zsel((size_t)n_jobs * QMC_MAX_DIM, 0);
    std::vector<double> amp((size_t)J * 4, 0.0);
    int64_t evals = 0;
    int rounds = 0, converged = 0;

    for (int round = 0; round < o.rounds; ++round) {
        // ---- the jobs whose lattice changed, with fresh candidates and shifts --------------------
        std::vector<int> batch;
        for (int i = 0; i < n_jobs; ++i) if (need[i]) batch.push_back(i);
        if (batch.empty()) break;
        const int nb = (int)batch.size();
        std::vector<qmc_job> bj(nb);
        std::vector<uint64_t> zc((size_t)nb * K * QMC_MAX_DIM, 0);
        std::vector<double> sh0((size_t)nb * QMC_MAX_DIM, 0.0), sh((size_t)nb * m * QMC_MAX_DIM, 0.0);
        for (int b = 0; b < nb; ++b) {
            const int i = batch[b];
            bj[b] = jobs[i];
            bj[b].n = n[i];
            bj[b].shift_offset = b * m;
            for (int c = 0; c < K; ++c)
                for (int k = 0; k < QMC_MAX_DIM; ++k)
                    zc[((size_t)b * K + c) * QMC_MAX_DIM + k] = 1 + draw(o.seed, round, i, 0, (uint64_t)c * 8 + k) % (n[i] - 1);
            for (int k = 0; k < QMC_MAX_DIM; ++k) sh0[(size_t)b * QMC_MAX_DIM + k] = draw_shift(draw(o.seed, round, i, 1, k));
            for (int s = 0; s < m; ++s)
                for (int k = 0; k < QMC_MAX_DIM; ++k)
                    sh[((size_t)b * m + s) * QMC_MAX_DIM + k] = draw_shift(draw(o.seed, round, i, 2, (uint64_t)s * 8 + k));
            for (int k = 0; k < QMC_MAX_DIM; ++k) bj[b].z[k] = zc[(size_t)b * K * QMC_MAX_DIM + k];
            evals += (int64_t)n[i] * (K + m);
        }
        int32_t rc = qmc_median_integrate_sectors(plan, bj.data(), nb, zc.data(), K, sh0.data(), sh.data(), nb * m, m,
                                                  reinterpret_cast<double*>(ds + S.cand_est), reinterpret_cast<double*>(ds + S.median),
                                                  reinterpret_cast<int32_t*>(ds + S.selected), reinterpret_cast<double*>(ds + S.sums),
                                                  reinterpret_cast<double*>(ds + S.results), nullptr, nullptr, cuda_stream);
        if (rc != QMC_OK) return rc;
        std::vector<double> bres((size_t)nb * J * 4);
        std::vector<int32_t> bsel(nb);
        if (cudaMemcpyAsync(bres.data(), ds + S.results, bres.size() * sizeof(double), cudaMemcpyDeviceToHost, stream) != cudaSuccess ||
            cudaMemcpyAsync(bsel.data(), ds + S.selected, bsel.size() * sizeof(int32_t), cudaMemcpyDeviceToHost, stream) != cudaSuccess ||
            cudaStreamSynchronize(stream) != cudaSuccess)
            return qmc::set_error(QMC_ERR_CUDA, std::string("qmc_adaptive_integrate: ") + cudaGetErrorString(cudaGetLastError()));
        if (measure_tau) {
            // tau_i "estimated on-line ... by tracking how fast a given integral is being evaluated":
            // CTA-cycles of the integral's tiles (m-shift stage + candidate stage) per evaluation, this round
            std::vector<int64_t> clk((size_t)2 * nb);
            rc = qmc_plan_last_job_clocks(plan, clk.data(), 2 * nb);
            if (rc != QMC_OK) return rc;
            for (int b = 0; b < nb; ++b) {
                const double t = (double)(clk[b] + clk[(size_t)nb + b]) / ((double)n[batch[b]] * (K + m));
                if (t > 0 && std::isfinite(t)) tau[batch[b]] = t;
            }
        }
        for (int b = 0; b < nb; ++b) {
            const int i = batch[b];
            std::memcpy(&res[(size_t)i * J * 4], &bres[(size_t)b * J * 4], (size_t)J * 4 * sizeof(double));
            n_done[i] = n[i];
            for (int k = 0; k < QMC_MAX_DIM; ++k) zsel[(size_t)i * QMC_MAX_DIM + k] = zc[((size_t)b * K + bsel[b]) * QMC_MAX_DIM + k];
        }
        ++rounds;

        // ---- A_j, var(A_j) (Eq. 4 with the measured variances), targets ---------------------------
        bool all_met = true;
        std::vector<double> Vt(J);
        for (int j = 0; j < J; ++j) {
            double are = 0, aim = 0, vre = 0, vim = 0;
            for (int i = 0; i < n_jobs; ++i) {
                const double* r = &res[((size_t)i * J + j) * 4];
                const double cr = jobs[i].coef_re, ci = jobs[i].coef_im;
                are += cr * r[0] - ci * r[1];
                aim += cr * r[1] + ci * r[0];
                vre += cr * cr * r[2] * r[2] + ci * ci * r[3] * r[3];
                vim += ci * ci * r[2] * r[2] + cr * cr * r[3] * r[3];
            }
            amp[j * 4 + 0] = are; amp[j * 4 + 1] = aim; amp[j * 4 + 2] = std::sqrt(vre); amp[j * 4 + 3] = std::sqrt(vim);
            const double target = std::max(o.epsabs, o.epsrel * std::hypot(are, aim));
            Vt[j] = target * target;
            if (!(vre + vim <= Vt[j])) all_met = false;
        }
        if (all_met) { converged = 1; break; }

        // ---- Eq. (2): w_ij = var(I_ij) n_i^alpha; Eq. (6) order by order; n_i never decreases ------
        std::vector<double> want(n_jobs), w(n_jobs), cand(n_jobs);
        for (int i = 0; i < n_jobs; ++i) want[i] = (double)n[i];
        for (int j = 0; j < J; ++j) {
            double any = 0;
            for (int i = 0; i < n_jobs; ++i) {
                const double* r = &res[((size_t)i * J + j) * 4];
                w[i] = (r[2] * r[2] + r[3] * r[3]) * std::pow((double)n_done[i], o.alpha);
                any += w[i] * c2[i];
            }
            if (!(any > 0)) continue;
            allocate(w.data(), tau.data(), c2.data(), n_jobs, o.alpha, o.safety * Vt[j], cand.data());
            for (int i = 0; i < n_jobs; ++i) want[i] = std::max(want[i], cand[i]);
        }
        bool any_grow = false;
        for (int i = 0; i < n_jobs; ++i) {
            const double cap = std::min((double)n_hi, o.growth * (double)n[i]);
            const uint64_t t = (uint64_t)std::ceil(std::min(want[i], cap));
            need[i] = 0;
            if (t > n[i]) {
                const uint64_t p = std::min(next_prime(t), n_hi);
                if (p > n[i]) { n[i] = p; need[i] = 1; any_grow = true; }
            }
        }
        if (!any_grow) break;
    }
    if (job_results) std::memcpy(job_results, res.data(), res.size() * sizeof(double));
    if (amplitude) std::memcpy(amplitude, amp.data(), amp.size() * sizeof(double));
    // a job whose n was raised for a round that never ran (max_rounds) reports the lattice of its latest result
    if (n_final) for (int i = 0; i < n_jobs; ++i) n_final[i] = n_done[i];
    if (z_final) std::memcpy(z_final, zsel.data(), zsel.size() * sizeof(uint64_t));
    if (info) { info->rounds = rounds; info->converged = converged; info->evaluations = evals; }
    return QMC_OK;
}

}  // extern "C"
