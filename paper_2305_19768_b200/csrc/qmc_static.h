// qmc_static.h -- host launchers of the nvcc-compiled kernels in qmc_static.cu.
#ifndef QMC_STATIC_H_
#define QMC_STATIC_H_

#include <cuda_runtime_api.h>
#include <stddef.h>
#include <stdint.h>

#include "qmc_job_dev.h"

namespace qmc {

cudaError_t launch_lattice_debug(uint64_t n, uint64_t barrett, const uint64_t* z, int dim, uint64_t k0, uint64_t count,
                                 uint64_t* d_out, cudaStream_t st);
cudaError_t launch_finalize(const QmcFinJob* d_fin, int n_jobs, int jout, const double* d_partials, double* d_shift_sums,
                            double* d_job_results, cudaStream_t st);
cudaError_t launch_piece_sums(const QmcPieceDev* d_pieces, const unsigned int* d_piece_lo, int n_jobs, int m, int jout,
                              const double* d_partials, double* d_out, cudaStream_t st);
cudaError_t launch_finalize_parts(const unsigned long long* d_n, int n_jobs, int m, int jout, const double* d_parts, int n_parts,
                                  size_t part_stride, double* d_shift_sums, double* d_job_results, cudaStream_t st);
struct PresampleHost {          // host-side description of one presampling launch (qmc_presample_lambda)
    int dim, transform, nF, n_cand;
    uint64_t n;
    double f_im, min_abs_f;
    uint64_t z[QMC_DEV_MAX_DIM];
    double shift[QMC_DEV_MAX_DIM];
    double kcoef[8], kinvb;
};
cudaError_t launch_presample(const PresampleHost& h, const double* d_F_coef, const unsigned char* d_F_exp, const double* d_lambdas,
                             unsigned int* d_fail, unsigned long long* d_worst, cudaStream_t st);
// qmc_presample_lambda_static: fixed layout of the file-scope scratch array of qmc_static.cu (96 KiB per device)
constexpr int kPresampleStaticMaxTerms = 4096;    // monomials of F
constexpr int kPresampleMaxCand = 1024;           // candidates lambda_j
constexpr size_t kPsOffCoef = 0;
constexpr size_t kPsOffExp = kPsOffCoef + (size_t)kPresampleStaticMaxTerms * sizeof(double);
constexpr size_t kPsOffLam = kPsOffExp + (size_t)kPresampleStaticMaxTerms * QMC_DEV_MAX_DIM;
constexpr size_t kPsOffFail = kPsOffLam + (size_t)kPresampleMaxCand * sizeof(double);
constexpr size_t kPsOffWorst = kPsOffFail + (size_t)2 * kPresampleMaxCand * sizeof(unsigned int);
constexpr size_t kPresampleStaticBytes = kPsOffWorst + (size_t)2 * kPresampleMaxCand * sizeof(unsigned long long);
static_assert(kPresampleStaticBytes == 96 * 1024 && kPsOffExp % 256 == 0 && kPsOffLam % 256 == 0 && kPsOffFail % 256 == 0 &&
              kPsOffWorst % 256 == 0, "layout of the static presampling scratch");
cudaError_t presample_static_scratch(unsigned char** d_ptr);
cudaError_t launch_presample_static(const PresampleHost& h, const double* h_F_coef, const unsigned char* h_F_exp,
                                    const double* h_lambdas, unsigned int* h_fail, unsigned long long* h_worst, cudaStream_t st);
cudaError_t launch_median_select(const QmcFinJob* d_fin, int n_jobs, int K, int jout, const double* d_cand_sums,
                                 double* d_cand_est, double* d_median, int* d_selected, cudaStream_t st);
cudaError_t launch_amplitude(const double* d_job_results, const double* d_coef, int n_jobs, int jout, double* d_amp,
                             cudaStream_t st);
cudaError_t launch_diag(const unsigned long long* d_diag, int n, long long* d_out, cudaStream_t st);
cudaError_t launch_dfma_peak(int blocks, int iters, cudaStream_t st, bool mixed = false);

}  // namespace qmc
#endif
