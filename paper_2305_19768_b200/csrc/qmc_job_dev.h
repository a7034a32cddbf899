// qmc_job_dev.h -- plain structs shared by the host side of libqmc and the device code.
// No includes: this text is also prepended to the NVRTC program of every plan module.
#ifndef QMC_JOB_DEV_H_
#define QMC_JOB_DEV_H_

#define QMC_DEV_MAX_DIM 8

// One internal job of a launch: a (sector, lattice, shift block) whose (shift, k-range)
// tiles occupy tile ids [tile_base, tile_base + m * tiles_per_shift) of the call.
struct QmcJobDev {
    unsigned long long n;          // lattice size, 1 <= n < 2^32 (or < 2^53 in a wide_lattice plan)
    unsigned long long barrett;    // floor((2^64 - 1) / n)   (32-bit index path)
    double inv_n;                  // 1 / n, correctly rounded
    unsigned int sector_case;      // case label of the sector inside its module's switch
    unsigned int z_row;            // row of the generating vector in the z table (8 x u64 per row)
    int sel_index;                 // >= 0: z_row += selected[sel_index]  (median rule, stage 2)
    unsigned int shift_row;        // first shift row of the job
    unsigned int m;                // number of shifts
    unsigned int tiles_per_shift;  // k-range tiles per shift
    unsigned int tile_points;      // lattice points per tile (last tile of a shift is ragged)
    unsigned int tile_base;        // first tile id of the job within the call
    unsigned int diag_slot;        // row of the int64[2] diagnostics counters
    unsigned int pad_;
    unsigned long long k_begin;    // lattice indices [k_begin, k_end) of this job are evaluated: the whole lattice
    unsigned long long k_end;      // (0, n), or one piece of a job that is shared between ranks
};

// Kernel argument block of the persistent evaluation kernels.
struct QmcLaunchArgs {
    const QmcJobDev* jobs;             // jobs of this module launch, ascending tile_base
    int n_jobs;
    unsigned int tile_lo, tile_hi;     // tile id range of this launch
    const unsigned long long* z_table; // rows x 8
    const int* selected;               // median-rule selections (may be null)
    const double* shifts;              // rows x 8
    double* partials;                  // tiles x (3 * J_out) x 2  (hi, lo)
    unsigned long long* diag;          // rows x 2
    unsigned int rare_row;             // diag row of the call's rare-path counters (checked evaluations, slow calls)
    unsigned long long* job_clocks;    // per diag row: SM clock cycles the CTAs spent in the job's tiles (tau_i)
    unsigned int* tile_counter;        // zeroed before the launch
};

// One piece of a sharded job, read by the piece-sum kernel: shifts [s0, s1) of job `job`, tiles as in QmcFinJob.
struct QmcPieceDev {
    unsigned int job, s0, s1, tile_base, tiles_per_shift, pad_;
};

// Per-output-job record read by the finalize kernel.
struct QmcFinJob {
    unsigned long long n;
    unsigned int tile_base, tiles_per_shift, m, pad_;
};

#endif
