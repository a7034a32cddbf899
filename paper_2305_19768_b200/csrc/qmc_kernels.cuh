// =====================================================================================
// qmc_kernels.cuh -- the two kernels of a plan module, appended after the generated sector
// structs (qmc_codegen.cpp) in the NVRTC program.  QMC_SECTOR_CASES(BODY) is generated too and
// expands to   case i: { BODY(Sector_i) } break;   for every sector of the module.
// =====================================================================================
// ------------------------------------------------------------------------------------ a6
// Persistent kernel of one plan module.  QMC_SECTOR_CASES(BODY) expands to
//   case i: BODY(Sector_i) break;   for the sectors compiled into this module.
#define QMC_TILE_CASE(S) qmc_tile_body<S>(ctx, ks0, ks1, tile_acc, red, diag_sh);
extern "C" __global__ void __launch_bounds__(QMC_THREADS, QMC_MIN_CTAS) qmc_eval_kernel(const QmcLaunchArgs a) {
    __shared__ QmcTileCtx ctx;
    __shared__ double red[QMC_WARPS * QMC_NCOMP * 2];
    __shared__ double tile_acc[QMC_NCOMP * 2];   // the tile's (hi, lo) sums, read and written by thread 0 only
    __shared__ u32 s_tile;
    __shared__ u32 diag_sh[3];   // zero-weight points, Im F >= 0 points, evaluations re-done by eval_checked
    qmc_math_init();
    for (;;) {
        __syncthreads();
        if (threadIdx.x == 0) {
            s_tile = a.tile_lo + atomicAdd(a.tile_counter, 1u);
            diag_sh[0] = 0u; diag_sh[1] = 0u; diag_sh[2] = 0u; qmc_sh_slow = 0u;
#pragma unroll
            for (int c = 0; c < QMC_NCOMP * 2; ++c) tile_acc[c] = 0.0;
        }
        __syncthreads();
        const u32 tile = s_tile;
        if (tile >= a.tile_hi) break;
        const long long tile_t0 = clock64();
        if (threadIdx.x < 32) qmc_setup_tile(a, tile, ctx);
        __syncthreads();
        // the tile in chunks of QMC_CHUNK points per thread (a4: bounded plain-FP64 chains, see qmc_tile_body)
        for (u64 ks0 = ctx.k0; ks0 < ctx.k1; ks0 += (u64)QMC_CHUNK * QMC_THREADS) {
            const u64 rest = ctx.k1 - ks0;
            const u64 ks1 = ks0 + (rest < (u64)QMC_CHUNK * QMC_THREADS ? rest : (u64)QMC_CHUNK * QMC_THREADS);
            switch (ctx.sector_case) { QMC_SECTOR_CASES(QMC_TILE_CASE) default: break; }
            __syncthreads();   // red[] is reused by the next chunk's block reduction
        }
        if (threadIdx.x == 0) {
            double* out = a.partials + (u64)tile * (QMC_NCOMP * 2);
#pragma unroll
            for (int c = 0; c < QMC_NCOMP * 2; ++c) out[c] = tile_acc[c];
            atomicAdd(&a.job_clocks[ctx.diag_slot], (u64)(clock64() - tile_t0));   // "tracking how fast a given integral is being evaluated"
            if (diag_sh[0]) atomicAdd(&a.diag[(u64)ctx.diag_slot * 2 + 0], (u64)diag_sh[0]);
            if (diag_sh[1]) atomicAdd(&a.diag[(u64)ctx.diag_slot * 2 + 1], (u64)diag_sh[1]);
            if (diag_sh[2]) atomicAdd(&a.diag[(u64)a.rare_row * 2 + 0], (u64)diag_sh[2]);
            if (qmc_sh_slow) atomicAdd(&a.diag[(u64)a.rare_row * 2 + 1], (u64)qmc_sh_slow);
        }
    }
}

#define QMC_DEBUG_CASE(S) qmc_debug_point<S>((qmc_idx)n, barrett, inv_n, z, delta, ks[i], out + (u64)i * (2 * QMC_DEV_MAX_DIM + 1 + 2 * QMC_JOUT));
extern "C" __global__ void qmc_debug_points_kernel(u32 sector_case, u64 n, u64 barrett, double inv_n, const u64* z,
                                                   const double* delta, const u64* ks, int count, double* out) {
    qmc_math_init();
    if (threadIdx.x == 0) qmc_sh_slow = 0u;
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= count) return;
    switch (sector_case) { QMC_SECTOR_CASES(QMC_DEBUG_CASE) default: break; }
}
