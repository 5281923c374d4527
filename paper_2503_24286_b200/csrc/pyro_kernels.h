// Launch interface between the C-ABI layer (pyro_api.cpp) and the kernels (pyro_kernels.cu).
#pragma once
#include <cuda_runtime.h>

#include <cstddef>
#include <cstdint>

#include "pyro_jac_tables.h"
#include "pyro_tables.h"

namespace pyro {

constexpr int kRatesMaxThreads = 256;   // threads (= points) per block of the rates kernel, a multiple of 32

struct RatesArgs {
    int64_t n, ld, n_chunks;     // n_chunks = ceil(n / 32): a warp takes 32 consecutive points at a time
    unsigned long long *work;    // device counter of the chunks handed out, zero at launch
    const double *rho, *T, *Y;
    double *omega;
    const unsigned char *gtab;   // device copy of the table blob in global memory
    uint32_t tab_bytes;          // blob size (a multiple of 16)
    uint32_t planes_off;         // byte offset of the A (and B) planes in dynamic shared memory
    uint32_t tmem_cols;          // tensor-memory columns the block allocates (a power of two >= 32)
    uint32_t off_spec, off_rxn_p, off_rxn_x, off_fall, off_eff;
    int32_t n_species;
    GroupCounts groups;
    // fused temperature + rates kernel only (pyro_source_terms): T is solved from (e, Y, T_guess) and written to T_out
    const double *e, *T_guess;
    double *T_out;
    int32_t *n_not_converged;
    const EnergyRow *energy;
    double tol, t_mid;
    int32_t max_iter, single_t_mid;
};

struct TempArgs {
    int64_t n, ld;
    const double *e, *Y, *T_guess;
    double *T;
    int32_t *n_not_converged;
    const EnergyRow *energy;     // device, [n_species]
    int32_t n_species, max_iter;
    double t_mid, tol;
    int32_t enthalpy;            // 0: e given, Newton with c_v (A.27); 1: h given, Newton with c_p
    int32_t single_t_mid;        // 1: every species switches NASA range at t_mid (streaming kernels); 0: general kernel
};

struct EosArgs {                 // (A.2)-(A.3): out = in / (Rm T) (density from pressure) or in Rm T (pressure from density)
    int64_t n, ld;
    const double *in, *T, *Y;
    double *out;
    const EnergyRow *energy;
    int32_t n_species, to_density;
};

struct ReactorArgs {             // batched RK4 reactor march (pyro_reactor_rk4)
    RatesArgs rates;             // tables, launch shape, rho, e, Newton controls, energy table, n_not_converged (Y, T, omega unused)
    double *Y;                   // [n_species][ld] state, in/out
    double *T;                   // [n] guess in, temperature of the final state out
    double *acc;                 // [n_species][ld] scratch: running sum of the weighted stage slopes
    double dt;
    int32_t n_steps;
    uint32_t energy_smem_off;    // byte offset of the staged energy table in dynamic shared memory (0: read it from global memory)
};

const void *reactor_kernel_ptr(bool tables_in_shared, bool b_in_tmem, bool singles);
cudaError_t launch_reactor(const ReactorArgs &a, int threads, int blocks, bool tables_in_shared, bool b_in_tmem, bool singles,
                           size_t smem_bytes, cudaStream_t stream);

// pyro_reactor_rk4_static: acc and rates.work are taken from the library's built-in device array (pyro_reactor_kernels.cu)
cudaError_t launch_reactor_static(const ReactorArgs &a, int device, int threads, int blocks, bool tables_in_shared, bool b_in_tmem,
                                  bool singles, size_t smem_bytes, cudaStream_t stream, const char **failed_at);

struct CnArgs {                  // implicit (Crank-Nicolson) reactor march: per-point linear algebra (pyro_cn_kernels.cu)
    int64_t n, ld;
    const double *rho, *omega;   // [n], [n_species][ld] rates at the current Newton iterate
    double *Y;                   // current iterate, updated in place
    double *Ym, *Sm, *F;         // [n_species][ld] each: state and right-hand side at the old time level, Newton residual / update
    double *J;                   // Jacobian in, LU factors out; blocked layout: element (i, k) of point p at
                                 // ((p / jblock) n_s^2 + i n_s + k) jblock + p % jblock
    int64_t jblock;
    double *last_update;         // [n] or NULL: max_k |dY_k| of this iteration
    int32_t *n_not_converged;
    const EnergyRow *energy;     // W_k
    double dt, update_tol;
    int32_t n_species, count_unconverged;
};
int cn_block_threads(int n_species);   // threads (= points) per block of cn_newton_kernel = the Jacobian's point block
cudaError_t launch_cn_begin_step(const CnArgs &a, cudaStream_t stream);
cudaError_t launch_cn_newton(const CnArgs &a, cudaStream_t stream);

constexpr int kJacMaxThreads = 128;
constexpr size_t kJacRingBytes = 8192;  // per warp: two segments of 32 records of up to 128 bytes (RecordRing)     // threads (= points) per block of the Jacobian kernel: one warp per tensor-memory lane quarter

struct JacArgs {                 // chemical Jacobian (pyro_jac_tables.h)
    int64_t n, ld, n_chunks;
    unsigned long long *work;    // chunk counter, zero at launch
    const double *rho, *T, *Y;
    double *J, *dSdT;            // J[(i n_s + k) ld + p]; dSdT[i ld + p] or NULL
    const unsigned char *gtab;   // rates blob (species rows at off_spec)
    const EnergyRow *energy;
    const unsigned char *jtab;   // Jacobian blob
    double *ext;                 // scratch of the [M] reactions: [1 + 2 n_ext][threads of the grid]
    uint32_t off_spec, tmem_cols;
    uint32_t planes_bytes;       // dynamic shared memory taken by the planes; the per-warp record rings (8 KB each) follow
    int32_t mode;                // 0: fixed (rho, T); 1: fixed (rho, e)
    int32_t ext_global;          // block kernel: the [M] scratch is ext[block][slot][32] in global memory, not in shared memory
    int64_t jblock;              // 0: J[(i n_s + k) ld + p]; else blocks of jblock points with contiguous matrices (implicit march)
    JacLayout lay;
};

constexpr size_t kJacBlockRingBytes = 4096;   // block kernel: per warp two segments of 16 records of up to 128 bytes
const void *jacobian_block_kernel_ptr(int warps);   // 16 or 8 warps on one chunk of 32 points (pyro_jac_block_kernels.cu)
cudaError_t launch_jacobian_block(const JacArgs &a, int warps, int blocks, size_t smem_bytes, cudaStream_t stream);
const void *jacobian_kernel_ptr(bool small);
cudaError_t launch_jacobian(const JacArgs &a, bool small, int threads, int blocks, size_t smem_bytes, cudaStream_t stream);

constexpr int kRates2Threads = 128;     // threads per block of the two-points-per-thread rates kernel (256 points)
const void *rates2_kernel_ptr(bool tables_in_shared, bool singles);
cudaError_t launch_rates2(const RatesArgs &a, int threads, int blocks, bool tables_in_shared, bool singles, size_t smem_bytes, cudaStream_t stream);
const void *rates_kernel_ptr(bool tables_in_shared, bool b_in_tmem, bool two_blocks);
const void *fused_kernel_ptr(bool tables_in_shared, bool b_in_tmem, bool two_blocks);
const void *temperature_kernel_ptr();
cudaError_t launch_rates(const RatesArgs &a, int threads, int blocks, bool tables_in_shared, bool b_in_tmem,
                         bool two_blocks, size_t smem_bytes, cudaStream_t stream, bool fused = false);
cudaError_t launch_temperature(const TempArgs &a, cudaStream_t stream);
cudaError_t launch_eos(const EosArgs &a, cudaStream_t stream);
cudaError_t launch_dfma_probe(double *out, int iters, int blocks, cudaStream_t stream);

}   // namespace pyro
