// Launch interface between the C-ABI layer (pyro_api.cpp) and the kernels (pyro_kernels.cu).
#pragma once
#include <cuda_runtime.h>

#include <cstddef>
#include <cstdint>

#include "pyro_tables.h"

namespace pyro {

struct RatesArgs {
    int64_t n, ld;
    const double *rho, *T, *Y;
    double *omega;
    const unsigned char *gtab;   // device copy of the table blob in global memory
    uint32_t off_spec, off_rxn_p, off_rxn_x, off_fall, off_eff_delta, off_eff_species;
    int32_t n_species, n_p, n_x;
    int32_t shape_quads[9], shape_pairs[9], shape_singles[9], ext_count[4];
};

struct TempArgs {
    int64_t n, ld;
    const double *e, *Y, *T_guess;
    double *T;
    int32_t *n_not_converged;
    const EnergyRow *energy;     // device, [n_species]
    int32_t n_species, max_iter;
    double t_mid, tol;
};

// variants: block_threads in {32, 64, 128}, points_per_thread in {1, 2}
const void *rates_kernel_ptr(int block_threads, int points_per_thread, bool tables_in_constant);
const void *temperature_kernel_ptr();
cudaError_t upload_const_table(const void *src_device, size_t bytes, cudaStream_t stream);
cudaError_t launch_rates(const RatesArgs &a, int block_threads, int points_per_thread, bool tables_in_constant,
                         size_t smem_bytes, cudaStream_t stream);
cudaError_t launch_temperature(const TempArgs &a, cudaStream_t stream);
cudaError_t launch_dfma_probe(double *out, int iters, int blocks, cudaStream_t stream);

}   // namespace pyro
