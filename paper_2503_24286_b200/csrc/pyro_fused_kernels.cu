// Instantiations of the fused temperature + rates kernel (rates_kernel<..., kFused = true>, pyro_rates_kernel.cuh):
// SURVEY.md 8(f) NEXT-1, (rho, e, Y, T_guess) -> (T, omega) in one launch.  A translation unit of
// its own so that the plain rates kernel's code is untouched by it.
#include "pyro_rates_kernel.cuh"

namespace pyro {

const void *fused_kernel_ptr(bool tables_in_shared, bool b_in_tmem, bool two_blocks) {
    if (two_blocks) {
        if (tables_in_shared)
            return b_in_tmem ? (const void *)rates_kernel<true, true, 2, true> : (const void *)rates_kernel<true, false, 2, true>;
        return b_in_tmem ? (const void *)rates_kernel<false, true, 2, true> : (const void *)rates_kernel<false, false, 2, true>;
    }
    if (tables_in_shared)
        return b_in_tmem ? (const void *)rates_kernel<true, true, 1, true> : (const void *)rates_kernel<true, false, 1, true>;
    return b_in_tmem ? (const void *)rates_kernel<false, true, 1, true> : (const void *)rates_kernel<false, false, 1, true>;
}

}   // namespace pyro
