// sm_100a kernel of the batched reactor march (per-point arithmetic: reactor_rk4_point in
// pyro_point.cuh): millions of independent adiabatic isochoric reactors (A.1) PAPER.md:886-888, classical RK4 at a
// fixed step, one thread per reactor.  Same on-chip layout, tables and chunk scheduling as the rates
// kernel (pyro_rates_kernel.cuh): the stage's mass fractions, then A_k, in shared memory; omega_k and B_k in tensor
// memory; the state Y0 and the running sum of the stage slopes in global memory (the caller's Y and scratch field),
// which a warp touches in 256-byte segments that stay in L2 over the four stages of a step.
#include <mutex>

#include "../../include/pyro.h"
#include "pyro_rates_kernel.cuh"

namespace pyro {

// kOwnScratch (pyro_reactor_rk4_static, end of this file): a.acc is the library's built-in scratch array, laid out
// [n_species][n rounded up to a whole chunk] instead of with the caller's leading dimension.
template <bool kTabSmem, bool kBTmem, bool kSingles, bool kOwnScratch = false>
__global__ void __launch_bounds__(kRatesMaxThreads, kSingles ? 2 : 1) reactor_kernel(const ReactorArgs a) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    __shared__ uint32_t s_tmem_base;
    const RatesArgs &r = a.rates;
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31, nthreads = blockDim.x;
    const int ns = r.n_species;
    const int64_t acc_ld = kOwnScratch ? ((r.n + 31) & ~(int64_t)31) : r.ld;
    if (kTabSmem) {
        const uint4 *src = reinterpret_cast<const uint4 *>(r.gtab);
        uint4 *dst = reinterpret_cast<uint4 *>(smem_raw);
        for (uint32_t i = tid; i < r.tab_bytes / 16u; i += nthreads) dst[i] = src[i];
    }
    // the energy table (128 bytes per species) next to the planes when it fits: the first sweep of a stage reads 13
    // coefficients per species at warp-uniform addresses, which from global memory is one long-scoreboard wait each
    const EnergyRow *energy = r.energy;
    if (a.energy_smem_off != 0u) {
        const uint4 *src = reinterpret_cast<const uint4 *>(r.energy);
        uint4 *dst = reinterpret_cast<uint4 *>(smem_raw + a.energy_smem_off);
        for (uint32_t i = tid; i < (uint32_t)ns * (uint32_t)(sizeof(EnergyRow) / 16); i += nthreads) dst[i] = src[i];
        energy = reinterpret_cast<const EnergyRow *>(smem_raw + a.energy_smem_off);
    }
    if (warp == 0) {
        asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(
                         (uint32_t)__cvta_generic_to_shared(&s_tmem_base)),
                     "r"(r.tmem_cols));
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;");
    }
    asm volatile("tcgen05.fence::before_thread_sync;");
    __syncthreads();
    asm volatile("tcgen05.fence::after_thread_sync;");
    const uint32_t tmem_base = s_tmem_base;
    DevTab tab{kTabSmem ? smem_raw : r.gtab, r.off_spec, r.off_rxn_p, r.off_rxn_x, r.off_fall, r.off_eff};
    const uint32_t planes = (uint32_t)__cvta_generic_to_shared(smem_raw) + r.planes_off;
    const uint32_t rows = (uint32_t)ns + 1u;
    DevMem<kBTmem> mem;
    mem.strideA = 8u * (uint32_t)nthreads;
    mem.baseA = planes + 8u * (uint32_t)tid;
    mem.baseB = mem.baseA + rows * mem.strideA;
    mem.tw = tmem_base + (((uint32_t)(warp & 3) * 32u) << 16) + (uint32_t)(warp >> 2) * (kBTmem ? 4u : 2u) * rows;

    auto grab = [&]() -> int64_t {
        unsigned long long c = 0;
        if (lane == 0) c = atomicAdd(r.work, 1ull);
        return (int64_t)__shfl_sync(0xffffffffu, c, 0);
    };
    for (int64_t chunk = grab(); chunk < r.n_chunks; chunk = grab()) {
        const int64_t p = chunk * 32 + lane;
        // Tail lanes stay in the warp's lockstep (the tensor-memory instructions are warp-collective) but touch no
        // field they do not own: they march a pure-species-0 state, read nothing that a live lane writes, store nothing.
        const bool live = p < r.n;
        const int64_t pc = live ? p : r.n - 1;
        double *Yp = a.Y + pc;
        double *Ap = a.acc + pc;
        double T = a.T[pc];
        const int bad = reactor_rk4_point<kSingles>(
            tab, r.groups, ns, r.single_t_mid != 0, r.t_mid, r.rho[pc], r.e[pc], &T, a.dt, a.n_steps, r.tol, r.max_iter, mem,
            [&](int k) { return live ? Yp[(int64_t)k * r.ld] : (k == 0 ? 1.0 : 0.0); },
            [&](int k, double v) {
                if (live) Yp[(int64_t)k * r.ld] = v;
            },
            [&](int k) { return live ? Ap[(int64_t)k * acc_ld] : 0.0; },
            [&](int k, double v) {
                if (live) Ap[(int64_t)k * acc_ld] = v;
            },
            [&](int k) -> const EnergyRow & { return energy[k]; });
        if (live) {
            a.T[p] = T;
            if (r.n_not_converged != nullptr && bad) atomicAdd(r.n_not_converged, bad);
        }
    }
    asm volatile("tcgen05.fence::before_thread_sync;");
    __syncthreads();
    if (warp == 0)
        asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tmem_base), "r"(r.tmem_cols));
}

const void *reactor_kernel_ptr(bool tables_in_shared, bool b_in_tmem, bool singles) {
    if (singles) {
        if (tables_in_shared) return b_in_tmem ? (const void *)reactor_kernel<true, true, true> : (const void *)reactor_kernel<true, false, true>;
        return b_in_tmem ? (const void *)reactor_kernel<false, true, true> : (const void *)reactor_kernel<false, false, true>;
    }
    if (tables_in_shared) return b_in_tmem ? (const void *)reactor_kernel<true, true, false> : (const void *)reactor_kernel<true, false, false>;
    return b_in_tmem ? (const void *)reactor_kernel<false, true, false> : (const void *)reactor_kernel<false, false, false>;
}

cudaError_t launch_reactor(const ReactorArgs &a, int threads, int blocks, bool tables_in_shared, bool b_in_tmem, bool singles,
                           size_t smem_bytes, cudaStream_t stream) {
    ReactorArgs copy = a;
    void *params[] = {&copy};
    return cudaLaunchKernel(reactor_kernel_ptr(tables_in_shared, b_in_tmem, singles), dim3((unsigned)blocks),
                            dim3((unsigned)threads), params, smem_bytes, stream);
}

// ---------------------------------------------------------------------------------------------------------------
// pyro_reactor_rk4_static (include/pyro.h): the same march for callers that have no device memory to lend as `work`
// and no way of getting any.  The stage-slope sums and the chunk counter live in the array below, which is part of
// the library image: the CUDA driver places it on every GPU that loads libpyro.so and keeps it there until the
// process exits, so using it costs no allocation at call time.
//
// g_rk4_static is a __device__ variable.  Inside host functions its name denotes a host-side shadow object, NOT the
// storage on the GPU: handing `g_rk4_static` (or `&g_rk4_static[0]`) to a kernel or to cudaMemsetAsync from host code
// would pass a host address.  The device address comes from cudaGetSymbolAddress, asked once per device with that
// device current (every device has its own copy at its own address), and is what the launch below passes on.
constexpr size_t kRk4StaticHeaderDoubles = 32;   // 256 bytes: [0] the chunk counter of the launch, rest unused
static __device__ __align__(256) double g_rk4_static[kRk4StaticHeaderDoubles + PYRO_RK4_STATIC_MAX_DOUBLES];

namespace {
constexpr int kStaticMaxDevices = 64;
struct Rk4StaticDevice {
    std::once_flag once;
    cudaError_t status = cudaErrorUnknown;
    const char *failed_at = "";
    double *base = nullptr;   // device address of g_rk4_static on this device
};
Rk4StaticDevice g_rk4_static_dev[kStaticMaxDevices];

const void *reactor_static_kernel_ptr(bool tables_in_shared, bool b_in_tmem, bool singles) {
    if (singles) {
        if (tables_in_shared) return b_in_tmem ? (const void *)reactor_kernel<true, true, true, true> : (const void *)reactor_kernel<true, false, true, true>;
        return b_in_tmem ? (const void *)reactor_kernel<false, true, true, true> : (const void *)reactor_kernel<false, false, true, true>;
    }
    if (tables_in_shared) return b_in_tmem ? (const void *)reactor_kernel<true, true, false, true> : (const void *)reactor_kernel<true, false, false, true>;
    return b_in_tmem ? (const void *)reactor_kernel<false, true, false, true> : (const void *)reactor_kernel<false, false, false, true>;
}

// Runs once per device, with that device current: looks up where this device keeps the array and lifts the dynamic
// shared-memory limit of the eight kernel variants to the device maximum (a property of the function, so no later
// call has to touch it).  Neither call allocates.
void rk4_static_setup(Rk4StaticDevice &d) {
    void *p = nullptr;
    d.failed_at = "cudaGetSymbolAddress(g_rk4_static)";
    if ((d.status = cudaGetSymbolAddress(&p, g_rk4_static)) != cudaSuccess) return;
    int dev = 0, optin = 0;
    d.failed_at = "cudaDeviceGetAttribute(MaxSharedMemoryPerBlockOptin)";
    if ((d.status = cudaGetDevice(&dev)) != cudaSuccess) return;
    if ((d.status = cudaDeviceGetAttribute(&optin, cudaDevAttrMaxSharedMemoryPerBlockOptin, dev)) != cudaSuccess) return;
    for (int v = 0; v < 8; ++v) {
        const void *fn = reactor_static_kernel_ptr((v & 1) != 0, (v & 2) != 0, (v & 4) != 0);
        cudaFuncAttributes fa{};
        d.failed_at = "cudaFuncGetAttributes(reactor, built-in scratch)";
        if ((d.status = cudaFuncGetAttributes(&fa, fn)) != cudaSuccess) return;
        d.failed_at = "cudaFuncSetAttribute(reactor, built-in scratch)";
        if ((d.status = cudaFuncSetAttribute(fn, cudaFuncAttributeMaxDynamicSharedMemorySize, optin - (int)fa.sharedSizeBytes)) != cudaSuccess) return;
        if ((d.status = cudaFuncSetAttribute(fn, cudaFuncAttributePreferredSharedMemoryCarveout, cudaSharedmemCarveoutMaxShared)) != cudaSuccess) return;
    }
    d.base = static_cast<double *>(p);
    d.failed_at = "";
}
}   // namespace

// `a` as for launch_reactor except acc and rates.work, which are set here.  `device` is the current device.
cudaError_t launch_reactor_static(const ReactorArgs &a, int device, int threads, int blocks, bool tables_in_shared, bool b_in_tmem,
                                  bool singles, size_t smem_bytes, cudaStream_t stream, const char **failed_at) {
    *failed_at = "device ordinal beyond the built-in scratch bookkeeping";
    if (device < 0 || device >= kStaticMaxDevices) return cudaErrorInvalidDevice;
    Rk4StaticDevice &d = g_rk4_static_dev[device];
    std::call_once(d.once, [&d] { rk4_static_setup(d); });
    *failed_at = d.failed_at;
    if (d.status != cudaSuccess) return d.status;
    ReactorArgs copy = a;
    copy.rates.work = reinterpret_cast<unsigned long long *>(d.base);
    copy.acc = d.base + kRk4StaticHeaderDoubles;
    // The array keeps whatever the last call left in it.  Only the chunk counter has to start at zero; the slope sums
    // are written (stage 2 of a step) before they are read (stages 3, 4 and the update), so they need no clearing.
    *failed_at = "cudaMemsetAsync(chunk counter of the built-in scratch)";
    cudaError_t ce = cudaMemsetAsync(copy.rates.work, 0, sizeof(unsigned long long), stream);
    if (ce != cudaSuccess) return ce;
    *failed_at = "launch of the reactor kernel (built-in scratch)";
    void *params[] = {&copy};
    return cudaLaunchKernel(reactor_static_kernel_ptr(tables_in_shared, b_in_tmem, singles), dim3((unsigned)blocks),
                            dim3((unsigned)threads), params, smem_bytes, stream);
}

}   // namespace pyro
