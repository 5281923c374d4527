// sm_100a kernels of libpyro and their launchers.
//
// Thread mapping: one thread per grid point, a warp reads 256
// contiguous bytes of every species plane of the SoA fields.  Per-point arrays that are
// indexed by a run-time species number live on chip (pyro_tables.h, pyro_point.cuh):
//   A_k = C_k E_k in shared memory as [k][thread] columns (conflict-free: lane l touches its own
//   banks), read-only while the reactions run;
//   omega_k and B_k = 1/E_k in TENSOR MEMORY: thread t of a warp owns lane 32 (warp % 4) + t,
//   species k is the four 32-bit columns 4k .. 4k+3 of that warp's column group (omega_k, B_k).
//   The stoichiometric accumulation is tcgen05.ld / add / tcgen05.st on warp-uniform column
//   addresses, which takes the read-modify-write traffic and the B loads (10 of the 14 indexed
//   accesses of a reaction) off the shared-memory pipe and lets 256 points (8 warps) be
//   resident per SM for the 53-species mechanism.
// The mechanism tables are staged once per block into shared memory and read with 128-bit
// loads at warp-uniform addresses; blocks are persistent (one per SM for the 53-species
// mechanism) and walk the tiles of points.
#include <cuda_runtime.h>

#include "pyro_kernels.h"
#include "pyro_point.cuh"
#include "pyro_rates_kernel.cuh"

namespace pyro {

// ---------------------------------------------------------------------------------------
// T[p] from e[p], Y[k][p], T_guess[p]   (row a4).  One streaming pass over Y builds the
// mixture energy polynomials of both NASA ranges; the Newton iterations then cost O(1).
// Each thread handles PPT points (BD apart, so every load stays coalesced) to amortise
// the warp-uniform reads of the energy table.
// ---------------------------------------------------------------------------------------
template <int BD, int PPT>
__global__ void __launch_bounds__(BD) temperature_kernel(const TempArgs a) {
    const int64_t base = (int64_t)blockIdx.x * (BD * PPT) + threadIdx.x;
    double Slo[PPT][6], Shi[PPT][6], Rm[PPT];
#pragma unroll
    for (int i = 0; i < PPT; ++i) {
        Rm[i] = 0.0;
#pragma unroll
        for (int m = 0; m < 6; ++m) Slo[i][m] = Shi[i][m] = 0.0;
    }
    int64_t pt[PPT];
#pragma unroll
    for (int i = 0; i < PPT; ++i) {
        const int64_t p = base + (int64_t)i * BD;
        pt[i] = p < a.n ? p : a.n - 1;   // tail lanes recompute the last point and store nothing
    }
    const int ns = a.n_species;
    constexpr int kAhead = 8;   // species planes prefetched into L2 ahead of the loads (the loop is latency-bound)
    for (int k = 0; k < ns; ++k) {
        if (k + kAhead < ns && (threadIdx.x & 15) == 0) {
#pragma unroll
            for (int i = 0; i < PPT; ++i)
                asm volatile("prefetch.global.L2 [%0];" ::"l"(a.Y + (int64_t)(k + kAhead) * a.ld + pt[i]));
        }
        double y[PPT];
#pragma unroll
        for (int i = 0; i < PPT; ++i) y[i] = a.Y[(int64_t)k * a.ld + pt[i]];
        const double2 *row = reinterpret_cast<const double2 *>(a.energy + k);
        double c[12];
#pragma unroll
        for (int m = 0; m < 6; ++m) {
            const double2 v = __ldg(row + m);
            c[2 * m] = v.x;
            c[2 * m + 1] = v.y;
        }
#pragma unroll
        for (int i = 0; i < PPT; ++i)
#pragma unroll
            for (int m = 0; m < 6; ++m) {
                Slo[i][m] = fma(y[i], c[m], Slo[i][m]);
                Shi[i][m] = fma(y[i], c[6 + m], Shi[i][m]);
            }
        if (a.enthalpy) {   // h(T) = e(T) + T sum_k Y_k R/W_k
            const double rw = __ldg(&a.energy[k].rw);
#pragma unroll
            for (int i = 0; i < PPT; ++i) Rm[i] = fma(y[i], rw, Rm[i]);
        }
    }
    if (a.enthalpy) {
#pragma unroll
        for (int i = 0; i < PPT; ++i) {
            Slo[i][1] += Rm[i];
            Shi[i][1] += Rm[i];
        }
    }
    int bad = 0;
#pragma unroll
    for (int i = 0; i < PPT; ++i) {
        const int64_t p = base + (int64_t)i * BD;
        double T;
        bool conv;
        newton_temperature(Slo[i], Shi[i], a.t_mid, a.e[pt[i]], a.T_guess[pt[i]], a.tol, a.max_iter, &T, &conv);
        if (p < a.n) {
            a.T[p] = T;
            bad += conv ? 0 : 1;
        }
    }
    if (a.n_not_converged != nullptr && bad) atomicAdd(a.n_not_converged, bad);
}

// ---------------------------------------------------------------------------------------
// Row a4 for mechanisms whose species have different break temperatures (reading G10): one
// thread per point, newton_temperature_general (pyro_point.cuh).  The first pass over Y streams from
// HBM (planes prefetched into L2 ahead of the loads); a repeated pass -- an iterate crossed a break
// temperature -- finds the point's column in L2.
// ---------------------------------------------------------------------------------------
template <int BD>
__global__ void __launch_bounds__(BD) temperature_general_kernel(const TempArgs a) {
    const int64_t p = (int64_t)blockIdx.x * BD + threadIdx.x;
    const int64_t pc = p < a.n ? p : a.n - 1;
    const int ns = a.n_species;
    constexpr int kAhead = 8;
    if ((threadIdx.x & 15) == 0)
        for (int k = 0; k < ns && k < kAhead; ++k) asm volatile("prefetch.global.L2 [%0];" ::"l"(a.Y + (int64_t)k * a.ld + pc));
    const double *Yp = a.Y + pc;
    double T;
    bool conv;
    newton_temperature_general(
        ns,
        [&](int k) {
            if (k + kAhead < ns && (threadIdx.x & 15) == 0)
                asm volatile("prefetch.global.L2 [%0];" ::"l"(Yp + (int64_t)(k + kAhead) * a.ld));
            return Yp[(int64_t)k * a.ld];
        },
        [&](int k) -> const EnergyRow & { return a.energy[k]; }, a.enthalpy != 0, a.e[pc], a.T_guess[pc], a.tol, a.max_iter, &T,
        &conv);
    if (p < a.n) {
        a.T[p] = T;
        if (a.n_not_converged != nullptr && !conv) atomicAdd(a.n_not_converged, 1);
    }
}

// ---------------------------------------------------------------------------------------
// The same solve as a software-pipelined stream (used when the Y planes are 16-byte aligned):
// thread t owns NV pairs of points (2t, 2t+1, then 2 BD further on, ...) of its block's 2 NV BD points and copies
// their 16 bytes of every species plane into its own slots of a D-deep shared-memory ring with cp.async, D
// species ahead of the arithmetic, so that the HBM latency is covered by D x NV x 16 bytes in flight per thread
// instead of by resident warps.  NV = 2: the twelve coefficients of a species serve four points per thread, which
// halves the warp-uniform table reads that bound the NV = 1 version (ncu: 14 of 18 shared-memory wavefronts per
// species and warp).  A thread only ever reads what it copied itself: no barrier
// in the loop.  The energy table is staged in shared memory once per block.
// ---------------------------------------------------------------------------------------
template <int BD, int D, int NV>
__global__ void __launch_bounds__(BD) temperature_stream_kernel(const TempArgs a) {
    static_assert((D & (D - 1)) == 0, "ring depth must be a power of two");
    constexpr int NP = 2 * NV;   // points per thread: NV 16-byte vectors, 2 BD points apart (every copy of a warp is 512 contiguous bytes)
    extern __shared__ __align__(16) unsigned char tsm[];
    EnergyRow *tab = reinterpret_cast<EnergyRow *>(tsm + (size_t)D * NV * BD * 16);
    const int tid = threadIdx.x, ns = a.n_species;
    {
        const double2 *src = reinterpret_cast<const double2 *>(a.energy);
        double2 *dst = reinterpret_cast<double2 *>(tab);
        for (int i = tid; i < ns * (int)(sizeof(EnergyRow) / 16); i += BD) dst[i] = __ldg(src + i);
    }
    const int64_t p0 = (int64_t)blockIdx.x * (BD * NP) + tid * 2;   // the launcher passes whole blocks only
    const double *Yp = a.Y + p0;
    const uint32_t slot0 = (uint32_t)__cvta_generic_to_shared(tsm) + (uint32_t)tid * 16u;
    auto issue = [&](int k) {
        if (k < ns) {
#pragma unroll
            for (int v = 0; v < NV; ++v)
                asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(slot0 + (uint32_t)((k & (D - 1)) * NV + v) * (BD * 16u)),
                             "l"(Yp + (int64_t)k * a.ld + v * (2 * BD))
                             : "memory");
        }
        asm volatile("cp.async.commit_group;" ::: "memory");   // one group per species, empty past the end
    };
#pragma unroll
    for (int s = 0; s < D; ++s) issue(s);
    __syncthreads();   // the energy table is in place
    double Slo[NP][6], Shi[NP][6], Rm[NP];
#pragma unroll
    for (int i = 0; i < NP; ++i) {
        Rm[i] = 0.0;
#pragma unroll
        for (int m = 0; m < 6; ++m) Slo[i][m] = Shi[i][m] = 0.0;
    }
#pragma unroll 1
    for (int k = 0; k < ns; ++k) {
        asm volatile("cp.async.wait_group %0;" ::"n"(D - 1) : "memory");
        double y[NP];
#pragma unroll
        for (int v = 0; v < NV; ++v)
            asm volatile("ld.shared.v2.f64 {%0, %1}, [%2];"
                         : "=d"(y[2 * v]), "=d"(y[2 * v + 1])
                         : "r"(slot0 + (uint32_t)((k & (D - 1)) * NV + v) * (BD * 16u)));
        issue(k + D);
        // the twelve coefficients of the species are read once (six warp-uniform 128-bit loads) for the thread's NP points
        const double2 *row = reinterpret_cast<const double2 *>(tab + k);
        double c[12];
#pragma unroll
        for (int m = 0; m < 6; ++m) {
            const double2 v = row[m];
            c[2 * m] = v.x;
            c[2 * m + 1] = v.y;
        }
#pragma unroll
        for (int i = 0; i < NP; ++i)
#pragma unroll
            for (int m = 0; m < 6; ++m) {
                Slo[i][m] = fma(y[i], c[m], Slo[i][m]);
                Shi[i][m] = fma(y[i], c[6 + m], Shi[i][m]);
            }
        if (a.enthalpy) {   // h(T) = e(T) + T sum_k Y_k R/W_k
            const double rw = tab[k].rw;
#pragma unroll
            for (int i = 0; i < NP; ++i) Rm[i] = fma(y[i], rw, Rm[i]);
        }
    }
    int bad = 0;
#pragma unroll
    for (int i = 0; i < NP; ++i) {
        if (a.enthalpy) {
            Slo[i][1] += Rm[i];
            Shi[i][1] += Rm[i];
        }
        const int64_t p = p0 + (i >> 1) * (2 * BD) + (i & 1);
        double T;
        bool conv;
        newton_temperature(Slo[i], Shi[i], a.t_mid, a.e[p], a.T_guess[p], a.tol, a.max_iter, &T, &conv);
        a.T[p] = T;
        bad += conv ? 0 : 1;
    }
    if (a.n_not_converged != nullptr && bad) atomicAdd(a.n_not_converged, bad);
}

// ---------------------------------------------------------------------------------------
// Ideal-gas equation of state (A.2)-(A.3) PAPER.md:892-899:
// Rm = sum_k Y_k R/W_k = R/W_mix per point, then rho = p/(Rm T) or p = rho Rm T.  One streaming
// pass over Y, HBM-bound; planes prefetched into L2 like the temperature kernel.
// ---------------------------------------------------------------------------------------
template <int BD, int PPT>
__global__ void __launch_bounds__(BD) eos_kernel(const EosArgs a) {
    const int64_t base = (int64_t)blockIdx.x * (BD * PPT) + threadIdx.x;
    int64_t pt[PPT];
    double Rm[PPT];
#pragma unroll
    for (int i = 0; i < PPT; ++i) {
        const int64_t p = base + (int64_t)i * BD;
        pt[i] = p < a.n ? p : a.n - 1;
        Rm[i] = 0.0;
    }
    constexpr int kAhead = 8;
    for (int k = 0; k < a.n_species; ++k) {
        if (k + kAhead < a.n_species && (threadIdx.x & 15) == 0) {
#pragma unroll
            for (int i = 0; i < PPT; ++i)
                asm volatile("prefetch.global.L2 [%0];" ::"l"(a.Y + (int64_t)(k + kAhead) * a.ld + pt[i]));
        }
        const double rw = __ldg(&a.energy[k].rw);
#pragma unroll
        for (int i = 0; i < PPT; ++i) Rm[i] = fma(a.Y[(int64_t)k * a.ld + pt[i]], rw, Rm[i]);
    }
#pragma unroll
    for (int i = 0; i < PPT; ++i) {
        const int64_t p = base + (int64_t)i * BD;
        if (p < a.n) {
            const double rt = Rm[i] * a.T[p];
            a.out[p] = a.to_density ? a.in[p] / rt : a.in[p] * rt;
        }
    }
}

// The same as a cp.async stream (16-byte aligned planes), like temperature_stream_kernel.
template <int BD, int D>
__global__ void __launch_bounds__(BD) eos_stream_kernel(const EosArgs a) {
    static_assert((D & (D - 1)) == 0, "ring depth must be a power of two");
    extern __shared__ __align__(16) unsigned char tsm[];
    double *rw = reinterpret_cast<double *>(tsm + (size_t)D * BD * 16);
    const int tid = threadIdx.x, ns = a.n_species;
    for (int k = tid; k < ns; k += BD) rw[k] = __ldg(&a.energy[k].rw);
    const int64_t p0 = ((int64_t)blockIdx.x * BD + tid) * 2;
    const double *Yp = a.Y + p0;
    const uint32_t slot0 = (uint32_t)__cvta_generic_to_shared(tsm) + (uint32_t)tid * 16u;
    auto issue = [&](int k) {
        if (k < ns)
            asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(slot0 + (uint32_t)(k & (D - 1)) * (BD * 16u)),
                         "l"(Yp + (int64_t)k * a.ld)
                         : "memory");
        asm volatile("cp.async.commit_group;" ::: "memory");
    };
#pragma unroll
    for (int s = 0; s < D; ++s) issue(s);
    __syncthreads();
    double Rm[2] = {0.0, 0.0};
#pragma unroll 1
    for (int k = 0; k < ns; ++k) {
        asm volatile("cp.async.wait_group %0;" ::"n"(D - 1) : "memory");
        double y[2];
        asm volatile("ld.shared.v2.f64 {%0, %1}, [%2];" : "=d"(y[0]), "=d"(y[1]) : "r"(slot0 + (uint32_t)(k & (D - 1)) * (BD * 16u)));
        issue(k + D);
        const double w = rw[k];
        Rm[0] = fma(y[0], w, Rm[0]);
        Rm[1] = fma(y[1], w, Rm[1]);
    }
#pragma unroll
    for (int i = 0; i < 2; ++i) {
        const double rt = Rm[i] * a.T[p0 + i];
        a.out[p0 + i] = a.to_density ? a.in[p0 + i] / rt : a.in[p0 + i] * rt;
    }
}

// ---------------------------------------------------------------------------------------
// FP64 FMA peak probe: 8 independent DFMA chains per thread.
// ---------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256) dfma_probe_kernel(double *out, int iters, double x0) {
    double v[8];
#pragma unroll
    for (int i = 0; i < 8; ++i) v[i] = x0 + i * 1e-3 + threadIdx.x * 1e-6;
    const double m = 0.999999, c = 1e-7;
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int u = 0; u < 8; ++u)
#pragma unroll
            for (int i = 0; i < 8; ++i) v[i] = fma(v[i], m, c);
    }
    double s = 0;
#pragma unroll
    for (int i = 0; i < 8; ++i) s += v[i];
    if (s == 12345.678) out[0] = s;   // never true; keeps the chains alive
}

// ---------------------------------------------------------------------------------------
// host side
// ---------------------------------------------------------------------------------------
// kMinBlocks = 2 caps the registers at 128 per thread so that small mechanisms (whose planes and
// tensor-memory columns leave room) keep two blocks of 256 threads resident per SM
const void *rates_kernel_ptr(bool tables_in_shared, bool b_in_tmem, bool two_blocks) {
    if (two_blocks) {
        if (tables_in_shared) return b_in_tmem ? (const void *)rates_kernel<true, true, 2> : (const void *)rates_kernel<true, false, 2>;
        return b_in_tmem ? (const void *)rates_kernel<false, true, 2> : (const void *)rates_kernel<false, false, 2>;
    }
    if (tables_in_shared) return b_in_tmem ? (const void *)rates_kernel<true, true, 1> : (const void *)rates_kernel<true, false, 1>;
    return b_in_tmem ? (const void *)rates_kernel<false, true, 1> : (const void *)rates_kernel<false, false, 1>;
}

cudaError_t launch_rates(const RatesArgs &a, int threads, int blocks, bool tables_in_shared, bool b_in_tmem,
                         bool two_blocks, size_t smem_bytes, cudaStream_t stream, bool fused) {
    const void *fn = fused ? fused_kernel_ptr(tables_in_shared, b_in_tmem, two_blocks)
                           : rates_kernel_ptr(tables_in_shared, b_in_tmem, two_blocks);
    RatesArgs copy = a;
    void *params[] = {&copy};
    return cudaLaunchKernel(fn, dim3((unsigned)blocks), dim3((unsigned)threads), params, smem_bytes, stream);
}

constexpr int kTempBD = 128, kTempPPT = 4;

constexpr int kStreamBD = 128, kStreamDepth = 8;
constexpr int kStreamNV = 2;   // 16-byte vectors (pairs of points) per thread of the temperature stream

cudaError_t launch_temperature(const TempArgs &a, cudaStream_t stream) {
    if (!a.single_t_mid) {   // species with different break temperatures: the interval-wise solve
        const int64_t blocks = (a.n + kTempBD - 1) / kTempBD;
        temperature_general_kernel<kTempBD><<<dim3((unsigned)blocks), dim3(kTempBD), 0, stream>>>(a);
        return cudaGetLastError();
    }
    // whole blocks of 2 x kStreamBD points go through the cp.async stream when every species plane
    // is 16-byte aligned; the rest (ragged tail, odd ld, unaligned Y) through the plain kernel
    TempArgs rest = a;
    const bool aligned = (a.ld % 2 == 0) && (reinterpret_cast<uintptr_t>(a.Y) % 16 == 0);
    // four points per thread pay off when the pass over the species dominates (measured: configs[2] 0.364 -> 0.349 ms);
    // for a handful of species the four Newton solves per thread do (configs[1] 0.53 -> 0.62 ms): two points there
    const int nv = a.n_species >= 24 ? kStreamNV : 1;
    const size_t smem = (size_t)kStreamDepth * nv * kStreamBD * 16 + (size_t)a.n_species * sizeof(EnergyRow);
    const int64_t main_blocks = aligned && smem <= 48 * 1024 ? a.n / (2 * nv * kStreamBD) : 0;
    if (main_blocks > 0) {
        if (nv == kStreamNV)
            temperature_stream_kernel<kStreamBD, kStreamDepth, kStreamNV><<<dim3((unsigned)main_blocks), dim3(kStreamBD), smem, stream>>>(a);
        else
            temperature_stream_kernel<kStreamBD, kStreamDepth, 1><<<dim3((unsigned)main_blocks), dim3(kStreamBD), smem, stream>>>(a);
        const int64_t done = main_blocks * 2 * nv * kStreamBD;
        rest.n = a.n - done;
        rest.e += done; rest.Y += done; rest.T_guess += done; rest.T += done;
    }
    if (rest.n > 0) {
        const int64_t per_block = (int64_t)kTempBD * kTempPPT;
        const int64_t blocks = (rest.n + per_block - 1) / per_block;
        temperature_kernel<kTempBD, kTempPPT><<<dim3((unsigned)blocks), dim3(kTempBD), 0, stream>>>(rest);
    }
    return cudaGetLastError();
}

const void *temperature_kernel_ptr() { return (const void *)temperature_kernel<kTempBD, kTempPPT>; }

cudaError_t launch_eos(const EosArgs &a, cudaStream_t stream) {
    EosArgs rest = a;
    const bool aligned = (a.ld % 2 == 0) && (reinterpret_cast<uintptr_t>(a.Y) % 16 == 0);
    const size_t smem = (size_t)kStreamDepth * kStreamBD * 16 + (size_t)a.n_species * sizeof(double);
    const int64_t main_blocks = aligned ? a.n / (2 * kStreamBD) : 0;
    if (main_blocks > 0) {
        eos_stream_kernel<kStreamBD, kStreamDepth><<<dim3((unsigned)main_blocks), dim3(kStreamBD), smem, stream>>>(a);
        const int64_t done = main_blocks * 2 * kStreamBD;
        rest.n = a.n - done;
        rest.in += done; rest.T += done; rest.Y += done; rest.out += done;
    }
    if (rest.n > 0) {
        const int64_t per_block = (int64_t)kTempBD * kTempPPT;
        const int64_t blocks = (rest.n + per_block - 1) / per_block;
        eos_kernel<kTempBD, kTempPPT><<<dim3((unsigned)blocks), dim3(kTempBD), 0, stream>>>(rest);
    }
    return cudaGetLastError();
}

cudaError_t launch_dfma_probe(double *out, int iters, int blocks, cudaStream_t stream) {
    dfma_probe_kernel<<<blocks, 256, 0, stream>>>(out, iters, 1.0);
    return cudaGetLastError();
}

}   // namespace pyro
