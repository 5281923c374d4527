// sm_100a kernels of libpyro and their launchers.
//
// Thread mapping: one thread per grid point, a warp reads 256
// contiguous bytes of every species plane of the SoA fields.  Per-point arrays that are
// indexed by a run-time species number (A_k = C_k E_k, B_k = 1/E_k, omega_k; pyro_tables.h)
// live in shared memory as [k][plane][tid] columns (conflict-free: lane l touches its own banks);
// mechanism tables are read at warp-uniform addresses from the __constant__ bank (or from
// global memory when a mechanism does not fit the 64 KB bank).
#include <cuda_runtime.h>

#include "pyro_kernels.h"
#include "pyro_point.cuh"

namespace pyro {

__constant__ __align__(16) unsigned char c_tab[kConstBankBytes];

template <bool kConst> struct DevTab {
    const unsigned char *base;   // global-memory copy of the blob (used when !kConst)
    uint32_t off_spec, off_rxn_p, off_rxn_x, off_fall, off_eff_delta, off_eff_species;

    __device__ __forceinline__ const unsigned char *at(uint32_t off) const {
        if constexpr (kConst)
            return c_tab + off;
        else
            return base + off;
    }
    __device__ __forceinline__ const SpecRow &spec(int k) const { return reinterpret_cast<const SpecRow *>(at(off_spec))[k]; }
    __device__ __forceinline__ const RxnP &rxn_p(int j) const { return reinterpret_cast<const RxnP *>(at(off_rxn_p))[j]; }
    __device__ __forceinline__ const RxnX &rxn_x(int j) const { return reinterpret_cast<const RxnX *>(at(off_rxn_x))[j]; }
    __device__ __forceinline__ const RxnFall &rxn_fall(int j) const { return reinterpret_cast<const RxnFall *>(at(off_fall))[j]; }
    __device__ __forceinline__ double eff_delta(int q) const { return reinterpret_cast<const double *>(at(off_eff_delta))[q]; }
    __device__ __forceinline__ int eff_species(int q) const { return (int)reinterpret_cast<const uint32_t *>(at(off_eff_species))[q]; }
};

// Shared-memory planes of one thread: species k, plane Q of its P points is the P-vector at
// base + (k kPlanes + Q) BD sizeof(Vec<P>), base = the thread's own column.  Explicit
// ld/st.shared on 32-bit window addresses: a handle costs one integer multiply-add and the
// planes are immediate offsets from it.  The accesses are volatile asm, so they keep their
// program order (the omega read-modify-writes of consecutive groups may touch one address).
template <int BD, int P> struct SmemPlanes {
    static constexpr uint32_t kPlaneBytes = BD * 8 * P, kSpeciesBytes = kPlanes * kPlaneBytes;
    uint32_t base;

    __device__ __forceinline__ uint32_t at(uint32_t k) const { return base + k * kSpeciesBytes; }
    template <int Q> __device__ __forceinline__ Vec<P> ld(uint32_t h) const {
        Vec<P> v;
        if constexpr (P == 1)
            asm volatile("ld.shared.f64 %0, [%1+%2];" : "=d"(v.v[0]) : "r"(h), "n"(Q * kPlaneBytes));
        else
            asm volatile("ld.shared.v2.f64 {%0, %1}, [%2+%3];" : "=d"(v.v[0]), "=d"(v.v[1]) : "r"(h), "n"(Q * kPlaneBytes));
        return v;
    }
    template <int Q> __device__ __forceinline__ void st(uint32_t h, const Vec<P> &v) const {
        if constexpr (P == 1)
            asm volatile("st.shared.f64 [%0+%1], %2;" ::"r"(h), "n"(Q * kPlaneBytes), "d"(v.v[0]));
        else
            asm volatile("st.shared.v2.f64 [%0+%1], {%2, %3};" ::"r"(h), "n"(Q * kPlaneBytes), "d"(v.v[0]), "d"(v.v[1]));
    }
};

// ---------------------------------------------------------------------------------------
// omega[k][p] from rho[p], T[p], Y[k][p]   (rows a1-a3, a5-a9)
// Thread t of a block owns the P adjacent points P t .. P t + P - 1 of the block's tile, so a
// warp reads 256 P contiguous bytes of every species plane (128-bit loads for P = 2 when the
// planes are 16-byte aligned) and every shared-memory access is conflict-free.  Tail threads
// recompute the last point and store nothing: control flow stays warp-uniform throughout.
// ---------------------------------------------------------------------------------------
template <int BD, int P, bool kConst>
__global__ void __launch_bounds__(BD) rates_kernel(const RatesArgs a) {
    static_assert(P == 1 || P == 2, "one or two points per thread");
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int tid = threadIdx.x;
    const int64_t p0 = ((int64_t)blockIdx.x * BD + tid) * P;
    const int ns = a.n_species;
    const SmemPlanes<BD, P> mem{(uint32_t)__cvta_generic_to_shared(smem_raw) + (uint32_t)tid * (8 * P)};
    DevTab<kConst> tab{a.gtab, a.off_spec, a.off_rxn_p, a.off_rxn_x, a.off_fall, a.off_eff_delta, a.off_eff_species};

    const bool full = p0 + P <= a.n;   // the last thread of a ragged tile owns fewer points
    const bool vec = P > 1 && full && (a.ld % P == 0) && ((reinterpret_cast<uintptr_t>(a.Y) % (8 * P)) == 0) &&
                     ((reinterpret_cast<uintptr_t>(a.omega) % (8 * P)) == 0);
    int64_t pi[P];
#pragma unroll
    for (int i = 0; i < P; ++i) pi[i] = (p0 + i < a.n) ? p0 + i : a.n - 1;
    double rho[P], T[P], ctot[P];
#pragma unroll
    for (int i = 0; i < P; ++i) {
        rho[i] = a.rho[pi[i]];
        T[i] = a.T[pi[i]];
        ctot[i] = 0.0;
    }
    const PointT<P> pt = make_point<P>(T);
    if (vec) {
        const Vec<P> *Yv = reinterpret_cast<const Vec<P> *>(a.Y + p0);
        const int64_t ldv = a.ld / P;
        fill_planes<P>(tab, ns, pt, rho, ctot, mem, [&](int k, double(&y)[P]) {
            const Vec<P> v = Yv[(int64_t)k * ldv];
#pragma unroll
            for (int i = 0; i < P; ++i) y[i] = v.v[i];
        });
    } else {
        fill_planes<P>(tab, ns, pt, rho, ctot, mem, [&](int k, double(&y)[P]) {
#pragma unroll
            for (int i = 0; i < P; ++i) y[i] = a.Y[(int64_t)k * a.ld + pi[i]];
        });
    }
    accumulate_reactions<P>(tab, a.shape_quads, a.shape_pairs, a.shape_singles, a.ext_count, pt, ctot, mem);
    if (vec) {
        Vec<P> *Wv = reinterpret_cast<Vec<P> *>(a.omega + p0);
        const int64_t ldv = a.ld / P;
#pragma unroll 4
        for (int k = 0; k < ns; ++k) Wv[(int64_t)k * ldv] = mem.template ld<kW>(mem.at((uint32_t)k));
    } else {
#pragma unroll 2
        for (int k = 0; k < ns; ++k) {
            const Vec<P> w = mem.template ld<kW>(mem.at((uint32_t)k));
#pragma unroll
            for (int i = 0; i < P; ++i)
                if (p0 + i < a.n) a.omega[(int64_t)k * a.ld + p0 + i] = w.v[i];
        }
    }
}

// ---------------------------------------------------------------------------------------
// T[p] from e[p], Y[k][p], T_guess[p]   (row a4).  One streaming pass over Y builds the
// mixture energy polynomials of both NASA ranges; the Newton iterations then cost O(1).
// Each thread handles PPT points (BD apart, so every load stays coalesced) to amortise
// the warp-uniform reads of the energy table.
// ---------------------------------------------------------------------------------------
template <int BD, int PPT>
__global__ void __launch_bounds__(BD) temperature_kernel(const TempArgs a) {
    const int64_t base = (int64_t)blockIdx.x * (BD * PPT) + threadIdx.x;
    double Slo[PPT][6], Shi[PPT][6];
#pragma unroll
    for (int i = 0; i < PPT; ++i)
#pragma unroll
        for (int m = 0; m < 6; ++m) Slo[i][m] = Shi[i][m] = 0.0;
    int64_t pt[PPT];
#pragma unroll
    for (int i = 0; i < PPT; ++i) {
        const int64_t p = base + (int64_t)i * BD;
        pt[i] = p < a.n ? p : a.n - 1;   // tail lanes recompute the last point and store nothing
    }
    const int ns = a.n_species;
    for (int k = 0; k < ns; ++k) {
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
template <int BD, int P> static const void *rates_fn(bool in_const) {
    return in_const ? (const void *)rates_kernel<BD, P, true> : (const void *)rates_kernel<BD, P, false>;
}

const void *rates_kernel_ptr(int bd, int points_per_thread, bool in_const) {
    if (points_per_thread == 1) {
        switch (bd) {
            case 32: return rates_fn<32, 1>(in_const);
            case 64: return rates_fn<64, 1>(in_const);
            case 128: return rates_fn<128, 1>(in_const);
            default: return nullptr;
        }
    }
    if (points_per_thread == 2) {
        switch (bd) {
            case 32: return rates_fn<32, 2>(in_const);
            case 64: return rates_fn<64, 2>(in_const);
            case 128: return rates_fn<128, 2>(in_const);
            default: return nullptr;
        }
    }
    return nullptr;
}

cudaError_t upload_const_table(const void *src_device, size_t bytes, cudaStream_t stream) {
    return cudaMemcpyToSymbolAsync(c_tab, src_device, bytes, 0, cudaMemcpyDeviceToDevice, stream);
}

cudaError_t launch_rates(const RatesArgs &a, int bd, int points_per_thread, bool in_const, size_t smem_bytes,
                         cudaStream_t stream) {
    const void *fn = rates_kernel_ptr(bd, points_per_thread, in_const);
    if (!fn) return cudaErrorInvalidValue;
    const int64_t per_block = (int64_t)bd * points_per_thread;
    const int64_t blocks = (a.n + per_block - 1) / per_block;
    RatesArgs copy = a;
    void *params[] = {&copy};
    return cudaLaunchKernel(fn, dim3((unsigned)blocks), dim3((unsigned)bd), params, smem_bytes, stream);
}

constexpr int kTempBD = 128, kTempPPT = 4;

cudaError_t launch_temperature(const TempArgs &a, cudaStream_t stream) {
    const int64_t per_block = (int64_t)kTempBD * kTempPPT;
    const int64_t blocks = (a.n + per_block - 1) / per_block;
    temperature_kernel<kTempBD, kTempPPT><<<dim3((unsigned)blocks), dim3(kTempBD), 0, stream>>>(a);
    return cudaGetLastError();
}

const void *temperature_kernel_ptr() { return (const void *)temperature_kernel<kTempBD, kTempPPT>; }

cudaError_t launch_dfma_probe(double *out, int iters, int blocks, cudaStream_t stream) {
    dfma_probe_kernel<<<blocks, 256, 0, stream>>>(out, iters, 1.0);
    return cudaGetLastError();
}

}   // namespace pyro
