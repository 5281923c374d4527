// The rates kernel template and its on-chip accessors (included by pyro_kernels.cu, which instantiates the
// plain kernel, and by pyro_fused_kernels.cu, which instantiates the fused temperature + rates kernel).
#pragma once
#include <cuda_runtime.h>

#include "pyro_kernels.h"
#include "pyro_point.cuh"

namespace pyro {

struct DevTab {
    const unsigned char *base;   // shared-memory copy of the blob, or the global one
    uint32_t off_spec, off_rxn_p, off_rxn_x, off_fall, off_eff;

    __device__ __forceinline__ const SpecRow &spec(int k) const { return reinterpret_cast<const SpecRow *>(base + off_spec)[k]; }
    __device__ __forceinline__ const RxnP &rxn_p(int j) const { return reinterpret_cast<const RxnP *>(base + off_rxn_p)[j]; }
    __device__ __forceinline__ const RxnX &rxn_x(int j) const { return reinterpret_cast<const RxnX *>(base + off_rxn_x)[j]; }
    __device__ __forceinline__ const RxnFall &rxn_fall(int j) const { return reinterpret_cast<const RxnFall *>(base + off_fall)[j]; }
    __device__ __forceinline__ const EffEntry &eff(int q) const { return reinterpret_cast<const EffEntry *>(base + off_eff)[q]; }
};

// On-chip planes of one thread.
//   Shared memory: species k of plane A is the double at baseA + k strideA (strideA = 8 bytes x
//   threads per block).
//   Tensor memory, kBTmem: species k is the four 32-bit columns tw + 4k .. 4k+3 of the thread's
//   lane, omega_k in the first pair and B_k in the second, so a reactant slot fetches both with
//   one LDTM.x4.  Very large mechanisms (!kBTmem: more than 127 species) keep B in a second
//   shared-memory plane and omega alone in tensor memory (columns tw + 2k).
// All accesses are volatile asm, so they keep their program order.
template <bool kBTmem> struct DevMem {
    typedef double V;
    struct WRaw {
        uint32_t lo, hi;
    };
    struct WBRaw {
        uint32_t wlo, whi, blo, bhi;
    };
    uint32_t baseA, baseB, strideA, tw;

    __device__ __forceinline__ uint32_t atA(uint32_t k) const { return baseA + k * strideA; }
    __device__ __forceinline__ uint32_t atB(uint32_t k) const { return kBTmem ? 0u : baseB + k * strideA; }
    __device__ __forceinline__ uint32_t atW(uint32_t k) const { return tw + (kBTmem ? 4u : 2u) * k; }
    __device__ __forceinline__ double lds(uint32_t h) const {
        double v;
        asm volatile("ld.shared.f64 %0, [%1];" : "=d"(v) : "r"(h));
        return v;
    }
    __device__ __forceinline__ void sts(uint32_t h, double v) const { asm volatile("st.shared.f64 [%0], %1;" ::"r"(h), "d"(v)); }
    __device__ __forceinline__ double ldA(uint32_t h) const { return lds(h); }
    __device__ __forceinline__ void stA(uint32_t h, double v) const { sts(h, v); }
    __device__ __forceinline__ WRaw ldtm2(uint32_t t) const {
        WRaw r;
        asm volatile("tcgen05.ld.sync.aligned.32x32b.x2.b32 {%0, %1}, [%2];" : "=r"(r.lo), "=r"(r.hi) : "r"(t));
        return r;
    }
    __device__ __forceinline__ WRaw ldW(uint32_t hW) const { return ldtm2(hW); }
    __device__ __forceinline__ WRaw ldB(uint32_t hW, uint32_t hB) const {
        if (kBTmem) return ldtm2(hW + 2u);
        const double b = lds(hB);
        return WRaw{(uint32_t)__double2loint(b), (uint32_t)__double2hiint(b)};
    }
    __device__ __forceinline__ WBRaw ldWB(uint32_t hW, uint32_t hB) const {
        WBRaw r;
        if (kBTmem) {
            asm volatile("tcgen05.ld.sync.aligned.32x32b.x4.b32 {%0, %1, %2, %3}, [%4];"
                         : "=r"(r.wlo), "=r"(r.whi), "=r"(r.blo), "=r"(r.bhi)
                         : "r"(hW));
        } else {
            const WRaw w = ldtm2(hW);
            const double b = lds(hB);
            r = WBRaw{w.lo, w.hi, (uint32_t)__double2loint(b), (uint32_t)__double2hiint(b)};
        }
        return r;
    }
    __device__ __forceinline__ void stW(uint32_t hW, double v) const {
        asm volatile("tcgen05.st.sync.aligned.32x32b.x2.b32 [%0], {%1, %2};" ::"r"(hW), "r"(__double2loint(v)), "r"(__double2hiint(v)));
    }
    __device__ __forceinline__ void st_species(uint32_t k, double a, double b) const {
        sts(atA(k), a);
        if (kBTmem) {
            asm volatile("tcgen05.st.sync.aligned.32x32b.x4.b32 [%0], {%1, %2, %3, %4};" ::"r"(atW(k)), "r"(0), "r"(0),
                         "r"(__double2loint(b)), "r"(__double2hiint(b)));
        } else {
            sts(atB(k), b);
            stW(atW(k), 0.0);
        }
    }
    // the registers of a tensor-memory load are defined only after the wait (ptxas turns it into the
    // scoreboard wait of the LDTMs); the value functions are only called after it
    __device__ __forceinline__ void fence_ld() const { asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory"); }
    __device__ __forceinline__ void fence_st() const { asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory"); }
    __device__ __forceinline__ double value(const WRaw &r) const { return __hiloint2double((int)r.hi, (int)r.lo); }
    __device__ __forceinline__ double value_w(const WBRaw &r) const { return __hiloint2double((int)r.whi, (int)r.wlo); }
    __device__ __forceinline__ double value_b(const WBRaw &r) const { return __hiloint2double((int)r.bhi, (int)r.blo); }
};

// ---------------------------------------------------------------------------------------
// omega[k][p] from rho[p], T[p], Y[k][p]   (rows a1-a3, a5-a9)
// Lane l of a warp owns point l of the warp's current chunk.  Tail lanes recompute the
// last point and store nothing: control flow stays warp-uniform throughout (the tensor-memory
// instructions are warp-collective).
// ---------------------------------------------------------------------------------------
// kFused: the point's temperature is not read but solved for first, from
// (e, Y, T_guess) by the Newton iteration of row a4 -- one extra sweep over the chunk's mass fractions, which the
// fill phase then finds in L2 -- and written to T_out: (rho, e, Y, T_guess) -> (T, omega) in one launch.
template <bool kTabSmem, bool kBTmem, int kMinBlocks, bool kFused = false>
__global__ void __launch_bounds__(kRatesMaxThreads, kMinBlocks) rates_kernel(const RatesArgs a) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    __shared__ uint32_t s_tmem_base;
    const int tid = threadIdx.x, warp = tid >> 5, nthreads = blockDim.x;
    const int ns = a.n_species;

    if (kTabSmem) {
        const uint4 *src = reinterpret_cast<const uint4 *>(a.gtab);
        uint4 *dst = reinterpret_cast<uint4 *>(smem_raw);
        for (uint32_t i = tid; i < a.tab_bytes / 16u; i += nthreads) dst[i] = src[i];
    }
    if (warp == 0) {
        asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(
                         (uint32_t)__cvta_generic_to_shared(&s_tmem_base)),
                     "r"(a.tmem_cols));
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;");
    }
    asm volatile("tcgen05.fence::before_thread_sync;");
    __syncthreads();
    asm volatile("tcgen05.fence::after_thread_sync;");
    const uint32_t tmem_base = s_tmem_base;

    DevTab tab{kTabSmem ? smem_raw : a.gtab, a.off_spec, a.off_rxn_p, a.off_rxn_x, a.off_fall, a.off_eff};
    const uint32_t planes = (uint32_t)__cvta_generic_to_shared(smem_raw) + a.planes_off;
    const uint32_t rows = (uint32_t)ns + 1u;
    DevMem<kBTmem> mem;
    mem.strideA = 8u * (uint32_t)nthreads;
    mem.baseA = planes + 8u * (uint32_t)tid;
    mem.baseB = mem.baseA + rows * mem.strideA;   // second plane, used when B is not in tensor memory
    mem.tw = tmem_base + (((uint32_t)(warp & 3) * 32u) << 16) + (uint32_t)(warp >> 2) * (kBTmem ? 4u : 2u) * rows;

    // Warps are independent (own shared-memory columns, own tensor-memory lanes): each takes the
    // next chunk of 32 consecutive points from a device-wide counter until none is left, which
    // balances warps that share a scheduler against warps that have one to themselves.
    const int lane = tid & 31;
    auto grab = [&]() -> int64_t {
        unsigned long long c = 0;
        if (lane == 0) c = atomicAdd(a.work, 1ull);
        return (int64_t)__shfl_sync(0xffffffffu, c, 0);
    };
    int64_t chunk = grab();
    while (chunk < a.n_chunks) {
        const int64_t p = chunk * 32 + lane;
        const int64_t pc = p < a.n ? p : a.n - 1;
        const double rho = a.rho[pc];
        const double *Yp = a.Y + pc;
        double Tpt;
        if (kFused) {
            bool conv;
            if (a.single_t_mid) {
                // one sweep builds the mixture energy polynomials of both NASA ranges (warp-uniform table reads,
                // four mass fractions in flight), then the Newton iteration costs O(1) per step (pyro_point.cuh)
                double Slo[6] = {0, 0, 0, 0, 0, 0}, Shi[6] = {0, 0, 0, 0, 0, 0};
                auto add = [&](int k, double y) {
                    const double2 *row = reinterpret_cast<const double2 *>(a.energy + k);
#pragma unroll
                    for (int m = 0; m < 3; ++m) {
                        const double2 lo = __ldg(row + m), hi = __ldg(row + 3 + m);
                        Slo[2 * m] = fma(y, lo.x, Slo[2 * m]);
                        Slo[2 * m + 1] = fma(y, lo.y, Slo[2 * m + 1]);
                        Shi[2 * m] = fma(y, hi.x, Shi[2 * m]);
                        Shi[2 * m + 1] = fma(y, hi.y, Shi[2 * m + 1]);
                    }
                };
                int k = 0;
#pragma unroll 1
                for (; k + 4 <= ns; k += 4) {
                    const double y0 = __ldg(Yp + (int64_t)k * a.ld), y1 = __ldg(Yp + (int64_t)(k + 1) * a.ld),
                                 y2 = __ldg(Yp + (int64_t)(k + 2) * a.ld), y3 = __ldg(Yp + (int64_t)(k + 3) * a.ld);
                    add(k, y0);
                    add(k + 1, y1);
                    add(k + 2, y2);
                    add(k + 3, y3);
                }
#pragma unroll 1
                for (; k < ns; ++k) add(k, __ldg(Yp + (int64_t)k * a.ld));
                newton_temperature(Slo, Shi, a.t_mid, a.e[pc], a.T_guess[pc], a.tol, a.max_iter, &Tpt, &conv);
            } else {
                newton_temperature_general(
                    ns, [&](int k) { return __ldg(Yp + (int64_t)k * a.ld); }, [&](int k) -> const EnergyRow & { return a.energy[k]; },
                    false, a.e[pc], a.T_guess[pc], a.tol, a.max_iter, &Tpt, &conv);
            }
            if (p < a.n) {
                a.T_out[p] = Tpt;
                if (a.n_not_converged != nullptr && !conv) atomicAdd(a.n_not_converged, 1);
            }
        } else {
            Tpt = a.T[pc];
        }
        const PointT pt = make_point(Tpt);
        const double ctot = fill_planes(tab, ns, pt, rho, mem, [&](int k) { return __ldg(Yp + (int64_t)k * a.ld); });
        const int64_t next = grab();
        if (next < a.n_chunks && (lane & 15) == 0) {   // bring the next chunk's inputs into L2 while the reactions run
            const int64_t pn = next * 32 + lane;
            asm volatile("prefetch.global.L2 [%0];" ::"l"(a.rho + pn));
            if (kFused) {
                asm volatile("prefetch.global.L2 [%0];" ::"l"(a.e + pn));
                asm volatile("prefetch.global.L2 [%0];" ::"l"(a.T_guess + pn));
            } else {
                asm volatile("prefetch.global.L2 [%0];" ::"l"(a.T + pn));
            }
            for (int k = 0; k < ns; ++k) asm volatile("prefetch.global.L2 [%0];" ::"l"(a.Y + (int64_t)k * a.ld + pn));
        }
        accumulate_reactions<kMinBlocks == 2>(tab, a.groups, pt, ctot, mem);   // singles: small mechanisms only
        double *Wp = a.omega + p;
        int k = 0;
#pragma unroll 1
        for (; k + 4 <= ns; k += 4) {
            typename DevMem<kBTmem>::WRaw r[4];
#pragma unroll
            for (int i = 0; i < 4; ++i) r[i] = mem.ldW(mem.atW((uint32_t)(k + i)));
            mem.fence_ld();
            if (p < a.n) {
#pragma unroll
                for (int i = 0; i < 4; ++i) Wp[(int64_t)(k + i) * a.ld] = mem.value(r[i]);
            }
        }
#pragma unroll 1
        for (; k < ns; ++k) {
            typename DevMem<kBTmem>::WRaw r[1];
            r[0] = mem.ldW(mem.atW((uint32_t)k));
            mem.fence_ld();
            if (p < a.n) Wp[(int64_t)k * a.ld] = mem.value(r[0]);
        }
        chunk = next;
    }
    asm volatile("tcgen05.fence::before_thread_sync;");
    __syncthreads();
    if (warp == 0)
        asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tmem_base), "r"(a.tmem_cols));
}

}   // namespace pyro
