// The rates kernel with TWO grid points per thread (rows a1-a3, a5-a9 of SURVEY.md 8(a)).
//
// Why.  The one-point kernel (pyro_rates_kernel.cuh) is bound by instruction issue, not by the FP64 pipe
// (profiles/r02_kernels.md: issue 66 %, FP64 pipe 45 %): of the 62 instructions of a plain 2+2 reaction only 23 are
// FP64, the rest is table reads, address arithmetic, R2UR and the tensor-memory / shared-memory accesses -- all of which
// are the same for every point.  Here a thread owns points l and l + 32 of a 64-point chunk; the per-point arithmetic
// (pyro_point.cuh, V = D2) runs both side by side, and one table read, one address, one LDS.128, one LDTM.x8 / STTM.x4
// serve two points.  The on-chip footprint per point is unchanged (A: 16 bytes per species and thread in shared
// memory; omega and B of both points: eight 32-bit tensor-memory columns per species), so a block of 128 threads
// holds the same 256 points per SM, with one warp per scheduler whose instruction-level parallelism is the two
// points times the lockstep group.
#include "pyro_rates_kernel.cuh"

namespace pyro {

struct DevMem2 {
    typedef D2 V;
    struct WRaw {
        uint32_t r[4];
    };
    struct WBRaw {
        uint32_t r[8];
    };
    uint32_t baseA, strideA, tw;

    __device__ __forceinline__ uint32_t atA(uint32_t k) const { return baseA + k * strideA; }
    __device__ __forceinline__ uint32_t atB(uint32_t) const { return 0u; }
    __device__ __forceinline__ uint32_t atW(uint32_t k) const { return tw + 8u * k; }
    __device__ __forceinline__ D2 ldA(uint32_t h) const {
        D2 v;
        asm volatile("ld.shared.v2.f64 {%0, %1}, [%2];" : "=d"(v.x), "=d"(v.y) : "r"(h));
        return v;
    }
    __device__ __forceinline__ void stA(uint32_t h, D2 v) const { asm volatile("st.shared.v2.f64 [%0], {%1, %2};" ::"r"(h), "d"(v.x), "d"(v.y)); }
    __device__ __forceinline__ WRaw ldtm4(uint32_t t) const {
        WRaw w;
        asm volatile("tcgen05.ld.sync.aligned.32x32b.x4.b32 {%0, %1, %2, %3}, [%4];"
                     : "=r"(w.r[0]), "=r"(w.r[1]), "=r"(w.r[2]), "=r"(w.r[3])
                     : "r"(t));
        return w;
    }
    __device__ __forceinline__ WRaw ldW(uint32_t hW) const { return ldtm4(hW); }
    __device__ __forceinline__ WRaw ldB(uint32_t hW, uint32_t) const { return ldtm4(hW + 4u); }
    __device__ __forceinline__ WBRaw ldWB(uint32_t hW, uint32_t) const {
        WBRaw w;
        asm volatile("tcgen05.ld.sync.aligned.32x32b.x8.b32 {%0, %1, %2, %3, %4, %5, %6, %7}, [%8];"
                     : "=r"(w.r[0]), "=r"(w.r[1]), "=r"(w.r[2]), "=r"(w.r[3]), "=r"(w.r[4]), "=r"(w.r[5]), "=r"(w.r[6]), "=r"(w.r[7])
                     : "r"(hW));
        return w;
    }
    __device__ __forceinline__ void stW(uint32_t hW, D2 v) const {
        asm volatile("tcgen05.st.sync.aligned.32x32b.x4.b32 [%0], {%1, %2, %3, %4};" ::"r"(hW), "r"(__double2loint(v.x)),
                     "r"(__double2hiint(v.x)), "r"(__double2loint(v.y)), "r"(__double2hiint(v.y)));
    }
    __device__ __forceinline__ void st_species(uint32_t k, D2 a, D2 b) const {
        stA(atA(k), a);
        asm volatile("tcgen05.st.sync.aligned.32x32b.x8.b32 [%0], {%1, %2, %3, %4, %5, %6, %7, %8};" ::"r"(atW(k)), "r"(0), "r"(0),
                     "r"(0), "r"(0), "r"(__double2loint(b.x)), "r"(__double2hiint(b.x)), "r"(__double2loint(b.y)),
                     "r"(__double2hiint(b.y)));
    }
    __device__ __forceinline__ void fence_ld() const { asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory"); }
    __device__ __forceinline__ void fence_st() const { asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory"); }
    __device__ __forceinline__ D2 value(const WRaw &w) const {
        return D2{__hiloint2double((int)w.r[1], (int)w.r[0]), __hiloint2double((int)w.r[3], (int)w.r[2])};
    }
    __device__ __forceinline__ D2 value_w(const WBRaw &w) const {
        return D2{__hiloint2double((int)w.r[1], (int)w.r[0]), __hiloint2double((int)w.r[3], (int)w.r[2])};
    }
    __device__ __forceinline__ D2 value_b(const WBRaw &w) const {
        return D2{__hiloint2double((int)w.r[5], (int)w.r[4]), __hiloint2double((int)w.r[7], (int)w.r[6])};
    }
};

// kSingles: the tables hold reactions that run one at a time (small mechanisms, pyro_pack.cpp) -- the loops for them
// are compiled in only then (instruction cache, as in the one-point kernel).
template <bool kTabSmem, bool kSingles> __global__ void __launch_bounds__(kRates2Threads, kSingles ? 3 : 1) rates2_kernel(const RatesArgs a) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    __shared__ uint32_t s_tmem_base;
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31, nthreads = blockDim.x;
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
    DevMem2 mem;
    mem.strideA = 16u * (uint32_t)nthreads;
    mem.baseA = (uint32_t)__cvta_generic_to_shared(smem_raw) + a.planes_off + 16u * (uint32_t)tid;
    mem.tw = tmem_base + (((uint32_t)warp * 32u) << 16);   // at most four warps: one per lane quarter

    auto grab = [&]() -> int64_t {
        unsigned long long c = 0;
        if (lane == 0) c = atomicAdd(a.work, 1ull);
        return (int64_t)__shfl_sync(0xffffffffu, c, 0);
    };
    int64_t chunk = grab();
    while (chunk < a.n_chunks) {   // chunks of 64 points: lane l owns points l and l + 32
        const int64_t p0 = chunk * 64 + lane, p1 = p0 + 32;
        const int64_t c0 = p0 < a.n ? p0 : a.n - 1, c1 = p1 < a.n ? p1 : a.n - 1;   // tail lanes recompute the last point, store nothing
        const D2 rho{a.rho[c0], a.rho[c1]};
        const PointTV<D2> pt = make_point(D2{a.T[c0], a.T[c1]});
        const double *Y0 = a.Y + c0, *Y1 = a.Y + c1;
        const D2 ctot = fill_planes(tab, ns, pt, rho, mem, [&](int k) { return D2{__ldg(Y0 + (int64_t)k * a.ld), __ldg(Y1 + (int64_t)k * a.ld)}; });
        const int64_t next = grab();
        if (next < a.n_chunks && (lane & 15) == 0) {   // bring the next chunk's inputs into L2 while the reactions run
            const int64_t pn = next * 64 + lane;
            asm volatile("prefetch.global.L2 [%0];" ::"l"(a.rho + pn));
            asm volatile("prefetch.global.L2 [%0];" ::"l"(a.rho + pn + 32));
            asm volatile("prefetch.global.L2 [%0];" ::"l"(a.T + pn));
            asm volatile("prefetch.global.L2 [%0];" ::"l"(a.T + pn + 32));
            for (int k = 0; k < ns; ++k) {
                asm volatile("prefetch.global.L2 [%0];" ::"l"(a.Y + (int64_t)k * a.ld + pn));
                asm volatile("prefetch.global.L2 [%0];" ::"l"(a.Y + (int64_t)k * a.ld + pn + 32));
            }
        }
        accumulate_reactions<kSingles, !kSingles>(tab, a.groups, pt, ctot, mem);   // small mechanisms: no four-in-lockstep loops
        int k = 0;
#pragma unroll 1
        for (; k < ns; k += 4) {
            DevMem2::WRaw r[4];
#pragma unroll
            for (int i = 0; i < 4; ++i) r[i] = mem.ldW(mem.atW((uint32_t)(k + i < ns ? k + i : ns)));
            mem.fence_ld();
#pragma unroll
            for (int i = 0; i < 4; ++i)
                if (k + i < ns) {
                    const D2 w = mem.value(r[i]);
                    if (p0 < a.n) a.omega[(int64_t)(k + i) * a.ld + p0] = w.x;
                    if (p1 < a.n) a.omega[(int64_t)(k + i) * a.ld + p1] = w.y;
                }
        }
        chunk = next;
    }
    asm volatile("tcgen05.fence::before_thread_sync;");
    __syncthreads();
    if (warp == 0)
        asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tmem_base), "r"(a.tmem_cols));
}

const void *rates2_kernel_ptr(bool tables_in_shared, bool singles) {
    if (singles) return tables_in_shared ? (const void *)rates2_kernel<true, true> : (const void *)rates2_kernel<false, true>;
    return tables_in_shared ? (const void *)rates2_kernel<true, false> : (const void *)rates2_kernel<false, false>;
}

cudaError_t launch_rates2(const RatesArgs &a, int threads, int blocks, bool tables_in_shared, bool singles, size_t smem_bytes, cudaStream_t stream) {
    RatesArgs copy = a;
    void *params[] = {&copy};
    return cudaLaunchKernel(rates2_kernel_ptr(tables_in_shared, singles), dim3((unsigned)blocks), dim3((unsigned)threads), params, smem_bytes, stream);
}

}   // namespace pyro
