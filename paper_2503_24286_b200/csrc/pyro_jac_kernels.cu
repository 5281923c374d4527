// sm_100a kernel of the chemical Jacobian (formulation: pyro_jac_tables.h, per-point
// arithmetic: pyro_jac.cuh).
//
// Thread mapping as in the rates kernel: one thread per point, lane l of a warp owns point l of the warp's
// current chunk of 32 consecutive points, so every load of a species plane and every store of a Jacobian
// plane J[(i n_s + k)] is one 256-byte segment.  Per-point arrays:
//   shared memory  [plane][k][thread]: C_k, G_k, dG_k/dT (read-only while the columns run), and -- for mechanisms
//                  of more than 84 species -- the default-efficiency plane V;
//   tensor memory  the accumulators: species k is columns tw + 6k .. 6k+5 (column W, V, dS/dT) of the thread's
//                  lane, so that the output loop fetches the three with one LDTM.x8; large mechanisms: 4 columns
//                  (W, dS/dT).
//   shared memory  one 8 KB record ring per warp behind the planes (RecordRing): the reaction and incidence tables
//                  stream through it;
//   global memory  the per-thread scratch of the third-body / falloff reactions, [slot][thread of the grid].
// Blocks are persistent; warps take chunks from a device-wide counter.
#include <cuda_runtime.h>

#include "pyro_jac_dev.cuh"

namespace pyro {

// kSmall: V in tensor memory (6 columns per species); else V in a fourth shared-memory plane (4 columns).
template <bool kSmall> struct DevJacMem {
    struct Raw {
        uint32_t lo, hi;
    };
    struct Out {
        uint32_t r[8];
    };
    uint32_t base, stride, plane;   // shared memory: byte address of this thread's entry 0 of plane C, bytes per species row, bytes per plane
    uint32_t tw;                    // tensor memory: lane and first column of this thread's group
    double *ext;                    // this thread's scratch column
    int64_t ext_stride;

    __device__ __forceinline__ double lds(uint32_t a) const {
        double v;
        asm volatile("ld.shared.f64 %0, [%1];" : "=d"(v) : "r"(a));
        return v;
    }
    __device__ __forceinline__ void sts(uint32_t a, double v) const { asm volatile("st.shared.f64 [%0], %1;" ::"r"(a), "d"(v)); }
    __device__ __forceinline__ double ldC(uint32_t k) const { return lds(base + k * stride); }
    __device__ __forceinline__ double ldG(uint32_t k) const { return lds(base + plane + k * stride); }
    __device__ __forceinline__ double ldDG(uint32_t k) const { return lds(base + 2u * plane + k * stride); }
    __device__ __forceinline__ uint32_t col(uint32_t k) const { return tw + (kSmall ? 6u : 4u) * k; }
    __device__ __forceinline__ Raw ldtm2(uint32_t t) const {
        Raw r;
        asm volatile("tcgen05.ld.sync.aligned.32x32b.x2.b32 {%0, %1}, [%2];" : "=r"(r.lo), "=r"(r.hi) : "r"(t));
        return r;
    }
    __device__ __forceinline__ void sttm2(uint32_t t, double v) const {
        asm volatile("tcgen05.st.sync.aligned.32x32b.x2.b32 [%0], {%1, %2};" ::"r"(t), "r"(__double2loint(v)), "r"(__double2hiint(v)));
    }
    template <int P> __device__ __forceinline__ Raw ld_acc(uint32_t k) const {
        if (!kSmall && P == PV) {
            const double v = lds(base + 3u * plane + k * stride);
            return Raw{(uint32_t)__double2loint(v), (uint32_t)__double2hiint(v)};
        }
        return ldtm2(col(k) + (kSmall ? 2u * P : (P == PDT ? 2u : 0u)));
    }
    template <int P> __device__ __forceinline__ void st_acc(uint32_t k, double v) const {
        if (!kSmall && P == PV) {
            sts(base + 3u * plane + k * stride, v);
            return;
        }
        sttm2(col(k) + (kSmall ? 2u * P : (P == PDT ? 2u : 0u)), v);
    }
    __device__ __forceinline__ void fill(uint32_t k, double c, double g, double dg) const {
        sts(base + k * stride, c);
        sts(base + plane + k * stride, g);
        sts(base + 2u * plane + k * stride, dg);
        st_acc<PW>(k, 0.0);
        st_acc<PV>(k, 0.0);
        st_acc<PDT>(k, 0.0);
    }
    __device__ __forceinline__ Out ld_out(uint32_t k) const {
        Out o;
        if (kSmall) {   // W, V, dS/dT and two columns of the next species (ignored)
            asm volatile("tcgen05.ld.sync.aligned.32x32b.x8.b32 {%0, %1, %2, %3, %4, %5, %6, %7}, [%8];"
                         : "=r"(o.r[0]), "=r"(o.r[1]), "=r"(o.r[2]), "=r"(o.r[3]), "=r"(o.r[4]), "=r"(o.r[5]), "=r"(o.r[6]), "=r"(o.r[7])
                         : "r"(col(k)));
        } else {
            asm volatile("tcgen05.ld.sync.aligned.32x32b.x4.b32 {%0, %1, %2, %3}, [%4];"
                         : "=r"(o.r[0]), "=r"(o.r[1]), "=r"(o.r[4]), "=r"(o.r[5])
                         : "r"(col(k)));
            const double v = lds(base + 3u * plane + k * stride);
            o.r[2] = (uint32_t)__double2loint(v);
            o.r[3] = (uint32_t)__double2hiint(v);
            o.r[6] = o.r[7] = 0u;
        }
        return o;
    }
    __device__ __forceinline__ double out_w(const Out &o) const { return __hiloint2double((int)o.r[1], (int)o.r[0]); }
    __device__ __forceinline__ double out_v(const Out &o) const { return __hiloint2double((int)o.r[3], (int)o.r[2]); }
    __device__ __forceinline__ double out_dt(const Out &o) const { return __hiloint2double((int)o.r[5], (int)o.r[4]); }
    __device__ __forceinline__ double value(const Raw &r) const { return __hiloint2double((int)r.hi, (int)r.lo); }
    __device__ __forceinline__ void fence_ld() const { asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory"); }
    __device__ __forceinline__ void fence_st() const { asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory"); }
    __device__ __forceinline__ double ld_ext(uint32_t s) const { return ext[(int64_t)s * ext_stride]; }
    __device__ __forceinline__ void st_ext(uint32_t s, double v) const { ext[(int64_t)s * ext_stride] = v; }
};

template <bool kSmall> __global__ void __launch_bounds__(kJacMaxThreads, 1) jacobian_kernel(const JacArgs a) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    __shared__ uint32_t s_tmem_base;
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31, nthreads = blockDim.x;
    const int ns = a.lay.n_species;
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

    const uint32_t rows = (uint32_t)ns + 1u;
    DevJacTab tab{a.gtab, a.off_spec, a.energy, a.jtab, a.lay.off_rxn, a.lay.off_inc, a.lay.off_eff, a.lay.off_fall, a.lay.off_col,
                  (uint32_t)a.lay.n_inc};
    // the warp's record ring sits behind the planes
    tab.ring.gen = smem_raw + (size_t)a.planes_bytes + (size_t)warp * RecordRing::kRingBytes;
    tab.ring.smem = (uint32_t)__cvta_generic_to_shared(tab.ring.gen);
    tab.ring.lane = (uint32_t)lane;
    DevJacMem<kSmall> mem;
    mem.stride = 8u * (uint32_t)nthreads;
    mem.plane = rows * mem.stride;
    mem.base = (uint32_t)__cvta_generic_to_shared(smem_raw) + 8u * (uint32_t)tid;
    // a block has at most four warps: warp w owns tensor-memory lanes 32 w .. 32 w + 31
    mem.tw = tmem_base + (((uint32_t)warp * 32u) << 16);
    mem.ext_stride = (int64_t)gridDim.x * nthreads;
    mem.ext = a.ext + (int64_t)blockIdx.x * nthreads + tid;

    auto grab = [&]() -> int64_t {
        unsigned long long c = 0;
        if (lane == 0) c = atomicAdd(a.work, 1ull);
        return (int64_t)__shfl_sync(0xffffffffu, c, 0);
    };
    for (int64_t chunk = grab(); chunk < a.n_chunks; chunk = grab()) {
        const int64_t p = chunk * 32 + lane;
        const int64_t pc = p < a.n ? p : a.n - 1;   // tail lanes recompute the last point and store nothing
        const bool live = p < a.n;
        const double *Yp = a.Y + pc;
        // J[(i n_s + k) ld + p] -- or, for the implicit march, blocks of jblock points: element (i, k) of point p at
        // ((p / jblock) n_s^2 + i n_s + k) jblock + p % jblock, so that the matrices of a block of points are contiguous
        double *Jp = a.jblock ? a.J + (pc / a.jblock) * ((int64_t)ns * ns * a.jblock) + pc % a.jblock : a.J + pc;
        const int64_t jstride = a.jblock ? a.jblock : a.ld;
        double *Tp = a.dSdT ? a.dSdT + pc : nullptr;
        jacobian_point(
            tab, a.lay, a.T[pc], a.rho[pc], a.mode, a.dSdT != nullptr, mem, [&](int k) { return __ldg(Yp + (int64_t)k * a.ld); },
            [&](int i, int k, double v) {
                if (live) __stcs(Jp + ((int64_t)i * ns + k) * jstride, v);
            },
            [&](int i, double v) {
                if (live) Tp[(int64_t)i * a.ld] = v;
            });
    }
    asm volatile("tcgen05.fence::before_thread_sync;");
    __syncthreads();
    if (warp == 0)
        asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tmem_base), "r"(a.tmem_cols));
}

const void *jacobian_kernel_ptr(bool small) { return small ? (const void *)jacobian_kernel<true> : (const void *)jacobian_kernel<false>; }

cudaError_t launch_jacobian(const JacArgs &a, bool small, int threads, int blocks, size_t smem_bytes, cudaStream_t stream) {
    JacArgs copy = a;
    void *params[] = {&copy};
    return cudaLaunchKernel(jacobian_kernel_ptr(small), dim3((unsigned)blocks), dim3((unsigned)threads), params, smem_bytes, stream);
}

}   // namespace pyro
