// Chemical Jacobian, block-cooperative kernel (formulation pyro_jac_tables.h, arithmetic
// pyro_jac.cuh).
//
// The one-thread-per-point kernel (pyro_jac_kernels.cu) keeps six planes per point on chip and therefore only 128
// points = one warp per scheduler per SM; ncu shows it bound by dependent-issue latency (profiles/r02_dead_ends.md).
// Here a BLOCK of NW warps works on ONE chunk of 32 points (lane l of every warp = point l of the chunk):
//   * the read-only planes of the chunk -- C, G, dG/dT, and after the first phases V and dS/dT -- are in shared memory
//     ONCE, [k][lane], whatever the number of warps;
//   * the columns of the Jacobian are independent of one another: every warp takes the next column (longest incidence
//     list first) from a block counter and accumulates it in its OWN tensor-memory plane (warp w: lane quarter w & 3,
//     column group w >> 2), then stores it -- sixteen warps per SM instead of four;
//   * the per-reaction phases (dS/dT and the default-efficiency plane V) are split by contiguous ranges of reactions,
//     accumulated per warp in tensor memory and added into the shared planes in warp order, eight rows at a time
//     through a shared scratch (a fixed order: the result does not depend on timing).
// Every column is accumulated by one warp in list order, so J is bit-for-bit what the other kernel writes.
#include "pyro_jac_dev.cuh"

namespace pyro {

struct BlkJacMem {
    struct Raw {
        uint32_t lo, hi;
    };
    const double *C, *G, *DG;   // this lane's entry of row 0 of the planes; row k is 32 doubles further on
    double *ext;                // this lane's entry of slot 0 of the scratch of the [M] reactions
    uint32_t tw;                // tensor memory: the warp's lanes and first column of its accumulator plane

    __device__ __forceinline__ double ldC(uint32_t k) const { return C[k * 32u]; }
    __device__ __forceinline__ double ldG(uint32_t k) const { return G[k * 32u]; }
    __device__ __forceinline__ double ldDG(uint32_t k) const { return DG[k * 32u]; }
    __device__ __forceinline__ double ld_ext(uint32_t s) const { return ext[s * 32u]; }
    __device__ __forceinline__ void st_ext(uint32_t s, double v) const { ext[s * 32u] = v; }
    template <int P> __device__ __forceinline__ Raw ld_acc(uint32_t k) const {   // P is always the warp's own plane here
        Raw r;
        asm volatile("tcgen05.ld.sync.aligned.32x32b.x2.b32 {%0, %1}, [%2];" : "=r"(r.lo), "=r"(r.hi) : "r"(tw + 2u * k));
        return r;
    }
    template <int P> __device__ __forceinline__ void st_acc(uint32_t k, double v) const {
        asm volatile("tcgen05.st.sync.aligned.32x32b.x2.b32 [%0], {%1, %2};" ::"r"(tw + 2u * k), "r"(__double2loint(v)), "r"(__double2hiint(v)));
    }
    __device__ __forceinline__ double value(const Raw &r) const { return __hiloint2double((int)r.hi, (int)r.lo); }
    __device__ __forceinline__ void fence_ld() const { asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory"); }
    __device__ __forceinline__ void fence_st() const { asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory"); }
};

// plane += the sum over the warps of their accumulators, which are cleared.  Eight rows at a time: every warp copies
// its eight partial rows to a shared scratch [NW][8][32], then warps 0-7 each add one row's NW partials in warp order (a
// fixed order: the result does not depend on timing).  Two short barriers per eight rows -- the first version let the
// warps take turns over the whole plane and spent 47 % of the kernel waiting at those barriers (ncu).
template <int NW>
__device__ __forceinline__ void blk_reduce(const BlkJacMem &mem, double *plane_lane, double *scratch, int ns, int warp, int lane) {
    mem.fence_st();
#pragma unroll 1
    for (int rb = 0; rb < ns; rb += 8) {
        BlkJacMem::Raw r[8];
#pragma unroll
        for (int u = 0; u < 8; ++u) r[u] = mem.ld_acc<PW>((uint32_t)(rb + u < ns ? rb + u : ns));
        mem.fence_ld();
#pragma unroll
        for (int u = 0; u < 8; ++u) {
            scratch[(warp * 8 + u) * 32 + lane] = mem.value(r[u]);
            if (rb + u < ns) mem.st_acc<PW>((uint32_t)(rb + u), 0.0);
        }
        __syncthreads();
        if (warp < 8 && rb + warp < ns) {
            double sum = plane_lane[(rb + warp) * 32];
#pragma unroll
            for (int w = 0; w < NW; ++w) sum += scratch[(w * 8 + warp) * 32 + lane];
            plane_lane[(rb + warp) * 32] = sum;
        }
        __syncthreads();
    }
}

template <int NW> __global__ void __launch_bounds__(32 * NW, 1) jacobian_block_kernel(const JacArgs a) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    __shared__ uint32_t s_tmem_base;
    __shared__ long long s_chunk;
    __shared__ int s_next;
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const int ns = a.lay.n_species, rows = ns + 1;
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

    // shared memory: five planes [rows][32], the [M] scratch [1 + 2 n_ext][32], two reduction rows [NW][32], the
    // reduction scratch [NW][8][32], NW rings
    double *sm = reinterpret_cast<double *>(smem_raw);
    double *pC = sm + lane, *pG = pC + rows * 32, *pDG = pG + rows * 32, *pV = pDG + rows * 32, *pDT = pV + rows * 32;
    // (the [M] scratch moves to global memory -- L2 -- for mechanisms whose planes leave no room for it)
    const int ext_rows = 1 + 2 * a.lay.n_ext;
    double *pExt = a.ext_global ? a.ext + ((int64_t)blockIdx.x * ext_rows) * 32 + lane : pDT + rows * 32;
    double *red = sm + (5 * rows + (a.ext_global ? 0 : ext_rows)) * 32;   // [2][NW][32]
    double *scratch = red + 2 * NW * 32;                         // [NW][8][32]: blk_reduce
    DevJacTab tab{a.gtab, a.off_spec, a.energy, a.jtab, a.lay.off_rxn, a.lay.off_inc, a.lay.off_eff, a.lay.off_fall, a.lay.off_col,
                  (uint32_t)a.lay.n_inc};
    tab.ring.seg_recs = 16;
    tab.ring.gen = smem_raw + (size_t)a.planes_bytes + (size_t)warp * kJacBlockRingBytes;
    tab.ring.smem = (uint32_t)__cvta_generic_to_shared(tab.ring.gen);
    tab.ring.lane = (uint32_t)lane;
    BlkJacMem mem{pC, pG, pDG, pExt, tmem_base + (((uint32_t)(warp & 3) * 32u) << 16) + (uint32_t)(warp >> 2) * 2u * (uint32_t)rows};
    const uint32_t *order = reinterpret_cast<const uint32_t *>(a.jtab + a.lay.off_order);
    // this warp's contiguous shares of the plain reactions and of the [M] reactions
    const int r0 = (int)((long long)a.lay.n_plain * warp / NW), r1 = (int)((long long)a.lay.n_plain * (warp + 1) / NW);
    const int x0 = a.lay.n_plain + (int)((long long)a.lay.n_ext * warp / NW), x1 = a.lay.n_plain + (int)((long long)a.lay.n_ext * (warp + 1) / NW);
    const int64_t jstride = a.jblock ? a.jblock : a.ld;

    for (;;) {
        if (tid == 0) s_chunk = (long long)atomicAdd(a.work, 1ull);
        __syncthreads();
        const int64_t chunk = s_chunk;
        if (chunk >= a.n_chunks) break;
        const int64_t p = chunk * 32 + lane;
        const int64_t pc = p < a.n ? p : a.n - 1;   // tail lanes recompute the last point and store nothing
        const bool live = p < a.n;
        const double T = a.T[pc], rho = a.rho[pc];
        const PointT pt = make_point(T);
        // ---- phase 0: the species' planes, split over the warps; C_tot and c_v by a fixed-order sum of the warps' parts
        double part_c = 0.0, part_cv = 0.0;
        for (int k = warp; k < ns; k += NW) {
            const SpecRow &row = tab.spec(k);
            const double *c = pt.T < row.t_mid ? row.lo : row.hi;
            const double y = __ldg(a.Y + (int64_t)k * a.ld + pc);
            const double C = rho * y * row.inv_w;
            part_c += C;
            pC[k * 32] = C;
            pG[k * 32] = species_log2E(c, pt.T, pt.L2T, pt.invT);
            pDG[k * 32] = species_log2E_dT(c, pt.T, pt.invT);
            pV[k * 32] = 0.0;
            pDT[k * 32] = 0.0;
            if (a.mode == 1) part_cv = fma(y, jac_species_cv(tab.energy(k), pt.T), part_cv);
        }
        if (warp == 0) {   // the dummy species and the constant multiplier
            pC[ns * 32] = 1.0;
            pG[ns * 32] = pDG[ns * 32] = pV[ns * 32] = pDT[ns * 32] = 0.0;
            pExt[0] = 1.0;
        }
        red[warp * 32 + lane] = part_c;
        red[(NW + warp) * 32 + lane] = part_cv;
#pragma unroll 1
        for (int i = 0; i <= ns; ++i) mem.st_acc<PW>((uint32_t)i, 0.0);
        if (tid == 0) s_next = 0;
        __syncthreads();
        double ctot = 0.0, cv = 0.0;
#pragma unroll
        for (int w = 0; w < NW; ++w) {
            ctot += red[w * 32 + lane];
            cv += red[(NW + w) * 32 + lane];
        }
        // ---- phase A: dS/dT of this warp's reactions; the [M] reactions leave their multiplier and dR/d[M] in the scratch
        // (a share of the plain reactions and a share of the [M] reactions each: the latter cost several times more)
        tab.begin_rxn(r0, r1 - r0);
#pragma unroll 1
        for (int j = r0; j < r1; ++j) {
            const JacRxn &r = tab.rxn(j);
            jac_scatter<PW>(mem, r.sc_species, r.sc_w, jac_plain_dRdT(r, pt, mem));
        }
        tab.begin_rxn(x0, x1 - x0);
#pragma unroll 1
        for (int j = x0; j < x1; ++j) {
            const JacRxn &r = tab.rxn(j);
            const JacExt x = jac_ext_reaction(tab, r, pt, ctot, mem);
            mem.st_ext(1u + 2u * r.ext, x.mul);
            mem.st_ext(2u + 2u * r.ext, x.g);
            jac_scatter<PW>(mem, r.sc_species, r.sc_w, x.dRdT);
        }
        blk_reduce<NW>(mem, pDT, scratch, ns, warp, lane);
        // ---- phase B: the default-efficiency part of every column, V_i = sum_x nu_ix W_i g_x eff_default,x
        tab.begin_rxn(x0, x1 - x0);
#pragma unroll 1
        for (int j = x0; j < x1; ++j) {
            const JacRxn &r = tab.rxn(j);
            jac_scatter<PW>(mem, r.sc_species, r.sc_w, mem.ld_ext(2u + 2u * r.ext) * r.eff_default);
        }
        blk_reduce<NW>(mem, pV, scratch, ns, warp, lane);
        if (a.dSdT != nullptr && live)
            for (int i = warp; i < ns; i += NW) a.dSdT[(int64_t)i * a.ld + p] = pDT[i * 32];
        // ---- phase 3: the columns, longest list first, one warp each
        const double rcv = a.mode == 1 ? 1.0 / cv : 0.0;
        double *Jp = a.jblock ? a.J + (pc / a.jblock) * ((int64_t)ns * ns * a.jblock) + pc % a.jblock : a.J + pc;
        for (;;) {
            int cidx = 0;
            if (lane == 0) cidx = atomicAdd(&s_next, 1);
            cidx = __shfl_sync(0xffffffffu, cidx, 0);
            if (cidx >= ns) break;
            const int k = (int)order[cidx];
            const JacCol &col = tab.col(k);
            tab.begin_inc_range(col.inc_begin, col.inc_end - col.inc_begin);
            jac_column(tab, col, pt, mem);
            mem.fence_st();
            const double scale = rho * tab.spec(k).inv_w;
            const double ekcv = a.mode == 1 ? jac_species_energy(tab.energy(k), pt.T) * rcv : 0.0;
            // four rows per tensor-memory round trip; the row pointer advances by n_s planes of J per row
            double *jp = Jp + (int64_t)k * jstride;
            const int64_t rstep = (int64_t)ns * jstride;
            const double *v = pV, *dt = pDT;
            int i = 0;
#pragma unroll 1
            for (; i + 4 <= ns; i += 4, jp += 4 * rstep, v += 128, dt += 128) {
                BlkJacMem::Raw r[4];
#pragma unroll
                for (int u = 0; u < 4; ++u) r[u] = mem.ld_acc<PW>((uint32_t)(i + u));
                double pv[4], pd[4];
#pragma unroll
                for (int u = 0; u < 4; ++u) pv[u] = v[u * 32], pd[u] = dt[u * 32];
                mem.fence_ld();
#pragma unroll
                for (int u = 0; u < 4; ++u) {
                    const double val = fma(mem.value(r[u]) + pv[u], scale, -(pd[u] * ekcv));
                    if (live) __stcs(jp + u * rstep, val);
                    mem.st_acc<PW>((uint32_t)(i + u), 0.0);
                }
            }
            if (i < ns) {   // the last one to three rows (the dummy row n_s stands in for the rows beyond)
                BlkJacMem::Raw r[3];
#pragma unroll
                for (int u = 0; u < 3; ++u) r[u] = mem.ld_acc<PW>((uint32_t)(i + u < ns ? i + u : ns));
                mem.fence_ld();
#pragma unroll
                for (int u = 0; u < 3; ++u)
                    if (i + u < ns) {
                        const double val = fma(mem.value(r[u]) + v[u * 32], scale, -(dt[u * 32] * ekcv));
                        if (live) __stcs(jp + u * rstep, val);
                        mem.st_acc<PW>((uint32_t)(i + u), 0.0);
                    }
            }
        }
        __syncthreads();   // every warp is done with the planes before the next chunk overwrites them
    }
    asm volatile("tcgen05.fence::before_thread_sync;");
    __syncthreads();
    if (warp == 0)
        asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tmem_base), "r"(a.tmem_cols));
}

const void *jacobian_block_kernel_ptr(int warps) {
    return warps == 16 ? (const void *)jacobian_block_kernel<16> : (const void *)jacobian_block_kernel<8>;
}

cudaError_t launch_jacobian_block(const JacArgs &a, int warps, int blocks, size_t smem_bytes, cudaStream_t stream) {
    JacArgs copy = a;
    void *params[] = {&copy};
    return cudaLaunchKernel(jacobian_block_kernel_ptr(warps), dim3((unsigned)blocks), dim3((unsigned)(32 * warps)), params, smem_bytes, stream);
}

}   // namespace pyro
