// Device-side table access shared by the two Jacobian kernels (pyro_jac_kernels.cu, pyro_jac_block_kernels.cu).
#pragma once
#include <cuda_runtime.h>

#include "pyro_jac.cuh"
#include "pyro_kernels.h"

namespace pyro {

// A table that one warp reads front to back, streamed through a two-segment ring in shared memory with cp.async:
// while the warp works on the records of one segment the next one is already on its way, so a record costs a
// shared-memory read instead of a dependent trip to L2 (the tables are far larger than L1: 190 KB of incidence
// records at 53 species, and a warp has nobody to hide that latency behind -- one warp per scheduler).
struct RecordRing {
    static constexpr uint32_t kSegRecs = 32, kRingBytes = 2u * kSegRecs * 128u;   // two segments of 32 records of up to 128 bytes
    uint32_t seg_recs = kSegRecs;   // records per segment (the block kernel uses 16: sixteen rings share the block's shared memory)
    const unsigned char *src;   // first record of the stream in global memory
    uint32_t smem;              // shared-memory address of this warp's ring
    unsigned char *gen;         // the same as a generic pointer
    uint32_t rec_bytes, seg_bytes, count;
    int32_t cur, ready;         // segment in buffer cur & 1 (cur + 1 in flight); last segment waited for
    uint32_t lane;

    __device__ __forceinline__ void issue(int32_t seg) {
        const uint32_t first = (uint32_t)seg * seg_recs;
        if (first < count) {
            const uint32_t recs = count - first < seg_recs ? count - first : seg_recs;
            const uint32_t bytes = recs * rec_bytes;
            const unsigned char *g = src + (size_t)first * rec_bytes;
            const uint32_t d = smem + (uint32_t)(seg & 1) * seg_bytes;
            for (uint32_t off = lane * 16u; off < bytes; off += 512u)
                asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(d + off), "l"(g + off) : "memory");
        }
        asm volatile("cp.async.commit_group;" ::: "memory");   // one group per segment, empty past the end
    }
    __device__ __forceinline__ void start(const unsigned char *first_record, uint32_t bytes_per_record, uint32_t n) {
        asm volatile("cp.async.wait_all;" ::: "memory");
        __syncwarp();
        src = first_record;
        rec_bytes = bytes_per_record;
        seg_bytes = seg_recs * bytes_per_record;
        count = n;
        cur = 0;
        ready = -1;
        issue(0);
        issue(1);
    }
    __device__ __forceinline__ const unsigned char *get(uint32_t q) {   // q never decreases between two start() calls
        const int32_t seg = (int32_t)(q / seg_recs);
        if (seg != ready) {
            while (cur < seg) {
                __syncwarp();        // every lane is done with the buffer that is refilled now
                issue(cur + 2);
                ++cur;
            }
            asm volatile("cp.async.wait_group 1;" ::: "memory");
            __syncwarp();
            ready = seg;
        }
        return gen + (uint32_t)(seg & 1) * seg_bytes + (q - (uint32_t)seg * seg_recs) * rec_bytes;
    }
    // record q and how many records from q on (below limit) lie contiguous in the ring: a loop over them only steps a pointer
    __device__ __forceinline__ const unsigned char *get_run(uint32_t q, uint32_t limit, uint32_t &n) {
        const unsigned char *p = get(q);
        const uint32_t seg_end = (q / seg_recs + 1u) * seg_recs;
        n = (limit < seg_end ? limit : seg_end) - q;
        return p;
    }
};

struct DevJacTab {
    const unsigned char *base;   // rates blob: species rows
    uint32_t off_spec;
    const EnergyRow *en;
    const unsigned char *jbase;
    uint32_t off_rxn, off_inc, off_eff, off_fall, off_col;
    uint32_t n_inc;
    mutable RecordRing ring;
    __device__ __forceinline__ const SpecRow &spec(int k) const { return reinterpret_cast<const SpecRow *>(base + off_spec)[k]; }
    __device__ __forceinline__ const EnergyRow &energy(int k) const { return en[k]; }
    __device__ __forceinline__ void begin_rxn(int first, int count) const {
        ring.start(jbase + off_rxn + (size_t)first * sizeof(JacRxn), (uint32_t)sizeof(JacRxn), (uint32_t)count);
        rxn_first = first;
    }
    __device__ __forceinline__ void begin_inc() const {
        ring.start(jbase + off_inc, (uint32_t)sizeof(JacInc), n_inc);
        inc_first = 0;
    }
    __device__ __forceinline__ void begin_inc_range(uint32_t first, uint32_t count) const {   // one column's list
        ring.start(jbase + off_inc + (size_t)first * sizeof(JacInc), (uint32_t)sizeof(JacInc), count);
        inc_first = (int)first;
    }
    __device__ __forceinline__ const JacRxn &rxn(int j) const { return *reinterpret_cast<const JacRxn *>(ring.get((uint32_t)(j - rxn_first))); }
    __device__ __forceinline__ const JacInc &inc(int q) const { return *reinterpret_cast<const JacInc *>(ring.get((uint32_t)(q - inc_first))); }
    // incidences q .. q + n - 1 (n >= 1, q + n <= end) at consecutive addresses
    __device__ __forceinline__ const JacInc *inc_run(uint32_t q, uint32_t end, uint32_t &n) const {
        return reinterpret_cast<const JacInc *>(ring.get_run(q - (uint32_t)inc_first, end - (uint32_t)inc_first, n));
    }
    __device__ __forceinline__ const EffEntry &eff(int q) const { return reinterpret_cast<const EffEntry *>(jbase + off_eff)[q]; }
    __device__ __forceinline__ const RxnFall &rxn_fall(int j) const { return reinterpret_cast<const RxnFall *>(jbase + off_fall)[j]; }
    __device__ __forceinline__ const JacCol &col(int k) const { return reinterpret_cast<const JacCol *>(jbase + off_col)[k]; }
    mutable int rxn_first = 0, inc_first = 0;
};

}   // namespace pyro
