// Measurement probes behind two design decisions (include/pyro.h: pyro_probe_dmma_peak, pyro_probe_indexed_rmw), so
// that the figures quoted in DESIGN.md and profiles/ can be reproduced from tracked code (`python bench.py --probes`).
//   * FP64 tensor cores: mma.sync.m8n8k4.f64 peak against the vector DFMA peak (the nu.R contraction)
//   * tensor memory as an indexed per-thread store: read-modify-write of doubles at warp-uniform run-time slots in
//     tensor memory (tcgen05.ld/st) against shared memory ([slot][thread], conflict-free)
#include <cuda_runtime.h>

#include <cstdint>
#include <string>

#include "../../include/pyro.h"

namespace pyro {
int set_last_error(int status, const std::string &msg);

// 8 independent accumulator fragments per warp: D(8x8) += A(8x4) B(4x8), 2 * 8 * 8 * 4 = 512 flops per mma per warp
__global__ void __launch_bounds__(256) dmma_probe_kernel(double *out, int iters) {
    double acc[8][2];
#pragma unroll
    for (int i = 0; i < 8; ++i) acc[i][0] = acc[i][1] = 1e-3 * (threadIdx.x + i);
    const double a = 0.999 + 1e-6 * threadIdx.x, b = 1.0e-3;
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int i = 0; i < 8; ++i)
            asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0, %1}, {%2}, {%3}, {%0, %1};"
                         : "+d"(acc[i][0]), "+d"(acc[i][1])
                         : "d"(a), "d"(b));
    }
    double s = 0;
#pragma unroll
    for (int i = 0; i < 8; ++i) s += acc[i][0] + acc[i][1];
    if (s == 12345.678) out[0] = s;
}

// mode 0: shared-memory RMW; 1: tensor-memory RMW (wait::ld before the add, wait::st before the next round);
// 2: tensor-memory loads only.  kRmwBatch independent slots per iteration out of 64, warp-uniform, pseudo-random: the
// batch the rates kernel issues for a lockstep group of four 2+2 reactions (16 loads, the adds, 16 stores).
constexpr int kRmwBatch = 16;
__global__ void __launch_bounds__(256) rmw_probe_kernel(int mode, int iters, long long *cycles, double *sink) {
    extern __shared__ __align__(16) unsigned char sm[];
    __shared__ uint32_t s_tmem;
    const int tid = threadIdx.x, warp = tid >> 5, nt = blockDim.x;
    if (warp == 0) {
        asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"((uint32_t)__cvta_generic_to_shared(&s_tmem)), "r"(512));
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;");
    }
    asm volatile("tcgen05.fence::before_thread_sync;");
    __syncthreads();
    asm volatile("tcgen05.fence::after_thread_sync;");
    const uint32_t tw = s_tmem + (((uint32_t)(warp & 3) * 32u) << 16) + (uint32_t)(warp >> 2) * 128u;
    const uint32_t base = (uint32_t)__cvta_generic_to_shared(sm) + 8u * tid, stride = 8u * nt;
    for (uint32_t k = 0; k < 64; ++k) {
        asm volatile("st.shared.f64 [%0], %1;" ::"r"(base + k * stride), "d"(1.0));
        asm volatile("tcgen05.st.sync.aligned.32x32b.x2.b32 [%0], {%1, %2};" ::"r"(tw + 2u * k), "r"(0), "r"(0x3ff00000));
    }
    asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory");
    __syncthreads();
    uint32_t lcg = 12345u + 977u * warp;
    double acc = 0.0;
    const long long t0 = clock64();
    for (int it = 0; it < iters; ++it) {
        uint32_t k[kRmwBatch];
#pragma unroll
        for (int i = 0; i < kRmwBatch; ++i) {
            lcg = lcg * 1664525u + 1013904223u;
            k[i] = (lcg >> 20) & 63u;
        }
        if (mode == 0) {
            double v[kRmwBatch];
#pragma unroll
            for (int i = 0; i < kRmwBatch; ++i) asm volatile("ld.shared.f64 %0, [%1];" : "=d"(v[i]) : "r"(base + k[i] * stride));
#pragma unroll
            for (int i = 0; i < kRmwBatch; ++i) asm volatile("st.shared.f64 [%0], %1;" ::"r"(base + k[i] * stride), "d"(v[i] + 1.0));
        } else {
            uint32_t lo[kRmwBatch], hi[kRmwBatch];
#pragma unroll
            for (int i = 0; i < kRmwBatch; ++i)
                asm volatile("tcgen05.ld.sync.aligned.32x32b.x2.b32 {%0, %1}, [%2];" : "=r"(lo[i]), "=r"(hi[i]) : "r"(tw + 2u * k[i]));
            asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
            if (mode == 1) {
#pragma unroll
                for (int i = 0; i < kRmwBatch; ++i) {
                    const double v = __hiloint2double((int)hi[i], (int)lo[i]) + 1.0;
                    asm volatile("tcgen05.st.sync.aligned.32x32b.x2.b32 [%0], {%1, %2};" ::"r"(tw + 2u * k[i]), "r"(__double2loint(v)), "r"(__double2hiint(v)));
                }
                asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory");
            } else {
#pragma unroll
                for (int i = 0; i < kRmwBatch; ++i) acc += __hiloint2double((int)hi[i], (int)lo[i]);
            }
        }
    }
    const long long t1 = clock64();
    if (tid == 0) cycles[blockIdx.x] = t1 - t0;
    if (acc == 12345.678) sink[0] = acc;
    asm volatile("tcgen05.fence::before_thread_sync;");
    __syncthreads();
    if (warp == 0) asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(s_tmem), "r"(512));
}

}   // namespace pyro

extern "C" {

int pyro_probe_dmma_peak(int device, double millis, double *tflops) {
    if (!tflops) return pyro::set_last_error(PYRO_ERR_NULL, "tflops is NULL");
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || device < 0 || device >= ndev) return pyro::set_last_error(PYRO_ERR_CUDA, "no such CUDA device");
    int prev = -1;
    cudaGetDevice(&prev);
    cudaSetDevice(device);
    cudaDeviceProp prop;
    cudaGetDeviceProperties(&prop, device);
    double *d_out = nullptr;
    cudaMalloc(&d_out, 8);
    cudaEvent_t t0, t1;
    cudaEventCreate(&t0);
    cudaEventCreate(&t1);
    const int blocks = prop.multiProcessorCount * 8;
    int iters = 2000;
    float ms = 0;
    for (int pass = 0; pass < 3; ++pass) {
        pyro::dmma_probe_kernel<<<blocks, 256>>>(d_out, iters);
        cudaEventRecord(t0);
        pyro::dmma_probe_kernel<<<blocks, 256>>>(d_out, iters);
        cudaEventRecord(t1);
        cudaEventSynchronize(t1);
        cudaEventElapsedTime(&ms, t0, t1);
        if (ms >= 0.5 * millis || pass == 2) break;
        iters = (int)(iters * (millis / (ms > 1e-3 ? ms : 1e-3))) + 1;
    }
    const cudaError_t ce = cudaGetLastError();
    *tflops = (double)blocks * 8.0 * (double)iters * 8.0 * 512.0 / (ms * 1e-3) / 1e12;   // blocks x warps x iters x 8 mma x 512 flops
    cudaEventDestroy(t0);
    cudaEventDestroy(t1);
    cudaFree(d_out);
    if (prev >= 0) cudaSetDevice(prev);
    return ce == cudaSuccess ? PYRO_OK : pyro::set_last_error(PYRO_ERR_CUDA, cudaGetErrorString(ce));
}

int pyro_probe_indexed_rmw(int device, int warps_per_sm, int mode, double *cycles_per_iteration) {
    if (!cycles_per_iteration) return pyro::set_last_error(PYRO_ERR_NULL, "cycles_per_iteration is NULL");
    if (warps_per_sm < 1 || warps_per_sm > 8 || mode < 0 || mode > 2) return pyro::set_last_error(PYRO_ERR_BAD_SIZE, "warps_per_sm in 1..8, mode in 0..2");
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || device < 0 || device >= ndev) return pyro::set_last_error(PYRO_ERR_CUDA, "no such CUDA device");
    int prev = -1;
    cudaGetDevice(&prev);
    cudaSetDevice(device);
    cudaDeviceProp prop;
    cudaGetDeviceProperties(&prop, device);
    const int blocks = prop.multiProcessorCount, threads = 32 * warps_per_sm, iters = 20000;
    long long *d_cycles = nullptr;
    double *d_sink = nullptr;
    cudaMalloc(&d_cycles, sizeof(long long) * blocks);
    cudaMalloc(&d_sink, 8);
    const size_t smem = (size_t)64 * 8 * threads;
    cudaFuncSetAttribute(pyro::rmw_probe_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    for (int pass = 0; pass < 2; ++pass) pyro::rmw_probe_kernel<<<blocks, threads, smem>>>(mode, iters, d_cycles, d_sink);
    long long h = 0;
    cudaMemcpy(&h, d_cycles, sizeof h, cudaMemcpyDeviceToHost);
    const cudaError_t ce = cudaGetLastError();
    *cycles_per_iteration = (double)h / iters;
    cudaFree(d_cycles);
    cudaFree(d_sink);
    if (prev >= 0) cudaSetDevice(prev);
    return ce == cudaSuccess ? PYRO_OK : pyro::set_last_error(PYRO_ERR_CUDA, cudaGetErrorString(ce));
}

}   // extern "C"
