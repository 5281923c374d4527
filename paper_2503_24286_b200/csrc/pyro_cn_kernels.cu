// Kernels of the implicit reactor march (include/pyro.h: pyro_reactor_cn): Crank-Nicolson (A.32) with Newton
// iterations (A.33)-(A.35) PAPER.md:1043-1062 on the analytic Jacobian (A.36) of pyro_get_jacobian.
// The temperature solve, the rates and the Jacobian of every Newton iteration are the library's own kernels; what
// is here is the per-point dense linear algebra between them.  One thread per point; every matrix element
// A[(i n_s + k) ld + p] is read and written in 256-byte segments per warp (the SoA layout of J), so the LU factorisation
// streams through L2 / HBM without any transpose.  No pivoting: the matrix is I - dt/(2 rho) J, a perturbation of the
// identity for the steps the scheme is used with (reading G32); a zero pivot shows up as a non-finite update and is
// counted in n_not_converged.
#include <cuda_runtime.h>

#include "pyro_kernels.h"

namespace pyro {

// start of a step: Ym = Y, Sm = W omega / rho (the right-hand side of (A.1) at the old time level)
__global__ void __launch_bounds__(256) cn_begin_step_kernel(const CnArgs a) {
    const int64_t p = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (p >= a.n) return;
    const double inv_rho = 1.0 / a.rho[p];
    for (int i = 0; i < a.n_species; ++i) {
        const int64_t at = (int64_t)i * a.ld + p;
        a.Ym[at] = a.Y[at];
        a.Sm[at] = a.energy[i].w * a.omega[at] * inv_rho;
    }
}

// one Newton iteration: F = Y - Ym - dt/2 (W omega/rho + Sm); (I - dt/(2 rho) J) dY = -F; Y += dY
//
// Left-looking LU in panels of NC columns.  A panel lives in shared memory as [column][row][thread] (conflict-free);
// the factors already computed (columns left of the panel) are read from global memory once per panel -- one global
// read serves NC multiply-adds, against three global accesses per multiply-add for the textbook in-place elimination
// (measured at 53 species: 440 ns per solve in global memory).  Threads never touch one another's data: no barrier.
#ifndef PYRO_CN_IN_FLIGHT
#define PYRO_CN_IN_FLIGHT 8
#endif
constexpr int kCnInFlight = PYRO_CN_IN_FLIGHT;
template <int NC, int TB> __global__ void __launch_bounds__(TB) cn_newton_kernel(const CnArgs a) {
    extern __shared__ double cn_cols[];   // [NC][n_species][TB]
    const int tid = threadIdx.x;
    const int64_t p = (int64_t)blockIdx.x * TB + tid;
    if (p >= a.n) return;
    const int ns = a.n_species;
    const int64_t ld = a.ld;
    // the block's matrices are contiguous: element (i, k) of this thread's point at (i n_s + k) TB + tid of the block
    double *A = a.J + (int64_t)blockIdx.x * ((int64_t)ns * ns * TB) + tid, *b = a.F + p;
    const double inv_rho = 1.0 / a.rho[p], half = 0.5 * a.dt, c = half * inv_rho;
    auto S = [&](int col, int i) -> double & { return cn_cols[((size_t)col * ns + i) * TB + tid]; };
    auto G = [&](int i, int k) -> double & { return A[((int64_t)i * ns + k) * TB]; };
    for (int j0 = 0; j0 < ns; j0 += NC) {
        const int nc = ns - j0 < NC ? ns - j0 : NC;
        for (int i = 0; i < ns; ++i)
#pragma unroll
            for (int cc = 0; cc < NC; ++cc) S(cc, i) = cc < nc ? (i == j0 + cc ? 1.0 : 0.0) - c * G(i, j0 + cc) : 0.0;
        for (int k = 0; k < j0; ++k) {   // eliminations of the columns left of the panel
            double ck[NC];
#pragma unroll
            for (int cc = 0; cc < NC; ++cc) ck[cc] = S(cc, k);
            // kCnInFlight factors in flight: with four warps per SM the loop is bound by the latency of these global reads
            int i = k + 1;
            for (; i + kCnInFlight <= ns; i += kCnInFlight) {
                double l[kCnInFlight];
#pragma unroll
                for (int u = 0; u < kCnInFlight; ++u) l[u] = G(i + u, k);
#pragma unroll
                for (int u = 0; u < kCnInFlight; ++u)
#pragma unroll
                    for (int cc = 0; cc < NC; ++cc) S(cc, i + u) = fma(-l[u], ck[cc], S(cc, i + u));
            }
            for (; i < ns; ++i) {
                const double l = G(i, k);
#pragma unroll
                for (int cc = 0; cc < NC; ++cc) S(cc, i) = fma(-l, ck[cc], S(cc, i));
            }
        }
        for (int jj = 0; jj < nc; ++jj) {   // the panel itself
            const int j = j0 + jj;
            for (int kk = 0; kk < jj; ++kk) {
                const int k = j0 + kk;
                const double ck = S(jj, k);
                for (int i = k + 1; i < ns; ++i) S(jj, i) = fma(-S(kk, i), ck, S(jj, i));
            }
            const double piv = 1.0 / S(jj, j);
            for (int i = j + 1; i < ns; ++i) S(jj, i) *= piv;
        }
        for (int i = 0; i < ns; ++i)
#pragma unroll
            for (int cc = 0; cc < NC; ++cc)
                if (cc < nc) G(i, j0 + cc) = S(cc, i);
    }
    // right-hand side in column 0 of the panel store: forward substitution with L, back substitution with U
    for (int i = 0; i < ns; ++i) {
        const int64_t at = (int64_t)i * ld + p;
        S(0, i) = -(a.Y[at] - a.Ym[at] - half * fma(a.energy[i].w * inv_rho, a.omega[at], a.Sm[at]));
    }
    for (int k = 0; k < ns; ++k) {
        const double bk = S(0, k);
#pragma unroll 4
        for (int i = k + 1; i < ns; ++i) S(0, i) = fma(-G(i, k), bk, S(0, i));
    }
    double worst = 0.0;
    bool finite = true;
    for (int r = ns - 1; r >= 0; --r) {
        double s = S(0, r);
#pragma unroll 4
        for (int j = r + 1; j < ns; ++j) s = fma(-G(r, j), S(0, j), s);
        s /= G(r, r);
        S(0, r) = s;
        b[(int64_t)r * ld] = s;
        a.Y[(int64_t)r * ld + p] += s;
        worst = fmax(worst, fabs(s));
        finite = finite && (s == s) && fabs(s) <= 1.7976931348623157e308;
    }
    if (a.last_update) a.last_update[p] = worst;
    if (a.count_unconverged && a.n_not_converged && (!finite || !(worst < a.update_tol))) atomicAdd(a.n_not_converged, 1);
}

constexpr int kCnPanel = 4;
int cn_block_threads(int n_species) { return (size_t)kCnPanel * n_species * 64 * sizeof(double) <= 200 * 1024 ? 64 : 32; }

cudaError_t launch_cn_begin_step(const CnArgs &a, cudaStream_t stream) {
    cn_begin_step_kernel<<<dim3((unsigned)((a.n + 255) / 256)), dim3(256), 0, stream>>>(a);
    return cudaGetLastError();
}
cudaError_t launch_cn_newton(const CnArgs &a, cudaStream_t stream) {
    const int tb = cn_block_threads(a.n_species);
    const size_t smem = (size_t)kCnPanel * a.n_species * tb * sizeof(double);
    // the limit is a property of the function on the current device: set it on every launch (cheap; no process-wide state)
    const void *fn = tb == 64 ? (const void *)cn_newton_kernel<kCnPanel, 64> : (const void *)cn_newton_kernel<kCnPanel, 32>;
    cudaError_t ce = cudaFuncSetAttribute(fn, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (ce != cudaSuccess) return ce;
    const dim3 grid((unsigned)((a.n + tb - 1) / tb));
    if (tb == 64) cn_newton_kernel<kCnPanel, 64><<<grid, dim3(64), smem, stream>>>(a);
    else cn_newton_kernel<kCnPanel, 32><<<grid, dim3(32), smem, stream>>>(a);
    return cudaGetLastError();
}

}   // namespace pyro
