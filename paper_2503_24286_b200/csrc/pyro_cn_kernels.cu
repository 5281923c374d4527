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
__global__ void __launch_bounds__(128) cn_newton_kernel(const CnArgs a) {
    const int64_t p = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (p >= a.n) return;
    const int ns = a.n_species;
    const int64_t ld = a.ld;
    double *A = a.J + p, *b = a.F + p;
    const double inv_rho = 1.0 / a.rho[p], half = 0.5 * a.dt, c = half * inv_rho;
    for (int i = 0; i < ns; ++i) {
        const int64_t at = (int64_t)i * ld + p;
        b[(int64_t)i * ld] = -(a.Y[at] - a.Ym[at] - half * fma(a.energy[i].w * inv_rho, a.omega[at], a.Sm[at]));
    }
    // elimination, column by column; the scaling A = I - c J is applied when an element is first touched (k == 0 for
    // rows below, on the pivot row before it is used)
    for (int i = 0; i < ns; ++i)
        for (int k = 0; k < ns; ++k) {
            double *e = A + ((int64_t)i * ns + k) * ld;
            *e = (i == k ? 1.0 : 0.0) - c * *e;
        }
    for (int k = 0; k < ns; ++k) {
        const double piv = 1.0 / A[((int64_t)k * ns + k) * ld];
        const double bk = b[(int64_t)k * ld];
        for (int i = k + 1; i < ns; ++i) {
            const double f = A[((int64_t)i * ns + k) * ld] * piv;
            double *ri = A + (int64_t)i * ns * ld;
            const double *rk = A + (int64_t)k * ns * ld;
#pragma unroll 4
            for (int j = k + 1; j < ns; ++j) ri[(int64_t)j * ld] = fma(-f, rk[(int64_t)j * ld], ri[(int64_t)j * ld]);
            b[(int64_t)i * ld] = fma(-f, bk, b[(int64_t)i * ld]);
        }
    }
    double worst = 0.0;
    bool finite = true;
    for (int r = ns - 1; r >= 0; --r) {
        double s = b[(int64_t)r * ld];
        const double *rr = A + (int64_t)r * ns * ld;
        for (int j = r + 1; j < ns; ++j) s = fma(-rr[(int64_t)j * ld], b[(int64_t)j * ld], s);
        s /= rr[(int64_t)r * ld];
        b[(int64_t)r * ld] = s;
        a.Y[(int64_t)r * ld + p] += s;
        worst = fmax(worst, fabs(s));
        finite = finite && (s == s) && fabs(s) <= 1.7976931348623157e308;
    }
    if (a.last_update) a.last_update[p] = worst;
    if (a.count_unconverged && a.n_not_converged && (!finite || !(worst < a.update_tol))) atomicAdd(a.n_not_converged, 1);
}

cudaError_t launch_cn_begin_step(const CnArgs &a, cudaStream_t stream) {
    cn_begin_step_kernel<<<dim3((unsigned)((a.n + 255) / 256)), dim3(256), 0, stream>>>(a);
    return cudaGetLastError();
}
cudaError_t launch_cn_newton(const CnArgs &a, cudaStream_t stream) {
    cn_newton_kernel<<<dim3((unsigned)((a.n + 127) / 128)), dim3(128), 0, stream>>>(a);
    return cudaGetLastError();
}

}   // namespace pyro
