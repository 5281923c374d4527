// Kernels of the implicit reactor march (include/pyro.h: pyro_reactor_cn): Crank-Nicolson (A.32) with Newton
// iterations (A.33)-(A.35) PAPER.md:1043-1062 on the analytic Jacobian (A.36) of pyro_get_jacobian.
// The temperature solve, the rates and the Jacobian of every Newton iteration are the library's own kernels; what
// is here is the per-point dense linear algebra between them.  One thread per point; every matrix element
// A[(i n_s + k) ld + p] is read and written in 256-byte segments per warp (the SoA layout of J), so the LU factorisation
// streams through L2 / HBM without any transpose.  No pivoting: the matrix is I - dt/(2 rho) J, a perturbation of the
// identity for the steps the scheme is used with (reading G32); a zero pivot shows up as a non-finite update and is
// counted in n_not_converged.
#include <cuda_runtime.h>

#include <cstdlib>

#include <mutex>

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
// (measured at 53 species: 440 ns per solve in global memory).  The right-hand side -F rides along as column n_s of the
// matrix, so the forward substitution is the elimination of that column and reads nothing of its own.
// Threads never touch one another's data: no barrier.
//
// Every global read of the factorisation has an address known in advance, and the kernel is bound by the latency of
// these reads (first version, eight plain loads in flight per thread: issue 4 %, long scoreboard 72 %).  So they
// stream through a per-thread ring in shared memory, filled by cp.async kCnGroups groups of kCnBatch elements ahead of
// their use; the consumer waits once per group and then has kCnBatch x NC independent multiply-adds.
constexpr int kCnRows = 4;               // rows of four columns per cp.async group
constexpr int kCnBatch = 4 * kCnRows;    // elements per cp.async group
constexpr int kCnGroups = 4;   // groups requested ahead (a power of two)
constexpr int kCnRing = kCnBatch * kCnGroups;

template <int TB> struct CnRing {
    uint32_t base;   // shared-memory byte address of this thread's element 0
    int issued, taken;
    __device__ __forceinline__ uint32_t at(int group, int e) const {
        return base + (uint32_t)((group & (kCnGroups - 1)) * kCnBatch + e) * (TB * 8u);
    }
    __device__ __forceinline__ void request(int e, const double *src) const {
        asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" ::"r"(at(issued, e)), "l"(src) : "memory");
    }
    __device__ __forceinline__ void commit() {   // one group per batch, empty past the end of the stream
        asm volatile("cp.async.commit_group;" ::: "memory");
        ++issued;
    }
    __device__ __forceinline__ void wait_front() const { asm volatile("cp.async.wait_group %0;" ::"n"(kCnGroups - 1) : "memory"); }
    __device__ __forceinline__ double take(int e) const {
        double v;
        asm volatile("ld.shared.f64 %0, [%1];" : "=d"(v) : "r"(at(taken, e)));
        return v;
    }
    __device__ __forceinline__ void drain() {
        asm volatile("cp.async.wait_all;" ::: "memory");
        issued = taken = 0;
    }
};

template <int NC, int TB> __global__ void __launch_bounds__(TB) cn_newton_kernel(const CnArgs a) {
    static_assert(NC % 4 == 0 && kCnBatch >= 6, "the eliminations left of a panel go by four columns");
    extern __shared__ double cn_cols[];   // [NC][n_species][TB], then the ring [kCnRing][TB]
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
    const int64_t row_step = (int64_t)ns * TB;
    CnRing<TB> ring{(uint32_t)__cvta_generic_to_shared(cn_cols + (size_t)NC * ns * TB) + 8u * (uint32_t)tid, 0, 0};

    int rhs_col = 0;
    for (int j0 = 0; j0 <= ns; j0 += NC) {   // columns 0 .. n_s - 1 of the matrix, column n_s = the right-hand side
        // the panel: J straight into its place (all reads in flight at once), then A = I - c J in place
        for (int i = 0; i < ns; ++i)
#pragma unroll
            for (int cc = 0; cc < NC; ++cc)
                if (j0 + cc < ns)
                    asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" ::"r"((uint32_t)__cvta_generic_to_shared(&S(cc, i))), "l"(&G(i, j0 + cc)) : "memory");
        // The factors left of the panel, L(i, k), k < j0, i > k, four columns (k .. k + 3) at a time, so that an element
        // of the panel is read and written once for four multiply-adds.  Order of the stream: the triangle
        // L(k+1,k); L(k+2,k), L(k+2,k+1); L(k+3,k), L(k+3,k+1), L(k+3,k+2) in a group of its own, then the rows i >= k + 4
        // in groups of kCnRows rows of four: L(i, k .. k+3), L(i + 1, k .. k+3), ...
        int gk = 0, gi = 1;
        const double *gp = &G(1, 0);   // &G(gi, gk); a row further is row_step doubles on, a column further TB
        auto request = [&]() {
            if (gk < j0) {
                if (gi == gk + 1) {
                    ring.request(0, gp);
                    ring.request(1, gp + row_step);
                    ring.request(2, gp + row_step + TB);
                    ring.request(3, gp + 2 * row_step);
                    ring.request(4, gp + 2 * row_step + TB);
                    ring.request(5, gp + 2 * row_step + 2 * TB);
                    gi += 3;
                    gp += 3 * row_step;
                } else {
#pragma unroll
                    for (int e = 0; e < kCnRows; ++e)
                        if (gi + e < ns) {
#pragma unroll
                            for (int q = 0; q < 4; ++q) ring.request(4 * e + q, gp + e * row_step + q * TB);
                        }
                    gi += kCnRows;
                    gp += kCnRows * row_step;
                }
                if (gi >= ns) {
                    gk += 4;
                    gi = gk + 1;
                    gp = &G(gi, gk);
                }
            }
            ring.commit();
        };
        asm volatile("cp.async.commit_group;" ::: "memory");
#pragma unroll 1
        for (int u = 0; u < kCnGroups; ++u) request();
        asm volatile("cp.async.wait_group %0;" ::"n"(kCnGroups) : "memory");   // the panel has landed
        {   // A = I - c J in place, four rows at a time (loads first: see below)
            int i = 0;
            for (; i + 4 <= ns; i += 4) {
                double v[4][NC];
#pragma unroll
                for (int e = 0; e < 4; ++e)
#pragma unroll
                    for (int cc = 0; cc < NC; ++cc) v[e][cc] = S(cc, i + e);
#pragma unroll
                for (int e = 0; e < 4; ++e)
#pragma unroll
                    for (int cc = 0; cc < NC; ++cc) S(cc, i + e) = j0 + cc < ns ? (i + e == j0 + cc ? 1.0 : 0.0) - c * v[e][cc] : 0.0;
            }
            for (; i < ns; ++i) {
#pragma unroll
                for (int cc = 0; cc < NC; ++cc) S(cc, i) = j0 + cc < ns ? (i == j0 + cc ? 1.0 : 0.0) - c * S(cc, i) : 0.0;
            }
        }
        if (j0 + NC > ns) {   // the last panel: the right-hand side -F behind the last column of the matrix
            rhs_col = ns - j0;
            for (int i = 0; i < ns; ++i) {
                const int64_t at = (int64_t)i * ld + p;
                S(rhs_col, i) = -(a.Y[at] - a.Ym[at] - half * fma(a.energy[i].w * inv_rho, a.omega[at], a.Sm[at]));
            }
        }
#pragma unroll 1
        for (int k = 0; k < j0; k += 4) {   // j0 is a multiple of NC, NC a multiple of four
            double c0[NC], c1[NC], c2[NC], c3[NC];   // rows k .. k + 3 of the panel, final after the triangle
            ring.wait_front();
            {
                double t[6];
#pragma unroll
                for (int e = 0; e < 6; ++e) t[e] = ring.take(e);
                ++ring.taken;
#pragma unroll
                for (int cc = 0; cc < NC; ++cc) c0[cc] = S(cc, k), c1[cc] = S(cc, k + 1), c2[cc] = S(cc, k + 2), c3[cc] = S(cc, k + 3);
                request();
#pragma unroll
                for (int cc = 0; cc < NC; ++cc) {
                    c1[cc] = fma(-t[0], c0[cc], c1[cc]);
                    c2[cc] = fma(-t[2], c1[cc], fma(-t[1], c0[cc], c2[cc]));
                    c3[cc] = fma(-t[5], c2[cc], fma(-t[4], c1[cc], fma(-t[3], c0[cc], c3[cc])));
                }
#pragma unroll
                for (int cc = 0; cc < NC; ++cc) S(cc, k + 1) = c1[cc], S(cc, k + 2) = c2[cc], S(cc, k + 3) = c3[cc];
            }
            // loads first, then the multiply-adds, then the stores: written out, because the compiler cannot tell that
            // the columns of the panel do not overlap and would otherwise wait for every load in turn
            int i0 = k + 4;
#pragma unroll 1
            for (; i0 + kCnRows <= ns; i0 += kCnRows) {
                ring.wait_front();
                double l[kCnRows][4], v[kCnRows][NC];
#pragma unroll
                for (int e = 0; e < kCnRows; ++e)
#pragma unroll
                    for (int q = 0; q < 4; ++q) l[e][q] = ring.take(4 * e + q);
                ++ring.taken;
#pragma unroll
                for (int e = 0; e < kCnRows; ++e)
#pragma unroll
                    for (int cc = 0; cc < NC; ++cc) v[e][cc] = S(cc, i0 + e);
                request();
#pragma unroll
                for (int e = 0; e < kCnRows; ++e)
#pragma unroll
                    for (int cc = 0; cc < NC; ++cc)
                        v[e][cc] = fma(-l[e][3], c3[cc], fma(-l[e][2], c2[cc], fma(-l[e][1], c1[cc], fma(-l[e][0], c0[cc], v[e][cc]))));
#pragma unroll
                for (int e = 0; e < kCnRows; ++e)
#pragma unroll
                    for (int cc = 0; cc < NC; ++cc) S(cc, i0 + e) = v[e][cc];
            }
            if (i0 < ns) {   // the ragged end of the four columns
                ring.wait_front();
#pragma unroll
                for (int e = 0; e < kCnRows - 1; ++e)
                    if (i0 + e < ns) {
                        double l[4], v[NC];
#pragma unroll
                        for (int q = 0; q < 4; ++q) l[q] = ring.take(4 * e + q);
#pragma unroll
                        for (int cc = 0; cc < NC; ++cc) v[cc] = S(cc, i0 + e);
#pragma unroll
                        for (int cc = 0; cc < NC; ++cc)
                            S(cc, i0 + e) = fma(-l[3], c3[cc], fma(-l[2], c2[cc], fma(-l[1], c1[cc], fma(-l[0], c0[cc], v[cc]))));
                    }
                ++ring.taken;
                request();
            }
        }
        ring.drain();
        for (int jj = 0; jj < NC; ++jj) {   // the panel itself
            const int j = j0 + jj;
            if (j > ns) break;
            for (int kk = 0; kk < jj; ++kk) {
                const int k = j0 + kk;
                const double ck = S(jj, k);
                int i = k + 1;
                for (; i + 4 <= ns; i += 4) {
                    double x[4], y[4];
#pragma unroll
                    for (int e = 0; e < 4; ++e) x[e] = S(kk, i + e), y[e] = S(jj, i + e);
#pragma unroll
                    for (int e = 0; e < 4; ++e) S(jj, i + e) = fma(-x[e], ck, y[e]);
                }
                for (; i < ns; ++i) S(jj, i) = fma(-S(kk, i), ck, S(jj, i));
            }
            if (j < ns) {
                const double piv = 1.0 / S(jj, j);
                for (int i = j + 1; i < ns; ++i) S(jj, i) *= piv;
            }
        }
        {   // the panel's columns back to their place in global memory, four rows at a time
            int i = 0;
            for (; i + 4 <= ns; i += 4) {
                double v[4][NC];
#pragma unroll
                for (int e = 0; e < 4; ++e)
#pragma unroll
                    for (int cc = 0; cc < NC; ++cc) v[e][cc] = S(cc, i + e);
#pragma unroll
                for (int e = 0; e < 4; ++e)
#pragma unroll
                    for (int cc = 0; cc < NC; ++cc)
                        if (j0 + cc < ns) G(i + e, j0 + cc) = v[e][cc];
            }
            for (; i < ns; ++i)
#pragma unroll
                for (int cc = 0; cc < NC; ++cc)
                    if (j0 + cc < ns) G(i, j0 + cc) = S(cc, i);
        }
    }
    // back substitution with U, row after row from the last: the diagonal element first, then the row right of it.
    // y = L^-1 (-F) is in column rhs_col of the panel store; x overwrites it.
    {
        int gr = ns - 1, gj = ns - 1;
        auto request = [&]() {
            if (gr >= 0) {
#pragma unroll
                for (int e = 0; e < kCnBatch; ++e)
                    if (gj + e < ns) ring.request(e, &G(gr, gj + e));
                gj += kCnBatch;
                if (gj >= ns) {
                    --gr;
                    gj = gr;
                }
            }
            ring.commit();
        };
#pragma unroll 1
        for (int u = 0; u < kCnGroups; ++u) request();
        double worst = 0.0;
        bool finite = true;
#pragma unroll 1
        for (int r = ns - 1; r >= 0; --r) {
            double s = S(rhs_col, r), diag = 1.0;
#pragma unroll 1
            for (int j0 = r; j0 < ns; j0 += kCnBatch) {
                ring.wait_front();
                double u[kCnBatch];
#pragma unroll
                for (int e = 0; e < kCnBatch; ++e) u[e] = j0 + e < ns ? ring.take(e) : 0.0;
                ++ring.taken;
                request();
#pragma unroll
                for (int e = 0; e < kCnBatch; ++e) {
                    if (j0 + e == r) diag = u[e];
                    else if (j0 + e < ns) s = fma(-u[e], S(rhs_col, j0 + e), s);
                }
            }
            s /= diag;
            S(rhs_col, r) = s;
            worst = fmax(worst, fabs(s));
            finite = finite && (s == s) && fabs(s) <= 1.7976931348623157e308;
        }
        ring.drain();
        {   // dY out, Y += dY: four rows at a time, so that the reads of Y do not wait for one another
            int i = 0;
            for (; i + 4 <= ns; i += 4) {
                double y[4], d[4];
#pragma unroll
                for (int e = 0; e < 4; ++e) y[e] = a.Y[(int64_t)(i + e) * ld + p], d[e] = S(rhs_col, i + e);
#pragma unroll
                for (int e = 0; e < 4; ++e) {
                    b[(int64_t)(i + e) * ld] = d[e];
                    a.Y[(int64_t)(i + e) * ld + p] = y[e] + d[e];
                }
            }
            for (; i < ns; ++i) {
                const double d = S(rhs_col, i);
                b[(int64_t)i * ld] = d;
                a.Y[(int64_t)i * ld + p] += d;
            }
        }
        if (a.last_update) a.last_update[p] = worst;
        if (a.count_unconverged && a.n_not_converged && (!finite || !(worst < a.update_tol))) atomicAdd(a.n_not_converged, 1);
    }
}

constexpr int kCnPanel = 4;
constexpr size_t kCnSmemLimit = 227 * 1024;   // dynamic shared memory a block can get on sm_100
static size_t cn_smem_bytes(int n_species, int tb) { return ((size_t)kCnPanel * n_species + kCnRing) * tb * sizeof(double); }
int cn_block_threads(int n_species) {
    // PYRO_CN_BLOCK is a test hook, read once per process (not per call: getenv is not safe against a concurrent setenv)
    static const int forced = [] {
        const char *env = std::getenv("PYRO_CN_BLOCK");
        return env ? (std::atoi(env) == 64 ? 64 : 32) : 0;
    }();
    // 64 points per block only where their panels fit the shared memory of one block (up to 97 species)
    if (forced == 64 && cn_smem_bytes(n_species, 64) <= kCnSmemLimit) return 64;
    return 32;   // measured at 53 species: 271 ns per reactor-iteration against 300 with 64 (more blocks, more loads in flight)
}

cudaError_t launch_cn_begin_step(const CnArgs &a, cudaStream_t stream) {
    cn_begin_step_kernel<<<dim3((unsigned)((a.n + 255) / 256)), dim3(256), 0, stream>>>(a);
    return cudaGetLastError();
}
namespace {
// The dynamic shared-memory limit is a property of the function on a device, shared by every mechanism and host thread:
// raised once per device to the device maximum, so that no launch ever lowers it under a concurrent one.
struct CnDeviceSetup {
    std::once_flag once;
    cudaError_t status = cudaSuccess;
};
CnDeviceSetup g_cn_setup[64];
void cn_setup_device(CnDeviceSetup &d, int dev) {
    int optin = 0;
    if ((d.status = cudaDeviceGetAttribute(&optin, cudaDevAttrMaxSharedMemoryPerBlockOptin, dev)) != cudaSuccess) return;
    for (const void *fn : {(const void *)cn_newton_kernel<kCnPanel, 64>, (const void *)cn_newton_kernel<kCnPanel, 32>}) {
        cudaFuncAttributes fa{};
        if ((d.status = cudaFuncGetAttributes(&fa, fn)) != cudaSuccess) return;
        if ((d.status = cudaFuncSetAttribute(fn, cudaFuncAttributeMaxDynamicSharedMemorySize, optin - (int)fa.sharedSizeBytes)) != cudaSuccess) return;
    }
}
}   // namespace

cudaError_t launch_cn_newton(const CnArgs &a, cudaStream_t stream) {
    const int tb = cn_block_threads(a.n_species);
    const size_t smem = cn_smem_bytes(a.n_species, tb);
    int dev = 0;
    cudaError_t ce = cudaGetDevice(&dev);
    if (ce != cudaSuccess) return ce;
    if (dev < 0 || dev >= 64) return cudaErrorInvalidDevice;
    CnDeviceSetup &d = g_cn_setup[dev];
    std::call_once(d.once, [&d, dev] { cn_setup_device(d, dev); });
    if (d.status != cudaSuccess) return d.status;
    const dim3 grid((unsigned)((a.n + tb - 1) / tb));
    if (tb == 64) cn_newton_kernel<kCnPanel, 64><<<grid, dim3(64), smem, stream>>>(a);
    else cn_newton_kernel<kCnPanel, 32><<<grid, dim3(32), smem, stream>>>(a);
    return cudaGetLastError();
}

}   // namespace pyro
