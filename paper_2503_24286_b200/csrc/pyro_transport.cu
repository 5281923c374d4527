// Mixture-averaged transport properties on sm_100a: (A.18)-(A.24) PAPER.md:968-996.
// Packer, kernel and C ABI (pyro_transport_create / pyro_get_transport / pyro_transport_destroy of include/pyro.h).
//
// What is computed per point, from T and Y:
//   X_k = W Y_k/W_k (A.3);  mu_k = sqrt(T) P_b,k(ln T)^2 (A.22);  kappa_k = sqrt(T) P_c,k(ln T) (A.24);
//   D_kj = sqrt(T) P_a,kj(ln T) (A.19);  Wilke factors Phi_kj (A.21);  mu (A.20), kappa (A.23), D_k,m (A.18).
//
// Formulation.  With v_k = Y_k/W_k (so X_k = W v_k) the mixture weight cancels out of (A.20), and with
// s_k = sqrt(mu_k) = T^(1/4) |P_b,k| the Wilke factor needs no square root per pair:
//   Phi_kj = (1 + s_k (1/s_j) q_kj)^2 c_kj,   q_kj = (W_j/W_k)^(1/4),  c_kj = 1/sqrt(8 (1 + W_k/W_j))   (pack time)
//   mu      = sum_k v_k mu_k / sum_j Phi_kj v_j
//   kappa   = 1/2 [ W sum_k v_k kappa_k + 1/(W sum_k v_k/kappa_k) ]
//   D_k,m   = (1 - v_k W_k) / (W sum_{j != k} v_j / D_kj)            ((W - X_k W_k)/W = 1 - Y_k)
// All of it is O(n_species^2) per point in plain FP64 arithmetic (bound: ALU): per pair one fused multiply-add and
// three multiplies for Phi, a degree-4 Horner polynomial and one reciprocal (hardware seed + two Newton steps) for
// 1/D_kj.
//
// Mapping.  One thread per point, a block of up to 256 points.  Per-point arrays v_j and 1/s_j live in shared
// memory as [j][thread] columns (conflict-free).  The pair tables (64 bytes per ordered pair: q, c, the five
// diffusion coefficients) are far larger than shared memory, but every thread of a block needs row k at the same
// time: the block walks k in lockstep and the rows stream through a two-deep cp.async ring (3.4 KB per row at 53
// species), one barrier per row.
#include <cuda_runtime.h>

#include <cmath>
#include <cstdio>
#include <cstring>
#include <string>
#include <vector>

#include "../../include/pyro.h"
#include "pyro_math.cuh"

namespace pyro {

struct alignas(16) TrSpecies {   // phase A, per species: viscosity fit and 1/W.  48 bytes
    double b[5];
    double inv_w;
};
struct alignas(16) TrRowHead {   // row k: the species' own fits and weight.  96 bytes
    double b[5], c[5];
    double w, pad;
};
struct alignas(16) TrPair {      // ordered pair (k, j).  64 bytes
    double q, c;                 // (W_j/W_k)^(1/4),  1/sqrt(8 (1 + W_k/W_j))
    double a[5];                 // D_kj = sqrt(T) sum_m a_m (ln T)^m
    double pad;
};

struct TransportArgs {
    int64_t n, ld;
    const double *T, *Y;
    double *mu, *kappa, *D;
    const unsigned char *spec;   // TrSpecies[n_species]
    const unsigned char *rows;   // n_species rows of TrRowHead + TrPair[n_species]
    int32_t n_species;
    uint32_t row_bytes;
};

__device__ __forceinline__ double horner4(const double *c, double x) {
    double p = fma(c[4], x, c[3]);
    p = fma(p, x, c[2]);
    p = fma(p, x, c[1]);
    return fma(p, x, c[0]);
}

__global__ void __launch_bounds__(256) transport_kernel(const TransportArgs a) {
    extern __shared__ __align__(16) unsigned char tsm[];
    const int tid = threadIdx.x, nt = blockDim.x, ns = a.n_species;
    // layout: plane v [ns][nt] | plane rs [ns][nt] | species table | row ring (2 rows)
    double *pv = reinterpret_cast<double *>(tsm) + tid;
    double *prs = pv + (size_t)ns * nt;
    unsigned char *spec_s = tsm + (size_t)2 * ns * nt * 8;
    unsigned char *ring = spec_s + (size_t)ns * sizeof(TrSpecies);
    for (int i = tid; i < ns * (int)(sizeof(TrSpecies) / 16); i += nt)
        reinterpret_cast<uint4 *>(spec_s)[i] = reinterpret_cast<const uint4 *>(a.spec)[i];
    auto prefetch_row = [&](int k) {
        const unsigned char *src = a.rows + (size_t)k * a.row_bytes;
        const uint32_t dst = (uint32_t)__cvta_generic_to_shared(ring + (size_t)(k & 1) * a.row_bytes);
        for (uint32_t i = tid; i < a.row_bytes / 16u; i += nt)
            asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(dst + 16u * i), "l"(src + 16u * i) : "memory");
        asm volatile("cp.async.commit_group;" ::: "memory");
    };
    prefetch_row(0);
    __syncthreads();   // species table in place

    const int64_t p = (int64_t)blockIdx.x * nt + tid;
    const int64_t pc = p < a.n ? p : a.n - 1;   // tail threads recompute the last point and store nothing
    const double T = a.T[pc];
    const double lnT = log(T), sqT = sqrt(T), qT = sqrt(sqT);
    const double *Yp = a.Y + pc;
    double s = 0.0;
    const TrSpecies *sp = reinterpret_cast<const TrSpecies *>(spec_s);
#pragma unroll 4
    for (int j = 0; j < ns; ++j) {
        const double v = Yp[(int64_t)j * a.ld] * sp[j].inv_w;
        s += v;
        pv[(size_t)j * nt] = v;
        prs[(size_t)j * nt] = rcp_newton(qT * fabs(horner4(sp[j].b, lnT)));   // 1/sqrt(mu_j)
    }
    double mu = 0.0, s1 = 0.0, s2 = 0.0;
#pragma unroll 1
    for (int k = 0; k < ns; ++k) {
        asm volatile("cp.async.wait_all;" ::: "memory");
        __syncthreads();   // row k has landed for everyone, and everyone is done with row k - 1
        if (k + 1 < ns) prefetch_row(k + 1);
        const unsigned char *row = ring + (size_t)(k & 1) * a.row_bytes;
        const TrRowHead &h = *reinterpret_cast<const TrRowHead *>(row);
        const TrPair *pr = reinterpret_cast<const TrPair *>(row + sizeof(TrRowHead));
        const double smu = qT * fabs(horner4(h.b, lnT));   // sqrt(mu_k)
        const double vk = pv[(size_t)k * nt];
        double den = 0.0, sd = 0.0;
        // eight pairs in flight per thread: the Horner -> reciprocal -> accumulate chain of a pair is ten dependent
        // FP64 operations, and a block in lockstep has nothing else to hide it behind (unroll 4: 8.8 ms per 2^20 points
        // at 53 species, 8: 5.2 ms, 16: 5.3 ms)
#pragma unroll 8
        for (int j = 0; j < ns; ++j) {
            const double vj = pv[(size_t)j * nt], rsj = prs[(size_t)j * nt];
            const double t = fma(smu * pr[j].q, rsj, 1.0);
            den = fma(t * t, pr[j].c * vj, den);                       // Phi_kj v_j   (A.21)
            const double r = rcp_newton(horner4(pr[j].a, lnT));        // sqrt(T) / D_kj   (A.19)
            sd = fma(j == k ? 0.0 : vj, r, sd);
        }
        mu = fma(vk * (smu * smu), rcp_newton(den), mu);               // (A.20): W cancels
        const double kap = sqT * horner4(h.c, lnT);                    // (A.24)
        s1 = fma(vk, kap, s1);
        s2 = fma(vk, rcp_newton(kap), s2);
        // (A.18): D_k,m = (1 - Y_k) / (W sum_{j != k} v_j / D_kj),  1/W = s,  1/D_kj = r / sqrt(T)
        if (p < a.n) a.D[(int64_t)k * a.ld + p] = (1.0 - vk * h.w) * (s * sqT) * rcp_newton(sd);
    }
    if (p < a.n) {
        a.mu[p] = mu;
        const double W = rcp_newton(s);
        a.kappa[p] = 0.5 * fma(W, s1, rcp_newton(W * s2));             // (A.23)
    }
}

}   // namespace pyro

// ------------------------------------------------------------------------------------------------- C ABI
namespace pyro {
int set_last_error(int status, const std::string &msg);   // pyro_api.cpp: the text behind pyro_last_error_string
}
namespace {
int tr_fail(int status, const std::string &msg) { return pyro::set_last_error(status, msg); }
}   // namespace

struct pyro_transport {
    int device = 0;
    int n_species = 0;
    unsigned char *d_spec = nullptr, *d_rows = nullptr;
    uint32_t row_bytes = 0;
    int threads = 0;
    size_t smem = 0;
};

extern "C" {

int pyro_transport_create(const pyro_transport_desc *d, int device, pyro_transport **out) {
    if (!out) return tr_fail(PYRO_ERR_NULL, "out is NULL");
    *out = nullptr;
    if (!d) return tr_fail(PYRO_ERR_NULL, "desc is NULL");
    const int ns = d->n_species;
    if (ns < 1) return tr_fail(PYRO_ERR_BAD_SIZE, "n_species < 1");
    if (!d->mol_weight || !d->visc || !d->cond || !d->diff) return tr_fail(PYRO_ERR_NULL, "a fit table is NULL");
    for (int k = 0; k < ns; ++k) {
        if (!(std::isfinite(d->mol_weight[k]) && d->mol_weight[k] > 0)) return tr_fail(PYRO_ERR_BAD_MECH, "mol_weight must be positive");
        for (int m = 0; m < 5; ++m)
            if (!std::isfinite(d->visc[5 * k + m]) || !std::isfinite(d->cond[5 * k + m]))
                return tr_fail(PYRO_ERR_BAD_MECH, "a viscosity / conductivity coefficient is not finite");
        for (int j = 0; j < ns; ++j)
            for (int m = 0; m < 5; ++m)
                if (j != k && !std::isfinite(d->diff[5 * ((size_t)k * ns + j) + m]))
                    return tr_fail(PYRO_ERR_BAD_MECH, "a diffusion coefficient is not finite");
    }
    int ndev = 0;
    cudaError_t ce = cudaGetDeviceCount(&ndev);
    if (ce != cudaSuccess || ndev == 0)
        return tr_fail(PYRO_ERR_CUDA, std::string("no CUDA device: ") + cudaGetErrorString(ce) + " (libpyro has no CPU fallback)");
    if (device < 0 || device >= ndev) return tr_fail(PYRO_ERR_BAD_SIZE, "device index out of range");
    int prev = -1;
    cudaGetDevice(&prev);
    if (cudaSetDevice(device) != cudaSuccess) return tr_fail(PYRO_ERR_CUDA, "cudaSetDevice failed");
    auto *t = new pyro_transport();
    t->device = device;
    t->n_species = ns;
    t->row_bytes = (uint32_t)(sizeof(pyro::TrRowHead) + (size_t)ns * sizeof(pyro::TrPair));
    std::vector<pyro::TrSpecies> spec(ns);
    std::vector<unsigned char> rows((size_t)ns * t->row_bytes, 0);
    for (int k = 0; k < ns; ++k) {
        for (int m = 0; m < 5; ++m) spec[k].b[m] = d->visc[5 * k + m];
        spec[k].inv_w = (double)(1.0L / (long double)d->mol_weight[k]);
        pyro::TrRowHead h;
        std::memset(&h, 0, sizeof h);
        for (int m = 0; m < 5; ++m) {
            h.b[m] = d->visc[5 * k + m];
            h.c[m] = d->cond[5 * k + m];
        }
        h.w = d->mol_weight[k];
        std::memcpy(rows.data() + (size_t)k * t->row_bytes, &h, sizeof h);
        for (int j = 0; j < ns; ++j) {
            pyro::TrPair pr;
            std::memset(&pr, 0, sizeof pr);
            const long double wk = d->mol_weight[k], wj = d->mol_weight[j];
            pr.q = (double)std::sqrt(std::sqrt(wj / wk));
            pr.c = (double)(1.0L / std::sqrt(8.0L * (1.0L + wk / wj)));
            for (int m = 0; m < 5; ++m) pr.a[m] = j == k ? (m == 0 ? 1.0 : 0.0) : d->diff[5 * ((size_t)k * ns + j) + m];   // diagonal never used
            std::memcpy(rows.data() + (size_t)k * t->row_bytes + sizeof(pyro::TrRowHead) + (size_t)j * sizeof pr, &pr, sizeof pr);
        }
    }
    cudaDeviceProp prop;
    auto bail = [&](const std::string &msg, int status) {
        cudaFree(t->d_spec);
        cudaFree(t->d_rows);
        delete t;
        if (prev >= 0) cudaSetDevice(prev);
        return tr_fail(status, msg);
    };
    if ((ce = cudaGetDeviceProperties(&prop, device)) != cudaSuccess) return bail(cudaGetErrorString(ce), PYRO_ERR_CUDA);
    const size_t fixed = (size_t)ns * sizeof(pyro::TrSpecies) + 2 * (size_t)t->row_bytes;
    const size_t smem_max = prop.sharedMemPerBlockOptin;
    if (fixed + 32 * 16 * (size_t)ns > smem_max) return bail("too many species for the on-chip staging of the transport kernel", PYRO_ERR_TOO_LARGE);
    size_t threads = (smem_max - fixed) / (16 * (size_t)ns);
    threads = (threads / 32) * 32;
    if (threads > 256) threads = 256;
    t->threads = (int)threads;
    t->smem = fixed + 16 * (size_t)ns * threads;
    if ((ce = cudaFuncSetAttribute(pyro::transport_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_max)) != cudaSuccess)
        return bail(cudaGetErrorString(ce), PYRO_ERR_CUDA);
    if ((ce = cudaMalloc(&t->d_spec, spec.size() * sizeof(pyro::TrSpecies))) != cudaSuccess ||
        (ce = cudaMalloc(&t->d_rows, rows.size())) != cudaSuccess ||
        (ce = cudaMemcpy(t->d_spec, spec.data(), spec.size() * sizeof(pyro::TrSpecies), cudaMemcpyHostToDevice)) != cudaSuccess ||
        (ce = cudaMemcpy(t->d_rows, rows.data(), rows.size(), cudaMemcpyHostToDevice)) != cudaSuccess)
        return bail(cudaGetErrorString(ce), PYRO_ERR_CUDA);
    if (prev >= 0) cudaSetDevice(prev);
    *out = t;
    return PYRO_OK;
}

int pyro_transport_destroy(pyro_transport *t) {
    if (!t) return PYRO_OK;
    int prev = -1;
    cudaGetDevice(&prev);
    cudaSetDevice(t->device);
    cudaFree(t->d_spec);
    cudaFree(t->d_rows);
    if (prev >= 0) cudaSetDevice(prev);
    delete t;
    return PYRO_OK;
}

int pyro_get_transport(const pyro_transport *t, int64_t n, int64_t ld, const double *T, const double *Y, double *mu,
                       double *kappa, double *Dkm, void *cuda_stream) {
    if (!t) return tr_fail(PYRO_ERR_NULL, "transport handle is NULL");
    if (n < 0 || ld < n) return tr_fail(PYRO_ERR_BAD_SIZE, "n < 0 or ld < n");
    if (n == 0) return PYRO_OK;
    if (!T || !Y || !mu || !kappa || !Dkm) return tr_fail(PYRO_ERR_NULL, "a field pointer is NULL");
    for (const void *q : {(const void *)T, (const void *)Y, (const void *)mu, (const void *)kappa, (const void *)Dkm})
        if (reinterpret_cast<uintptr_t>(q) & 7u) return tr_fail(PYRO_ERR_ALIGN, "field pointers must be 8-byte aligned");
    {
        const uintptr_t span = (uintptr_t)(((int64_t)t->n_species - 1) * ld + n) * sizeof(double);
        const uintptr_t y0 = reinterpret_cast<uintptr_t>(Y), d0 = reinterpret_cast<uintptr_t>(Dkm);
        if (y0 < d0 + span && d0 < y0 + span) return tr_fail(PYRO_ERR_BAD_SIZE, "D must not overlap Y");
    }
    int prev = -1;
    cudaGetDevice(&prev);
    if (cudaSetDevice(t->device) != cudaSuccess) return tr_fail(PYRO_ERR_CUDA, "cudaSetDevice failed");
    pyro::TransportArgs a{};
    a.n = n; a.ld = ld; a.T = T; a.Y = Y; a.mu = mu; a.kappa = kappa; a.D = Dkm;
    a.spec = t->d_spec; a.rows = t->d_rows; a.n_species = t->n_species; a.row_bytes = t->row_bytes;
    const int64_t blocks = (n + t->threads - 1) / t->threads;
    pyro::transport_kernel<<<dim3((unsigned)blocks), dim3((unsigned)t->threads), t->smem, static_cast<cudaStream_t>(cuda_stream)>>>(a);
    const cudaError_t ce = cudaGetLastError();
    if (prev >= 0) cudaSetDevice(prev);
    if (ce != cudaSuccess) return tr_fail(PYRO_ERR_CUDA, cudaGetErrorString(ce));
    return PYRO_OK;
}

}   // extern "C"
