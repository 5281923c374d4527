// C-ABI layer of libpyro (include/pyro.h): handle management, argument checks, the
// constant-bank residency protocol, launches, and the pipelined host-buffer entry point.
#include <cuda_runtime.h>

#include <atomic>
#include <chrono>
#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <mutex>
#include <string>
#include <vector>

#include "../../include/pyro.h"
#include "pyro_kernels.h"
#include "pyro_pack.h"

namespace {

thread_local std::string g_last_error;

int fail(int status, const std::string &msg) {
    g_last_error = msg;
    return status;
}

int cuda_fail(cudaError_t e, const char *what) {
    g_last_error = std::string(what) + ": " + cudaGetErrorString(e);
    return PYRO_ERR_CUDA;
}

#define PYRO_CUDA(call)                                      \
    do {                                                     \
        cudaError_t e_ = (call);                             \
        if (e_ != cudaSuccess) return cuda_fail(e_, #call);  \
    } while (0)

struct DeviceGuard {
    int prev = -1;
    bool ok = false;
    explicit DeviceGuard(int dev) {
        if (cudaGetDevice(&prev) == cudaSuccess && cudaSetDevice(dev) == cudaSuccess) ok = true;
    }
    ~DeviceGuard() {
        if (prev >= 0) cudaSetDevice(prev);
    }
};

// Who owns the __constant__ table bank of a device, and which streams may still be reading it.
struct ConstBank {
    std::mutex mu;
    uint64_t resident = 0;   // id of the mechanism whose tables are in the bank (0 = none)
    cudaStream_t upload_stream = nullptr;
    cudaEvent_t upload_done = nullptr;
    std::vector<std::pair<cudaStream_t, cudaEvent_t>> readers;
};

constexpr int kMaxDevices = 64;
ConstBank g_bank[kMaxDevices];
std::atomic<uint64_t> g_next_id{1};

struct HostPipe {   // staging of pyro_source_terms_host
    static constexpr int kBuf = 3;
    int64_t slab = 0;
    double *rho[kBuf] = {}, *e[kBuf] = {}, *Tg[kBuf] = {}, *T[kBuf] = {}, *Y[kBuf] = {}, *omega[kBuf] = {};
    cudaStream_t s_in = nullptr, s_run = nullptr, s_out = nullptr;
    cudaEvent_t in_done[kBuf] = {}, run_done[kBuf] = {}, out_done[kBuf] = {};
    int32_t *d_bad = nullptr;
    bool ready = false;
};

}   // namespace

struct pyro_mech {
    uint64_t id = 0;
    int device = 0;
    pyro::PackedMech packed;
    unsigned char *d_blob = nullptr;
    pyro::EnergyRow *d_energy = nullptr;
    bool in_const = false;
    int block_threads = 32;
    int points_per_thread = 1;
    size_t smem_bytes = 0;
    int blocks_per_sm = 0;
    int sm_count = 0;
    double newton_tol = 1e-6;
    int newton_max_iter = 10;
    std::mutex pipe_mu;
    HostPipe pipe;
};

namespace {

void free_pipe(HostPipe &p) {
    for (int b = 0; b < HostPipe::kBuf; ++b) {
        cudaFree(p.rho[b]); cudaFree(p.e[b]); cudaFree(p.Tg[b]); cudaFree(p.T[b]); cudaFree(p.Y[b]); cudaFree(p.omega[b]);
        if (p.in_done[b]) cudaEventDestroy(p.in_done[b]);
        if (p.run_done[b]) cudaEventDestroy(p.run_done[b]);
        if (p.out_done[b]) cudaEventDestroy(p.out_done[b]);
    }
    if (p.s_in) cudaStreamDestroy(p.s_in);
    if (p.s_run) cudaStreamDestroy(p.s_run);
    if (p.s_out) cudaStreamDestroy(p.s_out);
    cudaFree(p.d_bad);
    p = HostPipe{};
}

int check_fields(const pyro_mech *m, int64_t n, int64_t ld) {
    if (!m) return fail(PYRO_ERR_NULL, "mech is NULL");
    if (n < 0) return fail(PYRO_ERR_BAD_SIZE, "n < 0");
    if (ld < n) return fail(PYRO_ERR_BAD_SIZE, "ld < n");
    return PYRO_OK;
}

bool aligned8(const void *p) { return (reinterpret_cast<uintptr_t>(p) & 7u) == 0; }

// Enqueue the rates kernel of `m` on `stream`, making its tables resident first.
int enqueue_rates(const pyro_mech *m, const pyro::RatesArgs &a, cudaStream_t stream) {
    if (!m->in_const) {
        PYRO_CUDA(pyro::launch_rates(a, m->block_threads, m->points_per_thread, false, m->smem_bytes, stream));
        return PYRO_OK;
    }
    ConstBank &bank = g_bank[m->device];
    std::lock_guard<std::mutex> lock(bank.mu);
    if (!bank.upload_done) PYRO_CUDA(cudaEventCreateWithFlags(&bank.upload_done, cudaEventDisableTiming));
    if (bank.resident != m->id) {
        // order the overwrite after every launch that may still read the old tables
        for (auto &r : bank.readers)
            if (r.first != stream) PYRO_CUDA(cudaStreamWaitEvent(stream, r.second, 0));
        PYRO_CUDA(pyro::upload_const_table(m->d_blob, m->packed.lay.bytes, stream));
        PYRO_CUDA(cudaEventRecord(bank.upload_done, stream));
        bank.upload_stream = stream;
        bank.resident = m->id;
        for (auto &r : bank.readers) cudaEventDestroy(r.second);
        bank.readers.clear();
    } else if (stream != bank.upload_stream) {
        PYRO_CUDA(cudaStreamWaitEvent(stream, bank.upload_done, 0));
    }
    PYRO_CUDA(pyro::launch_rates(a, m->block_threads, m->points_per_thread, true, m->smem_bytes, stream));
    cudaEvent_t ev = nullptr;
    for (auto &r : bank.readers)
        if (r.first == stream) ev = r.second;
    if (!ev) {
        if (bank.readers.size() >= 64) {   // too many distinct streams: fall back to a device-wide fence
            PYRO_CUDA(cudaDeviceSynchronize());
            for (auto &r : bank.readers) cudaEventDestroy(r.second);
            bank.readers.clear();
        }
        PYRO_CUDA(cudaEventCreateWithFlags(&ev, cudaEventDisableTiming));
        bank.readers.emplace_back(stream, ev);
    }
    PYRO_CUDA(cudaEventRecord(ev, stream));
    return PYRO_OK;
}

pyro::RatesArgs rates_args(const pyro_mech *m, int64_t n, int64_t ld, const double *rho, const double *T,
                           const double *Y, double *omega) {
    const pyro::TableLayout &l = m->packed.lay;
    pyro::RatesArgs a{};
    a.n = n; a.ld = ld; a.rho = rho; a.T = T; a.Y = Y; a.omega = omega;
    a.gtab = m->d_blob;
    a.off_spec = l.off_spec; a.off_rxn_p = l.off_rxn_p; a.off_rxn_x = l.off_rxn_x; a.off_fall = l.off_fall;
    a.off_eff_delta = l.off_eff_delta; a.off_eff_species = l.off_eff_species;
    a.n_species = l.n_species; a.n_p = l.n_p; a.n_x = l.n_x;
    for (int s = 0; s < 9; ++s) {
        a.shape_quads[s] = l.shape_quads[s];
        a.shape_pairs[s] = l.shape_pairs[s];
        a.shape_singles[s] = l.shape_singles[s];
    }
    for (int k = 0; k < 4; ++k) a.ext_count[k] = l.ext_count[k];
    return a;
}

pyro::TempArgs temp_args(const pyro_mech *m, int64_t n, int64_t ld, const double *e, const double *Y,
                         const double *Tg, double *T, int32_t *bad) {
    pyro::TempArgs a{};
    a.n = n; a.ld = ld; a.e = e; a.Y = Y; a.T_guess = Tg; a.T = T; a.n_not_converged = bad;
    a.energy = m->d_energy;
    a.n_species = m->packed.n_species;
    a.max_iter = m->newton_max_iter;
    a.t_mid = m->packed.lay.t_mid;
    a.tol = m->newton_tol;
    return a;
}

}   // namespace

extern "C" {

int pyro_mech_create(const pyro_mech_desc *desc, int device, pyro_mech **out) {
    if (!out) return fail(PYRO_ERR_NULL, "out is NULL");
    *out = nullptr;
    if (!desc) return fail(PYRO_ERR_NULL, "desc is NULL");
    auto *m = new pyro_mech();
    std::string err;
    int st = pyro::pack_mechanism(desc, m->packed, err);
    if (st != PYRO_OK) {
        delete m;
        return fail(st, err);
    }
    int ndev = 0;
    cudaError_t ce = cudaGetDeviceCount(&ndev);
    if (ce != cudaSuccess || ndev == 0) {
        delete m;
        return fail(PYRO_ERR_CUDA, std::string("no CUDA device: ") + cudaGetErrorString(ce) +
                                       " (libpyro has no CPU fallback)");
    }
    if (device < 0 || device >= ndev || device >= kMaxDevices) {
        delete m;
        return fail(PYRO_ERR_BAD_SIZE, "device index out of range");
    }
    DeviceGuard guard(device);
    if (!guard.ok) {
        delete m;
        return fail(PYRO_ERR_CUDA, "cudaSetDevice failed");
    }
    m->device = device;
    m->id = g_next_id.fetch_add(1);
    const pyro::TableLayout &lay = m->packed.lay;
    auto bail = [&](cudaError_t e, const char *what) {
        cudaFree(m->d_blob);
        cudaFree(m->d_energy);
        delete m;
        return cuda_fail(e, what);
    };
    if ((ce = cudaMalloc(&m->d_blob, lay.bytes > 0 ? lay.bytes : 8)) != cudaSuccess) return bail(ce, "cudaMalloc(tables)");
    if ((ce = cudaMemcpy(m->d_blob, m->packed.blob.data(), lay.bytes, cudaMemcpyHostToDevice)) != cudaSuccess)
        return bail(ce, "cudaMemcpy(tables)");
    const size_t ebytes = m->packed.energy.size() * sizeof(pyro::EnergyRow);
    if ((ce = cudaMalloc(&m->d_energy, ebytes)) != cudaSuccess) return bail(ce, "cudaMalloc(energy table)");
    if ((ce = cudaMemcpy(m->d_energy, m->packed.energy.data(), ebytes, cudaMemcpyHostToDevice)) != cudaSuccess)
        return bail(ce, "cudaMemcpy(energy table)");

    m->in_const = lay.bytes <= (uint32_t)pyro::kConstBankBytes;
    if (const char *env = std::getenv("PYRO_TABLES")) {
        if (!std::strcmp(env, "global")) m->in_const = false;
    }
    cudaDeviceProp prop;
    if ((ce = cudaGetDeviceProperties(&prop, device)) != cudaSuccess) return bail(ce, "cudaGetDeviceProperties");
    m->sm_count = prop.multiProcessorCount;
    // launch shape (threads per block, points per thread): with the three planes of n_species + 1
    // doubles per point in shared memory, take the variant that keeps at least two warps per
    // scheduler resident with the most points in flight; below that, the most warps.
    int forced_bd = 0, forced_p = 0;
    if (const char *env = std::getenv("PYRO_RATES_BLOCK")) forced_bd = std::atoi(env);
    if (const char *env = std::getenv("PYRO_RATES_POINTS")) forced_p = std::atoi(env);
    long best_score = -1;
    for (int p = 1; p <= 2; ++p)
        for (int bd = 32; bd <= 128; bd *= 2) {
            if ((forced_bd && bd != forced_bd) || (forced_p && p != forced_p)) continue;
            const size_t smem = (size_t)pyro::kPlanes * (lay.n_species + 1) * sizeof(double) * p * bd;
            if (smem > (size_t)prop.sharedMemPerBlockOptin) continue;
            const void *fn = pyro::rates_kernel_ptr(bd, p, m->in_const);
            // the limit is a property of the function, shared by every mechanism: always raise it to the
            // device maximum so that a later, smaller mechanism cannot lower it under an earlier one
            if ((ce = cudaFuncSetAttribute(fn, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                           (int)prop.sharedMemPerBlockOptin)) != cudaSuccess)
                return bail(ce, "cudaFuncSetAttribute(MaxDynamicSharedMemorySize)");
            int nblk = 0;
            if ((ce = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&nblk, fn, bd, smem)) != cudaSuccess)
                return bail(ce, "cudaOccupancyMaxActiveBlocksPerMultiprocessor");
            const long warps = (long)nblk * bd / 32, points = (long)nblk * bd * p;
            const long score = (warps < 8 ? warps : 8) * 100000 + points;
            if (nblk > 0 && score > best_score) {
                best_score = score;
                m->block_threads = bd;
                m->points_per_thread = p;
                m->smem_bytes = smem;
                m->blocks_per_sm = nblk;
            }
        }
    if (best_score < 0) {
        cudaFree(m->d_blob);
        cudaFree(m->d_energy);
        delete m;
        return fail(PYRO_ERR_TOO_LARGE, "species arrays do not fit the shared memory of one block");
    }
    *out = m;
    return PYRO_OK;
}

int pyro_mech_destroy(pyro_mech *m) {
    if (!m) return PYRO_OK;
    DeviceGuard guard(m->device);
    {
        std::lock_guard<std::mutex> lock(m->pipe_mu);
        if (m->pipe.ready) free_pipe(m->pipe);
    }
    cudaFree(m->d_blob);
    cudaFree(m->d_energy);
    delete m;
    return PYRO_OK;
}

int pyro_mech_set_newton(pyro_mech *m, double abs_tol_K, int max_iter) {
    if (!m) return fail(PYRO_ERR_NULL, "mech is NULL");
    if (!(abs_tol_K >= 0) || max_iter < 1) return fail(PYRO_ERR_BAD_SIZE, "abs_tol_K must be >= 0 and max_iter >= 1");
    m->newton_tol = abs_tol_K;
    m->newton_max_iter = max_iter;
    return PYRO_OK;
}

int pyro_get_temperature(const pyro_mech *m, int64_t n, int64_t ld, const double *rho, const double *e,
                         const double *Y, const double *T_guess, double *T, int32_t *n_not_converged,
                         void *cuda_stream) {
    (void)rho;   // the ideal-gas caloric equation of state does not depend on density (G23)
    int st = check_fields(m, n, ld);
    if (st != PYRO_OK) return st;
    if (n == 0) return PYRO_OK;
    if (!e || !Y || !T_guess || !T) return fail(PYRO_ERR_NULL, "a field pointer is NULL");
    if (!aligned8(e) || !aligned8(Y) || !aligned8(T_guess) || !aligned8(T) ||
        (reinterpret_cast<uintptr_t>(n_not_converged) & 3u))
        return fail(PYRO_ERR_ALIGN, "field pointers must be 8-byte aligned");
    if (!m->packed.lay.single_t_mid)
        return fail(PYRO_ERR_UNSUPPORTED,
                    "species with different T_mid: the temperature solve of this build sums the energy "
                    "polynomials per NASA range and needs one T_mid per mechanism");
    DeviceGuard guard(m->device);
    PYRO_CUDA(pyro::launch_temperature(temp_args(m, n, ld, e, Y, T_guess, T, n_not_converged),
                                       static_cast<cudaStream_t>(cuda_stream)));
    return PYRO_OK;
}

int pyro_get_net_production_rates(const pyro_mech *m, int64_t n, int64_t ld, const double *rho, const double *T,
                                  const double *Y, double *omega, void *cuda_stream) {
    int st = check_fields(m, n, ld);
    if (st != PYRO_OK) return st;
    if (n == 0) return PYRO_OK;
    if (!rho || !T || !Y || !omega) return fail(PYRO_ERR_NULL, "a field pointer is NULL");
    if (!aligned8(rho) || !aligned8(T) || !aligned8(Y) || !aligned8(omega))
        return fail(PYRO_ERR_ALIGN, "field pointers must be 8-byte aligned");
    if (omega == Y) return fail(PYRO_ERR_BAD_SIZE, "omega must not alias Y");
    DeviceGuard guard(m->device);
    return enqueue_rates(m, rates_args(m, n, ld, rho, T, Y, omega), static_cast<cudaStream_t>(cuda_stream));
}

int pyro_source_terms_host(pyro_mech *m, int64_t n, int64_t ld, const double *rho, const double *e,
                           const double *Y, const double *T_guess, double *T, double *omega,
                           int64_t *n_not_converged) {
    int st = check_fields(m, n, ld);
    if (st != PYRO_OK) return st;
    if (n_not_converged) *n_not_converged = 0;
    if (n == 0) return PYRO_OK;
    if (!rho || !e || !Y || !T_guess || !T || !omega) return fail(PYRO_ERR_NULL, "a field pointer is NULL");
    DeviceGuard guard(m->device);
    std::lock_guard<std::mutex> lock(m->pipe_mu);
    HostPipe &p = m->pipe;
    const int ns = m->packed.n_species;
    if (!p.ready) {
        // slab of points: about 64 MB of mass fractions per buffer
        int64_t slab = (int64_t)(64.0 * 1024 * 1024 / (8.0 * ns));
        slab = (slab / 1024) * 1024;
        if (slab < 4096) slab = 4096;
        if (const char *env = std::getenv("PYRO_HOST_SLAB")) slab = std::atoll(env) > 0 ? std::atoll(env) : slab;
        p.slab = slab;
        for (int b = 0; b < HostPipe::kBuf; ++b) {
            PYRO_CUDA(cudaMalloc(&p.rho[b], slab * 8));
            PYRO_CUDA(cudaMalloc(&p.e[b], slab * 8));
            PYRO_CUDA(cudaMalloc(&p.Tg[b], slab * 8));
            PYRO_CUDA(cudaMalloc(&p.T[b], slab * 8));
            PYRO_CUDA(cudaMalloc(&p.Y[b], slab * 8 * ns));
            PYRO_CUDA(cudaMalloc(&p.omega[b], slab * 8 * ns));
            PYRO_CUDA(cudaEventCreateWithFlags(&p.in_done[b], cudaEventDisableTiming));
            PYRO_CUDA(cudaEventCreateWithFlags(&p.run_done[b], cudaEventDisableTiming));
            PYRO_CUDA(cudaEventCreateWithFlags(&p.out_done[b], cudaEventDisableTiming));
        }
        PYRO_CUDA(cudaStreamCreateWithFlags(&p.s_in, cudaStreamNonBlocking));
        PYRO_CUDA(cudaStreamCreateWithFlags(&p.s_run, cudaStreamNonBlocking));
        PYRO_CUDA(cudaStreamCreateWithFlags(&p.s_out, cudaStreamNonBlocking));
        PYRO_CUDA(cudaMalloc(&p.d_bad, sizeof(int32_t)));
        p.ready = true;
    }
    PYRO_CUDA(cudaMemsetAsync(p.d_bad, 0, sizeof(int32_t), p.s_run));
    const int64_t slab = p.slab;
    int64_t i = 0;
    for (int64_t s0 = 0; s0 < n; s0 += slab, ++i) {
        const int b = (int)(i % HostPipe::kBuf);
        const int64_t cnt = (n - s0 < slab) ? (n - s0) : slab;
        // the buffer is free once the results of its previous slab have left
        if (i >= HostPipe::kBuf) PYRO_CUDA(cudaStreamWaitEvent(p.s_in, p.out_done[b], 0));
        PYRO_CUDA(cudaMemcpyAsync(p.rho[b], rho + s0, cnt * 8, cudaMemcpyHostToDevice, p.s_in));
        PYRO_CUDA(cudaMemcpyAsync(p.e[b], e + s0, cnt * 8, cudaMemcpyHostToDevice, p.s_in));
        PYRO_CUDA(cudaMemcpyAsync(p.Tg[b], T_guess + s0, cnt * 8, cudaMemcpyHostToDevice, p.s_in));
        PYRO_CUDA(cudaMemcpy2DAsync(p.Y[b], slab * 8, Y + s0, ld * 8, cnt * 8, ns, cudaMemcpyHostToDevice, p.s_in));
        PYRO_CUDA(cudaEventRecord(p.in_done[b], p.s_in));
        PYRO_CUDA(cudaStreamWaitEvent(p.s_run, p.in_done[b], 0));
        PYRO_CUDA(pyro::launch_temperature(temp_args(m, cnt, slab, p.e[b], p.Y[b], p.Tg[b], p.T[b], p.d_bad), p.s_run));
        st = enqueue_rates(m, rates_args(m, cnt, slab, p.rho[b], p.T[b], p.Y[b], p.omega[b]), p.s_run);
        if (st != PYRO_OK) return st;
        PYRO_CUDA(cudaEventRecord(p.run_done[b], p.s_run));
        PYRO_CUDA(cudaStreamWaitEvent(p.s_out, p.run_done[b], 0));
        PYRO_CUDA(cudaMemcpyAsync(T + s0, p.T[b], cnt * 8, cudaMemcpyDeviceToHost, p.s_out));
        PYRO_CUDA(cudaMemcpy2DAsync(omega + s0, ld * 8, p.omega[b], slab * 8, cnt * 8, ns, cudaMemcpyDeviceToHost, p.s_out));
        PYRO_CUDA(cudaEventRecord(p.out_done[b], p.s_out));
    }
    int32_t bad = 0;
    PYRO_CUDA(cudaMemcpyAsync(&bad, p.d_bad, sizeof bad, cudaMemcpyDeviceToHost, p.s_run));
    PYRO_CUDA(cudaStreamSynchronize(p.s_run));
    PYRO_CUDA(cudaStreamSynchronize(p.s_out));
    PYRO_CUDA(cudaStreamSynchronize(p.s_in));
    if (n_not_converged) *n_not_converged = bad;
    return PYRO_OK;
}

int pyro_mech_info(const pyro_mech *m, int64_t *out, int cap) {
    if (!m || !out) return -fail(PYRO_ERR_NULL, "NULL argument");
    DeviceGuard guard(m->device);
    cudaFuncAttributes fa{};
    cudaFuncGetAttributes(&fa, pyro::rates_kernel_ptr(m->block_threads, m->points_per_thread, m->in_const));
    const int64_t v[13] = {m->packed.n_species, m->packed.n_reactions, m->packed.lay.n_p, m->packed.lay.n_x,
                           (int64_t)m->packed.lay.bytes, m->in_const ? 1 : 0, m->block_threads,
                           (int64_t)m->smem_bytes, m->blocks_per_sm, fa.numRegs, (int64_t)fa.localSizeBytes,
                           m->sm_count, m->points_per_thread};
    int cnt = cap < 13 ? cap : 13;
    for (int i = 0; i < cnt; ++i) out[i] = v[i];
    return cnt;
}

int pyro_probe_fp64_peak(int device, double millis, double *tflops) {
    if (!tflops) return fail(PYRO_ERR_NULL, "tflops is NULL");
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || device < 0 || device >= ndev)
        return fail(PYRO_ERR_CUDA, "no such CUDA device");
    DeviceGuard guard(device);
    cudaDeviceProp prop;
    PYRO_CUDA(cudaGetDeviceProperties(&prop, device));
    double *d_out = nullptr;
    PYRO_CUDA(cudaMalloc(&d_out, 8));
    cudaEvent_t t0, t1;
    PYRO_CUDA(cudaEventCreate(&t0));
    PYRO_CUDA(cudaEventCreate(&t1));
    const int blocks = prop.multiProcessorCount * 8;
    int iters = 2000;
    float ms = 0;
    for (int pass = 0; pass < 3; ++pass) {
        PYRO_CUDA(pyro::launch_dfma_probe(d_out, iters, blocks, nullptr));   // warm-up
        PYRO_CUDA(cudaEventRecord(t0, nullptr));
        PYRO_CUDA(pyro::launch_dfma_probe(d_out, iters, blocks, nullptr));
        PYRO_CUDA(cudaEventRecord(t1, nullptr));
        PYRO_CUDA(cudaEventSynchronize(t1));
        PYRO_CUDA(cudaEventElapsedTime(&ms, t0, t1));
        if (ms >= 0.5 * millis || pass == 2) break;
        iters = (int)(iters * (millis / (ms > 1e-3 ? ms : 1e-3))) + 1;
    }
    const double fmas = (double)blocks * 256.0 * (double)iters * 64.0;
    *tflops = 2.0 * fmas / (ms * 1e-3) / 1e12;
    cudaEventDestroy(t0);
    cudaEventDestroy(t1);
    cudaFree(d_out);
    return PYRO_OK;
}

const char *pyro_status_string(int status) {
    switch (status) {
        case PYRO_OK: return "PYRO_OK";
        case PYRO_ERR_NULL: return "PYRO_ERR_NULL: a required pointer is NULL";
        case PYRO_ERR_BAD_SIZE: return "PYRO_ERR_BAD_SIZE: a size or count is out of range";
        case PYRO_ERR_BAD_MECH: return "PYRO_ERR_BAD_MECH: the mechanism description is inconsistent";
        case PYRO_ERR_TOO_LARGE: return "PYRO_ERR_TOO_LARGE: mechanism beyond the compiled limits";
        case PYRO_ERR_ALIGN: return "PYRO_ERR_ALIGN: a field pointer is not 8-byte aligned";
        case PYRO_ERR_CUDA: return "PYRO_ERR_CUDA: CUDA runtime error";
        case PYRO_ERR_UNSUPPORTED: return "PYRO_ERR_UNSUPPORTED: no kernel for this input in this build";
        default: return "unknown pyro_status";
    }
}

const char *pyro_last_error_string(void) { return g_last_error.c_str(); }

}   // extern "C"
