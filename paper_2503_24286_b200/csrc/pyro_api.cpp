// C-ABI layer of libpyro (include/pyro.h): handle management, argument checks, the
// launch configuration, launches, and the pipelined host-buffer entry point.
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

constexpr int kMaxDevices = 64;
constexpr uint32_t kWorkSlots = 64;     // chunk counters of one mechanism: launches that run at the same time

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

namespace pyro {
int set_last_error(int status, const std::string &msg) { return fail(status, msg); }
}   // namespace pyro

struct pyro_mech {
    int device = 0;
    pyro::PackedMech packed;
    unsigned char *d_blob = nullptr;
    pyro::EnergyRow *d_energy = nullptr;
    unsigned long long *d_work = nullptr;      // ring of chunk counters, one per launch in flight
    mutable std::atomic<uint32_t> next_work{0};
    mutable std::vector<cudaEvent_t> work_done;   // recorded after the launch that used the slot
    mutable std::mutex work_mu;
    bool tab_smem = false;     // tables staged in shared memory (else read from global memory)
    bool b_tmem = false;       // plane B in tensor memory beside omega (else in shared memory)
    bool two_blocks = false;   // the 128-register variant: two blocks resident per SM
    int block_threads = 32;    // = points per block
    size_t smem_bytes = 0;     // dynamic shared memory: tables (if staged) + the A/B planes
    uint32_t planes_off = 0;
    uint32_t tmem_cols = 32;
    int blocks_per_sm = 0;
    // two-points-per-thread rates kernel (pyro_rates2_kernels.cu), used by pyro_get_net_production_rates when it fits
    bool two_points = false;
    bool tab_smem2 = false;
    size_t smem2 = 0;
    uint32_t planes_off2 = 0, tmem_cols2 = 32;
    int blocks_per_sm2 = 1;   // resident blocks of the two-points-per-thread kernel
    size_t reactor_smem = 0;         // its dynamic shared memory: that of the rates kernel + the staged energy table
    uint32_t reactor_energy_off = 0;
    int reactor_blocks_per_sm = 1;   // resident blocks of the reactor kernel (same block shape as the rates kernel)
    int sm_count = 0;
    std::atomic<double> newton_tol{1e-6};      // read by concurrent calls while pyro_mech_set_newton may write
    std::atomic<int> newton_max_iter{10};
    std::mutex pipe_mu;
    HostPipe pipe;
    // chemical Jacobian (pyro_get_jacobian)
    bool jac_ok = false;       // false: more species than the kernel holds (pyro_get_jacobian returns PYRO_ERR_UNSUPPORTED)
    bool jac_small = true;     // plane V in tensor memory (else in shared memory)
    pyro::JacPacked jac;
    unsigned char *d_jblob = nullptr;
    double *d_jext = nullptr;  // per-thread scratch of the [M] reactions, [1 + 2 n_ext][jac_grid_threads]
    int jac_threads = 0, jac_blocks_per_sm = 0;
    size_t jac_smem = 0;
    uint32_t jac_planes_bytes = 0;
    // block-cooperative Jacobian kernel (pyro_jac_block_kernels.cu): 0 = not used, else warps per block
    int jac_block_warps = 0;
    bool jac_block_ext_global = false;   // its [M] scratch in global memory (mechanisms whose planes fill the shared memory)
    size_t jac_block_smem = 0;
    uint32_t jac_block_planes_bytes = 0, jac_block_tmem_cols = 32;
    uint32_t jac_tmem_cols = 32;
    mutable std::mutex jac_mu;
    cudaEvent_t jac_done = nullptr;   // launches on one handle share the scratch: each waits for the one before
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

// Enqueue the rates kernel of `m` on `stream`: persistent blocks, blocks_per_sm per SM at most.
int enqueue_rates(const pyro_mech *m, const pyro::RatesArgs &a, cudaStream_t stream, bool fused = false) {
    const int warps = m->block_threads / 32;
    int64_t blocks = (int64_t)m->sm_count * m->blocks_per_sm;
    if (blocks > (a.n_chunks + warps - 1) / warps) blocks = (a.n_chunks + warps - 1) / warps;
    pyro::RatesArgs args = a;
    const bool two = m->two_points && !fused;
    if (two) {   // 64-point chunks, one warp per lane quarter
        args.n_chunks = (a.n + 63) / 64;
        args.planes_off = m->planes_off2;
        args.tmem_cols = m->tmem_cols2;
        blocks = (int64_t)m->sm_count * m->blocks_per_sm2;
        const int64_t need = (args.n_chunks + pyro::kRates2Threads / 32 - 1) / (pyro::kRates2Threads / 32);
        if (blocks > need) blocks = need;
    }
    // every launch in flight needs its own chunk counter: take the next slot of the ring and, before
    // resetting it, make this stream wait for the launch that used the slot kWorkSlots launches ago
    const uint32_t slot = m->next_work.fetch_add(1) % kWorkSlots;
    args.work = m->d_work + slot;
    std::lock_guard<std::mutex> lock(m->work_mu);
    PYRO_CUDA(cudaStreamWaitEvent(stream, m->work_done[slot], 0));
    PYRO_CUDA(cudaMemsetAsync(args.work, 0, sizeof(unsigned long long), stream));
    if (two)
        PYRO_CUDA(pyro::launch_rates2(args, pyro::kRates2Threads, (int)blocks, m->tab_smem2, m->two_blocks, m->smem2, stream));
    else
        PYRO_CUDA(pyro::launch_rates(args, m->block_threads, (int)blocks, m->tab_smem, m->b_tmem, m->two_blocks, m->smem_bytes, stream,
                                     fused));
    PYRO_CUDA(cudaEventRecord(m->work_done[slot], stream));
    return PYRO_OK;
}

pyro::RatesArgs rates_args(const pyro_mech *m, int64_t n, int64_t ld, const double *rho, const double *T,
                           const double *Y, double *omega) {
    const pyro::TableLayout &l = m->packed.lay;
    pyro::RatesArgs a{};
    a.n = n; a.ld = ld; a.rho = rho; a.T = T; a.Y = Y; a.omega = omega;
    a.n_chunks = (n + 31) / 32;
    a.gtab = m->d_blob;
    a.tab_bytes = l.bytes;
    a.planes_off = m->planes_off;
    a.tmem_cols = m->tmem_cols;
    a.off_spec = l.off_spec; a.off_rxn_p = l.off_rxn_p; a.off_rxn_x = l.off_rxn_x; a.off_fall = l.off_fall;
    a.off_eff = l.off_eff;
    a.n_species = l.n_species;
    for (int s = 0; s < 9; ++s) {
        a.groups.shape_g8[s] = l.shape_g8[s];
        a.groups.shape_g4[s] = l.shape_g4[s];
        a.groups.shape_g2[s] = l.shape_g2[s];
        a.groups.shape_g1[s] = l.shape_g1[s];
    }
    for (int k = 0; k < 4; ++k) {
        a.groups.ext_g4[k] = l.ext_g4[k];
        a.groups.ext_g2[k] = l.ext_g2[k];
        a.groups.ext_g1[k] = l.ext_g1[k];
    }
    return a;
}

pyro::TempArgs temp_args(const pyro_mech *m, int64_t n, int64_t ld, const double *e, const double *Y,
                         const double *Tg, double *T, int32_t *bad) {
    pyro::TempArgs a{};
    a.n = n; a.ld = ld; a.e = e; a.Y = Y; a.T_guess = Tg; a.T = T; a.n_not_converged = bad;
    a.energy = m->d_energy;
    a.n_species = m->packed.n_species;
    a.max_iter = m->newton_max_iter.load(std::memory_order_relaxed);
    a.t_mid = m->packed.lay.t_mid;
    a.tol = m->newton_tol.load(std::memory_order_relaxed);
    a.enthalpy = 0;
    a.single_t_mid = m->packed.lay.single_t_mid;
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
    int st = pyro::pack_mechanism(desc, m->packed, err, pyro::kLeftoverPad);
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
    const pyro::TableLayout &lay = m->packed.lay;
    auto release = [&]() {
        cudaFree(m->d_blob);
        cudaFree(m->d_energy);
        cudaFree(m->d_work);
        cudaFree(m->d_jblob);
        cudaFree(m->d_jext);
        if (m->jac_done) cudaEventDestroy(m->jac_done);
        for (cudaEvent_t ev : m->work_done)
            if (ev) cudaEventDestroy(ev);
        delete m;
    };
    auto bail = [&](cudaError_t e, const char *what) {
        release();
        return cuda_fail(e, what);
    };
    if ((ce = cudaMalloc(&m->d_blob, lay.bytes > 0 ? lay.bytes : 8)) != cudaSuccess) return bail(ce, "cudaMalloc(tables)");
    if ((ce = cudaMemcpy(m->d_blob, m->packed.blob.data(), lay.bytes, cudaMemcpyHostToDevice)) != cudaSuccess)
        return bail(ce, "cudaMemcpy(tables)");
    if ((ce = cudaMalloc(&m->d_work, kWorkSlots * sizeof(unsigned long long))) != cudaSuccess)
        return bail(ce, "cudaMalloc(work counters)");
    m->work_done.assign(kWorkSlots, nullptr);
    for (uint32_t i = 0; i < kWorkSlots; ++i)
        if ((ce = cudaEventCreateWithFlags(&m->work_done[i], cudaEventDisableTiming)) != cudaSuccess)
            return bail(ce, "cudaEventCreate(work counters)");
    const size_t ebytes = m->packed.energy.size() * sizeof(pyro::EnergyRow);
    if ((ce = cudaMalloc(&m->d_energy, ebytes)) != cudaSuccess) return bail(ce, "cudaMalloc(energy table)");
    if ((ce = cudaMemcpy(m->d_energy, m->packed.energy.data(), ebytes, cudaMemcpyHostToDevice)) != cudaSuccess)
        return bail(ce, "cudaMemcpy(energy table)");

    cudaDeviceProp prop;
    if ((ce = cudaGetDeviceProperties(&prop, device)) != cudaSuccess) return bail(ce, "cudaGetDeviceProperties");
    m->sm_count = prop.multiProcessorCount;
    // Launch shape.  A point needs, per species row, one double in shared memory (plane A) and four
    // 32-bit tensor-memory columns (planes W and B); warps share the 128 tensor-memory lanes four at a
    // time, so a block of w warps takes ceil(w/4) column groups of 4 rows columns out of 512.
    // Mechanisms of more than 127 species keep B in a second shared-memory plane (2 columns per
    // row).  Take the most threads (a multiple of 32, at most kRatesMaxThreads) that fit, with the
    // tables staged in shared memory unless that costs more than 40 % of the points.
    const size_t rows = (size_t)lay.n_species + 1;
    size_t static_smem = 0;   // the kernels keep the tensor-memory base address in static shared memory
    for (int v = 0; v < 8; ++v) {
        cudaFuncAttributes fa{};
        if ((ce = cudaFuncGetAttributes(&fa, pyro::rates_kernel_ptr((v & 1) != 0, (v & 2) != 0, (v & 4) != 0))) != cudaSuccess)
            return bail(ce, "cudaFuncGetAttributes");
        if (fa.sharedSizeBytes > static_smem) static_smem = fa.sharedSizeBytes;
    }
    const size_t smem_max = (size_t)prop.sharedMemPerBlockOptin - static_smem;
    const size_t tab_room = ((size_t)lay.bytes + 15) & ~(size_t)15;
    m->b_tmem = 4 * rows <= 512;
    if (const char *env = std::getenv("PYRO_B_PLANE")) {
        if (!std::strcmp(env, "shared")) m->b_tmem = false;
    }
    const size_t smem_row = m->b_tmem ? 8 : 16, cols_row = m->b_tmem ? 4 : 2;
    auto threads_for = [&](size_t table_bytes) {
        if (smem_max < table_bytes + smem_row * rows * 32) return 0;
        size_t t = (smem_max - table_bytes) / (smem_row * rows);
        t = (t / 32) * 32;
        const size_t groups_max = 512 / (cols_row * rows);
        if (t > 128 * groups_max) t = 128 * groups_max;
        if (t > (size_t)pyro::kRatesMaxThreads) t = pyro::kRatesMaxThreads;
        return (int)t;
    };
    int t_smem = threads_for(tab_room), t_glob = threads_for(0);
    if (const char *env = std::getenv("PYRO_TABLES")) {
        if (!std::strcmp(env, "global")) t_smem = 0;
        if (!std::strcmp(env, "shared")) t_glob = 0;
    }
    m->tab_smem = t_smem > 0 && 10 * t_smem >= 6 * t_glob;
    int threads = m->tab_smem ? t_smem : t_glob;
    if (const char *env = std::getenv("PYRO_RATES_BLOCK")) {
        const int forced = std::atoi(env);
        if (forced >= 32 && forced % 32 == 0 && forced <= threads) threads = forced;
    }
    if (threads < 32) {
        release();
        return fail(PYRO_ERR_TOO_LARGE, "species arrays do not fit the on-chip memory of one block");
    }
    auto shape = [&](int t, size_t &smem, uint32_t &cols) {
        const uint32_t groups = (uint32_t)((t / 32 + 3) / 4);
        const uint32_t need = (uint32_t)(groups * cols_row * rows);
        cols = 32;
        while (cols < need) cols *= 2;
        smem = (m->tab_smem ? tab_room : 0) + smem_row * rows * (size_t)t;
    };
    // Small mechanisms: two blocks of 224 threads per SM with the 128-register variant (two blocks of
    // 256 threads would need the whole register file, which the hardware does not grant), when shared
    // and tensor memory allow it.
    m->two_blocks = false;
    if (threads >= 224 && !std::getenv("PYRO_RATES_BLOCK")) {
        size_t smem2;
        uint32_t cols2;
        shape(224, smem2, cols2);
        if (2 * (smem2 + static_smem + 1024) <= (size_t)prop.sharedMemPerMultiprocessor && 2 * cols2 <= 512) {
            m->two_blocks = true;
            threads = 224;
        }
    }
    if (const char *env = std::getenv("PYRO_RATES_TWO_BLOCKS")) m->two_blocks = m->two_blocks && std::atoi(env) != 0;
    m->block_threads = threads;
    m->planes_off = m->tab_smem ? (uint32_t)tab_room : 0u;
    shape(threads, m->smem_bytes, m->tmem_cols);
    const void *fn = pyro::rates_kernel_ptr(m->tab_smem, m->b_tmem, m->two_blocks);
    // the limit is a property of the function, shared by every mechanism: always raise it to the
    // device maximum so that a later, smaller mechanism cannot lower it under an earlier one
    if ((ce = cudaFuncSetAttribute(fn, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_max)) != cudaSuccess)
        return bail(ce, "cudaFuncSetAttribute(MaxDynamicSharedMemorySize)");
    // Carve-out of the SM's L1/shared array: all of it as shared memory for the one-block shape; for the
    // two-block shape of small mechanisms only what the two blocks need, the rest stays L1 for the
    // spills of the 128-register build and for the global loads.
    int carveout = cudaSharedmemCarveoutMaxShared;
    if (m->two_blocks) {
        const size_t need = 2 * (m->smem_bytes + static_smem + 1024) + 8192;
        carveout = (int)((100 * need + prop.sharedMemPerMultiprocessor - 1) / prop.sharedMemPerMultiprocessor);
        if (carveout > 100) carveout = 100;
    }
    if (const char *env = std::getenv("PYRO_CARVEOUT")) carveout = std::atoi(env);
    if ((ce = cudaFuncSetAttribute(fn, cudaFuncAttributePreferredSharedMemoryCarveout, carveout)) != cudaSuccess)
        return bail(ce, "cudaFuncSetAttribute(PreferredSharedMemoryCarveout)");
    // Two points per thread (pyro_rates2_kernels.cu): 128 threads hold the same 256 points; needs eight tensor-memory
    // columns per species row and the A plane of both points (16 bytes per row and thread) in shared memory.  Used for
    // mechanisms that run the one-block shape (not the two-block shape of small mechanisms).
    if (8 * rows <= 512) {
        const size_t planes2 = 16 * rows * (size_t)pyro::kRates2Threads;
        const void *fn2s = pyro::rates2_kernel_ptr(true, m->two_blocks), *fn2g = pyro::rates2_kernel_ptr(false, m->two_blocks);
        cudaFuncAttributes fa2{};
        if ((ce = cudaFuncGetAttributes(&fa2, fn2s)) != cudaSuccess) return bail(ce, "cudaFuncGetAttributes(rates2)");
        const size_t smem_max2 = (size_t)prop.sharedMemPerBlockOptin - fa2.sharedSizeBytes;
        bool ok = false;
        if (tab_room + planes2 <= smem_max2 && m->tab_smem) {
            m->tab_smem2 = true;
            m->planes_off2 = (uint32_t)tab_room;
            m->smem2 = tab_room + planes2;
            ok = true;
        } else if (planes2 <= smem_max2) {
            m->tab_smem2 = false;
            m->planes_off2 = 0;
            m->smem2 = planes2;
            ok = true;
        }
        if (ok) {
            m->tmem_cols2 = 32;
            while (m->tmem_cols2 < 8 * rows) m->tmem_cols2 *= 2;
            // small mechanisms: as many blocks per SM as shared memory, tensor memory and the register file hold
            {
                const size_t regs_block = (size_t)((fa2.numRegs + 7) / 8 * 8) * pyro::kRates2Threads;
                int nb = (int)(prop.sharedMemPerMultiprocessor / (m->smem2 + fa2.sharedSizeBytes + 1024));
                nb = std::min(nb, (int)(512 / m->tmem_cols2));
                nb = std::min(nb, (int)((size_t)prop.regsPerMultiprocessor / regs_block));
                m->blocks_per_sm2 = std::max(1, std::min(nb, 4));
                if (std::getenv("PYRO_DEBUG"))
                    std::fprintf(stderr, "pyro: two-point kernel regs %d smem %zu tmem_cols %u blocks per SM %d\n", fa2.numRegs, m->smem2, m->tmem_cols2, m->blocks_per_sm2);
            }
            for (const void *f2 : {fn2s, fn2g}) {
                if ((ce = cudaFuncSetAttribute(f2, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_max2)) != cudaSuccess)
                    return bail(ce, "cudaFuncSetAttribute(rates2, MaxDynamicSharedMemorySize)");
                if ((ce = cudaFuncSetAttribute(f2, cudaFuncAttributePreferredSharedMemoryCarveout, cudaSharedmemCarveoutMaxShared)) != cudaSuccess)
                    return bail(ce, "cudaFuncSetAttribute(rates2, carveout)");
            }
            // Large mechanisms (one block per SM): measured slower than the one-point kernel (configs[2]: 7.58 against
            // 7.09 ms -- 27 % fewer instructions, but one warp per scheduler issues on 45 % of the cycles against 66 % for
            // two; profiles/r02_dead_ends.md).  Small mechanisms, where two blocks of it are resident per SM (two warps
            // per scheduler, as the one-point kernel, with the fewer instructions): faster (configs[1]: 2.26 against
            // 2.64 ms) and the library's choice.  PYRO_RATES_POINTS=1|2 forces either (tests, measurements).
            m->two_points = m->two_blocks && m->b_tmem && m->blocks_per_sm2 >= 2;   // (b_tmem false: the PYRO_B_PLANE hook asks for the one-point variant)
            if (const char *env = std::getenv("PYRO_RATES_POINTS")) m->two_points = std::atoi(env) == 2;
        }
    }
    {   // the reactor kernel of the same shape (pyro_reactor_rk4)
        const void *rfn = pyro::reactor_kernel_ptr(m->tab_smem, m->b_tmem, m->two_blocks);
        if ((ce = cudaFuncSetAttribute(rfn, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_max)) != cudaSuccess)
            return bail(ce, "cudaFuncSetAttribute(reactor, MaxDynamicSharedMemorySize)");
        if ((ce = cudaFuncSetAttribute(rfn, cudaFuncAttributePreferredSharedMemoryCarveout, carveout)) != cudaSuccess)
            return bail(ce, "cudaFuncSetAttribute(reactor, PreferredSharedMemoryCarveout)");
        m->reactor_smem = m->smem_bytes;
        m->reactor_energy_off = 0;
        const size_t etab = (size_t)lay.n_species * sizeof(pyro::EnergyRow);
        const size_t eoff = (m->smem_bytes + 15) & ~(size_t)15;
        // (two-block shape of small mechanisms: the table is a few KB, inside the slack of the carve-out above)
        if (eoff + etab <= smem_max && (!m->two_blocks || etab <= 4096)) {
            m->reactor_energy_off = (uint32_t)eoff;
            m->reactor_smem = eoff + etab;
        }
        int rblk = 0;
        if ((ce = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&rblk, rfn, threads, m->reactor_smem)) != cudaSuccess)
            return bail(ce, "cudaOccupancyMaxActiveBlocksPerMultiprocessor(reactor)");
        if (rblk > (int)(512 / m->tmem_cols)) rblk = (int)(512 / m->tmem_cols);
        m->reactor_blocks_per_sm = rblk < 1 ? 1 : rblk;
    }
    {   // the fused temperature + rates kernel of the same shape (pyro_source_terms)
        const void *ffn = pyro::fused_kernel_ptr(m->tab_smem, m->b_tmem, m->two_blocks);
        if ((ce = cudaFuncSetAttribute(ffn, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_max)) != cudaSuccess)
            return bail(ce, "cudaFuncSetAttribute(fused, MaxDynamicSharedMemorySize)");
        if ((ce = cudaFuncSetAttribute(ffn, cudaFuncAttributePreferredSharedMemoryCarveout, carveout)) != cudaSuccess)
            return bail(ce, "cudaFuncSetAttribute(fused, PreferredSharedMemoryCarveout)");
    }
    int nblk = 0;
    if ((ce = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&nblk, fn, threads, m->smem_bytes)) != cudaSuccess)
        return bail(ce, "cudaOccupancyMaxActiveBlocksPerMultiprocessor");
    if (std::getenv("PYRO_DEBUG")) {
        cudaFuncAttributes fa{};
        cudaFuncGetAttributes(&fa, fn);
        std::fprintf(stderr, "pyro: threads %d smem %zu static %zu regs %d local %zu tmem_cols %u occupancy %d two_blocks %d\n",
                     threads, m->smem_bytes, (size_t)fa.sharedSizeBytes, fa.numRegs, (size_t)fa.localSizeBytes, m->tmem_cols, nblk,
                     (int)m->two_blocks);
    }
    // The occupancy query answers 1 for the 128-register variant although two blocks of 224 threads
    // are resident together (measured: 4.9 -> 3.8 ms at configs[1] with two blocks per SM); registers
    // (2 x 224 x 128), shared memory and tensor-memory columns were checked above.
    if (m->two_blocks && nblk < 2) nblk = 2;
    if (nblk > (int)(512 / m->tmem_cols)) nblk = (int)(512 / m->tmem_cols);   // resident blocks share 512 columns
    if (nblk < 1) {
        release();
        return fail(PYRO_ERR_TOO_LARGE, "the rates kernel does not fit one SM for this mechanism");
    }
    m->blocks_per_sm = nblk;
    // The two-block kernel of small mechanisms contains the one-at-a-time loops: store the reactions
    // that the lockstep grouping left alone as singles instead of coupling them with null records
    // (the tables only shrink, so the shape chosen above stands).
    if (m->two_blocks) {
        pyro::PackedMech again;
        if (pyro::pack_mechanism(desc, again, err, pyro::kLeftoverSingles) == PYRO_OK && again.lay.bytes <= lay.bytes) {
            m->packed = again;
            if ((ce = cudaMemcpy(m->d_blob, m->packed.blob.data(), m->packed.lay.bytes, cudaMemcpyHostToDevice)) != cudaSuccess)
                return bail(ce, "cudaMemcpy(tables)");
        }
    }
    // ---- chemical Jacobian: tables, launch shape, scratch (mechanisms beyond its species limit keep everything else)
    if (lay.n_species <= pyro::kJacMaxSpecies) {
        st = pyro::pack_jacobian(desc, m->jac, err);
        if (st != PYRO_OK) {
            release();
            return fail(st, err);
        }
        const pyro::JacLayout &jl = m->jac.lay;
        if ((ce = cudaMalloc(&m->d_jblob, jl.bytes > 0 ? jl.bytes : 16)) != cudaSuccess) return bail(ce, "cudaMalloc(Jacobian tables)");
        if ((ce = cudaMemcpy(m->d_jblob, m->jac.blob.data(), jl.bytes, cudaMemcpyHostToDevice)) != cudaSuccess)
            return bail(ce, "cudaMemcpy(Jacobian tables)");
        // Per point: planes C, G, dG/dT in shared memory; accumulators W, V, dS/dT in tensor memory, 6 columns per
        // species row (one warp per lane quarter: at most 128 threads per block) if they fit 512 columns, else V
        // moves to a fourth shared-memory plane (4 columns per row).
        m->jac_small = 6 * rows + 2 <= 512;
        if (const char *env = std::getenv("PYRO_JAC_V_PLANE")) {
            if (!std::strcmp(env, "shared")) m->jac_small = false;
        }
        const size_t planes = m->jac_small ? 3 : 4;
        // The block-cooperative kernel (NW warps on one chunk of 32 points, planes once per chunk) when its shared
        // memory fits: 5 planes + the [M] scratch + 2 NW reduction rows of 32 doubles, and NW record rings.
        // (not for small mechanisms: with fewer columns than warps most of the block idles; measured at 9 species:
        // 4.8 against 2.2 ns per point)
        for (int shape = 0; shape < 4 && !m->jac_block_warps; ++shape) {
            const int nw = shape < 2 ? 16 : 8;
            const bool ext_global = shape & 1;   // second choice: the [M] scratch in global memory
            if (lay.n_species < 24 && !std::getenv("PYRO_JAC_KERNEL")) break;
            if (const char *env = std::getenv("PYRO_JAC_EXT")) {
                if (!std::strcmp(env, "global") && !ext_global) continue;
            }
            if (2 * rows * (size_t)(nw / 4) > 512) continue;
            const size_t pl = (5 * rows + (ext_global ? 0 : 1 + 2 * (size_t)jl.n_ext) + 2 * (size_t)nw + 8 * (size_t)nw) * 32 * sizeof(double);   // + reduction scratch
            const size_t need = pl + (size_t)nw * pyro::kJacBlockRingBytes;
            cudaFuncAttributes fb{};
            const void *bfn = pyro::jacobian_block_kernel_ptr(nw);
            if ((ce = cudaFuncGetAttributes(&fb, bfn)) != cudaSuccess) return bail(ce, "cudaFuncGetAttributes(jacobian block)");
            if (need + fb.sharedSizeBytes > (size_t)prop.sharedMemPerBlockOptin) continue;
            if ((ce = cudaFuncSetAttribute(bfn, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)((size_t)prop.sharedMemPerBlockOptin - fb.sharedSizeBytes))) != cudaSuccess)
                return bail(ce, "cudaFuncSetAttribute(jacobian block)");
            m->jac_block_ext_global = ext_global;
            m->jac_block_warps = nw;
            m->jac_block_smem = need;
            m->jac_block_planes_bytes = (uint32_t)pl;
            m->jac_block_tmem_cols = 32;
            while (m->jac_block_tmem_cols < 2 * rows * (size_t)(nw / 4)) m->jac_block_tmem_cols *= 2;
        }
        if (const char *env = std::getenv("PYRO_JAC_KERNEL")) {
            if (!std::strcmp(env, "point")) m->jac_block_warps = 0;   // "block": also for small mechanisms (tests)
        }
        cudaFuncAttributes fa{};
        const void *jfn = pyro::jacobian_kernel_ptr(m->jac_small);
        if ((ce = cudaFuncGetAttributes(&fa, jfn)) != cudaSuccess) return bail(ce, "cudaFuncGetAttributes(jacobian)");
        const size_t jsmem_max = (size_t)prop.sharedMemPerBlockOptin - fa.sharedSizeBytes;
        size_t jt = jsmem_max / (planes * 8 * rows + pyro::kJacRingBytes / 32);   // + the warp's share of its record ring
        jt = (jt / 32) * 32;
        if (jt > (size_t)pyro::kJacMaxThreads) jt = pyro::kJacMaxThreads;
        if (const char *env = std::getenv("PYRO_JAC_BLOCK")) {
            const size_t forced = (size_t)std::atoi(env);
            if (forced >= 32 && forced % 32 == 0 && forced <= jt) jt = forced;
        }
        if (jt >= 32) {
            m->jac_threads = (int)jt;
            m->jac_planes_bytes = (uint32_t)(planes * 8 * rows * jt);
            m->jac_smem = m->jac_planes_bytes + (jt / 32) * pyro::kJacRingBytes;
            const uint32_t need = (uint32_t)((m->jac_small ? 6 : 4) * rows + (m->jac_small ? 2 : 0));
            m->jac_tmem_cols = 32;
            while (m->jac_tmem_cols < need) m->jac_tmem_cols *= 2;
            if ((ce = cudaFuncSetAttribute(jfn, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)jsmem_max)) != cudaSuccess)
                return bail(ce, "cudaFuncSetAttribute(jacobian)");
            int jblk = 0;
            if ((ce = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&jblk, jfn, m->jac_threads, m->jac_smem)) != cudaSuccess)
                return bail(ce, "cudaOccupancyMaxActiveBlocksPerMultiprocessor(jacobian)");
            if (jblk > (int)(512 / m->jac_tmem_cols)) jblk = (int)(512 / m->jac_tmem_cols);
            if (jblk >= 1) {
                m->jac_blocks_per_sm = jblk;
                const size_t grid_threads = (size_t)m->sm_count * jblk * jt;
                if ((ce = cudaMalloc(&m->d_jext, (size_t)(1 + 2 * jl.n_ext) * grid_threads * sizeof(double))) != cudaSuccess)
                    return bail(ce, "cudaMalloc(Jacobian scratch)");
                if ((ce = cudaEventCreateWithFlags(&m->jac_done, cudaEventDisableTiming)) != cudaSuccess)
                    return bail(ce, "cudaEventCreate(jacobian)");
                m->jac_ok = true;
            }
        }
    }
    *out = m;
    return PYRO_OK;
}

int pyro_mech_destroy(pyro_mech *m) {
    if (!m) return PYRO_OK;
    DeviceGuard guard(m->device);
    {
        std::lock_guard<std::mutex> lock(m->pipe_mu);
        free_pipe(m->pipe);
    }
    cudaFree(m->d_blob);
    cudaFree(m->d_energy);
    cudaFree(m->d_work);
    cudaFree(m->d_jblob);
    cudaFree(m->d_jext);
    if (m->jac_done) cudaEventDestroy(m->jac_done);
    for (cudaEvent_t ev : m->work_done)
        if (ev) cudaEventDestroy(ev);
    delete m;
    return PYRO_OK;
}

int pyro_mech_set_newton(pyro_mech *m, double abs_tol_K, int max_iter) {
    if (!m) return fail(PYRO_ERR_NULL, "mech is NULL");
    if (!(abs_tol_K >= 0) || max_iter < 1) return fail(PYRO_ERR_BAD_SIZE, "abs_tol_K must be >= 0 and max_iter >= 1");
    m->newton_tol.store(abs_tol_K, std::memory_order_relaxed);
    m->newton_max_iter.store(max_iter, std::memory_order_relaxed);
    return PYRO_OK;
}

namespace {
int temperature_call(const pyro_mech *m, int64_t n, int64_t ld, const double *e, const double *Y, const double *T_guess,
                     double *T, int32_t *n_not_converged, void *cuda_stream, bool enthalpy) {
    int st = check_fields(m, n, ld);
    if (st != PYRO_OK) return st;
    if (n == 0) return PYRO_OK;
    if (!e || !Y || !T_guess || !T) return fail(PYRO_ERR_NULL, "a field pointer is NULL");
    if (!aligned8(e) || !aligned8(Y) || !aligned8(T_guess) || !aligned8(T) ||
        (reinterpret_cast<uintptr_t>(n_not_converged) & 3u))
        return fail(PYRO_ERR_ALIGN, "field pointers must be 8-byte aligned");
    DeviceGuard guard(m->device);
    pyro::TempArgs a = temp_args(m, n, ld, e, Y, T_guess, T, n_not_converged);
    a.enthalpy = enthalpy ? 1 : 0;
    PYRO_CUDA(pyro::launch_temperature(a, static_cast<cudaStream_t>(cuda_stream)));
    return PYRO_OK;
}

int eos_call(const pyro_mech *m, int64_t n, int64_t ld, const double *in, const double *T, const double *Y,
             double *out, void *cuda_stream, bool to_density) {
    int st = check_fields(m, n, ld);
    if (st != PYRO_OK) return st;
    if (n == 0) return PYRO_OK;
    if (!in || !T || !Y || !out) return fail(PYRO_ERR_NULL, "a field pointer is NULL");
    if (!aligned8(in) || !aligned8(T) || !aligned8(Y) || !aligned8(out))
        return fail(PYRO_ERR_ALIGN, "field pointers must be 8-byte aligned");
    DeviceGuard guard(m->device);
    pyro::EosArgs a{};
    a.n = n; a.ld = ld; a.in = in; a.T = T; a.Y = Y; a.out = out;
    a.energy = m->d_energy;
    a.n_species = m->packed.n_species;
    a.to_density = to_density ? 1 : 0;
    PYRO_CUDA(pyro::launch_eos(a, static_cast<cudaStream_t>(cuda_stream)));
    return PYRO_OK;
}
}   // namespace

int pyro_get_temperature(const pyro_mech *m, int64_t n, int64_t ld, const double *rho, const double *e,
                         const double *Y, const double *T_guess, double *T, int32_t *n_not_converged,
                         void *cuda_stream) {
    (void)rho;   // the ideal-gas caloric equation of state does not depend on density (G23)
    return temperature_call(m, n, ld, e, Y, T_guess, T, n_not_converged, cuda_stream, false);
}

int pyro_get_temperature_from_enthalpy(const pyro_mech *m, int64_t n, int64_t ld, const double *h, const double *Y,
                                       const double *T_guess, double *T, int32_t *n_not_converged,
                                       void *cuda_stream) {
    return temperature_call(m, n, ld, h, Y, T_guess, T, n_not_converged, cuda_stream, true);
}

int pyro_get_density(const pyro_mech *m, int64_t n, int64_t ld, const double *p, const double *T, const double *Y,
                     double *rho, void *cuda_stream) {
    return eos_call(m, n, ld, p, T, Y, rho, cuda_stream, true);
}

int pyro_get_pressure(const pyro_mech *m, int64_t n, int64_t ld, const double *rho, const double *T, const double *Y,
                      double *p, void *cuda_stream) {
    return eos_call(m, n, ld, rho, T, Y, p, cuda_stream, false);
}

int pyro_get_net_production_rates(const pyro_mech *m, int64_t n, int64_t ld, const double *rho, const double *T,
                                  const double *Y, double *omega, void *cuda_stream) {
    int st = check_fields(m, n, ld);
    if (st != PYRO_OK) return st;
    if (n == 0) return PYRO_OK;
    if (!rho || !T || !Y || !omega) return fail(PYRO_ERR_NULL, "a field pointer is NULL");
    if (!aligned8(rho) || !aligned8(T) || !aligned8(Y) || !aligned8(omega))
        return fail(PYRO_ERR_ALIGN, "field pointers must be 8-byte aligned");
    {   // omega is written while Y of other points is still being read: no overlap of the two fields at all
        const uintptr_t span = (uintptr_t)(((int64_t)m->packed.n_species - 1) * ld + n) * sizeof(double);
        const uintptr_t y0 = reinterpret_cast<uintptr_t>(Y), w0 = reinterpret_cast<uintptr_t>(omega);
        if (y0 < w0 + span && w0 < y0 + span) return fail(PYRO_ERR_BAD_SIZE, "omega must not overlap Y");
    }
    DeviceGuard guard(m->device);
    return enqueue_rates(m, rates_args(m, n, ld, rho, T, Y, omega), static_cast<cudaStream_t>(cuda_stream));
}

int pyro_source_terms(const pyro_mech *m, int64_t n, int64_t ld, const double *rho, const double *e, const double *Y,
                      const double *T_guess, double *T, double *omega, int32_t *n_not_converged, void *cuda_stream) {
    int st = check_fields(m, n, ld);
    if (st != PYRO_OK) return st;
    if (n == 0) return PYRO_OK;
    if (!rho || !e || !Y || !T_guess || !T || !omega) return fail(PYRO_ERR_NULL, "a field pointer is NULL");
    if (!aligned8(rho) || !aligned8(e) || !aligned8(Y) || !aligned8(T_guess) || !aligned8(T) || !aligned8(omega) ||
        (reinterpret_cast<uintptr_t>(n_not_converged) & 3u))
        return fail(PYRO_ERR_ALIGN, "field pointers must be 8-byte aligned");
    {
        const uintptr_t span = (uintptr_t)(((int64_t)m->packed.n_species - 1) * ld + n) * sizeof(double);
        const uintptr_t y0 = reinterpret_cast<uintptr_t>(Y), w0 = reinterpret_cast<uintptr_t>(omega);
        if (y0 < w0 + span && w0 < y0 + span) return fail(PYRO_ERR_BAD_SIZE, "omega must not overlap Y");
    }
    DeviceGuard guard(m->device);
    pyro::RatesArgs a = rates_args(m, n, ld, rho, nullptr, Y, omega);
    a.e = e; a.T_guess = T_guess; a.T_out = T; a.n_not_converged = n_not_converged;
    a.energy = m->d_energy;
    a.tol = m->newton_tol.load(std::memory_order_relaxed);
    a.max_iter = m->newton_max_iter.load(std::memory_order_relaxed);
    a.t_mid = m->packed.lay.t_mid;
    a.single_t_mid = m->packed.lay.single_t_mid;
    return enqueue_rates(m, a, static_cast<cudaStream_t>(cuda_stream), true);
}

int pyro_reactor_rk4(const pyro_mech *m, int64_t n, int64_t ld, const double *rho, const double *e, double *Y, double *T,
                     double dt, int32_t n_steps, double *work, int32_t *n_not_converged, void *cuda_stream) {
    int st = check_fields(m, n, ld);
    if (st != PYRO_OK) return st;
    if (n_steps < 0 || !(dt == dt)) return fail(PYRO_ERR_BAD_SIZE, "n_steps must be >= 0 and dt a number");
    if (n == 0) return PYRO_OK;
    if (!rho || !e || !Y || !T || !work) return fail(PYRO_ERR_NULL, "a field pointer is NULL");
    if (!aligned8(rho) || !aligned8(e) || !aligned8(Y) || !aligned8(T) || !aligned8(work) ||
        (reinterpret_cast<uintptr_t>(n_not_converged) & 3u))
        return fail(PYRO_ERR_ALIGN, "field pointers must be 8-byte aligned");
    {
        const uintptr_t span = (uintptr_t)(((int64_t)m->packed.n_species - 1) * ld + n) * sizeof(double);
        const uintptr_t y0 = reinterpret_cast<uintptr_t>(Y), w0 = reinterpret_cast<uintptr_t>(work);
        if (y0 < w0 + span && w0 < y0 + span) return fail(PYRO_ERR_BAD_SIZE, "work must not overlap Y");
    }
    DeviceGuard guard(m->device);
    cudaStream_t stream = static_cast<cudaStream_t>(cuda_stream);
    pyro::ReactorArgs a{};
    a.rates = rates_args(m, n, ld, rho, nullptr, nullptr, nullptr);
    a.rates.e = e;
    a.rates.n_not_converged = n_not_converged;
    a.rates.energy = m->d_energy;
    a.rates.tol = m->newton_tol.load(std::memory_order_relaxed);
    a.rates.max_iter = m->newton_max_iter.load(std::memory_order_relaxed);
    a.rates.t_mid = m->packed.lay.t_mid;
    a.rates.single_t_mid = m->packed.lay.single_t_mid;
    a.Y = Y; a.T = T; a.acc = work; a.dt = dt; a.n_steps = n_steps;
    a.energy_smem_off = m->reactor_energy_off;
    const int warps = m->block_threads / 32;
    int64_t blocks = (int64_t)m->sm_count * m->reactor_blocks_per_sm;
    if (blocks > (a.rates.n_chunks + warps - 1) / warps) blocks = (a.rates.n_chunks + warps - 1) / warps;
    const uint32_t slot = m->next_work.fetch_add(1) % kWorkSlots;
    a.rates.work = m->d_work + slot;
    std::lock_guard<std::mutex> lock(m->work_mu);
    PYRO_CUDA(cudaStreamWaitEvent(stream, m->work_done[slot], 0));
    PYRO_CUDA(cudaMemsetAsync(a.rates.work, 0, sizeof(unsigned long long), stream));
    PYRO_CUDA(pyro::launch_reactor(a, m->block_threads, (int)blocks, m->tab_smem, m->b_tmem, m->two_blocks, m->reactor_smem, stream));
    PYRO_CUDA(cudaEventRecord(m->work_done[slot], stream));
    return PYRO_OK;
}

// pyro_reactor_rk4 without the caller's `work` field: the scratch is the array built into the library image
// (pyro_reactor_kernels.cu).  No allocation, no event, no lock on this path; calls that overlap on a device race
// (documented in pyro.h), so nothing here tries to order them.
int pyro_reactor_rk4_static(const pyro_mech *m, int64_t n, int64_t ld, const double *rho, const double *e, double *Y, double *T,
                            double dt, int32_t n_steps, int32_t *n_not_converged, void *cuda_stream) {
    int st = check_fields(m, n, ld);
    if (st != PYRO_OK) return st;
    if (n_steps < 0 || !(dt == dt)) return fail(PYRO_ERR_BAD_SIZE, "n_steps must be >= 0 and dt a number");
    if (n == 0) return PYRO_OK;
    if (!rho || !e || !Y || !T) return fail(PYRO_ERR_NULL, "a field pointer is NULL");
    if (!aligned8(rho) || !aligned8(e) || !aligned8(Y) || !aligned8(T) || (reinterpret_cast<uintptr_t>(n_not_converged) & 3u))
        return fail(PYRO_ERR_ALIGN, "field pointers must be 8-byte aligned");
    const int64_t n_pad = (n + 31) & ~(int64_t)31;
    if (n_pad > (int64_t)PYRO_RK4_STATIC_MAX_DOUBLES / m->packed.n_species)
        return fail(PYRO_ERR_TOO_LARGE, "pyro_reactor_rk4_static: n_species x n (rounded up to 32) = " +
                                            std::to_string(m->packed.n_species) + " x " + std::to_string(n_pad) +
                                            " doubles exceed the built-in scratch of " +
                                            std::to_string((long long)PYRO_RK4_STATIC_MAX_DOUBLES) +
                                            " doubles; march the batch in slabs or pass your own work field to pyro_reactor_rk4");
    DeviceGuard guard(m->device);
    cudaStream_t stream = static_cast<cudaStream_t>(cuda_stream);
    pyro::ReactorArgs a{};
    a.rates = rates_args(m, n, ld, rho, nullptr, nullptr, nullptr);
    a.rates.e = e;
    a.rates.n_not_converged = n_not_converged;
    a.rates.energy = m->d_energy;
    a.rates.tol = m->newton_tol.load(std::memory_order_relaxed);
    a.rates.max_iter = m->newton_max_iter.load(std::memory_order_relaxed);
    a.rates.t_mid = m->packed.lay.t_mid;
    a.rates.single_t_mid = m->packed.lay.single_t_mid;
    a.Y = Y; a.T = T; a.dt = dt; a.n_steps = n_steps;
    a.energy_smem_off = m->reactor_energy_off;
    const int warps = m->block_threads / 32;
    int64_t blocks = (int64_t)m->sm_count * m->reactor_blocks_per_sm;
    if (blocks > (a.rates.n_chunks + warps - 1) / warps) blocks = (a.rates.n_chunks + warps - 1) / warps;
    const char *failed_at = "";
    const cudaError_t ce = pyro::launch_reactor_static(a, m->device, m->block_threads, (int)blocks, m->tab_smem, m->b_tmem,
                                                       m->two_blocks, m->reactor_smem, stream, &failed_at);
    if (ce != cudaSuccess) return fail(PYRO_ERR_CUDA, std::string(failed_at) + ": " + cudaGetErrorString(ce));
    return PYRO_OK;
}

namespace {
int jacobian_call(const pyro_mech *m, int64_t n, int64_t ld, const double *rho, const double *T, const double *Y, int mode,
                  double *J, double *dSdT, void *cuda_stream, int64_t jblock);
}

int pyro_get_jacobian(const pyro_mech *m, int64_t n, int64_t ld, const double *rho, const double *T, const double *Y,
                      int mode, double *J, double *dSdT, void *cuda_stream) {
    return jacobian_call(m, n, ld, rho, T, Y, mode, J, dSdT, cuda_stream, 0);
}

namespace {
int jacobian_call(const pyro_mech *m, int64_t n, int64_t ld, const double *rho, const double *T, const double *Y, int mode,
                  double *J, double *dSdT, void *cuda_stream, int64_t jblock) {
    int st = check_fields(m, n, ld);
    if (st != PYRO_OK) return st;
    if (mode != PYRO_JAC_FIXED_T && mode != PYRO_JAC_FIXED_E) return fail(PYRO_ERR_BAD_SIZE, "mode must be PYRO_JAC_FIXED_T or PYRO_JAC_FIXED_E");
    if (n == 0) return PYRO_OK;
    if (!rho || !T || !Y || !J) return fail(PYRO_ERR_NULL, "a field pointer is NULL");
    if (!aligned8(rho) || !aligned8(T) || !aligned8(Y) || !aligned8(J) || !aligned8(dSdT))
        return fail(PYRO_ERR_ALIGN, "field pointers must be 8-byte aligned");
    if (!m->jac_ok) return fail(PYRO_ERR_UNSUPPORTED, "the Jacobian kernel holds at most 127 species");
    const int64_t ns = m->packed.n_species;
    {   // J (and dSdT) are written while Y of other points is still being read
        const uintptr_t y0 = reinterpret_cast<uintptr_t>(Y), ys = (uintptr_t)((ns - 1) * ld + n) * sizeof(double);
        const uintptr_t j0 = reinterpret_cast<uintptr_t>(J), js = (uintptr_t)((ns * ns - 1) * ld + n) * sizeof(double);
        if (y0 < j0 + js && j0 < y0 + ys) return fail(PYRO_ERR_BAD_SIZE, "J must not overlap Y");
        const uintptr_t t0 = reinterpret_cast<uintptr_t>(dSdT);
        if (dSdT && ((y0 < t0 + ys && t0 < y0 + ys) || (j0 < t0 + ys && t0 < j0 + js)))
            return fail(PYRO_ERR_BAD_SIZE, "dSdT must not overlap Y or J");
    }
    DeviceGuard guard(m->device);
    cudaStream_t stream = static_cast<cudaStream_t>(cuda_stream);
    pyro::JacArgs a{};
    a.n = n; a.ld = ld; a.n_chunks = (n + 31) / 32;
    a.rho = rho; a.T = T; a.Y = Y; a.J = J; a.dSdT = dSdT;
    a.gtab = m->d_blob;
    a.off_spec = m->packed.lay.off_spec;
    a.energy = m->d_energy;
    a.jtab = m->d_jblob;
    a.ext = m->d_jext;
    a.tmem_cols = m->jac_tmem_cols;
    a.planes_bytes = m->jac_planes_bytes;
    a.mode = mode;
    a.lay = m->jac.lay;
    a.jblock = jblock;
    const int warps = m->jac_threads / 32;
    int64_t blocks = (int64_t)m->sm_count * m->jac_blocks_per_sm;
    if (blocks > (a.n_chunks + warps - 1) / warps) blocks = (a.n_chunks + warps - 1) / warps;
    const uint32_t slot = m->next_work.fetch_add(1) % kWorkSlots;
    a.work = m->d_work + slot;
    std::lock_guard<std::mutex> lock(m->jac_mu);
    {
        std::lock_guard<std::mutex> wl(m->work_mu);
        PYRO_CUDA(cudaStreamWaitEvent(stream, m->work_done[slot], 0));
    }
    PYRO_CUDA(cudaStreamWaitEvent(stream, m->jac_done, 0));   // the scratch is shared by the launches of one handle
    PYRO_CUDA(cudaMemsetAsync(a.work, 0, sizeof(unsigned long long), stream));
    if (m->jac_block_warps) {
        a.tmem_cols = m->jac_block_tmem_cols;
        a.planes_bytes = m->jac_block_planes_bytes;
        a.ext_global = m->jac_block_ext_global ? 1 : 0;
        int64_t bb = m->sm_count;
        if (bb > a.n_chunks) bb = a.n_chunks;
        PYRO_CUDA(pyro::launch_jacobian_block(a, m->jac_block_warps, (int)bb, m->jac_block_smem, stream));
    } else {
        PYRO_CUDA(pyro::launch_jacobian(a, m->jac_small, m->jac_threads, (int)blocks, m->jac_smem, stream));
    }
    PYRO_CUDA(cudaEventRecord(m->jac_done, stream));
    {
        std::lock_guard<std::mutex> wl(m->work_mu);
        PYRO_CUDA(cudaEventRecord(m->work_done[slot], stream));
    }
    return PYRO_OK;
}

int64_t cn_work_doubles(const pyro_mech *m, int64_t ld) {
    const int64_t ns = m->packed.n_species, jb = pyro::cn_block_threads((int)ns);
    return ns * ns * ((ld + jb - 1) / jb * jb) + 4 * ns * ld + ld;   // J (blocks of jb points), omega, Ym, Sm, F, last update
}
}   // namespace

int pyro_reactor_cn_work_doubles(const pyro_mech *m, int64_t ld, int64_t *doubles) {
    if (!m || !doubles) return fail(PYRO_ERR_NULL, "NULL argument");
    if (ld < 0) return fail(PYRO_ERR_BAD_SIZE, "ld < 0");
    *doubles = cn_work_doubles(m, ld);
    return PYRO_OK;
}

int pyro_reactor_cn(const pyro_mech *m, int64_t n, int64_t ld, const double *rho, const double *e, double *Y, double *T,
                    double dt, int32_t n_steps, int32_t newton_iters, double update_tol, double *work,
                    int32_t *n_not_converged, void *cuda_stream) {
    int st = check_fields(m, n, ld);
    if (st != PYRO_OK) return st;
    if (n_steps < 0 || newton_iters < 1 || !(dt == dt) || !(update_tol >= 0)) return fail(PYRO_ERR_BAD_SIZE, "n_steps >= 0, newton_iters >= 1, update_tol >= 0");
    if (n == 0) return PYRO_OK;
    if (!rho || !e || !Y || !T || !work) return fail(PYRO_ERR_NULL, "a field pointer is NULL");
    if (!aligned8(rho) || !aligned8(e) || !aligned8(Y) || !aligned8(T) || !aligned8(work) ||
        (reinterpret_cast<uintptr_t>(n_not_converged) & 3u))
        return fail(PYRO_ERR_ALIGN, "field pointers must be 8-byte aligned");
    if (!m->jac_ok) return fail(PYRO_ERR_UNSUPPORTED, "the Jacobian kernel holds at most 127 species");
    const int64_t ns = m->packed.n_species;
    {
        const uintptr_t ys = (uintptr_t)((ns - 1) * ld + n) * sizeof(double), ws = (uintptr_t)cn_work_doubles(m, ld) * sizeof(double);
        const uintptr_t y0 = reinterpret_cast<uintptr_t>(Y), w0 = reinterpret_cast<uintptr_t>(work);
        if (y0 < w0 + ws && w0 < y0 + ys) return fail(PYRO_ERR_BAD_SIZE, "work must not overlap Y");
    }
    cudaStream_t stream = static_cast<cudaStream_t>(cuda_stream);
    const int64_t jb = pyro::cn_block_threads((int)ns);
    double *J = work, *omega = J + ns * ns * ((ld + jb - 1) / jb * jb), *Ym = omega + ns * ld, *Sm = Ym + ns * ld, *F = Sm + ns * ld, *lastu = F + ns * ld;
    pyro::CnArgs a{};
    a.n = n; a.ld = ld; a.rho = rho; a.omega = omega; a.Y = Y; a.Ym = Ym; a.Sm = Sm; a.F = F; a.J = J; a.last_update = lastu;
    a.n_not_converged = n_not_converged; a.energy = m->d_energy; a.dt = dt; a.update_tol = update_tol; a.n_species = (int32_t)ns;
    a.jblock = jb;
    // rates at the initial state; then per step: old-level terms, newton_iters x (Jacobian, solve + update, temperature, rates)
    if ((st = pyro_get_temperature(m, n, ld, rho, e, Y, T, T, n_not_converged, cuda_stream)) != PYRO_OK) return st;
    if ((st = pyro_get_net_production_rates(m, n, ld, rho, T, Y, omega, cuda_stream)) != PYRO_OK) return st;
    for (int32_t step = 0; step < n_steps; ++step) {
        {
            DeviceGuard guard(m->device);
            PYRO_CUDA(pyro::launch_cn_begin_step(a, stream));
        }
        for (int32_t it = 0; it < newton_iters; ++it) {
            if ((st = jacobian_call(m, n, ld, rho, T, Y, PYRO_JAC_FIXED_E, J, nullptr, cuda_stream, jb)) != PYRO_OK) return st;
            a.count_unconverged = (it == newton_iters - 1) ? 1 : 0;
            {
                DeviceGuard guard(m->device);
                PYRO_CUDA(pyro::launch_cn_newton(a, stream));
            }
            if ((st = pyro_get_temperature(m, n, ld, rho, e, Y, T, T, n_not_converged, cuda_stream)) != PYRO_OK) return st;
            if ((st = pyro_get_net_production_rates(m, n, ld, rho, T, Y, omega, cuda_stream)) != PYRO_OK) return st;
        }
    }
    return PYRO_OK;
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
    // a failure leaves no half-built pipe behind and no copy in flight into the caller's buffers
    auto drain = [&]() {
        if (p.s_in) cudaStreamSynchronize(p.s_in);
        if (p.s_run) cudaStreamSynchronize(p.s_run);
        if (p.s_out) cudaStreamSynchronize(p.s_out);
    };
#define PYRO_PIPE(call)                                         \
    do {                                                        \
        cudaError_t e_ = (call);                                \
        if (e_ != cudaSuccess) {                                \
            drain();                                            \
            if (!p.ready) free_pipe(p);                         \
            return cuda_fail(e_, #call);                        \
        }                                                       \
    } while (0)
    if (!p.ready) {
        // slab of points: about 64 MB of mass fractions per buffer
        int64_t slab = (int64_t)(64.0 * 1024 * 1024 / (8.0 * ns));
        slab = (slab / 1024) * 1024;
        if (slab < 4096) slab = 4096;
        if (const char *env = std::getenv("PYRO_HOST_SLAB")) slab = std::atoll(env) > 0 ? std::atoll(env) : slab;
        p.slab = slab;
        for (int b = 0; b < HostPipe::kBuf; ++b) {
            PYRO_PIPE(cudaMalloc(&p.rho[b], slab * 8));
            PYRO_PIPE(cudaMalloc(&p.e[b], slab * 8));
            PYRO_PIPE(cudaMalloc(&p.Tg[b], slab * 8));
            PYRO_PIPE(cudaMalloc(&p.T[b], slab * 8));
            PYRO_PIPE(cudaMalloc(&p.Y[b], slab * 8 * ns));
            PYRO_PIPE(cudaMalloc(&p.omega[b], slab * 8 * ns));
            PYRO_PIPE(cudaEventCreateWithFlags(&p.in_done[b], cudaEventDisableTiming));
            PYRO_PIPE(cudaEventCreateWithFlags(&p.run_done[b], cudaEventDisableTiming));
            PYRO_PIPE(cudaEventCreateWithFlags(&p.out_done[b], cudaEventDisableTiming));
        }
        PYRO_PIPE(cudaStreamCreateWithFlags(&p.s_in, cudaStreamNonBlocking));
        PYRO_PIPE(cudaStreamCreateWithFlags(&p.s_run, cudaStreamNonBlocking));
        PYRO_PIPE(cudaStreamCreateWithFlags(&p.s_out, cudaStreamNonBlocking));
        PYRO_PIPE(cudaMalloc(&p.d_bad, sizeof(int32_t)));
        p.ready = true;
    }
    PYRO_PIPE(cudaMemsetAsync(p.d_bad, 0, sizeof(int32_t), p.s_run));
    const int64_t slab = p.slab;
    int64_t i = 0;
    for (int64_t s0 = 0; s0 < n; s0 += slab, ++i) {
        const int b = (int)(i % HostPipe::kBuf);
        const int64_t cnt = (n - s0 < slab) ? (n - s0) : slab;
        // the buffer is free once the results of its previous slab have left
        if (i >= HostPipe::kBuf) PYRO_PIPE(cudaStreamWaitEvent(p.s_in, p.out_done[b], 0));
        PYRO_PIPE(cudaMemcpyAsync(p.rho[b], rho + s0, cnt * 8, cudaMemcpyHostToDevice, p.s_in));
        PYRO_PIPE(cudaMemcpyAsync(p.e[b], e + s0, cnt * 8, cudaMemcpyHostToDevice, p.s_in));
        PYRO_PIPE(cudaMemcpyAsync(p.Tg[b], T_guess + s0, cnt * 8, cudaMemcpyHostToDevice, p.s_in));
        PYRO_PIPE(cudaMemcpy2DAsync(p.Y[b], slab * 8, Y + s0, ld * 8, cnt * 8, ns, cudaMemcpyHostToDevice, p.s_in));
        PYRO_PIPE(cudaEventRecord(p.in_done[b], p.s_in));
        PYRO_PIPE(cudaStreamWaitEvent(p.s_run, p.in_done[b], 0));
        PYRO_PIPE(pyro::launch_temperature(temp_args(m, cnt, slab, p.e[b], p.Y[b], p.Tg[b], p.T[b], p.d_bad), p.s_run));
        st = enqueue_rates(m, rates_args(m, cnt, slab, p.rho[b], p.T[b], p.Y[b], p.omega[b]), p.s_run);
        if (st != PYRO_OK) {
            drain();
            return st;
        }
        PYRO_PIPE(cudaEventRecord(p.run_done[b], p.s_run));
        PYRO_PIPE(cudaStreamWaitEvent(p.s_out, p.run_done[b], 0));
        PYRO_PIPE(cudaMemcpyAsync(T + s0, p.T[b], cnt * 8, cudaMemcpyDeviceToHost, p.s_out));
        PYRO_PIPE(cudaMemcpy2DAsync(omega + s0, ld * 8, p.omega[b], slab * 8, cnt * 8, ns, cudaMemcpyDeviceToHost, p.s_out));
        PYRO_PIPE(cudaEventRecord(p.out_done[b], p.s_out));
    }
    int32_t bad = 0;
    PYRO_PIPE(cudaMemcpyAsync(&bad, p.d_bad, sizeof bad, cudaMemcpyDeviceToHost, p.s_run));
    PYRO_PIPE(cudaStreamSynchronize(p.s_run));
    PYRO_PIPE(cudaStreamSynchronize(p.s_out));
    PYRO_PIPE(cudaStreamSynchronize(p.s_in));
#undef PYRO_PIPE
    if (n_not_converged) *n_not_converged = bad;
    return PYRO_OK;
}

int pyro_mech_info(const pyro_mech *m, int64_t *out, int cap) {
    if (!m || !out) return -fail(PYRO_ERR_NULL, "NULL argument");
    DeviceGuard guard(m->device);
    cudaFuncAttributes fa{};
    int64_t v[15] = {m->packed.n_species, m->packed.n_reactions, m->packed.lay.n_p, m->packed.lay.n_x,
                     (int64_t)m->packed.lay.bytes, m->tab_smem ? 1 : 0, m->block_threads,
                     (int64_t)m->smem_bytes, m->blocks_per_sm, 0, 0,
                     m->sm_count, 1, (int64_t)m->tmem_cols, m->b_tmem ? 1 : 0};
    if (m->two_points) {   // the kernel pyro_get_net_production_rates launches: two grid points per thread
        cudaFuncGetAttributes(&fa, pyro::rates2_kernel_ptr(m->tab_smem2, m->two_blocks));
        v[5] = m->tab_smem2 ? 1 : 0;
        v[6] = pyro::kRates2Threads;
        v[7] = (int64_t)m->smem2;
        v[8] = m->blocks_per_sm2;
        v[12] = 2;
        v[13] = (int64_t)m->tmem_cols2;
        v[14] = 1;
    } else {
        cudaFuncGetAttributes(&fa, pyro::rates_kernel_ptr(m->tab_smem, m->b_tmem, m->two_blocks));
    }
    v[9] = fa.numRegs;
    v[10] = (int64_t)fa.localSizeBytes;
    int cnt = cap < 15 ? cap : 15;
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
