// TEST-ONLY host build of libpyro's packer and per-point device functions.
//
// Compiles csrc/pyro_pack.cpp and the per-point arithmetic of csrc/pyro_point.cuh (the
// functions the kernels call for every thread) with g++, so that the packer, the table
// layout and the folded-coefficient arithmetic can be checked against the oracle on the
// CPU-only box ("host logic" tests, -m "not gpu").  It is NOT part of the product:
// libpyro.so does not contain it, the binding never loads it, and nothing outside tests/
// may use it.  The GPU parity tests (-m gpu) go through the C ABI of libpyro.so.
#include <cstdint>
#include <string>
#include <vector>

#include "../../paper_2503_24286_b200/csrc/pyro_pack.h"
#include "../../paper_2503_24286_b200/csrc/pyro_point.cuh"

namespace {
struct HostTab {
    const unsigned char *base;
    pyro::TableLayout lay;
    const pyro::RxnE &rxn_e(int j) const { return reinterpret_cast<const pyro::RxnE *>(base + lay.off_rxn_e)[j]; }
    const pyro::RxnX &rxn_x(int j) const { return reinterpret_cast<const pyro::RxnX *>(base + lay.off_rxn_x)[j]; }
    const pyro::RxnFall &rxn_fall(int j) const { return reinterpret_cast<const pyro::RxnFall *>(base + lay.off_fall)[j]; }
    double inv_w(int k) const { return reinterpret_cast<const double *>(base + lay.off_inv_w)[k]; }
    double eff_delta(int q) const { return reinterpret_cast<const double *>(base + lay.off_eff_delta)[q]; }
    int eff_species(int q) const { return reinterpret_cast<const uint16_t *>(base + lay.off_eff_species)[q]; }
};
thread_local std::string g_err;
}   // namespace

extern "C" {

const char *emu_last_error() { return g_err.c_str(); }

int emu_pack_status(const pyro_mech_desc *d, int64_t *info4) {
    pyro::PackedMech pm;
    int st = pyro::pack_mechanism(d, pm, g_err);
    if (st == PYRO_OK && info4) {
        info4[0] = pm.lay.n_e;
        info4[1] = pm.lay.n_x;
        info4[2] = pm.lay.bytes;
        info4[3] = pm.lay.n_eff;
    }
    return st;
}

int emu_rates(const pyro_mech_desc *d, int64_t n, int64_t ld, const double *rho, const double *T, const double *Y,
              double *omega) {
    constexpr int P = 2;   // as the kernel: one "thread" owns two adjacent points
    pyro::PackedMech pm;
    int st = pyro::pack_mechanism(d, pm, g_err);
    if (st != PYRO_OK) return st;
    HostTab tab{pm.blob.data(), pm.lay};
    const int ns = pm.n_species;
    std::vector<pyro::Vec<P>> C(ns + 1), W(ns + 1);   // + the dummy species
    for (int64_t p0 = 0; p0 < n; p0 += P) {
        double ctot[P], Tp[P];
        int64_t pi[P];
        for (int i = 0; i < P; ++i) {
            pi[i] = p0 + i < n ? p0 + i : n - 1;
            Tp[i] = T[pi[i]];
            ctot[i] = 0;
        }
        for (int k = 0; k < ns; ++k)
            for (int i = 0; i < P; ++i) {
                C[k].v[i] = rho[pi[i]] * Y[k * ld + pi[i]] * tab.inv_w(k);
                W[k].v[i] = 0;
                ctot[i] += C[k].v[i];
            }
        for (int i = 0; i < P; ++i) {
            C[ns].v[i] = 1.0;
            W[ns].v[i] = 0.0;
        }
        const pyro::PointT<P> pt = pyro::make_point<P>(Tp, pm.lay.t_mid);
        pyro::accumulate_reactions<P>(tab, pm.lay.shape_pairs, pm.lay.shape_singles, pm.lay.ext_count, pt, ctot,
                                      C.data(), W.data(), 1);
        for (int k = 0; k < ns; ++k)
            for (int i = 0; i < P; ++i)
                if (p0 + i < n) omega[k * ld + p0 + i] = W[k].v[i];
    }
    return PYRO_OK;
}

int emu_temperature(const pyro_mech_desc *d, int64_t n, int64_t ld, const double *e, const double *Y,
                    const double *Tg, double tol, int max_iter, double *T, int64_t *n_bad) {
    pyro::PackedMech pm;
    int st = pyro::pack_mechanism(d, pm, g_err);
    if (st != PYRO_OK) return st;
    const int ns = pm.n_species;
    int64_t bad = 0;
    for (int64_t p = 0; p < n; ++p) {
        double Slo[6] = {0, 0, 0, 0, 0, 0}, Shi[6] = {0, 0, 0, 0, 0, 0};
        for (int k = 0; k < ns; ++k)
            for (int m = 0; m < 6; ++m) {
                Slo[m] = std::fma(Y[k * ld + p], pm.energy[k].lo[m], Slo[m]);
                Shi[m] = std::fma(Y[k * ld + p], pm.energy[k].hi[m], Shi[m]);
            }
        bool conv;
        pyro::newton_temperature(Slo, Shi, pm.lay.t_mid, e[p], Tg[p], tol, max_iter, &T[p], &conv);
        bad += conv ? 0 : 1;
    }
    if (n_bad) *n_bad = bad;
    return PYRO_OK;
}

double emu_exp2(double y) { return pyro::exp2_poly(y); }
}
