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
    const pyro::SpecRow &spec(int k) const { return reinterpret_cast<const pyro::SpecRow *>(base + lay.off_spec)[k]; }
    const pyro::RxnP &rxn_p(int j) const { return reinterpret_cast<const pyro::RxnP *>(base + lay.off_rxn_p)[j]; }
    const pyro::RxnX &rxn_x(int j) const { return reinterpret_cast<const pyro::RxnX *>(base + lay.off_rxn_x)[j]; }
    const pyro::RxnFall &rxn_fall(int j) const { return reinterpret_cast<const pyro::RxnFall *>(base + lay.off_fall)[j]; }
    double eff_delta(int q) const { return reinterpret_cast<const double *>(base + lay.off_eff_delta)[q]; }
    int eff_species(int q) const { return (int)reinterpret_cast<const uint32_t *>(base + lay.off_eff_species)[q]; }
};
thread_local std::string g_err;

template <int P>
int emu_rates_p(const pyro_mech_desc *d, int64_t n, int64_t ld, const double *rho, const double *T, const double *Y,
                double *omega) {
    pyro::PackedMech pm;
    int st = pyro::pack_mechanism(d, pm, g_err);
    if (st != PYRO_OK) return st;
    HostTab tab{pm.blob.data(), pm.lay};
    const int ns = pm.n_species;
    std::vector<pyro::Vec<P>> s((size_t)pyro::kPlanes * (ns + 1));   // + the dummy species
    for (int64_t p0 = 0; p0 < n; p0 += P) {
        double ctot[P], Tp[P], rh[P];
        int64_t pi[P];
        for (int i = 0; i < P; ++i) {
            pi[i] = p0 + i < n ? p0 + i : n - 1;
            Tp[i] = T[pi[i]];
            rh[i] = rho[pi[i]];
            ctot[i] = 0;
        }
        const pyro::PointT<P> pt = pyro::make_point<P>(Tp);
        const pyro::ArrayMem<P> mem{s.data()};
        pyro::fill_planes<P>(tab, ns, pt, rh, ctot, mem, [&](int k, double (&y)[P]) {
            for (int i = 0; i < P; ++i) y[i] = Y[k * ld + pi[i]];
        });
        pyro::accumulate_reactions<P>(tab, pm.lay.shape_quads, pm.lay.shape_pairs, pm.lay.shape_singles,
                                      pm.lay.ext_count, pt, ctot, mem);
        for (int k = 0; k < ns; ++k)
            for (int i = 0; i < P; ++i)
                if (p0 + i < n) omega[k * ld + p0 + i] = s[k * pyro::kPlanes + 2].v[i];
    }
    return PYRO_OK;
}
}   // namespace

extern "C" {

const char *emu_last_error() { return g_err.c_str(); }

// info: [0] plain reactions [1] extended [2] table bytes [3] efficiencies
//       [4] plain reactions stored in groups of four [5] in couples [6] single T_mid
//       [7..15] per shape: reactions in fours, [16..24] in couples, [25..33] single
int emu_pack_status(const pyro_mech_desc *d, int64_t *info) {
    pyro::PackedMech pm;
    int st = pyro::pack_mechanism(d, pm, g_err);
    if (st == PYRO_OK && info) {
        info[0] = pm.lay.n_p;
        info[1] = pm.lay.n_x;
        info[2] = pm.lay.bytes;
        info[3] = pm.lay.n_eff;
        info[4] = info[5] = 0;
        for (int s = 0; s < 9; ++s) {
            info[4] += pm.lay.shape_quads[s];
            info[5] += pm.lay.shape_pairs[s];
            info[7 + s] = pm.lay.shape_quads[s];
            info[16 + s] = pm.lay.shape_pairs[s];
            info[25 + s] = pm.lay.shape_singles[s];
        }
        info[6] = pm.lay.single_t_mid;
    }
    return st;
}

// packed position -> reaction index of the description (order[n_reactions])
int emu_pack_order(const pyro_mech_desc *d, int32_t *order) {
    pyro::PackedMech pm;
    int st = pyro::pack_mechanism(d, pm, g_err);
    if (st == PYRO_OK)
        for (size_t i = 0; i < pm.order.size(); ++i) order[i] = pm.order[i];
    return st;
}

// points_per_thread selects the kernel variant that is emulated (1 or 2 points per "thread")
int emu_rates(const pyro_mech_desc *d, int points_per_thread, int64_t n, int64_t ld, const double *rho,
              const double *T, const double *Y, double *omega) {
    return points_per_thread == 2 ? emu_rates_p<2>(d, n, ld, rho, T, Y, omega)
                                  : emu_rates_p<1>(d, n, ld, rho, T, Y, omega);
}

int emu_temperature(const pyro_mech_desc *d, int64_t n, int64_t ld, const double *e, const double *Y,
                    const double *Tg, double tol, int max_iter, double *T, int64_t *n_bad) {
    pyro::PackedMech pm;
    int st = pyro::pack_mechanism(d, pm, g_err);
    if (st != PYRO_OK) return st;
    if (!pm.lay.single_t_mid) return PYRO_ERR_UNSUPPORTED;
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

void emu_exp2_pair(double y, double *e, double *b) {
    const double yy[1] = {y};
    double ee[1], bb[1];
    pyro::exp2_pair_n<1>(yy, ee, bb);
    *e = ee[0];
    *b = bb[0];
}
}
