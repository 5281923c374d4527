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
#include "../../paper_2503_24286_b200/csrc/pyro_jac.cuh"

namespace {
struct HostTab {
    const unsigned char *base;
    pyro::TableLayout lay;
    const pyro::SpecRow &spec(int k) const { return reinterpret_cast<const pyro::SpecRow *>(base + lay.off_spec)[k]; }
    const pyro::RxnP &rxn_p(int j) const { return reinterpret_cast<const pyro::RxnP *>(base + lay.off_rxn_p)[j]; }
    const pyro::RxnX &rxn_x(int j) const { return reinterpret_cast<const pyro::RxnX *>(base + lay.off_rxn_x)[j]; }
    const pyro::RxnFall &rxn_fall(int j) const { return reinterpret_cast<const pyro::RxnFall *>(base + lay.off_fall)[j]; }
    const pyro::EffEntry &eff(int q) const { return reinterpret_cast<const pyro::EffEntry *>(base + lay.off_eff)[q]; }
};
struct HostJacTab {
    const unsigned char *base;       // rates blob (species rows)
    pyro::TableLayout lay;
    const pyro::EnergyRow *en;
    const unsigned char *jbase;      // Jacobian blob
    pyro::JacLayout jl;
    const pyro::SpecRow &spec(int k) const { return reinterpret_cast<const pyro::SpecRow *>(base + lay.off_spec)[k]; }
    const pyro::EnergyRow &energy(int k) const { return en[k]; }
    const pyro::JacRxn &rxn(int j) const { return reinterpret_cast<const pyro::JacRxn *>(jbase + jl.off_rxn)[j]; }
    const pyro::JacInc &inc(int q) const { return reinterpret_cast<const pyro::JacInc *>(jbase + jl.off_inc)[q]; }
    const pyro::JacInc *inc_run(uint32_t q, uint32_t end, uint32_t &n) const {
        n = end - q;
        return &inc((int)q);
    }
    const pyro::EffEntry &eff(int q) const { return reinterpret_cast<const pyro::EffEntry *>(jbase + jl.off_eff)[q]; }
    const pyro::RxnFall &rxn_fall(int j) const { return reinterpret_cast<const pyro::RxnFall *>(jbase + jl.off_fall)[j]; }
    const pyro::JacCol &col(int k) const { return reinterpret_cast<const pyro::JacCol *>(jbase + jl.off_col)[k]; }
    void begin_rxn(int, int) const {}
    void begin_inc() const {}
};
thread_local std::string g_err;

pyro::GroupCounts group_counts(const pyro::TableLayout &l) {
    pyro::GroupCounts g;
    for (int s = 0; s < 9; ++s) {
        g.shape_g8[s] = l.shape_g8[s];
        g.shape_g4[s] = l.shape_g4[s];
        g.shape_g2[s] = l.shape_g2[s];
        g.shape_g1[s] = l.shape_g1[s];
    }
    for (int k = 0; k < 4; ++k) {
        g.ext_g4[k] = l.ext_g4[k];
        g.ext_g2[k] = l.ext_g2[k];
        g.ext_g1[k] = l.ext_g1[k];
    }
    return g;
}
}   // namespace

extern "C" {

const char *emu_last_error() { return g_err.c_str(); }

// info: [0] plain records [1] extended records [2] table bytes [3] efficiency entries
//       [4] plain records stored in groups of eight [5] of four [6] single T_mid
//       [7..15] per shape: records in eights, [16..24] in fours, [25..33] in couples
//       [34..37] extended records per kind in fours, [38..41] in couples
//       [42..50] plain records per shape alone, [51..54] extended records per kind alone
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
            info[4] += pm.lay.shape_g8[s];
            info[5] += pm.lay.shape_g4[s];
            info[7 + s] = pm.lay.shape_g8[s];
            info[16 + s] = pm.lay.shape_g4[s];
            info[25 + s] = pm.lay.shape_g2[s];
        }
        for (int k = 0; k < 4; ++k) {
            info[34 + k] = pm.lay.ext_g4[k];
            info[38 + k] = pm.lay.ext_g2[k];
            info[51 + k] = pm.lay.ext_g1[k];
        }
        for (int s = 0; s < 9; ++s) info[42 + s] = pm.lay.shape_g1[s];
        info[6] = pm.lay.single_t_mid;
    }
    return st;
}

// packed record -> reaction index of the description, -1 for a null record; order[cap]
int emu_pack_order(const pyro_mech_desc *d, int32_t *order, int32_t cap) {
    pyro::PackedMech pm;
    int st = pyro::pack_mechanism(d, pm, g_err);
    if (st == PYRO_OK)
        for (size_t i = 0; i < pm.order.size() && (int32_t)i < cap; ++i) order[i] = pm.order[i];
    return st;
}

// largest |sum over a reaction side of log2 E_k| over the guard temperatures, with (shift = 1) and without
// (shift = 0) the conserved-quantity shift of the species rows; the range guard is what may reject
int emu_pack_side_log2(const pyro_mech_desc *d, int shift, double *out) {
    pyro::PackedMech pm;
    int st = pyro::pack_mechanism(d, pm, g_err, pyro::kLeftoverAuto, shift ? pyro::kShiftOn : pyro::kShiftOff);
    out[0] = pm.max_side_log2; out[1] = pm.max_pair_log2; out[2] = pm.n_wide;
    return st;
}

int emu_rates2(const pyro_mech_desc *d, int64_t n, int64_t ld, const double *rho, const double *T, const double *Y,
               double *omega, int shift);

// the per-point functions of the rates kernel, one point after the other
int emu_rates(const pyro_mech_desc *d, int64_t n, int64_t ld, const double *rho, const double *T, const double *Y,
              double *omega) {
    return emu_rates2(d, n, ld, rho, T, Y, omega, 1);
}

int emu_rates2(const pyro_mech_desc *d, int64_t n, int64_t ld, const double *rho, const double *T, const double *Y,
               double *omega, int shift) {
    pyro::PackedMech pm;
    int st = pyro::pack_mechanism(d, pm, g_err, pyro::kLeftoverAuto, shift ? pyro::kShiftOn : pyro::kShiftOff);
    if (st != PYRO_OK) return st;
    HostTab tab{pm.blob.data(), pm.lay};
    const pyro::GroupCounts g = group_counts(pm.lay);
    const int ns = pm.n_species;
    std::vector<double> A(ns + 1), B(ns + 1), W(ns + 1);   // + the dummy species
    for (int64_t p = 0; p < n; ++p) {
        const pyro::PointT pt = pyro::make_point(T[p]);
        const pyro::ArrayMem mem{A.data(), B.data(), W.data()};
        const double ctot = pyro::fill_planes(tab, ns, pt, rho[p], mem, [&](int k) { return Y[k * ld + p]; });
        pyro::accumulate_reactions<true>(tab, g, pt, ctot, mem);
        for (int k = 0; k < ns; ++k) omega[k * ld + p] = W[k];
    }
    return PYRO_OK;
}

// enthalpy != 0: the enthalpy form, S1 += sum_k Y_k R/W_k as in the kernel
int emu_temperature2(const pyro_mech_desc *d, int64_t n, int64_t ld, const double *e, const double *Y,
                     const double *Tg, double tol, int max_iter, double *T, int64_t *n_bad, int enthalpy);

int emu_temperature(const pyro_mech_desc *d, int64_t n, int64_t ld, const double *e, const double *Y,
                    const double *Tg, double tol, int max_iter, double *T, int64_t *n_bad) {
    return emu_temperature2(d, n, ld, e, Y, Tg, tol, max_iter, T, n_bad, 0);
}

// the arithmetic of eos_kernel
int emu_eos(const pyro_mech_desc *d, int64_t n, int64_t ld, const double *in, const double *T, const double *Y,
            double *out, int to_density) {
    pyro::PackedMech pm;
    int st = pyro::pack_mechanism(d, pm, g_err);
    if (st != PYRO_OK) return st;
    for (int64_t p = 0; p < n; ++p) {
        double Rm = 0.0;
        for (int k = 0; k < pm.n_species; ++k) Rm = std::fma(Y[k * ld + p], pm.energy[k].rw, Rm);
        const double rt = Rm * T[p];
        out[p] = to_density ? in[p] / rt : in[p] * rt;
    }
    return PYRO_OK;
}

int emu_temperature2(const pyro_mech_desc *d, int64_t n, int64_t ld, const double *e, const double *Y,
                     const double *Tg, double tol, int max_iter, double *T, int64_t *n_bad, int enthalpy) {
    pyro::PackedMech pm;
    int st = pyro::pack_mechanism(d, pm, g_err);
    if (st != PYRO_OK) return st;
    const int ns = pm.n_species;
    int64_t bad = 0;
    if (!pm.lay.single_t_mid) {   // the arithmetic of temperature_general_kernel
        for (int64_t p = 0; p < n; ++p) {
            bool conv;
            pyro::newton_temperature_general(
                ns, [&](int k) { return Y[k * ld + p]; }, [&](int k) -> const pyro::EnergyRow & { return pm.energy[k]; },
                enthalpy != 0, e[p], Tg[p], tol, max_iter, &T[p], &conv);
            bad += conv ? 0 : 1;
        }
        if (n_bad) *n_bad = bad;
        return PYRO_OK;
    }
    for (int64_t p = 0; p < n; ++p) {
        double Slo[6] = {0, 0, 0, 0, 0, 0}, Shi[6] = {0, 0, 0, 0, 0, 0}, Rm = 0.0;
        for (int k = 0; k < ns; ++k) {
            for (int m = 0; m < 6; ++m) {
                Slo[m] = std::fma(Y[k * ld + p], pm.energy[k].lo[m], Slo[m]);
                Shi[m] = std::fma(Y[k * ld + p], pm.energy[k].hi[m], Shi[m]);
            }
            if (enthalpy) Rm = std::fma(Y[k * ld + p], pm.energy[k].rw, Rm);
        }
        if (enthalpy) {
            Slo[1] += Rm;
            Shi[1] += Rm;
        }
        bool conv;
        pyro::newton_temperature(Slo, Shi, pm.lay.t_mid, e[p], Tg[p], tol, max_iter, &T[p], &conv);
        bad += conv ? 0 : 1;
    }
    if (n_bad) *n_bad = bad;
    return PYRO_OK;
}

// the per-point functions of the Jacobian kernel, one point after the other; J[(i ns + k) ld + p], dSdT[i ld + p]
int emu_jacobian(const pyro_mech_desc *d, int64_t n, int64_t ld, const double *rho, const double *T, const double *Y,
                 int mode, double *J, double *dSdT) {
    pyro::PackedMech pm;
    int st = pyro::pack_mechanism(d, pm, g_err);
    if (st != PYRO_OK) return st;
    pyro::JacPacked jp;
    st = pyro::pack_jacobian(d, jp, g_err);
    if (st != PYRO_OK) return st;
    const HostJacTab tab{pm.blob.data(), pm.lay, pm.energy.data(), jp.blob.data(), jp.lay};
    const int ns = pm.n_species;
    std::vector<double> C(ns + 1), G(ns + 1), DG(ns + 1), a0(ns + 1), a1(ns + 1), a2(ns + 1), ext(1 + 2 * jp.lay.n_ext);
    for (int64_t p = 0; p < n; ++p) {
        const pyro::JacArrayMem mem{C.data(), G.data(), DG.data(), {a0.data(), a1.data(), a2.data()}, ext.data()};
        pyro::jacobian_point(
            tab, jp.lay, T[p], rho[p], mode, dSdT != nullptr, mem, [&](int k) { return Y[k * ld + p]; },
            [&](int i, int k, double v) { J[((int64_t)i * ns + k) * ld + p] = v; },
            [&](int i, double v) { dSdT[i * ld + p] = v; });
    }
    return PYRO_OK;
}

// the per-point reactor march of reactor_kernel, one point after the other; Y in/out, T in (guess) / out, work scratch
int emu_reactor(const pyro_mech_desc *d, int64_t n, int64_t ld, const double *rho, const double *e, double *Y, double *T,
                double dt, int n_steps, double tol, int max_iter, double *work, int64_t *n_bad) {
    pyro::PackedMech pm;
    int st = pyro::pack_mechanism(d, pm, g_err);
    if (st != PYRO_OK) return st;
    HostTab tab{pm.blob.data(), pm.lay};
    const pyro::GroupCounts g = group_counts(pm.lay);
    const int ns = pm.n_species;
    std::vector<double> A(ns + 1), B(ns + 1), W(ns + 1);
    int64_t bad = 0;
    for (int64_t p = 0; p < n; ++p) {
        const pyro::ArrayMem mem{A.data(), B.data(), W.data()};
        bad += pyro::reactor_rk4_point<true>(
            tab, g, ns, pm.lay.single_t_mid != 0, pm.lay.t_mid, rho[p], e[p], &T[p], dt, n_steps, tol, max_iter, mem,
            [&](int k) { return Y[k * ld + p]; }, [&](int k, double v) { Y[k * ld + p] = v; },
            [&](int k) { return work[k * ld + p]; }, [&](int k, double v) { work[k * ld + p] = v; },
            [&](int k) -> const pyro::EnergyRow & { return pm.energy[k]; });
    }
    if (n_bad) *n_bad = bad;
    return PYRO_OK;
}

double emu_exp2(double y) { return pyro::exp2_poly(y); }

double emu_log2(double x) { return pyro::log2_pos(x); }

double emu_exp2_rxn(double y) {
    double v[1] = {y};
    pyro::exp2_poly_n<1>(v);
    return v[0];
}

void emu_exp2_pair(double y, double *e, double *b) {
    const double yy[1] = {y};
    double ee[1], bb[1];
    pyro::exp2_pair_n<1>(yy, ee, bb);
    *e = ee[0];
    *b = bb[0];
}
}
