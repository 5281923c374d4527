// Mechanism packer (host): validates a pyro_mech_desc and flattens it into the device
// tables of pyro_tables.h.  Row a0 of the hot path.
#include "pyro_pack.h"

#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <algorithm>
#include <array>
#include <map>

namespace pyro {
namespace {

constexpr long double kMaxSideLog2 = 700.0L;    // plain class: largest |sum over a reaction side of log2 E_k| (FP64 holds 2^+-1022)
constexpr long double kMaxPairLog2 = 900.0L;    // extended class: largest |partial sum of product/reactant pair exponents|
constexpr long double kMaxExp2Arg = 1073741824.0L;   // 2^30: exp2_poly reduces |y| < 2^31
constexpr long double kR = 8314.46261815324L;   // J/(kmol K)
constexpr long double kP0 = 101325.0L;          // Pa
const long double kLog2e = 1.0L / std::log(2.0L);

struct Fail {
    int status;
    std::string msg;
};

#define PYRO_REQUIRE(cond, status, ...)                  \
    do {                                                 \
        if (!(cond)) {                                   \
            char buf_[256];                              \
            std::snprintf(buf_, sizeof buf_, __VA_ARGS__); \
            throw Fail{status, buf_};                    \
        }                                                \
    } while (0)

bool finite(double x) { return std::isfinite(x); }

template <class T> void put(std::vector<unsigned char> &blob, uint32_t off, const T *src, size_t count) {
    if (count) std::memcpy(blob.data() + off, src, count * sizeof(T));
}

// log2 E_k on the features (1, log2 T, 1/T, T, T^2, T^3, T^4), E_k = exp(g_k/RT) RT/p0 with
//   g/RT = a1 (1 - ln T) - a2/2 T - a3/6 T^2 - a4/12 T^3 - a5/20 T^4 + a6/T - a7
// which is h/RT - s/R of (A.12), (A.13) with the readings G2, G3.  The coefficient of log2 T
// needs no log2e factor (a ln T = a log2 T / log2e).
void species_row(const double *a, long double dst[7]) {
    const long double c0 = (long double)a[0] - (long double)a[6] + std::log(kR / kP0);
    dst[0] = c0 * kLog2e;
    dst[1] = 1.0L - (long double)a[0];
    dst[2] = (long double)a[5] * kLog2e;
    dst[3] = -(long double)a[1] / 2 * kLog2e;
    dst[4] = -(long double)a[2] / 6 * kLog2e;
    dst[5] = -(long double)a[3] / 12 * kLog2e;
    dst[6] = -(long double)a[4] / 20 * kLog2e;
}

// value of a row at T
long double row_value(const long double c[7], long double T) {
    const long double l2t = std::log2(T);
    return c[0] + c[1] * l2t + c[2] / T + T * (c[3] + T * (c[4] + T * (c[5] + T * c[6])));
}

// Temperatures at which the packer examines a mechanism: kGuardPoints values spaced geometrically over
// the supported range [PYRO_T_MIN, PYRO_T_MAX] of include/pyro.h.
constexpr int kGuardPoints = 64;
long double guard_temperature(int i) {
    return (long double)PYRO_T_MIN * std::pow((long double)PYRO_T_MAX / (long double)PYRO_T_MIN, (long double)i / (kGuardPoints - 1));
}

// Conserved-quantity shift of the species rows (see pyro_tables.h "Range").  nu[j] lists the net
// stoichiometric coefficients (species, coefficient) of the reversible reactions.  On return lam[k][f],
// f = 0..2, is what is subtracted from the (1, log2 T, 1/T) coefficients of BOTH rows of species k.
// Every lam[.][f] is orthogonal to every nu[j] (checked; all zeros are returned if the check fails), so
// sum_k nu_kj log2 E_k -- the equilibrium constant -- is unchanged.
void conserved_shift(int ns, const std::vector<std::vector<std::pair<int, int>>> &nu,
                     const std::vector<std::array<long double, 7>> &lo, const std::vector<std::array<long double, 7>> &hi,
                     const double *t_mid, std::vector<std::array<long double, 3>> &lam) {
    lam.assign(ns, {0.0L, 0.0L, 0.0L});
    // orthonormal basis Q of span{nu_j} by modified Gram-Schmidt (twice), in long double
    std::vector<std::vector<long double>> Q;
    std::vector<long double> v(ns);
    for (const auto &col : nu) {
        if ((int)Q.size() == ns) break;   // full rank: nothing is conserved, no shift possible
        std::fill(v.begin(), v.end(), 0.0L);
        long double n0 = 0;
        for (auto &kc : col) v[kc.first] += kc.second;
        for (int k = 0; k < ns; ++k) n0 += v[k] * v[k];
        if (n0 == 0) continue;
        for (int pass = 0; pass < 2; ++pass)
            for (const auto &q : Q) {
                long double d = 0;
                for (int k = 0; k < ns; ++k) d += q[k] * v[k];
                for (int k = 0; k < ns; ++k) v[k] -= d * q[k];
            }
        long double n1 = 0;
        for (int k = 0; k < ns; ++k) n1 += v[k] * v[k];
        if (n1 <= 1e-18L * n0) continue;   // dependent on the reactions seen so far
        const long double inv = 1.0L / std::sqrt(n1);
        for (int k = 0; k < ns; ++k) v[k] *= inv;
        Q.push_back(v);
    }
    if ((int)Q.size() == ns) return;
    auto project = [&](std::vector<long double> &x) {   // x <- (I - Q Q^T) x : the conserved part of x
        for (int pass = 0; pass < 2; ++pass)
            for (const auto &q : Q) {
                long double d = 0;
                for (int k = 0; k < ns; ++k) d += q[k] * x[k];
                for (int k = 0; k < ns; ++k) x[k] -= d * q[k];
            }
    };
    // least squares over the guard temperatures: lam_k(T) = lam[k][0] + lam[k][1] log2 T + lam[k][2]/T
    // approximates the conserved part of log2 E(T) (each species on the NASA range it is in at T)
    long double G[3][3] = {{0}}, phi[3];
    std::vector<std::array<long double, 3>> rhs(ns, {0.0L, 0.0L, 0.0L});
    std::vector<long double> L(ns);
    for (int i = 0; i < kGuardPoints; ++i) {
        const long double T = guard_temperature(i);
        for (int k = 0; k < ns; ++k) L[k] = row_value(T < (long double)t_mid[k] ? lo[k].data() : hi[k].data(), T);
        project(L);
        phi[0] = 1.0L; phi[1] = std::log2(T); phi[2] = 1.0L / T;
        for (int a = 0; a < 3; ++a) {
            for (int b = 0; b < 3; ++b) G[a][b] += phi[a] * phi[b];
            for (int k = 0; k < ns; ++k) rhs[k][a] += phi[a] * L[k];
        }
    }
    // solve the 3x3 normal equations (Gauss-Jordan with pivoting), the same matrix for every species
    long double inv[3][3] = {{1, 0, 0}, {0, 1, 0}, {0, 0, 1}};
    for (int c = 0; c < 3; ++c) {
        int piv = c;
        for (int r = c + 1; r < 3; ++r)
            if (std::fabs(G[r][c]) > std::fabs(G[piv][c])) piv = r;
        if (G[piv][c] == 0) return;
        for (int b = 0; b < 3; ++b) { std::swap(G[c][b], G[piv][b]); std::swap(inv[c][b], inv[piv][b]); }
        const long double d = 1.0L / G[c][c];
        for (int b = 0; b < 3; ++b) { G[c][b] *= d; inv[c][b] *= d; }
        for (int r = 0; r < 3; ++r)
            if (r != c) {
                const long double m = G[r][c];
                for (int b = 0; b < 3; ++b) { G[r][b] -= m * G[c][b]; inv[r][b] -= m * inv[c][b]; }
            }
    }
    std::vector<long double> col(ns);
    for (int f = 0; f < 3; ++f) {
        for (int k = 0; k < ns; ++k) col[k] = inv[f][0] * rhs[k][0] + inv[f][1] * rhs[k][1] + inv[f][2] * rhs[k][2];
        project(col);   // the solve amplifies rounding: put the coefficient vector back into the conserved space
        for (int k = 0; k < ns; ++k) lam[k][f] = col[k];
    }
    // the shift must cancel in every reversible reaction: |nu_j . lam_f| at rounding level, else no shift
    for (const auto &r : nu)
        for (int f = 0; f < 3; ++f) {
            long double dot = 0, mag = 0;
            for (auto &kc : r) {
                dot += kc.second * lam[kc.first][f];
                mag += std::fabs(kc.second * lam[kc.first][f]);
            }
            if (std::fabs(dot) > 1e-16L * mag + 1e-300L) {
                lam.assign(ns, {0.0L, 0.0L, 0.0L});
                return;
            }
        }
}

uint32_t align16(uint32_t x) { return (x + 15u) & ~15u; }

}   // namespace

// Falloff row of reaction j (type >= PYRO_FALLOFF_LINDEMANN): low-pressure Arrhenius coefficients in log2 form and
// the Troe parameters as slopes of base-2 exponents.
RxnFall fall_row(const pyro_mech_desc *d, int j) {
    RxnFall fl;
    std::memset(&fl, 0, sizeof fl);
    fl.l[0] = (double)(std::log((long double)d->A0[j]) * kLog2e);
    fl.l[1] = d->b0[j];
    fl.l[2] = (double)(-(long double)d->theta0[j] * kLog2e);
    if (d->type[j] == PYRO_FALLOFF_TROE) {
        const double *t = d->troe + 4 * j;
        fl.troe_alpha = t[0];
        // Sentinel temperatures of real mechanisms (T*** = 1e-30, T** = 1e30 ...) make the exponent
        // exceed what exp2 reduces (|y| < 2^31).  Clamp the coefficients where the term is exactly
        // zero in FP64 anyway: exp(-T/T***) with T*** < 1.4e-4 K is 0 for every T >= 1 K, and
        // exp(-T**/T) with T** > 7.4e8 K is 0 for every T <= 1e5 K; the clamped exponents stay
        // below 2^31 for 1 K <= T <= 1e5 K and still underflow to zero there.
        const long double kMaxSlope = 1.0e4L, kMaxT2 = 1073741824.0L;
        fl.troe_t3 = (double)std::max(-kLog2e / (long double)t[1], -kMaxSlope);
        fl.troe_t1 = std::isinf(t[2]) ? 0.0 : (double)std::max(-kLog2e / (long double)t[2], -kMaxSlope);
        fl.troe_has_t2 = std::isinf(t[3]) ? 0.0 : 1.0;
        fl.troe_t2 = std::isinf(t[3]) ? 0.0 : (double)std::max(-kLog2e * (long double)t[3], -kMaxT2);
    }
    return fl;
}

int pack_mechanism(const pyro_mech_desc *d, PackedMech &out, std::string &err, int leftover, int shift) {
    try {
        PYRO_REQUIRE(d != nullptr, PYRO_ERR_NULL, "desc is NULL");
        const int ns = d->n_species, nr = d->n_reactions, ne = d->n_elements;
        PYRO_REQUIRE(ns >= 1, PYRO_ERR_BAD_SIZE, "n_species = %d", ns);
        PYRO_REQUIRE(nr >= 0, PYRO_ERR_BAD_SIZE, "n_reactions = %d", nr);
        PYRO_REQUIRE(ne >= 0, PYRO_ERR_BAD_SIZE, "n_elements = %d", ne);
        PYRO_REQUIRE(d->mol_weight && d->nasa_lo && d->nasa_hi && d->t_mid, PYRO_ERR_NULL, "species table is NULL");
        if (nr > 0) {
            PYRO_REQUIRE(d->reac_ptr && d->reac_species && d->reac_coeff && d->prod_ptr && d->prod_species &&
                             d->prod_coeff,
                         PYRO_ERR_NULL, "stoichiometry CSR is NULL");
            PYRO_REQUIRE(d->A && d->b && d->theta && d->type && d->reversible, PYRO_ERR_NULL,
                         "rate table is NULL");
        }
        PYRO_REQUIRE(ns <= kMaxSpecies, PYRO_ERR_TOO_LARGE, "n_species %d > %d (on-chip staging limit)", ns,
                     kMaxSpecies);
        PYRO_REQUIRE(nr <= kMaxReactions, PYRO_ERR_TOO_LARGE, "n_reactions %d > %d", nr, kMaxReactions);

        // ---- species
        for (int k = 0; k < ns; ++k) {
            PYRO_REQUIRE(finite(d->mol_weight[k]) && d->mol_weight[k] > 0, PYRO_ERR_BAD_MECH,
                         "mol_weight[%d] is not positive", k);
            PYRO_REQUIRE(finite(d->t_mid[k]) && d->t_mid[k] > 0, PYRO_ERR_BAD_MECH, "t_mid[%d] is not positive", k);
            for (int m = 0; m < 7; ++m)
                PYRO_REQUIRE(finite(d->nasa_lo[7 * k + m]) && finite(d->nasa_hi[7 * k + m]), PYRO_ERR_BAD_MECH,
                             "NASA coefficient of species %d is not finite", k);
        }
        bool single_tmid = true;
        for (int k = 1; k < ns; ++k) single_tmid = single_tmid && d->t_mid[k] == d->t_mid[0];

        // ---- reactions: validation
        bool any_special = false;
        for (int j = 0; j < nr; ++j) {
            for (int side = 0; side < 2; ++side) {
                const int32_t *ptr = side ? d->prod_ptr : d->reac_ptr;
                const int32_t *sp = side ? d->prod_species : d->reac_species;
                const int32_t *co = side ? d->prod_coeff : d->reac_coeff;
                PYRO_REQUIRE(ptr[0] == 0 && ptr[j + 1] >= ptr[j], PYRO_ERR_BAD_MECH, "CSR pointer of reaction %d", j);
                int molecules = 0;
                for (int q = ptr[j]; q < ptr[j + 1]; ++q) {
                    PYRO_REQUIRE(sp[q] >= 0 && sp[q] < ns, PYRO_ERR_BAD_MECH,
                                 "species index %d out of range in reaction %d", sp[q], j);
                    PYRO_REQUIRE(co[q] >= 1, PYRO_ERR_BAD_MECH, "stoichiometric coefficient %d in reaction %d",
                                 co[q], j);
                    for (int q2 = ptr[j]; q2 < q; ++q2)
                        PYRO_REQUIRE(sp[q2] != sp[q], PYRO_ERR_BAD_MECH, "species %d listed twice on one side of reaction %d", sp[q], j);
                    molecules += co[q];
                }
                PYRO_REQUIRE(molecules >= 1, PYRO_ERR_BAD_MECH, "reaction %d has an empty side", j);
                PYRO_REQUIRE(molecules <= kMaxSide, PYRO_ERR_BAD_MECH,
                             "reaction %d has %d molecules on one side (slot width %d)", j, molecules, kMaxSide);
            }
            PYRO_REQUIRE(finite(d->A[j]) && d->A[j] > 0, PYRO_ERR_BAD_MECH, "A[%d] must be positive (ln A is taken)", j);
            PYRO_REQUIRE(finite(d->b[j]) && finite(d->theta[j]), PYRO_ERR_BAD_MECH, "b/theta of reaction %d", j);
            PYRO_REQUIRE(d->type[j] <= PYRO_FALLOFF_TROE, PYRO_ERR_BAD_MECH, "type[%d] = %d", j, d->type[j]);
            if (d->type[j] != PYRO_ELEMENTARY) {
                any_special = true;
                PYRO_REQUIRE(d->eff_default && d->eff_ptr, PYRO_ERR_NULL, "efficiency tables are NULL");
                PYRO_REQUIRE(finite(d->eff_default[j]), PYRO_ERR_BAD_MECH, "eff_default[%d]", j);
            }
            if (d->type[j] >= PYRO_FALLOFF_LINDEMANN) {
                PYRO_REQUIRE(d->A0 && d->b0 && d->theta0, PYRO_ERR_NULL, "low-pressure tables are NULL");
                PYRO_REQUIRE(finite(d->A0[j]) && d->A0[j] > 0, PYRO_ERR_BAD_MECH, "A0[%d] must be positive", j);
                PYRO_REQUIRE(finite(d->b0[j]) && finite(d->theta0[j]), PYRO_ERR_BAD_MECH, "b0/theta0 of reaction %d", j);
            }
            if (d->type[j] == PYRO_FALLOFF_TROE) {
                PYRO_REQUIRE(d->troe, PYRO_ERR_NULL, "troe table is NULL");
                const double *t = d->troe + 4 * j;
                PYRO_REQUIRE(finite(t[0]), PYRO_ERR_BAD_MECH, "Troe alpha of reaction %d", j);
                for (int m = 1; m < 4; ++m)
                    PYRO_REQUIRE(t[m] > 0 && !std::isnan(t[m]), PYRO_ERR_BAD_MECH,
                                 "Troe temperature %d of reaction %d is not positive", m, j);
                PYRO_REQUIRE(finite(t[1]), PYRO_ERR_BAD_MECH, "Troe T*** of reaction %d must be finite", j);
            }
        }
        if (any_special) {
            PYRO_REQUIRE(d->eff_ptr[0] == 0, PYRO_ERR_BAD_MECH, "eff_ptr[0] != 0");
            for (int j = 0; j < nr; ++j) {
                PYRO_REQUIRE(d->eff_ptr[j + 1] >= d->eff_ptr[j], PYRO_ERR_BAD_MECH, "eff_ptr of reaction %d", j);
                if (d->eff_ptr[j + 1] > d->eff_ptr[j])
                    PYRO_REQUIRE(d->eff_species && d->eff_value, PYRO_ERR_NULL, "efficiency lists are NULL");
                for (int q = d->eff_ptr[j]; q < d->eff_ptr[j + 1]; ++q) {
                    PYRO_REQUIRE(d->eff_species[q] >= 0 && d->eff_species[q] < ns, PYRO_ERR_BAD_MECH,
                                 "efficiency species %d out of range in reaction %d", d->eff_species[q], j);
                    PYRO_REQUIRE(finite(d->eff_value[q]), PYRO_ERR_BAD_MECH, "efficiency value in reaction %d", j);
                    for (int q2 = d->eff_ptr[j]; q2 < q; ++q2)
                        PYRO_REQUIRE(d->eff_species[q2] != d->eff_species[q], PYRO_ERR_BAD_MECH,
                                     "efficiency of species %d listed twice in reaction %d", d->eff_species[q], j);
                }
            }
        }
        if (d->elem_comp && ne > 0) {
            for (int j = 0; j < nr; ++j)
                for (int e = 0; e < ne; ++e) {
                    long long bal = 0;
                    for (int q = d->reac_ptr[j]; q < d->reac_ptr[j + 1]; ++q)
                        bal -= (long long)d->reac_coeff[q] * d->elem_comp[d->reac_species[q] * ne + e];
                    for (int q = d->prod_ptr[j]; q < d->prod_ptr[j + 1]; ++q)
                        bal += (long long)d->prod_coeff[q] * d->elem_comp[d->prod_species[q] * ne + e];
                    PYRO_REQUIRE(bal == 0, PYRO_ERR_BAD_MECH, "reaction %d does not balance element %d", j, e);
                }
        }

        // ---- species rows: log2 E_k folded in long double, shifted by the conserved part (pyro_tables.h
        // "Range"), rounded once
        std::vector<std::array<long double, 7>> rowLo(ns), rowHi(ns);
        for (int k = 0; k < ns; ++k) {
            species_row(d->nasa_lo + 7 * k, rowLo[k].data());
            species_row(d->nasa_hi + 7 * k, rowHi[k].data());
        }
        std::vector<std::vector<std::pair<int, int>>> nuRev;   // net coefficients of the reversible reactions
        for (int j = 0; j < nr; ++j) {
            if (!d->reversible[j]) continue;
            std::map<int, int> net;
            for (int q = d->reac_ptr[j]; q < d->reac_ptr[j + 1]; ++q) net[d->reac_species[q]] -= d->reac_coeff[q];
            for (int q = d->prod_ptr[j]; q < d->prod_ptr[j + 1]; ++q) net[d->prod_species[q]] += d->prod_coeff[q];
            std::vector<std::pair<int, int>> col;
            for (auto &kv : net)
                if (kv.second != 0) col.push_back(kv);
            if (!col.empty()) nuRev.push_back(col);
        }
        std::vector<std::array<long double, 3>> lam;
        conserved_shift(ns, nuRev, rowLo, rowHi, d->t_mid, lam);
        if (shift == kShiftOff) lam.assign(ns, {0.0L, 0.0L, 0.0L});
        for (int k = 0; k < ns; ++k)
            for (int f = 0; f < 3; ++f) {
                rowLo[k][f] -= lam[k][f];
                rowHi[k][f] -= lam[k][f];
            }
        // log2 E_k at the guard temperatures (row ns: the dummy species, E = 1); and the exponents of the rate
        // coefficients, which exp2 must be able to reduce
        std::vector<std::vector<long double>> Lg(kGuardPoints, std::vector<long double>(ns + 1, 0.0L));
        for (int i = 0; i < kGuardPoints; ++i) {
            const long double T = guard_temperature(i), l2t = std::log2(T);
            for (int k = 0; k < ns; ++k) {
                Lg[i][k] = row_value(T < (long double)d->t_mid[k] ? rowLo[k].data() : rowHi[k].data(), T);
                PYRO_REQUIRE(std::fabs(Lg[i][k]) <= kMaxPairLog2, PYRO_ERR_UNSUPPORTED,
                             "species %d: |log2 E| = %.0f at %.0f K is beyond what FP64 products of species factors can hold "
                             "(limit %.0f; supported range %g-%g K)", k, (double)std::fabs(Lg[i][k]), (double)T,
                             (double)kMaxPairLog2, (double)PYRO_T_MIN, (double)PYRO_T_MAX);
            }
            for (int j = 0; j < nr; ++j) {
                const long double yk = std::log((long double)d->A[j]) * kLog2e + d->b[j] * l2t - (long double)d->theta[j] * kLog2e / T;
                long double y0 = 0;
                if (d->type[j] >= PYRO_FALLOFF_LINDEMANN)
                    y0 = std::log((long double)d->A0[j]) * kLog2e + d->b0[j] * l2t - (long double)d->theta0[j] * kLog2e / T;
                PYRO_REQUIRE(std::fabs(yk) < kMaxExp2Arg && std::fabs(y0) < kMaxExp2Arg, PYRO_ERR_UNSUPPORTED,
                             "reaction %d: log2 of a rate coefficient reaches %.3g at %.0f K (exp2 reduces |y| < 2^30)", j,
                             (double)std::max(std::fabs(yk), std::fabs(y0)), (double)T);
            }
        }
        out.max_side_log2 = out.max_pair_log2 = 0.0;
        out.n_wide = 0;
        std::vector<SpecRow> spec(ns);
        for (int k = 0; k < ns; ++k) {
            spec[k].inv_w = (double)(1.0L / (long double)d->mol_weight[k]);
            spec[k].t_mid = d->t_mid[k];
            for (int f = 0; f < 7; ++f) {
                spec[k].lo[f] = (double)rowLo[k][f];
                spec[k].hi[f] = (double)rowHi[k][f];
            }
        }

        // ---- reactions: records
        std::vector<RxnP> recP;
        std::vector<RxnX> recX;
        std::vector<RxnFall> recFall;
        std::vector<std::vector<EffEntry>> effX;   // listed efficiencies of each extended record
        out.order.clear();
        std::vector<int> orderX, orderP, shapeP;
        std::vector<std::vector<int>> speciesP, speciesX;
        bool needs_ctot = false;
        for (int j = 0; j < nr; ++j) {
            uint32_t slot[6];
            for (int s = 0; s < 6; ++s) slot[s] = (uint32_t)ns;   // dummy species: A = B = 1, omega = sink
            std::map<int, int> net;
            bool repeated = false;   // a coefficient above 1 or a species on both sides
            int nreac = 0, nprod = 0;
            for (int q = d->reac_ptr[j]; q < d->reac_ptr[j + 1]; ++q) {
                for (int r = 0; r < d->reac_coeff[q]; ++r) slot[nreac++] = (uint32_t)d->reac_species[q];
                if (d->reac_coeff[q] > 1) repeated = true;
                net[d->reac_species[q]] -= d->reac_coeff[q];
            }
            for (int q = d->prod_ptr[j]; q < d->prod_ptr[j + 1]; ++q) {
                for (int r = 0; r < d->prod_coeff[q]; ++r) slot[3 + nprod++] = (uint32_t)d->prod_species[q];
                if (d->prod_coeff[q] > 1 || net.count(d->prod_species[q])) repeated = true;
                net[d->prod_species[q]] += d->prod_coeff[q];
            }
            const bool reversible = d->reversible[j] != 0;
            // (A.9): log2 k_f = log2 A + b log2 T - theta log2e / T
            double f[3];
            f[0] = (double)(std::log((long double)d->A[j]) * kLog2e);
            f[1] = d->b[j];
            f[2] = (double)(-(long double)d->theta[j] * kLog2e);
            const int type = d->type[j];
            // Range (pyro_tables.h): the plain class multiplies each side's species factors on their own, which
            // is safe while |sum over a side of log2 E_k| <= kMaxSideLog2 over the supported temperatures; a
            // reaction beyond that ("wide") goes to the extended class, whose products are formed in
            // reactant/product pairs.
            long double side = 0;
            for (int i = 0; i < kGuardPoints; ++i) {
                long double sr = 0, sp = 0;
                for (int m = 0; m < 3; ++m) {
                    sr += Lg[i][slot[m]];
                    sp += Lg[i][slot[3 + m]];
                }
                side = std::max(side, std::max(std::fabs(sr), reversible ? std::fabs(sp) : 0.0L));
            }
            const bool wide = side > kMaxSideLog2;
            if (wide && type == PYRO_ELEMENTARY && !repeated && reversible) ++out.n_wide;
            if (!wide && (double)side > out.max_side_log2) out.max_side_log2 = (double)side;
            if (type == PYRO_ELEMENTARY && !repeated && reversible && !wide) {
                RxnP p;
                std::memset(&p, 0, sizeof p);
                for (int m = 0; m < 3; ++m) p.f[m] = f[m];
                for (int m = 0; m < nreac; ++m) p.slot[m] = slot[m];
                for (int m = 0; m < nprod; ++m) p.slot[nreac + m] = slot[3 + m];
                for (int m = nreac + nprod; m < 6; ++m) p.slot[m] = (uint32_t)ns;
                recP.push_back(p);
                shapeP.push_back(3 * (nreac - 1) + (nprod - 1));
                orderP.push_back(j);
                std::vector<int> sp;
                for (auto &kv : net) sp.push_back(kv.first);
                speciesP.push_back(sp);
                continue;
            }
            RxnX x;
            std::memset(&x, 0, sizeof x);
            for (int m = 0; m < 3; ++m) x.f[m] = f[m];
            // The extended class forms the reverse product as prod_i (A_product,i B_reactant,i), i = 0..2 (padded
            // with the dummy species), so only the partial sums of d_i = log2 E_product,i - log2 E_reactant,i
            // must stay in range.  Order the slots so that the largest |d_i| and |partial sum| over the guard
            // temperatures is smallest (36 orderings), and refuse the mechanism if even that is too large.
            if (reversible) {
                const int perms[6][3] = {{0, 1, 2}, {0, 2, 1}, {1, 0, 2}, {1, 2, 0}, {2, 0, 1}, {2, 1, 0}};
                long double best = -1;
                int bestR = 0, bestP = 0;
                for (int pr = 0; pr < 6; ++pr)
                    for (int pp = 0; pp < 6; ++pp) {
                        long double cost = 0;
                        for (int i = 0; i < kGuardPoints; ++i) {
                            long double run = 0;
                            for (int m = 0; m < 3; ++m) {
                                const long double dm = Lg[i][slot[3 + perms[pp][m]]] - Lg[i][slot[perms[pr][m]]];
                                run += dm;
                                cost = std::max(cost, std::max(std::fabs(dm), std::fabs(run)));
                            }
                        }
                        if (best < 0 || cost < best) {
                            best = cost;
                            bestR = pr;
                            bestP = pp;
                        }
                    }
                PYRO_REQUIRE(best <= kMaxPairLog2, PYRO_ERR_UNSUPPORTED,
                             "reaction %d: products of its species factors reach 2^%.0f inside %g-%g K, beyond what FP64 "
                             "holds (limit 2^%.0f); its equilibrium constant is out of range there", j, (double)best,
                             (double)PYRO_T_MIN, (double)PYRO_T_MAX, (double)kMaxPairLog2);
                if ((double)best > out.max_pair_log2) out.max_pair_log2 = (double)best;
                uint32_t ordered[6];
                for (int m = 0; m < 3; ++m) {
                    ordered[m] = slot[perms[bestR][m]];
                    ordered[3 + m] = slot[3 + perms[bestP][m]];
                }
                for (int m = 0; m < 6; ++m) slot[m] = ordered[m];
            }
            for (int m = 0; m < 6; ++m) x.slot[m] = slot[m];
            x.rev = reversible ? 1 : 0;
            x.type = (int16_t)type;
            for (int s = 0; s < 6; ++s) x.sc_species[s] = (uint32_t)ns;
            int nsc = 0;
            std::vector<int> scs;
            for (auto &kv : net)
                if (kv.second != 0) {
                    x.sc_species[nsc] = (uint32_t)kv.first;
                    x.sc_nu[nsc] = (int16_t)kv.second;
                    scs.push_back(kv.first);
                    ++nsc;
                }
            x.eff_default = 1.0;
            std::vector<EffEntry> effs;
            if (type != PYRO_ELEMENTARY) {
                needs_ctot = true;
                x.eff_default = d->eff_default[j];
                for (int q = d->eff_ptr[j]; q < d->eff_ptr[j + 1]; ++q)
                    effs.push_back(EffEntry{d->eff_value[q] - d->eff_default[j], (uint32_t)d->eff_species[q], 0u});
            }
            if (type >= PYRO_FALLOFF_LINDEMANN) {
                const RxnFall fl = fall_row(d, j);
                x.fall_index = (uint32_t)recFall.size();
                recFall.push_back(fl);
            }
            recX.push_back(x);
            orderX.push_back(j);
            effX.push_back(effs);
            speciesX.push_back(scs);
        }
        // Lockstep groups.  The kernels run the reactions of a group side by side (their
        // exponentials interleaved, their omega read-modify-writes batched), which needs the
        // scatter lists of a group to be mutually disjoint.  Greedy: every reaction joins the first
        // open group it is disjoint from; a full group (eight) is closed.  What is left open is cut
        // into fours and couples; reactions left alone are re-coupled where possible.  The rest is either
        // coupled with a null record (index -1: every slot names the dummy species, so its rate is exactly
        // zero and it rides along in the partner's lockstep for free -- measured faster for mechanisms of
        // hundreds of reactions) or stored as singles that the kernels run one at a time (faster for small
        // mechanisms, where null records would be a large share of the work: configs[1] 3.7 -> 2.6 ms).
        bool pad_singles = leftover == kLeftoverPad;
        if (leftover == kLeftoverAuto) {
            pad_singles = nr >= 64;
            if (const char *env = std::getenv("PYRO_PACK_SINGLES")) pad_singles = std::atoi(env) == 0;
        }
        auto make_groups = [&](const std::vector<int> &members, const std::vector<std::vector<int>> &species,
                               int largest, std::vector<int> &g8, std::vector<int> &g4, std::vector<int> &g2,
                               std::vector<int> &g1) {
            auto disjoint = [&](int a, int b) {
                for (int x : species[a])
                    for (int y : species[b])
                        if (x == y) return false;
                return true;
            };
            std::vector<std::vector<int>> open;
            for (int i : members) {
                int home = -1;
                for (size_t g = 0; g < open.size() && home < 0; ++g) {
                    bool ok = true;
                    for (int member : open[g]) ok = ok && disjoint(member, i);
                    if (ok) home = (int)g;
                }
                if (home < 0) {
                    open.push_back({i});
                    continue;
                }
                open[home].push_back(i);
                if ((int)open[home].size() == largest) {
                    std::vector<int> &dst = largest == 8 ? g8 : g4;
                    dst.insert(dst.end(), open[home].begin(), open[home].end());
                    open.erase(open.begin() + home);
                }
            }
            std::vector<int> ones;
            for (auto &g : open) {
                size_t at = 0;
                if (g.size() - at >= 4) {
                    g4.insert(g4.end(), g.begin() + at, g.begin() + at + 4);
                    at += 4;
                }
                while (g.size() - at >= 2) {
                    g2.push_back(g[at]);
                    g2.push_back(g[at + 1]);
                    at += 2;
                }
                for (; at < g.size(); ++at) ones.push_back(g[at]);
            }
            std::vector<int> rest;
            for (int i : ones) {
                int partner = -1;
                for (size_t o = 0; o < rest.size() && partner < 0; ++o)
                    if (disjoint(rest[o], i)) partner = (int)o;
                if (partner >= 0) {
                    g2.push_back(rest[partner]);
                    g2.push_back(i);
                    rest.erase(rest.begin() + partner);
                } else {
                    rest.push_back(i);
                }
            }
            if (pad_singles) {
                for (int i : rest) {
                    g2.push_back(i);
                    g2.push_back(-1);
                }
            } else {
                g1 = rest;
            }
        };
        // plain class: by shape
        RxnP nullP;
        std::memset(&nullP, 0, sizeof nullP);
        for (int m = 0; m < 6; ++m) nullP.slot[m] = (uint32_t)ns;
        std::vector<RxnP> sortedP;
        int shape_g8[9] = {0}, shape_g4[9] = {0}, shape_g2[9] = {0}, shape_g1[9] = {0};
        for (int shape = 0; shape < 9; ++shape) {
            std::vector<int> members, g8, g4, g2, g1;
            for (size_t i = 0; i < recP.size(); ++i)
                if (shapeP[i] == shape) members.push_back((int)i);
            make_groups(members, speciesP, 4, g8, g4, g2, g1);   // (groups of eight: kept in the format, not formed yet)
            shape_g8[shape] = (int)g8.size();
            shape_g4[shape] = (int)g4.size();
            shape_g2[shape] = (int)g2.size();
            shape_g1[shape] = (int)g1.size();
            for (const std::vector<int> *g : {&g8, &g4, &g2, &g1})
                for (int i : *g) {
                    sortedP.push_back(i < 0 ? nullP : recP[i]);
                    out.order.push_back(i < 0 ? -1 : orderP[i]);
                }
        }
        recP.swap(sortedP);
        // extended class: by kind; the efficiency lists of a group are padded to one length
        RxnX nullX;
        std::memset(&nullX, 0, sizeof nullX);
        for (int m = 0; m < 6; ++m) nullX.slot[m] = nullX.sc_species[m] = (uint32_t)ns;
        nullX.rev = 1;
        nullX.eff_default = 1.0;
        std::vector<RxnX> sortedX;
        std::vector<EffEntry> effs;
        int ext_g4[4] = {0, 0, 0, 0}, ext_g2[4] = {0, 0, 0, 0}, ext_g1[4] = {0, 0, 0, 0};
        for (int kind = 0; kind < 4; ++kind) {
            std::vector<int> members, g8, g4, g2, g1;
            for (size_t i = 0; i < recX.size(); ++i)
                if ((int)recX[i].type == kind) members.push_back((int)i);
            make_groups(members, speciesX, 4, g8, g4, g2, g1);
            ext_g4[kind] = (int)g4.size();
            ext_g2[kind] = (int)g2.size();
            ext_g1[kind] = (int)g1.size();
            auto emit = [&](const std::vector<int> &g, size_t width) {
                for (size_t at = 0; at < g.size(); at += width) {
                    size_t longest = 0;
                    for (size_t m = 0; m < width; ++m)
                        if (g[at + m] >= 0) longest = std::max(longest, effX[g[at + m]].size());
                    longest = (longest + 3) / 4 * 4;   // the kernels read the lists four entries at a time
                    for (size_t m = 0; m < width; ++m) {
                        const int i = g[at + m];
                        RxnX x = i < 0 ? nullX : recX[i];
                        if (i < 0) {   // a null record next to a falloff reaction reads that reaction's falloff row
                            x.type = (int16_t)kind;
                            for (size_t m2 = 0; m2 < width; ++m2)
                                if (g[at + m2] >= 0) x.fall_index = recX[g[at + m2]].fall_index;
                        }
                        x.eff_begin = (uint32_t)effs.size();
                        x.eff_count = (uint32_t)longest;
                        if (i >= 0) effs.insert(effs.end(), effX[i].begin(), effX[i].end());
                        while (effs.size() < x.eff_begin + longest) effs.push_back(EffEntry{0.0, (uint32_t)ns, 0u});
                        sortedX.push_back(x);
                        out.order.push_back(i < 0 ? -1 : orderX[i]);
                    }
                }
            };
            emit(g4, 4);
            emit(g2, 2);
            emit(g1, 1);
        }
        recX.swap(sortedX);

        // ---- blob
        TableLayout &lay = out.lay;
        std::memset(&lay, 0, sizeof lay);
        lay.n_species = ns;
        lay.n_p = (int)recP.size();
        lay.n_x = (int)recX.size();
        lay.n_eff = (int)effs.size();
        lay.n_fall = (int)recFall.size();
        lay.needs_ctot = needs_ctot ? 1 : 0;
        lay.single_t_mid = single_tmid ? 1 : 0;
        lay.t_mid = d->t_mid[0];
        for (int s = 0; s < 9; ++s) {
            lay.shape_g8[s] = shape_g8[s];
            lay.shape_g4[s] = shape_g4[s];
            lay.shape_g2[s] = shape_g2[s];
            lay.shape_g1[s] = shape_g1[s];
        }
        for (int k = 0; k < 4; ++k) {
            lay.ext_g4[k] = ext_g4[k];
            lay.ext_g2[k] = ext_g2[k];
            lay.ext_g1[k] = ext_g1[k];
        }
        uint32_t off = 0;
        lay.off_spec = off;
        off = align16(off + (uint32_t)(spec.size() * sizeof(SpecRow)));
        lay.off_rxn_p = off;
        off = align16(off + (uint32_t)(recP.size() * sizeof(RxnP)));
        lay.off_rxn_x = off;
        off = align16(off + (uint32_t)(recX.size() * sizeof(RxnX)));
        lay.off_fall = off;
        off = align16(off + (uint32_t)(recFall.size() * sizeof(RxnFall)));
        lay.off_eff = off;
        off = align16(off + (uint32_t)(effs.size() * sizeof(EffEntry)));
        lay.bytes = off;
        out.blob.assign(off, 0);
        put(out.blob, lay.off_spec, spec.data(), spec.size());
        put(out.blob, lay.off_rxn_p, recP.data(), recP.size());
        put(out.blob, lay.off_rxn_x, recX.data(), recX.size());
        put(out.blob, lay.off_fall, recFall.data(), recFall.size());
        put(out.blob, lay.off_eff, effs.data(), effs.size());

        // ---- energy table of the temperature solve
        out.energy.assign(ns, EnergyRow{});
        for (int k = 0; k < ns; ++k) {
            const long double rw = kR / (long double)d->mol_weight[k];
            out.energy[k].rw = (double)rw;
            out.energy[k].t_mid = d->t_mid[k];
            out.energy[k].w = d->mol_weight[k];
            for (int range = 0; range < 2; ++range) {
                const double *a = (range ? d->nasa_hi : d->nasa_lo) + 7 * k;
                double *c = range ? out.energy[k].hi : out.energy[k].lo;
                c[0] = (double)((long double)a[5] * rw);
                c[1] = (double)(((long double)a[0] - 1) * rw);
                for (int m = 2; m <= 5; ++m) c[m] = (double)((long double)a[m - 1] / m * rw);
            }
        }
        out.n_species = ns;
        out.n_reactions = nr;
        return PYRO_OK;
    } catch (const Fail &f) {
        err = f.msg;
        return f.status;
    } catch (const std::exception &ex) {
        err = ex.what();
        return PYRO_ERR_BAD_MECH;
    }
}

}   // namespace pyro
