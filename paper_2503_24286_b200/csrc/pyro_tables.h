// Device table layout shared by the mechanism packer (host) and the kernels.
// Internal to libpyro; the public boundary is include/pyro.h.
//
// All rate exponents are stored in log2 units so that a rate coefficient is one exp2 of a
// short polynomial in the per-point features (1, log2 T, 1/T, T, T^2, T^3, T^4):
//   forward  (A.9)  PAPER.md:925   log2 k_f = f0 + f1 log2T + f2/T
//   reverse  (A.10) PAPER.md:932   log2 k_r = log2 k_f - log2 K_c, with the Gibbs sum
//            sum_i nu_ij g_i/(RT) of (A.11)-(A.13) folded per reaction at pack time into
//            7 coefficients for each NASA range (all species of a mechanism on the fast
//            path share one T_mid, so a reaction has exactly two ranges).
#pragma once
#include <cstdint>

namespace pyro {

constexpr int kMaxSide = 3;            // molecules per reaction side held in fixed-width slots
constexpr uint16_t kNoSpecies = 0xFFFF;
constexpr int kConstBankBytes = 63 * 1024;   // of the 64 KB __constant__ bank; the rest is left to the compiler

// Plain class: elementary reactions (reversible or not) whose net stoichiometry is the
// difference of the two slot lists.  152 bytes.
struct alignas(8) RxnE {
    double f[3];             // log2 k_f
    double rlo[7], rhi[7];   // log2 k_r for T < T_mid / T >= T_mid
    uint16_t slot[6];        // species of reactant molecules [0..2] and product molecules [3..5]
    uint8_t nreac, nprod;    // molecules per side (a coefficient 2 repeats the species)
    uint8_t reversible;
    uint8_t pad;
};

// Extended class: three-body and falloff reactions, and reactions with a species on both
// sides (whose scatter list differs from the slot lists).
struct alignas(8) RxnX {
    RxnE e;
    double l[3];             // log2 k_0 (low-pressure limit), falloff only
    double troe_alpha;       // Troe: Fcent = (1-alpha) 2^(t3 T) + alpha 2^(t1 T) + 2^(t2/T)
    double troe_t3, troe_t1, troe_t2;   // -log2e/T***, -log2e/T*, -log2e T**
    double eff_default;      // [M] = eff_default * C_tot + sum_listed eff_delta * C_k
    double sc_coef[6];       // scatter list: omega[sc_species] += sc_coef * R
    uint16_t sc_species[6];
    uint32_t eff_begin;      // range in the efficiency arrays
    uint16_t eff_count;
    uint8_t type;            // PYRO_ELEMENTARY .. PYRO_FALLOFF_TROE
    uint8_t n_scatter;
    uint8_t troe_has_t2;
    uint8_t pad[7];
};

// Byte offsets into the table blob (all 8-byte aligned).
struct TableLayout {
    uint32_t off_inv_w;      // double[n_species]   1/W_k
    uint32_t off_rxn_e;      // RxnE[n_e]
    uint32_t off_rxn_x;      // RxnX[n_x]
    uint32_t off_eff_delta;  // double[n_eff]       eff - eff_default
    uint32_t off_eff_species;// uint16[n_eff]
    uint32_t bytes;
    int32_t n_species, n_e, n_x, n_eff;
    int32_t needs_ctot;      // any extended reaction uses [M]
    double t_mid;            // the mechanism's single T_mid
};

// Energy table of the temperature solve: per species and NASA range the six coefficients
//   (a6, a1-1, a2/2, a3/3, a4/4, a5/5) * R/W_k
// so that  e(T) = sum_k Y_k (c0 + c1 T + ... + c5 T^5)   (A.25)-(A.26) PAPER.md:1008-1012
// and      c_v(T) = de/dT                                 (A.29)-(A.31) PAPER.md:1025-1034
struct alignas(8) EnergyRow {
    double lo[6], hi[6];
};

}   // namespace pyro
