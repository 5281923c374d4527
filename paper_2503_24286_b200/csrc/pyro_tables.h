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

#if defined(__CUDACC__)
#define PYRO_TAB_HD __host__ __device__ __forceinline__
#else
#define PYRO_TAB_HD inline
#endif

namespace pyro {

constexpr int kMaxSide = 3;            // molecules per reaction side held in fixed-width slots
constexpr uint16_t kNoSpecies = 0xFFFF;
constexpr int kConstBankBytes = 63 * 1024;   // of the 64 KB __constant__ bank; the rest is left to the compiler

// Plain class: reversible elementary reactions whose species are all distinct with unit
// coefficients (so the scatter list is the slot list and the slots of one reaction never
// collide).  Stored by shape (molecules per side), shape s = 3 (nreac-1) + (nprod-1); within a
// shape first the reactions the packer could pair with a species-disjoint partner (stored as
// consecutive couples), then the unpaired rest.  152 bytes.
// Slot words: sw[0] = reactant slots 0..2 and product slot 0 (16 bits each),
// sw[1] = product slots 1..2, then nreac, nprod, reversible (8 bits each).
struct alignas(8) RxnE {
    double f[3];             // log2 k_f
    double rlo[7], rhi[7];   // log2 k_r for T < T_mid / T >= T_mid
    uint64_t sw[2];
};

PYRO_TAB_HD int slot_of(const uint64_t w0, const uint64_t w1, int s) {
    return s < 4 ? (int)((w0 >> (16 * s)) & 0xFFFFu) : (int)((w1 >> (16 * (s - 4))) & 0xFFFFu);
}
PYRO_TAB_HD int nreac_of(const uint64_t w1) { return (int)((w1 >> 32) & 0xFFu); }
PYRO_TAB_HD int nprod_of(const uint64_t w1) { return (int)((w1 >> 40) & 0xFFu); }
PYRO_TAB_HD int reversible_of(const uint64_t w1) { return (int)((w1 >> 48) & 0xFFu); }

// Extended class: three-body and falloff reactions, irreversible reactions, and reactions
// with a repeated species (coefficient 2 or 3, or a species on both sides).  Stored by kind
// (kExtGeneral, kExtThreeBody, kExtLindemann, kExtTroe).  In `e` the six slots list every
// molecule (a coefficient 2 repeats the species); unused slots and unused scatter entries
// name the dummy species n_species, whose concentration is 1 and whose omega is a sink, so
// that the code is branch-free.  The scatter list holds each species once, with its net
// coefficient.
enum { kExtGeneral = 0, kExtThreeBody = 1, kExtLindemann = 2, kExtTroe = 3 };

struct alignas(8) RxnX {
    RxnE e;
    double eff_default;      // [M] = eff_default * C_tot + sum_listed eff_delta * C_k
    uint16_t sc_species[6];  // scatter list: omega[sc_species] += sc_nu * R
    int8_t sc_nu[6];
    uint32_t eff_begin;      // range in the efficiency arrays
    uint16_t eff_count;
    uint16_t fall_index;     // row of the falloff table (kinds kExtLindemann, kExtTroe)
    uint8_t type;            // PYRO_ELEMENTARY .. PYRO_FALLOFF_TROE
    uint8_t pad;
};

// Falloff parameters of an extended reaction.
struct alignas(8) RxnFall {
    double l[3];             // log2 k_0 (low-pressure limit)
    double troe_alpha;       // Troe: Fcent = (1-alpha) 2^(t3 T) + alpha 2^(t1 T) + has_t2 2^(t2/T)
    double troe_t3, troe_t1, troe_t2;   // -log2e/T***, -log2e/T*, -log2e T**
    double troe_has_t2;      // 1.0 or 0.0
};

// Byte offsets into the table blob (all 8-byte aligned).
struct TableLayout {
    uint32_t off_inv_w;      // double[n_species]   1/W_k
    uint32_t off_rxn_e;      // RxnE[n_e]
    uint32_t off_rxn_x;      // RxnX[n_x]
    uint32_t off_fall;       // RxnFall[n_fall]
    uint32_t off_eff_delta;  // double[n_eff]       eff - eff_default
    uint32_t off_eff_species;// uint16[n_eff]
    uint32_t bytes;
    int32_t n_species, n_e, n_x, n_eff, n_fall;
    int32_t shape_pairs[9];    // plain class, per shape: reactions stored as disjoint couples (even count)
    int32_t shape_singles[9];  // plain class, per shape: unpaired reactions
    int32_t ext_count[4];      // extended class, per kind
    int32_t needs_ctot;        // any extended reaction uses [M]
    double t_mid;              // the mechanism's single T_mid
};

// Energy table of the temperature solve: per species and NASA range the six coefficients
//   (a6, a1-1, a2/2, a3/3, a4/4, a5/5) * R/W_k
// so that  e(T) = sum_k Y_k (c0 + c1 T + ... + c5 T^5)   (A.25)-(A.26) PAPER.md:1008-1012
// and      c_v(T) = de/dT                                 (A.29)-(A.31) PAPER.md:1025-1034
struct alignas(8) EnergyRow {
    double lo[6], hi[6];
};

}   // namespace pyro
