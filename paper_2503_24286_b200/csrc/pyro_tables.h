// Device table layout shared by the mechanism packer (host) and the kernels.
// Internal to libpyro; the public boundary is include/pyro.h.
//
// Formulation.  With the per-species, per-point factor
//     E_k = exp(g_k/RT) * RT/p0          g = h - T s, NASA-7   (A.11)-(A.13) PAPER.md:936-945
// the equilibrium constant (A.10) PAPER.md:932 of reaction j factorises over its species,
//     1/K_c,j = prod_products E_k / prod_reactants E_k ,
// so the rate of progress (A.7) PAPER.md:916 becomes
//     R_j = k_f [prod_reac C_k - prod_prod C_k / K_c]
//         = k_f * prod_reac B_k * [prod_reac A_k - prod_prod A_k],   A_k = C_k E_k,  B_k = 1/E_k.
// The NASA range switch and the Gibbs polynomial are paid once per species and point; a
// reaction costs ONE exponential (k_f), three coefficients and its species slots.
// All exponents are stored in log2 units on the per-point features
//     (1, log2 T, 1/T, T, T^2, T^3, T^4).
//
// Range.  Taken literally the E_k are huge or tiny (|log2 E_k| ~ 1.44 |a6|/T: hundreds at 300 K) and a
// reaction side multiplies up to three of them, which overflows FP64 long before K_c -- which only holds
// the DIFFERENCE sum_k nu_kj log2 E_k -- does.  The identity above holds unchanged for
//     E'_k = E_k 2^(-lambda_k(T))   whenever   sum_k nu_kj lambda_k(T) = 0 for every reversible reaction j,
// i.e. for any lambda(T) in the left null space of the stoichiometric matrix (the conserved quantities:
// element counts, inert species, ...); C_k = A_k B_k is unchanged too.  The packer takes
//     lambda_k(T) = l_k0 + l_k1 log2 T + l_k2 / T
// as the least-squares fit, over the supported temperature range, of the projection of log2 E(T) onto that
// null space (pyro_pack.cpp: conserved_shift), and stores log2 E'_k: the same seven features, the first
// three coefficients shifted, both NASA ranges of a species by the same amount.  What is left in log2 E'_k
// is the part of the Gibbs energies that the reactions can actually see.  The packer then evaluates
// |sum over a side of log2 E'_k| of every reaction over the supported range: up to 700 the reaction may
// be in the plain class (sides multiplied on their own); beyond, it goes to the extended class, which
// multiplies in reactant/product pairs, so that only partial sums of log2 E'_p - log2 E'_r occur -- they
// end at -log2 K_c (up to the p0/RT factor), which is finite wherever the definition's own K_c is.  The
// packer orders the pairs for the smallest partial sums and refuses (PYRO_ERR_UNSUPPORTED) a mechanism whose
// partial sums exceed 900 inside [PYRO_T_MIN, PYRO_T_MAX] (include/pyro.h).
//
// Every record is a multiple of 16 bytes and 16-byte aligned: the kernels read the tables
// from shared memory with 128-bit loads at warp-uniform addresses (two wavefronts each, measured:
// a uniform load moves 8 bytes per wavefront, so record size is shared-memory bandwidth).
#pragma once
#include <cstdint>

#if defined(__CUDACC__)
#define PYRO_TAB_HD __host__ __device__ __forceinline__
#else
#define PYRO_TAB_HD inline
#endif

namespace pyro {

constexpr int kMaxSide = 3;   // molecules per reaction side held in fixed-width slots

// Per species: 1/W_k, T_mid,k and log2 E_k = c0 + c1 log2T + c2/T + c3 T + c4 T^2 + c5 T^3 + c6 T^4
// for each NASA range (T < T_mid: lo, else hi; reading G10).  Both coefficient sets start on
// a 16-byte boundary so that a thread fetches only the set of its own range.  128 bytes.
struct alignas(16) SpecRow {
    double lo[7];
    double inv_w;
    double hi[7];
    double t_mid;
};

// Plain class: reversible elementary reactions whose species are all distinct with unit
// coefficients (so the scatter list is the slot list and the slots of one reaction never
// collide).  Stored by shape (molecules per side), shape s = 3 (nreac-1) + (nprod-1); within a
// shape first the groups of eight mutually species-disjoint reactions, then the groups of
// four, then the couples, then the reactions left alone.  Large mechanisms couple a reaction
// left alone with a null record instead (every slot names the dummy species, so its rate is
// exactly zero).  48 bytes.
struct alignas(16) RxnP {
    double f[3];        // log2 k_f = f0 + f1 log2T + f2/T          (A.9) PAPER.md:925
    uint32_t slot[6];   // species: reactants 0..nreac-1, then products nreac..nreac+nprod-1
};

// Extended class: three-body and falloff reactions, irreversible reactions, reactions
// with a repeated species (coefficient 2 or 3, or a species on both sides), and "wide" reactions
// (a side's sum of log2 E_k exceeds 700 somewhere in the supported temperature range).  The rate is
// formed in reactant/product pairs, R = k [prod_i (A_ri B_ri) - prod_i (A_pi B_ri)], i = 0..2 left to
// right, with the slots ordered by the packer so that the partial products stay in range.  Stored by kind,
// within a kind first the groups of four reactions with mutually disjoint scatter lists, then
// the couples, then the reactions left alone.  The six slots list every molecule (a
// coefficient 2 repeats the species), reactants in 0..2 and products in 3..5; unused slots and
// unused scatter entries name the dummy species n_species (A = B = 1, omega = sink), so that
// the code is branch-free.  The scatter list holds each species once, with its net
// coefficient.  112 bytes.
enum { kExtGeneral = 0, kExtThreeBody = 1, kExtLindemann = 2, kExtTroe = 3 };

struct alignas(16) RxnX {
    double f[3];             // log2 k_f (high-pressure limit for falloff kinds)
    uint32_t slot[6];
    uint32_t sc_species[6];  // omega[sc_species] += sc_nu * R
    double eff_default;      // [M] = eff_default * C_tot + sum_listed eff_delta * C_k
    int16_t sc_nu[6];        // net stoichiometric coefficients of the scatter list (one I2F each)
    int16_t rev;             // 1 reversible, 0 irreversible (r_r = 0)
    int16_t type;            // PYRO_ELEMENTARY .. PYRO_FALLOFF_TROE
    uint32_t eff_begin;      // first entry of the efficiency list
    uint32_t eff_count;      // entries, padded with (0, dummy) to the maximum of the lockstep group, a multiple of 4
    uint32_t fall_index;     // row of the falloff table (kinds kExtLindemann, kExtTroe)
    uint32_t pad;
};

// Falloff parameters of an extended reaction.  64 bytes.
struct alignas(16) RxnFall {
    double l[3];             // log2 k_0 (low-pressure limit)
    double troe_alpha;       // Troe: Fcent = (1-alpha) 2^(t3 T) + alpha 2^(t1 T) + has_t2 2^(t2/T)
    double troe_t3, troe_t1, troe_t2;   // -log2e/T***, -log2e/T*, -log2e T**
    double troe_has_t2;      // 1.0 or 0.0
};

// One listed third-body efficiency: delta = eff - eff_default of the reaction.  16 bytes.
struct alignas(16) EffEntry {
    double delta;
    uint32_t species;
    uint32_t pad;
};

// Byte offsets into the table blob (all 16-byte aligned) and the loop counts of the kernels.
struct TableLayout {
    uint32_t off_spec;       // SpecRow[n_species]
    uint32_t off_rxn_p;      // RxnP[n_p]
    uint32_t off_rxn_x;      // RxnX[n_x]
    uint32_t off_fall;       // RxnFall[n_fall]
    uint32_t off_eff;        // EffEntry[n_eff]
    uint32_t bytes;
    int32_t n_species;
    int32_t n_p, n_x, n_eff, n_fall;   // stored records (null records included)
    int32_t shape_g8[9];     // plain class, per shape: records stored as disjoint groups of eight
    int32_t shape_g4[9];     // ... of four
    int32_t shape_g2[9];     // ... as couples
    int32_t shape_g1[9];     // ... alone
    int32_t ext_g4[4];       // extended class, per kind: records stored as disjoint groups of four
    int32_t ext_g2[4];       // ... as couples
    int32_t ext_g1[4];       // ... alone
    int32_t needs_ctot;      // any extended reaction uses [M]
    int32_t single_t_mid;    // 1 if every species has the same T_mid (needed by the temperature solve)
    double t_mid;            // that T_mid
};

static_assert(sizeof(SpecRow) == 128 && sizeof(RxnP) == 48 && sizeof(RxnX) == 112 && sizeof(RxnFall) == 64 &&
                  sizeof(EffEntry) == 16,
              "table records are read with 128-bit loads");

// Loop counts of one mechanism, as the kernels take them (copied from TableLayout).
struct GroupCounts {
    int32_t shape_g8[9], shape_g4[9], shape_g2[9], shape_g1[9], ext_g4[4], ext_g2[4], ext_g1[4];
};

// Energy table of the temperature solve: per species and NASA range the six coefficients
//   (a6, a1-1, a2/2, a3/3, a4/4, a5/5) * R/W_k
// so that  e(T) = sum_k Y_k (c0 + c1 T + ... + c5 T^5)   (A.25)-(A.26) PAPER.md:1008-1012
// and      c_v(T) = de/dT                                 (A.29)-(A.31) PAPER.md:1025-1034
// rw = R/W_k serves the enthalpy form (h_k = e_k + R T/W_k) and the equation of
// state (A.2)-(A.3) PAPER.md:892-899: sum_k Y_k R/W_k = R / W_mix.
// t_mid: the species' own break temperature (the general solve for mechanisms with several of them).
// w = W_k serves the reactor march (A.1): dY_k/dt = W_k omega_k / rho.  128 bytes.
struct alignas(16) EnergyRow {
    double lo[6], hi[6];
    double rw, t_mid;
    double w, pad;
};

}   // namespace pyro
