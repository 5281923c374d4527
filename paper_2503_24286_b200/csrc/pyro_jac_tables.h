// Device tables of the chemical-Jacobian kernel, shared by its packer (host) and
// the kernel.  Internal to libpyro; the public boundary is include/pyro.h (pyro_get_jacobian).
//
// What is computed (eq. (6); (A.36) PAPER.md:1057; S_i = W_i omega_i (A.1) PAPER.md:888):
//     J_ik = dS_i/dY_k = W_i (rho/W_k) sum_j nu_ij dR_j/dC_k  [ - dS_i/dT e_k/c_v  at fixed (rho, e) ]
//     dS_i/dT = W_i sum_j nu_ij dR_j/dT
// with R_j of (A.7) and its rate-coefficient forms (A.9), (A.10), readings G6-G8.
//
// Formulation.  One thread owns one point and walks the Jacobian COLUMN BY COLUMN, because a column
// (n_species values) fits on chip per thread while the matrix (n_species^2) does not.  Column k collects
//     d omega_i / dC_k = sum over the reactions in which species k takes part (as a molecule of one side)
//                        + sum over the third-body / falloff reactions, through [M] = sum eff_k C_k
// so the packer transposes the mechanism: per species the list of its INCIDENCES (reaction, side).  An
// incidence costs one exponential:  d q_f/dC_k = mult k_f prod(other reactant molecules)  and
// d q_r/dC_k = mult k_f/K_c prod(other product molecules), k_f/K_c = 2^(log2 k_f + sum_prod G - sum_reac G) with
// the per-species G_k = log2 E_k of pyro_tables.h (the plain definition's second exponential; no products of
// species factors, hence no range limit beyond that of K_c itself).
// Third-body / falloff reactions are evaluated once per point (phase 1), which leaves two numbers per
// reaction in a per-thread scratch: the multiplier of the incidence terms (mul = [M] or L F) and the
// coefficient of eff_k (g = dR/d[M]); the part of sum_x nu_ix g_x eff_xk that comes from the default efficiency
// is the same for every column and is accumulated once (plane V); the listed efficiencies are incidences
// of their own.  The temperature derivative is one more accumulation over all reactions (plane DT).
#pragma once
#include <cstdint>

#include "pyro_tables.h"

namespace pyro {

// One reaction of any type (phases 1 and 2).  Type 0 reactions come first, then the [M] reactions.  128 bytes.
struct alignas(16) JacRxn {
    double f[3];              // log2 k_f = f0 + f1 log2 T + f2 / T   (A.9)
    double sc_w[6];           // nu_i W_i of the scatter list (W_i folded in: the planes hold dS, not d omega)
    double eff_default;
    uint16_t slot[6];         // molecules: reactants 0..2, products 3..5; unused = dummy species n_species (C = 1, G = 0)
    uint16_t sc_species[6];   // each species once, with its net coefficient; unused = dummy (sink)
    uint16_t rev, type;       // reversible flag; PYRO_ELEMENTARY .. PYRO_FALLOFF_TROE
    uint32_t eff_begin, eff_count;   // listed efficiencies (EffEntry: delta = eff - eff_default)
    uint32_t fall_index;      // RxnFall row (falloff types)
    uint32_t ext;             // [M] reactions: scratch slots 1 + 2 ext (mul) and 2 + 2 ext (g); slot 0 holds 1.0
    uint32_t pad;
};

// Species k is a molecule of one side of reaction r.  112 bytes.
//   d = coef * scratch[mul] * 2^(f . features + sum G[gslot 3..5] - sum G[gslot 0..2]) * C[other0] * C[other1]
//   column_k[sc_species] += sc_w * d
struct alignas(16) JacInc {
    double f[3];
    double coef;              // + multiplicity of k among the reactants, or - multiplicity among the products
    double sc_w[6];
    uint16_t other[2];        // the other molecules of that side (dummy: C = 1)
    uint16_t gslot[6];        // product-side incidence: the reaction's molecule slots; reactant side: all dummy (G = 0)
    uint16_t sc_species[6];
    uint16_t mul;             // scratch slot of the multiplier (0: the constant 1)
    uint16_t pad;
};

// The incidence list of one species: records [inc_begin, inc_end) of the JacInc table, in the order the kernel walks
// them (the whole table is read front to back once per point).  A species that is listed in the efficiency list of
// an [M]-reaction x has one more incidence for it: d = delta * scratch[g_x], stored as a JacInc whose exponent is 0
// (2^0 = 1 exactly), whose other molecules are the dummy species and whose multiplier slot is g_x.
// Within a list the records are sorted into four classes, each with a loop of its own in the kernel (no per-record
// branch): class = 2 * (has a Gibbs sum: product-side incidence) + (more than four scatter entries); n_class[c] records
// of class c follow one another in the order 0, 1, 2, 3.  A record of a class without a Gibbs sum has all its gslot =
// dummy, one with at most four scatter entries has sc_species[4..5] = dummy: the short loops skip work whose result
// is exactly zero.  16 bytes.
struct alignas(16) JacCol {
    uint32_t inc_begin, inc_end;
    uint16_t n_class[4];
};

struct JacLayout {
    uint32_t off_rxn, off_inc, off_eff, off_fall, off_col, off_order, bytes;   // off_order: uint32[n_species], the columns by decreasing list length
    int32_t n_species, n_plain, n_ext, n_inc, n_eff, n_fall;
};

static_assert(sizeof(JacRxn) == 128 && sizeof(JacInc) == 112 && sizeof(JacCol) == 16,
              "Jacobian table records are multiples of 16 bytes");

}   // namespace pyro
