// Mechanism packer interface (host side of libpyro).
#pragma once
#include <string>
#include <vector>

#include "../../include/pyro.h"
#include "pyro_jac_tables.h"
#include "pyro_tables.h"

namespace pyro {

// Limits of the on-chip staging: per point n_species + 1 values of plane W in tensor memory (512
// 32-bit columns per thread at most) and of planes A, B in shared / tensor memory.
constexpr int kMaxSpecies = 255;
constexpr int kMaxReactions = 1 << 20;

struct PackedMech {
    TableLayout lay;
    std::vector<unsigned char> blob;   // rates tables, laid out by `lay`
    std::vector<EnergyRow> energy;     // temperature-solve table [n_species]
    std::vector<int> order;            // packed record -> reaction index of the description (-1: null record)
    int n_species = 0, n_reactions = 0;
    double max_side_log2 = 0.0;        // plain class: largest |sum over a reaction side of log2 E_k| over the guard temperatures
    double max_pair_log2 = 0.0;        // extended class: largest |partial sum of pair exponents| (pyro_tables.h "Range")
    int n_wide = 0;                    // reactions that are in the extended class only because a side sum exceeds the plain limit
};

// Returns a pyro_status; on failure `err` says which entry was rejected.
// `leftover` says what happens to reactions that end up alone after the lockstep grouping:
// kLeftoverPad couples each with a null record, kLeftoverSingles stores them as singles (the
// kernel variant must then contain the one-at-a-time loops), kLeftoverAuto takes singles for
// fewer than 64 reactions (environment PYRO_PACK_SINGLES=0/1 overrides; host tests).
enum { kLeftoverAuto = -1, kLeftoverPad = 0, kLeftoverSingles = 1 };
// `shift`: kShiftOn subtracts the conserved part of log2 E_k from the species rows (pyro_tables.h "Range");
// kShiftOff leaves the rows as folded (host tests: the two must give the same rates).
enum { kShiftOn = 1, kShiftOff = 0 };
int pack_mechanism(const pyro_mech_desc *desc, PackedMech &out, std::string &err, int leftover = kLeftoverAuto,
                   int shift = kShiftOn);

// Tables of the chemical-Jacobian kernel (pyro_jac_tables.h) of a description that pack_mechanism accepted.
// The kernel keeps two accumulators per species in tensor memory: at most kJacMaxSpecies species.
constexpr int kJacMaxSpecies = 127;
struct JacPacked {
    JacLayout lay;
    std::vector<unsigned char> blob;
};
int pack_jacobian(const pyro_mech_desc *desc, JacPacked &out, std::string &err);

// Falloff row of reaction j of a validated description (shared by the rates and the Jacobian tables).
RxnFall fall_row(const pyro_mech_desc *desc, int j);

}   // namespace pyro
