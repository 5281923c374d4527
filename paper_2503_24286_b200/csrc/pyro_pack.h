// Mechanism packer interface (host side of libpyro).
#pragma once
#include <string>
#include <vector>

#include "../../include/pyro.h"
#include "pyro_tables.h"

namespace pyro {

// Limits of the on-chip staging: three FP64 planes of n_species + 1 per point in shared memory,
// 32 points per block at least, 227 KB per block at most.
constexpr int kMaxSpecies = 300;
constexpr int kMaxReactions = 1 << 20;

struct PackedMech {
    TableLayout lay;
    std::vector<unsigned char> blob;   // rates tables, laid out by `lay`
    std::vector<EnergyRow> energy;     // temperature-solve table [n_species]
    std::vector<int> order;            // packed position -> reaction index of the description
    int n_species = 0, n_reactions = 0;
};

// Returns a pyro_status; on failure `err` says which entry was rejected.
int pack_mechanism(const pyro_mech_desc *desc, PackedMech &out, std::string &err);

}   // namespace pyro
