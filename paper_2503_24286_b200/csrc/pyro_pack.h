// Mechanism packer interface (host side of libpyro).
#pragma once
#include <string>
#include <vector>

#include "../../include/pyro.h"
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
};

// Returns a pyro_status; on failure `err` says which entry was rejected.
int pack_mechanism(const pyro_mech_desc *desc, PackedMech &out, std::string &err);

}   // namespace pyro
