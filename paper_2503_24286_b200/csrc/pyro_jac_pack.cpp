// Packer of the chemical-Jacobian tables (pyro_jac_tables.h): transposes a validated mechanism into per-species
// incidence lists.  Called by pyro_mech_create after pack_mechanism has accepted the description.
#include <algorithm>
#include <cmath>
#include <cstring>
#include <map>

#include "pyro_pack.h"

namespace pyro {
namespace {
uint32_t align16j(uint32_t x) { return (x + 15u) & ~15u; }
}   // namespace

int pack_jacobian(const pyro_mech_desc *d, JacPacked &out, std::string &err) {
    const int ns = d->n_species, nr = d->n_reactions;
    if (ns > kJacMaxSpecies) {
        err = "the Jacobian kernel holds at most " + std::to_string(kJacMaxSpecies) + " species";
        return PYRO_ERR_TOO_LARGE;
    }
    const long double log2e = 1.0L / std::log(2.0L);
    const uint16_t dummy = (uint16_t)ns;
    std::vector<JacRxn> rxn_plain, rxn_ext;
    std::vector<EffEntry> effs;
    std::vector<RxnFall> falls;
    std::vector<std::vector<JacInc>> inc(ns);
    std::vector<std::vector<JacInc>> effinc(ns);   // incidences through a listed third-body efficiency
    for (int j = 0; j < nr; ++j) {
        JacRxn r;
        std::memset(&r, 0, sizeof r);
        r.f[0] = (double)(std::log((long double)d->A[j]) * log2e);
        r.f[1] = d->b[j];
        r.f[2] = (double)(-(long double)d->theta[j] * log2e);
        for (int m = 0; m < 6; ++m) r.slot[m] = r.sc_species[m] = dummy;
        std::map<int, int> net, nreac_of, nprod_of;
        int nreac = 0, nprod = 0;
        for (int q = d->reac_ptr[j]; q < d->reac_ptr[j + 1]; ++q) {
            for (int c = 0; c < d->reac_coeff[q]; ++c) r.slot[nreac++] = (uint16_t)d->reac_species[q];
            net[d->reac_species[q]] -= d->reac_coeff[q];
            nreac_of[d->reac_species[q]] += d->reac_coeff[q];
        }
        for (int q = d->prod_ptr[j]; q < d->prod_ptr[j + 1]; ++q) {
            for (int c = 0; c < d->prod_coeff[q]; ++c) r.slot[3 + nprod++] = (uint16_t)d->prod_species[q];
            net[d->prod_species[q]] += d->prod_coeff[q];
            nprod_of[d->prod_species[q]] += d->prod_coeff[q];
        }
        int nsc = 0;
        for (auto &kv : net)
            if (kv.second != 0) {
                r.sc_species[nsc] = (uint16_t)kv.first;
                r.sc_w[nsc] = (double)((long double)kv.second * (long double)d->mol_weight[kv.first]);
                ++nsc;
            }
        r.rev = d->reversible[j] ? 1 : 0;
        r.type = d->type[j];
        r.eff_default = 1.0;
        const bool ext = r.type != PYRO_ELEMENTARY;
        uint16_t mul_slot = 0;
        if (ext) {
            r.ext = (uint32_t)rxn_ext.size();
            mul_slot = (uint16_t)(1u + 2u * r.ext);
            r.eff_default = d->eff_default[j];
            r.eff_begin = (uint32_t)effs.size();
            for (int q = d->eff_ptr[j]; q < d->eff_ptr[j + 1]; ++q) {
                const double delta = d->eff_value[q] - d->eff_default[j];
                effs.push_back(EffEntry{delta, (uint32_t)d->eff_species[q], 0u});
                // species eff_species[q] enters R through [M]: d = delta * g_x, written as an incidence whose
                // exponent is 0 (2^0 = 1 exactly) and whose other molecules are the dummy species (C = 1)
                JacInc e;
                std::memset(&e, 0, sizeof e);
                e.coef = delta;
                for (int m = 0; m < 6; ++m) {
                    e.sc_w[m] = r.sc_w[m];
                    e.sc_species[m] = r.sc_species[m];
                    e.gslot[m] = dummy;
                }
                e.other[0] = e.other[1] = dummy;
                e.mul = (uint16_t)(2u + 2u * r.ext);
                effinc[d->eff_species[q]].push_back(e);
            }
            r.eff_count = (uint32_t)effs.size() - r.eff_begin;
            if (r.type >= PYRO_FALLOFF_LINDEMANN) {
                r.fall_index = (uint32_t)falls.size();
                falls.push_back(fall_row(d, j));
            }
        }
        // incidences: species k as a molecule of the reactant side (forward rate) / product side (reverse rate)
        for (int side = 0; side < 2; ++side) {
            if (side == 1 && !r.rev) continue;
            const std::map<int, int> &cnt = side ? nprod_of : nreac_of;
            for (auto &kv : cnt) {
                JacInc e;
                std::memset(&e, 0, sizeof e);
                for (int m = 0; m < 3; ++m) e.f[m] = r.f[m];
                e.coef = side ? -(double)kv.second : (double)kv.second;
                for (int m = 0; m < 6; ++m) {
                    e.sc_w[m] = r.sc_w[m];
                    e.sc_species[m] = r.sc_species[m];
                    e.gslot[m] = side ? r.slot[m] : dummy;
                }
                int no = 0;
                bool skipped = false;
                e.other[0] = e.other[1] = dummy;
                for (int m = 0; m < 3; ++m) {
                    const uint16_t s = r.slot[3 * side + m];
                    if (s == dummy) continue;
                    if (!skipped && s == (uint16_t)kv.first) {
                        skipped = true;   // one molecule of k is differentiated away
                        continue;
                    }
                    e.other[no++] = s;
                }
                e.mul = mul_slot;
                inc[kv.first].push_back(e);
            }
        }
        (ext ? rxn_ext : rxn_plain).push_back(r);
    }
    if (1 + 2 * rxn_ext.size() > 65535) {
        err = "too many third-body / falloff reactions for the Jacobian tables";
        return PYRO_ERR_TOO_LARGE;
    }
    JacLayout &lay = out.lay;
    std::memset(&lay, 0, sizeof lay);
    lay.n_species = ns;
    lay.n_plain = (int)rxn_plain.size();
    lay.n_ext = (int)rxn_ext.size();
    lay.n_eff = (int)effs.size();
    lay.n_fall = (int)falls.size();
    std::vector<JacCol> cols(ns);
    std::vector<JacInc> inc_all;
    auto inc_class = [&](const JacInc &e) {
        bool gibbs = false;
        for (int m = 0; m < 6; ++m) gibbs = gibbs || e.gslot[m] != dummy;
        const bool wide = e.sc_species[4] != dummy || e.sc_species[5] != dummy;   // the scatter list is filled from the front
        return 2 * (gibbs ? 1 : 0) + (wide ? 1 : 0);
    };
    for (int k = 0; k < ns; ++k) {
        std::vector<JacInc> list(inc[k]);
        list.insert(list.end(), effinc[k].begin(), effinc[k].end());
        std::memset(&cols[k], 0, sizeof cols[k]);
        cols[k].inc_begin = (uint32_t)inc_all.size();
        for (int c = 0; c < 4; ++c) {
            size_t n = 0;
            for (const JacInc &e : list)
                if (inc_class(e) == c) {
                    inc_all.push_back(e);
                    ++n;
                }
            if (n > 65535) {
                err = "too many incidences of one species for the Jacobian tables";
                return PYRO_ERR_TOO_LARGE;
            }
            cols[k].n_class[c] = (uint16_t)n;
        }
        cols[k].inc_end = (uint32_t)inc_all.size();
    }
    lay.n_inc = (int)inc_all.size();
    std::vector<JacRxn> rxn(rxn_plain);
    rxn.insert(rxn.end(), rxn_ext.begin(), rxn_ext.end());
    uint32_t off = 0;
    lay.off_rxn = off;
    off = align16j(off + (uint32_t)(rxn.size() * sizeof(JacRxn)));
    lay.off_inc = off;
    off = align16j(off + (uint32_t)(inc_all.size() * sizeof(JacInc)));
    lay.off_eff = off;
    off = align16j(off + (uint32_t)(effs.size() * sizeof(EffEntry)));
    lay.off_fall = off;
    off = align16j(off + (uint32_t)(falls.size() * sizeof(RxnFall)));
    lay.off_col = off;
    off = align16j(off + (uint32_t)(cols.size() * sizeof(JacCol)));
    // the columns by decreasing list length: the block kernel hands them to its warps in this order (longest first)
    std::vector<uint32_t> order(ns);
    for (int k = 0; k < ns; ++k) order[k] = (uint32_t)k;
    std::stable_sort(order.begin(), order.end(), [&](uint32_t x, uint32_t y) {
        return cols[x].inc_end - cols[x].inc_begin > cols[y].inc_end - cols[y].inc_begin;
    });
    lay.off_order = off;
    off = align16j(off + (uint32_t)(order.size() * sizeof(uint32_t)));
    lay.bytes = off;
    out.blob.assign(off, 0);
    auto put = [&](uint32_t at, const void *src, size_t bytes) {
        if (bytes) std::memcpy(out.blob.data() + at, src, bytes);
    };
    put(lay.off_rxn, rxn.data(), rxn.size() * sizeof(JacRxn));
    put(lay.off_inc, inc_all.data(), inc_all.size() * sizeof(JacInc));
    put(lay.off_eff, effs.data(), effs.size() * sizeof(EffEntry));
    put(lay.off_fall, falls.data(), falls.size() * sizeof(RxnFall));
    put(lay.off_col, cols.data(), cols.size() * sizeof(JacCol));
    put(lay.off_order, order.data(), order.size() * sizeof(uint32_t));
    return PYRO_OK;
}

}   // namespace pyro
