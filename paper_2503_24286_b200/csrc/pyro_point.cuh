// Per-point arithmetic of the hot path, shared by the kernels and the host test build.
//
// One thread owns one grid point.  Per-point arrays indexed by a run-time species number live
// on chip as three planes per species:
//     plane A  A_k = C_k E_k      plane B  B_k = 1/E_k      plane W  omega_k
// with E_k = exp(g_k/RT) RT/p0 (pyro_tables.h).  The functions below reach them through a
// `Mem` accessor (A in shared memory, W and B side by side in tensor memory in the kernels --
// or B in shared memory for very large mechanisms -- plain arrays in the host build):
//     hA = mem.atA(k), hW = mem.atW(k), hB = mem.atB(k)    handles of species k for this thread
//     mem.ldA(hA)
//     r = mem.ldW(hW), mem.ldB(hW, hB), mem.ldWB(hW, hB)   raw values; readable by mem.value(r),
//         mem.value_w(r), mem.value_b(r) only after mem.fence_ld()   (tensor-memory loads are asynchronous)
//     mem.stW(hW, v); mem.fence_st() before a later load may see the stored value
//     mem.st_species(k, a, b)                              fill: A_k = a, B_k = b, omega_k = 0
#pragma once
#include "../../include/pyro.h"
#include "pyro_math.cuh"
#include "pyro_tables.h"

namespace pyro {

constexpr double kLog10of2 = 0.30102999566398119521;   // log10(2)

// Per-thread temperature features of its point (V = double) or of its two points (V = D2, pyro_math.cuh).
template <class V> struct PointTV {
    V T, invT, L2T;
};
typedef PointTV<double> PointT;

PYRO_HD PointT make_point(double T) {
    PointT pt;
    pt.T = T;
    pt.invT = 1.0 / T;
    pt.L2T = log2(T);
    return pt;
}
PYRO_HD PointTV<D2> make_point(D2 T) {
    PointTV<D2> pt;
    pt.T = T;
    pt.invT = D2{1.0 / T.x, 1.0 / T.y};
    pt.L2T = D2{log2(T.x), log2(T.y)};
    return pt;
}

// log2 k = c0 + c1 log2T + c2/T                               (A.9) PAPER.md:925
template <class V> PYRO_HD V arrhenius_log2(double c0, double c1, double c2, V L2T, V invT) {
    return fma(c1, L2T, fma(c2, invT, c0));
}

// log2 E_k = c0 + c1 log2T + c2/T + c3 T + c4 T^2 + c5 T^3 + c6 T^4     (A.11)-(A.13) folded
PYRO_HD double species_log2E(const double *c, double T, double L2T, double invT) {
    double h = fma(c[6], T, c[5]);
    h = fma(h, T, c[4]);
    h = fma(h, T, c[3]);
    double y = fma(h, T, c[0]);
    y = fma(c[1], L2T, y);
    return fma(c[2], invT, y);
}
// the same with the NASA range chosen per point (T < T_mid,k: low; G10) by fetching only that coefficient set
PYRO_HD double species_log2E_row(const SpecRow &row, const PointT &pt) {
    return species_log2E(pt.T < row.t_mid ? row.lo : row.hi, pt.T, pt.L2T, pt.invT);
}
PYRO_HD D2 species_log2E_row(const SpecRow &row, const PointTV<D2> &pt) {
    return D2{species_log2E(pt.T.x < row.t_mid ? row.lo : row.hi, pt.T.x, pt.L2T.x, pt.invT.x),
              species_log2E(pt.T.y < row.t_mid ? row.lo : row.hi, pt.T.y, pt.L2T.y, pt.invT.y)};
}

// Rows a2, a3 of SURVEY.md 8(a) for NK species in lockstep: C_k = rho Y_k / W_k (A.8)
// PAPER.md:921, the NASA range chosen per point, E_k and 1/E_k by one paired exponential.  Writes A_k = C_k E_k,
// B_k = 1/E_k, omega_k = 0 and adds C_k to ctot.
template <int NK, class Tab, class Mem, class PT, class V>
PYRO_HD void species_planes(const Tab &tab, int k0, const PT &pt, V rho, const V (&Y)[NK], V &ctot, const Mem &mem) {
    V y[NK], e[NK], b[NK], C[NK];
#pragma unroll
    for (int i = 0; i < NK; ++i) {
        const SpecRow &row = tab.spec(k0 + i);
        y[i] = species_log2E_row(row, pt);
        C[i] = rho * Y[i] * row.inv_w;
    }
    exp2_pair_nv<NK>(y, e, b);
#pragma unroll
    for (int i = 0; i < NK; ++i) {
        ctot += C[i];
        mem.st_species((uint32_t)(k0 + i), C[i] * e[i], b[i]);
    }
}

// The first N species slots of a record, fetched two at a time (the records are 16-byte aligned).
template <int N> PYRO_HD void load_slots(const uint32_t (&src)[6], uint32_t (&dst)[6]) {
#pragma unroll
    for (int m = 0; m < N; m += 2) {
        const unsigned long long p = *reinterpret_cast<const unsigned long long *>(&src[m]);
        dst[m] = (uint32_t)p;
        dst[m + 1] = (uint32_t)(p >> 32);
    }
}

// Plain-class reactions of one shape (NR reactant molecules, NP product molecules), NB in
// lockstep (the packer stores groups of mutually species-disjoint reactions):
//   R = k_f prod_reac B_k [prod_reac A_k - prod_prod A_k]    (A.7), (A.10) as in pyro_tables.h
//   omega -= R on reactants, += R on products                (A.5)
// Branch-free.  The NB exponentials run as interleaved Horner chains; all species touched in
// one iteration are distinct, so the omega read-modify-writes are one batch of loads, the
// adds, one batch of stores.  V = typename Mem::V: one point per thread or two.
template <int NR, int NP, int NB, class Tab, class Mem, class PT>
PYRO_HD void plain_reactions(const Tab &tab, int j0, int count, const PT &pt, const Mem &mem) {
    typedef typename Mem::V V;
    constexpr int NS = NR + NP;
#pragma unroll 1
    for (int j = j0; j < j0 + count; j += NB) {
        uint32_t hA[NB][NS], hB[NB][NR], hW[NB][NS];
        V y[NB];
#pragma unroll
        for (int b = 0; b < NB; ++b) {
            const RxnP &r = tab.rxn_p(j + b);
            uint32_t slot[6];
            load_slots<NS>(r.slot, slot);
#pragma unroll
            for (int m = 0; m < NS; ++m) {
                hA[b][m] = mem.atA(slot[m]);
                if (m < NR) hB[b][m] = mem.atB(slot[m]);
                hW[b][m] = mem.atW(slot[m]);
            }
            y[b] = arrhenius_log2(r.f[0], r.f[1], r.f[2], pt.L2T, pt.invT);
        }
        mem.fence_st();
        typename Mem::WBRaw wbr[NB][NR];   // reactants: omega and B together
        typename Mem::WRaw wr[NB][NP];     // products: omega
#pragma unroll
        for (int b = 0; b < NB; ++b) {
#pragma unroll
            for (int m = 0; m < NR; ++m) wbr[b][m] = mem.ldWB(hW[b][m], hB[b][m]);
#pragma unroll
            for (int m = 0; m < NP; ++m) wr[b][m] = mem.ldW(hW[b][NR + m]);
        }
        V a[NB][NS];
#pragma unroll
        for (int b = 0; b < NB; ++b)
#pragma unroll
            for (int m = 0; m < NS; ++m) a[b][m] = mem.ldA(hA[b][m]);
        exp2_poly_nv<NB>(y);
        V pd[NB];   // k_f (prod_reac A - prod_prod A)
#pragma unroll
        for (int b = 0; b < NB; ++b) {
            V pf = a[b][0], pr = a[b][NR];
#pragma unroll
            for (int m = 1; m < NR; ++m) pf *= a[b][m];
#pragma unroll
            for (int m = 1; m < NP; ++m) pr *= a[b][NR + m];
            pd[b] = y[b] * (pf - pr);
        }
        mem.fence_ld();
#pragma unroll
        for (int b = 0; b < NB; ++b) {
            V pb = mem.value_b(wbr[b][0]);
#pragma unroll
            for (int m = 1; m < NR; ++m) pb *= mem.value_b(wbr[b][m]);
            const V R = pb * pd[b];
#pragma unroll
            for (int m = 0; m < NR; ++m) mem.stW(hW[b][m], mem.value_w(wbr[b][m]) - R);
#pragma unroll
            for (int m = 0; m < NP; ++m) mem.stW(hW[b][NR + m], mem.value(wr[b][m]) + R);
        }
    }
}

// One shape of the plain class: its groups of eight and of four run four in lockstep, its
// couples two in lockstep, the rest one at a time.
// kSingles = false leaves the one-at-a-time loops out (the packer then stores no singles): for
// large mechanisms their code alone costs 8 % (measured on configs[2]: instruction cache).
// kQuads = false runs the groups of eight and of four two in lockstep as well (they are stored as consecutive
// disjoint couples): small mechanisms hardly have such groups, and without the four-in-lockstep loops the
// two-points-per-thread kernel is half the code and far fewer registers.
template <int NR, int NP, bool kSingles, bool kQuads, class Tab, class Mem, class PT>
PYRO_HD int plain_shape(const Tab &tab, int j, int g8, int g4, int g2, int g1, const PT &pt, const Mem &mem) {
    if (kQuads) {
        plain_reactions<NR, NP, 4>(tab, j, g8 + g4, pt, mem);
        plain_reactions<NR, NP, 2>(tab, j + g8 + g4, g2, pt, mem);
    } else {
        plain_reactions<NR, NP, 2>(tab, j, g8 + g4 + g2, pt, mem);
    }
    if (kSingles) plain_reactions<NR, NP, 1>(tab, j + g8 + g4 + g2, g1, pt, mem);
    return j + g8 + g4 + g2 + g1;
}

// Extended-class reactions of one kind, NB in lockstep: third body, falloff (Lindemann /
// Troe), and general elementary reactions (irreversible, repeated species).  Forms per
// reading G6-G8 (PAPER.md:928 only cites them).  Slots and scatter entries are padded with the
// dummy species and the efficiency lists of a group have one length, so there are no
// data-dependent branches; logarithms and divisions are the branch-free log2_pos and
// rcp_newton of pyro_math.cuh.
template <int KIND, int NB, class Tab, class Mem, class PT, class V>
PYRO_HD void extended_reactions(const Tab &tab, int j0, int count, const PT &pt, V ctot, const Mem &mem) {
    constexpr int NE = KIND == kExtTroe ? 5 : (KIND == kExtLindemann ? 2 : 1);   // exponentials per reaction
#pragma unroll 1
    for (int j = j0; j < j0 + count; j += NB) {
        uint32_t hA[NB][6], hB[NB][3], hWs[NB][3], hW[NB][6];   // hWs: tensor-memory handle of a reactant slot (its B)
        double nu[NB][6], rev[NB], alpha[NB], has_t2[NB];
        V M[NB];
        V y[NB * NE];
        uint32_t q0[NB], nq = 0;
#pragma unroll
        for (int b = 0; b < NB; ++b) {
            const RxnX &x = tab.rxn_x(j + b);
            uint32_t slot[6], sc[6];
            load_slots<6>(x.slot, slot);
            load_slots<6>(x.sc_species, sc);
#pragma unroll
            for (int m = 0; m < 6; ++m) {
                hA[b][m] = mem.atA(slot[m]);
                if (m < 3) {
                    hB[b][m] = mem.atB(slot[m]);
                    hWs[b][m] = mem.atW(slot[m]);
                }
                hW[b][m] = mem.atW(sc[m]);
                nu[b][m] = (double)x.sc_nu[m];
            }
            rev[b] = (double)x.rev;
            y[b * NE] = arrhenius_log2(x.f[0], x.f[1], x.f[2], pt.L2T, pt.invT);
            M[b] = x.eff_default * ctot;
            q0[b] = x.eff_begin;
            nq = x.eff_count;   // one length per group
            if (KIND >= kExtLindemann) {
                const RxnFall &fl = tab.rxn_fall((int)x.fall_index);
                y[b * NE + 1] = arrhenius_log2(fl.l[0], fl.l[1], fl.l[2], pt.L2T, pt.invT) - y[b * NE];   // log2(k0/k_inf)
                if (KIND == kExtTroe) {
                    alpha[b] = fl.troe_alpha;
                    has_t2[b] = fl.troe_has_t2;
                    y[b * NE + 2] = fl.troe_t3 * pt.T;
                    y[b * NE + 3] = fl.troe_t1 * pt.T;
                    y[b * NE + 4] = fl.troe_t2 * pt.invT;
                }
            }
        }
        mem.fence_st();
        typename Mem::WRaw wr[NB][6], br[NB][3];
#pragma unroll
        for (int b = 0; b < NB; ++b)
#pragma unroll
            for (int m = 0; m < 6; ++m) {
                wr[b][m] = mem.ldW(hW[b][m]);
                if (m < 3) br[b][m] = mem.ldB(hWs[b][m], hB[b][m]);
            }
        V a[NB][6];
#pragma unroll
        for (int b = 0; b < NB; ++b)
#pragma unroll
            for (int m = 0; m < 6; ++m) a[b][m] = mem.ldA(hA[b][m]);
        if (KIND != kExtGeneral) {
            // [M] = sum_k eff_k C_k = eff_default C_tot + sum_listed (eff_k - eff_default) C_k with
            // C_k = A_k B_k; the lists of a group are padded to one length, a multiple of four
#pragma unroll 1
            for (uint32_t q = 0; q < nq; q += 4) {
                typename Mem::WRaw cb[NB * 4];
                double dl[NB * 4];
                V ca[NB * 4];
#pragma unroll
                for (int b = 0; b < NB; ++b)
#pragma unroll
                    for (int u = 0; u < 4; ++u) {
                        const EffEntry &en = tab.eff((int)(q0[b] + q) + u);
                        cb[b * 4 + u] = mem.ldB(mem.atW(en.species), mem.atB(en.species));
                        ca[b * 4 + u] = mem.ldA(mem.atA(en.species));
                        dl[b * 4 + u] = en.delta;
                    }
                mem.fence_ld();
#pragma unroll
                for (int b = 0; b < NB; ++b)
#pragma unroll
                    for (int u = 0; u < 4; ++u) M[b] = fma(dl[b * 4 + u], ca[b * 4 + u] * mem.value(cb[b * 4 + u]), M[b]);
            }
        }
        exp2_poly_nv<NB * NE>(y);
        V fall[NB];
#pragma unroll
        for (int b = 0; b < NB; ++b) fall[b] = splat<V>(1.0);
        if (KIND >= kExtLindemann) {
            V Pr[NB];
#pragma unroll
            for (int b = 0; b < NB; ++b) {
                Pr[b] = y[b * NE + 1] * M[b];                    // Pr = k0 [M] / k_inf
                fall[b] = Pr[b] * rcp_newton(1.0 + Pr[b]);       // k = k_inf Pr/(1+Pr) F
            }
            if (KIND == kExtTroe) {
                V z[NB];
#pragma unroll
                for (int b = 0; b < NB; ++b) {
                    const V Fc = fma(1.0 - alpha[b], y[b * NE + 2], fma(alpha[b], y[b * NE + 3], has_t2[b] * y[b * NE + 4]));
                    const V l2Fc = log2_pos(Fc);
                    const V lFc = l2Fc * kLog10of2;
                    const V cc = -0.4 - 0.67 * lFc;
                    const V n = 0.75 - 1.27 * lFc;
                    const V lPr = log2_pos(Pr[b]) * kLog10of2 + cc;
                    // F = Fcent^(1/(1+f1^2)), f1 = lPr/d, d = n - 0.14 lPr:  1/(1+f1^2) = d^2/(d^2 + lPr^2)
                    const V d = n - 0.14 * lPr;
                    const V d2 = d * d;
                    z[b] = l2Fc * (d2 * rcp_newton(fma(lPr, lPr, d2)));
                }
                exp2_poly_nv<NB>(z);
#pragma unroll
                for (int b = 0; b < NB; ++b) fall[b] *= z[b];
            }
        }
        mem.fence_ld();
#pragma unroll
        for (int b = 0; b < NB; ++b) {
            // Pair form (pyro_tables.h "Range"): prod_reac C_k = prod_i (A_ri B_ri) and
            // prod_prod C_k / K_c = prod_i (A_pi B_ri), multiplied left to right in the slot order the packer
            // chose, so that no partial product leaves the FP64 range while the rate itself is in it.
            const V b0 = mem.value(br[b][0]), b1 = mem.value(br[b][1]), b2 = mem.value(br[b][2]);
            const V pf = (a[b][0] * b0) * (a[b][1] * b1) * (a[b][2] * b2);
            const V pr = rev[b] != 0.0 ? (a[b][3] * b0) * (a[b][4] * b1) * (a[b][5] * b2) : splat<V>(0.0);   // irreversible: r_r = 0 (G19)
            V R = y[b * NE] * (pf - pr) * fall[b];
            if (KIND == kExtThreeBody) R *= M[b];   // R = [M](q_f - q_r), reading G8
#pragma unroll
            for (int m = 0; m < 6; ++m) mem.stW(hW[b][m], fma(nu[b][m], R, mem.value(wr[b][m])));
        }
    }
}

template <int KIND, bool kSingles, bool kCouples, class Tab, class Mem, class PT, class V>
PYRO_HD int extended_kind(const Tab &tab, int j, int g4, int g2, int g1, const PT &pt, V ctot, const Mem &mem) {
    // groups of four and couples alike run two in lockstep, in ONE loop per kind: four in lockstep
    // gains less than the second copy of the loop costs (instruction cache; measured on configs[2]).
    // kCouples = false (small mechanisms in the two-points-per-thread kernel, where a reaction already is two chains):
    // every record one at a time -- one loop per kind and the registers of one reaction.
    if (kCouples) {
        extended_reactions<KIND, 2>(tab, j, g4 + g2, pt, ctot, mem);
        if (kSingles) extended_reactions<KIND, 1>(tab, j + g4 + g2, g1, pt, ctot, mem);
    } else {
        extended_reactions<KIND, 1>(tab, j, g4 + g2 + g1, pt, ctot, mem);
    }
    return j + g4 + g2 + g1;
}

// Rows a5-a9 of SURVEY.md 8(a): rates of progress of every reaction and their stoichiometric
// accumulation into plane W, (A.5)-(A.10) PAPER.md:908-934.  The planes hold n_species + 1
// entries: the last one is the dummy species (A = B = 1, omega = sink) that pads the
// extended records and the efficiency lists.
template <bool kSingles, bool kQuads = true, class Tab, class Mem, class PT, class V>
PYRO_HD void accumulate_reactions(const Tab &tab, const GroupCounts &g, const PT &pt, V ctot, const Mem &mem) {
    int j = 0;
    j = plain_shape<1, 1, kSingles, kQuads>(tab, j, g.shape_g8[0], g.shape_g4[0], g.shape_g2[0], g.shape_g1[0], pt, mem);
    j = plain_shape<1, 2, kSingles, kQuads>(tab, j, g.shape_g8[1], g.shape_g4[1], g.shape_g2[1], g.shape_g1[1], pt, mem);
    j = plain_shape<1, 3, kSingles, kQuads>(tab, j, g.shape_g8[2], g.shape_g4[2], g.shape_g2[2], g.shape_g1[2], pt, mem);
    j = plain_shape<2, 1, kSingles, kQuads>(tab, j, g.shape_g8[3], g.shape_g4[3], g.shape_g2[3], g.shape_g1[3], pt, mem);
    j = plain_shape<2, 2, kSingles, kQuads>(tab, j, g.shape_g8[4], g.shape_g4[4], g.shape_g2[4], g.shape_g1[4], pt, mem);
    j = plain_shape<2, 3, kSingles, kQuads>(tab, j, g.shape_g8[5], g.shape_g4[5], g.shape_g2[5], g.shape_g1[5], pt, mem);
    j = plain_shape<3, 1, kSingles, kQuads>(tab, j, g.shape_g8[6], g.shape_g4[6], g.shape_g2[6], g.shape_g1[6], pt, mem);
    j = plain_shape<3, 2, kSingles, kQuads>(tab, j, g.shape_g8[7], g.shape_g4[7], g.shape_g2[7], g.shape_g1[7], pt, mem);
    j = plain_shape<3, 3, kSingles, kQuads>(tab, j, g.shape_g8[8], g.shape_g4[8], g.shape_g2[8], g.shape_g1[8], pt, mem);
    int x = 0;
    x = extended_kind<kExtGeneral, kSingles, kQuads>(tab, x, g.ext_g4[0], g.ext_g2[0], g.ext_g1[0], pt, ctot, mem);
    x = extended_kind<kExtThreeBody, kSingles, kQuads>(tab, x, g.ext_g4[1], g.ext_g2[1], g.ext_g1[1], pt, ctot, mem);
    x = extended_kind<kExtLindemann, kSingles, kQuads>(tab, x, g.ext_g4[2], g.ext_g2[2], g.ext_g1[2], pt, ctot, mem);
    x = extended_kind<kExtTroe, kSingles, kQuads>(tab, x, g.ext_g4[3], g.ext_g2[3], g.ext_g1[3], pt, ctot, mem);
    mem.fence_st();
}

// Rows a2, a3 for every species, then the dummy species (A = B = 1, omega = sink): fills the
// three planes.  `load_y(k)` fetches the thread's mass fraction(s) of species k.  Returns C_tot.
template <class Tab, class Mem, class PT, class V, class LoadY>
PYRO_HD V fill_planes(const Tab &tab, int ns, const PT &pt, V rho, const Mem &mem, const LoadY &load_y) {
    V ctot = splat<V>(0.0);
    int k = 0;
#pragma unroll 1
    for (; k + 4 <= ns; k += 4) {
        const V y[4] = {load_y(k), load_y(k + 1), load_y(k + 2), load_y(k + 3)};
        species_planes<4>(tab, k, pt, rho, y, ctot, mem);
    }
#pragma unroll 1
    for (; k < ns; ++k) {
        const V y[1] = {load_y(k)};
        species_planes<1>(tab, k, pt, rho, y, ctot, mem);
    }
    mem.st_species((uint32_t)ns, splat<V>(1.0), splat<V>(1.0));
    return ctot;
}

// Plain arrays of n_species + 1 entries per plane (host build, tests).
struct ArrayMem {
    typedef double V;
    typedef double WRaw;
    struct WBRaw {
        double w, b;
    };
    double *A, *B, *W;
    PYRO_HD uint32_t atA(uint32_t k) const { return k; }
    PYRO_HD uint32_t atB(uint32_t k) const { return k; }
    PYRO_HD uint32_t atW(uint32_t k) const { return k; }
    PYRO_HD double ldA(uint32_t h) const { return A[h]; }
    PYRO_HD void stA(uint32_t h, double v) const { A[h] = v; }
    PYRO_HD WRaw ldW(uint32_t h) const { return W[h]; }
    PYRO_HD WRaw ldB(uint32_t, uint32_t hB) const { return B[hB]; }
    PYRO_HD WBRaw ldWB(uint32_t hW, uint32_t hB) const { return WBRaw{W[hW], B[hB]}; }
    PYRO_HD void stW(uint32_t h, double v) const { W[h] = v; }
    PYRO_HD void st_species(uint32_t k, double a, double b) const {
        A[k] = a;
        B[k] = b;
        W[k] = 0.0;
    }
    PYRO_HD void fence_ld() const {}
    PYRO_HD void fence_st() const {}
    PYRO_HD double value(WRaw r) const { return r; }
    PYRO_HD double value_w(const WBRaw &r) const { return r.w; }
    PYRO_HD double value_b(const WBRaw &r) const { return r.b; }
};

// Newton iteration on the mixture energy polynomial (row a4): (A.27)-(A.28) PAPER.md:1017-1021,
// stop rule per reading G11 (update, then test |dT| < tol; cap max_iter).
//   e(T)   = S[0] + S[1] T + ... + S[5] T^5,  S = sum_k Y_k * EnergyRow   (A.25)-(A.26)
//   c_v(T) = S[1] + 2 S[2] T + ... + 5 S[5] T^4                           (A.29)-(A.31)
// with the low-range sums for T < t_mid and the high-range sums otherwise (G10), chosen
// again at every iterate.  Returns the number of iterations; *converged says whether the
// stop rule fired.
PYRO_HD int newton_temperature(const double *Slo, const double *Shi, double t_mid, double e, double T, double tol,
                               int max_iter, double *T_out, bool *converged) {
    int it = 0;
    bool conv = false;
    while (it < max_iter) {
        const bool low = T < t_mid;
        const double s0 = low ? Slo[0] : Shi[0], s1 = low ? Slo[1] : Shi[1], s2 = low ? Slo[2] : Shi[2],
                     s3 = low ? Slo[3] : Shi[3], s4 = low ? Slo[4] : Shi[4], s5 = low ? Slo[5] : Shi[5];
        double eT = fma(s5, T, s4);
        eT = fma(eT, T, s3);
        eT = fma(eT, T, s2);
        eT = fma(eT, T, s1);
        eT = fma(eT, T, s0);
        double cv = fma(5.0 * s5, T, 4.0 * s4);
        cv = fma(cv, T, 3.0 * s3);
        cv = fma(cv, T, 2.0 * s2);
        cv = fma(cv, T, s1);
        const double dT = -(eT - e) / cv;
        T += dT;
        ++it;
        if (fabs(dT) < tol) {
            conv = true;
            break;
        }
    }
    *T_out = T;
    *converged = conv;
    return it;
}

// The same solve for mechanisms whose species switch NASA range at different temperatures (G10: the
// range is chosen per species at every iterate).  The mixture polynomial S = sum_k Y_k c_k(range of k at T) is
// valid on the whole interval [t_below, t_above) between the two break temperatures that enclose T, so it
// is summed once (one pass over the species: `load_y(k)` and the energy row of k) and the Newton
// iteration continues on it at O(1) per step until an iterate leaves the interval; then the pass is
// repeated for the interval the iterate fell into.  Iterates, stop rule and count are those of
// newton_temperature.  `enthalpy`: S[1] += sum_k Y_k R/W_k (h = e + T R/W_mix).
template <class LoadY, class Row>
PYRO_HD int newton_temperature_general(int ns, const LoadY &load_y, const Row &row_of, bool enthalpy, double e, double T,
                                       double tol, int max_iter, double *T_out, bool *converged) {
    int it = 0;
    bool conv = false;
    while (it < max_iter && !conv) {
        double S[6] = {0.0, 0.0, 0.0, 0.0, 0.0, 0.0}, Rm = 0.0;
        double t_below = -1.0, t_above = 1.7976931348623157e308;
        auto add_species = [&](int k, double y) {
            const EnergyRow &r = row_of(k);
            const double tm = r.t_mid;
            const bool low = T < tm;
            const double *c = low ? r.lo : r.hi;
#pragma unroll
            for (int m = 0; m < 6; ++m) S[m] = fma(y, c[m], S[m]);
            Rm = fma(y, r.rw, Rm);
            t_above = low && tm < t_above ? tm : t_above;
            t_below = !low && tm > t_below ? tm : t_below;
        };
        int k = 0;
#pragma unroll 1
        for (; k + 4 <= ns; k += 4) {   // four mass fractions in flight: the pass is bound by the latency of these loads
            const double y0 = load_y(k), y1 = load_y(k + 1), y2 = load_y(k + 2), y3 = load_y(k + 3);
            add_species(k, y0);
            add_species(k + 1, y1);
            add_species(k + 2, y2);
            add_species(k + 3, y3);
        }
#pragma unroll 1
        for (; k < ns; ++k) add_species(k, load_y(k));
        if (enthalpy) S[1] += Rm;
        do {
            double eT = fma(S[5], T, S[4]);
            eT = fma(eT, T, S[3]);
            eT = fma(eT, T, S[2]);
            eT = fma(eT, T, S[1]);
            eT = fma(eT, T, S[0]);
            double cv = fma(5.0 * S[5], T, 4.0 * S[4]);
            cv = fma(cv, T, 3.0 * S[3]);
            cv = fma(cv, T, 2.0 * S[2]);
            cv = fma(cv, T, S[1]);
            const double dT = -(eT - e) / cv;
            T += dT;
            ++it;
            conv = fabs(dT) < tol;
        } while (!conv && it < max_iter && T >= t_below && T < t_above);   // NaN leaves the loop and the pass repeats until the cap
    }
    *T_out = T;
    *converged = conv;
    return it;
}

// n_steps classical Runge-Kutta steps of one adiabatic isochoric reactor (A.1) PAPER.md:886-888,
//     rho dY_k/dt = W_k omega_k(rho, T(e, Y), Y),     rho, e constant      (RK4 at a fixed step).
// The state stays where the rates path keeps it: a stage's mass fractions are written into plane A, the Newton solve
// of row a4 runs on them, fill_planes turns plane A into A_k = C_k E_k in place, accumulate_reactions leaves the
// stage's omega in plane W, and the next stage's first sweep reads it from there.  Only Y0 (the caller's Y, updated in
// place once per step) and the running sum of the weighted stage slopes (`acc`, a caller-provided scratch field)
// live in global memory, one coalesced access per species and stage.
//   y0_ld(k), y0_st(k, v)    mass fraction of species k at the start of the step (caller's Y)
//   acc_ld(k), acc_st(k, v)  dt/6 k1 + dt/3 k2 + dt/3 k3 so far
//   row_of(k)                energy row of species k (c_v polynomial, W_k, T_mid)
// Returns the number of Newton solves that hit the iteration cap; *T is the guess on entry and the temperature of
// the final state on return.
template <bool kSingles, class Tab, class Mem, class Y0Ld, class Y0St, class AccLd, class AccSt, class Row>
PYRO_HD int reactor_rk4_point(const Tab &tab, const GroupCounts &g, int ns, bool single_t_mid, double t_mid, double rho,
                              double e, double *T, double dt, int n_steps, double tol, int max_iter, const Mem &mem,
                              const Y0Ld &y0_ld, const Y0St &y0_st, const AccLd &acc_ld, const AccSt &acc_st, const Row &row_of) {
    const double inv_rho = 1.0 / rho;
    const double dt6 = dt / 6.0, dt3 = dt / 3.0, dth = dt / 2.0;
    double Tc = *T;
    int bad = 0;
    for (int step = 0; step <= n_steps; ++step) {
        const int n_stage = step < n_steps ? 4 : 1;   // after the last step: the final update and its temperature
#pragma unroll 1
        for (int s = 0; s < n_stage; ++s) {
            double Slo[6] = {0.0, 0.0, 0.0, 0.0, 0.0, 0.0}, Shi[6] = {0.0, 0.0, 0.0, 0.0, 0.0, 0.0};
            const bool have_slope = step > 0 || s > 0;   // plane W holds the omega of the stage before
            if (have_slope) mem.fence_st();
            // eight species at a time: their omega (tensor memory) and their two global values are requested
            // together, so the L2 latency of the state is paid once per batch
            constexpr int NB = 8;
            const bool need_acc = s != 1 && have_slope;
#pragma unroll 1
            for (int k = 0; k < ns; k += NB) {
                typename Mem::WRaw wr[NB];
                double y0v[NB], accv[NB];
                if (have_slope) {
#pragma unroll
                    for (int i = 0; i < NB; ++i) wr[i] = mem.ldW(mem.atW((uint32_t)(k + i < ns ? k + i : ns)));
                }
#pragma unroll
                for (int i = 0; i < NB; ++i) {
                    const int ki = k + i < ns ? k + i : ns - 1;
                    y0v[i] = y0_ld(ki);
                    accv[i] = need_acc ? acc_ld(ki) : 0.0;
                }
                if (have_slope) mem.fence_ld();
#pragma unroll
                for (int i = 0; i < NB; ++i) {
                    const int ki = k + i;
                    if (ki < ns) {
                        const EnergyRow &er = row_of(ki);
                        const double slope = have_slope ? mem.value(wr[i]) * (er.w * inv_rho) : 0.0;   // W_k omega_k / rho
                        double y0 = y0v[i], ys;
                        if (s == 0) {
                            if (have_slope) {   // Y1 = Y0 + dt/6 (k1 + 2 k2 + 2 k3 + k4)
                                y0 = y0 + fma(dt6, slope, accv[i]);
                                y0_st(ki, y0);
                            }
                            ys = y0;
                        } else if (s == 1) {
                            acc_st(ki, dt6 * slope);
                            ys = fma(dth, slope, y0);
                        } else {
                            acc_st(ki, fma(dt3, slope, accv[i]));
                            ys = fma(s == 2 ? dth : dt, slope, y0);
                        }
                        mem.stA(mem.atA((uint32_t)ki), ys);
                        if (single_t_mid) {
#pragma unroll
                            for (int m = 0; m < 6; ++m) {
                                Slo[m] = fma(ys, er.lo[m], Slo[m]);
                                Shi[m] = fma(ys, er.hi[m], Shi[m]);
                            }
                        }
                    }
                }
            }
            bool conv;
            if (single_t_mid)
                newton_temperature(Slo, Shi, t_mid, e, Tc, tol, max_iter, &Tc, &conv);
            else
                newton_temperature_general(
                    ns, [&](int q) { return mem.ldA(mem.atA((uint32_t)q)); }, row_of, false, e, Tc, tol, max_iter, &Tc, &conv);
            bad += conv ? 0 : 1;
            if (step == n_steps) break;
            const PointT pt = make_point(Tc);
            const double ctot = fill_planes(tab, ns, pt, rho, mem, [&](int q) { return mem.ldA(mem.atA((uint32_t)q)); });
            accumulate_reactions<kSingles>(tab, g, pt, ctot, mem);
        }
    }
    *T = Tc;
    return bad;
}

}   // namespace pyro
