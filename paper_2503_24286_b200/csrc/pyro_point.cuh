// Per-point arithmetic of the hot path, shared by every kernel variant.
//
// One thread owns P grid points.  Per-point arrays indexed by a run-time species number live
// on chip as three planes per species, each a column of P-vectors:
//     plane kA  A_k = C_k E_k      plane kB  B_k = 1/E_k      plane kW  omega_k
// with E_k = exp(g_k/RT) RT/p0 (pyro_tables.h).  The functions below reach them through a
// `Mem` accessor (shared memory in the kernels, a plain array in the host build):
//     h = mem.at(k)                  handle of species k for this thread
//     mem.template ld<Q>(h)          the thread's P-vector of plane Q
//     mem.template st<Q>(h, v)
#pragma once
#include "../../include/pyro.h"
#include "pyro_math.cuh"
#include "pyro_tables.h"

namespace pyro {

constexpr double kLog10of2 = 0.30102999566398119521;   // log10(2)
enum { kA = 0, kB = 1, kW = 2 };

template <int P> struct alignas(8 * P) Vec {
    double v[P];
};

// Per-thread temperature features of its P points.
template <int P> struct PointT {
    double T[P], invT[P], L2T[P];
};

template <int P> PYRO_HD PointT<P> make_point(const double (&T)[P]) {
    PointT<P> pt;
#pragma unroll
    for (int i = 0; i < P; ++i) {
        pt.T[i] = T[i];
        pt.invT[i] = 1.0 / T[i];
        pt.L2T[i] = log2(T[i]);
    }
    return pt;
}

// log2 k = c0 + c1 log2T + c2/T                               (A.9) PAPER.md:925
PYRO_HD double arrhenius_log2(double c0, double c1, double c2, double L2T, double invT) {
    return fma(c1, L2T, fma(c2, invT, c0));
}

// log2 E_k = c0 + c1 log2T + c2/T + c3 T + c4 T^2 + c5 T^3 + c6 T^4     (A.11)-(A.13) folded
PYRO_HD double species_log2E(const double (&c)[7], double T, double L2T, double invT) {
    double h = fma(c[6], T, c[5]);
    h = fma(h, T, c[4]);
    h = fma(h, T, c[3]);
    double y = fma(h, T, c[0]);
    y = fma(c[1], L2T, y);
    return fma(c[2], invT, y);
}

// Rows a2, a3 of SURVEY.md 8(a) for one species: C_k = rho Y_k / W_k (A.8) PAPER.md:921,
// the NASA range chosen per point (T < T_mid,k: low; G10), E_k and 1/E_k by one paired
// exponential.  Returns A_k = C_k E_k, B_k = 1/E_k and adds C_k to ctot.
template <int P>
PYRO_HD void species_planes(const SpecRow &row, const PointT<P> &pt, const double (&rho)[P], const double (&Y)[P],
                            double (&ctot)[P], Vec<P> &A, Vec<P> &B) {
    double y[P], e[P], b[P];
#pragma unroll
    for (int i = 0; i < P; ++i) {
        const bool low = pt.T[i] < row.t_mid;
        double c[7];
#pragma unroll
        for (int m = 0; m < 7; ++m) c[m] = low ? row.lo[m] : row.hi[m];
        y[i] = species_log2E(c, pt.T[i], pt.L2T[i], pt.invT[i]);
    }
    exp2_pair_n<P>(y, e, b);
#pragma unroll
    for (int i = 0; i < P; ++i) {
        const double C = rho[i] * Y[i] * row.inv_w;
        ctot[i] += C;
        A.v[i] = C * e[i];
        B.v[i] = b[i];
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

template <int P> PYRO_HD Vec<P> splat(double x) {
    Vec<P> v;
#pragma unroll
    for (int i = 0; i < P; ++i) v.v[i] = x;
    return v;
}

// Plain-class reactions of one shape (NR reactant molecules, NP product molecules), NB in
// lockstep (the packer stores groups of NB mutually species-disjoint reactions):
//   R = k_f prod_reac B_k [prod_reac A_k - prod_prod A_k]    (A.7), (A.10) as in pyro_tables.h
//   omega -= R on reactants, += R on products                (A.5)
// Branch-free.  The NB P exponentials run as interleaved Horner chains; all species touched in
// one iteration are distinct, so the omega read-modify-writes are one batch of loads, the
// adds, one batch of stores.
template <int P, int NR, int NP, int NB, class Tab, class Mem>
PYRO_HD void plain_reactions(const Tab &tab, int j0, int count, const PointT<P> &pt, const Mem &mem) {
    constexpr int NS = NR + NP;
#pragma unroll 1
    for (int j = j0; j < j0 + count; j += NB) {
        uint32_t h[NB][NS];
        double y[NB * P];
#pragma unroll
        for (int b = 0; b < NB; ++b) {
            const RxnP &r = tab.rxn_p(j + b);
            uint32_t slot[6];
            load_slots<NS>(r.slot, slot);
#pragma unroll
            for (int m = 0; m < NS; ++m) h[b][m] = mem.at(slot[m]);
            const double f0 = r.f[0], f1 = r.f[1], f2 = r.f[2];
#pragma unroll
            for (int i = 0; i < P; ++i) y[b * P + i] = arrhenius_log2(f0, f1, f2, pt.L2T[i], pt.invT[i]);
        }
        Vec<P> a[NB][NS], bb[NB][NR], w[NB][NS];
#pragma unroll
        for (int b = 0; b < NB; ++b)
#pragma unroll
            for (int m = 0; m < NS; ++m) {
                a[b][m] = mem.template ld<kA>(h[b][m]);
                if (m < NR) bb[b][m] = mem.template ld<kB>(h[b][m]);
                w[b][m] = mem.template ld<kW>(h[b][m]);
            }
        exp2_poly_n<NB * P>(y);
#pragma unroll
        for (int b = 0; b < NB; ++b) {
            double R[P];
#pragma unroll
            for (int i = 0; i < P; ++i) {
                double pf = a[b][0].v[i], pb = bb[b][0].v[i], pr = a[b][NR].v[i];
#pragma unroll
                for (int m = 1; m < NR; ++m) {
                    pf *= a[b][m].v[i];
                    pb *= bb[b][m].v[i];
                }
#pragma unroll
                for (int m = 1; m < NP; ++m) pr *= a[b][NR + m].v[i];
                R[i] = (y[b * P + i] * pb) * (pf - pr);
            }
#pragma unroll
            for (int m = 0; m < NS; ++m)
#pragma unroll
                for (int i = 0; i < P; ++i) w[b][m].v[i] = m < NR ? w[b][m].v[i] - R[i] : w[b][m].v[i] + R[i];
        }
#pragma unroll
        for (int b = 0; b < NB; ++b)
#pragma unroll
            for (int m = 0; m < NS; ++m) mem.template st<kW>(h[b][m], w[b][m]);
    }
}

template <int P, int NR, int NP, class Tab, class Mem>
PYRO_HD int plain_shape(const Tab &tab, int j, int quads, int pairs, int singles, const PointT<P> &pt,
                        const Mem &mem) {
    plain_reactions<P, NR, NP, 4>(tab, j, quads, pt, mem);
    plain_reactions<P, NR, NP, 2>(tab, j + quads, pairs, pt, mem);
    plain_reactions<P, NR, NP, 1>(tab, j + quads + pairs, singles, pt, mem);
    return j + quads + pairs + singles;
}

// Extended-class reactions of one kind: third body, falloff (Lindemann / Troe), and general
// elementary reactions (irreversible, repeated species).  Forms per reading G6-G8
// (PAPER.md:928 only cites them).  One reaction per iteration, its exponentials batched;
// slots and scatter entries are padded with the dummy species so there are no branches.
template <int P, int KIND, class Tab, class Mem>
PYRO_HD void extended_reactions(const Tab &tab, int j0, int count, const PointT<P> &pt, const double (&ctot)[P],
                                const Mem &mem) {
    constexpr int NE = KIND == kExtTroe ? 5 : (KIND == kExtLindemann ? 2 : 1);   // exponentials per point
#pragma unroll 1
    for (int j = j0; j < j0 + count; ++j) {
        const RxnX &x = tab.rxn_x(j);
        uint32_t h[6], hsc[6], slot[6], sc[6];
        double nu[6];
        load_slots<6>(x.slot, slot);
        load_slots<6>(x.sc_species, sc);
#pragma unroll
        for (int m = 0; m < 6; ++m) {
            h[m] = mem.at(slot[m]);
            hsc[m] = mem.at(sc[m]);
            nu[m] = x.sc_nu[m];
        }
        const bool reversible = x.rev != 0.0;
        double y[NE * P];
#pragma unroll
        for (int i = 0; i < P; ++i) y[i] = arrhenius_log2(x.f[0], x.f[1], x.f[2], pt.L2T[i], pt.invT[i]);
        double M[P];
#pragma unroll
        for (int i = 0; i < P; ++i) M[i] = 1.0;
        if (KIND != kExtGeneral) {
            // [M] = sum_k eff_k C_k = eff_default C_tot + sum_listed (eff_k - eff_default) C_k,  C_k = A_k B_k
#pragma unroll
            for (int i = 0; i < P; ++i) M[i] = x.eff_default * ctot[i];
            const int q0 = (int)x.eff_begin, q1 = q0 + (int)x.eff_count;
            for (int q = q0; q < q1; ++q) {
                const double d = tab.eff_delta(q);
                const uint32_t he = mem.at((uint32_t)tab.eff_species(q));
                const Vec<P> ak = mem.template ld<kA>(he), bk = mem.template ld<kB>(he);
#pragma unroll
                for (int i = 0; i < P; ++i) M[i] = fma(d, ak.v[i] * bk.v[i], M[i]);
            }
        }
        double alpha = 0.0, has_t2 = 0.0;
        if (KIND >= kExtLindemann) {
            const RxnFall &fl = tab.rxn_fall((int)x.fall_index);
#pragma unroll
            for (int i = 0; i < P; ++i)   // log2(k0 / k_inf)
                y[P + i] = arrhenius_log2(fl.l[0], fl.l[1], fl.l[2], pt.L2T[i], pt.invT[i]) - y[i];
            if (KIND == kExtTroe) {
                alpha = fl.troe_alpha;
                has_t2 = fl.troe_has_t2;
#pragma unroll
                for (int i = 0; i < P; ++i) {
                    y[2 * P + i] = fl.troe_t3 * pt.T[i];
                    y[3 * P + i] = fl.troe_t1 * pt.T[i];
                    y[4 * P + i] = fl.troe_t2 * pt.invT[i];
                }
            }
        }
        Vec<P> a[6], bb[3], w[6];
#pragma unroll
        for (int m = 0; m < 6; ++m) {
            a[m] = mem.template ld<kA>(h[m]);
            if (m < 3) bb[m] = mem.template ld<kB>(h[m]);
            w[m] = mem.template ld<kW>(hsc[m]);
        }
        exp2_poly_n<NE * P>(y);
        double fall[P];
#pragma unroll
        for (int i = 0; i < P; ++i) fall[i] = 1.0;
        if (KIND >= kExtLindemann) {
            double Pr[P];
#pragma unroll
            for (int i = 0; i < P; ++i) {
                Pr[i] = y[P + i] * M[i];              // Pr = k0 [M] / k_inf
                fall[i] = Pr[i] / (1.0 + Pr[i]);      // k = k_inf Pr/(1+Pr) F
            }
            if (KIND == kExtTroe) {
                double z[P];
#pragma unroll
                for (int i = 0; i < P; ++i) {
                    const double Fc = fma(1.0 - alpha, y[2 * P + i], fma(alpha, y[3 * P + i], has_t2 * y[4 * P + i]));
                    const double l2Fc = log2(Fc);
                    const double lFc = l2Fc * kLog10of2;
                    const double cc = -0.4 - 0.67 * lFc;
                    const double n = 0.75 - 1.27 * lFc;
                    const double lPr = log2(Pr[i]) * kLog10of2 + cc;
                    // F = Fcent^(1/(1+f1^2)), f1 = lPr/d, d = n - 0.14 lPr:  1/(1+f1^2) = d^2/(d^2 + lPr^2)
                    const double d = n - 0.14 * lPr;
                    const double d2 = d * d;
                    z[i] = l2Fc * (d2 / fma(lPr, lPr, d2));
                }
                exp2_poly_n<P>(z);
#pragma unroll
                for (int i = 0; i < P; ++i) fall[i] *= z[i];
            }
        }
        double R[P];
#pragma unroll
        for (int i = 0; i < P; ++i) {
            const double pf = a[0].v[i] * a[1].v[i] * a[2].v[i];
            const double pr = reversible ? a[3].v[i] * a[4].v[i] * a[5].v[i] : 0.0;
            const double pb = bb[0].v[i] * bb[1].v[i] * bb[2].v[i];
            R[i] = (y[i] * pb) * (pf - pr) * fall[i];
            if (KIND == kExtThreeBody) R[i] *= M[i];   // R = [M](q_f - q_r), reading G8
        }
#pragma unroll
        for (int m = 0; m < 6; ++m) {
#pragma unroll
            for (int i = 0; i < P; ++i) w[m].v[i] = fma(nu[m], R[i], w[m].v[i]);
            mem.template st<kW>(hsc[m], w[m]);
        }
    }
}

// Rows a5-a9 of SURVEY.md 8(a): rates of progress of every reaction and their stoichiometric
// accumulation into plane kW, (A.5)-(A.10) PAPER.md:908-934.  The planes hold n_species + 1
// entries: the last one is the dummy species (A = B = 1, omega = sink) that pads the
// extended records.
template <int P, class Tab, class Mem>
PYRO_HD void accumulate_reactions(const Tab &tab, const int (&quads)[9], const int (&pairs)[9],
                                  const int (&singles)[9], const int (&ext)[4], const PointT<P> &pt,
                                  const double (&ctot)[P], const Mem &mem) {
    int j = 0;
    j = plain_shape<P, 1, 1>(tab, j, quads[0], pairs[0], singles[0], pt, mem);
    j = plain_shape<P, 1, 2>(tab, j, quads[1], pairs[1], singles[1], pt, mem);
    j = plain_shape<P, 1, 3>(tab, j, quads[2], pairs[2], singles[2], pt, mem);
    j = plain_shape<P, 2, 1>(tab, j, quads[3], pairs[3], singles[3], pt, mem);
    j = plain_shape<P, 2, 2>(tab, j, quads[4], pairs[4], singles[4], pt, mem);
    j = plain_shape<P, 2, 3>(tab, j, quads[5], pairs[5], singles[5], pt, mem);
    j = plain_shape<P, 3, 1>(tab, j, quads[6], pairs[6], singles[6], pt, mem);
    j = plain_shape<P, 3, 2>(tab, j, quads[7], pairs[7], singles[7], pt, mem);
    j = plain_shape<P, 3, 3>(tab, j, quads[8], pairs[8], singles[8], pt, mem);
    int x = 0;
    extended_reactions<P, kExtGeneral>(tab, x, ext[0], pt, ctot, mem); x += ext[0];
    extended_reactions<P, kExtThreeBody>(tab, x, ext[1], pt, ctot, mem); x += ext[1];
    extended_reactions<P, kExtLindemann>(tab, x, ext[2], pt, ctot, mem); x += ext[2];
    extended_reactions<P, kExtTroe>(tab, x, ext[3], pt, ctot, mem);
}

// Rows a2, a3 for every species, then the dummy species (A = B = 1, omega = sink): fills the
// three planes.  `load_y(k, y)` fetches the thread's mass fractions of species k.
template <int P, class Tab, class Mem, class LoadY>
PYRO_HD void fill_planes(const Tab &tab, int ns, const PointT<P> &pt, const double (&rho)[P], double (&ctot)[P],
                         const Mem &mem, const LoadY &load_y) {
    const Vec<P> zero = splat<P>(0.0);
#pragma unroll 2
    for (int k = 0; k < ns; ++k) {
        double y[P];
        load_y(k, y);
        Vec<P> A, B;
        species_planes<P>(tab.spec(k), pt, rho, y, ctot, A, B);
        const uint32_t h = mem.at((uint32_t)k);
        mem.template st<kA>(h, A);
        mem.template st<kB>(h, B);
        mem.template st<kW>(h, zero);
    }
    const uint32_t h = mem.at((uint32_t)ns);
    mem.template st<kA>(h, splat<P>(1.0));
    mem.template st<kB>(h, splat<P>(1.0));
    mem.template st<kW>(h, zero);
}

// Plain array of kPlanes * (n_species + 1) P-vectors (host build, tests).
template <int P> struct ArrayMem {
    Vec<P> *s;
    PYRO_HD uint32_t at(uint32_t k) const { return k * kPlanes; }
    template <int Q> PYRO_HD Vec<P> ld(uint32_t h) const { return s[h + Q]; }
    template <int Q> PYRO_HD void st(uint32_t h, const Vec<P> &v) const { s[h + Q] = v; }
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

}   // namespace pyro
