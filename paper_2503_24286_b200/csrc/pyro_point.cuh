// Per-point arithmetic of the hot path, shared by every kernel variant.
//
// One thread owns P grid points.  Per-point arrays indexed by a run-time species number
// (concentrations C_k and production rates omega_k) live in the block's shared memory as
// columns: species k of the thread's points is the P-vector at sC[k * stride].  P = 2 makes
// every shared-memory access a 128-bit one, halves the warp-uniform table reads and the
// index arithmetic per point, and gives every thread two independent dependency chains.
#pragma once
#include "../../include/pyro.h"
#include "pyro_math.cuh"
#include "pyro_tables.h"

namespace pyro {

constexpr double kLog10of2 = 0.30102999566398119521;   // log10(2)

template <int P> struct alignas(8 * P) Vec {
    double v[P];
};

// Per-thread temperature features of its P points.
template <int P> struct PointT {
    double T[P], invT[P], L2T[P];
    bool low[P];   // T < T_mid: low NASA range (G10)
};

template <int P> PYRO_HD PointT<P> make_point(const double (&T)[P], double t_mid) {
    PointT<P> pt;
#pragma unroll
    for (int i = 0; i < P; ++i) {
        pt.T[i] = T[i];
        pt.invT[i] = 1.0 / T[i];
        pt.L2T[i] = log2(T[i]);
        pt.low[i] = T[i] < t_mid;
    }
    return pt;
}

// log2 k = c0 + c1 log2T + c2/T                               (A.9) PAPER.md:925
PYRO_HD double arrhenius_log2(double c0, double c1, double c2, double L2T, double invT) {
    return fma(c1, L2T, fma(c2, invT, c0));
}

// log2 k_r = c0 + c1 log2T + c2/T + c3 T + c4 T^2 + c5 T^3 + c6 T^4   (A.10)-(A.13) folded
PYRO_HD double reverse_log2(const double (&lo)[7], const double (&hi)[7], bool low, double T, double L2T,
                            double invT) {
    double h = fma(low ? lo[6] : hi[6], T, low ? lo[5] : hi[5]);
    h = fma(h, T, low ? lo[4] : hi[4]);
    h = fma(h, T, low ? lo[3] : hi[3]);
    double y = fma(h, T, low ? lo[0] : hi[0]);
    y = fma(low ? lo[1] : hi[1], L2T, y);
    return fma(low ? lo[2] : hi[2], invT, y);
}

// Register image of the rate part of one reaction record.
struct RateCoef {
    double f0, f1, f2;
    double lo[7], hi[7];
};

template <class Rec> PYRO_HD RateCoef load_rate(const Rec &r) {
    RateCoef c;
    c.f0 = r.f[0];
    c.f1 = r.f[1];
    c.f2 = r.f[2];
#pragma unroll
    for (int m = 0; m < 7; ++m) {
        c.lo[m] = r.rlo[m];
        c.hi[m] = r.rhi[m];
    }
    return c;
}

// Plain-class reactions of one shape (NR reactant molecules, NP product molecules), NB in
// lockstep (NB = 2 for the species-disjoint couples formed by the packer, 1 for the rest):
//   R = k_f prod C^nu' - k_r prod C^nu''   (A.7);  omega -= R on reactants, += R on products (A.5)
// Branch-free.  All 2 NB P exponentials run as interleaved Horner chains; all species touched
// in one iteration are distinct, so the omega read-modify-writes are one batch of loads, the
// adds, one batch of stores.
template <int P, int NR, int NP, int NB, class Tab>
PYRO_HD void plain_reactions(const Tab &tab, int j0, int count, const PointT<P> &pt, const Vec<P> *__restrict__ sC,
                             Vec<P> *__restrict__ sW, int stride) {
    constexpr int NS = NR + NP;
#pragma unroll 1
    for (int j = j0; j < j0 + count; j += NB) {
        int s[NB][NS];
        double y[NB * 2 * P];
#pragma unroll
        for (int b = 0; b < NB; ++b) {
            const RxnE &r = tab.rxn_e(j + b);
            const uint64_t w0 = r.sw[0], w1 = r.sw[1];
#pragma unroll
            for (int m = 0; m < NR; ++m) s[b][m] = slot_of(w0, w1, m) * stride;
#pragma unroll
            for (int m = 0; m < NP; ++m) s[b][NR + m] = slot_of(w0, w1, 3 + m) * stride;
            const RateCoef c = load_rate(r);
#pragma unroll
            for (int i = 0; i < P; ++i) {
                y[(2 * b) * P + i] = arrhenius_log2(c.f0, c.f1, c.f2, pt.L2T[i], pt.invT[i]);
                y[(2 * b + 1) * P + i] = reverse_log2(c.lo, c.hi, pt.low[i], pt.T[i], pt.L2T[i], pt.invT[i]);
            }
        }
        Vec<P> c[NB][NS], w[NB][NS];
#pragma unroll
        for (int b = 0; b < NB; ++b)
#pragma unroll
            for (int m = 0; m < NS; ++m) {
                c[b][m] = sC[s[b][m]];
                w[b][m] = sW[s[b][m]];
            }
        exp2_poly_n<NB * 2 * P>(y);
#pragma unroll
        for (int b = 0; b < NB; ++b) {
            double R[P];
#pragma unroll
            for (int i = 0; i < P; ++i) {
                double qf = y[(2 * b) * P + i] * c[b][0].v[i];
#pragma unroll
                for (int m = 1; m < NR; ++m) qf *= c[b][m].v[i];
                double qr = y[(2 * b + 1) * P + i] * c[b][NR].v[i];
#pragma unroll
                for (int m = 1; m < NP; ++m) qr *= c[b][NR + m].v[i];
                R[i] = qf - qr;
            }
#pragma unroll
            for (int m = 0; m < NS; ++m)
#pragma unroll
                for (int i = 0; i < P; ++i) w[b][m].v[i] = m < NR ? w[b][m].v[i] - R[i] : w[b][m].v[i] + R[i];
        }
#pragma unroll
        for (int b = 0; b < NB; ++b)
#pragma unroll
            for (int m = 0; m < NS; ++m) sW[s[b][m]] = w[b][m];
    }
}

template <int P, int NR, int NP, class Tab>
PYRO_HD int plain_shape(const Tab &tab, int j, int pairs, int singles, const PointT<P> &pt,
                        const Vec<P> *__restrict__ sC, Vec<P> *__restrict__ sW, int stride) {
    plain_reactions<P, NR, NP, 2>(tab, j, pairs, pt, sC, sW, stride);
    plain_reactions<P, NR, NP, 1>(tab, j + pairs, singles, pt, sC, sW, stride);
    return j + pairs + singles;
}

// Extended-class reactions of one kind: third body, falloff (Lindemann / Troe), and general
// elementary reactions (irreversible, repeated species).  Forms per reading G6-G8
// (PAPER.md:928 only cites them).  One reaction per iteration, its exponentials batched;
// slots and scatter entries are padded with the dummy species so there are no branches.
template <int P, int KIND, class Tab>
PYRO_HD void extended_reactions(const Tab &tab, int j0, int count, const PointT<P> &pt, const double (&ctot)[P],
                                const Vec<P> *__restrict__ sC, Vec<P> *__restrict__ sW, int stride) {
    constexpr int NE = KIND == kExtTroe ? 6 : (KIND == kExtLindemann ? 3 : 2);   // exponentials per point
#pragma unroll 1
    for (int j = j0; j < j0 + count; ++j) {
        const RxnX &x = tab.rxn_x(j);
        const uint64_t w0 = x.e.sw[0], w1 = x.e.sw[1];
        const double rev = reversible_of(w1) ? 1.0 : 0.0;
        int s[6], sc[6];
        double nu[6];
#pragma unroll
        for (int m = 0; m < 6; ++m) {
            s[m] = slot_of(w0, w1, m) * stride;
            sc[m] = x.sc_species[m] * stride;
            nu[m] = (double)x.sc_nu[m];
        }
        const RateCoef rc = load_rate(x.e);
        double y[NE * P];
#pragma unroll
        for (int i = 0; i < P; ++i) {
            y[i] = arrhenius_log2(rc.f0, rc.f1, rc.f2, pt.L2T[i], pt.invT[i]);
            y[P + i] = reverse_log2(rc.lo, rc.hi, pt.low[i], pt.T[i], pt.L2T[i], pt.invT[i]);
        }
        double M[P];
#pragma unroll
        for (int i = 0; i < P; ++i) M[i] = 1.0;
        if (KIND != kExtGeneral) {
            // [M] = sum_k eff_k C_k = eff_default C_tot + sum_listed (eff_k - eff_default) C_k
#pragma unroll
            for (int i = 0; i < P; ++i) M[i] = x.eff_default * ctot[i];
            const int q0 = (int)x.eff_begin, q1 = q0 + x.eff_count;
            for (int q = q0; q < q1; ++q) {
                const double d = tab.eff_delta(q);
                const Vec<P> c = sC[tab.eff_species(q) * stride];
#pragma unroll
                for (int i = 0; i < P; ++i) M[i] = fma(d, c.v[i], M[i]);
            }
        }
        double alpha = 0.0, has_t2 = 0.0;
        if (KIND >= kExtLindemann) {
            const RxnFall &fl = tab.rxn_fall(x.fall_index);
#pragma unroll
            for (int i = 0; i < P; ++i)   // log2(k0 / k_inf)
                y[2 * P + i] = arrhenius_log2(fl.l[0], fl.l[1], fl.l[2], pt.L2T[i], pt.invT[i]) - y[i];
            if (KIND == kExtTroe) {
                alpha = fl.troe_alpha;
                has_t2 = fl.troe_has_t2;
#pragma unroll
                for (int i = 0; i < P; ++i) {
                    y[3 * P + i] = fl.troe_t3 * pt.T[i];
                    y[4 * P + i] = fl.troe_t1 * pt.T[i];
                    y[5 * P + i] = fl.troe_t2 * pt.invT[i];
                }
            }
        }
        Vec<P> c[6], w[6];
#pragma unroll
        for (int m = 0; m < 6; ++m) {
            c[m] = sC[s[m]];
            w[m] = sW[sc[m]];
        }
        exp2_poly_n<NE * P>(y);
        double fall[P];
#pragma unroll
        for (int i = 0; i < P; ++i) fall[i] = 1.0;
        if (KIND >= kExtLindemann) {
            double Pr[P];
#pragma unroll
            for (int i = 0; i < P; ++i) {
                Pr[i] = y[2 * P + i] * M[i];          // Pr = k0 [M] / k_inf
                fall[i] = Pr[i] / (1.0 + Pr[i]);      // k = k_inf Pr/(1+Pr) F
            }
            if (KIND == kExtTroe) {
                double z[P], l2Fc[P];
#pragma unroll
                for (int i = 0; i < P; ++i) {
                    const double Fc = fma(1.0 - alpha, y[3 * P + i], fma(alpha, y[4 * P + i], has_t2 * y[5 * P + i]));
                    l2Fc[i] = log2(Fc);
                    const double lFc = l2Fc[i] * kLog10of2;
                    const double cc = -0.4 - 0.67 * lFc;
                    const double n = 0.75 - 1.27 * lFc;
                    const double lPr = log2(Pr[i]) * kLog10of2 + cc;
                    const double f1 = lPr / (n - 0.14 * lPr);
                    z[i] = l2Fc[i] / (1.0 + f1 * f1);
                }
                exp2_poly_n<P>(z);
#pragma unroll
                for (int i = 0; i < P; ++i) fall[i] *= z[i];
            }
        }
        double R[P];
#pragma unroll
        for (int i = 0; i < P; ++i) {
            const double qf = y[i] * c[0].v[i] * c[1].v[i] * c[2].v[i];
            const double qr = rev * y[P + i] * c[3].v[i] * c[4].v[i] * c[5].v[i];
            R[i] = (qf - qr) * fall[i];
            if (KIND == kExtThreeBody) R[i] *= M[i];   // R = [M](q_f - q_r), reading G8
        }
#pragma unroll
        for (int m = 0; m < 6; ++m) {
#pragma unroll
            for (int i = 0; i < P; ++i) w[m].v[i] = fma(nu[m], R[i], w[m].v[i]);
            sW[sc[m]] = w[m];
        }
    }
}

// Rows a5-a9 of SURVEY.md 8(a): rates of progress of every reaction and their stoichiometric
// accumulation into sW, (A.5)-(A.10) PAPER.md:908-934.  sC and sW hold n_species + 1 entries:
// the last one is the dummy species (C = 1, omega = sink) that pads the extended records.
template <int P, class Tab>
PYRO_HD void accumulate_reactions(const Tab &tab, const int (&pairs)[9], const int (&singles)[9], const int (&ext)[4],
                                  const PointT<P> &pt, const double (&ctot)[P], const Vec<P> *__restrict__ sC,
                                  Vec<P> *__restrict__ sW, int stride) {
    int j = 0;
    j = plain_shape<P, 1, 1>(tab, j, pairs[0], singles[0], pt, sC, sW, stride);
    j = plain_shape<P, 1, 2>(tab, j, pairs[1], singles[1], pt, sC, sW, stride);
    j = plain_shape<P, 1, 3>(tab, j, pairs[2], singles[2], pt, sC, sW, stride);
    j = plain_shape<P, 2, 1>(tab, j, pairs[3], singles[3], pt, sC, sW, stride);
    j = plain_shape<P, 2, 2>(tab, j, pairs[4], singles[4], pt, sC, sW, stride);
    j = plain_shape<P, 2, 3>(tab, j, pairs[5], singles[5], pt, sC, sW, stride);
    j = plain_shape<P, 3, 1>(tab, j, pairs[6], singles[6], pt, sC, sW, stride);
    j = plain_shape<P, 3, 2>(tab, j, pairs[7], singles[7], pt, sC, sW, stride);
    j = plain_shape<P, 3, 3>(tab, j, pairs[8], singles[8], pt, sC, sW, stride);
    int x = 0;
    extended_reactions<P, kExtGeneral>(tab, x, ext[0], pt, ctot, sC, sW, stride); x += ext[0];
    extended_reactions<P, kExtThreeBody>(tab, x, ext[1], pt, ctot, sC, sW, stride); x += ext[1];
    extended_reactions<P, kExtLindemann>(tab, x, ext[2], pt, ctot, sC, sW, stride); x += ext[2];
    extended_reactions<P, kExtTroe>(tab, x, ext[3], pt, ctot, sC, sW, stride);
}

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
