// Per-point arithmetic of the hot path, shared by every kernel variant.
// One thread owns one grid point; `sC` and `sW` are that thread's columns of the
// block's shared-memory arrays C[k][tid] and omega[k][tid] (element k at k*stride).
#pragma once
#include "../../include/pyro.h"
#include "pyro_math.cuh"
#include "pyro_tables.h"

namespace pyro {

constexpr double kLog10of2 = 0.30102999566398119521;   // log10(2)

// log2 k = c0 + c1 log2T + c2/T                               (A.9) PAPER.md:925
PYRO_HD double arrhenius_log2(const double *c, double L2T, double invT) {
    return fma(c[1], L2T, fma(c[2], invT, c[0]));
}

// log2 k_r = c0 + c1 log2T + c2/T + c3 T + c4 T^2 + c5 T^3 + c6 T^4   (A.10)-(A.13) folded
PYRO_HD double reverse_log2(const double *lo, const double *hi, bool low, double T, double L2T, double invT) {
    const double c6 = low ? lo[6] : hi[6], c5 = low ? lo[5] : hi[5], c4 = low ? lo[4] : hi[4],
                 c3 = low ? lo[3] : hi[3], c2 = low ? lo[2] : hi[2], c1 = low ? lo[1] : hi[1],
                 c0 = low ? lo[0] : hi[0];
    double h = fma(c6, T, c5);
    h = fma(h, T, c4);
    h = fma(h, T, c3);
    double y = fma(h, T, c0);
    y = fma(c1, L2T, y);
    return fma(c2, invT, y);
}

// Rates of progress of every reaction and their stoichiometric accumulation into sW
// (rows a5-a9 of SURVEY.md 8(a)): (A.5)-(A.10) PAPER.md:908-934; third-body and falloff
// forms per reading G6-G8 (PAPER.md:928 only cites them).
template <class Tab>
PYRO_HD void accumulate_reactions(const Tab &tab, int n_e, int n_x, double t_mid, double T, double ctot,
                                  const double *sC, double *sW, int stride) {
    const double invT = 1.0 / T;
    const double L2T = log2(T);
    const bool low = T < t_mid;

    // ---- plain class: R = k_f prod C^nu' - k_r prod C^nu''
#pragma unroll 2
    for (int j = 0; j < n_e; ++j) {
        const RxnE &r = tab.rxn_e(j);
        const int nreac = r.nreac, nprod = r.nprod;
        const int s0 = r.slot[0] * stride, s1 = r.slot[1] * stride, s2 = r.slot[2] * stride;
        const int p0 = r.slot[3] * stride, p1 = r.slot[4] * stride, p2 = r.slot[5] * stride;
        double qf = exp2_poly(arrhenius_log2(r.f, L2T, invT)) * sC[s0];
        if (nreac > 1) qf *= sC[s1];
        if (nreac > 2) qf *= sC[s2];
        double qr = 0.0;
        if (r.reversible) {
            qr = exp2_poly(reverse_log2(r.rlo, r.rhi, low, T, L2T, invT)) * sC[p0];
            if (nprod > 1) qr *= sC[p1];
            if (nprod > 2) qr *= sC[p2];
        }
        const double R = qf - qr;
        sW[s0] -= R;
        if (nreac > 1) sW[s1] -= R;
        if (nreac > 2) sW[s2] -= R;
        sW[p0] += R;
        if (nprod > 1) sW[p1] += R;
        if (nprod > 2) sW[p2] += R;
    }

    // ---- extended class: third body, falloff, species on both sides
    for (int j = 0; j < n_x; ++j) {
        const RxnX &x = tab.rxn_x(j);
        const RxnE &r = x.e;
        const int type = x.type;
        const double yf = arrhenius_log2(r.f, L2T, invT);
        double kf = exp2_poly(yf);
        double kr = 0.0;
        if (r.reversible) kr = exp2_poly(reverse_log2(r.rlo, r.rhi, low, T, L2T, invT));
        double M = 1.0;
        if (type != PYRO_ELEMENTARY) {
            M = x.eff_default * ctot;
            const int q0 = (int)x.eff_begin, q1 = q0 + x.eff_count;
            for (int q = q0; q < q1; ++q) M = fma(tab.eff_delta(q), sC[tab.eff_species(q) * stride], M);
        }
        if (type >= PYRO_FALLOFF_LINDEMANN) {
            // Pr = k0 [M] / k_inf;  k = k_inf Pr/(1+Pr) F
            const double Pr = exp2_poly(arrhenius_log2(x.l, L2T, invT) - yf) * M;
            double fall = Pr / (1.0 + Pr);
            if (type == PYRO_FALLOFF_TROE) {
                double Fc = (1.0 - x.troe_alpha) * exp2_poly(x.troe_t3 * T) + x.troe_alpha * exp2_poly(x.troe_t1 * T);
                if (x.troe_has_t2) Fc += exp2_poly(x.troe_t2 * invT);
                const double l2Fc = log2(Fc);
                const double lFc = l2Fc * kLog10of2;
                const double c = -0.4 - 0.67 * lFc;
                const double n = 0.75 - 1.27 * lFc;
                const double lPr = log2(Pr) * kLog10of2 + c;
                const double f1 = lPr / (n - 0.14 * lPr);
                fall *= exp2_poly(l2Fc / (1.0 + f1 * f1));
            }
            kf *= fall;
            kr *= fall;
        }
        const int nreac = r.nreac, nprod = r.nprod;
        double qf = kf * sC[r.slot[0] * stride];
        if (nreac > 1) qf *= sC[r.slot[1] * stride];
        if (nreac > 2) qf *= sC[r.slot[2] * stride];
        double qr = kr * sC[r.slot[3] * stride];
        if (nprod > 1) qr *= sC[r.slot[4] * stride];
        if (nprod > 2) qr *= sC[r.slot[5] * stride];
        double R = qf - qr;
        if (type == PYRO_THREE_BODY) R *= M;   // R = [M](q_f - q_r), reading G8
        const int nsc = x.n_scatter;
        for (int s = 0; s < nsc; ++s) {
            const int k = x.sc_species[s] * stride;
            sW[k] = fma(x.sc_coef[s], R, sW[k]);
        }
    }
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
