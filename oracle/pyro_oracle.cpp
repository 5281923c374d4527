// CPU ORACLE -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
//
// Plain, slow, scalar C++17 restatement of the thermochemistry of arXiv 2503.24286
// (Pyrometheus), Appendix A, point by point, in the order and notation of the paper.
// Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference
// legs may call it.  It shares no code, header, table or constant with the CUDA
// library (paper_2503_24286_b200/csrc); it has its own mechanism struct and is built
// with g++ -O2 -ffp-contract=off (no FMA contraction, no fast-math, no blocking or
// reordering).  The only concession to speed is `#pragma omp parallel for` over the
// independent points ("no loop-carried dependencies").
//
// Every function is instantiated for Real = double (the oracle proper) and
// Real = long double (80-bit; the arbiter of pin P14).
//
// What pins each function (tests/test_oracle_pins.py):
//   species_thermo      P1 continuity at T_mid, P2 c_p = dh/dT, P3 c_p/T = ds/dT, W2 g/RT values
//   mixture_e / cv      P4 c_v = de/dT, W4 closed form
//   get_temperature     P8 recovers generating T, W4 one-step convergence
//   rate coefficient    W1 (the Arrhenius triple printed at PAPER.md:205-208)
//   equilibrium const   W2 hand computation, P7 K_c(fwd) K_c(bwd) = 1, P6 detailed balance
//   third body/falloff  W3 hand computation, P9 [M] = p/RT, P10 Lindemann limits, P11 Troe -> Lindemann,
//                       W5 where [M] multiplies: q_f, q_r, omega of a three-body and of falloff reactions (G8)
//   production rates    P5 mass + element conservation, P12 scaling, P15 dense nu brute force, P16
//   mixture_h / cp      N1 h - e = R T sum_k Y_k/W_k, N2 c_p = dh/dT, N3 c_p - c_v = R sum_k Y_k/W_k
//   get_temperature_h   N4 recovers generating T, closed form for a constant-c_p species
//   density / pressure  N5 single species rho = p W/(R T), N6 p(rho(p)) = p, N7 sum_k C_k = p/(R T)
//   jacobian            J1 differences of the oracle's omega (long double), J2 closed forms (W6), J3 conservation
//                       per column, J4 the (rho, e) form through the Newton solve, J5 dS/dT by central differences
//   transport           X1 single species, X2 identical species, X3 the W7 fixture (50-digit evaluation), X4 binary
//                       D_1,m = W_2 D_12/W, X5 permutation of the species, X6 Wilke limits
//   reactor_rk4         R1 a step = degree-4 Taylor polynomial for a linear decay, R2 fourth order in dt, R3 mass and
//                       element conservation, R4 energy, R5 equilibrium is a fixed point
//   reactor_cn          C1 a step of a linear decay = y (1 - z/2)/(1 + z/2), C2 second order in dt, C3 conservation,
//                       C4 bounded where RK4 diverges
//   No function is "parity unpinned".
//
// Readings of garbled / silent passages are
// marked (Gn) where they are used.
//
// Units: SI with kmol.  R = 8314.46261815324 J/(kmol K), p0 = 101325 Pa (G5).

#include <cmath>
#include <cstdint>
#include <vector>
#ifdef _OPENMP
#include <omp.h>
#endif

extern "C" {
// The oracle's own description of a mechanism: borrowed host pointers.
struct oracle_mech {
    int32_t n_species, n_reactions;
    const double *mol_weight;            // [n_species] kg/kmol
    const double *nasa_lo, *nasa_hi;     // [n_species][7]  a1..a7
    const double *t_mid;                 // [n_species]
    const int32_t *reac_ptr, *reac_species, *reac_coeff;   // nu'  (CSR over reactions)
    const int32_t *prod_ptr, *prod_species, *prod_coeff;   // nu''
    const double *A, *b, *theta;         // [n_reactions]
    const uint8_t *type;                 // 0 elementary, 1 three-body, 2 Lindemann, 3 Troe
    const uint8_t *reversible;
    const double *eff_default;           // [n_reactions]
    const int32_t *eff_ptr, *eff_species;
    const double *eff_value;
    const double *A0, *b0, *theta0;      // low-pressure limit (type >= 2)
    const double *troe;                  // [n_reactions][4] alpha, T***, T*, T**
};
}

namespace {

template <class Real> struct Const {
    static constexpr Real R = Real(8314.46261815324L);   // J/(kmol K)            (G5)
    static constexpr Real p0 = Real(101325.0L);          // Pa, 1 atm
};

// NASA-7 polynomials of species k at temperature T.
//   (A.31; G3)  cp/R = a1 + a2 T + a3 T^2 + a4 T^3 + a5 T^4
//   (A.12)      h/RT = a1 + a2/2 T + a3/3 T^2 + a4/4 T^3 + a5/5 T^4 + a6/T
//   (A.13; G2)  s/R  = a1 ln T + a2 T + a3/2 T^2 + a4/3 T^3 + a5/4 T^4 + a7
//   (A.11)      g/RT = h/RT - s/R
// Range choice (G10): T < T_mid ? low : high.
template <class Real>
void species_thermo(const oracle_mech &m, int k, Real T, Real &cp_R, Real &h_RT, Real &s_R, Real &g_RT) {
    const double *c = (T < Real(m.t_mid[k])) ? (m.nasa_lo + 7 * k) : (m.nasa_hi + 7 * k);
    const Real a1 = c[0], a2 = c[1], a3 = c[2], a4 = c[3], a5 = c[4], a6 = c[5], a7 = c[6];
    const Real T2 = T * T, T3 = T2 * T, T4 = T3 * T;
    cp_R = a1 + a2 * T + a3 * T2 + a4 * T3 + a5 * T4;
    h_RT = a1 + a2 / Real(2) * T + a3 / Real(3) * T2 + a4 / Real(4) * T3 + a5 / Real(5) * T4 + a6 / T;
    s_R = a1 * std::log(T) + a2 * T + a3 / Real(2) * T2 + a4 / Real(3) * T3 + a5 / Real(4) * T4 + a7;
    g_RT = h_RT - s_R;
}

// (A.25), (A.26): e = sum_k Y_k e_k,  e_k = (h_k - R T)/W_k = (h_RT_k - 1) R T / W_k
template <class Real>
Real mixture_e(const oracle_mech &m, Real T, const Real *Y, int64_t ld) {
    Real e = 0;
    for (int k = 0; k < m.n_species; ++k) {
        Real cp_R, h_RT, s_R, g_RT;
        species_thermo<Real>(m, k, T, cp_R, h_RT, s_R, g_RT);
        e += Y[k * ld] * (h_RT - Real(1)) * Const<Real>::R * T / Real(m.mol_weight[k]);
    }
    return e;
}

// (A.29), (A.30) per unit mass (G4): c_v = sum_k Y_k (c_p,k - R)/W_k
template <class Real>
Real mixture_cv(const oracle_mech &m, Real T, const Real *Y, int64_t ld) {
    Real cv = 0;
    for (int k = 0; k < m.n_species; ++k) {
        Real cp_R, h_RT, s_R, g_RT;
        species_thermo<Real>(m, k, T, cp_R, h_RT, s_R, g_RT);
        cv += Y[k * ld] * (cp_R - Real(1)) * Const<Real>::R / Real(m.mol_weight[k]);
    }
    return cv;
}

// Enthalpy form ("minor modifications"; `do_energy=False` of listing 22, :674):
//   h = sum_k Y_k h_k,  h_k = h_RT_k R T / W_k  (J/kg; A.12 with PAPER.md:939),  c_p = sum_k Y_k c_p,k  (A.30)
template <class Real>
Real mixture_h(const oracle_mech &m, Real T, const Real *Y, int64_t ld) {
    Real h = 0;
    for (int k = 0; k < m.n_species; ++k) {
        Real cp_R, h_RT, s_R, g_RT;
        species_thermo<Real>(m, k, T, cp_R, h_RT, s_R, g_RT);
        h += Y[k * ld] * h_RT * Const<Real>::R * T / Real(m.mol_weight[k]);
    }
    return h;
}

template <class Real>
Real mixture_cp(const oracle_mech &m, Real T, const Real *Y, int64_t ld) {
    Real cp = 0;
    for (int k = 0; k < m.n_species; ++k) {
        Real cp_R, h_RT, s_R, g_RT;
        species_thermo<Real>(m, k, T, cp_R, h_RT, s_R, g_RT);
        cp += Y[k * ld] * cp_R * Const<Real>::R / Real(m.mol_weight[k]);
    }
    return cp;
}

// Ideal-gas equation of state (A.2), (A.3) PAPER.md:892-899:  p = rho R T / W,  W = (sum_k Y_k/W_k)^-1
template <class Real>
Real mean_molecular_weight(const oracle_mech &m, const Real *Y, int64_t ld) {
    Real s = 0;
    for (int k = 0; k < m.n_species; ++k) s += Y[k * ld] / Real(m.mol_weight[k]);
    return Real(1) / s;
}

template <class Real>
Real density_point(const oracle_mech &m, Real p, Real T, const Real *Y, int64_t ld) {
    return p * mean_molecular_weight<Real>(m, Y, ld) / (Const<Real>::R * T);
}

template <class Real>
Real pressure_point(const oracle_mech &m, Real rho, Real T, const Real *Y, int64_t ld) {
    return rho * Const<Real>::R * T / mean_molecular_weight<Real>(m, Y, ld);
}

// (A.27), (A.28); listing 22; per-point stop rule (G11):
// apply the update, then test |dT| < tol; cap max_iter; last iterate returned.
// `enthalpy`: the same iteration on h(T) = h with c_p in place of c_v.
template <class Real>
void get_temperature_point(const oracle_mech &m, Real e, const Real *Y, int64_t ld, Real T_guess, Real tol,
                           int max_iter, Real &T_out, int &iters, int &converged, bool enthalpy = false) {
    Real T = T_guess;
    iters = 0;
    converged = 0;
    for (int it = 1; it <= max_iter; ++it) {
        const Real dT = enthalpy ? -(mixture_h<Real>(m, T, Y, ld) - e) / mixture_cp<Real>(m, T, Y, ld)
                                 : -(mixture_e<Real>(m, T, Y, ld) - e) / mixture_cv<Real>(m, T, Y, ld);
        T = T + dT;
        iters = it;
        if (std::fabs(dT) < tol) {
            converged = 1;
            break;
        }
    }
    T_out = T;
}

// Everything the rate of one reaction is made of, for the pins.
template <class Real> struct ReactionDetail {
    Real kf;       // effective forward rate coefficient (after falloff)
    Real k_inf;    // A T^b exp(-theta/T)
    Real k0;       // low-pressure coefficient (falloff) else 0
    Real M;        // third-body concentration
    Real Pr;       // reduced pressure (falloff) else 0
    Real F;        // broadening factor (falloff) else 1
    Real Kc;       // equilibrium constant (reversible) else 0
    Real qf, qr;   // forward / reverse rates of progress (after the three-body factor)
};

// One reaction at one point, following SURVEY.md 8(c) "Oracle algorithm".
//   C[k]  molar concentrations (A.8),  g[k] = g_k/(R T) (A.11)
template <class Real>
ReactionDetail<Real> reaction_rate(const oracle_mech &m, int j, Real T, const Real *C, const Real *g) {
    ReactionDetail<Real> d{};
    // (A.9): k = A T^b exp(-theta/T)  -- literal form with pow (G13, G15)
    Real kf = Real(m.A[j]) * std::pow(T, Real(m.b[j])) * std::exp(-Real(m.theta[j]) / T);
    d.k_inf = kf;
    // third-body concentration [M] = sum_k eff_jk C_k, eff = default unless listed (G6)
    // (the listed efficiencies of a reaction may come in any order: plain search)
    Real M = 0;
    for (int k = 0; k < m.n_species; ++k) {
        Real eff = Real(m.eff_default[j]);
        for (int q = m.eff_ptr[j]; q < m.eff_ptr[j + 1]; ++q)
            if (m.eff_species[q] == k) eff = Real(m.eff_value[q]);
        M += eff * C[k];
    }
    d.M = M;
    d.F = 1;
    const int type = m.type[j];
    if (type >= 2) {   // falloff (G6-G9)
        const Real k0 = Real(m.A0[j]) * std::pow(T, Real(m.b0[j])) * std::exp(-Real(m.theta0[j]) / T);
        const Real Pr = k0 * M / kf;   // kf is k_inf here
        Real F = 1;                    // Lindemann
        if (type == 3) {               // Troe
            const Real alpha = m.troe[4 * j + 0], T3 = m.troe[4 * j + 1], T1 = m.troe[4 * j + 2],
                       T2 = m.troe[4 * j + 3];
            Real Fc = (Real(1) - alpha) * std::exp(-T / T3) + alpha * std::exp(-T / T1);
            if (std::isfinite(m.troe[4 * j + 3])) Fc += std::exp(-T2 / T);   // 4-parameter form (G7)
            const Real lFc = std::log10(Fc);
            const Real c = Real(-0.4L) - Real(0.67L) * lFc;
            const Real n = Real(0.75L) - Real(1.27L) * lFc;
            const Real lPr = std::log10(Pr) + c;
            const Real f1 = lPr / (n - Real(0.14L) * lPr);
            F = std::pow(Real(10), lFc / (Real(1) + f1 * f1));
        }
        d.k0 = k0;
        d.Pr = Pr;
        d.F = F;
        kf = kf * (Pr / (Real(1) + Pr)) * F;
    }
    d.kf = kf;
    // (A.7) forward: kf prod C^nu'   (integer powers by repeated multiplication, G16)
    Real qf = kf;
    for (int q = m.reac_ptr[j]; q < m.reac_ptr[j + 1]; ++q)
        for (int r = 0; r < m.reac_coeff[q]; ++r) qf *= C[m.reac_species[q]];
    Real qr = 0;
    if (m.reversible[j]) {
        // (A.10; G1): Kc = (p0/RT)^(sum nu) exp(-sum nu g/RT)
        int dnu = 0;
        Real dg = 0;
        for (int q = m.prod_ptr[j]; q < m.prod_ptr[j + 1]; ++q) {
            dnu += m.prod_coeff[q];
            dg += Real(m.prod_coeff[q]) * g[m.prod_species[q]];
        }
        for (int q = m.reac_ptr[j]; q < m.reac_ptr[j + 1]; ++q) {
            dnu -= m.reac_coeff[q];
            dg -= Real(m.reac_coeff[q]) * g[m.reac_species[q]];
        }
        const Real Kc = std::pow(Const<Real>::p0 / (Const<Real>::R * T), Real(dnu)) * std::exp(-dg);
        d.Kc = Kc;
        qr = kf / Kc;
        for (int q = m.prod_ptr[j]; q < m.prod_ptr[j + 1]; ++q)
            for (int r = 0; r < m.prod_coeff[q]; ++r) qr *= C[m.prod_species[q]];
    }
    if (type == 1) {   // three-body: R = [M](qf - qr)  (G8)
        qf *= M;
        qr *= M;
    }
    d.qf = qf;
    d.qr = qr;
    return d;
}

// omega_i = sum_j nu_ij R_j (A.5), nu = nu'' - nu' (A.6), summed in reaction order (G22);
// bound_i = sum_j |nu_ij| (|r_f,j| + |r_r,j|) is the scale of the parity tolerance (north_star).
template <class Real>
void production_rates_point(const oracle_mech &m, Real rho, Real T, const Real *Y, int64_t ld, Real *omega,
                            Real *bound, int64_t ldo, Real *rf_out, Real *rr_out, int64_t ldr) {
    const int ns = m.n_species, nr = m.n_reactions;
    std::vector<Real> C(ns), g(ns), nu(ns);
    for (int k = 0; k < ns; ++k) {
        C[k] = rho * Y[k * ld] / Real(m.mol_weight[k]);   // (A.8)
        Real cp_R, h_RT, s_R;
        species_thermo<Real>(m, k, T, cp_R, h_RT, s_R, g[k]);
        omega[k * ldo] = 0;
        if (bound) bound[k * ldo] = 0;
    }
    for (int j = 0; j < nr; ++j) {
        const ReactionDetail<Real> d = reaction_rate<Real>(m, j, T, C.data(), g.data());
        if (rf_out) rf_out[j * ldr] = d.qf;
        if (rr_out) rr_out[j * ldr] = d.qr;
        const Real Rj = d.qf - d.qr;   // (A.7)
        // net coefficients of this reaction
        for (int q = m.reac_ptr[j]; q < m.reac_ptr[j + 1]; ++q) nu[m.reac_species[q]] = 0;
        for (int q = m.prod_ptr[j]; q < m.prod_ptr[j + 1]; ++q) nu[m.prod_species[q]] = 0;
        for (int q = m.reac_ptr[j]; q < m.reac_ptr[j + 1]; ++q) nu[m.reac_species[q]] -= Real(m.reac_coeff[q]);
        for (int q = m.prod_ptr[j]; q < m.prod_ptr[j + 1]; ++q) nu[m.prod_species[q]] += Real(m.prod_coeff[q]);
        auto add = [&](int k) {
            if (nu[k] == Real(0)) return;
            omega[k * ldo] += nu[k] * Rj;
            if (bound) bound[k * ldo] += std::fabs(nu[k]) * (std::fabs(d.qf) + std::fabs(d.qr));
            nu[k] = 0;   // a species listed on both sides is visited once
        };
        for (int q = m.reac_ptr[j]; q < m.reac_ptr[j + 1]; ++q) add(m.reac_species[q]);
        for (int q = m.prod_ptr[j]; q < m.prod_ptr[j + 1]; ++q) add(m.prod_species[q]);
    }
}

template <class Real>
void get_net_production_rates(const oracle_mech &m, int64_t n, int64_t ld, const Real *rho, const Real *T,
                              const Real *Y, Real *omega, Real *bound, Real *rf, Real *rr) {
#pragma omp parallel for schedule(static)
    for (int64_t p = 0; p < n; ++p)
        production_rates_point<Real>(m, rho[p], T[p], Y + p, ld, omega + p, bound ? bound + p : nullptr, ld,
                                     rf ? rf + p : nullptr, rr ? rr + p : nullptr, ld);
}

template <class Real>
void get_temperature(const oracle_mech &m, int64_t n, int64_t ld, const Real *e, const Real *Y,
                     const Real *T_guess, Real tol, int max_iter, Real *T, int32_t *iters, int32_t *conv,
                     bool enthalpy = false) {
#pragma omp parallel for schedule(static)
    for (int64_t p = 0; p < n; ++p) {
        int it, cv;
        get_temperature_point<Real>(m, e[p], Y + p, ld, T_guess[p], tol, max_iter, T[p], it, cv, enthalpy);
        if (iters) iters[p] = it;
        if (conv) conv[p] = cv;
    }
}

// ---------------------------------------------------------------------------------------------------
// the chemical Jacobian, analytic.  PAPER.md:697-714 eq. (6) J = dS/dY with
// S_i = W_i omega_i (A.1) PAPER.md:888; (A.36) PAPER.md:1057.  Written out from (A.5)-(A.13) by the chain and
// product rules, reaction by reaction, dense in the species index (slow and plain on purpose).
//   C_k = rho Y_k / W_k (A.8): at fixed rho,  d/dY_k = (rho/W_k) d/dC_k ; the Y_k are independent variables
//   (no sum-to-one constraint is applied, as automatic differentiation of (A.5) would not apply one).
// Readings: G26 what is held fixed -- mode 0: (rho, T); mode 1: (rho, e), the paper's J: listing 23
// differentiates through the temperature inversion, i.e.  dT/dY_k|_e = -e_k(T)/c_v  from (A.25): 0 = e_k dY_k + c_v dT.
// Pins (tests/test_oracle_pins.py): J1 finite differences of this oracle's own omega in long double, error linear in
// delta for one-sided differences as in eq. (7) / fig. 8 and quadratic for central ones; J2 closed forms of the
// single reaction W2/W6 (dR/dC_A = k C_B); J3 mass and element conservation per column; J4 the
// (rho, e) form against differences through the oracle's own Newton solve; J5 dS/dT by central differences for
// every reaction type.
// Every derivative comes with the sum of the absolute values of the terms it is made of ("a..." twins); the
// harness scales the parity tolerance of the CUDA path with them, exactly as bound_i does for omega.
template <class Real> struct ReactionDerivative {
    std::vector<Real> dqf_dC, dqr_dC, aqf_dC, aqr_dC;   // [n_species]
    Real dqf_dT = 0, dqr_dT = 0, aqf_dT = 0, aqr_dT = 0;
};

template <class Real>
ReactionDerivative<Real> reaction_derivative(const oracle_mech &m, int j, Real T, const Real *C, const Real *g,
                                             const Real *h_RT) {
    const int ns = m.n_species;
    ReactionDerivative<Real> d;
    d.dqf_dC.assign(ns, Real(0)); d.dqr_dC.assign(ns, Real(0)); d.aqf_dC.assign(ns, Real(0)); d.aqr_dC.assign(ns, Real(0));
    const Real ln10 = std::log(Real(10));
    // (A.9): k = A T^b exp(-theta/T);  d ln k / dT = (b + theta/T)/T
    const Real kinf = Real(m.A[j]) * std::pow(T, Real(m.b[j])) * std::exp(-Real(m.theta[j]) / T);
    const Real dlnkinf_dT = (Real(m.b[j]) + Real(m.theta[j]) / T) / T;
    const Real a_dlnkinf_dT = (std::fabs(Real(m.b[j])) + std::fabs(Real(m.theta[j])) / T) / T;
    // [M] = sum_k eff_k C_k  (G6):  d[M]/dC_k = eff_k
    std::vector<Real> eff(ns);
    Real M = 0;
    for (int k = 0; k < ns; ++k) {
        eff[k] = Real(m.eff_default[j]);
        for (int q = m.eff_ptr[j]; q < m.eff_ptr[j + 1]; ++q)
            if (m.eff_species[q] == k) eff[k] = Real(m.eff_value[q]);
        M += eff[k] * C[k];
    }
    const int type = m.type[j];
    Real k = kinf, dlnk_dT = dlnkinf_dT, a_dlnk_dT = a_dlnkinf_dT, dlnk_dM = 0, a_dlnk_dM = 0;
    if (type >= 2) {   // falloff (G6-G8): k = k_inf L(Pr) F(T, Pr), L = Pr/(1+Pr), Pr = k0 [M]/k_inf
        const Real k0 = Real(m.A0[j]) * std::pow(T, Real(m.b0[j])) * std::exp(-Real(m.theta0[j]) / T);
        const Real dlnk0_dT = (Real(m.b0[j]) + Real(m.theta0[j]) / T) / T;
        const Real a_dlnk0_dT = (std::fabs(Real(m.b0[j])) + std::fabs(Real(m.theta0[j])) / T) / T;
        const Real Pr = k0 * M / kinf;
        const Real dlnPr_dT = dlnk0_dT - dlnkinf_dT;          // at fixed concentrations
        const Real a_dlnPr_dT = a_dlnk0_dT + a_dlnkinf_dT;
        const Real dlnL_dlnPr = Real(1) / (Real(1) + Pr);     // d ln[Pr/(1+Pr)] / d ln Pr
        Real F = 1, dlnF_dlnPr = 0, dlnF_dT = 0, a_dlnF_dT = 0;   // dlnF_dT: at fixed Pr
        if (type == 3) {
            const Real alpha = m.troe[4 * j + 0], T3 = m.troe[4 * j + 1], T1 = m.troe[4 * j + 2], T2 = m.troe[4 * j + 3];
            const Real e3 = std::exp(-T / T3), e1 = std::exp(-T / T1);
            const bool has2 = std::isfinite(m.troe[4 * j + 3]);
            const Real e2 = has2 ? std::exp(-T2 / T) : Real(0);
            const Real Fc = (Real(1) - alpha) * e3 + alpha * e1 + e2;
            const Real t3 = -(Real(1) - alpha) / T3 * e3, t1 = -alpha / T1 * e1, t2 = has2 ? T2 / (T * T) * e2 : Real(0);
            const Real dlFc_dT = (t3 + t1 + t2) / (Fc * ln10);             // lFc = log10 Fc
            const Real a_dlFc_dT = (std::fabs(t3) + std::fabs(t1) + std::fabs(t2)) / (std::fabs(Fc) * ln10);
            const Real lFc = std::log10(Fc);
            const Real c = Real(-0.4L) - Real(0.67L) * lFc;
            const Real n = Real(0.75L) - Real(1.27L) * lFc;
            const Real x = std::log10(Pr) + c;
            const Real den = n - Real(0.14L) * x;
            const Real f1 = x / den;
            const Real gg = Real(1) / (Real(1) + f1 * f1);                 // log10 F = lFc gg
            F = std::pow(Real(10), lFc * gg);
            const Real df1_dx = n / (den * den), df1_dn = -x / (den * den);
            const Real dgg_df1 = -Real(2) * f1 * gg * gg;
            // vary Pr at fixed T: dx/d ln Pr = 1/ln 10, so d ln F/d ln Pr = ln10 lFc dgg/df1 df1/dx / ln10
            dlnF_dlnPr = lFc * dgg_df1 * df1_dx;
            // vary T at fixed Pr: c and n move with lFc
            const Real dx_dT = -Real(0.67L) * dlFc_dT, dn_dT = -Real(1.27L) * dlFc_dT;
            dlnF_dT = ln10 * (dlFc_dT * gg + lFc * dgg_df1 * (df1_dx * dx_dT + df1_dn * dn_dT));
            a_dlnF_dT = ln10 * a_dlFc_dT *
                        (gg + std::fabs(lFc * dgg_df1) * (std::fabs(df1_dx) * Real(0.67L) + std::fabs(df1_dn) * Real(1.27L)));
        }
        k = kinf * (Pr / (Real(1) + Pr)) * F;
        dlnk_dT = dlnkinf_dT + (dlnL_dlnPr + dlnF_dlnPr) * dlnPr_dT + dlnF_dT;
        a_dlnk_dT = a_dlnkinf_dT + (std::fabs(dlnL_dlnPr) + std::fabs(dlnF_dlnPr)) * a_dlnPr_dT + a_dlnF_dT;
        dlnk_dM = (dlnL_dlnPr + dlnF_dlnPr) / M;              // d ln Pr / d[M] = 1/[M]
        a_dlnk_dM = (std::fabs(dlnL_dlnPr) + std::fabs(dlnF_dlnPr)) / std::fabs(M);
    }
    // dense nu', nu'' of this reaction
    std::vector<int> nup(ns, 0), nupp(ns, 0);
    for (int q = m.reac_ptr[j]; q < m.reac_ptr[j + 1]; ++q) nup[m.reac_species[q]] += m.reac_coeff[q];
    for (int q = m.prod_ptr[j]; q < m.prod_ptr[j + 1]; ++q) nupp[m.prod_species[q]] += m.prod_coeff[q];
    // P = prod_l C_l^nu_l  and  dP/dC_k = nu_k C_k^(nu_k - 1) prod_{l != k} C_l^nu_l   (no division: C_k may be 0)
    auto power_product = [&](const std::vector<int> &nu, int skip_one_of) {
        Real P = 1;
        for (int l = 0; l < ns; ++l)
            for (int r = 0; r < nu[l] - (l == skip_one_of ? 1 : 0); ++r) P *= C[l];
        return P;
    };
    const Real Pf = power_product(nup, -1);
    Real kr = 0, Pr_ = 0, dlnKc_dT = 0, a_dlnKc_dT = 0;
    if (m.reversible[j]) {
        int dnu = 0;
        Real dg = 0, dh = 0, adh = 0;
        for (int l = 0; l < ns; ++l) {
            const int nu = nupp[l] - nup[l];
            if (nu == 0) continue;
            dnu += nu;
            dg += Real(nu) * g[l];
            dh += Real(nu) * h_RT[l];
            adh += std::fabs(Real(nu) * h_RT[l]);
        }
        const Real Kc = std::pow(Const<Real>::p0 / (Const<Real>::R * T), Real(dnu)) * std::exp(-dg);   // (A.10; G1)
        kr = k / Kc;
        Pr_ = power_product(nupp, -1);
        // ln Kc = dnu ln(p0/RT) - sum nu g/RT, d(g/RT)/dT = -(h/RT)/T  (from (A.11)-(A.13)):
        dlnKc_dT = (-Real(dnu) + dh) / T;
        a_dlnKc_dT = (std::fabs(Real(dnu)) + adh) / T;
    }
    const Real qf0 = k * Pf, qr0 = kr * Pr_;
    const Real Mfac = (type == 1) ? M : Real(1);   // three-body: R = [M](qf0 - qr0)  (G8)
    for (int l = 0; l < ns; ++l) {
        const Real direct_f = nup[l] > 0 ? k * Real(nup[l]) * power_product(nup, l) : Real(0);
        const Real direct_r = (m.reversible[j] && nupp[l] > 0) ? kr * Real(nupp[l]) * power_product(nupp, l) : Real(0);
        const Real viaM_f = qf0 * dlnk_dM * eff[l], viaM_r = qr0 * dlnk_dM * eff[l];
        d.dqf_dC[l] = Mfac * (direct_f + viaM_f);
        d.dqr_dC[l] = Mfac * (direct_r + viaM_r);
        d.aqf_dC[l] = std::fabs(Mfac) * (std::fabs(direct_f) + std::fabs(qf0 * a_dlnk_dM * eff[l]));
        d.aqr_dC[l] = std::fabs(Mfac) * (std::fabs(direct_r) + std::fabs(qr0 * a_dlnk_dM * eff[l]));
        if (type == 1) {
            d.dqf_dC[l] += eff[l] * qf0;
            d.dqr_dC[l] += eff[l] * qr0;
            d.aqf_dC[l] += std::fabs(eff[l] * qf0);
            d.aqr_dC[l] += std::fabs(eff[l] * qr0);
        }
    }
    d.dqf_dT = Mfac * qf0 * dlnk_dT;
    d.dqr_dT = Mfac * qr0 * (dlnk_dT - dlnKc_dT);
    d.aqf_dT = std::fabs(Mfac * qf0) * a_dlnk_dT;
    d.aqr_dT = std::fabs(Mfac * qr0) * (a_dlnk_dT + a_dlnKc_dT);
    return d;
}

// One point.  J[(i n_s + k) ldj] = dS_i/dY_k, dSdT[i ldj] = dS_i/dT at fixed (rho, Y); the same shapes for the
// bounds.  mode 0: Y-derivatives at fixed (rho, T); mode 1: at fixed (rho, e)  (reading G26).
template <class Real>
void jacobian_point(const oracle_mech &m, Real rho, Real T, const Real *Y, int64_t ld, int mode, Real *J, Real *dSdT,
                    Real *boundJ, Real *bounddSdT, int64_t ldj) {
    const int ns = m.n_species, nr = m.n_reactions;
    std::vector<Real> C(ns), g(ns), h_RT(ns), cp_R(ns), Yv(ns);
    for (int k = 0; k < ns; ++k) {
        Yv[k] = Y[k * ld];
        C[k] = rho * Yv[k] / Real(m.mol_weight[k]);
        Real s_R;
        species_thermo<Real>(m, k, T, cp_R[k], h_RT[k], s_R, g[k]);
    }
    std::vector<Real> dwdC((size_t)ns * ns, Real(0)), adwdC((size_t)ns * ns, Real(0)), dwdT(ns, Real(0)), adwdT(ns, Real(0));
    for (int j = 0; j < nr; ++j) {
        const ReactionDerivative<Real> d = reaction_derivative<Real>(m, j, T, C.data(), g.data(), h_RT.data());
        std::vector<int> nu(ns, 0);
        for (int q = m.reac_ptr[j]; q < m.reac_ptr[j + 1]; ++q) nu[m.reac_species[q]] -= m.reac_coeff[q];
        for (int q = m.prod_ptr[j]; q < m.prod_ptr[j + 1]; ++q) nu[m.prod_species[q]] += m.prod_coeff[q];
        for (int i = 0; i < ns; ++i) {
            if (nu[i] == 0) continue;
            for (int k = 0; k < ns; ++k) {   // (A.5): d omega_i/dC_k = sum_j nu_ij (dqf_j/dC_k - dqr_j/dC_k)
                dwdC[(size_t)i * ns + k] += Real(nu[i]) * (d.dqf_dC[k] - d.dqr_dC[k]);
                adwdC[(size_t)i * ns + k] += std::fabs(Real(nu[i])) * (d.aqf_dC[k] + d.aqr_dC[k]);
            }
            dwdT[i] += Real(nu[i]) * (d.dqf_dT - d.dqr_dT);
            adwdT[i] += std::fabs(Real(nu[i])) * (d.aqf_dT + d.aqr_dT);
        }
    }
    Real cv = 0;
    if (mode == 1) cv = mixture_cv<Real>(m, T, Yv.data(), 1);
    for (int i = 0; i < ns; ++i) {
        const Real Wi = Real(m.mol_weight[i]);
        const Real sT = Wi * dwdT[i], asT = Wi * adwdT[i];
        if (dSdT) dSdT[i * ldj] = sT;
        if (bounddSdT) bounddSdT[i * ldj] = asT;
        for (int k = 0; k < ns; ++k) {
            const Real scale = Wi * rho / Real(m.mol_weight[k]);
            Real v = scale * dwdC[(size_t)i * ns + k], a = scale * adwdC[(size_t)i * ns + k];
            if (mode == 1) {   // + dS_i/dT dT/dY_k|_e,  dT/dY_k|_e = -e_k/c_v,  e_k = (h_RT_k - 1) R T / W_k  (A.26)
                const Real ek = (h_RT[k] - Real(1)) * Const<Real>::R * T / Real(m.mol_weight[k]);
                v -= sT * ek / cv;
                a += std::fabs(asT * ek / cv);
            }
            J[((size_t)i * ns + k) * ldj] = v;
            if (boundJ) boundJ[((size_t)i * ns + k) * ldj] = a;
        }
    }
}

template <class Real>
void get_jacobian(const oracle_mech &m, int64_t n, int64_t ld, const Real *rho, const Real *T, const Real *Y, int mode,
                  Real *J, Real *dSdT, Real *boundJ, Real *bounddSdT) {
#pragma omp parallel for schedule(static)
    for (int64_t p = 0; p < n; ++p)
        jacobian_point<Real>(m, rho[p], T[p], Y + p, ld, mode, J + p, dSdT ? dSdT + p : nullptr,
                             boundJ ? boundJ + p : nullptr, bounddSdT ? bounddSdT + p : nullptr, ld);
}

// ---------------------------------------------------------------------------------------------------
// homogeneous adiabatic isochoric reactors (A.1) PAPER.md:886-888,
//     rho dY_k/dt = W_k omega_k(rho, T, Y),   rho and e constant,   T from (e, Y) by the Newton inversion (A.25)-(A.28),
// marched with the classical fourth-order Runge-Kutta scheme at a fixed step ("standard fourth-order
// accurate explicit Runge-Kutta ... a time step of 10 ns").  Written out stage by stage:
//     k1 = f(Y0), k2 = f(Y0 + dt/2 k1), k3 = f(Y0 + dt/2 k2), k4 = f(Y0 + dt k3),  Y1 = Y0 + dt/6 (k1 + 2 k2 + 2 k3 + k4),
//     f_k(Y) = W_k omega_k(rho, T(e, Y), Y) / rho.
// Readings (G27): every stage inverts the temperature from the stage's mass fractions, starting the Newton
// iteration from the temperature of the stage before (stop rule G11); mass fractions are neither clipped nor
// renormalised (G17); the temperature returned is that of the final state.
// Ybound_k accumulates the sizes of the terms that were added into Y_k (dt/6 (B1 + 2 B2 + 2 B3 + B4) W_k/rho with B the
// bound_i of (A.5)): the scale of the parity tolerance.
// Pins (tests/test_oracle_reactor_pins.py): R1 one irreversible reaction with constant rate coefficient: a step is
// the degree-4 Taylor polynomial of exp(-k dt) exactly; R2 fourth-order convergence in dt; R3 mass and element
// conservation; R4 energy: e(T_final, Y_final) = e; R5 a steady state (equilibrium composition) stays put.
template <class Real>
void reactor_rk4_point(const oracle_mech &m, Real rho, Real e, Real *Y, int64_t ld, Real &T, Real dt, int n_steps, Real tol,
                       int max_iter, Real *Ybound, int64_t ldb, int &not_converged) {
    const int ns = m.n_species;
    std::vector<Real> Y0(ns), Ys(ns), om(ns), bd(ns), k1(ns), k2(ns), k3(ns), k4(ns), B(ns);
    not_converged = 0;
    auto f = [&](const std::vector<Real> &y, std::vector<Real> &k, Real weight) {
        int it, cv;
        Real Tn;
        get_temperature_point<Real>(m, e, y.data(), 1, T, tol, max_iter, Tn, it, cv);
        if (!cv) ++not_converged;
        T = Tn;
        production_rates_point<Real>(m, rho, T, y.data(), 1, om.data(), bd.data(), 1, nullptr, nullptr, 1);
        for (int i = 0; i < ns; ++i) {
            k[i] = Real(m.mol_weight[i]) * om[i] / rho;
            B[i] += weight * Real(m.mol_weight[i]) * bd[i] / rho;
        }
    };
    for (int i = 0; i < ns; ++i) {
        Y0[i] = Y[i * ld];
        if (Ybound) Ybound[i * ldb] = 0;
    }
    for (int step = 0; step < n_steps; ++step) {
        for (int i = 0; i < ns; ++i) B[i] = 0;
        f(Y0, k1, Real(1));
        for (int i = 0; i < ns; ++i) Ys[i] = Y0[i] + dt / Real(2) * k1[i];
        f(Ys, k2, Real(2));
        for (int i = 0; i < ns; ++i) Ys[i] = Y0[i] + dt / Real(2) * k2[i];
        f(Ys, k3, Real(2));
        for (int i = 0; i < ns; ++i) Ys[i] = Y0[i] + dt * k3[i];
        f(Ys, k4, Real(1));
        for (int i = 0; i < ns; ++i) {
            Y0[i] = Y0[i] + dt / Real(6) * (k1[i] + Real(2) * k2[i] + Real(2) * k3[i] + k4[i]);
            if (Ybound) Ybound[i * ldb] += dt / Real(6) * B[i];
        }
    }
    {   // temperature of the final state
        int it, cv;
        Real Tn;
        get_temperature_point<Real>(m, e, Y0.data(), 1, T, tol, max_iter, Tn, it, cv);
        if (!cv) ++not_converged;
        T = Tn;
    }
    for (int i = 0; i < ns; ++i) Y[i * ld] = Y0[i];
}

template <class Real>
void reactor_rk4(const oracle_mech &m, int64_t n, int64_t ld, const Real *rho, const Real *e, Real *Y, Real *T, Real dt,
                 int n_steps, Real tol, int max_iter, Real *Ybound, int64_t *n_not_converged) {
    int64_t bad = 0;
#pragma omp parallel for schedule(static) reduction(+ : bad)
    for (int64_t p = 0; p < n; ++p) {
        int nc;
        reactor_rk4_point<Real>(m, rho[p], e[p], Y + p, ld, T[p], dt, n_steps, tol, max_iter, Ybound ? Ybound + p : nullptr, ld, nc);
        bad += nc;
    }
    if (n_not_converged) *n_not_converged = bad;
}

// ---------------------------------------------------------------------------------------------------
// mixture-averaged transport properties, Appendix A.2, as printed:
//   X_k = W Y_k / W_k,  W = (sum_i Y_i/W_i)^-1                                              (A.3)
//   mu_k    = sqrt(T) [sum_{m=0..4} b_km (ln T)^m]^2                                         (A.22)
//   Phi_kj  = [1 + sqrt((mu_k/mu_j) sqrt(W_j/W_k))]^2 / sqrt(8 (1 + W_k/W_j))                (A.21)
//   mu      = sum_k X_k mu_k / sum_j Phi_kj X_j                                              (A.20)
//   kappa_k = sqrt(T) sum_m c_km (ln T)^m                                                    (A.24)
//   kappa   = 1/2 [sum_k X_k kappa_k + (sum_k X_k/kappa_k)^-1]                               (A.23)
//   D_kj    = sqrt(T) sum_m a_kjm (ln T)^m                                                   (A.19)
//   D_k,m   = (W - X_k W_k)/W (sum_{j != k} X_j/D_kj)^-1                                     (A.18)
// Readings: G28 the binary diffusivities are taken exactly as (A.19) prints them (sqrt(T) times the
// polynomial, no pressure factor: the fits are the caller's, at the caller's pressure); G29 (A.18) is singular for a
// pure species (0/0): left as printed, a mixture of at least two species is a documented precondition; G30 the
// polynomial is evaluated by Horner's rule in ln T.
// Pins (tests/test_oracle_transport_pins.py): X1 a single species returns its own mu_k, kappa_k; X2 identical species
// mix to the species value at any composition; X3 the W7 fixture (50-digit mpmath evaluation of a three-species
// mixture); X4 binary mixture D_1,m = W_2 D_12 / W; X5 permuting the species permutes the result; X6 Wilke's
// identity Phi_jk = (mu_j/mu_k)(W_k/W_j) Phi_kj through the mixture formula (equal-mass, equal-viscosity limits).
extern "C" {
struct oracle_transport {
    int32_t n_species;
    const double *mol_weight;   // [n_species]
    const double *visc;         // [n_species][5]  b_km
    const double *cond;         // [n_species][5]  c_km
    const double *diff;         // [n_species][n_species][5]  a_kjm
};
}

template <class Real> Real poly4(const double *c, Real x) {   // sum_{m=0..4} c_m x^m, Horner (G30)
    Real p = Real(c[4]);
    for (int m = 3; m >= 0; --m) p = p * x + Real(c[m]);
    return p;
}

template <class Real>
void transport_point(const oracle_transport &t, Real T, const Real *Y, int64_t ld, Real &mu, Real &kappa, Real *Dkm,
                     int64_t ldd) {
    const int ns = t.n_species;
    const Real lnT = std::log(T), sqT = std::sqrt(T);
    std::vector<Real> X(ns), muk(ns), kak(ns);
    Real s = 0;
    for (int k = 0; k < ns; ++k) s += Y[k * ld] / Real(t.mol_weight[k]);
    const Real W = Real(1) / s;                                                   // (A.3)
    for (int k = 0; k < ns; ++k) {
        X[k] = W * Y[k * ld] / Real(t.mol_weight[k]);
        const Real pb = poly4<Real>(t.visc + 5 * k, lnT);
        muk[k] = sqT * pb * pb;                                                   // (A.22)
        kak[k] = sqT * poly4<Real>(t.cond + 5 * k, lnT);                          // (A.24)
    }
    mu = 0;
    for (int k = 0; k < ns; ++k) {
        Real den = 0;
        for (int j = 0; j < ns; ++j) {
            const Real Wk = t.mol_weight[k], Wj = t.mol_weight[j];
            const Real a = Real(1) + std::sqrt(muk[k] / muk[j] * std::sqrt(Wj / Wk));
            den += a * a / std::sqrt(Real(8) * (Real(1) + Wk / Wj)) * X[j];       // (A.21)
        }
        mu += X[k] * muk[k] / den;                                                // (A.20)
    }
    Real s1 = 0, s2 = 0;
    for (int k = 0; k < ns; ++k) {
        s1 += X[k] * kak[k];
        s2 += X[k] / kak[k];
    }
    kappa = (s1 + Real(1) / s2) / Real(2);                                        // (A.23)
    for (int k = 0; k < ns; ++k) {
        Real sum = 0;
        for (int j = 0; j < ns; ++j) {
            if (j == k) continue;
            sum += X[j] / (sqT * poly4<Real>(t.diff + 5 * ((size_t)k * ns + j), lnT));   // (A.19)
        }
        Dkm[k * ldd] = (W - X[k] * Real(t.mol_weight[k])) / W / sum;              // (A.18)
    }
}

template <class Real>
void get_transport(const oracle_transport &t, int64_t n, int64_t ld, const Real *T, const Real *Y, Real *mu, Real *kappa,
                   Real *Dkm) {
#pragma omp parallel for schedule(static)
    for (int64_t p = 0; p < n; ++p) transport_point<Real>(t, T[p], Y + p, ld, mu[p], kappa[p], Dkm + p, ld);
}

// Implicit march of the same reactors with the Crank-Nicolson scheme of Appendix A.3.2:
//     F_k = Y_k^{m+1} - Y_k^m - dt/2 (s_k^{m+1} + s_k^m) = 0,   s_k = W_k omega_k / rho  (the right-hand side of (A.1)),   (A.32)
// solved per step by Newton iterations (A.33)-(A.35) started from Y^m:
//     (delta_jk - dt/2 ds_j/dY_k) dY_k = -F_j,    Y <- Y + dY,
// with the chemical Jacobian (A.36) at fixed (rho, e) (reading G26: ds_j/dY_k = J_jk / rho of jacobian_point, mode 1).
// Readings (G31): a fixed number of Newton iterations per step (data-independent control flow, as the paper's
// JAX version needs); the temperature is re-inverted from (e, Y) before every evaluation of omega
// and J, starting from the last temperature; the linear system is solved by Gaussian elimination with partial
// pivoting; the size of the last Newton update max_k |dY_k| is returned per point.
// Pins (tests/test_oracle_reactor_pins.py): C1 linear decay: a step is y (1 - z/2)/(1 + z/2) exactly, after one Newton
// iteration; C2 second-order convergence in dt; C3 mass and element conservation; C4 bounded at dt where RK4 diverges.
template <class Real>
void solve_dense(int n, std::vector<Real> &A, std::vector<Real> &b) {   // A x = b, partial pivoting; x returned in b
    for (int c = 0; c < n; ++c) {
        int piv = c;
        for (int r = c + 1; r < n; ++r)
            if (std::fabs(A[(size_t)r * n + c]) > std::fabs(A[(size_t)piv * n + c])) piv = r;
        if (piv != c) {
            for (int j = 0; j < n; ++j) std::swap(A[(size_t)c * n + j], A[(size_t)piv * n + j]);
            std::swap(b[c], b[piv]);
        }
        for (int r = c + 1; r < n; ++r) {
            const Real f = A[(size_t)r * n + c] / A[(size_t)c * n + c];
            for (int j = c; j < n; ++j) A[(size_t)r * n + j] -= f * A[(size_t)c * n + j];
            b[r] -= f * b[c];
        }
    }
    for (int r = n - 1; r >= 0; --r) {
        Real s = b[r];
        for (int j = r + 1; j < n; ++j) s -= A[(size_t)r * n + j] * b[j];
        b[r] = s / A[(size_t)r * n + r];
    }
}

template <class Real>
void reactor_cn_point(const oracle_mech &m, Real rho, Real e, Real *Y, int64_t ld, Real &T, Real dt, int n_steps,
                      int newton_iters, Real tol, int max_iter, Real *Ybound, int64_t ldb, Real &last_update, int &not_converged) {
    const int ns = m.n_species;
    std::vector<Real> Ym(ns), Yn(ns), sm(ns), om(ns), bd(ns), bdm(ns), J((size_t)ns * ns), A((size_t)ns * ns), F(ns);
    not_converged = 0;
    last_update = 0;
    auto rates = [&](const std::vector<Real> &y, std::vector<Real> &w, std::vector<Real> &b) {
        int it, cv;
        Real Tn;
        get_temperature_point<Real>(m, e, y.data(), 1, T, tol, max_iter, Tn, it, cv);
        if (!cv) ++not_converged;
        T = Tn;
        production_rates_point<Real>(m, rho, T, y.data(), 1, w.data(), b.data(), 1, nullptr, nullptr, 1);
    };
    for (int i = 0; i < ns; ++i) {
        Yn[i] = Y[i * ld];
        if (Ybound) Ybound[i * ldb] = 0;
    }
    rates(Yn, om, bd);
    for (int step = 0; step < n_steps; ++step) {
        for (int i = 0; i < ns; ++i) {
            Ym[i] = Yn[i];
            sm[i] = Real(m.mol_weight[i]) * om[i] / rho;
            bdm[i] = bd[i];
        }
        for (int it = 0; it < newton_iters; ++it) {
            jacobian_point<Real>(m, rho, T, Yn.data(), 1, 1, J.data(), nullptr, nullptr, nullptr, 1);
            for (int i = 0; i < ns; ++i) {
                F[i] = -(Yn[i] - Ym[i] - dt / Real(2) * (Real(m.mol_weight[i]) * om[i] / rho + sm[i]));      // (A.32)
                for (int k = 0; k < ns; ++k)
                    A[(size_t)i * ns + k] = (i == k ? Real(1) : Real(0)) - dt / Real(2) * J[(size_t)i * ns + k] / rho;   // (A.35)
            }
            solve_dense<Real>(ns, A, F);                                                                      // (A.34)
            last_update = 0;
            for (int i = 0; i < ns; ++i) {
                Yn[i] += F[i];                                                                                 // (A.33)
                last_update = std::fmax(last_update, std::fabs(F[i]));
            }
            rates(Yn, om, bd);
        }
        if (Ybound)
            for (int i = 0; i < ns; ++i) Ybound[i * ldb] += dt / Real(2) * Real(m.mol_weight[i]) * (bd[i] + bdm[i]) / rho;
    }
    for (int i = 0; i < ns; ++i) Y[i * ld] = Yn[i];
}

template <class Real>
void reactor_cn(const oracle_mech &m, int64_t n, int64_t ld, const Real *rho, const Real *e, Real *Y, Real *T, Real dt,
                int n_steps, int newton_iters, Real tol, int max_iter, Real *Ybound, Real *last_update, int64_t *n_not_converged) {
    int64_t bad = 0;
#pragma omp parallel for schedule(static) reduction(+ : bad)
    for (int64_t p = 0; p < n; ++p) {
        int nc;
        Real lu;
        reactor_cn_point<Real>(m, rho[p], e[p], Y + p, ld, T[p], dt, n_steps, newton_iters, tol, max_iter,
                               Ybound ? Ybound + p : nullptr, ld, lu, nc);
        if (last_update) last_update[p] = lu;
        bad += nc;
    }
    if (n_not_converged) *n_not_converged = bad;
}

template <class Real>
void reaction_detail(const oracle_mech &m, int j, Real rho, Real T, const Real *Y, Real *out9) {
    const int ns = m.n_species;
    std::vector<Real> C(ns), g(ns);
    for (int k = 0; k < ns; ++k) {
        C[k] = rho * Y[k] / Real(m.mol_weight[k]);
        Real cp_R, h_RT, s_R;
        species_thermo<Real>(m, k, T, cp_R, h_RT, s_R, g[k]);
    }
    const ReactionDetail<Real> d = reaction_rate<Real>(m, j, T, C.data(), g.data());
    out9[0] = d.kf; out9[1] = d.k_inf; out9[2] = d.k0; out9[3] = d.M; out9[4] = d.Pr;
    out9[5] = d.F; out9[6] = d.Kc; out9[7] = d.qf; out9[8] = d.qr;
}

}   // namespace

extern "C" {

int oracle_num_threads() {
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}
void oracle_set_num_threads(int n) {
#ifdef _OPENMP
    omp_set_num_threads(n);
#else
    (void)n;
#endif
}
int oracle_sizeof_real80() { return (int)sizeof(long double); }

#define ORACLE_API(SUFFIX, Real)                                                                              \
    void oracle_species_thermo_##SUFFIX(const oracle_mech *m, int k, Real T, Real *out4) {                    \
        species_thermo<Real>(*m, k, T, out4[0], out4[1], out4[2], out4[3]);                                   \
    }                                                                                                         \
    Real oracle_mixture_e_##SUFFIX(const oracle_mech *m, Real T, const Real *Y) {                             \
        return mixture_e<Real>(*m, T, Y, 1);                                                                  \
    }                                                                                                         \
    Real oracle_mixture_cv_##SUFFIX(const oracle_mech *m, Real T, const Real *Y) {                            \
        return mixture_cv<Real>(*m, T, Y, 1);                                                                 \
    }                                                                                                         \
    void oracle_reaction_detail_##SUFFIX(const oracle_mech *m, int j, Real rho, Real T, const Real *Y,        \
                                         Real *out9) {                                                        \
        reaction_detail<Real>(*m, j, rho, T, Y, out9);                                                        \
    }                                                                                                         \
    void oracle_get_temperature_##SUFFIX(const oracle_mech *m, int64_t n, int64_t ld, const Real *e,          \
                                         const Real *Y, const Real *T_guess, Real tol, int max_iter, Real *T, \
                                         int32_t *iters, int32_t *converged) {                                \
        get_temperature<Real>(*m, n, ld, e, Y, T_guess, tol, max_iter, T, iters, converged);                  \
    }                                                                                                         \
    Real oracle_mixture_h_##SUFFIX(const oracle_mech *m, Real T, const Real *Y) {                             \
        return mixture_h<Real>(*m, T, Y, 1);                                                                  \
    }                                                                                                         \
    Real oracle_mixture_cp_##SUFFIX(const oracle_mech *m, Real T, const Real *Y) {                            \
        return mixture_cp<Real>(*m, T, Y, 1);                                                                 \
    }                                                                                                         \
    void oracle_get_temperature_h_##SUFFIX(const oracle_mech *m, int64_t n, int64_t ld, const Real *h,        \
                                           const Real *Y, const Real *T_guess, Real tol, int max_iter,       \
                                           Real *T, int32_t *iters, int32_t *converged) {                    \
        get_temperature<Real>(*m, n, ld, h, Y, T_guess, tol, max_iter, T, iters, converged, true);            \
    }                                                                                                         \
    void oracle_get_density_##SUFFIX(const oracle_mech *m, int64_t n, int64_t ld, const Real *p,              \
                                     const Real *T, const Real *Y, Real *rho) {                               \
        for (int64_t i = 0; i < n; ++i) rho[i] = density_point<Real>(*m, p[i], T[i], Y + i, ld);              \
    }                                                                                                         \
    void oracle_get_pressure_##SUFFIX(const oracle_mech *m, int64_t n, int64_t ld, const Real *rho,           \
                                      const Real *T, const Real *Y, Real *p) {                                \
        for (int64_t i = 0; i < n; ++i) p[i] = pressure_point<Real>(*m, rho[i], T[i], Y + i, ld);             \
    }                                                                                                         \
    void oracle_get_jacobian_##SUFFIX(const oracle_mech *m, int64_t n, int64_t ld, const Real *rho, const Real *T, \
                                      const Real *Y, int mode, Real *J, Real *dSdT, Real *boundJ,              \
                                      Real *bounddSdT) {                                                       \
        get_jacobian<Real>(*m, n, ld, rho, T, Y, mode, J, dSdT, boundJ, bounddSdT);                            \
    }                                                                                                         \
    void oracle_reactor_rk4_##SUFFIX(const oracle_mech *m, int64_t n, int64_t ld, const Real *rho, const Real *e,    \
                                     Real *Y, Real *T, Real dt, int n_steps, Real tol, int max_iter, Real *Ybound, \
                                     int64_t *n_not_converged) {                                              \
        reactor_rk4<Real>(*m, n, ld, rho, e, Y, T, dt, n_steps, tol, max_iter, Ybound, n_not_converged);      \
    }                                                                                                         \
    void oracle_get_transport_##SUFFIX(const oracle_transport *t, int64_t n, int64_t ld, const Real *T, const Real *Y, \
                                       Real *mu, Real *kappa, Real *Dkm) {                                   \
        get_transport<Real>(*t, n, ld, T, Y, mu, kappa, Dkm);                                                 \
    }                                                                                                         \
    void oracle_reactor_cn_##SUFFIX(const oracle_mech *m, int64_t n, int64_t ld, const Real *rho, const Real *e,     \
                                    Real *Y, Real *T, Real dt, int n_steps, int newton_iters, Real tol,           \
                                    int max_iter, Real *Ybound, Real *last_update, int64_t *n_not_converged) {     \
        reactor_cn<Real>(*m, n, ld, rho, e, Y, T, dt, n_steps, newton_iters, tol, max_iter, Ybound, last_update,  \
                         n_not_converged);                                                                    \
    }                                                                                                         \
    void oracle_get_net_production_rates_##SUFFIX(const oracle_mech *m, int64_t n, int64_t ld,                \
                                                  const Real *rho, const Real *T, const Real *Y, Real *omega, \
                                                  Real *bound, Real *rf, Real *rr) {                          \
        get_net_production_rates<Real>(*m, n, ld, rho, T, Y, omega, bound, rf, rr);                           \
    }

ORACLE_API(f64, double)
ORACLE_API(f80, long double)

}   // extern "C"
