// Per-point arithmetic of the chemical-Jacobian kernel, shared by the kernel and the
// host test build.  Formulation and table records: pyro_jac_tables.h.
//
// One thread owns one point.  Per-point arrays indexed by a run-time species number, n_species + 1 entries
// each (the last one is the dummy species: C = 1, G = DG = 0, accumulators = sink):
//     read-only after the fill:   C_k (A.8),  G_k = log2 E_k (pyro_tables.h),  DG_k = dG_k/dT
//     accumulators:               PW  the current column  dS_i/dC_k,
//                                 PV  the part of every column that comes from the default efficiencies,
//                                 PDT dS_i/dT
// reached through a `Mem` accessor (kernel: shared and tensor memory; host build: plain arrays):
//     mem.ldC(k), mem.ldG(k), mem.ldDG(k)                   doubles
//     mem.fill(k, C, G, DG)                                 also zeroes the three accumulators of k
//     r = mem.template ld_acc<P>(k); mem.fence_ld(); mem.value(r);  mem.template st_acc<P>(k, v); mem.fence_st()
//     o = mem.ld_out(k); mem.fence_ld(); mem.out_w(o), out_v(o), out_dt(o)     the three accumulators of k at once
//     mem.ld_ext(slot), mem.st_ext(slot, v)                 per-thread scratch of the [M] reactions
#pragma once
#include "pyro_jac_tables.h"
#include "pyro_point.cuh"

namespace pyro {

enum { PW = 0, PV = 1, PDT = 2 };

constexpr double kLn2 = 0.69314718055994530942;
constexpr double kLog2e = 1.4426950408889634074;
constexpr double kLn10 = 2.3025850929940456840;

// d/dT of log2 k = c0 + c1 log2T + c2/T
PYRO_HD double arrhenius_log2_dT(double c1, double c2, double invT) { return invT * fma(-c2, invT, c1 * kLog2e); }

// d/dT of species_log2E
PYRO_HD double species_log2E_dT(const double *c, double T, double invT) {
    double h = fma(4.0 * c[6], T, 3.0 * c[5]);
    h = fma(h, T, 2.0 * c[4]);
    h = fma(h, T, c[3]);
    return fma(invT, fma(-c[2], invT, c[1] * kLog2e), h);
}

// column[sc_species[m]] += sc_w[m] * d  for the first N scatter entries (unused entries name the dummy species)
template <int P, int N, class Mem>
PYRO_HD void jac_scatter_n(const Mem &mem, const uint16_t (&sp)[6], const double (&w)[6], double d) {
    typename Mem::Raw r[N];
    uint32_t s[N];   // read once: the fences below are compiler barriers, behind which the record would be read again
    double c[N];
#pragma unroll
    for (int m = 0; m < N; ++m) {
        s[m] = sp[m];
        c[m] = w[m];
    }
    mem.fence_st();
#pragma unroll
    for (int m = 0; m < N; ++m) r[m] = mem.template ld_acc<P>(s[m]);
    mem.fence_ld();
#pragma unroll
    for (int m = 0; m < N; ++m) mem.template st_acc<P>(s[m], fma(c[m], d, mem.value(r[m])));
}
template <int P, class Mem>
PYRO_HD void jac_scatter(const Mem &mem, const uint16_t (&sp)[6], const double (&w)[6], double d) {
    jac_scatter_n<P, 6>(mem, sp, w, d);
}

struct JacRates {   // what phases 1 and 2 need of one reaction at one point
    double yf, dyf;      // log2 k_f and its temperature derivative
    double qf, qr;       // k_f prod C_reac,  k_f/K_c prod C_prod (0 if irreversible)
    double ddG;          // d/dT of sum_prod G - sum_reac G  (log2 units)
};

template <class Mem>
PYRO_HD JacRates jac_reaction_rates(const JacRxn &r, const PointT &pt, const Mem &mem) {
    JacRates o;
    o.yf = arrhenius_log2(r.f[0], r.f[1], r.f[2], pt.L2T, pt.invT);
    o.dyf = arrhenius_log2_dT(r.f[1], r.f[2], pt.invT);
    double c[6], g[6], dg[6];
#pragma unroll
    for (int m = 0; m < 6; ++m) {
        c[m] = mem.ldC(r.slot[m]);
        g[m] = mem.ldG(r.slot[m]);
        dg[m] = mem.ldDG(r.slot[m]);
    }
    const double dG = ((g[3] + g[4]) + g[5]) - ((g[0] + g[1]) + g[2]);
    o.ddG = ((dg[3] + dg[4]) + dg[5]) - ((dg[0] + dg[1]) + dg[2]);
    double y[2] = {o.yf, o.yf + dG};
    exp2_poly_n<2>(y);
    o.qf = y[0] * ((c[0] * c[1]) * c[2]);
    o.qr = r.rev ? y[1] * ((c[3] * c[4]) * c[5]) : 0.0;
    return o;
}

struct JacExt {      // a third-body / falloff reaction at one point
    double mul;      // multiplier of its incidence terms: [M] or L F
    double g;        // dR/d[M]: the coefficient of the efficiency eff_k in dR/dC_k
    double dRdT;     // dR/dT at fixed concentrations
};

// Third-body and falloff forms (readings G6-G8) and their derivatives with respect to [M] and T.
template <class Tab, class Mem>
PYRO_HD JacExt jac_ext_reaction(const Tab &tab, const JacRxn &r, const PointT &pt, double ctot, const Mem &mem) {
    const JacRates q = jac_reaction_rates(r, pt, mem);
    double M = r.eff_default * ctot;
#pragma unroll 1
    for (uint32_t e = r.eff_begin; e < r.eff_begin + r.eff_count; ++e) {
        const EffEntry &en = tab.eff((int)e);
        M = fma(en.delta, mem.ldC(en.species), M);
    }
    const double net = q.qf - q.qr;
    const double dnet_dT = kLn2 * (q.qf * q.dyf - q.qr * (q.dyf + q.ddG));   // at fixed rate-coefficient multiplier
    double mul, g, dRdT;
    if (r.type == PYRO_THREE_BODY) {   // R = [M] (q_f - q_r)
        mul = M;
        g = net;
        dRdT = M * dnet_dT;
    } else {                           // R = L F (q_f - q_r), L = Pr/(1+Pr), Pr = k_0 [M]/k_inf
        const RxnFall &fl = tab.rxn_fall((int)r.fall_index);
        const double y0 = arrhenius_log2(fl.l[0], fl.l[1], fl.l[2], pt.L2T, pt.invT);
        const double dy0 = arrhenius_log2_dT(fl.l[1], fl.l[2], pt.invT);
        double e[4] = {y0 - q.yf, fl.troe_t3 * pt.T, fl.troe_t1 * pt.T, fl.troe_t2 * pt.invT};
        exp2_poly_n<4>(e);
        const double Pr = e[0] * M;
        const double dlnL = rcp_newton(1.0 + Pr);   // d ln L / d ln Pr
        double LF = Pr * dlnL, dlnF_dlnPr = 0.0, dlnF_dT = 0.0;
        if (r.type == PYRO_FALLOFF_TROE) {
            const double a3 = (1.0 - fl.troe_alpha) * e[1], a1 = fl.troe_alpha * e[2], a2 = fl.troe_has_t2 * e[3];
            const double Fc = a3 + a1 + a2;
            const double dFc = kLn2 * fma(fl.troe_t3, a3, fma(fl.troe_t1, a1, -fl.troe_t2 * pt.invT * pt.invT * a2));
            const double l2Fc = log2_pos(Fc), lFc = l2Fc * kLog10of2;
            const double dlFc = dFc * rcp_newton(Fc * kLn10);
            const double cc = -0.4 - 0.67 * lFc, n = 0.75 - 1.27 * lFc;
            const double xx = fma(log2_pos(Pr), kLog10of2, cc);
            const double rden = rcp_newton(n - 0.14 * xx);
            const double f1 = xx * rden;
            const double gg = rcp_newton(fma(f1, f1, 1.0));
            double z[1] = {l2Fc * gg};
            exp2_poly_n<1>(z);
            LF *= z[0];
            const double df1_dx = n * rden * rden, df1_dn = -xx * rden * rden;
            const double dgg = -2.0 * f1 * gg * gg;
            dlnF_dlnPr = lFc * dgg * df1_dx;
            dlnF_dT = kLn10 * dlFc * fma(lFc * dgg, fma(df1_dx, -0.67, df1_dn * -1.27), gg);
        }
        mul = LF;
        const double s = dlnL + dlnF_dlnPr;
        g = LF * s * rcp_newton(M) * net;
        dRdT = LF * fma(fma(s, kLn2 * (dy0 - q.dyf), dlnF_dT), net, dnet_dT);
    }
    return JacExt{mul, g, dRdT};
}

// dR/dT of a reaction without [M]
template <class Mem> PYRO_HD double jac_plain_dRdT(const JacRxn &r, const PointT &pt, const Mem &mem) {
    const JacRates q = jac_reaction_rates(r, pt, mem);
    return kLn2 * (q.qf * q.dyf - q.qr * (q.dyf + q.ddG));
}

// e_k(T) of the energy rows (A.26)
PYRO_HD double jac_species_energy(const EnergyRow &er, double T) {
    const double *ec = T < er.t_mid ? er.lo : er.hi;
    double ek = fma(ec[5], T, ec[4]);
    ek = fma(ek, T, ec[3]);
    ek = fma(ek, T, ec[2]);
    ek = fma(ek, T, ec[1]);
    return fma(ek, T, ec[0]);
}
// c_v,k(T) = de_k/dT (A.29)-(A.31)
PYRO_HD double jac_species_cv(const EnergyRow &er, double T) {
    const double *ec = T < er.t_mid ? er.lo : er.hi;
    double cvk = fma(5.0 * ec[5], T, 4.0 * ec[4]);
    cvk = fma(cvk, T, 3.0 * ec[3]);
    cvk = fma(cvk, T, 2.0 * ec[2]);
    return fma(cvk, T, ec[1]);
}

// The incidences [begin, end) of one class of one column: column[sc_species] += sc_w * d  (pyro_jac_tables.h)
// kGibbs: the records have a Gibbs sum (product side); N: scatter entries in use (4 or 6)
template <bool kGibbs, int N, class Tab, class Mem>
PYRO_HD void jac_column_accumulate(const Tab &tab, uint32_t begin, uint32_t end, const PointT &pt, const Mem &mem) {
#pragma unroll 1
    for (uint32_t q = begin; q < end;) {
        uint32_t n;
        const JacInc *run = tab.inc_run(q, end, n);   // the records the table has at consecutive addresses
        q += n;
#pragma unroll 1
        for (const JacInc *stop = run + n; run != stop; ++run) {
            const JacInc &e = *run;
            double y[1] = {arrhenius_log2(e.f[0], e.f[1], e.f[2], pt.L2T, pt.invT)};
            if (kGibbs)
                y[0] += ((mem.ldG(e.gslot[3]) + mem.ldG(e.gslot[4])) + mem.ldG(e.gslot[5])) -
                        ((mem.ldG(e.gslot[0]) + mem.ldG(e.gslot[1])) + mem.ldG(e.gslot[2]));
            const double others = mem.ldC(e.other[0]) * mem.ldC(e.other[1]);
            const double m = e.coef * mem.ld_ext(e.mul);
            exp2_poly_n<1>(y);
            jac_scatter_n<PW, N>(mem, e.sc_species, e.sc_w, (m * y[0]) * others);
        }
    }
}

// One column: its four classes of records one after the other.
template <class Tab, class Mem>
PYRO_HD void jac_column(const Tab &tab, const JacCol &col, const PointT &pt, const Mem &mem) {
    uint32_t q = col.inc_begin;
    jac_column_accumulate<false, 4>(tab, q, q + col.n_class[0], pt, mem);
    q += col.n_class[0];
    jac_column_accumulate<false, 6>(tab, q, q + col.n_class[1], pt, mem);
    q += col.n_class[1];
    jac_column_accumulate<true, 4>(tab, q, q + col.n_class[2], pt, mem);
    q += col.n_class[2];
    jac_column_accumulate<true, 6>(tab, q, q + col.n_class[3], pt, mem);
}

// The whole Jacobian of one point.
//   load_y(k)               mass fraction of species k at this point
//   store_J(i, k, v)        J_ik = dS_i/dY_k;  store_T(i, v)  dS_i/dT (called only if want_T)
//   mode 0: Y-derivatives at fixed (rho, T); mode 1: at fixed (rho, e) (reading G26)
template <class Tab, class Mem, class LoadY, class StoreJ, class StoreT>
PYRO_HD void jacobian_point(const Tab &tab, const JacLayout &lay, double T, double rho, int mode, bool want_T, const Mem &mem,
                            const LoadY &load_y, const StoreJ &store_J, const StoreT &store_T) {
    const int ns = lay.n_species;
    const PointT pt = make_point(T);
    // ---- phase 0: C_k, G_k, dG_k/dT; C_tot; c_v (mode 1)
    double ctot = 0.0, cv = 0.0;
#pragma unroll 1
    for (int k = 0; k < ns; ++k) {
        const SpecRow &row = tab.spec(k);
        const double *c = pt.T < row.t_mid ? row.lo : row.hi;
        const double y = load_y(k);
        const double C = rho * y * row.inv_w;
        ctot += C;
        mem.fill((uint32_t)k, C, species_log2E(c, pt.T, pt.L2T, pt.invT), species_log2E_dT(c, pt.T, pt.invT));
        if (mode == 1) {   // c_v = sum_k Y_k de_k/dT  (A.29)-(A.31), energy rows of pyro_tables.h
            cv = fma(y, jac_species_cv(tab.energy(k), pt.T), cv);
        }
    }
    mem.fill((uint32_t)ns, 1.0, 0.0, 0.0);
    mem.st_ext(0u, 1.0);
    // ---- phase 1: third-body and falloff reactions (readings G6-G8), once per point
    tab.begin_rxn(lay.n_plain, lay.n_ext);   // the records of a phase are read front to back (kernel: streamed through shared memory)
#pragma unroll 1
    for (int x = 0; x < lay.n_ext; ++x) {
        const JacRxn &r = tab.rxn(lay.n_plain + x);
        const JacExt x_ = jac_ext_reaction(tab, r, pt, ctot, mem);
        const double mul = x_.mul, g = x_.g, dRdT = x_.dRdT;
        mem.st_ext(1u + 2u * r.ext, mul);
        mem.st_ext(2u + 2u * r.ext, g);
        jac_scatter<PDT>(mem, r.sc_species, r.sc_w, dRdT);
        jac_scatter<PV>(mem, r.sc_species, r.sc_w, g * r.eff_default);
    }
    // ---- phase 2: temperature derivative of the other reactions
    tab.begin_rxn(0, lay.n_plain);
#pragma unroll 1
    for (int j = 0; j < lay.n_plain; ++j) {
        const JacRxn &r = tab.rxn(j);
        jac_scatter<PDT>(mem, r.sc_species, r.sc_w, jac_plain_dRdT(r, pt, mem));
    }
    mem.fence_st();
    if (want_T) {
#pragma unroll 1
        for (int i = 0; i < ns; ++i) {
            const typename Mem::Raw r = mem.template ld_acc<PDT>((uint32_t)i);
            mem.fence_ld();
            store_T(i, mem.value(r));
        }
    }
    // ---- phase 3: the columns
    const double rcv = mode == 1 ? 1.0 / cv : 0.0;
    tab.begin_inc();
#pragma unroll 1
    for (int k = 0; k < ns; ++k) {
        const JacCol &col = tab.col(k);
        jac_column(tab, col, pt, mem);
        mem.fence_st();
        // J_ik = (column_i + V_i) rho/W_k - dS_i/dT e_k/c_v ; the column accumulator is cleared for the next one
        const double scale = rho * tab.spec(k).inv_w;
        double ekcv = 0.0;
        if (mode == 1) {
            ekcv = jac_species_energy(tab.energy(k), pt.T) * rcv;
        }
#pragma unroll 1
        for (int i = 0; i < ns; i += 4) {   // four rows in flight per tensor-memory round trip
            typename Mem::Out o[4];
#pragma unroll
            for (int u = 0; u < 4; ++u) o[u] = mem.ld_out((uint32_t)(i + u < ns ? i + u : ns));
            mem.fence_ld();
#pragma unroll
            for (int u = 0; u < 4; ++u)
                if (i + u < ns) {
                    store_J(i + u, k, fma(mem.out_w(o[u]) + mem.out_v(o[u]), scale, -(mem.out_dt(o[u]) * ekcv)));
                    mem.template st_acc<PW>((uint32_t)(i + u), 0.0);
                }
        }
    }
}

// Plain arrays of n_species + 1 entries per plane (host build, tests).
struct JacArrayMem {
    typedef double Raw;
    struct Out {
        double w, v, dt;
    };
    double *C, *G, *DG, *acc[3], *ext;
    PYRO_HD double ldC(uint32_t k) const { return C[k]; }
    PYRO_HD double ldG(uint32_t k) const { return G[k]; }
    PYRO_HD double ldDG(uint32_t k) const { return DG[k]; }
    PYRO_HD void fill(uint32_t k, double c, double g, double dg) const {
        C[k] = c;
        G[k] = g;
        DG[k] = dg;
        acc[0][k] = acc[1][k] = acc[2][k] = 0.0;
    }
    template <int P> PYRO_HD Raw ld_acc(uint32_t k) const { return acc[P][k]; }
    template <int P> PYRO_HD void st_acc(uint32_t k, double v) const { acc[P][k] = v; }
    PYRO_HD Out ld_out(uint32_t k) const { return Out{acc[PW][k], acc[PV][k], acc[PDT][k]}; }
    PYRO_HD double out_w(const Out &o) const { return o.w; }
    PYRO_HD double out_v(const Out &o) const { return o.v; }
    PYRO_HD double out_dt(const Out &o) const { return o.dt; }
    PYRO_HD double value(Raw r) const { return r; }
    PYRO_HD void fence_ld() const {}
    PYRO_HD void fence_st() const {}
    PYRO_HD double ld_ext(uint32_t s) const { return ext[s]; }
    PYRO_HD void st_ext(uint32_t s, double v) const { ext[s] = v; }
};

}   // namespace pyro
