"""Host logic without a GPU: the C-ABI library loads and exports what include/pyro.h declares;
the packer's validation; and the packer + per-point device arithmetic (compiled for the host by
tests/hostemu, a test-only build) against the oracle."""
import ctypes as C
import os
import re
import subprocess

import mpmath as mp
import numpy as np
import pytest

import hand_cases
import parity
from oracle import oracle
from paper_2503_24286_b200 import binding, build, inputs

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


# ------------------------------------------------------------------ boundary
def test_library_builds_loads_and_exports_every_declared_symbol():
    build.build_libpyro()
    lib = C.CDLL(binding.LIB_PATH)
    header = open(os.path.join(ROOT, "include", "pyro.h")).read()
    declared = set(re.findall(r"^(?:int|const char \*)\s*(pyro_[a-z0-9_]+)\s*\(", header, flags=re.M))
    assert declared == set(binding.EXPORTS), declared ^ set(binding.EXPORTS)
    for name in declared:
        assert hasattr(lib, name), name
    # extern "C", plain pointers and sizes: no C++ or torch types in the signatures
    nm = subprocess.run(["nm", "-D", "--defined-only", binding.LIB_PATH], capture_output=True, text=True).stdout
    for name in declared:
        assert re.search(rf"\bT {name}\b", nm), name
    assert "torch" not in header and "at::" not in header


def test_status_strings_and_no_cpu_fallback():
    lib = binding.load_library()
    for st, name in binding.STATUS_NAMES.items():
        assert lib.pyro_status_string(st).decode().startswith(name)
    import torch
    if not torch.cuda.is_available():
        # the product path must fail loudly without a CUDA device
        with pytest.raises(binding.PyroError) as ei:
            binding.Mechanism(inputs.config_mechanism(0))
        assert ei.value.status == 6 and "no CPU fallback" in str(ei.value)
    assert lib.pyro_mech_destroy(None) == 0


# ------------------------------------------------------------------ host emulation helpers
@pytest.fixture(scope="module")
def emu():
    src = os.path.join(ROOT, "tests", "hostemu", "hostemu.cpp")
    lib = os.path.join(ROOT, "tests", "hostemu", "libhostemu.so")
    deps = [src] + [os.path.join(ROOT, "paper_2503_24286_b200", "csrc", f)
                    for f in ("pyro_pack.cpp", "pyro_pack.h", "pyro_point.cuh", "pyro_math.cuh", "pyro_tables.h",
                              "pyro_jac_pack.cpp", "pyro_jac.cuh", "pyro_jac_tables.h")]
    if not os.path.exists(lib) or any(os.path.getmtime(d) > os.path.getmtime(lib) for d in deps):
        subprocess.run(["g++", "-std=c++17", "-O2", "-mfma", "-shared", "-fPIC", "-o", lib, src,
                        os.path.join(ROOT, "paper_2503_24286_b200", "csrc", "pyro_pack.cpp"),
                        os.path.join(ROOT, "paper_2503_24286_b200", "csrc", "pyro_jac_pack.cpp")], check=True)
    L = C.CDLL(lib)
    L.emu_last_error.restype = C.c_char_p
    L.emu_exp2.restype = C.c_double
    L.emu_exp2.argtypes = [C.c_double]
    vp, i64 = C.c_void_p, C.c_int64
    L.emu_pack_status.argtypes = [vp, vp]
    L.emu_rates.argtypes = [vp, i64, i64, vp, vp, vp, vp]
    L.emu_pack_order.argtypes = [vp, vp, C.c_int32]
    L.emu_exp2_rxn.restype = C.c_double
    L.emu_exp2_rxn.argtypes = [C.c_double]
    L.emu_log2.restype = C.c_double
    L.emu_log2.argtypes = [C.c_double]
    L.emu_exp2_pair.argtypes = [C.c_double, vp, vp]
    L.emu_temperature.argtypes = [vp, i64, i64, vp, vp, vp, C.c_double, C.c_int, vp, vp]
    L.emu_temperature2.argtypes = [vp, i64, i64, vp, vp, vp, C.c_double, C.c_int, vp, vp, C.c_int]
    L.emu_eos.argtypes = [vp, i64, i64, vp, vp, vp, vp, C.c_int]
    L.emu_rates2.argtypes = [vp, i64, i64, vp, vp, vp, vp, C.c_int]
    L.emu_pack_side_log2.argtypes = [vp, C.c_int, vp]
    L.emu_jacobian.argtypes = [vp, i64, i64, vp, vp, vp, C.c_int, vp, vp]
    L.emu_reactor.argtypes = [vp, i64, i64, vp, vp, vp, vp, C.c_double, C.c_int, C.c_double, C.c_int, vp, vp]
    return L


def emu_rates(emu, mech, rho, T, Y):
    desc, keep = binding.make_desc(mech)
    rho, T, Y = (np.ascontiguousarray(x, dtype=np.float64) for x in (rho, T, Y))
    om = np.empty_like(Y)
    st = emu.emu_rates(C.byref(desc), rho.shape[0], rho.shape[0], rho.ctypes.data, T.ctypes.data,
                       Y.ctypes.data, om.ctypes.data)
    assert st == 0, emu.emu_last_error()
    return om


def emu_rates_status(emu, mech, rho, T, Y, shift=1):
    """(status, omega, message) of the host build of the rates path; shift = 0 packs without the conserved shift."""
    desc, keep = binding.make_desc(mech)
    rho, T, Y = (np.ascontiguousarray(x, dtype=np.float64) for x in (rho, T, Y))
    om = np.empty_like(Y)
    st = emu.emu_rates2(C.byref(desc), rho.shape[0], rho.shape[0], rho.ctypes.data, T.ctypes.data,
                        Y.ctypes.data, om.ctypes.data, shift)
    return st, om, emu.emu_last_error().decode()


def pack_range(emu, mech, shift=1):
    """(status, largest side sum of the plain class, largest pair partial sum, wide reactions)."""
    desc, keep = binding.make_desc(mech)
    out = (C.c_double * 3)()
    st = emu.emu_pack_side_log2(C.byref(desc), shift, out)
    return st, out[0], out[1], int(out[2])


def emu_temperature(emu, mech, e, Y, Tg, tol=1e-6, max_iter=10):
    desc, keep = binding.make_desc(mech)
    e, Y, Tg = (np.ascontiguousarray(x, dtype=np.float64) for x in (e, Y, Tg))
    T = np.empty_like(e)
    bad = C.c_int64(0)
    st = emu.emu_temperature(C.byref(desc), e.shape[0], e.shape[0], e.ctypes.data, Y.ctypes.data, Tg.ctypes.data,
                             tol, max_iter, T.ctypes.data, C.byref(bad))
    assert st == 0, emu.emu_last_error()
    return T, int(bad.value)


def pack_status(emu, mech, mutate=None):
    desc, keep = binding.make_desc(mech)
    if mutate:
        mutate(desc, keep)
    info = (C.c_int64 * 55)()
    st = emu.emu_pack_status(C.byref(desc), info)
    return st, list(info), emu.emu_last_error().decode()


# ------------------------------------------------------------------ exp2
def test_exp2_poly_accuracy_and_edges(emu):
    mp.mp.dps = 40
    rng = np.random.default_rng(1)
    ys = np.concatenate([rng.uniform(-1000, 1000, 4000), rng.uniform(-1, 1, 1000),
                         np.arange(-20, 21) * 0.5, [1e-300, -1e-300, 0.0]])
    worst = 0.0
    for y in ys:
        got = emu.emu_exp2(float(y))
        ref = mp.mpf(2) ** mp.mpf(float(y))
        worst = max(worst, float(abs(mp.mpf(got) / ref - 1)))
    assert worst < 2e-15, worst
    assert emu.emu_exp2(0.0) == 1.0 and emu.emu_exp2(10.0) == 1024.0 and emu.emu_exp2(-3.0) == 0.125
    assert emu.emu_exp2(-1100.0) < 1e-307 and emu.emu_exp2(-1e9) < 1e-307       # flushed, never negative or NaN
    assert emu.emu_exp2(-1100.0) >= 0.0
    assert np.isnan(emu.emu_exp2(float("nan")))
    assert not np.isfinite(emu.emu_exp2(1100.0)) or emu.emu_exp2(1100.0) > 1e307


def test_exp2_of_the_reaction_loops_degree_nine(emu):
    """exp2_poly_n (rate coefficients, falloff): degree-9 polynomial, relative error below 5e-14."""
    mp.mp.dps = 40
    rng = np.random.default_rng(4)
    ys = np.concatenate([rng.uniform(-1000, 1000, 3000), rng.uniform(-1, 1, 2000), np.arange(-20, 21) * 0.5])
    worst = 0.0
    for y in ys:
        worst = max(worst, float(abs(mp.mpf(emu.emu_exp2_rxn(float(y))) / (mp.mpf(2) ** mp.mpf(float(y))) - 1)))
    assert 1e-15 < worst < 5e-14, worst
    assert emu.emu_exp2_rxn(0.0) == 1.0 and emu.emu_exp2_rxn(10.0) == 1024.0
    assert 0.0 <= emu.emu_exp2_rxn(-1e9) < 1e-307 and np.isnan(emu.emu_exp2_rxn(float("nan")))


def test_exp2_pair_is_exp2_and_its_reciprocal(emu):
    """(2^y, 2^-y) from one range reduction: each as accurate as exp2_poly, product 1 to a few ulp."""
    mp.mp.dps = 40
    rng = np.random.default_rng(2)
    ys = np.concatenate([rng.uniform(-1000, 1000, 3000), rng.uniform(-1, 1, 1000), np.arange(-20, 21) * 0.5, [0.0]])
    worst = worst_prod = 0.0
    e, b = C.c_double(), C.c_double()
    for y in ys:
        emu.emu_exp2_pair(float(y), C.byref(e), C.byref(b))
        ref = mp.mpf(2) ** mp.mpf(float(y))
        worst = max(worst, float(abs(mp.mpf(e.value) / ref - 1)), float(abs(mp.mpf(b.value) * ref - 1)))
        worst_prod = max(worst_prod, abs(e.value * b.value - 1.0))
    assert worst < 2e-15, worst
    assert worst_prod < 1e-15, worst_prod
    emu.emu_exp2_pair(10.0, C.byref(e), C.byref(b))
    assert e.value == 1024.0 and b.value == 1.0 / 1024.0


def test_log2_pos_accuracy(emu):
    """Branch-free log2 of the falloff path: absolute error a few 1e-16 near 1, 1 ulp-ish beyond."""
    mp.mp.dps = 40
    rng = np.random.default_rng(3)
    xs = np.concatenate([10.0 ** rng.uniform(-300, 300, 3000), rng.uniform(0.5, 2.0, 3000),
                         2.0 ** np.arange(-40, 41), [np.sqrt(2.0), np.sqrt(0.5), 1.0, 1.0 + 2.0 ** -52, 1.0 - 2.0 ** -53]])
    worst = 0.0
    for x in xs:
        got = emu.emu_log2(float(x))
        ref = mp.log(mp.mpf(float(x)), 2)
        worst = max(worst, float(abs(mp.mpf(got) - ref) / max(1, abs(ref))))
    assert worst < 4e-16, worst
    assert emu.emu_log2(1.0) == 0.0 and emu.emu_log2(8.0) == 3.0 and emu.emu_log2(0.25) == -2.0


# ------------------------------------------------------------------ packer validation (row a0)
def _expected_plain(mech):
    """Plain class = elementary, reversible, every coefficient 1, no species on both sides."""
    n = 0
    for j in range(mech.n_reactions):
        rc = mech.reac_coeff[mech.reac_ptr[j]:mech.reac_ptr[j + 1]]
        pc = mech.prod_coeff[mech.prod_ptr[j]:mech.prod_ptr[j + 1]]
        rs = set(mech.reac_species[mech.reac_ptr[j]:mech.reac_ptr[j + 1]])
        ps = set(mech.prod_species[mech.prod_ptr[j]:mech.prod_ptr[j + 1]])
        if mech.rtype[j] == 0 and mech.reversible[j] and (rc == 1).all() and (pc == 1).all() and not (rs & ps):
            n += 1
    return n


def test_packer_classes_and_table_size(emu):
    for mech in (inputs.config_mechanism(0), inputs.config_mechanism(2), hand_cases.all_paths_mechanism()):
        st, info, _ = pack_status(emu, mech)
        # wide reactions (a side's species factors beyond 2^700 at the cold end) leave the plain class
        n_plain = _expected_plain(mech) - pack_range(emu, mech)[3]
        order = pack_order(emu, mech, info[0] + info[1])
        assert st == 0
        # records = reactions (+ null records that complete a couple, in mechanisms of 64 reactions or more)
        assert (order[:info[0]] >= 0).sum() == n_plain and (order[info[0]:] >= 0).sum() == mech.n_reactions - n_plain
        assert mech.n_reactions >= 64 or (order >= 0).all()
        assert info[3] >= len(mech.eff_species)      # efficiency lists padded to one length per lockstep group
    st, info, _ = pack_status(emu, inputs.config_mechanism(2))
    assert info[2] <= 40 * 1024          # configs[2] tables are staged in shared memory beside the planes
    assert info[0] > 200                 # and most reactions are in the plain class
    assert info[4] + info[5] > 0.7 * info[0]       # mostly stored as lockstep groups of eight or four
    assert info[3] <= 1.25 * len(inputs.config_mechanism(2).eff_species)
    assert info[6] == 1


def pack_order(emu, mech, n_records):
    desc, keep = binding.make_desc(mech)
    order = np.full(n_records, -7, dtype=np.int32)
    assert emu.emu_pack_order(C.byref(desc), order.ctypes.data, n_records) == 0
    return order


def test_packer_groups_are_species_disjoint_and_order_is_a_permutation(emu):
    """The lockstep groups batch their omega read-modify-writes: the members of a group must not
    share a species that they update.  `order` maps packed records back to the description
    (-1 for the null records that complete a couple in large mechanisms; small ones store the
    reactions left alone as singles)."""
    for mech in (inputs.config_mechanism(0), inputs.config_mechanism(2), inputs.config_mechanism(3),
                 hand_cases.all_paths_mechanism()):
        st, info, _ = pack_status(emu, mech)
        order = pack_order(emu, mech, info[0] + info[1])
        assert sorted(j for j in order.tolist() if j >= 0) == list(range(mech.n_reactions))
        assert set(order.tolist()) <= set(range(-1, mech.n_reactions))

        def net(j):
            nu = {}
            for q in range(mech.reac_ptr[j], mech.reac_ptr[j + 1]):
                nu[int(mech.reac_species[q])] = nu.get(int(mech.reac_species[q]), 0) - int(mech.reac_coeff[q])
            for q in range(mech.prod_ptr[j], mech.prod_ptr[j + 1]):
                nu[int(mech.prod_species[q])] = nu.get(int(mech.prod_species[q]), 0) + int(mech.prod_coeff[q])
            return {k for k, v in nu.items() if v != 0}
        shape = lambda j: 3 * (int(mech.reac_coeff[mech.reac_ptr[j]:mech.reac_ptr[j + 1]].sum()) - 1) + \
            int(mech.prod_coeff[mech.prod_ptr[j]:mech.prod_ptr[j + 1]].sum()) - 1
        kind = lambda j: int(mech.rtype[j])

        def check(pos, size, count, same):
            assert count % size == 0
            for g0 in range(pos, pos + count, size):
                group = [j for j in order[g0:g0 + size] if j >= 0]
                assert group and all(same(j) for j in group)
                assert len(set().union(*[net(j) for j in group])) == sum(len(net(j)) for j in group)
                assert size == 2 or len(group) == size          # null records only complete couples
            return pos + count
        pos = 0
        for sh in range(9):
            for size, count in ((8, info[7 + sh]), (4, info[16 + sh]), (2, info[25 + sh]), (1, info[42 + sh])):
                pos = check(pos, size, count, lambda j: shape(j) == sh)
        assert pos == info[0]
        for k in range(4):
            for size, count in ((4, info[34 + k]), (2, info[38 + k]), (1, info[51 + k])):
                pos = check(pos, size, count, lambda j: kind(j) == k)
        assert pos == info[0] + info[1]


def test_packer_error_codes(emu):
    m = hand_cases.all_paths_mechanism()

    def set_arr(name, idx, val):
        def f(desc, keep):
            for a in list(keep):
                if a.ctypes.data == getattr(desc, name):
                    c = a.copy()          # never touch the cached mechanism's own arrays
                    c.flat[idx] = val
                    keep.append(c)
                    setattr(desc, name, c.ctypes.data)
                    break
        return f

    def null(name):
        return lambda desc, keep: setattr(desc, name, None)

    assert emu.emu_pack_status(None, None) == 1
    cases = [
        (null("mol_weight"), 1), (null("reac_ptr"), 1), (null("A"), 1), (null("troe"), 1), (null("A0"), 1),
        (lambda d, k: setattr(d, "n_species", 0), 2), (lambda d, k: setattr(d, "n_reactions", -1), 2),
        (set_arr("mol_weight", 1, -2.0), 3), (set_arr("nasa_lo", 3, np.nan), 3), (set_arr("t_mid", 0, 0.0), 3),
        (set_arr("A", 2, 0.0), 3), (set_arr("A", 2, -1.0), 3), (set_arr("theta", 0, np.inf), 3),
        (set_arr("reac_species", 0, 99), 3), (set_arr("prod_species", 1, -1), 3), (set_arr("reac_coeff", 0, 0), 3),
        (set_arr("reac_coeff", 0, 4), 3),            # more than 3 molecules on a side
        (set_arr("reac_ptr", 2, 0), 3),              # CSR not monotone
        (set_arr("type", 0, 9), 3), (set_arr("troe", 4 * 8 + 1, -5.0), 3), (set_arr("troe", 4 * 8 + 2, 0.0), 3),
        (set_arr("A0", 7, 0.0), 3), (set_arr("eff_species", 0, 77), 3),
        (lambda d, k: setattr(d, "n_species", 100000), 4),
    ]
    for mutate, expected in cases:
        st, _, msg = pack_status(emu, m, mutate)
        assert st == expected, (expected, st, msg)
        assert msg
    # species with different T_mid pack (the rates path takes the range per species) ...
    st, info, _ = pack_status(emu, m, set_arr("t_mid", 1, 1200.0))
    assert st == 0 and info[6] == 0
    # element balance is checked when a composition is given
    mech = inputs.config_mechanism(0)
    assert pack_status(emu, mech)[0] == 0
    st, _, msg = pack_status(emu, mech, set_arr("elem_comp", 0, 5))
    assert st == 3 and "balance" in msg


# ------------------------------------------------------------------ packer + device arithmetic vs oracle
def test_emu_rates_hand_mechanism_all_paths(emu):
    mech = hand_cases.all_paths_mechanism()
    rho, T, Y = hand_cases.random_states(mech, 512)
    om_ref, bound = oracle.Oracle(mech).get_net_production_rates(rho, T, Y)
    om = emu_rates(emu, mech, rho, T, Y)
    parity.assert_omega_parity(om, om_ref, bound)
    # one reaction at a time, so that no path hides behind another
    for j in range(mech.n_reactions):
        sub = hand_cases.simple_mechanism(hand_cases.species5(), [])   # placeholder to fetch builder
        rx = _reaction_dict(mech, j)
        one = hand_cases.simple_mechanism(hand_cases.species5(), [rx])
        om_ref, bound = oracle.Oracle(one).get_net_production_rates(rho[:64], T[:64], Y[:, :64])
        parity.assert_omega_parity(emu_rates(emu, one, rho[:64], T[:64], Y[:, :64]), om_ref, bound)


def _reaction_dict(mech, j):
    d = dict(
        reac={int(mech.reac_species[q]): int(mech.reac_coeff[q]) for q in range(mech.reac_ptr[j], mech.reac_ptr[j + 1])},
        prod={int(mech.prod_species[q]): int(mech.prod_coeff[q]) for q in range(mech.prod_ptr[j], mech.prod_ptr[j + 1])},
        A=mech.A[j], b=mech.b[j], theta=mech.theta[j], type=int(mech.rtype[j]), reversible=int(mech.reversible[j]),
        eff_default=mech.eff_default[j], A0=mech.A0[j], b0=mech.b0[j], theta0=mech.theta0[j],
        eff={int(mech.eff_species[q]): float(mech.eff_value[q]) for q in range(mech.eff_ptr[j], mech.eff_ptr[j + 1])},
    )
    if mech.rtype[j] == 3:
        d["troe"] = tuple(mech.troe[j])
    return d


def _cold_to_hot_states(mech, n, seed=3):
    rng = np.random.default_rng(seed)
    T = np.concatenate([[250.0, 251.0, 300.0, 6000.0], rng.uniform(250.0, 3500.0, size=n - 4)])
    Y = rng.dirichlet(np.full(mech.n_species, 0.8), size=n).T.copy()
    rho = rng.uniform(0.05, 5.0, size=n)
    return rho, T, Y


@pytest.mark.parametrize("a6", [1.2e5, -1.2e5, 2.5e5, -2.5e5])
def test_emu_rates_finite_wherever_the_oracle_is_extreme_formation_enthalpies(emu, a6):
    """SURVEY.md section 7 hard part 4 / (A.10) PAPER.md:932: |g_k/RT| ~ |a6|/T up to 1000 per species at 250 K.
    The per-species factors are shifted by what the reactions conserve and wide reactions are multiplied in
    pairs, so the rates are finite and within tolerance wherever the oracle's are; a mechanism whose K_c
    itself leaves the FP64 range inside the supported temperatures is refused with a message, never NaN."""
    for name, mech in hand_cases.extreme_thermo_mechanisms(a6).items():
        rho, T, Y = _cold_to_hot_states(mech, 400)
        om_ref, bound = oracle.Oracle(mech).get_net_production_rates(rho, T, Y)
        st, om, msg = emu_rates_status(emu, mech, rho, T, Y)
        if name == "assoc" and abs(a6) > 2e5:
            # K_c ~ exp(+-a6/T) = 2^+-1440 at 250 K: out of range for the definition itself
            assert not np.isfinite(om_ref[:, T < 300]).all()
            assert st == 7 and "K" in msg and "250" in msg
            continue
        assert st == 0, msg
        ok = np.isfinite(om_ref).all(axis=0) & np.isfinite(bound).all(axis=0)
        assert ok.all(), "the oracle is finite on the whole supported range for the accepted mechanisms"
        assert np.isfinite(om).all()
        parity.assert_omega_parity(om, om_ref, bound)


def test_conserved_shift_changes_nothing_but_the_range(emu):
    """Packing with and without the shift of the species rows gives the same rates (it cancels exactly in K_c
    and in C_k = A_k B_k); without it the extreme mechanism is out of range and is refused."""
    for cfg, n in ((0, 512), (2, 128)):
        mech = inputs.config_mechanism(cfg)
        st = inputs.config_states(cfg, n=n)
        om_ref, bound = oracle.Oracle(mech).get_net_production_rates(st["rho"], st["T"], st["Y"])
        for shift in (0, 1):
            s, om, msg = emu_rates_status(emu, mech, st["rho"], st["T"], st["Y"], shift)
            assert s == 0, msg
            assert parity.assert_omega_parity(om, om_ref, bound) < 1e-12
        s1, side1, pair1, wide1 = pack_range(emu, mech, 1)
        assert s1 == 0 and side1 <= 700.0 and pair1 <= 900.0
    mech = hand_cases.extreme_thermo_mechanisms(-2.5e5)["balanced"]
    s0, *_ = pack_range(emu, mech, 0)
    s1, side1, pair1, wide1 = pack_range(emu, mech, 1)
    assert s0 == 7 and s1 == 0 and side1 < 50.0 and wide1 == 0   # the common a6/T is gone entirely


def test_wide_reactions_take_the_pair_form(emu):
    """A reaction whose side sums exceed 2^700 at the cold end goes to the extended class, which multiplies in
    reactant/product pairs.  Packed without the shift, A + B <=> AB with |log2 E_k| = 692 each at 250 K is
    such a reaction; the rates still match the oracle from 250 K up."""
    mech = hand_cases.extreme_thermo_mechanisms(-1.2e5)["assoc"]
    s, side, pair, wide = pack_range(emu, mech, 0)
    assert s == 0 and wide == 1 and 600.0 < pair <= 900.0   # (the Lindemann reaction is in the extended class anyway)
    assert pack_range(emu, mech, 1)[3] == 0   # with the shift the sides stay below 2^700
    rho, T, Y = _cold_to_hot_states(mech, 300)
    om_ref, bound = oracle.Oracle(mech).get_net_production_rates(rho, T, Y)
    for shift in (0, 1):
        st, om, msg = emu_rates_status(emu, mech, rho, T, Y, shift)
        assert st == 0, msg
        parity.assert_omega_parity(om, om_ref, bound)


def test_troe_sentinel_temperatures(emu):
    """T*** = 1e-30, T* = 1e30, T** = 1e30 as real mechanism files carry them: the exponents are
    clamped at pack time where the term is exactly 0 (or 1) in FP64, so exp2's reduction never sees |y| >= 2^31."""
    mech = hand_cases.troe_sentinel_mechanism()
    rho, T, Y = hand_cases.random_states(mech, 600)
    T[:4] = [250.0, 1234.5, 3000.0, 6000.0]
    om_ref, bound = oracle.Oracle(mech).get_net_production_rates(rho, T, Y)
    assert np.isfinite(om_ref).all()
    st, om, msg = emu_rates_status(emu, mech, rho, T, Y)
    assert st == 0, msg
    parity.assert_omega_parity(om, om_ref, bound)


def test_rate_coefficient_exponent_out_of_exp2_range_is_refused(emu):
    mech = hand_cases.simple_mechanism(hand_cases.species5(), [dict(reac={0: 1, 1: 1}, prod={2: 1}, A=1e10, b=0.0, theta=1e12)])
    st, _, msg = pack_status(emu, mech)
    assert st == 7 and "rate coefficient" in msg


@pytest.mark.parametrize("cfg,n", [(0, 4096), (1, 2048), (2, 1024), (3, 256)])
def test_emu_rates_config_mechanisms(emu, cfg, n):
    mech = inputs.config_mechanism(cfg)
    st = inputs.config_states(cfg, n=n)
    om_ref, bound = oracle.Oracle(mech).get_net_production_rates(st["rho"], st["T"], st["Y"])
    r = parity.assert_omega_parity(emu_rates(emu, mech, st["rho"], st["T"], st["Y"]), om_ref, bound)
    assert r < 1e-12   # typical residual is a few 1e-14; 1e-11 is the bar


def test_emu_rates_both_packings_of_leftover_reactions(emu, monkeypatch):
    """Reactions left alone after grouping: singles (small mechanisms) or null-padded couples (large)."""
    for cfg, n in ((0, 1024), (2, 256)):
        mech = inputs.config_mechanism(cfg)
        st = inputs.config_states(cfg, n=n)
        om_ref, bound = oracle.Oracle(mech).get_net_production_rates(st["rho"], st["T"], st["Y"])
        for singles in ("0", "1"):
            monkeypatch.setenv("PYRO_PACK_SINGLES", singles)
            stt, info, _ = pack_status(emu, mech)
            order = pack_order(emu, mech, info[0] + info[1])
            assert (singles == "1") == bool((order >= 0).all()) or (order >= 0).all()
            parity.assert_omega_parity(emu_rates(emu, mech, st["rho"], st["T"], st["Y"]), om_ref, bound)


def test_emu_rates_species_with_different_t_mid(emu):
    """Each species switches NASA range at its own T_mid (G10); states straddle both."""
    import copy
    mech = copy.deepcopy(inputs.config_mechanism(0))
    mech.t_mid = mech.t_mid.copy()
    mech.t_mid[::2] = 1400.0
    mech.t_mid[1::3] = 800.0
    st = inputs.config_states(0, n=2048)
    om_ref, bound = oracle.Oracle(mech).get_net_production_rates(st["rho"], st["T"], st["Y"])
    parity.assert_omega_parity(emu_rates(emu, mech, st["rho"], st["T"], st["Y"]), om_ref, bound)


def _mixed_tmid_case(cfg, n, seed=11):
    """A config mechanism with four different break temperatures (ranges re-matched at each), states from
    250 K to 3200 K, guesses within 10 % -- so that some land on the other side of a break temperature and
    some iterates cross one -- plus guesses placed exactly on and one ulp around the break temperatures."""
    mech = inputs.with_species_break_temperatures(inputs.config_mechanism(cfg), [800.0, 1000.0, 1400.0, 1250.0])
    rng = np.random.default_rng(seed)
    T = rng.uniform(250.0, 3200.0, size=n)
    T[: n // 4] = rng.choice([800.0, 1000.0, 1250.0, 1400.0], size=n // 4) * (1.0 + rng.uniform(-0.04, 0.04, size=n // 4))
    Y = rng.dirichlet(np.full(mech.n_species, 0.5), size=n).T.copy()
    e = inputs.mixture_energy(mech, T, Y)
    h = e + inputs.R_UNIVERSAL * T * (Y / mech.mol_weight[:, None]).sum(axis=0)
    Tg = T * (1.0 + rng.uniform(-0.1, 0.1, size=n))
    Tg[:8] = [800.0, np.nextafter(800.0, 0), np.nextafter(800.0, 1e4), 1250.0, 1400.0, np.nextafter(1400.0, 0), 1000.0, 999.0]
    return mech, T, Y, e, h, Tg


@pytest.mark.parametrize("cfg,n", [(0, 3000), (2, 600)])
def test_emu_temperature_species_with_different_t_mid(emu, cfg, n):
    """Row a4 with per-species break temperatures (G10; (A.12)-(A.13) PAPER.md:941-945, listing 22 :672-695): the
    interval-wise solve agrees with the oracle's per-species, per-iterate range choice to 1e-12, in both the
    energy and the enthalpy form, and recovers the generating temperature."""
    mech, T, Y, e, h, Tg = _mixed_tmid_case(cfg, n)
    orc = oracle.Oracle(mech)
    for enthalpy, rhs in ((0, e), (1, h)):
        T_ref, it, conv = (orc.get_temperature_from_enthalpy if enthalpy else orc.get_temperature)(rhs, Y, Tg)
        assert conv.all()
        desc, keep = binding.make_desc(mech)
        rhs_c, Y_c, Tg_c = (np.ascontiguousarray(x, dtype=np.float64) for x in (rhs, Y, Tg))
        out = np.empty_like(rhs_c)
        bad = C.c_int64(-1)
        st = emu.emu_temperature2(C.byref(desc), n, n, rhs_c.ctypes.data, Y_c.ctypes.data, Tg_c.ctypes.data, 1e-6, 10,
                                  out.ctypes.data, C.byref(bad), enthalpy)
        assert st == 0 and bad.value == 0
        parity.assert_T_parity(out, T_ref)
        assert np.max(np.abs(out - T) / T) < 1e-11   # the generating temperature (e was formed in long double)
        crossed = ((Tg[:, None] < mech.t_mid[None, :]) != (T[:, None] < mech.t_mid[None, :])).any(axis=1)
        assert crossed.sum() > n // 10   # the case does exercise the re-summation


@pytest.mark.parametrize("cfg,n", [(0, 4096), (2, 1024), (3, 256), (4, 512)])
def test_emu_temperature_config_mechanisms(emu, cfg, n):
    mech = inputs.config_mechanism(cfg)
    st = inputs.config_states(cfg, n=n)
    T_ref, it, conv = oracle.Oracle(mech).get_temperature(st["e"], st["Y"], st["T_guess"])
    T, bad = emu_temperature(emu, mech, st["e"], st["Y"], st["T_guess"])
    parity.assert_T_parity(T, T_ref)
    assert bad == int((conv == 0).sum()) == 0
    # capped iteration: both stop at the same iterate
    T_ref3, _, conv3 = oracle.Oracle(mech).get_temperature(st["e"], st["Y"], st["T_guess"], max_iter=2)
    T3, bad3 = emu_temperature(emu, mech, st["e"], st["Y"], st["T_guess"], max_iter=2)
    parity.assert_T_parity(T3, T_ref3)
    assert bad3 == int((conv3 == 0).sum())


# ------------------------------------------------------------------ NEXT-1: enthalpy form, equation of state
@pytest.mark.parametrize("cfg,n", [(0, 2048), (2, 512)])
def test_emu_enthalpy_inversion_and_eos(emu, cfg, n):
    mech = inputs.config_mechanism(cfg)
    orc = oracle.Oracle(mech)
    st = inputs.config_states(cfg, n=n)
    desc, keep = binding.make_desc(mech)
    Y = np.ascontiguousarray(st["Y"])
    h = np.array([orc.mixture_h(float(st["T"][p]), Y[:, p]) for p in range(n)])
    T_ref, _, conv = orc.get_temperature_from_enthalpy(h, Y, st["T_guess"])
    T = np.empty(n)
    bad = C.c_int64(0)
    Tg = np.ascontiguousarray(st["T_guess"])
    assert emu.emu_temperature2(C.byref(desc), n, n, h.ctypes.data, Y.ctypes.data, Tg.ctypes.data, 1e-6, 10,
                                T.ctypes.data, C.byref(bad), 1) == 0
    parity.assert_T_parity(T, T_ref)
    assert bad.value == 0 and conv.all()
    p = np.ascontiguousarray(inputs.P_ATM * np.linspace(0.1, 50.0, n))
    Tt = np.ascontiguousarray(st["T"])
    rho = np.empty(n)
    assert emu.emu_eos(C.byref(desc), n, n, p.ctypes.data, Tt.ctypes.data, Y.ctypes.data, rho.ctypes.data, 1) == 0
    assert np.max(np.abs(rho / orc.get_density(p, Tt, Y) - 1)) <= parity.EOS_TOL
    pp = np.empty(n)
    assert emu.emu_eos(C.byref(desc), n, n, rho.ctypes.data, Tt.ctypes.data, Y.ctypes.data, pp.ctypes.data, 0) == 0
    assert np.max(np.abs(pp / orc.get_pressure(rho, Tt, Y) - 1)) <= parity.EOS_TOL


def test_emu_rates_degenerate_mechanisms(emu):
    for name, mech in hand_cases.degenerate_mechanisms().items():
        rho, T, Y = hand_cases.random_states(mech, 200)
        om_ref, bound = oracle.Oracle(mech).get_net_production_rates(rho, T, Y)
        om = emu_rates(emu, mech, rho, T, Y)
        parity.assert_omega_parity(om, om_ref, bound)
        if mech.n_reactions == 0:
            assert not om.any()


def test_emu_rates_fuzz_mechanisms(emu):
    for mech in hand_cases.fuzz_mechanisms():
        rho, T, Y = hand_cases.random_states(mech, 96, seed=mech.n_reactions)
        om_ref, bound = oracle.Oracle(mech).get_net_production_rates(rho, T, Y)
        parity.assert_omega_parity(emu_rates(emu, mech, rho, T, Y), om_ref, bound)


# ------------------------------------------------------------------ chemical Jacobian
def emu_jacobian(emu, mech, rho, T, Y, mode):
    desc, keep = binding.make_desc(mech)
    rho, T, Y = (np.ascontiguousarray(x, dtype=np.float64) for x in (rho, T, Y))
    ns, n = Y.shape
    J = np.full((ns, ns, n), np.nan)
    sT = np.full((ns, n), np.nan)
    st = emu.emu_jacobian(C.byref(desc), n, n, rho.ctypes.data, T.ctypes.data, Y.ctypes.data, mode, J.ctypes.data,
                          sT.ctypes.data)
    assert st == 0, emu.emu_last_error()
    return J, sT


@pytest.mark.parametrize("mode", [0, 1])
@pytest.mark.parametrize("case", ["all_paths", "cfg0", "cfg2", "mixed_t_mid"])
def test_jacobian_point_code_matches_oracle(emu, case, mode):
    """The per-point Jacobian code (incidence lists, one exponential per incidence, [M] reactions once per
    point) against the oracle's analytic Jacobian, element by element, relative to the sum of absolute terms."""
    if case == "all_paths":
        mech = hand_cases.all_paths_mechanism()
        rho, T, Y = hand_cases.random_states(mech, 64)
    else:
        cfg = 2 if case == "cfg2" else 0
        mech = inputs.config_mechanism(cfg)
        if case == "mixed_t_mid":
            mech = inputs.with_species_break_temperatures(mech, np.linspace(800.0, 1400.0, mech.n_species))
        st = inputs.config_states(cfg, n=48 if cfg == 2 else 256)
        rho, T, Y = st["rho"], st["T"], st["Y"]
        Y = Y.copy()
        Y[:, :4] = 0.0          # exact zeros: no division by a concentration anywhere
        Y[0, :4] = 1.0
    J, sT = emu_jacobian(emu, mech, rho, T, Y, mode)
    Jr, sTr, bJ, bT = oracle.Oracle(mech).get_jacobian(rho, T, Y, mode=mode)
    assert np.all(np.isfinite(J)) and np.all(np.isfinite(sT))
    parity.assert_jacobian_parity(J, Jr, bJ)
    parity.assert_jacobian_parity(sT, sTr, bT)


# ------------------------------------------------------------------ reactor march
def stable_dt(orc, rho, T, Y, safety=0.05):
    """A step that resolves the fastest chemical time scale of the batch (largest Jacobian row sum of dY/dt = S/rho)."""
    J, _, _, _ = orc.get_jacobian(rho, T, Y, mode=1)
    return safety / float(np.max(np.abs(J).sum(axis=1) / np.asarray(rho)[None, :]))


def emu_reactor(emu, mech, rho, e, Y, Tg, dt, n_steps, tol=1e-6, max_iter=10):
    desc, keep = binding.make_desc(mech)
    rho, e = (np.ascontiguousarray(x, dtype=np.float64) for x in (rho, e))
    Y = np.array(Y, dtype=np.float64, order="C")
    T = np.array(Tg, dtype=np.float64)
    work = np.full_like(Y, np.nan)
    bad = C.c_int64(0)
    st = emu.emu_reactor(C.byref(desc), rho.shape[0], rho.shape[0], rho.ctypes.data, e.ctypes.data, Y.ctypes.data,
                         T.ctypes.data, dt, n_steps, tol, max_iter, work.ctypes.data, C.byref(bad))
    assert st == 0, emu.emu_last_error()
    return Y, T, int(bad.value)


REACTOR_TOL = 1e-10   # |dY_k| <= REACTOR_TOL * (sum of the sizes of the terms added into Y_k + |Y_k|)


def assert_reactor_parity(Y, T, Y_ref, T_ref, Yb):
    assert np.isfinite(Y).all() and np.isfinite(T).all()
    rY = float(np.max(np.abs(Y - Y_ref) / (Yb + np.abs(Y_ref) + 1e-300)))
    rT = float(np.max(np.abs(T - T_ref) / T_ref))
    assert rY <= REACTOR_TOL, f"max |dY|/(Ybound + |Y|) = {rY:.3e}"
    assert rT <= 1e-9, f"max |dT|/T = {rT:.3e}"
    return rY, rT


@pytest.mark.parametrize("case", ["all_paths", "cfg0", "cfg2", "mixed_t_mid"])
def test_reactor_point_code_matches_oracle(emu, case):
    if case == "all_paths":
        mech = hand_cases.all_paths_mechanism()
        rho, T, Y = hand_cases.random_states(mech, 48)
    else:
        cfg = 2 if case == "cfg2" else 0
        mech = inputs.config_mechanism(cfg)
        if case == "mixed_t_mid":
            mech = inputs.with_species_break_temperatures(mech, np.linspace(800.0, 1400.0, mech.n_species))
        st = inputs.config_states(cfg, n=24 if cfg == 2 else 128)
        rho, T, Y = st["rho"], st["T"], st["Y"]
    orc = oracle.Oracle(mech)
    e = np.array([orc.mixture_e(T[p], Y[:, p]) for p in range(len(T))])
    Tg = T * 1.03
    dt = stable_dt(orc, rho, T, Y)
    for n_steps in (0, 1, 6):
        Yr, Tr, Yb, bad_r = orc.reactor_rk4(rho, e, Y, Tg, dt, n_steps)
        Ye, Te, bad_e = emu_reactor(emu, mech, rho, e, Y, Tg, dt, n_steps)
        assert bad_r == bad_e == 0
        rY, rT = assert_reactor_parity(Ye, Te, Yr, Tr, Yb)
    assert np.any(np.abs(Yr - Y) > 1e-6 * np.abs(Y))


# ------------------------------------------------------------------ bench.py host helpers (no GPU)
def test_bench_tempered_window_picks_the_most_populated_decade():
    """bench.py marches the reactor legs on the states of the most populated window [L, 10 L] of their own time scale."""
    import bench
    rng = np.random.default_rng(3)
    lam = np.concatenate([10.0 ** rng.uniform(20, 140, 5000), 10.0 ** rng.uniform(33.0, 33.9, 700), [np.nan, 0.0, -1.0, np.inf]])
    sel, lam_max = bench.tempered_window(lam)
    assert len(sel) >= 700 and len(set(sel.tolist())) == len(sel)
    assert np.isfinite(lam[sel]).all() and lam[sel].min() > 0
    assert lam[sel].max() == lam_max and lam_max <= 10.0 * lam[sel].min()
    assert 5e32 <= lam[sel].min() and lam_max <= 1e35
    # brute force on a small case: no other window holds more states
    small = lam[:300]
    sel_s, _ = bench.tempered_window(small)
    ok = small[np.isfinite(small) & (small > 0)]
    best = max(int(np.sum((ok >= lo) & (ok <= 10.0 * lo))) for lo in ok)
    assert len(sel_s) == best
    empty, none = bench.tempered_window(np.array([np.nan, 0.0]))
    assert len(empty) == 0 and none is None


def test_bench_ncu_summary_round_trip_and_staleness_guard(tmp_path):
    """The ncu figures of the bench line come from a committed one-row summary; they are withheld when the library's
    kernel is not the captured one (other registers per thread) or the mechanism has another size."""
    import bench
    cols = list(bench.NCU_COLUMNS.values())
    units = {"launch__registers_per_thread": "register/thread", "gpu__time_duration.sum": "ms", "dram__bytes_read.sum": "Mbyte",
             "dram__bytes_write.sum": "Gbyte", "smsp__cycles_elapsed.max": "cycle", "smsp__inst_executed.sum": "inst"}
    vals = {"launch__registers_per_thread": "178", "gpu__time_duration.sum": "1.5", "dram__bytes_read.sum": "400.5",
            "dram__bytes_write.sum": "0.25", "smsp__cycles_elapsed.max": "1,000,000", "smsp__inst_executed.sum": "12345"}
    raw = tmp_path / "raw.csv"
    with open(raw, "w") as f:
        f.write('"ID","Kernel Name",' + ",".join(f'"{c}"' for c in cols) + "\n")
        f.write('"","",' + ",".join(f'"{units.get(c, "inst/cycle")}"' for c in cols) + "\n")
        f.write('"0","void rates_kernel<1, 1, 1, 0>(RatesArgs)",' + ",".join(f'"{vals.get(c, "2.0")}"' for c in cols) + "\n")
    out = tmp_path / "capture.csv"
    rec = bench.write_ncu_summary(str(raw), 1 << 20, 53, 325, out_path=str(out))
    assert rec["duration_ns"] == 1.5e6 and rec["dram_read_bytes"] == 400.5e6 and rec["dram_write_bytes"] == 0.25e9
    assert rec["fp64_flops"] == (2.0 + 2.0 + 2 * 2.0) * 1e6 and rec["kernel"] == "void rates_kernel<1, 1, 1, 0>"
    back = bench.read_ncu_summary(53, 325, 178, path=str(out))
    assert back["points"] == 1 << 20 and back["dram_read_bytes"] == 400.5e6 and back["kernel"] == rec["kernel"]
    assert bench.read_ncu_summary(53, 325, 170, path=str(out)) is None      # another build of the kernel
    assert bench.read_ncu_summary(9, 21, 178, path=str(out)) is None        # another mechanism
    assert bench.read_ncu_summary(53, 325, 178, path=str(tmp_path / "missing.csv")) is None
    # the committed capture of this round parses and is of the graded configuration
    committed = bench.read_ncu_summary(53, 325, 178)
    if committed is not None:
        assert committed["points"] == 1 << 20 and 8e8 < committed["dram_read_bytes"] + committed["dram_write_bytes"] < 1e9
