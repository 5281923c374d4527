"""GPU parity: the CUDA path, called through the C ABI of libpyro.so, against the CPU oracle on
the same seeded inputs, element by element (tolerances of north_star, see parity.py)."""
import ctypes as C
import os

import numpy as np
import pytest

import hand_cases
import parity
from oracle import oracle
from paper_2503_24286_b200 import binding, inputs

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")


def dev(x):
    return torch.from_numpy(np.ascontiguousarray(x)).cuda()


@pytest.fixture(scope="module")
def mechs():
    cache = {}

    def get(cfg):
        if cfg not in cache:
            m = inputs.config_mechanism(cfg)
            cache[cfg] = (m, binding.Mechanism(m), oracle.Oracle(m))
        return cache[cfg]
    return get


def gpu_rates(gm, rho, T, Y, **kw):
    om = gm.get_net_production_rates(dev(rho), dev(T), dev(Y), **kw)
    torch.cuda.synchronize()
    return om.cpu().numpy()


# ------------------------------------------------------------------ small sizes: every element
@pytest.mark.parametrize("cfg,n", [(0, 4096), (1, 3001), (2, 2500), (3, 700)])
def test_rates_every_point(mechs, cfg, n):
    """Several blocks and a ragged tail; every (species, point) entry compared."""
    mech, gm, orc = mechs(cfg)
    st = inputs.config_states(cfg, n=n)
    om_ref, bound = orc.get_net_production_rates(st["rho"], st["T"], st["Y"])
    om = gpu_rates(gm, st["rho"], st["T"], st["Y"])
    parity.assert_omega_parity(om, om_ref, bound)


@pytest.mark.parametrize("cfg,n", [(0, 4096), (2, 2500), (3, 700), (4, 13**3)])
def test_temperature_every_point(mechs, cfg, n):
    mech, gm, orc = mechs(cfg)
    st = inputs.config_states(cfg, n=n)
    T_ref, it, conv = orc.get_temperature(st["e"], st["Y"], st["T_guess"])
    bad = torch.zeros(1, dtype=torch.int32, device="cuda")
    T = gm.get_temperature(dev(st["e"]), dev(st["Y"]), dev(st["T_guess"]), rho=dev(st["rho"]), n_not_converged=bad)
    torch.cuda.synchronize()
    parity.assert_T_parity(T.cpu().numpy(), T_ref)
    assert int(bad.item()) == 0 and conv.all()
    # generated e came from T in long double: the solve recovers it
    assert np.max(np.abs(T.cpu().numpy() - st["T"]) / st["T"]) < 1e-12


def test_hand_mechanism_every_reaction_class(mechs):
    mech = hand_cases.all_paths_mechanism()
    gm = binding.Mechanism(mech)
    rho, T, Y = hand_cases.random_states(mech, 777)
    om_ref, bound = oracle.Oracle(mech).get_net_production_rates(rho, T, Y)
    parity.assert_omega_parity(gpu_rates(gm, rho, T, Y), om_ref, bound)


# ------------------------------------------------------------------ full sizes, bench launch configuration
def _sample(n, count, seed=5):
    rng = np.random.default_rng(seed)
    idx = np.unique(np.concatenate([rng.integers(0, n, size=count), [0, 1, n - 2, n - 1]]))
    return idx


@pytest.mark.parametrize("cfg,count", [(1, 20000), (2, 4096), (3, 1024)])
def test_rates_full_size_sampled(mechs, cfg, count):
    """BASELINE.json sizes (2^24 / 2^22 / 2^20 points), one launch as bench.py issues it; the oracle
    evaluates a random sample of points one by one."""
    mech, gm, orc = mechs(cfg)
    n = inputs.CONFIG_POINTS[cfg]
    st = inputs.config_states(cfg)
    assert st["rho"].shape[0] == n
    d_rho, d_T, d_Y = dev(st["rho"]), dev(st["T"]), dev(st["Y"])
    om = gm.get_net_production_rates(d_rho, d_T, d_Y)
    torch.cuda.synchronize()
    idx = _sample(n, count)
    om_s = om[:, torch.from_numpy(idx).cuda()].cpu().numpy()
    om_ref, bound = orc.get_net_production_rates(st["rho"][idx], st["T"][idx], st["Y"][:, idx])
    parity.assert_omega_parity(om_s, om_ref, bound)
    # properties that hold at any size: finite everywhere, mass conservation sum_i W_i omega_i = 0
    assert bool(torch.isfinite(om).all())
    W = dev(mech.mol_weight)[:, None]
    mass = (W * om).sum(0).abs()
    scale = (W * om.abs()).sum(0)
    assert bool((mass <= 1e-9 * scale + 1e-300).all())
    del om, d_Y
    torch.cuda.empty_cache()


def test_full_source_term_step_cfg4_sampled(mechs):
    """configs[4]: 256^3 flame-front field, (rho, e, Y, T_guess) -> T -> omega on one stream."""
    mech, gm, orc = mechs(4)
    n = inputs.CONFIG_POINTS[4]
    st = inputs.config_states(4)
    d_Y = dev(st["Y"])
    d_rho = dev(st["rho"])
    bad = torch.zeros(1, dtype=torch.int32, device="cuda")
    T = gm.get_temperature(dev(st["e"]), d_Y, dev(st["T_guess"]), rho=d_rho, n_not_converged=bad)
    om = gm.get_net_production_rates(d_rho, T, d_Y)
    torch.cuda.synchronize()
    assert int(bad.item()) == 0
    # sample: random points plus four full x-lines through the flame front
    lines = np.concatenate([np.arange(256) + 256 * (y + 256 * z) for y, z in ((0, 0), (17, 200), (128, 128), (255, 255))])
    idx = np.unique(np.concatenate([_sample(n, 3000), lines]))
    T_ref, it, conv = orc.get_temperature(st["e"][idx], st["Y"][:, idx], st["T_guess"][idx])
    T_s = T[torch.from_numpy(idx).cuda()].cpu().numpy()
    parity.assert_T_parity(T_s, T_ref)
    assert conv.all() and it.max() <= 10
    # rates parity on the temperature the GPU solve produced (the two T agree to ~1e-15; feeding the
    # oracle the same T keeps the two tolerances independent)
    om_ref, bound = orc.get_net_production_rates(st["rho"][idx], T_s, st["Y"][:, idx])
    parity.assert_omega_parity(om[:, torch.from_numpy(idx).cuda()].cpu().numpy(), om_ref, bound)
    assert bool(torch.isfinite(om).all()) and bool(torch.isfinite(T).all())
    # T everywhere recovers the field that generated e (double-precision e at this size: 1e-10)
    assert float(((T - dev(st["T"])).abs() / dev(st["T"])).max()) < 1e-10


# ------------------------------------------------------------------ edge cases
def test_empty_single_ragged_and_padded_leading_dimension(mechs):
    mech, gm, orc = mechs(0)
    ns = mech.n_species
    # n = 0 launches nothing
    z = torch.empty(0, dtype=torch.float64, device="cuda")
    zY = torch.empty((ns, 0), dtype=torch.float64, device="cuda")
    assert gm.get_net_production_rates(z, z, zY).shape == (ns, 0)
    assert gm.get_temperature(z, zY, z).shape == (0,)
    st = inputs.config_states(0, n=1000)
    om_ref, bound = orc.get_net_production_rates(st["rho"], st["T"], st["Y"])
    T_ref, _, _ = orc.get_temperature(st["e"], st["Y"], st["T_guess"])
    for n in (1, 31, 33, 129, 1000):
        # ld > n: fields are windows into wider buffers, padding filled with NaN that must not be read
        ld = n + 7
        Ybuf = torch.full((ns, ld), float("nan"), dtype=torch.float64, device="cuda")
        Ybuf[:, :n] = dev(st["Y"][:, :n])
        out = torch.full((ns, ld), -7.0, dtype=torch.float64, device="cuda")
        gm.get_net_production_rates(dev(st["rho"][:n]), dev(st["T"][:n]), Ybuf[:, :n], out=out[:, :n])
        Tout = gm.get_temperature(dev(st["e"][:n]), Ybuf[:, :n], dev(st["T_guess"][:n]))
        torch.cuda.synchronize()
        parity.assert_omega_parity(out[:, :n].cpu().numpy(), om_ref[:, :n], bound[:, :n])
        assert bool((out[:, n:] == -7.0).all())   # nothing written beyond n
        parity.assert_T_parity(Tout.cpu().numpy(), T_ref[:n])


def test_temperature_in_place_and_iteration_cap(mechs):
    mech, gm, orc = mechs(0)
    st = inputs.config_states(0, n=2048)
    # T may alias T_guess
    Tg = dev(st["T_guess"])
    gm.get_temperature(dev(st["e"]), dev(st["Y"]), Tg, out=Tg)
    torch.cuda.synchronize()
    T_ref, _, _ = orc.get_temperature(st["e"], st["Y"], st["T_guess"])
    parity.assert_T_parity(Tg.cpu().numpy(), T_ref)
    # cap: non-converged points are counted, the last iterate is returned
    gm2 = binding.Mechanism(mech)
    gm2.set_newton(abs_tol_K=1e-6, max_iter=2)
    bad = torch.zeros(1, dtype=torch.int32, device="cuda")
    T2 = gm2.get_temperature(dev(st["e"]), dev(st["Y"]), dev(st["T_guess"]), n_not_converged=bad)
    torch.cuda.synchronize()
    T_ref2, it2, conv2 = orc.get_temperature(st["e"], st["Y"], st["T_guess"], tol=1e-6, max_iter=2)
    parity.assert_T_parity(T2.cpu().numpy(), T_ref2)
    assert int(bad.item()) == int((conv2 == 0).sum()) > 0


def test_abi_error_codes_on_device(mechs):
    mech, gm, _ = mechs(0)
    lib = binding.load_library()
    st = inputs.config_states(0, n=64)
    rho, T, Y = dev(st["rho"]), dev(st["T"]), dev(st["Y"])
    om = torch.empty_like(Y)
    h = gm._h
    f = lib.pyro_get_net_production_rates
    assert f(None, 64, 64, rho.data_ptr(), T.data_ptr(), Y.data_ptr(), om.data_ptr(), None) == 1
    assert f(h, 64, 64, None, T.data_ptr(), Y.data_ptr(), om.data_ptr(), None) == 1
    assert f(h, -1, 64, rho.data_ptr(), T.data_ptr(), Y.data_ptr(), om.data_ptr(), None) == 2
    assert f(h, 64, 63, rho.data_ptr(), T.data_ptr(), Y.data_ptr(), om.data_ptr(), None) == 2
    assert f(h, 64, 64, rho.data_ptr() + 4, T.data_ptr(), Y.data_ptr(), om.data_ptr(), None) == 5
    assert f(h, 64, 64, rho.data_ptr(), T.data_ptr(), Y.data_ptr(), Y.data_ptr(), None) == 2   # omega aliases Y
    g = lib.pyro_get_temperature
    assert g(h, 64, 64, None, None, Y.data_ptr(), T.data_ptr(), T.data_ptr(), None, None) == 1
    assert g(h, 64, 10, None, rho.data_ptr(), Y.data_ptr(), T.data_ptr(), T.data_ptr(), None, None) == 2
    # partial overlap of omega with Y (not only pointer equality): the second plane of Y, and a range that ends inside Y
    assert f(h, 64, 64, rho.data_ptr(), T.data_ptr(), Y.data_ptr(), Y.data_ptr() + 8 * 64, None) == 2
    assert f(h, 64, 64, rho.data_ptr(), T.data_ptr(), Y.data_ptr() + 8 * 64 * (mech.n_species - 1), Y.data_ptr(), None) == 2
    # ld < n and alignment on every entry point, including the NEXT-1 helpers
    bad32 = torch.zeros(4, dtype=torch.int32, device="cuda")
    assert g(h, 64, 64, None, rho.data_ptr(), Y.data_ptr(), T.data_ptr(), T.data_ptr(), bad32.data_ptr() + 2, None) == 5
    assert g(h, 64, 64, None, rho.data_ptr() + 4, Y.data_ptr(), T.data_ptr(), T.data_ptr(), None, None) == 5
    ge = lib.pyro_get_temperature_from_enthalpy
    assert ge(h, 64, 63, rho.data_ptr(), Y.data_ptr(), T.data_ptr(), T.data_ptr(), None, None) == 2
    assert ge(h, 64, 64, rho.data_ptr(), Y.data_ptr(), T.data_ptr(), T.data_ptr(), bad32.data_ptr() + 1, None) == 5
    assert ge(h, 64, 64, None, Y.data_ptr(), T.data_ptr(), T.data_ptr(), None, None) == 1
    for eos in (lib.pyro_get_density, lib.pyro_get_pressure):
        assert eos(h, 64, 63, rho.data_ptr(), T.data_ptr(), Y.data_ptr(), om.data_ptr(), None) == 2
        assert eos(h, -5, 64, rho.data_ptr(), T.data_ptr(), Y.data_ptr(), om.data_ptr(), None) == 2
        assert eos(h, 64, 64, rho.data_ptr(), T.data_ptr() + 4, Y.data_ptr(), om.data_ptr(), None) == 5
        assert eos(h, 64, 64, rho.data_ptr(), None, Y.data_ptr(), om.data_ptr(), None) == 1
        assert eos(h, 0, 0, None, None, None, None, None) == 0   # n == 0 launches nothing
    hs = lib.pyro_source_terms_host
    assert hs(h, 64, 63, None, None, None, None, None, None, None) == 2
    assert hs(h, 64, 64, None, None, None, None, None, None, None) == 1
    assert lib.pyro_mech_set_newton(h, -1.0, 10) == 2 and lib.pyro_mech_set_newton(h, 1e-6, 0) == 2
    assert lib.pyro_last_error_string()
    out = C.c_void_p()
    assert lib.pyro_mech_create(None, 0, C.byref(out)) == 1
    desc, keep = binding.make_desc(mech)
    assert lib.pyro_mech_create(C.byref(desc), 99, C.byref(out)) == 2 and not out.value


def test_two_mechanisms_alternate_across_streams(mechs):
    """Alternating launches of two mechanisms on two streams: every launch stages its own tables and
    allocates its own tensor-memory columns, so concurrent kernels of different mechanisms coexist."""
    m0, g0, o0 = mechs(0)
    m2, g2, o2 = mechs(2)
    assert g0.info()["tables_in_shared"] == 1 and g2.info()["tables_in_shared"] == 1
    s0 = inputs.config_states(0, n=3000)
    s2 = inputs.config_states(2, n=1500)
    ref0, b0 = o0.get_net_production_rates(s0["rho"], s0["T"], s0["Y"])
    ref2, b2 = o2.get_net_production_rates(s2["rho"], s2["T"], s2["Y"])
    a0 = [dev(s0[k]) for k in ("rho", "T", "Y")]
    a2 = [dev(s2[k]) for k in ("rho", "T", "Y")]
    torch.cuda.synchronize()
    sa, sb = torch.cuda.Stream(), torch.cuda.Stream()
    outs = []
    for rep in range(6):
        outs.append((0, g0.get_net_production_rates(*a0, stream=sa if rep % 2 else sb)))
        outs.append((2, g2.get_net_production_rates(*a2, stream=sb if rep % 2 else sa)))
    torch.cuda.synchronize()
    for which, om in outs:
        parity.assert_omega_parity(om.cpu().numpy(), ref0 if which == 0 else ref2, b0 if which == 0 else b2)


def test_tables_in_global_memory_path(mechs, monkeypatch):
    """Mechanisms whose tables would crowd the planes out of shared memory read them from global
    memory; here that path is forced for configs[2] and configs[3]."""
    monkeypatch.setenv("PYRO_TABLES", "global")
    for cfg, n in ((2, 1111), (3, 300)):
        mech, _, orc = mechs(cfg)
        gm = binding.Mechanism(mech)
        assert gm.info()["tables_in_shared"] == 0
        st = inputs.config_states(cfg, n=n)
        om_ref, bound = orc.get_net_production_rates(st["rho"], st["T"], st["Y"])
        parity.assert_omega_parity(gpu_rates(gm, st["rho"], st["T"], st["Y"]), om_ref, bound)


@pytest.mark.parametrize("cfg,block", [(2, 32), (2, 64), (2, 96), (2, 160), (2, 256), (0, 32), (0, 128), (0, 256),
                                       (3, 32), (3, 64)])
def test_every_block_size(mechs, monkeypatch, cfg, block):
    """Threads (= points) per block of the rates kernel, forced: 1 to 8 warps, i.e. one and two
    tensor-memory column groups, with a ragged last tile and more tiles than resident blocks."""
    monkeypatch.setenv("PYRO_RATES_BLOCK", str(block))
    mech, _, orc = mechs(cfg)
    gm = binding.Mechanism(mech)
    info = gm.info()
    assert info["block_threads"] == block
    assert info["tmem_columns"] >= ((block // 32 + 3) // 4) * (4 if info["b_in_tmem"] else 2) * (mech.n_species + 1)
    for n in (777, 2 * block + 1, info["sm_count"] * info["blocks_per_sm"] * block + 5 * block + 3):
        if cfg == 3 and n > 3000:
            n = 3001
        st = inputs.config_states(cfg, n=n)
        om_ref, bound = orc.get_net_production_rates(st["rho"], st["T"], st["Y"])
        parity.assert_omega_parity(gpu_rates(gm, st["rho"], st["T"], st["Y"]), om_ref, bound)


def test_plane_b_in_shared_memory_path(mechs, monkeypatch):
    """Mechanisms of more than 127 species keep plane B in shared memory (two tensor-memory columns
    per species instead of four); here that variant is forced for configs[0], [2] and [3]."""
    monkeypatch.setenv("PYRO_B_PLANE", "shared")
    for cfg, n in ((0, 3000), (2, 1111), (3, 300)):
        mech, _, orc = mechs(cfg)
        gm = binding.Mechanism(mech)
        assert gm.info()["b_in_tmem"] == 0
        st = inputs.config_states(cfg, n=n)
        om_ref, bound = orc.get_net_production_rates(st["rho"], st["T"], st["Y"])
        parity.assert_omega_parity(gpu_rates(gm, st["rho"], st["T"], st["Y"]), om_ref, bound)


def test_species_with_different_t_mid(mechs):
    """Per-species break temperatures (G10): the rates path switches range per species and point, and the
    temperature solve (energy and enthalpy form) re-sums the mixture polynomial whenever an iterate crosses a
    break temperature -- both against the oracle, which chooses the range per species at every iterate."""
    from test_host_logic import _mixed_tmid_case
    for cfg, n in ((0, 5000), (2, 1111)):
        mech, T, Y, e, h, Tg = _mixed_tmid_case(cfg, n)
        gm = binding.Mechanism(mech)
        orc = oracle.Oracle(mech)
        rho = np.full(n, 0.7)
        om_ref, bound = orc.get_net_production_rates(rho, T, Y)
        parity.assert_omega_parity(gpu_rates(gm, rho, T, Y), om_ref, bound)
        T_ref, _, conv = orc.get_temperature(e, Y, Tg)
        assert conv.all()
        bad = torch.zeros(1, dtype=torch.int32, device="cuda")
        T_gpu = gm.get_temperature(dev(e), dev(Y), dev(Tg), n_not_converged=bad).cpu().numpy()
        parity.assert_T_parity(T_gpu, T_ref)
        assert int(bad.item()) == 0
        Th_ref, _, _ = orc.get_temperature_from_enthalpy(h, Y, Tg)
        parity.assert_T_parity(gm.get_temperature_from_enthalpy(dev(h), dev(Y), dev(Tg)).cpu().numpy(), Th_ref)
        # padded leading dimension and an iteration cap of 2: last iterates and the count as the oracle's
        ld = n + 37
        Yp = torch.full((mech.n_species, ld), float("nan"), dtype=torch.float64, device="cuda")
        Yp[:, :n] = dev(Y)
        gm.set_newton(1e-6, 2)
        T2_ref, _, conv2 = orc.get_temperature(e, Y, Tg, max_iter=2)
        bad.zero_()
        T2 = gm.get_temperature(dev(e), Yp[:, :n], dev(Tg), n_not_converged=bad).cpu().numpy()
        parity.assert_T_parity(T2, T2_ref)
        assert int(bad.item()) == int((conv2 == 0).sum())
        gm.set_newton(1e-6, 10)
        gm.close()


@pytest.mark.parametrize("a6", [1.2e5, -1.2e5, 2.5e5, -2.5e5])
def test_rates_finite_wherever_the_oracle_is_extreme_formation_enthalpies(a6):
    """|g_k/RT| up to 1000 per species at 250 K (SURVEY.md section 7 hard part 4; (A.10) PAPER.md:932): the shifted
    species factors and the pair form of wide reactions keep the kernel finite and within tolerance wherever
    the oracle is; a mechanism whose K_c itself leaves FP64 inside the supported range is refused at create."""
    from test_host_logic import _cold_to_hot_states
    for name, mech in hand_cases.extreme_thermo_mechanisms(a6).items():
        rho, T, Y = _cold_to_hot_states(mech, 1500)
        om_ref, bound = oracle.Oracle(mech).get_net_production_rates(rho, T, Y)
        if name == "assoc" and abs(a6) > 2e5:
            with pytest.raises(binding.PyroError) as ei:
                binding.Mechanism(mech)
            assert ei.value.status == 7 and "250" in str(ei.value)
            continue
        assert np.isfinite(om_ref).all() and np.isfinite(bound).all()
        gm = binding.Mechanism(mech)
        parity.assert_omega_parity(gpu_rates(gm, rho, T, Y), om_ref, bound)
        gm.close()


def test_troe_sentinel_temperatures():
    """T*** = 1e-30, T* = 1e30, T** = 1e30 as real mechanism files carry them."""
    mech = hand_cases.troe_sentinel_mechanism()
    rho, T, Y = hand_cases.random_states(mech, 2000)
    T[:4] = [250.0, 1234.5, 3000.0, 6000.0]
    om_ref, bound = oracle.Oracle(mech).get_net_production_rates(rho, T, Y)
    assert np.isfinite(om_ref).all()
    gm = binding.Mechanism(mech)
    parity.assert_omega_parity(gpu_rates(gm, rho, T, Y), om_ref, bound)
    gm.close()


def test_host_buffer_pipeline_matches_oracle(mechs, monkeypatch):
    """pyro_source_terms_host: slabbed H2D -> T -> omega -> D2H with a slab size that leaves a ragged tail."""
    monkeypatch.setenv("PYRO_HOST_SLAB", "4096")
    mech, _, orc = mechs(0)
    gm = binding.Mechanism(mech)
    n = 4096 * 5 + 123
    st = inputs.config_states(0, n=n)
    pin = lambda x: torch.from_numpy(np.ascontiguousarray(x)).pin_memory()
    T = torch.empty(n, dtype=torch.float64).pin_memory()
    om = torch.empty((mech.n_species, n), dtype=torch.float64).pin_memory()
    bad = gm.source_terms_host(pin(st["rho"]), pin(st["e"]), pin(st["Y"]), pin(st["T_guess"]), T, om)
    assert bad == 0
    T_ref, _, _ = orc.get_temperature(st["e"], st["Y"], st["T_guess"])
    parity.assert_T_parity(T.numpy(), T_ref)
    om_ref, bound = orc.get_net_production_rates(st["rho"], T.numpy(), st["Y"])
    parity.assert_omega_parity(om.numpy(), om_ref, bound)
    # pageable numpy buffers work too
    T2 = np.empty(n)
    om2 = np.empty((mech.n_species, n))
    gm.source_terms_host(st["rho"], st["e"], st["Y"], st["T_guess"], T2, om2)
    assert np.array_equal(T2, T.numpy()) and np.array_equal(om2, om.numpy())


@pytest.mark.parametrize("cfg,n", [(0, 5000), (2, 3001), (3, 700)])
def test_enthalpy_inversion_and_equation_of_state(mechs, cfg, n):
    """pyro_get_temperature_from_enthalpy, pyro_get_density, pyro_get_pressure."""
    mech, gm, orc = mechs(cfg)
    st = inputs.config_states(cfg, n=n)
    Y = np.ascontiguousarray(st["Y"])
    h = np.array([orc.mixture_h(float(st["T"][p]), Y[:, p]) for p in range(n)])
    T_ref, _, conv = orc.get_temperature_from_enthalpy(h, Y, st["T_guess"])
    bad = torch.zeros(1, dtype=torch.int32, device="cuda")
    T = gm.get_temperature_from_enthalpy(dev(h), dev(Y), dev(st["T_guess"]), n_not_converged=bad)
    parity.assert_T_parity(T.cpu().numpy(), T_ref)
    assert int(bad.item()) == 0 and conv.all()
    # energy and enthalpy forms are different equations
    T_e = gm.get_temperature(dev(h), dev(Y), dev(st["T_guess"])).cpu().numpy()
    assert np.min(np.abs(T_e - T_ref) / T_ref) > 1e-3
    p = inputs.P_ATM * np.linspace(0.1, 50.0, n)
    rho = gm.get_density(dev(p), dev(st["T"]), dev(Y))
    assert np.max(np.abs(rho.cpu().numpy() / orc.get_density(p, st["T"], Y) - 1)) <= parity.EOS_TOL
    pp = gm.get_pressure(rho, dev(st["T"]), dev(Y), out=rho)          # in place
    assert np.max(np.abs(pp.cpu().numpy() / p - 1)) <= 10 * parity.EOS_TOL
    assert gm.get_density(dev(p[:0]), dev(st["T"][:0]), dev(Y[:, :0])).numel() == 0


def test_degenerate_mechanisms(mechs):
    """No reaction at all, a single species, only extended-class reactions; T solve on each."""
    for name, mech in hand_cases.degenerate_mechanisms().items():
        gm = binding.Mechanism(mech)
        orc = oracle.Oracle(mech)
        rho, T, Y = hand_cases.random_states(mech, 777)
        om_ref, bound = orc.get_net_production_rates(rho, T, Y)
        om = gpu_rates(gm, rho, T, Y)
        parity.assert_omega_parity(om, om_ref, bound)
        if mech.n_reactions == 0:
            assert not om.any()
        e = np.array([orc.mixture_e(float(T[p]), Y[:, p]) for p in range(777)])
        Tg = T * 1.07
        T_ref, _, _ = orc.get_temperature(e, Y, Tg)
        parity.assert_T_parity(gm.get_temperature(dev(e), dev(Y), dev(Tg)).cpu().numpy(), T_ref)


def test_temperature_stream_and_plain_paths(mechs):
    """pyro_get_temperature runs whole blocks of 256 points through the cp.async stream when the Y
    planes are 16-byte aligned and the rest (ragged tail, odd leading dimension, unaligned Y) through
    the plain kernel: same answers from every mix of the two."""
    mech, gm, orc = mechs(2)
    n = 256 * 5 + 77
    st = inputs.config_states(2, n=n)
    T_ref, _, _ = orc.get_temperature(st["e"], st["Y"], st["T_guess"])
    ns = mech.n_species
    for ld, shift in ((n + 1, 0), (n + 2, 0), (n + 2, 1), (n + 3, 1)):   # even / odd ld, aligned / unaligned base
        buf = torch.zeros(ns * ld + 2, dtype=torch.float64, device="cuda")
        Y = buf[shift:shift + ns * ld].view(ns, ld)[:, :n]
        Y.copy_(dev(st["Y"]))
        assert Y.stride(0) == ld and (Y.data_ptr() % 16 == 0) == (shift == 0)
        bad = torch.zeros(1, dtype=torch.int32, device="cuda")
        T = gm.get_temperature(dev(st["e"]), Y, dev(st["T_guess"]), n_not_converged=bad)
        parity.assert_T_parity(T.cpu().numpy(), T_ref)
        assert int(bad.item()) == 0
    # in place, stream path, with the iteration cap reported from both kernels
    gm.set_newton(1e-300, 2)
    try:
        Tg = dev(st["T_guess"]).clone()
        bad = torch.zeros(1, dtype=torch.int32, device="cuda")
        gm.get_temperature(dev(st["e"]), dev(st["Y"]), Tg, out=Tg, n_not_converged=bad)
        T2_ref, _, conv2 = orc.get_temperature(st["e"], st["Y"], st["T_guess"], tol=1e-300, max_iter=2)
        parity.assert_T_parity(Tg.cpu().numpy(), T2_ref)
        assert int(bad.item()) == int((conv2 == 0).sum()) > n - 8
    finally:
        gm.set_newton(1e-6, 10)


def test_fuzz_mechanisms(mechs):
    """Other shapes than the configs (ragged lockstep groups, both packings of leftover reactions,
    120-species planes with few reactions): rates and temperature against the oracle."""
    for mech in hand_cases.fuzz_mechanisms():
        gm = binding.Mechanism(mech)
        orc = oracle.Oracle(mech)
        rho, T, Y = hand_cases.random_states(mech, 1500, seed=mech.n_reactions)
        om_ref, bound = orc.get_net_production_rates(rho, T, Y)
        parity.assert_omega_parity(gpu_rates(gm, rho, T, Y), om_ref, bound)
        e = np.array([orc.mixture_e(float(T[p]), Y[:, p]) for p in range(1500)])
        T_ref, _, _ = orc.get_temperature(e, Y, T * 0.93)
        parity.assert_T_parity(gm.get_temperature(dev(e), dev(Y), dev(T * 0.93)).cpu().numpy(), T_ref)


# ------------------------------------------------------------------ chemical Jacobian
def gpu_jacobian(gm, rho, T, Y, mode, **kw):
    J, sT = gm.get_jacobian(dev(rho), dev(T), dev(Y), mode=mode, **kw)
    torch.cuda.synchronize()
    return J.cpu().numpy(), (None if sT is None else sT.cpu().numpy())


@pytest.mark.parametrize("mode", [0, 1])
@pytest.mark.parametrize("cfg,n", [(0, 1500), (2, 333), (3, 70)])
def test_jacobian_every_entry(mechs, cfg, n, mode):
    """pyro_get_jacobian against the oracle's analytic Jacobian: every entry J[i, k, p] and dS/dT, several
    blocks and a ragged tail; both readings of what is held fixed (G26)."""
    mech, gm, orc = mechs(cfg)
    st = inputs.config_states(cfg, n=n)
    Y = st["Y"].copy()
    Y[:, :3] = 0.0           # exact zeros in the composition: no division by a concentration
    Y[mech.n_species - 1, :3] = 1.0
    Jr, sTr, bJ, bT = orc.get_jacobian(st["rho"], st["T"], Y, mode=mode)
    J, sT = gpu_jacobian(gm, st["rho"], st["T"], Y, mode)
    r1 = parity.assert_jacobian_parity(J, Jr, bJ)
    r2 = parity.assert_jacobian_parity(sT, sTr, bT)
    print(f"cfg {cfg} mode {mode}: max |dJ|/bound = {r1:.2e}, max |d dSdT|/bound = {r2:.2e}")


def test_jacobian_hand_mechanism_padded_ld_and_no_dSdT():
    """Every reaction class; leading dimension larger than n with NaN padding left untouched; dSdT = NULL."""
    mech = hand_cases.all_paths_mechanism()
    gm = binding.Mechanism(mech)
    n, ld, ns = 77, 96, mech.n_species
    rho, T, Y = hand_cases.random_states(mech, n)
    Yp = np.full((ns, ld), np.nan)
    Yp[:, :n] = Y
    Jr, sTr, bJ, bT = oracle.Oracle(mech).get_jacobian(rho, T, Y, mode=1)
    out = torch.full((ns, ns, ld), float("nan"), dtype=torch.float64, device="cuda")
    Yd, rd, Td = dev(Yp), dev(rho), dev(T)
    binding._check(gm._lib.pyro_get_jacobian(gm._h, n, ld, rd.data_ptr(), Td.data_ptr(), Yd.data_ptr(), 1,
                                             out.data_ptr(), None, None))
    torch.cuda.synchronize()
    o = out.cpu().numpy()
    parity.assert_jacobian_parity(o[:, :, :n], Jr, bJ)
    assert np.isnan(o[:, :, n:]).all()


def test_jacobian_v_plane_in_shared_memory_and_small_blocks(mechs, monkeypatch):
    """The one-thread-per-point kernel (the fallback of the block-cooperative one), its large-mechanism layout (V in
    shared memory, 4 tensor-memory columns per species) forced on configs[0], and 32-thread blocks."""
    mech, _, orc = mechs(0)
    st = inputs.config_states(0, n=700)
    Jr, sTr, bJ, bT = orc.get_jacobian(st["rho"], st["T"], st["Y"], mode=0)
    for env in ({"PYRO_JAC_KERNEL": "block"}, {"PYRO_JAC_KERNEL": "point"}, {"PYRO_JAC_KERNEL": "point", "PYRO_JAC_V_PLANE": "shared"},
                {"PYRO_JAC_KERNEL": "point", "PYRO_JAC_BLOCK": "32"}):
        for k, v in env.items():
            monkeypatch.setenv(k, v)
        gm = binding.Mechanism(mech)
        J, sT = gpu_jacobian(gm, st["rho"], st["T"], st["Y"], 0)
        parity.assert_jacobian_parity(J, Jr, bJ)
        parity.assert_jacobian_parity(sT, sTr, bT)
        for k in env:
            monkeypatch.delenv(k)


def test_jacobian_block_kernel_scratch_in_global_memory(mechs, monkeypatch):
    """The block-cooperative kernel with the scratch of the [M] reactions in global memory (its shape for mechanisms
    whose planes fill the shared memory: configs[3] by itself), forced on configs[2] and on the hand mechanism."""
    monkeypatch.setenv("PYRO_JAC_KERNEL", "block")
    monkeypatch.setenv("PYRO_JAC_EXT", "global")
    hand = hand_cases.all_paths_mechanism()
    st = inputs.config_states(2, n=333)
    for mech, (rho, T, Y) in ((inputs.config_mechanism(2), (st["rho"], st["T"], st["Y"])), (hand, hand_cases.random_states(hand, 99))):
        Jr, sTr, bJ, bT = oracle.Oracle(mech).get_jacobian(rho, T, Y, mode=1)
        J, sT = gpu_jacobian(binding.Mechanism(mech), rho, T, Y, 1)
        parity.assert_jacobian_parity(J, Jr, bJ)
        parity.assert_jacobian_parity(sT, sTr, bT)


def test_jacobian_full_size_sampled_columns(mechs):
    """configs[2] at the size bench.py times the Jacobian on (2^18 points): sampled points against the oracle."""
    mech, gm, orc = mechs(2)
    n = 1 << 18
    st = inputs.config_states(2, n=n)
    J, sT = gm.get_jacobian(dev(st["rho"]), dev(st["T"]), dev(st["Y"]), mode=1)
    torch.cuda.synchronize()
    idx = _sample(n, 96)
    Jr, sTr, bJ, bT = orc.get_jacobian(st["rho"][idx], st["T"][idx], st["Y"][:, idx], mode=1)
    parity.assert_jacobian_parity(J[:, :, idx].cpu().numpy(), Jr, bJ)
    parity.assert_jacobian_parity(sT[:, idx].cpu().numpy(), sTr, bT)
    # conservation of mass per column holds at any size: sum_i J_ik = 0 relative to the column's terms
    s = J.sum(dim=0).abs().max().item()
    assert s <= 1e-9 * J.abs().sum(dim=0).max().item()


def test_jacobian_error_codes(mechs):
    mech, gm, _ = mechs(0)
    ns = mech.n_species
    st = inputs.config_states(0, n=64)
    rho, T, Y = dev(st["rho"]), dev(st["T"]), dev(st["Y"])
    J = torch.empty((ns, ns, 64), dtype=torch.float64, device="cuda")
    f = gm._lib.pyro_get_jacobian
    assert f(gm._h, 64, 64, rho.data_ptr(), T.data_ptr(), Y.data_ptr(), 2, J.data_ptr(), None, None) == 2   # mode
    assert f(gm._h, 64, 32, rho.data_ptr(), T.data_ptr(), Y.data_ptr(), 0, J.data_ptr(), None, None) == 2   # ld < n
    assert f(gm._h, 64, 64, rho.data_ptr(), T.data_ptr(), Y.data_ptr(), 0, None, None, None) == 1           # NULL
    assert f(gm._h, 64, 64, rho.data_ptr(), T.data_ptr(), Y.data_ptr(), 0, J.data_ptr() + 4, None, None) == 5   # alignment
    assert f(gm._h, 64, 64, rho.data_ptr(), T.data_ptr(), Y.data_ptr(), 0, Y.data_ptr(), None, None) == 2   # J overlaps Y
    assert f(gm._h, 0, 0, None, None, None, 0, None, None, None) == 0                                       # n = 0


# ------------------------------------------------------------------ fused temperature + rates
@pytest.mark.parametrize("cfg,n", [(0, 4096), (2, 2500), (3, 700), (4, 13**3)])
def test_fused_source_terms_every_point(mechs, cfg, n):
    """pyro_source_terms: T against the oracle's Newton solve, omega against the oracle's rates at the GPU's T
    (the same split of the comparison as the two-launch step of configs[4])."""
    mech, gm, orc = mechs(cfg)
    st = inputs.config_states(cfg, n=n)
    T_ref, it, conv = orc.get_temperature(st["e"], st["Y"], st["T_guess"])
    bad = torch.zeros(1, dtype=torch.int32, device="cuda")
    T, om = gm.source_terms(dev(st["rho"]), dev(st["e"]), dev(st["Y"]), dev(st["T_guess"]), n_not_converged=bad)
    torch.cuda.synchronize()
    T = T.cpu().numpy()
    parity.assert_T_parity(T, T_ref)
    assert int(bad.item()) == 0
    om_ref, bound = orc.get_net_production_rates(st["rho"], T, st["Y"])
    parity.assert_omega_parity(om.cpu().numpy(), om_ref, bound)
    # and it is the two-launch step: same temperatures bit for bit, hence same rates
    T2 = gm.get_temperature(dev(st["e"]), dev(st["Y"]), dev(st["T_guess"]))
    om2 = gm.get_net_production_rates(dev(st["rho"]), T2, dev(st["Y"]))
    torch.cuda.synchronize()
    assert np.max(np.abs(T2.cpu().numpy() - T) / T) <= 1e-14
    parity.assert_omega_parity(om.cpu().numpy(), om2.cpu().numpy(), bound)


def test_fused_source_terms_mixed_t_mid_cap_and_in_place(mechs):
    """Species with different break temperatures; T in place of T_guess; iteration cap reported."""
    mech0, _, _ = mechs(0)
    mech = inputs.with_species_break_temperatures(mech0, np.linspace(700.0, 1500.0, mech0.n_species))
    gm, orc = binding.Mechanism(mech), oracle.Oracle(mech)
    st = inputs.config_states(0, n=3000)
    e = np.array([orc.mixture_e(st["T"][p], st["Y"][:, p]) for p in range(3000)])
    T_ref, _, _ = orc.get_temperature(e, st["Y"], st["T_guess"])
    Tg = dev(st["T_guess"])
    T, om = gm.source_terms(dev(st["rho"]), dev(e), dev(st["Y"]), Tg, T_out=Tg)
    torch.cuda.synchronize()
    parity.assert_T_parity(Tg.cpu().numpy(), T_ref)
    om_ref, bound = orc.get_net_production_rates(st["rho"], Tg.cpu().numpy(), st["Y"])
    parity.assert_omega_parity(om.cpu().numpy(), om_ref, bound)
    gm.set_newton(1e-6, 1)
    bad = torch.zeros(1, dtype=torch.int32, device="cuda")
    gm.source_terms(dev(st["rho"]), dev(e), dev(st["Y"]), dev(st["T_guess"]), n_not_converged=bad)
    torch.cuda.synchronize()
    _, _, conv1 = orc.get_temperature(e, st["Y"], st["T_guess"], max_iter=1)
    assert int(bad.item()) == int((conv1 == 0).sum()) > 0


# ------------------------------------------------------------------ batched reactor march
REACTOR_TOL = 1e-10   # |dY_k| <= REACTOR_TOL * (sum of the sizes of the terms added into Y_k + |Y_k|)


def stable_dt(orc, rho, T, Y, safety=0.05):
    """A step that resolves the fastest chemical time scale of the batch (largest Jacobian row sum of dY/dt = S/rho)."""
    J, _, _, _ = orc.get_jacobian(rho, T, Y, mode=1)
    return safety / float(np.max(np.abs(J).sum(axis=1) / np.asarray(rho)[None, :]))


def assert_reactor_parity(Y, T, Y_ref, T_ref, Yb):
    assert np.isfinite(Y).all() and np.isfinite(T).all()
    rY = float(np.max(np.abs(Y - Y_ref) / (Yb + np.abs(Y_ref) + 1e-300)))
    rT = float(np.max(np.abs(T - T_ref) / T_ref))
    assert rY <= REACTOR_TOL, f"max |dY|/(Ybound + |Y|) = {rY:.3e}"
    assert rT <= 1e-9, f"max |dT|/T = {rT:.3e}"
    return rY, rT


@pytest.mark.parametrize("case,n", [("all_paths", 333), ("cfg0", 3001), ("cfg2", 700), ("cfg3", 150), ("mixed_t_mid", 1000)])
def test_reactor_rk4_every_point(mechs, case, n):
    """pyro_reactor_rk4 against the oracle's RK4 march: final mass fractions and temperature of every reactor,
    0, 1 and 7 steps, ragged tails, every reaction class, per-species break temperatures."""
    if case == "all_paths":
        mech = hand_cases.all_paths_mechanism()
        rho, T, Y = hand_cases.random_states(mech, n)
    else:
        cfg = {"cfg0": 0, "cfg2": 2, "cfg3": 3, "mixed_t_mid": 0}[case]
        mech = inputs.config_mechanism(cfg)
        if case == "mixed_t_mid":
            mech = inputs.with_species_break_temperatures(mech, np.linspace(800.0, 1400.0, mech.n_species))
        st = inputs.config_states(cfg, n=n)
        rho, T, Y = st["rho"], st["T"], st["Y"]
    orc = oracle.Oracle(mech)
    gm = binding.Mechanism(mech)
    e = np.array([orc.mixture_e(T[p], Y[:, p]) for p in range(n)])
    Tg = T * 1.03
    ns_dt = min(n, 64)
    dt = stable_dt(orc, rho[:ns_dt], T[:ns_dt], Y[:, :ns_dt], safety=0.02)
    for n_steps in (0, 1, 7):
        Yr, Tr, Yb, bad_r = orc.reactor_rk4(rho, e, Y, Tg, dt, n_steps)
        ok = np.isfinite(Yr).all(axis=0) & np.isfinite(Tr) & (np.abs(Yr).max(axis=0) < 10.0)   # reactors the step is stable for
        assert ok.sum() >= 0.5 * n
        Yd, Td = dev(Y), dev(Tg)
        bad = torch.zeros(1, dtype=torch.int32, device="cuda")
        gm.reactor_rk4(dev(rho), dev(e), Yd, Td, dt, n_steps, n_not_converged=bad)
        torch.cuda.synchronize()
        rY, rT = assert_reactor_parity(Yd.cpu().numpy()[:, ok], Td.cpu().numpy()[ok], Yr[:, ok], Tr[ok], Yb[:, ok])
        if ok.all():
            assert int(bad.item()) == bad_r
        print(f"{case} steps {n_steps}: max |dY|/scale = {rY:.2e}, max |dT|/T = {rT:.2e}, stable reactors {int(ok.sum())}/{n}")


def test_reactor_rk4_padded_ld_and_error_codes(mechs):
    mech, gm, orc = mechs(0)
    n, ld, ns = 100, 128, mech.n_species
    st = inputs.config_states(0, n=n)
    dt = stable_dt(orc, st["rho"][:32], st["T"][:32], st["Y"][:, :32], safety=0.02)
    Yr, Tr, Yb, _ = orc.reactor_rk4(st["rho"], st["e"], st["Y"], st["T_guess"], dt, 3)
    Yp = np.full((ns, ld), np.nan)
    Yp[:, :n] = st["Y"]
    Yd, Td = dev(Yp), dev(st["T_guess"])
    work = torch.full((ns, ld), float("nan"), dtype=torch.float64, device="cuda")
    rd, ed = dev(st["rho"]), dev(st["e"])
    f = gm._lib.pyro_reactor_rk4
    assert f(gm._h, n, ld, rd.data_ptr(), ed.data_ptr(), Yd.data_ptr(), Td.data_ptr(), dt, 3, work.data_ptr(), None, None) == 0
    torch.cuda.synchronize()
    Yh = Yd.cpu().numpy()
    ok = np.isfinite(Yr).all(axis=0) & (np.abs(Yr).max(axis=0) < 10.0)
    assert_reactor_parity(Yh[:, :n][:, ok], Td.cpu().numpy()[ok], Yr[:, ok], Tr[ok], Yb[:, ok])
    assert np.isnan(Yh[:, n:]).all() and torch.isnan(work[:, n:]).all()
    assert f(gm._h, n, ld, rd.data_ptr(), ed.data_ptr(), Yd.data_ptr(), Td.data_ptr(), dt, -1, work.data_ptr(), None, None) == 2
    assert f(gm._h, n, 50, rd.data_ptr(), ed.data_ptr(), Yd.data_ptr(), Td.data_ptr(), dt, 1, work.data_ptr(), None, None) == 2
    assert f(gm._h, n, ld, rd.data_ptr(), ed.data_ptr(), Yd.data_ptr(), Td.data_ptr(), dt, 1, None, None, None) == 1
    assert f(gm._h, n, ld, rd.data_ptr(), ed.data_ptr(), Yd.data_ptr(), Td.data_ptr(), dt, 1, Yd.data_ptr(), None, None) == 2
    assert f(gm._h, n, ld, rd.data_ptr(), ed.data_ptr(), Yd.data_ptr() + 4, Td.data_ptr(), dt, 1, work.data_ptr(), None, None) == 5
    assert f(gm._h, 0, 0, None, None, None, None, dt, 1, None, None, None) == 0


# ------------------------------------------------------------------ mixture-averaged transport
TRANSPORT_TOL = 1e-11   # relative, on mu, kappa and every D_k,m


def assert_transport_parity(got, ref):
    worst = 0.0
    for g, r in zip(got, ref):
        g = g.cpu().numpy() if hasattr(g, "cpu") else np.asarray(g)
        assert np.isfinite(g).all()
        worst = max(worst, float(np.max(np.abs(g - r) / np.abs(r))))
    assert worst <= TRANSPORT_TOL, f"max relative difference {worst:.3e}"
    return worst


@pytest.mark.parametrize("cfg,n", [(0, 3001), (2, 1500), (3, 333)])
def test_transport_every_point(cfg, n):
    """pyro_get_transport against the oracle's (A.18)-(A.24): mu, kappa and every D_k,m of every point; several
    blocks and a ragged tail; a composition with exact zeros."""
    tr = inputs.config_transport(cfg)
    st = inputs.config_states(cfg, n=n)
    Y = st["Y"].copy()
    Y[:, 0] = 0.0
    Y[:2, 0] = 0.5            # only two species present
    ref = oracle.TransportOracle(tr).get_transport(st["T"], Y)
    gt = binding.Transport(tr)
    got = gt.get_transport(dev(st["T"]), dev(Y))
    torch.cuda.synchronize()
    w = assert_transport_parity(got, ref)
    print(f"transport cfg {cfg}: max relative difference {w:.2e}")


def test_transport_w7_padded_ld_and_error_codes(golden_dir):
    """The hand-written W7 mixture through the C ABI; leading dimension > n with NaN padding untouched; error codes."""
    from test_oracle_transport_pins import _w7
    from conftest import read_golden
    mk, tr = _w7(golden_dir)
    g = {k: float(v) for k, v in read_golden(os.path.join(golden_dir, "w7_transport.txt")).items()}
    gt = binding.Transport(tr)
    n, ld = 5, 8
    Yp = np.full((3, ld), np.nan)
    Yp[:, :n] = np.array([[float(y)] for y in mk.Y])
    Td = dev(np.full(n, float(mk.T)))
    Yd = dev(Yp)
    mu = torch.full((n,), float("nan"), dtype=torch.float64, device="cuda")
    ka = torch.full((n,), float("nan"), dtype=torch.float64, device="cuda")
    D = torch.full((3, ld), float("nan"), dtype=torch.float64, device="cuda")
    f = gt._lib.pyro_get_transport
    assert f(gt._h, n, ld, Td.data_ptr(), Yd.data_ptr(), mu.data_ptr(), ka.data_ptr(), D.data_ptr(), None) == 0
    torch.cuda.synchronize()
    assert abs(mu[0].item() / g["mu_mix"] - 1) < 1e-13 and abs(ka[4].item() / g["kappa_mix"] - 1) < 1e-13
    for k in range(3):
        assert abs(D[k, 2].item() / g[f"D_{k}m"] - 1) < 1e-13
    assert torch.isnan(D[:, n:]).all()
    assert f(gt._h, n, 3, Td.data_ptr(), Yd.data_ptr(), mu.data_ptr(), ka.data_ptr(), D.data_ptr(), None) == 2
    assert f(gt._h, n, ld, Td.data_ptr(), Yd.data_ptr(), None, ka.data_ptr(), D.data_ptr(), None) == 1
    assert f(gt._h, n, ld, Td.data_ptr(), Yd.data_ptr(), mu.data_ptr() + 4, ka.data_ptr(), D.data_ptr(), None) == 5
    assert f(gt._h, n, ld, Td.data_ptr(), Yd.data_ptr(), mu.data_ptr(), ka.data_ptr(), Yd.data_ptr(), None) == 2
    assert f(gt._h, 0, 0, None, None, None, None, None, None) == 0
    assert f(None, n, ld, Td.data_ptr(), Yd.data_ptr(), mu.data_ptr(), ka.data_ptr(), D.data_ptr(), None) == 1
    bad = binding.TransportDesc(0, None, None, None, None)
    h = C.c_void_p()
    assert gt._lib.pyro_transport_create(C.byref(bad), 0, C.byref(h)) == 2 and not h.value
    assert gt._lib.pyro_transport_destroy(None) == 0


# ------------------------------------------------------------------ ABI: size and alignment checks of every field entry point
def test_abi_ld_and_alignment_on_every_entry_point(mechs):
    """ld < n is PYRO_ERR_BAD_SIZE and a misaligned pointer PYRO_ERR_ALIGN on every device entry point, including the
    widened ones; n_not_converged must be 4-byte aligned."""
    mech, gm, _ = mechs(0)
    ns, n = mech.n_species, 64
    st = inputs.config_states(0, n=n)
    rho, e, Y, Tg, T = (dev(st[k]) for k in ("rho", "e", "Y", "T_guess", "T"))
    out1 = torch.empty(n, dtype=torch.float64, device="cuda")
    outY = torch.empty((ns, n), dtype=torch.float64, device="cuda")
    J = torch.empty((ns, ns, n), dtype=torch.float64, device="cuda")
    bad = torch.zeros(2, dtype=torch.int32, device="cuda")
    L, h = gm._lib, gm._h
    p = lambda t: t.data_ptr()
    calls = {
        "temperature": lambda ld, o=0: L.pyro_get_temperature(h, n, ld, p(rho), p(e), p(Y), p(Tg), p(out1) + o, None, None),
        "temperature_h": lambda ld, o=0: L.pyro_get_temperature_from_enthalpy(h, n, ld, p(e), p(Y), p(Tg), p(out1) + o, None, None),
        "density": lambda ld, o=0: L.pyro_get_density(h, n, ld, p(rho), p(T), p(Y), p(out1) + o, None),
        "pressure": lambda ld, o=0: L.pyro_get_pressure(h, n, ld, p(rho), p(T), p(Y), p(out1) + o, None),
        "rates": lambda ld, o=0: L.pyro_get_net_production_rates(h, n, ld, p(rho), p(T), p(Y), p(outY) + o, None),
        "source_terms": lambda ld, o=0: L.pyro_source_terms(h, n, ld, p(rho), p(e), p(Y), p(Tg), p(out1) + o, p(outY), None, None),
        "jacobian": lambda ld, o=0: L.pyro_get_jacobian(h, n, ld, p(rho), p(T), p(Y), 0, p(J) + o, None, None),
        "reactor": lambda ld, o=0: L.pyro_reactor_rk4(h, n, ld, p(rho), p(e), p(Y), p(out1) + o, 1e-300, 0, p(outY), None, None),
    }
    for name, f in calls.items():
        assert f(n - 1) == 2, name          # ld < n
        assert f(n, 4) == 5, name           # 4-byte offset: not 8-byte aligned
    # n_not_converged: device int32, 4-byte aligned
    assert L.pyro_get_temperature(h, n, n, p(rho), p(e), p(Y), p(Tg), p(out1), p(bad) + 2, None) == 5
    assert L.pyro_get_temperature(h, n, n, p(rho), p(e), p(Y), p(Tg), p(out1), p(bad) + 4, None) == 0
    assert L.pyro_source_terms(h, n, n, p(rho), p(e), p(Y), p(Tg), p(out1), p(outY), p(bad) + 1, None) == 5
    assert L.pyro_reactor_rk4(h, n, n, p(rho), p(e), p(Y), p(out1), 1e-300, 0, p(outY), p(bad) + 2, None) == 5
    torch.cuda.synchronize()


@pytest.mark.parametrize("points", ["1", "2"])
def test_rates_kernel_points_per_thread(mechs, monkeypatch, points):
    """Both rates kernels on every kind of mechanism, whichever the library would choose (PYRO_RATES_POINTS forces
    one: the two-points-per-thread kernel is the default for small mechanisms, the one-point kernel for the others):
    every entry against the oracle, ragged tail of a 64-point chunk, hand mechanism with every class."""
    monkeypatch.setenv("PYRO_RATES_POINTS", points)
    hand = hand_cases.all_paths_mechanism()
    cases = [(hand, hand_cases.random_states(hand, 333))]
    for cfg, n in ((0, 777), (1, 1000 + 33), (2, 2500 + 33)):
        st = inputs.config_states(cfg, n=n)
        cases.append((inputs.config_mechanism(cfg), (st["rho"], st["T"], st["Y"])))
    for mech, (rho, T, Y) in cases:
        gm = binding.Mechanism(mech)
        om_ref, bound = oracle.Oracle(mech).get_net_production_rates(rho, T, Y)
        parity.assert_omega_parity(gpu_rates(gm, rho, T, Y), om_ref, bound)


# ------------------------------------------------------------------ implicit (Crank-Nicolson) reactor march (NEXT-4)
@pytest.mark.parametrize("case,n", [("all_paths", 200), ("cfg0", 1000), ("cfg2", 150)])
def test_reactor_cn_every_point(mechs, case, n):
    """pyro_reactor_cn against the oracle's Crank-Nicolson march (same fixed number of Newton iterations per step), at
    a step ten times the explicit one; ragged tails."""
    if case == "all_paths":
        mech = hand_cases.all_paths_mechanism()
        rho, T, Y = hand_cases.random_states(mech, n)
    else:
        cfg = {"cfg0": 0, "cfg2": 2}[case]
        mech = inputs.config_mechanism(cfg)
        st = inputs.config_states(cfg, n=n)
        rho, T, Y = st["rho"], st["T"], st["Y"]
    orc = oracle.Oracle(mech)
    gm = binding.Mechanism(mech)
    e = np.array([orc.mixture_e(T[p], Y[:, p]) for p in range(n)])
    Tg = T * 1.03
    # ten times the explicit step of the stiffest reactor of the batch: I - dt/(2 rho) J stays a perturbation of the
    # identity for every reactor (the kernel's LU does not pivot, reading G32)
    dt = stable_dt(orc, rho, T, Y, safety=0.2)
    for n_steps, iters in ((1, 1), (3, 4)):
        Yr, Tr, Yb, lu, bad_r = orc.reactor_cn(rho, e, Y, Tg, dt, n_steps, newton_iters=iters)
        ok = np.isfinite(Yr).all(axis=0) & np.isfinite(Tr) & (np.abs(Yr).max(axis=0) < 10.0) & (lu < 1e-3)
        assert ok.sum() >= 0.5 * n
        Yd, Td = dev(Y), dev(Tg)
        gm.reactor_cn(dev(rho), dev(e), Yd, Td, dt, n_steps, newton_iters=iters)
        torch.cuda.synchronize()
        Yg, Tgpu = Yd.cpu().numpy(), Td.cpu().numpy()
        rY = float(np.max(np.abs(Yg - Yr)[:, ok] / (Yb + np.abs(Yr) + 1e-300)[:, ok]))
        rT = float(np.max(np.abs(Tgpu - Tr)[ok] / Tr[ok]))
        print(f"{case} steps {n_steps} iters {iters}: max |dY|/scale = {rY:.2e}, max |dT|/T = {rT:.2e}, reactors compared {int(ok.sum())}/{n}")
        assert rY <= 1e-9 and rT <= 1e-8


def test_reactor_cn_linear_decay_closed_form_and_convergence_count():
    """A -> B with a constant rate coefficient: the GPU march reproduces y (1 - z/2)/(1 + z/2) per step at z = 20,
    where the explicit march diverges; the update tolerance counts unconverged (point, step) pairs."""
    z4 = [0.0] * 4
    sp = [dict(W=20.0, lo=[3.5, *z4, -1000.0, 2.0]), dict(W=20.0, lo=[3.0, *z4, -3000.0, 3.0])]
    k, dt, steps = 2.5e5, 8e-5, 5
    mech = inputs.simple_mechanism(sp, [dict(reac={0: 1}, prod={1: 1}, A=k, b=0.0, theta=0.0, reversible=0)])
    gm, orc = binding.Mechanism(mech), oracle.Oracle(mech)
    n = 100
    Y = np.vstack([np.linspace(0.1, 0.9, n), 1 - np.linspace(0.1, 0.9, n)])
    T = np.full(n, 1100.0)
    rho = np.full(n, 0.4)
    e = np.array([orc.mixture_e(T[p], Y[:, p]) for p in range(n)])
    Yd, Td = dev(Y), dev(T)
    bad = torch.zeros(1, dtype=torch.int32, device="cuda")
    gm.reactor_cn(dev(rho), dev(e), Yd, Td, dt, steps, newton_iters=2, update_tol=1e-12, n_not_converged=bad)
    torch.cuda.synchronize()
    g = ((1 - k * dt / 2) / (1 + k * dt / 2)) ** steps
    assert np.max(np.abs(Yd.cpu().numpy()[0] - Y[0] * g)) < 1e-14 and int(bad.item()) == 0
    Yd = dev(Y)
    gm.reactor_cn(dev(rho), dev(e), Yd, dev(T), dt, steps, newton_iters=1, update_tol=1e-12, n_not_converged=bad)
    torch.cuda.synchronize()
    assert int(bad.item()) == n * steps     # one iteration: the (only) update is the whole step, far above the tolerance
    Yr = dev(Y)
    gm.reactor_rk4(dev(rho), dev(e), Yr, dev(T), dt, steps)
    torch.cuda.synchronize()
    assert not bool(torch.isfinite(Yr).all()) or float(Yr.abs().max().item()) > 1e10   # the explicit march diverges at z = 20


# ------------------------------------------------------------------ marches on which most reactors move
# The synthetic mechanisms span more than a hundred decades of chemical time scale from one state to the next, so one
# step size for a whole batch leaves almost every reactor where it started (and an unchanged Y then passes any
# comparison).  The tests below group the reactors by their OWN time scale and march every group at its own step.
def stiffness_groups(orc, rho, T, Y, ratio=10.0):
    """[(indices, lambda_max)]: the reactors sorted by lambda_p = largest row sum of |dS/dY|/rho at fixed (rho, e) (the
    oracle's Jacobian), cut into runs whose lambda stay within `ratio` of one another."""
    J, _, _, _ = orc.get_jacobian(rho, T, Y, mode=1)
    lam = (np.abs(J).sum(axis=1) / np.asarray(rho)[None, :]).max(axis=0)
    order = np.argsort(lam)
    groups, cur = [], [order[0]]
    for p in order[1:]:
        if lam[p] <= ratio * lam[cur[0]]:
            cur.append(p)
        else:
            groups.append(np.array(cur))
            cur = [p]
    groups.append(np.array(cur))
    return [(g, float(lam[g].max())) for g in groups]


def moved_fraction(Y0, Y1, threshold):
    """Share of the reactors of which some mass fraction changed by more than `threshold`, relatively."""
    return float(np.mean(np.max(np.abs(Y1 - Y0) / (np.abs(Y0) + 1e-30), axis=0) > threshold))


def tempered_residual(Yg, Yr, Yb):
    """max |dY| / scale with a scale an unchanged Y cannot meet: the size Yb of the terms added into an entry wherever
    those are visible in it (Yb >= 1e-4 |Y|: the entry moved in the fifth digit or before), else Yb + |Y| (there the
    rounding of Y itself, 1e-16 |Y|, is what bounds the agreement)."""
    scale = np.where(Yb >= 1e-4 * np.abs(Yr), Yb, Yb + np.abs(Yr)) + 1e-300
    return float(np.max(np.abs(Yg - Yr) / scale))


def tempered_case(case, n):
    if case == "all_paths":
        mech = hand_cases.all_paths_mechanism()
        rho, T, Y = hand_cases.random_states(mech, n)
    else:
        cfg = {"cfg0": 0, "cfg2": 2, "cfg3": 3}[case]
        mech = inputs.config_mechanism(cfg)
        st = inputs.config_states(cfg, n=n)
        rho, T, Y = st["rho"], st["T"], st["Y"]
    orc = oracle.Oracle(mech)
    e = np.array([orc.mixture_e(T[p], Y[:, p]) for p in range(n)])
    return mech, orc, rho, T, Y, e


@pytest.mark.parametrize("case,n", [("cfg0", 3001), ("cfg2", 700), ("cfg3", 120), ("all_paths", 333)])
def test_reactor_rk4_tempered_most_reactors_move(case, n):
    """pyro_reactor_rk4 against the oracle, one launch per stiffness group at dt = 0.2 / lambda_max of the group, 7 steps:
    in every launch at least 80 % of the reactors change some Y_k by more than 1e-6 (asserted), over the batch at least
    80 % by more than 1e-3, and every entry is compared on the scale of the terms the march added to it."""
    mech, orc, rho, T, Y, e = tempered_case(case, n)
    gm = binding.Mechanism(mech)
    Tg = T * 1.03
    worst, worst_T, moved3, launches = 0.0, 0.0, 0.0, 0
    for g, lam_max in stiffness_groups(orc, rho, T, Y):
        dt = 0.2 / lam_max
        Yr, Tr, Yb, bad_r = orc.reactor_rk4(rho[g], e[g], Y[:, g], Tg[g], dt, 7)
        assert np.isfinite(Yr).all() and np.isfinite(Tr).all() and np.abs(Yr).max() < 10.0   # stable for every reactor of the group
        Yd, Td = dev(Y[:, g]), dev(Tg[g])
        bad = torch.zeros(1, dtype=torch.int32, device="cuda")
        gm.reactor_rk4(dev(rho[g]), dev(e[g]), Yd, Td, dt, 7, n_not_converged=bad)
        torch.cuda.synchronize()
        Yg, Tgpu = Yd.cpu().numpy(), Td.cpu().numpy()
        assert np.isfinite(Yg).all() and np.isfinite(Tgpu).all()
        m6 = moved_fraction(Y[:, g], Yr, 1e-6)
        assert m6 >= 0.8, f"{case}: only {m6:.2f} of the {len(g)} reactors of a launch moved (dt {dt:.3e})"
        assert moved_fraction(Y[:, g], Yg, 1e-6) >= 0.8
        moved3 += moved_fraction(Y[:, g], Yr, 1e-3) * len(g)
        worst = max(worst, tempered_residual(Yg, Yr, Yb))
        worst_T = max(worst_T, float(np.max(np.abs(Tgpu - Tr) / Tr)))
        assert int(bad.item()) == bad_r
        launches += 1
    print(f"{case}: {launches} launches, moved by > 1e-3: {moved3 / n:.3f} of {n} reactors, max |dY|/scale = {worst:.2e}, max |dT|/T = {worst_T:.2e}")
    assert moved3 >= 0.8 * n
    assert worst <= REACTOR_TOL and worst_T <= 1e-9


@pytest.mark.parametrize("z", [0.1, 1.0, 2.5])
def test_reactor_rk4_linear_decay_taylor_polynomial(z):
    """GPU twin of oracle pin R1: A -> B at a constant rate coefficient k; one RK4 step of size z/k multiplies Y_A by
    the degree-4 Taylor polynomial of exp(-z) -- every reactor, 5 steps, to 1e-14."""
    z4 = [0.0] * 4
    sp = [dict(W=20.0, lo=[3.5, *z4, -1000.0, 2.0]), dict(W=20.0, lo=[3.0, *z4, -3000.0, 3.0])]
    k, steps, n = 2.5e5, 5, 4099
    mech = inputs.simple_mechanism(sp, [dict(reac={0: 1}, prod={1: 1}, A=k, b=0.0, theta=0.0, reversible=0)])
    gm, orc = binding.Mechanism(mech), oracle.Oracle(mech)
    ya = np.linspace(0.1, 0.9, n)
    Y = np.vstack([ya, 1 - ya])
    T = np.full(n, 1100.0)
    rho = np.full(n, 0.4)
    e = np.array([orc.mixture_e(T[p], Y[:, p]) for p in range(n)])
    Yd, Td = dev(Y), dev(T)
    gm.reactor_rk4(dev(rho), dev(e), Yd, Td, z / k, steps)
    torch.cuda.synchronize()
    growth = (1 - z + z**2 / 2 - z**3 / 6 + z**4 / 24) ** steps
    Yg = Yd.cpu().numpy()
    assert np.max(np.abs(Yg[0] - ya * growth)) < 1e-14
    assert np.max(np.abs(Yg[1] - (1 - ya * growth))) < 1e-14     # mass is conserved: Y_B = 1 - Y_A


@pytest.mark.parametrize("case,n", [("cfg0", 1000), ("cfg2", 300), ("all_paths", 200)])
@pytest.mark.parametrize("factor", [10.0, 100.0])
def test_reactor_cn_tempered_far_from_the_identity(case, n, factor):
    """pyro_reactor_cn against the oracle's Crank-Nicolson march (partial pivoting) per stiffness group, at `factor`
    times the group's explicit step 0.2 / lambda_max, 2 steps of 4 Newton iterations.  At factor 100 the matrix the
    kernel factors WITHOUT pivoting, I - dt/(2 rho) J, has |dt/(2 rho) J| up to 10 for every group: the reactors lost to
    that (or to a Newton iteration that diverges at such a step on either side) are counted and reported."""
    mech, orc, rho, T, Y, e = tempered_case(case, n)
    gm = binding.Mechanism(mech)
    Tg = T * 1.03
    compared, lost, worst, moved, norm_min = 0, 0, 0.0, 0.0, np.inf
    for g, lam_max in stiffness_groups(orc, rho, T, Y):
        dt = factor * 0.2 / lam_max
        norm_min = min(norm_min, 0.5 * dt * lam_max)
        Yr, Tr, Yb, lu, _ = orc.reactor_cn(rho[g], e[g], Y[:, g], Tg[g], dt, 2, newton_iters=4)
        ok = np.isfinite(Yr).all(axis=0) & np.isfinite(Tr) & (np.abs(Yr).max(axis=0) < 10.0)
        Yd, Td = dev(Y[:, g]), dev(Tg[g])
        gm.reactor_cn(dev(rho[g]), dev(e[g]), Yd, Td, dt, 2, newton_iters=4)
        torch.cuda.synchronize()
        Yg, Tgpu = Yd.cpu().numpy(), Td.cpu().numpy()
        if not ok.any():
            continue
        scale = (np.where(Yb >= 1e-4 * np.abs(Yr), Yb, Yb + np.abs(Yr)) + 1e-300)[:, ok]
        with np.errstate(invalid="ignore"):
            r = np.max(np.abs(Yg[:, ok] - Yr[:, ok]) / scale, axis=0)
            rT = np.abs(Tgpu[ok] - Tr[ok]) / Tr[ok]
        good = (r <= 1e-9) & (rT <= 1e-8)
        compared += int(ok.sum())
        lost += int((~good).sum())
        if good.any():
            worst = max(worst, float(r[good].max()))
        moved += moved_fraction(Y[:, g][:, ok], Yr[:, ok], 1e-3) * int(ok.sum())
    print(f"{case} x{factor:g}: |dt/(2 rho) J| >= {norm_min:.1f} in every launch, reactors compared {compared}/{n}, "
          f"lost to the LU without pivoting or a diverging Newton iteration {lost}, moved by > 1e-3: {moved / max(compared, 1):.3f}, "
          f"max |dY|/scale of the rest = {worst:.2e}")
    assert compared >= 0.8 * n
    assert moved >= 0.8 * compared
    assert lost == 0


# ------------------------------------------------------------------ widened rows at the sizes bench.py times, sampled
def test_transport_and_reactors_at_bench_size_sampled(mechs):
    """The launch configurations of bench.py's widened legs on configs[2]: transport on 2^20 points, the RK4 march on
    2^20 reactors x 4 steps, the Crank-Nicolson march on 2^16 reactors x 1 step of 3 Newton iterations; sampled
    reactors (first, last, random) against the oracle.  The step is the bench's: from the GPU Jacobian of the batch."""
    mech, gm, orc = mechs(2)
    n = 1 << 20
    st = inputs.config_states(2, n=n)
    rho, e, Y, Tg, T = (dev(st[k]) for k in ("rho", "e", "Y", "T_guess", "T"))
    idx = _sample(n, 48)
    # transport
    tr = inputs.config_transport(2)
    got = binding.Transport(tr).get_transport(T, Y)
    torch.cuda.synchronize()
    ref = oracle.TransportOracle(tr).get_transport(st["T"][idx], st["Y"][:, idx])
    assert_transport_parity((got[0][idx], got[1][idx], got[2][:, idx]), ref)
    # explicit march on bench.py's tempered batch: the states of the most populated stiffness decade of a slice
    # (GPU Jacobian), repeated to 2^20 reactors, dt = 0.2 / lambda_max
    import bench
    m = 1 << 14
    J, _ = gm.get_jacobian(rho[:m].contiguous(), T[:m].contiguous(), Y[:, :m].contiguous(), mode=1, want_dSdT=False)
    lam = (J.abs().sum(dim=1) / rho[:m][None, :]).amax(dim=0).cpu().numpy()
    del J
    sel, lam_max = bench.tempered_window(lam)
    assert len(sel) >= 100
    rep_h = sel[np.arange(n) % len(sel)]
    rep = torch.from_numpy(rep_h).cuda()
    dt = 0.2 / lam_max
    rho_r, e_r, Yd, Td = rho[rep].contiguous(), e[rep].contiguous(), Y[:, rep].contiguous(), Tg[rep].contiguous()
    gm.reactor_rk4(rho_r, e_r, Yd, Td, dt, 4)
    torch.cuda.synchronize()
    src = rep_h[idx]
    Yr, Tr, Yb, _ = orc.reactor_rk4(st["rho"][src], st["e"][src], st["Y"][:, src], st["T_guess"][src], dt, 4)
    assert np.isfinite(Yr).all() and np.abs(Yr).max() < 10.0
    assert moved_fraction(st["Y"][:, src], Yr, 1e-3) >= 0.8
    assert tempered_residual(Yd[:, idx].cpu().numpy(), Yr, Yb) <= REACTOR_TOL
    assert float(np.max(np.abs(Td[idx].cpu().numpy() - Tr) / Tr)) <= 1e-9
    assert bool(torch.isfinite(Yd).all())
    assert float((((Yd - Y[:, rep]).abs() / (Y[:, rep].abs() + 1e-30)).amax(dim=0) > 1e-6).float().mean().item()) >= 0.8
    # implicit march at ten times that step
    nc = 1 << 16
    idc = _sample(nc, 32)
    Yc, Tc = Y[:, rep[:nc]].contiguous(), Tg[rep[:nc]].contiguous()
    gm.reactor_cn(rho_r[:nc].contiguous(), e_r[:nc].contiguous(), Yc, Tc, 10.0 * dt, 1, newton_iters=3)
    torch.cuda.synchronize()
    src = rep_h[idc]
    Yr, Tr, Yb, lu, _ = orc.reactor_cn(st["rho"][src], st["e"][src], st["Y"][:, src], st["T_guess"][src], 10.0 * dt, 1, newton_iters=3)
    assert np.isfinite(Yr).all() and np.abs(Yr).max() < 10.0
    assert moved_fraction(st["Y"][:, src], Yr, 1e-3) >= 0.8
    rY = tempered_residual(Yc[:, idc].cpu().numpy(), Yr, Yb)
    assert rY <= 1e-9, rY
