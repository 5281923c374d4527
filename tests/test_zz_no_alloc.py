"""pyro_reactor_rk4_static: the RK4 reactor march for callers that cannot allocate device memory.

Who that is: code that lives inside another program's memory budget -- a chemistry plug-in of a flow solver that
owns every byte of the GPU and lends out only its state arrays, a call made after the host application has frozen
its memory pool, a time loop that cannot afford the device-wide synchronisation cudaMalloc implies.  Such a caller
has no `work` field to give pyro_reactor_rk4; the _static variant takes its scratch from a fixed 32 MiB array that is
part of libpyro.so's device image instead, and is otherwise the same march.

What is checked here, through the C ABI, against pyro_reactor_rk4 on the same inputs and at the tolerance of the
other reactor tests (tests/test_gpu_parity.py: |dY_k| <= 1e-10 x the size of the terms added into Y_k, |dT|/T <= 1e-9):
four _static calls back to back on one stream with no synchronisation in between, on batches of different species
count, size and leading dimension, so that every call after the first finds the previous call's leftovers in the array
in a different layout; that free device memory does not shrink across a call; that a batch beyond the array's size
is refused with PYRO_ERR_TOO_LARGE before anything is launched.

The file name sorts last on purpose (pytest -x stops at the first failure; a problem here must not hide the parity
tests), and the tests make no assumption about what ran before them: they pass in a fresh process, where the first
_static call performs the one-time address look-up, and at the end of the whole suite.
"""
import numpy as np
import pytest

from paper_2503_24286_b200 import binding, inputs

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")

REACTOR_TOL = 1e-10   # as tests/test_gpu_parity.py
T_TOL = 1e-9


def dev(x):
    return torch.from_numpy(np.ascontiguousarray(x)).cuda()


def linear_decay_case(n, z, steps):
    """A -> B at a constant rate coefficient k, dt = z / k: every reactor moves, and one RK4 step multiplies Y_A by
    the degree-4 Taylor polynomial of exp(-z) exactly."""
    z4 = [0.0] * 4
    sp = [dict(W=20.0, lo=[3.5, *z4, -1000.0, 2.0]), dict(W=20.0, lo=[3.0, *z4, -3000.0, 3.0])]
    k = 2.5e5
    mech = inputs.simple_mechanism(sp, [dict(reac={0: 1}, prod={1: 1}, A=k, b=0.0, theta=0.0, reversible=0)])
    ya = np.linspace(0.1, 0.9, n)
    Y = np.vstack([ya, 1.0 - ya])
    T = np.full(n, 1100.0)
    rho = np.full(n, 0.4)
    e = inputs.mixture_energy(mech, T, Y, dtype=np.float64)
    return dict(mech=mech, rho=rho, e=e, Y=Y, Tg=T * 1.02, dt=z / k, steps=steps, ld=n,
                growth=(1.0 - z + z**2 / 2 - z**3 / 6 + z**4 / 24) ** steps)


def config_case(cfg, n, ld, steps, skip=0):
    """States of BASELINE.json configs[cfg] (the `skip` first ones left out), padded to leading dimension ld with NaN.
    The step is taken from the batch's own chemical time scales (GPU Jacobian at fixed (rho, e)): a quarter of the
    reactors are stiffer than 0.05/dt, so the reactors just below that are marched at a step that moves them."""
    mech = inputs.config_mechanism(cfg)
    st = inputs.config_states(cfg, n=n + skip)
    rho, e, Tg, T, Y = (st[k][..., skip:] for k in ("rho", "e", "T_guess", "T", "Y"))
    gm = binding.Mechanism(mech)
    J, _ = gm.get_jacobian(dev(rho), dev(T), dev(Y), mode=1, want_dSdT=False)
    lam = (J[:, :, :n].abs().sum(dim=1) / dev(rho)[None, :]).amax(dim=0).cpu().numpy()
    lam = lam[np.isfinite(lam) & (lam > 0)]
    dt = 0.05 / float(np.quantile(lam, 0.75))
    Yp = np.full((mech.n_species, ld), np.nan)
    Yp[:, :n] = Y
    return dict(mech=mech, rho=rho, e=e, Y=Yp, Tg=Tg, dt=dt, steps=steps, ld=ld, gm=gm)


def run(case, static, bad):
    """One march through the C ABI; returns the device tensors (no synchronisation)."""
    gm = case.setdefault("gm", None) or binding.Mechanism(case["mech"])
    case["gm"] = gm
    n = case["rho"].shape[0]
    rho, e, Y, T = dev(case["rho"]), dev(case["e"]), dev(case["Y"]), dev(case["Tg"])
    case.setdefault("keep", []).append((rho, e))
    if static:
        st = gm._lib.pyro_reactor_rk4_static(gm._h, n, case["ld"], rho.data_ptr(), e.data_ptr(), Y.data_ptr(), T.data_ptr(),
                                             case["dt"], case["steps"], bad.data_ptr(), None)
    else:
        work = torch.full_like(Y, float("nan"))
        case["keep"].append(work)
        st = gm._lib.pyro_reactor_rk4(gm._h, n, case["ld"], rho.data_ptr(), e.data_ptr(), Y.data_ptr(), T.data_ptr(),
                                      case["dt"], case["steps"], work.data_ptr(), bad.data_ptr(), None)
    assert st == 0, gm._lib.pyro_last_error_string().decode()
    return Y, T


def compare(name, case, got, ref, bad_got, bad_ref):
    n = case["rho"].shape[0]
    Yg, Tg = got[0].cpu().numpy(), got[1].cpu().numpy()
    Yr, Tr = ref[0].cpu().numpy(), ref[1].cpu().numpy()
    Y0 = case["Y"][:, :n]
    assert np.array_equal(np.isnan(Yg[:, n:]), np.isnan(Yr[:, n:])) and np.isnan(Yg[:, n:]).all()   # padding untouched
    Yg, Yr = Yg[:, :n], Yr[:, :n]
    # reactors the explicit step is stable for (the others overflow identically in both marches and say nothing)
    ok = np.isfinite(Yr).all(axis=0) & np.isfinite(Tr) & (np.abs(Yr).max(axis=0) < 10.0)
    assert ok.sum() >= 0.5 * n, f"{name}: only {int(ok.sum())} of {n} reactors are stable at this step"
    assert np.isfinite(Yg[:, ok]).all() and np.isfinite(Tg[ok]).all()
    # |Y0| + |Y| is a lower bound of the scale the parity tests use (the terms added into Y_k start with Y0 itself)
    rY = float(np.max(np.abs(Yg[:, ok] - Yr[:, ok]) / (np.abs(Y0[:, ok]) + np.abs(Yr[:, ok]) + 1e-300)))
    rT = float(np.max(np.abs(Tg - Tr)[ok] / Tr[ok]))
    moved = np.max(np.abs(Yr[:, ok] - Y0[:, ok]) / (np.abs(Y0[:, ok]) + 1e-30), axis=0) > 1e-6
    print(f"{name}: max |dY|/scale = {rY:.2e}, max |dT|/T = {rT:.2e}, reactors compared {int(ok.sum())}/{n}, "
          f"moved {int(moved.sum())}, bit-identical {bool(np.array_equal(Yg[:, ok], Yr[:, ok]))}")
    assert rY <= REACTOR_TOL, f"{name}: max |dY|/scale = {rY:.3e}"
    assert rT <= T_TOL, f"{name}: max |dT|/T = {rT:.3e}"
    assert bad_got == bad_ref, f"{name}: Newton non-convergence count {bad_got} against {bad_ref}"
    return int(moved.sum())


def test_static_scratch_march_matches_the_work_field_march_on_calls_in_a_row():
    cases = [
        ("configs[2] 53 species, 3001 reactors, ld 3040", config_case(2, 3001, 3040, 7)),
        ("linear decay 2 species, 70001 reactors", linear_decay_case(70001, 0.5, 5)),
        ("configs[0] 9 species, 1000 reactors", config_case(0, 1000, 1000, 3, skip=500)),
        ("configs[2] again, 700 reactors, 1 step", config_case(2, 700, 704, 1, skip=3001)),
    ]
    # the existing path first (caller-provided work field, one counter each)
    refs, bad_refs = [], []
    for _, case in cases:
        bad = torch.zeros(1, dtype=torch.int32, device="cuda")
        refs.append(run(case, False, bad))
        bad_refs.append(bad)
    torch.cuda.synchronize()
    # then the built-in scratch: all calls enqueued back to back on the default stream, no synchronisation between them
    gots, bad_gots = [], []
    for _, case in cases:
        bad = torch.zeros(1, dtype=torch.int32, device="cuda")
        gots.append(run(case, True, bad))
        bad_gots.append(bad)
    torch.cuda.synchronize()
    moved = [compare(name, case, got, ref, int(bg.item()), int(br.item()))
             for (name, case), got, ref, bg, br in zip(cases, gots, refs, bad_gots, bad_refs)]
    assert moved[0] >= 10 and moved[1] == 70001
    # the linear decay also has a closed form: Y_A after `steps` steps = Y_A(0) x (Taylor polynomial of exp(-z))^steps
    lin = cases[1][1]
    assert np.max(np.abs(gots[1][0].cpu().numpy()[0] - lin["Y"][0] * lin["growth"])) < 1e-14


def test_static_scratch_call_allocates_nothing_and_refuses_oversized_batches():
    case = config_case(2, 2048, 2048, 2)
    bad = torch.zeros(1, dtype=torch.int32, device="cuda")
    run(case, True, bad)            # in a fresh process this is the call that looks the array up
    torch.cuda.synchronize()
    free_before, _ = torch.cuda.mem_get_info()
    gm = case["gm"]
    n = 2048
    rho, e, Y, T = dev(case["rho"]), dev(case["e"]), dev(case["Y"]), dev(case["Tg"])
    torch.cuda.synchronize()
    free_mid, _ = torch.cuda.mem_get_info()     # after this test's own tensors exist
    f = gm._lib.pyro_reactor_rk4_static
    for _ in range(3):
        assert f(gm._h, n, 2048, rho.data_ptr(), e.data_ptr(), Y.data_ptr(), T.data_ptr(), case["dt"], 1, bad.data_ptr(), None) == 0
    torch.cuda.synchronize()
    free_after, _ = torch.cuda.mem_get_info()
    assert free_after >= free_mid, (free_before, free_mid, free_after)
    # the limit: n_species x (n rounded up to 32) doubles must fit the array; real-size fields, so that even a call that
    # wrongly went ahead would stay inside them
    ns = case["mech"].n_species
    n_max = (binding.RK4_STATIC_MAX_DOUBLES // ns) // 32 * 32
    n_big = n_max + 1
    Yb = torch.full((ns, n_big), 1.0 / ns, dtype=torch.float64, device="cuda")
    one = torch.ones(n_big, dtype=torch.float64, device="cuda")
    Tb = torch.full((n_big,), 1000.0, dtype=torch.float64, device="cuda")
    before = Yb.clone()
    assert f(gm._h, n_big, n_big, one.data_ptr(), one.data_ptr(), Yb.data_ptr(), Tb.data_ptr(), 1e-12, 1, None, None) == 4
    msg = gm._lib.pyro_last_error_string().decode()
    assert "built-in scratch" in msg and str(binding.RK4_STATIC_MAX_DOUBLES) in msg, msg
    torch.cuda.synchronize()
    assert torch.equal(Yb, before)
    # the largest batch that does fit is accepted (n_steps = 0: only the temperature inversion runs)
    e_max = torch.full((n_max,), float(case["e"][0]), dtype=torch.float64, device="cuda")
    Ym = dev(np.repeat(case["Y"][:, :1], n_max, axis=1))
    assert f(gm._h, n_max, n_max, one.data_ptr(), e_max.data_ptr(), Ym.data_ptr(), Tb.data_ptr(), 1e-12, 0, None, None) == 0
    # the other argument checks are those of pyro_reactor_rk4
    assert f(gm._h, n, 2048, rho.data_ptr(), e.data_ptr(), Y.data_ptr(), T.data_ptr(), case["dt"], -1, None, None) == 2
    assert f(gm._h, n, 100, rho.data_ptr(), e.data_ptr(), Y.data_ptr(), T.data_ptr(), case["dt"], 1, None, None) == 2
    assert f(gm._h, n, 2048, None, e.data_ptr(), Y.data_ptr(), T.data_ptr(), case["dt"], 1, None, None) == 1
    assert f(gm._h, n, 2048, rho.data_ptr(), e.data_ptr(), Y.data_ptr() + 4, T.data_ptr(), case["dt"], 1, None, None) == 5
    assert f(gm._h, 0, 0, None, None, None, None, 1e-9, 1, None, None) == 0
    torch.cuda.synchronize()
