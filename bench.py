#!/usr/bin/env python
"""bench.py -- source-term points/sec of the thermochemistry hot path on B200.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config C] [--impl ours|reference]

A *step* is one pass of the whole hot path over one batch of synthetic input:
pyro_get_temperature (rho, e, Y, T_guess -> T) followed by pyro_get_net_production_rates
(rho, T, Y -> omega) on the same stream, through the C ABI of libpyro.so.  The default workload
is BASELINE.json configs[2] (53 species / 325 reactions, 2^22 points), the configuration the
metric is quoted on.  `value` is points/s with the inputs resident in HBM; `e2e` is the same
metric through pyro_source_terms_host with pinned HOST buffers (copies inside the timed region).
One JSON line is printed by rank 0.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

from paper_2503_24286_b200 import inputs, sharding  # noqa: E402

METRIC = "source-term points/sec (FP64, 53 sp/325 rxn) and % of B200 FP64/HBM roofline"

# FP64 cost of the transcendental functions, counted in SASS of nvcc 12.9 -O3 for sm_100a
# (DADD + DMUL + 2 DFMA on the fast path of CUDA's exp / log / division).
FLOPS_EXP, FLOPS_LOG, FLOPS_DIV = 30, 46, 15

# DRAM traffic of the rates kernel measured once with `ncu --set full` (dram__bytes_read.sum +
# dram__bytes_write.sum = 866.3 MB for 2^20 points of configs[2]; profiles/r01_v8_kernels.md).
# Reported as `traffic` for the configs[2]/[4] mechanism only, scaled to the points of one launch.
NCU_RATES_DRAM_BYTES_PER_POINT_53SP = 864.1e6 / 1048576
# Executed FP64 work of the rates kernel from the same ncu capture (profiles/r02_kernels.md): DADD + DMUL + 2 DFMA
# thread instructions per point, and the busy share of the FP64 pipe.  configs[2]/[4] mechanism only.
NCU_RATES_EXECUTED_FLOPS_PER_POINT_53SP = 24.2e3
NCU_RATES_FP64_PIPE_PCT_53SP = 45.0

# FP64 roof of one B200: 148 SMs x 64 FP64 FMA lanes x 2 flop x 1.965 GHz.
FP64_PEAK_TFLOPS = 148 * 64 * 2 * 1.965e9 / 1e12


def algorithmic_flops_per_point(mech):
    """F_rates of SURVEY.md section 8(d): what the method itself must compute per point."""
    E, L, D = FLOPS_EXP, FLOPS_LOG, FLOPS_DIV
    ns = mech.n_species
    f = (D + L + 1) + ns * (2 + 12) + (ns - 1)
    for j in range(mech.n_reactions):
        m_j = int(mech.reac_coeff[mech.reac_ptr[j]:mech.reac_ptr[j + 1]].sum()
                  + mech.prod_coeff[mech.prod_ptr[j]:mech.prod_ptr[j + 1]].sum())
        n_j = int(mech.eff_ptr[j + 1] - mech.eff_ptr[j])
        t = int(mech.rtype[j])
        if mech.reversible[j]:
            f += 8 + 3 * m_j + 2 * E
        else:
            f += 4 + 2 * m_j + E
        if t == inputs.THREE_BODY:
            f += 2 * n_j + 2
        if t >= inputs.FALLOFF_LINDEMANN:
            f += 8 + 2 * n_j + E + 2 * D
        if t == inputs.FALLOFF_TROE:
            f += 21 + 4 * E + 2 * L + 2 * D
    return float(f)


def algorithmic_bytes_per_point(ns):
    """Compulsory HBM traffic, FP64: rates 8(2 N_s + 2), T-solve 8(N_s + 3)."""
    return {"rates": 8.0 * (2 * ns + 2), "temperature": 8.0 * (ns + 3)}


class ClockSampler:
    """Samples nvidia-smi SM clocks and throttle reasons while the timed region runs."""

    FIELDS = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
              "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
              "clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.index = index
        self.rows = []
        self._stop = threading.Event()
        self._t = None

    def _run(self):
        while not self._stop.is_set():
            try:
                out = subprocess.run(["nvidia-smi", f"--id={self.index}", f"--query-gpu={self.FIELDS}",
                                      "--format=csv,noheader,nounits"], capture_output=True, text=True, timeout=5).stdout
                parts = [p.strip() for p in out.strip().split(",")]
                if len(parts) >= 7:
                    self.rows.append(parts)
            except Exception:
                pass
            self._stop.wait(0.1)

    def __enter__(self):
        self._t = threading.Thread(target=self._run, daemon=True)
        self._t.start()
        return self

    def __exit__(self, *a):
        self._stop.set()
        self._t.join(timeout=6)

    def summary(self):
        if not self.rows:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["unsampled"]}
        sm = sorted(float(r[0]) for r in self.rows)
        reasons = []
        for name, col in (("hw_slowdown", 3), ("hw_thermal_slowdown", 4), ("sw_thermal_slowdown", 5),
                          ("sw_power_cap", 6)):
            if any(r[col].lower().startswith("active") for r in self.rows):
                reasons.append(name)
        pw = [float(r[2]) for r in self.rows if r[2].replace(".", "", 1).isdigit()]
        return {"sm_mhz": sm[len(sm) // 2], "sm_max_mhz": float(self.rows[0][1]), "reasons": reasons,
                "samples": len(self.rows), "power_w_max": max(pw) if pw else None}


def time_oracle(cfg, target_seconds, with_temperature=True):
    """The CPU oracle as it stands, on a bounded sample of the workload.  Returns (points/s, dict)."""
    from oracle import oracle
    mech = inputs.config_mechanism(cfg)
    orc = oracle.Oracle(mech)
    cores = oracle.num_threads()
    st = inputs.config_states(cfg, n=1024 * 16 if mech.n_species < 20 else 4096, e_dtype=np.float64)

    def run(s):
        t0 = time.perf_counter()
        T = s["T"]
        if with_temperature:
            T, _, _ = orc.get_temperature(s["e"], s["Y"], s["T_guess"])
        orc.get_net_production_rates(s["rho"], T, s["Y"], want_bound=False)
        return time.perf_counter() - t0
    run(st)
    rate = st["rho"].shape[0] / run(st)
    n = int(min(inputs.CONFIG_POINTS[cfg], max(4096, rate * target_seconds)))
    if cfg == 4:
        n = round(n ** (1 / 3)) ** 3
    st = inputs.config_states(cfg, n=n, e_dtype=np.float64)
    dt = run(st)
    return n / dt, {"cores": cores, "sample": f"{n} points of configs[{cfg}] (seeded as the GPU workload), "
                                              f"{'temperature solve + ' if with_temperature else ''}production rates, "
                                              f"{dt:.1f} s", "n": n, "seconds": dt}


def _event_times(fn, stream, reps, warm=2):
    import torch
    for _ in range(warm):
        fn()
    torch.cuda.synchronize()
    ts = []
    for _ in range(reps):
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record(stream)
        fn()
        b.record(stream)
        torch.cuda.synchronize()
        ts.append(a.elapsed_time(b))
    return float(np.median(ts)), float(min(ts))


def time_widened_rows(gm, mech, cfg, d, T, stream, device):
    """SURVEY.md 8(f) rows beyond the step, each timed on its own (CUDA events, median of 5 after 2 warm-ups) on a
    bounded slice of the same states: NEXT-2 chemical Jacobian, NEXT-3 mixture-averaged transport, NEXT-4 batched
    RK4 reactors.  Rooflines: DESIGN.md section 7."""
    import torch
    from paper_2503_24286_b200 import binding
    ns = mech.n_species
    n = d["rho"].shape[0]
    peaks = {}
    try:
        peaks = json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))
    except Exception:
        pass
    hbm_peak = float(peaks.get("hbm_gbs", 6650.0))
    out = {}
    # ---- NEXT-2: J = dS/dY at fixed (rho, e) and dS/dT; output 8 ns^2 bytes per point dominates the traffic
    nj = int(min(n, max(4096, (6 << 30) // (8 * ns * ns))))
    nj = 1 << (nj.bit_length() - 1)
    sl = lambda x: x[..., :nj].contiguous()
    rho_j, T_j, Y_j = sl(d["rho"]), sl(T), sl(d["Y"])
    J = torch.empty((ns, ns, nj), dtype=torch.float64, device="cuda")
    sT = torch.empty((ns, nj), dtype=torch.float64, device="cuda")
    try:
        ms, mn = _event_times(lambda: gm.get_jacobian(rho_j, T_j, Y_j, mode=1, out=J, dSdT=sT, stream=stream), stream, 5)
        byt = 8.0 * (ns * ns + 3 * ns + 2) * nj
        out["next2_jacobian"] = {
            "points": nj, "ms": ms, "ms_min": mn, "points_per_s": nj / (ms * 1e-3), "mode": "fixed (rho, e)",
            "roofline": {"bound": "hbm", "achieved": byt / (ms * 1e-3) / 1e9, "peak": hbm_peak, "unit": "GB/s",
                         "frac": byt / (ms * 1e-3) / 1e9 / hbm_peak, "bytes_per_point": 8.0 * (ns * ns + 3 * ns + 2)}}
        # a stable explicit step for the reactors: the largest row sum of |J|/rho over the slice bounds the stiffness
        rate = float((J.abs().sum(dim=1) / rho_j[None, :]).max().item())
    except binding.PyroError as ex:
        out["next2_jacobian"] = {"unavailable": str(ex)}
        rate = None
    del J, sT
    # ---- NEXT-3: mixture-averaged transport, O(ns^2) FP64 per point
    tr = inputs.config_transport(cfg)
    gt = binding.Transport(tr, device=device)
    nt = int(min(n, 1 << 20))
    T_t, Y_t = T[:nt].contiguous(), d["Y"][:, :nt].contiguous()
    mu, ka, D = torch.empty_like(T_t), torch.empty_like(T_t), torch.empty_like(Y_t)
    ms, mn = _event_times(lambda: gt.get_transport(T_t, Y_t, mu, ka, D, stream=stream), stream, 5)
    # per ordered pair: Phi 7 flops, Horner 8, reciprocal counted as a division, accumulate 2; per species 2 Horner + 3 divisions
    fl = ns * ns * (7 + 8 + FLOPS_DIV + 2) + ns * (16 + 3 * FLOPS_DIV + 12) + FLOPS_LOG + 2 * FLOPS_DIV
    out["next3_transport"] = {
        "points": nt, "ms": ms, "ms_min": mn, "points_per_s": nt / (ms * 1e-3),
        "roofline": {"bound": "alu", "achieved": fl * nt / (ms * 1e-3) / 1e12, "peak": FP64_PEAK_TFLOPS, "unit": "TFLOP/s",
                     "frac": fl * nt / (ms * 1e-3) / 1e12 / FP64_PEAK_TFLOPS, "flops_per_point": float(fl)}}
    gt.close()
    # ---- NEXT-4: RK4 reactors, 4 stages (Newton solve + rates) per step
    if rate:
        nr = int(min(n, 1 << 20))
        steps = 4
        dt = 1e-3 / rate
        rho_r, e_r = d["rho"][:nr].contiguous(), d["e"][:nr].contiguous()
        work = torch.empty((ns, nr), dtype=torch.float64, device="cuda")
        Y_r, T_r = d["Y"][:, :nr].clone(), d["T_guess"][:nr].clone()

        def march():
            Y_r.copy_(d["Y"][:, :nr])
            T_r.copy_(d["T_guess"][:nr])
            gm.reactor_rk4(rho_r, e_r, Y_r, T_r, dt, steps, work=work, stream=stream)
        copy_ms, _ = _event_times(lambda: (Y_r.copy_(d["Y"][:, :nr]), T_r.copy_(d["T_guess"][:nr])), stream, 5)
        ms, mn = _event_times(march, stream, 5)
        ms, mn = ms - copy_ms, mn - copy_ms
        fl = 4 * algorithmic_flops_per_point(mech) + 4 * (25 * ns + FLOPS_DIV + 4) * 4
        out["next4_reactor_rk4"] = {
            "reactors": nr, "steps": steps, "dt": dt, "ms": ms, "ms_min": mn,
            "reactor_steps_per_s": nr * steps / (ms * 1e-3), "ns_per_reactor_stage": ms * 1e6 / nr / steps / 4,
            "finite_fraction": float(torch.isfinite(Y_r).all(dim=0).float().mean().item()),
            "roofline": {"bound": "alu", "achieved": fl * nr * steps / (ms * 1e-3) / 1e12, "peak": FP64_PEAK_TFLOPS,
                         "unit": "TFLOP/s", "frac": fl * nr * steps / (ms * 1e-3) / 1e12 / FP64_PEAK_TFLOPS,
                         "flops_per_reactor_step": float(fl)}}
        # implicit march: one Crank-Nicolson step of 3 Newton iterations (temperature + rates + Jacobian + LU each)
        nc = int(min(n, 1 << 16))
        rho_c, e_c = d["rho"][:nc].contiguous(), d["e"][:nc].contiguous()
        Y_c, T_c = d["Y"][:, :nc].clone(), d["T_guess"][:nc].clone()
        iters = 3
        try:
            def cn():
                Y_c.copy_(d["Y"][:, :nc])
                T_c.copy_(d["T_guess"][:nc])
                gm.reactor_cn(rho_c, e_c, Y_c, T_c, 10.0 * dt, 1, newton_iters=iters, stream=stream)
            ms, mn = _event_times(cn, stream, 3, warm=1)
            lu_bytes = 8.0 * (ns ** 3 / 12.0 + 2.5 * ns * ns)   # panel LU: one factor read per four multiply-adds + panel load/store + back substitution
            out["next4_reactor_cn"] = {
                "reactors": nc, "steps": 1, "newton_iters": iters, "dt": 10.0 * dt, "ms": ms, "ms_min": mn,
                "ns_per_reactor_iteration": ms * 1e6 / nc / iters,
                "finite_fraction": float(torch.isfinite(Y_c).all(dim=0).float().mean().item()),
                "roofline": {"bound": "hbm", "achieved": lu_bytes * nc * iters / (ms * 1e-3) / 1e9, "peak": hbm_peak, "unit": "GB/s",
                             "frac": lu_bytes * nc * iters / (ms * 1e-3) / 1e9 / hbm_peak,
                             "note": "the per-point panel LU dominates; bytes = factor reads of the left-looking LU as written (ns^3/12 + 2.5 ns^2 doubles per solve); compulsory traffic is 16 ns^2 bytes"}}
        except binding.PyroError as ex:
            out["next4_reactor_cn"] = {"unavailable": str(ex)}
    return out


def reference_arm(args, rank):
    """--impl reference: the oracle timed on the host cores (this tier's reference arm)."""
    if rank != 0:
        return
    cfg = args.config
    per_step = 4.0
    vals = []
    info = None
    for i in range(args.warmup + args.steps):
        v, info = time_oracle(cfg, per_step)
        if i >= args.warmup:
            vals.append(v)
    value = float(np.mean(vals))
    mech = inputs.config_mechanism(cfg)
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": "points/s", "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * info["seconds"],
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": f"configs[{cfg}]: {mech.n_species} species / {mech.n_reactions} reactions; "
                               f"each step a bounded sample ({info['n']} points) of the {inputs.CONFIG_POINTS[cfg]}-point workload",
                   "step": "temperature Newton solve + net production rates"},
        "cpu_baseline": {"value": value, "unit": "points/s", "cores": info["cores"], "kind": "oracle",
                         "sample": info["sample"]},
        "e2e": {"value": value, "unit": "points/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line), flush=True)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", type=int, default=2, choices=[0, 1, 2, 3, 4])
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-widened", action="store_true", help="skip the SURVEY 8(f) rows (Jacobian, transport, reactors)")
    ap.add_argument("--probes", action="store_true", help="print the design probes (DMMA peak, indexed RMW) and exit")
    ap.add_argument("--points", type=int, default=0, help="override the number of points (profiling runs)")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3) if args.impl == "ours" else args.warmup

    rank = int(os.environ.get("RANK", "0"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))

    if args.impl == "reference":
        reference_arm(args, rank)
        return

    import torch
    import torch.distributed as dist

    from paper_2503_24286_b200 import binding

    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: libpyro has no CPU fallback")
    torch.cuda.set_device(local_rank)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local_rank))

    if args.probes:
        if rank == 0:
            out = {"fp64_dfma_tflops": binding.probe_fp64_peak(local_rank, 200.0),
                   "fp64_dmma_m8n8k4_tflops": binding.probe_dmma_peak(local_rank, 200.0),
                   "indexed_rmw_cycles_per_iteration": {
                       f"{w}_warps": {name: binding.probe_indexed_rmw(local_rank, w, mode)
                                      for mode, name in ((0, "shared_rmw"), (1, "tensor_rmw"), (2, "tensor_loads"))}
                       for w in (1, 4, 8)}}
            print(json.dumps(out), flush=True)
        return

    cfg = args.config
    mech = inputs.config_mechanism(cfg)
    ns = mech.n_species
    n = args.points or inputs.CONFIG_POINTS[cfg]
    # weak scaling: every rank owns a full-size batch of independent points (own seed), no collective
    st = inputs.config_states(cfg, n=n, seed=sharding.rank_state_seed(cfg, rank), e_dtype=np.float64)
    gm = binding.Mechanism(mech, device=local_rank)
    info = gm.info()

    pin = lambda x: torch.from_numpy(np.ascontiguousarray(x)).pin_memory()
    h = {k: pin(st[k]) for k in ("rho", "e", "Y", "T_guess")}
    d = {k: v.cuda(non_blocking=True) for k, v in h.items()}
    T = torch.empty(n, dtype=torch.float64, device="cuda")
    omega = torch.empty((ns, n), dtype=torch.float64, device="cuda")
    bad = torch.zeros(1, dtype=torch.int32, device="cuda")
    stream = torch.cuda.current_stream()

    def step():
        gm.get_temperature(d["e"], d["Y"], d["T_guess"], rho=d["rho"], out=T, n_not_converged=bad, stream=stream)
        gm.get_net_production_rates(d["rho"], T, d["Y"], out=omega, stream=stream)

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    for _ in range(args.warmup):
        step()
    barrier()
    ev = [[torch.cuda.Event(enable_timing=True) for _ in range(3)] for _ in range(args.steps)]
    with ClockSampler(local_rank) as clocks:
        barrier()
        t_begin = torch.cuda.Event(enable_timing=True)
        t_end = torch.cuda.Event(enable_timing=True)
        t_begin.record(stream)
        for i in range(args.steps):
            ev[i][0].record(stream)
            gm.get_temperature(d["e"], d["Y"], d["T_guess"], rho=d["rho"], out=T, n_not_converged=bad, stream=stream)
            ev[i][1].record(stream)
            gm.get_net_production_rates(d["rho"], T, d["Y"], out=omega, stream=stream)
            ev[i][2].record(stream)
        t_end.record(stream)
        barrier()
    total_ms = t_begin.elapsed_time(t_end)
    temp_all = [e[0].elapsed_time(e[1]) for e in ev]
    rates_all = [e[1].elapsed_time(e[2]) for e in ev]
    temp_ms = float(np.median(temp_all))      # per-launch CUDA-event times: median (and min) over the timed steps
    rates_ms = float(np.median(rates_all))
    total_ms = sharding.max_over_ranks(total_ms, device="cuda")
    ms_per_step = total_ms / args.steps
    value = sharding.job_throughput(n, world, ms_per_step)
    not_converged = int(bad.item())

    # end to end through the host-buffer entry point (pinned host memory, copies inside the timed region)
    e2e = None
    if not args.no_e2e:
        T_h = torch.empty(n, dtype=torch.float64).pin_memory()
        om_h = torch.empty((ns, n), dtype=torch.float64).pin_memory()
        e2e_steps = max(2, min(args.steps, 5))
        gm.source_terms_host(h["rho"], h["e"], h["Y"], h["T_guess"], T_h, om_h)   # warm-up (allocates staging)
        barrier()
        t0 = time.perf_counter()
        for _ in range(e2e_steps):
            gm.source_terms_host(h["rho"], h["e"], h["Y"], h["T_guess"], T_h, om_h)
        torch.cuda.synchronize()
        dt = time.perf_counter() - t0
        dt = sharding.max_over_ranks(dt, device="cuda")
        e2e = {"value": world * n * e2e_steps / dt, "unit": "points/s",
               "h2d_bytes_per_step": int(8 * n * (ns + 3)), "d2h_bytes_per_step": int(8 * n * (ns + 1)),
               "steps": e2e_steps, "ms_per_step": 1e3 * dt / e2e_steps,
               "api": "pyro_source_terms_host (pinned host buffers, 3-stage slab pipeline)"}
        # the host path and the device path compute the same thing
        assert torch.equal(om_h[:, :1024], omega[:, :1024].cpu()), "host pipeline and device path disagree"

    # SURVEY.md 8(f) NEXT-1 helpers, outside the timed step: enthalpy form of the inversion and the
    # equation of state (streaming kernels; algorithmic bytes 8(N_s + 3) per point each)
    helpers = {}
    if rank == 0:
        p_in = torch.full((n,), 101325.0, dtype=torch.float64, device="cuda")
        rho_out = torch.empty(n, dtype=torch.float64, device="cuda")
        calls = {
            "temperature_from_enthalpy": lambda: gm.get_temperature_from_enthalpy(d["e"], d["Y"], d["T_guess"], out=T,
                                                                                  stream=stream),
            "density": lambda: gm.get_density(p_in, T, d["Y"], out=rho_out, stream=stream),
            "pressure": lambda: gm.get_pressure(rho_out, T, d["Y"], out=p_in, stream=stream),
        }
        for name, fn in calls.items():
            fn()
            t0, t1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            t0.record(stream)
            for _ in range(5):
                fn()
            t1.record(stream)
            torch.cuda.synchronize()
            helpers[name] = t0.elapsed_time(t1) / 5
        gm.get_temperature(d["e"], d["Y"], d["T_guess"], rho=d["rho"], out=T, n_not_converged=bad, stream=stream)
        torch.cuda.synchronize()

    widened = {}
    if rank == 0 and not args.no_widened:
        widened = time_widened_rows(gm, mech, cfg, d, T, stream, local_rank)

    if rank == 0:
        flops_pt = algorithmic_flops_per_point(mech)
        bytes_pt = algorithmic_bytes_per_point(ns)
        achieved_tflops = flops_pt * n / (rates_ms * 1e-3) / 1e12
        measured_peak = None
        try:
            measured_peak = binding.probe_fp64_peak(local_rank, 200.0)
        except Exception as ex:   # the probe is a cross-check, never the result
            measured_peak = f"unavailable: {ex}"
        peaks = {}
        try:
            peaks = json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))
        except Exception:
            pass
        hbm_peak = float(peaks.get("hbm_gbs", 6650.0))
        line = {
            "metric": METRIC, "value": value, "unit": "points/s", "n_gpus": world, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {
                "workload": f"configs[{cfg}]: {ns} species / {mech.n_reactions} reactions, {n} points per GPU, "
                            f"synthetic mechanism and states (DESIGN.md input recipe)",
                "step": "pyro_get_temperature then pyro_get_net_production_rates on one stream",
                "l2": "inputs (%.2f GB per step) are larger than the 126 MB L2; no flush needed" % (8e-9 * n * (ns + 3)),
                "block_threads": info["block_threads"], "blocks_per_sm": info["blocks_per_sm"],
                "smem_bytes_per_block": info["smem_bytes"], "tables_in_shared": info["tables_in_shared"], "tmem_columns": info["tmem_columns"],
                "registers": info["registers"], "spill_bytes": info["local_bytes"],
                "points_per_thread": info["points_per_thread"],
                "newton_not_converged": not_converged,
            },
            "kernels_ms": {"temperature": temp_ms, "rates": rates_ms, "temperature_min": float(min(temp_all)),
                           "rates_min": float(min(rates_all)), "statistic": "median and min of the per-launch event times"},
            "roofline": {
                "bound": "alu", "kernel": "rates2_kernel" if info["points_per_thread"] == 2 else "rates_kernel", "achieved": achieved_tflops, "peak": FP64_PEAK_TFLOPS,
                "unit": "TFLOP/s", "frac": achieved_tflops / FP64_PEAK_TFLOPS,
                "traffic": NCU_RATES_DRAM_BYTES_PER_POINT_53SP * n if ns == 53 else None,
                "traffic_note": "bytes per launch, ncu dram read + write of one profiled launch scaled by points; "
                                "algorithmic bytes per launch = %.4g" % (bytes_pt["rates"] * n),
                "flops_per_point": flops_pt,
                "frac_is": "algorithmic flops (SURVEY 8(d): two libm exponentials per reversible reaction) / time / peak",
                "executed_frac": (NCU_RATES_EXECUTED_FLOPS_PER_POINT_53SP * n / (rates_ms * 1e-3) / 1e12 / FP64_PEAK_TFLOPS
                                  if ns == 53 else None),
                "fp64_pipe_pct": NCU_RATES_FP64_PIPE_PCT_53SP if ns == 53 else None,
                "executed_note": "executed flops per point and FP64-pipe busy share from the committed ncu capture "
                                 "(profiles/r02_kernels.md), scaled by this run's time",
                "peak_source": "148 SMs x 64 FP64 FMA lanes x 2 x 1.965 GHz (DESIGN.md); measured DFMA probe alongside",
                "measured_dfma_tflops": measured_peak,
                "hbm": {"achieved_gbs": bytes_pt["rates"] * n / (rates_ms * 1e-3) / 1e9, "peak_gbs": hbm_peak,
                        "frac": bytes_pt["rates"] * n / (rates_ms * 1e-3) / 1e9 / hbm_peak,
                        "peak_source": "MEASURED_PEAKS.json" if peaks else "fallback 6.65 TB/s"},
                "temperature_kernel_hbm": {"achieved_gbs": bytes_pt["temperature"] * n / (temp_ms * 1e-3) / 1e9,
                                           "frac": bytes_pt["temperature"] * n / (temp_ms * 1e-3) / 1e9 / hbm_peak},
            },
            "next1_helpers_ms": {k: {"ms": v, "hbm_frac": min(1.0, 8.0 * (ns + 3) * n / (v * 1e-3) / 1e9 / hbm_peak),
                                     "gbs": 8.0 * (ns + 3) * n / (v * 1e-3) / 1e9,
                                     "note": "peak = measured COPY bandwidth; a read-only stream can exceed it: fraction capped at 1"}
                                 for k, v in helpers.items()},
            "clocks": clocks.summary(),
            "gpu_launches": 2 * args.steps,
        }
        line.update(widened)
        if e2e:
            line["e2e"] = e2e
        if not args.no_cpu_baseline and world == 1:
            v, binfo = time_oracle(cfg, 15.0)
            line["cpu_baseline"] = {"value": v, "unit": "points/s", "cores": binfo["cores"], "kind": "oracle",
                                    "sample": binfo["sample"]}
        print(json.dumps(line), flush=True)
    if world > 1:
        dist.barrier()
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
