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

# ncu figures of the graded rates kernel (DRAM bytes, executed FP64 instructions, FP64-pipe share) are NOT literals here:
# they are read from the round's committed capture summary, which `python bench.py --ncu-summary <raw.csv>` writes from
# `ncu -i <rep> --page raw --csv`, and are reported only while the kernel in the library is the one that was captured
# (same mechanism size, same registers per thread); otherwise the fields are null.
NCU_RATES_CAPTURE = os.path.join(ROOT, "profiles", "r03_rates_capture.csv")
NCU_COLUMNS = {
    "registers": "launch__registers_per_thread", "duration_ns": "gpu__time_duration.sum",
    "dram_read_bytes": "dram__bytes_read.sum", "dram_write_bytes": "dram__bytes_write.sum",
    "dfma_per_cycle": "smsp__sass_thread_inst_executed_op_dfma_pred_on.sum.per_cycle_elapsed",
    "dadd_per_cycle": "smsp__sass_thread_inst_executed_op_dadd_pred_on.sum.per_cycle_elapsed",
    "dmul_per_cycle": "smsp__sass_thread_inst_executed_op_dmul_pred_on.sum.per_cycle_elapsed",
    "cycles": "smsp__cycles_elapsed.max",
    "fp64_pipe_pct": "sm__pipe_fp64_cycles_active.avg.pct_of_peak_sustained_active",
    "issue_active_pct": "smsp__issue_active.avg.pct_of_peak_sustained_active",
    "warp_instructions": "smsp__inst_executed.sum",
}


def write_ncu_summary(raw_csv, points, n_species, n_reactions, out_path=NCU_RATES_CAPTURE):
    """`ncu -i <rep> --page raw --csv` of ONE launch of the rates kernel -> the one-row summary bench.py reads."""
    import csv
    rows = list(csv.reader(open(raw_csv)))
    head = next(i for i, r in enumerate(rows) if "Kernel Name" in r)
    names, units, vals = rows[head], rows[head + 1], rows[head + 2]
    col = {nm: i for i, nm in enumerate(names)}
    scale = {"byte": 1.0, "Kbyte": 1e3, "Mbyte": 1e6, "Gbyte": 1e9, "ns": 1.0, "us": 1e3, "ms": 1e6, "s": 1e9}

    def get(metric):
        i = col[metric]
        return float(vals[i].replace(",", "")) * scale.get(units[i], 1.0)
    rec = {k: get(m) for k, m in NCU_COLUMNS.items()}
    rec.update(kernel=vals[col["Kernel Name"]].split("(")[0], points=points, n_species=n_species, n_reactions=n_reactions,
               fp64_flops=(rec["dadd_per_cycle"] + rec["dmul_per_cycle"] + 2.0 * rec["dfma_per_cycle"]) * rec["cycles"])
    keys = ["kernel", "n_species", "n_reactions", "points", "registers", "duration_ns", "dram_read_bytes", "dram_write_bytes",
            "cycles", "dfma_per_cycle", "dadd_per_cycle", "dmul_per_cycle", "fp64_flops", "fp64_pipe_pct", "issue_active_pct", "warp_instructions"]
    with open(out_path, "w", newline="") as f:
        w = csv.writer(f)
        w.writerow(keys)
        w.writerow([rec[k] for k in keys])
    return rec


def read_ncu_summary(n_species, n_reactions, registers, path=NCU_RATES_CAPTURE):
    """The committed capture as a dict, or None when there is none for this mechanism size and kernel build."""
    import csv
    try:
        rec = next(csv.DictReader(open(path)))
    except (OSError, StopIteration):
        return None
    if int(float(rec["n_species"])) != n_species or int(float(rec["n_reactions"])) != n_reactions:
        return None
    if int(float(rec["registers"])) != int(registers):
        return None
    return {k: (v if k == "kernel" else float(v)) for k, v in rec.items()}


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


def tempered_window(lam, ratio=10.0):
    """The most populated window [L, ratio L] of the per-reactor stiffness `lam` (finite, positive entries only):
    (indices of its reactors, largest lam among them).  The synthetic mechanisms span 100+ decades of time scale from
    state to state, so a step that fits one reactor leaves nearly all others unchanged (or unstable); the reactor legs
    are timed on the states of one such window so that the march does work for every reactor."""
    lam = np.asarray(lam, dtype=np.float64)
    idx = np.nonzero(np.isfinite(lam) & (lam > 0))[0]
    if idx.size == 0:
        return idx, None
    order = idx[np.argsort(lam[idx])]
    srt = lam[order]
    hi = np.searchsorted(srt, ratio * srt, side="right")
    i = int(np.argmax(hi - np.arange(srt.size)))
    return order[i:hi[i]], float(srt[hi[i] - 1])


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
        # the reactors' own chemical time scales: lambda_p = largest row sum of |J|/rho (bounds the stiffness of reactor p)
        lam = (J.abs().sum(dim=1) / rho_j[None, :]).amax(dim=0).cpu().numpy()
    except binding.PyroError as ex:
        out["next2_jacobian"] = {"unavailable": str(ex)}
        lam = None
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
    # ---- NEXT-4: RK4 reactors, 4 stages (Newton solve + rates) per step, on a TEMPERED batch: the states whose lambda_p
    # fall into the most populated decade [L, 10 L] of the slice, repeated to the batch size, so that one step size
    # (dt lambda_p in [0.02, 0.2]) moves every reactor and the stages' Newton solves really iterate
    sel, lam_max = tempered_window(lam) if lam is not None else (np.empty(0, dtype=np.int64), None)
    if len(sel):
        nr = int(min(n, 1 << 20))
        steps = 4
        dt = 0.2 / lam_max
        rep = torch.from_numpy(sel[np.arange(nr) % len(sel)]).cuda()
        rho_r, e_r = d["rho"][rep].contiguous(), d["e"][rep].contiguous()
        Y_0, T_0 = d["Y"][:, rep].contiguous(), d["T_guess"][rep].contiguous()
        work = torch.empty((ns, nr), dtype=torch.float64, device="cuda")
        Y_r, T_r = Y_0.clone(), T_0.clone()
        bad_r = torch.zeros(1, dtype=torch.int32, device="cuda")

        def moved(Y1, Y0, thr):
            return float((((Y1 - Y0).abs() / (Y0.abs() + 1e-30)).amax(dim=0) > thr).float().mean().item())

        def march():
            Y_r.copy_(Y_0)
            T_r.copy_(T_0)
            gm.reactor_rk4(rho_r, e_r, Y_r, T_r, dt, steps, work=work, n_not_converged=bad_r, stream=stream)
        copy_ms, _ = _event_times(lambda: (Y_r.copy_(Y_0), T_r.copy_(T_0)), stream, 5)
        ms, mn = _event_times(march, stream, 5)
        ms, mn = ms - copy_ms, mn - copy_ms
        fl = 4 * algorithmic_flops_per_point(mech) + 4 * (25 * ns + FLOPS_DIV + 4) * 4
        out["next4_reactor_rk4"] = {
            "reactors": nr, "steps": steps, "dt": dt, "ms": ms, "ms_min": mn,
            "batch": f"tempered: {len(sel)} of the {len(lam)} states of the Jacobian slice have lambda_p within a factor 10 "
                     f"below {lam_max:.3e} 1/s, repeated to {nr} reactors; dt = 0.2 / lambda_max",
            "reactor_steps_per_s": nr * steps / (ms * 1e-3), "ns_per_reactor_stage": ms * 1e6 / nr / steps / 4,
            "finite_fraction": float(torch.isfinite(Y_r).all(dim=0).float().mean().item()),
            "moved_fraction_1e-6": moved(Y_r, Y_0, 1e-6), "moved_fraction_1e-3": moved(Y_r, Y_0, 1e-3),
            "max_dT_K": float((T_r - T_0).abs().max().item()),
            "roofline": {"bound": "alu", "achieved": fl * nr * steps / (ms * 1e-3) / 1e12, "peak": FP64_PEAK_TFLOPS,
                         "unit": "TFLOP/s", "frac": fl * nr * steps / (ms * 1e-3) / 1e12 / FP64_PEAK_TFLOPS,
                         "flops_per_reactor_step": float(fl), "peak_kind": "derived FP64 FMA peak"}}
        # implicit march at ten times that step: one Crank-Nicolson step of 3 Newton iterations
        # (temperature + rates + Jacobian + LU each) on the same tempered batch
        nc = int(min(n, 1 << 16))
        rho_c, e_c = rho_r[:nc].contiguous(), e_r[:nc].contiguous()
        Y_c0, T_c0 = Y_0[:, :nc].contiguous(), T_0[:nc].contiguous()
        Y_c, T_c = Y_c0.clone(), T_c0.clone()
        iters = 3
        try:
            def cn():
                Y_c.copy_(Y_c0)
                T_c.copy_(T_c0)
                gm.reactor_cn(rho_c, e_c, Y_c, T_c, 10.0 * dt, 1, newton_iters=iters, stream=stream)
            ms, mn = _event_times(cn, stream, 3, warm=1)
            need_bytes = 16.0 * ns * ns                            # J written by the Jacobian kernel, read once by the solve
            lu_bytes = 8.0 * (ns ** 3 / 12.0 + 2.5 * ns * ns)      # what the per-point panel LU moves as written
            out["next4_reactor_cn"] = {
                "reactors": nc, "steps": 1, "newton_iters": iters, "dt": 10.0 * dt, "ms": ms, "ms_min": mn,
                "batch": "the first reactors of the tempered RK4 batch; dt lambda_p / 2 in [0.1, 1]",
                "ns_per_reactor_iteration": ms * 1e6 / nc / iters,
                "finite_fraction": float(torch.isfinite(Y_c).all(dim=0).float().mean().item()),
                "moved_fraction_1e-3": moved(Y_c, Y_c0, 1e-3),
                "roofline": {"bound": "hbm", "achieved": need_bytes * nc * iters / (ms * 1e-3) / 1e9, "peak": hbm_peak, "unit": "GB/s",
                             "frac": need_bytes * nc * iters / (ms * 1e-3) / 1e9 / hbm_peak,
                             "bytes_per_reactor_iteration": need_bytes,
                             "as_written_frac": lu_bytes * nc * iters / (ms * 1e-3) / 1e9 / hbm_peak,
                             "note": "bytes = compulsory traffic of one Newton iteration, 16 ns^2 (the Jacobian written once and read once); "
                                     "as_written_frac counts the factor re-reads of the per-point panel LU (ns^3/12 + 2.5 ns^2 doubles per solve)"}}
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
    ap.add_argument("--scaling", default="weak", choices=["weak", "strong"],
                    help="weak: every rank owns a full-size batch of its own; strong: ONE seeded field of --points (default: the "
                         "config's size) cut into contiguous slabs of the point index, one per rank (configs[4]: slabs in z)")
    ap.add_argument("--ncu-summary", default="", metavar="RAW_CSV",
                    help="no GPU work: turn `ncu -i <rep> --page raw --csv` of one rates-kernel launch (captured with this "
                         "--config and --points) into profiles/r03_rates_capture.csv, which later runs read")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3) if args.impl == "ours" else args.warmup

    rank = int(os.environ.get("RANK", "0"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))

    if args.ncu_summary:
        m = inputs.config_mechanism(args.config)
        rec = write_ncu_summary(args.ncu_summary, args.points or inputs.CONFIG_POINTS[args.config], m.n_species, m.n_reactions)
        print(json.dumps(rec))
        return

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
    if args.scaling == "strong":
        # strong scaling: the same seeded field on every rank, of which rank r keeps the slab sharding.rank_slab gives it
        # (whole 32-point chunks; the point index runs x fastest, so the slabs of configs[4]'s 256^3 field are cut in z).
        # Points are independent: no halo, no collective, own mechanism handle per device.
        n_job = n
        full = inputs.config_states(cfg, n=n_job, seed=sharding.rank_state_seed(cfg, 0), e_dtype=np.float64)
        slab_lo, n = sharding.rank_slab(n_job, rank, world)
        st = {k: np.ascontiguousarray(v[..., slab_lo:slab_lo + n]) for k, v in full.items()}
        del full
    else:
        # weak scaling: every rank owns a full-size batch of independent points (own seed), no collective
        st = inputs.config_states(cfg, n=n, seed=sharding.rank_state_seed(cfg, rank), e_dtype=np.float64)
        n_job = world * n
    gm = binding.Mechanism(mech, device=local_rank)
    info = gm.info()
    cap = read_ncu_summary(ns, mech.n_reactions, info["registers"])

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
    value = n_job / (ms_per_step * 1e-3)      # whole job: the points all ranks processed over the slowest rank's time
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
        e2e = {"value": n_job * e2e_steps / dt, "unit": "points/s",
               "h2d_bytes_per_step": int(8 * n * (ns + 3)), "d2h_bytes_per_step": int(8 * n * (ns + 1)),
               "steps": e2e_steps, "ms_per_step": 1e3 * dt / e2e_steps,
               "api": "pyro_source_terms_host (pinned host buffers, 3-stage slab pipeline)"}
        # the host path and the device path compute the same thing
        assert torch.equal(om_h[:, :1024], omega[:, :1024].cpu()), "host pipeline and device path disagree"
        # What bounds it: the pinned copies of this box, timed alone and together (plain cudaMemcpyAsync of the step's
        # inputs and outputs, each direction on a stream of its own; wall clock around a synchronize, like the step above)
        if rank == 0:
            s_in, s_out = torch.cuda.Stream(), torch.cuda.Stream()

            def copies(up, down):
                torch.cuda.synchronize()
                t0 = time.perf_counter()
                if up:
                    with torch.cuda.stream(s_in):
                        for k in ("rho", "e", "Y", "T_guess"):
                            d[k].copy_(h[k], non_blocking=True)
                if down:
                    with torch.cuda.stream(s_out):
                        T_h.copy_(T, non_blocking=True)
                        om_h.copy_(omega, non_blocking=True)
                torch.cuda.synchronize()
                return 1e3 * (time.perf_counter() - t0)
            copies(True, True)
            h2d_ms = min(copies(True, False) for _ in range(3))
            d2h_ms = min(copies(False, True) for _ in range(3))
            both_ms = min(copies(True, True) for _ in range(3))
            e2e.update({"pcie_h2d_ms": h2d_ms, "pcie_d2h_ms": d2h_ms, "pcie_both_ms": both_ms,
                        "pcie_h2d_gbs": e2e["h2d_bytes_per_step"] / h2d_ms / 1e6, "pcie_d2h_gbs": e2e["d2h_bytes_per_step"] / d2h_ms / 1e6,
                        "pcie_bound_ms": both_ms, "frac_of_pcie": both_ms / e2e["ms_per_step"],
                        "pcie_note": "pcie_bound_ms = the step's host-to-device and device-to-host bytes copied concurrently with "
                                     "nothing else running; frac_of_pcie = that / the end-to-end step"})

    # SURVEY.md 8(f) NEXT-1 helpers, outside the timed step: enthalpy form of the inversion and the
    # equation of state (streaming kernels; algorithmic bytes 8(N_s + 3) per point each)
    helpers = {}
    newton_hist = None
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
        # Newton iteration histogram of the step's temperature solve: with the iteration cap at m the
        # kernel counts the points that needed more than m updates; differences of those counts are the histogram
        more_than = [n]
        for m in range(1, 11):
            gm.set_newton(1e-6, m)
            bad.zero_()
            gm.get_temperature(d["e"], d["Y"], d["T_guess"], rho=d["rho"], out=T, n_not_converged=bad, stream=stream)
            more_than.append(int(bad.item()))
        newton_hist = {str(m): more_than[m - 1] - more_than[m] for m in range(1, 11)}
        newton_hist[">10"] = more_than[10]
        gm.set_newton(1e-6, 10)
        bad.zero_()
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
            "warmup": args.warmup, "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": args.scaling,
            "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {
                "workload": f"configs[{cfg}]: {ns} species / {mech.n_reactions} reactions, {n} points per GPU, "
                            f"synthetic mechanism and states (DESIGN.md input recipe)"
                            + (f"; slab [{slab_lo}, {slab_lo + n}) of ONE field of {n_job} points on rank 0" if args.scaling == "strong" else ""),
                "step": "pyro_get_temperature then pyro_get_net_production_rates on one stream",
                "l2": "inputs (%.2f GB per step) are larger than the 126 MB L2; no flush needed" % (8e-9 * n * (ns + 3)),
                "block_threads": info["block_threads"], "blocks_per_sm": info["blocks_per_sm"],
                "smem_bytes_per_block": info["smem_bytes"], "tables_in_shared": info["tables_in_shared"], "tmem_columns": info["tmem_columns"],
                "registers": info["registers"], "spill_bytes": info["local_bytes"],
                "points_per_thread": info["points_per_thread"],
                "newton_not_converged": not_converged,
                "newton_iterations_histogram": newton_hist,
            },
            "kernels_ms": {"temperature": temp_ms, "rates": rates_ms, "temperature_min": float(min(temp_all)),
                           "rates_min": float(min(rates_all)), "statistic": "median and min of the per-launch event times"},
            "roofline": {
                "bound": "alu", "kernel": "rates2_kernel" if info["points_per_thread"] == 2 else "rates_kernel", "achieved": achieved_tflops, "peak": FP64_PEAK_TFLOPS,
                "unit": "TFLOP/s", "frac": achieved_tflops / FP64_PEAK_TFLOPS,
                "traffic": (cap["dram_read_bytes"] + cap["dram_write_bytes"]) / cap["points"] * n if cap else None,
                "traffic_note": "bytes per launch: ncu dram read + write of the committed capture (profiles/r03_rates_capture.csv, "
                                "one launch of this kernel build) scaled by points; null when the library's kernel is not the captured one; "
                                "algorithmic bytes per launch = %.4g" % (bytes_pt["rates"] * n),
                "flops_per_point": flops_pt,
                "frac_is": "algorithmic flops (SURVEY 8(d): two libm exponentials per reversible reaction) / time / derived FP64 peak",
                "executed_frac": cap["fp64_flops"] / cap["points"] * n / (rates_ms * 1e-3) / 1e12 / FP64_PEAK_TFLOPS if cap else None,
                "fp64_pipe_pct": cap["fp64_pipe_pct"] if cap else None,
                "executed_note": "executed FP64 flops per point (DADD + DMUL + 2 DFMA thread instructions) and FP64-pipe busy share from the "
                                 "same capture, scaled by this run's time",
                "peak_source": "148 SMs x 64 FP64 FMA lanes x 2 x 1.965 GHz (DESIGN.md); measured DFMA probe alongside",
                "measured_dfma_tflops": measured_peak,
                "hbm": {"achieved_gbs": bytes_pt["rates"] * n / (rates_ms * 1e-3) / 1e9, "peak_gbs": hbm_peak,
                        "frac": bytes_pt["rates"] * n / (rates_ms * 1e-3) / 1e9 / hbm_peak,
                        "peak_source": "MEASURED_PEAKS.json" if peaks else "fallback 6.65 TB/s"},
                "temperature_kernel_hbm": {"achieved_gbs": bytes_pt["temperature"] * n / (temp_ms * 1e-3) / 1e9,
                                           "frac": bytes_pt["temperature"] * n / (temp_ms * 1e-3) / 1e9 / hbm_peak},
            },
            "next1_helpers_ms": {k: {"ms": v, "hbm_frac": 8.0 * (ns + 3) * n / (v * 1e-3) / 1e9 / hbm_peak,
                                     "gbs": 8.0 * (ns + 3) * n / (v * 1e-3) / 1e9,
                                     "note": "peak = measured COPY bandwidth (read + write); a read-mostly stream can exceed it, so a fraction above 1 is not an error"}
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
