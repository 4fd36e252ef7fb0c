#!/usr/bin/env python3
"""bench.py -- MD steps/s and SCF iterations/s of the B200 Thomas-Fermi OFMD hot path (fp64, 1 B200).

  python bench.py [--gpus N] [--steps K] [--warmup W] [--workload c5|c1|c2|c3|c4] [--grid G] [--impl ours|reference]

A "step" is one velocity-Verlet MD step = one pass of the whole hot path (structure factor, ionic potential, Ewald,
one-center density initialisation, the SCF iterations to the stop rule, profile store, forces, integrator).
Default workload: BASELINE.json configs[4] at its largest grid -- "c5", 2000 Al ions, 384^3 grid (56.6 M points, 5.6 GB of
fields: the HBM-bound regime), T = 50 eV -- the largest single-GPU configuration.  The same line carries, under
"configs", a short run of every other MD configuration (c1..c4) unless --no-other-configs.
Prints ONE JSON line.  N > 1: independent replicas, one per rank (the
path does not shard without an FFT transpose; replicas only), launched under torchrun.
"""
from __future__ import annotations

import argparse
import csv
import json
import os
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)
import arche_inputs as ai  # noqa: E402

# Stop rule of the throughput runs: BASELINE.json's 1e-10 Ha on the free energy and 1e-8 on the relative density
# residual (reading D4).  Mixing: More's w after a warm-up with the fixed w.
TOL = dict(scf_tol_F=1e-10, scf_tol_dn=1e-8, scf_max_iter=2000, mix_warmup=3, mix_w_fixed=0.95, xc=2)
# c4 (T = 1 eV, 61-bohr cell): the longest wave has lambda = chi0/(pi k_min^2) ~ 110, so the fixed w of the warm-up must
# exceed (lambda-1)/(lambda+1): automatic w = lambda/(1+lambda), More's w once |mu_k - mu_{k-1}| < 1e-3 kT (1 - w) (reading A11b)
TOL_BY_WORKLOAD = {"c4": dict(scf_max_iter=12000, mix_w_fixed=0.0, mix_mu_tol=1e-3)}
NCU_TRAFFIC_CSV = os.path.join(ROOT, "profiles", "r02b_c5_384_ncu_full.csv")


XC_NAME = {1: "PZ81 LDA (constants as printed; eps_c, V_c jump 3e-5 Ha at r_s=1)",
           2: "PZ81 LDA (C, D at full precision from PZ's continuity conditions at r_s=1: reading A13b)"}


def tol_for(workload):
    t = dict(TOL); t.update(TOL_BY_WORKLOAD.get(workload, {}))
    return t


def bytes_per_point(nx, fused=True):
    """algorithmic HBM bytes per REAL grid point and launch of each kernel class; a half-spectrum
    complex array costs h = 16*P/nx bytes per real point (P = padded row pitch of the nx/2+1 stored columns)"""
    h = 16.0 * ((nx // 2 + 1 + 7) // 8 * 8) / nx
    if fused:
        return {"fft_inv_z_potential": 5 * h,  # read nhat_i, nhat_a, Vhat_ie; write nhat_i (fused mixing), work
                "fft_y": 2 * h,                # read + write work
                "fft_inv_x_vi": h + 32,        # read work, n_i, n_a; write n_i (fused mixing), V_i
                "mu_pass": 8,                  # per evaluation of N(mu): read V_i (L2/register-cached on small grids)
                "density": 24 + h,             # read V_i, n_i; write n_a, work (r2c x pass with the density prologue)
                "fft_fwd_z_reduce": 4 * h,     # read work, nhat_i, Vhat_ie; write nhat_a
                "mix": 16 + 3 * h,
                "stress_fields": 3 * h + 8}    # f1: read nhat_a, S_Z, S2 and n_a once
    return {"potential_g": 5 * h,              # streaming: read nhat_i, nhat_a, Vhat_ie; write nhat_i, work
            "fft_inv_z_potential": 2 * h, "fft_y": 2 * h, "fft_inv_x_vi": h + 8,      # plain passes
            "vi_r": 40,                        # read V_H, n_i, n_a; write n_i, V_i
            "mu_pass": 8,
            "density_r": 24,                   # read V_i, n_i; write n_a
            "fft_fwd_x_real": 8 + h, "fft_fwd_z_reduce": 2 * h,                        # plain passes
            "reduce_g": 3 * h,                 # read nhat_a, nhat_i, Vhat_ie
            "mix": 16 + 3 * h,
            "stress_fields": 3 * h + 8}


# fp64 work per grid point of the arithmetic-bound classes, counted from the kernels (an FMA = 2 flops): one
# Fermi-Dirac function = 11 FMA Horner + ~8 flops to locate the segment; PZ81 = cbrt + log or sqrt + 2 divisions
# ~ 90 flops; the reductions ~ 20.
FLOPS_PER_POINT = {"mu_pass": 32, "density": 3 * 30 + 90 + 20, "density_r": 3 * 30 + 90 + 20, "vi_r": 30 + 90 + 10,
                   "fft_inv_x_vi": 30 + 90 + 10}     # fft_inv_x_vi carries the V_i epilogue only in the fused form
# fp64 work per (ion, stored half-spectrum point) of the ion-grid sums in FMA-slot units (2 x fp64 pipe instructions:
# a lone multiply or add occupies the same issue slot as an FMA, and the measured peak counts an FMA as 2): S_Z one
# complex multiply-add = 4 FMAs; forces t = W a_j (2 mul + 2 FMA), P += t (2 add), Q += kx t (2 FMA) = 8 instructions
FLOPS_PER_PAIR = {"structure_factor": 8.0, "force": 16.0}
FP64_DERIVED_TFLOPS = 148 * 64 * 2 * 1.965e9 / 1e12   # unit count x clock (B200_PROFILING.md), used only if not measured


def peaks():
    try:
        with open(os.path.join(ROOT, "MEASURED_PEAKS.json")) as fh:
            return float(json.load(fh)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    except Exception:
        return 6650.0, "fallback (B200_PROFILING.md 6.65 TB/s)"


def ncu_traffic():
    """DRAM bytes per launch of each kernel class from the committed `ncu --set full` capture of this workload
    (profiles/r02b_c5_384_ncu_full.csv, written by paper_2606_13283_b200/ncu_summary.py): class -> bytes"""
    out = {}
    try:
        with open(NCU_TRAFFIC_CSV) as fh:
            for row in csv.DictReader(fh):
                if row.get("class"):
                    out.setdefault(row["class"], []).append(float(row["dram_bytes_read"]) + float(row["dram_bytes_write"]))
    except Exception:
        return {}
    return {k: float(np.mean(v)) for k, v in out.items()}


def roofline_entry(name, ms_per_launch, ng, bpp, peak_gbs, peak_src, fp64_peak, fp64_src, evals_per_launch=1.0,
                   pairs=None, flops_per_point=None):
    """roofline object of one kernel class: HBM bytes for the streaming/FFT classes, fp64 flops for the
    arithmetic-bound ones (whichever bound is the higher fraction is the binding one and is reported)"""
    t = ms_per_launch * 1e-3
    if name in FLOPS_PER_PAIR:
        tf = FLOPS_PER_PAIR[name] * pairs / t / 1e12 if t > 0 and pairs else 0.0
        return {"bound": "alu", "kernel": name, "achieved": tf, "peak": fp64_peak, "unit": "TFLOP/s",
                "frac": tf / fp64_peak, "traffic": None, "peak_source": fp64_src}
    hbm = bpp.get(name, 0.0) * evals_per_launch * ng / t / 1e9 if t > 0 else 0.0
    out = {"bound": "hbm", "kernel": name, "achieved": hbm, "peak": peak_gbs, "unit": "GB/s",
           "frac": hbm / peak_gbs, "traffic": None, "peak_source": peak_src}
    fpp = flops_per_point or FLOPS_PER_POINT
    if name in fpp and t > 0 and not (name == "fft_inv_x_vi" and "vi_r" in bpp):
        tf = fpp[name] * evals_per_launch * ng / t / 1e12
        if tf / fp64_peak > out["frac"]:
            out = {"bound": "alu", "kernel": name, "achieved": tf, "peak": fp64_peak, "unit": "TFLOP/s",
                   "frac": tf / fp64_peak, "traffic": None, "peak_source": fp64_src, "hbm_gbs": hbm}
    return out


class ClockSampler:
    """polls SM clock / throttle reasons through NVML while the timed region runs"""

    def __init__(self, index=0, period=0.02):
        self.samples, self.reasons, self.max_mhz, self._stop = [], set(), None, threading.Event()
        self.index, self.period, self.th = index, period, None

    def _run(self):
        try:
            import pynvml as nv
            nv.nvmlInit()
            h = nv.nvmlDeviceGetHandleByIndex(self.index)
            self.max_mhz = nv.nvmlDeviceGetMaxClockInfo(h, nv.NVML_CLOCK_SM)
            names = {"hw_slowdown": 0x8, "sw_power_cap": 0x4, "hw_thermal_slowdown": 0x40,
                     "sw_thermal_slowdown": 0x20, "hw_power_brake": 0x80}
            while not self._stop.is_set():
                self.samples.append(nv.nvmlDeviceGetClockInfo(h, nv.NVML_CLOCK_SM))
                r = nv.nvmlDeviceGetCurrentClocksThrottleReasons(h)
                for k, bit in names.items():
                    if r & bit:
                        self.reasons.add(k)
                time.sleep(self.period)
        except Exception as e:  # NVML missing: report it instead of inventing numbers
            self.reasons.add(f"nvml_unavailable:{type(e).__name__}")

    def __enter__(self):
        self.th = threading.Thread(target=self._run, daemon=True); self.th.start(); return self

    def __exit__(self, *a):
        self._stop.set(); self.th.join(timeout=2)

    def summary(self):
        return {"sm_mhz": float(np.median(self.samples)) if self.samples else None, "sm_max_mhz": self.max_mhz,
                "reasons": sorted(self.reasons)}


# ------------------------------------------------------------------------------------------------ oracle legs
ORACLE_SAMPLE_GRID = {"c5": 32, "c4": 32, "c3": 32}   # bounded samples of the large workloads run on a coarser grid


def oracle_sample(cfg, workload, iters_per_step=None, target_s=12.0, max_iters=40):
    """Bounded oracle sample of one MD step of `workload` (the oracle as it stands, all host cores): the per-step
    ion-grid work, a few SCF iterations from the uniform start and the forces.  Workloads whose grid the oracle cannot
    do in seconds (c3, c4, c5) are sampled on a coarser grid of the SAME cell and ions and scaled linearly in N_g
    (every stage of the oracle is O(N_g) or O(N_i N_g)) -- labelled extrapolated.  MD step = ion work +
    iterations/step x time per iteration + forces, with the iterations per step the GPU run observed (when given) or the
    oracle's own count of a converged solve on a 16^3 grid of the same cell."""
    import oracle
    tol = tol_for(workload)
    full_ng = int(np.prod(cfg["grid"]))
    g = ORACLE_SAMPLE_GRID.get(workload)
    scfg = dict(cfg)
    if g and g ** 3 < full_ng:
        scfg["grid"] = np.array([g, g, g], dtype=np.int32)
    scale = full_ng / float(np.prod(scfg["grid"]))
    o = oracle.Oracle(scfg, **tol)
    t0 = time.perf_counter(); o.scf_begin(scfg["pos"]); t_ion = time.perf_counter() - t0
    t0 = time.perf_counter(); o.scf_iter(); t_first = time.perf_counter() - t0
    iters = max(1, min(max_iters, int((target_s - t_ion) / max(t_first, 1e-3)) - 1))
    t0 = time.perf_counter()
    for _ in range(iters):
        o.scf_iter()
    t_it = (time.perf_counter() - t0 + t_first) / (iters + 1)
    t0 = time.perf_counter(); o.forces(); t_force = time.perf_counter() - t0
    src = "iterations per step observed by the GPU run"
    if iters_per_step is None:
        tiny = dict(cfg); tiny["grid"] = np.array([16, 16, 16], dtype=np.int32)
        ot = oracle.Oracle(tiny, **tol)
        iters_per_step = float(ot.scf_solve(tiny["pos"])["scf_iters"])
        src = "the oracle's own iteration count of a converged solve on a 16^3 grid of the same cell"
    step_s = scale * (iters_per_step * t_it + t_ion + t_force)
    gs = [int(x) for x in scfg["grid"]]
    return dict(value=1.0 / step_s, unit="md_steps/s", cores=oracle.lib().oracle_num_threads(), kind="oracle",
                sample=f"{iters + 1} SCF iterations ({t_it:.2f} s each) + structure factor/Ewald ({t_ion:.2f} s) + forces "
                       f"({t_force:.2f} s) of {workload} on grid {gs}"
                       + (f", EXTRAPOLATED x{scale:.0f} linearly in N_g to the full grid" if scale > 1 else "")
                       + f"; MD step = ion work + {iters_per_step:.0f} iterations + forces ({src})",
                scf_iters_per_s=1.0 / (scale * t_it), extrapolated=True)


def run_reference(args, cfg):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    vals = []
    for _ in range(args.warmup + args.steps):
        vals.append(oracle_sample(cfg, args.workload, target_s=4.0, max_iters=3))   # one bounded sample per "step"
    use = vals[args.warmup:] or vals
    v = float(np.mean([x["value"] for x in use]))
    cb = dict(use[-1]); cb["value"] = v
    line = {"impl": "reference", "metric": "md_steps_per_s", "value": v, "unit": "md_steps/s", "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 / v, "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": dict(workload_config(cfg, args.workload), free_energy="evaluated in every SCF iteration (the oracle)"),
            "cpu_baseline": cb,
            "e2e": {"value": v, "unit": "md_steps/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "note": "the CPU oracle as it stands; ms_per_step is the extrapolated full-size MD step, not an observed time"}
    print(json.dumps(line))


def workload_config(cfg, name):
    tol = tol_for(name)
    ng = int(np.prod(cfg["grid"]))
    mix = ("More w = U/(K+U) after 3 warm-up iterations at w = 0.95" if tol.get("mix_mu_tol", 0) <= 0 else
           f"warm-up at the automatic w = lambda/(1+lambda), More w = U/(K+U) once |d mu| < {tol['mix_mu_tol']:g} kT (1 - w) (P:311)")
    return {"workload": f"{name}: {len(cfg['Z'])} Al ions (Z=3), cell {[round(float(x), 4) for x in cfg['cell']]} bohr, "
                        f"grid {[int(g) for g in cfg['grid']]} ({ng / 1e6:.2f} M points), T={cfg['T_eV']} eV, "
                        f"dt={cfg['dt'] / ai.FS_AU:.2f} fs, TF + {XC_NAME[tol['xc']]} + Ashcroft rc=1.12, one-center init; one step = one "
                        f"velocity-Verlet MD step with the SCF run to its stop rule",
            "stop_rule": f"|dF|<{tol['scf_tol_F']:g} Ha and ||n_i-n_a||/||n_a||<{tol['scf_tol_dn']:g}" +
                         (" (widened by two PZ81 branch-flip quanta when a flip is detected: DESIGN.md reading A13; "
                          "flagged per run as flip_steps)" if tol["xc"] == 1 else " (strict: the XC potential is continuous)"),
            "mixing": mix,
            "free_energy": ("evaluated in every SCF iteration" if tol["xc"] == 1 or os.environ.get("ARCHE_LAZY_F", "1")[0] == "0" else
                            "evaluated only in the iterations where the stop rule can use it (the last ones of a solve; "
                            "free_energy_evals_per_step in the line; DESIGN.md section 5)"),
            "l2": ("L2 flushed between timed steps (256 MiB write); fields of %.1f GB per step exceed the 126 MB L2"
                   % (99.0 * ng / 1e9) if ng >= 192 ** 3 else
                   "L2 flushed between timed steps (256 MiB write); the working set is L2-resident within a step")}


def replica_config(cfg, rank, world):
    """N > 1 runs independent replicas: same recipe, rank-dependent thermal displacement"""
    if world > 1:
        rng = np.random.default_rng(1000 + rank)
        cfg = dict(cfg)
        cfg["pos"] = np.mod(cfg["pos"] + 0.05 * rng.standard_normal(cfg["pos"].shape), cfg["cell"])
    return cfg


def max_over_ranks(values, device=None):
    """element-wise MAX of a list of floats over all ranks of the default process group (NCCL on GPUs, gloo in tests)"""
    import torch
    import torch.distributed as dist
    t = torch.tensor(values, dtype=torch.float64, device=device)
    if dist.is_available() and dist.is_initialized() and dist.get_world_size() > 1:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return t.tolist()


# ------------------------------------------------------------------------------------------------ GPU legs
class MdRun:
    """device-timed MD steps of one workload through the C ABI"""

    def __init__(self, cfg, workload, dev, flush):
        import torch
        from paper_2606_13283_b200 import Arche
        self.torch, self.cfg, self.workload, self.dev, self.flush = torch, cfg, workload, dev, flush
        self.g = Arche(cfg, device=dev, **tol_for(workload))
        self.pos = torch.as_tensor(cfg["pos"].copy(), device=dev)
        self.vel = torch.as_tensor(cfg["vel"].copy(), device=dev)
        self.dt = cfg["dt"]

    def timed(self, K, step_fn):
        torch = self.torch
        ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(K)]
        out = dict(iters=0, mu_evals=0, not_converged=0, flips=0, F_evals=0)
        for a, b in ev:
            self.flush.fill_(1)                      # evict L2 between timed steps
            a.record(self.g.stream)
            r = step_fn()
            b.record(self.g.stream)
            out["iters"] += r["scf_iters"]; out["mu_evals"] += r["mu_evals"]; out["F_evals"] += r.get("F_evals", r["scf_iters"])
            out["not_converged"] += int(r["converged"] != 1 or r["rc"] != 0); out["flips"] += int(r["flip_seen"])
        torch.cuda.synchronize()
        out["seconds"] = sum(a.elapsed_time(b) for a, b in ev) * 1e-3
        return out

    def device_arm(self, K, W):
        for _ in range(W):
            self.g.md_step(self.dt, self.pos, self.vel)
        self.torch.cuda.synchronize()
        l0 = self.g.launch_count()
        out = self.timed(K, lambda: self.g.md_step(self.dt, self.pos, self.vel))
        out["launches"] = self.g.launch_count() - l0
        return out

    def host_arm(self, K, W=2):
        """the same step through arche_md_step_host: pinned host buffers, H2D of positions/velocities and D2H of
        positions/velocities/forces + the result struct inside the timed region"""
        torch = self.torch
        n = self.g.n_ions
        self.hp = torch.empty((n, 3), dtype=torch.float64).pin_memory(); self.hv = torch.empty_like(self.hp).pin_memory()
        self.hF = torch.empty_like(self.hp).pin_memory()
        self.hp.copy_(self.pos.cpu()); self.hv.copy_(self.vel.cpu())
        for _ in range(W):
            self.g.md_step_host(self.dt, self.hp, self.hv, self.hF)
        out = self.timed(K, lambda: self.g.md_step_host(self.dt, self.hp, self.hv, self.hF))
        out["h2d_bytes_per_step"] = 2 * 3 * n * 8
        out["d2h_bytes_per_step"] = 3 * 3 * n * 8 + 144
        return out

    def profile_arm(self, K):
        """second pass over the following K steps with CUDA events around every launch of each kernel class"""
        pos2 = self.torch.as_tensor(self.hp.numpy().copy(), device=self.dev) if hasattr(self, "hp") else self.pos
        vel2 = self.torch.as_tensor(self.hv.numpy().copy(), device=self.dev) if hasattr(self, "hv") else self.vel
        self.g.profile_enable(True)
        out = self.timed(K, lambda: self.g.md_step(self.dt, pos2, vel2))
        out["prof"] = self.g.profile_get()
        self.g.profile_enable(False)
        self.vel2 = vel2
        return out


def class_table(run, prof_out, K, dev_out, peak, peak_src, fp64_peak, fp64_src, traffic):
    g = run.g
    prof = prof_out["prof"]
    ng = g.ng
    bpp = bytes_per_point(g.grid[0], g.is_fused())
    tot = sum(v[0] for v in prof.values()) or 1.0
    evals_per_iter = dev_out["mu_evals"] / max(dev_out["iters"], 1)
    # lazy free energy: only the fraction f_F of the iterations evaluates I_{3/2}, eps_xc (density classes) and E_ie
    # (the Vhat_ie read of the S5 reduction); the launches of a class are timed together, so the work per launch is
    # the mix of the two forms
    f_F = prof_out["F_evals"] / max(prof_out["iters"], 1)
    bpp = dict(bpp)
    h = 16.0 * ((g.grid[0] // 2 + 1 + 7) // 8 * 8) / g.grid[0]
    if "reduce_g" in bpp:
        bpp["reduce_g"] = (2.0 + f_F) * h
    elif "fft_fwd_z_reduce" in bpp:
        bpp["fft_fwd_z_reduce"] = (3.0 + f_F) * h
    flops = dict(FLOPS_PER_POINT)
    for k in ("density", "density_r"):
        flops[k] = (2 * 30 + 14) + f_F * (30 + 90 + 6)
    P = (g.grid[0] // 2 + 1 + 7) // 8 * 8
    pairs = float(g.n_ions) * P * g.grid[1] * g.grid[2]
    rl, kernels = {}, {}
    for k, (ms, n) in prof.items():
        if not n:
            continue
        ent = {"ms_total": round(ms, 4), "launches": n, "share": round(ms / tot, 4), "us_per_launch": round(1e3 * ms / n, 2)}
        if k in bpp or k in FLOPS_PER_POINT or k in FLOPS_PER_PAIR:
            # the mu kernel's launches carry (evals_per_iter - 1) evaluations each: the first rides in the S2 pass
            per = max(evals_per_iter - 1.0, 1e-9) if k == "mu_pass" else 1.0
            e = roofline_entry(k, ms / n, ng, bpp, peak, peak_src, fp64_peak, fp64_src, per, pairs, flops)
            e["traffic"] = traffic.get(k)
            rl[k] = e
            ent.update({"bound": e["bound"], "achieved": round(e["achieved"], 2), "unit": e["unit"], "frac": round(e["frac"], 4)})
            if e["traffic"] is not None:
                ent["ncu_dram_bytes_per_launch"] = e["traffic"]
                ent["algorithmic_bytes_per_launch"] = bpp.get(k, 0.0) * per * ng
        kernels[k] = ent
    for k in ("density", "density_r", "reduce_g", "fft_fwd_z_reduce"):
        if k in kernels:
            kernels[k]["free_energy_fraction_of_launches"] = round(f_F, 4)
    return rl, kernels, tot, evals_per_iter, bpp


def persistent_roofline(run, prof, rl_bpp, evals_per_iter, tot_prof, l2_peak, peak, peak_src):
    """c1 / c2: the SCF loop is ONE kernel on an L2-resident grid.  Its bound is the L2, not HBM: the iteration's
    algorithmic traffic over the kernel's time against the measured L2 read bandwidth (and, for the record, HBM)."""
    g = run.g
    scf_classes = ("fft_inv_z_potential", "fft_y", "fft_inv_x_vi", "mu_pass", "density", "fft_fwd_z_reduce")
    bpi = sum(rl_bpp[k] * (2 if k == "fft_y" else max(evals_per_iter - 1.0, 0.0) if k == "mu_pass" else 1)
              for k in scf_classes) * g.ng
    t_scf = sum(prof[k][0] for k in scf_classes) * 1e-3
    n_it = max(prof["density"][1], 1)
    ach = bpi * n_it / t_scf / 1e9
    return {"bound": "l2", "kernel": f"scf_persistent_kernel<{g.grid[0]},{g.grid[1]},{g.grid[2]}> (whole SCF loop, one launch "
            "per solve)", "achieved": ach, "peak": l2_peak, "unit": "GB/s", "frac": ach / l2_peak,
            "peak_source": "measured in this run (arche_peak_l2: 32 MiB swept 64 times by all SMs)",
            "frac_of_hbm_peak": ach / peak, "share_of_step": round(t_scf * 1e3 / tot_prof, 4), "bytes_per_iteration": bpi,
            "us_per_iteration": round(1e6 * t_scf / n_it, 2), "traffic": None,
            "note": "fields are L2-resident: latency/barrier-bound, not HBM-bound (DESIGN.md section 5)"}


def bench_config_block(name, dev, flush, K, W, peak, peak_src, fp64_peak, fp64_src, l2_peak):
    """short run of one of the other MD configurations for the "configs" block of the line"""
    cfg = ai.make_config(name)
    run = MdRun(cfg, name, dev, flush)
    d = run.device_arm(K, W)
    h = run.host_arm(K, 1)
    p = run.profile_arm(K)
    rl, kernels, tot, epi, bpp = class_table(run, p, K, d, peak, peak_src, fp64_peak, fp64_src, {})
    blk = {"workload": workload_config(cfg, name)["workload"], "steps": K, "warmup": W,
           "md_steps_per_s": K / d["seconds"], "ms_per_step": 1e3 * d["seconds"] / K,
           "scf_iterations_per_s": d["iters"] / d["seconds"], "scf_iters_per_step": d["iters"] / K,
           "free_energy_evals_per_step": d["F_evals"] / K, "e2e_md_steps_per_s": K / h["seconds"], "not_converged_steps": d["not_converged"], "flip_steps": d["flips"],
           "gpu_launches": int(d["launches"]), "mixing": workload_config(cfg, name)["mixing"],
           "form": "persistent" if run.g.is_persistent() else ("fused" if run.g.is_fused() else "streamed"),
           "kernels": {k: {kk: v[kk] for kk in ("share", "us_per_launch", "bound", "frac") if kk in v} for k, v in kernels.items()}}
    if run.g.is_persistent():
        blk["roofline"] = persistent_roofline(run, p["prof"], bpp, epi, tot, l2_peak, peak, peak_src)
    elif rl:
        dom = max(rl, key=lambda k: p["prof"][k][0])
        blk["roofline"] = dict(rl[dom]); blk["roofline"]["share_of_step"] = round(p["prof"][dom][0] / tot, 4)
    del run
    return blk


def sweep_point(grid, dev, iters=20):
    """BASELINE.json configs[4] as written: ONE SCF iteration (from the uniform start, after 3 warm-up iterations) and one
    force evaluation of the 2000-ion cell on a grid^3 mesh -- the linear-scaling check in the number of grid points"""
    import torch
    from paper_2606_13283_b200 import Arche
    cfg = ai.make_config("c5", grid=grid)
    g = Arche(cfg, device=dev, **tol_for("c5"))
    pos = torch.as_tensor(cfg["pos"], device=dev)
    ev = [torch.cuda.Event(enable_timing=True) for _ in range(6)]
    g.scf_begin(pos)                                   # warm-up of the ion-grid kernels
    ev[0].record(g.stream); g.scf_begin(pos); ev[1].record(g.stream)
    for _ in range(3):
        g.scf_iter()
    ev[2].record(g.stream)
    for _ in range(iters):
        g.scf_iter()
    ev[3].record(g.stream)
    g.forces()
    ev[4].record(g.stream); g.forces(); ev[5].record(g.stream)
    torch.cuda.synchronize()
    it_ms = ev[2].elapsed_time(ev[3]) / iters
    out = {"grid": grid, "ms_per_scf_iteration": it_ms, "scf_iterations_per_s": 1e3 / it_ms,
           "grid_points_per_s": g.ng / it_ms * 1e3, "ion_grid_work_ms": ev[0].elapsed_time(ev[1]),
           "force_evaluation_ms": ev[4].elapsed_time(ev[5]), "form": "fused" if g.is_fused() else "streamed"}
    del g
    return out


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--workload", default="c5")
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-other-configs", action="store_true", help="skip the short c1..c4 runs of the 'configs' block")
    ap.add_argument("--grid", type=int, default=0, help="with --workload c5: grid size (default 384)")
    ap.add_argument("--xc", type=int, default=2, choices=[1, 2],
                    help="2 (default): PZ81 with C, D at full precision (continuous at r_s = 1, strict stop rule); 1: as printed")
    args = ap.parse_args()
    TOL["xc"] = args.xc
    cfg = ai.make_config(args.workload, grid=(args.grid or None) if args.workload == "c5" else None)
    if args.impl == "reference":
        return run_reference(args, cfg)

    import torch
    import torch.distributed as dist
    world = int(os.environ.get("WORLD_SIZE", "1")); rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device(f"cuda:{local}"))
    torch.cuda.set_device(local)
    dev = f"cuda:{local}"
    cfg = replica_config(cfg, rank, world)
    flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev)
    W = max(args.warmup, 3)
    K = args.steps

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    run = MdRun(cfg, args.workload, dev, flush)
    g = run.g
    # ---- measured rooflines of this run: fp64 FMA rate of the vector pipe, L2 read bandwidth (HBM: MEASURED_PEAKS.json)
    pk = g.peak_fp64(1.0)
    fp64_peak, fp64_src = pk["sustained_tflops"], "measured in this run (arche_peak_fp64: dependent DFMA chains on all SMs for 1 s)"
    l2_peak = g.peak_l2()
    peak, peak_src = peaks()
    # ---- device-resident arm
    for _ in range(W):
        g.md_step(run.dt, run.pos, run.vel)
    barrier()
    l0 = g.launch_count()
    with ClockSampler(local) as cs:
        d = run.timed(K, lambda: g.md_step(run.dt, run.pos, run.vel))
    launches = g.launch_count() - l0
    barrier()
    # ---- end-to-end arm: host buffers through the C ABI
    h = run.host_arm(K, 2)
    barrier()
    # ---- per-kernel-class timing of the following steps (second pass, CUDA events around every launch)
    p = run.profile_arm(K)
    # ---- f1: stress tensor + pressure of the last step's state (reported beside the step, not inside its timed region)
    for _ in range(2):
        g.stress(run.vel2)
    s0 = torch.cuda.Event(enable_timing=True); s1 = torch.cuda.Event(enable_timing=True)
    ls = g.launch_count()
    s0.record(g.stream)
    for _ in range(5):
        st = g.stress(run.vel2)
    s1.record(g.stream); torch.cuda.synchronize()
    stress = {"ms_per_call": s0.elapsed_time(s1) / 5, "launches_per_call": (g.launch_count() - ls) / 5,
              "pressure_Ha_per_bohr3": st["P"], "note": "arche_stress incl. its D2H of 55 doubles; outside the timed MD step"}

    t_dev_max, t_e2e_max = max_over_ranks([d["seconds"], h["seconds"]], device=dev)
    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return
    traffic = ncu_traffic() if (args.workload == "c5" and g.grid[0] == 384) else {}
    rl, kernels, tot_prof, evals_per_iter, bpp = class_table(run, p, K, d, peak, peak_src, fp64_peak, fp64_src, traffic)
    if g.is_persistent():
        roof = persistent_roofline(run, p["prof"], bpp, evals_per_iter, tot_prof, l2_peak, peak, peak_src)
    else:
        dom = max(rl, key=lambda k: p["prof"][k][0])
        roof = dict(rl[dom])
        roof["share_of_step"] = round(p["prof"][dom][0] / tot_prof, 4)
        hbm_classes = [k for k in rl if rl[k]["bound"] == "hbm"]
        tot_b = sum(bpp[k] * g.ng * p["prof"][k][1] for k in hbm_classes)
        tot_t = sum(p["prof"][k][0] for k in hbm_classes) * 1e-3
        roof["hbm_classes_aggregate_gbs"] = tot_b / tot_t / 1e9 if tot_t > 0 else None
        roof["hbm_classes_aggregate_frac"] = roof["hbm_classes_aggregate_gbs"] / peak if tot_t > 0 else None
        roof["hbm_classes_share_of_step"] = round(tot_t * 1e3 / tot_prof, 4)
        if roof.get("traffic") is not None:
            roof["traffic_source"] = "dram__bytes_read.sum + dram__bytes_write.sum per launch, parsed at run time from " \
                                     "profiles/r02b_c5_384_ncu_full.csv (ncu --set full capture of this command)"
    roof["measured"] = ("second pass over the following steps with per-class timing: CUDA events on the library's stream "
                        "around every launch of the class")
    line = {"metric": "md_steps_per_s", "value": world * K / t_dev_max, "unit": "md_steps/s",
            "n_gpus": world, "steps": K, "warmup": W, "ms_per_step": 1e3 * t_dev_max / K,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": workload_config(cfg, args.workload),
            "scf_iterations_per_s": world * d["iters"] / t_dev_max, "scf_iters_per_step": d["iters"] / K,
            "ms_per_scf_iteration_incl_ion_work": 1e3 * t_dev_max / max(d["iters"], 1),
            "grid_points_per_s": world * d["iters"] * g.ng / t_dev_max,
            "not_converged_steps": d["not_converged"], "flip_steps": d["flips"],
            "free_energy_evals_per_step": d["F_evals"] / K,
            "clocks": cs.summary(),
            "e2e": {"value": world * K / t_e2e_max, "unit": "md_steps/s",
                    "h2d_bytes_per_step": h["h2d_bytes_per_step"], "d2h_bytes_per_step": h["d2h_bytes_per_step"],
                    "scf_iters_per_step": h["iters"] / K, "api": "arche_md_step_host (pinned host buffers)"},
            "gpu_launches": int(launches),
            "mu_evals_per_iter": evals_per_iter, "roofline": roof, "kernels": kernels, "stress": stress,
            "peaks": {"hbm_gbs": peak, "hbm_source": peak_src, "fp64_tflops_sustained": pk["sustained_tflops"],
                      "fp64_tflops_burst": pk["burst_tflops"], "fp64_tflops_derived": FP64_DERIVED_TFLOPS,
                      "l2_read_gbs": l2_peak}}
    if d["not_converged"]:
        line["warning"] = f"{d['not_converged']} timed step(s) hit scf_max_iter: the value is not a converged-MD rate"
    del run, g
    if world == 1 and not args.no_other_configs:
        others = [w for w in ("c1", "c2", "c3", "c4") if w != args.workload]
        line["configs"] = {}
        for w in others:
            try:
                line["configs"][w] = bench_config_block(w, dev, flush, 3 if w == "c4" else 10, 1 if w == "c4" else 3,
                                                        peak, peak_src, fp64_peak, fp64_src, l2_peak)
            except Exception as e:   # a failing side config must not lose the headline line; it is reported, not hidden
                line["configs"][w] = {"error": f"{type(e).__name__}: {e}"}
    if world == 1 and not args.no_other_configs and args.workload == "c5":
        try:
            line["c5_sweep"] = [sweep_point(n, dev) for n in (64, 128, 192, 256, 384)]
        except Exception as e:
            line["c5_sweep"] = {"error": f"{type(e).__name__}: {e}"}
    if not args.no_cpu_baseline:
        line["cpu_baseline"] = oracle_sample(cfg, args.workload, iters_per_step=d["iters"] / K)
    print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
