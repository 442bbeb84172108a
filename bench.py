"""bench.py -- throughput of the fp64 directional wavelet transform (forward + inverse) on B200.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--workload C3|C2|C1|C4|C5|T2]

`--gpus N` (N > 1) outside a launcher starts the N ranks itself (torch.distributed.run, one rank per GPU, rendezvous on
127.0.0.1); under a launcher (WORLD_SIZE set) N must equal WORLD_SIZE.

One "step" = one forward + one inverse transform of one batch of the workload (all hot-path steps a1-a8 of DESIGN.md).
The default workload is BASELINE.json's metric configuration: L = 1024, N = 5, lambda = 2, J0 = 2, multiresolution,
real fp64 signals, batch of 4 (configs[2]) -> 4 transforms per step.  Prints ONE JSON line (rank 0).

`value`  : transforms/s with inputs resident in HBM (plan-level C-ABI calls, CUDA events, max over ranks).
`e2e`    : the same metric through the host-buffer C-ABI calls (s2wav_forward_host / s2wav_inverse_host), pinned
           host memory, H2D and D2H copies inside the timed region.
`roofline`: dominant kernel class (on-the-fly Wigner contraction), bound "alu": algorithmic FP64 flops per launch
           / device time per launch measured with cudaEvents inside the library (s2w_timing_*), against the
           nominal DFMA peak 148 SMs x 64 lanes x 2 x sm_max_mhz.
`cpu_baseline`: the oracle (oracle/, double instance, OpenMP) timed on a bounded sample of the same workload.
N > 1: replicas only: every rank transforms its own batch, no data-path collective, scaling "weak".
`--impl reference` times the oracle itself (rank 0 only).
"""
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

METRIC = "fp64 wavelet fwd+inv transforms/sec"
# dram__bytes_read.sum + dram__bytes_write.sum of the dominant kernel class, summed over the launches of ONE step (like
# `achieved`, which is flops per step / ms per step), from the `ncu --set full` captures of profiles/r01j_wigner_ncu.md
# (C3, on-the-fly) and profiles/r02d_* (C4): (workload, class) -> bytes per step.  Other workloads have no capture: traffic = null.
NCU_TRAFFIC = {("C3", "wigner_forward"): 1.299e9 + 0.070e9, ("C3", "wigner_inverse"): 0.519e9 + 0.679e9,
               ("C4", "wigner_forward"): 1.618e9}   # C4: the nine forward launches of a step, profiles/r02d_*.md
NCU_TRAFFIC_SOURCE = {"C3": "profiles/r01j_wigner_ncu.md (the C3 Wigner kernels are unchanged since that capture)",
                      "C4": "profiles/r02d_wigner_forward_few_columns.md"}
UNIT = "transforms/s"


def parse_args():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="C3", choices=["C1", "C2", "C3", "C4", "C5", "T2"])
    ap.add_argument("--precompute", action="store_true",
                    help="sphere workloads: the precomputed-kernel variant (S2W_PRECOMPUTE, step a9)")
    ap.add_argument("--recursion", action="store_true",
                    help="ball workloads: S2W_RECURSION, the on-the-fly Wigner recursion where the plan would precompute")
    ap.add_argument("--adjoint", action="store_true",
                    help="sphere workloads: time the adjoint pair S^H (signal -> coefficients) + A^H (coefficients -> "
                         "signal) of the workload's plan (SURVEY 8(f)-1); no e2e / cpu_baseline")
    ap.add_argument("--dry-run-cpu", action="store_true",
                    help="launcher check without GPUs: the N ranks rendezvous over gloo, report rank / seed offset / pid, "
                         "run the MAX-over-ranks exchange on the CPU and rank 0 prints what it gathered")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    return ap.parse_args()


# ---------------------------------------------------------------------------------------------------------------
# clocks during the timed region (B200_PROFILING.md recipe)
# ---------------------------------------------------------------------------------------------------------------
class ClockSampler:
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.index = index
        self.rows = []
        self.proc = None
        self.thread = None

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), "--query-gpu=" + self.Q,
                                          "--format=csv,noheader,nounits", "-lms", "100"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
        except OSError:
            self.proc = None
            return
        self.thread = threading.Thread(target=self._read, daemon=True)
        self.thread.start()

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append(line.strip())

    def stop(self):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except subprocess.TimeoutExpired:
            self.proc.kill()
        sm, smax, reasons, power = [], [], set(), []
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for r in self.rows:
            p = [x.strip() for x in r.split(",")]
            if len(p) < 7:
                continue
            try:
                sm.append(float(p[0]))
                smax.append(float(p[1]))
                power.append(float(p[2]))
            except ValueError:
                continue
            for k, nm in enumerate(names):
                if p[3 + k].lower().startswith("active"):
                    reasons.add(nm)
        if not sm:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["no samples"]}
        return {"sm_mhz": float(np.median(sm)), "sm_max_mhz": float(max(smax)), "reasons": sorted(reasons),
                "power_w_max": float(max(power)), "samples": len(sm)}


# ---------------------------------------------------------------------------------------------------------------
# workload description and algorithmic work (tuples and flops per launch class)
# ---------------------------------------------------------------------------------------------------------------
def stage_tuples(Lg, n_list, lmin, real):
    """(t, m, l, n) tuples of one Wigner contraction launch: all Lg rings, l in [max(|m|,|n|,lmin), Lg),
    m >= 0 (the (-m,-n) column shares the recursion: d^l_{-m,-n} = (-1)^{m+n} d^l_{mn})."""
    m = np.arange(Lg)
    tot = 0
    for n in n_list:
        lo = np.maximum(np.maximum(m, abs(n)), lmin)
        tot += int(np.clip(Lg - lo, 0, None).sum()) * Lg
    return tot


def workload_stages(cfg, api):
    """[(Lg, n_list, lmin)] for the contraction launches of ONE direction of one transform pair: the set is the same
    for the inverse-type kernel (a7 at L_s, a5 per scale, a7 at L) and the forward-type kernel (a3, a6, a3)."""
    L, N, lam, J0, mr = cfg["L"], cfg["N"], cfg["lam"], cfg["J0"], cfg["multires"]
    psi, phi = api.s2wav_kernels(L, N, lam, J0)
    J = api.s2w_scale_count(L, lam)

    def bl(e):
        return L if not mr else int(min(int(np.ceil(lam ** e - 1e-9)), L))
    stages = [(L, [0], 0), (bl(J0), [0], 0)]
    for j in range(J0, J + 1):
        Lj = bl(j + 1)
        a = np.abs(psi[j - J0][:Lj])
        ns = [n for n in range(-(N - 1), N, 2) if abs(n) < Lj and a[:, n + N - 1].any()]
        nz = np.nonzero(a.any(axis=1))[0]
        if len(ns) and len(nz):
            stages.append((Lj, ns, int(nz[0])))
    return stages


def contraction_flops_per_step(cfg, api):
    """Algorithmic FP64 flops of the Wigner contraction kernels in one step, per kernel class:
    per tuple 5 flops for the recursion step (shared by all columns) + 4 flops per complex column
    (2 DFMA: d * (re, im)); columns = batch (real) or 2 * batch (complex: (m,n) and (-m,-n))."""
    cols = cfg["batch"] * (1 if cfg["real"] else 2)
    tup = sum(stage_tuples(Lg, ns, lmin, cfg["real"]) for (Lg, ns, lmin) in workload_stages(cfg, api))
    return tup, tup * (5.0 + 4.0 * cols)


def make_signals(cfg, api, torch, device, seed_offset=0):
    """Band-limited synthetic signals of the workload, resident on `device`: coefficients from the seeded recipe of
    paper_2402_01282_b200.inputs, synthesised to MW pixels by the library's own inverse
    harmonic transform (set-up, outside every timed region)."""
    from paper_2402_01282_b200 import inputs
    L, B, real = cfg["L"], cfg["batch"], cfg["real"]
    gen = inputs.flm_real if real else inputs.flm_complex
    flm = gen(L, cfg["seed"] + 1000 * seed_offset, B, cfg["spectrum"])
    plan = api.s2wav_plan_create(L, 1, cfg["lam"], 0, True, real, B, device.index or 0)
    f = plan.harmonic_inverse(torch.from_numpy(flm).to(device))
    torch.cuda.synchronize()
    plan.close()
    return f.reshape(B, L, 2 * L - 1)


# ---------------------------------------------------------------------------------------------------------------
# CPU baseline: the oracle as it stands (double instance, OpenMP), on a bounded sample of the workload
# ---------------------------------------------------------------------------------------------------------------
def _scale_stages(cfg):
    """[(Lg, n_list, lmin)] of the oracle's contraction stages in ONE direction (all m of both signs)."""
    from oracle import sphere as S
    L, N, lam, J0, mr = cfg["L"], cfg["N"], cfg["lam"], cfg["J0"], cfg["multires"]
    psi, phi, J = S.filters(L, N, lam, J0, "f64")
    stages = [(L, [0], 0), (S.bandlimit_of_scaling(L, lam, J0, mr), [0], 0)]
    for j in range(J0, J + 1):
        Lj = S.bandlimit_of_scale(j, L, lam, mr)
        a = np.abs(np.asarray(psi[j - J0][:Lj], dtype=np.complex128))
        ns = [n for n in range(-(N - 1), N, 2) if abs(n) < Lj and a[:, n + N - 1].any()]
        nz = np.nonzero(a.any(axis=1))[0]
        if len(ns) and len(nz):
            stages.append((Lj, ns, int(nz[0])))
    return stages


def _tuples_per_ring(Lg, ns, lmin):
    m = np.abs(np.arange(-(Lg - 1), Lg))
    return sum(int(np.clip(Lg - np.maximum(np.maximum(m, abs(n)), lmin), 0, None).sum()) for n in ns)


def cpu_baseline(cfg, budget=1.0):
    """The oracle as it stands (double instance, OpenMP, all host cores) on a bounded sample of the workload, every
    O(L^3)-class part of it timed: (1) analysis-side contraction: oracle.sphere.analysis_from_flm of one signal on a
    subset of the top scale's beta rings; (2) synthesis-side contraction: oracle.sphere.dl_forward of one row n on a
    subset of rings; (3) the MW reweighting (R3 (ii)-(vi), O(L^2) per column) on a batch of columns of the top grid.
    Each part is scaled to one full forward + inverse transform -- (1), (2) by (t, m, l, n) tuple count, (3) by column
    count x (L_j / L_top)^2 -- and the three are added.  `budget` scales the sample sizes (1.0: about 10-30 s)."""
    from oracle import sphere as S
    from paper_2402_01282_b200 import inputs
    L, N, lam, J0, mr, real = cfg["L"], cfg["N"], cfg["lam"], cfg["J0"], cfg["multires"], cfg["real"]
    gen = inputs.flm_real if real else inputs.flm_complex
    flm = gen(L, cfg["seed"], 1, cfg["spectrum"])[0]
    filt = S.filters(L, N, lam, J0, "f64")
    psi, phi, J = filt
    stages = _scale_stages(cfg)
    Lj, ns, lmin = stages[-1]
    S.wigner_d(8, 1, 0, 0.3, "f64")  # loads / builds the library outside the timed region
    dir_tuples = sum(_tuples_per_ring(Lg, n_, lm_) * Lg for (Lg, n_, lm_) in stages)
    # (1) analysis-side contraction
    nr1 = max(1, min(Lj, int(round(budget * 6.0e9 / (N * float(Lj) ** 2 * 4.0)))))
    rings = np.unique(np.linspace(0, Lj - 1, nr1).astype(int))
    t0 = time.perf_counter()
    S.analysis_from_flm(flm, L, N, lam, J0, mr, "f64", filt, scales=[J], rings={J: rings})
    dt1 = time.perf_counter() - t0
    tup1 = _tuples_per_ring(Lj, ns, lmin) * len(rings)
    # (2) synthesis-side contraction: one row n, a subset of rings, all (l, m)
    rng = np.random.default_rng(0)
    nr2 = max(1, min(Lj, int(round(budget * 2.0e9 / (float(Lj) ** 2 * 2.0)))))
    betas = S.mw_thetas(Lj, "f64")[np.unique(np.linspace(0, Lj - 1, nr2).astype(int))]
    H = rng.standard_normal((2 * Lj - 1, betas.size)) + 1j * rng.standard_normal((2 * Lj - 1, betas.size))
    t0 = time.perf_counter()
    S.dl_forward(H, Lj, ns[-1], betas, "f64")
    dt2 = time.perf_counter() - t0
    tup2 = _tuples_per_ring(Lj, [ns[-1]], 0) * betas.size
    # (3) reweighting columns of the top grid
    nc = max(1, min(2 * Lj - 1, int(round(budget * 1.6e8 / float(Lj) ** 2))))
    Fc = rng.standard_normal((nc, Lj)) + 1j * rng.standard_normal((nc, Lj))
    t0 = time.perf_counter()
    S.mw_reweight(Fc, Lj, np.ones(nc, dtype=np.int32), "f64")
    dt3 = time.perf_counter() - t0
    # forward transforms with reweighting: SHT of f at L (analysis), SHT of W^Phi at L_s and every scale (synthesis)
    col_equiv = sum((2 * Lg - 1) * len(n_) * (Lg / float(Lj)) ** 2 for (Lg, n_, lm_) in stages)
    est = dt1 * dir_tuples / max(tup1, 1) + dt2 * dir_tuples / max(tup2, 1) + dt3 * col_equiv / nc
    return {"value": 1.0 / est, "unit": UNIT, "cores": S.num_threads("f64"), "kind": "oracle",
            "sample": "contraction + reweighting, extrapolated: (1) oracle analysis of 1 signal, top scale j=%d (L_j=%d), "
                      "%d of %d beta rings, %.1f s; (2) synthesis-side contraction dl_forward, row n=%d, %d rings, %.1f s; "
                      "(3) MW reweighting of %d of the top grid's columns, %.1f s; scaled to one fwd+inv transform by "
                      "tuple count (%.3g per direction) and column count -> %.0f s (contraction %.0f + %.0f, "
                      "reweighting %.0f)"
                      % (J, Lj, len(rings), Lj, dt1, ns[-1], betas.size, dt2, nc, dt3, dir_tuples, est,
                         dt1 * dir_tuples / max(tup1, 1), dt2 * dir_tuples / max(tup2, 1), dt3 * col_equiv / nc)}


def oracle_measured_small():
    """One un-extrapolated oracle forward + inverse transform (double instance, all cores) of BASELINE config 2
    (L = 256, N = 3, complex): the measured companion of the extrapolated C3 figure."""
    from oracle import sphere as S
    from paper_2402_01282_b200 import inputs
    c = inputs.CONFIGS["C2"]
    L, N, lam, J0 = c["L"], c["N"], c["lam"], c["J0"]
    flm = inputs.config_coefficients("C2")[0]
    filt = S.filters(L, N, lam, J0, "f64")
    f = S.sht_inverse(flm, L, "f64")
    t0 = time.perf_counter()
    phi, psi = S.analysis(f, L, N, lam, J0, True, "f64", filt)
    back = S.synthesis(phi, psi, L, N, lam, J0, True, "f64", filt)
    dt = time.perf_counter() - t0
    return {"workload": "C2: sphere L=256 N=3 lambda=2 J0=2 multires complex, forward+inverse, whole transform timed",
            "value": 1.0 / dt, "unit": UNIT, "seconds": dt, "cores": S.num_threads("f64"),
            "roundtrip_rel_err": float(np.abs(back - f).max() / np.abs(f).max())}


def run_reference(args, cfg):
    """--impl reference: the oracle as it stands on the host cores; each step is one bounded sample."""
    from paper_2402_01282_b200 import api
    world = int(os.environ.get("WORLD_SIZE", "1"))
    args.gpus = world
    cfg["coeff_gb"] = (api._coeff_elems_sphere(cfg["L"], cfg["N"], cfg["lam"], cfg["J0"], cfg["multires"])
                       * cfg["batch"] * (8 if cfg["real"] else 16) / 1e9)
    vals, base = [], None
    for i in range(args.warmup + args.steps):
        base = cpu_baseline(cfg, budget=0.25)
        if i >= args.warmup:
            vals.append(base["value"])
    v = float(np.mean(vals))
    base["value"] = v
    base["measured_small"] = oracle_measured_small()
    line = {"impl": "reference", "metric": METRIC, "value": v, "unit": UNIT, "n_gpus": world,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * cfg["batch"] / v,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": workload_config(cfg, args), "cpu_baseline": base,
            "e2e": {"value": v, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}}
    print(json.dumps(line))


def workload_config(cfg, args):
    return {"workload": "%s: sphere L=%d N=%d lambda=%g J0=%d multires=%s %s fp64 batch=%d, %s"
                        % (cfg["name"], cfg["L"], cfg["N"], cfg["lam"], cfg["J0"], cfg["multires"],
                           "real" if cfg["real"] else "complex", cfg["batch"],
                           "adjoint pair S^H + A^H" if getattr(args, "adjoint", False) else "forward+inverse"),
            "L": cfg["L"], "N": cfg["N"], "lambda": cfg["lam"], "J0": cfg["J0"], "multiresolution": cfg["multires"],
            "batch_per_gpu": cfg["batch"],
            "mode": "precomputed Wigner-d table (DMMA)" if getattr(args, "precompute", False) else "on-the-fly Wigner recursion",
            "parallelism": "replicas x%d (no data-path collective)" % args.gpus,
            "l2": "coefficient block per step (%.2f GB) exceeds the 126 MB L2; no explicit flush" % cfg.get("coeff_gb", 0.0)}


# ---------------------------------------------------------------------------------------------------------------
# multi-GPU bookkeeping: replicas only -- every rank transforms its own batch of signals, there is
# no data-path collective; the only exchange is this MAX over the ranks' device times.
# ---------------------------------------------------------------------------------------------------------------
def replica_seed_offset(rank):
    """Seed offset of rank r (make_signals draws its signals from seed + 1000 r): independent signals per replica."""
    return int(rank)


def max_over_ranks(values, world, device):
    """Element-wise MAX of a list of floats over all ranks (identity for world == 1)."""
    import torch
    t = torch.tensor([float(v) for v in values], dtype=torch.float64, device=device)
    if world > 1:
        import torch.distributed as dist
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return [float(v) for v in t]


def whole_job_value(world, batch_per_rank, steps, ms_max):
    """transforms/s of the whole job: the units ALL ranks processed over the slowest rank's device time."""
    return world * batch_per_rank * steps / (ms_max * 1e-3)


# ---------------------------------------------------------------------------------------------------------------
# our arm
# ---------------------------------------------------------------------------------------------------------------
def run_ours(args, cfg):
    import torch
    import torch.distributed as dist
    from paper_2402_01282_b200 import api

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise RuntimeError("bench.py needs a CUDA device (there is no CPU fallback); use --impl reference for the oracle")
    torch.cuda.set_device(local)
    device = torch.device("cuda", local)
    if world > 1:
        dist.init_process_group("nccl", device_id=device)

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    adj = bool(getattr(args, "adjoint", False))
    if adj:  # no host-buffer entry point and no timed oracle for the adjoints
        args.no_e2e = args.no_cpu_baseline = True
    L, N, lam, J0, mr, real, B = cfg["L"], cfg["N"], cfg["lam"], cfg["J0"], cfg["multires"], cfg["real"], cfg["batch"]
    f = make_signals(cfg, api, torch, device, seed_offset=replica_seed_offset(rank))     # independent signals per replica
    plan = api.s2wav_plan_create(L, N, lam, J0, mr, real, B, local,
                                 flags=api.S2W_PRECOMPUTE if args.precompute else 0)
    cfg["coeff_gb"] = plan.coeff_elems * B * (8 if real else 16) / 1e9
    w = torch.empty((B, plan.coeff_elems), dtype=plan.dtype, device=device)
    back = torch.empty((B, plan.signal_elems), dtype=plan.dtype, device=device)

    def step():
        if adj:
            plan.inverse_adjoint(f, out=w)
            plan.forward_adjoint(w, out=back)
        else:
            plan.forward(f, out=w)
            plan.inverse(w, out=back)

    for _ in range(max(args.warmup, 3)):
        step()
    barrier()
    if adj:  # A^H S^H is not the identity; the check is the defining identity <A f, y> = <f, A^H y> with y = S^H f
        Af = plan.forward(f)
        rt_err = float((torch.vdot(Af.flatten(), w.flatten()) - torch.vdot(f.flatten(), back.flatten())).abs()
                       / (Af.norm() * w.norm()))
        del Af
    else:
        rt_err = float((back.view_as(f) - f).abs().max() / f.abs().max())

    # ---- device-resident timing: exactly K steps, CUDA events on the launching (current) stream ----
    sampler = ClockSampler(local)
    if rank == 0:
        sampler.start()
    l0 = api.launch_count()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    e0.record()
    for _ in range(args.steps):
        step()
    e1.record()
    barrier()
    ms = e0.elapsed_time(e1)
    launches = api.launch_count() - l0
    clocks = sampler.stop() if rank == 0 else None

    # ---- per-class kernel times (same steps, event pairs around every launch; a separate pass so that the
    #      event records do not sit inside the headline number) ----
    api.timing_enable(True)
    api.timing_read()
    ksteps = max(2, min(args.steps, 5))
    for _ in range(ksteps):
        step()
    torch.cuda.synchronize()
    classes = api.timing_read()
    api.timing_enable(False)

    # ---- end to end through the host-buffer C ABI calls (pinned memory; H2D + D2H inside) ----
    e2e = None
    if not args.no_e2e and not args.precompute:
        # pinned host buffers for the signals, the coefficients and the reconstruction
        fh = torch.empty(f.shape, dtype=f.dtype, pin_memory=True)
        fh.copy_(f)
        fh_np = fh.numpy()
        wh_np = torch.empty((B, plan.coeff_elems), dtype=f.dtype, pin_memory=True).numpy()
        fb_np = torch.empty(f.shape, dtype=f.dtype, pin_memory=True).numpy()
        api.s2wav_inverse_host(api.s2wav_forward_host(fh_np, L, N, lam, J0, mr, out=wh_np), L, N, lam, J0, mr,
                               out=fb_np)  # warm-up (builds the cached plan and its staging buffers)
        barrier()
        nrep = max(1, min(args.steps, 3))
        t0 = time.perf_counter()
        for _ in range(nrep):
            wh = api.s2wav_forward_host(fh_np, L, N, lam, J0, mr, out=wh_np)
            fb = api.s2wav_inverse_host(wh, L, N, lam, J0, mr, out=fb_np)
        torch.cuda.synchronize()
        dt = time.perf_counter() - t0
        esz = 8 if real else 16
        sig_b, cof_b = plan.signal_elems * B * esz, plan.coeff_elems * B * esz
        e2e = {"dt": dt / nrep, "h2d": sig_b + cof_b, "d2h": sig_b + cof_b,
               "rt_err": float(np.abs(fb - fh_np).max() / np.abs(fh_np).max())}

    # ---- max over ranks ----
    ms, e2e_dt = max_over_ranks([ms, e2e["dt"] if e2e else 0.0], world, device)
    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return

    value = whole_job_value(world, B, args.steps, ms)
    tup, flops = contraction_flops_per_step(cfg, api)   # per class per step
    dom = max(("wigner_inverse", "wigner_forward"), key=lambda k: classes[k][0])
    dom_ms, dom_n = classes[dom]
    sm_max = (clocks or {}).get("sm_max_mhz") or 1965.0
    peak = 148 * 64 * 2 * sm_max * 1e6 / 1e12          # nominal DFMA peak, TFLOP/s
    achieved = flops * ksteps / (dom_ms * 1e-3) / 1e12 if dom_ms > 0 else 0.0
    try:
        probe = {"dfma_tflops": api.probe_fp64(0, local), "dmma_tflops": api.probe_fp64(1, local)}
    except Exception as e:  # noqa: BLE001
        probe = {"error": str(e)}
    total_kms = sum(v[0] for v in classes.values())
    roofline = {"bound": "alu", "kernel": dom, "achieved": achieved, "peak": peak, "unit": "TFLOP/s",
                "frac": achieved / peak if peak else None,
                "traffic": NCU_TRAFFIC.get((cfg["name"], dom)) if not (args.precompute or adj) else None,
                "traffic_unit": "bytes per step (all launches of the class), ncu --set full, "
                                + NCU_TRAFFIC_SOURCE.get(cfg["name"], "no capture for this workload"),
                "peak_source": "derived: 148 SMs x 64 FP64 lanes x 2 flop x sm_max_mhz (DESIGN.md); "
                               "measured DFMA-chain probe beside it",
                "probe": probe, "tuples_per_step": tup, "flops_per_step": flops,
                "launches_per_step": dom_n / ksteps, "ms_per_step": dom_ms / ksteps}
    if args.precompute:
        # the precomputed-kernel variant streams 8 B of Wigner-d table per (ring, m, l, n) tuple
        hbm = None
        try:
            hbm = json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))["hbm_gbs"]
            src = "measured copy bandwidth of MEASURED_PEAKS.json"
        except Exception:  # noqa: BLE001
            hbm, src = 6650.0, "fallback of B200_PROFILING.md (MEASURED_PEAKS.json absent)"
        gbs = 8.0 * tup * ksteps / (dom_ms * 1e-3) / 1e9 if dom_ms > 0 else 0.0
        roofline = {"bound": "hbm", "kernel": dom, "achieved": gbs, "peak": hbm, "unit": "GB/s",
                    "frac": gbs / hbm, "traffic": None, "peak_source": src, "tuples_per_step": tup,
                    "bytes_per_step": 8.0 * tup, "launches_per_step": dom_n / ksteps, "ms_per_step": dom_ms / ksteps}
    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
        "warmup": max(args.warmup, 3), "ms_per_step": ms / args.steps, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f64", "data": "synthetic", "config": workload_config(cfg, args),
        "clocks": clocks, "gpu_launches": int(launches),
        ("adjoint_identity_rel_err" if adj else "roundtrip_rel_err"): rt_err,
        "roofline": roofline,
        "kernel_ms_per_step": {k: round(v[0] / ksteps, 4) for k, v in classes.items()},
        "kernel_share": {k: round(v[0] / total_kms, 4) for k, v in classes.items()} if total_kms else None,
    }
    if e2e:
        line["e2e"] = {"value": world * B / e2e_dt, "unit": UNIT, "h2d_bytes_per_step": e2e["h2d"],
                       "d2h_bytes_per_step": e2e["d2h"], "roundtrip_rel_err": e2e["rt_err"]}
    if not args.no_cpu_baseline and world == 1:
        line["cpu_baseline"] = cpu_baseline(cfg, budget=3.0)   # about 10-30 s of host work
        line["cpu_baseline"]["measured_small"] = oracle_measured_small()
    print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()


# ---------------------------------------------------------------------------------------------------------------
# ball workload (C5): one step = forward + inverse Fourier-Laguerre wavelet transform of one [P][L][2L-1] field
# ---------------------------------------------------------------------------------------------------------------
def ball_stages(cfg, api):
    """[(Lg, n_list, lmin, shells)] of the contraction launches of one direction (Alg. 2): Z at (L, P), the scaling
    part at (L, P), then every (j', j) with P_j' shells."""
    L, P, N, lam, nu, J0 = cfg["L"], cfg["P"], cfg["N"], cfg["lam"], cfg["nu"], cfg["J0"]
    kl = api.s2ball_kernels(L, P, N, lam, nu, J0)["kappa_l"]
    J, Jp = api.s2w_scale_count(L, lam), api.s2w_scale_count(P, nu)

    def bl(base, e, cap):
        return int(min(int(np.ceil(base ** e - 1e-9)), cap))
    stages = [(L, [0], 0, P), (L, [0], 0, P)]
    for jp in range(J0, Jp + 1):
        Pj = bl(nu, jp + 1, P)
        for j in range(J0, J + 1):
            Lj = bl(lam, j + 1, L)
            k = np.abs(kl[j - J0][:Lj])
            nz = np.nonzero(k)[0]
            ns = [n for n in range(-(N - 1), N, 2) if abs(n) < Lj]
            if len(nz) and len(ns):
                stages.append((Lj, ns, int(nz[0]), Pj))
    return stages


def run_ball(args, cfg):
    import torch
    from paper_2402_01282_b200 import api, inputs
    if not torch.cuda.is_available():
        raise RuntimeError("bench.py needs a CUDA device (there is no CPU fallback)")
    if int(os.environ.get("WORLD_SIZE", "1")) > 1:
        raise RuntimeError("the ball workload is single-GPU (replicas only); run it with --gpus 1")
    torch.cuda.set_device(0)
    device = torch.device("cuda", 0)
    L, P, N, lam, nu, J0, tau = cfg["L"], cfg["P"], cfg["N"], cfg["lam"], cfg["nu"], cfg["J0"], cfg["tau"]
    flags = api.S2W_PRECOMPUTE if getattr(args, "precompute", False) else (api.S2W_RECURSION if getattr(args, "recursion", False) else 0)
    plan = api.s2ball_plan_create(L, P, N, lam, nu, J0, tau, flags=flags)
    pre = bool(flags & api.S2W_PRECOMPUTE) or (not (flags & api.S2W_RECURSION) and L <= 256)
    if flags:
        args.no_e2e = True                          # the host-buffer entry points build their plan with flags = 0
    flmp = inputs.config_coefficients(cfg["name"])
    f = plan.harmonic_inverse(torch.from_numpy(flmp).to(device).reshape(1, -1))
    w = torch.empty((1, plan.coeff_elems), dtype=plan.dtype, device=device)
    back = torch.empty((1, plan.signal_elems), dtype=plan.dtype, device=device)

    adj = bool(getattr(args, "adjoint", False))
    if adj:
        args.no_e2e = args.no_cpu_baseline = True

    def step():
        if adj:
            plan.inverse_adjoint(f, out=w)
            plan.forward_adjoint(w, out=back)
        else:
            plan.forward(f, out=w)
            plan.inverse(w, out=back)
    for _ in range(max(args.warmup, 3)):
        step()
    torch.cuda.synchronize()
    if adj:  # the defining identity <A f, y> = <f, A^H y> with y = S^H f
        Af = plan.forward(f)
        rt_err = float((torch.vdot(Af.flatten(), w.flatten()) - torch.vdot(f.flatten(), back.flatten())).abs()
                       / (Af.norm() * w.norm()))
        del Af
    else:
        rt_err = float((back - f).abs().max() / f.abs().max())
    sampler = ClockSampler(0)
    sampler.start()
    l0 = api.launch_count()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    torch.cuda.synchronize()
    e0.record()
    for _ in range(args.steps):
        step()
    e1.record()
    torch.cuda.synchronize()
    ms = e0.elapsed_time(e1)
    launches = api.launch_count() - l0
    clocks = sampler.stop()
    api.timing_enable(True)
    api.timing_read()
    ksteps = max(2, min(args.steps, 5))
    for _ in range(ksteps):
        step()
    torch.cuda.synchronize()
    classes = api.timing_read()
    api.timing_enable(False)
    # algorithmic flops of one contraction class: 5 per tuple (recursion) + 4 per tuple and complex column; a complex
    # shell is 2 columns ((m,n) and (-m,-n))
    flops = 0.0
    for (Lg, ns, lmin, shells) in ball_stages(cfg, api):
        flops += stage_tuples(Lg, ns, lmin, False) * (5.0 + 4.0 * 2 * shells)
    dom = max(("wigner_inverse", "wigner_forward"), key=lambda k: classes[k][0])
    dom_ms = classes[dom][0]
    sm_max = (clocks or {}).get("sm_max_mhz") or 1965.0
    peak = 148 * 64 * 2 * sm_max * 1e6 / 1e12
    achieved = flops * ksteps / (dom_ms * 1e-3) / 1e12 if dom_ms > 0 else 0.0
    e2e = None
    if not args.no_e2e:
        fh = torch.empty((P, L, 2 * L - 1), dtype=f.dtype, pin_memory=True)
        fh.copy_(f.reshape(P, L, 2 * L - 1))
        fh_np = fh.numpy()
        wh_np = torch.empty(plan.coeff_elems, dtype=f.dtype, pin_memory=True).numpy()
        fb_np = torch.empty((P, L, 2 * L - 1), dtype=f.dtype, pin_memory=True).numpy()
        api.s2ball_inverse_host(api.s2ball_forward_host(fh_np, L, P, N, lam, nu, J0, tau, out=wh_np), L, P, N, lam, nu,
                                J0, tau, out=fb_np)
        t0 = time.perf_counter()
        wh = api.s2ball_forward_host(fh_np, L, P, N, lam, nu, J0, tau, out=wh_np)
        fb = api.s2ball_inverse_host(wh, L, P, N, lam, nu, J0, tau, out=fb_np)
        dt = time.perf_counter() - t0
        nbytes = (plan.signal_elems + plan.coeff_elems) * 16
        e2e = {"value": 1.0 / dt, "unit": UNIT, "h2d_bytes_per_step": nbytes, "d2h_bytes_per_step": nbytes,
               "roundtrip_rel_err": float(np.abs(fb - fh_np).max() / np.abs(fh_np).max())}
    total_kms = sum(v[0] for v in classes.values())
    line = {
        "metric": METRIC, "value": args.steps / (ms * 1e-3), "unit": UNIT, "n_gpus": 1, "steps": args.steps,
        "warmup": max(args.warmup, 3), "ms_per_step": ms / args.steps, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": "%s: ball L=%d P=%d N=%d lambda_l=%g lambda_p=%g J0=%d tau=%g complex fp64, "
                               "%s" % (cfg["name"], L, P, N, lam, nu, J0, tau, "adjoint pair S^H + A^H" if adj else "forward+inverse"),
                   "L": L, "P": P, "N": N, "parallelism": "replicas x1 (no data-path collective)",
                   "mode": ("precomputed Wigner-d tables, theta quadrature folded into the table on grids with L_j <= 256 "
                            "(the default of ball plans with L <= 256)" if pre else "on-the-fly Wigner recursion"),
                   "l2": "coefficient block per step (%.2f GB) exceeds the 126 MB L2; no explicit flush"
                         % (plan.coeff_elems * 16 / 1e9)},
        "clocks": clocks, "gpu_launches": int(launches),
        ("adjoint_identity_rel_err" if adj else "roundtrip_rel_err"): rt_err,
        "roofline": {"bound": "alu", "kernel": dom, "achieved": achieved, "peak": peak, "unit": "TFLOP/s",
                     "frac": achieved / peak if peak else None, "traffic": None,
                     "peak_source": "derived: 148 SMs x 64 FP64 lanes x 2 flop x sm_max_mhz (DESIGN.md)",
                     "flops_per_step": flops, "ms_per_step": dom_ms / ksteps},
        "kernel_ms_per_step": {k: round(v[0] / ksteps, 4) for k, v in classes.items()},
        "kernel_share": {k: round(v[0] / total_kms, 4) for k, v in classes.items()} if total_kms else None,
    }
    if e2e:
        line["e2e"] = e2e
    print(json.dumps(line))



def free_port():
    import socket
    with socket.socket(socket.AF_INET, socket.SOCK_STREAM) as sk:
        sk.bind(("127.0.0.1", 0))
        return sk.getsockname()[1]


def spawn_ranks(args):
    """`python bench.py --gpus N` outside a launcher: start N ranks of this same command, one per GPU, under
    torch.distributed.run (what the driver does itself for N > 1) and return its exit code."""
    env = dict(os.environ)
    env.setdefault("NCCL_DEBUG", "INFO")            # the communicator log shows the N ranks (stderr)
    env.setdefault("NCCL_DEBUG_SUBSYS", "INIT")
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", str(args.gpus),
           "--master-addr", "127.0.0.1", "--master-port", str(free_port()), os.path.abspath(__file__)] + sys.argv[1:]
    return subprocess.call(cmd, env=env)


def run_dry(args):
    """--dry-run-cpu: every rank joins a gloo group and reports itself; no transform runs."""
    import torch
    import torch.distributed as dist
    rank, world = int(os.environ.get("RANK", "0")), int(os.environ.get("WORLD_SIZE", "1"))
    if world > 1:
        dist.init_process_group("gloo")
    me = {"rank": rank, "local_rank": int(os.environ.get("LOCAL_RANK", "0")), "pid": os.getpid(),
          "seed_offset": replica_seed_offset(rank)}
    everyone = [me]
    if world > 1:
        everyone = [None] * world
        dist.all_gather_object(everyone, me)
    ms, = max_over_ranks([10.0 + rank], world, torch.device("cpu"))
    if rank == 0:
        print(json.dumps({"dry_run": True, "n_gpus": world, "ranks": everyone, "ms_max": ms,
                          "value": whole_job_value(world, 4, args.steps, ms), "unit": UNIT}))
    if world > 1:
        dist.destroy_process_group()


def main():
    args = parse_args()
    world_env = os.environ.get("WORLD_SIZE")
    if world_env is None and args.gpus > 1:
        raise SystemExit(spawn_ranks(args))
    if world_env is not None and int(world_env) != args.gpus:
        raise SystemExit("bench.py: --gpus %d but the launcher started WORLD_SIZE=%s ranks" % (args.gpus, world_env))
    if args.dry_run_cpu:
        run_dry(args)
        return
    from paper_2402_01282_b200 import inputs
    cfg = dict(inputs.CONFIGS[args.workload])
    cfg["name"] = args.workload
    if cfg.get("kind") == "ball":
        if args.impl == "reference":
            raise SystemExit("--impl reference times the sphere workloads (the metric configuration is C3)")
        run_ball(args, cfg)
        return
    if args.impl == "reference":
        if int(os.environ.get("RANK", "0")) == 0:
            run_reference(args, cfg)
        return
    run_ours(args, cfg)


if __name__ == "__main__":
    main()
