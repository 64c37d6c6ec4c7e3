#!/usr/bin/env python
"""bench.py -- the nuSHT hot path on synthetic BASELINE.json workloads.

A step = one synthesis (Eq. 3) + one adjoint (Eq. 2) of arXiv 2406.14542 on the same plan, back
to back, inputs resident in HBM.  Default workload: BASELINE.json configs[2] (the configuration
the metric "nuSHT synth+adjoint ms at lmax=4095" is quoted on): lmax = mmax = 4095, FP64,
eps = 1e-10, 67,108,864 uniform random points, white a_lm.  Planning (point sort, tables, cuFFT
plans) is excluded from the timed region, as in the paper.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config 1|2|3|4|6] [--impl reference]

Prints ONE JSON line (rank 0).  Multi-GPU: the method is single-GPU: N ranks run N
independent replicas ("replicas only"), no collective on the data path.
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

from paper_2406_14542_b200 import inputs  # noqa: E402

METRIC = "nusht_synth_plus_adjoint_ms"
FP64_FMA_PER_CLK_PER_SM = 64          # B200: 148 SMs x 64 FP64 FMA/clk
N_SM = 148


def parse():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", type=int, default=3)
    ap.add_argument("--npts", type=int, default=None, help="override the point count (debugging)")
    ap.add_argument("--impl", default="b200", choices=["b200", "reference"])
    ap.add_argument("--cpu-seconds", type=float, default=20.0, help="target CPU time of the oracle sample")
    ap.add_argument("--sigma", type=float, default=None,
                    help="up-sampling factor of the nuFFT grid: 2 (default) or 1.25, the paper's own (PAPER.md:152)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--eps-sweep", action="store_true",
                    help="BASELINE.json configs[4]: lmax=4095 on 67M points, eps in {1e-4, 1e-6} FP32 and "
                         "{1e-8, 1e-10, 1e-12} FP64; one JSON line per eps (accuracy on an oracle subset + timing)")
    ap.add_argument("--sweep-subset", type=int, default=1500, help="points of the oracle subset of the sweep")
    ap.add_argument("--ring", default=None, choices=["gl", "equi", "healpix", "healpix-lens"],
                    help="ring-grid transforms (SURVEY 8(f) rank 3/4) instead of the nuSHT step: 'gl' = Gauss-Legendre grid "
                         "(lmax+1 rings x 2 lmax+2 pixels, the paper's output grid, PAPER.md:154): step = synthesis + "
                         "analysis; 'healpix' = the same on a HEALPix-style ring layout (PAPER.md:218), nside = (lmax+1)/2; "
                         "'equi' = the 2(lmax+1)^2 equi-angular grid of config 2: step = gradient (Eq. C2) + pointing; "
                         "'healpix-lens' = the paper's use case (Eq. 8, Appendix C) on the HEALPix-style layout: step = "
                         "deflection field of a lensing potential (Eq. C2) + pointing (Eq. C1) + nusht_set_points + "
                         "synthesis of the unlensed field at the deflected pixel centres")
    ap.add_argument("--lmax", type=int, default=4095, help="band limit of the --ring modes")
    return ap.parse_args()


class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled during the timed region (B200_PROFILING.md)."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.rows, self.proc, self.index = [], None, index

    def start(self):
        try:
            self.proc = subprocess.Popen(
                ["nvidia-smi", "-i", str(self.index), "--query-gpu=" + self.Q, "--format=csv,noheader,nounits",
                 "-lms", "100"], stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.th = threading.Thread(target=self._read, daemon=True)
            self.th.start()
        except OSError:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append([c.strip() for c in line.split(",")])

    def stop(self):
        if not self.proc:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        self.th.join(timeout=2)
        sm, mx, reasons = [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for r in self.rows:
            try:
                sm.append(float(r[0])); mx.append(float(r[1]))
            except (ValueError, IndexError):
                continue
            for n, v in zip(names, r[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(n)
        busy = sorted(sm)[len(sm) // 2:] if sm else []      # upper half = samples under load
        return {"sm_mhz": float(np.median(busy)) if busy else None, "sm_max_mhz": max(mx) if mx else None,
                "samples": len(sm), "reasons": sorted(reasons)}


def oracle_sample(cfg, theta, phi, alm, x, seconds):
    """Time the oracle as it stands on a bounded sample of the same workload; extrapolate to the
    full point count.  Returns (ms per full step extrapolated, description dict)."""
    from oracle import oracle as o
    L, M = cfg["lmax"], cfg["mmax"]
    nlm = inputs.nlm(L, M)
    # One sampling rule for both legs (cpu_baseline and --impl reference): at least 64 points per OpenMP thread (the
    # oracle's synthesis loop hands out chunks of 64 points: fewer leaves threads idle and under-reports it), then
    # grown until synthesis + adjoint take about `seconds` of wall time (bounded by the sample given).
    n = max(64 * max(1, o.num_threads()), int(2.0e8 * max(1, o.num_threads()) * 0.25 / nlm))
    n = min(len(theta), n)
    while True:
        t0 = time.perf_counter()
        o.synthesis(L, M, theta[:n], phi[:n], alm)
        t_syn = time.perf_counter() - t0
        t0 = time.perf_counter()
        o.adjoint(L, M, theta[:n], phi[:n], x[:n])
        t_adj = time.perf_counter() - t0
        tot = t_syn + t_adj
        if tot >= 0.5 * seconds or n >= len(theta):
            break
        n = int(min(len(theta), max(2 * n, n * 0.9 * seconds / max(tot, 1e-3))))
    scale = len(theta) / n
    ms_full = (t_syn + t_adj) * scale * 1e3
    return ms_full, {"value": ms_full, "unit": "ms", "cores": o.num_threads(), "kind": "oracle",
                     "sample": "direct sums (oracle/nusht_oracle.c, binary64, OpenMP) on the first %d of %d points "
                               "at lmax=%d: synthesis %.2f s + adjoint %.2f s, extrapolated x%.0f to the full point count"
                               % (n, len(theta), L, t_syn, t_adj, scale),
                     "steps_per_s": 2 * nlm * n / (t_syn + t_adj)}


def oracle_points(cfg, theta, phi, sl=slice(None)):
    """The checker's point set: Eq. C1 by oracle.pointing for the lensing-like config, the points themselves else."""
    if cfg.get("deflection") is None:
        return theta[sl], phi[sl]
    from oracle import oracle as o
    a_t, a_p = cfg["deflection"]
    t2, p2 = o.pointing(theta[sl], phi[sl], a_t[sl], a_p[sl])
    return np.asarray(t2, dtype=np.float64), np.asarray(p2, dtype=np.float64)


def run_reference(args, rank):
    if rank != 0:
        return
    cfg = dict(inputs.CONFIGS[args.config])
    npts_full = args.npts or cfg["npts"]
    # the oracle only ever sees a sample: generate just a prefix-sized workload with the config's recipe
    nsample = min(npts_full, 1 << 16)
    cfg2, theta, phi, alm, x = inputs.make_config(args.config, npts=nsample)
    theta, phi = oracle_points(cfg2, theta, phi)
    vals, last = [], None
    per_step = max(2.0, min(args.cpu_seconds, 120.0 / max(1, args.steps + args.warmup)))
    for i in range(args.warmup + args.steps):
        ms, desc = oracle_sample(cfg2, theta, phi, alm, x, per_step)
        ms *= npts_full / len(theta)
        desc["value"] = ms
        desc["sample"] += "; then x%.0f from the %d-point generated prefix to %d points" % (
            npts_full / len(theta), len(theta), npts_full)
        if i >= args.warmup:
            vals.append(ms)
            last = desc
    v = float(np.mean(vals))
    last["value"] = v
    out = {"impl": "reference", "metric": METRIC, "value": v, "unit": "ms", "n_gpus": args.gpus, "steps": args.steps,
           "warmup": args.warmup, "ms_per_step": v, "higher_is_better": False, "scaling": "weak",
           "vs_baseline": None, "dtype": "f64", "data": "synthetic",
           "config": workload_config(cfg, npts_full), "cpu_baseline": last,
           "e2e": {"value": v, "unit": "ms", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
           "gpu_launches": 0}
    print(json.dumps(out))


def workload_config(cfg, npts):
    origin = "BASELINE.json config" if cfg["lmax"] <= 8191 else "beyond BASELINE.json (inputs.CONFIGS[6]):"
    return {"workload": "%s lmax=%d eps=%g: %d %s points, %s a_lm; step = synthesis + adjoint"
                        % (origin, cfg["lmax"], cfg["eps"], npts, cfg["points"], cfg["spectrum"]),
            "lmax": cfg["lmax"], "mmax": cfg["mmax"], "npts": int(npts), "eps": cfg["eps"],
            "l2": "inputs larger than L2 (alm %.0f MB, map %.0f MB, fine grid > 126 MB at lmax >= 1023)"
                  % (inputs.nlm(cfg["lmax"], cfg["mmax"]) * 16 / 1e6, npts * 8 / 1e6),
            "parallelism": "replicas"}


def measured_peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        d = json.load(open(path))
        return float(d["hbm_gbs"]), "measured (MEASURED_PEAKS.json)", float(d.get("sm_max_mhz", 1965.0))
    return 6650.0, "fallback (B200_PROFILING.md)", 1965.0


def ncu_traffic(cfg, npts):
    """DRAM bytes per launch (dram__bytes_read.sum + dram__bytes_write.sum) of our kernels from the committed
    `ncu --set full` capture (profiles/ncu_traffic.json); only valid for the workload it was captured on."""
    path = os.path.join(ROOT, "profiles", "ncu_traffic.json")
    if not os.path.exists(path):
        return {}
    d = json.load(open(path))
    if d.get("lmax") != cfg["lmax"] or d.get("npts") != npts or d.get("eps") != cfg["eps"]:
        return {}
    return d.get("bytes_per_launch", {})


def stage_rooflines(cfg, info, npts, syn_ms, adj_ms, sm_mhz, probe):
    """Algorithmic work per stage over its CUDA-event time."""
    hbm, hbm_src, sm_max = measured_peaks()
    L, M = cfg["lmax"], cfg["mmax"]
    nlm = inputs.nlm(L, M)
    npairs = (info.n_rings + 1) // 2
    fp64_peak = N_SM * FP64_FMA_PER_CLK_PER_SM * 2 * sm_max * 1e6 / 1e12        # TFLOP/s at max clock
    leg_flop = 2.0 * 3.0 * nlm * npairs                                           # 3 FMA per (l, m, ring pair)
    nth2, nth, nph = info.n_theta, info.n_theta_fine, info.n_phi_fine
    grid_bytes = (nth // 2 + 1) * nph * 8
    nu_bytes = npts * (16 + 8) + grid_bytes
    out = {}

    def alu(name, ms, fma_executed):
        # `achieved` / `frac`: the FP64 FMAs the launch EXECUTES (nusht_plan_info: the (l, m, ring pair) steps left
        # after the plan-time fast-forward x 3) over its CUDA-event time: at most 1 by construction.  `nominal`: the
        # SURVEY.md 8(d) count nlm x ceil(N_r/2) x 3 FMA, which includes the below-range steps the kernel skips, so
        # its ratio to the peak is a speed-up over the plain loop, not a pipe fraction (it exceeds 1 at lmax = 8191).
        a = 2.0 * fma_executed / (ms * 1e-3) / 1e12
        an = leg_flop / (ms * 1e-3) / 1e12
        out[name] = {"bound": "alu", "achieved": a, "peak": fp64_peak, "unit": "TFLOP/s", "frac": a / fp64_peak,
                     "traffic": None, "ms": ms,
                     "peak_source": "derived: 148 SM x 64 FP64 FMA/clk x 2 x %.0f MHz (max SM clock)" % sm_max,
                     "peak_measured_dfma": probe.get("dfma"), "peak_measured_dmma": probe.get("dmma"),
                     "frac_of_measured_dfma": (a / probe["dfma"]) if probe.get("dfma") else None,
                     "frac_executed": a / fp64_peak,
                     "executed_fma_per_launch": int(fma_executed),
                     "nominal": {"fma_per_launch": leg_flop / 2.0, "tflops": an, "ratio_to_peak": an / fp64_peak,
                                 "note": "SURVEY 8(d) count incl. the below-range steps the kernel skips"},
                     "frac_at_sampled_clock": (a / (fp64_peak * sm_mhz / sm_max)) if sm_mhz else None}

    def mem(name, ms, nbytes):
        a = nbytes / (ms * 1e-3) / 1e9
        out[name] = {"bound": "hbm", "achieved": a, "peak": hbm, "unit": "GB/s", "frac": a / hbm, "traffic": None,
                     "ms": ms, "peak_source": hbm_src, "algorithmic_bytes": nbytes}

    traffic = ncu_traffic(cfg, npts)

    alu("legendre_synthesis", syn_ms["legendre"], info.legendre_fma_synthesis)
    alu("legendre_adjoint", adj_ms["legendre"], info.legendre_fma_adjoint)
    mem("interp", syn_ms["interp"], nu_bytes)
    mem("spread", adj_ms["spread"], nu_bytes + grid_bytes)      # + zeroing the grid
    fft_ms = syn_ms["fft_theta"] + syn_ms["deconv_pad"] + syn_ms["fft_fine_theta"] + syn_ms["fft_fine_phi"]
    fft_bytes = (2 * (M + 1) * nth2 * 16 + (M + 1) * (2 * L + 1) * 16 + (M + 1) * nth * 16
                 + 2 * (M + 1) * nth * 16 + (nth // 2 + 1) * ((M + 1) * 16 + nph * 8))
    mem("fourier_synthesis", fft_ms, fft_bytes)
    fft_ms_a = adj_ms["fft_theta"] + adj_ms["deconv_trunc"] + adj_ms["fft_fine_theta"] + adj_ms["fft_fine_phi"]
    mem("fourier_adjoint", fft_ms_a, fft_bytes)
    for k in out:
        out[k]["traffic"] = traffic.get(k)
    # interpolation / spreading at w >= 9 in FP64 are bound by the FP64 pipe (DMMA + kernel evaluation), not by
    # HBM: report that fraction too.  Executed FMA per point: 4 KS NT 256/8 (interp) or
    # 2 MT NT 256/4 (spread) tensor-core FMA + 2 (w/2)(deg+1) evaluation FMA.
    w = info.kernel_width
    nt = 2 if w <= 8 else (3 if w <= 14 else 4)
    ks = 2 if w <= 6 else (3 if w <= 11 else (4 if w <= 14 else 5))
    mt = 1 if w <= 6 else (2 if w <= 14 else 3)
    ev = 2 * ((w + 1) // 2) * (max(w, 5) + 1)
    for name, fma in (("interp", ks * nt * 256 / 8 + ev), ("spread", mt * nt * 256 / 4 + ev)):
        tf = 2.0 * fma * npts / (out[name]["ms"] * 1e-3) / 1e12
        out[name]["fp64_executed_tflops"] = tf
        out[name]["fp64_frac"] = tf / fp64_peak
        out[name]["fp64_frac_of_measured_dmma"] = (tf / probe["dmma"]) if probe.get("dmma") else None
    return out


def max_over_ranks(ms, world, device):
    """Replicas only: every rank times the same per-rank workload; the job time of a step is
    the slowest rank's (CUDA-event ms, MAX all-reduce).  Works with any backend (gloo on CPU in the tests)."""
    if world <= 1:
        return float(ms)
    import torch
    import torch.distributed as dist
    t = torch.tensor([float(ms)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def job_value(ms, world):
    """`value` for N replicas: time per (synthesis + adjoint) pair delivered by the whole job."""
    return ms / world


def run_b200(args, rank, world):
    import torch
    import torch.distributed as dist
    from paper_2406_14542_b200 import nusht

    local = int(os.environ.get("LOCAL_RANK", 0))
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl")
    cfg, theta, phi, alm, x = inputs.make_config(args.config, npts=args.npts)
    npts = len(theta)
    L, M, eps = cfg["lmax"], cfg["mmax"], cfg["eps"]
    d_theta, d_phi = torch.from_numpy(theta).cuda(), torch.from_numpy(phi).cuda()
    if cfg["deflection"] is not None:      # lensing-like config: the points are the deflected pixels, Eq. C1 on the GPU
        d_theta, d_phi = nusht.nusht_pointing(d_theta, d_phi, *(torch.from_numpy(a).cuda() for a in cfg["deflection"]))
    plan = nusht.Plan(L, M, d_theta, d_phi, eps, cfg["dtype"], sigma=args.sigma)
    del d_theta, d_phi
    d_alm, d_x = torch.from_numpy(alm).cuda(), torch.from_numpy(x).cuda()
    d_map = torch.empty(npts, dtype=torch.float64, device="cuda")
    d_out = torch.empty(plan.nlm, dtype=torch.complex128, device="cuda")
    stream = torch.cuda.current_stream()

    def step():
        plan.synthesis(d_alm, d_map, stream)
        plan.adjoint(d_x, d_out, stream)

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    # FP64 throughput of this device (denominator of the Legendre / nuFFT rooflines), outside the timed region
    probe = {"dfma": nusht.probe_fp64("dfma"), "dmma": nusht.probe_fp64("dmma")}
    plan.set_stage_timing(False)
    for _ in range(max(args.warmup, 3)):
        step()
    barrier()
    sampler = ClockSampler(local)
    sampler.start()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    launches0 = nusht.launch_count()
    e0.record(stream)
    for _ in range(args.steps):                 # the timed region: exactly K steps, nothing else
        step()
    e1.record(stream)
    launches = nusht.launch_count() - launches0   # kernels of libnusht.so launched inside the timed region (counted)
    barrier()
    ms = e0.elapsed_time(e1) / args.steps
    ms = max_over_ranks(ms, world, "cuda")
    # per-stage CUDA-event times: a second pass over the same K steps with the plan's stage events on
    # (reading them needs a sync after each step, so this pass is not the one `value` comes from)
    plan.set_stage_timing(True)
    syn_acc, adj_acc = {}, {}
    for _ in range(args.steps):
        step()
        for acc, t in ((syn_acc, plan.stage_times("synthesis")), (adj_acc, plan.stage_times("adjoint"))):
            for k, v in t.items():
                acc[k] = acc.get(k, 0.0) + v / args.steps
    barrier()
    clocks = sampler.stop()

    # end to end through the host-buffer C-ABI calls: pinned host inputs, H2D + D2H inside the region
    e2e = None
    if not args.no_e2e:
        h_alm, h_x = torch.from_numpy(alm).pin_memory(), torch.from_numpy(x).pin_memory()
        h_map = torch.empty(npts, dtype=torch.float64).pin_memory()
        h_out = torch.empty(plan.nlm, dtype=torch.complex128).pin_memory()
        plan.set_stage_timing(False)
        for _ in range(2):
            plan.synthesis_host(h_alm, h_map, stream)
            plan.adjoint_host(h_x, h_out, stream)
        barrier()
        t0 = time.perf_counter()
        for _ in range(args.steps):
            plan.synthesis_host(h_alm, h_map, stream)
            plan.adjoint_host(h_x, h_out, stream)
            plan.host_sync()          # both results are in host memory
        barrier()
        e2e_ms = (time.perf_counter() - t0) * 1e3 / args.steps
        e2e_ms = max_over_ranks(e2e_ms, world, "cuda")
        # the same K steps as a pipeline: no synchronisation between steps, each step in flight has host output
        # buffers of its own (two sets, as the library has two sets of staging buffers), one nusht_host_sync at the end
        h_map2 = torch.empty(npts, dtype=torch.float64).pin_memory()
        h_out2 = torch.empty(plan.nlm, dtype=torch.complex128).pin_memory()
        outs = [(h_map, h_out), (h_map2, h_out2)]
        barrier()
        t0 = time.perf_counter()
        for k in range(args.steps):
            plan.synthesis_host(h_alm, outs[k & 1][0], stream)
            plan.adjoint_host(h_x, outs[k & 1][1], stream)
        plan.host_sync()
        barrier()
        pipe_ms = max_over_ranks((time.perf_counter() - t0) * 1e3 / args.steps, world, "cuda")
        nb = plan.nlm * 16 + npts * 8
        e2e = {"value": job_value(e2e_ms, world), "unit": "ms", "h2d_bytes_per_step": nb, "d2h_bytes_per_step": nb,
               "how": "nusht_synthesis_host + nusht_adjoint_host + nusht_host_sync every step (both results in host "
                      "memory before the next step starts)",
               "pipelined": {"value": job_value(pipe_ms, world), "unit": "ms",
                             "how": "the same calls and copies, K steps without a synchronisation between them, one "
                                    "nusht_host_sync at the end; two sets of pinned host output buffers"},
               "checksum": float(h_map[:1024].double().sum().item()),
               "checksum_pipelined": float(outs[(args.steps - 1) & 1][0][:1024].double().sum().item())}
    # pointing (Eq. C1): not part of a step; timed on its own over the same number of points
    pointing = None
    if rank == 0:
        gen = torch.Generator(device="cuda")
        gen.manual_seed(1234)
        sig = 2.5 * np.pi / (180 * 60)
        p_t = torch.from_numpy(theta).cuda()
        p_p = torch.from_numpy(phi).cuda()
        a_t = sig * torch.randn(npts, dtype=torch.float64, device="cuda", generator=gen)
        a_p = sig * torch.randn(npts, dtype=torch.float64, device="cuda", generator=gen)
        for _ in range(3):
            nusht.nusht_pointing(p_t, p_p, a_t, a_p, stream)
        p0, p1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        torch.cuda.synchronize()
        p0.record(stream)
        for _ in range(args.steps):
            nusht.nusht_pointing(p_t, p_p, a_t, a_p, stream)
        p1.record(stream)
        torch.cuda.synchronize()
        pt_ms = p0.elapsed_time(p1) / args.steps
        peak, src, _ = measured_peaks()
        pointing = {"kernel": "k_pointing", "npts": npts, "ms": pt_ms, "bound": "hbm", "algorithmic_bytes": 48 * npts,
                    "achieved": 48 * npts / (pt_ms * 1e-3) / 1e9, "peak": peak, "unit": "GB/s",
                    "frac": 48 * npts / (pt_ms * 1e-3) / 1e9 / peak, "peak_source": src,
                    "note": "outside the timed step; output allocation (2 x npts x 8 B) inside the timed calls"}
        del a_t, a_p
        # re-pointing a finished plan (Appendix C: one point set per deflection field)
        sort_ms0 = plan.info.sort_ms
        torch.cuda.synchronize()
        plan.set_points(p_t, p_p)
        set_points_ms = plan.info.set_points_ms
        del p_t, p_p
    if rank != 0:
        return
    roofs = stage_rooflines(cfg, plan.info, npts, syn_acc, adj_acc, clocks.get("sm_mhz"), probe)
    own = ["legendre_synthesis", "legendre_adjoint", "interp", "spread"]
    dominant = max(own, key=lambda k: roofs[k]["ms"])
    roof = dict(roofs[dominant])
    roof["kernel"] = dominant
    out = {
        "metric": METRIC, "value": job_value(ms, world), "unit": "ms", "n_gpus": world, "steps": args.steps,
        "warmup": max(args.warmup, 3), "ms_per_step": ms, "higher_is_better": False, "scaling": "weak",
        "vs_baseline": None, "dtype": "f64", "data": "synthetic", "config": workload_config(cfg, npts),
        "transforms_per_s": 2e3 * world / ms, "points_per_s": 2.0 * npts * world / (ms * 1e-3),
        "synthesis_ms": sum(syn_acc.values()), "adjoint_ms": sum(adj_acc.values()),
        "stage_ms": {"synthesis": syn_acc, "adjoint": adj_acc},
        "roofline": roof, "stage_rooflines": roofs, "clocks": clocks, "e2e": e2e,
        # kernels of libnusht.so launched inside the timed region, counted by the library (nusht_launch_count);
        # cuFFT's kernels and memsets are not included
        "gpu_launches": int(launches),
        "fp64_probe": {"dfma_tflops": probe["dfma"], "dmma_tflops": probe["dmma"],
                       "how": "nusht_probe_fp64: dependent-free DFMA / mma.sync.m8n8k4.f64 streams on every SM, CUDA "
                              "events, best of 10, measured in this run before the timed region"},
        "pointing": pointing,
        "plan": {"ms": plan.info.plan_ms, "workspace_gb": plan.info.workspace_bytes / 1e9,
                 "sort_ms": sort_ms0, "sort_algorithmic_bytes": 60 * npts,
                 "sort_gbs": (60 * npts / (sort_ms0 * 1e-3) / 1e9) if sort_ms0 > 0 else None,
                 "sort_frac_of_hbm": (60 * npts / (sort_ms0 * 1e-3) / 1e9 / measured_peaks()[0])
                 if sort_ms0 > 0 else None,
                 # nusht_set_points: the same points handed to the finished plan again (wall time incl. allocation,
                 # device synchronised on both sides; outside the timed region)
                 "set_points_ms": set_points_ms,
                 "n_rings": plan.info.n_rings, "n_theta": plan.info.n_theta, "n_theta_fine": plan.info.n_theta_fine,
                 "n_phi_fine": plan.info.n_phi_fine, "kernel_width": plan.info.kernel_width,
                 "sigma": plan.info.sigma},
    }
    if not args.no_cpu_baseline and world == 1:
        ns = min(npts, 1 << 16)
        o_theta, o_phi = oracle_points(cfg, theta, phi, slice(0, ns))
        _, desc = oracle_sample(cfg, o_theta, o_phi, alm, x[:ns], args.cpu_seconds)
        desc["value"] *= npts / ns
        desc["sample"] += "; then x%.0f from the %d-point prefix to %d points" % (npts / ns, ns, npts)
        out["cpu_baseline"] = desc
    print(json.dumps(out))
    if world > 1:
        dist.destroy_process_group()


def run_eps_sweep(args):
    """Config 5: accuracy (Eq. 9-10 against the long-double oracle on a seeded subset of the points; the
    paper's own subset is 1e6 points, which a direct sum cannot afford here) and throughput per eps."""
    import torch
    from oracle import oracle as o
    from paper_2406_14542_b200 import nusht
    torch.cuda.set_device(0)
    cfg, theta, phi, alm, x = inputs.make_config(args.config, npts=args.npts)
    L, M, npts = cfg["lmax"], cfg["mmax"], len(theta)
    rng = np.random.default_rng(12345)
    sub = np.sort(rng.choice(npts, min(args.sweep_subset, npts), replace=False))
    o_theta, o_phi = oracle_points(cfg, theta, phi, sub)
    f_ref = o.synthesis(L, M, o_theta, o_phi, alm, "ld")
    xs = np.zeros(npts)
    xs[sub] = x[sub]
    c_ref = o.adjoint(L, M, o_theta, o_phi, x[sub], "ld")
    d_theta, d_phi = torch.from_numpy(theta).cuda(), torch.from_numpy(phi).cuda()
    if cfg["deflection"] is not None:
        d_theta, d_phi = nusht.nusht_pointing(d_theta, d_phi, *(torch.from_numpy(a).cuda() for a in cfg["deflection"]))
    for dtype, eps in (("f32", 1e-4), ("f32", 1e-6), ("f64", 1e-8), ("f64", 1e-10), ("f64", 1e-12)):
        plan = nusht.Plan(L, M, d_theta, d_phi, eps, dtype)
        rd, cd = (np.float32, np.complex64) if dtype == "f32" else (np.float64, np.complex128)
        d_alm, d_x, d_xs = (torch.from_numpy(alm.astype(cd)).cuda(), torch.from_numpy(x.astype(rd)).cuda(),
                            torch.from_numpy(xs.astype(rd)).cuda())
        f = plan.synthesis(d_alm)
        c = plan.adjoint(d_xs)
        e_syn = float(np.linalg.norm(f[torch.from_numpy(sub).cuda()].cpu().numpy().astype(np.float64) - f_ref)
                      / np.linalg.norm(f_ref))
        e_adj = float(np.linalg.norm(c.cpu().numpy().astype(np.complex128) - c_ref) / np.linalg.norm(c_ref))
        d_map = torch.empty_like(f)
        d_out = torch.empty_like(c)
        plan.set_stage_timing(True)
        for _ in range(3):
            plan.synthesis(d_alm, d_map)
            plan.adjoint(d_x, d_out)
        torch.cuda.synchronize()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        for _ in range(args.steps):
            plan.synthesis(d_alm, d_map)
            plan.adjoint(d_x, d_out)
        e1.record()
        torch.cuda.synchronize()
        ms = e0.elapsed_time(e1) / args.steps
        print(json.dumps({"metric": METRIC, "value": ms, "unit": "ms", "dtype": dtype, "eps": eps,
                          "kernel_width": plan.info.kernel_width, "eps_eff_synthesis": e_syn, "eps_eff_adjoint": e_adj,
                          "subset_points": int(len(sub)), "points_per_s": 2.0 * npts / (ms * 1e-3),
                          "stage_ms": {"synthesis": plan.stage_times("synthesis"), "adjoint": plan.stage_times("adjoint")},
                          "config": workload_config(dict(cfg, eps=eps), npts)}))
        plan.destroy()
        del d_alm, d_x, d_xs, f, c, d_map, d_out


def run_ring(args):
    """Ring-grid modes: not the headline metric; one JSON line with CUDA-event times and the Legendre share."""
    import torch
    from paper_2406_14542_b200 import nusht
    torch.cuda.set_device(0)
    L = args.lmax
    stream = torch.cuda.current_stream()
    phi0 = None
    if args.ring == "gl":
        xg, wg = np.polynomial.legendre.leggauss(L + 1)
        theta = np.arccos(xg[::-1])
        half = (L + 1) // 2
        theta[L + 1 - half:] = np.pi - theta[:half][::-1]
        nphi = np.full(L + 1, 2 * L + 2)
        weight = wg[::-1] * (2 * np.pi / (2 * L + 2))
    elif args.ring in ("healpix", "healpix-lens"):   # nside = (lmax + 1) / 2: 2 (nside - 1) cap rings of distinct lengths
        theta, nphi, phi0, weight = inputs.healpix_ring_layout((L + 1) // 2)
    else:
        nr = 2 * (L + 1)
        theta = np.pi * (np.arange(nr) + 0.5) / nr
        nphi = np.full(nr, nr)
        weight = None
    plan = nusht.RingPlan(L, L, theta, nphi, phi0, weight)
    alm = torch.from_numpy(inputs.random_alm(L, L, 7, "inv_l2")).cuda()
    f = torch.empty(plan.npix, dtype=torch.float64, device="cuda")
    out = torch.empty(plan.nlm, dtype=torch.complex128, device="cuda")
    if args.ring in ("gl", "healpix"):
        def step():
            plan.synthesis(alm, f, stream)
            plan.analysis(f, out, stream)
        what = "ring synthesis + analysis on " + ("a Gauss-Legendre grid" if args.ring == "gl" else
                                                 "a HEALPix-style ring layout, nside = (lmax + 1) / 2")
    elif args.ring == "healpix-lens":
        th = torch.from_numpy(np.repeat(theta, nphi)).cuda()
        ph = torch.from_numpy(np.concatenate([p0 + 2 * np.pi * np.arange(n) / n for n, p0 in zip(nphi, phi0)])).cuda()
        philm = torch.from_numpy(inputs.random_alm(L, L, 8, "inv_l2")).cuda() * 2e-5      # a few arcminutes rms
        eps = 1e-10
        lens = nusht.Plan(L, L, th, ph, eps)          # planned once; every step re-points it (nusht_set_points)

        def step():
            a_t, a_p = plan.gradient(philm, stream)
            t2, p2 = nusht.nusht_pointing(th, ph, a_t, a_p, stream)
            lens.set_points(t2, p2)
            lens.synthesis(alm, f, stream)
        what = ("lensed map on a HEALPix-style layout, nside = (lmax + 1) / 2: Eq. C2 (two ring syntheses) + Eq. C1 + "
                "nusht_set_points + nuSHT synthesis at eps = %g" % eps)
    else:
        th = torch.from_numpy(np.repeat(theta, nphi)).cuda()
        ph = torch.from_numpy(np.tile(2 * np.pi * np.arange(nphi[0]) / nphi[0], len(theta))).cuda()
        philm = alm * 2e-5

        def step():
            a_t, a_p = plan.gradient(philm, stream)
            nusht.nusht_pointing(th, ph, a_t, a_p, stream)
        what = "deflection field (Eq. C2) + pointing (Eq. C1) on the 2(lmax+1)^2 equi-angular grid"
    for _ in range(max(args.warmup, 3)):
        step()
    torch.cuda.synchronize()
    n0 = nusht.launch_count()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record(stream)
    for _ in range(args.steps):
        step()
    e1.record(stream)
    torch.cuda.synchronize()
    ms = e0.elapsed_time(e1) / args.steps
    print(json.dumps({"metric": "ring_%s_ms" % args.ring.replace("-", "_"), "value": ms, "unit": "ms", "n_gpus": 1, "steps": args.steps,
                      "warmup": max(args.warmup, 3), "higher_is_better": False, "dtype": "f64", "data": "synthetic",
                      "config": {"workload": what, "lmax": L, "nrings": int(len(theta)), "npix": int(plan.npix)},
                      "pixels_per_s": plan.npix / (ms * 1e-3), "gpu_launches": int(nusht.launch_count() - n0),
                      "plan": {"ms": plan.info.plan_ms, "workspace_gb": plan.info.workspace_bytes / 1e9,
                               "npairs": plan.info.npairs, "nruns": plan.info.nruns}}))
    plan.destroy()


def main():
    args = parse()
    if args.ring:
        run_ring(args)
        return
    if args.eps_sweep:
        run_eps_sweep(args)
        return
    rank = int(os.environ.get("RANK", 0))
    world = int(os.environ.get("WORLD_SIZE", 1))
    if args.impl == "reference":
        run_reference(args, rank)
        return
    run_b200(args, rank, world)


if __name__ == "__main__":
    main()
