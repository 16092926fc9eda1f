#!/usr/bin/env python
"""bench.py -- NUFFT-Radon forward+adjoint pairs/s on B200 (BASELINE.json metric).

A step = one pass of the whole hot path (radon_forward_batch then radon_adjoint_batch: stages
F1-F4 and A1-A4 of SURVEY.md 8(a)) over one batch of `--slices` synthetic 2048^2 slices with
1025 x 2048 projections (BASELINE.json configs[3] shape, batched as configs[4]).  `value` is
whole-job pairs/s with inputs resident in HBM; `e2e` is the same metric through the host-buffer
C-ABI calls (pinned host memory, copies inside the timed region).  Beside the contract's keys the
line carries `stages` (per-stage CUDA events of a second, untimed pass), `roofline` (the dominant
stage against the measured HBM peak), `gridding_kernels` (the bare interpolation / gridding kernels
on complex data, SURVEY 8(d)'s 151 MB, north_star's 50 % target), `paper_shape` (PAPER.md:59's own
180 x 1024 shape, context), `next_rows` (radon_inverse, solver loop, filter), `library_context` (cuFFT timed beside the FFT passes:
a yardstick, never on the product path) and `cpu_baseline` (the oracle, sampled).

  python bench.py [--gpus N] [--steps K] [--warmup W] [--slices B] [--impl reference]
  torchrun ... bench.py --gpus N ...      one rank per GPU; slice-parallel replicas (weak scaling)
"""
import argparse
import json
import os
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

METRIC = "nufft_radon_fwd_adj_pairs_per_s"
UNIT = "pairs/s"
WORKLOAD = "config4_beamline_2048 (2048^2 fp32, 1025 angles x 2048 bins, sigma=2, W=6)"


def measured_peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        with open(path) as f:
            return float(json.load(f)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    return 6650.0, "fallback (B200_PROFILING.md: 6.65 TB/s)"


def stage_bytes(N, G, M, n_angles, W=6):
    """Algorithmic bytes per launch of each stage of radon_forward / radon_adjoint (DESIGN.md
    section 7).  Image and sinogram are real, so the path moves the HERMITIAN HALF of the
    spectrum: grid rows ky = 0..G/2 (+ W halo rows for the gather), T = (G/2+1) x N, polar
    samples j >= 0 in the forward direction.  These are half of SURVEY.md 8(d)'s full-complex
    figures (kept for the bare gridding kernels, see gridding_bytes)."""
    H = G // 2 + 1
    return {
        "F1_colfft": 4 * N * N + 8 * H * N, "F2_rowfft": 8 * H * N + 8 * (H + W) * G,
        "F3_gather": 8 * (H + W) * G + 8 * (M // 2 + n_angles), "F4_proj_ifft": 8 * (M // 2 + n_angles) + 4 * M,
        "A1_proj_fft": 4 * M + 8 * M, "A2_scatter": 8 * M + 8 * H * G,
        "A3_rowifft": 8 * H * G + 8 * H * N, "A4_colifft": 8 * H * N + 4 * N * N,
    }


# dram__bytes_read.sum + dram__bytes_write.sum per launch at config 4: NOT measured by this run
# (ncu cannot run inside it) but copied from the ncu --set full capture named below, one slice at a
# time.  Values below the algorithmic bytes mean that part of a stage's output was still in the
# 126 MB L2 when the kernel ended (one-slice capture: the grid written by A2 is read by A3 from L2).
NCU_TRAFFIC_SOURCE = "profiles/r02_kernels.md (ncu --set full, one slice at a time; copied, not measured by this run)"
NCU_DRAM_BYTES = {
    "F1_colfft": 17.06e6, "F2_rowfft": 44.63e6, "F3_gather": 69.30e6, "F4_proj_ifft": 8.59e6,
    "A1_proj_fft": 8.46e6, "A2_scatter": 40.66e6, "A3_rowifft": 71.60e6, "A4_colifft": 33.74e6,
}


def gridding_bytes(G, M):
    """bare gridding / inverse gridding on arbitrary complex data."""
    return 8 * G * G + 8 * M


class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled during the timed region."""

    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.index, self.proc, self.lines = index, None, []

    def start(self):
        try:
            self.proc = subprocess.Popen(
                ["nvidia-smi", "-i", str(self.index), f"--query-gpu={self.Q}", "--format=csv,noheader,nounits",
                 "-lms", "20"], stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.t = threading.Thread(target=self._read, daemon=True)
            self.t.start()
        except OSError:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.lines.append((time.perf_counter(), line.strip()))

    def wait_first(self, timeout=5.0):
        """nvidia-smi takes a moment to start: block until its first sample arrives."""
        t0 = time.perf_counter()
        while self.proc and not self.lines and time.perf_counter() - t0 < timeout:
            time.sleep(0.01)

    def stop(self, t_begin=None, t_end=None):
        """Samples taken in [t_begin, t_end] (host clock); all samples if the window is None."""
        if not self.proc:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except subprocess.TimeoutExpired:
            self.proc.kill()
        sm, mx, reasons = [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for ts, ln in self.lines:
            if t_begin is not None and not (t_begin <= ts <= t_end):
                continue
            f = [x.strip() for x in ln.split(",")]
            if len(f) < 7:
                continue
            try:
                sm.append(float(f[0])); mx.append(float(f[1]))
            except ValueError:
                continue
            for n, v in zip(names, f[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(n)
        sm.sort()
        return {"sm_mhz": sm[len(sm) // 2] if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "samples": len(sm), "reasons": sorted(reasons)}


def cpu_oracle_pairs_per_s(cfg, n_sample, seed=77):
    """The oracle as it stands (closed-form O-direct, the routine the full-size parity tests
    use) on a bounded sample: n_sample sinogram entries + n_sample pixels of one slice;
    cost is exactly linear in the number of outputs, so pairs/s is extrapolated."""
    import numpy as np

    import oracle
    import workloads

    x = workloads.make_batch_slice(0, cfg.N).astype(np.float64)
    rng = np.random.default_rng(seed)
    idx = rng.choice(cfg.M, n_sample, replace=False)
    pix = rng.choice(cfg.N * cfg.N, n_sample, replace=False)
    y = rng.standard_normal((cfg.n_angles, cfg.n_det))
    t0 = time.perf_counter(); oracle.dirichlet_forward_subset(x, cfg.n_angles, cfg.n_det, idx)
    t1 = time.perf_counter(); oracle.dirichlet_adjoint(y, cfg.N, pix=pix)
    t2 = time.perf_counter()
    t_pair = (t1 - t0) / n_sample * cfg.M + (t2 - t1) / n_sample * cfg.N * cfg.N
    return 1.0 / t_pair, oracle.num_threads(), (t2 - t0)


def run_reference(args):
    """--impl reference: the CPU oracle on the host cores, same metric/config."""
    import workloads

    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return 0
    cfg = workloads.get_config(4)
    n_sample = args.ref_sample
    for _ in range(args.warmup and 1):
        cpu_oracle_pairs_per_s(cfg, max(n_sample // 8, 8))
    vals, t_total = [], 0.0
    for _ in range(args.steps):
        v, cores, dt = cpu_oracle_pairs_per_s(cfg, n_sample)
        vals.append(v); t_total += dt
    value = len(vals) / sum(1.0 / v for v in vals)
    sample = (f"{n_sample} sinogram entries + {n_sample} pixels of one slice per step, closed-form "
              f"O-direct (oracle.dirichlet_forward_subset / dirichlet_adjoint), extrapolated x M/{n_sample}, x N^2/{n_sample}")
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 / value * args.slices,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": WORKLOAD, "slices_per_step_per_gpu": args.slices, "kind": "cpu oracle, extrapolated"},
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0, "gpus_used": 0,
    }
    print(json.dumps(line))
    return 0


def respawn_under_torchrun(args):
    """`python bench.py --gpus N` without a torchrun environment: start N ranks on this node (the
    driver's own launch line) and hand over to them."""
    import socket

    with socket.socket() as sk:
        sk.bind(("127.0.0.1", 0))
        port = sk.getsockname()[1]
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={args.gpus}",
           "--master-addr", "127.0.0.1", "--master-port", str(port), os.path.abspath(__file__)] + sys.argv[1:]
    return subprocess.call(cmd)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--slices", type=int, default=32, help="slices per step per GPU (configs[4]: 32)")
    ap.add_argument("--impl", default="b200", choices=["b200", "reference"])
    ap.add_argument("--ref-sample", type=int, default=512)
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-library-context", action="store_true", help="skip the cuFFT yardstick (context only)")
    ap.add_argument("--no-clock-load", action="store_true",
                    help="skip the 0.5 s of untimed identical steps that give nvidia-smi time to sample "
                         "(profiling runs: keeps the kernel launch list short and deterministic)")
    args = ap.parse_args()
    if args.impl == "reference":
        return run_reference(args)
    if args.gpus > 1 and "WORLD_SIZE" not in os.environ:
        return respawn_under_torchrun(args)

    import numpy as np
    import torch

    import paper_1009_1380_b200 as rb
    import workloads
    from paper_1009_1380_b200 import dist as rdist

    rb.lib()                                   # fail loudly if the CUDA library is missing
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; there is no CPU fallback (use --impl reference for the oracle)")
    rank, local_rank, world = rdist.init("nccl")
    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    cfg = workloads.get_config(4)
    B = args.slices
    # the first plan of a process also pays for the CUDA context and for loading the library's kernels
    t_plan = time.perf_counter()
    rb.RadonPlan(64, 90, 91).close()
    torch.cuda.synchronize()
    first_plan_ms = (time.perf_counter() - t_plan) * 1e3
    t_plan = time.perf_counter()
    plan = rb.RadonPlan(cfg.N, cfg.n_angles, cfg.n_det)
    torch.cuda.synchronize()
    plan_create_ms = (time.perf_counter() - t_plan) * 1e3

    # synthetic slices (configs[4] recipe), distinct per rank; resident in HBM before timing
    n_unique = min(B, 8)
    uniq = np.stack([workloads.make_batch_slice(rank * B + i, cfg.N) for i in range(n_unique)])
    hx = torch.from_numpy(np.concatenate([uniq] * ((B + n_unique - 1) // n_unique))[:B].copy())
    # every slice distinct in memory (no aliasing): scale repeats slightly
    for i in range(B):
        hx[i] *= 1.0 + 1e-3 * (i // n_unique)
    x = hx.to(dev)
    sino = torch.empty((B, cfg.n_angles, cfg.n_det), dtype=torch.float32, device=dev)
    xt = torch.empty_like(x)

    def step():
        plan.radon_forward_batch(x, sino)
        plan.radon_adjoint_batch(sino, xt)

    for _ in range(max(args.warmup, 3)):
        step()
    torch.cuda.synchronize()
    plan.stage_times()                          # clear

    sampler = ClockSampler(local_rank)
    sampler.start()
    sampler.wait_first()
    stream = torch.cuda.current_stream()
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    rdist.barrier(); torch.cuda.synchronize()
    n0 = rb.kernel_launch_count()
    t_host0 = time.perf_counter()
    ev0.record(stream)
    for _ in range(args.steps):
        step()
    ev1.record(stream)
    torch.cuda.synchronize(); rdist.barrier()
    launches = rb.kernel_launch_count() - n0
    # per-stage times: a second, untimed pass of the same steps with CUDA events recorded
    # between the stages inside the C ABI (the events cost a few us per pair, so they stay out
    # of the timed region above)
    plan.stage_timing(True)
    for _ in range(args.steps):
        step()
    torch.cuda.synchronize()
    plan.stage_timing(False)
    stages = plan.stage_times()
    # the timed region is tens of ms: keep the GPU under the identical load a little longer so
    # that nvidia-smi (20 ms period) sees the clocks this workload runs at
    t_load_end = time.perf_counter() + 0.5
    while not args.no_clock_load and time.perf_counter() < t_load_end:
        step()
        torch.cuda.synchronize()
    clocks = sampler.stop(t_host0, time.perf_counter())
    clocks["window"] = "timed region + 0.5 s of identical untimed steps, nvidia-smi -lms 20"
    t_ms = rdist.max_over_ranks(ev0.elapsed_time(ev1), dev)
    pairs = world * B * args.steps
    value = pairs / (t_ms * 1e-3)

    # ---- e2e: host buffers through the C ABI, copies inside the timed region ------------
    e2e = None
    if not args.no_e2e:
        hxp = hx.pin_memory()
        hs = torch.empty((B, cfg.n_angles, cfg.n_det), dtype=torch.float32).pin_memory()
        hxt = torch.empty((B, cfg.N, cfg.N), dtype=torch.float32).pin_memory()

        def step_host():
            plan.radon_forward_adjoint_host(hxp, hs, hxt)

        def step_host_separate():
            plan.radon_forward_host(hxp, hs)
            plan.radon_adjoint_host(hs, hxt)

        n_e2e = max(1, min(args.steps, 3))
        rates = {}
        for name, fn in (("pair_call", step_host), ("separate_calls", step_host_separate)):
            fn()
            rdist.barrier(); torch.cuda.synchronize()
            t0 = time.perf_counter()
            for _ in range(n_e2e):
                fn()
            torch.cuda.synchronize()
            rates[name] = world * B * n_e2e / rdist.max_over_ranks(time.perf_counter() - t0, dev)
        e2e = {"value": rates["pair_call"], "unit": UNIT,
               "h2d_bytes_per_step": int(hxp.numel() * 4),
               "d2h_bytes_per_step": int(hs.numel() * 4 + hxt.numel() * 4),
               "steps": n_e2e, "api": "radon_forward_adjoint_host (pinned host buffers; image up, sinogram and adjoint image down)",
               "separate_calls": {"value": rates["separate_calls"], "h2d_bytes_per_step": int(hxp.numel() * 4 + hs.numel() * 4),
                                  "d2h_bytes_per_step": int(hs.numel() * 4 + hxt.numel() * 4),
                                  "api": "radon_forward_host + radon_adjoint_host"}}

    # ---- roofline of the dominant kernel (stage with the largest device time) -----------
    peak, peak_src = measured_peaks()
    sbytes = stage_bytes(cfg.N, plan.G, cfg.M, cfg.n_angles)
    per_stage = {}
    for k, (ms, n) in stages.items():
        if n:
            us = ms / n * 1e3
            per_stage[k] = {"us_per_launch": round(us, 2), "launches_timed": n,
                            "algorithmic_MB": round(sbytes[k] / 1e6, 1),
                            "GBps": round(sbytes[k] / (us * 1e-6) / 1e9, 1),
                            "frac_of_hbm_peak": round(sbytes[k] / (us * 1e-6) / 1e9 / peak, 4)}
    dom = max(per_stage, key=lambda k: per_stage[k]["us_per_launch"] * per_stage[k]["launches_timed"]) if per_stage else None
    traffic = NCU_DRAM_BYTES.get(dom) if (dom and cfg.N == 2048) else None
    roofline = None
    if dom:
        ach = per_stage[dom]["GBps"]
        roofline = {"bound": "hbm", "kernel": dom, "achieved": ach, "peak": peak, "unit": "GB/s",
                    "frac": round(ach / peak, 4), "traffic": traffic, "traffic_source": NCU_TRAFFIC_SOURCE,
                    "peak_source": peak_src,
                    "algorithmic_bytes_per_launch": sbytes[dom],
                    "us_per_launch": per_stage[dom]["us_per_launch"]}

    # ---- the bare gridding kernels on arbitrary complex data (north_star: >= 50 % of the HBM
    #      roofline at this config): radon_interp_only (F3) and radon_grid_only (A2 + merge + dc),
    #      full grid / every sample, timed alone with CUDA events on the launching stream -----
    gk = {}
    gen = torch.Generator(device=dev); gen.manual_seed(1234 + rank)
    NBUF = 3     # 3 x 134 MB of grids: a call's grid was evicted from the 126 MB L2 by the two calls before it
    cgrid = [torch.view_as_complex(torch.randn((plan.G, plan.G, 2), device=dev, generator=gen)) for _ in range(NBUF)]
    cpol = [torch.view_as_complex(torch.randn((cfg.n_angles, cfg.n_det, 2), device=dev, generator=gen)) for _ in range(NBUF)]
    ogrid = [torch.empty_like(cgrid[0]) for _ in range(NBUF)]
    opol = [torch.empty_like(cpol[0]) for _ in range(NBUF)]
    gbytes = gridding_bytes(plan.G, cfg.M)
    for name, fn in (("interp_only", lambda i: plan.radon_interp_only(cgrid[i % NBUF], opol[i % NBUF])),
                     ("grid_only", lambda i: plan.radon_grid_only(cpol[i % NBUF], ogrid[i % NBUF]))):
        for i in range(2 * NBUF):
            fn(i)
        times, reps, calls = [], 5, 4 * NBUF
        for _ in range(reps):
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record(stream)
            for i in range(calls):
                fn(i)
            e1.record(stream)
            torch.cuda.synchronize()
            times.append(e0.elapsed_time(e1) / calls)
        times.sort()
        us = times[reps // 2] * 1e3                      # median of 5 runs of 12 back-to-back calls
        gk[name] = {"us_per_call": round(us, 2), "algorithmic_MB": round(gbytes / 1e6, 1),
                    "GBps": round(gbytes / (us * 1e-6) / 1e9, 1),
                    "frac_of_hbm_peak": round(gbytes / (us * 1e-6) / 1e9 / peak, 4),
                    "samples_per_s": cfg.M / (us * 1e-6),
                    "us_min": round(times[0] * 1e3, 2), "us_max": round(times[-1] * 1e3, 2),
                    "l2": "12 back-to-back calls rotating over 3 grid buffers (402 MB > 126 MB L2); median of 5 runs"}
    del cgrid, cpol, ogrid, opol

    # ---- the paper's own timing shape ("1024x1024 grid sampled with 180 angles, 1024
    #      pixels per angle", 3 ms FFTs + 6 ms gridding on a Tesla C1060): context, not the headline.
    #      Both readings of "1024x1024 grid": the oversampled grid, or the image. ------
    paper_shape = {}
    gen_p = torch.Generator(device=dev); gen_p.manual_seed(99)
    for label, Np in (("grid_1024 (N=512, G=1024)", 512), ("image_1024 (N=1024, G=2048)", 1024)):
        pp = rb.RadonPlan(Np, 180, 1024)
        xp = torch.from_numpy(workloads.make_batch_slice(1, Np)).to(dev)
        sp = torch.empty((180, 1024), dtype=torch.float32, device=dev)
        xo = torch.empty_like(xp)
        for _ in range(5):
            pp.radon_forward(xp, sp); pp.radon_adjoint(sp, xo)
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(stream)
        for _ in range(50):
            pp.radon_forward(xp, sp); pp.radon_adjoint(sp, xo)
        e1.record(stream)
        torch.cuda.synchronize()
        us = e0.elapsed_time(e1) / 50 * 1e3
        paper_shape[label] = {"us_per_pair": round(us, 1), "pairs_per_s": round(1e6 / us, 1),
                              "paper_C1060_us_per_pair": 9000.0,
                              "note": "working set fits the 126 MB L2; 180 x 1024 samples, sigma=2, W=6"}
        # the paper's own design for the gridding step (load-balanced quadtree bins, one
        # thread block per bin, two per-bin strategies) against this library's, same sum, same data
        cp = torch.view_as_complex(torch.randn((180, 1024, 2), device=dev, generator=gen_p))
        cg = torch.empty((pp.G, pp.G), dtype=torch.complex64, device=dev)
        cmpv = {}
        for name, fn in (("radon_grid_only", lambda: pp.radon_grid_only(cp, cg)),
                         ("radon_grid_only_paper_bins_4096", lambda: pp.radon_grid_only_paper_bins(cp, cg, n_bins=4096))):
            for _ in range(3):
                fn()
            e0.record(stream)
            for _ in range(10):
                fn()
            e1.record(stream)
            torch.cuda.synchronize()
            cmpv[name + "_us"] = round(e0.elapsed_time(e1) / 10 * 1e3, 1)
        cmpv["bins"] = pp.paper_bins_stats()
        paper_shape[label]["gridding_design_comparison"] = cmpv
        del pp

    # ---- the density-compensated inverse Radon transform at this config ----
    xi = torch.empty((cfg.N, cfg.N), dtype=torch.float32, device=dev)
    plan.radon_inverse(sino[0], xi)                       # builds D (host, fp64) on first use
    for _ in range(3):
        plan.radon_inverse(sino[0], xi)
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record(stream)
    for i in range(20):
        plan.radon_inverse(sino[i % B], xi)
    e1.record(stream)
    torch.cuda.synchronize()
    next_rows = {"radon_inverse_us_per_call": round(e0.elapsed_time(e1) / 20 * 1e3, 1),
                 "note": "A1 with density weights (PAPER.md:89) + A2-A4; one slice at a time"}

    # ---- SURVEY 8(f) items 3-4 / BASELINE.json configs[2]: the solver iteration
    #      x <- S_tau(x - alpha A^T F (A x - b)) inside the library:
    #      radon_solver_run = one iteration (8 kernels, residual / filter / update fused into the
    #      epilogues) captured as a CUDA graph and launched n times; F = the polynomial sinogram filter ----
    c3 = workloads.get_config(3)
    p3 = rb.RadonPlan(c3.N, c3.n_angles, c3.n_det)
    xt3 = torch.from_numpy(workloads.make_image(3)).float().to(dev)
    b3 = p3.radon_forward(xt3).clone()
    v3 = torch.ones_like(xt3)
    for _ in range(8):
        w3 = p3.radon_adjoint(p3.radon_forward(v3)).clone()
        lam = float(w3.norm() / v3.norm())
        v3 = w3 / w3.norm()
    alpha, tau = 1.0 / lam, 1e-4
    solver = {}
    for label, filtered in (("plain", False), ("filtered_order3", True)):
        x3 = torch.zeros_like(xt3)
        p3.radon_solver_run(x3, b3, alpha, tau, 10, filtered)
        n0 = rb.kernel_launch_count()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(stream)
        p3.radon_solver_run(x3, b3, alpha, tau, 100, filtered)     # 200 alternating operator calls
        e1.record(stream)
        torch.cuda.synchronize()
        r = p3.radon_forward(x3) - b3
        solver[label] = {"iterations_per_s": round(100 / (e0.elapsed_time(e1) * 1e-3), 1),
                         "us_per_iteration": round(e0.elapsed_time(e1) * 10, 1),
                         "library_kernels_in_loop": int(rb.kernel_launch_count() - n0),
                         "relative_residual_after_110": round(float(r.norm() / b3.norm()), 4)}
    next_rows["solver_loop_config3"] = {**solver["plain"], "operator_calls": 200, "filtered": solver["filtered_order3"],
                                        "note": "radon_solver_run on configs[2] (1024^2, 64 x 1449): graph-captured "
                                                "iteration, no kernel outside the library; latency bound at this size"}
    del p3
    # filter(Radon{x}) against Radon{x} at config 4 (the filter runs in the epilogue of the F4 kernel)
    xf, sf = x[0], sino[0]
    sf_out = torch.empty_like(sf)
    ft = {}
    for label, fn in (("radon_forward", lambda: plan.radon_forward(xf, sf)),
                      ("radon_forward_filtered", lambda: plan.radon_forward_filtered(xf, sf)),
                      ("radon_filter_axis0", lambda: plan.radon_filter(sf, out=sf_out, axis=0)),
                      ("radon_filter_axis1", lambda: plan.radon_filter(sf, out=sf_out, axis=1))):
        for _ in range(3):
            fn()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(stream)
        for _ in range(20):
            fn()
        e1.record(stream)
        torch.cuda.synchronize()
        ft[label] = round(e0.elapsed_time(e1) / 20 * 1e3, 1)
    next_rows["sinogram_filter_us_per_call_config4"] = ft

    if rank != 0:
        return 0
    # ---- context only, never on the product path: the vendor FFT library (cuFFT through torch.fft)
    #      on the transforms F1-F2 and A3-A4 stand for, same sizes, inputs cycling through HBM ----
    library_context = None
    if not args.no_library_context and per_stage:
        G = cfg.G
        imgs = [torch.randn(cfg.N, cfg.N, device=dev) for _ in range(4)]
        spec = [torch.fft.rfft2(im, s=(G, G)) for im in imgs]
        rows_c = [torch.randn(1024, G, device=dev, dtype=torch.complex64) for _ in range(8)]
        lc = {}
        for label, fn in (("rfft2_zero_padded_N_to_G", lambda i: torch.fft.rfft2(imgs[i % 4], s=(G, G))),
                          ("irfft2_G", lambda i: torch.fft.irfft2(spec[i % 4], s=(G, G))),
                          ("fft_1024_contiguous_rows_of_G", lambda i: torch.fft.fft(rows_c[i % 8], dim=1))):
            for i in range(3):
                fn(i)
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record()
            for i in range(20):
                fn(i)
            e1.record()
            torch.cuda.synchronize()
            lc[label] = round(e0.elapsed_time(e1) / 20 * 1e3, 1)
        lc["this_library_us"] = {"F1+F2 (de-apodise, pad, 2-D FFT, Hermitian half)": round(per_stage["F1_colfft"]["us_per_launch"] + per_stage["F2_rowfft"]["us_per_launch"], 1),
                                 "A3+A4 (2-D inverse FFT, crop, de-apodise)": round(per_stage["A3_rowifft"]["us_per_launch"] + per_stage["A4_colifft"]["us_per_launch"], 1),
                                 "one column pass = 1024 FFTs of length G on column pairs": per_stage["F1_colfft"]["us_per_launch"]}
        lc["note"] = "cuFFT via torch.fft, us per call; a yardstick for the FFT passes, not used by the library"
        library_context = lc
        del imgs, spec, rows_c
    cpu_baseline = None
    if not args.no_cpu_baseline and world == 1:
        v, cores, dt = cpu_oracle_pairs_per_s(cfg, args.ref_sample)
        cpu_baseline = {"value": v, "unit": UNIT, "cores": cores, "kind": "oracle",
                        "sample": f"{args.ref_sample} sinogram entries + {args.ref_sample} pixels of one slice "
                                  f"({dt:.1f} s of CPU work), closed-form O-direct, extrapolated linearly to M and N^2 outputs"}
    t_pair_us = t_ms * 1e3 / (B * args.steps)
    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
        "warmup": max(args.warmup, 3), "ms_per_step": t_ms / args.steps, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "f32", "data": "synthetic",
        "config": {"workload": WORKLOAD, "slices_per_step_per_gpu": B, "parallelism": f"slice-parallel replicas x{world}",
                   "l2": f"inputs {B * cfg.N * cfg.N * 4 / 1e6:.0f} MB/step cycle through HBM (> 126 MB L2); per-slice grid 134 MB > L2"},
        "samples_per_s": 2.0 * cfg.M * value, "us_per_pair": t_pair_us,
        "e2e": e2e, "gpu_launches": int(launches), "clocks": clocks,
        "plan": {"plan_create_ms": round(plan_create_ms, 1), "first_plan_of_the_process_ms_config1": round(first_plan_ms, 1), "schedules_ms": round(plan.schedule_check(True, verify=False)[2], 1),
                 "schedules_built_on_device": bool(plan.schedule_check(True, verify=False)[1]), "plan_device_bytes": int(plan.workspace_bytes),
                 "plan_device_bytes_after_run": int(plan.device_bytes()),
                 "note": "radon_plan_create: tables + schedules (CUDA kernels, plan_device.cu) + first workspace; the batched calls "
                         "add three more workspaces on first use"},
        "roofline": roofline, "stages": per_stage, "gridding_kernels": gk, "paper_shape": paper_shape, "next_rows": next_rows,
        "library_context": library_context, "cpu_baseline": cpu_baseline,
    }
    print(json.dumps(line))
    return 0


if __name__ == "__main__":
    sys.exit(main())
