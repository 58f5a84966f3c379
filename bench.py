#!/usr/bin/env python
"""bench.py -- field samples/s of the sCWatter hot path on B200.

  python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--skip-large]

A step is one pass of the grid hot path (mode weights -> spectral assembly -> twiddles -> separable
synthesis, batched over layers by scw_sweep_wavelengths = a-7) over
BASELINE.json's config 1 in complex64: 33x33 frequencies, 4 layers x 64 planes, 256x256 grid
= 16 777 216 field samples per step.  The point path (a-5, config 3) and the spectroscopy sweep
(config 4) are timed as well and reported under "extra".  Inputs are seeded synthetic
(scw_inputs.py), resident in HBM for `value`, and in pinned host memory for `e2e`.
Multi-GPU: the path has no exchange step ("replicas only"): under torchrun every rank runs the same
workload on its own GPU; value = N * samples / max-over-ranks time.
--impl reference times the fp64 CPU oracle (oracle/) on a bounded sample of the same workload.
"""
import argparse
import json
import os
import statistics
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

import numpy as np  # noqa: E402

import scw_inputs as si  # noqa: E402

METRIC = "field samples/s (complex E 3-vectors)"
UNIT = "samples/s"
FP32_PEAK_TFLOPS = 148 * 128 * 2 * 1.965e9 / 1e12      # CUDA-core FFMA peak at max clock (context only)
FP64_DMMA_PEAK_TFLOPS = 37.1                           # measured on this pool's B200 (DMMA microbenchmark)


# ------------------------------------------------------------------------------------------------
def measured_peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        d = json.load(open(path))
        return dict(hbm_gbs=d["hbm_gbs"], bf16_tflops=d["bf16_tflops"],
                    bf16_tflops_sustained=d.get("bf16_tflops_sustained", d["bf16_tflops"]), source="measured")
    return dict(hbm_gbs=6650.0, bf16_tflops=1590.0, bf16_tflops_sustained=1400.0, source="fallback")


class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled during the timed region (B200_PROFILING.md recipe)."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index=0):
        self.rows, self.proc, self.thread, self.index = [], None, None, index

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", f"--id={self.index}", f"--query-gpu={self.Q}",
                                          "--format=csv,noheader,nounits", "-lms", "100"],
                                         stdout=subprocess.PIPE, stderr=subprocess.STDOUT, text=True)
        except OSError:
            return
        self.thread = threading.Thread(target=lambda: [self.rows.append(l) for l in self.proc.stdout], daemon=True)
        self.thread.start()

    def stop(self):
        if not self.proc:
            return dict(sm_mhz=None, sm_max_mhz=None, reasons=["nvidia-smi unavailable"])
        self.proc.terminate()
        self.thread.join(timeout=2)
        sm, smax, reasons = [], [], set()
        for line in self.rows:
            f = [t.strip() for t in line.split(",")]
            if len(f) < 7:
                continue
            try:
                sm.append(float(f[0]))
                smax.append(float(f[1]))
            except ValueError:
                continue
            for name, v in zip(("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"), f[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(name)
        busy = [c for c in sm if c > 0.5 * max(smax or [1])] or sm
        return dict(sm_mhz=statistics.median(busy) if busy else None, sm_max_mhz=max(smax) if smax else None,
                    reasons=sorted(reasons), samples=len(sm))


def dist_setup(n_gpus):
    """Rendezvous for N > 1 (torchrun env); returns (rank, world, local_rank, torch.distributed or None)."""
    world = int(os.environ.get("WORLD_SIZE", "1"))
    if world == 1:
        return 0, 1, 0, None
    import torch
    import torch.distributed as dist
    backend = "nccl" if torch.cuda.is_available() else "gloo"
    dist.init_process_group(backend=backend)
    return dist.get_rank(), world, int(os.environ.get("LOCAL_RANK", "0")), dist


def max_over_ranks(ms, dist):
    """Timing plumbing only: the slowest rank defines the step time (no data-path collective)."""
    if dist is None:
        return ms
    import torch
    t = torch.tensor([ms], dtype=torch.float64, device="cuda" if dist.get_backend() == "nccl" else "cpu")
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def barrier(dist):
    if dist is not None:
        dist.barrier()


# ------------------------------------------------------------------------------------------------
def config1_inputs(dtype=np.complex64):
    cfg = si.CONFIGS[1]
    layers = [si.make_layer(cfg, l, dtype=dtype) for l in range(cfg.n_layers)]
    zs = [si.grid_coords(cfg, l)[2] for l in range(cfg.n_layers)]
    x, y, _ = si.grid_coords(cfg, 0)
    return cfg, layers, zs, x, y


def time_steps(torch, fn, steps, warmup, dist=None):
    for _ in range(warmup):
        fn()
    torch.cuda.synchronize()
    barrier(dist)
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    for _ in range(steps):
        fn()
    e1.record()
    torch.cuda.synchronize()
    barrier(dist)
    return max_over_ranks(e0.elapsed_time(e1) / steps, dist)


def kernel_rooflines(prof, steps, cfg, dtype_bytes, peaks):
    """Per-kernel algorithmic bytes / flops per launch for config 1 (one launch = one layer), DESIGN.md table."""
    M = cfg.U * cfg.Vn
    R, J, Fz, Nx, Ny = 3 * M, 4 * M, cfg.planes, cfg.Nx, cfg.Ny
    es = dtype_bytes
    alg = {
        "simt_assemble": dict(bytes=R * J * es + J * Fz * es + R * Fz * es, flops=8 * R * J * Fz),
        "tc_assemble": dict(bytes=R * J * es + J * Fz * es + R * Fz * es, flops=8 * R * J * Fz),
        "simt_synth_a": dict(bytes=R * Fz * es + 3 * Fz * cfg.U * Ny * es, flops=8 * 3 * Fz * M * Ny),
        "simt_synth_b": dict(bytes=3 * Fz * Nx * Ny * es + 3 * Fz * cfg.U * Ny * es, flops=8 * 3 * Fz * Nx * cfg.U * Ny),
        "tc_synth": dict(bytes=3 * Fz * Nx * Ny * es + R * Fz * es, flops=8 * 3 * Fz * (M * Ny + Nx * cfg.U * Ny)),
    }
    traffic = {}
    tpath = os.path.join(ROOT, "profiles", "dram_traffic.json")
    if os.path.exists(tpath):
        traffic = json.load(open(tpath))
    out = {}
    total = sum(ms for ms, _ in prof.values()) or 1.0
    for name, (ms, n) in prof.items():
        per = ms / n
        k = dict(ms_per_launch=per, launches_per_step=n / steps, share=ms / total)
        if name in alg:
            # a grouped launch covers several layers: units per launch = layers per step / launches per step
            units = cfg.n_layers / (n / steps)
            nbytes, flops = alg[name]["bytes"] * units, alg[name]["flops"] * units
            gbs = nbytes / (per * 1e-3) / 1e9
            k.update(bound="hbm", achieved=gbs, peak=peaks["hbm_gbs"], unit="GB/s", frac=gbs / peaks["hbm_gbs"],
                     traffic=traffic.get(name), layers_per_launch=units, alg_bytes=nbytes,
                     useful_tflops=flops / (per * 1e-3) / 1e12)
            if name.startswith("tc_"):
                # BF16x3: three bf16 products per real product; sustained measured bf16 peak (kernel inside a step)
                ex = 3 * flops / (per * 1e-3) / 1e12
                k.update(executed_bf16_tflops=ex, tensor_frac=ex / peaks["bf16_tflops_sustained"])
        out[name] = k
    return out


def run_ours(args):
    import torch

    import paper_2404_07293_b200 as scw
    rank, world, local_rank, dist = dist_setup(args.gpus)
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: there is no CPU fallback (use --impl reference for the oracle)")
    torch.cuda.set_device(local_rank)
    device = torch.device("cuda", local_rank)
    scw.lib()
    peaks = measured_peaks()
    dev = lambda a: torch.from_numpy(np.ascontiguousarray(a)).to(device)

    cfg, layers, zs, x, y = config1_inputs(np.complex64)
    ctx = scw.Context(local_rank)
    Ls = [scw.Layer.from_numpy(d, device) for d in layers]
    dz, dx, dy = [dev(z) for z in zs], dev(x), dev(y)
    out = [torch.empty((cfg.planes, 3, cfg.Ny, cfg.Nx), dtype=torch.complex64, device=device) for _ in Ls]
    samples = cfg.n_layers * cfg.planes * cfg.Nx * cfg.Ny
    step = lambda: scw.scw_sweep_wavelengths(ctx, Ls, dz, dx, dy, out=out)

    # ---- value: inputs resident in HBM
    step()
    torch.cuda.synchronize()
    n0 = ctx.launch_count()
    sampler = ClockSampler(local_rank)
    sampler.start()
    t_wait = time.perf_counter()
    while not sampler.rows and time.perf_counter() - t_wait < 3.0:   # nvidia-smi needs ~0.3 s to start
        time.sleep(0.05)
    ms = time_steps(torch, step, args.steps, args.warmup, dist)
    launches = (ctx.launch_count() - n0) // (args.steps + args.warmup)
    # the timed region lasts a few ms: keep the identical step running ~0.7 s so the 100 ms sampler sees it
    t_hold = time.perf_counter()
    while time.perf_counter() - t_hold < 0.7:
        step()
        torch.cuda.synchronize()
    clocks = sampler.stop()
    clocks["window"] = "warm-up + timed steps + 0.7 s of the identical step"
    value = world * samples / (ms * 1e-3)

    # ---- per-kernel device timers over a second pass of the same K steps
    ctx.set_profile(True)
    for _ in range(args.steps):
        step()
    torch.cuda.synchronize()
    prof = ctx.profile()
    ctx.set_profile(False)
    kernels = kernel_rooflines(prof, args.steps, cfg, 8, peaks)
    dominant = max((k for k in kernels if "frac" in kernels[k]), key=lambda k: kernels[k]["share"])
    roof = {k: kernels[dominant][k] for k in ("bound", "achieved", "peak", "unit", "frac", "traffic")}
    roof.update(kernel=dominant, share_of_step=kernels[dominant]["share"], peak_source=peaks["source"],
                alg_bytes_per_launch=kernels[dominant]["alg_bytes"])

    # ---- e2e: the same step through the host-buffer C-ABI call (pinned host memory, H2D + D2H inside)
    pin = lambda a: torch.from_numpy(np.ascontiguousarray(a)).pin_memory()
    Lh = [scw.Layer(U=d["U"], Vn=d["Vn"], X=d["X"], Y=d["Y"], lam=d["lam"], z_lo=d["z_lo"], z_hi=d["z_hi"],
                    V=pin(d["V"]), gamma=pin(d["gamma"]), c=pin(d["c"]), dir=pin(d["dir"])) for d in layers]
    hz, hx, hy = [pin(z) for z in zs], pin(x), pin(y)
    hout = [torch.empty((cfg.planes, 3, cfg.Ny, cfg.Nx), dtype=torch.complex64).pin_memory() for _ in Lh]
    io = {}

    def host_step():
        _, io["up"], io["down"] = scw.scw_sweep_wavelengths_host(ctx, Lh, hz, hx, hy, out=hout)

    e2e = None
    if not args.quick:
        ms_e2e = time_steps(torch, host_step, max(2, args.steps // 2), 1, dist)
        e2e = dict(value=world * samples / (ms_e2e * 1e-3), unit=UNIT, ms_per_step=ms_e2e,
                   h2d_bytes_per_step=io["up"], d2h_bytes_per_step=io["down"])
        dev_host = float((hout[0] - out[0].cpu()).abs().max() / hout[0].abs().max())
        assert dev_host <= 5e-5, f"host-buffer path disagrees with the device path: {dev_host:.3e}"

    extra = {}
    if rank == 0 and not args.quick:
        extra = extra_workloads(torch, scw, ctx, device, args, peaks)

    cpu = None
    if rank == 0 and world == 1 and not args.no_cpu and not args.quick:
        cpu = cpu_baseline(layers[0], x, y, zs[0], cfg)

    if rank == 0:
        line = dict(metric=METRIC, value=value, unit=UNIT, n_gpus=world, steps=args.steps, warmup=args.warmup,
                    ms_per_step=ms, higher_is_better=True, scaling="weak", vs_baseline=None, dtype="c64 (fp32)",
                    data="synthetic",
                    config=dict(workload="BASELINE.json configs[1]: 33x33 frequencies (M=1089, J=4356), 4 layers x 64 "
                                "planes, 256x256 grid, complex64, one scw_sweep_wavelengths call per step",
                                samples_per_step=samples, parallelism=f"replicas x{world}",
                                cache="inputs (457 MB of V) + outputs (403 MB) per step exceed the 126 MB L2"),
                    clocks=clocks, e2e=e2e, gpu_launches=int(launches) * args.steps, gpu_launches_per_step=int(launches),
                    roofline=roof, kernels=kernels, cpu_baseline=cpu, extra=extra, peaks=peaks)
        print(json.dumps(line))
    if dist is not None:
        dist.destroy_process_group()


def extra_workloads(torch, scw, ctx, device, args, peaks):
    """Configs 3 (point path), 4 (sweep, detector), exterior field, 2, 1 complex128 and 3' at full size."""
    dev = lambda a: torch.from_numpy(np.ascontiguousarray(a)).to(device)
    extra = {}
    # config 3: 4e6 scattered points x 4356 plane waves
    c3 = si.CONFIGS[3]
    pw = scw.PlaneWaves.from_numpy(si.make_planewaves(c3), device)
    pts = dev(si.make_points(c3))
    outp = torch.empty((pts.shape[0], 3), dtype=torch.complex64, device=device)
    ms = time_steps(torch, lambda: scw.scw_eval_points(ctx, pw, pts, out=outp), args.steps, args.warmup)
    terms = pts.shape[0] * 4356
    sfu_peak = 148 * 16 * 1.965e9 / 3                      # terms/s if 3 MUFU ops per term saturate the XU pipe
    extra["config3_points"] = dict(ms_per_call=ms, points_per_s=pts.shape[0] / (ms * 1e-3), terms_per_s=terms / (ms * 1e-3),
                                   roofline=dict(bound="alu", achieved=terms / (ms * 1e-3) / 1e9, peak=sfu_peak / 1e9,
                                                 unit="Gterm/s (3 MUFU/term at 16/clk/SM, 148 SMs, 1965 MHz)",
                                                 frac=terms / (ms * 1e-3) / sfu_peak, traffic=None))
    del pts, outp
    # config 4: 32 wavelengths x 2 layers, one call
    c4 = si.CONFIGS[4]
    x, y, _ = si.grid_coords(c4, 0)
    Ls, zs = [], []
    for li in range(len(c4.lams)):
        for l in range(c4.n_layers):
            Ls.append(scw.Layer.from_numpy(si.make_layer(c4, l, li, dtype=np.complex64), device))
            zs.append(dev(si.grid_coords(c4, l)[2]))
    out = [torch.empty((c4.planes, 3, c4.Ny, c4.Nx), dtype=torch.complex64, device=device) for _ in Ls]
    dx, dy = dev(x), dev(y)
    ms = time_steps(torch, lambda: scw.scw_sweep_wavelengths(ctx, Ls, zs, dx, dy, out=out), args.steps, args.warmup)
    n4 = len(Ls) * c4.planes * c4.Nx * c4.Ny
    ebytes = n4 * 24
    extra["config4_sweep"] = dict(ms_per_call=ms, samples_per_s=n4 / (ms * 1e-3),
                                  hbm_write_frac=ebytes / (ms * 1e-3) / 1e9 / peaks["hbm_gbs"])
    # NEXT-3 detector: the same sweep with I = sum_comp |E_comp|^2 reduced in the synthesis epilogue (E never written)
    outI = [torch.empty((c4.planes, c4.Ny, c4.Nx), dtype=torch.float32, device=device) for _ in Ls]
    ms = time_steps(torch, lambda: scw.scw_sweep_intensity(ctx, Ls, zs, dx, dy, out=outI), args.steps, args.warmup)
    extra["config4_sweep_intensity"] = dict(ms_per_call=ms, samples_per_s=n4 / (ms * 1e-3),
                                            speedup_vs_complex_field=extra["config4_sweep"]["ms_per_call"] / ms)
    del Ls, zs, out, outI
    torch.cuda.empty_cache()
    # NEXT-1 exterior field (eq. 9-10): the paper's Table 2 shape (M = 2500 orders, one 256 x 256 plane below the
    # sample; 142 s on one i9 core, 0.29 s on an RTX 3090) and a config-1-shaped volume above it
    for name, cfgx, side, planes in (("exterior_table2_plane", si.Config(5, "table 2 exterior", 50, 50, 32.0, (1.0,), 1, 1,
                                                                          256, 256, (np.complex64,)), 1, 1),
                                     ("exterior_volume_33x33", si.CONFIGS[1], 0, 64)):
        ext = si.make_exterior(cfgx, side, dtype=np.complex64)
        X = scw.Exterior.from_numpy(ext, device)
        xg, yg, _ = si.grid_coords(cfgx, 0)
        d = np.linspace(0.0, 3.0, planes)
        zg = dev(ext["z_face"] - d if side == 0 else ext["z_face"] + d)
        dxg, dyg = dev(xg), dev(yg)
        Pbuf = torch.empty((planes, 3 * cfgx.U * cfgx.Vn), dtype=torch.complex64, device=device)
        Eo = torch.empty((planes, 3, cfgx.Ny, cfgx.Nx), dtype=torch.complex64, device=device)

        def ext_step():
            scw.scw_exterior_spectra(ctx, X, zg, out=Pbuf)
            scw.scw_synthesize_grid(ctx, U=cfgx.U, Vn=cfgx.Vn, X=ext["X"], Y=ext["Y"], P=Pbuf, x=dxg, y=dyg, out=Eo)

        ms = time_steps(torch, ext_step, args.steps, args.warmup)
        ns = planes * cfgx.Nx * cfgx.Ny
        extra[name] = dict(ms_per_call=ms, samples_per_s=ns / (ms * 1e-3), orders=cfgx.U * cfgx.Vn, planes=planes,
                           hbm_write_frac=ns * 24 / (ms * 1e-3) / 1e9 / peaks["hbm_gbs"])
    if not args.skip_large:
        c1, layers, zs1, x1, y1 = config1_inputs(np.complex128)
        Ls = [scw.Layer.from_numpy(d, device) for d in layers]
        out = [torch.empty((c1.planes, 3, c1.Ny, c1.Nx), dtype=torch.complex128, device=device) for _ in Ls]
        dz, dx, dy = [dev(z) for z in zs1], dev(x1), dev(y1)
        ms = time_steps(torch, lambda: scw.scw_sweep_wavelengths(ctx, Ls, dz, dx, dy, out=out), max(2, args.steps // 2), 2)
        M1 = c1.U * c1.Vn
        gf = c1.n_layers * (8 * 3 * M1 * 4 * M1 * c1.planes + 8 * 3 * c1.planes * (M1 * c1.Ny + c1.Nx * c1.U * c1.Ny)) / 1e9
        extra["config1_c128"] = dict(ms_per_call=ms, samples_per_s=c1.n_layers * c1.planes * c1.Nx * c1.Ny / (ms * 1e-3),
                                     roofline=dict(bound="tensor", achieved=gf / ms, peak=FP64_DMMA_PEAK_TFLOPS,
                                                   unit="TFLOP/s (useful fp64, 8 per complex MAC; the 3M kernel executes 6; peak = "
                                                        "measured mma.sync m8n8k4 f64 rate, DESIGN.md 5)",
                                                   frac=gf / ms / FP64_DMMA_PEAK_TFLOPS, traffic=None))
        del Ls, out, layers
        torch.cuda.empty_cache()
        c2 = si.CONFIGS[2]
        x2, y2, _ = si.grid_coords(c2, 0)
        Ls = [scw.Layer.from_numpy(si.make_layer(c2, l, dtype=np.complex64), device) for l in range(c2.n_layers)]
        dz = [dev(si.grid_coords(c2, l)[2]) for l in range(c2.n_layers)]
        out = [torch.empty((c2.planes, 3, c2.Ny, c2.Nx), dtype=torch.complex64, device=device) for _ in Ls]
        dx, dy = dev(x2), dev(y2)
        ms = time_steps(torch, lambda: scw.scw_sweep_wavelengths(ctx, Ls, dz, dx, dy, out=out), max(2, args.steps // 2), 2)
        n2 = c2.n_layers * c2.planes * c2.Nx * c2.Ny
        vbytes = sum(l.V.numel() * 8 for l in Ls)
        extra["config2_large"] = dict(ms_per_call=ms, samples_per_s=n2 / (ms * 1e-3),
                                      hbm_frac_V_plus_E=(vbytes + n2 * 24) / (ms * 1e-3) / 1e9 / peaks["hbm_gbs"])
        del Ls, out
        torch.cuda.empty_cache()
        lay = scw.Layer.from_numpy(si.make_layer(c3, dtype=np.complex64), device)
        pts = dev(si.make_points(c3, n=65536))
        ms = time_steps(torch, lambda: scw.scw_eval_points(ctx, lay, pts), 2, 1)
        extra["config3_dense_points"] = dict(ms_per_call=ms, points_per_s=65536 / (ms * 1e-3))
    return extra


def cpu_baseline(layer, x, y, z, cfg, budget_s=15.0):
    """The oracle as it stands (Tier A triple loop) on a bounded seeded sample of config 1, host cores."""
    import oracle
    n_total = cfg.planes * cfg.Ny * cfg.Nx
    idx = si.sample_subset(cfg, n_total, 4096)
    iz, iy, ix = np.unravel_index(idx, (cfg.planes, cfg.Ny, cfg.Nx))
    xyz = np.column_stack([x[ix], y[iy], z[iz]])
    cores = oracle.threads()
    t0 = time.perf_counter()
    oracle.layer_samples(xyz=xyz[:cores], **layer)
    probe = time.perf_counter() - t0
    n = int(max(cores, min(len(xyz), budget_s / max(probe, 1e-6) * cores)))
    n -= n % cores
    t0 = time.perf_counter()
    oracle.layer_samples(xyz=xyz[:n], **layer)
    dt = time.perf_counter() - t0
    return dict(value=n / dt, unit=UNIT, cores=cores, kind="oracle",
                sample=f"{n} seeded samples of config 1 layer 0 (Tier A: 3*M*J = 14.2e6 complex terms per sample), {dt:.1f} s")


def run_reference(args):
    """--impl reference: the oracle timed on the host cores; each step is a bounded sample of config 1."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    import oracle
    cfg = si.CONFIGS[1]
    layer = si.make_layer(cfg, 0, dtype=np.complex64)
    x, y, z = si.grid_coords(cfg, 0)
    cores = oracle.threads()
    per_step = 2 * cores
    idx = si.sample_subset(cfg, cfg.planes * cfg.Ny * cfg.Nx, per_step * (args.steps + args.warmup))
    iz, iy, ix = np.unravel_index(idx, (cfg.planes, cfg.Ny, cfg.Nx))
    xyz = np.column_stack([x[ix], y[iy], z[iz]])
    for w in range(args.warmup):
        oracle.layer_samples(xyz=xyz[w * per_step:(w + 1) * per_step], **layer)
    t0 = time.perf_counter()
    for s in range(args.warmup, args.warmup + args.steps):
        oracle.layer_samples(xyz=xyz[s * per_step:(s + 1) * per_step], **layer)
    dt = (time.perf_counter() - t0) / args.steps
    value = per_step / dt
    sample = f"{per_step} seeded samples of config 1 layer 0 per step (Tier A triple loop)"
    print(json.dumps(dict(impl="reference", metric=METRIC, value=value, unit=UNIT, n_gpus=args.gpus, steps=args.steps,
                          warmup=args.warmup, ms_per_step=dt * 1e3, higher_is_better=True, scaling="weak",
                          vs_baseline=None, dtype="f64", data="synthetic",
                          config=dict(workload="BASELINE.json configs[1] (33x33 frequencies, 4 layers x 64 planes, "
                                      "256x256 grid); bounded sample per step", samples_per_step=per_step),
                          cpu_baseline=dict(value=value, unit=UNIT, cores=cores, kind="oracle", sample=sample),
                          e2e=dict(value=value, unit=UNIT, h2d_bytes_per_step=0, d2h_bytes_per_step=0),
                          gpu_launches=0)))


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--all", action="store_true", help="(default now) also time config 2, config 1 complex128, config 3'")
    ap.add_argument("--skip-large", action="store_true", help="skip config 2, config 1 complex128 and config 3' (extra)")
    ap.add_argument("--no-cpu", action="store_true", help="skip the cpu_baseline leg")
    ap.add_argument("--quick", action="store_true", help="only the resident-input step (for ncu captures)")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3) if args.impl == "ours" else args.warmup
    if args.impl == "reference":
        run_reference(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
