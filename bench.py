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


# ------------------------------------------------------------------------------------------------
def measured_peaks(ctx=None):
    """Roofline denominators: MEASURED_PEAKS.json (driver-written: HBM copy, dense bf16) plus the library's own
    microbenchmarks run on this device right now (scw_measure_peak: FP64 DMMA, FP32 FMA, MUFU, HBM read / write streams)."""
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        d = json.load(open(path))
        out = dict(hbm_gbs=d["hbm_gbs"], bf16_tflops=d["bf16_tflops"],
                   bf16_tflops_sustained=d.get("bf16_tflops_sustained", d["bf16_tflops"]), source="measured")
    else:
        out = dict(hbm_gbs=6650.0, bf16_tflops=1590.0, bf16_tflops_sustained=1400.0, source="fallback")
    if ctx is not None:
        out.update(ctx.measure_peaks(reps=5))
        out["microbenchmarks"] = "scw_measure_peak (csrc/scw_peaks.cu), best of 5 launches each, run before the timed step"
    return out


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


def time_each(torch, fn, n=20):
    """n individually timed calls (an event pair each, back to back): best and median, SURVEY 8(d) "Timing"."""
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(n)]
    for a, b in ev:
        a.record()
        fn()
        b.record()
    torch.cuda.synchronize()
    t = sorted(a.elapsed_time(b) for a, b in ev)
    return dict(best_ms=t[0], median_ms=t[len(t) // 2], n=n)


def sweep_shape(cfg, n_inst):
    """Sizes of one grouped sweep: n_inst (wavelength, layer) instances of cfg's shape."""
    M = cfg.U * cfg.Vn
    pad16 = lambda v: (v + 15) // 16 * 16
    chunks = lambda nf: (2 * nf + 79) // 80                          # frequency chunks of the synthesis (K <= 80)
    nuc, nvc = chunks(cfg.U), chunks(cfg.Vn)
    K2p, K1p = pad16(2 * -(-cfg.U // nuc)), pad16(2 * -(-cfg.Vn // nvc))
    tiles = -(-cfg.Nx // 128) * -(-cfg.Ny // 128)
    return dict(M=M, R=3 * M, J=4 * M, Fz=cfg.planes, Nx=cfg.Nx, Ny=cfg.Ny, U=cfg.U, Vn=cfg.Vn, n_inst=n_inst,
                # executed tensor flops of the synthesis per plane and 128 x 128 tile: GEMM1 (M = 128, N = K2p, K = K1p per
                # v chunk) for every u chunk, GEMM2 (two 64-y halves, N = 128, K = K2p) per u chunk; three bf16 products each
                synth_exec_per_plane_tile=3 * 2 * 128 * (nuc * nvc * K2p * K1p + nuc * 128 * K2p), tiles=tiles)


def kernel_rooflines(prof, steps, sh, peaks, traffic=None):
    """Per-kernel algorithmic bytes / flops per launch of a grouped complex64 sweep (bytes per unit), against
    BOTH rooflines: HBM (measured copy peak) and bf16 tensor (sustained measured peak; useful and executed flops)."""
    es = 8
    R, J, Fz, Nx, Ny, M, U, n = sh["R"], sh["J"], sh["Fz"], sh["Nx"], sh["Ny"], sh["M"], sh["U"], sh["n_inst"]
    alg = {
        # fused a-1 + a-2 (+ fix-up into the synthesis images): read V once, read c / gamma / z, spectra stay on chip / in L2
        "tc_assemble": dict(bytes=n * (R * J * es + J * (es + 17) + Fz * 8), flops=n * 8 * R * J * Fz,
                            executed=n * 3 * 8 * R * J * Fz),
        "simt_assemble": dict(bytes=n * (R * J * es + J * Fz * es + R * Fz * es), flops=n * 8 * R * J * Fz, executed=None),
        # a-4: write E once (the spectrum images are L2-resident)
        "tc_synth": dict(bytes=n * 3 * Fz * Nx * Ny * es, flops=n * 8 * 3 * Fz * (M * Ny + Nx * U * Ny),
                         executed=n * 3 * Fz * sh["tiles"] * sh["synth_exec_per_plane_tile"]),
    }
    traffic = traffic or {}
    out = {}
    total = sum(ms for ms, _ in prof.values()) or 1.0
    for name, (ms, cnt) in prof.items():
        per = ms / cnt
        launches = cnt / steps
        k = dict(ms_per_launch=per, launches_per_step=launches, share=ms / total)
        if name in alg:
            a = alg[name]
            nbytes, flops = a["bytes"] / launches, a["flops"] / launches
            gbs = nbytes / (per * 1e-3) / 1e9
            k.update(alg_bytes=nbytes, hbm_gbs=gbs, hbm_frac=gbs / peaks["hbm_gbs"],
                     useful_tflops=flops / (per * 1e-3) / 1e12, traffic=traffic.get(name))
            if a["executed"]:
                ex = a["executed"] / launches / (per * 1e-3) / 1e12
                # against BOTH measured bf16 peaks: `sustained` (a long cuBLAS run, clocks settled under the power cap) is
                # the denominator for a kernel timed inside a long step; `burst` (a short run at boost clocks) is the
                # harsher one and the right one for a kernel that runs alone for ~100 us
                k.update(executed_bf16_tflops=ex, tensor_frac_executed=ex / peaks["bf16_tflops_sustained"],
                         tensor_frac_useful=k["useful_tflops"] / peaks["bf16_tflops_sustained"],
                         tensor_frac_executed_burst=ex / peaks["bf16_tflops"],
                         tensor_frac_useful_burst=k["useful_tflops"] / peaks["bf16_tflops"])
                k["binding"] = "hbm" if k["hbm_frac"] >= k["tensor_frac_executed"] else "tensor"
            else:
                k["binding"] = "hbm"
        out[name] = k
    return out


def dominant_roofline(kernels, peaks):
    """The `roofline` object of the JSON line for the kernel with the largest share of the step."""
    dom = max((k for k in kernels if "hbm_frac" in kernels[k]), key=lambda k: kernels[k]["share"])
    k = kernels[dom]
    if k["binding"] == "tensor":
        roof = dict(bound="tensor", achieved=k["executed_bf16_tflops"], peak=peaks["bf16_tflops_sustained"], unit="TFLOP/s",
                    frac=k["tensor_frac_executed"])
    else:
        roof = dict(bound="hbm", achieved=k["hbm_gbs"], peak=peaks["hbm_gbs"], unit="GB/s", frac=k["hbm_frac"])
    roof.update(traffic=k.get("traffic"), kernel=dom, share_of_step=k["share"], alg_bytes_per_launch=k["alg_bytes"],
                ms_per_launch=k["ms_per_launch"], peak_source=peaks["source"])
    return roof


def profile_sweep_events(torch, ctx, step, steps):
    """Per-kernel device milliseconds over `steps` further calls with a CUDA event between consecutive kernels (the
    library's event timers).  The events serialise the launches: the programmatic overlap of a kernel's prologue with its
    predecessor's tail is lost, so these intervals add up to MORE than the plain step."""
    ctx.set_profile(True)
    for _ in range(steps):
        step()
    torch.cuda.synchronize()
    prof = ctx.profile()
    ctx.set_profile(False)
    return prof


def profile_from_ring(ctx, steps):
    """{kernel: (ms over the steps, launches)}, steps covered: the device-clock intervals of the LAST `steps` sweep calls,
    read from the ring every tensor-core sweep kernel stamps with the globaltimer of its last CTA's exit
    (scw_profile_timeline).  A kernel's interval runs from the end of its predecessor in the stream to its own end, so the
    intervals add up to the CUDA-event time of the same steps, and nothing sits between the kernels (a CUDA event between
    two launches would undo their programmatic overlap).  Call it right after the timed loop: it reads, it runs nothing."""
    tl = ctx.kernel_timeline()
    names = [name for _, name in tl]
    if "tc_assemble" not in names:
        return {}, 0
    per_step = names[::-1].index("tc_assemble") + 1               # a step's launches: from its assembly to its last synthesis
    use = min(steps, (len(tl) - 1) // per_step) * per_step
    prof = {}
    for i in range(len(tl) - use, len(tl)):
        ms = (tl[i][0] - tl[i - 1][0]) * 1e-6
        a = prof.get(tl[i][1], (0.0, 0))
        prof[tl[i][1]] = (a[0] + ms, a[1] + 1)
    return prof, use // per_step


def load_traffic():
    path = os.path.join(ROOT, "profiles", "dram_traffic.json")
    return json.load(open(path)) if os.path.exists(path) else {}


def run_ours(args):
    import torch

    import paper_2404_07293_b200 as scw
    rank, world, local_rank, dist = dist_setup(args.gpus)
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: there is no CPU fallback (use --impl reference for the oracle)")
    torch.cuda.set_device(local_rank)
    device = torch.device("cuda", local_rank)
    scw.lib()
    dev = lambda a: torch.from_numpy(np.ascontiguousarray(a)).to(device)

    cfg, layers, zs, x, y = config1_inputs(np.complex64)
    ctx = scw.Context(local_rank)
    peaks = measured_peaks(None if args.quick else ctx)
    Ls = [scw.Layer.from_numpy(d, device) for d in layers]
    dz, dx, dy = [dev(z) for z in zs], dev(x), dev(y)
    out = [torch.empty((cfg.planes, 3, cfg.Ny, cfg.Nx), dtype=torch.complex64, device=device) for _ in Ls]
    samples = cfg.n_layers * cfg.planes * cfg.Nx * cfg.Ny
    # two output sets used alternately: a step never overwrites lines of its predecessor that are still dirty in the
    # 126 MB L2 (re-using one set would let those lines be overwritten in place and never reach the DRAM)
    outs = (out, [torch.empty_like(o) for o in out])
    n_calls = [0]

    def step():
        n_calls[0] += 1
        return scw.scw_sweep_wavelengths(ctx, Ls, dz, dx, dy, out=outs[n_calls[0] & 1])

    # ---- set-up (untimed, once per context): twiddle cache on (x, y do not change between steps) and the stream-K split
    # of the assembly calibrated on this very sweep (scw_calibrate: 3 rounds of 6 sweeps)
    ctx.set_cache(True)
    scw.scw_calibrate(ctx, Ls, dz, dx, dy, out=out, reps=5)

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
    prof, nsteps = profile_from_ring(ctx, max(1, min(args.steps, 60) - 1))  # the kernels of these timed steps (bar the first, whose
                                                                     # assembly interval holds the host's launch latency)
    launches = (ctx.launch_count() - n0) // (args.steps + args.warmup)
    each = time_each(torch, step, max(20, args.steps))
    # the timed region lasts a few ms: keep the identical step running ~0.7 s so the 100 ms sampler sees it
    t_hold = time.perf_counter()
    while time.perf_counter() - t_hold < 0.7:
        step()
        torch.cuda.synchronize()
    clocks = sampler.stop()
    clocks["window"] = "warm-up + timed steps + 0.7 s of the identical step"
    value = world * samples / (ms * 1e-3)

    # ---- per-kernel device timers over a second pass of the same K steps
    # per kernel: device clock inside the timed steps above (sums to their CUDA-event time); then a further pass with a
    # CUDA event between the kernels
    kernels = kernel_rooflines(prof, nsteps, sweep_shape(cfg, cfg.n_layers), peaks, load_traffic())
    roof = dominant_roofline(kernels, peaks)
    roof["timing"] = ("device clock (globaltimer) inside the timed steps themselves: interval from the previous kernel's end "
                      "to this kernel's end (scw_profile_timeline), the intervals add up to ms_per_step; "
                      "`kernels_cuda_events` = a further pass with a CUDA event between the kernels, which removes their "
                      "programmatic overlap")
    ev = profile_sweep_events(torch, ctx, step, args.steps)
    kernels_ev = {k: dict(ms_per_launch=v["ms_per_launch"], hbm_frac=v.get("hbm_frac"))
                  for k, v in kernel_rooflines(ev, args.steps, sweep_shape(cfg, cfg.n_layers), peaks).items()}
    vbytes = sum(l.V.numel() * 8 for l in Ls)
    # where the fused assembly kernel's time goes: per-CTA timeline of its last launch (scw_profile_assembly)
    tl = np.array(ctx.assembly_timeline())
    asm_phases = None
    if len(tl):
        main, fix = tl[:, 2] - tl[:, 1], tl[:, 3] - tl[:, 2]
        asm_phases = dict(unit="us since the CTA's start, over the persistent CTAs of the last assembly launch",
                          weights_and_padding_done=dict(median=float(np.median(tl[:, 1])), max=float(tl[:, 1].max())),
                          main_loop=dict(min=float(main.min()), median=float(np.median(main)), max=float(main.max())),
                          fixup=dict(median=float(np.median(fix)), max=float(fix.max())),
                          exit=dict(min=float(tl[:, 3].min()), median=float(np.median(tl[:, 3])), max=float(tl[:, 3].max())),
                          main_loop_hbm_frac_at_median=vbytes / (float(np.median(main)) * 1e-6) / 1e9 / peaks["hbm_gbs"],
                          note="main loop = V streamed through TMA + tensor cores; its median is what the kernel would take "
                               "if every SM streamed at the same rate and the weight / fix-up phases were free")
    # ---- the same step WITHOUT the untimed set-up: a fresh ctx with no calibrated split, first with nothing cached (the
    # twiddle tables are rebuilt and the control block cleared every step: 3 launches), then with SCW_OPT_CACHE only
    value_cold = value_uncal = None
    if not args.quick:
        ctx2 = scw.Context(local_rank)
        step2 = lambda: scw.scw_sweep_wavelengths(ctx2, Ls, dz, dx, dy, out=outs[0])
        ms_cold = time_steps(torch, step2, args.steps, args.warmup, dist)
        ctx2.set_cache(True)
        ms_uncal = time_steps(torch, step2, args.steps, args.warmup, dist)
        ctx2.close()
        del ctx2
        value_cold = dict(value=world * samples / (ms_cold * 1e-3), ms_per_step=ms_cold,
                          note="no scw_calibrate, no SCW_OPT_CACHE: twiddle kernel + assembly + synthesis every step")
        value_uncal = dict(value=world * samples / (ms_uncal * 1e-3), ms_per_step=ms_uncal,
                           note="SCW_OPT_CACHE on, equal stream-K split (no scw_calibrate)")
    whole = dict(alg_bytes=vbytes + samples * 24, hbm_frac=(vbytes + samples * 24) / (ms * 1e-3) / 1e9 / peaks["hbm_gbs"],
                 note="V read once + E written once per step, over the step time: the step's HBM floor fraction")

    # ---- e2e: the same step through the host-buffer C-ABI call (pinned host memory, H2D + D2H inside)
    e2e = None
    if not args.quick:
        pin = lambda a: torch.from_numpy(np.ascontiguousarray(a)).pin_memory()
        Lh = [scw.Layer(U=d["U"], Vn=d["Vn"], X=d["X"], Y=d["Y"], lam=d["lam"], z_lo=d["z_lo"], z_hi=d["z_hi"],
                        V=pin(d["V"]), gamma=pin(d["gamma"]), c=pin(d["c"]), dir=pin(d["dir"])) for d in layers]
        hz, hx, hy = [pin(z) for z in zs], pin(x), pin(y)
        hout = [torch.empty((cfg.planes, 3, cfg.Ny, cfg.Nx), dtype=torch.complex64).pin_memory() for _ in Lh]
        io = {}

        def host_step():
            _, io["up"], io["down"] = scw.scw_sweep_wavelengths_host(ctx, Lh, hz, hx, hy, out=hout)

        ms_e2e = time_steps(torch, host_step, max(2, args.steps // 2), 1, dist)
        e2e = dict(value=world * samples / (ms_e2e * 1e-3), unit=UNIT, ms_per_step=ms_e2e,
                   h2d_bytes_per_step=io["up"], d2h_bytes_per_step=io["down"])
        dev_host = float((hout[0] - out[0].cpu()).abs().max() / hout[0].abs().max())
        assert dev_host <= 5e-5, f"host-buffer path disagrees with the device path: {dev_host:.3e}"
        del Lh, hout

    extra = {}
    if rank == 0 and not args.quick:
        extra = extra_workloads(torch, scw, ctx, device, args, peaks)

    cpu = None
    if rank == 0 and world == 1 and not args.no_cpu and not args.quick:
        cpu = cpu_baseline(layers[0], x, y, zs[0], cfg)

    if rank == 0:
        per_config = summarise_configs(ms, value / world, roof, extra)
        line = dict(metric=METRIC, value=value, unit=UNIT, n_gpus=world, steps=args.steps, warmup=args.warmup,
                    ms_per_step=ms, value_uncalibrated=value_uncal, value_cold=value_cold, per_config=per_config, step_ms_best=each["best_ms"], step_ms_median=each["median_ms"],
                    value_at_median=world * samples / (each["median_ms"] * 1e-3), individually_timed_steps=each["n"],
                    higher_is_better=True, scaling="weak", vs_baseline=None, dtype="c64 (fp32)", data="synthetic",
                    config=dict(workload="BASELINE.json configs[1]: 33x33 frequencies (M=1089, J=4356), 4 layers x 64 "
                                "planes, 256x256 grid, complex64, one scw_sweep_wavelengths call per step",
                                samples_per_step=samples, parallelism=f"replicas x{world}",
                                cache="inputs (457 MB of V) + outputs (403 MB) per step exceed the 126 MB L2; outputs alternate between two buffer sets",
                                setup="untimed, once: SCW_OPT_CACHE=1 (twiddle tables kept between steps, step a-3 'cached in ctx') "
                                      "and scw_calibrate (per-SM stream-K split of the assembly)",
                                why_config1="configs[1] is the largest config that runs in BOTH dtypes and the only one "
                                            "whose assembly is balanced between HBM and tensor work (Fz = 64); configs[2], [4] "
                                            "(HBM-bound, Fz = 16), [3], [3'] and configs[1] complex128 are under `extra`, "
                                            "each with its own roofline"),
                    clocks=clocks, e2e=e2e, gpu_launches=int(launches) * args.steps, gpu_launches_per_step=int(launches),
                    roofline=roof, whole_step=whole, assembly_phases=asm_phases, kernels=kernels,
                    kernels_cuda_events=kernels_ev, cpu_baseline=cpu, extra=extra, peaks=peaks)
        print(json.dumps(line))
    if dist is not None:
        dist.destroy_process_group()


def summarise_configs(ms, value, roof, extra):
    """One row per BASELINE.json config (the headline step first): time per call, throughput, the kernel that dominates
    the call, the roofline that bounds it and the fraction reached -- the figures a reader would otherwise dig out of
    `extra`.  Fractions are those computed where the config is measured (same peaks, same algorithmic bytes / flops)."""
    rows = {"config1_c64": dict(ms=ms, samples_per_s=value, kernel=roof["kernel"], bound=roof["bound"], frac=roof["frac"],
                                headline=True)}

    def sweep_row(e):                                     # a grouped complex64 sweep: the kernel with the largest share
        name = max(e["kernels"], key=lambda k: e["kernels"][k]["share"])
        k = e["kernels"][name]
        tensor = k.get("binding") == "tensor"
        return dict(ms=e["ms_per_call"], samples_per_s=e["samples_per_s"], kernel=name, bound="tensor" if tensor else "hbm",
                    frac=k["tensor_frac_executed"] if tensor else k.get("hbm_frac"), whole_call_hbm_frac=e.get("hbm_frac_V_plus_E"))

    def roof_row(e, rate_key, kernel):
        r = e["roofline"]
        return dict(ms=e.get("ms_per_call", e.get("ms_per_layer")), **{rate_key: e.get(rate_key)}, kernel=kernel,
                    bound=r["bound"], frac=r.get("frac_executed", r["frac"]), frac_useful=r["frac"] if "frac_executed" in r else None)

    if "config2_large" in extra:
        rows["config2_c64"] = sweep_row(extra["config2_large"])
    if "config4_sweep" in extra:
        rows["config4_c64"] = sweep_row(extra["config4_sweep"])
    if "config4_sweep_intensity" in extra:
        rows["config4_intensity"] = sweep_row(extra["config4_sweep_intensity"])
    if "config1_c128" in extra:
        rows["config1_c128"] = roof_row(extra["config1_c128"], "samples_per_s", "dmma_cgemm")
    if "config3_points" in extra:
        rows["config3_points"] = roof_row(extra["config3_points"], "points_per_s", "points_pw_c64")
    if "config3_dense_points" in extra:
        rows["config3_dense_points"] = roof_row(extra["config3_dense_points"], "points_per_s", "tc_assemble")
    if "vbuild_config1_shape" in extra:
        rows["next2_vbuild"] = roof_row(extra["vbuild_config1_shape"], "modes_per_s", "tc_assemble (generic GEMM)")
    if "alpha_propagation_config1_size" in extra:
        rows["next4_alpha_lu"] = roof_row(extra["alpha_propagation_config1_size"], "n", "lu_panel + dmma_cgemm")
    return rows


def extra_workloads(torch, scw, ctx, device, args, peaks):
    """Configs 3 (point path), 4 (sweep, detector), exterior field, 2, 1 complex128 and 3' at full size, each with the
    rooflines SURVEY 8(d) asks for (tensor useful / executed, HBM, which one binds)."""
    dev = lambda a: torch.from_numpy(np.ascontiguousarray(a)).to(device)
    traffic = load_traffic()
    mufu = peaks.get("mufu_gops", 148 * 16 * 1.965)           # Gop/s, measured by scw_measure_peak
    extra = {}
    # config 3: 4e6 scattered points x 4356 plane waves
    c3 = si.CONFIGS[3]
    pw = scw.PlaneWaves.from_numpy(si.make_planewaves(c3), device)
    pts = dev(si.make_points(c3))
    outp = torch.empty((pts.shape[0], 3), dtype=torch.complex64, device=device)
    ms = time_steps(torch, lambda: scw.scw_eval_points(ctx, pw, pts, out=outp), args.steps, args.warmup)
    terms = pts.shape[0] * 4356
    gterm = terms / (ms * 1e-3) / 1e9
    extra["config3_points"] = dict(ms_per_call=ms, points_per_s=pts.shape[0] / (ms * 1e-3), terms_per_s=gterm * 1e9,
                                   roofline=dict(bound="alu", achieved=gterm, peak=mufu / 3,
                                                 unit="Gterm/s (3 MUFU per term: sin, cos, ex2; peak = measured MUFU rate / 3)",
                                                 frac=gterm / (mufu / 3), traffic=None,
                                                 note="the XU floor is the demanding bound; what binds in practice is the "
                                                      "issue port (FFMA2 and DFMA hold it 2 cycles each: ~28.5 issue cycles "
                                                      "per warp-term against 24 XU cycles, DESIGN.md 5.3)",
                                                 fp32_fma_frac=gterm * 28 / 1e3 / peaks.get("fp32_fma_tflops", 70.7)))
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
    sweep4 = lambda: scw.scw_sweep_wavelengths(ctx, Ls, zs, dx, dy, out=out)
    scw.scw_calibrate(ctx, Ls, zs, dx, dy, out=out, reps=3)
    ms = time_steps(torch, sweep4, args.steps, args.warmup)
    n4 = len(Ls) * c4.planes * c4.Nx * c4.Ny
    vbytes = sum(l.V.numel() * 8 for l in Ls)
    k4 = kernel_rooflines(*profile_from_ring(ctx, max(1, args.steps - 1)), sweep_shape(c4, len(Ls)), peaks)   # of the steps just timed
    extra["config4_sweep"] = dict(ms_per_call=ms, samples_per_s=n4 / (ms * 1e-3), kernels=k4,
                                  hbm_frac_V_plus_E=(vbytes + n4 * 24) / (ms * 1e-3) / 1e9 / peaks["hbm_gbs"])
    # NEXT-3 detector: the same sweep with I = sum_comp |E_comp|^2 reduced in the synthesis epilogue (E never written)
    outI = [torch.empty((c4.planes, c4.Ny, c4.Nx), dtype=torch.float32, device=device) for _ in Ls]
    det4 = lambda: scw.scw_sweep_intensity(ctx, Ls, zs, dx, dy, out=outI)
    ms_i = time_steps(torch, det4, args.steps, args.warmup)
    kI = kernel_rooflines(*profile_from_ring(ctx, max(1, args.steps - 1)), sweep_shape(c4, len(Ls)), peaks)
    if "tc_synth" in kI:                                     # detector: 4 bytes per sample leave the SM instead of 24
        kI["tc_synth"]["alg_bytes"] = n4 * 4
        kI["tc_synth"]["hbm_gbs"] = n4 * 4 / (kI["tc_synth"]["ms_per_launch"] * 1e-3) / 1e9
        kI["tc_synth"]["hbm_frac"] = kI["tc_synth"]["hbm_gbs"] / peaks["hbm_gbs"]
        kI["tc_synth"]["binding"] = "tensor"
    extra["config4_sweep_intensity"] = dict(ms_per_call=ms_i, samples_per_s=n4 / (ms_i * 1e-3), kernels=kI,
                                            speedup_vs_complex_field=ms / ms_i)
    # window sums only: the detector reading S(lambda, z) of a 192 x 192 window, no per-sample output at all
    win = (32, 224, 32, 224)
    outS = [torch.empty((c4.planes,), dtype=torch.float32, device=device) for _ in Ls]
    detw = lambda: scw.scw_sweep_detector(ctx, Ls, zs, dx, dy, window=win, want_I=False, out_S=outS)
    ms_w = time_steps(torch, detw, args.steps, args.warmup)
    extra["config4_sweep_window_sums"] = dict(ms_per_call=ms_w, samples_per_s=n4 / (ms_w * 1e-3), window=win,
                                              speedup_vs_complex_field=ms / ms_w)
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

        def ext_two_calls():
            scw.scw_exterior_spectra(ctx, X, zg, out=Pbuf)
            scw.scw_synthesize_grid(ctx, U=cfgx.U, Vn=cfgx.Vn, X=ext["X"], Y=ext["Y"], P=Pbuf, x=dxg, y=dyg, out=Eo)

        ms2 = time_steps(torch, ext_two_calls, args.steps, args.warmup)
        ms = time_steps(torch, lambda: scw.scw_exterior_grid(ctx, X, zg, dxg, dyg, out=Eo), args.steps, args.warmup)
        ns = planes * cfgx.Nx * cfgx.Ny
        extra[name] = dict(ms_per_call=ms, samples_per_s=ns / (ms * 1e-3), orders=cfgx.U * cfgx.Vn, planes=planes,
                           hbm_write_frac=ns * 24 / (ms * 1e-3) / 1e9 / peaks["hbm_gbs"], call="scw_exterior_grid (twiddles cached)",
                           ms_spectra_then_synthesize=ms2)
    # NEXT-2 V builder (eq. 33) at config-1 shape: V = T Q, an M x M by M x 4M complex GEMM (BF16x3 on tcgen05) + row copy
    c1s = si.CONFIGS[1]
    M1 = c1s.U * c1s.Vn
    gq = torch.Generator(device=device).manual_seed(7293)
    Qd = torch.view_as_complex(torch.randn((4 * M1, 4 * M1, 2), generator=gq, device=device) / (8 * M1) ** 0.5)
    psid = torch.view_as_complex(torch.randn((M1, 2), generator=gq, device=device) / (2 * M1) ** 0.5)
    Vout = torch.empty((4 * M1, 3 * M1), dtype=torch.complex64, device=device)
    vb = lambda: scw.scw_build_V(ctx, U=c1s.U, Vn=c1s.Vn, X=c1s.L, Y=c1s.L, lam=1.0, Q=Qd, psi=psid, out=Vout)
    ms = time_steps(torch, vb, args.steps, args.warmup)
    useful = 8 * M1 * M1 * 4 * M1 / (ms * 1e-3) / 1e12
    qbytes = (Qd.numel() + Vout.numel()) * 8
    extra["vbuild_config1_shape"] = dict(
        ms_per_call=ms, modes_per_s=4 * M1 / (ms * 1e-3),
        roofline=dict(bound="tensor", achieved=3 * useful, peak=peaks["bf16_tflops_sustained"], unit="TFLOP/s executed (BF16x3)",
                      frac=3 * useful / peaks["bf16_tflops_sustained"], useful_tflops=useful,
                      hbm_frac=qbytes / (ms * 1e-3) / 1e9 / peaks["hbm_gbs"], traffic=None,
                      note="reads Q once (152 MB), writes V (114 MB); 41 GF useful"))
    del Qd, psid, Vout
    torch.cuda.empty_cache()
    # NEXT-4 alpha propagation (eq. 24-26) at config-1 size: one layer = one 4356 x 4356 complex128 LU + two triangular solves
    n_a = 4 * M1
    ga = torch.Generator(device=device).manual_seed(7294)
    # plain complex Gaussian Q (an eigenvector matrix is not diagonally dominant): partial pivoting exchanges nearly every
    # row, so the timed LU includes the cross-CTA pivot search and the k_lu_laswp traffic
    Qa = torch.view_as_complex(torch.randn((n_a, n_a, 2), generator=ga, device=device, dtype=torch.float64) / 2 ** 0.5)
    gma = torch.view_as_complex(torch.rand((n_a, 2), generator=ga, device=device, dtype=torch.float64))
    r0a = torch.view_as_complex(torch.randn((n_a, 2), generator=ga, device=device, dtype=torch.float64))
    al = lambda: scw.scw_propagate_alpha(ctx, lam=1.0, z_if=[0.0, 1.5], Q=[Qa], gamma=[gma], r0=r0a)
    ms = time_steps(torch, al, 3, 1)
    lu_tf = (8.0 / 3.0) * n_a ** 3 / (ms * 1e-3) / 1e12
    extra["alpha_propagation_config1_size"] = dict(
        ms_per_layer=ms, n=n_a,
        roofline=dict(bound="tensor", achieved=lu_tf, peak=peaks.get("fp64_dmma_tflops"), unit="TFLOP/s (fp64, 8/3 n^3 for the complex LU)",
                      frac=lu_tf / peaks["fp64_dmma_tflops"] if peaks.get("fp64_dmma_tflops") else None, traffic=None,
                      note="bound by the grid barrier per column of the cooperative panel kernel (half of the time) and by K = 64 trailing GEMMs, not by the tensor-core rate"))
    del Qa, gma, r0a
    torch.cuda.empty_cache()
    if not args.skip_large:
        c1, layers, zs1, x1, y1 = config1_inputs(np.complex128)
        Ls = [scw.Layer.from_numpy(d, device) for d in layers]
        out = [torch.empty((c1.planes, 3, c1.Ny, c1.Nx), dtype=torch.complex128, device=device) for _ in Ls]
        dz, dx, dy = [dev(z) for z in zs1], dev(x1), dev(y1)
        ms = time_steps(torch, lambda: scw.scw_sweep_wavelengths(ctx, Ls, dz, dx, dy, out=out), max(2, args.steps // 2), 2)
        M1 = c1.U * c1.Vn
        gf = c1.n_layers * (8 * 3 * M1 * 4 * M1 * c1.planes + 8 * 3 * c1.planes * (M1 * c1.Ny + c1.Nx * c1.U * c1.Ny)) / 1e9
        dmma = peaks.get("fp64_dmma_tflops")
        extra["config1_c128"] = dict(ms_per_call=ms, samples_per_s=c1.n_layers * c1.planes * c1.Nx * c1.Ny / (ms * 1e-3),
                                     roofline=dict(bound="tensor", achieved=gf / ms, peak=dmma,
                                                   unit="TFLOP/s (useful fp64, 8 per complex MAC; the 3M kernel executes 6; peak = "
                                                        "mma.sync m8n8k4 f64 rate measured by scw_measure_peak in this run)",
                                                   frac=gf / ms / dmma if dmma else None,
                                                   frac_executed=0.75 * gf / ms / dmma if dmma else None, traffic=None))
        del Ls, out, layers
        torch.cuda.empty_cache()
        c2 = si.CONFIGS[2]
        x2, y2, _ = si.grid_coords(c2, 0)
        Ls = [scw.Layer.from_numpy(si.make_layer(c2, l, dtype=np.complex64), device) for l in range(c2.n_layers)]
        dz = [dev(si.grid_coords(c2, l)[2]) for l in range(c2.n_layers)]
        out = [torch.empty((c2.planes, 3, c2.Ny, c2.Nx), dtype=torch.complex64, device=device) for _ in Ls]
        dx, dy = dev(x2), dev(y2)
        sweep2 = lambda: scw.scw_sweep_wavelengths(ctx, Ls, dz, dx, dy, out=out)
        scw.scw_calibrate(ctx, Ls, dz, dx, dy, out=out, reps=2)
        ms = time_steps(torch, sweep2, max(2, args.steps // 2), 2)
        n2 = c2.n_layers * c2.planes * c2.Nx * c2.Ny
        vbytes = sum(l.V.numel() * 8 for l in Ls)
        k2 = kernel_rooflines(*profile_from_ring(ctx, max(1, max(2, args.steps // 2) - 1)), sweep_shape(c2, len(Ls)), peaks, traffic.get("config2"))
        extra["config2_large"] = dict(ms_per_call=ms, samples_per_s=n2 / (ms * 1e-3), kernels=k2,
                                      hbm_frac_V_plus_E=(vbytes + n2 * 24) / (ms * 1e-3) / 1e9 / peaks["hbm_gbs"])
        del Ls, out
        torch.cuda.empty_cache()
        # config 3': dense eq. 34 at 65 536 scattered points: per point 3*M*J complex MACs on the tensor cores (a-1/a-2 with
        # one column per point, BF16x3) + an M-term sum per point
        lay = scw.Layer.from_numpy(si.make_layer(c3, dtype=np.complex64), device)
        pts = dev(si.make_points(c3, n=65536))
        ms = time_steps(torch, lambda: scw.scw_eval_points(ctx, lay, pts), 2, 1)
        M3 = c3.U * c3.Vn
        useful = 65536 * 8 * 3 * M3 * 4 * M3 / (ms * 1e-3) / 1e12
        extra["config3_dense_points"] = dict(
            ms_per_call=ms, points_per_s=65536 / (ms * 1e-3),
            roofline=dict(bound="tensor", achieved=3 * useful, peak=peaks["bf16_tflops_sustained"],
                          unit="TFLOP/s executed (BF16x3; useful = achieved / 3)", frac=3 * useful / peaks["bf16_tflops_sustained"],
                          useful_tflops=useful, hbm_frac=(65536 / 4096) * lay.V.numel() * 8 / (ms * 1e-3) / 1e9 / peaks["hbm_gbs"],
                          traffic=None, note="V is re-read once per chunk of 4096 points (16 chunks): hbm_frac counts those reads"))
    return extra


def blas_threads():
    try:
        from threadpoolctl import threadpool_info
        n = [p.get("num_threads", 1) for p in threadpool_info() if p.get("user_api") == "blas"]
        return max(n) if n else (os.cpu_count() or 1)
    except Exception:
        return os.cpu_count() or 1


def time_tier_b(layer, x, y, z, repeats=1):
    """Tier B of the oracle (the paper's own factored algorithm O(M^2 Fz + M F), numpy complex128 / BLAS) on
    the full grid of one config-1 layer; returns (samples, seconds)."""
    import oracle
    best = None
    for _ in range(repeats):
        t0 = time.perf_counter()
        oracle.tier_b_grid(x=x, y=y, z=z, **layer)
        dt = time.perf_counter() - t0
        best = dt if best is None else min(best, dt)
    return len(z) * len(y) * len(x), best


def time_tier_a(layer, xyz, threads, budget_s):
    """Tier A (the plain definition, triple loop) on as many of the seeded samples as fit the budget."""
    import oracle
    oracle.set_threads(threads)
    t0 = time.perf_counter()
    oracle.layer_samples(xyz=xyz[:threads], **layer)
    probe = time.perf_counter() - t0
    n = int(max(threads, min(len(xyz), budget_s / max(probe, 1e-6) * threads)))
    n -= n % threads
    t0 = time.perf_counter()
    oracle.layer_samples(xyz=xyz[:n], **layer)
    return n, time.perf_counter() - t0


def cpu_baseline(layer, x, y, z, cfg):
    """The oracle as it stands on the box's host cores, on config 1 layer 0 (~25 s in all).  Headline: Tier B, the paper's
    own factored algorithm, on the full 256 x 256 x 64 grid of the layer with all cores (the "fair" CPU baseline of SURVEY
    8(d)); beside it Tier A, the plain triple loop, on a bounded seeded sample with all cores and with one thread."""
    import oracle
    n_total = cfg.planes * cfg.Ny * cfg.Nx
    idx = si.sample_subset(cfg, n_total, 4096)
    iz, iy, ix = np.unravel_index(idx, (cfg.planes, cfg.Ny, cfg.Nx))
    xyz = np.column_stack([x[ix], y[iy], z[iz]])
    cores = oracle.threads()
    nb, tb = time_tier_b(layer, x, y, z, repeats=2)
    na, ta = time_tier_a(layer, xyz, cores, 10.0)
    n1, t1 = time_tier_a(layer, xyz, 1, 5.0)
    oracle.set_threads(cores)
    return dict(value=nb / tb, unit=UNIT, cores=blas_threads(), kind="oracle",
                tier="B (factored, O(M^2 Fz + M F), PAPER.md:418; numpy complex128 + BLAS)",
                sample=f"all {nb} samples of config 1 layer 0 (256 x 256 x 64), best of 2, {tb:.2f} s",
                definition=dict(value=na / ta, unit=UNIT, cores=cores, kind="oracle",
                                tier="A (the plain definition: 3*M*J = 14.2e6 complex terms per sample, OpenMP over samples)",
                                sample=f"{na} seeded samples of config 1 layer 0, {ta:.1f} s"),
                definition_1thread=dict(value=n1 / t1, unit=UNIT, cores=1, kind="oracle", tier="A, one thread",
                                        sample=f"{n1} seeded samples of config 1 layer 0, {t1:.1f} s"))


def run_reference(args):
    """--impl reference: the oracle timed on the host cores.  Each step evaluates ONE full layer of config 1 (4 194 304
    samples) with Tier B, the factored CPU algorithm the GPU path also runs; Tier A (the plain definition,
    O(M J) per sample) is reported beside it on a bounded sample."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    import oracle
    cfg = si.CONFIGS[1]
    layer = si.make_layer(cfg, 0, dtype=np.complex64)
    x, y, z = si.grid_coords(cfg, 0)
    per_step = cfg.planes * cfg.Ny * cfg.Nx
    for _ in range(args.warmup):
        oracle.tier_b_grid(x=x, y=y, z=z, **layer)
    t0 = time.perf_counter()
    for _ in range(args.steps):
        oracle.tier_b_grid(x=x, y=y, z=z, **layer)
    dt = (time.perf_counter() - t0) / args.steps
    value = per_step / dt
    cores = oracle.threads()
    idx = si.sample_subset(cfg, per_step, 4096)
    iz, iy, ix = np.unravel_index(idx, (cfg.planes, cfg.Ny, cfg.Nx))
    na, ta = time_tier_a(layer, np.column_stack([x[ix], y[iy], z[iz]]), cores, 6.0)
    sample = f"one full layer of config 1 per step ({per_step} samples), Tier B (factored, numpy complex128 + BLAS)"
    print(json.dumps(dict(impl="reference", metric=METRIC, value=value, unit=UNIT, n_gpus=args.gpus, steps=args.steps,
                          warmup=args.warmup, ms_per_step=dt * 1e3, higher_is_better=True, scaling="weak",
                          vs_baseline=None, dtype="f64", data="synthetic",
                          config=dict(workload="BASELINE.json configs[1] (33x33 frequencies, 4 layers x 64 planes, "
                                      "256x256 grid); one of its four layers per step", samples_per_step=per_step),
                          cpu_baseline=dict(value=value, unit=UNIT, cores=blas_threads(), kind="oracle",
                                            tier="B (factored)", sample=sample,
                                            definition=dict(value=na / ta, unit=UNIT, cores=cores, kind="oracle", tier="A",
                                                            sample=f"{na} seeded samples of config 1 layer 0, {ta:.1f} s")),
                          e2e=dict(value=value, unit=UNIT, h2d_bytes_per_step=0, d2h_bytes_per_step=0),
                          gpu_launches=0)))


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
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
