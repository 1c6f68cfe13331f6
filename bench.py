#!/usr/bin/env python
"""bench.py -- AFNO spectral layer fwd+bwd samples/s at 90x180x768 bf16 (BASELINE.json metric).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference]

One "step" = one pass of the whole hot path (afno_spectral_fwd then afno_spectral_bwd, i.e.
every row F1-F9 and B1-B8 of DESIGN.md S1) over one batch of synthetic FourCastNet-shaped
activations.  Workload: BASELINE.json configs[4] (B=4, 90x180x768, 8 blocks of 96, bf16,
lambda 0.01, kept fraction 1.0).  Prints ONE JSON line (contract in the task prompt).

N > 1: the path does not shard ("replicas only", S6): every rank runs an
independent replica on its own GPU, no data-path collective; value = all ranks' samples /
max-over-ranks device time.  `--parallel dp` (not the contract line) adds what data
parallelism needs on top: ONE all-reduce(SUM) of the 1.19 MB of parameter gradients per step, inside the timed region.
"""
from __future__ import annotations

import argparse
import re
import json
import os
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import numpy as np  # noqa: E402

METRIC = "afno_spectral_fwd_bwd_samples_per_s_90x180x768_bf16"
UNIT = "samples/s"
WL_NAME = "fcn_b4_bwd"


def _peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        p = json.load(open(path))
        return dict(hbm_gbs=float(p["hbm_gbs"]), tensor_tflops=float(p["bf16_tflops"]),
                    tensor_tflops_sustained=float(p.get("bf16_tflops_sustained", p["bf16_tflops"])),
                    sm_max_mhz=float(p.get("sm_max_mhz", 1965.0)), source="measured")
    return dict(hbm_gbs=6650.0, tensor_tflops=1590.0, tensor_tflops_sustained=1400.0, sm_max_mhz=1965.0,
                source="fallback")


def kept_counts(wl):
    f = float(np.float32(wl.kept_fraction))
    Kh = max(1, min(wl.H // 2 + 1, int(np.floor(f * (wl.H // 2 + 1)))))
    Kw = max(1, min(wl.W // 2 + 1, int(np.floor(f * (wl.W // 2 + 1)))))
    rows = 2 * Kh - 1 if Kh <= wl.H // 2 else wl.H
    return Kh, Kw, rows * Kw


def layer_work(B, H, W, C, nb, kept_modes, ctx=True):
    """Algorithmic work of one fwd+bwd step (S5.4): COMPULSORY HBM bytes (the five
    activation tensors x, y, x again, dy, dx and the parameters / gradients) and MODEL MLP FLOPs."""
    act = B * H * W * C * 2                                  # one bf16 activation tensor
    params = 2 * (nb * (C // nb) ** 2 * 2 + C * 2) * 4       # w1,b1,w2,b2 fp32
    bytes_fwd = 2 * act + params                             # x in, y out
    bytes_bwd = 3 * act + 2 * params                         # x, dy in, dx out; params in, grads out
    bs = C // nb
    gemm = 2 * (2 * bs) * (2 * bs) * nb * kept_modes * B     # one complex block GEMM over all modes
    flops_fwd = 2 * gemm                                     # F3, F5
    flops_bwd_model = 4 * gemm                               # B4, B5, B6, B7
    return dict(bytes=bytes_fwd + bytes_bwd, flops_model=flops_fwd + flops_bwd_model, gemm=gemm, act=act,
                params=params)


def executed_tensor_flops(B, wl, Kw, ctx=True):
    """Tensor FLOPs the tcgen05 path EXECUTES per step, counted from the UMMA instructions the kernels issue
    (S5.3): every transform is a dense DFT GEMM and M is padded to 128."""
    umma96, umma192 = 2.0 * 128 * 96 * 16, 2.0 * 128 * 192 * 16
    groups = (wl.C + 95) // 96                               # the kernels tile over GROUPS of 96 channels (a group holds
                                                             # 96 / bs blocks when the blocks are narrower: 32 blocks of 32 = 11 groups)
    t_mode = B * Kw * groups                                 # (b, kw, group) tiles of tc_mix2 / tc_wgrad
    t_row = B * wl.H * groups                                # (b, h, group) tiles of the W-direction kernels
    mix_fwd = 96 * umma96 * t_mode                           # H-DFT 24 + layer 1 24 + layer 2 24 + inverse H-DFT 24
    mix_bwd = (96 if ctx else 168) * umma96 * t_mode
    wdft = 24 * umma96 * t_row                               # one launch; fwd has 2 (x -> A, A -> y), bwd 2 (+1 stateless)
    wgrad = 2 * 12 * umma192 * t_mode
    n_w = 4 if ctx else 5
    return dict(total=mix_fwd + mix_bwd + n_w * wdft + wgrad, tc_mix_fwd=mix_fwd, tc_mix_bwd=mix_bwd,
                tc_wdft_per_launch=wdft, tc_wgrad=wgrad)


def fft_flops_per_step(B, wl):
    """fp32 butterfly FLOPs a mixed-radix FFT implementation of the five 2-D transforms would execute
    (SURVEY.md S8(d) estimate: r2/r3/r5 butterflies 4/16/44 real FLOPs + 6 per non-trivial twiddle;
    cfft(90) ~ 3,084, cfft(180) ~ 7,068, rfft(W) = cfft(W/2) + 10 W/2); None for other grids."""
    cfft = {45: 1300.0, 90: 3084.0, 180: 7068.0}
    if wl.H not in cfft or wl.W // 2 not in cfft:
        return None
    rfft_w = cfft[wl.W // 2] + 10.0 * (wl.W // 2)
    per_channel = wl.H * rfft_w + (wl.W // 2 + 1) * cfft[wl.H]
    return 5.0 * per_channel * wl.C * B


class ClockSampler:
    """Samples SM clock and throttle reasons through NVML while the timed region runs."""

    def __init__(self, index):
        self.samples, self.reasons, self.max_mhz = [], set(), None
        self._stop = threading.Event()
        self._thread = None
        try:
            import pynvml
            pynvml.nvmlInit()
            self.nv = pynvml
            self.h = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.max_mhz = pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM)
        except Exception:
            self.nv = None

    def _run(self):
        nv = self.nv
        names = {
            "hw_slowdown": getattr(nv, "nvmlClocksThrottleReasonHwSlowdown", 0x8),
            "hw_thermal_slowdown": getattr(nv, "nvmlClocksThrottleReasonHwThermalSlowdown", 0x40),
            "sw_thermal_slowdown": getattr(nv, "nvmlClocksThrottleReasonSwThermalSlowdown", 0x20),
            "sw_power_cap": getattr(nv, "nvmlClocksThrottleReasonSwPowerCap", 0x4),
        }
        while not self._stop.is_set():
            try:
                self.samples.append(nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM))
                r = nv.nvmlDeviceGetCurrentClocksThrottleReasons(self.h)
                for k, bit in names.items():
                    if r & bit:
                        self.reasons.add(k)
            except Exception:
                pass
            self._stop.wait(0.02)

    def __enter__(self):
        if self.nv is not None:
            self._thread = threading.Thread(target=self._run, daemon=True)
            self._thread.start()
        return self

    def __exit__(self, *a):
        self._stop.set()
        if self._thread is not None:
            self._thread.join()

    def summary(self):
        if not self.samples:
            return {"sm_mhz": None, "sm_max_mhz": self.max_mhz, "reasons": ["nvml unavailable"]}
        return {"sm_mhz": float(np.median(self.samples)), "sm_max_mhz": self.max_mhz,
                "reasons": sorted(self.reasons)}


def max_over_ranks(value: float, dist, device) -> float:
    """Max of a per-rank scalar over all ranks (the N > 1 timing rule); dist = torch.distributed or None."""
    if dist is None:
        return float(value)
    import torch
    t = torch.tensor([float(value)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def whole_job_value(world: int, samples_per_rank_step: int, steps: int, ms_max: float) -> float:
    """Replicas only: every rank processes its own batch; value = all ranks' samples / max time."""
    return world * samples_per_rank_step * steps / (ms_max * 1e-3)


def oracle_time(n_samples: int):
    """Times the fp64 CPU oracle (as it stands) fwd+bwd on n_samples samples of the workload."""
    from oracle import afno_oracle
    from paper_2208_05419_b200 import inputs
    wl = inputs.WORKLOADS[WL_NAME]
    d = inputs.make_inputs(wl, B=n_samples)
    cfg = afno_oracle.Config(n_samples, wl.H, wl.W, wl.C, wl.num_blocks, lam=float(np.float32(wl.lam)),
                             kept_fraction=wl.kept_fraction)
    afno_oracle.lib()
    t0 = time.perf_counter()
    afno_oracle.forward(cfg, d["x"], d["w1"], d["b1"], d["w2"], d["b2"])
    afno_oracle.backward(cfg, d["x"], d["dy"], d["w1"], d["b1"], d["w2"], d["b2"])
    dt = time.perf_counter() - t0
    return n_samples / dt, dt, afno_oracle.num_threads()


def run_reference(args):
    """--impl reference: the oracle on the host cores, same metric/config, bounded sample per step."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return 0
    from paper_2208_05419_b200 import inputs
    wl = inputs.WORKLOADS[WL_NAME]
    steps = max(1, args.steps)
    for _ in range(args.warmup):
        oracle_time(1)
    tot_s, tot_t, cores = 0, 0.0, 0
    for _ in range(steps):
        v, dt, cores = oracle_time(1)
        tot_s += 1
        tot_t += dt
    value = tot_s / tot_t
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
        "steps": steps, "warmup": args.warmup, "ms_per_step": 1e3 * tot_t / steps,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
        "data": "synthetic",
        "config": {"workload": f"BASELINE.json configs[4]: {wl.name}; one sample per step (bounded sample)",
                   "H": wl.H, "W": wl.W, "C": wl.C, "num_blocks": wl.num_blocks, "lambda": wl.lam,
                   "kept_fraction": wl.kept_fraction},
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle",
                         "sample": f"{steps} x (1 sample fwd+bwd at 90x180x768, fp64, mixed-radix FFT mode)"},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line))
    return 0


def run_ours(args):
    import torch

    from paper_2208_05419_b200 import binding, inputs

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the AFNO path has no CPU fallback")
    torch.cuda.set_device(local_rank)
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device("cuda", local_rank))

    wl = inputs.WORKLOADS[WL_NAME]
    B = wl.B
    desc = binding.Desc(B, wl.H, wl.W, wl.C, wl.num_blocks, wl.hidden_factor, wl.lam, wl.kept_fraction,
                        binding.AFNO_BF16, 0)
    binding.afno_plan_warmup(desc)
    path = binding.afno_spectral_path(desc)
    peaks = _peaks()

    # --- inputs resident in HBM; rotate NSETS disjoint buffer sets (1.6 GB >> 126 MB L2) so reads are cold ----
    data = inputs.make_inputs(wl)
    NSETS = 4
    dev = torch.device("cuda", local_rank)
    to_bf16 = lambda a: torch.from_numpy(a).to(dev).to(torch.bfloat16)
    x0, dy0 = to_bf16(data["x"]), to_bf16(data["dy"])
    sets = []
    for s in range(NSETS):
        # distinct data per set (a roll along the batch axis keeps the statistics)
        sets.append(dict(x=torch.roll(x0, s, 0).contiguous(), dy=torch.roll(dy0, s, 0).contiguous(),
                         y=torch.empty_like(x0), dx=torch.empty_like(x0)))
    params = [torch.from_numpy(data[k]).to(dev) for k in ("w1", "b1", "w2", "b2")]
    from paper_2208_05419_b200 import sharding
    bucket = sharding.GradBucket.allocate(wl.num_blocks, wl.C // wl.num_blocks, wl.hidden_factor, device=dev)
    grads = bucket.views      # one flat buffer: --parallel dp reduces it with a single collective
    ws_f = torch.empty(binding.afno_spectral_workspace_bytes(desc, False), dtype=torch.uint8, device=dev)
    ws_b = torch.empty(binding.afno_spectral_workspace_bytes(desc, True), dtype=torch.uint8, device=dev)
    stream = torch.cuda.current_stream()
    launches = [0]

    # a training step: fwd leaves Xh, O1 and the activation masks in the workspace, bwd reads them
    # (SURVEY.md S8(a) row B1 "or load saved context"); --stateless times the recomputing bwd
    ctx = not args.stateless
    desc_f = binding.Desc(**{**desc.__dict__, "flags": binding.FLAG_SAVE_CONTEXT}) if ctx else desc
    desc_b = binding.Desc(**{**desc.__dict__, "flags": binding.FLAG_USE_CONTEXT}) if ctx else desc

    def step(i, st=stream):
        s = sets[i % NSETS]
        binding.afno_spectral_fwd(desc_f, s["x"], *params, s["y"], ws_b if ctx else ws_f, st)
        n = binding.afno_last_launch_count()
        binding.afno_spectral_bwd(desc_b, s["x"], s["dy"], *params, s["dx"], *grads, ws_b, st)
        launches[0] = n + binding.afno_last_launch_count()
        if args.parallel == "dp":
            bucket.all_reduce(dist, stream=st)   # PAPER.md:134; NCCL, on the step's stream (no-op at world size 1)

    def barrier():
        torch.cuda.synchronize()
        if dist is not None:
            dist.barrier()
            torch.cuda.synchronize()

    for i in range(args.warmup):
        step(i)
    barrier()
    # EXACTLY args.steps steps between two events; an event after every step gives the per-step spread
    evs = [torch.cuda.Event(enable_timing=True) for _ in range(args.steps + 1)]
    with ClockSampler(local_rank) as clocks:
        evs[0].record(stream)
        for i in range(args.steps):
            step(i)
            evs[i + 1].record(stream)
        barrier()
    ms = max_over_ranks(evs[0].elapsed_time(evs[-1]), dist, dev)
    per_step = np.array([evs[i].elapsed_time(evs[i + 1]) for i in range(args.steps)])
    ms_per_step = ms / args.steps
    value = whole_job_value(world, B, args.steps, ms)

    # --- the same step captured in CUDA graphs, one graph per buffer set: reported beside ---
    graph_info = None
    try:
        if args.timed_only:
            raise RuntimeError("skipped (--timed-only)")
        gs = torch.cuda.Stream()
        graphs = []
        with torch.cuda.stream(gs):
            for k in range(NSETS):
                gk = torch.cuda.CUDAGraph()
                with torch.cuda.graph(gk, stream=gs):
                    step(k, gs)
                graphs.append(gk)
            for k in range(NSETS):
                graphs[k].replay()
            torch.cuda.synchronize()
            g0, g1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            g0.record(gs)
            for i in range(args.steps):
                graphs[i % NSETS].replay()
            g1.record(gs)
            torch.cuda.synchronize()
        gms = g0.elapsed_time(g1) / args.steps
        graph_info = {"ms_per_step": gms, "value": B / (gms * 1e-3), "unit": UNIT,
                      "note": "fwd+bwd captured once per buffer set and replayed (reported, not the headline)"}
    except Exception as ex:  # capture is an extra: never lose the bench line to it
        graph_info = {"error": str(ex)[:200]}
    torch.cuda.synchronize()

    # --- per-kernel durations, measured live with CUDA events around every launch -----------
    # (the events sit between the kernels of a call and so disable the programmatic-dependent-launch overlap:
    #  the per-kernel times add up to more than ms_per_step; their SHARES are what the roofline uses)
    binding.afno_profile_start()
    PROF_STEPS = max(2, min(args.steps, 5))
    for i in range(PROF_STEPS):
        step(i)
    prof = binding.afno_profile_stop()
    total_prof_ms = sum(v[1] for v in prof.values())
    Kh, Kw, kept_modes = kept_counts(wl)
    work = layer_work(B, wl.H, wl.W, wl.C, wl.num_blocks, kept_modes, ctx)
    exe = executed_tensor_flops(B, wl, Kw, ctx)
    traffic = TrafficTable()
    clk = clocks.summary()
    per_kernel = {}
    for k, (n, ms_k) in sorted(prof.items()):
        per_kernel[k] = kernel_roofline(k, n, ms_k, PROF_STEPS, work, exe, peaks, traffic, total_prof_ms)
    dom = max(prof, key=lambda k: prof[k][1])

    # --- whole-layer roofline of BASELINE.json's metric: the headline fraction -----------
    t_step = ms_per_step * 1e-3
    t_hbm = work["bytes"] / (peaks["hbm_gbs"] * 1e9)
    t_tensor = work["flops_model"] / (peaks["tensor_tflops"] * 1e12)
    t_tensor_sus = work["flops_model"] / (peaks["tensor_tflops_sustained"] * 1e12)
    fp32_peak = 148 * 128 * 2 * peaks["sm_max_mhz"] * 1e6
    fft = fft_flops_per_step(B, wl)
    t_fft = fft / fp32_peak if fft else None
    t_roof = max(t_hbm, t_tensor)
    step_traffic = traffic.step_total(prof, PROF_STEPS)
    roofline = {
        "scope": "layer: all launches of one fwd+bwd step (SURVEY.md S8(d) contractual 2-term roofline)",
        "bound": "hbm" if t_hbm >= t_tensor else "tensor",
        "achieved": work["bytes"] / t_step / 1e9, "peak": peaks["hbm_gbs"], "unit": "GB/s",
        "frac": t_roof / t_step,
        "algorithmic_bytes_per_step": work["bytes"],
        "traffic": step_traffic,
        "traffic_ratio": (step_traffic / work["bytes"]) if step_traffic else None,
        "traffic_source": traffic.source,
        "t_roof_us_per_step": 1e6 * t_roof,
        "peaks": f"{peaks['hbm_gbs']} GB/s copy, {peaks['tensor_tflops']} TFLOP/s bf16 burst, "
                 f"{peaks['tensor_tflops_sustained']} sustained ({peaks['source']}, MEASURED_PEAKS.json)",
        "variants": {
            "two_term_burst": {"t_hbm_us": 1e6 * t_hbm, "t_tensor_us": 1e6 * t_tensor, "frac": max(t_hbm, t_tensor) / t_step},
            "two_term_sustained_tensor": {"t_tensor_us": 1e6 * t_tensor_sus, "frac": max(t_hbm, t_tensor_sus) / t_step},
            "three_term_with_fp32_fft": ({"t_fft_us": 1e6 * t_fft, "fp32_peak_tflops": fp32_peak / 1e12, "fft_flops": fft,
                                          "frac": max(t_hbm, t_tensor, t_fft) / t_step,
                                          "note": "bound of a plain fp32-ALU mixed-radix FFT design (SURVEY.md S0 finding 3); "
                                                  "this path runs its transforms on the tensor cores instead"} if t_fft else None),
            "executed_tensor_floor": {"t_us": 1e6 * exe["total"] / (peaks["tensor_tflops"] * 1e12),
                                      "note": "tensor FLOPs the kernels execute (dense DFT GEMMs, M padded to 128) at the burst peak"},
        },
        "mlp_flops_model_per_step": work["flops_model"],
        "tensor_flops_executed_per_step": exe["total"],
        "executed_over_model": exe["total"] / work["flops_model"],
        "achieved_tbs": work["bytes"] / t_step / 1e12,
        "achieved_tflops_model": work["flops_model"] / t_step / 1e12,
        "achieved_tflops_executed": exe["total"] / t_step / 1e12,
        "dominant_kernel": dict(per_kernel[dom], kernel=dom),
        "kernels_ms_per_step": {k: round(v[1] / PROF_STEPS, 4) for k, v in sorted(prof.items())},
        "per_kernel": per_kernel,
        "per_kernel_note": "CUDA events around every launch (afno_profile_*): no PDL overlap between kernels, so the sum "
                           "exceeds ms_per_step; algorithmic bytes = COMPULSORY bytes of the launch only (activations in / "
                           "out, parameters), intermediates (half-spectra, saved context, operand images) are traffic",
    }

    # --- end to end through the C ABI with HOST buffers -----------------------------------------
    e2e = None
    if (rank == 0 or world > 1) and not args.timed_only:
        pin = lambda t: t.cpu().pin_memory()
        hx, hdy = pin(x0), pin(dy0)
        hp = [pin(p) for p in params]
        hy, hdx = torch.empty_like(hx).pin_memory(), torch.empty_like(hx).pin_memory()
        hg = [torch.empty_like(p).pin_memory() for p in hp]
        arena = torch.empty(binding.afno_spectral_host_arena_bytes(desc, 2), dtype=torch.uint8, device=dev)
        act = hx.numel() * 2
        pbytes = sum(p.numel() * 4 for p in hp)
        E2E_STEPS = max(1, min(args.steps, 5))

        def host_step():
            # one call per training step: x and dy in, y, dx and the parameter gradients out, the two directions of the
            # link busy across the forward / backward boundary (x is uploaded once)
            binding.afno_spectral_step_host(desc, hx, hdy, *hp, hy, hdx, *hg, arena, stream)

        host_step()
        barrier()
        t0 = time.perf_counter()
        for _ in range(E2E_STEPS):
            host_step()
        torch.cuda.synchronize()
        dt = max_over_ranks(time.perf_counter() - t0, dist, dev)
        e2e = {"value": whole_job_value(world, B, E2E_STEPS, dt * 1e3), "unit": UNIT,
               "h2d_bytes_per_step": 2 * act + 2 * pbytes, "d2h_bytes_per_step": 2 * act + pbytes,
               "steps": E2E_STEPS, "note": "afno_spectral_step_host (one C-ABI call per step: fwd + bwd from pinned host buffers, x uploaded once, results back on the host), wall clock"}

    cpu_baseline = None
    if rank == 0 and world == 1 and not args.no_cpu_baseline and not args.timed_only:
        v, dt, cores = oracle_time(8)
        cpu_baseline = {"value": v, "unit": UNIT, "cores": cores, "kind": "oracle",
                        "sample": f"8 samples fwd+bwd at 90x180x768 (fp64 oracle, mixed-radix FFT mode), {dt:.1f} s"}

    if rank == 0:
        line = {
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "bf16", "data": "synthetic",
            "ms_per_step_median": float(np.median(per_step)), "ms_per_step_best": float(per_step.min()),
            "config": {"workload": f"BASELINE.json configs[4]: {wl.name}", "B_per_gpu": B, "H": wl.H, "W": wl.W,
                       "C": wl.C, "num_blocks": wl.num_blocks, "lambda": wl.lam, "kept_fraction": wl.kept_fraction,
                       "path": path, "backward": "saved context (fwd keeps Xh, O1 and the activation masks; bwd runs the gradient stages only)" if ctx
                       else "stateless (recomputes the spectrum of x)", "parallelism": ("single GPU" if world == 1 else "replicas only" if args.parallel == "replicas" else
                                       "data parallel: one all-reduce(SUM) of the parameter gradients per step"),
                       "l2": f"{NSETS} rotating input/output buffer sets of {4 * x0.numel() * 2 / 1e6:.0f} MB "
                             "each (> 126 MB L2), no explicit flush"},
            "clocks": clk, "e2e": e2e, "gpu_launches": launches[0] * args.steps,
            "roofline": roofline, "cuda_graph": graph_info, "cpu_baseline": cpu_baseline,
        }
        print(json.dumps(line))
    if dist is not None:
        dist.destroy_process_group()
    return 0


TRAFFIC_CSV = os.path.join("profiles", "r3_dram_traffic.csv")


def kernel_source_hash():
    """sha256 (first 16 hex digits) over the names and contents of every file under paper_2208_05419_b200/csrc/: what a
    stored ncu capture must have been taken on to describe this tree's kernels."""
    import hashlib
    h = hashlib.sha256()
    csrc = os.path.join(ROOT, "paper_2208_05419_b200", "csrc")
    for name in sorted(os.listdir(csrc)):
        if name.endswith((".cu", ".cuh", ".h")):
            h.update(name.encode() + b"\0")
            h.update(open(os.path.join(csrc, name), "rb").read())
    return h.hexdigest()[:16]


class TrafficTable:
    """dram__bytes_read.sum + dram__bytes_write.sum per launch from the committed ncu capture (profiles/r3_dram_traffic.csv,
    written by `bench.py --write-traffic`: '# src <hash of csrc/>' and '# git <commit>' header lines, then
    kernel,bytes_per_launch).  A stored capture, not a live measurement, so it only counts for the kernels it was taken
    on: when the hash of this tree's kernel sources differs from the header's, every figure is None and `source` says
    why (a stale capture is never quoted)."""

    def __init__(self, path=None, src_hash=None):
        self.rows, self.source = {}, None
        rel = TRAFFIC_CSV if path is None else path
        path = rel if os.path.isabs(rel) else os.path.join(ROOT, rel)
        try:
            git, src, rows = "unknown", None, {}
            for line in open(path).read().splitlines():
                if line.startswith("#"):
                    w = line[1:].split()
                    if len(w) >= 2 and w[0] == "git":
                        git = w[1]
                    if len(w) >= 2 and w[0] == "src":
                        src = w[1]
                    continue
                k, v = line.split(",")[:2]
                if k != "kernel":
                    rows[k] = int(float(v))
            have = kernel_source_hash() if src_hash is None else src_hash
            if src != have:
                self.source = (f"null: {rel} was captured on kernel sources {src} (commit {git}), this tree's are {have}; "
                               f"re-capture with the command in {os.path.splitext(rel)[0]}.md")
            else:
                self.rows = rows
                self.source = f"{rel} (ncu capture of kernel sources {src}, commit {git}; stored, not measured by this run)"
        except Exception as ex:
            self.source = f"unavailable: {ex}"

    def get(self, name):
        if name not in self.rows:
            if self.rows:
                sys.stderr.write(f"bench.py: {TRAFFIC_CSV} has no row for kernel {name!r}\n")
            return None
        return self.rows[name]

    def step_total(self, prof, steps):
        tot = 0
        for k, (n, _) in prof.items():
            t = self.get(k)
            if t is None:
                if k.startswith("tc_"):
                    return None
                continue
            tot += t * n / steps
        return int(tot) if tot else None


def write_traffic(raw_csv, out_path):
    """profiles/r3_dram_traffic.csv from ncu's raw page (`ncu -i X.ncu-rep --page raw --csv > raw.csv`) of a capture of
    `bench.py --timed-only` that starts on a step boundary: mean dram__bytes_read.sum + dram__bytes_write.sum per launch
    and kernel.  ncu names both chain launches tc_mix2; within a step the first is the forward's (tc_mix_fwd), the
    second the backward's (tc_mix_bwd), which is how the library's own profiler names them."""
    import csv
    import subprocess
    rows = list(csv.reader(open(raw_csv)))
    hdr = next(i for i, r in enumerate(rows) if "Kernel Name" in r)
    cols = {c: i for i, c in enumerate(rows[hdr])}
    units = rows[hdr + 1]
    scale = {"byte": 1.0, "Kbyte": 1e3, "Mbyte": 1e6, "Gbyte": 1e9}
    acc, mix = {}, 0
    for r in rows[hdr + 2:]:
        if len(r) <= cols["Kernel Name"]:
            continue
        m = re.search(r"(\w+)(?:<[^<>]*>)?\(", r[cols["Kernel Name"]])     # 'void afno::<unnamed>::tc_mix2<2, 0>(...)' -> tc_mix2
        name = m.group(1) if m else r[cols["Kernel Name"]].strip()
        if name == "tc_mix2":
            name = "tc_mix_fwd" if mix % 2 == 0 else "tc_mix_bwd"
            mix += 1
        name = {"tc_wdft_fwd2": "tc_wdft_fwd", "tc_wdft_inv2": "tc_wdft_inv"}.get(name, name)
        tot = 0.0
        for m in ("dram__bytes_read.sum", "dram__bytes_write.sum"):
            tot += float(r[cols[m]].replace(",", "")) * scale[units[cols[m]]]
        acc.setdefault(name, []).append(tot)
    try:
        git = subprocess.run(["git", "-C", ROOT, "rev-parse", "--short", "HEAD"], capture_output=True, text=True).stdout.strip() or "unknown"
    except Exception:
        git = "unknown"
    with open(out_path, "w") as f:
        f.write(f"# src {kernel_source_hash()}\n# git {git}\n")
        f.write("# dram__bytes_read.sum + dram__bytes_write.sum per launch (mean over the captured launches), ncu --set full\n")
        f.write("kernel,bytes_per_launch\n")
        for k, v in acc.items():
            f.write(f"{k},{int(sum(v) / len(v))}\n")
    return acc


def kernel_work(name, work, exe):
    """Algorithmic work of ONE launch: COMPULSORY HBM bytes only (activations into / out of
    the launch and parameters; half-spectra, saved context and operand images are intermediates) and the
    model FLOPs of the complex block GEMMs it evaluates (8 per complex MAC; padding and DFT-as-GEMM excluded)."""
    act, params, gemm = work["act"], work["params"], work["gemm"]
    table = {
        "tc_wdft_fwd": dict(bound="hbm", bytes=act, flops=0.0, executed=exe["tc_wdft_per_launch"]),
        "tc_wdft_inv": dict(bound="hbm", bytes=2 * act, flops=0.0, executed=exe["tc_wdft_per_launch"]),   # residual in, y / dx out
        "tc_mix_fwd": dict(bound="tensor", bytes=params, flops=2 * gemm, executed=exe["tc_mix_fwd"]),
        "tc_mix_bwd": dict(bound="tensor", bytes=params, flops=2 * gemm, executed=exe["tc_mix_bwd"]),
        "tc_wgrad": dict(bound="tensor", bytes=params, flops=2 * gemm, executed=exe["tc_wgrad"]),
        "k_block_gemm": dict(bound="alu", bytes=0, flops=gemm, executed=0.0),
        "k_block_wgrad": dict(bound="alu", bytes=0, flops=gemm, executed=0.0),
    }
    return table.get(name)


def kernel_roofline(name, n_launch, total_ms, steps, work, exe, peaks, traffic, total_prof_ms):
    """Per-kernel roofline entry: achieved = algorithmic work of one launch / its average duration measured with
    CUDA events around every launch (afno_profile_*); traffic = stored ncu DRAM bytes per launch."""
    per_launch_s = total_ms * 1e-3 / n_launch
    kw = kernel_work(name, work, exe)
    tr = traffic.get(name)
    out = {"launches_per_step": n_launch / steps, "avg_launch_us": round(per_launch_s * 1e6, 2),
           "share_of_step": total_ms / total_prof_ms if total_prof_ms > 0 else None, "traffic": tr}
    if kw is None:
        out.update({"bound": None, "frac": None})
        return out
    out["algorithmic_bytes"] = kw["bytes"]
    out["traffic_ratio"] = (tr / kw["bytes"]) if tr and kw["bytes"] else None
    out["dram_gbs_from_traffic"] = (tr / per_launch_s / 1e9) if tr else None
    if kw["bound"] == "tensor":
        ach = kw["flops"] / per_launch_s / 1e12
        out.update({"bound": "tensor", "achieved": ach, "peak": peaks["tensor_tflops"], "unit": "TFLOP/s",
                    "frac": ach / peaks["tensor_tflops"], "algorithmic_flops": kw["flops"],
                    "executed_flops": kw["executed"], "executed_tflops": kw["executed"] / per_launch_s / 1e12})
    elif kw["bound"] == "hbm":
        ach = kw["bytes"] / per_launch_s / 1e9
        out.update({"bound": "hbm", "achieved": ach, "peak": peaks["hbm_gbs"], "unit": "GB/s",
                    "frac": ach / peaks["hbm_gbs"], "executed_flops": kw["executed"]})
    else:
        peak = 148 * 128 * 2 * peaks["sm_max_mhz"] * 1e6 / 1e12
        ach = kw["flops"] / per_launch_s / 1e12
        out.update({"bound": "alu", "achieved": ach, "peak": peak, "unit": "TFLOP/s", "frac": ach / peak})
    return out


# ---- the other configurations of BASELINE.json and SURVEY.md S8(f): `bench.py --workload NAME` -----------------------
# name -> (what it is, B, H, W, C, num_blocks, hidden_factor, kept_fraction, dtype, backward, saved context)
WORKLOAD_TABLE = {
    "fcn_b1": ("BASELINE.json configs[1]: 90x180x768 bf16 fwd B=1", 1, 90, 180, 768, 8, 1, 1.0, "bf16", False, False),
    "fcn_b8": ("BASELINE.json configs[2]: 90x180x768 bf16 fwd B=8, kept 1.0", 8, 90, 180, 768, 8, 1, 1.0, "bf16", False, False),
    "fcn_b8_half": ("BASELINE.json configs[2]: 90x180x768 bf16 fwd B=8, kept 0.5", 8, 90, 180, 768, 8, 1, 0.5, "bf16", False, False),
    "hires_b2": ("BASELINE.json configs[3]: 180x360x768 bf16 fwd B=2 (hybrid path)", 2, 180, 360, 768, 8, 1, 1.0, "bf16", False, False),
    "fcn_b4_fwd": ("90x180x768 bf16 fwd B=4", 4, 90, 180, 768, 8, 1, 1.0, "bf16", False, False),
    "fcn_b4_bwd_stateless": ("BASELINE.json configs[4] with the stateless backward (recomputes the spectrum of x)", 4, 90, 180, 768, 8, 1, 1.0, "bf16", True, False),
    "fcn_b8_bwd": ("90x180x768 bf16 fwd+bwd B=8, saved context", 8, 90, 180, 768, 8, 1, 1.0, "bf16", True, True),
    "paper_ch_b4": ("paper channel structure 90x180x1024, 32 blocks of 32, fwd B=4", 4, 90, 180, 1024, 32, 1, 1.0, "bf16", False, False),
    "paper_ch_b4_bwd": ("paper channel structure 90x180x1024, 32 blocks of 32, fwd+bwd B=4, saved context", 4, 90, 180, 1024, 32, 1, 1.0, "bf16", True, True),
    "hires_b2_bwd": ("180x360x768 bf16 fwd+bwd B=2 (hybrid path)", 2, 180, 360, 768, 8, 1, 1.0, "bf16", True, False),
    "paper_shape_b2": ("paper layer shape 180x360x1024, 32 blocks of 32, fwd B=2 (hybrid path)", 2, 180, 360, 1024, 32, 1, 1.0, "bf16", False, False),
    "paper_shape_b1_bwd": ("paper layer shape 180x360x1024, 32 blocks of 32, fwd+bwd B=1 (hybrid path)", 1, 180, 360, 1024, 32, 1, 1.0, "bf16", True, False),
    "hf2_b4": ("hidden factor 2, 90x180x768 bf16 fwd B=4 (hybrid path)", 4, 90, 180, 768, 8, 2, 1.0, "bf16", False, False),
    "hf2_b4_bwd": ("hidden factor 2, 90x180x768 bf16 fwd+bwd B=4 (hybrid path)", 4, 90, 180, 768, 8, 2, 1.0, "bf16", True, False),
    "fp32_b2_bwd": ("fp32 activations 90x180x768 fwd+bwd B=2 (generic fp32 path)", 2, 90, 180, 768, 8, 1, 1.0, "f32", True, False),
    "p1_b1": ("p -> 1 token grid 720x1440x768 bf16 fwd B=1 (hybrid path)", 1, 720, 1440, 768, 8, 1, 1.0, "bf16", False, False),
    "p1_b1_bwd": ("p -> 1 token grid 720x1440x768 bf16 fwd+bwd B=1 (hybrid path)", 1, 720, 1440, 768, 8, 1, 1.0, "bf16", True, False),
}


def workload_roofline(B, H, W, C, nb, hf, f, f32, backward):
    """2-term layer roofline of any configuration: compulsory bytes (x in, y out; x, dy in, dx out;
    parameters in, gradients out) and the model FLOPs of the block MLP (2 GEMMs forward, 4 more backward)."""
    bs = C // nb
    hid = bs * hf
    a_bytes = B * H * W * C * (4 if f32 else 2)
    pbytes = 2 * (nb * bs * hid * 2 + (hid + bs) * nb) * 4
    nbytes = (2 * a_bytes + pbytes) + ((3 * a_bytes + 2 * pbytes) if backward else 0)
    Kh = max(1, min(H // 2 + 1, int(np.floor(float(np.float32(f)) * (H // 2 + 1)))))
    Kw = max(1, min(W // 2 + 1, int(np.floor(float(np.float32(f)) * (W // 2 + 1)))))
    kept = (2 * Kh - 1 if Kh <= H // 2 else H) * Kw
    gemm = 2 * (2 * bs) * (2 * hid) * nb * kept * B
    return nbytes, 2 * gemm + (4 * gemm if backward else 0)


def run_workload(args):
    """One of the other configurations through the C ABI, same JSON line as the headline (single GPU; inputs resident in
    HBM and rotated over buffer sets larger than the L2; EXACTLY --steps steps between two CUDA events after --warmup
    warm-up steps).  No e2e / cpu_baseline legs: they belong to the headline run."""
    import torch

    from paper_2208_05419_b200 import binding

    if int(os.environ.get("WORLD_SIZE", "1")) != 1 or args.gpus != 1:
        raise SystemExit("bench.py --workload other than the headline runs on one GPU")
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the AFNO path has no CPU fallback")
    what, B, H, W, C, nb, hf, f, dtype, backward, ctx = WORKLOAD_TABLE[args.workload]
    f32 = dtype == "f32"
    peaks = _peaks()
    adt = torch.float32 if f32 else torch.bfloat16
    desc = binding.Desc(B, H, W, C, nb, hf, 0.01, f, binding.AFNO_F32 if f32 else binding.AFNO_BF16, 0)
    binding.afno_plan_warmup(desc)
    dev = torch.device("cuda", 0)
    torch.cuda.set_device(0)
    g = torch.Generator(device="cuda").manual_seed(220805419)
    act = B * H * W * C
    nsets = int(np.ceil(300e6 / (act * (4 if f32 else 2) * (4 if backward else 2))))
    nsets = min(max(2, nsets), 8)
    bs, hid = C // nb, (C // nb) * hf
    sets = []
    for _ in range(nsets):
        s = dict(x=torch.randn((B, H, W, C), device=dev, generator=g).to(adt), y=torch.empty((B, H, W, C), device=dev, dtype=adt))
        if backward:
            s["dy"] = torch.randn((B, H, W, C), device=dev, generator=g).to(adt)
            s["dx"] = torch.empty_like(s["x"])
        sets.append(s)
    params = [0.02 * torch.randn(shape, device=dev, generator=g) for shape in
              [(nb, bs, hid, 2), (nb, hid, 2), (nb, hid, bs, 2), (nb, bs, 2)]]
    grads = [torch.empty_like(p) for p in params]
    desc_f = binding.Desc(**{**desc.__dict__, "flags": binding.FLAG_SAVE_CONTEXT if ctx else 0})
    desc_b = binding.Desc(**{**desc.__dict__, "flags": binding.FLAG_USE_CONTEXT if ctx else 0})
    ws = torch.empty(max(16, binding.afno_spectral_workspace_bytes(desc_f, backward)), dtype=torch.uint8, device=dev)
    stream = torch.cuda.current_stream()
    launches = [0]

    def step(i):
        s = sets[i % nsets]
        binding.afno_spectral_fwd(desc_f, s["x"], *params, s["y"], ws, stream)
        launches[0] = binding.afno_last_launch_count()
        if backward:
            binding.afno_spectral_bwd(desc_b, s["x"], s["dy"], *params, s["dx"], *grads, ws, stream)
            launches[0] += binding.afno_last_launch_count()

    for i in range(args.warmup):
        step(i)
    torch.cuda.synchronize()
    evs = [torch.cuda.Event(enable_timing=True) for _ in range(args.steps + 1)]
    with ClockSampler(0) as clocks:
        evs[0].record(stream)
        for i in range(args.steps):
            step(i)
            evs[i + 1].record(stream)
        torch.cuda.synchronize()
    ms = evs[0].elapsed_time(evs[-1])
    per_step = np.array([evs[i].elapsed_time(evs[i + 1]) for i in range(args.steps)])
    ms_per_step = ms / args.steps
    binding.afno_profile_start()
    PROF_STEPS = max(2, min(args.steps, 3))
    for i in range(PROF_STEPS):
        step(i)
    prof = binding.afno_profile_stop()
    nbytes, flops = workload_roofline(B, H, W, C, nb, hf, f, f32, backward)
    t_step = ms_per_step * 1e-3
    t_hbm, t_tensor = nbytes / (peaks["hbm_gbs"] * 1e9), flops / (peaks["tensor_tflops"] * 1e12)
    hbm_bound = t_hbm >= t_tensor
    dom = max(prof, key=lambda k: prof[k][1])
    line = {
        "metric": f"afno_spectral_{'fwd_bwd' if backward else 'fwd'}_samples_per_s_{H}x{W}x{C}_{dtype}",
        "value": B * args.steps / (ms * 1e-3), "unit": UNIT, "n_gpus": 1, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f32" if f32 else "bf16", "data": "synthetic N(0,1) activations and 0.02 N(0,1) parameters drawn on the device (seeded)",
        "ms_per_step_median": float(np.median(per_step)), "ms_per_step_best": float(per_step.min()),
        "config": {"workload": f"{args.workload}: {what}", "B_per_gpu": B, "H": H, "W": W, "C": C, "num_blocks": nb,
                   "hidden_factor": hf, "lambda": 0.01, "kept_fraction": f, "path": binding.afno_spectral_path(desc),
                   "backward": ("saved context" if ctx else "stateless") if backward else "none (forward only)",
                   "parallelism": "single GPU",
                   "l2": f"{nsets} rotating buffer sets of {(4 if backward else 2) * act * (4 if f32 else 2) / 1e6:.0f} MB "
                         "(together > 126 MB L2), no explicit flush"},
        "clocks": clocks.summary(),
        "e2e": None, "e2e_note": "the host-buffer leg is measured on the headline workload (python bench.py)",
        "gpu_launches": launches[0] * args.steps,
        "roofline": {
            "scope": "layer: all launches of one step (SURVEY.md S8(d) 2-term roofline of this shape)",
            "bound": "hbm" if hbm_bound else "tensor",
            "achieved": (nbytes / t_step / 1e9) if hbm_bound else (flops / t_step / 1e12),
            "peak": peaks["hbm_gbs"] if hbm_bound else peaks["tensor_tflops"], "unit": "GB/s" if hbm_bound else "TFLOP/s",
            "frac": max(t_hbm, t_tensor) / t_step, "traffic": None,
            "traffic_source": "null: no ncu DRAM capture is stored for this workload",
            "algorithmic_bytes_per_step": nbytes, "mlp_flops_model_per_step": flops,
            "t_roof_us_per_step": 1e6 * max(t_hbm, t_tensor),
            "peaks": f"{peaks['hbm_gbs']} GB/s copy, {peaks['tensor_tflops']} TFLOP/s bf16 burst ({peaks['source']}, MEASURED_PEAKS.json)",
            "dominant_kernel": {"kernel": dom, "ms_per_step": prof[dom][1] / PROF_STEPS, "launches_per_step": prof[dom][0] / PROF_STEPS},
            "kernels_ms_per_step": {k: round(v[1] / PROF_STEPS, 4) for k, v in sorted(prof.items())},
        },
        "cuda_graph": None,
        "cpu_baseline": None, "cpu_baseline_note": "skipped: the oracle leg is timed on the headline workload (python bench.py)",
    }
    print(json.dumps(line))
    return 0


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=50)
    ap.add_argument("--warmup", type=int, default=10)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--write-traffic", metavar="RAW_CSV", default=None,
                    help="no benchmark: turn ncu's raw page of a --timed-only capture into " + TRAFFIC_CSV)
    ap.add_argument("--workload", default=WL_NAME, choices=[WL_NAME] + sorted(WORKLOAD_TABLE),
                    help="default: the BASELINE.json headline (configs[4], fwd+bwd B=4 at 90x180x768 bf16); the other names "
                         "time the remaining BASELINE.json configs and the SURVEY.md S8(f) shapes (single GPU, same JSON line)")
    ap.add_argument("--timed-only", action="store_true",
                    help="warm-up, the timed steps and the per-kernel event pass only (no CUDA-graph replay, e2e or "
                         "cpu_baseline legs): the command the ncu captures under profiles/ run")
    ap.add_argument("--parallel", default="replicas", choices=["replicas", "dp"],
                    help="N > 1: independent replicas (the contract line; DESIGN.md S6) or data parallelism with one "
                         "all-reduce of the parameter gradients per step (SURVEY.md S8(f) item 4)")
    ap.add_argument("--stateless", action="store_true",
                    help="time the stateless afno_spectral_bwd (recomputes F1) instead of the saved-context step")
    args = ap.parse_args()
    if args.write_traffic:
        acc = write_traffic(args.write_traffic, os.path.join(ROOT, TRAFFIC_CSV))
        print(json.dumps({"written": TRAFFIC_CSV, "src": kernel_source_hash(), "launches": {k: len(v) for k, v in acc.items()}}))
        return 0
    if args.warmup < 3 and args.impl == "ours":
        args.warmup = 3
    if args.impl == "reference":
        return run_reference(args)
    if args.workload != WL_NAME:
        return run_workload(args)
    return run_ours(args)


if __name__ == "__main__":
    sys.exit(main())
