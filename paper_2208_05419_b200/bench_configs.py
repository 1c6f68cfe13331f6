"""Times the OTHER configurations of BASELINE.json and SURVEY.md S8(f) through the C ABI (bench.py times the headline).

    python -m paper_2208_05419_b200.bench_configs [--calls 20] [--only NAME ...]

One JSON line per configuration: us per call (CUDA events on the launching stream over `--calls` calls, best of 3
repetitions, inputs rotated over buffer sets larger than the 126 MB L2), samples/s, the path that served it, the
fraction of the 2-term layer roofline (compulsory bytes at the measured HBM copy bandwidth, model MLP FLOPs at the
measured bf16 peak) and the per-kernel durations (CUDA events around every launch).  Inputs are
resident in HBM; no oracle, no CPU fallback.  The numbers of BASELINE.md S4 come from this script.
"""
from __future__ import annotations

import argparse
import json
import os
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        p = json.load(open(path))
        return float(p["hbm_gbs"]), float(p["bf16_tflops"]), "measured"
    return 6650.0, 1590.0, "fallback"


# name -> (B, H, W, C, num_blocks, hidden_factor, kept_fraction, backward, context)
CONFIGS = {
    "configs[1] fwd B=1": (1, 90, 180, 768, 8, 1, 1.0, False, False),
    "configs[2] fwd B=8 kept 1.0": (8, 90, 180, 768, 8, 1, 1.0, False, False),
    "configs[2] fwd B=8 kept 0.5": (8, 90, 180, 768, 8, 1, 0.5, False, False),
    "configs[3] fwd B=2 180x360": (2, 180, 360, 768, 8, 1, 1.0, False, False),
    "configs[4] fwd+bwd B=4 context": (4, 90, 180, 768, 8, 1, 1.0, True, True),
    "configs[4] fwd+bwd B=4 stateless": (4, 90, 180, 768, 8, 1, 1.0, True, False),
    "fwd+bwd B=8 context": (8, 90, 180, 768, 8, 1, 1.0, True, True),
    "paper channels 90x180x1024 nb=32 fwd+bwd B=4 context": (4, 90, 180, 1024, 32, 1, 1.0, True, True),
    "paper channels 90x180x1024 nb=32 fwd B=4": (4, 90, 180, 1024, 32, 1, 1.0, False, False),
    "180x360x768 fwd+bwd B=2 (hybrid)": (2, 180, 360, 768, 8, 1, 1.0, True, False),
    "paper shape 180x360x1024 nb=32 fwd B=2 (hybrid)": (2, 180, 360, 1024, 32, 1, 1.0, False, False),
    "paper shape 180x360x1024 nb=32 fwd+bwd B=1 (hybrid)": (1, 180, 360, 1024, 32, 1, 1.0, True, False),
    "hidden factor 2, 90x180x768 fwd B=4 (hybrid)": (4, 90, 180, 768, 8, 2, 1.0, False, False),
    "hidden factor 2, 90x180x768 fwd+bwd B=4 (hybrid)": (4, 90, 180, 768, 8, 2, 1.0, True, False),
    "fp32 activations 90x180x768 fwd+bwd B=2 (generic)": (2, 90, 180, 768, 8, 1, 1.0, True, False),
    "p->1 token grid 720x1440x768 fwd B=1 (hybrid)": (1, 720, 1440, 768, 8, 1, 1.0, False, False),
    "p->1 token grid 720x1440x768 fwd+bwd B=1 (hybrid)": (1, 720, 1440, 768, 8, 1, 1.0, True, False),
}


def kept_modes(H, W, f):
    f = float(np.float32(f))
    Kh = max(1, min(H // 2 + 1, int(np.floor(f * (H // 2 + 1)))))
    Kw = max(1, min(W // 2 + 1, int(np.floor(f * (W // 2 + 1)))))
    rows = 2 * Kh - 1 if Kh <= H // 2 else H
    return rows * Kw


def run(name, cfg, calls, reps):
    import torch

    from paper_2208_05419_b200 import binding

    B, H, W, C, nb, hf, f, backward, ctx = cfg
    hbm, tensor, src = _peaks()
    f32 = name.startswith("fp32")
    adt = torch.float32 if f32 else torch.bfloat16
    desc = binding.Desc(B, H, W, C, nb, hf, 0.01, f, binding.AFNO_F32 if f32 else binding.AFNO_BF16, 0)
    binding.afno_plan_warmup(desc)
    dev = torch.device("cuda")
    g = torch.Generator(device="cuda").manual_seed(1)
    act = B * H * W * C
    nsets = max(2, int(np.ceil(300e6 / (act * (4 if name.startswith("fp32") else 2) * (4 if backward else 2)))))
    nsets = min(nsets, 8)
    bs = C // nb
    hid = bs * hf
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
    fl_f = binding.FLAG_SAVE_CONTEXT if ctx else 0
    fl_b = binding.FLAG_USE_CONTEXT if ctx else 0
    desc_f = binding.Desc(**{**desc.__dict__, "flags": fl_f})
    desc_b = binding.Desc(**{**desc.__dict__, "flags": fl_b})
    ws = torch.empty(max(16, binding.afno_spectral_workspace_bytes(desc_f, backward)), dtype=torch.uint8, device=dev)
    stream = torch.cuda.current_stream()
    launches = [0]

    def call(i):
        s = sets[i % nsets]
        binding.afno_spectral_fwd(desc_f, s["x"], *params, s["y"], ws, stream)
        launches[0] = binding.afno_last_launch_count()
        if backward:
            binding.afno_spectral_bwd(desc_b, s["x"], s["dy"], *params, s["dx"], *grads, ws, stream)
            launches[0] += binding.afno_last_launch_count()

    for i in range(3):
        call(i)
    torch.cuda.synchronize()
    best = None
    for _ in range(reps):
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(stream)
        for i in range(calls):
            call(i)
        e1.record(stream)
        torch.cuda.synchronize()
        ms = e0.elapsed_time(e1) / calls
        best = ms if best is None else min(best, ms)
    binding.afno_profile_start()
    for i in range(3):
        call(i)
    prof = binding.afno_profile_stop()
    # 2-term layer roofline: compulsory bytes and model MLP FLOPs
    a_bytes = act * (4 if f32 else 2)
    pbytes = 2 * (nb * bs * hid * 2 + (hid + bs) * nb) * 4
    nbytes = (2 * a_bytes + pbytes) + ((3 * a_bytes + 2 * pbytes) if backward else 0)
    gemm = 2 * (2 * bs) * (2 * hid) * nb * kept_modes(H, W, f) * B
    flops = 2 * gemm + (4 * gemm if backward else 0)
    t_roof = max(nbytes / (hbm * 1e9), flops / (tensor * 1e12))
    line = {
        "config": name, "B": B, "H": H, "W": W, "C": C, "num_blocks": nb, "hidden_factor": hf, "kept_fraction": f,
        "backward": backward, "context": ctx, "path": binding.afno_spectral_path(desc),
        "us_per_call": round(best * 1e3, 1), "samples_per_s": round(B / (best * 1e-3), 1),
        "us_per_sample": round(best * 1e3 / B, 1), "launches_per_call": launches[0],
        "roofline_us_per_call": round(t_roof * 1e6, 1), "frac": round(t_roof / (best * 1e-3), 4),
        "compulsory_bytes": nbytes, "mlp_flops_model": flops, "peaks": f"{hbm} GB/s, {tensor} TFLOP/s ({src})",
        "kernels_us_per_call": {k: round(1e3 * v[1] / 3, 1) for k, v in sorted(prof.items())},
        "calls": calls, "reps": reps, "buffer_sets": nsets, "data": "synthetic N(0,1) activations resident in HBM",
    }
    del sets, ws
    torch.cuda.empty_cache()
    return line


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--calls", type=int, default=20)
    ap.add_argument("--reps", type=int, default=3)
    ap.add_argument("--only", nargs="*", default=None, help="substrings of the configuration names to run")
    args = ap.parse_args()
    import torch
    if not torch.cuda.is_available():
        raise SystemExit("bench_configs needs a CUDA device: the AFNO path has no CPU fallback")
    for name, cfg in CONFIGS.items():
        if args.only and not any(s in name for s in args.only):
            continue
        print(json.dumps(run(name, cfg, args.calls, args.reps)), flush=True)
    return 0


if __name__ == "__main__":
    sys.exit(main())
