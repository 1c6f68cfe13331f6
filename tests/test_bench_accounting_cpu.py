"""CPU checks of bench.py's roofline accounting: the compulsory bytes, model FLOPs, executed
UMMA FLOPs and FFT-FLOP estimate of the headline workload are the figures DESIGN.md S5.4 derives by hand."""
import importlib.util
import os

import numpy as np

from paper_2208_05419_b200 import inputs

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
spec = importlib.util.spec_from_file_location("bench", os.path.join(ROOT, "bench.py"))
bench = importlib.util.module_from_spec(spec)
spec.loader.exec_module(bench)


def test_headline_work_figures():
    wl = inputs.WORKLOADS[bench.WL_NAME]
    assert (wl.B, wl.H, wl.W, wl.C, wl.num_blocks) == (4, 90, 180, 768, 8)
    Kh, Kw, kept = bench.kept_counts(wl)
    assert (Kh, Kw, kept) == (46, 91, 8190)
    work = bench.layer_work(wl.B, wl.H, wl.W, wl.C, wl.num_blocks, kept)
    act = 4 * 90 * 180 * 768 * 2
    params = 2 * (8 * 96 * 96 * 2 + 768 * 2) * 4
    assert work["bytes"] == 5 * act + 3 * params == 501_239_808          # 128.0 MB per sample x 4
    assert work["flops_model"] == 6 * 2 * 192 * 192 * 8 * 8190 * 4       # 29.0 GF per sample x 4
    assert abs(work["flops_model"] / 4 - 28.98e9) < 0.01e9
    exe = bench.executed_tensor_flops(wl.B, wl, Kw)
    # 96 UMMAs of 128x96x16 per mode tile (2 chain launches), 24 per row tile (4 W launches), 12 of 128x192x16 per
    # (layer, mode tile): 110.0 + 110.0 + 4 x 27.2 + 55.0 GF
    assert abs(exe["tc_mix_fwd"] - 109.9e9) < 0.2e9 and abs(exe["tc_wdft_per_launch"] - 27.18e9) < 0.05e9
    assert abs(exe["tc_wgrad"] - 54.97e9) < 0.1e9
    assert abs(exe["total"] / work["flops_model"] - 3.31) < 0.01
    fft = bench.fft_flops_per_step(wl.B, wl)
    assert abs(fft / 4 - 2.45e9) < 0.02e9                                 # 2.45 GFLOP per sample


def test_kernel_work_counts_compulsory_bytes_only():
    wl = inputs.WORKLOADS[bench.WL_NAME]
    _, Kw, kept = bench.kept_counts(wl)
    work = bench.layer_work(wl.B, wl.H, wl.W, wl.C, wl.num_blocks, kept)
    exe = bench.executed_tensor_flops(wl.B, wl, Kw)
    act = work["act"]
    assert bench.kernel_work("tc_wdft_fwd", work, exe)["bytes"] == act            # x (or dy) in; the half-spectrum is an intermediate
    assert bench.kernel_work("tc_wdft_inv", work, exe)["bytes"] == 2 * act        # residual in, y (or dx) out
    for k in ("tc_mix_fwd", "tc_mix_bwd", "tc_wgrad"):
        kw = bench.kernel_work(k, work, exe)
        assert kw["bytes"] == work["params"] and kw["flops"] == 2 * work["gemm"]
    # the layer's compulsory bytes are the sum of what the W kernels move plus the parameters
    assert 2 * act + 3 * act + 3 * work["params"] == work["bytes"]


def test_whole_job_value_and_reference_line_shape():
    assert bench.whole_job_value(2, 4, 10, 5.0) == 2 * 4 * 10 / 5e-3
    assert np.isclose(bench.whole_job_value(1, 4, 20, 20 * 0.4568), 4 / 0.4568e-3)


def test_executed_flops_count_groups_of_96_channels_not_blocks():
    """32 blocks of 32 channels are 11 groups of 96 (the kernels' tile), not 32: the executed-FLOP figure of the paper's
    channel structure follows the groups."""
    wl = inputs.WORKLOADS["paper_ch_b2"]
    assert (wl.C, wl.num_blocks) == (1024, 32)
    _, Kw, _ = bench.kept_counts(wl)
    exe = bench.executed_tensor_flops(wl.B, wl, Kw)
    umma96 = 2.0 * 128 * 96 * 16
    assert exe["tc_mix_fwd"] == 96 * umma96 * wl.B * Kw * 11
    assert exe["tc_wdft_per_launch"] == 24 * umma96 * wl.B * wl.H * 11


def test_stale_traffic_capture_is_never_quoted(tmp_path):
    """The stored ncu DRAM-traffic table carries the hash of the kernel sources it was captured on; with another hash
    in the tree every figure is None and the source string says so."""
    p = tmp_path / "t.csv"
    p.write_text("# src 0123456789abcdef\n# git abc1234\nkernel,bytes_per_launch\ntc_wdft_fwd,1000\ntc_mix_fwd,2000\n")
    fresh = bench.TrafficTable(str(p), src_hash="0123456789abcdef")
    assert fresh.get("tc_wdft_fwd") == 1000 and "stored" in fresh.source
    assert fresh.step_total({"tc_wdft_fwd": (4, 0.1), "tc_mix_fwd": (2, 0.1)}, 2) == 2 * 1000 + 2000
    stale = bench.TrafficTable(str(p), src_hash="ffffffffffffffff")
    assert stale.rows == {} and stale.source.startswith("null:") and "ffffffffffffffff" in stale.source
    assert stale.step_total({"tc_wdft_fwd": (4, 0.1)}, 2) is None
    assert len(bench.kernel_source_hash()) == 16
    # the committed table, whatever its state, never raises
    t = bench.TrafficTable()
    assert t.source is not None


def test_workload_table_is_valid_and_its_roofline_agrees_with_the_headline_accounting():
    """Every `bench.py --workload` entry is a descriptor the C ABI accepts (host-side check, no GPU), and the generic
    roofline formula reproduces the headline's hand-derived figures."""
    from paper_2208_05419_b200 import binding
    for name, (what, B, H, W, C, nb, hf, f, dtype, backward, ctx) in bench.WORKLOAD_TABLE.items():
        d = binding.Desc(B, H, W, C, nb, hf, 0.01, f, binding.AFNO_F32 if dtype == "f32" else binding.AFNO_BF16, 0)
        path = binding.afno_spectral_path(d)
        assert path is not None, name
        assert ("hybrid" in what) == (path == "hybrid-fft32-tcgen05"), (name, path)
        assert not ctx or backward, name
    wl = inputs.WORKLOADS[bench.WL_NAME]
    _, _, kept = bench.kept_counts(wl)
    work = bench.layer_work(wl.B, wl.H, wl.W, wl.C, wl.num_blocks, kept)
    assert bench.workload_roofline(wl.B, wl.H, wl.W, wl.C, wl.num_blocks, 1, wl.kept_fraction, False, True) == (
        work["bytes"], work["flops_model"])
    # forward only: x in, y out, parameters in; two block GEMMs
    nbytes, flops = bench.workload_roofline(1, 90, 180, 768, 8, 1, 1.0, False, False)
    assert nbytes == 2 * 90 * 180 * 768 * 2 + work["params"] and flops == 2 * work["gemm"] // 4
