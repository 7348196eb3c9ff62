#!/usr/bin/env python
"""bench.py -- FK convolution hot path on B200: achieved HBM GB/s (BASELINE.json metric).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--extras none|fast|all]

One "step" = one pass of the whole hot path over one batch of synthetic input on BASELINE config 2
(hadronic FK, N=512, nx=50, 100 of 196 flavour pairs, ~1.0 GB, fp64, R=1): the convolution
(Eq. (1): luminosity on the fly -> streaming contraction -> two-level reduction) AND its
gradient (the VJP), i.e. two full reads of the table per step.  `value` = algorithmic
bytes per step / device time with everything resident in HBM; `e2e` = the same through the
host-buffer C-ABI calls (H2D of f and g, D2H of sigma and df inside the timed region; the FK table
itself stays resident, as in a fit: PAPER.md:29, :47).  Prints exactly one JSON line on stdout.

`--impl reference` times the CPU oracle (oracle/, as it stands) on a bounded sample of the same
workload.  N > 1: one process per GPU; when WORLD_SIZE is not set, bench.py re-executes itself under
torch.distributed.run with N ranks (and fails loudly when the node has fewer than N GPUs).  Default mode
"replicas": every rank runs the same step on its own copy of the table, no data-path
collective, value = N * bytes / max-over-ranks time, "scaling": "weak".  `--shard rows`: BASELINE config 4 with
whole tables owned by ranks (sharded.ShardedFkGroup), forward + VJP + the ONE all-reduce that assembles df per
step, total work fixed: "scaling": "strong".
"""
from __future__ import annotations

import argparse
import json
import os
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

from paper_1909_10547_b200 import synth  # noqa: E402  (seeded inputs only; no method arithmetic)

FP64_PEAK_TFLOPS = 37.2  # 148 SM x 64 FMA/clk x 2 x 1.965 GHz (probe: profiles/r01_fp64_peak.md)
METRIC = "fk_convolution_achieved_hbm_bandwidth"
UNIT = "GB/s"
# kernels of the config-2 step as the library's timing hook names them -> (what they are, S 8(a) rows, bound)
STEP_KERNELS = {
    "fk_fwd_column": ("forward column kernel: luminosity + streaming contraction + level-1 reduction", "a1+a2+a3", "hbm"),
    "fk_reduce_chunks": ("level-2 reduction of the forward partials", "a3", "latency"),
    "fk_colsum": ("VJP stage 1: column sums G = g^T FK", "a6", "hbm"),
    "fk_vjp_foldk": ("VJP stage 2: one pass over G for both legs", "a6", "latency"),
    "fk_vjp_foldk_final": ("VJP stage 2: fixed-order sum over channels", "a6", "latency"),
}
TRAFFIC_CSV = os.path.join("profiles", "r02_traffic.csv")
WORKLOAD = "config2: hadronic FK N=512 nx=50 nfl=14 C=100 R=1 fp64 (1.024 GB), forward + VJP per step"


def _measured_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        with open(p) as fh:
            d = json.load(fh)
        return float(d["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs, STREAM-style copy)"
    return 6650.0, "fallback (B200_PROFILING.md, 6.65 TB/s)"


def _tf32_peak():
    """Dense TF32 tensor peak in TFLOP/s: the measured bf16 cuBLAS burst figure x the guide's nominal TF32 / bf16 ratio (1/2)."""
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        with open(p) as fh:
            return 0.5 * float(json.load(fh)["bf16_tflops"])
    return 0.5 * 1590.0


# ------------------------------------------------------------------------------------------ clocks
class ClockSampler:
    """Samples SM clock and throttle reasons through NVML while the timed region runs."""

    def __init__(self, index: int):
        self.index = index
        self.samples, self.reasons = [], set()
        self.max_mhz = None
        self._stop = threading.Event()
        self._thr = None
        try:
            import pynvml
            pynvml.nvmlInit()
            self.nv = pynvml
            self.h = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.max_mhz = pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM)
        except Exception:
            self.nv = None

    def _names(self, mask):
        nv = self.nv
        table = [
            ("hw_slowdown", getattr(nv, "nvmlClocksEventReasonHwSlowdown", getattr(nv, "nvmlClocksThrottleReasonHwSlowdown", 0x8))),
            ("hw_thermal_slowdown", getattr(nv, "nvmlClocksEventReasonHwThermalSlowdown", getattr(nv, "nvmlClocksThrottleReasonHwThermalSlowdown", 0x40))),
            ("sw_thermal_slowdown", getattr(nv, "nvmlClocksEventReasonSwThermalSlowdown", getattr(nv, "nvmlClocksThrottleReasonSwThermalSlowdown", 0x20))),
            ("sw_power_cap", getattr(nv, "nvmlClocksEventReasonSwPowerCap", getattr(nv, "nvmlClocksThrottleReasonSwPowerCap", 0x4))),
        ]
        return [n for n, bit in table if mask & bit]

    def _run(self):
        nv = self.nv
        while not self._stop.is_set():
            try:
                self.samples.append(nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM))
                try:
                    mask = nv.nvmlDeviceGetCurrentClocksEventReasons(self.h)
                except Exception:
                    mask = nv.nvmlDeviceGetCurrentClocksThrottleReasons(self.h)
                self.reasons.update(self._names(mask))
            except Exception:
                pass
            time.sleep(0.002)

    def __enter__(self):
        if self.nv is not None:
            self._thr = threading.Thread(target=self._run, daemon=True)
            self._thr.start()
        return self

    def __exit__(self, *a):
        self._stop.set()
        if self._thr is not None:
            self._thr.join()

    def summary(self):
        if not self.samples:
            return {"sm_mhz": None, "sm_max_mhz": self.max_mhz, "reasons": [], "samples": 0}
        return {"sm_mhz": float(np.median(self.samples)), "sm_max_mhz": self.max_mhz,
                "reasons": sorted(self.reasons), "samples": len(self.samples)}


# ------------------------------------------------------------------------------------------ helpers
def step_bytes(case) -> int:
    """Algorithmic bytes of one step: FK once per pass, two passes, plus
    f, sigma (forward) and f, g, df (VJP)."""
    fkb = case.fk.nbytes
    return 2 * fkb + 2 * case.f.nbytes + case.f.nbytes + 2 * case.N * case.R * 8


def aggregate_max(ms_local: float, world: int) -> float:
    """max over ranks of the device time (gloo on CPU in the tests, nccl under torchrun)."""
    if world <= 1:
        return ms_local
    import torch
    import torch.distributed as dist
    dev = "cuda" if dist.get_backend() == "nccl" else "cpu"
    t = torch.tensor([ms_local], dtype=torch.float64, device=dev)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def _oracle_step_seconds(case, reps_target_s=10.0, max_reps=5):
    from oracle import fk_oracle as O  # the one place bench.py may execute oracle/
    O.hadronic(case.fk[:8], case.pairs, case.f)  # load + warm
    t_tot, reps = 0.0, 0
    while reps < max_reps and (reps == 0 or t_tot < reps_target_s):
        t0 = time.perf_counter()
        O.hadronic(case.fk, case.pairs, case.f)
        O.hadronic_vjp(case.fk, case.pairs, case.f, case.g)
        t_tot += time.perf_counter() - t0
        reps += 1
    return t_tot / reps, reps, O.num_threads()


# ------------------------------------------------------------------------------------------ reference arm
def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return 0
    rows = 128
    case = synth.config2(R=1, N=rows)
    from oracle import fk_oracle as O
    O.hadronic(case.fk[:8], case.pairs, case.f)
    for _ in range(max(0, min(args.warmup, 1))):
        O.hadronic(case.fk, case.pairs, case.f); O.hadronic_vjp(case.fk, case.pairs, case.f, case.g)
    steps = max(1, min(args.steps, 8))
    t0 = time.perf_counter()
    for _ in range(steps):
        O.hadronic(case.fk, case.pairs, case.f)
        O.hadronic_vjp(case.fk, case.pairs, case.f, case.g)
    sec = (time.perf_counter() - t0) / steps
    gbs = step_bytes(case) / sec / 1e9
    sample = f"first {rows} of 512 datapoints of config 2, forward + VJP, {steps} timed steps"
    line = {
        "impl": "reference", "metric": METRIC, "value": gbs, "unit": UNIT, "n_gpus": 1,   # rank 0's host cores, whatever --gpus says
        "steps": steps, "warmup": min(args.warmup, 1), "ms_per_step": sec * 1e3, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": WORKLOAD, "sample": sample},
        "cpu_baseline": {"value": gbs, "unit": UNIT, "cores": O.num_threads(), "kind": "oracle", "sample": sample},
        "e2e": {"value": gbs, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
    }
    print(json.dumps(line))
    return 0


# ------------------------------------------------------------------------------------------ our arm
def _time_loop(fn, steps, stream):
    import torch
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record(stream)
    for _ in range(steps):
        fn()
    e1.record(stream)
    e1.synchronize()
    return e0.elapsed_time(e1) / steps  # ms per call


def _bench_call(fn, stream, steps=20, warmup=3):
    for _ in range(warmup):
        fn()
    return _time_loop(fn, steps, stream)


def run_extras(K, torch, level, table2, case2, peak):
    """Other BASELINE configs (device-resident, CUDA events, median-free mean over 20 calls)."""
    out = {}
    stream = torch.cuda.current_stream()
    flush = torch.empty(256 * 1024 * 1024, dtype=torch.uint8, device="cuda")

    def cold(fn, reps=10):
        # small tables fit in L2 (126 MB): flush it before every timed call
        ts = []
        for _ in range(3):
            fn()
        for _ in range(reps):
            flush.zero_()
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record(stream); fn(); e1.record(stream); e1.synchronize()
            ts.append(e0.elapsed_time(e1))
        return float(np.median(ts))

    # config 2 split into its two passes
    f2 = torch.from_numpy(case2.f).cuda(); g2 = torch.from_numpy(case2.g).cuda()
    s2 = torch.empty((case2.N, 1), dtype=torch.float64, device="cuda"); d2 = torch.empty_like(f2)
    fkb = case2.fk.nbytes
    ms = _bench_call(lambda: table2.conv(f2, s2), stream)
    out["cfg2_forward"] = {"ms": ms, "GBps": fkb / ms / 1e6, "frac_of_peak": fkb / ms / 1e6 / peak,
                           "predictions_per_s": case2.N / ms * 1e3}
    ms = _bench_call(lambda: table2.vjp(f2, g2, d2), stream)
    out["cfg2_vjp"] = {"ms": ms, "GBps": fkb / ms / 1e6, "frac_of_peak": fkb / ms / 1e6 / peak}

    # the step replayed from a CUDA graph (capture of the two calls on a side stream): launch gaps removed by the driver
    graph, side = torch.cuda.CUDAGraph(), torch.cuda.Stream()
    with torch.cuda.graph(graph, stream=side):
        table2.conv(f2, s2)
        table2.vjp(f2, g2, d2)
    ms = _bench_call(graph.replay, stream)
    out["cfg2_step_cuda_graph"] = {"ms": ms, "GBps": 2 * fkb / ms / 1e6, "frac_of_peak": 2 * fkb / ms / 1e6 / peak}
    del graph
    # forward + VJP from ONE read of FK (fk_table_conv_vjp: g known before the forward pass).
    # GBps counts the FK bytes that really move (once); step_equiv_GBps the two-pass step it replaces.
    ms = _bench_call(lambda: table2.conv_vjp(f2, g2, s2, d2), stream)
    out["cfg2_conv_vjp_one_read"] = {"ms": ms, "GBps": fkb / ms / 1e6, "frac_of_peak": fkb / ms / 1e6 / peak,
                                     "step_equiv_GBps": 2 * fkb / ms / 1e6}
    # one fit iteration (fk_table_fit_step): forward -> chi2 and its gradient -> VJP, all on the device
    rng = np.random.default_rng(190910547 + 2001)
    a_ = rng.standard_normal(size=(case2.N, case2.N))
    cinv2 = torch.from_numpy(a_ @ a_.T / case2.N + np.eye(case2.N)).cuda()
    data2 = torch.from_numpy(rng.standard_normal(size=case2.N)).cuda()
    gg = torch.empty_like(s2); c2 = torch.empty(1, dtype=torch.float64, device="cuda")
    ms = _bench_call(lambda: table2.fit_step(f2, data2, cinv2, s2, gg, c2, d2), stream)
    out["cfg2_fit_step"] = {"ms": ms, "GBps": 2 * fkb / ms / 1e6, "frac_of_peak": 2 * fkb / ms / 1e6 / peak,
                            "fit_iterations_per_s": 1e3 / ms}
    # config 2 with the table stored in fp32 and everything else fp64 (FK_F32S64): half the bytes
    t32 = K.FkTable(K.FK_KIND_HADRONIC, torch.from_numpy(case2.fk).cuda(), case2.pairs, case2.nfl, K.FK_F32S64, K.FK_STORE_PACK)
    torch.cuda.empty_cache()
    ms = _bench_call(lambda: t32.conv(f2, s2), stream)
    out["cfg2_forward_fp32_storage"] = {"ms": ms, "GBps": fkb / 2 / ms / 1e6, "frac_of_peak": fkb / 2 / ms / 1e6 / peak,
                                        "predictions_per_s": case2.N / ms * 1e3, "tolerance": 1e-7}
    ms = _bench_call(lambda: t32.vjp(f2, g2, d2), stream)
    out["cfg2_vjp_fp32_storage"] = {"ms": ms, "GBps": fkb / 2 / ms / 1e6, "frac_of_peak": fkb / 2 / ms / 1e6 / peak}
    t32.destroy()
    # element-sparse storage (FK_STORE_SPARSE): the config-2 table with 30 % of its entries zeroed (config 1's
    # fraction) and with 60 %: bytes counted AS STORED (values + masks + headers); dense_equiv_GBps = the dense bytes / time
    gen = torch.Generator(device="cuda"); gen.manual_seed(190910547 + 2300)
    fk_dense = torch.from_numpy(case2.fk).cuda()
    for zf in (0.3, 0.6):
        fkz = fk_dense * (torch.rand(fk_dense.shape, device="cuda", generator=gen) >= zf)
        nnz = int(torch.count_nonzero(fkz).item())
        tsp = K.FkTable(K.FK_KIND_HADRONIC, fkz, case2.pairs, case2.nfl, K.FK_F64, K.FK_STORE_SPARSE)
        del fkz
        torch.cuda.empty_cache()
        stored = 8 * nnz + case2.N * ((case2.fk[0].size + 511) // 512) * 80
        for name, fn in (("forward", lambda: tsp.conv(f2, s2)), ("vjp", lambda: tsp.vjp(f2, g2, d2))):
            ms = _bench_call(fn, stream)
            out[f"cfg2_sparse{int(zf * 100)}_{name}"] = {"ms": ms, "stored_bytes": stored, "stored_over_dense": stored / fkb, "GBps": stored / ms / 1e6,
                                                        "frac_of_peak": stored / ms / 1e6 / peak, "dense_equiv_GBps": fkb / ms / 1e6}
        tsp.destroy()
    del fk_dense
    torch.cuda.empty_cache()
    # latency floors next to the microsecond-scale configs (SURVEY 8(d), L2 caveat): an empty launch, and one streaming
    # read of the same number of bytes (cold: L2 flushed before every call), through the same C-ABI library
    sink = torch.zeros(1, dtype=torch.float64, device="cuda")
    out["floor_empty_kernel_launch"] = {"ms": _bench_call(lambda: K.probe_launch(0), stream, steps=50),
                                        "ms_cold": cold(lambda: K.probe_launch(0))}
    c0 = synth.config0()
    fk0_d = torch.from_numpy(c0.fk).cuda()
    out["floor_read_probe_cfg0_bytes_cold"] = {"ms": cold(lambda: K.probe_launch(1, fk0_d, sink)), "bytes": c0.fk.nbytes}
    t0 = K.FkTable(K.FK_KIND_HADRONIC, fk0_d, c0.pairs, c0.nfl)
    f0 = torch.from_numpy(c0.f).cuda(); s0 = torch.empty((c0.N, 1), dtype=torch.float64, device="cuda")
    ms = cold(lambda: t0.conv(f0, s0))
    out["cfg0_forward_cold"] = {"ms": ms, "GBps": c0.fk.nbytes / ms / 1e6, "predictions_per_s": c0.N / ms * 1e3}
    ms = _bench_call(lambda: t0.conv(f0, s0), stream)
    out["cfg0_forward_L2warm"] = {"ms": ms, "GBps": c0.fk.nbytes / ms / 1e6}
    for R in (1, 100):
        c1 = synth.config1(R=R)
        fk1_d = torch.from_numpy(c1.fk).cuda()
        if R == 1:
            out["floor_read_probe_cfg1_bytes_cold"] = {"ms": cold(lambda: K.probe_launch(1, fk1_d, sink)), "bytes": c1.fk.nbytes}
        t1 = K.FkTable(K.FK_KIND_DIS, fk1_d, c1.flav, c1.nfl, R_hint=R)
        f1 = torch.from_numpy(c1.f).cuda(); s1 = torch.empty((c1.N, R), dtype=torch.float64, device="cuda")
        ms = cold(lambda: t1.conv(f1, s1))
        out[f"cfg1_dis_R{R}_cold"] = {"ms": ms, "GBps": c1.fk.nbytes / ms / 1e6,
                                      "predictions_per_s": c1.N * R / ms * 1e3,
                                      "GFLOPs": 2.0 * c1.N * c1.nx * c1.nA * R / ms / 1e6}
        t1.destroy()
    # config 3: same table as config 2, R=128 replicas
    R = 128
    f3 = torch.from_numpy(synth.pdf_grid(synth.pdf_params(synth.rng_for(2, synth.T_PDF, 0), R), 50)).cuda()
    s3 = torch.empty((case2.N, R), dtype=torch.float64, device="cuda")
    ms = _bench_call(lambda: table2.conv(f3, s3), stream, steps=5, warmup=2)
    flops = 2.0 * case2.N * case2.fk[0].size * R
    out["cfg3_forward_R128"] = {"ms": ms, "TFLOPs": flops / ms / 1e9, "replica_evals_per_s": R / ms * 1e3,
                                "predictions_per_s": case2.N * R / ms * 1e3, "frac_of_fp64_peak": flops / ms / 1e9 / FP64_PEAK_TFLOPS}
    g3 = torch.from_numpy(np.ascontiguousarray(np.broadcast_to(case2.g, (case2.N, R)))).cuda()
    d3 = torch.empty_like(f3)
    ms = _bench_call(lambda: table2.vjp(f3, g3, d3), stream, steps=5, warmup=2)
    out["cfg3_vjp_R128"] = {"ms": ms, "TFLOPs": flops / ms / 1e9, "frac_of_fp64_peak": flops / ms / 1e9 / FP64_PEAK_TFLOPS}
    # config 3, fp32 variant (BASELINE cfg3: "fp64 and fp32 variant"): tcgen05 3xTF32 contraction (fk_tc32.cu) against the
    # column-kernel passes it replaces.  HBM roofline: the 0.512 GB fp32 table once; tensor roofline: 3 TF32 products.
    t32v = K.FkTable(K.FK_KIND_HADRONIC, torch.from_numpy(case2.fk).cuda(), case2.pairs, case2.nfl, K.FK_F32, K.FK_STORE_PACK, R_hint=R)
    torch.cuda.empty_cache()
    f3s = f3.to(torch.float32); s3s = torch.empty((case2.N, R), dtype=torch.float32, device="cuda")
    ms = _bench_call(lambda: t32v.conv(f3s, s3s), stream, steps=10, warmup=3)
    tf32_peak = _tf32_peak()
    # tensor floor of the split: one TF32 product + two bf16 correction products (bf16 = 2 x the TF32 rate)
    tensor_floor_ms = flops / (tf32_peak * 1e9) + 2 * flops / (2 * tf32_peak * 1e9)
    out["cfg3_forward_R128_fp32"] = {
        "ms": ms, "launches": t32v.last_launches(), "GBps": fkb / 2 / ms / 1e6, "frac_of_peak": fkb / 2 / ms / 1e6 / peak,
        "TFLOPs_useful": flops / ms / 1e9, "tensor_floor_ms": tensor_floor_ms, "frac_of_tensor_peak": tensor_floor_ms / ms,
        "tf32_peak_TFLOPs": tf32_peak, "replica_evals_per_s": R / ms * 1e3, "tolerance": 1e-5}
    K.set_option(K.FK_OPT_TC32, 0)
    try:
        ms = _bench_call(lambda: t32v.conv(f3s, s3s), stream, steps=3, warmup=1)
        out["cfg3_forward_R128_fp32_column_passes"] = {"ms": ms, "launches": t32v.last_launches()}
    finally:
        K.set_option(K.FK_OPT_TC32, 1)
    # fp32 variant, VJP: FP64 tensor-core contraction over the fp32 table (widened in the fragment loads) + fp64 fold
    g3s = g3.to(torch.float32); d3s = torch.empty_like(f3s)
    ms = _bench_call(lambda: t32v.vjp(f3s, g3s, d3s), stream, steps=5, warmup=2)
    out["cfg3_vjp_R128_fp32"] = {"ms": ms, "launches": t32v.last_launches(), "TFLOPs": flops / ms / 1e9,
                                 "frac_of_fp64_peak": flops / ms / 1e9 / FP64_PEAK_TFLOPS, "tolerance": 1e-5}
    K.set_option(K.FK_OPT_GEMM_MIN_R, 1 << 20)
    try:
        ms = _bench_call(lambda: t32v.vjp(f3s, g3s, d3s), stream, steps=3, warmup=1)
        out["cfg3_vjp_R128_fp32_column_passes"] = {"ms": ms, "launches": t32v.last_launches()}
    finally:
        K.set_option(K.FK_OPT_GEMM_MIN_R, 0)
    t32v.destroy()
    # fp32 STORAGE, fp64 everything else (FK_F32S64) at R = 128: the FP64 contractions over the table as stored
    t32s = K.FkTable(K.FK_KIND_HADRONIC, torch.from_numpy(case2.fk).cuda(), case2.pairs, case2.nfl, K.FK_F32S64, K.FK_STORE_PACK, R_hint=R)
    torch.cuda.empty_cache()
    ms = _bench_call(lambda: t32s.conv(f3, s3), stream, steps=5, warmup=2)
    out["cfg3_forward_R128_f32s64"] = {"ms": ms, "launches": t32s.last_launches(), "TFLOPs": flops / ms / 1e9,
                                       "frac_of_fp64_peak": flops / ms / 1e9 / FP64_PEAK_TFLOPS, "tolerance": 1e-7}
    ms = _bench_call(lambda: t32s.vjp(f3, g3, d3), stream, steps=5, warmup=2)
    out["cfg3_vjp_R128_f32s64"] = {"ms": ms, "launches": t32s.last_launches(), "TFLOPs": flops / ms / 1e9,
                                   "frac_of_fp64_peak": flops / ms / 1e9 / FP64_PEAK_TFLOPS, "tolerance": 1e-7}
    t32s.destroy()
    if level == "all":
        out.update(run_config4(K, torch, peak))
    return out


def run_config4(K, torch, peak):
    """BASELINE config 4 (reading R15: the explicit distributions; ~14.8 GB): grouped forward + VJP at
    R=1 (HBM-bound) and R=100 (FP64-bound)."""
    out = {}
    shapes = synth.config4_shapes()
    stream = torch.cuda.current_stream()
    Rmax = 100
    params = synth.pdf_params(synth.rng_for(4, synth.T_PDF), Rmax)
    tabs, tabs32, fs, gs = [], [], [], []
    for t in range(shapes.T):
        c = synth.config4_table(t, shapes, Rmax, params)
        fk_d = torch.from_numpy(c.fk).cuda()
        tabs.append(K.FkTable(K.FK_KIND_HADRONIC, fk_d, c.pairs, c.nfl, R_hint=1))
        tabs32.append(K.FkTable(K.FK_KIND_HADRONIC, fk_d, c.pairs, c.nfl, K.FK_F32, K.FK_STORE_PACK, R_hint=1))
        del fk_d
        fs.append(c.f); gs.append(c.g)
    torch.cuda.empty_cache()
    grp = K.FkGroup(tabs, R_hint=Rmax)
    nbytes = shapes.fk_elements() * 8
    for R in (1, Rmax):
        f_cat = torch.cat([torch.from_numpy(np.ascontiguousarray(f[:R])).reshape(-1) for f in fs]).cuda()
        g_cat = torch.cat([torch.from_numpy(np.ascontiguousarray(g[:, :R])).reshape(-1) for g in gs]).cuda()
        _, so = grp.offsets(R)
        sig = torch.empty(int(so[-1]), dtype=torch.float64, device="cuda"); df = torch.empty_like(f_cat)
        flops = 2.0 * shapes.fk_elements() * R
        nst = 10 if R == 1 else 3
        ms = _bench_call(lambda: grp.conv(f_cat, R, sig), stream, steps=nst, warmup=3)
        out[f"cfg4_grouped_forward_R{R}"] = {"ms": ms, "GBps": nbytes / ms / 1e6, "frac_of_peak": nbytes / ms / 1e6 / peak,
                                             "TFLOPs": flops / ms / 1e9, "frac_of_fp64_peak": flops / ms / 1e9 / FP64_PEAK_TFLOPS,
                                             "sumN": int(shapes.N.sum()), "GB": nbytes / 1e9, "launches": grp.last_launches()}
        ms = _bench_call(lambda: grp.vjp(f_cat, g_cat, R, df), stream, steps=nst, warmup=3)
        out[f"cfg4_grouped_vjp_R{R}"] = {"ms": ms, "GBps": nbytes / ms / 1e6, "frac_of_peak": nbytes / ms / 1e6 / peak,
                                         "TFLOPs": flops / ms / 1e9, "frac_of_fp64_peak": flops / ms / 1e9 / FP64_PEAK_TFLOPS,
                                         "launches": grp.last_launches()}
        if R == 1:   # forward + VJP from one read of every table (fk_conv_grouped_conv_vjp)
            ms = _bench_call(lambda: grp.conv_vjp(f_cat, g_cat, R, sig, df), stream, steps=nst, warmup=3)
            out["cfg4_grouped_conv_vjp_one_read_R1"] = {"ms": ms, "GBps": nbytes / ms / 1e6, "frac_of_peak": nbytes / ms / 1e6 / peak,
                                                        "step_equiv_GBps": 2 * nbytes / ms / 1e6, "launches": grp.last_launches()}
    grp.destroy()
    for t in tabs:
        t.destroy()
    # fp32 variant of the group at R = 100: one grouped tcgen05 launch (3xTF32) over all 60 tables
    grp32 = K.FkGroup(tabs32, R_hint=Rmax)
    f32_cat = torch.cat([torch.from_numpy(np.ascontiguousarray(f[:Rmax])).reshape(-1) for f in fs]).cuda().float()
    _, so = grp32.offsets(Rmax)
    sig32 = torch.empty(int(so[-1]), dtype=torch.float32, device="cuda")
    ms = _bench_call(lambda: grp32.conv(f32_cat, Rmax, sig32), stream, steps=5, warmup=3)
    flops = 2.0 * shapes.fk_elements() * Rmax
    floor = 2 * flops / (_tf32_peak() * 1e9)   # one TF32 product + two bf16 correction products at twice the rate
    out[f"cfg4_grouped_forward_R{Rmax}_fp32"] = {"ms": ms, "TFLOPs_useful": flops / ms / 1e9, "tensor_floor_ms": floor, "frac_of_tensor_peak": floor / ms,
                                                 "launches": grp32.last_launches(), "tolerance": 1e-5}
    # ... and its VJP: the grouped FP64 tensor-core contraction over the fp32 tables as stored + the fp64 fold
    g32_cat = torch.cat([torch.from_numpy(np.ascontiguousarray(g[:, :Rmax])).reshape(-1) for g in gs]).cuda().float()
    df32 = torch.empty_like(f32_cat)
    ms = _bench_call(lambda: grp32.vjp(f32_cat, g32_cat, Rmax, df32), stream, steps=3, warmup=2)
    out[f"cfg4_grouped_vjp_R{Rmax}_fp32"] = {"ms": ms, "TFLOPs": flops / ms / 1e9, "frac_of_fp64_peak": flops / ms / 1e9 / FP64_PEAK_TFLOPS,
                                             "launches": grp32.last_launches(), "tolerance": 1e-5}
    grp32.destroy()
    for t in tabs32:
        t.destroy()
    return out


# Table 3 of the paper: flat FK[N x K] . PDF[K x R] with a PRE-BUILT PDF matrix (the paper's own
# shapes; K = 49 * 27^2 = 35721).  Run through fk_conv_dis with one pseudo-flavour and nx = K:
# sigma[n][r] = sum_k FK[n][k][0] f[r][0][k], i.e. f = PDF^T.  (K, R, N, paper's best seconds, whose)
TABLE3 = [
    (35721, 1, 8, 1.57e-4, "AVX"), (10**6, 1, 8, 5.00e-3, "AVX"), (10**7, 1, 8, 5.70e-2, "AVX"), (10**8, 1, 8, 5.70e-1, "AVX"),
    (35721, 10**2, 8, 1.60e-2, "AVX"), (35721, 10**3, 8, 1.50e-1, "TF-CPU"), (35721, 10**4, 8, 1.12, "TF-CPU"),
    (35721, 5 * 10**4, 10, 5.33, "TF-CPU"), (35721, 1, 10**2, 2.43e-3, "AVX"), (35721, 1, 10**3, 2.14e-2, "AVX"),
    (35721, 1, 10**4, 2.16e-1, "AVX"), (35721, 10**2, 10**2, 6.20e-2, "TF-CPU"), (35721, 10**3, 10**3, 3.00e-1, "TF-CPU"),
    (35721, 2 * 10**3, 2 * 10**3, 1.38, "TF-GPU"),
]


def run_table3(K, torch, peak):
    """Kernel-only times (operands resident, L2 flushed before each call when they fit in it) next to the paper's
    best time of each row (other hardware, H2D included for its GPU variants: context, not a target)."""
    out = []
    stream = torch.cuda.current_stream()
    gen = torch.Generator(device="cuda"); gen.manual_seed(190910547 + 3000)
    flush = torch.empty(256 * 1024 * 1024, dtype=torch.uint8, device="cuda")
    flav = np.zeros(1, dtype=np.int32)
    for (Kc, R, N, paper_s, who) in TABLE3:
        # the flat product is symmetric in its operands: the LARGER one is streamed as the table (read once from
        # HBM), the smaller one plays the PDF grid; for R > N that computes sigma^T[R][N]
        swapped = R > N
        rows, cols = (R, N) if swapped else (N, R)
        fk = torch.randn((rows, Kc, 1), dtype=torch.float64, device="cuda", generator=gen)
        f = torch.randn((cols, 1, Kc), dtype=torch.float64, device="cuda", generator=gen)
        sig = torch.empty((rows, cols), dtype=torch.float64, device="cuda")
        # rows of odd length (K = 35721) are not 16-byte aligned in place: the packed copy pads them (128-bit loads)
        store = K.FK_STORE_PACK if (Kc % 2 and rows * Kc * 8 < 40e9) else K.FK_STORE_BORROW
        tab = K.FkTable(K.FK_KIND_DIS, fk, flav, 1, K.FK_F64, store, R_hint=cols)
        for _ in range(2):
            tab.conv(f, sig)
        ts = []
        for _ in range(5):
            flush.zero_()
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record(stream); tab.conv(f, sig); e1.record(stream); e1.synchronize()
            ts.append(e0.elapsed_time(e1))
        ms = float(np.median(ts))
        nbytes = 8.0 * (N * Kc + Kc * R + N * R)
        # H2D-inclusive, as the paper's GPU numbers are ("the time required for the memory transfer to the
        # GPU" is included): both operands come from pinned host memory and the result goes back, inside the timed region
        fk_h = torch.empty(fk.shape, dtype=fk.dtype, pin_memory=True); fk_h.copy_(fk)
        f_h = torch.empty(f.shape, dtype=f.dtype, pin_memory=True); f_h.copy_(f)
        sig_h = torch.empty(sig.shape, dtype=sig.dtype, pin_memory=True)
        ts = []
        for it in range(3):
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            t0 = time.perf_counter()
            e0.record(stream)
            fk.copy_(fk_h, non_blocking=True); f.copy_(f_h, non_blocking=True)
            tab.conv(f, sig)
            sig_h.copy_(sig, non_blocking=True)
            e1.record(stream); e1.synchronize()
            if it:
                ts.append(max(e0.elapsed_time(e1), (time.perf_counter() - t0) * 1e3))
        ms_h2d = float(np.median(ts))
        out.append({"K": Kc, "R": R, "N": N, "ms": ms, "GBps": nbytes / ms / 1e6, "TFLOPs": 2.0 * N * Kc * R / ms / 1e9,
                    "ms_h2d_inclusive": ms_h2d, "h2d_GBps": 8.0 * (N * Kc + Kc * R) / ms_h2d / 1e6,
                    "launches": tab.last_launches(), "streamed": "PDF matrix" if swapped else "FK", "paper_best_s": paper_s, "paper_best": who,
                    "paper_over_ours": paper_s * 1e3 / ms, "paper_over_ours_h2d_inclusive": paper_s * 1e3 / ms_h2d})
        tab.destroy()
        del fk, f, sig, fk_h, f_h, sig_h
        torch.cuda.empty_cache()
    return out


def run_ours(args):
    import torch
    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device - the FK convolution has no CPU fallback")
    torch.cuda.set_device(local)
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    from paper_1909_10547_b200 import fkconv as K

    case = synth.config2(R=1)
    fk_d = torch.from_numpy(case.fk).cuda()
    table = K.FkTable(K.FK_KIND_HADRONIC, fk_d, case.pairs, case.nfl, K.FK_F64, K.FK_STORE_PACK, R_hint=1)
    del fk_d
    torch.cuda.empty_cache()
    f_d = torch.from_numpy(case.f).cuda(); g_d = torch.from_numpy(case.g).cuda()
    sig = torch.empty((case.N, 1), dtype=torch.float64, device="cuda"); df = torch.empty_like(f_d)
    stream = torch.cuda.current_stream()
    nbytes = step_bytes(case)
    peak, peak_src = _measured_peaks()

    launches_per_step = 0

    def step():
        nonlocal launches_per_step
        table.conv(f_d, sig, stream)
        n = table.last_launches()
        table.vjp(f_d, g_d, df, stream)
        launches_per_step = n + table.last_launches()

    for _ in range(max(3, args.warmup)):
        step()
    torch.cuda.synchronize()
    if world > 1:
        torch.distributed.barrier()

    # timed region: K steps, CUDA events on the launching stream, nothing between the launches of a step
    with ClockSampler(local) as clk:
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        torch.cuda.synchronize()
        e0.record(stream)
        for _ in range(args.steps):
            step()
        e1.record(stream)
        e1.synchronize()
        torch.cuda.synchronize()
    ms_local = e0.elapsed_time(e1) / args.steps
    # the same K steps once more with the library's per-launch event pairs (fk_profile_enable): every kernel of the
    # step timed on the launching stream.  Separate from the region above because an event record between two
    # launches serialises them (no programmatic dependent launch overlap), which would tax the headline number.
    K.profile_enable(True)
    e2, e3 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e2.record(stream)
    for _ in range(args.steps):
        step()
    e3.record(stream)
    e3.synchronize()
    ms_profiled = e2.elapsed_time(e3) / args.steps
    kernel_times = K.profile_report()
    K.profile_enable(False)
    if world > 1:
        torch.distributed.barrier()
    ms = aggregate_max(ms_local, world)
    value = world * nbytes / ms / 1e6  # GB/s, whole job

    # e2e: the host-buffer C-ABI calls (pinned staging, H2D + D2H + wait inside every step)
    f_h, g_h = case.f.copy(), case.g.copy()
    sig_h, df_h = np.empty((case.N, 1)), np.empty_like(case.f)
    # One host call per step: fk_table_conv_vjp_host (f and g up in one copy, sigma and df back in one copy, one wait).  With
    # FK_OPT_FUSED = 0 it runs the SAME two passes as the device-timed step (two reads of the table per step); the library's
    # default for this call, forward + VJP from one read, is timed next to it as `one_read_ms_per_step`.
    def e2e_time(fused):
        K.set_option(K.FK_OPT_FUSED, fused)
        try:
            for _ in range(3):
                table.conv_vjp_host(f_h, g_h, sig_h, df_h, stream)
            torch.cuda.synchronize()
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            t0 = time.perf_counter()
            e0.record(stream)
            for _ in range(args.steps):
                table.conv_vjp_host(f_h, g_h, sig_h, df_h, stream)
            e1.record(stream)
            e1.synchronize()
            return max(e0.elapsed_time(e1) / args.steps, (time.perf_counter() - t0) * 1e3 / args.steps)
        finally:
            K.set_option(K.FK_OPT_FUSED, 1)
    e2e_ms = aggregate_max(e2e_time(0), world)
    e2e_one_read_ms = aggregate_max(e2e_time(1), world)
    e2e = {"value": world * nbytes / e2e_ms / 1e6, "unit": UNIT,
           "h2d_bytes_per_step": int(case.f.nbytes + case.g.nbytes),
           "d2h_bytes_per_step": int(sig_h.nbytes + df_h.nbytes), "ms_per_step": e2e_ms,
           "call": "fk_table_conv_vjp_host, FK_OPT_FUSED=0 (two passes = two reads of the table, as the device-timed step)",
           "one_read_ms_per_step": e2e_one_read_ms}

    if rank != 0:
        return 0

    fkb = case.fk.nbytes
    traffic = _ncu_traffic()
    kernels = []
    for name, (n, tot_ms) in kernel_times.items():
        what, rows, bound = STEP_KERNELS.get(name, (name, "?", "?"))
        k_ms = tot_ms / n
        kb = fkb if bound == "hbm" else None   # algorithmic bytes per launch: the FK table once
        kernels.append({"name": name, "what": what, "rows": rows, "bound": bound, "launches": n, "ms": k_ms,
                        "share_of_profiled_step": tot_ms / args.steps / ms_profiled, "bytes": kb,
                        "achieved": (kb / k_ms / 1e6) if kb else None, "frac": (kb / k_ms / 1e6 / peak) if kb else None,
                        "traffic": traffic.get(name)})
    kernels.sort(key=lambda k: -k["ms"])
    dom = kernels[0] if kernels else None
    roofline = {
        "bound": "hbm", "kernel": (dom["name"] + " (" + dom["what"] + ", rows " + dom["rows"] + ")") if dom else None,
        "achieved": dom["achieved"] if dom else None, "peak": peak, "unit": "GB/s",
        "frac": dom["frac"] if dom else None, "peak_source": peak_src,
        "kernel_ms": dom["ms"] if dom else None, "kernel_launches_timed": dom["launches"] if dom else 0,
        "bytes_per_launch": fkb, "traffic": dom["traffic"] if dom else None,
        "traffic_source": "committed ncu --set full capture, " + TRAFFIC_CSV + " (dram read + write bytes per launch; not measured in this run)",
        "timed_in": "second pass of the same K steps with per-launch CUDA event pairs on the launching stream",
        "ms_per_step_profiled": ms_profiled, "kernels": kernels,
    }
    cpu_baseline = None
    if not args.no_cpu_baseline:
        rows = 256
        sub = synth.HadronicCase("cfg2-sample", case.fk[:rows], case.pairs, case.f, case.g[:rows])
        sec, reps, cores = _oracle_step_seconds(sub)
        cpu_baseline = {"value": step_bytes(sub) / sec / 1e9, "unit": UNIT, "cores": cores, "kind": "oracle",
                        "sample": f"first {rows} of 512 datapoints of config 2, forward + VJP, {reps} reps, {sec:.2f} s each"}
    extras = {}
    if args.extras != "none" and world == 1:
        try:
            extras = {"table3": run_table3(K, torch, peak)} if args.extras == "table3" else run_extras(K, torch, args.extras, table, case, peak)
        except Exception as exc:  # extras never take the headline down
            extras = {"error": repr(exc)}
    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
        "warmup": max(3, args.warmup), "ms_per_step": ms, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": WORKLOAD, "table_bytes": fkb, "bytes_per_step": nbytes,
                   "l2": "inputs (1.024 GB table, read twice per step) are larger than the 126 MB L2; no flush needed",
                   "storage": "fk_table PACK (channel-major, x innermost, 16-byte padded rows)",
                   "multi_gpu": "replicas only"},
        "frac_of_hbm_peak": value / world / peak, "predictions_per_s": world * case.N / ms * 1e3,
        "roofline": roofline, "cpu_baseline": cpu_baseline, "e2e": e2e,
        "gpu_launches": launches_per_step * args.steps, "clocks": clk.summary(), "extras": extras,
    }
    print(json.dumps(line))
    return 0


def _ncu_traffic():
    """{kernel name: dram__bytes_read.sum + dram__bytes_write.sum per launch} from the committed summary of the
    ncu --set full capture (profiles/r02_traffic.csv: name,dram_read_bytes,dram_write_bytes,ncu kernel name), {} if absent."""
    out = {}
    try:
        with open(os.path.join(ROOT, TRAFFIC_CSV)) as fh:
            for ln in fh:
                c = ln.strip().split(",")
                if len(c) >= 3 and c[0] in STEP_KERNELS:
                    out[c[0]] = int(float(c[1])) + int(float(c[2]))
    except Exception:
        pass
    return out


def _spawn(args, argv):
    """--gpus N > 1 without a torchrun environment: re-execute under torch.distributed.run with N ranks on 127.0.0.1."""
    import socket
    import subprocess
    import torch
    have = torch.cuda.device_count() if torch.cuda.is_available() else 0
    if args.impl != "reference" and have < args.gpus:
        raise SystemExit(f"bench.py: --gpus {args.gpus} but this node has {have} CUDA device(s): refusing to report an "
                         f"N-GPU number from fewer GPUs")
    with socket.socket() as sk:
        sk.bind(("127.0.0.1", 0))
        port = sk.getsockname()[1]
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={args.gpus}",
           "--master-addr", "127.0.0.1", "--master-port", str(port), os.path.abspath(__file__)] + argv
    return subprocess.call(cmd)


def run_sharded(args):
    """--shard rows: BASELINE config 4 (R = 1) with whole tables owned by ranks ('whole tables of a ragged
    group, balanced by bytes').  Step = grouped forward (no exchange) + grouped VJP + the one all-reduce that assembles
    df_cat on every rank.  Total work is fixed as N grows: "scaling": "strong"."""
    import torch
    import torch.distributed as dist
    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device - the FK convolution has no CPU fallback")
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    from paper_1909_10547_b200 import fkconv as K
    from paper_1909_10547_b200 import sharded
    shapes = synth.config4_shapes()
    R = 1
    params = synth.pdf_params(synth.rng_for(4, synth.T_PDF), R)
    plan = sharded.GroupPlan([(int(shapes.N[t]), int(shapes.nx[t]), 14, int(shapes.C[t])) for t in range(shapes.T)], world)
    mine = set(plan.owner_tables[rank])
    cases, fs, gs = [], [], []
    for t in range(shapes.T):
        # tables of other ranks: shapes only (never generated or uploaded); f and g are needed in the global layout
        c = synth.config4_table(t, shapes, R, params, with_fk=t in mine)
        cases.append((K.FK_KIND_HADRONIC, c.fk, c.pairs, c.nfl))
        fs.append(c.f); gs.append(c.g)
    grp = sharded.ShardedFkGroup(cases, R_hint=R)
    f_cat = torch.cat([torch.from_numpy(np.ascontiguousarray(f[:R])).reshape(-1) for f in fs]).cuda()
    g_cat = torch.cat([torch.from_numpy(np.ascontiguousarray(g[:, :R])).reshape(-1) for g in gs]).cuda()
    stream = torch.cuda.current_stream()
    peak, peak_src = _measured_peaks()
    nbytes = 2 * shapes.fk_elements() * 8   # whole job: every table read once per pass, two passes

    def step():
        grp.conv(f_cat, R)
        grp.vjp(f_cat, g_cat, R)

    for _ in range(max(3, args.warmup)):
        step()
    torch.cuda.synchronize()
    if world > 1:
        dist.barrier()
    with ClockSampler(local) as clk:
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(stream)
        for _ in range(args.steps):
            step()
        e1.record(stream)
        e1.synchronize()
        torch.cuda.synchronize()
    if world > 1:
        dist.barrier()
    ms = aggregate_max(e0.elapsed_time(e1) / args.steps, world)
    launches = grp.local.last_launches()
    if rank == 0:
        value = nbytes / ms / 1e6
        print(json.dumps({
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": max(3, args.warmup),
            "ms_per_step": ms, "higher_is_better": True, "scaling": "strong", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": "config4: 60 ragged hadronic tables (14.83 GB) R=1, grouped forward + grouped VJP + all-reduce of df per step",
                       "shard": "rows (whole tables to ranks by FK bytes, LPT greedy)", "tables_on_rank0": len(mine),
                       "l2": "per-rank tables are larger than the 126 MB L2; no flush needed", "multi_gpu": "datapoint-sharded, one all-reduce"},
            "frac_of_hbm_peak": value / world / peak, "roofline": None, "cpu_baseline": None, "e2e": None,
            "gpu_launches_last_call_rank0": launches, "clocks": clk.summary()}))
    grp.destroy()
    if world > 1:
        dist.destroy_process_group()
    return 0


def main(argv=None):
    argv = list(sys.argv[1:] if argv is None else argv)
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=200)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--extras", default="fast", choices=["none", "fast", "all", "table3"])
    ap.add_argument("--shard", default="replicas", choices=["replicas", "rows"])
    ap.add_argument("--no-cpu-baseline", action="store_true")
    args = ap.parse_args(argv)
    if args.gpus < 1:
        raise SystemExit("bench.py: --gpus must be >= 1")
    if args.impl == "reference":
        return run_reference(args)   # rank 0's host cores only; never spawns
    world = int(os.environ.get("WORLD_SIZE", "0") or 0)
    if args.gpus > 1 and world == 0:
        return _spawn(args, argv)
    if world and world != args.gpus:
        raise SystemExit(f"bench.py: --gpus {args.gpus} but WORLD_SIZE={world}")
    if args.shard == "rows":
        return run_sharded(args)
    return run_ours(args)


if __name__ == "__main__":
    sys.exit(main())
