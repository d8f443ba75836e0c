#!/usr/bin/env python
"""bench.py -- documents scored/sec and achieved fraction of the B200 roofline, next to the CPU oracle.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload NAME] [--impl reference]

A "step" is one pass of the hot path over one batch of seeded synthetic input: one tms_maxsim call
(dense workloads) or tms_pq_build_lut + tms_pq_maxsim (PQ workload).  The default workload is
BASELINE.json configs[1] (ColBERT-scale: Q=8, Nq=32, d=128, bf16, B=500,000 documents of Nd=128).  Inputs are
far larger than L2 (126 MB), so consecutive timed steps cannot reuse cached documents.

One JSON line on stdout (rank 0): the driver contract plus `roofline`, `cpu_baseline`, `e2e`, `clocks`.
`--impl reference` times the fp64 CPU oracle, as it stands, on the host cores.
"""
from __future__ import annotations

import argparse
import json
import os
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import numpy as np
import torch

METRIC = "documents scored/sec and achieved HBM GB/s (% of B200 peak) vs CPU oracle"
UNIT = "docs/s"

# name -> parameters.  c2* = configs[1], c3* = configs[2], c4* = configs[3], c5 = configs[4], c1 = configs[0].
WORKLOADS = {
    "c1": dict(kind="dense", Q=1, Nq=32, d=128, dtype="fp32", B=1000, Nd=128, lengths="uniform"),
    "c2": dict(kind="dense", Q=8, Nq=32, d=128, dtype="bf16", B=500_000, Nd=128, lengths="uniform"),
    "c2-fp16": dict(kind="dense", Q=8, Nq=32, d=128, dtype="fp16", B=500_000, Nd=128, lengths="uniform"),
    "c2-fp32": dict(kind="dense", Q=8, Nq=32, d=128, dtype="fp32", B=500_000, Nd=128, lengths="uniform"),
    "c2-q4": dict(kind="dense", Q=4, Nq=32, d=128, dtype="bf16", B=500_000, Nd=128, lengths="uniform"),
    "c2-q1": dict(kind="dense", Q=1, Nq=32, d=128, dtype="bf16", B=500_000, Nd=128, lengths="uniform"),
    "c3-100k": dict(kind="dense", Q=8, Nq=32, d=128, dtype="bf16", B=100_000, Nd=None, lengths="lognormal"),
    "c3-250k": dict(kind="dense", Q=8, Nq=32, d=128, dtype="bf16", B=250_000, Nd=None, lengths="lognormal"),
    "c3-500k": dict(kind="dense", Q=8, Nq=32, d=128, dtype="bf16", B=500_000, Nd=None, lengths="lognormal"),
    "c4-d64": dict(kind="dense", Q=4, Nq=32, d=64, dtype="bf16", B=100_000, Nd=128, lengths="uniform"),
    "c4-d256": dict(kind="dense", Q=4, Nq=32, d=256, dtype="bf16", B=100_000, Nd=128, lengths="uniform"),
    "c4-d512": dict(kind="dense", Q=4, Nq=32, d=512, dtype="bf16", B=100_000, Nd=128, lengths="uniform"),
    "c4-d768": dict(kind="dense", Q=4, Nq=32, d=768, dtype="bf16", B=100_000, Nd=128, lengths="uniform"),
    # NEXT-1: the paper's query-length and document-length sweeps (Tables 10, 11), Q=1 as in the paper
    "n1-nq8": dict(kind="dense", Q=1, Nq=8, d=128, dtype="bf16", B=100_000, Nd=128, lengths="uniform"),
    "n1-nq16": dict(kind="dense", Q=1, Nq=16, d=128, dtype="bf16", B=100_000, Nd=128, lengths="uniform"),
    "n1-nq64": dict(kind="dense", Q=1, Nq=64, d=128, dtype="bf16", B=100_000, Nd=128, lengths="uniform"),
    "n1-b1k": dict(kind="dense", Q=1, Nq=32, d=128, dtype="bf16", B=1_000, Nd=128, lengths="uniform"),
    "n1-b10k": dict(kind="dense", Q=1, Nq=32, d=128, dtype="bf16", B=10_000, Nd=128, lengths="uniform"),
    "n1-b100k": dict(kind="dense", Q=1, Nq=32, d=128, dtype="bf16", B=100_000, Nd=128, lengths="uniform"),
    "n1-nd32": dict(kind="dense", Q=1, Nq=32, d=128, dtype="bf16", B=100_000, Nd=32, lengths="uniform"),
    "n1-nd64": dict(kind="dense", Q=1, Nq=32, d=128, dtype="bf16", B=100_000, Nd=64, lengths="uniform"),
    "n1-nd256": dict(kind="dense", Q=1, Nq=32, d=128, dtype="bf16", B=100_000, Nd=256, lengths="uniform"),
    "n1-nd512": dict(kind="dense", Q=1, Nq=32, d=128, dtype="bf16", B=100_000, Nd=512, lengths="uniform"),
    # NEXT-2: scoring followed by per-query top-100 (the paper's 500K end-to-end case)
    "c2-topk": dict(kind="dense", Q=8, Nq=32, d=128, dtype="bf16", B=500_000, Nd=128, lengths="uniform", topk=100),
    "c2-q1-topk": dict(kind="dense", Q=1, Nq=32, d=128, dtype="bf16", B=500_000, Nd=128, lengths="uniform", topk=100),
    # NEXT-4: the same scores as c5 from the decode-and-contract variant (codebook in shared memory, tensor cores)
    "c5-decode": dict(kind="pq", Q=8, Nq=32, d=128, dtype="bf16", B=1_000_000, Nd=128, lengths="uniform", M=16, K=256,
                      decode=True),
    "c5": dict(kind="pq", Q=8, Nq=32, d=128, dtype="bf16", B=1_000_000, Nd=128, lengths="uniform", M=16, K=256),
}
TORCH_DTYPES = {"bf16": torch.bfloat16, "fp16": torch.float16, "fp32": torch.float32}
ELEM_BYTES = {"bf16": 2, "fp16": 2, "fp32": 4}
FALLBACK_HBM_GBS = 6650.0  # /opt/skills/guides/B200_PROFILING.md, used only when MEASURED_PEAKS.json is absent
FALLBACK_BF16_TFLOPS = 1590.0
FALLBACK_BF16_TFLOPS_SUSTAINED = 1400.0
SMEM_PIPE_PEAK_GBS = 148 * 128 * 1.965  # shared-memory load pipe: SMs x bytes/clk x max SM clock (GHz) = 37,229 GB/s


# ---- inputs ----------------------------------------------------------------------------------------------------------

def make_offsets(w, B, seed):
    from paper_2606_26439_b200 import synth

    if w["lengths"] == "uniform":
        return synth.uniform_offsets(B, w["Nd"])
    return synth.offsets_from_lengths(synth.lognormal_lengths(B, seed=seed))


def make_inputs(w, B, seed, device):
    """Seeded synthetic inputs for workload `w` with B documents."""
    from paper_2606_26439_b200 import synth

    dt = TORCH_DTYPES[w["dtype"]]
    off = make_offsets(w, B, seed)
    T = int(off[-1])
    q = synth.unit_tokens(w["Q"] * w["Nq"], w["d"], dt, seed=seed + 1, device=device).view(w["Q"], w["Nq"], w["d"])
    if w["kind"] == "dense":
        store = synth.unit_tokens(T, w["d"], dt, seed=seed + 2, device=device)
        return dict(q=q, off=off, store=store, T=T)
    C = synth.pq_codebooks(w["M"], w["K"], w["d"] // w["M"], seed=seed + 3).to(device)
    codes = synth.pq_codes(T, w["M"], seed=seed + 4, device=device, K=w["K"])
    return dict(q=q, off=off, store=codes, C=C, T=T)


def algorithmic_bytes(w, T, B):
    from paper_2606_26439_b200 import accounting

    if w["kind"] == "dense":
        return accounting.dense_bytes(w["Q"], w["Nq"], w["d"], T, B, ELEM_BYTES[w["dtype"]])
    return accounting.pq_bytes(w["Q"], w["Nq"], w["M"], w["K"], T, B)


# ---- clocks ----------------------------------------------------------------------------------------------------------

class ClockSampler:
    """Samples SM clock and throttle reasons of one GPU through NVML while the timed region runs."""

    REASONS = {0x1: "gpu_idle", 0x2: "applications_clocks_setting", 0x4: "sw_power_cap", 0x8: "hw_slowdown",
               0x10: "sync_boost", 0x20: "sw_thermal_slowdown", 0x40: "hw_thermal_slowdown",
               0x80: "hw_power_brake_slowdown", 0x100: "display_clock_setting"}

    def __init__(self, device_index: int, period_s: float = 0.005):
        self.period, self.samples, self.mask, self.h, self.max_mhz = period_s, [], 0, None, None
        self._stop = threading.Event()
        self._thread = None
        try:
            import pynvml

            pynvml.nvmlInit()
            uuid = str(torch.cuda.get_device_properties(device_index).uuid)
            uuid = uuid if uuid.startswith("GPU-") else "GPU-" + uuid
            try:
                self.h = pynvml.nvmlDeviceGetHandleByUUID(uuid.encode())
            except Exception:
                self.h = pynvml.nvmlDeviceGetHandleByIndex(device_index)
            self.nv = pynvml
            self.max_mhz = int(pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM))
        except Exception:
            self.h = None

    def _run(self):
        while not self._stop.is_set():
            try:
                self.samples.append(int(self.nv.nvmlDeviceGetClockInfo(self.h, self.nv.NVML_CLOCK_SM)))
                self.mask |= int(self.nv.nvmlDeviceGetCurrentClocksEventReasons(self.h))
            except Exception:
                pass
            time.sleep(self.period)

    def start(self):
        if self.h is not None:
            self._thread = threading.Thread(target=self._run, daemon=True)
            self._thread.start()

    def stop(self):
        if self._thread is not None:
            self._stop.set()
            self._thread.join()
        reasons = [name for bit, name in self.REASONS.items() if self.mask & bit and name != "gpu_idle"]
        med = int(np.median(self.samples)) if self.samples else None
        return {"sm_mhz": med, "sm_max_mhz": self.max_mhz, "reasons": reasons, "samples": len(self.samples)}


# ---- the CPU oracle legs (the only places bench.py touches oracle/) --------------------------------------------------

def oracle_time(w, q, store, off, C=None):
    import oracle

    t0 = time.perf_counter()
    if w["kind"] == "dense":
        _, used = oracle.maxsim(q, store, off, return_threads=True)
    else:
        _, used = oracle.pq_maxsim(q, C, store, off, return_threads=True)
    return time.perf_counter() - t0, used


def oracle_sample(w, inp, n_docs):
    """First n_docs documents of the workload as host tensors."""
    off = inp["off"][:n_docs + 1].copy()
    t_hi = int(off[-1])
    store = inp["store"][:t_hi].cpu()
    C = inp["C"].cpu() if "C" in inp else None
    return inp["q"].cpu(), store, off, C


def cpu_baseline(w, inp, B, target_s=15.0):
    """The oracle, as it stands, on a bounded prefix of the same workload (about target_s of CPU work)."""
    n0 = min(B, 500)
    q, store, off, C = oracle_sample(w, inp, n0)
    t, used = oracle_time(w, q, store, off, C)
    n = int(max(n0, min(B, n0 * target_s / max(t, 1e-6))))
    if n > n0:
        q, store, off, C = oracle_sample(w, inp, n)
        t, used = oracle_time(w, q, store, off, C)
    return {"value": n / t, "unit": UNIT, "cores": int(used), "kind": "oracle",
            "sample": f"first {n} of {B} documents of the same store, all {w['Q']} queries, {t:.2f} s wall, "
                      f"fp64, OpenMP over documents"}


def run_reference(args, w, rank):
    """--impl reference: the oracle on the host cores; rank 0 only."""
    if rank != 0:
        return
    from paper_2606_26439_b200 import synth  # input generators only

    import oracle

    B = args.B or w["B"]
    # calibrate the per-step sample so that steps + warmup end within ~2 minutes
    small = dict(w)
    n0 = min(B, 300)
    inp = make_inputs(small, n0, args.seed, "cpu")
    t, used = oracle_time(w, inp["q"], inp["store"], inp["off"], inp.get("C"))
    budget = 120.0 / max(1, args.steps + args.warmup)
    n = int(max(50, min(B, n0 * budget / max(t, 1e-6))))
    inp = make_inputs(small, n, args.seed, "cpu")
    for _ in range(args.warmup):
        oracle_time(w, inp["q"], inp["store"], inp["off"], inp.get("C"))
    t0 = time.perf_counter()
    for _ in range(args.steps):
        _, used = oracle_time(w, inp["q"], inp["store"], inp["off"], inp.get("C"))
    el = time.perf_counter() - t0
    value = n * args.steps / el
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": 1e3 * el / args.steps, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": config_dict(args, w, B, int(make_offsets(w, B, args.seed)[-1]), sample_docs_per_step=n),
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": int(used), "kind": "oracle",
                         "sample": f"{n} documents per step (same recipe as the workload), all {w['Q']} queries, fp64"},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    _ = oracle, synth
    print(json.dumps(line), flush=True)


def config_dict(args, w, B, T, **extra):
    c = {"workload": f"{args.workload}: " + ("dense MaxSim" if w["kind"] == "dense" else "fused PQ MaxSim"),
         "Q": w["Q"], "Nq": w["Nq"], "d": w["d"], "store_dtype": w["dtype"], "B_per_gpu": B, "total_tokens_per_gpu": T,
         "lengths": ("uniform Nd=%d" % w["Nd"]) if w["lengths"] == "uniform" else "lognormal(median 64, sigma 0.5) clip [8,180]",
         "l2": "inputs larger than L2 (no flush needed)" if T * w["d"] * ELEM_BYTES[w["dtype"]] > (512 << 20) or
               (w["kind"] == "pq" and T * w.get("M", 0) > (512 << 20)) else "L2 flushed between timed steps",
         "parallelism": f"dp{args.gpus} (documents sharded, no data-path collective)"}
    if w["kind"] == "pq":
        c.update({"M": w["M"], "K": w["K"]})
    c.update(extra)
    return c


# ---- the CUDA arm ----------------------------------------------------------------------------------------------------

def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=50)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--workload", default="c2", choices=sorted(WORKLOADS))
    ap.add_argument("--impl", default="tms", choices=["tms", "reference"])
    ap.add_argument("--B", type=int, default=0, help="override the number of documents per GPU")
    ap.add_argument("--variant", default="auto")
    ap.add_argument("--seed", type=int, default=0)
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-cpu", action="store_true")
    ap.add_argument("--e2e-steps", type=int, default=3)
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3) if args.impl == "tms" else args.warmup
    w = WORKLOADS[args.workload]

    rank = int(os.environ.get("RANK", "0"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))

    if args.impl == "reference":
        run_reference(args, w, rank)
        return

    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (there is no CPU fallback; use --impl reference for the oracle)")
    import torch.distributed as dist

    from paper_2606_26439_b200 import build as tms_build
    from paper_2606_26439_b200 import shard, tms

    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    if world > 1:
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        dist.init_process_group("nccl", device_id=dev)
    if rank == 0:
        tms_build.build()
    if world > 1:
        dist.barrier()
    tms.load()

    B = args.B or w["B"]
    inp = make_inputs(w, B, args.seed + 1000 * rank, dev)  # weak scaling: every rank owns its own B-document shard
    T = inp["T"]
    off_d = torch.from_numpy(inp["off"]).to(dev)
    scores = torch.empty((w["Q"], B), dtype=torch.float32, device=dev)
    flush = None
    small = "flushed" in config_dict(args, w, B, T)["l2"]
    if small:
        flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev)

    if w["kind"] == "dense":
        need = tms.tms_maxsim_workspace_bytes(w["Q"], w["Nq"], w["d"], B, TORCH_DTYPES[w["dtype"]])
        dws = torch.empty(need, dtype=torch.uint8, device=dev) if need else None  # only queries longer than 32 tokens

        k = w.get("topk", 0)
        if k:
            tk_v = torch.empty((w["Q"], k), dtype=torch.float32, device=dev)
            tk_i = torch.empty((w["Q"], k), dtype=torch.int64, device=dev)
            tk_ws = torch.empty(max(tms.tms_topk_workspace_bytes(w["Q"], B, k), 8), dtype=torch.uint8, device=dev)

        def step():
            tms.tms_maxsim(inp["q"], inp["store"], off_d, scores=scores, variant=args.variant, workspace=dws)
            if k:
                tms.tms_topk(scores, k, values=tk_v, indices=tk_i, workspace=tk_ws)
    else:
        lut = torch.empty((w["Q"], w["Nq"], w["M"], w["K"]), dtype=torch.float32, device=dev)
        ws = torch.empty(max(tms.tms_pq_workspace_bytes(w["Q"], w["Nq"], w["M"], w["K"], B), 16), dtype=torch.uint8,
                         device=dev)

        if w.get("decode"):
            def step():
                tms.tms_pq_maxsim_decode(inp["q"], inp["C"], inp["store"], off_d, scores=scores)
        else:
            def step():
                tms.tms_pq_build_lut(inp["q"], inp["C"], lut=lut)
                tms.tms_pq_maxsim(lut, inp["store"], off_d, scores=scores, workspace=ws, variant=args.variant)

    def sync_all():
        torch.cuda.synchronize()
        if world > 1:
            dist.barrier()
            torch.cuda.synchronize()

    for _ in range(args.warmup):
        step()
    sync_all()

    # ---- timed region: exactly K steps; per-step CUDA events on the launching stream --------------------------------
    sampler = ClockSampler(local_rank)
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(args.steps)]
    t_start, t_end = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    n0 = tms.tms_launch_count()
    sampler.start()
    sync_all()
    t_start.record()
    for a, b in ev:
        if flush is not None:
            flush.fill_(1)
        a.record()
        step()
        b.record()
    t_end.record()
    sync_all()
    clocks = sampler.stop()
    launches = tms.tms_launch_count() - n0
    step_ms = np.array([a.elapsed_time(b) for a, b in ev])
    total_ms = float(step_ms.sum()) if flush is not None else float(t_start.elapsed_time(t_end))
    total_ms = shard.max_over_ranks(total_ms, dev)
    ms_per_step = total_ms / args.steps
    value = world * B / (ms_per_step * 1e-3)

    # ---- roofline of the dominant kernel ------------------------------------------------------------------------------
    # Each step is timed alone (events around one call), so the burst peaks of MEASURED_PEAKS.json apply.
    from paper_2606_26439_b200 import accounting

    peaks_path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(peaks_path):
        pk = json.load(open(peaks_path))
        hbm_peak, tc_peak, peak_src = float(pk["hbm_gbs"]), float(pk["bf16_tflops"]), "MEASURED_PEAKS.json (of measured)"
        tc_sustained = float(pk.get("bf16_tflops_sustained", tc_peak))
    else:
        hbm_peak, tc_peak, peak_src = FALLBACK_HBM_GBS, FALLBACK_BF16_TFLOPS, "B200_PROFILING.md fallback (of fallback)"
        tc_sustained = FALLBACK_BF16_TFLOPS_SUSTAINED
    # Tensor peak by regime (B200_PROFILING.md): the burst figure for kernels timed alone; when the timed region is a
    # long back-to-back loop that ran under the power cap -- the regime of the sustained cuBLAS measurement -- the
    # sustained figure.  The HBM peak is the measured copy rate in both regimes.
    tc_regime = "burst"
    if total_ms > 100.0 and "sw_power_cap" in clocks.get("reasons", []):
        tc_peak, tc_regime = tc_sustained, "sustained (timed region %.0f ms under sw_power_cap)" % total_ms
    peak_src += ", tensor peak: " + tc_regime
    abytes = algorithmic_bytes(w, T, B)
    kern_ms = float(step_ms.mean())
    kern_s = kern_ms * 1e-3
    hbm_gbs = abytes / kern_s / 1e9
    traffic = None
    tpath = os.path.join(ROOT, "profiles", "traffic.csv")  # ncu dram__bytes_read.sum + dram__bytes_write.sum per launch
    if os.path.exists(tpath):
        for ln in open(tpath).read().splitlines()[1:]:
            name, _, val = ln.partition(",")
            if name == args.workload:
                traffic = int(val)
    common = {"traffic": traffic, "peak_source": peak_src, "algorithmic_bytes_per_launch": abytes,
              "kernel_ms_mean": kern_ms, "kernel_ms_min": float(step_ms.min()),
              "kernel_ms_median": float(np.median(step_ms)),
              "hbm": {"achieved_GBps": hbm_gbs, "peak_GBps": hbm_peak, "frac": hbm_gbs / hbm_peak,
                      "frac_of_nominal_8000": hbm_gbs / 8000.0}}
    if w["kind"] == "dense":
        # tensor work: 2*Q*Nq*T*d algorithmic FLOP; fp32 inputs cost three bf16 MMAs per product, so
        # their tensor peak is a third of the bf16 peak.  The roofline that binds is the one with the larger ideal time.
        fl = accounting.dense_flops(w["Q"], w["Nq"], w["d"], T)
        tc_eff_peak = tc_peak / (3.0 if w["dtype"] == "fp32" else 1.0)
        tfl = fl / kern_s / 1e12
        common["tensor"] = {"achieved_TFLOPs": tfl, "peak_TFLOPs": tc_eff_peak, "frac": tfl / tc_eff_peak,
                            "algorithmic_flops_per_launch": fl}
        if fl / (tc_eff_peak * 1e12) > abytes / (hbm_peak * 1e9):
            roofline = {"bound": "tensor", "achieved": tfl, "peak": tc_eff_peak, "unit": "TFLOP/s",
                        "frac": tfl / tc_eff_peak}
        else:
            roofline = {"bound": "hbm", "achieved": hbm_gbs, "peak": hbm_peak, "unit": "GB/s", "frac": hbm_gbs / hbm_peak}
        roofline["tensor_tflops"] = tfl
        if w["Q"] * w["Nq"] > 128 and w["dtype"] != "fp32":
            roofline["note"] = ("two query blocks: HBM and tensor ideal times are within 1 % of each other at the burst peaks; the "
                                "kernel's read stream alone draws 750-950 W of the 1000 W cap, so the tensor pipe runs at a "
                                "power-capped SM clock of ~1.3 GHz (~1.05 GHz sustained) and binds (DESIGN.md 5.1)")
    elif w.get("decode"):
        # decode-and-contract PQ: 2*Q*Nq*T*d FLOP at two bf16 MMAs per product for bf16 queries (hi*hi + hi*lo)
        fl = accounting.dense_flops(w["Q"], w["Nq"], w["d"], T)
        tc_eff_peak = tc_peak / 2.0
        tfl = fl / kern_s / 1e12
        roofline = {"bound": "tensor", "achieved": tfl, "peak": tc_eff_peak, "unit": "TFLOP/s", "frac": tfl / tc_eff_peak,
                    "note": "codes decoded in shared memory and contracted on tcgen05; two bf16 MMAs per product "
                            "(centroids split hi/lo), so the tensor peak is half the bf16 peak (DESIGN.md 10)"}
    else:
        # fused PQ: Q*Nq*T*M four-byte shared-memory gathers against M bytes of codes per token -- bound by the
        # shared-memory load pipe (128 B/clk/SM), not by HBM and not by tensor cores
        lookups = accounting.pq_lookups(w["Q"], w["Nq"], w["M"], T)
        smem_peak = SMEM_PIPE_PEAK_GBS
        g = lookups * 4 / kern_s / 1e9
        roofline = {"bound": "alu", "achieved": g, "peak": smem_peak, "unit": "GB/s", "frac": g / smem_peak,
                    "note": "shared-memory gather bytes/s against 148 SMs x 128 B/clk x 1.965 GHz; step = LUT build + "
                            "relayout + fused lookup kernel (DESIGN.md 5.4)"}
    roofline.update(common)

    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": w["dtype"] if w["kind"] == "dense" else "f32", "data": "synthetic",
        "config": config_dict(args, w, B, T), "pairs_per_s": value * w["Q"],
        "roofline": roofline, "clocks": clocks, "gpu_launches": int(launches),
    }

    # ---- end to end through the host-buffer entry point: H2D of the store + D2H of the scores every step -------------
    if not args.no_e2e:
        if w.get("decode"):  # no host-buffer entry point for the decode variant: its end-to-end number is c5's copy-bound one
            line["e2e"] = {"value": None, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0,
                           "unavailable": "tms_pq_maxsim_decode has no host-buffer entry point; see workload c5"}
        else:
            line["e2e"] = run_e2e(args, w, inp, B, T, dev, world, tms, shard)
    if rank == 0 and not args.no_cpu and world >= 1:
        line["cpu_baseline"] = cpu_baseline(w, inp, B)
    if world > 1:
        dist.barrier()
        dist.destroy_process_group()
    if rank == 0:
        print(json.dumps(line), flush=True)


def run_e2e(args, w, inp, B, T, dev, world, tms, shard):
    row = w["d"] * ELEM_BYTES[w["dtype"]] if w["kind"] == "dense" else w["M"]
    try:
        import psutil

        avail = psutil.virtual_memory().available
    except Exception:
        avail = 64 << 30
    budget = int(min(avail * 0.4, 96 << 30) / max(world, 1))
    Be = B
    if T * row > budget:  # host memory cannot pin the whole shard: use a document prefix and say so
        Be = max(1, int(B * budget / (T * row)))
    off_h = torch.from_numpy(inp["off"][:Be + 1].copy())
    Te = int(off_h[-1])
    store_h = torch.empty((Te, inp["store"].shape[1]), dtype=inp["store"].dtype, pin_memory=True)
    store_h.copy_(inp["store"][:Te])
    q_h = inp["q"].cpu().pin_memory()
    scores_h = torch.empty((w["Q"], Be), dtype=torch.float32, pin_memory=True)
    ws = torch.empty(2 << 30, dtype=torch.uint8, device=dev)
    if w["kind"] == "dense":
        def call():
            tms.tms_maxsim_host(q_h, store_h, off_h, scores_h, ws)
        h2d = q_h.numel() * q_h.element_size() + Te * row + (Be + 1) * 8
    else:
        C_h = inp["C"].cpu().pin_memory()

        def call():
            tms.tms_pq_maxsim_host(q_h, C_h, store_h, off_h, scores_h, ws)
        h2d = q_h.numel() * q_h.element_size() + C_h.numel() * 4 + Te * row + (Be + 1) * 8
    d2h = w["Q"] * Be * 4
    call()
    torch.cuda.synchronize()
    if world > 1:
        torch.distributed.barrier()
    t0 = time.perf_counter()
    a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    a.record()
    for _ in range(args.e2e_steps):
        call()  # returns after the scores have landed in host memory
    b.record()
    torch.cuda.synchronize()
    ms = shard.max_over_ranks(max(a.elapsed_time(b), 1e3 * (time.perf_counter() - t0)), dev)
    return {"value": world * Be * args.e2e_steps / (ms * 1e-3), "unit": UNIT, "h2d_bytes_per_step": int(h2d),
            "d2h_bytes_per_step": int(d2h), "steps": args.e2e_steps, "docs_per_step_per_gpu": Be,
            "api": "tms_maxsim_host" if w["kind"] == "dense" else "tms_pq_maxsim_host",
            "ms_per_step": ms / args.e2e_steps}


if __name__ == "__main__":
    main()
