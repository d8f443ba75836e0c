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
    # the dimension sweep at Q=8: two query blocks do not fit tensor memory next to the accumulators for d > 256, so the
    # kernel runs as CTA pairs that share every document tile by TMA multicast (the store is still read once)
    "c4-d512-q8": dict(kind="dense", Q=8, Nq=32, d=512, dtype="bf16", B=100_000, Nd=128, lengths="uniform"),
    "c4-d768-q8": dict(kind="dense", Q=8, Nq=32, d=768, dtype="bf16", B=100_000, Nd=128, lengths="uniform"),
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
    "c5-decode-fp16": dict(kind="pq", Q=8, Nq=32, d=128, dtype="bf16", B=1_000_000, Nd=128, lengths="uniform", M=16,
                           K=256, decode=True, precision="fp16"),
    # configs[4] through tms_pq_maxsim as a caller gets it (TMS_VARIANT_AUTO: the paper's fp32 table, in shared
    # memory); the kernel name and bytes per entry come from tms_pq_maxsim_variant_used, not from this table
    "c5": dict(kind="pq", Q=8, Nq=32, d=128, dtype="bf16", B=1_000_000, Nd=128, lengths="uniform", M=16, K=256),
    # the opt-in LUT kernel over fp16 table entries (SURVEY 7.3 H6's A/B: half the shared-memory gather bytes, lossy)
    "c5-f16": dict(kind="pq", Q=8, Nq=32, d=128, dtype="bf16", B=1_000_000, Nd=128, lengths="uniform", M=16, K=256,
                   pq_variant="pq_smem_f16"),
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
        self.power, self.power_limit = [], None
        self.stamps, self.masks = [], []  # host time and throttle-reason mask of every sample
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
            try:
                self.power_limit = pynvml.nvmlDeviceGetEnforcedPowerLimit(self.h) / 1000.0
            except Exception:
                self.power_limit = None
        except Exception:
            self.h = None

    def _run(self):
        while not self._stop.is_set():
            try:
                mhz = int(self.nv.nvmlDeviceGetClockInfo(self.h, self.nv.NVML_CLOCK_SM))
                mask = int(self.nv.nvmlDeviceGetCurrentClocksEventReasons(self.h))
                pw = self._power_w()
                self.stamps.append(time.perf_counter())
                self.samples.append(mhz)
                self.masks.append(mask)
                self.power.append(pw)
            except Exception:
                pass
            time.sleep(self.period)

    def _power_w(self):
        """Instantaneous board power when the driver exposes it (NVML_FI_DEV_POWER_INSTANT), else the ~1 s average."""
        try:
            fid = getattr(self.nv, "NVML_FI_DEV_POWER_INSTANT", 186)
            v = self.nv.nvmlDeviceGetFieldValues(self.h, [fid])[0]
            if v.nvmlReturn == 0 and v.value.uiVal > 0:
                self.power_kind = "instant"
                return v.value.uiVal / 1000.0
        except Exception:
            pass
        self.power_kind = "1 s average"
        return self.nv.nvmlDeviceGetPowerUsage(self.h) / 1000.0

    def start(self):
        if self.h is not None:
            self._thread = threading.Thread(target=self._run, daemon=True)
            self._thread.start()

    def stop(self, t_first=None, t_last=None):
        """Ends sampling.  With [t_first, t_last] (host times between which the GPU was running the timed steps) only the
        samples taken inside that window count: a sample read before the first step started shows the idle board."""
        if self._thread is not None:
            self._stop.set()
            self._thread.join()
        if t_first is not None:
            keep = [i for i, t in enumerate(self.stamps) if t_first <= t <= t_last]
            self.samples = [self.samples[i] for i in keep]
            self.power = [self.power[i] for i in keep]
            self.masks = [self.masks[i] for i in keep]
        self.mask = 0
        for m in self.masks:
            self.mask |= m
        reasons = [name for bit, name in self.REASONS.items() if self.mask & bit and name != "gpu_idle"]
        med = int(np.median(self.samples)) if self.samples else None
        out = {"sm_mhz": med, "sm_max_mhz": self.max_mhz, "reasons": reasons, "samples": len(self.samples)}
        if self.power:
            out.update({"power_w_mean": float(np.mean(self.power)), "power_w_max": float(np.max(self.power)),
                        "power_limit_w": self.power_limit, "power_kind": getattr(self, "power_kind", None)})
        return out


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
        "config": config_dict(args, w, B, int(make_offsets(w, B, args.seed)[-1]), 1, sample_docs_per_step=n),
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": int(used), "kind": "oracle",
                         "sample": f"{n} documents per step (same recipe as the workload), all {w['Q']} queries, fp64"},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    _ = oracle, synth
    print(json.dumps(line), flush=True)


def config_dict(args, w, B, T, world=1, **extra):
    c = {"workload": f"{args.workload}: " + ("dense MaxSim" if w["kind"] == "dense" else "fused PQ MaxSim"),
         "Q": w["Q"], "Nq": w["Nq"], "d": w["d"], "store_dtype": w["dtype"], "B_per_gpu": B, "total_tokens_per_gpu": T,
         "lengths": ("uniform Nd=%d" % w["Nd"]) if w["lengths"] == "uniform" else "lognormal(median 64, sigma 0.5) clip [8,180]",
         "l2": config_l2(w, T),
         "parallelism": f"dp{world} (one process per GPU, documents sharded, no data-path collective)"}
    if w["kind"] == "pq":
        c.update({"M": w["M"], "K": w["K"]})
    c.update(extra)
    return c


# ---- the CUDA arm ----------------------------------------------------------------------------------------------------

def load_peaks():
    peaks_path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(peaks_path):
        pk = json.load(open(peaks_path))
        return {"hbm": float(pk["hbm_gbs"]), "tc_burst": float(pk["bf16_tflops"]),
                "tc_sustained": float(pk.get("bf16_tflops_sustained", pk["bf16_tflops"])),
                "source": "MEASURED_PEAKS.json (HBM: device-to-device copy rate, read+write bytes; tensor: cuBLAS bf16 8192^3)"}
    return {"hbm": FALLBACK_HBM_GBS, "tc_burst": FALLBACK_BF16_TFLOPS, "tc_sustained": FALLBACK_BF16_TFLOPS_SUSTAINED,
            "source": "B200_PROFILING.md fallback"}


def profiled_traffic(name):
    """DRAM bytes per launch from the committed ncu capture (not measured in this run): (bytes, source) or (None, None)."""
    tpath = os.path.join(ROOT, "profiles", "traffic.csv")
    if not os.path.exists(tpath):
        return None, None
    lines = open(tpath).read().splitlines()
    src = "profiles/traffic.csv (ncu dram__bytes_read.sum + dram__bytes_write.sum, one launch; %s)" % (
        lines[0].split("#", 1)[1].strip() if "#" in lines[0] else "see profiles/*.md for the capture")
    for ln in lines[1:]:
        nm, _, val = ln.partition(",")
        if nm == name:
            return int(val), src
    return None, None


class Workload:
    """One workload's device-resident inputs and its step function (one pass of the hot path through the C ABI)."""

    def __init__(self, name, w, B, seed, dev, tms, variant="auto", reuse=None):
        self.name, self.w, self.B, self.dev, self.tms = name, w, B, dev, tms
        if reuse is not None and reuse.w["kind"] == w["kind"] == "dense" and reuse.B == B and \
                all(reuse.w[k] == w[k] for k in ("d", "dtype", "lengths", "Nd")):
            # same store (same recipe, seed and shape); only the queries differ
            from paper_2606_26439_b200 import synth

            q = synth.unit_tokens(w["Q"] * w["Nq"], w["d"], TORCH_DTYPES[w["dtype"]], seed=seed + 1,
                                  device=dev).view(w["Q"], w["Nq"], w["d"])
            self.inp = dict(reuse.inp, q=q)
        else:
            self.inp = make_inputs(w, B, seed, dev)
        inp = self.inp
        self.T = inp["T"]
        self.off_d = torch.from_numpy(inp["off"]).to(dev)
        self.scores = torch.empty((w["Q"], B), dtype=torch.float32, device=dev)
        self.l2 = config_l2(w, self.T)
        self.flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev) if "flushed" in self.l2 else None
        Q, Nq, d = w["Q"], w["Nq"], w["d"]
        if w["kind"] == "dense":
            need = tms.tms_maxsim_workspace_bytes(Q, Nq, d, B, TORCH_DTYPES[w["dtype"]])
            dws = torch.empty(need, dtype=torch.uint8, device=dev) if need else None  # only queries longer than 32 tokens
            k = w.get("topk", 0)
            if k:
                tk_v = torch.empty((Q, k), dtype=torch.float32, device=dev)
                tk_i = torch.empty((Q, k), dtype=torch.int64, device=dev)
                tk_ws = torch.empty(max(tms.tms_topk_workspace_bytes(Q, B, k), 8), dtype=torch.uint8, device=dev)

            def step():
                tms.tms_maxsim(inp["q"], inp["store"], self.off_d, scores=self.scores, variant=variant, workspace=dws)
                if k:
                    tms.tms_topk(self.scores, k, values=tk_v, indices=tk_i, workspace=tk_ws)
            self.kernel = tms.tms_maxsim_variant_used(Q, Nq, d, B, self.T, TORCH_DTYPES[w["dtype"]]) \
                if variant == "auto" else variant
        elif w.get("decode"):
            def step():
                tms.tms_pq_maxsim_decode(inp["q"], inp["C"], inp["store"], self.off_d, scores=self.scores,
                                         precision=w.get("precision", "split_bf16"))
            self.kernel = "tcgen05 (decode-and-contract, %s operands)" % w.get("precision", "split_bf16")
        else:
            lut = torch.empty((Q, Nq, w["M"], w["K"]), dtype=torch.float32, device=dev)
            ws = torch.empty(max(tms.tms_pq_workspace_bytes(Q, Nq, w["M"], w["K"], B), 16), dtype=torch.uint8, device=dev)

            # "c5" calls with variant "auto" and asks the library what that runs; "c5-f16" opts into fp16 entries
            pq_variant = variant if variant != "auto" else w.get("pq_variant", "auto")

            def step():
                tms.tms_pq_build_lut(inp["q"], inp["C"], lut=lut)
                tms.tms_pq_maxsim(lut, inp["store"], self.off_d, scores=self.scores, workspace=ws, variant=pq_variant)
            self.kernel = tms.tms_pq_maxsim_variant_used(Q, Nq, w["M"], w["K"]) if pq_variant == "auto" else pq_variant
            self.entry_bytes = 2 if self.kernel == "pq_smem_f16" else 4
        self.step = step


def config_l2(w, T):
    big = T * w["d"] * ELEM_BYTES[w["dtype"]] > (512 << 20) or (w["kind"] == "pq" and T * w.get("M", 0) > (512 << 20))
    return "inputs larger than L2 (no flush needed)" if big else "L2 flushed between timed steps"


def timed_region(wl, steps, warmup, local_rank, sync_all, shard, min_ms=0.0, max_steps=2000):
    """W warm-up steps, then exactly K steps with per-step CUDA events on the launching stream; clocks, throttle reasons and
    board power are sampled through NVML while the steps run (samples taken before the first step starts or after the
    last one ends are dropped).  min_ms > 0 (secondary workloads): K is raised until the region lasts about min_ms, so
    that the 5 ms NVML sampler sees it (at most max_steps); a region that still comes out short is timed again with K
    scaled up.  Returns per-step times and the max-over-ranks total."""
    for _ in range(warmup):
        wl.step()
    sync_all()
    if min_ms > 0:  # a few more untimed steps, measured, to size the region (flush included; first-call costs excluded)
        w0, w1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        w0.record()
        for _ in range(5):
            if wl.flush is not None:
                wl.flush.fill_(1)
            wl.step()
        w1.record()
        sync_all()
        est = max(w0.elapsed_time(w1) / 5, 1e-3)
        steps = int(min(max_steps, max(steps, np.ceil(min_ms / est))))
    for _attempt in range(3):
        out = _timed_steps(wl, steps, local_rank, sync_all, shard)
        region_ms = out[4]
        if min_ms <= 0 or region_ms >= 0.7 * min_ms or steps >= max_steps:
            break
        steps = int(min(max_steps, np.ceil(steps * 1.1 * min_ms / max(region_ms, 1e-3))))
    return out[:4]


def _timed_steps(wl, steps, local_rank, sync_all, shard):
    sampler = ClockSampler(local_rank)
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(steps)]
    t_start, t_end = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    n0 = wl.tms.tms_launch_count()
    sampler.start()
    sync_all()
    t_first = time.perf_counter() + 1e-3  # the GPU is idle here: the first step starts as soon as it is enqueued
    t_start.record()
    for a, b in ev:
        if wl.flush is not None:
            wl.flush.fill_(1)
        a.record()
        wl.step()
        b.record()
    t_end.record()
    torch.cuda.synchronize()
    t_last = time.perf_counter()
    sync_all()
    clocks = sampler.stop(t_first, t_last)
    launches = wl.tms.tms_launch_count() - n0
    step_ms = np.array([a.elapsed_time(b) for a, b in ev])
    region_ms = float(t_start.elapsed_time(t_end))  # flushes included: what the clock sampler saw
    total_ms = float(step_ms.sum()) if wl.flush is not None else region_ms
    _, total_ms = shard.aggregate_throughput(1.0, total_ms, wl.dev)  # MAX over ranks of the device-timed region
    return step_ms, total_ms, clocks, int(launches), region_ms


def roofline_of(wl, step_ms, total_ms, clocks, peaks):
    """The binding roofline of the dominant kernel: algorithmic bytes (or FLOP) per launch / mean launch time."""
    from paper_2606_26439_b200 import accounting

    w, T, B = wl.w, wl.T, wl.B
    hbm_peak, tc_burst, tc_sust = peaks["hbm"], peaks["tc_burst"], peaks["tc_sustained"]
    abytes = algorithmic_bytes(w, T, B)
    kern_ms = float(step_ms.mean())
    kern_s = kern_ms * 1e-3
    hbm_gbs = abytes / kern_s / 1e9
    traffic, traffic_src = profiled_traffic(wl.name)
    common = {"traffic": traffic, "traffic_source": traffic_src, "peak_source": peaks["source"],
              "algorithmic_bytes_per_launch": abytes, "kernel": wl.kernel,
              "kernel_ms_mean": kern_ms, "kernel_ms_min": float(step_ms.min()), "kernel_ms_median": float(np.median(step_ms)),
              "hbm": {"achieved_GBps": hbm_gbs, "peak_GBps": hbm_peak, "frac": hbm_gbs / hbm_peak,
                      "frac_of_nominal_8000": hbm_gbs / 8000.0, "ideal_ms": abytes / (hbm_peak * 1e9) * 1e3}}
    notes = []
    if hbm_gbs > hbm_peak:
        notes.append("achieved exceeds the HBM 'peak' because that figure is a copy rate (reads + writes share the bus "
                     "and turn it around) while this kernel only reads")
    if w["kind"] == "dense" or w.get("decode"):
        # tensor work: 2*Q*Nq*T*d algorithmic FLOP.  fp32 inputs cost three bf16 MMAs per product, the PQ
        # decode variant two (bf16 queries), so their tensor peaks are a third / half of the bf16 peak.
        fl = accounting.dense_flops(w["Q"], w["Nq"], w["d"], T)
        div = (1.0 if w.get("precision") == "fp16" else 2.0) if w.get("decode") else (3.0 if w["dtype"] == "fp32" else 1.0)
        tfl = fl / kern_s / 1e12
        common["tensor"] = {"achieved_TFLOPs": tfl, "mma_per_product": div, "algorithmic_flops_per_launch": fl,
                            "peak_TFLOPs_burst": tc_burst / div, "frac_burst": tfl / (tc_burst / div),
                            "peak_TFLOPs_sustained": tc_sust / div, "frac_sustained": tfl / (tc_sust / div),
                            "ideal_ms_burst": fl / (tc_burst / div * 1e12) * 1e3}
        if w.get("decode") or fl / (tc_burst / div * 1e12) > abytes / (hbm_peak * 1e9):
            roofline = {"bound": "tensor", "achieved": tfl, "peak": tc_burst / div, "unit": "TFLOP/s",
                        "frac": tfl / (tc_burst / div)}
        else:
            roofline = {"bound": "hbm", "achieved": hbm_gbs, "peak": hbm_peak, "unit": "GB/s", "frac": hbm_gbs / hbm_peak}
        ih, it = common["hbm"]["ideal_ms"], common["tensor"]["ideal_ms_burst"]
        if abs(ih - it) < 0.1 * max(ih, it):
            notes.append("HBM and tensor ideal times are within 10 %% of each other (%.3f vs %.3f ms at the burst peaks): "
                         "read `frac` as the fraction of either" % (ih, it))
    else:
        # fused PQ (LUT form): Q*Nq*T*M four-byte shared-memory gathers against M bytes of codes per token -- bound by
        # the shared-memory load pipe (128 B/clk/SM), not by HBM and not by tensor cores
        lookups = accounting.pq_lookups(w["Q"], w["Nq"], w["M"], T)
        entry_bytes = wl.entry_bytes
        g = lookups * entry_bytes / kern_s / 1e9
        roofline = {"bound": "alu", "achieved": g, "peak": SMEM_PIPE_PEAK_GBS, "unit": "GB/s", "frac": g / SMEM_PIPE_PEAK_GBS}
        notes.append("shared-memory gather bytes/s (%d-byte table entries) against 148 SMs x 128 B/clk x 1.965 GHz; step = "
                     "LUT build + relayout + fused lookup kernel" % entry_bytes)
    # what THIS run observed about clocks and power (NVML samples taken while the timed steps ran)
    p_w, p_lim = clocks.get("power_w_mean"), clocks.get("power_limit_w")
    obs = "this run: NVML SM clock median %s MHz (max %s), throttle reasons %s" % (
        clocks.get("sm_mhz"), clocks.get("sm_max_mhz"), clocks.get("reasons") or "none")
    if p_w and p_lim:
        obs += ", board power (%s) mean %.0f W / max %.0f W of a %.0f W limit over %d samples" % (
            clocks.get("power_kind"), p_w, clocks.get("power_w_max", p_w), p_lim, clocks.get("samples", 0))
        if clocks.get("power_w_max", 0) >= 0.93 * p_lim:
            obs += " -- the run sits at the board power limit; NVML's clock field does not show the sub-millisecond " \
                   "clock reductions the power controller applies (DESIGN.md 5.1 has the in-kernel measurement)"
    notes.append(obs)
    roofline["note"] = "; ".join(notes)
    roofline["timed_region_ms"] = total_ms
    roofline.update(common)
    return roofline


SECONDARY = ["c2-q4", "c2-q1", "c2-fp16", "c2-fp32", "c3-100k", "c3-250k", "c3-500k", "c4-d64", "c4-d256", "c4-d512",
             "c4-d768", "c4-d512-q8", "c4-d768-q8", "c5", "c5-f16", "c5-decode", "c5-decode-fp16",
             "c2-topk", "c1", "n1-b1k", "n1-nq64", "n1-nd32", "n1-nd512"]
SECONDARY_MIN_MS = 150.0  # each secondary timed region lasts at least this long (>= 20 NVML samples under load)


def run_secondary(args, main_wl, dev, local_rank, tms, shard, sync_all, peaks):
    """The other BASELINE.json configs and the NEXT-1 sweeps' end points, each timed on its own (its own warm-up, at least
    --secondary-steps steps and at least SECONDARY_MIN_MS of device time, its own clock samples taken under load) AFTER
    and outside the headline's timed region: {name: {ms_per_step, docs_per_s, bound, frac, ...}}."""
    out = {}
    prev = main_wl
    for name in SECONDARY:
        if name == args.workload:
            continue
        w = WORKLOADS[name]
        try:
            same_store = [c for c in (prev, main_wl) if c.w["kind"] == w["kind"] == "dense" and c.B == w["B"] and
                          all(c.w[k] == w[k] for k in ("d", "dtype", "lengths", "Nd"))]
            wl = Workload(name, w, w["B"], args.seed, dev, tms, reuse=same_store[0] if same_store else None)
            torch.cuda.synchronize()
            time.sleep(1.0)  # let the board's power controller settle after the previous workload (each config is timed
            #                  on its own: a 0.4 ms kernel measured right behind a power-capped one inherits its clocks)
            step_ms, total_ms, clocks, launches = timed_region(wl, args.secondary_steps, 3, local_rank, sync_all, shard,
                                                               min_ms=SECONDARY_MIN_MS)
            r = roofline_of(wl, step_ms, total_ms, clocks, peaks)
            out[name] = {"ms_per_step": float(step_ms.mean()), "ms_min": float(step_ms.min()),
                         "ms_median": float(np.median(step_ms)),
                         "docs_per_s": w["B"] / (float(step_ms.mean()) * 1e-3), "steps": int(step_ms.size),
                         "bound": r["bound"], "frac": r["frac"], "achieved": r["achieved"], "peak": r["peak"],
                         "unit": r["unit"], "hbm_GBps": r["hbm"]["achieved_GBps"], "hbm_frac": r["hbm"]["frac"],
                         "tensor_frac_burst": r.get("tensor", {}).get("frac_burst"), "kernel": r["kernel"],
                         "gpu_launches": launches, "traffic": r["traffic"],
                         "clocks": {k: clocks.get(k) for k in ("sm_mhz", "reasons", "samples", "power_w_mean",
                                                               "power_w_max")},
                         "B": w["B"], "total_tokens": wl.T}
            if prev is not main_wl and prev is not wl:
                del prev
            prev = wl
        except Exception as e:  # a secondary workload never takes the headline down with it
            out[name] = {"error": repr(e)[:200]}
        torch.cuda.empty_cache()
    return out


def spawn_ranks(args):
    """`python bench.py --gpus N` without a launcher: start the N ranks here (same command line under
    torch.distributed.run, one rank per GPU over NCCL) and pass rank 0's JSON line through."""
    import socket
    import subprocess

    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        port = s.getsockname()[1]
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={args.gpus}",
           "--master-addr", "127.0.0.1", "--master-port", str(port), os.path.abspath(__file__)] + sys.argv[1:]
    env = dict(os.environ)
    env.setdefault("NCCL_DEBUG", "INFO")        # communicator / transport lines (NVLS, P2P) for whoever checks the ranks
    env.setdefault("NCCL_DEBUG_SUBSYS", "INIT")
    # NCCL writes to stdout, from every rank and also at teardown: pass everything through as it comes, but hold rank 0's
    # JSON line back so that it is the LAST line of this process's stdout
    proc = subprocess.Popen(cmd, env=env, stdout=subprocess.PIPE, text=True, bufsize=1)
    final = None
    for ln in proc.stdout:
        if ln.startswith("{") and '"metric"' in ln:
            final = ln
        else:
            sys.stdout.write(ln)
            sys.stdout.flush()
    rc = proc.wait()
    if final is not None:
        sys.stdout.write(final)
        sys.stdout.flush()
    raise SystemExit(rc)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--workload", default="c2", choices=sorted(WORKLOADS))
    ap.add_argument("--impl", default="tms", choices=["tms", "reference"])
    ap.add_argument("--B", type=int, default=0, help="override the number of documents per GPU")
    ap.add_argument("--variant", default="auto")
    ap.add_argument("--seed", type=int, default=0)
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-cpu", action="store_true")
    ap.add_argument("--no-secondary", action="store_true", help="skip the brief timings of the other configs")
    ap.add_argument("--secondary-steps", type=int, default=20)
    ap.add_argument("--sustained-steps", type=int, default=200,
                    help="steps of the headline's separate long run (0 = skip)")
    ap.add_argument("--e2e-steps", type=int, default=3)
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3) if args.impl == "tms" else args.warmup
    w = WORKLOADS[args.workload]

    launched = "WORLD_SIZE" in os.environ
    rank = int(os.environ.get("RANK", "0"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))

    if args.impl == "reference":
        run_reference(args, w, rank)
        return
    if args.gpus > 1 and not launched:
        spawn_ranks(args)  # does not return
    if launched and world != args.gpus and rank == 0:
        print(f"bench.py: --gpus {args.gpus} but WORLD_SIZE={world}; reporting n_gpus={world}", file=sys.stderr)

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

    def sync_all():
        torch.cuda.synchronize()
        if world > 1:
            dist.barrier()
            torch.cuda.synchronize()

    B = args.B or w["B"]
    # weak scaling: every rank owns its own B-document shard (token-balanced shards of a world*B store have this size)
    wl = Workload(args.workload, w, B, shard.rank_seed(args.seed, rank), dev, tms, variant=args.variant)
    T = wl.T
    step_ms, total_ms, clocks, launches = timed_region(wl, args.steps, args.warmup, local_rank, sync_all, shard)
    ms_per_step = total_ms / args.steps
    value = world * B / (ms_per_step * 1e-3)  # = shard.aggregate_throughput(B, ms_per_step): whole-job documents/s
    peaks = load_peaks()
    roofline = roofline_of(wl, step_ms, total_ms, clocks, peaks)

    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": w["dtype"] if w["kind"] == "dense" else "f32", "data": "synthetic",
        "config": config_dict(args, w, B, T, world), "pairs_per_s": value * w["Q"],
        "roofline": roofline, "clocks": clocks, "gpu_launches": launches,
    }

    # ---- end to end through the host-buffer entry point: H2D of the store + D2H of the scores every step -------------
    if not args.no_e2e:
        line["e2e"] = run_e2e(args, w, wl.inp, B, T, dev, world, tms, shard)
    if rank == 0 and not args.no_cpu:
        line["cpu_baseline"] = cpu_baseline(w, wl.inp, B)
    # ---- the other configs, briefly, outside the headline's timed region (single-GPU runs only) ----------------------
    if world == 1 and not args.no_secondary and args.workload == "c2" and not args.B:
        line["secondary"] = run_secondary(args, wl, dev, local_rank, tms, shard, sync_all, peaks)
    # ---- the headline again as one long run ("sustains", north_star): outside the K-step region, after a pause ---------
    line["step_ms"] = [round(float(x), 4) for x in step_ms]
    if args.sustained_steps > 0:
        torch.cuda.synchronize()
        time.sleep(1.0)
        s_ms, s_total, s_clk, _ = timed_region(wl, args.sustained_steps, 3, local_rank, sync_all, shard)
        rs = roofline_of(wl, s_ms, s_total, s_clk, peaks)
        line["sustained"] = {"steps": int(s_ms.size), "ms_per_step": s_total / s_ms.size,
                             "ms_median": float(np.median(s_ms)), "bound": rs["bound"], "frac_burst": rs["frac"],
                             "tensor_frac_burst": rs.get("tensor", {}).get("frac_burst"),
                             "tensor_frac_sustained": rs.get("tensor", {}).get("frac_sustained"),
                             "hbm_frac": rs["hbm"]["frac"],
                             "sm_mhz": s_clk.get("sm_mhz"), "reasons": s_clk.get("reasons"),
                             "samples": s_clk.get("samples"), "power_w_mean": s_clk.get("power_w_mean")}
    # compact copy of every secondary result, LAST in the line so that a truncated record still carries all of them:
    # name -> [ms mean, ms median, bound, fraction of that bound's peak, steps, NVML samples under load, median SM MHz]
    if "secondary" in line:
        line["secondary_summary"] = {
            n: ([round(v["ms_per_step"], 5), round(v["ms_median"], 5), v["bound"], round(v["frac"], 4), v["steps"],
                 v["clocks"].get("samples"), v["clocks"].get("sm_mhz")] if "error" not in v else ["error"])
            for n, v in line["secondary"].items()}
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
        host_fn = tms.tms_pq_maxsim_decode_host if w.get("decode") else tms.tms_pq_maxsim_host

        def call():
            host_fn(q_h, C_h, store_h, off_h, scores_h, ws)
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
            "api": "tms_maxsim_host" if w["kind"] == "dense" else
                   ("tms_pq_maxsim_decode_host" if w.get("decode") else "tms_pq_maxsim_host"),
            "ms_per_step": ms / args.e2e_steps}


if __name__ == "__main__":
    main()
