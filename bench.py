#!/usr/bin/env python
"""bench.py -- one JSON line per run for the mixed-step MLA attention path (BASELINE.json `metric`).

A "step" = one pass of the whole hot path over one synthetic batch:
kairos_append_latent(chunk) + kairos_mixed_step (host planner or cached plan, persistent tcgen05 kernels, LSE combine).

Headline workload at N=1: BASELINE.json configs[4] ("long-context stress": 32 decodes at 32768 + a 4096-token chunk over
a 28672-token prefix), the largest single-GPU configuration (BASELINE.json's `metric` names no config).  The same run
also times every other gated workload -- configs[1], configs[2], all seven chunk sizes of configs[3] -- and reports them
in `sweep` (step time, attention-kernel bracket, host enqueue time, fraction of the roofline against the BURST tensor
peak).  Inputs are seeded synthetic stand-ins for the paper's proprietary traces.  N>1: one replica per
GPU (requests shard by sequence with no data-path collective: "replicas only"), value aggregated over ranks.

  python bench.py [--gpus N] [--steps K] [--warmup W] [--config I] [--chunk C] [--no-sweep] [--fp8-only] [--impl kairos|reference]
  torchrun --nnodes=1 --nproc-per-node N ... bench.py --gpus N ...

Timing: W >= 3 warm-up steps, then exactly K steps bracketed by barrier + torch.cuda.synchronize, CUDA events on the
launching stream, max over ranks.  L2: a workload whose step touches more than 2x the 126 MB L2 needs nothing; smaller
ones rotate over R disjoint copies of the pool / queries so that more than 2x L2 is touched between two uses of a copy
(stated per point in `l2`).
"""
from __future__ import annotations

import argparse
import hashlib
import json
import os
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

from paper_2607_02043_b200 import workloads as W  # noqa: E402

L2_BYTES = 126 * 2 ** 20
METRIC = "mixed_step_mla_attention_us"
UNIT = "us/step"
HEADLINE = (4, None)
SWEEP = [(1, None), (2, None)] + [(3, c) for c in W.SWEEP_CHUNKS] + [(4, None)]


def load_peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        with open(path) as f:
            p = json.load(f)
        return dict(hbm_gbs=float(p["hbm_gbs"]), bf16_tflops=float(p["bf16_tflops"]),
                    bf16_tflops_sustained=float(p.get("bf16_tflops_sustained", p["bf16_tflops"])), source="measured")
    # fallback stated in /opt/skills/guides/B200_PROFILING.md
    return dict(hbm_gbs=6650.0, bf16_tflops=1590.0, bf16_tflops_sustained=1400.0, source="fallback")


KERNEL_SOURCES = ["append.cu", "attn_pair.cu", "attn_umma.cu", "plan.cpp", "umma_ptx.cuh", "fp8.cu"]


def csrc_sha() -> str:
    """Hash of the device code and the planner (what decides a kernel's DRAM traffic): an ncu capture under profiles/ is
    only quoted for the sources it measured."""
    h = hashlib.sha256()
    d = os.path.join(ROOT, "paper_2607_02043_b200", "csrc")
    for f in KERNEL_SOURCES:
        with open(os.path.join(d, f), "rb") as fh:
            h.update(fh.read())
    return h.hexdigest()[:16]


def measured_traffic(key: str):
    """DRAM read+write bytes of one launch of the dominant kernel from the committed `ncu --set full` capture of exactly
    this point (profiles/r02_traffic.csv: key,kernel,dram_bytes,csrc_sha), or (None, why)."""
    path = os.path.join(ROOT, "profiles", "r02_traffic.csv")
    if not os.path.exists(path):
        return None, "no ncu capture committed for this point"
    sha = csrc_sha()
    with open(path) as f:
        for line in f.read().splitlines()[1:]:
            parts = line.split(",")
            if len(parts) >= 4 and parts[0] == key:
                if parts[3] != sha:
                    return None, "capture predates the current kernel sources"
                return int(parts[2]), parts[1]
    return None, "no ncu capture committed for this point"


def point_key(index: int, chunk) -> str:
    return f"config{index}" + (f"_C{chunk}" if chunk is not None else "")


def make_workload(index: int, chunk, seed_shift: int = 0):
    inp = W.make_config(index, chunk_len=chunk)
    if seed_shift and index == 1:  # other replicas: same shapes, different seed (independent batches)
        inp = W.make_inputs("steady_state", 1 + seed_shift, None, 512, 0, n_dec=64,
                            lognormal=dict(median=1024, sigma=0.8, lo=64, hi=8192), q_scale=0.1)
    return inp


def workload_label(index: int, inp) -> str:
    return (f"configs[{index}] {inp.name}: {inp.n_dec} decodes (sum L = {int(inp.dec_ctx_lens.astype(np.int64).sum())})"
            f" + {inp.chunk_len}-token chunk over {inp.prefix_len}-token prefix; MLA 16 heads, 512+64, page 64, bf16")


class ClockSampler(threading.Thread):
    """Samples SM clock / throttle reasons through NVML while the timed region runs."""

    def __init__(self, index: int):
        super().__init__(daemon=True)
        self.samples, self.reasons, self.max_mhz = [], set(), None
        self._stop_evt = threading.Event()
        self.ok = False
        try:
            import pynvml
            pynvml.nvmlInit()
            self.nv = pynvml
            self.h = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.max_mhz = pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM)
            self.ok = True
        except Exception:
            pass

    def run(self):
        if not self.ok:
            return
        nv = self.nv
        names = {nv.nvmlClocksThrottleReasonSwPowerCap: "sw_power_cap", nv.nvmlClocksThrottleReasonHwSlowdown: "hw_slowdown",
                 nv.nvmlClocksThrottleReasonHwThermalSlowdown: "hw_thermal_slowdown",
                 nv.nvmlClocksThrottleReasonSwThermalSlowdown: "sw_thermal_slowdown",
                 nv.nvmlClocksThrottleReasonHwPowerBrakeSlowdown: "hw_power_brake"}
        while not self._stop_evt.is_set():
            try:
                self.samples.append(nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM))
                r = nv.nvmlDeviceGetCurrentClocksThrottleReasons(self.h)
                for bit, name in names.items():
                    if r & bit:
                        self.reasons.add(name)
            except Exception:
                pass
            time.sleep(0.002)

    def stop(self):
        self._stop_evt.set()
        self.join(timeout=2)
        med = float(np.median(self.samples)) if self.samples else None
        return {"sm_mhz": med, "sm_max_mhz": self.max_mhz, "reasons": sorted(self.reasons), "samples": len(self.samples)}


# ---------------------------------------------------------------------------------------------- CPU oracle legs
def oracle_sample(inp, budget_pairs: float = 6.0e6):
    """A bounded sample of the workload for the oracle: every decode and every chunk row when the whole step fits the
    budget, else evenly spaced decodes / chunk rows; returns (dec_idx, chunk_idx, pairs_in_sample, pairs_total, label)."""
    L = inp.dec_ctx_lens.astype(np.int64)
    C, P = inp.chunk_len, inp.prefix_len
    dec_pairs, chunk_pairs = int(L.sum()), C * P + C * (C + 1) // 2
    total = dec_pairs + chunk_pairs
    if total <= budget_pairs:
        return np.arange(inp.n_dec, dtype=np.int32), np.arange(C, dtype=np.int32), total, total, "every decode and chunk row"
    fd = min(1.0, budget_pairs / 2 / max(dec_pairs, 1))
    fc = min(1.0, budget_pairs / 2 / max(chunk_pairs, 1))
    nd = max(1, int(round(inp.n_dec * fd))) if inp.n_dec else 0
    nc = max(1, int(round(C * fc))) if C else 0
    di = np.unique(np.linspace(0, inp.n_dec - 1, nd).astype(np.int32)) if nd else np.zeros(0, np.int32)
    ci = np.unique(np.linspace(0, C - 1, nc).astype(np.int32)) if nc else np.zeros(0, np.int32)
    pairs = int(L[di].sum()) + int((P + ci.astype(np.int64) + 1).sum())
    return di, ci, pairs, total, (f"{len(di)} of {inp.n_dec} decodes and {len(ci)} of {C} chunk rows, evenly spaced; "
                                  f"time scaled by (query, key) pairs {total}/{pairs}")


def oracle_step_seconds(inp, reps: int):
    """Times the oracle as it stands on the host cores; returns (per-rep seconds scaled to the full step, threads, label)."""
    from oracle import oracle
    di, ci, pairs, total, label = oracle_sample(inp)
    full = pairs == total
    ts = []
    pool = inp.pool.copy()
    oracle.append(pool, inp.chunk_latent, inp.chunk_k_rope, inp.chunk_page_table, inp.prefix_len)
    for _ in range(reps):
        t0 = time.perf_counter()
        if full:
            oracle.append(pool, inp.chunk_latent, inp.chunk_k_rope, inp.chunk_page_table, inp.prefix_len)
            oracle.mixed_step(pool, inp.q_dec, inp.dec_page_tables, inp.dec_ctx_lens, inp.chunk_len, inp.prefix_len,
                              inp.q_chunk, inp.chunk_page_table, inp.softmax_scale)
        else:
            if len(di):
                oracle.attend_rows(pool, inp.dec_page_tables, inp.dec_table_stride, di, inp.q_dec[di], inp.dec_ctx_lens[di],
                                   inp.softmax_scale)
            if len(ci):
                oracle.attend_rows(pool, inp.chunk_page_table[None, :], inp.chunk_page_table.shape[0],
                                   np.zeros(len(ci), np.int32), inp.q_chunk[ci], (inp.prefix_len + ci + 1).astype(np.int32),
                                   inp.softmax_scale)
        ts.append((time.perf_counter() - t0) * (total / pairs))
    return ts, oracle.num_threads(), label


def run_reference(args, rank: int):
    """--impl reference: the CPU oracle timed on the host cores (rank 0 only), on this arm's config / metric / unit."""
    if rank != 0:
        return
    inp = make_workload(args.config, args.chunk)
    steps = min(args.steps, 5)
    oracle_step_seconds(inp, 1)
    ts, cores, label = oracle_step_seconds(inp, steps)
    us = float(np.mean(ts)) * 1e6
    sample = f"{inp.name}: {label}; {steps} timed reps"
    line = {"impl": "reference", "metric": METRIC, "value": us, "unit": UNIT, "n_gpus": args.gpus, "steps": steps,
            "warmup": 1, "ms_per_step": us / 1e3, "higher_is_better": False, "scaling": "weak",
            "vs_baseline": None, "dtype": "f32", "data": "synthetic",
            "config": {"workload": workload_label(args.config, inp), "what": "CPU oracle (oracle/oracle_mla.c) on host cores"},
            "cpu_baseline": {"value": us, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
            "e2e": {"value": us, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)


# ---------------------------------------------------------------------------------------------- the GPU arm
class Point:
    """One workload resident on the device (R rotating copies) with its timed regions."""

    def __init__(self, index, chunk, rank_seed_shift, dev, K, torch):
        self.index, self.chunk, self.K, self.torch, self.dev = index, chunk, K, torch, dev
        inp = self.inp = make_workload(index, chunk, seed_shift=rank_seed_shift)
        self.alg_bytes, self.alg_flops = inp.algorithmic_bytes(), inp.algorithmic_flops()
        step_touch = inp.pool.nbytes + inp.q_dec.nbytes + inp.q_chunk.nbytes
        if step_touch > 2 * L2_BYTES:
            replicas = 1
            self.l2 = f"one step touches {step_touch / 2**20:.0f} MiB > 2x L2: no flush needed"
        else:
            replicas = int(np.ceil(2.0 * L2_BYTES / max(step_touch, 1))) + 1
            self.l2 = f"inputs rotate over {replicas} disjoint pool/query copies ({replicas * step_touch / 2**20:.0f} MiB > 2x L2)"
        self.replicas = replicas

        class Rep:
            pass
        self.reps = []
        for _ in range(replicas):
            R = Rep()
            R.pool = K.bf16_tensor(inp.pool, dev)
            R.ws = torch.empty(K.workspace_bytes(max(inp.n_dec, 1), max(inp.chunk_len, 1)), dtype=torch.uint8, device=dev)
            R.ctx = K.Kairos(R.pool, R.ws, inp.softmax_scale)
            R.q_dec = K.bf16_tensor(inp.q_dec, dev)
            R.q_chunk = K.bf16_tensor(inp.q_chunk, dev)
            R.dec_pt = torch.from_numpy(inp.dec_page_tables).to(dev)
            R.chunk_pt = torch.from_numpy(inp.chunk_page_table).to(dev)
            R.latent = K.bf16_tensor(inp.chunk_latent, dev)
            R.k_rope = K.bf16_tensor(inp.chunk_k_rope, dev)
            R.out_dec = torch.empty((inp.n_dec, 16, 512), dtype=torch.bfloat16, device=dev)
            R.out_chunk = torch.empty((inp.chunk_len, 16, 512), dtype=torch.bfloat16, device=dev)
            R.lse_dec = torch.empty((inp.n_dec, 16), dtype=torch.float32, device=dev)
            R.lse_chunk = torch.empty((inp.chunk_len, 16), dtype=torch.float32, device=dev)
            # the step as a serving loop issues it: the same buffers every time, marshalled once (Kairos.bind_step)
            R.bound = R.ctx.bind_step(R.q_dec, R.dec_pt, inp.dec_ctx_lens, R.q_chunk, R.chunk_pt, inp.chunk_len, inp.prefix_len,
                                      R.out_dec, R.out_chunk, R.lse_dec, R.lse_chunk, R.latent, R.k_rope)
            self.reps.append(R)
        self.lens = inp.dec_ctx_lens

    def step(self, R):
        R.bound.run()  # kairos_append_latent(chunk) + kairos_mixed_step

    def warm(self, n, tune=True):
        inp = self.inp
        self.tuned = None
        if tune and inp.chunk_len and inp.n_dec and self.alg_flops <= 2.0e12:
            # kairos_tune_step (public API): each context measures the candidate launch orders of its step once and pins the fastest.
            # Not on configs[4] (4.4 TFLOP per step: the planner's order is the best one there and the candidate runs take seconds).
            for R in self.reps:
                R.ctx.append_latent(R.latent, R.k_rope, R.chunk_pt, inp.prefix_len)
                self.tuned = R.ctx.tune_step(R.q_dec, R.dec_pt, self.lens, R.q_chunk, R.chunk_pt, inp.chunk_len, inp.prefix_len,
                                             R.out_dec, R.out_chunk, reps=5)
            if self.alg_flops > 1.0e11:
                # the candidate runs of a tensor-bound step are tens of ms at full power: under the power cap the region that
                # follows them directly runs 5-15 % slower, so the chip idles for a second before the warm-up
                self.torch.cuda.synchronize()
                time.sleep(1.0)
        for i in range(max(n, 3) * self.replicas):  # every copy plans, hits its cache and captures its graph before timing
            self.step(self.reps[i % self.replicas])
        self.torch.cuda.synchronize()
        self.info = self.reps[0].ctx.last_plan_info()

    def timed(self, n_steps, barrier, profile=False, settle=0.0):
        """(device ms over n_steps, host seconds spent issuing them, summed attention-bracket us, brackets).
        settle > 0: the region starts from the state the first region of a point starts from -- that many seconds of idle, then
        three untimed steps.  Under its power cap this chip drops its clocks ~7 % after ~70 ms of back-to-back tensor-bound
        steps (measured: two 20-step regions of configs[4] in a row give 3.66 and 3.92 ms/step, whichever runs second), so a
        region that follows another one without a pause is not comparable with it."""
        torch = self.torch
        for R in self.reps:
            R.ctx.profile_enable(profile)
        if settle > 0:
            barrier()
            time.sleep(settle)
            for i in range(3):
                self.step(self.reps[i % self.replicas])
            if profile:
                barrier()
                for R in self.reps:
                    R.ctx.profile_read()  # drop the brackets of the untimed steps
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        barrier()
        t0 = time.perf_counter()
        e0.record()
        for i in range(n_steps):
            self.step(self.reps[i % self.replicas])
        e1.record()
        host_s = time.perf_counter() - t0
        barrier()
        ms = e0.elapsed_time(e1)
        k_us, k_n = 0.0, 0
        if profile:
            for R in self.reps:
                us, n = R.ctx.profile_read()
                k_us += us
                k_n += n
                R.ctx.profile_enable(False)
        return ms, host_s, k_us, k_n

    def close(self):
        for R in self.reps:
            R.ctx.close()
        self.reps = []
        self.torch.cuda.empty_cache()


def roofline_entry(pt: Point, us_per_step: float, kern_us: float, peaks) -> dict:
    t_hbm = pt.alg_bytes / (peaks["hbm_gbs"] * 1e9) * 1e6
    t_tc_burst = pt.alg_flops / (peaks["bf16_tflops"] * 1e12) * 1e6
    t_tc_sus = pt.alg_flops / (peaks["bf16_tflops_sustained"] * 1e12) * 1e6
    bound = "hbm" if t_hbm >= t_tc_burst else "tensor"
    roof = max(t_hbm, t_tc_burst)
    return {"bound": bound, "roofline_us": roof, "roofline_us_sustained_tensor_peak": max(t_hbm, t_tc_sus),
            "frac": roof / us_per_step, "frac_sustained": max(t_hbm, t_tc_sus) / us_per_step,
            "kernel_frac": roof / kern_us if kern_us > 0 else None}


FP8_TOKEN_BYTES = 512 + 4 + 128  # e4m3 latent codes + one f32 scale + bf16 RoPE key (include/kairos.h, G23)


def fp8_decode_leg(K, torch, dev, peaks, steps, warmup):
    """configs[3] over the fp8 latent cache -- the decodes alone (C = 0, kairos_fp8_decode) and, under "mixed",
    the step with a chunk of 256 / 512 tokens (kairos_fp8_append of the chunk + kairos_fp8_mixed_step).  The cache is built on the
    device by kairos_fp8_append from the same synthetic tokens; one step reads >= 338 MiB (> 2x L2: no flush)."""
    def one(C):
        inp = W.make_config(3, chunk_len=C)
        pool16 = K.bf16_tensor(inp.pool)
        ws = torch.empty(K.workspace_bytes(inp.n_dec + C, 0), dtype=torch.uint8, device=dev)
        ctx = K.Kairos(pool16, ws, inp.softmax_scale)
        pool8 = torch.zeros((inp.num_pages, K.FP8_PAGE_BYTES), dtype=torch.uint8, device=dev)
        ctx.fp8_attach(pool8)
        dpt = torch.from_numpy(inp.dec_page_tables).to(dev)
        for i in range(inp.n_dec):
            tok = ctx.gather_latent(dpt[i], int(inp.dec_ctx_lens[i]))
            ctx.fp8_append(tok[:, :512].contiguous(), tok[:, 512:].contiguous(), dpt[i], 0)
        qd = K.bf16_tensor(inp.q_dec)
        od = torch.empty((inp.n_dec, 16, 512), dtype=torch.bfloat16, device=dev)
        if C:
            cpt = torch.from_numpy(inp.chunk_page_table).to(dev)
            lat, rope, qc = K.bf16_tensor(inp.chunk_latent), K.bf16_tensor(inp.chunk_k_rope), K.bf16_tensor(inp.q_chunk)
            oc = torch.empty((C, 16, 512), dtype=torch.bfloat16, device=dev)

            def step():
                ctx.fp8_append(lat, rope, cpt, inp.prefix_len)
                ctx.fp8_mixed_step(qd, dpt, inp.dec_ctx_lens, qc, cpt, C, inp.prefix_len, out_dec=od, out_chunk=oc, want_lse=False)
        else:
            def step():
                ctx.fp8_decode(qd, dpt, inp.dec_ctx_lens, out_dec=od, want_lse=False)
        for _ in range(max(warmup, 3)):
            step()
        torch.cuda.synchronize()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        n = max(steps, 200)
        e0.record()
        for _ in range(n):
            step()
        e1.record()
        torch.cuda.synchronize()
        us = e0.elapsed_time(e1) * 1e3 / n
        tokens = int(inp.dec_ctx_lens.astype(np.int64).sum())
        alg = (tokens + (inp.prefix_len + C if C else 0)) * FP8_TOKEN_BYTES + (inp.n_dec + C) * (W.Q_BYTES + W.OUT_BYTES)
        roof_us = max(alg / peaks["hbm_gbs"] / 1e3, inp.algorithmic_flops() / peaks["bf16_tflops"] / 1e6)
        info = ctx.last_plan_info()
        return {"workload": f"configs[3] C={C} over the fp8 latent cache", "B": inp.n_dec, "C": C, "P": inp.prefix_len, "cached_tokens": tokens,
                "step_us": us, "steps": n, "algorithmic_bytes": alg, "bytes_per_token": FP8_TOKEN_BYTES,
                "roofline": {"bound": "hbm", "achieved": alg / (us * 1e-6) / 1e9, "peak": peaks["hbm_gbs"], "unit": "GB/s",
                             "frac": roof_us / us, "roofline_us": roof_us,
                             "note": "whole step over max(HBM time of its algorithmic bytes, tensor time of its FLOPs at the bf16 peak)"},
                "kernels_per_step": info["kernels"] + (1 if C else 0), "graph": info["graph"], "work_items": info["work_items"]}

    head = one(0)
    head["workload"] = "configs[3] C=0 decodes over the fp8 latent cache (kairos_fp8_decode)"
    head["traffic"] = measured_traffic("fp8_config3_C0")[0]
    head["dtype"] = "e4m3 cache, bf16 q / out, f32 accumulation"
    head["l2"] = "one step reads 338 MiB > 2x L2: no flush needed"
    head["mixed"] = [one(256), one(512)]
    return head


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--config", type=int, default=HEADLINE[0], help="BASELINE.json configs index of the headline workload")
    ap.add_argument("--chunk", type=int, default=None, help="chunk size for configs[3]")
    ap.add_argument("--impl", default="kairos", choices=["kairos", "reference"])
    ap.add_argument("--no-sweep", action="store_true", help="time the headline workload only")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--fp8-only", action="store_true", help="run the fp8 latent-cache decode leg alone and print its entry (profiling)")
    ap.add_argument("--no-tune", action="store_true", help="keep the planner's own launch order (skip kairos_tune_step in the warm-up)")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3)

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))

    if args.impl == "reference":
        run_reference(args, rank)
        return

    import torch
    import torch.distributed as dist
    from paper_2607_02043_b200 import kairos as K  # raises if libkairos.so is missing: no fallback
    from paper_2607_02043_b200 import replicas as R_

    assert torch.cuda.is_available(), "bench.py needs a CUDA device (no CPU fallback)"
    torch.cuda.set_device(local_rank)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local_rank))
    dev = torch.device("cuda", local_rank)
    peaks = load_peaks()

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    if args.fp8_only:
        print(json.dumps({"fp8_decode": fp8_decode_leg(K, torch, dev, peaks, args.steps, args.warmup)}), flush=True)
        return

    # ---- headline workload first (clock / throttle reasons are sampled over its timed regions only)
    pt = Point(args.config, args.chunk, R_.replica_seed_shift(rank), dev, K, torch)
    inp = pt.inp
    pt.warm(args.warmup, tune=not args.no_tune)
    info = pt.info
    sampler = ClockSampler(local_rank)
    sampler.start()
    ms_head, host_head, _, _ = pt.timed(args.steps, barrier)
    # roofline leg: the same K steps again with the attention kernels bracketed by CUDA events on their stream
    ms_prof, _, kern_us, kern_n = pt.timed(args.steps, barrier, profile=True, settle=1.0)
    clocks = sampler.stop()
    # the same step issued back to back for 5x as long, with no pause before it: what a long serving loop sees under the power cap
    ms_sus, _, _, _ = pt.timed(5 * args.steps, barrier)


    # ---- the other gated workloads (rank 0's own GPU, N = 1 only): same protocol, their own step counts
    sweep = []
    headline_key = point_key(args.config, args.chunk)
    if world == 1 and not args.no_sweep:
        for (ci, cc) in SWEEP:
            if point_key(ci, cc) == headline_key:
                continue
            sp = Point(ci, cc, 0, dev, K, torch)
            sp.warm(args.warmup, tune=not args.no_tune)
            ms, _, _, _ = sp.timed(10, barrier)  # sizes the timed region: at least K steps and about 30 ms
            n = int(min(max(args.steps, 30e3 / max(ms * 1e3 / 10, 1.0)), 400))
            ms, host_s, _, _ = sp.timed(n, barrier)
            _, _, k_us, k_n = sp.timed(n, barrier, profile=True, settle=0.5)
            us, kern = ms * 1e3 / n, k_us / max(k_n, 1)
            e = {"workload": point_key(ci, cc), "B": sp.inp.n_dec, "C": sp.inp.chunk_len, "P": sp.inp.prefix_len,
                 "step_us": us, "kernel_us": kern, "host_enqueue_us": host_s * 1e6 / n, "steps": n, "l2": sp.l2,
                 "chunk_pairs": sp.info["chunk_pairs"], "dec_ctas_first": sp.info["dec_ctas_first"],
                 "kernels_per_step": sp.info["kernels"], "graph": sp.info["graph"],
                 "tuned_order": None if sp.tuned is None else {"mode": sp.tuned[0], "us": sp.tuned[1], "planner_us": sp.tuned[2]}}
            e.update(roofline_entry(sp, us, kern, peaks))
            sweep.append(e)
            sp.close()
            del sp

    fp8 = None
    if world == 1 and not args.no_sweep:
        fp8 = fp8_decode_leg(K, torch, dev, peaks, args.steps, args.warmup)

    ms_max = R_.max_over_ranks(ms_head, dev)
    us_per_step = R_.whole_job_us_per_step(ms_head, args.steps, world, dev)  # world replicas advance one step per iteration

    # ---- end-to-end leg: same step through the C ABI with HOST buffers (pinned), copies inside the timed region
    e2e = None
    if not args.no_e2e:
        R = pt.reps[0]
        pin = lambda a: torch.from_numpy(np.ascontiguousarray(a)).pin_memory().numpy()
        h_qd, h_qc = pin(inp.q_dec), pin(inp.q_chunk)
        h_dpt, h_cpt = pin(inp.dec_page_tables), pin(inp.chunk_page_table)
        h_lat, h_rope = pin(inp.chunk_latent), pin(inp.chunk_k_rope)
        h_od = torch.empty((inp.n_dec, 16, 512), dtype=torch.int16).pin_memory().numpy().view(np.uint16)
        h_oc = torch.empty((inp.chunk_len, 16, 512), dtype=torch.int16).pin_memory().numpy().view(np.uint16)
        e2e_steps = max(10, min(args.steps, 100))
        for _ in range(3):
            h2d, d2h = R.ctx.mixed_step_host(h_qd, h_dpt, pt.lens, h_qc, h_lat, h_rope, h_cpt, inp.chunk_len, inp.prefix_len, h_od, h_oc)
        barrier()
        t0 = time.perf_counter()
        for i in range(e2e_steps):
            pt.reps[i % pt.replicas].ctx.mixed_step_host(h_qd, h_dpt, pt.lens, h_qc, h_lat, h_rope, h_cpt, inp.chunk_len,
                                                         inp.prefix_len, h_od, h_oc)
        torch.cuda.synchronize()
        e2e_s = time.perf_counter() - t0
        e2e_us = R_.max_over_ranks(e2e_s, dev) * 1e6 / (e2e_steps * world)
        e2e = {"value": e2e_us, "unit": UNIT, "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h,
               "api": "kairos_mixed_step_host (pinned host buffers, synchronous; a large chunk runs in slices whose copies overlap the attention)",
               "steps": e2e_steps}

    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return

    # ---- roofline of the attention kernels of the step (kairos_mixed_kernel, plus the concurrent kairos_chunk_pair_kernel
    # when the planner moves the chunk onto SM pairs): algorithmic bytes / flops per step over the live CUDA-event
    # duration of that bracket inside the second timed region.  Tensor peak = the BURST cuBLAS figure of MEASURED_PEAKS.json
    # (a step lasts milliseconds at full clocks); the fraction against the sustained figure is reported beside it.
    kern_avg_us = kern_us / max(kern_n, 1)
    own_us = ms_max * 1e3 / args.steps
    re = roofline_entry(pt, own_us, kern_avg_us, peaks)
    traffic, traffic_note = measured_traffic(headline_key)
    if re["bound"] == "hbm":
        achieved = pt.alg_bytes / (kern_avg_us * 1e-6) / 1e9
        roof = {"bound": "hbm", "achieved": achieved, "peak": peaks["hbm_gbs"], "unit": "GB/s", "frac": achieved / peaks["hbm_gbs"]}
    else:
        achieved = pt.alg_flops / (kern_avg_us * 1e-6) / 1e12
        roof = {"bound": "tensor", "achieved": achieved, "peak": peaks["bf16_tflops"], "unit": "TFLOP/s",
                "frac": achieved / peaks["bf16_tflops"], "peak_kind": "burst",
                "peak_sustained": peaks["bf16_tflops_sustained"], "frac_sustained": achieved / peaks["bf16_tflops_sustained"]}
    kname = ("kairos_chunk_pair_kernel (chunk, %d 2-CTA clusters) + kairos_mixed_kernel (decode splits), concurrent grids"
             % info["chunk_pairs"]) if info.get("chunk_pairs", 0) > 0 else "kairos_mixed_kernel"
    roof.update({"traffic": traffic, "traffic_note": traffic_note, "kernel": kname, "kernel_us": kern_avg_us,
                 "launches_timed": kern_n, "peak_source": peaks["source"], "algorithmic_bytes": pt.alg_bytes,
                 "algorithmic_flops": pt.alg_flops, "step_roofline_us": re["roofline_us"], "step_frac_of_roofline": re["frac"],
                 "step_frac_of_roofline_sustained_tensor_peak": re["frac_sustained"],
                 "us_per_step_with_kernel_events": ms_prof * 1e3 / args.steps})
    head = {"workload": headline_key, "B": inp.n_dec, "C": inp.chunk_len, "P": inp.prefix_len, "step_us": own_us,
            "kernel_us": kern_avg_us, "host_enqueue_us": host_head * 1e6 / args.steps, "steps": args.steps, "l2": pt.l2,
            "chunk_pairs": info["chunk_pairs"], "dec_ctas_first": info["dec_ctas_first"],
            "kernels_per_step": info["kernels"], "graph": info["graph"],
            "tuned_order": None if pt.tuned is None else {"mode": pt.tuned[0], "us": pt.tuned[1], "planner_us": pt.tuned[2]}}
    head.update(re)
    order = {point_key(ci, cc): i for i, (ci, cc) in enumerate(SWEEP)}
    sweep = sorted(sweep + [head], key=lambda e: order.get(e["workload"], 99))

    cpu = None
    if not args.no_cpu_baseline:
        ts, cores, label = oracle_step_seconds(inp, 1)
        cpu = {"value": float(np.median(ts)) * 1e6, "unit": UNIT, "cores": cores, "kind": "oracle",
               "sample": f"{inp.name}: {label}"}

    line = {
        "metric": METRIC, "value": us_per_step, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": ms_max / args.steps, "higher_is_better": False, "scaling": "weak", "vs_baseline": None,
        "dtype": "bf16", "data": "synthetic",
        "config": {"workload": workload_label(args.config, inp), "parallelism": f"replicas x{world} (no collective)",
                   "l2": pt.l2,
                   "step": "kairos_append_latent(chunk) + kairos_mixed_step (cached plan replayed as a CUDA graph: attention grid(s) + combine)",
                   "plan": info, "library": K.version()},
        "clocks": clocks,
        "host_enqueue_us": host_head * 1e6 / args.steps,
        "sustained": {"us_per_step": ms_sus * 1e3 / (5 * args.steps), "steps": 5 * args.steps,
                      "note": "back to back behind the two timed regions, no pause: the power cap has dropped the clocks by then; "
                              "the timed regions each start after >= 1 s of idle + 3 untimed steps"},
        "e2e": e2e,
        "gpu_launches": int(args.steps * info["kernels"]),  # the bound step's kernels: append + attention grid(s) + combine
        "roofline": roof,
        "cpu_baseline": cpu,
        "achieved": {"algorithmic_GBps": pt.alg_bytes / (us_per_step * world * 1e-6) / 1e9,
                     "algorithmic_TFLOPs": pt.alg_flops / (us_per_step * world * 1e-6) / 1e12},
        "sweep": sweep,
        "fp8_decode": fp8,
    }
    print(json.dumps(line), flush=True)
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
