#!/usr/bin/env python
"""bench.py -- one JSON line per run for the mixed-step MLA attention path (BASELINE.json `metric`).

A "step" = one pass of the whole hot path over one synthetic batch:
kairos_append_latent(chunk) + kairos_mixed_step (host planner, persistent tcgen05 kernels, LSE combine).
Workload at N=1: BASELINE.json configs[1] ("decode-node steady state": 64 lognormal decodes + one 512-token chunk),
seeded synthetic inputs standing in for the paper's proprietary traces.  N>1: one replica per GPU
(requests shard by sequence with no data-path collective: "replicas only"), value aggregated over ranks.

  python bench.py [--gpus N] [--steps K] [--warmup W] [--config I] [--chunk C] [--impl kairos|reference]
  torchrun --nnodes=1 --nproc-per-node N ... bench.py --gpus N ...

Timing: W >= 3 warm-up steps, then exactly K steps bracketed by barrier + torch.cuda.synchronize, CUDA events on
the launching stream, max over ranks.  Between steps the inputs rotate over R disjoint copies of the pool / queries
so that the bytes touched between two uses of a copy exceed 2x the 126 MB L2 (stated in `config.l2`).
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

from paper_2607_02043_b200 import workloads as W  # noqa: E402

L2_BYTES = 126 * 2 ** 20
METRIC = "mixed_step_mla_attention_us"
UNIT = "us/step"


def load_peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        with open(path) as f:
            p = json.load(f)
        return dict(hbm_gbs=float(p["hbm_gbs"]), bf16_tflops=float(p["bf16_tflops"]),
                    bf16_tflops_sustained=float(p.get("bf16_tflops_sustained", p["bf16_tflops"])), source="measured")
    # fallback stated in /opt/skills/guides/B200_PROFILING.md
    return dict(hbm_gbs=6650.0, bf16_tflops=1590.0, bf16_tflops_sustained=1400.0, source="fallback")


def make_workload(index: int, chunk, seed_shift: int = 0):
    inp = W.make_config(index, chunk_len=chunk)
    if seed_shift:  # other replicas: same shapes, different seed (independent batches)
        kw = dict(q_scale=0.1)
        if index == 1:
            inp = W.make_inputs("steady_state", 1 + seed_shift, None, 512, 0, n_dec=64,
                                lognormal=dict(median=1024, sigma=0.8, lo=64, hi=8192), **kw)
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


def oracle_step_seconds(inp, reps: int):
    """Times the oracle as it stands on the host cores for one full step (append + mixed step)."""
    from oracle import oracle
    ts = []
    for _ in range(reps):
        pool = inp.pool.copy()
        t0 = time.perf_counter()
        oracle.append(pool, inp.chunk_latent, inp.chunk_k_rope, inp.chunk_page_table, inp.prefix_len)
        oracle.mixed_step(pool, inp.q_dec, inp.dec_page_tables, inp.dec_ctx_lens, inp.chunk_len, inp.prefix_len,
                          inp.q_chunk, inp.chunk_page_table, inp.softmax_scale)
        ts.append(time.perf_counter() - t0)
    return ts, oracle.num_threads()


def run_reference(args, rank: int):
    """--impl reference: the CPU oracle timed on the host cores (rank 0 only)."""
    if rank != 0:
        return
    inp = make_workload(args.config, args.chunk)
    for _ in range(max(args.warmup, 0)):
        oracle_step_seconds(inp, 1)
    ts, cores = oracle_step_seconds(inp, args.steps)
    us = float(np.mean(ts)) * 1e6
    sample = f"full {inp.name} step (append + every decode and chunk row), {args.steps} timed reps"
    line = {"impl": "reference", "metric": METRIC, "value": us, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": us / 1e3, "higher_is_better": False, "scaling": "weak",
            "vs_baseline": None, "dtype": "f32", "data": "synthetic",
            "config": {"workload": workload_label(args.config, inp), "what": "CPU oracle (oracle/oracle_mla.c) on host cores"},
            "cpu_baseline": {"value": us, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
            "e2e": {"value": us, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=2000)
    ap.add_argument("--warmup", type=int, default=20)
    ap.add_argument("--config", type=int, default=1, help="BASELINE.json configs index (default 1: steady state)")
    ap.add_argument("--chunk", type=int, default=None, help="chunk size for configs[3]")
    ap.add_argument("--impl", default="kairos", choices=["kairos", "reference"])
    ap.add_argument("--no-cpu-baseline", action="store_true")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3)

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))

    if args.impl == "reference":
        if args.steps > 50:
            args.steps = 20  # bounded: each reference step is a full CPU pass over the workload
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

    inp = make_workload(args.config, args.chunk, seed_shift=R_.replica_seed_shift(rank))
    alg_bytes, alg_flops = inp.algorithmic_bytes(), inp.algorithmic_flops()
    pool_bytes = inp.pool.nbytes
    step_touch = pool_bytes + inp.q_dec.nbytes + inp.q_chunk.nbytes
    replicas = max(2, int(np.ceil(2.0 * L2_BYTES / max(step_touch, 1))) + 1)
    free_b, _ = torch.cuda.mem_get_info()
    replicas = int(min(replicas, max(1, (free_b * 0.6) // max(step_touch * 1.3, 1))))

    class Rep:
        pass
    reps = []
    lens = inp.dec_ctx_lens
    for r in range(replicas):
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
        reps.append(R)

    def step(R):
        if inp.chunk_len:
            R.ctx.append_latent(R.latent, R.k_rope, R.chunk_pt, inp.prefix_len)
        R.ctx.mixed_step(R.q_dec, R.dec_pt, lens, R.q_chunk, R.chunk_pt, inp.chunk_len, inp.prefix_len,
                         out_dec=R.out_dec, out_chunk=R.out_chunk, lse_dec=R.lse_dec, lse_chunk=R.lse_chunk)

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    def timed_region(n_steps: int, profile: bool):
        for R in reps:
            R.ctx.profile_enable(profile)
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        barrier()
        e0.record()
        for i in range(n_steps):
            step(reps[i % replicas])
        e1.record()
        barrier()
        ms = e0.elapsed_time(e1)
        k_us, k_n = 0.0, 0
        if profile:
            for R in reps:
                us, n = R.ctx.profile_read()
                k_us += us
                k_n += n
                R.ctx.profile_enable(False)
        return ms, k_us, k_n

    # warm-up
    for i in range(args.warmup):
        step(reps[i % replicas])
    barrier()
    info = reps[0].ctx.last_plan_info()

    sampler = ClockSampler(local_rank)
    sampler.start()
    ms, _, _ = timed_region(args.steps, profile=False)
    # roofline leg: the same K steps again with the main kernel bracketed by CUDA events on its stream
    ms_prof, kern_us, kern_n = timed_region(args.steps, profile=True)
    clocks = sampler.stop()

    ms_max = R_.max_over_ranks(ms, dev)
    us_per_step = R_.whole_job_us_per_step(ms, args.steps, world, dev)  # world replicas advance one step per iteration

    # ---- end-to-end leg: same step through the C ABI with HOST buffers (pinned), copies inside the timed region
    R = reps[0]
    pin = lambda a: torch.from_numpy(np.ascontiguousarray(a)).pin_memory().numpy()
    h_qd, h_qc = pin(inp.q_dec), pin(inp.q_chunk)
    h_dpt, h_cpt = pin(inp.dec_page_tables), pin(inp.chunk_page_table)
    h_lat, h_rope = pin(inp.chunk_latent), pin(inp.chunk_k_rope)
    h_od = torch.empty((inp.n_dec, 16, 512), dtype=torch.int16).pin_memory().numpy().view(np.uint16)
    h_oc = torch.empty((inp.chunk_len, 16, 512), dtype=torch.int16).pin_memory().numpy().view(np.uint16)
    e2e_steps = max(20, min(args.steps, 200))
    for _ in range(3):
        h2d, d2h = R.ctx.mixed_step_host(h_qd, h_dpt, lens, h_qc, h_lat, h_rope, h_cpt, inp.chunk_len, inp.prefix_len, h_od, h_oc)
    barrier()
    t0 = time.perf_counter()
    for i in range(e2e_steps):
        reps[i % replicas].ctx.mixed_step_host(h_qd, h_dpt, lens, h_qc, h_lat, h_rope, h_cpt, inp.chunk_len,
                                               inp.prefix_len, h_od, h_oc)
    torch.cuda.synchronize()
    e2e_s = time.perf_counter() - t0
    e2e_us = R_.max_over_ranks(e2e_s, dev) * 1e6 / (e2e_steps * world)

    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return

    # ---- roofline of the attention kernels of the step (kairos_mixed_kernel, plus the concurrent kairos_chunk_pair_kernel
    # when the planner moves the chunk onto SM pairs): algorithmic bytes / flops per step over the live CUDA-event
    # duration of that bracket inside the second timed region
    kern_avg_us = kern_us / max(kern_n, 1)
    t_hbm_us = alg_bytes / (peaks["hbm_gbs"] * 1e9) * 1e6
    # the kernels are timed inside the long step loop, so the tensor peak is the SUSTAINED cuBLAS figure of MEASURED_PEAKS.json
    # (the burst figure is for a kernel timed alone); the burst fraction is reported beside it
    tc_peak = peaks["bf16_tflops_sustained"]
    t_tc_us = alg_flops / (tc_peak * 1e12) * 1e6
    bound = "hbm" if t_hbm_us >= t_tc_us else "tensor"
    traffic = None  # DRAM bytes of one launch of the dominant kernel from the committed ncu capture of this configuration
    tpath = os.path.join(ROOT, "profiles", "r01_traffic.csv")
    if os.path.exists(tpath):
        key = f"config{args.config}" + (f"_C{args.chunk}" if args.chunk is not None else "")
        with open(tpath) as f:
            for line in f.read().splitlines()[1:]:
                k, _, v = line.split(",")
                if k == key:
                    traffic = int(v)
    if bound == "hbm":
        achieved = alg_bytes / (kern_avg_us * 1e-6) / 1e9
        roof = {"bound": "hbm", "achieved": achieved, "peak": peaks["hbm_gbs"], "unit": "GB/s",
                "frac": achieved / peaks["hbm_gbs"], "traffic": traffic}
    else:
        achieved = alg_flops / (kern_avg_us * 1e-6) / 1e12
        roof = {"bound": "tensor", "achieved": achieved, "peak": tc_peak, "unit": "TFLOP/s",
                "frac": achieved / tc_peak, "traffic": traffic, "peak_kind": "sustained (kernel timed inside the step loop)",
                "peak_burst": peaks["bf16_tflops"], "frac_of_burst": achieved / peaks["bf16_tflops"]}
    kname = ("kairos_chunk_pair_kernel (chunk, %d 2-CTA clusters) + kairos_mixed_kernel (decode splits), concurrent grids"
             % info["chunk_pairs"]) if info.get("chunk_pairs", 0) > 0 else "kairos_mixed_kernel"
    roof.update({"kernel": kname, "kernel_us": kern_avg_us, "launches_timed": kern_n,
                 "peak_source": peaks["source"], "algorithmic_bytes": alg_bytes, "algorithmic_flops": alg_flops,
                 "step_roofline_us": max(t_hbm_us, t_tc_us),
                 "step_frac_of_roofline": max(t_hbm_us, t_tc_us) / (ms_max * 1e3 / args.steps),
                 "us_per_step_with_kernel_events": ms_prof * 1e3 / args.steps})

    cpu = None
    if not args.no_cpu_baseline:
        n_rep = 3 if args.config <= 1 else 1
        ts, cores = oracle_step_seconds(inp, n_rep)
        cpu = {"value": float(np.median(ts)) * 1e6, "unit": UNIT, "cores": cores, "kind": "oracle",
               "sample": f"full {inp.name} step (append + every decode and chunk row), median of {n_rep}"}

    line = {
        "metric": METRIC, "value": us_per_step, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": ms_max / args.steps, "higher_is_better": False, "scaling": "weak", "vs_baseline": None,
        "dtype": "bf16", "data": "synthetic",
        "config": {"workload": workload_label(args.config, inp), "parallelism": f"replicas x{world} (no collective)",
                   "l2": f"inputs rotate over {replicas} disjoint pool/query copies ({replicas * step_touch / 2**20:.0f} MiB > 2x L2)",
                   "step": "kairos_append_latent(chunk) + kairos_mixed_step (planner H2D + persistent attention kernel(s) + combine)",
                   "plan": info, "library": K.version()},
        "clocks": clocks,
        "e2e": {"value": e2e_us, "unit": UNIT, "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h,
                "api": "kairos_mixed_step_host (pinned host buffers, synchronous)", "steps": e2e_steps},
        "gpu_launches": int(args.steps * ((1 if inp.chunk_len else 0) + info["kernels"])),
        "roofline": roof,
        "cpu_baseline": cpu,
        "achieved": {"algorithmic_GBps": alg_bytes / (us_per_step * world * 1e-6) / 1e9,
                     "algorithmic_TFLOPs": alg_flops / (us_per_step * world * 1e-6) / 1e12},
    }
    print(json.dumps(line), flush=True)
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
