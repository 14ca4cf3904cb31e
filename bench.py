#!/usr/bin/env python
"""bench.py -- Lomb-Scargle term-evaluation throughput on B200 (BASELINE.json metric).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload C5] [--impl ours|reference] [--shard series|freq]
    python bench.py --sweep | --back-to-back N      (N_t scaling sweep; call latency of the small configs)

One "step" = one pass of the whole hot path (moments -> records -> accumulate -> finish, all rows of
SURVEY.md section 8(a)) over one seeded synthetic workload.  N = 1 times BASELINE.json's headline config
C5 (Nt = Nf = 1e6, one series).

The line of record (top-level `value`, `dtype`, `roofline`) is the FP32-pipe form of the path (LSP_PIPE_FP32): the
paper's arithmetic -- fp32 throughout, SFU sin/cos at the anchors -- against the FP32 +
MUFU issue roofline BASELINE.json's metric names.  The same run then times the library's automatic plan, which on this
workload is the tensor-core factorisation with fp16 hi + e5m2 correction operands, and reports it as the sub-record
`fast_path` (its own events, clocks, roofline and parity): narrower operand arithmetic than the paper's, so it is never
the headline.  `parity` carries max|P_gpu - P_oracle| / max P_oracle and the arg-max agreement of each timed
configuration on the oracle subset this run computes for `cpu_baseline` (outside the timed regions).

N > 1 (torchrun): --shard series (default): every rank runs its own series of the same shape (weak scaling, no data-path
collective: the path shards by independent series); value = all ranks' terms / max-over-ranks
time.  --shard freq: ONE series, rank g computes the contiguous frequency slice (f_min + k_g df, df, Nf_g) and the global
peak is merged by an 8-byte MAXLOC exchange (strong scaling).

Prints ONE JSON line (rank 0).  `--impl reference` times the fp64 oracle (oracle/, the CPU baseline)
on a bounded sample of the same workload instead.
"""
from __future__ import annotations

import argparse
import json
import os
import statistics
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import workloads  # noqa: E402  (seeded input generators; hold none of the method's arithmetic)

METRIC = "lomb_scargle_term_evals_per_s"
UNIT = "terms/s"
TENSOR_FLOP_PER_TERM = 16            # complex MAC for W = XC + i XS plus complex MAC for V = (CC-SS) + 2i CS: 8 real MACs
TENSOR_FLOP_PER_TERM_EXECUTED = 32   # W runs as three fp16 passes (hi*hi + lo*hi + hi*lo), V as one
TENSOR_FLOP_PER_TERM_EXECUTED_CORR8 = 24   # fp16-rate equivalent when both correction products share one e5m2 MMA of K = 32
                                           # (16 FLOP per term at twice the fp16 rate): hi*hi 8 + corrections 8 + V 8
FP32_LANES_PER_SM = 128          # B200: 4 SMSPs x 32 FP32 lanes (guide: blackwell_cuda_programming.md)
MUFU_LANES_PER_SM = 16           # 4 SMSPs x 4
NOMINAL_FP16_TFLOPS = 2250.0     # dense fp16/bf16 tensor peak of B200 (B200_PROFILING.md)
PIPE_FP32, PIPE_TENSOR = 1, 2


# ----------------------------------------------------------------------------- helpers (host logic)
def rank_seed(workload: str, rank: int):
    """Seed of rank r's series: the config's own seed for rank 0, +1000*r for the others."""
    idx = {"C1": 1, "C2": 2, "C3": 3, "C4": 4, "C4S": 4, "C5": 5, "P0": 0}[workload.upper()]
    return None if rank == 0 else workloads.BASE_SEED + idx + 1000 * rank


def reduce_max(value: float, dist=None) -> float:
    """Max over ranks of a scalar (device time); identity when not distributed."""
    if dist is None or not dist.is_initialized() or dist.get_world_size() == 1:
        return float(value)
    import torch
    t = torch.tensor([float(value)], dtype=torch.float64)
    if dist.get_backend() == "nccl":
        t = t.cuda()
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def aggregate_value(terms_per_rank: int, world: int, max_seconds: float) -> float:
    return terms_per_rank * world / max_seconds


def freq_slice(Nf: int, world: int, rank: int):
    """--shard freq: rank g owns the contiguous grid indices [k0, k0 + n) -- every k once, sizes
    differing by at most one -- and calls the library with (f_min + k0 df, df, n)."""
    base, extra = divmod(int(Nf), int(world))
    n = base + (1 if rank < extra else 0)
    k0 = rank * base + min(rank, extra)
    return k0, n


def merge_peaks(local_val: float, local_idx: int, dist=None):
    """Global peak of a frequency-sharded periodogram: MAXLOC over the ranks' (value, global index) pairs, the LOWEST
    index among equal maxima (reading G9).  8 bytes of payload per rank (fp32 value + int32 index)."""
    if dist is None or not dist.is_initialized() or dist.get_world_size() == 1:
        return float(local_val), int(local_idx)
    import torch
    mine = torch.tensor([float(local_val), float(local_idx)], dtype=torch.float64)      # the index is exact in fp64 (< 2^31)
    if dist.get_backend() == "nccl":
        mine = mine.cuda()
    allp = [torch.empty_like(mine) for _ in range(dist.get_world_size())]
    dist.all_gather(allp, mine)
    pairs = [(float(p[0]), int(p[1])) for p in allp]
    best = max(v for v, _ in pairs)
    return best, min(i for v, i in pairs if v == best)


def measured_peaks() -> dict:
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        with open(path) as fh:
            return json.load(fh)
    return {}


class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled DURING the timed region."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int = 0):
        self.proc = None
        self.lines = []
        self.index = index

    def start(self):
        try:
            self.proc = subprocess.Popen(
                ["nvidia-smi", "-i", str(self.index), "--query-gpu=" + self.Q,
                 "--format=csv,noheader,nounits", "-lms", "20"],
                stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.thread = threading.Thread(target=self._read, daemon=True)
            self.thread.start()
        except OSError:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.lines.append(line.strip())

    def stop(self) -> dict:
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except Exception:
            self.proc.kill()
        sm, smax, pw, reasons = [], [], [], set()
        names = ("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap")
        for ln in self.lines:
            parts = [p.strip() for p in ln.split(",")]
            if len(parts) < 7:
                continue
            try:
                sm.append(float(parts[0])); smax.append(float(parts[1])); pw.append(float(parts[2]))
            except ValueError:
                continue
            for n, v in zip(names, parts[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(n)
        if not sm:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["no samples"]}
        return {"sm_mhz": statistics.median(sm), "sm_max_mhz": max(smax), "power_w_max": max(pw),
                "samples": len(sm), "reasons": sorted(reasons)}


# ----------------------------------------------------------------------------- oracle legs (CPU)
def time_oracle(w, seconds_target: float = 12.0, max_freqs: int = 4096, keep: bool = False):
    """Time the fp64 oracle, as it stands, on a strided subset of the workload's frequency grid.

    Returns (terms_per_s, cores, sample_description, elapsed_s[, ks, P_ref of series 0 when keep])."""
    import oracle
    t = w.t[0] if (w.B > 1 and w.t.ndim == 2) else w.t          # batch: series 0 (shared-time batch: the one time vector)
    x = w.x[0] if w.B > 1 else w.x
    cores = oracle.host_threads()
    oracle.periodogram(t[:1000], x[:1000], w.f_min, w.df, 8)          # build + warm the library
    done, elapsed, n = 0, 0.0, max(8, cores * 4)
    kept_ks, kept_P = [], []
    while elapsed < seconds_target and done < max_freqs:
        n = min(n, max_freqs - done)
        stride = max(1, w.Nf // n)
        ks = (np.arange(n, dtype=np.int64) * stride + done % stride) % w.Nf
        t0 = time.perf_counter()
        P, used = oracle.periodogram(t, x, w.f_min, w.df, w.Nf, ks=ks, return_threads=True)
        dt = time.perf_counter() - t0
        elapsed += dt; done += n; cores = used
        if keep:
            kept_ks.append(ks); kept_P.append(P)
        rate = n * w.Nt / dt
        n = int(min(max_freqs, max(n, rate * (seconds_target - elapsed) / w.Nt * 0.9))) or 1
        if seconds_target - elapsed < 0.5:
            break
    terms = done * w.Nt
    sample = "%d of %d frequencies (strided) x Nt=%d samples of %s%s" % (
        done, w.Nf, w.Nt, w.name, " series 0" if w.B > 1 else "")
    if keep:
        return terms / elapsed, cores, sample, elapsed, np.concatenate(kept_ks), np.concatenate(kept_P)
    return terms / elapsed, cores, sample, elapsed


def parity_record(w, P_gpu, ks, P_ref, peak_gpu: int):
    """max|P_gpu - P_oracle| / max P_oracle on the oracle subset of this run, plus the arg-max: the oracle over a dense
    window of +-32 bins around the GPU's peak (and the expected bin) must put its maximum at the GPU's index."""
    import oracle
    t = w.t[0] if (w.B > 1 and w.t.ndim == 2) else w.t
    x = w.x[0] if w.B > 1 else w.x
    centres = [peak_gpu] + ([int(round(w.expected_peak_bin))] if w.expected_peak_bin is not None else [])
    win = np.unique(np.concatenate([np.arange(max(0, c - 32), min(w.Nf, c + 33), dtype=np.int64) for c in centres]))
    P_win = oracle.periodogram(t, x, w.f_min, w.df, w.Nf, ks=win)
    all_ks = np.concatenate([ks, win]); all_ref = np.concatenate([P_ref, P_win])
    err = float(np.max(np.abs(P_gpu[all_ks].astype(np.float64) - all_ref)) / np.max(all_ref))
    k_ref = int(all_ks[int(np.argmax(all_ref))])
    return {"max_rel_err": err, "tolerance": 1e-4, "argmax_equal": bool(k_ref == int(peak_gpu)), "argmax_gpu": int(peak_gpu),
            "argmax_oracle_on_sample": k_ref, "frequencies_compared": int(all_ks.size)}


def run_reference(args):
    """--impl reference: the oracle on the host cores, bounded sample per step; rank 0 only."""
    if int(os.environ.get("RANK", "0")) != 0:
        return 0
    w = workloads.make(args.workload)
    per_step = max(1.0, min(20.0, 120.0 / max(1, args.steps + args.warmup)))
    for _ in range(args.warmup):
        time_oracle(w, seconds_target=min(per_step, 2.0))
    rates, cores, sample = [], 1, ""
    t0 = time.perf_counter()
    for _ in range(args.steps):
        r, cores, sample, _ = time_oracle(w, seconds_target=per_step)
        rates.append(r)
    wall = time.perf_counter() - t0
    value = statistics.mean(rates)
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * wall / max(1, args.steps),
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": w.name, "Nt": w.Nt, "Nf": w.Nf, "series": w.B,
                   "note": "fp64 two-pass oracle (oracle/lsp_oracle.c, OpenMP) on a strided frequency subset"},
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line))
    return 0


# ----------------------------------------------------------------------------- our arm (GPU)
def roofline_record(terms, B, Nt, Nf, plan, k_ms, all_ms, clocks, peaks, n_sm, workload_name):
    """Roofline of the dominant (accumulate) kernel of one timed configuration."""
    sm_max = float(peaks.get("sm_max_mhz", 1965.0))
    peak_tflops = n_sm * FP32_LANES_PER_SM * 2 * sm_max * 1e6 / 1e12
    lane_ops = plan["lane_ops_per_term"]
    sm_mhz = clocks.get("sm_mhz") if clocks else None
    if lane_ops:                                             # FP32-pipe form: 6 lane-ops (FMA = 2 FLOP) per term
        achieved = terms * lane_ops * 2 / (k_ms * 1e-3) / 1e12
        mufu_per_s = terms * 2.0 / plan["K"] / (k_ms * 1e-3)            # one MUFU.SIN + one MUFU.COS per anchor = per K terms
        mufu_peak = n_sm * MUFU_LANES_PER_SM * sm_max * 1e6
        rec = {
            "bound": "alu", "achieved": achieved, "peak": peak_tflops, "unit": "TFLOP/s", "frac": achieved / peak_tflops,
            "lane_ops_per_term": lane_ops,
            "peak_basis": "FP32 issue: %d SMs x 128 FP32 lanes x 2 FLOP x %.0f MHz (sm_max_mhz of MEASURED_PEAKS.json%s)"
                          % (n_sm, sm_max, "" if peaks else "; fallback"),
            "frac_at_measured_clock": (achieved / (n_sm * FP32_LANES_PER_SM * 2 * sm_mhz * 1e6 / 1e12)) if sm_mhz else None,
            "mufu_frac": mufu_per_s / mufu_peak,
            "mufu_basis": "2 MUFU per K = %d terms against %d SMs x 16 lanes x %.0f MHz" % (plan["K"], n_sm, sm_max),
        }
    else:                                                    # tensor-core form: 8 real MACs = 16 FLOP per term
        tpeak = float(peaks.get("bf16_tflops_sustained", peaks.get("bf16_tflops", 1590.0)))   # fp16 rate = bf16 rate
        burst = float(peaks.get("bf16_tflops", tpeak))
        alg_flop = TENSOR_FLOP_PER_TERM
        executed = TENSOR_FLOP_PER_TERM_EXECUTED_CORR8 if "e5m2corr" in plan["kernel"] else TENSOR_FLOP_PER_TERM_EXECUTED
        if "shared_gemm" in plan["kernel"]:                  # shared-time batch: only W = XC + i XS is per series (one real MAC each for
            alg_flop, executed = 4, 8                        # cos and sin: 4 FLOP per term); executed: main product 4 + e5m2 corrections 4
        achieved = terms * alg_flop / (k_ms * 1e-3) / 1e12
        rec = {
            "bound": "tensor", "achieved": achieved, "peak": tpeak, "unit": "TFLOP/s", "frac": achieved / tpeak,
            "frac_vs_burst_peak": achieved / burst, "frac_vs_nominal_fp16_peak": achieved / NOMINAL_FP16_TFLOPS,
            "flop_per_term_algorithmic": alg_flop, "flop_per_term_executed": executed,
            "frac_executed": achieved * executed / alg_flop / tpeak,
            "peak_basis": "MEASURED_PEAKS.json bf16_tflops_sustained (cuBLAS bf16 back to back; fp16 has the same nominal "
                          "rate; the kernel is timed inside a step that is itself power-capped): %s"
                          % ("measured" if peaks else "fallback 1590"),
            "fp32_alu_equivalent_frac": terms * 12 / (k_ms * 1e-3) / 1e12 / peak_tflops,
        }
    alg_bytes = 12.0 * B * Nt + 4.0 * B * Nf
    rec.update({
        "traffic": None, "kernel": plan["kernel"], "kernel_ms": k_ms,
        "kernel_share_of_step": k_ms / statistics.mean(all_ms),
        "algorithmic_bytes": alg_bytes, "hbm_GBps_algorithmic": alg_bytes / (k_ms * 1e-3) / 1e9,
    })
    prof = os.path.join(ROOT, "profiles", "traffic.json")
    if os.path.exists(prof):
        try:
            with open(prof) as fh:
                rec["traffic"] = json.load(fh).get("%s/%s" % (workload_name, plan["kernel"]))
        except Exception:
            pass
    if rec["traffic"]:
        rec["traffic_over_algorithmic"] = rec["traffic"] / alg_bytes
    return rec


def dtype_of(plan) -> str:
    if plan["lane_ops_per_term"]:
        return "f32"
    return "f16 + e5m2 correction operands, f32 accumulate" if "e5m2corr" in plan["kernel"] else "f16 hi+lo operands, f32 accumulate"


def run_ours(args):
    import torch
    import torch.distributed as dist
    import paper_1007_1658_b200 as lsp

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device -- the product path has no CPU fallback")
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    dd = dist if world > 1 else None

    shard_freq = args.shard == "freq" and world > 1
    w = workloads.make(args.workload, seed=None if shard_freq else rank_seed(args.workload, rank))
    if shard_freq and w.B > 1:
        raise SystemExit("--shard freq is for a single series")
    batched = w.B > 1
    k0, Nf_local = freq_slice(w.Nf, world, rank) if shard_freq else (0, w.Nf)
    f_min_local = w.f_min + k0 * w.df
    terms_local = w.B * w.Nt * Nf_local
    h = lsp.Handle(local)
    for key, val in ((lsp.PARAM_K, args.K), (lsp.PARAM_THREADS, args.threads), (lsp.PARAM_NSPLIT, args.nsplit),
                     (lsp.PARAM_FLUSH, args.flush), (lsp.PARAM_TABLE_MB, args.table_mb), (lsp.PARAM_COARSE, args.coarse),
                     (lsp.PARAM_TRUNC, args.trunc), (lsp.PARAM_CORR, args.corr)):
        if val:
            h.set_param(key, val)
    h.set_param(lsp.PARAM_TIMING, 1)

    t_h = torch.from_numpy(np.ascontiguousarray(w.t)).pin_memory()
    x_h = torch.from_numpy(np.ascontiguousarray(w.x)).pin_memory()
    t_d, x_d = t_h.cuda(), x_h.cuda()
    flush_buf = torch.empty(256 << 20, dtype=torch.uint8, device="cuda")        # > 126 MB L2
    shape = (w.B, Nf_local) if batched else (Nf_local,)
    P_d = torch.empty(shape, dtype=torch.float32, device="cuda")
    P_h = torch.empty(shape, dtype=torch.float32).pin_memory()
    pi_h = torch.empty(w.B, dtype=torch.int32).pin_memory()
    pv_h = torch.empty(w.B, dtype=torch.float32).pin_memory()
    out = {}

    def step_device():
        if batched:
            out["P"], out["pi"], out["pv"] = h.periodogram_batched(t_d, x_d, f_min_local, w.df, Nf_local)
        else:
            out["P"] = h.periodogram(t_d, x_d, f_min_local, w.df, Nf_local, out=P_d)

    def step_host():
        if batched:
            h.periodogram_batched_host(t_h, x_h, f_min_local, w.df, Nf_local, P=P_h, peak_idx=pi_h, peak_val=pv_h)
        else:
            h.periodogram_host(t_h, x_h, f_min_local, w.df, Nf_local, out=P_h)

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    def time_config(pipe: int):
        """Warm up, then time exactly `steps` device-resident steps (CUDA events, L2 flushed between them, clocks sampled
        during), then the end-to-end host-buffer steps.  Returns the raw measurements of this configuration."""
        h.set_param(lsp.PARAM_PIPE, pipe)
        for _ in range(max(3, args.warmup)):
            step_device()
        torch.cuda.synchronize()
        sampler = ClockSampler(local)
        if rank == 0:
            sampler.start()
            time.sleep(0.3)
        evs = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(args.steps)]
        barrier()
        for ea, eb in evs:
            flush_buf.zero_()                                   # L2 flush between timed iterations (outside the step's events)
            ea.record()
            step_device()                                       # enqueue only: no host sync inside the timed region
            eb.record()
        barrier()
        total_ms = sum(ea.elapsed_time(eb) for ea, eb in evs)   # device time of exactly K steps, flushes excluded
        kern_ms, all_ms = [], []
        for back in range(min(args.steps, 64)):                 # per-kernel CUDA events recorded by the library on
            tm = h.call_timing(back)                            # the launching stream during the timed region
            kern_ms.append(tm["accumulate"]); all_ms.append(sum(tm.values()))
        clocks = sampler.stop() if rank == 0 else None
        plan = h.last_plan()
        P_last = out["P"].clone()
        peak = None
        if not batched:                                         # global peak; merged over the ranks when the grid is sharded
            pv, pi = torch.max(P_last, dim=0)
            peak = merge_peaks(float(pv), int(pi) + k0, dd if shard_freq else None)
        # end to end through the host-buffer C-ABI call (H2D + compute + D2H inside the timed region)
        for _ in range(2):
            step_host()
        barrier()
        t0 = time.perf_counter()
        for _ in range(args.steps):
            step_host()
        torch.cuda.synchronize()
        e2e_s = reduce_max((time.perf_counter() - t0) / args.steps, dd)
        return {"pipe": pipe, "ms_per_step": reduce_max(total_ms / args.steps, dd), "kern_ms": kern_ms, "all_ms": all_ms,
                "clocks": clocks, "plan": plan, "P": P_last, "peak": peak, "e2e_s": e2e_s}

    def time_config_checked(pipe: int):
        """time_config, re-measured ONCE (after a pause) if the clocks sampled during the timed region show a thermal or
        hardware slowdown, or sit well below the maximum with no reason given (a leftover clock lock).  sw_power_cap is kept."""
        m = time_config(pipe)
        bad = lambda c: c is not None and c.get("sm_mhz") is not None and (
            any(r in ("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown") for r in c["reasons"])
            or (not c["reasons"] and c["sm_mhz"] < 0.8 * c["sm_max_mhz"]))
        flag = torch.tensor([1.0 if bad(m["clocks"]) else 0.0], device="cuda")
        if world > 1:
            dist.broadcast(flag, src=0)                                   # every rank takes rank 0's decision
        if flag.item() > 0:
            time.sleep(3.0)
            first = m["clocks"]
            m = time_config(pipe)
            if m["clocks"] is not None:
                m["clocks"]["remeasured_after"] = first
        return m

    rec = time_config_checked(args.pipe if args.pipe else PIPE_FP32)      # the line of record: the paper's fp32 arithmetic
    fast = None
    if not args.pipe and not args.no_fast_path:
        fast = time_config_checked(0)                                     # the library's automatic plan
        if fast["plan"]["kernel"] == rec["plan"]["kernel"]:
            fast = None                                                   # (same kernel: nothing to add)
    fast16 = None
    if fast is not None and "pair2" in fast["plan"]["kernel"] and not args.no_fast_path:
        # the same tensor form with the corrections as two fp16 MMAs: 22 significant operand bits in every product of XC, XS
        h.set_param(lsp.PARAM_CORR, 1)
        fast16 = time_config_checked(0)
        h.set_param(lsp.PARAM_CORR, 0)
    h2d = t_h.numel() * 8 + x_h.numel() * 4
    d2h = P_h.numel() * 4 + (pi_h.numel() * 8 if batched else 0)

    if rank != 0:
        h.close()
        if world > 1:
            dist.destroy_process_group()
        return 0

    peaks = measured_peaks()
    n_sm = torch.cuda.get_device_properties(local).multi_processor_count

    cpu, oracle_keep = None, None
    if world == 1 and not args.no_cpu_baseline:
        r, cores, sample, _, ks, P_ref = time_oracle(w, seconds_target=args.cpu_seconds, keep=True)
        cpu = {"value": r, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample}
        oracle_keep = (ks, P_ref)

    def whole_job(seconds):
        return w.terms / seconds if shard_freq else aggregate_value(terms_local, world, seconds)

    def finish_record(m):
        k_ms = statistics.mean(m["kern_ms"])
        roof = roofline_record(terms_local, w.B, w.Nt, Nf_local, m["plan"], k_ms, m["all_ms"], m["clocks"], peaks, n_sm, w.name)
        d = {"dtype": dtype_of(m["plan"]), "value": whole_job(m["ms_per_step"] * 1e-3), "unit": UNIT, "ms_per_step": m["ms_per_step"],
             "plan": m["plan"], "clocks": m["clocks"],
             "e2e": {"value": whole_job(m["e2e_s"]), "unit": UNIT, "ms_per_step": m["e2e_s"] * 1e3,
                     "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h},
             "gpu_launches": m["plan"]["launches"] * args.steps, "roofline": roof}
        if oracle_keep is not None:
            Pg = m["P"].cpu().numpy()
            Pg0 = Pg[0] if batched else Pg
            d["parity"] = parity_record(w, Pg0, oracle_keep[0], oracle_keep[1], int(np.argmax(Pg0)))
        if m["peak"] is not None:
            d["peak"] = {"value": m["peak"][0], "index": m["peak"][1]}
        return d

    r0 = finish_record(rec)
    line = {
        "metric": METRIC, "value": r0["value"], "unit": UNIT, "n_gpus": world, "steps": args.steps,
        "warmup": max(3, args.warmup), "ms_per_step": r0["ms_per_step"], "higher_is_better": True,
        "scaling": "strong" if shard_freq else "weak",
        "vs_baseline": None, "dtype": r0["dtype"], "data": "synthetic",
        "config": {"workload": w.name, "Nt": w.Nt, "Nf": w.Nf, "series": w.B,
                   "terms_per_step": w.terms * (1 if shard_freq else world),
                   "l2": "flushed between timed iterations (256 MB write)", "plan": r0["plan"],
                   "arithmetic": "line of record = LSP_PIPE_FP32 (the paper's fp32 arithmetic, PAPER.md:140, :290); "
                                 "fast_path = the library's automatic plan, timed in the same run",
                   "parallelism": ("single GPU" if world == 1 else
                                   ("one series, contiguous frequency slices per rank, MAXLOC peak merge" if shard_freq
                                    else "independent series per rank"))},
        "clocks": r0["clocks"], "e2e": r0["e2e"], "gpu_launches": r0["gpu_launches"], "roofline": r0["roofline"],
        "cpu_baseline": cpu,
    }
    for k in ("parity", "peak"):
        if k in r0:
            line[k] = r0[k]
    if fast is not None:
        f0 = finish_record(fast)
        f0["note"] = ("tensor-core factorisation of the same sums (DESIGN.md section 6b): operand arithmetic narrower than "
                      "the paper's fp32, inside the path's 1e-4 max P tolerance; reported, not the headline")
        f0["speedup_over_line_of_record"] = r0["ms_per_step"] / f0["ms_per_step"]
        line["fast_path"] = f0
    if fast16 is not None:
        f1 = finish_record(fast16)
        f1["note"] = ("the fast path with LSP_PARAM_CORR = 1: first-order corrections of the fp16 hi + lo operand split as two fp16 MMAs "
                      "(22 significant operand bits per product of XC, XS -- no less than the paper's fp32 with SFU trig, PAPER.md:290; "
                      "CC, CS in one fp16 pass, fp32 accumulation in the tensor core); reported, not the headline")
        f1["speedup_over_line_of_record"] = r0["ms_per_step"] / f1["ms_per_step"]
        line["fast_path_fp16x3"] = f1
    if world == 1 and w.name == "C5" and not args.pipe and not args.no_extras:
        # SURVEY.md section 8(f) row 3 in the driver's own run: the paper-shaped P0 in the FP32 form and the automatic
        # plan (whole-call device time, median of 5, L2 flushed), and the N_t sweep of this workload in the FP32 form (slope -> 2)
        extras = {}
        p0 = workloads.make("P0")
        t0_d, x0_d = torch.from_numpy(p0.t).cuda(), torch.from_numpy(p0.x).cuda()
        P0_d = torch.empty(p0.Nf, dtype=torch.float32, device="cuda")
        for name, pipe in (("fp32", PIPE_FP32), ("automatic", 0)):
            h.set_param(lsp.PARAM_PIPE, pipe)
            for _ in range(2):
                h.periodogram(t0_d, x0_d, p0.f_min, p0.df, p0.Nf, out=P0_d)
            ms = []
            for _ in range(5):
                flush_buf.zero_()
                ea, eb = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                ea.record(); h.periodogram(t0_d, x0_d, p0.f_min, p0.df, p0.Nf, out=P0_d); eb.record()
                torch.cuda.synchronize()
                ms.append(ea.elapsed_time(eb))
            med = statistics.median(ms)
            extras["P0_" + name] = {"ms": med, "terms_per_s": p0.terms / (med * 1e-3), "kernel": h.last_plan()["kernel"],
                                    "peak_index": int(torch.argmax(P0_d)), "expected_peak_bin": p0.expected_peak_bin}
        extras["P0_note"] = "paper-shaped run: Nt = 382,003, Nf = 1,528,064 (5.84e11 terms, the count behind the paper's Table 2)"
        h.set_param(lsp.PARAM_PIPE, PIPE_FP32)
        extras["sweep_fp32"] = sweep_rows(h, w, 5, steps=(16, 8, 4, 2), flush_buf=flush_buf)
        h.set_param(lsp.PARAM_PIPE, 0)
        line["extras"] = extras
    if batched:
        # BASELINE config 4: "report per-series peak power distribution" -- the peaks the last host-buffer step returned,
        # and their false-alarm probabilities by eq. (3) with N_ind = Nf (lsp_false_alarm)
        pv = pv_h.numpy().astype(np.float64)
        fap = h.false_alarm(pv_h.cuda(), w.Nt, float(w.Nf)).cpu().numpy().astype(np.float64)
        q = np.quantile(pv, [0.05, 0.25, 0.5, 0.75, 0.95])
        line["peak_power_distribution"] = {
            "series": int(pv.size), "mean": float(pv.mean()), "std": float(pv.std()), "min": float(pv.min()), "max": float(pv.max()),
            "q05": float(q[0]), "q25": float(q[1]), "q50": float(q[2]), "q75": float(q[3]), "q95": float(q[4]),
            "mean_power_all_bins": float(P_h.numpy().mean(dtype=np.float64)),
            "false_alarm_eq3_median": float(np.median(fap)), "fraction_with_fap_below_0.01": float((fap < 0.01).mean()),
            # the Monte-Carlo use of PAPER.md:369: the number of independent frequencies that makes eq. (3) give a false-alarm
            # probability of 1/2 at the median peak of the noise ensemble (report only; host arithmetic on the device's peaks)
            "n_ind_from_median_peak": float(np.log(0.5) / np.log1p(-(1.0 - 2.0 * q[2] / (w.Nt - 1)) ** ((w.Nt - 3) / 2.0))),
        }
    print(json.dumps(line))
    h.close()
    if world > 1:
        dist.destroy_process_group()
    return 0


def run_sweep(args):
    """N_t scaling sweep (the paper's Fig. 4): the workload is uniformly
    down-sampled by 64, 32, ..., 1 with N_f in proportion to N_t; whole-call device time (all kernels, CUDA events) per
    size, and the log-log slope d log t / d log N_t, which the paper expects to approach 2.  One JSON line."""
    import paper_1007_1658_b200 as lsp
    base = workloads.make(args.workload)
    h = lsp.Handle(0)
    if args.pipe:
        h.set_param(lsp.PARAM_PIPE, args.pipe)
    rows = sweep_rows(h, base, max(5, args.steps // 2))
    h.close()
    print(json.dumps({"metric": "lomb_scargle_Nt_sweep", "workload": base.name, "unit": "ms", "data": "synthetic",
                      "note": "uniform down-sampling, Nf proportional to Nt (PAPER.md:351-353, eq. (11)); expected slope -> 2",
                      "sweep": rows}))
    return 0


def sweep_rows(h, base, reps, steps=(64, 32, 16, 8, 4, 2, 1), flush_buf=None):
    """Whole-call device time of `base` down-sampled by each of `steps` (Nf in proportion), L2 flushed between calls."""
    import torch
    if flush_buf is None:
        flush_buf = torch.empty(256 << 20, dtype=torch.uint8, device="cuda")
    rows = []
    for step in steps:
        w = workloads.downsample(base, step) if step > 1 else base
        t_d = torch.from_numpy(np.ascontiguousarray(w.t)).cuda()
        x_d = torch.from_numpy(np.ascontiguousarray(w.x)).cuda()
        P_d = torch.empty(w.Nf, dtype=torch.float32, device="cuda")
        for _ in range(3):
            h.periodogram(t_d, x_d, w.f_min, w.df, w.Nf, out=P_d)
        torch.cuda.synchronize()
        ms = []
        for _ in range(reps):
            flush_buf.zero_()
            ea, eb = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            ea.record(); h.periodogram(t_d, x_d, w.f_min, w.df, w.Nf, out=P_d); eb.record()
            torch.cuda.synchronize()
            ms.append(ea.elapsed_time(eb))
        med = statistics.median(ms)
        rows.append({"Nt": w.Nt, "Nf": w.Nf, "ms_median": med, "ms_min": min(ms), "terms_per_s": w.terms / (med * 1e-3),
                     "kernel": h.last_plan()["kernel"]})
    for a, b in zip(rows[:-1], rows[1:]):
        b["slope_vs_previous"] = float(np.log(b["ms_median"] / a["ms_median"]) / np.log(b["Nt"] / a["Nt"]))
    return rows


def run_back_to_back(args):
    """SURVEY.md section 8(d) protocol for the small configs: N back-to-back device-pointer calls on one stream, no L2 flush, no
    host synchronisation in between (separates launch latency from arithmetic); eager, and captured once into a CUDA graph and
    replayed.  One JSON line."""
    import torch
    import paper_1007_1658_b200 as lsp
    w = workloads.make(args.workload)
    if w.B > 1:
        raise SystemExit("--back-to-back is for a single series")
    h = lsp.Handle(0)
    for key, val in ((lsp.PARAM_PIPE, args.pipe), (lsp.PARAM_NSPLIT, args.nsplit), (lsp.PARAM_COARSE, args.coarse), (lsp.PARAM_K, args.K),
                     (lsp.PARAM_THREADS, args.threads)):
        if val:
            h.set_param(key, val)
    t_d = torch.from_numpy(np.ascontiguousarray(w.t)).cuda()
    x_d = torch.from_numpy(np.ascontiguousarray(w.x)).cuda()
    P_d = torch.empty(w.Nf, dtype=torch.float32, device="cuda")
    n = args.back_to_back
    for _ in range(20):
        h.periodogram(t_d, x_d, w.f_min, w.df, w.Nf, out=P_d)
    torch.cuda.synchronize()
    ea, eb = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    ea.record()
    for _ in range(n):
        h.periodogram(t_d, x_d, w.f_min, w.df, w.Nf, out=P_d)
    eb.record(); torch.cuda.synchronize()
    eager_ms = ea.elapsed_time(eb) / n
    plan = h.last_plan()
    st = torch.cuda.Stream()
    with torch.cuda.stream(st):
        for _ in range(3):
            h.periodogram(t_d, x_d, w.f_min, w.df, w.Nf, out=P_d, stream=st)
        g = torch.cuda.CUDAGraph()
        with torch.cuda.graph(g, stream=st):
            h.periodogram(t_d, x_d, w.f_min, w.df, w.Nf, out=P_d, stream=st)
        torch.cuda.synchronize()
        ea.record(st)
        for _ in range(n):
            g.replay()
        eb.record(st); torch.cuda.synchronize()
    graph_ms = ea.elapsed_time(eb) / n
    h.close()
    print(json.dumps({"metric": "lomb_scargle_back_to_back_call_ms", "workload": w.name, "calls": n, "unit": "ms per call", "data": "synthetic",
                      "eager_ms_per_call": eager_ms, "graph_replay_ms_per_call": graph_ms, "terms_per_s_eager": w.terms / (eager_ms * 1e-3),
                      "plan": plan, "note": "device-pointer calls back to back on one stream, no L2 flush, no host sync between calls"}))
    return 0


def run_variants(args):
    """SURVEY.md section 8(f) row 1 beside the classical periodogram, same workload, same protocol: whole-call device time (CUDA
    events, L2 flushed between calls) of lsp_periodogram, lsp_periodogram_gls and lsp_periodogram_gls_weighted in the FP32-pipe
    form and under the automatic plan, each checked against ITS oracle function on sampled series; for a single series within its
    limits also lsp_periodogram_static.  One JSON line."""
    import torch
    import paper_1007_1658_b200 as lsp
    import oracle
    w = workloads.make(args.workload)
    batched = w.B > 1
    t2 = np.ascontiguousarray(w.t if w.t.ndim == 2 or not batched else np.broadcast_to(w.t, w.x.shape)).reshape(w.B, -1) if batched else w.t.reshape(1, -1)
    x2 = np.ascontiguousarray(w.x).reshape(w.B, -1)
    wts = np.random.default_rng(20100716).uniform(0.2, 3.0, x2.shape).astype(np.float32)      # heteroscedastic weights 1 / sigma^2
    t_d = torch.from_numpy(np.ascontiguousarray(w.t)).cuda()
    x_d = torch.from_numpy(np.ascontiguousarray(w.x)).cuda()
    w_d = torch.from_numpy(wts if batched else wts[0]).cuda()
    flush_buf = torch.empty(256 << 20, dtype=torch.uint8, device="cuda")
    h = lsp.Handle(0)
    sample = sorted(set([0, w.B // 2, w.B - 1]))
    ks = np.unique(np.linspace(0, w.Nf - 1, min(w.Nf, 2048)).astype(np.int64))
    refs = {}

    def ref_of(kind, b):
        if (kind, b) not in refs:
            tb, xb = t2[b if t2.shape[0] > 1 else 0], x2[b]
            if kind == "classical":
                refs[(kind, b)] = oracle.periodogram(tb, xb, w.f_min, w.df, w.Nf, ks=ks)
            elif kind == "generalised":
                refs[(kind, b)] = oracle.periodogram_gls(tb, xb, w.f_min, w.df, w.Nf, ks=ks)
            else:
                refs[(kind, b)] = oracle.periodogram_gls_weighted(tb, xb, wts[b], w.f_min, w.df, w.Nf, ks=ks)
        return refs[(kind, b)]

    def call(kind):
        gls = kind != "classical"
        wt = w_d if kind == "weighted" else None
        if batched:
            return h.periodogram_batched(t_d, x_d, w.f_min, w.df, w.Nf, gls=gls, weights=wt)[0]
        return h.periodogram(t_d, x_d, w.f_min, w.df, w.Nf, gls=gls, weights=wt).reshape(1, -1)

    def timed(fn):
        for _ in range(3):
            P = fn()
        torch.cuda.synchronize()
        ms = []
        for _ in range(max(5, args.steps)):
            flush_buf.zero_()
            ea, eb = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            ea.record(); P = fn(); eb.record()
            torch.cuda.synchronize()
            ms.append(ea.elapsed_time(eb))
        return statistics.median(ms), P

    rows = []
    for pipe, form in ((lsp.PIPE_FP32, "FP32 pipe"), (0, "automatic")):
        h.set_param(lsp.PARAM_PIPE, pipe)
        for kind in ("classical", "generalised", "weighted"):
            ms, P = timed(lambda: call(kind))
            plan = h.last_plan()
            Pn = P.cpu().numpy()
            err = max(float(np.max(np.abs(Pn[b][ks] - ref_of(kind, b))) / max(np.max(Pn[b]), np.max(ref_of(kind, b)))) for b in sample)
            rows.append({"form": form, "periodogram": kind, "ms": ms, "terms_per_s": w.terms / (ms * 1e-3), "kernel": plan["kernel"],
                         "launches": plan["launches"], "max_rel_err_vs_oracle": err, "series_checked": len(sample), "frequencies_checked": int(ks.size)})
    if not batched and w.Nt <= lsp.STATIC_MAX_NT and w.Nf <= lsp.STATIC_MAX_NF:
        P_s = torch.empty(w.Nf, dtype=torch.float32, device="cuda")
        ms, P = timed(lambda: lsp.periodogram_static(t_d, x_d, w.f_min, w.df, w.Nf, out=P_s).reshape(1, -1))
        Pn = P.cpu().numpy()[0]
        err = float(np.max(np.abs(Pn[ks] - ref_of("classical", 0))) / max(np.max(Pn), np.max(ref_of("classical", 0))))
        rows.append({"form": "FP32 pipe, lsp_periodogram_static (no allocation)", "periodogram": "classical", "ms": ms,
                     "terms_per_s": w.terms / (ms * 1e-3), "kernel": "accum_z_kernel", "launches": 3, "max_rel_err_vs_oracle": err,
                     "series_checked": 1, "frequencies_checked": int(ks.size)})
    h.close()
    print(json.dumps({"metric": "lomb_scargle_variants_ms", "workload": w.name, "unit": "ms per call", "data": "synthetic",
                      "config": {"workload": w.name, "series": w.B, "Nt": w.Nt, "Nf": w.Nf, "l2_flush_between_calls": True},
                      "tolerance": 1e-4, "rows": rows,
                      "note": "whole-call device time (median); weights U[0.2, 3) per sample; each row checked against its own oracle function on a strided frequency subset, the error relative to max P of the series (the largest value the GPU returned over the whole grid)"}))
    return 0


def main(argv=None):
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="C5")
    ap.add_argument("--shard", default="series", choices=["series", "freq"],
                    help="N > 1: independent series per rank (weak scaling) or frequency slices of one series (strong scaling)")
    ap.add_argument("--pipe", type=int, default=0, help="time ONLY this form (1 = FP32 pipe, 2 = tensor cores) instead of the line of record + fast path")
    ap.add_argument("--no-fast-path", action="store_true", help="skip the automatic-plan sub-record")
    ap.add_argument("--no-extras", action="store_true", dest="no_extras", help="default C5 run: skip the P0 and N_t-sweep sub-records")
    ap.add_argument("--K", type=int, default=0)
    ap.add_argument("--threads", type=int, default=0)
    ap.add_argument("--nsplit", type=int, default=0)
    ap.add_argument("--flush", type=int, default=0)
    ap.add_argument("--table-mb", type=int, default=0, dest="table_mb")
    ap.add_argument("--coarse", type=int, default=0)
    ap.add_argument("--trunc", type=int, default=0)
    ap.add_argument("--corr", type=int, default=0, help="with --pipe 2: 1 = LSP_PARAM_CORR (fp16 hi + lo corrections in the CTA-pair kernel)")
    ap.add_argument("--sweep", action="store_true", help="N_t scaling sweep of --workload (single series) instead of the bench line")
    ap.add_argument("--back-to-back", type=int, default=0, dest="back_to_back",
                    help="N back-to-back calls of --workload (single series), eager and as a replayed CUDA graph, instead of the bench line")
    ap.add_argument("--variants", action="store_true",
                    help="time the classical, generalised and weighted periodograms (and the no-allocation entry point) on --workload instead of the bench line")
    ap.add_argument("--cpu-seconds", type=float, default=12.0)
    ap.add_argument("--no-cpu-baseline", action="store_true")
    args = ap.parse_args(argv)
    if args.impl == "reference":
        return run_reference(args)
    if args.sweep:
        return run_sweep(args)
    if args.back_to_back:
        return run_back_to_back(args)
    if args.variants:
        return run_variants(args)
    return run_ours(args)


if __name__ == "__main__":
    sys.exit(main())
