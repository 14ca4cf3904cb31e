"""N > 1 host logic of bench.py on CPU: two gloo ranks, distinct per-rank series, max-over-ranks timing.

The path shards by independent series: no data-path collective exists, so what is
covered here is the plumbing bench.py uses under torchrun -- rank seeds, the MAX all-reduce of the device
time and the whole-job aggregate.  No CUDA, no oracle.
"""
import os
import socket
import sys

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    port = s.getsockname()[1]
    s.close()
    return port


def _worker(rank, world, port, q):
    import torch.distributed as dist
    import bench
    import workloads
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        seed = bench.rank_seed("C1", rank)
        w = workloads.make("C1", Nt=200, Nf=50, seed=seed)
        my_ms = 10.0 + 5.0 * rank                      # pretend device times: rank 1 is slower
        mx = bench.reduce_max(my_ms, dist)
        value = bench.aggregate_value(w.terms, world, mx * 1e-3)
        q.put((rank, seed, float(w.t.sum()), mx, value, w.terms))
    finally:
        dist.destroy_process_group()


def test_two_rank_gloo_max_time_and_aggregate():
    import torch.multiprocessing as mp
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    out = sorted(q.get(timeout=120) for _ in procs)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    (r0, s0, t0, m0, v0, n0), (r1, s1, t1, m1, v1, n1) = out
    assert s0 is None and s1 is not None               # rank 0 keeps the config's own seed
    assert t0 != t1                                    # ranks hold different series
    assert m0 == m1 == 15.0                            # MAX over ranks, seen by both
    assert v0 == v1 == pytest.approx(2 * n0 / 15e-3)   # whole-job units / max time


def _worker_freq(rank, world, port, q):
    """--shard freq host logic: every rank takes its contiguous slice of ONE series' grid, finds its
    local peak (a numpy stand-in for the device's P: this test is about slice bounds and the peak merge, not arithmetic) and the
    ranks merge by MAXLOC, lowest index on ties."""
    import torch.distributed as dist
    import bench
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        Nf = 1001                                      # ragged: 501 + 500
        k0, n = bench.freq_slice(Nf, world, rank)
        P = np.zeros(Nf, dtype=np.float32)
        P[[137, 700, 900]] = [5.0, 9.0, 9.0]           # the global maximum is tied between bins 700 and 900, both on rank 1
        P[400] = 8.5                                   # rank 0's local peak
        local = P[k0:k0 + n]
        val, idx = bench.merge_peaks(float(local.max()), int(local.argmax()) + k0, dist)
        # a tie ACROSS ranks: equal maxima at 300 (rank 0) and 800 (rank 1)
        P2 = np.zeros(Nf, dtype=np.float32); P2[[300, 800]] = 4.0
        l2 = P2[k0:k0 + n]
        val2, idx2 = bench.merge_peaks(float(l2.max()), int(l2.argmax()) + k0, dist)
        q.put((rank, k0, n, val, idx, val2, idx2))
    finally:
        dist.destroy_process_group()


def test_two_rank_gloo_frequency_slices_and_peak_merge():
    import torch.multiprocessing as mp
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker_freq, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    out = sorted(q.get(timeout=120) for _ in procs)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    (r0, k0a, na, v0, i0, w0, j0), (r1, k0b, nb, v1, i1, w1, j1) = out
    assert (k0a, na, k0b, nb) == (0, 501, 501, 500)    # every k owned exactly once, ragged Nf
    assert v0 == v1 == 9.0 and i0 == i1 == 700         # global MAXLOC, lowest index among equal maxima, seen by both ranks
    assert w0 == w1 == 4.0 and j0 == j1 == 300         # tie across ranks: the lower rank's (lower) index wins


def test_frequency_slices_cover_the_grid_once():
    import bench
    for Nf in (1, 7, 1000, 1000003):
        for world in (1, 2, 3, 8):
            seen, total = 0, 0
            for r in range(world):
                k0, n = bench.freq_slice(Nf, world, r)
                assert k0 == seen and n >= 0
                seen += n; total += n
            assert total == Nf
    assert bench.merge_peaks(3.0, 5, None) == (3.0, 5)


def test_single_process_helpers():
    import bench
    assert bench.reduce_max(3.5, None) == 3.5
    assert bench.aggregate_value(10, 4, 2.0) == 20.0
    assert bench.rank_seed("C5", 0) is None
    assert bench.rank_seed("C5", 3) != bench.rank_seed("C5", 2)


def test_reference_arm_is_rank0_only(monkeypatch, capsys):
    import bench
    monkeypatch.setenv("RANK", "1")
    args = bench.argparse.Namespace(workload="C1", steps=1, warmup=0, gpus=2)
    assert bench.run_reference(args) == 0
    assert capsys.readouterr().out == ""               # other ranks exit 0 without work


def test_roofline_record_is_recomputable():
    """The bench line's roofline numbers follow from terms, kernel time and the stated peaks: the FP32 form
    against 148 x 128 lanes x 2 FLOP x clock at 6 lane-ops per term, with the MUFU fraction from 2 MUFU per K terms; the tensor
    form against the measured sustained bf16 figure at 16 FLOP per term."""
    import bench
    peaks = {"sm_max_mhz": 1965.0, "bf16_tflops_sustained": 1376.4, "bf16_tflops": 1628.7}
    clocks = {"sm_mhz": 1965.0, "sm_max_mhz": 1965.0, "reasons": []}
    plan = {"lane_ops_per_term": 6, "K": 32, "kernel": "accum_z_kernel<K=32,fp32,three-term>"}
    r = bench.roofline_record(1e12, 1, 10**6, 10**6, plan, 194.81, [195.0], clocks, peaks, 148, "C5")
    peak = 148 * 128 * 2 * 1.965e9 / 1e12
    assert r["bound"] == "alu" and abs(r["peak"] - peak) < 1e-9
    assert abs(r["achieved"] - 1e12 * 12 / 0.19481 / 1e12) < 1e-6 and abs(r["frac"] - r["achieved"] / peak) < 1e-12
    assert abs(r["frac"] - 0.827) < 2e-3
    assert abs(r["mufu_frac"] - (1e12 * 2 / 32 / 0.19481) / (148 * 16 * 1.965e9)) < 1e-12
    assert r["algorithmic_bytes"] == 16e6 and abs(r["kernel_share_of_step"] - 194.81 / 195.0) < 1e-12
    tplan = {"lane_ops_per_term": 0, "K": 128, "kernel": "accum_umma_pair2_kernel<tcgen05.cta_group2.m256n256.f16+e5m2corr,fine-table>"}
    t = bench.roofline_record(1e12, 1, 10**6, 10**6, tplan, 18.37, [19.4], clocks, peaks, 148, "C5")
    assert t["bound"] == "tensor" and t["peak"] == 1376.4 and t["flop_per_term_algorithmic"] == 16 and t["flop_per_term_executed"] == 24
    assert abs(t["achieved"] - 1e12 * 16 / 0.01837 / 1e12) < 1e-6 and abs(t["frac"] - t["achieved"] / 1376.4) < 1e-12
    assert bench.dtype_of(plan) == "f32" and bench.dtype_of(tplan).startswith("f16 + e5m2")
    assert bench.dtype_of({"lane_ops_per_term": 0, "kernel": "accum_umma_pair2_kernel<tcgen05.cta_group2.m256n256.f16,hi+lo,fine-table>"}).startswith("f16 hi+lo")
