"""Host-only launch planner (csrc/lsp_plan.h through lsp_plan_query): no GPU needed."""
import os
import re

import pytest

import paper_1007_1658_b200 as pkg

SM = 148
FP32, TENSOR = pkg.PIPE_FP32, pkg.PIPE_TENSOR


@pytest.mark.parametrize("B,Nt,Nf", [(1, 1000, 1000), (1, 10000, 10000), (1, 100000, 1000000),
                                     (4096, 1000, 2000), (1, 1000000, 1000000), (1, 2, 1), (3, 77, 5),
                                     (1, 382003, 1528064)])
def test_plan_is_valid_and_covers_the_problem(B, Nt, Nf):
    p = pkg.plan_query_form(SM, B, Nt, Nf, FP32)
    assert p["pipe"] == FP32
    assert p["K"] in (4, 8, 12, 16, 20, 24, 28, 32)
    assert p["threads"] % 32 == 0 and 32 <= p["threads"] <= 256
    assert p["n_freq_blocks"] * p["K"] * p["threads"] >= Nf                 # every frequency is owned
    assert (p["n_freq_blocks"] - 1) * p["K"] * p["threads"] < Nf            # no empty block
    assert p["nsplit"] >= 1 and p["nsplit"] * p["split_len"] >= Nt          # every sample is covered
    assert (p["nsplit"] - 1) * p["split_len"] < Nt                          # no empty split
    assert p["split_len"] % 256 == 0                                        # whole tiles
    assert p["chunks_or_ctas_per_sm"] >= 1
    assert B * p["nsplit"] * 16 * Nf <= (1 << 31) + 16 * Nf                 # workspace cap


def test_big_problems_use_wide_threads_and_fill_the_machine():
    p = pkg.plan_query_form(SM, 1, 1000000, 1000000, FP32)
    assert p["K"] >= 24                                                     # anchor amortised
    units = p["nsplit"] * p["n_freq_blocks"]
    slots = p["chunks_or_ctas_per_sm"] * SM
    waves = units / slots
    assert waves > 8 and (waves % 1.0 > 0.85 or waves % 1.0 == 0.0)         # last wave nearly full


def test_small_problems_split_the_time_axis():
    p = pkg.plan_query_form(SM, 1, 10000, 10000, FP32)
    assert p["nsplit"] * p["n_freq_blocks"] >= SM                           # enough CTAs to touch every SM
    p1 = pkg.plan_query_form(SM, 4096, 1000, 2000, FP32)
    assert p1["nsplit"] == 1                                                # the batch already fills the GPU


def test_plan_query_rejects_bad_sizes():
    with pytest.raises(pkg.LspError):
        pkg.plan_query(SM, 1, 1, 10)
    with pytest.raises(pkg.LspError):
        pkg.plan_query(0, 1, 10, 10)
    with pytest.raises(pkg.LspError):
        pkg.plan_query_form(SM, 1, 10, 10, 3)


@pytest.mark.parametrize("B,Nt,Nf", [(1, 10000, 10000), (1, 100000, 1000000), (4096, 1000, 2000),
                                     (1, 1000000, 1000000), (1, 382003, 1528064), (2, 700, 40000), (1, 5000000, 300000)])
def test_tensor_core_plans_cover_the_problem(B, Nt, Nf):
    """tcgen05 forms: K reports the coarse extent L, a CTA owns 128 L frequencies; L = 128 is the CTA-pair form (even block
    count), whose 3 KB-per-sample table is bounded by time chunks."""
    p = pkg.plan_query_form(SM, B, Nt, Nf, TENSOR)
    L = p["K"]
    assert L in (16, 32, 64, 128) and p["pipe"] == TENSOR
    fpb, threads = 128 * L, (544 if L == 128 else 288)
    assert p["threads"] == threads
    nfb = p["n_freq_blocks"]
    if L == 128:
        assert nfb % 2 == 0 and nfb * fpb >= Nf and (nfb - 2) * fpb < Nf
        nchunks = p["chunks_or_ctas_per_sm"]
        chunk_len = -(-Nt // nchunks)
        chunk_len = -(-chunk_len // 128) * 128
        assert nchunks >= 1 and chunk_len * 3072 <= (1 << 30) + 128 * 3072            # the table of a chunk fits the default budget
        assert (nchunks - 1) * chunk_len < Nt <= nchunks * chunk_len
        assert p["nsplit"] * p["split_len"] >= min(Nt, chunk_len) and (p["nsplit"] - 1) * p["split_len"] < chunk_len
    else:
        assert p["chunks_or_ctas_per_sm"] == {64: 2, 32: 2, 16: 3}[L]
        assert nfb * fpb >= Nf and (nfb - 1) * fpb < Nf
        assert p["nsplit"] >= 1 and p["nsplit"] * p["split_len"] >= Nt and (p["nsplit"] - 1) * p["split_len"] < Nt
    assert p["split_len"] % (128 if L == 128 else 32) == 0
    assert B * p["nsplit"] * 16 * Nf <= (1 << 31) + 16 * Nf
    assert p["est_cycles"] > 0


def test_table_chunks():
    """C5 (3.07 GB of table) runs in three chunks under the default 1 GiB budget, P0 in two, C3 in one."""
    assert pkg.plan_query_form(SM, 1, 1000000, 1000000, TENSOR)["chunks_or_ctas_per_sm"] == 3
    assert pkg.plan_query_form(SM, 1, 382003, 1528064, TENSOR)["chunks_or_ctas_per_sm"] == 2
    assert pkg.plan_query_form(SM, 1, 100000, 1000000, TENSOR)["chunks_or_ctas_per_sm"] == 1


def test_automatic_form():
    """pipe = 0: a tcgen05 form for large accurate-enough problems, the FP32 form for tiny Nt; explicit forms are honoured."""
    big = pkg.plan_query(SM, 1, 1000000, 1000000)
    assert big["pipe"] == TENSOR
    units = big["nsplit"] * big["n_freq_blocks"]
    assert units / SM > 2 and ((units / SM) % 1.0 > 0.85 or units % SM == 0)  # last wave of a chunk nearly full
    assert pkg.plan_query(SM, 1, 100000, 1000000)["pipe"] == TENSOR
    assert pkg.plan_query(SM, 1, 300, 1000000)["pipe"] == FP32               # Nt < 512: V's single fp16 pass is too coarse
    assert pkg.plan_query(SM, 1, 2, 1)["pipe"] == FP32
    auto = pkg.plan_query_form(SM, 1, 1000000, 1000000, 0)
    z = pkg.plan_query_form(SM, 1, 1000000, 1000000, FP32)
    assert auto["pipe"] == TENSOR and auto["est_cycles"] < z["est_cycles"]


def test_tcgen05_coarse_extent_follows_the_grid():
    """Long grids take the CTA-pair tile (tensor-pipe bound); a Monte-Carlo batch of short grids (C4) takes a
    narrow tile that the grid fills, three CTAs per SM."""
    assert pkg.plan_query_form(SM, 1, 1000000, 1000000, TENSOR)["K"] == 128
    c4 = pkg.plan_query_form(SM, 4096, 1000, 2000, TENSOR)
    assert c4["K"] == 16 and c4["n_freq_blocks"] == 1 and c4["nsplit"] == 1
    assert pkg.plan_query(SM, 4096, 1000, 2000)["pipe"] == TENSOR


def test_occupancy_model_matches_the_compiled_kernels():
    """The planner's register table (plan_regs in csrc/lsp_plan.h) is what ptxas reported for accum_z_kernel<K> in the build
    that produced the library (paper_1007_1658_b200/build_ptxas.log), and the loaded library is not older than its sources."""
    import importlib
    b = importlib.import_module("paper_1007_1658_b200.build")
    b.build()
    assert not b.is_stale()
    log = open(os.path.join(b.PKG, "build_ptxas.log")).read()
    src = open(os.path.join(b.CSRC, "lsp_plan.h")).read()
    table = [int(v) for v in re.search(r"static const int z\[9\] = \{([^}]*)\}", src).group(1).split(",")]
    seen = {}
    for m in re.finditer(r"Compiling entry function '_ZN3lsp14accum_z_kernelILi(\d+)ELi\d+ELi\d+ELb0ELb0ELb0EEEvNS_11AccumParamsE'.*?Used (\d+) registers", log, re.S):
        seen[int(m.group(1))] = int(m.group(2))
    assert sorted(seen) == [4, 8, 12, 16, 20, 24, 28, 32]
    for K, regs in seen.items():
        assert table[K // 4] == regs, "plan_regs(K=%d) = %d, ptxas says %d" % (K, table[K // 4], regs)
