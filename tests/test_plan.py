"""Host-only launch planner (csrc/lsp_plan.h through lsp_plan_query): no GPU needed."""
import pytest

import paper_1007_1658_b200 as pkg

SM = 148


@pytest.mark.parametrize("B,Nt,Nf", [(1, 1000, 1000), (1, 10000, 10000), (1, 100000, 1000000),
                                     (4096, 1000, 2000), (1, 1000000, 1000000), (1, 2, 1), (3, 77, 5),
                                     (1, 382003, 1528064)])
def test_plan_is_valid_and_covers_the_problem(B, Nt, Nf):
    p = pkg.plan_query_form(SM, B, Nt, Nf, 3)              # the FP32 z form
    assert p["recurrence"] == 3
    assert p["K"] in (4, 8, 12, 16, 20, 24, 28, 32)
    assert p["threads"] % 32 == 0 and 32 <= p["threads"] <= 256
    assert p["n_freq_blocks"] * p["K"] * p["threads"] >= Nf                 # every frequency is owned
    assert (p["n_freq_blocks"] - 1) * p["K"] * p["threads"] < Nf            # no empty block
    assert p["nsplit"] >= 1 and p["nsplit"] * p["split_len"] >= Nt          # every sample is covered
    assert (p["nsplit"] - 1) * p["split_len"] < Nt                          # no empty split
    assert p["split_len"] % 256 == 0                                        # whole tiles
    assert p["ctas_per_sm"] >= 1
    assert B * p["nsplit"] * 16 * Nf <= (1 << 31) + 16 * Nf                 # workspace cap


def test_big_problems_use_wide_threads_and_fill_the_machine():
    p = pkg.plan_query_form(SM, 1, 1000000, 1000000, 3)
    assert p["K"] >= 24                                                     # anchor amortised
    units = p["nsplit"] * p["n_freq_blocks"]
    slots = p["ctas_per_sm"] * SM
    waves = units / slots
    assert waves > 8 and (waves % 1.0 > 0.85 or waves % 1.0 == 0.0)         # last wave nearly full


def test_small_problems_split_the_time_axis():
    p = pkg.plan_query_form(SM, 1, 10000, 10000, 3)
    assert p["nsplit"] * p["n_freq_blocks"] >= SM                           # enough CTAs to touch every SM
    p1 = pkg.plan_query_form(SM, 4096, 1000, 2000, 3)
    assert p1["nsplit"] == 1                                                # the batch already fills the GPU


def test_plan_query_rejects_bad_sizes():
    with pytest.raises(pkg.LspError):
        pkg.plan_query(SM, 1, 1, 10)
    with pytest.raises(pkg.LspError):
        pkg.plan_query(0, 1, 10, 10)


@pytest.mark.parametrize("B,Nt,Nf", [(1, 10000, 10000), (1, 100000, 1000000), (4096, 1000, 2000),
                                     (1, 1000000, 1000000), (1, 382003, 1528064), (2, 700, 40000)])
@pytest.mark.parametrize("rec", [4, 5])
def test_tensor_core_plans_cover_the_problem(B, Nt, Nf, rec):
    p = pkg.plan_query_form(SM, B, Nt, Nf, rec)
    if rec == 4:
        fpb, threads, cps = 8192, 256, 1
    else:                                                  # tcgen05: K reports the coarse extent L; a CTA owns 128 L frequencies
        assert p["K"] in (16, 32, 64, 128)
        fpb, threads, cps = 128 * p["K"], (544 if p["K"] == 128 else 288), {128: 1, 64: 2, 32: 2, 16: 3}[p["K"]]
    assert p["recurrence"] == rec and p["threads"] == threads and p["ctas_per_sm"] == cps
    assert p["n_freq_blocks"] * fpb >= Nf and (p["n_freq_blocks"] - 1) * fpb < Nf
    assert p["nsplit"] >= 1 and p["nsplit"] * p["split_len"] >= Nt and (p["nsplit"] - 1) * p["split_len"] < Nt
    assert p["split_len"] % 128 == 0
    assert B * p["nsplit"] * 16 * Nf <= (1 << 31) + 16 * Nf
    assert p["est_cycles"] > 0


def test_automatic_form():
    """rec = 0: tcgen05 form for large accurate-enough problems, FP32 z form for tiny Nt; explicit forms are honoured."""
    big = pkg.plan_query(SM, 1, 1000000, 1000000)
    assert big["recurrence"] == 5
    units = big["nsplit"] * big["n_freq_blocks"]
    assert units / SM > 4 and ((units / SM) % 1.0 > 0.85 or units % SM == 0)  # last wave nearly full
    assert pkg.plan_query(SM, 1, 100000, 1000000)["recurrence"] == 5
    assert pkg.plan_query(SM, 1, 300, 1000000)["recurrence"] == 3            # Nt < 512: V's single fp16 pass is too coarse
    assert pkg.plan_query(SM, 1, 2, 1)["recurrence"] == 3
    auto = pkg.plan_query_form(SM, 1, 1000000, 1000000, 0)
    z = pkg.plan_query_form(SM, 1, 1000000, 1000000, 3)
    assert auto["recurrence"] == 5 and auto["est_cycles"] < z["est_cycles"]
    with pytest.raises(pkg.LspError):
        pkg.plan_query_form(SM, 1, 10, 10, 6)


def test_tcgen05_coarse_extent_follows_the_grid():
    """Long grids take the 128 x 128 tile (tensor-pipe bound); a Monte-Carlo batch of short grids (C4) takes a
    narrow tile that the grid fills, two CTAs per SM."""
    assert pkg.plan_query_form(SM, 1, 1000000, 1000000, 5)["K"] == 128
    c4 = pkg.plan_query_form(SM, 4096, 1000, 2000, 5)
    assert c4["K"] == 16 and c4["n_freq_blocks"] == 1 and c4["nsplit"] == 1
    assert pkg.plan_query(SM, 4096, 1000, 2000)["recurrence"] == 5
