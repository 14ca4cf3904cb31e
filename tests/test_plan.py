"""Host-only launch planner (csrc/lsp_plan.h through lsp_plan_query): no GPU needed."""
import pytest

import paper_1007_1658_b200 as pkg

SM = 148


@pytest.mark.parametrize("B,Nt,Nf", [(1, 1000, 1000), (1, 10000, 10000), (1, 100000, 1000000),
                                     (4096, 1000, 2000), (1, 1000000, 1000000), (1, 2, 1), (3, 77, 5),
                                     (1, 382003, 1528064)])
def test_plan_is_valid_and_covers_the_problem(B, Nt, Nf):
    p = pkg.plan_query(SM, B, Nt, Nf)
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
    p = pkg.plan_query(SM, 1, 1000000, 1000000)
    assert p["K"] >= 24                                                     # anchor amortised
    units = p["nsplit"] * p["n_freq_blocks"]
    slots = p["ctas_per_sm"] * SM
    waves = units / slots
    assert waves > 8 and (waves % 1.0 > 0.85 or waves % 1.0 == 0.0)         # last wave nearly full


def test_small_problems_split_the_time_axis():
    p = pkg.plan_query(SM, 1, 10000, 10000)
    assert p["nsplit"] * p["n_freq_blocks"] >= SM                           # enough CTAs to touch every SM
    p1 = pkg.plan_query(SM, 4096, 1000, 2000)
    assert p1["nsplit"] == 1                                                # the batch already fills the GPU


def test_plan_query_rejects_bad_sizes():
    with pytest.raises(pkg.LspError):
        pkg.plan_query(SM, 1, 1, 10)
    with pytest.raises(pkg.LspError):
        pkg.plan_query(0, 1, 10, 10)
