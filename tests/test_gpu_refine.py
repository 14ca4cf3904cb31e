"""GPU parity where the single-pass sums are ill-conditioned (csrc/lsp_refine.cuh): f T << 1, the aliases of regular sampling,
and the generalised periodogram's determinant -> 0.

Eq. (5) divides (S - D) by (Nt - R); as R -> Nt both are small differences of the sums of eq. (8), and the
rounding of fp32 sums is amplified by Nt/(Nt - R).  The library recomputes such frequencies from the raw series in fp64
(LSP_PARAM_REFINE = 0, the default).  Every form of the accumulate step and both places the refinement runs -- inside
finish_kernel, and refine_kernel behind the fused epilogues -- are compared here with the fp64 oracle on grids that start at
f = 0, on series with a drift (so that the low-frequency power is the LARGEST on the grid and the arg-max falls among the
refined bins).  How far up the refinement reaches depends on the form (refine_amplification in lsp_refine.cuh): R > 0.8 Nt
for the FP32-pipe form, down to R > 0.26 Nt at Nt = 512 for the tensor-core forms, whose cos 2 theta sums come from one fp16 pass."""
import numpy as np
import pytest

import oracle

pytestmark = pytest.mark.gpu

TOL = 1e-4          # north_star
TIGHT = 2e-6        # refined bins: fp64 sums, rounded once to fp32


def _series(B, Nt, T, seed, shared_t=False, even=False, drift=2.0):
    rng = np.random.default_rng(seed)
    if even:
        t = np.broadcast_to(np.arange(Nt) * (T / Nt), (B, Nt)).copy()
    else:
        t = np.sort(rng.uniform(0.0, T, (1 if shared_t else B, Nt)), axis=1)
        t = np.broadcast_to(t, (B, Nt)).copy()
    x = rng.standard_normal((B, Nt)) + drift * (t / T) * rng.uniform(0.7, 1.5, (B, 1))
    return t, x.astype(np.float32)


def _gpu(h, pkg, t, x, f_min, df, Nf, shared_t=False, gls=False, w=None, **params):
    import torch
    keys = {k: getattr(pkg, "PARAM_" + k.upper()) for k in params}
    for k, v in params.items():
        h.set_param(keys[k], v)
    try:
        td = torch.from_numpy(np.ascontiguousarray(t[0] if shared_t else t)).cuda()
        xd = torch.from_numpy(x).cuda()
        wd = torch.from_numpy(w).cuda() if w is not None else None
        P, pi, pv = h.periodogram_batched(td, xd, f_min, df, Nf, gls=gls, weights=wd)
        torch.cuda.synchronize()
        plan = h.last_plan()
    finally:
        for k in params:
            h.set_param(keys[k], 0)
    return P.cpu().numpy().astype(np.float64), pi.cpu().numpy(), pv.cpu().numpy(), plan


def _ref(t, x, f_min, df, Nf, gls=False, w=None):
    out = []
    for b in range(x.shape[0]):
        if w is not None:
            out.append(oracle.periodogram_gls_weighted(t[b], x[b], w[b], f_min, df, Nf))
        elif gls:
            out.append(oracle.periodogram_gls(t[b], x[b], f_min, df, Nf))
        else:
            out.append(oracle.periodogram(t[b], x[b], f_min, df, Nf))
    return np.array(out)


def _peaks_consistent(P, pi, pv, ref):
    """The arg-max was merged correctly between the epilogue and the refinement: (peak_idx, peak_val) is the maximum of the P the
    call returned, lowest index on ties, and the oracle's power at that index is its maximum to fp32 rounding (neighbouring
    low-frequency bins differ by less than an fp32 ulp, so the index itself is not unique)."""
    for b in range(P.shape[0]):
        assert int(pi[b]) == int(np.argmax(P[b])) and float(pv[b]) == float(np.float32(P[b].max()))
        assert ref[b][int(pi[b])] >= ref[b].max() * (1.0 - 2 * TOL)


FORMS = [  # name, B, Nt, shared_t, params, kernel substring, launches the refinement as its own kernel
    ("fp32", 2, 3000, False, dict(pipe=1), "accum_z_kernel", False),
    ("fp32-splits", 1, 9000, False, dict(pipe=1, nsplit=5), "accum_z_kernel", False),
    ("small", 1, 3000, False, dict(pipe=2), "accum_umma_small_kernel", False),
    ("small-automatic", 1, 1000, False, dict(), "accum_umma_small_kernel", False),
    ("pair", 2, 3000, False, dict(pipe=2, coarse=128), "accum_umma_pair2_kernel", False),
    ("duo-fused", 7, 1000, False, dict(pipe=2, coarse=16, nsplit=1), "fused-finish", True),
    ("duo", 7, 3000, False, dict(pipe=2, coarse=16), "accum_umma_duo_kernel", False),
    ("shared-gemm-fused", 21, 1000, True, dict(), "shared-times,fused-finish", True),
    ("shared-gemm", 21, 9000, True, dict(), "shared_gemm_kernel", False),
    # Nt > 16,384: finish_kernel lists the flagged frequencies for refine_kernel instead of redoing them inside its block
    ("fp32-long", 1, 20000, False, dict(pipe=1), "accum_z_kernel", False),
    ("pair-long", 2, 20000, False, dict(pipe=2, coarse=128), "accum_umma_pair2_kernel", False),
    ("shared-gemm-long", 17, 20000, True, dict(), "shared_gemm_kernel", False),
]


@pytest.mark.parametrize("name,B,Nt,shared_t,params,kernel,own_kernel", FORMS, ids=[f[0] for f in FORMS])
def test_low_frequencies_every_form(lsp, name, B, Nt, shared_t, params, kernel, own_kernel):
    """Grid from f = 0 in steps of 0.004 / T (f T = 0 ... 1.2): the bins below f T ~ 0.09 have R > 0.95 Nt and are refined in every form."""
    pkg, h = lsp
    T = 50.0
    t, x = _series(B, Nt, T, seed=900 + Nt + B, shared_t=shared_t)
    f_min, df, Nf = 0.0, 0.004 / T, 301
    ref = _ref(t, x, f_min, df, Nf)
    P, pi, pv, plan = _gpu(h, pkg, t, x, f_min, df, Nf, shared_t=shared_t, **params)
    assert kernel in plan["kernel"], plan
    assert ("fused-finish" in plan["kernel"]) == own_kernel
    low = slice(0, 20)                                       # f T <= 0.076: all refined
    for b in range(B):
        top = ref[b].max()
        assert ref[b][1] > 0.5 * top                          # the drift: the low-frequency power is what the tolerance is measured against
        assert np.max(np.abs(P[b][low] - ref[b][low])) <= TIGHT * top, (name, b)
        assert np.max(np.abs(P[b] - ref[b])) <= (TOL if Nt >= 512 else 1e-3) * top, (name, b)
        assert P[b][0] <= 1e-20                              # f = 0: X has zero mean (reading G7)
    _peaks_consistent(P, pi, pv, ref)
    # the refinement is what achieves it: without it the tensor-core forms miss the tolerance on these bins
    P0, pi0, pv0, _ = _gpu(h, pkg, t, x, f_min, df, Nf, shared_t=shared_t, refine=1, **params)
    e_on = max(np.max(np.abs(P[b][low] - ref[b][low])) / ref[b].max() for b in range(B))
    e_off = max(np.max(np.abs(P0[b][low] - ref[b][low])) / ref[b].max() for b in range(B))
    assert e_off > 10 * e_on, (e_on, e_off)
    if "accum_z" not in plan["kernel"]:
        assert e_off > TOL
    # f T >= 0.6: R is small; only the strong bins of the tensor forms are flagged there (P > 0.0118 Nt or more: refine_power,
    # lsp_refine.cuh), nothing else changes
    weak = (P0[:, 150:] <= 0.0118 * Nt) if "accum_z" not in plan["kernel"] else np.ones_like(P0[:, 150:], dtype=bool)
    assert np.array_equal(P[:, 150:][weak], P0[:, 150:][weak])
    assert np.max(np.abs(P[:, 150:] - P0[:, 150:])) <= TOL * ref.max()


@pytest.mark.parametrize("Nt", [2500, 20000], ids=["in-block", "listed"])
@pytest.mark.parametrize("weighted", [False, True])
@pytest.mark.parametrize("params,kernel", [(dict(pipe=1), "accum_z_kernel"), (dict(pipe=2, coarse=128), "accum_umma_pair2_kernel")],
                         ids=["fp32", "pair"])
def test_generalised_periodogram_low_frequencies(lsp, weighted, params, kernel, Nt):
    """The floating-mean fit as f T -> 0 tends to that of a quadratic trend (not to 0): large on a series with a drift.  The
    closed-form determinant of the fp32 sums is useless there; the refinement sums the centred basis directly in fp64.
    Oracle: the least-squares definition in its well-conditioned form (reading G15, pin GP6)."""
    pkg, h = lsp
    B, T = 2, 80.0
    t, x = _series(B, Nt, T, seed=41)
    rng = np.random.default_rng(5)
    w = rng.uniform(0.2, 3.0, (B, Nt)).astype(np.float32) if weighted else None
    f_min, df, Nf = 0.0, 0.0007 / T, (400 if Nt < 10000 else 150)   # f T = 0 ... 0.28 (0.1)
    ref = _ref(t, x, f_min, df, Nf, gls=True, w=w)
    P, pi, pv, plan = _gpu(h, pkg, t, x, f_min, df, Nf, gls=True, w=w, **params)
    assert kernel in plan["kernel"]
    for b in range(B):
        assert ref[b][1] > 10.0                              # f T = 7e-4: the power of the trend
        assert P[b][0] == 0.0 and ref[b][0] == 0.0           # f = 0 itself: singular fit (reading G7)
        assert np.max(np.abs(P[b] - ref[b])) <= TIGHT * ref[b].max(), b
    _peaks_consistent(P, pi, pv, ref)
    # one frequency at a time down to f T = 1e-6 (single-series entry point)
    import torch
    td, xd = torch.from_numpy(t[0]).cuda(), torch.from_numpy(x[0]).cuda()
    wd = torch.from_numpy(w[0]).cuda() if weighted else None
    for fT in (1e-6, 1e-4, 1e-2):
        got = float(h.periodogram(td, xd, fT / T, df, 1, gls=True, weights=wd).cpu()[0])
        want = (oracle.periodogram_gls_weighted(t[0], x[0], w[0], fT / T, df, 1) if weighted else oracle.periodogram_gls(t[0], x[0], fT / T, df, 1))[0]
        assert abs(got - want) <= TIGHT * want and want > 10.0, (fT, got, want)


@pytest.mark.parametrize("B,params,kernel", [(3, dict(pipe=1), "accum_z_kernel"), (1, dict(pipe=2), "accum_umma_small_kernel"),
                                             (3, dict(pipe=2, coarse=16, nsplit=1), "fused-finish")], ids=["fp32", "small", "duo-fused"])
def test_alias_of_regular_sampling(lsp, B, params, kernel):
    """Regular sampling: at f = 1/dt every phase repeats and R -> Nt again; P(1/dt + d) mirrors P(d).  A grid across the alias
    (f T' from -0.3 to +0.3 around it, the alias itself on the grid) against the oracle."""
    pkg, h = lsp
    Nt, T = 1600, 40.0
    t, x = _series(B, Nt, T, seed=77, even=True)
    fs = Nt / T
    df = 0.003 / T
    f_min, Nf = fs - 100 * df, 201
    ref = _ref(t, x, f_min, df, Nf)
    P, pi, pv, plan = _gpu(h, pkg, t, x, f_min, df, Nf, **params)
    assert kernel in plan["kernel"]
    for b in range(B):
        assert ref[b][90] > 10.0 and ref[b][110] > 10.0       # the mirrored low-frequency power of the drift
        assert np.max(np.abs(P[b] - ref[b])) <= TOL * ref[b].max(), b
        assert np.max(np.abs(P[b][95:106] - ref[b][95:106])) <= TIGHT * ref[b].max(), b      # |f - 1/dt| T <= 0.015: refined in every form
    _peaks_consistent(P, pi, pv, ref)


def test_refinement_is_reproducible_and_clears_its_list(lsp):
    """The fused epilogues append to the list in whatever order their warps finish; the refined values and the merged peak do
    not depend on it (bit-identical repeats), and the list is empty again for the next call (a call on another form follows)."""
    pkg, h = lsp
    T = 50.0
    t, x = _series(9, 1000, T, seed=3)
    args = (t, x, 0.0, 0.004 / T, 301)
    a = _gpu(h, pkg, *args, pipe=2, coarse=16, nsplit=1)
    assert "fused-finish" in a[3]["kernel"]
    for _ in range(3):
        b = _gpu(h, pkg, *args, pipe=2, coarse=16, nsplit=1)
        assert np.array_equal(a[0], b[0]) and np.array_equal(a[1], b[1]) and np.array_equal(a[2], b[2])
    ts, xs = _series(20, 1000, T, seed=4, shared_t=True)
    c = _gpu(h, pkg, ts, xs, 0.0, 0.004 / T, 301, shared_t=True)
    assert "shared-times,fused-finish" in c[3]["kernel"]
    ref = _ref(ts, xs, 0.0, 0.004 / T, 301)
    for b in range(20):
        assert np.max(np.abs(c[0][b] - ref[b])) <= TOL * ref[b].max()
    _peaks_consistent(c[0], c[1], c[2], ref)


def test_list_overflow_keeps_the_fp32_sum_values(lsp):
    """More flagged (series, frequency) pairs than the fused epilogues' list holds (1,048,576): the rest keep the value of the
    fp32 sums (which at f T ~ 0.01 is poor on the tensor-core forms: lsp.h says so) and take part in the arg-max as they are;
    nothing is written out of bounds, the pairs that did fit are refined, and the next call starts from an empty list."""
    pkg, h = lsp
    B, Nt, T, Nf = 9000, 600, 50.0, 128                      # 128 bins below f T = 0.08: 1,152,000 pairs
    t, x = _series(B, Nt, T, seed=8)
    f_min, df = 0.0, 0.0006 / T
    P, pi, pv, plan = _gpu(h, pkg, t, x, f_min, df, Nf, pipe=2, coarse=16)
    assert "fused-finish" in plan["kernel"]
    assert np.all(np.isfinite(P)) and np.all(P >= 0.0)
    for b in range(0, B, 97):
        assert int(pi[b]) == int(np.argmax(P[b])) and float(pv[b]) == float(np.float32(P[b].max()))
    sample = np.arange(0, B, 449)
    ref = _ref(t[sample], x[sample], f_min, df, Nf)
    good = np.array([[abs(P[b][k] - ref[i][k]) <= 2e-6 * ref[i].max() for k in range(Nf)] for i, b in enumerate(sample)])
    assert 0.80 <= good.mean() < 1.0                         # 91 % fit the list; the rest are the fp32-sum values
    # the next call: list empty again, every flagged bin refined
    t2, x2 = _series(5, 1000, T, seed=9)
    P2, pi2, pv2, _ = _gpu(h, pkg, t2, x2, 0.0, 0.004 / T, 301, pipe=2, coarse=16, nsplit=1)
    ref2 = _ref(t2, x2, 0.0, 0.004 / T, 301)
    for b in range(5):
        assert np.max(np.abs(P2[b][:20] - ref2[b][:20])) <= TIGHT * ref2[b].max()
    _peaks_consistent(P2, pi2, pv2, ref2)


def test_host_entry_points_refine_too(lsp):
    """The host-buffer calls stage the series in device memory and run the same path: the refinement reads the staged copy."""
    import torch
    pkg, h = lsp
    T = 50.0
    t, x = _series(1, 2000, T, seed=12)
    f_min, df, Nf = 0.0, 0.004 / T, 301
    ref = _ref(t, x, f_min, df, Nf)
    P = h.periodogram_host(torch.from_numpy(t[0]).pin_memory(), torch.from_numpy(x[0]).pin_memory(), f_min, df, Nf).numpy().astype(np.float64)
    assert np.max(np.abs(P[:20] - ref[0][:20])) <= TIGHT * ref[0].max()
    assert np.max(np.abs(P - ref[0])) <= TOL * ref[0].max()
    tb, xb = _series(70, 1000, T, seed=13)
    refb = _ref(tb, xb, f_min, df, Nf)
    Pb = torch.empty((70, Nf), dtype=torch.float32).pin_memory()
    h.periodogram_batched_host(torch.from_numpy(tb).pin_memory(), torch.from_numpy(xb).pin_memory(), f_min, df, Nf, P=Pb)
    Pb = Pb.numpy().astype(np.float64)
    for b in range(70):
        assert np.max(np.abs(Pb[b][:20] - refb[b][:20])) <= TIGHT * refb[b].max()
        assert np.max(np.abs(Pb[b] - refb[b])) <= TOL * refb[b].max()


def test_refine_param(lsp):
    pkg, h = lsp
    assert h.get_param(pkg.PARAM_REFINE) == 0
    h.set_param(pkg.PARAM_REFINE, 1)
    assert h.get_param(pkg.PARAM_REFINE) == 1
    h.set_param(pkg.PARAM_REFINE, 0)
    with pytest.raises(pkg.LspError):
        h.set_param(pkg.PARAM_REFINE, 2)


def test_listed_refinement_in_a_cuda_graph(lsp):
    """Long series (refine_kernel behind finish_kernel) on a fresh handle whose memory comes from lsp_reserve alone: the call
    is captured into a CUDA graph, replayed three times (the list must be empty again after every replay) and compared with the
    eager call and the oracle."""
    import torch
    pkg, _ = lsp
    T, Nt, Nf = 50.0, 20000, 301
    t, x = _series(1, Nt, T, seed=21)
    f_min, df = 0.0, 0.004 / T
    ref = _ref(t, x, f_min, df, Nf)[0]
    td, xd = torch.from_numpy(t[0]).cuda(), torch.from_numpy(x[0]).cuda()
    P = torch.empty(Nf, dtype=torch.float32, device="cuda")
    with pkg.Handle(0) as h:
        h.reserve(1, Nt, Nf)
        g, s = torch.cuda.CUDAGraph(), torch.cuda.Stream()
        with torch.cuda.stream(s):
            torch.cuda.synchronize()
            with torch.cuda.graph(g, stream=s):
                h.periodogram(td, xd, f_min, df, Nf, out=P)
        first = None
        for _ in range(3):
            P.zero_()
            g.replay()
            torch.cuda.synchronize()
            first = P.clone() if first is None else first
            assert torch.equal(P, first)
        got = P.cpu().numpy().astype(np.float64)
        assert np.max(np.abs(got[:20] - ref[:20])) <= TIGHT * ref.max()
        assert np.max(np.abs(got - ref)) <= TOL * ref.max()
        eager = h.periodogram(td, xd, f_min, df, Nf)
        torch.cuda.synchronize()
        assert torch.equal(eager, first)


TREND_FORMS = [  # name, B, Nt, Nf, span, f_max, shared_t, params, kernel substring
    ("small-1k", 1, 1000, 1000, 100.0, 0.1, False, dict(), "accum_umma_small_kernel"),
    ("small-20k", 1, 20000, 20000, 100.0, 0.1, False, dict(), "accum_umma_small_kernel"),
    ("small-long-splits", 2, 250001, 65536, 1000.0, 0.05, False, dict(nsplit=3), "accum_umma_small_kernel"),
    ("duo", 8, 6000, 2000, 50.0, 0.2, False, dict(), "accum_umma_duo_kernel"),
    ("shared-gemm", 32, 9000, 3000, 50.0, 0.2, True, dict(), "shared_gemm_kernel"),
    ("pair", 1, 100000, 1000003, 100.0, 1.0, False, dict(), "accum_umma_pair2_kernel"),
    ("pair-long-splits", 1, 250001, 1000003, 1000.0, 0.5, False, dict(nsplit=7), "accum_umma_pair2_kernel"),
    ("pair-fp16x3", 1, 100000, 1000003, 100.0, 1.0, False, dict(corr=1), "accum_umma_pair2_kernel"),
    ("fp32", 1, 250001, 1000003, 1000.0, 0.5, False, dict(pipe=1), "accum_z_kernel"),
]


@pytest.mark.parametrize("name,B,Nt,Nf,span,f_max,shared_t,params,kernel", TREND_FORMS, ids=[f[0] for f in TREND_FORMS])
def test_series_with_a_trend(lsp, name, B, Nt, Nf, span, f_max, shared_t, params, kernel):
    """A linear drift of one sigma over the span: the low-frequency power is the largest on the grid (P of thousands), every sum
    there is COHERENT, and R / Nt takes every value between 0 and 1 on a grid that starts at f = 0.  This is where the tensor
    core's round-toward-zero accumulation shows: a randomised sweep found errors up to 1e-3 of max P at R = 0.3 ... 0.9 Nt that
    grew with the length of the time splits (D_V was drained once per split and the refinement started at R = 0.9 Nt).  Since then
    D_V is drained with D_W at every window and the tensor forms refine from R = 0.45 Nt (CTA-pair kernel) / 0.6 Nt on.
    Dense low-frequency bins (f T < 3), the end of the grid and random bins against the oracle."""
    pkg, h = lsp
    rng = np.random.default_rng(1100 + Nt % 977 + B)
    tt = np.sort(rng.uniform(0.0, span, Nt))
    t = np.broadcast_to(tt, (B, Nt)).copy()
    x = (rng.standard_normal((B, Nt)) + 1.0 * t / span).astype(np.float32)
    f_min, df = 0.0, f_max / (Nf - 1)
    P, pi, pv, plan = _gpu(h, pkg, t, x, f_min, df, Nf, shared_t=shared_t, **params)
    assert kernel in plan["kernel"], plan
    fT = np.arange(Nf) * df * span
    low = np.where(fT < 3.0)[0]
    ks = np.unique(np.concatenate([low[::max(1, len(low) // 400)], rng.integers(0, Nf, 100), np.arange(Nf - 64, Nf)])).astype(np.int64)
    worst = 0.0
    for b in sorted({0, B - 1}):
        ref = oracle.periodogram(tt, x[b], f_min, df, Nf, ks=ks)
        top = max(float(ref.max()), float(P[b].max()))
        assert top > 30.0                                        # the trend's power
        worst = max(worst, float(np.max(np.abs(P[b][ks] - ref))) / top)
        assert int(pi[b]) == int(np.argmax(P[b]))
    print("%s: max |dP| / max P = %.2e" % (name, worst))
    assert worst <= TOL


STRONG_FORMS = [  # name, Nt, Nf, span, f_max, params, kernel substring
    ("pair", 100000, 1000003, 100.0, 1.0, dict(), "accum_umma_pair2_kernel"),
    ("pair-fp16x3", 100000, 1000003, 100.0, 1.0, dict(corr=1), "accum_umma_pair2_kernel"),
    ("small-20k", 20000, 20000, 100.0, 0.1, dict(), "accum_umma_small_kernel"),
]


@pytest.mark.parametrize("kind,a", [("drift", 3.0), ("drift", 100.0), ("sine", 30.0), ("parabola", 10.0), ("drift", 0.5)],
                         ids=["drift-3-sigma", "drift-100-sigma", "slow-sine-30-sigma", "parabola-10-sigma", "drift-half-sigma"])
@pytest.mark.parametrize("name,Nt,Nf,span,f_max,params,kernel", STRONG_FORMS, ids=[f[0] for f in STRONG_FORMS])
def test_strong_slow_signals(lsp, name, Nt, Nf, span, f_max, params, kernel, kind, a):
    """Signals that are strong AND slow (a drift of many sigma, a sinusoid of 1.3 cycles over the span, a parabola; time-sorted samples):
    every drain window of the tensor forms then sums products whose signs are fixed over the window, the case the truncation
    compensation cannot model from the window sum alone.  Before bins with P > 0.0118 Nt were refined (refine_power, lsp_refine.cuh)
    the CTA-pair kernel was off by 1.1e-4 ... 1.6e-4 of max P on these inputs (an error proportional to P_k itself, so the largest bins
    carried it); now every form stays within half the tolerance.  The half-sigma drift is just below the threshold (nothing refined for
    its power): there the CTA-pair kernel measured 6.7e-5 ... 7.1e-5 -- an error of sum e^{2i theta}, not of the data: round-to-nearest
    of the fine operand's fp16 (cos 2b, sin 2b) makes the same error in every sample where b hardly moves -- until the table was
    rounded stochastically (umma_ftable_pair_kernel): 2.5e-5 ... 3.3e-5."""
    pkg, h = lsp
    rng = np.random.default_rng(1100 + Nt % 977 + 1)
    tt = np.sort(rng.uniform(0.0, span, Nt))
    sig = {"drift": a * tt / span, "sine": a * np.sin(2 * np.pi * (1.3 / span) * tt + 0.4), "parabola": a * (tt / span - 0.5) ** 2}[kind]
    x = (rng.standard_normal(Nt) + sig).astype(np.float32)[None, :]
    f_min, df = 0.0, f_max / (Nf - 1)
    P, pi, pv, plan = _gpu(h, pkg, tt[None, :], x, f_min, df, Nf, **params)
    assert kernel in plan["kernel"], plan
    fT = np.arange(Nf) * df * span
    low = np.where(fT < 6.0)[0]
    ks = np.unique(np.concatenate([low[::max(1, len(low) // 500)], rng.integers(0, Nf, 100), [int(pi[0])]])).astype(np.int64)
    ref = oracle.periodogram(tt, x[0], f_min, df, Nf, ks=ks)
    top = max(float(ref.max()), float(P[0].max()))
    worst = float(np.max(np.abs(P[0][ks] - ref))) / top
    print("%s, %s %g sigma: max P = %.4g (%.1f %% of (Nt - 1)/2), max |dP| / max P = %.2e" % (name, kind, a, top, 200.0 * top / (Nt - 1), worst))
    assert int(pi[0]) == int(np.argmax(P[0])) and float(pv[0]) == float(P[0].max())
    assert worst <= 0.5 * TOL


@pytest.mark.parametrize("params", [dict(), dict(corr=1)], ids=["pair", "pair-fp16x3"])
@pytest.mark.parametrize("kind,a", [("sine", 20.0), ("drift", 30.0)], ids=["slow-sine-20-sigma", "drift-30-sigma"])
def test_strong_slow_signal_below_the_grid(lsp, params, kind, a):
    """A strong slow component whose frequency the grid does NOT contain (f_min T = 65; the signal has 1.7 cycles per span, or is a drift):
    no bin holds its power, so nothing is refined for it, but every bin sees it inside each accumulation window.  With time-sorted
    samples the tensor core's running accumulator swings with it far from the window's final value and the truncation loss is not what
    the compensation reads off that value: 1.1e-4 ... 2.0e-4 of max P on the CTA-pair kernel (found by a randomised sweep with strong
    signals).  The records are therefore laid out in a golden-ratio stride order (record_order_stride, lsp_prepass.cuh; LSP_PARAM_ORDER):
    every window holds samples from all over the span.  Both orders are measured here."""
    pkg, h = lsp
    Nt, Nf, span, f_min, f_max = 250001, 239999, 5000.0, 0.013, 5.0
    rng = np.random.default_rng(7)
    tt = np.sort(rng.uniform(0.0, span, Nt))
    sig = a * np.sin(2 * np.pi * 1.7 / span * tt + 1.0) if kind == "sine" else a * tt / span
    x = (rng.standard_normal(Nt) + sig).astype(np.float32)[None, :]
    df = (f_max - f_min) / (Nf - 1)
    ks = np.unique(np.concatenate([np.arange(40), rng.integers(0, Nf, 400), np.arange(Nf - 20, Nf)])).astype(np.int64)
    ref = oracle.periodogram(tt, x[0], f_min, df, Nf, ks=ks)
    err = {}
    for order in (0, 1):
        P, pi, pv, plan = _gpu(h, pkg, tt[None, :], x, f_min, df, Nf, order=order, **params)
        assert "accum_umma_pair2_kernel" in plan["kernel"], plan
        err[order] = float(np.max(np.abs(P[0][ks] - ref))) / max(float(ref.max()), float(P[0].max()))
        assert int(pi[0]) == int(np.argmax(P[0]))
    print("%s %g sigma, %s: max |dP| / max P = %.2e in stride order, %.2e in the order given" % (kind, a, params, err[0], err[1]))
    assert err[0] <= 0.5 * TOL
    assert err[1] > 2.0 * err[0]
