"""CPU checks of the seeded input generators added for the section 8(f) rows (no arithmetic of the method lives there)."""
import numpy as np

import oracle
import workloads


def test_c4s_is_c4_on_one_time_vector():
    a, s = workloads.c4(B=7, Nt=300, Nf=50), workloads.make("C4S", B=7, Nt=300, Nf=50)
    assert s.name == "C4S" and s.B == 7 and s.t.ndim == 1 and s.t.shape == (300,)
    assert np.array_equal(s.t, a.t[0]) and np.array_equal(s.x, a.x)
    assert (s.f_min, s.df, s.Nf) == (a.f_min, a.df, a.Nf) and s.terms == 7 * 300 * 50
    # the oracle's batched call accepts the shared vector and equals series-by-series evaluation on it
    P, idx, val = oracle.periodogram_batched(s.t, s.x, s.f_min, s.df, s.Nf)
    for b in (0, 6):
        assert np.allclose(P[b], oracle.periodogram(s.t, s.x[b], s.f_min, s.df, s.Nf), rtol=0, atol=1e-12)


def test_downsample_keeps_resolution_and_scales_the_grid():
    w = workloads.p0(Nt=4000, Nf=16000)
    d = workloads.downsample(w, 4)
    assert d.Nt == 1000 and d.Nf == 4000 and (d.f_min, d.df) == (w.f_min, w.df)
    assert np.array_equal(d.t, w.t[::4]) and np.array_equal(d.x, w.x[::4])
    assert workloads.downsample(w, 1).Nt == w.Nt
    # the injected period is still found at the same bin after down-sampling (same light curve, fewer points); the
    # nearly even sampling also puts an equally high alias at f_sampling - f_inj, so the check is the power AT the expected bin
    P = oracle.periodogram(d.t, d.x, d.f_min, d.df, d.Nf)
    k = int(round(w.expected_peak_bin))
    assert P[k - 1:k + 2].max() >= 0.9 * P.max() and P.max() > 50.0
