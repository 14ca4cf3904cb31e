"""Pins for the fp64 oracle (oracle/lsp_oracle.c and its numpy twin), CPU only.

Each test fixes the oracle against something that is NOT the oracle: a least-squares
fit, numpy's FFT, a closed form, scipy's own Lomb-Scargle, an invariance, mpmath
brute force, Gaussian-noise statistics.  Numbering P1..P9 follows DESIGN.md ("Pins").
Equation / line references are to /root/reference/PAPER.md (Townsend 2010).
"""
import json
import os

import numpy as np
import pytest

import oracle
import workloads

HERE = os.path.dirname(os.path.abspath(__file__))


def _series(Nt, seed, T=20.0, f_inj=0.9):
    rng = np.random.Generator(np.random.PCG64(seed))
    t = np.sort(rng.uniform(0.0, T, Nt))
    x = (np.sin(2 * np.pi * f_inj * t + 0.3) + rng.normal(0.0, 0.7, Nt)).astype(np.float32)
    return t, x


def _grid(f_lo, f_hi, Nf):
    return f_lo, (f_hi - f_lo) / (Nf - 1)


def _c_and_numpy(t, x, f_min, df, Nf):
    Pc = oracle.periodogram(t, x, f_min, df, Nf)
    Pn = oracle.periodogram_numpy(t, x, f_min + np.arange(Nf) * df)
    return Pc, Pn


# ------------------------------------------------------------------ C build vs numpy twin
def test_c_oracle_matches_numpy_twin():
    t, x = _series(257, 11)
    f_min, df = _grid(0.05, 6.0, 301)
    Pc, Pn = _c_and_numpy(t, x, f_min, df, 301)
    assert np.max(np.abs(Pc - Pn)) <= 1e-11 * np.max(Pn)


def test_subset_indices_match_full_grid():
    t, x = _series(300, 12)
    f_min, df = _grid(0.05, 6.0, 400)
    full = oracle.periodogram(t, x, f_min, df, 400)
    ks = np.array([0, 3, 17, 399, 200, 200], dtype=np.int64)
    sub = oracle.periodogram(t, x, f_min, df, 400, ks=ks)
    assert np.array_equal(sub, full[ks])


def test_thread_count_does_not_change_result():
    t, x = _series(300, 13)
    f_min, df = _grid(0.05, 6.0, 64)
    a = oracle.periodogram(t, x, f_min, df, 64, nthreads=1)
    b, used = oracle.periodogram(t, x, f_min, df, 64, nthreads=2, return_threads=True)
    assert used == 2
    assert np.array_equal(a, b)


# ------------------------------------------------------------------ P1 least squares
@pytest.mark.parametrize("Nt,seed", [(10, 1), (23, 2), (40, 3)])
def test_P1_least_squares_chi2_reduction(Nt, seed):
    """P*2*var = sum X^2 - min chi^2 of the fit X ~ a cos wt + b sin wt (2x2 normal equations).

    Fixes eq. (1) including tau of eq. (2) and both denominators."""
    t, x = _series(Nt, seed, T=10.0)
    X = x.astype(np.float64)
    X = X - X.mean()
    var = (X * X).sum() / (Nt - 1)
    freqs = np.linspace(0.07, 3.1, 37)
    expect = np.empty_like(freqs)
    for i, f in enumerate(freqs):
        A = np.stack([np.cos(2 * np.pi * f * t), np.sin(2 * np.pi * f * t)], axis=1)
        N = A.T @ A
        rhs = A.T @ X
        ab = np.linalg.solve(N, rhs)
        chi2 = ((X - A @ ab) ** 2).sum()
        expect[i] = ((X * X).sum() - chi2) / (2.0 * var)
    got_np = oracle.periodogram_numpy(t, x, freqs)
    assert np.max(np.abs(got_np - expect)) <= 1e-11 * np.max(expect)
    f_min, df = freqs[0], freqs[1] - freqs[0]
    got_c = oracle.periodogram(t, x, f_min, df, freqs.size)
    assert np.max(np.abs(got_c - expect)) <= 1e-10 * np.max(expect)


# ------------------------------------------------------------------ P2 FFT periodogram
@pytest.mark.parametrize("N", [64, 250])
def test_P2_even_sampling_equals_fft_periodogram(N):
    """t_j = j*dt, Fourier frequencies k/(N dt), 0<k<N/2:  P_k = |FFT(X)_k|^2 / (N var)."""
    w = workloads.even_sampling(N, dt=0.25, seed=5)
    X = w.x.astype(np.float64)
    X = X - X.mean()
    var = (X * X).sum() / (N - 1)
    F = np.fft.fft(X)
    k = np.arange(1, N // 2)
    expect = np.abs(F[k]) ** 2 / (N * var)
    got = oracle.periodogram(w.t, w.x, w.f_min, w.df, w.Nf)
    assert got.shape == expect.shape
    assert np.max(np.abs(got - expect)) <= 1e-11 * np.max(expect)


# ------------------------------------------------------------------ P3 shift invariance
def test_P3_time_shift_invariance():
    """P[t] = P[t + c] (tau of eq. (2) absorbs the origin)."""
    t, x = _series(500, 21, T=50.0)
    f_min, df = _grid(0.02, 5.0, 500)
    a = oracle.periodogram(t, x, f_min, df, 500)
    b = oracle.periodogram(t + 1234.567, x, f_min, df, 500)
    c = oracle.periodogram(t - 77.25, x, f_min, df, 500)
    assert np.max(np.abs(a - b)) <= 1e-9 * np.max(a)
    assert np.max(np.abs(a - c)) <= 1e-9 * np.max(a)


def test_affine_invariance_in_x():
    """The series is 'scaled and shifted' to zero mean, unit variance: P[a x + b] = P[x]."""
    t, x = _series(300, 22)
    f_min, df = _grid(0.05, 4.0, 200)
    a = oracle.periodogram(t, x, f_min, df, 200)
    x2 = (4.0 * x.astype(np.float64) + 8.0).astype(np.float32)      # exact in fp32: power-of-two scale, small shift
    b = oracle.periodogram(t, x2, f_min, df, 200)
    assert np.max(np.abs(a - b)) <= 1e-5 * np.max(a)                 # fp32 rounding of x2 only


# ------------------------------------------------------------------ P4 closed form
def test_P4_pure_sinusoid_closed_form():
    """Even sampling, whole cycles: P = (Nt-1)/2 at its own Fourier frequency, 0 at the others (pins G1)."""
    N, dt, k0 = 128, 0.5, 9
    t = np.arange(N) * dt
    x = np.sin(2 * np.pi * k0 / (N * dt) * t + 0.4).astype(np.float64)
    df = 1.0 / (N * dt)
    # feed float64-exact values through the numpy twin (float32 cast perturbs at 1e-7)
    P32 = oracle.periodogram(t, x.astype(np.float32), df, df, N // 2 - 1)
    assert abs(P32[k0 - 1] - (N - 1) / 2.0) <= 1e-5
    others = np.delete(P32, k0 - 1)
    assert np.max(np.abs(others)) <= 1e-10
    assert np.all(P32 <= (N - 1) / 2.0 + 1e-9)


# ------------------------------------------------------------------ P5 scipy
def test_P5_scipy_lombscargle():
    """scipy.signal.lombscargle (independent code) / var equals the oracle."""
    from scipy.signal import lombscargle
    t, x = _series(400, 31, T=40.0)
    f_min, df = _grid(0.03, 4.0, 300)
    freqs = f_min + np.arange(300) * df
    X = x.astype(np.float64)
    X = X - X.mean()
    var = (X * X).sum() / (X.size - 1)
    expect = lombscargle(t, X, 2 * np.pi * freqs) / var
    got = oracle.periodogram(t, x, f_min, df, 300)
    assert np.max(np.abs(got - expect)) <= 1e-10 * np.max(expect)


# ------------------------------------------------------------------ P6 noise statistics
def test_P6_gaussian_noise_mean_power_is_one():
    """Pure Gaussian noise: P is beta-distributed with mean 1 under the N-1 variance (G1)."""
    w = workloads.c4(B=96, Nt=200, Nf=150, seed=99)
    P, idx, val = oracle.periodogram_batched(w.t, w.x, w.f_min, w.df, w.Nf)
    assert P.shape == (96, 150)
    m = P.mean()
    assert abs(m - 1.0) < 0.03, m
    assert np.all(P >= 0.0) and np.all(P <= (200 - 1) / 2.0)
    assert np.array_equal(idx, P.argmax(axis=1))
    assert np.array_equal(val, P.max(axis=1))
    # peaks of ~100 independent frequencies: Gumbel-like, mean ~ ln(Nind)+0.58, std ~ pi/sqrt(6)
    assert 3.5 < val.mean() < 7.5
    assert 0.6 < val.std() < 2.2


# ------------------------------------------------------------------ P7 injected sinusoid
def test_P7_injected_sinusoid_recovered_C1():
    w = workloads.c1()
    P = oracle.periodogram(w.t, w.x, w.f_min, w.df, w.Nf)
    k = oracle.argmax(P)
    assert abs(k - w.expected_peak_bin) <= 1.0
    # amplitude 1, noise 0.5: var ~ 0.75, P_peak ~ Nt A^2 / (4 var)
    assert 0.8 * 1000 / (4 * 0.75) < P[k] < 1.2 * 1000 / (4 * 0.75)


# ------------------------------------------------------------------ P8 single-pass form
def test_P8_single_pass_and_trigfree_forms_agree():
    """eqs (1)-(2) == eqs (5)-(8) == the atan2-free combine used by the CUDA finish step.

    Written out here from the paper, independent of both implementations."""
    t, x = _series(333, 41, T=30.0)
    X = x.astype(np.float64)
    X = X - X.mean()
    Nt = X.size
    var = (X * X).sum() / (Nt - 1)
    freqs = np.linspace(0.04, 5.0, 211)
    ref = oracle.periodogram_numpy(t, x, freqs)
    for i, f in enumerate(freqs):
        w = 2 * np.pi * f
        c, s = np.cos(w * t), np.sin(w * t)
        XC, XS, CC, SS, CS = (X * c).sum(), (X * s).sum(), (c * c).sum(), (s * s).sum(), (c * s).sum()
        wt = 0.5 * np.arctan2(2 * CS, CC - SS)                       # eq. (6)
        ct, st = np.cos(wt), np.sin(wt)                              # eq. (7)
        p5 = 0.5 * ((ct * XC + st * XS) ** 2 / (ct * ct * CC + 2 * ct * st * CS + st * st * SS)
                    + (ct * XS - st * XC) ** 2 / (ct * ct * SS - 2 * ct * st * CS + st * st * CC))  # eq. (5)
        assert abs(p5 / var - ref[i]) <= 1e-10 * max(1.0, ref[i])
        A, B = 2 * CC - Nt, 2 * CS                                   # SS = Nt - CC
        R = np.hypot(A, B)
        S = XC * XC + XS * XS
        D = ((XC * XC - XS * XS) * A + 2 * XC * XS * B) / R
        p6 = ((S + D) / (Nt + R) + (S - D) / (Nt - R)) / (2 * var)
        assert abs(p6 - ref[i]) <= 1e-10 * max(1.0, ref[i])


# ------------------------------------------------------------------ P9 mpmath brute force
def test_P9_mpmath_brute_force_tiny():
    import mpmath as mp
    mp.mp.dps = 50
    t, x = _series(12, 51, T=7.0)
    freqs = [0.11, 0.73, 2.9]
    got = oracle.periodogram_numpy(t, x, freqs)
    f_min, df = 0.11, 0.62
    got_c = oracle.periodogram(t, x, f_min, df, 2)                   # 0.11, 0.73
    tm = [mp.mpf(float(v)) for v in t]
    xm = [mp.mpf(float(v)) for v in x]
    N = len(tm)
    mean = sum(xm) / N
    Xm = [v - mean for v in xm]
    var = sum(v * v for v in Xm) / (N - 1)
    for i, f in enumerate(freqs):
        w = 2 * mp.pi * mp.mpf(f)
        tau = mp.atan2(sum(mp.sin(2 * w * tj) for tj in tm), sum(mp.cos(2 * w * tj) for tj in tm)) / (2 * w)
        cs = [mp.cos(w * (tj - tau)) for tj in tm]
        ss = [mp.sin(w * (tj - tau)) for tj in tm]
        p = (sum(a * b for a, b in zip(Xm, cs)) ** 2 / sum(c * c for c in cs)
             + sum(a * b for a, b in zip(Xm, ss)) ** 2 / sum(s * s for s in ss)) / (2 * var)
        assert abs(float(p) - got[i]) <= 1e-12 * max(1.0, float(p))
        if i < 2:
            assert abs(float(p) - got_c[i]) <= 1e-11 * max(1.0, float(p))


# ------------------------------------------------------------------ degenerate readings
def test_G7_zero_frequency_and_nyquist_are_finite():
    N = 32
    t = np.arange(N, dtype=np.float64)
    rng = np.random.Generator(np.random.PCG64(3))
    x = rng.normal(size=N).astype(np.float32)
    P0 = oracle.periodogram(t, x, 0.0, 0.5, 2)        # f = 0 and f = Nyquist (sin wt = 0 for all j)
    assert np.all(np.isfinite(P0))
    assert abs(P0[0]) < 1e-12                          # zero-mean series: XC = 0 at f = 0
    X = x.astype(np.float64) - x.astype(np.float64).mean()
    var = (X * X).sum() / (N - 1)
    alt = (X * np.cos(np.pi * t)).sum() ** 2 / N / (2 * var)
    assert abs(P0[1] - alt) <= 1e-9 * max(1.0, alt)


def test_G9_argmax_lowest_index_on_ties():
    assert oracle.argmax(np.array([1.0, 5.0, 5.0, 2.0])) == 1
    assert oracle.argmax(np.array([7.0])) == 0


def test_moments_sample_variance():
    rng = np.random.Generator(np.random.PCG64(8))
    x = rng.normal(3.0, 2.0, 1001).astype(np.float32)
    m, v = oracle.moments(x)
    xd = x.astype(np.float64)
    assert abs(m - xd.mean()) < 1e-12
    assert abs(v - xd.var(ddof=1)) < 1e-12


def test_fap_eq3_limits():
    """Eq. (3): Q(0) = 1, Q decreasing in P, Q(P_max) = 0 (reading G13: the base is the normalised power
    p = 2P/(Nt - 1) under the sample-variance scaling G1), Q -> Nf * s for small single-trial probability s."""
    Q = oracle.false_alarm_probability(np.array([0.0, 5.0, 10.0, 20.0, 499.5]), 1000, 500)
    assert Q[0] == 1.0 and Q[4] == 0.0
    assert np.all(np.diff(Q) < 0)
    assert abs(Q[3] / (500 * oracle.false_alarm_probability(np.array([20.0]), 1000, 1.0)[0]) - 1.0) < 1e-3


def test_fap_F1_single_trial_is_the_beta_survival_function():
    """Pin F1 (not the formula retyped: scipy's regularised incomplete beta function).  PAPER.md:50: for Gaussian noise P_n is
    beta distributed (Schwarzenberg-Czerny 1998): p = chi^2 reduction / total chi^2 ~ Beta(1, (Nt-3)/2) for a two-parameter
    fit to Nt - 1 degrees of freedom.  With N_f = 1, eq. (3) must be that law's survival function at p = 2P/(Nt - 1)."""
    from scipy.special import betainc
    from scipy.stats import beta
    for Nt in (10, 12, 17, 100, 1000):
        z = np.linspace(0.0, (Nt - 1) / 2.0, 41)
        Q = oracle.false_alarm_probability(z, Nt, 1.0)
        p = 2.0 * z / (Nt - 1)
        assert np.max(np.abs(Q - (1.0 - betainc(1.0, (Nt - 3) / 2.0, p)))) < 1e-12
        assert np.max(np.abs(Q - beta.sf(p, 1.0, (Nt - 3) / 2.0))) < 1e-12
        # the literal 2P/Nt of the paper's print (N-variance convention) is a different function of this library's P
        wrong = np.clip(1.0 - 2.0 * z / Nt, 0, 1) ** ((Nt - 3) / 2.0)
        if Nt <= 17:
            assert np.max(np.abs(Q - wrong)) > 0.02


def _mc_noise_powers(Nt, n_series, seed, gls):
    """Oracle periodograms of Gaussian-noise series at a few frequencies (uneven sampling for the floating-mean fit, for which
    the beta law is exact at ANY frequency; even sampling at Fourier frequencies for eq. (1), where the sample mean is
    orthogonal to the sinusoids and the law is exact too)."""
    rng = np.random.default_rng(seed)
    if gls:
        t = np.sort(rng.uniform(0.0, 10.0, Nt))
        f_min, df, Nf = 0.31, 0.47, 4
    else:
        t = np.arange(Nt, dtype=np.float64) * 0.5
        f_min = df = 1.0 / (Nt * 0.5)
        Nf = 4                                             # Fourier frequencies k = 1..4 < Nt/2
    out = np.empty((n_series, Nf))
    for m in range(n_series):
        x = rng.standard_normal(Nt).astype(np.float32)
        out[m] = (oracle.periodogram_gls if gls else oracle.periodogram)(t, x, f_min, df, Nf, nthreads=1)
    return out


@pytest.mark.parametrize("gls", [False, True])
def test_fap_F2_monte_carlo_single_trial_exceedance(gls):
    """Pin F2: at Nt = 12 the N vs N-1 convention, the exponent and the base are all visible.  The fraction of the oracle's own
    noise periodograms exceeding z must be eq. (3) with N_f = 1 within 4.5 standard errors -- and must NOT be the variants
    (2P/Nt in the base; exponent (Nt-2)/2 or (Nt-1)/2), which sit 8+ standard errors away at some z."""
    Nt, M = 12, 20000
    P = _mc_noise_powers(Nt, M, 20261104 + int(gls), gls).reshape(-1)
    n = P.size
    far = {"base_N": 0.0, "exp_Nm2": 0.0, "exp_Nm1": 0.0}
    for z in (0.5, 1.0, 2.0, 3.0, 4.0):
        emp = float((P > z).mean())
        q = float(oracle.false_alarm_probability(np.array([z]), Nt, 1.0)[0])
        se = np.sqrt(max(q * (1 - q), 1e-9) / (n / 4.0))   # 4 frequencies of one series share its variance estimate: count series, not values
        assert abs(emp - q) <= 4.5 * se, (z, emp, q, se)
        p = 2 * z / (Nt - 1)
        variants = {"base_N": (1 - 2 * z / Nt) ** ((Nt - 3) / 2), "exp_Nm2": (1 - p) ** ((Nt - 2) / 2), "exp_Nm1": (1 - p) ** ((Nt - 1) / 2)}
        for name, v in variants.items():
            far[name] = max(far[name], abs(emp - v) / se)
    assert min(far.values()) > 8.0, far


def test_fap_F3_monte_carlo_many_independent_frequencies():
    """Pin F3: the [...]^N_f of eq. (3) is the chance that the LARGEST of N_f independent powers exceeds z.  Independent
    powers are made honestly: one frequency from each of N_f independent noise series (distinct variance estimates)."""
    Nt, Nf, M = 12, 8, 4000
    P = _mc_noise_powers(Nt, M * Nf, 777, True)[:, 0].reshape(M, Nf)
    peak = P.max(axis=1)
    for z in (2.0, 3.0, 4.0):
        emp = float((peak > z).mean())
        q = float(oracle.false_alarm_probability(np.array([z]), Nt, float(Nf))[0])
        se = np.sqrt(q * (1 - q) / M)
        assert abs(emp - q) <= 4.5 * se, (z, emp, q, se)
        q1 = float(oracle.false_alarm_probability(np.array([z]), Nt, 1.0)[0])
        assert abs(emp - q1) > 8 * se                      # N_f really enters


def test_paper_facts_fixture():
    """Numbers printed in the paper (tests/golden/paper_facts.json) are self-consistent."""
    with open(os.path.join(HERE, "golden", "paper_facts.json")) as fh:
        facts = json.load(fh)
    Nt, Nf = facts["validation_Nt"]["value"], facts["validation_Nf"]["value"]
    assert Nf % facts["block_size"]["value"] == 0          # reading G8: Nf rounded up to blocks of 256
    assert Nf * (4 * Nt + 1) > Nf * (2 * Nt + 3)           # PAPER.md:59 vs :86, "factor ~2"
    assert abs(Nf * (4 * Nt + 1) / (Nf * (2 * Nt + 3)) - 2.0) < 1e-4
    tc = facts["t_calc_s"]
    assert abs(tc["cpu8"] / tc["C1060"] - 28) < 1.0        # "approaching thirty" (abstract)


# ------------------------------------------------------------------ generalised (floating-mean) periodogram
def _gappy(Nt, seed, span=30.0):
    rng = np.random.default_rng(seed)
    t = np.sort(rng.uniform(0.0, span, Nt))
    return rng, t


def test_GP1_c_gls_matches_numpy_lstsq():
    """C normal equations + elimination vs numpy's SVD least squares (independent solver), random sampling."""
    rng, t = _gappy(57, 11)
    x = (1.3 + np.sin(2 * np.pi * 0.41 * t + 0.3) + 0.4 * rng.standard_normal(t.size)).astype(np.float32)
    f_min, df, Nf = 0.02, 0.013, 90
    P = oracle.periodogram_gls(t, x, f_min, df, Nf)
    ref = oracle.periodogram_gls_numpy(t, x, f_min + df * np.arange(Nf))
    assert np.max(np.abs(P - ref)) <= 1e-11 * max(1.0, ref.max())
    ks = np.array([0, 7, 89, 44], dtype=np.int64)
    assert np.array_equal(oracle.periodogram_gls(t, x, f_min, df, Nf, ks=ks), P[ks])


def test_GP2_scipy_floating_mean():
    """Library special case: scipy.signal.lombscargle(floating_mean=True, normalize=True) is the fraction of the
    variance the fit explains; times (Nt - 1)/2 it is this normalisation."""
    from scipy.signal import lombscargle
    rng, t = _gappy(200, 12, span=50.0)
    x = (5.0 + 0.8 * np.sin(2 * np.pi * 0.23 * t) + rng.standard_normal(t.size)).astype(np.float32)
    f = 0.01 + 0.004 * np.arange(400)
    P = oracle.periodogram_gls(t, x, f[0], 0.004, f.size)
    X = x.astype(np.float64)
    p = lombscargle(t, X, 2 * np.pi * f, floating_mean=True, normalize=True)
    assert np.max(np.abs(P - p * (t.size - 1) / 2.0)) <= 1e-9 * P.max()


def test_GP3_sinusoid_plus_offset_reaches_the_maximum():
    """x = c + A sin(w t + phi) sampled over a FRACTION of a cycle: the floating-mean fit is exact, so
    P = (Nt - 1)/2 (the largest possible value), whereas eq. (1) (mean fixed at the sample mean) falls short."""
    t = np.linspace(0.0, 0.6, 41) ** 1.3                       # uneven, 0.3 of a cycle of f0
    f0 = 0.5
    x = (2.0 + 0.7 * np.sin(2 * np.pi * f0 * t + 0.9)).astype(np.float64)
    x32 = x.astype(np.float32)
    P = oracle.periodogram_gls(t, x32, f0, 1.0, 1)[0]
    assert abs(P - (t.size - 1) / 2.0) <= 1e-5 * (t.size - 1) / 2.0      # fp32 rounding of x is the only residual
    assert oracle.periodogram(t, x32, f0, 1.0, 1)[0] < 0.99 * P


def test_GP4_equals_eq1_on_even_sampling_at_fourier_frequencies():
    """Even sampling, Fourier frequencies 0 < k < N/2: sum cos = sum sin = 0, the constant is orthogonal to the
    sinusoids and the generalised periodogram reduces to eq. (1)."""
    N, dt = 64, 0.25
    rng = np.random.default_rng(13)
    t = dt * np.arange(N)
    x = rng.standard_normal(N).astype(np.float32)
    df = 1.0 / (N * dt)
    P1 = oracle.periodogram(t, x, df, df, N // 2 - 1)
    Pg = oracle.periodogram_gls(t, x, df, df, N // 2 - 1)
    assert np.max(np.abs(P1 - Pg)) <= 1e-12 * P1.max()


def test_GP5_zechmeister_kuerster_closed_form():
    """The closed form of the cited paper (Zechmeister & Kuerster 2009, eqs 4-13, unit weights w = 1/N), typed here:
    p = [SS YC^2 + CC YS^2 - 2 CS YC YS] / (YY D), D = CC SS - CS^2, with mean-corrected sums; P = p (Nt-1)/2."""
    rng, t = _gappy(83, 14, span=12.0)
    x = (0.2 + np.cos(2 * np.pi * 0.9 * t) + 0.5 * rng.standard_normal(t.size)).astype(np.float32)
    y = x.astype(np.float64)
    N = t.size
    f = 0.05 + 0.021 * np.arange(120)
    out = np.empty(f.size)
    for i, fi in enumerate(f):
        c, s = np.cos(2 * np.pi * fi * t), np.sin(2 * np.pi * fi * t)
        Y, C, S = y.mean(), c.mean(), s.mean()
        YY = (y * y).mean() - Y * Y
        YC = (y * c).mean() - Y * C
        YS = (y * s).mean() - Y * S
        CC = (c * c).mean() - C * C
        SS = (s * s).mean() - S * S
        CS = (c * s).mean() - C * S
        D = CC * SS - CS * CS
        out[i] = (SS * YC ** 2 + CC * YS ** 2 - 2 * CS * YC * YS) / (YY * D) * (N - 1) / 2.0
    P = oracle.periodogram_gls(t, x, f[0], 0.021, f.size)
    assert np.max(np.abs(P - out)) <= 1e-10 * P.max()
    assert P.min() >= 0.0 and P.max() <= (N - 1) / 2.0
    assert oracle.periodogram_gls(t, x, 0.0, 0.1, 1)[0] == 0.0                  # singular at f = 0 (G7)


def test_GP6_low_frequencies_against_60_digit_least_squares():
    """Reading G15 (oracle/lsp_oracle.c, lsp_oracle_gls_fit): the fit is posed in a centred, scaled basis so that it stays
    accurate as f T -> 0.  Pin: the SAME fit on the RAW basis {cos(w t), sin(w t), 1} and raw times, solved in 60-digit
    arithmetic (there the raw normal equations have digits to spare), with and without weights, on a series with a drift
    (whose low-frequency power is large: the fit tends to that of a quadratic trend), from f T = 1e-6 to 2.5."""
    import mpmath as mp
    mp.mp.dps = 60
    rng = np.random.default_rng(77)
    Nt, T = 40, 9.0
    t = 1000.0 + np.sort(rng.uniform(0.0, T, Nt))                          # far from the origin: the centring has work to do
    x = (rng.standard_normal(Nt) + 0.4 * (t - 1000.0)).astype(np.float32)
    wts = rng.uniform(0.2, 3.0, Nt).astype(np.float32)

    def exact(weights, f):
        w = [mp.mpf(float(v)) for v in weights]
        tm = [mp.mpf(float(v)) for v in t]
        xm = [mp.mpf(float(v)) for v in x]
        W = sum(w)
        mean = sum(a * b for a, b in zip(w, xm)) / W
        d = [v - mean for v in xm]
        chi0 = sum(a * b * b for a, b in zip(w, d))
        A, rhs = mp.zeros(3, 3), mp.zeros(3, 1)
        for tj, dj, wj in zip(tm, d, w):
            a = 2 * mp.pi * mp.mpf(f) * tj
            g = [mp.cos(a), mp.sin(a), mp.mpf(1)]
            for r in range(3):
                for c in range(3):
                    A[r, c] += wj * g[r] * g[c]
                rhs[r] += wj * g[r] * dj
        beta = mp.lu_solve(A, rhs)
        return float((Nt - 1) / 2 * sum(beta[r] * rhs[r] for r in range(3)) / chi0)

    for fT in (1e-6, 1e-4, 1e-2, 0.3, 2.5):
        f = fT / T
        want_w, want_u = exact(wts, f), exact(np.ones(Nt), f)
        got_w = oracle.periodogram_gls_weighted(t, x, wts, f, 0.1, 1)[0]
        got_u = oracle.periodogram_gls(t, x, f, 0.1, 1)[0]
        assert abs(got_w - want_w) <= 1e-7 * want_w, (fT, got_w, want_w)
        assert abs(got_u - want_u) <= 1e-7 * want_u, (fT, got_u, want_u)
        assert fT > 0.3 or want_u > 1.0                                    # the drift: low-frequency power is not negligible
    assert oracle.periodogram_gls(t, x, 0.0, 0.1, 1)[0] == 0.0             # f = 0 itself: singular, reading G7


# ----------------------------------------------------------------------------- weighted generalised periodogram (GW1-GW5)
def _weighted_case(Nt=120, seed=31, span=40.0):
    rng, t = _gappy(Nt, seed, span=span)
    sig = rng.uniform(0.3, 2.0, t.size)                                   # per-sample error bars
    x = (3.0 + 0.9 * np.sin(2 * np.pi * 0.31 * t + 0.4) + sig * rng.standard_normal(t.size)).astype(np.float32)
    w = (1.0 / sig ** 2).astype(np.float32)
    return rng, t, x, w


def test_GW1_constant_weights_reduce_to_the_unweighted_periodogram():
    """w_j = const must reproduce lsp_oracle_gls (pins GP1-GP5), whatever the constant: only weight RATIOS matter."""
    rng, t, x, _ = _weighted_case()
    f0, df, Nf = 0.02, 0.007, 300
    ref = oracle.periodogram_gls(t, x, f0, df, Nf)
    for c in (1.0, 0.125, 37.0):
        P = oracle.periodogram_gls_weighted(t, x, np.full(t.size, c, np.float32), f0, df, Nf)
        assert np.max(np.abs(P - ref)) <= 1e-11 * ref.max()


def test_GW2_integer_weights_equal_repeated_samples():
    """A sample with weight n is n copies of that sample: the chi^2 ratio of the weighted fit equals the chi^2 ratio of
    the UNWEIGHTED generalised periodogram (pinned on its own) of the expanded series.  Catches a weight applied to the
    wrong factor, squared, or left out of one of the sums."""
    rng, t, x, _ = _weighted_case(Nt=60, seed=5)
    n = rng.integers(1, 5, t.size)
    f0, df, Nf = 0.03, 0.011, 150
    Pw = oracle.periodogram_gls_weighted(t, x, n.astype(np.float32), f0, df, Nf)
    te, xe = np.repeat(t, n), np.repeat(x, n)
    Pe = oracle.periodogram_gls(te, xe, f0, df, Nf)
    ratio_w = Pw / ((t.size - 1) / 2.0)
    ratio_e = Pe / ((te.size - 1) / 2.0)
    assert np.max(np.abs(ratio_w - ratio_e)) <= 1e-11


def test_GW3_numpy_lstsq_on_sqrt_weighted_rows():
    """Independent solver: minimise |sqrt(w) (x - A beta)|^2 by numpy.linalg.lstsq (SVD) row-scaled by sqrt(w)."""
    rng, t, x, w = _weighted_case(Nt=90, seed=77)
    f0, df, Nf = 0.04, 0.013, 120
    P = oracle.periodogram_gls_weighted(t, x, w, f0, df, Nf)
    y, wd = x.astype(np.float64), w.astype(np.float64)
    sw = np.sqrt(wd)
    ybar = (wd * y).sum() / wd.sum()
    chi0 = (wd * (y - ybar) ** 2).sum()
    out = np.empty(Nf)
    for i in range(Nf):
        om = 2 * np.pi * (f0 + i * df)
        A = np.stack([np.cos(om * t), np.sin(om * t), np.ones(t.size)], axis=1)
        beta = np.linalg.lstsq(A * sw[:, None], y * sw, rcond=None)[0]
        chi = (wd * (y - A @ beta) ** 2).sum()
        out[i] = 0.5 * (t.size - 1) * (chi0 - chi) / chi0
    assert np.max(np.abs(P - out)) <= 1e-10 * P.max()
    assert P.min() >= 0.0 and P.max() <= (t.size - 1) / 2.0


def test_GW4_scipy_lombscargle_weights():
    """Library special case: scipy.signal.lombscargle(weights=w, floating_mean=True, normalize=True) is the fraction of the
    weighted variance the fit explains; times (Nt - 1)/2 it is this normalisation (as GP2 for unit weights)."""
    from scipy.signal import lombscargle
    rng, t, x, w = _weighted_case(Nt=200, seed=12, span=50.0)
    f = 0.01 + 0.004 * np.arange(400)
    P = oracle.periodogram_gls_weighted(t, x, w, f[0], 0.004, f.size)
    p = lombscargle(t, x.astype(np.float64), 2 * np.pi * f, weights=w.astype(np.float64), floating_mean=True, normalize=True)
    assert np.max(np.abs(P - p * (t.size - 1) / 2.0)) <= 1e-9 * P.max()


def test_GW5_zechmeister_kuerster_closed_form_with_weights():
    """The closed form of the cited paper (Zechmeister & Kuerster 2009) with normalised weights w_j / sum w, typed here:
    p = [SS YC^2 + CC YS^2 - 2 CS YC YS] / (YY D); plus: a zero weight removes the sample from the fit, and a noise-free
    sinusoid + offset reaches the maximum (Nt - 1)/2 whatever the weights."""
    rng, t, x, w = _weighted_case(Nt=83, seed=14, span=12.0)
    y, wn = x.astype(np.float64), w.astype(np.float64) / w.astype(np.float64).sum()
    f = 0.05 + 0.021 * np.arange(120)
    out = np.empty(f.size)
    for i, fi in enumerate(f):
        c, s = np.cos(2 * np.pi * fi * t), np.sin(2 * np.pi * fi * t)
        Y, C, S = (wn * y).sum(), (wn * c).sum(), (wn * s).sum()
        YY = (wn * y * y).sum() - Y * Y
        YC = (wn * y * c).sum() - Y * C
        YS = (wn * y * s).sum() - Y * S
        CC = (wn * c * c).sum() - C * C
        SS = (wn * s * s).sum() - S * S
        CS = (wn * c * s).sum() - C * S
        D = CC * SS - CS * CS
        out[i] = (SS * YC ** 2 + CC * YS ** 2 - 2 * CS * YC * YS) / (YY * D) * (t.size - 1) / 2.0
    P = oracle.periodogram_gls_weighted(t, x, w, f[0], 0.021, f.size)
    assert np.max(np.abs(P - out)) <= 1e-10 * P.max()
    # zero weights: same chi^2 ratio as the series without those samples
    w0 = w.copy(); w0[::3] = 0.0
    keep = w0 > 0
    Pz = oracle.periodogram_gls_weighted(t, x, w0, f[0], 0.021, f.size) / ((t.size - 1) / 2.0)
    Pk = oracle.periodogram_gls_weighted(t[keep], x[keep], w0[keep], f[0], 0.021, f.size) / ((keep.sum() - 1) / 2.0)
    assert np.max(np.abs(Pz - Pk)) <= 1e-11
    # exact model: the fit is perfect at its own frequency
    xs = (2.0 + 1.5 * np.cos(2 * np.pi * 0.4 * t - 0.3)).astype(np.float32)
    Pm = oracle.periodogram_gls_weighted(t, xs, w, 0.4, 0.1, 1)[0]
    assert abs(Pm - (t.size - 1) / 2.0) <= 1e-5 * (t.size - 1) / 2.0     # x is fp32: the model is exact to ~1e-7 per sample
    assert oracle.periodogram_gls_weighted(t, x, w, 0.0, 0.1, 1)[0] == 0.0          # singular at f = 0 (G7)
