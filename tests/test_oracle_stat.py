"""Pins for the oracle's statistic core (oracle/sc_oracle.c: sco_stat_from_arrays, sco_inner) -- SURVEY.md 8(c) O1/O6.

None of these retype the oracle's formula: they use identities the paper states, brute force over the phase
that Eq. 8/10 maximise, exact closed forms, and the sampling distributions the paper prints (Eq. 11-12).
"""
import json
import os

import numpy as np
import pytest

import sc_synth as sy

GOLD = json.load(open(os.path.join(os.path.dirname(__file__), "golden", "paper_values.json")))


def _rand_arrays(rng, n):
    d = rng.standard_normal(n) + 1j * rng.standard_normal(n)
    h = (rng.standard_normal(n) + 1j * rng.standard_normal(n)) * rng.uniform(0.5, 2.0, n)
    S = rng.uniform(0.5, 3.0, n)
    return d, h, S


def _bracket(a, b, S, df, lo, hi):
    """Literal Eq. 7 for one channel list: [a|b]_n = sum_alpha 4 Re sum_j a b^dagger / S df."""
    tot = 0.0
    for aa, bb, SS in zip(a, b, S):
        for j in range(lo, hi):
            tot += 4.0 * (aa[j] * np.conj(bb[j]) / SS[j]).real * df
    return tot


def test_bruteforce_phase_maximisation_tiny_grids(oracle):
    """(vi) Eq. 10 by explicit grid search over phi_n on n_bins <= 16, N <= 4."""
    rng = np.random.default_rng(11)
    phis = np.linspace(0.0, 2.0 * np.pi, 7201)
    for trial in range(6):
        n = int(rng.integers(5, 17))
        N = int(rng.integers(1, 5))
        df = rng.uniform(0.1, 2.0)
        dA, hA, SA = _rand_arrays(rng, n)
        dE, hE, SE = _rand_arrays(rng, n)
        cuts = np.sort(rng.choice(np.arange(1, n), size=N - 1, replace=False)) if N > 1 else np.array([], dtype=int)
        edges = np.concatenate([[0], cuts, [n]]).astype(np.int64)
        ups = 0.0
        for k in range(N):
            lo, hi = int(edges[k]), int(edges[k + 1])
            best = max(_bracket([dA, dE], [hA * np.exp(1j * p), hE * np.exp(1j * p)], [SA, SE], df, lo, hi)
                       for p in phis)
            # refine the grid maximum: [d|h e^{i phi}] = R cos(phi - phi0); grid error <= R (dphi/2)^2/2
            hh = _bracket([hA, hE], [hA, hE], [SA, SE], df, lo, hi)
            ups += best ** 2 / hh
        got = oracle.stat_from_arrays(dA, dE, hA, hE, SA, SE, df, edges)
        assert got == pytest.approx(ups, rel=2e-7)          # (2pi/7200/2)^2 = 1.9e-7 worst-case grid error
        assert got >= ups * (1 - 1e-12)                      # the grid can only under-estimate the maximum


def test_single_channel_matches_two_channel_with_zero_E(oracle):
    rng = np.random.default_rng(5)
    n = 40
    d, h, S = _rand_arrays(rng, n)
    e = sy.edges(n, 4)
    one = oracle.stat_from_arrays(d, None, h, None, S, None, 0.3, e)
    two = oracle.stat_from_arrays(d, d * 0, h, h * 0, S, S, 0.3, e)
    assert one == pytest.approx(two, rel=1e-15)


def test_exact_match_gives_rho_squared_for_any_edges(oracle):
    """(i),(ii) d = h, no noise: Upsilon_N = <h|h> = rho^2 for N = 1 and for any segmentation."""
    rng = np.random.default_rng(3)
    n = 5000
    _, hA, SA = _rand_arrays(rng, n)
    _, hE, SE = _rand_arrays(rng, n)
    df = 0.37
    rho2 = oracle.inner(hA, hE, hA, hE, SA, SE, df)
    # sco_inner against the library routine Eq. 1 reduces to: 4 df Re vdot
    assert rho2 == pytest.approx(4 * df * (np.vdot(hA / SA, hA) + np.vdot(hE / SE, hE)).real, rel=1e-13)
    for N in (1, 2, 7, 100, 5000):
        assert oracle.stat_from_arrays(hA, hE, hA, hE, SA, SE, df, sy.edges(n, N)) == pytest.approx(rho2, rel=1e-12)
    # partial coverage: only the covered bins count
    e = np.array([100, 900, 901, 901, 2500], dtype=np.int64)
    part = oracle.inner(hA[100:2500], hE[100:2500], hA[100:2500], hE[100:2500], SA[100:2500], SE[100:2500], df)
    assert oracle.stat_from_arrays(hA, hE, hA, hE, SA, SE, df, e) == pytest.approx(part, rel=1e-12)


def test_invariances(oracle):
    """(iii) overall phase, amplitude (1/D_L) and per-segment complex rescaling leave Upsilon unchanged
    (the phase is maximised in each segment independently)."""
    rng = np.random.default_rng(4)
    n, N, df = 3000, 30, 1.3
    dA, hA, SA = _rand_arrays(rng, n)
    dE, hE, SE = _rand_arrays(rng, n)
    e = sy.edges(n, N)
    base = oracle.stat_from_arrays(dA, dE, hA, hE, SA, SE, df, e)
    ph = np.exp(1j * 0.7311)
    assert oracle.stat_from_arrays(dA, dE, hA * ph, hE * ph, SA, SE, df, e) == pytest.approx(base, rel=1e-12)
    assert oracle.stat_from_arrays(dA, dE, hA * 3e-21, hE * 3e-21, SA, SE, df, e) == pytest.approx(base, rel=1e-12)
    fac = np.repeat(rng.standard_normal(N) + 1j * rng.standard_normal(N), np.diff(e))
    assert oracle.stat_from_arrays(dA, dE, hA * fac, hE * fac, SA, SE, df, e) == pytest.approx(base, rel=1e-11)
    # a phase applied to ONE channel only is NOT an invariance (Q1: one common phase per segment, channels summed inside)
    assert abs(oracle.stat_from_arrays(dA, dE, hA * ph, hE, SA, SE, df, e) / base - 1) > 1e-3


def test_refinement_monotone_and_cauchy_schwarz(oracle):
    """(iv) nested refinement never decreases Upsilon; (v) Upsilon_N <= <d|d>."""
    rng = np.random.default_rng(8)
    n, df = 6000, 0.9
    dA, hA, SA = _rand_arrays(rng, n)
    dE, hE, SE = _rand_arrays(rng, n)
    vals = [oracle.stat_from_arrays(dA, dE, hA, hE, SA, SE, df, sy.edges(n, N)) for N in (1, 10, 100, 1000, 6000)]
    assert all(b >= a * (1 - 1e-13) for a, b in zip(vals, vals[1:]))
    dd = oracle.inner(dA, dE, dA, dE, SA, SE, df)
    assert all(v <= dd * (1 + 1e-13) for v in vals)
    # N = n_bins with one channel: each bin matches perfectly -> equality in Cauchy-Schwarz
    one = oracle.stat_from_arrays(dA, None, hA, None, SA, None, df, sy.edges(n, n))
    assert one == pytest.approx(oracle.inner(dA, None, dA, None, SA, None, df), rel=1e-12)


def test_impulse_segment_indexing_bit_exact(oracle):
    """(vii) a one-bin impulse lands in exactly the segment k with e_k <= j < e_{k+1}, incl. empty and 1-bin segments."""
    n = 1000
    rng = np.random.default_rng(9)
    h = np.ones(n) * (1 + 0.5j)
    S = np.ones(n)
    for edges in (sy.edges(n, 7), sy.edges(n, 333), np.array([0, 0, 1, 1, 2, 500, 500, 999, 1000], dtype=np.int64),
                  np.array([10, 20, 990], dtype=np.int64)):
        for j in list(rng.integers(0, n, 20)) + [0, 1, 2, 9, 10, 19, 20, 499, 500, 989, 990, 998, 999]:
            d = np.zeros(n, dtype=complex)
            d[j] = 2.0 - 1.0j
            _, seg = oracle.stat_from_arrays(d, None, h, None, S, None, 1.0, edges, want_seg=True)
            nz = np.nonzero(seg[:, 0] ** 2 + seg[:, 1] ** 2)[0]
            k = np.searchsorted(edges, j, side="right") - 1
            if 0 <= k < len(edges) - 1 and edges[k] <= j < edges[k + 1]:
                assert list(nz) == [k]
                assert complex(seg[k, 0], seg[k, 1]) == d[j] * np.conj(h[j])     # exact: one term, S = 1
            else:
                assert len(nz) == 0
            # sigma_k is the plain count of |h|^2 over the segment
            assert np.array_equal(seg[:, 2], np.diff(edges) * 1.25)


def test_empty_and_zero_template_segments_contribute_zero(oracle):
    """Q8."""
    n = 64
    rng = np.random.default_rng(1)
    d, h, S = _rand_arrays(rng, n)
    h[16:32] = 0
    e = np.array([0, 16, 32, 32, 64], dtype=np.int64)
    full = oracle.stat_from_arrays(d, None, h, None, S, None, 1.0, e)
    a = oracle.stat_from_arrays(d, None, h, None, S, None, 1.0, np.array([0, 16], dtype=np.int64))
    b = oracle.stat_from_arrays(d, None, h, None, S, None, 1.0, np.array([32, 64], dtype=np.int64))
    assert np.isfinite(full) and full == pytest.approx(a + b, rel=1e-14)
    assert oracle.stat_from_arrays(d, None, h * 0, None, S, None, 1.0, e) == 0.0


@pytest.mark.parametrize("N", [1, 10, 100])
def test_sampling_distribution_moments(oracle, N):
    """O6 normalisation against Eq. 11-12 and chi^2_2:
    noise only: mean 2N, sd 2 sqrt N; signal of SNR rho at theta_*: mean 2N + rho^2, sd 2 sqrt(N + rho^2).
    (For Gaussian noise the first two moments are exact for every N, not only in the CLT limit.)"""
    assert GOLD["sampling_distributions"]["mu_k"] == 2.0
    n, rho = 4000, 12.0
    f = 0.02 + np.arange(n) * 1e-7
    S = sy.psd_AE(f)
    df = 1e-7
    rng = np.random.default_rng(100 + N)
    hA = (rng.standard_normal(n) + 1j * rng.standard_normal(n)) * 1e-20
    hE = (rng.standard_normal(n) + 1j * rng.standard_normal(n)) * 1e-20
    kappa = rho / np.sqrt(oracle.inner(hA, hE, hA, hE, S, S, df))
    e = sy.edges(n, N)
    trials = 1500
    noise_only, with_signal = [], []
    for t in range(trials):
        nA = sy.draw_noise(7000 + 2 * t, S, df)
        nE = sy.draw_noise(7001 + 2 * t, S, df)
        noise_only.append(oracle.stat_from_arrays(nA, nE, hA, hE, S, S, df, e))
        with_signal.append(oracle.stat_from_arrays(nA + kappa * hA, nE + kappa * hE, hA, hE, S, S, df, e))
    for vals, mean, var in ((noise_only, 2 * N, 4 * N), (with_signal, 2 * N + rho ** 2, 4 * N + 4 * rho ** 2)):
        m, v = np.mean(vals), np.var(vals)
        assert abs(m - mean) < 5 * np.sqrt(var / trials)          # 5 sigma on the mean
        assert v == pytest.approx(var, rel=0.25)
    if N == 1:
        # chi^2_2: P(Upsilon_1 > x) = exp(-x/2)
        frac = np.mean(np.array(noise_only) > 2 * np.log(2))
        assert frac == pytest.approx(0.5, abs=0.07)
