"""Pins for the oracle's Eq. 8 / Eq. 9 quantities and for the equal-SNR^2 segment edges of PAPER.md:120 / App. A
(oracle/sc_oracle.c: sco_components_from_seg, sco_loglike, sco_equal_snr_edges, sco_eval_stat_adaptive).

Nothing here retypes the oracle's loops: the pins are brute force over the phases Eq. 8 maximises, closed forms
(noise-free match, analytic amplitude maximum, quantiles of flat and power-law spectra), the paper's Appendix A
statement and invariants that hold for any input.
"""
import numpy as np
import pytest

import sc_synth as sy


def _rand(rng, n):
    d = rng.standard_normal(n) + 1j * rng.standard_normal(n)
    h = (rng.standard_normal(n) + 1j * rng.standard_normal(n)) * rng.uniform(0.5, 2.0, n)
    S = rng.uniform(0.5, 3.0, n)
    return d, h, S


def _bracket(a, b, S, df, lo, hi):
    """Literal Eq. 7."""
    tot = 0.0
    for aa, bb, SS in zip(a, b, S):
        tot += 4.0 * df * float(np.sum((aa[lo:hi] * np.conj(bb[lo:hi]) / SS[lo:hi]).real))
    return tot


# ------------------------------------------------------------------------------------------ Eq. 8, Eq. 9
def test_overlap_is_sum_of_phase_maxima_bruteforce(oracle):
    """Eq. 8: O_hat_N = sum_n max_phi [d | h e^{i phi}]_n, by grid search over phi in every segment."""
    rng = np.random.default_rng(21)
    phis = np.linspace(0.0, 2.0 * np.pi, 3601)
    for _ in range(5):
        n, N = int(rng.integers(6, 20)), int(rng.integers(1, 5))
        df = rng.uniform(0.2, 2.0)
        dA, hA, SA = _rand(rng, n)
        dE, hE, SE = _rand(rng, n)
        cuts = np.sort(rng.choice(np.arange(1, n), size=N - 1, replace=False)) if N > 1 else np.array([], dtype=int)
        e = np.concatenate([[0], cuts, [n]]).astype(np.int64)
        _, seg = oracle.stat_from_arrays(dA, dE, hA, hE, SA, SE, df, e, want_seg=True)
        ups, ohat, hh = oracle.components_from_seg(seg, df)
        want = sum(max(_bracket([dA, dE], [hA * np.exp(1j * p), hE * np.exp(1j * p)], [SA, SE], df, int(e[k]), int(e[k + 1]))
                       for p in phis) for k in range(N))
        assert ohat == pytest.approx(want, rel=5e-7) and ohat >= want * (1 - 1e-12)
        assert hh == pytest.approx(_bracket([hA, hE], [hA, hE], [SA, SE], df, 0, n), rel=1e-12)       # Eq. 3
        assert ups == pytest.approx(oracle.stat_from_arrays(dA, dE, hA, hE, SA, SE, df, e), rel=1e-13)


def test_loglike_closed_forms(oracle):
    """Eq. 9 against Eq. 4-5 where they must agree, and its analytic amplitude maximum."""
    rng = np.random.default_rng(22)
    n, df = 64, 0.7
    dA, hA, SA = _rand(rng, n)
    dE, hE, SE = _rand(rng, n)
    e = sy.edges(n, 8)
    # (i) noise-free exact match d = A0 h: every segment is in phase, so log L_hat_N(A0) = -1/2 <d - A0 h|d - A0 h> = 0
    A0 = 3.7
    _, seg = oracle.stat_from_arrays(A0 * hA, A0 * hE, hA, hE, SA, SE, df, e, want_seg=True)
    ups, ohat, hh = oracle.components_from_seg(seg, df)
    dd = oracle.inner(A0 * hA, A0 * hE, A0 * hA, A0 * hE, SA, SE, df)
    assert abs(oracle.loglike(dd, hh, ohat, A0)) <= 1e-10 * dd
    assert ups == pytest.approx(A0 ** 2 * hh, rel=1e-12)                       # Upsilon = rho^2 for any edges
    # (ii) N = 1 and the best common phase: Eq. 9 equals the coherent Eq. 4, -1/2 <d - h e^{i phi*}|d - h e^{i phi*}>
    e1 = sy.edges(n, 1)
    _, seg1 = oracle.stat_from_arrays(dA, dE, hA, hE, SA, SE, df, e1, want_seg=True)
    ups1, ohat1, hh1 = oracle.components_from_seg(seg1, df)
    dd = oracle.inner(dA, dE, dA, dE, SA, SE, df)
    phis = np.linspace(0, 2 * np.pi, 20001)
    coh = max(-0.5 * _bracket([dA - 1.3 * hA * np.exp(1j * p), dE - 1.3 * hE * np.exp(1j * p)],
                              [dA - 1.3 * hA * np.exp(1j * p), dE - 1.3 * hE * np.exp(1j * p)], [SA, SE], df, 0, n)
              for p in phis)
    assert oracle.loglike(dd, hh1, ohat1, 1.3) == pytest.approx(coh, abs=1e-6 * dd)
    # (iii) maximum over the amplitude: A* = O_hat/<h|h>, value -1/2<d|d> + 1/2 O_hat^2/<h|h>; at N = 1 that is Upsilon_1/2
    a_star = ohat1 / hh1
    top = oracle.loglike(dd, hh1, ohat1, a_star)
    assert top == pytest.approx(-0.5 * dd + 0.5 * ups1, rel=1e-12)
    assert top >= oracle.loglike(dd, hh1, ohat1, a_star * 1.01) and top >= oracle.loglike(dd, hh1, ohat1, a_star * 0.99)
    # (iv) N > 1: O_hat^2/<h|h> <= Upsilon_N (Cauchy-Schwarz over segments), so the amplitude-maximised likelihood is bounded
    _, seg = oracle.stat_from_arrays(dA, dE, hA, hE, SA, SE, df, e, want_seg=True)
    ups, ohat, hh = oracle.components_from_seg(seg, df)
    assert ohat ** 2 / hh <= ups * (1 + 1e-12) and ohat >= ohat1 * (1 - 1e-12)      # more segments, more freedom


# ------------------------------------------------------------------------------------------ PAPER.md:120, App. A
def test_edges_flat_spectrum_closed_form(oracle):
    """Equal s_j (linear chirp + white PSD, App. A: |h(f)|^2 flat, t proportional to f): the
    equal-SNR^2 edges are equal-width in frequency = equal-duration in time, e_n = ceil(n n_bins / N).
    (s_j = 2^-3 is exact in floating point, so the comparison C_j >= C n/N is exact too.)"""
    for n, N in ((1000, 10), (1000, 7), (97, 13), (64, 64), (50, 1)):
        h = np.full(n, 0.25 + 0.25j)            # |h|^2 = 1/8
        S = np.ones(n)
        e = oracle.equal_snr_edges(h, None, S, None, N)
        want = [-(-k * n // N) for k in range(N + 1)]
        assert list(e) == want


def test_edges_power_law_quantiles(oracle):
    """s(f) ~ f^-7/3 (the inspiral |h|^2 with white noise): C(f) ~ f_lo^-4/3 - f^-4/3, so the quantile frequencies
    are closed form; the discrete edges must sit within one bin of them."""
    f = np.linspace(0.017, 0.030, 200001)
    h = f ** (-7.0 / 6.0) * np.exp(1j * 0.3)
    S = np.ones_like(f)
    N = 37
    e = oracle.equal_snr_edges(h, None, S, None, N)
    a, b = f[0] ** (-4.0 / 3.0), f[-1] ** (-4.0 / 3.0)
    fq = (a - (a - b) * np.arange(N + 1) / N) ** (-0.75)
    jq = (fq - f[0]) / (f[1] - f[0])
    assert e[0] == 0 and e[-1] == len(f)
    # first bin AT OR AFTER the quantile (ceil: up to +1) and left-Riemann sum vs integral of a decreasing s (up to ~+1)
    dj = e[1:-1] - jq[1:-1]
    assert dj.min() >= 0.0 and dj.max() <= 2.0


def test_edges_invariants_random_templates(oracle):
    rng = np.random.default_rng(23)
    for _ in range(4):
        n, N = int(rng.integers(200, 600)), int(rng.integers(2, 40))
        _, hA, SA = _rand(rng, n)
        _, hE, SE = _rand(rng, n)
        hA[: n // 7] = 0; hE[: n // 7] = 0                  # a time-window-like empty stretch
        e = oracle.equal_snr_edges(hA, hE, SA, SE, N)
        s = np.abs(hA) ** 2 / SA + np.abs(hE) ** 2 / SE
        assert e[0] == 0 and e[-1] == n and np.all(np.diff(e) >= 0)
        C = np.concatenate([[0.0], np.cumsum(s)])
        for k in range(1, N):
            t = C[-1] * k / N
            assert C[e[k]] >= t * (1 - 1e-12)               # the edge reaches the quantile ...
            assert e[k] == 0 or C[e[k] - 1] < t * (1 + 1e-12)   # ... and is the first bin that does
        per = np.array([s[e[k]:e[k + 1]].sum() for k in range(N)])
        assert np.abs(per - C[-1] / N).max() <= s.max() * (1 + 1e-9)      # each segment holds C/N up to one bin
        # scaling the template (D_L) or the PSD does not move the edges
        e2 = oracle.equal_snr_edges(4.0 * hA, 4.0 * hE, 0.5 * SA, 0.5 * SE, N)
        assert np.array_equal(e, e2)
    z = np.zeros(50, dtype=complex)
    assert list(oracle.equal_snr_edges(z, z, np.ones(50), np.ones(50), 4)) == [0, 0, 0, 0, 50]


def test_adaptive_statistic_consistency(oracle):
    """sco_eval_stat_adaptive = template -> equal-SNR^2 edges -> Eq. 10 on those edges; N = 1 equals the fixed-edge
    statistic; the noise-free exact match still gives rho^2."""
    inp = sy.config_inputs(1, P=3)
    cfg = oracle.make_config(inp["cfg"])
    rng = np.random.default_rng(24)
    nb = cfg.n_bins
    dA = inp["noise_A"]; dE = inp["noise_E"]
    th = inp["particles"]
    N = 25
    ups, edges, comp = oracle.eval_stat_adaptive(cfg, dA, dE, inp["S_A"], inp["S_E"], th, N, want_edges=True, want_comp=True)
    for p in range(3):
        hA, hE, _ = oracle.template(cfg, th[p])
        e = oracle.equal_snr_edges(hA, hE, inp["S_A"], inp["S_E"], N)
        assert np.array_equal(e, edges[p])
        u, seg = oracle.stat_from_arrays(dA, dE, hA, hE, inp["S_A"], inp["S_E"], inp["df"], e, want_seg=True)
        assert u == ups[p]
        assert np.allclose(comp[p], oracle.components_from_seg(seg, inp["df"]), rtol=1e-14)
        # the supplied-edges path reproduces it
    again = oracle.eval_stat_adaptive(cfg, dA, dE, inp["S_A"], inp["S_E"], th, N, in_edges=edges)
    assert np.array_equal(again, ups)
    one = oracle.eval_stat_adaptive(cfg, dA, dE, inp["S_A"], inp["S_E"], th, 1)
    assert np.array_equal(one, oracle.eval_stat(cfg, dA, dE, inp["S_A"], inp["S_E"], th, sy.edges(nb, 1)))
    # noise-free exact match
    hA, hE, _ = oracle.template(cfg, th[0])
    rho2 = oracle.inner(hA, hE, hA, hE, inp["S_A"], inp["S_E"], inp["df"])
    got = oracle.eval_stat_adaptive(cfg, hA, hE, inp["S_A"], inp["S_E"], th[:1], 50)
    assert got[0] == pytest.approx(rho2, rel=1e-12)
    # equal-SNR^2 segments of the matching template: every term of Eq. 10 is rho^2/N (up to one bin)
    _, e0 = oracle.eval_stat_adaptive(cfg, hA, hE, inp["S_A"], inp["S_E"], th[:1], 50, want_edges=True)
    _, seg = oracle.stat_from_arrays(hA, hE, hA, hE, inp["S_A"], inp["S_E"], inp["df"], e0[0], want_seg=True)
    terms = 4 * inp["df"] * seg[:, 2]
    assert np.abs(terms / (rho2 / 50) - 1).max() < 5e-3
