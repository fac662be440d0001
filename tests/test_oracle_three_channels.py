"""Pins for the three-channel (A, E, T) variants of the oracle and for the harness PSDs: the
closed forms of sc_synth.psd_AE / psd_T against the TDI combination of 12 uncorrelated link noises written out."""
import numpy as np
import pytest

import sc_synth as sy


def _tdi_noise_psd(f):
    """S_A, S_E, S_T from first principles: 6 optical-metrology noises n_sr and 6 test-mass noises, uncorrelated.
    Link s->r carries y_sr = n_sr + delta_r(s) + D delta_s(r)  (the receiving test mass and the delayed sending one),
    D = e^{-2 pi i f L}; X = (1 - D^2)[(y31 + D y13) - (y21 + D y12)], Y, Z cyclic (O4)."""
    x = 2 * np.pi * f * sy.ARM_L_S
    D = np.exp(-1j * x)
    S_oms, S_acc = sy.link_noise_sources(f)
    links = [(1, 2), (2, 1), (2, 3), (3, 2), (3, 1), (1, 3)]                 # (s, r)
    src = {("n", s, r): i for i, (s, r) in enumerate(links)}
    src.update({("d", a, b): 6 + i for i, (a, b) in enumerate(links)})        # test mass of s/c a facing b
    def y(s, r):
        v = np.zeros(12, dtype=complex)
        v[src[("n", s, r)]] += 1.0
        v[src[("d", r, s)]] += 1.0
        v[src[("d", s, r)]] += D
        return v
    def michelson(a, b, c):                                                   # X for (a, b, c) = (1, 2, 3)
        return (1 - D * D) * ((y(c, a) + D * y(a, c)) - (y(b, a) + D * y(a, b)))
    X, Y, Z = michelson(1, 2, 3), michelson(2, 3, 1), michelson(3, 1, 2)
    w = np.concatenate([np.full(6, S_oms), np.full(6, S_acc)])
    out = []
    for comb in ((Z - X) / np.sqrt(2), (X - 2 * Y + Z) / np.sqrt(6), (X + Y + Z) / np.sqrt(3)):
        out.append(float((np.abs(comb) ** 2 * w).sum()))
    cross = float(np.abs((((Z - X) / np.sqrt(2)) * np.conj((X + Y + Z) / np.sqrt(3)) * w).sum()))
    return out, cross


@pytest.mark.parametrize("f", [0.003, 0.010, 0.017, 0.02, 0.03, 0.04, 0.055])
def test_psd_closed_forms_from_uncorrelated_link_noises(f):
    (SA, SE, ST), cross = _tdi_noise_psd(f)
    assert sy.psd_AE(f) == pytest.approx(SA, rel=1e-12)
    assert sy.psd_AE(f) == pytest.approx(SE, rel=1e-12)                        # A and E have the same PSD
    assert sy.psd_T(f) == pytest.approx(ST, rel=1e-11)
    assert cross <= 1e-12 * np.sqrt(SA * ST)                                   # ... and the channels are uncorrelated


def _tiny(oracle, seed=0):
    cfgd = sy.grid_config(0.02, 0.0180, 0.0182)
    cfg = oracle.make_config(cfgd)
    f = sy.freqs(cfgd)
    S3 = (sy.psd_AE(f), sy.psd_AE(f), sy.psd_T(f))
    rng = np.random.default_rng(seed)
    th = np.array([30.0, 0.24, 0.9e8, 1.0, 0.3, 0.7, -1.0, 0.0])
    return cfgd, cfg, f, S3, th, rng


def test_template3_extends_template_and_T_is_the_tdi_T(oracle):
    cfgd, cfg, f, S3, th, rng = _tiny(oracle)
    cfg0 = oracle.make_config(dict(cfgd, window_mode=0))
    hA, hE, hT, w3 = oracle.template3(cfg0, th)
    gA, gE, w2 = oracle.template(cfg0, th)
    assert np.array_equal(hA, gA) and np.array_equal(hE, gE) and w2 == w3
    for j in (0, len(f) // 2, len(f) - 1):                                     # h_T = T(f; t_f) f^(-7/6) e^{-i Psi}
        t = oracle.tf(cfg0, th, f[j])
        T = oracle.tdi(cfg0, th, f[j], t)["T"]
        want = T * f[j] ** (-7.0 / 6.0) * np.exp(-1j * oracle.phase(cfg0, th, f[j]))
        assert hT[j] == pytest.approx(want, rel=1e-12)
    assert 0 < np.abs(hT).max() < np.abs(hA).max()                             # suppressed at these frequencies, not zero


def test_stat3_identities_and_reduction_to_two_channels(oracle):
    cfgd, cfg, f, S3, th, rng = _tiny(oracle, 1)
    df = 1.0 / cfgd["T_obs_s"]
    n = len(f)
    h3 = oracle.template3(oracle.make_config(dict(cfgd, window_mode=0)), th)[:3]
    z = np.zeros(n, dtype=complex)
    for edges in (sy.edges(n, 1), sy.edges(n, 7), np.array([0, 3, 3, 9, n])):
        rho2 = oracle.inner3(h3, h3, S3, df)
        assert oracle.stat_from_arrays3(h3, h3, S3, df, edges) == pytest.approx(rho2, rel=1e-12)   # d = h, any edges
        noise = [np.sqrt(S / (4 * df)) * (rng.standard_normal(n) + 1j * rng.standard_normal(n)) for S in S3]
        d3 = [a + b for a, b in zip(h3, noise)]
        # T data and T template switched off: the two-channel definition
        u2 = oracle.stat_from_arrays(d3[0], d3[1], h3[0], h3[1], S3[0], S3[1], df, edges)
        assert oracle.stat_from_arrays3((d3[0], d3[1], z), (h3[0], h3[1], z), S3, df, edges) == pytest.approx(u2, rel=1e-13)
        # per-segment phase invariance and the channel sum inside |.| (Q1): rotating ALL channels together changes nothing
        u3 = oracle.stat_from_arrays3(d3, h3, S3, df, edges)
        rot = [x * np.exp(0.7j) for x in h3]
        assert oracle.stat_from_arrays3(d3, rot, S3, df, edges) == pytest.approx(u3, rel=1e-12)
        # ... rotating only T does change it (one common phase per segment)
        rotT = [h3[0], h3[1], h3[2] * np.exp(1.3j)]
        assert abs(oracle.stat_from_arrays3(d3, rotT, S3, df, edges) - u3) > 1e-6 * u3
    # brute force on a tiny grid: max over a phase grid of [d|h e^{i phi}] per segment (Eq. 8/10)
    m = 12
    e = np.array([0, 5, m])
    d3 = [rng.standard_normal(m) + 1j * rng.standard_normal(m) for _ in range(3)]
    g3 = [rng.standard_normal(m) + 1j * rng.standard_normal(m) for _ in range(3)]
    Ss = [np.abs(rng.standard_normal(m)) + 0.5 for _ in range(3)]
    phis = np.linspace(0, 2 * np.pi, 20001)
    want = 0.0
    for k in range(2):
        sl = slice(e[k], e[k + 1])
        ip = lambda a, b: 4 * df * sum(np.real((x[sl] * np.conj(y[sl]) / S[sl]).sum()) for x, y, S in zip(a, b, Ss))
        x_k = max(ip(d3, [g * np.exp(1j * p) for g in g3]) for p in phis[::40])
        want += x_k ** 2 / ip(g3, g3)
    assert oracle.stat_from_arrays3(d3, g3, Ss, df, e) == pytest.approx(want, rel=1e-4)


def test_eval_stat3_matches_composition(oracle):
    cfgd, cfg, f, S3, th, rng = _tiny(oracle, 2)
    df = 1.0 / cfgd["T_obs_s"]
    n = len(f)
    d3 = [np.sqrt(S / (4 * df)) * (rng.standard_normal(n) + 1j * rng.standard_normal(n)) for S in S3]
    P = np.vstack([th, th * np.array([1.001, 1, 1, 1.1, 1, 1, 1, 1])])
    e = sy.edges(n, 5)
    out, seg = oracle.eval_stat3(cfg, d3, S3, P, e, want_seg=True)
    for p in range(2):
        h3 = oracle.template3(cfg, P[p])[:3]
        u, s = oracle.stat_from_arrays3(d3, h3, S3, df, e, want_seg=True)
        assert out[p] == u and np.array_equal(seg[p], s)


def test_equal_snr_edges3_pins(oracle):
    """PAPER.md:120 over three channels: (i) without T the rule is sco_equal_snr_edges; (ii) every segment holds C/N to within
    one bin's s_j, with s_j written out here from the definition; (iii) flat s_j split over three channels gives
    e_n = ceil(n n_bins / N); (iv) T matters: switching it on moves edges of a real template."""
    cfgd, cfg, f, S3, th, rng = _tiny(oracle, 3)
    n = len(f)
    h3 = oracle.template3(oracle.make_config(dict(cfgd, window_mode=0)), th)[:3]
    for N in (1, 2, 7, 40):
        e2 = oracle.equal_snr_edges(h3[0], h3[1], S3[0], S3[1], N)
        assert np.array_equal(oracle.equal_snr_edges3((h3[0], h3[1], None), S3, N), e2)
        # make T count: scale it up so that it carries a third of the total
        sA = np.abs(h3[0]) ** 2 / S3[0] + np.abs(h3[1]) ** 2 / S3[1]
        sT = np.abs(h3[2]) ** 2 / S3[2]
        g = np.sqrt(0.5 * sA.sum() / sT.sum())
        hT = g * h3[2] * (1.0 + 0.5 * np.sin(np.arange(n) / 7.0))          # and give it a shape of its own
        e3 = oracle.equal_snr_edges3((h3[0], h3[1], hT), S3, N)
        s = sA + np.abs(hT) ** 2 / S3[2]
        cum = np.concatenate([[0.0], np.cumsum(s)])
        C = cum[-1]
        assert e3[0] == 0 and e3[-1] == n and np.all(np.diff(e3) >= 0)
        for k in range(1, N):
            j = e3[k]
            assert cum[j] >= C * k / N * (1 - 1e-12) and (j == 0 or cum[j - 1] < C * k / N * (1 + 1e-12))
        if N == 40:
            assert not np.array_equal(e3, e2)
    ones = np.ones(n, dtype=complex)
    for N in (3, 10):
        e = oracle.equal_snr_edges3((ones, 2 * ones, 3 * ones), (np.ones(n), np.ones(n), np.ones(n)), N)
        assert np.array_equal(e[1:-1], np.ceil(np.arange(1, N) * n / N).astype(np.int64))


def test_eval_stat_adaptive3_composition_and_identities(oracle):
    cfgd, cfg, f, S3, th, rng = _tiny(oracle, 4)
    df = 1.0 / cfgd["T_obs_s"]
    n = len(f)
    h3 = oracle.template3(cfg, th)[:3]
    d3 = [h + np.sqrt(S / (4 * df)) * (rng.standard_normal(n) + 1j * rng.standard_normal(n)) for h, S in zip(h3, S3)]
    P = np.vstack([th, th * np.array([1.001, 1, 1, 1.1, 1, 1, 1, 1])])
    for N in (1, 6):
        out, ed, comp = oracle.eval_stat_adaptive3(cfg, d3, S3, P, N, want_edges=True, want_comp=True)
        for p in range(2):
            g3 = oracle.template3(cfg, P[p])[:3]
            e = oracle.equal_snr_edges3(g3, S3, N)
            assert np.array_equal(ed[p], e)
            u, seg = oracle.stat_from_arrays3(d3, g3, S3, df, e, want_seg=True)
            assert out[p] == u and np.array_equal(comp[p], oracle.components_from_seg(seg, df))
        # given edges override the choice: the shared equal-width list reproduces sco_eval_stat3
        sh = sy.edges(n, N)
        assert np.array_equal(oracle.eval_stat_adaptive3(cfg, d3, S3, P, N, in_edges=np.tile(sh, (2, 1))), oracle.eval_stat3(cfg, d3, S3, P, sh))
    # d = h over three channels: rho^2 on its own equal-SNR^2 edges, whatever N
    rho2 = oracle.inner3(h3, h3, S3, df)
    for N in (1, 5, 30):
        assert oracle.eval_stat_adaptive3(cfg, h3, S3, th[None, :], N)[0] == pytest.approx(rho2, rel=1e-12)
