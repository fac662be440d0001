"""Pins for the oracle's orbit / single-link / TDI response (sco_orbit, sco_link, sco_tdi, sco_template) -- O4.

The paper cites the BBHx implementation of [56] (Eq. 16) and prints no formula, so parity with
BBHx is UNPINNED.  What is pinned: orbit geometry, the two-pulse Doppler identity behind the single-link formula,
the long-wavelength (Michelson) limit built here from explicit 3x3 polarisation tensors, T -> 0 in that limit,
cyclic symmetry under relabelling the spacecraft, and the absence of a Doppler term at the ecliptic poles.
"""
import numpy as np
import pytest

import sc_synth as sy


def _cfg(oracle, **kw):
    d = sy.grid_config(1.0, 0.017, 0.025)
    d.update(kw)
    return oracle.make_config(d)


THETA = np.array([30.0, 0.2469, 1.0e8, 2.01, 0.6, 2.498, -1.85, 0.0])


def test_orbit_geometry(oracle):
    """Equal arms (= L to first order in e = L/(2 sqrt3 AU) ~ 0.0048) and centroid on the 1-AU circle (Q6)."""
    cfg = _cfg(oracle)
    for t in np.linspace(0, 4 * sy.YEAR_S, 23):
        p = oracle.orbit(cfg, t)
        a = 2 * np.pi * t / sy.YEAR_S
        assert np.allclose(p[0], sy.AU_S * np.array([np.cos(a), np.sin(a), 0.0]), rtol=0, atol=1e-9)
        assert np.allclose(p[1:].mean(axis=0), p[0], rtol=0, atol=1e-9)
        for i, j in ((1, 2), (2, 3), (3, 1)):
            assert np.linalg.norm(p[i] - p[j]) == pytest.approx(sy.ARM_L_S, rel=2e-5)
    # the constellation counter-rotates once per year: spacecraft n at t equals spacecraft n+1 a third of a year ... no;
    # what IS exact: lambda0 -> lambda0 + 2pi/3 relabels n -> n+1
    p = oracle.orbit(cfg, 1.234e7)
    q = oracle.orbit(_cfg(oracle, orbit_lambda0=2 * np.pi / 3), 1.234e7)
    assert np.allclose(q[1], p[2], atol=1e-9) and np.allclose(q[2], p[3], atol=1e-9) and np.allclose(q[3], p[1], atol=1e-9)


def _pol_tensors(theta):
    """explicit 3x3 polarisation tensors eps+, epsx for (lambda, beta, psi) -- built independently of the oracle."""
    lam, bet, psi = theta[3], theta[4], theta[6]
    n_hat = np.array([np.cos(bet) * np.cos(lam), np.cos(bet) * np.sin(lam), np.sin(bet)])
    k = -n_hat
    u = np.array([-np.sin(bet) * np.cos(lam), -np.sin(bet) * np.sin(lam), np.cos(bet)])
    v = np.cross(k, u)                          # right-handed (u, v, k)
    ep = np.outer(u, u) - np.outer(v, v)
    ex = np.outer(u, v) + np.outer(v, u)
    return k, np.cos(2 * psi) * ep + np.sin(2 * psi) * ex, -np.sin(2 * psi) * ep + np.cos(2 * psi) * ex


def _zeta(theta, n):
    k, Ep, Ex = _pol_tensors(theta)
    ci = np.cos(theta[5])
    return 0.5 * (1 + ci * ci) * (n @ Ep @ n) - 1j * ci * (n @ Ex @ n)


def test_single_link_two_pulse_identity(oracle):
    """y_sr = zeta [e^{-2 pi i f (L + k.p_s)} - e^{-2 pi i f k.p_r}] / (2 (1 - k.n))  (two-pulse Doppler response of a
    plane wave, emission at s delayed by L) -- equals the oracle's sinc form when |p_r - p_s| = L."""
    cfg = _cfg(oracle)
    rng = np.random.default_rng(2)
    for _ in range(12):
        th = THETA.copy()
        th[3], th[4], th[5], th[6] = rng.uniform(0, 6.28), rng.uniform(-1.5, 1.5), rng.uniform(0, 3.1), rng.uniform(-3.1, 0)
        f, t = rng.uniform(0.01, 0.04), rng.uniform(0, 1.2e8)
        s, r = rng.choice([1, 2, 3], size=2, replace=False)
        p = oracle.orbit(cfg, t)
        k, _, _ = _pol_tensors(th)
        n = (p[r] - p[s]) / np.linalg.norm(p[r] - p[s])
        L = sy.ARM_L_S
        # use the exact-arm geometry the sinc form assumes: p_r' = p_s + L n differs from p_r by ~1e-5 L
        mid = 0.5 * (p[r] + p[s])
        ps, pr = mid - 0.5 * L * n, mid + 0.5 * L * n
        two_pulse = _zeta(th, n) * (np.exp(-2j * np.pi * f * (L + k @ ps)) - np.exp(-2j * np.pi * f * (k @ pr))) / (2 * (1 - k @ n))
        got = oracle.link(cfg, th, f, t, s, r)
        assert got == pytest.approx(two_pulse, rel=1e-9)


def test_long_wavelength_michelson_limit_and_T_null(oracle):
    """f L -> 0:  X/(2 pi f L)^2 -> 2 (zeta_13 - zeta_12) e^{-2 pi i f k.p0}  (textbook Michelson response times the
    common Doppler factor); the T combination vanishes relative to A, E."""
    cfg = _cfg(oracle, arm_L_s=1e-4)          # shrink the arms: x = 2 pi f L ~ 1e-5
    f, t = 0.02, 3.3e7
    p = oracle.orbit(cfg, t)
    k, _, _ = _pol_tensors(THETA)
    n12 = (p[2] - p[1]) / np.linalg.norm(p[2] - p[1])
    n13 = (p[3] - p[1]) / np.linalg.norm(p[3] - p[1])
    tdi = oracle.tdi(cfg, THETA, f, t)
    x = 2 * np.pi * f * 1e-4
    want = 2 * (_zeta(THETA, n13) - _zeta(THETA, n12)) * np.exp(-2j * np.pi * f * (k @ p[0]))
    assert tdi["X"] / x ** 2 == pytest.approx(want, rel=1e-4)
    assert abs(tdi["T"]) < 1e-4 * max(abs(tdi["A"]), abs(tdi["E"]))
    # A, E, T are the stated combinations of X, Y, Z
    assert tdi["A"] == pytest.approx((tdi["Z"] - tdi["X"]) / np.sqrt(2), rel=1e-13)
    assert tdi["E"] == pytest.approx((tdi["X"] - 2 * tdi["Y"] + tdi["Z"]) / np.sqrt(6), rel=1e-13)
    assert tdi["T"] == pytest.approx((tdi["X"] + tdi["Y"] + tdi["Z"]) / np.sqrt(3), abs=1e-13 * abs(tdi["X"]))


def test_tdi_X_from_links(oracle):
    """X = (1 - D^2)[(y31 + D y13) - (y21 + D y12)], D = e^{-2 pi i f L} (TDI 1st generation, Q6), assembled here
    from the oracle's single links."""
    cfg = _cfg(oracle)
    f, t = 0.0234, 7.7e7
    y = {(s, r): oracle.link(cfg, THETA, f, t, s, r) for s in (1, 2, 3) for r in (1, 2, 3) if s != r}
    D = np.exp(-2j * np.pi * f * sy.ARM_L_S)
    tdi = oracle.tdi(cfg, THETA, f, t)
    assert tdi["X"] == pytest.approx((1 - D * D) * ((y[3, 1] + D * y[1, 3]) - (y[2, 1] + D * y[1, 2])), rel=1e-12)
    assert tdi["Y"] == pytest.approx((1 - D * D) * ((y[1, 2] + D * y[2, 1]) - (y[3, 2] + D * y[2, 3])), rel=1e-12)
    assert tdi["Z"] == pytest.approx((1 - D * D) * ((y[2, 3] + D * y[3, 2]) - (y[1, 3] + D * y[3, 1])), rel=1e-12)


def test_cyclic_symmetry(oracle):
    """Relabelling spacecraft 1->2->3->1 (lambda0 += 2pi/3) maps X->Y->Z->X."""
    cfg = _cfg(oracle)
    cfg2 = _cfg(oracle, orbit_lambda0=2 * np.pi / 3)
    a = oracle.tdi(cfg, THETA, 0.021, 5.0e7)
    b = oracle.tdi(cfg2, THETA, 0.021, 5.0e7)
    assert b["X"] == pytest.approx(a["Y"], rel=1e-10)
    assert b["Y"] == pytest.approx(a["Z"], rel=1e-10)
    assert b["Z"] == pytest.approx(a["X"], rel=1e-10)


def test_no_doppler_at_ecliptic_pole(oracle):
    """beta = +-pi/2  =>  k.p0 = 0: the link phase carries no 2 pi f AU term, so shifting the whole constellation
    by removing the centroid changes nothing.  Away from the pole the same phase swings by ~2 pi f AU = 63 rad."""
    cfg = _cfg(oracle)
    f = 0.02
    for beta in (np.pi / 2, -np.pi / 2):
        th = THETA.copy()
        th[4] = beta
        for t in (0.0, 1.1e7, 2.9e7):
            p = oracle.orbit(cfg, t)
            k, _, _ = _pol_tensors(th)
            assert abs(k @ p[0]) < 1e-10
            n = (p[2] - p[1]) / np.linalg.norm(p[2] - p[1])
            L = sy.ARM_L_S
            x = np.pi * f * L * (1 - k @ n)
            centred = -1j * np.pi * f * L * np.sin(x) / x * np.exp(-1j * np.pi * f * (L + k @ (p[1] + p[2] - 2 * p[0]))) * _zeta(th, n)
            assert oracle.link(cfg, th, f, t, 1, 2) == pytest.approx(centred, rel=1e-9)
    th = THETA.copy()
    th[4] = 0.0
    ph = [np.angle(oracle.link(cfg, th, f, t, 1, 2) / _zeta(th, (oracle.orbit(cfg, t)[2] - oracle.orbit(cfg, t)[1]) / sy.ARM_L_S))
          for t in np.linspace(0, sy.YEAR_S, 2000)]
    assert np.ptp(np.unwrap(ph)) == pytest.approx(2 * 2 * np.pi * f * sy.AU_S, rel=0.02)


def test_template_is_transfer_times_amplitude_times_phase(oracle):
    """Eq. 16: h_alpha(f_j) = T_alpha(f_j; t_f) f^(-7/6) e^{-i Psi(f_j)} at the bins inside the window."""
    inp = sy.config_inputs(1, P=2)
    cfg = oracle.make_config(inp["cfg"])
    th = inp["injections"][0]["theta"]
    hA, hE, w = oracle.template(cfg, th)
    assert w > 1000
    for j in np.nonzero(np.abs(hA) > 0)[0][:: max(1, w // 7)]:
        f = inp["f"][j]
        t = oracle.tf(cfg, th, f)
        tdi = oracle.tdi(cfg, th, f, t)
        carrier = f ** (-7.0 / 6.0) * np.exp(-1j * oracle.phase(cfg, th, f))
        assert hA[j] == pytest.approx(tdi["A"] * carrier, rel=1e-12)
        assert hE[j] == pytest.approx(tdi["E"] * carrier, rel=1e-12)
    # sub-range evaluation agrees with the full one
    hA2, hE2, _ = oracle.template(cfg, th, j_begin=12000, n=500)
    assert np.array_equal(hA2, hA[12000:12500]) and np.array_equal(hE2, hE[12000:12500])


def test_injection_at_snr_gives_rho_squared(oracle):
    """north_star pin: no noise, template at the injected parameters, N = 1: |<d|h>|^2/<h|h> = rho^2; and the same for
    every refinement.  Table V: max Upsilon_1 ~ rho^2 = 1444 at rho = 38."""
    inp = sy.config_inputs(1, P=2)
    cfg = oracle.make_config(inp["cfg"])
    th = inp["injections"][0]["theta"]
    hA, hE, _ = oracle.template(cfg, th)
    S, df = inp["S_A"], inp["df"]
    rho = 38.0
    kappa = rho / np.sqrt(oracle.inner(hA, hE, hA, hE, S, S, df))
    for N in (1, 10, 100, 1000):
        u = oracle.eval_stat(cfg, kappa * hA, kappa * hE, S, S, th[None, :], sy.edges(cfg.n_bins, N))
        assert u[0] == pytest.approx(rho ** 2, rel=1e-10)
    # with noise the value at theta_inj scatters around 2N + rho^2 with sd 2 sqrt(N + rho^2) (Eq. 12): N = 1
    vals = []
    for s in range(40):
        dA = kappa * hA + sy.draw_noise(900 + 2 * s, S, df)
        dE = kappa * hE + sy.draw_noise(901 + 2 * s, S, df)
        vals.append(oracle.stat_from_arrays(dA, dE, hA, hE, S, S, df, sy.edges(cfg.n_bins, 1)))
    assert np.mean(vals) == pytest.approx(2 + rho ** 2, abs=4 * 2 * np.sqrt(1 + rho ** 2) / np.sqrt(40))
    # the paper's four search maxima (1390..1450) sit within ~1 sd (2*38 = 76) of rho^2
    assert all(abs(v - rho ** 2) < 76 for v in [1450.1, 1390.3, 1422.3, 1434.1])
