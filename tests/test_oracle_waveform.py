"""Pins for the oracle's phase and time-frequency map (sco_phase, sco_tf) -- SURVEY.md 8(c) O2/O3.

The paper names TaylorF2Ecc [49] and prints no formula, so the pins are: the Newtonian closed
forms, the textbook TaylorT2 time-to-coalescence through 3.5PN (an independently stated series with its own
coefficients), the t_c values the paper prints in Tables I and III, the SPA identity t(f) = Psi'(f)/2pi by finite
differences, and the GW cycle count.  The leading eccentric coefficient is pinned by Peters' small-e equations.  The constant part
of psi_5 (degenerate with phi_c, irrelevant to Upsilon) and parity with the LALSimulation / TaylorF2Ecc code stay UNPINNED.
"""
import json
import os

import numpy as np
import pytest

import sc_synth as sy

GOLD = json.load(open(os.path.join(os.path.dirname(__file__), "golden", "paper_values.json")))
MS = sy.MSUN_S


def _cfg(oracle, pn=7, ecc=0, f_ref=0.018):
    return oracle.make_config(sy.grid_config(1.0, 0.017, 0.025, pn_order_x2=pn, ecc_leading=ecc, f_ref_ecc=f_ref))


def _theta(Mc=30.0, eta=0.2469, tc=1.0e8, e0=0.0):
    return np.array([Mc, eta, tc, 1.0, 0.3, 0.5, -0.4, e0])


def test_tf_newtonian_closed_form(oracle):
    """pn_order 0: t_c - t(f) = (5/256) M_c^(-5/3) (pi f)^(-8/3)."""
    cfg = _cfg(oracle, pn=0)
    for Mc, eta in ((20.0, 0.2), (30.0, 0.2469), (95.0, 0.234)):
        th = _theta(Mc, eta, tc=2.0e8)
        for f in (0.010, 0.0175, 0.03, 0.04):
            tau = 5.0 / 256.0 * (Mc * MS) ** (-5.0 / 3.0) * (np.pi * f) ** (-8.0 / 3.0)
            assert th[2] - oracle.tf(cfg, th, f) == pytest.approx(tau, rel=1e-12)


def test_tf_taylorT2_series_through_2pn(oracle):
    """Textbook TaylorT2 time: t_c - t = tau_0 [1 + (743/252 + 11 eta/3) v^2 - (32 pi/5) v^3
    + (3058673/508032 + 5429 eta/504 + 617 eta^2/72) v^4]; pins psi_2, psi_3, psi_4 and the derivative rule."""
    for pn, terms in ((2, 1), (3, 2), (4, 3)):
        cfg = _cfg(oracle, pn=pn)
        for Mc, eta in ((25.0, 0.21), (36.0, 0.25)):
            th = _theta(Mc, eta, tc=0.0)
            for f in (0.012, 0.02, 0.035):
                M = Mc * MS * eta ** -0.6
                v = (np.pi * M * f) ** (1.0 / 3.0)
                series = [(743.0 / 252.0 + 11.0 * eta / 3.0) * v ** 2, -(32.0 * np.pi / 5.0) * v ** 3,
                          (3058673.0 / 508032.0 + 5429.0 * eta / 504.0 + 617.0 * eta ** 2 / 72.0) * v ** 4]
                tau0 = 5.0 / 256.0 * (Mc * MS) ** (-5.0 / 3.0) * (np.pi * f) ** (-8.0 / 3.0)
                assert -oracle.tf(cfg, th, f) == pytest.approx(tau0 * (1.0 + sum(series[:terms])), rel=1e-12)


def test_tf_taylorT2_series_2p5_to_3p5pn(oracle):
    """The same published TaylorT2 timing series continued to 3.5PN (its own rational coefficients, not those of the
    TaylorF2 phase): -(7729/252 - 13 eta/3) pi v^5, the 3PN term with 128 pi^2/3, 6848 gamma_E/105 and
    (3424/105) ln(16 v^2), and the 3.5PN term.  Pins psi_5's logarithm, psi_6 (every eta power, the Euler-gamma and log
    terms) and psi_7 through t = Psi'/2pi -- a wrong digit in any of them moves t(f) by >> 1e-10 relative."""
    gam = 0.5772156649015329
    for pn, terms in ((5, 1), (6, 2), (7, 3)):
        cfg = _cfg(oracle, pn=pn)
        for Mc, eta in ((25.0, 0.21), (36.0, 0.25), (30.0, 0.2469)):
            th = _theta(Mc, eta, tc=0.0)
            for f in (0.012, 0.02, 0.035):
                M = Mc * MS * eta ** -0.6
                v = (np.pi * M * f) ** (1.0 / 3.0)
                low = ((743.0 / 252.0 + 11.0 * eta / 3.0) * v ** 2 - (32.0 * np.pi / 5.0) * v ** 3
                       + (3058673.0 / 508032.0 + 5429.0 * eta / 504.0 + 617.0 * eta ** 2 / 72.0) * v ** 4)
                high = [-(7729.0 / 252.0 - 13.0 * eta / 3.0) * np.pi * v ** 5,
                        (-10052469856691.0 / 23471078400.0 + 128.0 * np.pi ** 2 / 3.0 + 6848.0 * gam / 105.0
                         + (3147553127.0 / 3048192.0 - 451.0 * np.pi ** 2 / 12.0) * eta - 15211.0 * eta ** 2 / 1728.0
                         + 25565.0 * eta ** 3 / 1296.0 + 3424.0 / 105.0 * np.log(16.0 * v * v)) * v ** 6,
                        (-15419335.0 / 127008.0 - 75703.0 * eta / 756.0 + 14809.0 * eta ** 2 / 378.0) * np.pi * v ** 7]
                tau0 = 5.0 / 256.0 * (Mc * MS) ** (-5.0 / 3.0) * (np.pi * f) ** (-8.0 / 3.0)
                assert -oracle.tf(cfg, th, f) == pytest.approx(tau0 * (1.0 + low + sum(high[:terms])), rel=1e-11)


@pytest.mark.parametrize("table", ["table_I", "table_III"])
def test_paper_tc_values(oracle, table):
    """Tables I / III: t_c [30-day months, Q14] of the source that enters at f_low at t = 0."""
    g = GOLD[table]
    month = GOLD["month_convention"]["month_s"]
    for ecc in (0, 1):
        cfg = _cfg(oracle, pn=7, ecc=ecc, f_ref=g["f_low_hz"])
        th = np.array([g["Mc_msun"], g["eta"], 0.0, g["lambda"], g["beta"], g["iota"], g["psi"], g["e0"]])
        tc = -oracle.tf(cfg, th, g["f_low_hz"])            # t(f_low) = 0  <=>  t_c = -t(f_low)|_{t_c = 0}
        assert tc / month == pytest.approx(g["tc_months"], rel=5e-3)


@pytest.mark.parametrize("pn,ecc", [(0, 0), (2, 0), (5, 0), (6, 0), (7, 0), (7, 1)])
def test_tf_is_phase_derivative(oracle, pn, ecc):
    """O3 identity t(f) = (1/2pi) dPsi/df by 4th-order central differences (pins every derivative term incl. the log
    terms).  t_c = 0 keeps Psi ~ 1e7 rad so the FP64 difference quotient is good to ~1e-11."""
    cfg = _cfg(oracle, pn=pn, ecc=ecc, f_ref=0.017)
    th = _theta(28.0, 0.24, tc=0.0, e0=0.08)
    for f in (0.011, 0.0175, 0.022, 0.039):
        h = 4e-6
        P = lambda x: oracle.phase(cfg, th, x)
        num = (-P(f + 2 * h) + 8 * P(f + h) - 8 * P(f - h) + P(f - 2 * h)) / (12 * h) / (2 * np.pi)   # 4th order
        assert oracle.tf(cfg, th, f) == pytest.approx(num, rel=1e-9)
    # and the t_c term
    th2 = th.copy()
    th2[2] = 12345.678
    assert oracle.tf(cfg, th2, 0.02) - oracle.tf(cfg, th, 0.02) == pytest.approx(12345.678, rel=1e-9)
    assert oracle.phase(cfg, th2, 0.02) - oracle.phase(cfg, th, 0.02) == pytest.approx(2 * np.pi * 0.02 * 12345.678, rel=1e-7)


def test_newtonian_cycle_count(oracle):
    """SPA: Psi(f) = 2 pi f t(f) - phi(t(f)) - pi/4, so the GW phase accumulated between f_lo and f_hi,
    [2 pi f t(f) - Psi(f)]_lo^hi / 2pi, must equal the Newtonian cycle count
    (1/(32 pi^(8/3))) M_c^(-5/3) (f_lo^(-5/3) - f_hi^(-5/3))   (1.95e6 for 30 Msun over 0.017-0.030 Hz).
    Pins the sign and the 3/(128 eta) v^-5 normalisation of the phase."""
    cfg = _cfg(oracle, pn=0)
    for Mc in (20.0, 30.0, 40.0):
        th = _theta(Mc, 0.2469, tc=1.1e8)
        acc = lambda f: 2 * np.pi * f * oracle.tf(cfg, th, f) - oracle.phase(cfg, th, f)
        ncyc = (acc(0.030) - acc(0.017)) / (2 * np.pi)
        closed = (Mc * MS) ** (-5.0 / 3.0) / (32 * np.pi ** (8.0 / 3.0)) * (0.017 ** (-5.0 / 3.0) - 0.030 ** (-5.0 / 3.0))
        assert ncyc == pytest.approx(closed, rel=1e-8)
        if Mc == 30.0:
            assert closed == pytest.approx(1.95e6, rel=5e-3)


def test_tf_monotone_in_band(oracle):
    """t(f) increases with f over every config band (needed by the Q4 window)."""
    cfg = _cfg(oracle)
    for Mc, eta in ((18.5, 0.15), (30.0, 0.2495), (41.5, 0.2222)):
        th = _theta(Mc, eta, tc=1.0e8)
        t = np.array([oracle.tf(cfg, th, f) for f in np.linspace(0.010, 0.040, 400)])
        assert np.all(np.diff(t) > 0)


def test_eccentric_term_scaling(oracle):
    """Q5: the e0^2 term is quadratic in e0, vanishes at e0 = 0, scales as f^(-34/9) and is NEGATIVE relative to the
    Newtonian term with ratio -(2355/1462) e0^2 at f = f_ref."""
    c0 = _cfg(oracle, pn=0, ecc=0, f_ref=0.02)
    c1 = _cfg(oracle, pn=0, ecc=1, f_ref=0.02)
    base = lambda f: oracle.phase(c0, _theta(tc=0.0), f) + np.pi / 4
    d = lambda e0, f: oracle.phase(c1, _theta(tc=0.0, e0=e0), f) - oracle.phase(c0, _theta(tc=0.0, e0=e0), f)
    assert d(0.0, 0.02) == 0.0
    assert d(0.1, 0.02) / d(0.05, 0.02) == pytest.approx(4.0, rel=1e-6)
    assert d(0.1, 0.02) / base(0.02) == pytest.approx(-(2355.0 / 1462.0) * 0.01, rel=1e-6)
    assert d(0.1, 0.03) / d(0.1, 0.02) == pytest.approx(1.5 ** (-34.0 / 9.0), rel=1e-6)


def test_eccentric_coefficient_from_peters_equations(oracle):
    """Pins 2355/1462 from quantities it is not written in: at small e Peters' equations give e = e_0 (f/f_ref)^(-19/18)
    and df/dt = (96/5) pi^(8/3) M_c^(5/3) f^(11/3) (1 + 157 e^2/24); integrating dt = df/(df/dt) from f to infinity,
    t_c - t(f) = tau_0(f) [1 - (157/43) e(f)^2]   (157/24 x (8/3)/(8/3 + 19/9) = 157/43).
    The oracle gets t(f) from its phase term by t = Psi'/2pi; both must agree at Newtonian order."""
    f_ref = 0.0175
    cfg = _cfg(oracle, pn=0, ecc=1, f_ref=f_ref)
    for Mc, eta, e0 in ((30.0, 0.2469, 0.1), (22.0, 0.23, 0.03)):
        th = _theta(Mc, eta, tc=0.0, e0=e0)
        for f in (0.012, 0.0175, 0.03):
            tau0 = 5.0 / 256.0 * (Mc * MS) ** (-5.0 / 3.0) * (np.pi * f) ** (-8.0 / 3.0)
            e2 = e0 ** 2 * (f / f_ref) ** (-19.0 / 9.0)
            assert -oracle.tf(cfg, th, f) == pytest.approx(tau0 * (1.0 - 157.0 / 43.0 * e2), rel=1e-12)


def test_invalid_theta_gives_zero_template(oracle):
    cfg = oracle.make_config(sy.grid_config(0.01, 0.018, 0.0185))
    for bad in (dict(i=1, v=0.26), dict(i=1, v=0.0), dict(i=0, v=-3.0), dict(i=2, v=np.nan), dict(i=4, v=np.inf)):
        th = _theta(tc=3e5)
        th[bad["i"]] = bad["v"]
        hA, hE, w = oracle.template(cfg, th)
        assert w == 0 and not hA.any() and not hE.any()


def test_time_window_is_contiguous_and_matches_tf(oracle):
    """Q4: bins with 0 <= t(f_j) <= T_obs form one contiguous block; nothing else is non-zero."""
    inp = sy.config_inputs(1, P=4)
    cfg = oracle.make_config(inp["cfg"])
    th = inp["particles"][0]
    hA, hE, w = oracle.template(cfg, th)
    t = np.array([oracle.tf(cfg, th, f) for f in inp["f"][::97]])
    inside = (t >= 0) & (t <= cfg.T_obs_s)
    nz = (np.abs(hA) > 0)
    assert np.array_equal(nz[::97], inside)
    idx = np.nonzero(nz)[0]
    assert len(idx) == w and (w == 0 or idx[-1] - idx[0] + 1 == w)
    cfg0 = oracle.make_config(dict(inp["cfg"], window_mode=0))
    assert oracle.template(cfg0, th)[2] == cfg.n_bins
