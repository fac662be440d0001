"""Pins for the oracle's "truth" mode (sco_phase_ld, sco_tf_ld, sco_config.truth_mode) and for sco_eval_stat_levels.

SURVEY.md 7 step 1 / 8(c) O1: an optional long-double phase mode for the corner where the FP64 rounding of a 1e7-rad phase
(3e-9 rad per bin) is the larger error -- N = 1 at small Upsilon.  The long-double
functions restate O2 / O3 line for line, so the pins are (i) the ones that pin the FP64 functions, run on them: Newtonian
closed form, the published TaylorT2 timing series through 3.5PN, the finite-difference identity t = Psi'/2pi; (ii) the
PRECISION claim: agreement with a 40-digit evaluation to 1e-11 rad where the FP64 function is off by ~1e-9 rad, and the
exactly representable part 2 pi f t_c against rational arithmetic; (iii) the statistic in truth mode against the FP64 mode
to the predicted size of the FP64 rounding effect.
"""
from fractions import Fraction

import mpmath as mp
import numpy as np
import pytest

import sc_synth as sy

MS = sy.MSUN_S


def _cfg(oracle, pn=7, ecc=0, f_ref=0.018, T=4.0, truth=False):
    return oracle.make_config(sy.grid_config(T, 0.017, 0.030, pn_order_x2=pn, ecc_leading=ecc, f_ref_ecc=f_ref), truth=truth)


def _theta(Mc=30.0, eta=0.2469, tc=1.2e8, e0=0.0):
    return np.array([Mc, eta, tc, 1.0, 0.3, 0.5, -0.4, e0])


def test_tf_truth_newtonian_and_taylorT2(oracle):
    """As test_oracle_waveform: t_c - t(f) = tau_0 [1 + TaylorT2 series through 3.5PN] (its own published coefficients)."""
    gam = 0.5772156649015329
    for pn, terms in ((0, 0), (2, 1), (3, 2), (4, 3), (5, 4), (6, 5), (7, 6)):
        cfg = _cfg(oracle, pn=pn)
        for Mc, eta in ((25.0, 0.21), (36.0, 0.25), (30.0, 0.2469)):
            th = _theta(Mc, eta, tc=0.0)
            for j in (cfg.j0 + 5, cfg.j0 + 700001, cfg.j0 + cfg.n_bins - 1):
                f = j / cfg.T_obs_s
                v = (np.pi * Mc * MS * eta ** -0.6 * f) ** (1.0 / 3.0)
                ser = [(743.0 / 252.0 + 11.0 * eta / 3.0) * v ** 2, -(32.0 * np.pi / 5.0) * v ** 3,
                       (3058673.0 / 508032.0 + 5429.0 * eta / 504.0 + 617.0 * eta ** 2 / 72.0) * v ** 4,
                       -(7729.0 / 252.0 - 13.0 * eta / 3.0) * np.pi * v ** 5,
                       (-10052469856691.0 / 23471078400.0 + 128.0 * np.pi ** 2 / 3.0 + 6848.0 * gam / 105.0
                        + (3147553127.0 / 3048192.0 - 451.0 * np.pi ** 2 / 12.0) * eta - 15211.0 * eta ** 2 / 1728.0
                        + 25565.0 * eta ** 3 / 1296.0 + 3424.0 / 105.0 * np.log(16.0 * v * v)) * v ** 6,
                       (-15419335.0 / 127008.0 - 75703.0 * eta / 756.0 + 14809.0 * eta ** 2 / 378.0) * np.pi * v ** 7]
                tau0 = 5.0 / 256.0 * (Mc * MS) ** (-5.0 / 3.0) * (np.pi * f) ** (-8.0 / 3.0)
                assert -oracle.tf_truth(cfg, th, j) == pytest.approx(tau0 * (1.0 + sum(ser[:terms])), rel=1e-11)


@pytest.mark.parametrize("pn,ecc", [(0, 0), (5, 0), (6, 0), (7, 0), (7, 1)])
def test_tf_truth_is_phase_derivative(oracle, pn, ecc):
    """t(f) = Psi'(f)/2pi by 4th-order central differences over whole bins of the long-double phase (hi + lo parts)."""
    cfg = _cfg(oracle, pn=pn, ecc=ecc, f_ref=0.017)
    th = _theta(28.0, 0.24, tc=0.0, e0=0.08)
    k = 128                                             # step of 128 bins = 1.0e-6 Hz on the 4-yr grid
    h = k / cfg.T_obs_s
    for j in (cfg.j0 + 2 * k, cfg.j0 + 400000, cfg.j0 + cfg.n_bins - 2 * k - 1):
        P = lambda jj: mp.mpf(float(oracle.phase_truth(cfg, th, jj)[0])) + mp.mpf(float(oracle.phase_truth(cfg, th, jj)[1]))
        num = (-P(j + 2 * k) + 8 * P(j + k) - 8 * P(j - k) + P(j - 2 * k)) / (12 * h) / (2 * mp.pi)
        assert oracle.tf_truth(cfg, th, j) == pytest.approx(float(num), rel=1e-10)


def _psi_mp(cfg, th, j):
    """40-digit evaluation of O2 (3.5PN, optional leading eccentric term) at f = j / T_obs: a PRECISION reference for the
    long-double code (the formula itself is pinned by the timing series and the finite-difference identity above)."""
    mp.mp.dps = 40
    f = mp.mpf(int(j)) / mp.mpf(float(cfg.T_obs_s))
    Mc, eta, tc, e0 = mp.mpf(float(th[0])) * mp.mpf(MS), mp.mpf(float(th[1])), mp.mpf(float(th[2])), mp.mpf(float(th[7]))
    M = Mc * eta ** mp.mpf("-0.6")
    v = mp.cbrt(mp.pi * M * f)
    g = mp.euler
    psi = [1, 0, mp.mpf(3715) / 756 + 55 * eta / 9, -16 * mp.pi,
           mp.mpf(15293365) / 508032 + 27145 * eta / 504 + 3085 * eta ** 2 / 72,
           mp.pi * (mp.mpf(38645) / 756 - 65 * eta / 9) * (1 + 3 * mp.log(v)),
           mp.mpf(11583231236531) / 4694215680 - 640 * mp.pi ** 2 / 3 - 6848 * g / 21 - mp.mpf(6848) / 21 * mp.log(4 * v)
           + (-mp.mpf(15737765635) / 3048192 + 2255 * mp.pi ** 2 / 12) * eta + 76055 * eta ** 2 / 1728 - 127825 * eta ** 3 / 1296,
           mp.pi * (mp.mpf(77096675) / 254016 + 378515 * eta / 1512 - 74045 * eta ** 2 / 756)]
    s = sum(psi[k] * v ** (k - 5) for k in range(cfg.pn_order_x2 + 1))
    Psi = 2 * mp.pi * f * tc - mp.pi / 4 + 3 / (128 * eta) * s
    if cfg.ecc_leading:
        vref = mp.cbrt(mp.pi * M * mp.mpf(float(cfg.f_ref_ecc)))
        Psi += -3 / (128 * eta) * v ** -5 * (mp.mpf(2355) / 1462) * e0 ** 2 * (vref / v) ** (mp.mpf(19) / 3)
    return Psi


def test_phase_truth_precision(oracle):
    """Long double holds a 2e7-rad phase to < 2e-11 rad (the FP64 function is off by up to ~1e-8 rad there): the claim
    the truth mode exists for.  Also cos/sin of the long-double phase."""
    worst_ld, worst_64 = 0.0, 0.0
    for ecc in (0, 1):
        cfg = _cfg(oracle, ecc=ecc, f_ref=0.017)
        for Mc, eta, tc in ((30.0, 0.2469, 1.2e8), (21.0, 0.23, 1.6e8), (39.0, 0.2495, 0.9e8)):
            th = _theta(Mc, eta, tc, e0=0.05 * ecc)
            for j in np.linspace(cfg.j0, cfg.j0 + cfg.n_bins - 1, 23).astype(np.int64):
                ref = _psi_mp(cfg, th, j)
                hi, lo, c, s = oracle.phase_truth(cfg, th, j)
                err_ld = abs(float(mp.mpf(float(hi)) + mp.mpf(float(lo)) - ref))
                err_64 = abs(float(mp.mpf(oracle.phase(cfg, th, float(j) / cfg.T_obs_s)) - ref))
                worst_ld, worst_64 = max(worst_ld, err_ld), max(worst_64, err_64)
                assert abs(c - float(mp.cos(ref))) < 3e-11 and abs(s - float(mp.sin(ref))) < 3e-11
    assert worst_ld < 2e-11, worst_ld
    assert 5e-10 < worst_64 < 5e-8, worst_64          # the FP64 rounding the truth mode removes (3e-9 rad typical)


def test_f_tc_term_exact(oracle):
    """pn_order 0 with an enormous chirp mass leaves Psi = 2 pi f t_c - pi/4 + (tiny): the f t_c product against exact
    rational arithmetic on the doubles that enter (T_obs, t_c) and the integer bin index."""
    cfg = _cfg(oracle, pn=0)
    th = _theta(Mc=1e12, eta=0.25, tc=123456789.125)
    for j in (cfg.j0, cfg.j0 + 999983, cfg.j0 + cfg.n_bins - 1):
        turns = Fraction(int(j)) * Fraction(float(th[2])) / Fraction(float(cfg.T_obs_s))      # f t_c, exact
        frac = float(turns - int(turns))
        hi, lo, c, s = oracle.phase_truth(cfg, th, j)
        v = (np.pi * th[0] * MS * 0.25 ** -0.6 * j / cfg.T_obs_s) ** (1.0 / 3.0)
        rest = -np.pi / 4 + 3.0 / (128 * 0.25) * v ** -5.0                                   # ~ -pi/4 + 1e-17
        assert c == pytest.approx(np.cos(2 * np.pi * frac + rest), abs=2e-11)
        assert s == pytest.approx(np.sin(2 * np.pi * frac + rest), abs=2e-11)


def test_truth_mode_statistic_differs_by_the_fp64_phase_rounding(oracle):
    """Upsilon_N in truth mode vs FP64 mode on the c2 grid (1 yr: phases ~5e6 rad, FP64 rounding ~1e-9 rad per bin): the two
    agree to a few 1e-9/sqrt(Upsilon) (independent per-bin phase errors eps change Upsilon by ~2.8 eps/sqrt(Upsilon),
    DESIGN.md "Error model"), are not identical, and the window (decided in FP64 in both modes) is the same."""
    inp = sy.config_inputs(2, P=6)
    c64, cld = oracle.make_config(inp["cfg"]), oracle.make_config(inp["cfg"], truth=True)
    dA, dE = inp["noise_A"], inp["noise_E"]
    e = sy.edges(inp["cfg"]["n_bins"], 1)
    a, wa = oracle.eval_stat(c64, dA, dE, inp["S_A"], inp["S_E"], inp["particles"], e, want_inwin=True)
    b, wb = oracle.eval_stat(cld, dA, dE, inp["S_A"], inp["S_E"], inp["particles"], e, want_inwin=True)
    assert np.array_equal(wa, wb)
    ok = a > 0
    rel = np.abs(a - b)[ok] / b[ok] * np.sqrt(b[ok])
    assert rel.max() < 3e-8 and rel.max() > 1e-12, rel


def test_eval_stat_levels_equals_eval_stat_and_numpy(oracle):
    """sco_eval_stat_levels (the reference of the c2-c5 parity tests): level by level it is sco_eval_stat on that edge
    list (lists of different lengths, incl. partial coverage and empty segments), and both equal a numpy bin sum of
    Eq. 7/10 over the oracle's template."""
    inp = sy.config_inputs(1, P=5)
    cfg = oracle.make_config(inp["cfg"])
    nb = inp["cfg"]["n_bins"]
    rng = np.random.default_rng(7)
    ragged = np.sort(rng.integers(100, nb - 100, size=38)).astype(np.int64)
    ragged[5] = ragged[4]                                                    # an empty segment
    lists = [sy.edges(nb, 1), sy.edges(nb, 7), sy.edges(nb, 1000), ragged, sy.edges(nb, 64)]
    dA = inp["noise_A"] + 0.3 * oracle.template(cfg, inp["particles"][0])[0]
    dE = inp["noise_E"]
    lev = oracle.eval_stat_levels(cfg, dA, dE, inp["S_A"], inp["S_E"], inp["particles"], lists)
    assert lev.shape == (len(lists), 5)
    for l, e in enumerate(lists):
        one = oracle.eval_stat(cfg, dA, dE, inp["S_A"], inp["S_E"], inp["particles"], e)
        assert np.array_equal(lev[l], one)
    for p in range(5):
        hA, hE, _ = oracle.template(cfg, inp["particles"][p])
        zj = dA * np.conj(hA) / inp["S_A"] + dE * np.conj(hE) / inp["S_E"]
        sj = np.abs(hA) ** 2 / inp["S_A"] + np.abs(hE) ** 2 / inp["S_E"]
        for l, e in enumerate(lists):
            ups = 0.0
            for k in range(len(e) - 1):
                z, sg = zj[e[k]:e[k + 1]].sum(), sj[e[k]:e[k + 1]].sum()
                if sg > 0:
                    ups += abs(z) ** 2 / sg
            assert lev[l, p] == pytest.approx(4.0 * inp["df"] * ups, rel=1e-10)
