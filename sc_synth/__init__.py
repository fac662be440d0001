"""Seeded synthetic inputs for the semi-coherent statistic (SURVEY.md 8(d) recipe).

This module serves BOTH the CPU oracle's tests and the CUDA path's tests / bench and therefore holds none of
the method's arithmetic: no waveform, no response, no inner product, no PSO update.  It only makes numbers that
are inputs to both sides: the FFT grid, the noise PSD (harness-side model, PAPER.md:245 -> SURVEY O5), Gaussian
noise (O6), parameter draws inside prior boxes shaped like the paper's tiles (Table I
PAPER.md:263-279), segment edges (Q2) and PSO hyper-parameters (Table IV).
Injected signals are added by the caller, who supplies the template arrays (tests: from oracle/; bench: from the
CUDA library's own sc_gen_template).

The paper uses only simulated data: no public dataset stands behind these inputs.
"""
import math

import numpy as np

MASTER_SEED = 240813170
YEAR_S = 31557600.0                     # Julian year (Q6)
C_M_S = 299792458.0
AU_S = 1.495978707e11 / C_M_S           # 499.004783836 s
ARM_L_S = 2.5e9 / C_M_S                 # 8.33910238 s
MSUN_S = 4.925491025543576e-06
MONTH_S = 30.0 * 86400.0                # Q14: the paper's "months" are 30-day months

STREAMS = {"noise": 1, "injection": 2, "particles": 3, "velocities": 4, "pso": 5}


def seed_for(stream, config_id, extra=0):
    return MASTER_SEED + STREAMS[stream] + 100 * int(config_id) + 1000003 * int(extra)


# ---------------------------------------------------------------------------------------------- grid
def grid_config(T_obs_yr, f_lo, f_hi, window_mode=1, pn_order_x2=7, ecc_leading=0, f_ref_ecc=None):
    """FFT grid f_j = (j0 + j)/T_obs, j0 = ceil(f_lo T_obs), last bin floor(f_hi T_obs) (SURVEY 8 grid table)."""
    T = T_obs_yr * YEAR_S
    j0 = int(math.ceil(f_lo * T - 1e-6))
    j1 = int(math.floor(f_hi * T + 1e-6))
    return {
        "T_obs_s": T, "j0": j0, "n_bins": j1 - j0 + 1, "n_channels": 2, "window_mode": window_mode,
        "pn_order_x2": pn_order_x2, "ecc_leading": ecc_leading,
        "f_ref_ecc": float(f_lo if f_ref_ecc is None else f_ref_ecc),
        "arm_L_s": ARM_L_S, "au_s": AU_S, "orbit_alpha0": 0.0, "orbit_lambda0": 0.0, "year_s": YEAR_S,
    }


def freqs(cfg):
    return (cfg["j0"] + np.arange(cfg["n_bins"], dtype=np.float64)) / cfg["T_obs_s"]


def edges(n_bins, n_seg):
    """Q2: shared integer edges e_k = floor(k n_bins / N), exact integer arithmetic; nested for nested N."""
    k = np.arange(n_seg + 1, dtype=object)
    return np.array([(int(kk) * int(n_bins)) // int(n_seg) for kk in k], dtype=np.int64)


# ---------------------------------------------------------------------------------------------- noise
def psd_AE(f):
    """O5: analytic instrumental PSD of the TDI-1 A/E channels (no confusion noise)."""
    f = np.asarray(f, dtype=np.float64)
    x = 2.0 * np.pi * f * ARM_L_S
    S_oms = (15e-12) ** 2 * (1.0 + (2e-3 / f) ** 4) * (2.0 * np.pi * f / C_M_S) ** 2
    S_acc = (3e-15) ** 2 * (1.0 + (0.4e-3 / f) ** 2) * (1.0 + (f / 8e-3) ** 4) / (2.0 * np.pi * f * C_M_S) ** 2
    return 8.0 * np.sin(x) ** 2 * (2.0 * S_acc * (3.0 + 2.0 * np.cos(x) + np.cos(2.0 * x)) + S_oms * (2.0 + np.cos(x)))


def psd_T(f):
    """The third TDI-1 channel T = (X + Y + Z)/sqrt(3), same link-noise model: S_T = S_X + 2 S_XY."""
    f = np.asarray(f, dtype=np.float64)
    x = 2.0 * np.pi * f * ARM_L_S
    S_oms = (15e-12) ** 2 * (1.0 + (2e-3 / f) ** 4) * (2.0 * np.pi * f / C_M_S) ** 2
    S_acc = (3e-15) ** 2 * (1.0 + (0.4e-3 / f) ** 2) * (1.0 + (f / 8e-3) ** 4) / (2.0 * np.pi * f * C_M_S) ** 2
    return 16.0 * np.sin(x) ** 2 * ((1.0 - np.cos(x)) * S_oms + 2.0 * (1.0 - np.cos(x)) ** 2 * S_acc)


def link_noise_sources(f):
    """(S_oms, S_acc) per link / test mass in fractional-frequency units: the two inputs of psd_AE and psd_T."""
    f = np.asarray(f, dtype=np.float64)
    S_oms = (15e-12) ** 2 * (1.0 + (2e-3 / f) ** 4) * (2.0 * np.pi * f / C_M_S) ** 2
    S_acc = (3e-15) ** 2 * (1.0 + (0.4e-3 / f) ** 2) * (1.0 + (f / 8e-3) ** 4) / (2.0 * np.pi * f * C_M_S) ** 2
    return S_oms, S_acc


def draw_noise(seed, S, df):
    """O6: Re n, Im n ~ N(0, S/(4 df)) independent per bin (so <n|h> ~ N(0, <h|h>))."""
    rng = np.random.default_rng(seed)
    sd = np.sqrt(np.asarray(S) / (4.0 * df))
    return sd * rng.standard_normal(len(sd)) + 1j * sd * rng.standard_normal(len(sd))


# ---------------------------------------------------------------------------------------------- parameters
# Upper end [s] of the t_c range each config's injections are drawn from, per (config, injection index): the time a chirp of
# the injection's M_c needs from the band's lower edge to coalescence, so that the track enters the band at t ~ 0 (SURVEY
# 8(d) recipe).  Tabulated numbers -- this module holds none of the method's arithmetic; a caller with another source
# (tests/test_gpu_fuzz.py) passes its own value to draw_injection.
TC_UPPER_S = {(1, 0): 100381200.86424167, (2, 0): 116909178.85339002, (3, 0): 142024571.46033856,
              (5, 0): 712395601.66902, (5, 1): 394859670.4492147}


def eta_of_q(q):
    return q / (1.0 + q) ** 2


def draw_sky(rng):
    lam = rng.uniform(0.0, 2.0 * np.pi)
    beta = math.asin(rng.uniform(-1.0, 1.0))
    iota = math.acos(rng.uniform(-1.0, 1.0))
    psi = rng.uniform(-np.pi, 0.0)                     # Table I range
    return lam, beta, iota, psi


def draw_injection(rng, Mc, q, tc_upper, e0=0.0):
    """theta = (M_c, eta, t_c, lambda, beta, iota, psi, e0); t_c ~ U[tc_upper - 0.25 yr, tc_upper] (the caller's bound)."""
    tau = float(tc_upper)
    tc = rng.uniform(tau - 0.25 * YEAR_S, tau)
    lam, beta, iota, psi = draw_sky(rng)
    return np.array([Mc, eta_of_q(q), tc, lam, beta, iota, psi, e0], dtype=np.float64)


def prior_box(Mc_c, tc_c, eta_lo=0.15, eta_hi=0.2495, e0_range=(0.0, 0.0), dMc=1.5, dtc=3.0 * MONTH_S,
              Mc_range=None, tc_range=None):
    """Tile-shaped box (PAPER.md:253 '~3 Msun x 6 months', Table I ranges for the rest) -> lo[8], hi[8]."""
    Mc_lo, Mc_hi = Mc_range if Mc_range else (Mc_c - dMc, Mc_c + dMc)
    tc_lo, tc_hi = tc_range if tc_range else (tc_c - dtc, tc_c + dtc)
    lo = np.array([Mc_lo, eta_lo, tc_lo, 0.0, -np.pi / 2, 0.0, -np.pi, e0_range[0]])
    hi = np.array([Mc_hi, eta_hi, tc_hi, 2 * np.pi, np.pi / 2, np.pi, 0.0, e0_range[1]])
    return lo, hi


def draw_particles(seed, n, lo, hi):
    rng = np.random.default_rng(seed)
    return lo + (hi - lo) * rng.random((n, 8))


def draw_velocities(seed, n, lo, hi):
    """Q9: v0 ~ U(-0.1, 0.1) (hi - lo)."""
    rng = np.random.default_rng(seed)
    return (hi - lo) * rng.uniform(-0.1, 0.1, (n, 8))


# Table IV; column order (M_c, eta, beta, lambda, iota, psi, f_low, e0) per Q12, re-ordered
# to the theta layout (M_c, eta, t_c, lambda, beta, iota, psi, e0).  The paper's eps^{f_low} has no t_c
# counterpart (Q3): the t_c clamp is left to the caller (0 here).
TABLE_IV = {
    100: dict(omega=0.5, phi_p=0.2, phi_g=0.3, eps=[0.1, 0.05, 0.0, 0.1, 0.1, 0.2, 0.1, 0.1]),
    50: dict(omega=0.5, phi_p=0.2, phi_g=0.4, eps=[0.01, 0.05, 0.0, 0.01, 0.01, 0.2, 0.1, 0.1]),
    10: dict(omega=0.3, phi_p=0.2, phi_g=0.5, eps=[0.001, 0.05, 0.0, 0.001, 0.001, 0.01, 0.1, 0.1]),
    1: dict(omega=0.72, phi_p=1.193, phi_g=1.193, eps=[0.0] * 8),
}

# ---------------------------------------------------------------------------------------------- configs
# BASELINE.json "configs" 0..4 == c1..c5 of SURVEY.md section 8.
CONFIGS = {
    1: dict(T_obs_yr=0.5, band=(0.018, 0.020), P=64, n_segs=[1000], n_swarms=1,
            inj=[dict(Mc=30.0, q=0.8, rho=20.0)]),
    2: dict(T_obs_yr=1.0, band=(0.017, 0.025), P=1024, n_segs=[10000, 1000, 100], n_swarms=1,
            inj=[dict(Mc=30.0, q=0.8, rho=17.0)]),
    3: dict(T_obs_yr=4.0, band=(0.017, 0.030), P=10000, n_segs=[5000], n_swarms=1,
            inj=[dict(Mc=(20.0, 40.0), q=(0.5, 1.0), rho=17.0)],
            pso=dict(omega=0.7, phi_p=1.5, phi_g=1.5, eps=[0.0] * 8, iters=100)),
    4: dict(T_obs_yr=4.0, band=(0.017, 0.030), P=10000, n_segs=[50000, 5000, 500], n_swarms=1,
            inj=[], box=dict(Mc_range=(28.5, 31.5), tc_range=(3.2 * YEAR_S, 3.7 * YEAR_S)),
            pso=dict(omega=0.7, phi_p=1.5, phi_g=1.5, eps=[0.0] * 8, iters=200)),
    5: dict(T_obs_yr=4.0, band=(0.010, 0.040), P=40000, n_segs=[50000, 5000, 500, 50, 1], n_swarms=4,
            inj=[dict(Mc=(20.0, 40.0), q=(0.5, 1.0), rho=25.0), dict(Mc=(20.0, 40.0), q=(0.5, 1.0), rho=17.0)]),
}


def config_inputs(config_id, P=None, replica=0):
    """Everything about config c<id> that does not need a template: grid, PSD, noise, injection parameters
    (un-scaled), prior box, particles, velocities, edge lists.  The caller adds kappa*h(theta_inj) to 'noise'.
    replica > 0 draws an independent noise realisation and population (other GPUs / repeated noise seeds, config 4)."""
    spec = CONFIGS[config_id]
    f_lo, f_hi = spec["band"]
    cfg = grid_config(spec["T_obs_yr"], f_lo, f_hi)
    f = freqs(cfg)
    S = psd_AE(f)
    df = 1.0 / cfg["T_obs_s"]
    nA = draw_noise(seed_for("noise", config_id, 2 * replica), S, df)
    nE = draw_noise(seed_for("noise", config_id, 2 * replica + 1), S, df)
    rng = np.random.default_rng(seed_for("injection", config_id))
    injections = []
    for i, s in enumerate(spec["inj"]):
        Mc = s["Mc"] if not isinstance(s["Mc"], tuple) else rng.uniform(*s["Mc"])
        q = s["q"] if not isinstance(s["q"], tuple) else rng.uniform(*s["q"])
        injections.append(dict(theta=draw_injection(rng, Mc, q, TC_UPPER_S[(config_id, i)]), rho=s["rho"]))
    if "box" in spec:
        lo, hi = prior_box(0.0, 0.0, **spec["box"])
    else:
        th0 = injections[0]["theta"]
        eta_lo = 0.15 if config_id <= 2 else eta_of_q(0.5)
        lo, hi = prior_box(th0[0], th0[2], eta_lo=eta_lo)
    n = spec["P"] if P is None else P
    return dict(id=config_id, spec=spec, cfg=cfg, f=f, S_A=S, S_E=S.copy(), df=df, noise_A=nA, noise_E=nE,
                injections=injections, lo=lo, hi=hi,
                particles=draw_particles(seed_for("particles", config_id, replica), max(spec["P"], n), lo, hi)[:n].copy(),
                velocities=draw_velocities(seed_for("velocities", config_id, replica), max(spec["P"], n), lo, hi)[:n].copy(),
                edges={N: edges(cfg["n_bins"], N) for N in spec["n_segs"]},
                pso_seed=seed_for("pso", config_id, replica))
