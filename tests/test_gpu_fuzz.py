"""Randomised GPU-vs-oracle parity (all `-m gpu`): grids, tiles, populations and edge lists the named configs do not
visit -- odd bin counts, bands and observation times that give other node spacings, particles whose time windows
(Q4) lie partly or wholly outside the band, irregular / partial / repeated segment edges, populations that are not
a multiple of the 128-particle block.  Every particle is compared (<= 1e-6 relative, north_star, flat: the reference is the oracle's long-double truth mode);
inputs are seeded."""
import numpy as np
import pytest

import sc_synth as sy
from helpers import gpu_handle, make_data, rel_err

pytestmark = pytest.mark.gpu

TOL = 1e-6


def _case(seed):
    rng = np.random.default_rng(9000 + seed)
    T_yr = float(rng.choice([0.31, 0.5, 0.77, 1.0, 1.63]))
    f_lo = float(rng.uniform(0.012, 0.024))
    width = float(rng.uniform(0.0012, 0.004)) / T_yr ** 0.5
    cfg = sy.grid_config(T_yr, f_lo, f_lo + width)
    f = sy.freqs(cfg)
    S = sy.psd_AE(f)
    df = 1.0 / cfg["T_obs_s"]
    Mc, q = float(rng.uniform(18.0, 45.0)), float(rng.uniform(0.5, 1.0))
    # t_c such that the track enters the band near t = 0: Newtonian time to coalescence from f_lo (closed form of
    # test_oracle_waveform.test_tf_newtonian_closed_form)
    tau = 5.0 / 256.0 * (Mc * sy.MSUN_S) ** (-5.0 / 3.0) * (np.pi * f_lo) ** (-8.0 / 3.0)
    th = sy.draw_injection(rng, Mc, q, tau)
    # a tile around the source, wide enough in t_c that many windows start or end inside the band or miss it
    lo, hi = sy.prior_box(th[0], th[2], eta_lo=0.16, dMc=float(rng.uniform(0.2, 2.0)),
                          dtc=float(rng.uniform(0.2, 1.5)) * T_yr * sy.YEAR_S)
    P = int(rng.choice([131, 257, 300, 515]))
    parts = sy.draw_particles(int(rng.integers(1 << 30)), P, lo, hi)
    inp = dict(cfg=cfg, S_A=S, S_E=S.copy(), df=df, lo=lo, hi=hi, particles=parts,
               noise_A=sy.draw_noise(int(rng.integers(1 << 30)), S, df), noise_E=sy.draw_noise(int(rng.integers(1 << 30)), S, df),
               injections=[dict(theta=th, rho=float(rng.uniform(8.0, 30.0)))])
    nb = cfg["n_bins"]
    lists = [sy.edges(nb, 1), sy.edges(nb, int(rng.integers(2, 8))), sy.edges(nb, int(rng.integers(8, 64))),
             sy.edges(nb, int(rng.integers(64, 5000)))]
    # irregular edges covering part of the band, with repeated entries (empty segments)
    n_e = int(rng.integers(3, 400))
    a, b = sorted(rng.integers(0, nb + 1, size=2))
    irr = np.sort(rng.integers(a, b + 1, size=n_e)).astype(np.int64)
    lists.append(irr)
    return inp, lists


@pytest.mark.parametrize("seed", range(12))
def test_random_grids_tiles_and_edges(oracle, seed):
    import torch
    import paper_2408_13170_b200 as sc
    inp, lists = _case(seed)
    if oracle.template(oracle.make_config(inp["cfg"]), inp["injections"][0]["theta"])[2] == 0:
        inp["injections"] = []                      # the drawn source never enters this band within T_obs: noise only
    cfg, dA, dE = make_data(oracle, inp)
    H = gpu_handle(inp, dA, dE)
    if seed % 2:
        H.set_option(sc.SC_OPT_TC_MAX_S, int(np.ceil(max(inp["hi"][2], 1.0))))
    par = torch.from_numpy(inp["particles"]).to("cuda:0")
    # reference in the oracle's truth mode (long-double phase): Psi ~ 2 pi f t_c reaches 5e7 rad on these tiles, where the
    # FP64 oracle's own per-bin rounding (1.3e-8 rad rms) would exceed the bar for Upsilon << 1; with it the bar is flat
    cfg_truth = oracle.make_config(inp["cfg"], truth=True)
    ref = oracle.eval_stat_levels(cfg_truth, dA, dE, inp["S_A"], inp["S_E"], inp["particles"], lists)
    n_live = 0
    # second round: the caller states the measured window fraction (SC_OPT_WINDOW_FRACTION_PPM), which widens the node spacing of
    # the FP32-amplitude path with the number of segments -- on tiles whose windows partly leave the band, the hard case of that rule
    for hint in (False, True):
        if hint:
            H.eval_stat(par, lists[0].astype(np.int32))                      # whole band: evaluated bins = the windows
            phi = H.counters()[0] / (len(inp["particles"]) * inp["cfg"]["n_bins"])
            H.set_option(sc.SC_OPT_WINDOW_FRACTION_PPM, max(1, int(round(1e6 * phi))))
        for e, r in zip(lists, ref):
            got = H.eval_stat(par, e.astype(np.int32)).cpu().numpy()
            assert np.all(np.isfinite(got)) and np.all(got >= 0.0)
            assert np.array_equal(got == 0.0, r == 0.0), (seed, len(e))          # same particles see an empty window
            ok = r > 0
            n_live += int(ok.sum())
            if ok.any():
                err = rel_err(got[ok], r[ok])
                assert np.all(err <= TOL), (seed, hint, len(e), float(err.max()), float(r[ok][np.argmax(err)]))
    assert n_live > 0
    H.close()


@pytest.mark.parametrize("seed", range(5))
def test_wide_grids_with_node_spacing_hint_and_quadratic_runs(oracle, seed):
    """Multi-year grids (3.5e5 - 1.1e6 bins) where the window-fraction statement widens the node spacing (stride 512 - 2048) and
    the long segments switch the pair loop to its quadratic-amplitude runs (SC_FLAVOUR_QUAD): random tiles, random numbers of
    equal segments from 8 to n_bins/130 and one irregular edge list; a seeded sample of particles against the oracle's truth
    mode, flat 1e-6 bar."""
    import torch
    import paper_2408_13170_b200 as sc
    rng = np.random.default_rng(500 + seed)
    T_yr = float(rng.choice([2.0, 3.0, 4.0]))
    f_lo, width = float(rng.uniform(0.014, 0.022)), float(rng.uniform(0.004, 0.012))
    cfg = sy.grid_config(T_yr, f_lo, f_lo + width)
    S = sy.psd_AE(sy.freqs(cfg))
    df = 1.0 / cfg["T_obs_s"]
    Mc, q = float(rng.uniform(20.0, 40.0)), float(rng.uniform(0.5, 1.0))
    tau = 5.0 / 256.0 * (Mc * sy.MSUN_S) ** (-5.0 / 3.0) * (np.pi * f_lo) ** (-8.0 / 3.0)     # Newtonian time to coalescence from f_lo
    th = sy.draw_injection(rng, Mc, q, tau)
    lo, hi = sy.prior_box(th[0], th[2], eta_lo=0.16, dMc=float(rng.uniform(0.3, 1.5)), dtc=float(rng.uniform(0.05, 0.4)) * T_yr * sy.YEAR_S)
    P = 384
    parts = sy.draw_particles(int(rng.integers(1 << 30)), P, lo, hi)
    inp = dict(cfg=cfg, S_A=S, S_E=S.copy(), df=df, lo=lo, hi=hi, particles=parts,
               noise_A=sy.draw_noise(int(rng.integers(1 << 30)), S, df), noise_E=sy.draw_noise(int(rng.integers(1 << 30)), S, df),
               injections=[dict(theta=th, rho=float(rng.uniform(10.0, 30.0)))])
    if oracle.template(oracle.make_config(cfg), th)[2] == 0:
        inp["injections"] = []
    nb = cfg["n_bins"]
    lists = [sy.edges(nb, int(np.exp(rng.uniform(np.log(8), np.log(nb / 130))))) for _ in range(3)]
    n_e = int(rng.integers(20, 3000))
    a, b = sorted(rng.integers(0, nb + 1, size=2))
    if b - a > 200 * n_e:
        lists.append(np.sort(rng.integers(a, b + 1, size=n_e)).astype(np.int64))      # irregular, long on average, short pieces among them
    _, dA, dE = make_data(oracle, inp)
    H = gpu_handle(inp, dA, dE)
    H.set_option(sc.SC_OPT_TC_MAX_S, int(np.ceil(hi[2])))
    par = torch.from_numpy(parts).to("cuda:0")
    H.eval_stat(par, sy.edges(nb, 1).astype(np.int32))
    H.set_option(sc.SC_OPT_WINDOW_FRACTION_PPM, max(1, int(round(1e6 * H.counters()[0] / (P * nb)))))
    idx = np.sort(rng.choice(P, 12, replace=False))
    ref = oracle.eval_stat_levels(oracle.make_config(cfg, truth=True), dA, dE, S, S, parts[idx], lists)
    quad_seen = 0
    for e, r in zip(lists, ref):
        got = H.eval_stat(par, e.astype(np.int32)).cpu().numpy()[idx]
        quad_seen += bool(H.launch_info()[1] & sc.SC_FLAVOUR_QUAD)
        assert np.array_equal(got == 0.0, r == 0.0), (seed, len(e))
        ok = r > 0
        if ok.any():
            err = rel_err(got[ok], r[ok])
            assert np.all(err <= TOL), (seed, len(e), H.launch_info(), float(err.max()), float(r[ok][np.argmax(err)]))
    H.close()
    assert quad_seen >= 1
