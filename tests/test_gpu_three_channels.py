"""Three TDI channels A, E, T on the GPU against the oracle's sco_*3 functions (all `-m gpu`)."""
import numpy as np
import pytest

import sc_synth as sy
from helpers import rel_err

pytestmark = pytest.mark.gpu
TOL = 1e-6


def _dev(torch, a):
    return torch.from_numpy(np.ascontiguousarray(a)).to("cuda:0")


def _setup(oracle, cid, P, rho, seed):
    import torch
    import paper_2408_13170_b200 as sc
    sc.load_library()
    inp = sy.config_inputs(cid, P=P)
    cfgd = dict(inp["cfg"], n_channels=3)
    cfg = oracle.make_config(cfgd)
    f = sy.freqs(cfgd)
    S3 = (inp["S_A"], inp["S_E"], sy.psd_T(f))
    nT = sy.draw_noise(seed, S3[2], inp["df"])
    d3 = [inp["noise_A"].copy(), inp["noise_E"].copy(), nT]
    th = inp["injections"][0]["theta"]
    h3 = oracle.template3(cfg, th)[:3]
    kappa = rho / np.sqrt(oracle.inner3(h3, h3, S3, inp["df"]))
    d3 = [d + kappa * h for d, h in zip(d3, h3)]
    t = lambda a: _dev(torch, a)
    ri = lambda z: torch.view_as_real(t(z)).contiguous()
    H = sc.Handle(cfgd, ri(d3[0]), ri(d3[1]), t(S3[0]), t(S3[1]), dT=ri(d3[2]), S_T=t(S3[2]))
    return torch, sc, inp, cfgd, cfg, S3, d3, th, kappa, h3, H


def test_c1_three_channels_full_population(oracle):
    torch, sc, inp, cfgd, cfg, S3, d3, th, kappa, h3, H = _setup(oracle, 1, None, 20.0, 901)
    nb = cfgd["n_bins"]
    parts = np.vstack([inp["particles"], th[None, :]])
    par = _dev(torch, parts)
    for N in (1, 5, 100, 1000):
        e = sy.edges(nb, N)
        ref, refseg = oracle.eval_stat3(cfg, d3, S3, parts, e, want_seg=True)
        got = H.eval_stat(par, e).cpu().numpy()
        assert rel_err(got, ref).max() <= TOL, (N, rel_err(got, ref).max())
        seg = H.eval_segments(par, e).cpu().numpy()
        scale = np.abs(refseg).max(axis=1, keepdims=True)
        assert (np.abs(seg - refseg) / scale).max() <= 2e-6
        comp = H.eval_components(par, e).cpu().numpy()
        cref = np.array([oracle.components_from_seg(s, inp["df"]) for s in refseg])
        assert rel_err(comp, cref).max() <= TOL
    # the T channel matters here: dropping it changes the statistic at the injection by more than the tolerance
    e = sy.edges(nb, 100)
    u3 = H.eval_stat(par[-1:].contiguous(), e).item()
    u2 = oracle.eval_stat(oracle.make_config(inp["cfg"]), d3[0], d3[1], S3[0], S3[1], th[None, :], e)[0]
    assert abs(u3 - u2) > 1e-3 * u3
    dd = oracle.inner3(d3, d3, S3, inp["df"])
    assert H.data_norm() == pytest.approx(dd, rel=1e-12)
    H.close()


def test_three_channel_template_and_noise_free_match(oracle):
    torch, sc, inp, cfgd, cfg, S3, d3, th, kappa, h3, H = _setup(oracle, 1, 4, 20.0, 902)
    gA, gE, gT = (x.cpu().numpy()[0] for x in H.gen_template3(_dev(torch, th[None, :])))
    for g, h in zip((gA, gE, gT), h3):
        assert np.abs(g - h).max() <= 1e-7 * np.abs(h).max()
    assert np.array_equal(np.abs(gT) > 0, np.abs(h3[2]) > 0)
    H.close()
    # d = kappa h in all three channels: Upsilon_N(theta_inj) = rho^2 for every N
    import paper_2408_13170_b200 as scm
    t = lambda a: _dev(torch, a)
    ri = lambda z: torch.view_as_real(t(z)).contiguous()
    H2 = scm.Handle(cfgd, ri(kappa * h3[0]), ri(kappa * h3[1]), t(S3[0]), t(S3[1]), dT=ri(kappa * h3[2]), S_T=t(S3[2]))
    for N in (1, 10, 1000):
        got = H2.eval_stat(_dev(torch, th[None, :]), sy.edges(cfgd["n_bins"], N)).item()
        assert got == pytest.approx(400.0, rel=TOL)
    H2.close()


def test_fused_and_two_pass_agree(oracle):
    """SC_OPT_FUSED_AET: the one-pass kernel (A, E, T in the pair loop) and the two passes with combined segment tables are
    the same definition -- statistic, segments and components agree to FP32 rounding for the whole population, at levels
    that take the polynomial (N = 10) and the hardware (N = 100, 1000) sin/cos flavour."""
    torch, sc, inp, cfgd, cfg, S3, d3, th, kappa, h3, H = _setup(oracle, 2, 512, 17.0, 906)
    H.set_option(sc.SC_OPT_TC_MAX_S, int(np.ceil(inp["hi"][2])))
    H.set_option(sc.SC_OPT_ESCALATE, 0)
    par = _dev(torch, inp["particles"])
    for N in (10, 100, 1000):
        e = sy.edges(cfgd["n_bins"], N)
        res = {}
        for fused in (1, 0):
            H.set_option(sc.SC_OPT_FUSED_AET, fused)
            res[fused] = (H.eval_stat(par, e).cpu().numpy(), H.eval_segments(par, e).cpu().numpy(), H.eval_components(par, e).cpu().numpy())
        a, b = res[1], res[0]
        ok = b[0] > 1.0
        assert ok.sum() > 400 and rel_err(a[0][ok], b[0][ok]).max() <= 2e-6 / np.sqrt(b[0][ok]).min()
        scale = np.abs(b[1]).max(axis=1, keepdims=True)
        assert (np.abs(a[1] - b[1]) / scale).max() <= 2e-6
        assert rel_err(a[2][ok], b[2][ok]).max() <= 2e-6
    H.close()


def test_c2_three_channels_sampled(oracle):
    torch, sc, inp, cfgd, cfg, S3, d3, th, kappa, h3, H = _setup(oracle, 2, None, 17.0, 903)
    H.set_option(sc.SC_OPT_TC_MAX_S, int(np.ceil(inp["hi"][2])))
    P = inp["particles"].shape[0]
    idx = np.sort(np.random.default_rng(9).choice(P, 8, replace=False))
    par = _dev(torch, inp["particles"])
    for N in (1000, 100):
        e = sy.edges(cfgd["n_bins"], N)
        ref = oracle.eval_stat3(cfg, d3, S3, inp["particles"][idx], e)
        got = H.eval_stat(par, e).cpu().numpy()                     # whole population
        assert rel_err(got[idx], ref).max() <= TOL
        assert np.all(np.isfinite(got)) and np.all(got >= 0)
    H.close()


@pytest.mark.parametrize("N", [8, 16])
def test_three_channel_escalation_of_ill_conditioned_particles(oracle, N):
    """SC_OPT_ESCALATE on a three-channel handle: both passes run the FP32-amplitude kernels (segment tables), so a particle
    whose COMBINED statistic is below tau is re-evaluated by the all-FP64 kernels (both passes) -- c2's population at a
    coarse rung has such particles; every particle must meet the bar, an escalated one carries the all-FP64 value."""
    torch, sc, inp, cfgd, cfg, S3, d3, th, kappa, h3, H = _setup(oracle, 2, 256, 17.0, 905)
    e = sy.edges(cfgd["n_bins"], N)
    par = _dev(torch, inp["particles"])
    ref = oracle.eval_stat3(cfg, d3, S3, inp["particles"], e)
    auto = H.eval_stat(par, e).cpu().numpy()
    H.set_option(sc.SC_OPT_ESCALATE, 0)
    plain = H.eval_stat(par, e).cpu().numpy()
    H.set_option(sc.SC_OPT_PRECISION, 2)
    f64 = H.eval_stat(par, e).cpu().numpy()
    H.close()
    esc = (plain > 0) & (plain < 6.0)
    assert esc.sum() > 0                                           # the case is exercised
    assert rel_err(auto[esc], f64[esc]).max() <= 1e-11 and np.array_equal(auto[~esc], plain[~esc])
    ok = ref > 0
    assert rel_err(auto[ok], ref[ok]).max() <= TOL


@pytest.mark.parametrize("N", [2, 10, 50, 100, 1000])
def test_c1_three_channels_adaptive_segments(oracle, N):
    """Per-particle equal-SNR^2 segments over A, E, T (PAPER.md:120 with the channel sums of PAPER.md:36, 59 -- the paper's
    own configuration): the device decides the integer edges in FP64 from all three channels; they must EQUAL
    sco_equal_snr_edges3, and the statistic and the components must match the oracle on those edges."""
    torch, sc, inp, cfgd, cfg, S3, d3, th, kappa, h3, H = _setup(oracle, 1, None, 20.0, 907)
    nb = cfgd["n_bins"]
    parts = np.vstack([inp["particles"], th[None, :]])
    par = _dev(torch, parts)
    got, ged, comp = H.eval_stat_adaptive(par, N, want_edges=True, want_comp=True)
    got, ged, comp = got.cpu().numpy(), ged.cpu().numpy().astype(np.int64), comp.cpu().numpy()
    H.close()
    ref_own, oed = oracle.eval_stat_adaptive3(cfg, d3, S3, parts, N, want_edges=True)
    assert np.all(ged[:, 0] == 0) and np.all(ged[:, -1] == nb) and np.all(np.diff(ged, axis=1) >= 0)
    d = np.abs(ged - oed)
    assert np.array_equal(ged, oed), (int(d.max()), float((d != 0).mean()))
    ref, rc = oracle.eval_stat_adaptive3(cfg, d3, S3, parts, N, in_edges=ged, want_comp=True)
    assert rel_err(got, ref).max() <= TOL, (N, rel_err(got, ref).max())
    assert rel_err(comp, rc).max() <= TOL
    # the T channel moves the edges: the two-channel rule on the same templates gives other edges somewhere
    if N >= 50:
        e2 = oracle.eval_stat_adaptive(oracle.make_config(inp["cfg"]), d3[0], d3[1], S3[0], S3[1], parts[-1:], N, want_edges=True)[1]
        assert not np.array_equal(e2[0], oed[-1])


def test_c3_three_channels_bench_configuration(oracle):
    """The bench's three-channel extra at full size: c3 (4 yr, 1.64 M bins, node stride 512), whole population through the
    one-pass kernel at N = 5000 and through the per-particle-segment kernels at N = 100; the oracle (truth mode) on a sample."""
    torch, sc, inp, cfgd, cfg, S3, d3, th, kappa, h3, H = _setup(oracle, 3, None, 17.0, 908)
    H.set_option(sc.SC_OPT_TC_MAX_S, int(np.ceil(inp["hi"][2])))
    P = inp["particles"].shape[0]
    par = _dev(torch, inp["particles"])
    cfg_t = oracle.make_config(cfgd, truth=True)
    e = sy.edges(cfgd["n_bins"], 5000)
    got = H.eval_stat(par, e).cpu().numpy()
    idx = np.unique(np.concatenate([np.random.default_rng(12).choice(P, 12, replace=False), np.argsort(got)[:4]]))
    ref = oracle.eval_stat3(cfg_t, d3, S3, inp["particles"][idx], e)
    assert rel_err(got[idx], ref).max() <= TOL, rel_err(got[idx], ref).max()
    assert np.all(np.isfinite(got)) and np.all(got >= 0)
    # per-particle segments over the three channels
    ga, ged = H.eval_stat_adaptive(par, 100, want_edges=True)
    ga, ged = ga.cpu().numpy(), ged.cpu().numpy().astype(np.int64)
    H.close()
    sub = idx[:8]
    ref_own, oed = oracle.eval_stat_adaptive3(cfg, d3, S3, inp["particles"][sub], 100, want_edges=True)
    dlt = np.abs(ged[sub] - oed)
    assert dlt.max() <= 1 and (dlt == 0).mean() >= 0.999, (int(dlt.max()), float((dlt != 0).mean()))
    ref_a = oracle.eval_stat_adaptive3(cfg_t, d3, S3, inp["particles"][sub], 100, in_edges=ged[sub])
    assert rel_err(ga[sub], ref_a).max() <= TOL, rel_err(ga[sub], ref_a).max()


def test_three_channel_restrictions_and_search(oracle):
    torch, sc, inp, cfgd, cfg, S3, d3, th, kappa, h3, H = _setup(oracle, 1, None, 20.0, 904)
    par = _dev(torch, inp["particles"])
    got = H.eval_stat_adaptive(par, 1).cpu().numpy()                # one segment: the edges are (0, n_bins)
    assert np.array_equal(got, H.eval_stat(par, np.array([0, cfgd["n_bins"]])).cpu().numpy())
    with pytest.raises(sc.SCError):
        sc.Handle(dict(cfgd, n_channels=2), par, par, par, par, dT=par, S_T=par)
    # a short search on the paper's own configuration (A, E, T with per-particle equal-SNR^2 segments) runs through
    hyper = [sy.TABLE_IV[100], sy.TABLE_IV[1]]
    scfg = sc.ScSearchConfig.make([100, 1], hyper, adaptive_edges=True, conv_window=3, max_iters_per_rung=5, seed=1)
    P = inp["particles"].shape[0]
    lab = torch.zeros(P, dtype=torch.int32, device="cuda:0")
    res = H.search_run(scfg, par.clone(), _dev(torch, inp["velocities"]), lab, 1, _dev(torch, inp["lo"]), _dev(torch, inp["hi"]))
    ref = oracle.eval_stat3(cfg, d3, S3, res["best_pos"], sy.edges(cfgd["n_bins"], 1))
    assert res["best_val"][0] == pytest.approx(ref[0], rel=TOL)
    H.close()
