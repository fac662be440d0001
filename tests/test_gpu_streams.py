"""Second workload (Fig. 3 of the paper): many data streams x one template,
through the C ABI, against the oracle stream by stream, plus the sampling distributions the paper checks with it."""
import numpy as np
import pytest

import sc_synth as sy
from helpers import gpu_handle, rel_err

pytestmark = pytest.mark.gpu
TOL = 1e-6


def _dev(torch, a):
    return torch.from_numpy(np.ascontiguousarray(a)).to("cuda:0")


@pytest.fixture(scope="module")
def env(oracle):
    import torch
    import paper_2408_13170_b200 as sc
    assert torch.cuda.is_available()
    sc.load_library()
    inp = sy.config_inputs(1, P=1)
    cfg = oracle.make_config(inp["cfg"])
    th = inp["injections"][0]["theta"]
    hA, hE, _ = oracle.template(cfg, th)
    rho2 = oracle.inner(hA, hE, hA, hE, inp["S_A"], inp["S_E"], inp["df"])
    H = gpu_handle(inp, inp["noise_A"], inp["noise_E"])          # the handle only lends its PSD to this path
    yield dict(torch=torch, sc=sc, inp=inp, cfg=cfg, th=th, hA=hA, hE=hE, rho2=rho2, H=H)
    H.close()


def _streams(env, D, rho, seed):
    """D independent noise realisations (sc_synth recipe, O6) + the ORACLE's template scaled to SNR rho."""
    inp = env["inp"]
    rng = np.random.default_rng(seed)
    nb = inp["cfg"]["n_bins"]
    sd = np.sqrt(inp["S_A"] / (4 * inp["df"]))
    sdE = np.sqrt(inp["S_E"] / (4 * inp["df"]))
    kappa = rho / np.sqrt(env["rho2"])
    dA = (rng.standard_normal((D, nb)) + 1j * rng.standard_normal((D, nb))) * sd + kappa * env["hA"]
    dE = (rng.standard_normal((D, nb)) + 1j * rng.standard_normal((D, nb))) * sdE + kappa * env["hE"]
    return dA, dE


@pytest.mark.parametrize("f64", [False, True], ids=["f32streams", "f64streams"])
def test_streams_parity(env, oracle, f64):
    torch, H, inp = env["torch"], env["H"], env["inp"]
    nb = inp["cfg"]["n_bins"]
    D = 24
    dA, dE = _streams(env, D, 20.0, 11)
    dA[3] *= 0; dE[3] *= 0                                        # an all-zero stream gives exactly 0
    W = H.whiten_streams(_dev(torch, dA), _dev(torch, dE), f64=f64)
    levels = [1, 10, 100, 1000] if f64 else [10, 100, 1000, 7919]
    for N in levels + ["partial"]:
        e = sy.edges(nb, N) if N != "partial" else np.array([5, 5, 1029, 1030, 9000, 9000, 20001], dtype=np.int64)
        got = H.eval_stat_streams(_dev(torch, env["th"]), W, e).cpu().numpy()
        ref = np.array([oracle.stat_from_arrays(dA[d], dE[d], env["hA"], env["hE"], inp["S_A"], inp["S_E"], inp["df"], e)
                        for d in range(D)])
        assert got[3] == 0.0 and ref[3] == 0.0
        m = np.arange(D) != 3
        assert rel_err(got[m], ref[m]).max() <= TOL, (N, rel_err(got[m], ref[m]).max())
    # same template path as the particle workload: one stream == the handle's own data evaluated by sc_eval_stat
    H2 = gpu_handle(inp, dA[0], dE[0])
    e = sy.edges(nb, 100)
    a = H2.eval_stat(_dev(torch, env["th"][None, :]), e).cpu().numpy()[0]
    b = H.eval_stat_streams(_dev(torch, env["th"]), W, e).cpu().numpy()[0]
    assert a == pytest.approx(b, rel=2e-7)
    H2.close()


def test_streams_sampling_distributions(env):
    """Eq. 11-12 and the chi^2_2 of N = 1 over 1500 noise realisations, as in Fig. 3:
    noise only mean 2N, var 4N; with the signal mean 2N + rho^2, var 4N + 4 rho^2."""
    torch, H, inp = env["torch"], env["H"], env["inp"]
    nb = inp["cfg"]["n_bins"]
    D = 1500
    g = torch.Generator(device="cuda:0").manual_seed(240813170)
    sdA = _dev(torch, np.sqrt(inp["S_A"] / (4 * inp["df"])))
    sdE = _dev(torch, np.sqrt(inp["S_E"] / (4 * inp["df"])))
    nA = torch.view_as_complex(torch.randn((D, nb, 2), dtype=torch.float64, device="cuda:0", generator=g)) * sdA
    nE = torch.view_as_complex(torch.randn((D, nb, 2), dtype=torch.float64, device="cuda:0", generator=g)) * sdE
    hA, hE = _dev(torch, env["hA"]), _dev(torch, env["hE"])
    th = _dev(torch, env["th"])
    # segments over the template's support (the time window leaves part of this band empty, and an empty segment
    # contributes nothing, Q8): N equal-width segments between the first and the last non-zero bin
    nz = np.nonzero(np.abs(env["hA"]) > 0)[0]
    j0, j1 = int(nz[0]), int(nz[-1]) + 1
    for rho in (0.0, 10.0, 20.0):
        kappa = rho / np.sqrt(env["rho2"])
        W = H.whiten_streams(nA + kappa * hA, nE + kappa * hE, f64=True)
        for N in (1, 10, 50, 100):
            u = H.eval_stat_streams(th, W, j0 + sy.edges(j1 - j0, N)).cpu().numpy()
            mean, var = 2 * N + rho ** 2, 4 * N + 4 * rho ** 2
            assert abs(u.mean() - mean) < 5 * np.sqrt(var / D), (rho, N, u.mean(), mean)
            assert abs(u.var() / var - 1) < 5 * np.sqrt(2.0 / D) + 0.05, (rho, N, u.var(), var)
        del W


def test_streams_argument_errors(env):
    torch, sc, H, inp = env["torch"], env["sc"], env["H"], env["inp"]
    nb = inp["cfg"]["n_bins"]
    W = torch.zeros((2, nb, 4), dtype=torch.float32, device="cuda:0")
    th = _dev(torch, env["th"])
    with pytest.raises(sc.SCError):
        H.eval_stat_streams(th, W, np.array([0, 10, 5, nb]))
    with pytest.raises(sc.SCError):
        H.eval_stat_streams(th, W, np.array([0, nb + 1]))
    assert np.array_equal(H.eval_stat_streams(th, W, np.array([7, 7])).cpu().numpy(), np.zeros(2))
