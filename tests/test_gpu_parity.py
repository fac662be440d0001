"""GPU-vs-oracle parity through the C ABI (all `-m gpu`).

Bar (BASELINE.json north_star): |Upsilon_gpu - Upsilon_oracle| <= 1e-6 * Upsilon_oracle for EVERY particle, on every
config; bit-exact segment-boundary indexing.  Data streams are assembled from sc_synth noise plus the ORACLE's
templates (tests/helpers.py); nothing the oracle sees comes from the CUDA path.
Full-size cases run the GPU in bench.py's launch configuration (whole population) and compare a seeded sample of
particles the oracle can afford, plus properties that hold at any size.
"""
import numpy as np
import pytest

import sc_synth as sy
from helpers import gpu_handle, make_data, rel_err

pytestmark = pytest.mark.gpu

TOL = 1e-6          # relative, per particle (north_star)


@pytest.fixture(scope="module")
def torch_cuda():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    return torch


@pytest.fixture(scope="module")
def sc():
    import paper_2408_13170_b200 as sc
    sc.load_library()          # fails loudly if the extension is missing
    return sc


def _dev(torch, a):
    return torch.from_numpy(np.ascontiguousarray(a)).to("cuda:0")


def _sample_idx(P, n, seed):
    return np.sort(np.random.default_rng(seed).choice(P, size=min(n, P), replace=False))


# ---------------------------------------------------------------------------------------------- config 1 (full)
@pytest.fixture(scope="module")
def c1(oracle, torch_cuda, sc):
    inp = sy.config_inputs(1)
    cfg, dA, dE = make_data(oracle, inp)
    H = gpu_handle(inp, dA, dE)
    yield dict(inp=inp, cfg=cfg, dA=dA, dE=dE, H=H)
    H.close()


@pytest.mark.parametrize("prec", [1, 2], ids=["fp32amp", "allfp64"])
def test_c1_full_population(c1, oracle, torch_cuda, sc, prec):
    inp, H = c1["inp"], c1["H"]
    e = inp["edges"][1000]
    ref, refseg = oracle.eval_stat(c1["cfg"], c1["dA"], c1["dE"], inp["S_A"], inp["S_E"], inp["particles"], e, want_seg=True)
    H.set_option(sc.SC_OPT_PRECISION, prec)
    par = _dev(torch_cuda, inp["particles"])
    got = H.eval_stat(par, e).cpu().numpy()
    assert rel_err(got, ref).max() <= TOL
    seg = H.eval_segments(par, e).cpu().numpy()
    scale = np.abs(refseg).max(axis=1, keepdims=True)            # per particle, per component
    tol_seg = 2e-6 if prec == 1 else 1e-7
    assert (np.abs(seg - refseg) / scale).max() <= tol_seg
    # the statistic recomputed from the GPU's own segments agrees with the GPU's statistic (stitch = definition)
    z2 = seg[:, :, 0] ** 2 + seg[:, :, 1] ** 2
    with np.errstate(invalid="ignore", divide="ignore"):
        u = 4 * inp["df"] * np.where(seg[:, :, 2] > 0, z2 / seg[:, :, 2], 0.0).sum(axis=1)
    # (the FP32 path evaluates the statistic with hardware sin/cos and the segments with the polynomial one)
    assert rel_err(u, got).max() <= (1e-12 if prec == 2 else 2e-7)
    H.set_option(sc.SC_OPT_PRECISION, 0)


def test_c1_template_elementwise(c1, oracle, torch_cuda):
    """sc_gen_template (same node tables / interpolants as the statistic) against the oracle's direct evaluation."""
    inp, H = c1["inp"], c1["H"]
    thetas = np.vstack([inp["injections"][0]["theta"][None, :], inp["particles"][:3]])
    gA, gE = H.gen_template(_dev(torch_cuda, thetas))
    gA, gE = gA.cpu().numpy(), gE.cpu().numpy()
    for i, th in enumerate(thetas):
        hA, hE, w = oracle.template(c1["cfg"], th)
        assert np.array_equal(np.abs(gA[i]) > 0, np.abs(hA) > 0)          # identical time window, bin for bin
        assert int((np.abs(gA[i]) > 0).sum()) == w
        assert np.abs(gA[i] - hA).max() <= 1e-7 * np.abs(hA).max()
        assert np.abs(gE[i] - hE).max() <= 1e-7 * np.abs(hE).max()


def test_c1_hierarchy_levels_and_single_segment(c1, oracle, torch_cuda, sc):
    inp, H = c1["inp"], c1["H"]
    nb = inp["cfg"]["n_bins"]
    par = _dev(torch_cuda, inp["particles"])
    levels = [1, 3, 10, 100, 1000, 7919, nb]                 # N = n_bins: one bin per segment
    elist = [sy.edges(nb, N) for N in levels]
    ref = oracle.eval_stat_levels(c1["cfg"], c1["dA"], c1["dE"], inp["S_A"], inp["S_E"], inp["particles"], elist)
    prev = None
    for N, e, r in zip(levels, elist, ref):
        got = H.eval_stat(par, e).cpu().numpy()               # auto precision: all-FP64 below 8 segments
        assert rel_err(got, r).max() <= TOL, N
        if prev is not None and N % prev[0] == 0:
            assert np.all(got >= prev[1] * (1 - 1e-9))        # nested refinement never decreases Upsilon
        prev = (N, got)


@pytest.mark.parametrize("N", [8, 10, 16, 32, 50])
def test_escalation_of_ill_conditioned_particles(oracle, torch_cuda, sc, N):
    """Automatic precision: the FP32 path's relative error grows like c / sqrt(Upsilon), so every
    particle with 0 < Upsilon < tau is re-evaluated by the all-FP64 path on the device.  c2's population at the paper's
    coarse rungs (N = 50, 10) has such particles: the bar must hold for all of them, an escalated particle
    must carry the all-FP64 value (to 1e-11), every other one exactly the FP32 path's."""
    inp = sy.config_inputs(2, P=384)
    cfg, dA, dE = make_data(oracle, inp)
    H = gpu_handle(inp, dA, dE)
    e = sy.edges(inp["cfg"]["n_bins"], N)
    par = _dev(torch_cuda, inp["particles"])
    ref = oracle.eval_stat(cfg, dA, dE, inp["S_A"], inp["S_E"], inp["particles"], e)
    auto = H.eval_stat(par, e).cpu().numpy()
    auto2 = H.eval_stat(par, e).cpu().numpy()                 # second call: grid hint now known, same result
    H.set_option(sc.SC_OPT_ESCALATE, 0)
    plain = H.eval_stat(par, e).cpu().numpy()
    H.set_option(sc.SC_OPT_PRECISION, 2)
    f64 = H.eval_stat(par, e).cpu().numpy()
    H.close()
    tau = 16.0 if N >= 32 else 6.0
    esc = (plain > 0) & (plain < tau)
    assert np.array_equal(auto, auto2)
    # (the escalation pass runs the all-FP64 kernels on the compacted list: same formula, other warp neighbours)
    assert rel_err(auto[esc], f64[esc]).max(initial=0.0) <= 1e-11 and np.array_equal(auto[~esc], plain[~esc])
    ok = ref > 0
    assert rel_err(auto[ok], ref[ok]).max() <= TOL
    assert rel_err(auto[ok], ref[ok]).max() <= 6e-7           # design margin: c_max / sqrt(tau) <= 4.1e-7
    if N <= 16:
        assert esc.sum() > 0                                  # the case is exercised


def test_window_sort_is_a_pure_reordering(oracle, torch_cuda, sc):
    """SC_OPT_WINDOW_SORT: batches are processed in the order of the window centres.  Against the oracle nothing changes;
    against the input order only the rounding of the FP32 path does (the sigma of a sub-interval comes from the weight
    moments when all 32 particles of the warp are inside their windows, from the per-bin sum otherwise); the all-FP64
    path has one formula and agrees to its own rounding (a lane's phase differences are rebuilt or stepped on depending
    on whether a neighbour is active before its window opens).  Re-running and re-batching in input order is bitwise stable."""
    inp = sy.config_inputs(2, P=640)
    cfg, dA, dE = make_data(oracle, inp)
    H = gpu_handle(inp, dA, dE)
    par = _dev(torch_cuda, inp["particles"])
    idx = _sample_idx(640, 48, 11)
    for N in (100, 1):
        e = sy.edges(inp["cfg"]["n_bins"], N)
        ref = oracle.eval_stat(cfg, dA, dE, inp["S_A"], inp["S_E"], inp["particles"][idx], e)
        H.set_option(sc.SC_OPT_WINDOW_SORT, 1)
        a = H.eval_stat(par, e).cpu().numpy()
        assert np.array_equal(a, H.eval_stat(par, e).cpu().numpy())
        H.set_option(sc.SC_OPT_WINDOW_SORT, 0)
        b = H.eval_stat(par, e).cpu().numpy()
        H.set_option(sc.SC_OPT_SCRATCH_BYTES, 8 << 20)           # several batches, input order: same warps, same bits
        c = H.eval_stat(par, e).cpu().numpy()
        H.set_option(sc.SC_OPT_SCRATCH_BYTES, 8 << 30)
        assert np.array_equal(b, c)
        ok = ref > 0
        assert rel_err(a[idx][ok], ref[ok]).max() <= TOL and rel_err(b[idx][ok], ref[ok]).max() <= TOL
        if N == 1:
            assert rel_err(a[b > 0], b[b > 0]).max() <= 1e-11
        else:
            assert rel_err(a[b > 0], b[b > 0]).max() <= 2e-7
    H.close()


def test_short_windows_skip_logic_c5(oracle, torch_cuda, sc):
    """c5: every particle's time window covers a few per cent of the band, at its own place.  With the window sort most
    (chunk, 128-particle block) CTAs and most (node, block) entries are skipped and k_stitch reads only the chunks of the
    window; in input order nearly nothing is.  Both orders must give the same statistic for EVERY particle (to 1e-11
    on the all-FP64 path, to FP32 rounding otherwise), the components included, and the oracle's on a sample."""
    inp = sy.config_inputs(5, P=1536)
    cfg, dA, dE = make_data(oracle, inp)
    H = gpu_handle(inp, dA, dE)
    H.set_option(sc.SC_OPT_TC_MAX_S, int(np.ceil(inp["hi"][2])))
    par = _dev(torch_cuda, inp["particles"])
    idx = _sample_idx(1536, 6, 55)
    for N in (500, 1):
        e = sy.edges(inp["cfg"]["n_bins"], N)
        ref = oracle.eval_stat(cfg, dA, dE, inp["S_A"], inp["S_E"], inp["particles"][idx], e)
        res = {}
        for srt in (1, 0):
            H.set_option(sc.SC_OPT_WINDOW_SORT, srt)
            res[srt] = (H.eval_stat(par, e).cpu().numpy(), H.eval_components(par, e).cpu().numpy())
        a, b = res[1][0], res[0][0]
        assert (a > 0).sum() > 1400
        if N == 1:      # all-FP64: only the rounding of the phase forward differences depends on the warp's company
            assert rel_err(a[b > 0], b[b > 0]).max() <= 1e-11
            assert rel_err(res[1][1][:, 1:][b > 0], res[0][1][:, 1:][b > 0]).max() <= 1e-11
        else:
            assert rel_err(a[b > 0], b[b > 0]).max() <= 2e-7
            assert rel_err(res[1][1][:, 1:][b > 0], res[0][1][:, 1:][b > 0]).max() <= 2e-7
        ok = ref > 0
        assert rel_err(a[idx][ok], ref[ok]).max() <= TOL
    H.close()


def test_c1_partial_and_empty_edges(c1, oracle, torch_cuda):
    inp, H = c1["inp"], c1["H"]
    nb = inp["cfg"]["n_bins"]
    par = _dev(torch_cuda, inp["particles"][:9])               # ragged population
    for e in (np.array([5000, 5000, 5001, 9000, 9000, 20000, 20000], dtype=np.int64),      # empties, 1-bin, partial cover
              np.array([0, 1, 2, 3, nb], dtype=np.int64),
              np.array([2047, 2048, 2049, 4096, 6144, 6145], dtype=np.int64),              # edges on / next to chunk borders
              np.array([nb - 1, nb], dtype=np.int64),
              np.array([17, 17], dtype=np.int64)):                                          # nothing covered
        ref, refseg = oracle.eval_stat(c1["cfg"], c1["dA"], c1["dE"], inp["S_A"], inp["S_E"], inp["particles"][:9], e, want_seg=True)
        got = H.eval_stat(par, e).cpu().numpy()
        assert np.all(np.abs(got - ref) <= TOL * np.abs(ref)), e
        seg = H.eval_segments(par, e).cpu().numpy()
        scale = max(np.abs(refseg).max(), 1e-300)
        assert np.abs(seg - refseg).max() <= 2e-6 * scale
        assert np.array_equal(seg[:, np.diff(e) == 0, :], np.zeros_like(seg[:, np.diff(e) == 0, :]))


@pytest.mark.parametrize("N,prec", [(1, 0), (50, 0), (1000, 0), (1000, 2), (100, 1)])
def test_c1_components_and_loglike(c1, oracle, torch_cuda, sc, N, prec):
    """Eq. 8 (O_hat_N), Eq. 3 (<h|h>) and Eq. 9 (log L_hat_N) from the same per-segment sums, against the oracle's
    sco_components_from_seg / sco_loglike applied to the ORACLE's segments."""
    inp, H = c1["inp"], c1["H"]
    e = sy.edges(inp["cfg"]["n_bins"], N)
    ref, refseg = oracle.eval_stat(c1["cfg"], c1["dA"], c1["dE"], inp["S_A"], inp["S_E"], inp["particles"], e, want_seg=True)
    comp_ref = np.array([oracle.components_from_seg(s, inp["df"]) for s in refseg])
    dd = oracle.inner(c1["dA"], c1["dE"], c1["dA"], c1["dE"], inp["S_A"], inp["S_E"], inp["df"])
    assert H.data_norm() == pytest.approx(dd, rel=1e-12)
    H.set_option(sc.SC_OPT_PRECISION, prec)
    par = _dev(torch_cuda, inp["particles"])
    comp = H.eval_components(par, e).cpu().numpy()
    assert rel_err(comp[:, 0], ref).max() <= TOL
    assert np.array_equal(comp[:, 0], H.eval_stat(par, e).cpu().numpy())      # same kernels, same order
    assert rel_err(comp[:, 1], comp_ref[:, 1]).max() <= TOL
    assert rel_err(comp[:, 2], comp_ref[:, 2]).max() <= TOL
    # amplitude that maximises Eq. 9: A = O_hat/<h|h>; also an arbitrary one
    for amp in (comp_ref[:, 1] / comp_ref[:, 2], np.full(len(ref), 3.0e-3 * np.median(comp_ref[:, 1] / comp_ref[:, 2]))):
        want = np.array([oracle.loglike(dd, c[2], c[1], a) for c, a in zip(comp_ref, amp)])
        got = H.eval_loglike(par, _dev(torch_cuda, amp), e).cpu().numpy()
        # log L_hat = -dd/2 + (small): the bar is relative to the data-independent part that the template controls
        assert (np.abs(got - want) / np.maximum(np.abs(want + 0.5 * dd), 1e-300)).max() <= 2 * TOL
    H.set_option(sc.SC_OPT_PRECISION, 0)


def test_invalid_particles_give_zero(c1, torch_cuda):
    inp, H = c1["inp"], c1["H"]
    p = inp["particles"][:6].copy()
    p[0, 1] = 0.26; p[1, 0] = -1.0; p[2, 2] = np.nan; p[3, 5] = np.inf; p[4, 1] = 0.0
    got = H.eval_stat(_dev(torch_cuda, p), inp["edges"][1000]).cpu().numpy()
    assert np.array_equal(got[:5], np.zeros(5)) and got[5] > 0 and np.all(np.isfinite(got))


def test_determinism_batching_and_host_entry(c1, torch_cuda, sc):
    inp, H = c1["inp"], c1["H"]
    e = inp["edges"][1000]
    par = _dev(torch_cuda, inp["particles"])
    a = H.eval_stat(par, e).cpu().numpy()
    b = H.eval_stat(par, e).cpu().numpy()
    assert np.array_equal(a, b)                                 # no atomics in the bin loop: bitwise reproducible
    H.set_option(sc.SC_OPT_SCRATCH_BYTES, 1 << 20)              # force several particle batches
    c = H.eval_stat(par, e).cpu().numpy()
    H.set_option(sc.SC_OPT_SCRATCH_BYTES, 8 << 30)
    assert np.array_equal(a, c)
    d = H.eval_stat_host(inp["particles"], e)                   # host-buffer entry point
    assert np.array_equal(a, d)
    e_dev = torch_cuda.from_numpy(e.astype(np.int32)).to("cuda:0")
    f = H.eval_stat(par, e_dev).cpu().numpy()                   # device-resident edges
    assert np.array_equal(a, f)
    for P in (1, 5, 33, 64):
        g = H.eval_stat(par[:P].contiguous(), e).cpu().numpy()
        assert np.array_equal(g, a[:P])


def test_error_codes(c1, torch_cuda, sc):
    inp, H = c1["inp"], c1["H"]
    par = _dev(torch_cuda, inp["particles"][:4])
    nb = inp["cfg"]["n_bins"]
    for bad in (np.array([0, 10, 5, nb]), np.array([-1, 10, nb]), np.array([0, nb + 1])):
        with pytest.raises(sc.SCError) as ei:
            H.eval_stat(par, bad)
        assert ei.value.code == -1
    with pytest.raises(sc.SCError):
        sc.Handle(dict(inp["cfg"], n_channels=3), par, par, par, par)
    # the handle still works after argument errors
    assert H.eval_stat(par, inp["edges"][1000]).shape[0] == 4


# ---------------------------------------------------------------------------------------------- bit-exact indexing
def test_segment_indexing_bit_exact(oracle, torch_cuda, sc):
    """One-bin impulse data: exactly one segment may be non-zero, the k with e_k <= j < e_{k+1} (Q2, Q7)."""
    cfgd = sy.grid_config(0.5, 0.018, 0.020, window_mode=0)
    nb = cfgd["n_bins"]
    S = sy.psd_AE(sy.freqs(cfgd))
    th = sy.config_inputs(1, P=1)["particles"]
    rng = np.random.default_rng(12)
    edge_sets = [sy.edges(nb, 1000), sy.edges(nb, 7),
                 np.array([0, 0, 1, 1, 2, 2047, 2048, 2048, 2049, 4095, 4097, 30000, nb], dtype=np.int64),
                 np.array([100, 2048, 4096, 31000], dtype=np.int64)]
    bins = sorted(set([0, 1, 2, 2046, 2047, 2048, 2049, 4095, 4096, 4097, 99, 100, 30999, 31000, nb - 1]
                      + list(rng.integers(0, nb, 10))))
    for j in bins:
        dA = np.zeros(nb, dtype=complex)
        dA[j] = (1.0 - 2.0j) * np.sqrt(S[j])
        H = gpu_handle(dict(cfg=cfgd, S_A=S, S_E=S), dA, dA * 0)
        for e in edge_sets:
            seg = H.eval_segments(_dev(torch_cuda, th), e).cpu().numpy()[0]
            nz = np.nonzero(seg[:, 0] ** 2 + seg[:, 1] ** 2)[0]
            k = np.searchsorted(e, j, side="right") - 1
            inside = 0 <= k < len(e) - 1 and e[k] <= j < e[k + 1]
            assert list(nz) == ([k] if inside else []), (j, e[:6])
        H.close()


# ---------------------------------------------------------------------------------------------- configs 2..5
# escalation thresholds of the automatic mode (sc_stat.cu esc_tau_poly / esc_tau_mufu)
ESC_TAU = {"poly": 6.0, "mufu": 16.0}


def _hard_particles(got, N, n_each=8):
    """Where this design can fail is in the tails: the particles with the smallest non-zero statistic (the FP32 path's
    error grows as 1/sqrt(Upsilon)) and the ones nearest the escalation threshold tau of the level (just above it a
    particle keeps its FP32 value).  Chosen from the GPU's values; their reference is computed by the oracle alone."""
    live = np.nonzero(got > 0)[0]
    if live.size == 0:
        return live
    small = live[np.argsort(got[live], kind="stable")[:n_each]]
    tau = ESC_TAU["mufu"] if N >= 32 else ESC_TAU["poly"]
    near = live[np.argsort(np.abs(got[live] - tau), kind="stable")[:n_each]] if N >= 8 else live[:0]
    return np.concatenate([small, near])


def _full_launch_case(oracle, torch, sc, cid, n_sample, seed, tc_hint=True, opts=(), win_hint=True):
    """GPU: the whole population in bench.py's launch configuration, every level.  Oracle (truth mode: long-double phase,
    so the 1e-6 bar holds flat down to the smallest Upsilon): a seeded random sample of n_sample particles plus, per level,
    the 8 smallest non-zero and the 8 nearest the escalation threshold."""
    inp = sy.config_inputs(cid)
    cfg, dA, dE = make_data(oracle, inp)
    H = gpu_handle(inp, dA, dE)
    if tc_hint:
        H.set_option(sc.SC_OPT_TC_MAX_S, int(np.ceil(inp["hi"][2])))      # what bench.py sets: the tile's t_c bound
    for o, v in opts:
        H.set_option(o, v)
    P = inp["particles"].shape[0]
    levels = inp["spec"]["n_segs"]
    par = _dev(torch, inp["particles"])
    if win_hint:                       # ... and the measured share of the band inside the time windows (node spacing for N' segments)
        H.eval_stat(par, inp["edges"][levels[0]])
        H.set_option(sc.SC_OPT_WINDOW_FRACTION_PPM, int(round(1e6 * H.counters()[0] / (P * inp["cfg"]["n_bins"]))))
    got = {}
    for N in levels:
        got[N] = H.eval_stat(par, inp["edges"][N]).cpu().numpy()            # whole population, bench launch config
    inp["evaluated_fraction"] = H.counters()[0] / (P * inp["cfg"]["n_bins"])      # share of bins inside the time windows
    H.close()
    idx = np.unique(np.concatenate([_sample_idx(P, n_sample, seed)] + [_hard_particles(got[N], N) for N in levels]))
    cfg_truth = oracle.make_config(inp["cfg"], truth=True)
    ref = oracle.eval_stat_levels(cfg_truth, dA, dE, inp["S_A"], inp["S_E"], inp["particles"][idx], [inp["edges"][N] for N in levels])
    dd = oracle.inner(dA, dE, dA, dE, inp["S_A"], inp["S_E"], inp["df"])
    return inp, levels, idx, ref, got, dd


def _check_case(inp, levels, idx, ref, got, dd):
    for l, N in enumerate(levels):
        assert np.array_equal(got[N][idx] == 0.0, ref[l] == 0.0), N        # the same particles see an empty window
        live = ref[l] > 0
        err = rel_err(got[N][idx][live], ref[l][live])
        assert err.size and err.max() <= TOL, (N, err.max(), float(ref[l][live][np.argmax(err)]))
        assert np.all(np.isfinite(got[N])) and np.all(got[N] >= 0) and np.all(got[N] <= dd * (1 + 1e-9))   # Cauchy-Schwarz
    for a, b in zip(levels, levels[1:]):                       # levels are listed fine -> coarse and nest
        if a % b == 0:
            # levels may run in different precision modes; for Upsilon << 1 the FP32 path's error ~ 2.8 eps sqrt(Upsilon)
            # is not relative, hence the absolute floor
            assert np.all(got[a] >= got[b] - TOL * np.maximum(got[b], 1.0))


def test_c2_levels(oracle, torch_cuda, sc):
    _check_case(*_full_launch_case(oracle, torch_cuda, sc, 2, 64, 2))


def test_c3_bench_configuration(oracle, torch_cuda, sc):
    inp, levels, idx, ref, got, dd = _full_launch_case(oracle, torch_cuda, sc, 3, 64, 3)
    _check_case(inp, levels, idx, ref, got, dd)
    # Eq. 11: away from the source Upsilon_N ~ N(2N', 4N') with N' the segments the time window leaves
    # non-empty (Q8): the population median sits at 2 N'
    N = levels[0] * inp["evaluated_fraction"]
    assert abs(np.median(got[levels[0]]) - 2 * N) < 5 * 2 * np.sqrt(N)


def test_c4_noise_only_levels(oracle, torch_cuda, sc):
    inp, levels, idx, ref, got, dd = _full_launch_case(oracle, torch_cuda, sc, 4, 64, 4)
    _check_case(inp, levels, idx, ref, got, dd)
    for N in levels:            # pure noise: mean 2N', sd 2 sqrt N' (Eq. 11), N' = segments inside the time window (Q8)
        Np = N * inp["evaluated_fraction"]
        # all particles see ONE noise realisation, whose segment powers fluctuate in common: 0.5 % is ~5 sigma of that
        assert abs(got[N].mean() / (2 * Np) - 1) < 5e-3 + 2 / Np


def test_c5_full_hierarchy_with_coherent_level(oracle, torch_cuda, sc):
    inp, levels, idx, ref, got, dd = _full_launch_case(oracle, torch_cuda, sc, 5, 64, 5)
    assert levels[-1] == 1
    _check_case(inp, levels, idx, ref, got, dd)


@pytest.mark.parametrize("cid", [3, 4])
def test_tensor_core_flavour(oracle, torch_cuda, sc, cid):
    """SC_OPT_TENSOR_CORES = 1 (k_dense2_tc: the amplitude x data factor as a split-TF32 contraction on tcgen05, accumulators in
    TMEM, 8192-bin chunks): same definition, same bar against the oracle -- c3 (N = 5000) and c4 (N = 50000, 5000, 500)."""
    _check_case(*_full_launch_case(oracle, torch_cuda, sc, cid, 24, 10 + cid, opts=((sc.SC_OPT_TENSOR_CORES, 1),)))


def test_default_stride_without_tile_hint(oracle, torch_cuda, sc):
    """Without SC_OPT_TC_MAX_S the conservative default (t_c <= 10 yr) must meet the same bar."""
    inp, levels, idx, ref, got, dd = _full_launch_case(oracle, torch_cuda, sc, 2, 16, 7, tc_hint=False, win_hint=False)
    _check_case(inp, levels, idx, ref, got, dd)


# ---------------------------------------------------------------------------------------------- model variants
@pytest.mark.parametrize("window_mode,ecc", [(0, 0), (1, 1), (0, 1)])
def test_window_off_and_eccentric_term(oracle, torch_cuda, sc, window_mode, ecc):
    base = sy.config_inputs(1, P=24)
    cfgd = dict(base["cfg"], window_mode=window_mode, ecc_leading=ecc, f_ref_ecc=0.018)
    inp = dict(base, cfg=cfgd)
    parts = base["particles"].copy()
    if ecc:
        parts[:, 7] = np.random.default_rng(5).uniform(0.005, 0.1, len(parts))      # Table I prior
        inp["injections"] = [dict(theta=np.concatenate([base["injections"][0]["theta"][:7], [0.05]]), rho=20.0)]
    cfg, dA, dE = make_data(oracle, inp)
    H = gpu_handle(inp, dA, dE)
    for N in (1, 100, 1000):
        e = sy.edges(cfgd["n_bins"], N)
        ref = oracle.eval_stat(cfg, dA, dE, inp["S_A"], inp["S_E"], parts, e)
        got = H.eval_stat(_dev(torch_cuda, parts), e).cpu().numpy()
        assert rel_err(got, ref).max() <= TOL, (N, window_mode, ecc)
    H.close()


@pytest.mark.parametrize("pn", [0, 4])
def test_lower_pn_orders(oracle, torch_cuda, sc, pn):
    base = sy.config_inputs(1, P=8)
    inp = dict(base, cfg=dict(base["cfg"], pn_order_x2=pn, window_mode=0))
    cfg, dA, dE = make_data(oracle, inp)
    H = gpu_handle(inp, dA, dE)
    e = sy.edges(inp["cfg"]["n_bins"], 100)
    ref = oracle.eval_stat(cfg, dA, dE, inp["S_A"], inp["S_E"], base["particles"], e)
    got = H.eval_stat(_dev(torch_cuda, base["particles"]), e).cpu().numpy()
    assert rel_err(got, ref).max() <= TOL
    H.close()


# ---------------------------------------------------------------------------------------------- north_star identities on the GPU
def test_noise_free_exact_match_gives_rho_squared(oracle, torch_cuda, sc):
    """d = kappa h(theta_inj), no noise: Upsilon_N(theta_inj) = rho^2 for N = 1 and every refinement."""
    inp = sy.config_inputs(1, P=1)
    cfg = oracle.make_config(inp["cfg"])
    th = inp["injections"][0]["theta"]
    hA, hE, _ = oracle.template(cfg, th)
    rho = 20.0
    kappa = rho / np.sqrt(oracle.inner(hA, hE, hA, hE, inp["S_A"], inp["S_E"], inp["df"]))
    H = gpu_handle(inp, kappa * hA, kappa * hE)
    for N in (1, 10, 1000):
        got = H.eval_stat(_dev(torch_cuda, th[None, :]), sy.edges(cfg.n_bins, N)).cpu().numpy()[0]
        assert got == pytest.approx(rho ** 2, rel=TOL)
    H.close()


# ---------------------------------------------------------------------------------------------- PSO
def _pso_state(torch, pos, vel, S):
    P = pos.shape[0]
    return dict(pos=_dev(torch, pos), vel=_dev(torch, vel), pbest_pos=_dev(torch, pos + 0.0),
                pbest_val=torch.full((P,), -np.inf, dtype=torch.float64, device="cuda:0"),
                gbest_pos=torch.zeros((S, 8), dtype=torch.float64, device="cuda:0"),
                gbest_val=torch.zeros(S, dtype=torch.float64, device="cuda:0"))


@pytest.mark.parametrize("P,S", [(64, 1), (4000, 4), (40000, 4), (10007, 1)])
def test_pso_step_parity(c1, oracle, torch_cuda, P, S):
    H = c1["H"]
    rng = np.random.default_rng(P)
    lo, hi = c1["inp"]["lo"], c1["inp"]["hi"].copy()
    hi[7] = 0.1
    pos = lo + (hi - lo) * rng.random((P, 8))
    vel = (hi - lo) * rng.uniform(-0.4, 0.4, (P, 8))           # large velocities: the boundary rule fires often
    eps = np.array([0.1, 0.05, 0.0, 0.1, 0.1, 0.2, 0.1, 0.1]) * 0.1
    st = _pso_state(torch_cuda, pos, vel, S)
    o = dict(pos=pos.copy(), vel=vel.copy(), pbp=pos.copy(), pbv=np.full(P, -np.inf), gp=np.zeros((S, 8)), gv=np.zeros(S))
    for it in range(3):
        stat = np.round(rng.normal(100, 10, P), 0)              # rounded: many exact ties
        H.pso_step(st, _dev(torch_cuda, stat), _dev(torch_cuda, lo), _dev(torch_cuda, hi), _dev(torch_cuda, eps),
                   0.5, 0.2, 0.3, 12345678901234567, it, S)
        oracle.pso_step(o["pos"], o["vel"], o["pbp"], o["pbv"], stat, o["gp"], o["gv"], lo, hi, eps, 0.5, 0.2, 0.3,
                        12345678901234567, it, S)
        assert np.array_equal(st["pbest_val"].cpu().numpy(), o["pbv"])
        assert np.array_equal(st["pbest_pos"].cpu().numpy(), o["pbp"])
        assert np.array_equal(st["gbest_val"].cpu().numpy(), o["gv"])
        assert np.array_equal(st["gbest_pos"].cpu().numpy(), o["gp"])          # arg max incl. lowest-index tie rule
        # Eq. 13-15: identical uniforms (bit-equal Philox) and the same association -> <= 1e-13 relative
        span = hi - lo + 1e-300
        assert (np.abs(st["pos"].cpu().numpy() - o["pos"]) / span).max() <= 1e-13
        assert (np.abs(st["vel"].cpu().numpy() - o["vel"]) / span).max() <= 1e-13


@pytest.mark.parametrize("P,S,shards", [(10000, 1, 2), (40000, 4, 2), (4096, 1, 8), (600, 2, 3)])
def test_pso_step_sharded_is_bit_identical(c1, torch_cuda, P, S, shards):
    """every swarm cut into `shards` contiguous pieces (one per rank), evaluated piece by piece with
    sc_pso_best -> (all-gather, here a concatenation on one GPU) -> sc_pso_pick -> sc_pso_move: personal bests, swarm
    bests, positions and velocities are BIT-identical to one sc_pso_step on the whole population (global indices break
    ties and are the Philox counters).  Three iterations with many exact ties in the statistic."""
    from paper_2408_13170_b200 import dist as scd
    H = c1["H"]
    rng = np.random.default_rng(100 + P)
    lo, hi = c1["inp"]["lo"], c1["inp"]["hi"].copy()
    hi[7] = 0.1
    pos = lo + (hi - lo) * rng.random((P, 8))
    vel = (hi - lo) * rng.uniform(-0.4, 0.4, (P, 8))
    eps = np.array([0.1, 0.05, 0.0, 0.1, 0.1, 0.2, 0.1, 0.1]) * 0.1
    d = lambda a: _dev(torch_cuda, a)
    whole = _pso_state(torch_cuda, pos, vel, S)
    per, piece = P // S, P // S // shards
    # "rank" r = (swarm s, piece k) owns particles [s per + k piece, s per + (k+1) piece)
    ranks = []
    for s_ in range(S):
        for k in range(shards):
            a = s_ * per + k * piece
            ranks.append(dict(a=a, swarm=s_, st=_pso_state(torch_cuda, pos[a:a + piece], vel[a:a + piece], 1)))
    args = (d(lo), d(hi), d(eps), 0.5, 0.2, 0.3, 12345678901234567)
    for it in range(3):
        stat = np.round(rng.normal(100, 3, P), 0)                 # rounded: many exact ties, also across shards
        H.pso_step(whole, d(stat), *args, it, S)
        cands = []
        for r in ranks:
            c = torch_cuda.empty((1, 10), dtype=torch_cuda.float64, device="cuda:0")
            H.pso_best(r["st"], d(stat[r["a"]:r["a"] + piece]), c, 1, r["a"])
            cands.append(c)
        for r in ranks:
            allc = torch_cuda.stack([c for c, q in zip(cands, ranks) if q["swarm"] == r["swarm"]])     # the all-gather
            H.pso_pick(allc, r["st"])
            H.pso_move(r["st"], *args, it, 1, r["a"])
        for key in ("pos", "vel", "pbest_pos", "pbest_val"):
            got = torch_cuda.cat([r["st"][key] for r in ranks]).cpu().numpy()
            assert np.array_equal(got, whole[key].cpu().numpy()), (key, it)
        for r in ranks:
            assert np.array_equal(r["st"]["gbest_val"].cpu().numpy(), whole["gbest_val"][r["swarm"]:r["swarm"] + 1].cpu().numpy())
            assert np.array_equal(r["st"]["gbest_pos"].cpu().numpy(), whole["gbest_pos"][r["swarm"]:r["swarm"] + 1].cpu().numpy())
    # the same through dist.pso_step_sharded without a process group (one shard = the whole population)
    one = _pso_state(torch_cuda, pos, vel, S)
    ref = _pso_state(torch_cuda, pos, vel, S)
    stat = d(np.round(rng.normal(100, 3, P), 0))
    scd.pso_step_sharded(H, one, stat, *args, 9, S, 0)
    H.pso_step(ref, stat, *args, 9, S)
    for key in ("pos", "vel", "pbest_pos", "pbest_val", "gbest_pos", "gbest_val"):
        assert np.array_equal(one[key].cpu().numpy(), ref[key].cpu().numpy()), key


def test_pso_uniforms_bit_equal(c1, oracle, torch_cuda):
    """omega = phi_p = 0, phi_g = 1, pos = 0, gbest = 1 in every dimension: the new position IS r_G (Q10)."""
    H = c1["H"]
    P = 257
    z = np.zeros((P, 8))
    st = _pso_state(torch_cuda, z, z, 1)
    st["pbest_pos"] = _dev(torch_cuda, np.ones((P, 8)))
    st["pbest_val"] = _dev(torch_cuda, np.full(P, 5.0))
    lo, hi = np.full(8, -10.0), np.full(8, 10.0)
    H.pso_step(st, _dev(torch_cuda, np.zeros(P)), _dev(torch_cuda, lo), _dev(torch_cuda, hi), _dev(torch_cuda, np.zeros(8)),
               0.0, 0.0, 1.0, 987654321, 77, 1)
    got = st["pos"].cpu().numpy()
    for p in (0, 1, 100, 256):
        _, rG = oracle.pso_uniforms(987654321, p, 77)
        assert np.array_equal(got[p], rG)


def test_device_resident_search_improves_best(c1, torch_cuda, sc):
    """A short device-resident loop (eval + PSO, no host round trip) on config 1: the swarm best never decreases and
    ends above the initial best (trajectory parity with the oracle is not required: arg-max flips amplify 1e-6)."""
    inp, H = c1["inp"], c1["H"]
    e = inp["edges"][1000]
    st = _pso_state(torch_cuda, inp["particles"], inp["velocities"], 1)
    lo, hi, eps = (_dev(torch_cuda, a) for a in (inp["lo"], inp["hi"], np.zeros(8)))
    stat = torch_cuda.empty(64, dtype=torch_cuda.float64, device="cuda:0")
    best = []
    for it in range(12):
        H.eval_stat(st["pos"], e, out=stat)
        H.pso_step(st, stat, lo, hi, eps, 0.7, 1.5, 1.5, inp["pso_seed"], it, 1)
        best.append(st["gbest_val"].item())
    assert all(b >= a for a, b in zip(best, best[1:])) and best[-1] >= best[0]
    pos = st["pos"].cpu().numpy()
    assert np.all(pos >= inp["lo"]) and np.all(pos <= inp["hi"])


# ---------------------------------------------------------------------------------------------- per-particle segments
def _check_adaptive(oracle, cfg, dA, dE, inp, parts, N, got, ged, comp=None, exact=True):
    """PAPER.md:120 segments.  Floating point decides the integer edges, and both sides take the decision in FP64: the
    device's edges must EQUAL the oracle's (sco_equal_snr_edges) -- everywhere when `exact`, else in >= 99.9 % of the edges
    and never more than one bin away (a cumulative sum within the interpolation error, ~1e-12 relative, of its target may
    fall on the other side: probability ~1e-12 x n_bins per edge).  The statistic is then compared with the oracle evaluated
    on the device's edges (sco_eval_stat_adaptive in_edges), which are the oracle's own wherever they agree."""
    nb = inp["cfg"]["n_bins"]
    ref_own, oed = oracle.eval_stat_adaptive(cfg, dA, dE, inp["S_A"], inp["S_E"], parts, N, want_edges=True)
    assert np.all(ged[:, 0] == 0) and np.all(ged[:, -1] == nb) and np.all(np.diff(ged, axis=1) >= 0)
    d = np.abs(ged.astype(np.int64) - oed)
    if exact:
        assert np.array_equal(ged.astype(np.int64), oed), (int(d.max()), float((d != 0).mean()))
    else:
        assert d.max() <= 1 and (d == 0).mean() >= 0.999, (int(d.max()), float((d != 0).mean()))
    ref, rc = oracle.eval_stat_adaptive(cfg, dA, dE, inp["S_A"], inp["S_E"], parts, N, in_edges=ged, want_comp=True)
    assert rel_err(got, ref).max() <= TOL, (N, rel_err(got, ref).max())
    # moving an edge by one bin changes Upsilon by O(1/bins-per-segment): the two choices give nearby statistics
    assert np.all(np.abs(got - ref_own) <= 0.05 * np.maximum(ref_own, 1.0))
    if comp is not None:
        assert rel_err(comp[:, 0], ref).max() <= TOL
        assert rel_err(comp[:, 1], rc[:, 1]).max() <= TOL and rel_err(comp[:, 2], rc[:, 2]).max() <= TOL


@pytest.mark.parametrize("N", [2, 10, 50, 100, 1000])
def test_c1_adaptive_segments(c1, oracle, torch_cuda, sc, N):
    inp, H = c1["inp"], c1["H"]
    parts = inp["particles"]
    got, ged, comp = H.eval_stat_adaptive(_dev(torch_cuda, parts), N, want_edges=True, want_comp=True)
    _check_adaptive(oracle, c1["cfg"], c1["dA"], c1["dE"], inp, parts, N, got.cpu().numpy(), ged.cpu().numpy(), comp.cpu().numpy())
    # each segment holds C/N of the template's squared SNR to within one bin (the definition, checked on the device's
    # own per-segment sums): sigma_k of the GPU components sum to <h|h>
    got2 = H.eval_stat_adaptive(_dev(torch_cuda, parts), N).cpu().numpy()
    assert np.array_equal(got2, got.cpu().numpy())                # deterministic; edges output does not change the result


def test_c1_adaptive_single_segment_and_invalid(c1, oracle, torch_cuda, sc):
    inp, H = c1["inp"], c1["H"]
    nb = inp["cfg"]["n_bins"]
    par = _dev(torch_cuda, inp["particles"])
    got, ged = H.eval_stat_adaptive(par, 1, want_edges=True)
    assert np.array_equal(got.cpu().numpy(), H.eval_stat(par, np.array([0, nb])).cpu().numpy())
    assert np.array_equal(ged.cpu().numpy(), np.tile([0, nb], (len(inp["particles"]), 1)))
    p = inp["particles"][:5].copy()
    p[0, 1] = 0.3; p[1, 2] = -5e8                                 # invalid eta; t_c far before the data: empty window
    got, ged = H.eval_stat_adaptive(_dev(torch_cuda, p), 10, want_edges=True)
    got, ged = got.cpu().numpy(), ged.cpu().numpy()
    assert got[0] == 0.0 and got[1] == 0.0 and np.all(got[2:] > 0)
    assert np.array_equal(ged[0], [0] * 10 + [nb]) and np.array_equal(ged[1], [0] * 10 + [nb])   # the oracle's convention
    with pytest.raises(sc.SCError):
        H.eval_stat_adaptive(par, 0)


def test_adaptive_noise_free_match_and_equal_shares(oracle, torch_cuda, sc):
    """d = kappa h(theta_inj): Upsilon_N = rho^2 on the particle's own equal-SNR^2 segments, and every segment holds
    rho^2/N of it to within one bin's contribution."""
    inp = sy.config_inputs(1, P=1)
    cfg = oracle.make_config(inp["cfg"])
    th = inp["injections"][0]["theta"]
    hA, hE, _ = oracle.template(cfg, th)
    rho = 20.0
    kappa = rho / np.sqrt(oracle.inner(hA, hE, hA, hE, inp["S_A"], inp["S_E"], inp["df"]))
    H = gpu_handle(inp, kappa * hA, kappa * hE)
    s = 4 * inp["df"] * kappa ** 2 * (np.abs(hA) ** 2 / inp["S_A"] + np.abs(hE) ** 2 / inp["S_E"])
    for N in (10, 100):
        got, ged = H.eval_stat_adaptive(_dev(torch_cuda, th[None, :]), N, want_edges=True)
        assert got.item() == pytest.approx(rho ** 2, rel=TOL)
        e = ged.cpu().numpy()[0]
        share = np.add.reduceat(s, e[:-1])[: N]
        assert np.abs(share - rho ** 2 / N).max() <= 2.5 * s.max()
    H.close()


def test_c3_adaptive_bench_configuration(oracle, torch_cuda, sc):
    """Config 3 population (10^4 particles, 1.64 M bins) in the launch configuration bench.py times, N = 100 (the first
    rung of the paper's ladder): sampled particles against the oracle."""
    inp = sy.config_inputs(3)
    cfg, dA, dE = make_data(oracle, inp)
    H = gpu_handle(inp, dA, dE)
    H.set_option(sc.SC_OPT_TC_MAX_S, int(np.ceil(inp["hi"][2])))
    P = inp["particles"].shape[0]
    idx = _sample_idx(P, 32, 33)
    N = 100
    got, ged = H.eval_stat_adaptive(_dev(torch_cuda, inp["particles"]), N, want_edges=True)
    got, ged = got.cpu().numpy(), ged.cpu().numpy()
    _check_adaptive(oracle, cfg, dA, dE, inp, inp["particles"][idx], N, got[idx], ged[idx], exact=False)
    assert np.all(np.isfinite(got)) and np.all(got >= 0)
    assert np.all(np.diff(ged, axis=1) >= 0) and np.all(ged[:, -1] == inp["cfg"]["n_bins"])
    H.close()


def test_c5_adaptive_short_windows(oracle, torch_cuda, sc):
    """Per-particle segments on c5's short, scattered time windows: the window sort, the empty-CTA exits, the skipped node
    blocks and the windowed stitch of the adaptive path.  A sample against the oracle (edges equal, statistic to 1e-6);
    sort on / off over the whole population: same edges, and where every edge agrees the same statistic to FP32 rounding."""
    inp = sy.config_inputs(5, P=1280)
    cfg, dA, dE = make_data(oracle, inp)
    H = gpu_handle(inp, dA, dE)
    H.set_option(sc.SC_OPT_TC_MAX_S, int(np.ceil(inp["hi"][2])))
    par = _dev(torch_cuda, inp["particles"])
    idx = _sample_idx(1280, 24, 77)
    N = 50
    res = {}
    for srt in (1, 0):
        H.set_option(sc.SC_OPT_WINDOW_SORT, srt)
        g, e = H.eval_stat_adaptive(par, N, want_edges=True)
        res[srt] = (g.cpu().numpy(), e.cpu().numpy())
    H.close()
    (a, ea), (b, eb) = res[1], res[0]
    _check_adaptive(oracle, cfg, dA, dE, inp, inp["particles"][idx], N, a[idx], ea[idx], exact=False)
    assert np.abs(ea - eb).max() <= 1 and (ea == eb).mean() >= 0.9999          # the FP64 decision does not depend on the order
    same = np.all(ea == eb, axis=1) & (b > 0)
    assert same.sum() > 1200
    assert rel_err(a[same], b[same]).max() <= 2e-7
    assert np.all(np.diff(ea, axis=1) >= 0) and np.all(ea[:, -1] == inp["cfg"]["n_bins"]) and np.all(ea[:, 0] == 0)


def test_node_spacing_error_model(oracle, torch_cuda, sc):
    """with the coarse node spacing forced (all-FP64 kernels, so nothing but the interpolation shows), the
    error of Upsilon stays below K days^6 / sqrt(N') -- days = signal time per coarse interval at the slowest-chirping corner,
    N' = segments inside the window, K = 7.5e-10 (N' = 1) and 1.4e-10 (N' >= 8) as measured -- which is what the spacing rules
    (2 days all-FP64, 4 (N'/8)^(1/12) days FP32 amplitudes) are derived from.  c5: every window sits at that corner."""
    inp = sy.config_inputs(5, P=160)
    cfg, dA, dE = make_data(oracle, inp)
    par = _dev(torch_cuda, inp["particles"])
    nb, T = inp["cfg"]["n_bins"], inp["cfg"]["T_obs_s"]
    tc_max = float(np.ceil(inp["hi"][2]))
    s_per_bin = (8.0 / 3.0) * tc_max / ((inp["cfg"]["j0"] / T) * T)
    levels = [1, 5000, 50000]
    edges = [sy.edges(nb, N) for N in levels]
    ref = oracle.eval_stat_levels(oracle.make_config(inp["cfg"], truth=True), dA, dE, inp["S_A"], inp["S_E"], inp["particles"], edges)
    worst = {}
    for lg in (7, 8, 9):
        H = gpu_handle(inp, dA, dE)
        H.set_option(sc.SC_OPT_TC_MAX_S, int(tc_max))
        H.set_option(sc.SC_OPT_STRIDE_LOG2, lg)
        H.set_option(sc.SC_OPT_PRECISION, 2)
        days = (1 << lg) * s_per_bin / 86400.0
        for N, e, r in zip(levels, edges, ref):
            got = H.eval_stat(par, e).cpu().numpy()
            phi = H.counters()[0] / (len(r) * nb)
            live = r > 0
            n_eff = max(1.0, N * phi)
            K = 7.5e-10 if N == 1 else 1.4e-10
            worst[(lg, N)] = rel_err(got[live], r[live]).max()
            assert worst[(lg, N)] <= 2.0 * K * days ** 6 / np.sqrt(n_eff) + 2e-9, (lg, N, days, n_eff, worst[(lg, N)])
        H.close()
    assert worst[(9, 1)] > 50 * worst[(7, 1)]             # ~ days^6: the model is not vacuous


@pytest.mark.parametrize("N,prec", [(1, 0), (100, 0), (2000, 0), (2000, 2)])
def test_c2_components_many_chunks(oracle, torch_cuda, sc, N, prec):
    """Eq. 8 / Eq. 3 on c2 (123 chunks of 2048 bins, 247 of 1024: the chunk walk of a particle is folded in parts by k_stitch_parts /
    k_stitch_join, with the partial sums of |z_k| and sigma_k) against the oracle's segments, 24 particles."""
    inp = sy.config_inputs(2, P=24)
    cfg, dA, dE = make_data(oracle, inp)
    H = gpu_handle(inp, dA, dE)
    H.set_option(sc.SC_OPT_TC_MAX_S, int(np.ceil(inp["hi"][2])))
    H.set_option(sc.SC_OPT_PRECISION, prec)
    e = sy.edges(inp["cfg"]["n_bins"], N)
    ref, refseg = oracle.eval_stat(oracle.make_config(inp["cfg"], truth=True), dA, dE, inp["S_A"], inp["S_E"], inp["particles"], e, want_seg=True)
    comp_ref = np.array([oracle.components_from_seg(s, inp["df"]) for s in refseg])
    par = _dev(torch_cuda, inp["particles"])
    comp = H.eval_components(par, e).cpu().numpy()
    live = ref > 0
    assert live.sum() >= 12 and np.array_equal(comp[:, 0] == 0, ~live)
    assert rel_err(comp[live, 0], ref[live]).max() <= TOL
    assert np.array_equal(comp[:, 0], H.eval_stat(par, e).cpu().numpy())      # same kernels, same order
    assert rel_err(comp[live, 1], comp_ref[live, 1]).max() <= TOL
    assert rel_err(comp[live, 2], comp_ref[live, 2]).max() <= TOL
    H.close()
