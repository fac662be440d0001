"""sc_kmeans_static (`-m gpu`): the allocation-free variant of sc_kmeans -- scratch in a file-scope static device array of the
library -- against the existing path.  Same kernels on the same inputs: labels, counts and iteration counts must be equal and
the centroids bit-equal (the bar test_gpu_search.py holds sc_kmeans to against the oracle).  Two calls in a row: the array is
shared and keeps the previous call's contents.  Collected last on purpose (the suite runs with pytest -x)."""
import numpy as np
import pytest

import sc_synth as sy

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def env():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    import paper_2408_13170_b200 as sc
    sc.load_library()          # fails loudly if the extension is missing
    inp = sy.config_inputs(1)
    t = lambda a: torch.from_numpy(np.ascontiguousarray(a)).to("cuda:0")
    H = sc.Handle(inp["cfg"], torch.view_as_real(t(inp["noise_A"])).contiguous(), torch.view_as_real(t(inp["noise_E"])).contiguous(),
                  t(inp["S_A"]), t(inp["S_E"]))
    yield torch, sc, H, inp, t
    H.close()


def _problem(inp, seed, P, K):
    """Particles in K blobs inside the prior box (plus a uniform background), initial centroids = K of the particles."""
    rng = np.random.default_rng(seed)
    lo, hi = inp["lo"], inp["hi"]
    centres = lo + rng.uniform(0.1, 0.9, size=(K, 8)) * (hi - lo)
    which = rng.integers(0, K, size=P)
    pos = centres[which] + 0.04 * rng.standard_normal((P, 8)) * (hi - lo)
    bg = rng.random(P) < 0.2
    pos[bg] = lo + rng.random((int(bg.sum()), 8)) * (hi - lo)
    pos = np.clip(pos, lo, hi)
    cent0 = pos[rng.choice(P, K, replace=False)].copy()
    return pos, cent0


def _run(torch, sc, H, t, fn, pos, cent0, lo, hi, max_iter):
    P, K = pos.shape[0], cent0.shape[0]
    cent = t(cent0.copy())
    label = torch.full((P,), 12345, dtype=torch.int32, device="cuda:0")
    count = torch.full((K,), -7, dtype=torch.int64, device="cuda:0")
    dpos = t(pos)
    torch.cuda.synchronize()
    free0 = torch.cuda.mem_get_info()[0]                    # inputs and outputs exist: what changes now is the call's own
    it = fn(H.h, dpos, P, lo, hi, cent, K, max_iter, label, count)
    torch.cuda.synchronize()
    grabbed = free0 - torch.cuda.mem_get_info()[0]
    return it, label.cpu().numpy(), count.cpu().numpy(), cent.cpu().numpy(), grabbed


def test_static_scratch_variant_matches_sc_kmeans_on_two_calls_in_a_row(env):
    torch, sc, H, inp, t = env
    lo, hi = t(inp["lo"]), t(inp["hi"])
    # the second call is smaller in P and K than the first and stops on max_iter: whatever the first left in the array
    # (a non-zero "changed" counter, counts of clusters the second call does not have) must not leak into it
    cases = [(11, 6000, 7, 100), (12, 777, 3, 2), (13, 4097, sc.SC_KMEANS_STATIC_MAX_K, 100)]
    for i, (seed, P, K, max_iter) in enumerate(cases):
        pos, cent0 = _problem(inp, seed, P, K)
        got = _run(torch, sc, H, t, sc.sc_kmeans_static, pos, cent0, lo, hi, max_iter)
        if i > 0:              # (the very first call on a device may load the module lazily)
            assert got[4] <= 0, got[4]                     # the call took no device memory
        want = _run(torch, sc, H, t, sc.sc_kmeans, pos, cent0, lo, hi, max_iter)
        assert got[0] == want[0] and 1 <= got[0] <= max_iter, (seed, got[0], want[0])
        assert np.array_equal(got[1], want[1]) and got[1].min() >= 0 and got[1].max() < K
        assert np.array_equal(got[2], want[2]) and got[2].sum() == P
        assert np.array_equal(got[3], want[3])                             # same kernels, same order: bit-equal centroids
        assert np.array_equal(got[2], np.bincount(got[1], minlength=K))    # counts are those of the labels
        # and the definition: every label is a nearest centroid of the LAST assignment step's input ... after convergence
        # (max_iter not hit) the centroids are the member means
        if got[0] < max_iter:
            for k in range(K):
                if got[2][k]:
                    assert np.allclose(got[3][k], pos[got[1] == k].mean(axis=0), rtol=1e-12, atol=0)


def test_sizes_beyond_the_static_array_are_rejected(env):
    torch, sc, H, inp, t = env
    K = sc.SC_KMEANS_STATIC_MAX_K + 1
    pos, cent0 = _problem(inp, 5, 1000, K)
    label = torch.empty(1000, dtype=torch.int32, device="cuda:0")
    with pytest.raises(sc.SCError) as ei:
        sc.sc_kmeans_static(H.h, t(pos), 1000, t(inp["lo"]), t(inp["hi"]), t(cent0), K, 10, label)
    assert "SC_KMEANS_STATIC_MAX_K" in str(ei.value)
    # the handle stays usable
    pos, cent0 = _problem(inp, 6, 500, 4)
    it = sc.sc_kmeans_static(H.h, t(pos), 500, t(inp["lo"]), t(inp["hi"]), t(cent0), 4, 50, label[:500].contiguous())
    assert it >= 1
