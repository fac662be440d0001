"""Pins of the oracle's multi-swarm bookkeeping: labelled PSO step, k-means regrouping and the
convergence rule -- against hand-computed values, invariants and scikit-learn's Lloyd iterations."""
import numpy as np
import pytest


def _state(rng, P, S):
    lo = np.array([28.5, 0.15, 1.0e8, 0.0, -1.5, 0.0, -3.1, 0.0])
    hi = np.array([31.5, 0.2495, 1.2e8, 6.28, 1.5, 3.14, 0.0, 0.1])
    pos = lo + (hi - lo) * rng.random((P, 8))
    vel = (hi - lo) * rng.uniform(-0.3, 0.3, (P, 8))
    return lo, hi, pos, vel


def test_labeled_step_equals_block_step_for_contiguous_labels(oracle):
    rng = np.random.default_rng(1)
    P, S = 120, 4
    lo, hi, pos, vel = _state(rng, P, S)
    eps = np.array([0.1, 0.05, 0.0, 0.1, 0.1, 0.2, 0.1, 0.1]) * 0.01
    a = dict(pos=pos.copy(), vel=vel.copy(), pbp=pos.copy(), pbv=np.full(P, -np.inf), gp=np.zeros((S, 8)), gv=np.zeros(S))
    b = {k: v.copy() for k, v in a.items()}
    lab = np.repeat(np.arange(S, dtype=np.int32), P // S)
    for it in range(3):
        stat = np.round(rng.normal(50, 5, P))
        oracle.pso_step(a["pos"], a["vel"], a["pbp"], a["pbv"], stat, a["gp"], a["gv"], lo, hi, eps, 0.5, 0.2, 0.3, 99, it, S)
        oracle.pso_step_labeled(b["pos"], b["vel"], b["pbp"], b["pbv"], stat, b["gp"], b["gv"], lab, lo, hi, eps, 0.5, 0.2, 0.3, 99, it)
        for k in a:
            assert np.array_equal(a[k], b[k]), k


def test_labeled_step_scattered_membership_and_empty_swarm(oracle):
    """Hand-checkable case: omega = phi_p = 0, phi_g = 1, so v = r_G (gbest_of_own_swarm - theta) (Eq. 14)."""
    rng = np.random.default_rng(2)
    P, S = 9, 3
    lo, hi = np.full(8, -100.0), np.full(8, 100.0)
    pos = rng.normal(0, 1, (P, 8))
    lab = np.array([2, 0, 2, 0, 0, 2, 0, 2, 2], dtype=np.int32)          # swarm 1 is empty
    stat = np.array([5.0, 1.0, 7.0, 3.0, 3.0, 7.0, 2.0, 1.0, 0.0])
    st = dict(pos=pos.copy(), vel=np.zeros((P, 8)), pbp=pos.copy(), pbv=np.full(P, -np.inf), gp=np.full((S, 8), 42.0), gv=np.zeros(S))
    oracle.pso_step_labeled(st["pos"], st["vel"], st["pbp"], st["pbv"], stat, st["gp"], st["gv"], lab, lo, hi, np.zeros(8),
                            0.0, 0.0, 1.0, 7, 3)
    assert st["gv"][0] == 3.0 and np.array_equal(st["gp"][0], pos[3])     # tie 3.0 at particles 3 and 4: lowest index
    assert st["gv"][2] == 7.0 and np.array_equal(st["gp"][2], pos[2])     # tie 7.0 at particles 2 and 5
    assert st["gv"][1] == -np.inf and np.array_equal(st["gp"][1], np.full(8, 42.0))
    for p in range(P):
        _, rG = oracle.pso_uniforms(7, p, 3)
        g = pos[3] if lab[p] == 0 else pos[2]
        assert np.allclose(st["vel"][p], rG * (g - pos[p]), rtol=1e-15, atol=0)
        assert np.allclose(st["pos"][p], pos[p] + rG * (g - pos[p]), rtol=1e-15, atol=0)


def test_kmeans_hand_example_1d(oracle):
    """Only M_c varies: points 0,1,2 | 10,11,12 in a box of width 12 from centroids at 1.5 and 2.5:
    iteration 1: labels by nearest of (1.5, 2.5) -> {0,1,2(tie -> lowest k)} | {10,11,12}: 2 is equidistant (0.5 each):
    lowest k wins, so cluster 0 = {0,1,2}, cluster 1 = {10,11,12}; centroids 1 and 11; iteration 2: no change."""
    lo, hi = np.zeros(8), np.array([12.0, 0, 0, 0, 0, 0, 0, 0])
    pos = np.zeros((6, 8)); pos[:, 0] = [0, 1, 2, 10, 11, 12]
    cent = np.zeros((2, 8)); cent[:, 0] = [1.5, 2.5]
    lab, c, cnt, it = oracle.kmeans(pos, lo, hi, cent)
    assert list(lab) == [0, 0, 0, 1, 1, 1] and list(cnt) == [3, 3] and it == 2
    assert c[0, 0] == 1.0 and c[1, 0] == 11.0


def test_kmeans_recovers_separated_blobs_and_fixed_point(oracle):
    rng = np.random.default_rng(3)
    lo, hi, _, _ = _state(rng, 1, 1)
    K, per = 5, 400
    centres = lo + (hi - lo) * rng.uniform(0.15, 0.85, (K, 8))
    truth = np.repeat(np.arange(K), per)
    pos = centres[truth] + (hi - lo) * rng.normal(0, 0.004, (K * per, 8))
    perm = rng.permutation(K * per)
    pos, truth = pos[perm], truth[perm]
    init = centres + (hi - lo) * rng.normal(0, 0.02, (K, 8))
    lab, c, cnt, it = oracle.kmeans(pos, lo, hi, init)
    assert np.array_equal(lab, truth) and list(cnt) == [per] * K
    w = 1.0 / (hi - lo)
    d = (((pos[:, None, :] - c[None, :, :]) * w) ** 2).sum(-1)
    assert np.array_equal(d.argmin(1), lab)                                # nearest-centroid labels
    for k in range(K):
        assert np.allclose(c[k], pos[lab == k].mean(0), rtol=1e-13)        # centroids are the member means


def test_kmeans_objective_never_increases_and_matches_sklearn(oracle):
    sk = pytest.importorskip("sklearn.cluster")
    rng = np.random.default_rng(4)
    lo, hi, pos, _ = _state(rng, 3000, 1)
    pos[:1000] = lo + (hi - lo) * (0.3 + 0.05 * rng.normal(size=(1000, 8)))   # one dense clump in a uniform background
    pos = np.clip(pos, lo, hi)
    init = pos[rng.choice(3000, 6, replace=False)].copy()
    w = 1.0 / (hi - lo)
    prev = np.inf
    for mi in (1, 2, 3, 5, 8, 100):
        lab, c, cnt, it = oracle.kmeans(pos, lo, hi, init, max_iter=mi)
        # objective with the labels of iteration `it` and the centroids they produced
        J = ((((pos - c[lab]) * w) ** 2).sum())
        assert J <= prev * (1 + 1e-12)
        prev = J
    km = sk.KMeans(n_clusters=6, init=(init - lo) * w, n_init=1, algorithm="lloyd", max_iter=300, tol=0.0).fit((pos - lo) * w)
    assert np.array_equal(km.labels_, lab)
    assert np.allclose(km.cluster_centers_, (c - lo) * w, atol=1e-12)


def test_kmeans_ignores_degenerate_dimensions_and_keeps_empty_clusters(oracle):
    rng = np.random.default_rng(5)
    lo, hi, pos, _ = _state(rng, 200, 1)
    lo2, hi2 = lo.copy(), hi.copy()
    hi2[7] = lo2[7]                                                        # e_0 not searched: zero width
    pos[:, 7] = rng.normal(0, 1e6, 200)                                    # garbage there must not matter
    init = np.vstack([pos[:2], (hi + 10 * (hi - lo))[None, :]])            # third centroid far away: stays empty
    lab, c, cnt, it = oracle.kmeans(pos, lo2, hi2, init)
    pos0 = pos.copy(); pos0[:, 7] = 0.0
    init0 = init.copy(); init0[:, 7] = 0.0
    lab0, c0, cnt0, it0 = oracle.kmeans(pos0, lo2, hi2, init0)
    assert np.array_equal(lab, lab0) and cnt[2] == 0 and np.array_equal(c[2], init[2])


def test_convergence_rule(oracle):
    """converged if the best has not improved by more than 2 over 50 iterations."""
    h = np.concatenate([np.linspace(100, 200, 30), np.full(50, 200.0)])
    assert not oracle.converged(h[:50], 50, 2.0)                           # fewer than window + 1 entries
    assert not oracle.converged(h[:79], 50, 2.0)                           # 200 - h[28] = 3.4 > 2
    assert oracle.converged(h[:80], 50, 2.0)                               # 200 - h[29] = 0
    g = 100 + 0.05 * np.arange(200)                                        # creeping up by 2.5 per 50 iterations
    assert not oracle.converged(g, 50, 2.0) and oracle.converged(g, 50, 2.5)
