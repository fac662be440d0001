"""Pins for the oracle's PSO step and its counter-based RNG (sco_philox4x32_10, sco_pso_uniforms, sco_pso_step) -- O7/Q9/Q10.

Eq. 13-15 are checked on hand-computed one-particle examples; the RNG against the published
algorithm's known-answer vectors and its moments.
"""
import json
import os

import numpy as np
import pytest

GOLD = json.load(open(os.path.join(os.path.dirname(__file__), "golden", "paper_values.json")))


def test_philox_known_answers(oracle):
    for case in GOLD["philox4x32_10_kat"]["cases"]:
        got = oracle.philox4x32_10([int(x, 16) for x in case["ctr"]], [int(x, 16) for x in case["key"]])
        assert got == [int(x, 16) for x in case["out"]]


def test_uniform_mapping_and_moments(oracle):
    """Q10: counter = (particle, iter, block 0..3, 0), key = seed; u = (word + 0.5) 2^-32 in (0,1), 16 per (particle, iter)."""
    seed, p, it = 0x0123456789ABCDEF, 77, 5
    rP, rG = oracle.pso_uniforms(seed, p, it)
    words = []
    for b in range(4):
        words += oracle.philox4x32_10([p, it, b, 0], [seed & 0xFFFFFFFF, seed >> 32])
    assert np.array_equal(rP, (np.array(words[:8], dtype=np.float64) + 0.5) / 2.0 ** 32)
    assert np.array_equal(rG, (np.array(words[8:], dtype=np.float64) + 0.5) / 2.0 ** 32)
    u = np.concatenate([np.concatenate(oracle.pso_uniforms(42, q, i)) for q in range(400) for i in range(5)])
    assert u.min() > 0.0 and u.max() < 1.0
    assert u.mean() == pytest.approx(0.5, abs=4 / np.sqrt(12 * len(u)))
    assert u.var() == pytest.approx(1 / 12, rel=0.03)
    # independence across particle / iteration / dimension: lag correlations vanish
    m = u.reshape(-1, 16)
    c = np.corrcoef(m.T)
    assert np.abs(c - np.eye(16)).max() < 0.1
    assert not np.array_equal(oracle.pso_uniforms(42, 1, 0)[0], oracle.pso_uniforms(42, 0, 1)[0])
    assert not np.array_equal(oracle.pso_uniforms(42, 1, 0)[0], oracle.pso_uniforms(43, 1, 0)[0])


def _one(oracle, pos, vel, pbest_pos, pbest_val, stat, lo, hi, eps, omega, php, phg, seed=1, it=0, n_swarms=1):
    pos, vel, pbp = (np.array(a, dtype=np.float64).reshape(-1, 8).copy() for a in (pos, vel, pbest_pos))
    pbv = np.array(pbest_val, dtype=np.float64).copy()
    gp = np.zeros((n_swarms, 8))
    gv = np.full(n_swarms, -np.inf)
    oracle.pso_step(pos, vel, pbp, pbv, np.array(stat, dtype=np.float64), gp, gv, lo, hi, eps, omega, php, phg, seed, it, n_swarms)
    return pos, vel, pbp, pbv, gp, gv


def test_hand_computed_single_particle(oracle):
    """One particle: Xi = Psi = its own best, so u = Omega v + (Phi_P r_P + Phi_G r_G)(Psi - theta)  (Eq. 14)."""
    lo, hi = np.full(8, -100.0), np.full(8, 100.0)
    eps = np.zeros(8)
    pos = np.arange(8.0)
    vel = np.full(8, 0.5)
    pb = pos + 2.0
    rP, rG = oracle.pso_uniforms(9, 0, 3)
    # stat below the stored best: the best stays where it was
    p, v, pbp, pbv, gp, gv = _one(oracle, pos, vel, pb, [10.0], [3.0], lo, hi, eps, 0.7, 1.5, 1.25, seed=9, it=3)
    u = 0.7 * 0.5 + 1.5 * rP * 2.0 + 1.25 * rG * 2.0
    assert np.allclose(v[0], u, rtol=1e-15, atol=0) and np.allclose(p[0], pos + u, rtol=1e-15)
    assert pbv[0] == 10.0 and np.array_equal(pbp[0], pb) and gv[0] == 10.0 and np.array_equal(gp[0], pb)
    # stat above the stored best (strict): the best moves to the current position BEFORE Eq. 14, so u = Omega v
    p, v, pbp, pbv, gp, gv = _one(oracle, pos, vel, pb, [10.0], [11.0], lo, hi, eps, 0.7, 1.5, 1.25, seed=9, it=3)
    assert np.array_equal(v[0], np.full(8, 0.35)) and np.array_equal(pbp[0], pos) and pbv[0] == 11.0 and gv[0] == 11.0
    # equality is not an improvement
    *_, pbp, pbv, gp, gv = _one(oracle, pos, vel, pb, [10.0], [10.0], lo, hi, eps, 0.7, 1.5, 1.25)
    assert np.array_equal(pbp[0], pb)


def test_minimum_velocity_clamp_and_zero(oracle):
    """Eq. 15: v = max(eps, |u|) u/|u|; Q9: u = 0 -> +eps (or 0 if eps = 0)."""
    lo, hi = np.full(8, -100.0), np.full(8, 100.0)
    pos = np.zeros(8)
    vel = np.array([0.01, -0.01, 1.0, -1.0, 0.0, 0.0, 0.3, -0.3])
    eps = np.array([0.1, 0.1, 0.1, 0.1, 0.1, 0.0, 0.3, 0.5])
    # Phi_P = Phi_G = 0 and Omega = 1: u = v exactly
    p, v, *_ = _one(oracle, pos, vel, pos, [0.0], [-1.0], lo, hi, eps, 1.0, 0.0, 0.0)
    assert np.array_equal(v[0], np.array([0.1, -0.1, 1.0, -1.0, 0.1, 0.0, 0.3, -0.5]))
    assert np.array_equal(p[0], v[0])


def test_reflecting_boundary(oracle):
    """Q9: clamp to [lo, hi] and reverse that component's velocity."""
    lo, hi = np.zeros(8), np.ones(8)
    pos = np.array([0.9, 0.1, 0.5, 0.5, 1.0, 0.0, 0.5, 0.5])
    vel = np.array([0.3, -0.3, 0.3, -0.3, 0.2, -0.2, 0.5, -0.5])
    p, v, *_ = _one(oracle, pos, vel, pos, [0.0], [-1.0], lo, hi, np.zeros(8), 1.0, 0.0, 0.0)
    assert np.array_equal(p[0], np.array([1.0, 0.0, 0.8, 0.2, 1.0, 0.0, 1.0, 0.0]))
    assert np.array_equal(v[0], np.array([-0.3, 0.3, 0.3, -0.3, -0.2, 0.2, 0.5, -0.5]))


def test_swarm_best_bookkeeping(oracle):
    """Per-swarm arg max over personal bests, lowest index on ties; swarms are equal contiguous blocks; synchronous:
    Eq. 14 uses the bests of iteration i-1 inputs (updated with this call's stat) for every particle alike."""
    P, S = 12, 3
    rng = np.random.default_rng(0)
    pos = rng.uniform(0.2, 0.8, (P, 8))
    vel = np.zeros((P, 8))
    pbp = pos.copy() + 0.01
    pbv = np.array([1, 5, 5, 2, 9, 3, 3, 9.5, 0, 0, 0, 0], dtype=float)
    stat = np.array([0, 0, 7, 0, 0, 0, 0, 0, -1, -1, -1, -1], dtype=float)
    gp, gv = np.zeros((S, 8)), np.full(S, -np.inf)
    lo, hi = np.zeros(8), np.ones(8)
    pos0 = pos.copy()
    oracle.pso_step(pos, vel, pbp, pbv, stat, gp, gv, lo, hi, np.zeros(8), 0.0, 0.0, 1.0, 5, 0, S)
    assert list(gv) == [7.0, 9.5, 0.0]
    assert np.array_equal(gp[0], pos0[2])                 # particle 2 improved to 7 at its current position
    assert np.array_equal(gp[1], pos0[7] + 0.01)          # particle 7's stored best
    assert np.array_equal(gp[2], pos0[8] + 0.01)          # tie among 8..11 -> lowest index
    # Omega = Phi_P = 0, Phi_G = 1: every particle moved a fraction r_G of the way to ITS swarm's best
    for p in range(P):
        _, rG = oracle.pso_uniforms(5, p, 0)
        want = pos0[p] + rG * (gp[p // 4] - pos0[p])
        assert np.allclose(pos[p], want, rtol=1e-15, atol=1e-18)


def test_table_iv_rows_are_the_papers(oracle):
    import sc_synth as sy
    for N, row in GOLD["table_IV"]["rows"].items():
        h = sy.TABLE_IV[int(N)]
        assert [h["omega"], h["phi_p"], h["phi_g"]] == row
