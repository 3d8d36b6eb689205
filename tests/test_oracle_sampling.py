"""Pins of the oracle's temperature / top-k sampler (dfo_sample; R23) -- the paper implies a generation loop but
gives no sampler, so the function is pinned by what the definition fixes: special cases that reduce to argmax, a closed form
for a flat distribution, the softmax probabilities themselves (float64 numpy) through a sweep of the uniform input, support
restricted to the top k, tie order, permutation equivariance, and an independent sort-based restatement."""
import numpy as np
import pytest


def test_greedy_special_cases(oracle_mod):
    g = np.random.default_rng(0)
    for _ in range(50):
        lg = g.standard_normal(97).astype(np.float32)
        lg[g.integers(0, 97, 3)] = lg.max()                       # ties for the maximum: the lowest index wins
        want = int(np.flatnonzero(lg == lg.max())[0])
        assert oracle_mod.sample(lg, 1.0, 1, 0.77) == want          # top_k = 1
        assert oracle_mod.sample(lg, 0.0, 8, 0.77) == want          # temperature <= 0
        assert oracle_mod.sample(lg, 0.7, 8, 0.0) == want           # u = 0 always picks rank 0
        assert oracle_mod.sample(lg, 0.7, 8, 0.3) in np.argsort(-lg, kind="stable")[:8]


def test_flat_distribution_closed_form(oracle_mod):
    # temperature -> infinity: every weight is exactly 1, c_r = r + 1, the pick is rank floor(u k)
    lg = np.array([3.0, -1.0, 2.5, 2.5, 0.0, 7.0, 1.0], np.float32)
    order = np.argsort(-lg, kind="stable")                           # value descending, index ascending
    k = 5
    for u in (0.0, 0.19, 0.2, 0.39999, 0.5, 0.79, 0.8, 0.999):
        assert oracle_mod.sample(lg, 1e30, k, u) == int(order[int(np.floor(np.float64(np.float32(u)) * k))]), u


def test_frequencies_are_the_softmax_probabilities(oracle_mod):
    g = np.random.default_rng(1)
    lg = (g.standard_normal(40) * 2).astype(np.float32)
    temperature, k, N = 0.8, 12, 20000
    order = np.argsort(-lg, kind="stable")[:k]
    p = np.exp((lg[order].astype(np.float64) - np.float64(lg[order[0]])) / temperature)
    p /= p.sum()
    counts = np.zeros(lg.size)
    for i in range(N):
        counts[oracle_mod.sample(lg, temperature, k, (i + 0.5) / N)] += 1
    assert counts[np.setdiff1d(np.arange(lg.size), order)].sum() == 0          # nothing outside the top k
    assert np.abs(counts[order] / N - p).max() <= 2.0 / N + 1e-5               # inverse-CDF sampling of exactly these probabilities
    # and in rank order: the picks are monotone in u
    picks = [int(np.flatnonzero(order == oracle_mod.sample(lg, temperature, k, (i + 0.5) / 200))[0]) for i in range(200)]
    assert picks == sorted(picks)


def test_against_sort_based_restatement_with_ties_and_permutation(oracle_mod):
    g = np.random.default_rng(2)

    def restated(lg, temperature, k, u):
        order = np.lexsort((np.arange(lg.size), -lg.astype(np.float64)))[:k]   # value descending, then index ascending
        d = ((lg[order] - lg[order[0]]).astype(np.float32) / np.float32(temperature)).astype(np.float32)
        w = np.array([oracle_mod.sp_expf(float(x)) for x in d], np.float64)
        c = np.cumsum(w)
        r = np.flatnonzero(c > np.float64(np.float32(u)) * c[-1])
        return int(order[r[0] if r.size else k - 1])

    for trial in range(200):
        n = int(g.integers(5, 200))
        lg = np.round(g.standard_normal(n) * 3, 1).astype(np.float32)           # rounded: plenty of ties
        k = int(g.integers(1, min(n, 64) + 1))
        temperature = float(g.uniform(0.2, 3.0))
        u = float(g.uniform(0, 1))
        got = oracle_mod.sample(lg, temperature, k, u)
        assert got == restated(lg, temperature, k, u), (trial, n, k, temperature, u)
    # permutation equivariance (distinct logits)
    lg = g.permutation(np.arange(64)).astype(np.float32) * 0.25
    perm = g.permutation(64)
    for u in (0.1, 0.5, 0.9):
        a = oracle_mod.sample(lg, 1.3, 10, u)
        b = oracle_mod.sample(lg[perm], 1.3, 10, u)
        assert perm[b] == a
