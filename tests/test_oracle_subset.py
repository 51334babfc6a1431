"""Pins of the oracle's stochastic viewgraph sub-sampling (Alg. 3 l.3-6; PAPER.md:500 A1.3:
"a fresh uniform random subset S of E of size min(|E|, M) ... a fresh subset is drawn every step").  None of
these re-types the oracle's own routine: the keys are checked against the scene generator's SplitMix64 class (an
independent implementation of the published generator), the subset against a brute-force rank count, and the
distribution against what "uniform" fixes."""
import numpy as np

import oracle
from epo_scenes import SplitMix64


def test_S0_keys_are_splitmix64_outputs():
    """key(0, p) is output number p + 1 of SplitMix64(seed); key(s, p) is output number s * 2^32 + p + 1."""
    for seed in (0, 1, 2607005790, 0xFFFFFFFFFFFFFFFF):
        ref = SplitMix64(seed).raw(64)
        got = [oracle.subset_key(seed, 0, p) for p in range(64)]
        assert got == [int(x) for x in ref]
        g = SplitMix64(seed); g.counter = 3 * 2 ** 32 + 10          # skip ahead: an explicit counter
        assert oracle.subset_key(seed, 3, 10) == int(g.raw(1)[0])
    assert SplitMix64(1234567).raw(1)[0] == np.uint64(6457827717110365317)   # published test vector of SplitMix64


def test_S1_subset_is_the_M_smallest_keys_brute_force():
    seed, P, M = 99, 300, 37
    for step in (0, 1, 17):
        keys = [oracle.subset_key(seed, step, p) for p in range(P)]
        rank = [sum((keys[q], q) < (keys[p], p) for q in range(P)) for p in range(P)]   # O(P^2), by definition
        want = np.array([r < M for r in rank])
        got = oracle.pair_subset(seed, step, P, M)
        assert got.sum() == M and np.array_equal(got, want)


def test_S2_size_rule_and_freshness():
    assert oracle.pair_subset(5, 0, 10, 1024).all()                 # |E| <= M: S = E (Alg. 3 l.5)
    assert oracle.pair_subset(5, 0, 10, 10).all()
    assert oracle.pair_subset(5, 0, 10, 0).all()                    # budget 0 = off
    a, b = oracle.pair_subset(5, 0, 5000, 1024), oracle.pair_subset(5, 1, 5000, 1024)
    assert a.sum() == b.sum() == 1024
    # two independent uniform 1024-subsets of 5000 share 1024^2/5000 = 210 elements on average (sd ~ 12)
    assert 140 <= int((a & b).sum()) <= 280
    assert not np.array_equal(a, oracle.pair_subset(6, 0, 5000, 1024))   # the seed matters
    assert np.array_equal(a, oracle.pair_subset(5, 0, 5000, 1024))       # a pure function of (seed, step)


def test_S3_uniform_inclusion_and_pair_independence():
    """Every pair is included with probability M/P (the estimator is unbiased) and inclusions of two
    pairs are those of sampling without replacement: P(both) = M(M-1)/(P(P-1))."""
    P, M, T = 200, 50, 4000
    inc = np.zeros(P); both = 0
    for s in range(T):
        f = oracle.pair_subset(2024, s, P, M)
        inc += f; both += int(f[3] and f[150])
    p = M / P
    z = (inc - T * p) / np.sqrt(T * p * (1 - p))
    assert np.abs(z).max() < 4.5, np.abs(z).max()                  # 200 cells, 4.5 sigma
    assert abs(np.mean(z ** 2) - 1.0) < 0.35                       # chi-square / dof close to 1
    pb = M * (M - 1) / (P * (P - 1))
    assert abs(both - T * pb) < 4.5 * np.sqrt(T * pb * (1 - pb))
