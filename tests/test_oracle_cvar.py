"""Pins for the oracle's CVaR reducer and sensitivity scaling (no GPU).

PAPER.md (10)-(13) :97-111, Alg.1 l.24-26 :204-207, (18)-(19) :144-148.
"""
import os

import numpy as np
import pytest

from oracle import oracle as O

GOLDEN = os.path.join(os.path.dirname(__file__), "golden")


def _golden_gaussian():
    rows = [l.split() for l in open(os.path.join(GOLDEN, "gaussian_cvar.txt")) if not l.startswith("#")]
    return {float(a): float(v) for a, v in rows}


def _paper_hp():
    rows = [l.split() for l in open(os.path.join(GOLDEN, "paper_hyperparameters.txt")) if not l.startswith("#")]
    return {k: float(v) for k, v in rows}


def test_tail_count_configs_and_robustness():
    # BASELINE configs: C0, C1, C2, C3, C4 sweep
    assert O.tail_count(0.9, 16) == 2
    assert O.tail_count(0.95, 64) == 4
    assert O.tail_count(0.95, 128) == 7
    assert O.tail_count(0.9, 128) == 13
    assert O.tail_count(0.95, 16) == 1
    assert O.tail_count(0.95, 256) == 13
    # naive ceil((1-0.7)*10) is 4 in fp64; the count must be 3
    assert O.tail_count(0.7, 10) == 3
    # the paper's own N=300, alpha=0.9: (1-alpha)N = 30 exactly
    hp = _paper_hp()
    assert O.tail_count(0.9, int(hp["realisations"])) == 30
    assert int(hp["samples"]) * int(hp["realisations"]) == int(hp["trajectories_total"])
    # clamped to [1, M]
    assert O.tail_count(0.999999, 8) == 1
    assert O.tail_count(1e-9, 8) == 8


def test_cvar_hand_arrays():
    # hand-checkable, incl. ties and all-zero
    assert O.cvar_topk([1, 2, 3, 4, 5, 6, 7, 8], 2) == 7.5
    assert O.cvar_topk([8, 1, 7, 2, 6, 3, 5, 4], 3) == 7.0
    assert O.cvar_topk([0, 0, 0, 0], 2) == 0.0
    assert O.cvar_topk([7, 0, 0, 0, 0, 0, 0, 0], 2) == 3.5
    assert O.cvar_topk([5, 5, 5, 1], 2) == 5.0  # ties: value independent of which tied items are picked
    assert O.cvar_topk([-3, -1, -2], 1) == -1.0
    assert O.cvar_topk([2.5], 1) == 2.5
    assert O.cvar_topk([1, 2, 3], 3) == 2.0


def test_cvar_brute_force_random():
    rng = np.random.default_rng(0)
    for _ in range(200):
        M = int(rng.integers(1, 9))
        k = int(rng.integers(1, M + 1))
        L = rng.integers(0, 4, size=M).astype(float) if rng.random() < 0.5 else rng.normal(size=M)
        # brute force: maximum over all size-k subsets of the subset mean
        from itertools import combinations
        best = max(sum(c) / k for c in combinations(L.tolist(), k))
        assert O.cvar_topk(L, k) == pytest.approx(best, abs=1e-14)


def test_rockafellar_uryasev_identity():
    # paper ref [10]: when (1-alpha)M is an integer,
    # CVaR = min_c { c + sum_m max(L_m - c, 0) / ((1-alpha) M) }, minimum attained at a sample value
    rng = np.random.default_rng(1)
    for M, alpha in [(10, 0.7), (20, 0.9), (300, 0.9), (64, 0.75)]:
        L = rng.exponential(size=M)
        k = O.tail_count(alpha, M)
        assert abs(k - (1 - alpha) * M) < 1e-9
        ru = min(c + np.maximum(L - c, 0).sum() / k for c in L)
        assert O.cvar_topk(L, k) == pytest.approx(ru, rel=1e-13)


@pytest.mark.parametrize("alpha", [0.9, 0.95, 0.99])
def test_gaussian_closed_form(alpha):
    # definitions (10)-(11) for L ~ N(0,1): CVaR = pdf(ppf(alpha))/(1-alpha)
    closed = _golden_gaussian()[alpha]
    M = 1 << 20
    L = np.random.default_rng(int(alpha * 100)).normal(size=M)
    k = O.tail_count(alpha, M)
    mc_sigma = 2.5 / np.sqrt(k)  # generous bound on the tail-mean MC error
    assert abs(O.cvar_topk(L, k) - closed) < 4 * mc_sigma / 2
    assert abs(O.cvar_literal12(L, alpha) - closed) < 4 * mc_sigma / 2
    # affine equivariance with mu, sigma (north_star: mu + sigma*phi(Phi^-1(alpha))/(1-alpha))
    assert O.cvar_topk(3.0 + 2.0 * L, k) == pytest.approx(3.0 + 2.0 * O.cvar_topk(L, k), rel=1e-12)


def test_literal_12_vs_topk():
    rng = np.random.default_rng(3)
    # no ties, (1-alpha)M non-integer -> the two estimators coincide (G11)
    for M, alpha in [(16, 0.9), (64, 0.95), (128, 0.95), (128, 0.9), (256, 0.95)]:
        L = rng.normal(size=M)
        assert O.cvar_literal12(L, alpha) == pytest.approx(O.cvar_topk(L, O.tail_count(alpha, M)), rel=1e-13)
    # (1-alpha)M integer: literal (12) averages one more value (N_o = (1-alpha)M + 1)
    L = np.arange(1.0, 11.0)
    assert O.cvar_literal12(L, 0.7) == pytest.approx(np.mean([7, 8, 9, 10]))
    assert O.cvar_topk(L, O.tail_count(0.7, 10)) == pytest.approx(np.mean([8, 9, 10]))
    # ties at VaR: literal (12) averages all tied values
    L = np.zeros(16); L[3] = 7.0
    assert O.cvar_literal12(L, 0.9) == pytest.approx(7.0 / 16)
    assert O.cvar_topk(L, 2) == 3.5


def test_sensitivity_scaling():
    rng = np.random.default_rng(4)
    L = rng.exponential(size=64)
    assert np.array_equal(O.sensitivity_scale(L, 1.0), (L - L.mean()) + L.mean()) or \
        np.allclose(O.sensitivity_scale(L, 1.0), L, rtol=1e-15)
    for B in (0.5, 2.0, 7.0):
        La = O.sensitivity_scale(L, B)
        assert La.mean() == pytest.approx(L.mean(), rel=1e-13)           # "maintaining their mean" :142
        assert La.std() == pytest.approx(B * L.std(), rel=1e-12)          # variance scaled up
        k = 4
        # B>0 is affine-monotone: CVaR(L_a) = B (CVaR(L) - Lbar) + Lbar
        assert O.cvar_topk(La, k) == pytest.approx(B * (O.cvar_topk(L, k) - L.mean()) + L.mean(), rel=1e-12)
