"""K-sharded update: the oracle's per-shard restatement of (17)/(4) against the oracle's own whole-K update
(partition invariance), and the host-side shard arithmetic of the product (no GPU)."""
import numpy as np
import pytest

from oracle import oracle as O
from paper_2209_12842_b200 import sharded
from paper_2209_12842_b200 import workloads as W


@pytest.mark.parametrize("K,world", [(1, 1), (7, 1), (7, 2), (8, 8), (10, 3), (16384, 8), (65537, 5)])
def test_shard_bounds_partition_exactly(K, world):
    b = [sharded.shard_bounds(K, world, r) for r in range(world)]
    assert b[0][0] == 0 and b[-1][1] == K
    assert all(b[i][1] == b[i + 1][0] for i in range(world - 1))          # contiguous, no gap, no overlap
    sizes = [e - s for s, e in b]
    assert max(sizes) - min(sizes) <= 1 and min(sizes) >= 1 and sizes == sorted(sizes, reverse=True)


def test_shard_bounds_rejects_empty_shards():
    with pytest.raises(ValueError):
        sharded.shard_bounds(3, 4, 0)
    with pytest.raises(ValueError):
        sharded.shard_bounds(8, 2, 2)


def test_shard_problem_names_its_place():
    p = W.config0(K=10)
    s = sharded.shard_problem(p, 3, 2)
    assert (s.K, s.k_offset, s.K_total) == (3, 7, 10) and s.seed == p.seed and s.M == p.M


@pytest.mark.parametrize("lam,scale", [(1.0, 1.0), (0.5, 1e4), (100.0, 10.0)])
def test_partition_invariance_of_the_update(lam, scale):
    """combine(partials of any partition) == (17)/(4) on all K samples, soft and one-hot weights alike."""
    rng = np.random.default_rng(0)
    p = W.config0(K=97, T=9).replace(lam=lam)
    orc = O.Oracle(p)
    S = scale * rng.uniform(0.0, 5.0, p.K)
    u = rng.normal(size=(p.K, p.T, 2)) * np.array([0.2, 1.5])
    ref = orc.weights_update(S, u)
    for cuts in ([0, 97], [0, 40, 97], [0, 1, 2, 50, 96, 97], list(range(98))):
        parts = np.stack([O.shard_partial(S[a:b], u[a:b], lam) for a, b in zip(cuts[:-1], cuts[1:])])
        vp = O.combine_partials(parts, lam, p.u_min, p.u_max)
        assert np.abs(vp - ref["v_plus"]).max() < 1e-12
        vp_perm = O.combine_partials(parts[::-1], lam, p.u_min, p.u_max)   # the order of the shards is irrelevant
        assert np.abs(vp_perm - ref["v_plus"]).max() < 1e-12
    # the shard that holds the argmin carries scale 1; Z of the union is the oracle's Z
    parts = np.stack([O.shard_partial(S[a:b], u[a:b], lam) for a, b in ((0, 40), (40, 97))])
    s = np.exp(-(parts[:, 0] - parts[:, 0].min()) / lam)
    assert s.max() == 1.0 and abs((s * parts[:, 1]).sum() - ref["Z"]) < 1e-9 * ref["Z"]
