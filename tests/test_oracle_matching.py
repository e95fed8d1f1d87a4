"""Pins for the oracle's batch-level matching replay: exhaustive enumeration on tiny
batches, the unconstrained case (= row-wise maxima, "the objective decomposes per request"), filtered entries
and infeasibility.  No GPU."""
import itertools

import numpy as np
import pytest


def _brute(S, quota):
    B, I = S.shape
    best = -np.inf
    for a in itertools.product(range(I), repeat=B):
        if any(a.count(i) > quota[i] for i in range(I)):
            continue
        v = sum(float(S[r, a[r]]) for r in range(B))
        best = max(best, v)
    return best


def test_matching_equals_exhaustive_optimum_on_tiny_batches(orc):
    rng = np.random.default_rng(0)
    for _ in range(40):
        B, I = int(rng.integers(1, 7)), int(rng.integers(1, 4))
        S = rng.uniform(0, 1, (B, I)).astype(np.float32)
        if rng.uniform() < 0.3:
            S[rng.integers(0, B), rng.integers(0, I)] = -np.inf
        quota = rng.integers(0, B + 1, I)
        while quota.sum() < B:
            quota[rng.integers(0, I)] += 1
        best = _brute(S, quota)
        if best == -np.inf:
            with pytest.raises(ValueError):
                orc.matching_replay(S, quota)
            continue
        out = orc.matching_replay(S, quota)
        assert abs(out["objective"] - best) <= 1e-9
        assert all((out["match"] == i).sum() <= quota[i] for i in range(I))
        assert np.isfinite(S[np.arange(B), out["match"]]).all()


def test_loose_quotas_give_row_maxima_and_tight_quotas_cost_something(orc):
    """With room for the whole batch on every instance the objective decomposes per request: the matching is
    the row-wise argmax.  A quota of one request per instance can only lower the optimum."""
    rng = np.random.default_rng(1)
    S = rng.uniform(0, 1, (8, 12)).astype(np.float32)
    loose = orc.matching_replay(S, [8] * 12, greedy=S.argmax(axis=1))
    assert np.array_equal(loose["match"], S.argmax(axis=1)) and loose["diverged"] == 0
    assert abs(loose["objective"] - float(S.astype(np.float64).max(axis=1).sum())) <= 1e-12
    tight = orc.matching_replay(S, [1] * 12, greedy=S.argmax(axis=1))
    assert tight["objective"] <= loose["objective"] and len(set(tight["match"].tolist())) == 8
    # hand-made: both requests prefer instance 0; one slot there -> the request that loses less moves
    S2 = np.array([[0.9, 0.5], [0.8, 0.1]], np.float32)
    out = orc.matching_replay(S2, [1, 1], greedy=[0, 0])
    assert out["match"].tolist() == [1, 0] and abs(out["objective"] - (0.5 + 0.8)) < 1e-7 and out["diverged"] == 1
    with pytest.raises(ValueError):
        orc.matching_replay(S2, [1, 0])
