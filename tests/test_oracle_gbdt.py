"""Pins for the oracle's gradient-boosted TPOT head: the forest evaluation rule against
scikit-learn's gradient boosting, a hand-built tree, the summation order, and the whole dispatch against the pinned
linear head through a forest that tabulates it.  No GPU."""
import numpy as np
import pytest

from paper_2606_17949_b200 import synth
from test_oracle_score import _rand_case


def _export_sklearn(gbr, tiers=1):
    """scikit-learn GradientBoostingRegressor -> node arrays.  sklearn goes left when x <= thr (x is float32, thr
    float64); the oracle's rule is XGBoost's x < thr', so thr' = the smallest float32 above thr."""
    feat, val, left, right, roots = [], [], [], [], []
    lr = gbr.learning_rate
    for est in gbr.estimators_[:, 0]:
        tr = est.tree_
        off = len(feat)
        roots.append(off)
        for n in range(tr.node_count):
            if tr.children_left[n] < 0:
                feat.append(-1), val.append(lr * float(tr.value[n, 0, 0])), left.append(-1), right.append(-1)
            else:
                thr = tr.threshold[n]
                t32 = np.float32(thr)
                if float(t32) <= thr:
                    t32 = np.nextafter(t32, np.float32(np.inf))
                feat.append(int(tr.feature[n])), val.append(float(t32))
                left.append(off + int(tr.children_left[n])), right.append(off + int(tr.children_right[n]))
    return feat, val, left, right, roots


def test_forest_rule_matches_sklearn_gradient_boosting(orc):
    from sklearn.ensemble import GradientBoostingRegressor
    rng = np.random.default_rng(0)
    n, Fa = 4000, 2
    b = rng.integers(0, 33, n)
    d = rng.integers(0, 20001, n).astype(np.float32)
    aux = rng.uniform(0, 1, (n, Fa)).astype(np.float32)
    X = np.column_stack([b.astype(np.float32), d, aux]).astype(np.float32)
    y = 13.9 * (1 + 0.02 * b) + 2.0 * aux[:, 0] + 1e-4 * d + rng.normal(0, 0.2, n)
    gbr = GradientBoostingRegressor(n_estimators=40, max_depth=4, learning_rate=0.2, random_state=0).fit(X, y)
    feat, val, left, right, roots = _export_sklearn(gbr)
    I = 500
    inst = orc.Instances(tier=[0] * I, cap=[16] * I, price_in=[1], price_out=[1], pre=[0], dec=[1], slope=[0])
    forest = orc.Forest(feat, val, left, right, roots, [0, len(roots)], [float(gbr.init_.constant_[0, 0])], 2 + Fa,
                        aux=X[:I, 2:])
    got = orc.gbdt_tpot(inst, forest, X[:I, 1], X[:I, 0].astype(np.int32))
    np.testing.assert_allclose(got, gbr.predict(X[:I]), rtol=2e-6)
    assert got.std() > 1.0   # a real, input-dependent predictor


def test_hand_built_tree_and_summation_order(orc):
    # x0 = b < 2.5 ? (x1 = d < 100 ? 1.0 : 2.0) : (aux0 < 0.5 ? 3.0 : 4.0)
    feat, val = [0, 1, -1, -1, 2, -1, -1], [2.5, 100.0, 1.0, 2.0, 0.5, 3.0, 4.0]
    left, right = [1, 2, -1, -1, 5, -1, -1], [4, 3, -1, -1, 6, -1, -1]
    inst = orc.Instances(tier=[0] * 5, cap=[9] * 5, price_in=[1], price_out=[1], pre=[0], dec=[1], slope=[0])
    aux = np.array([[0.1], [0.9], [0.1], [0.9], [0.5]], np.float32)
    forest = orc.Forest(feat, val, left, right, [0], [0, 1], [10.0], 3, aux=aux)
    got = orc.gbdt_tpot(inst, forest, [50.0, 100.0, 0.0, 0.0, 0.0], [2, 2, 3, 3, 3])
    assert got.tolist() == [11.0, 12.0, 13.0, 14.0, 14.0]   # 100 < 100 and 0.5 < 0.5 are false -> right
    # fp32 sum, sequential, from the base: (0 + 1e8) + 1 = 1e8 (1 is lost), then - 1e8 = 0 -> floor 1e-6;
    # any other order would give 1
    f2 = orc.Forest([-1, -1, -1], [1e8, 1.0, -1e8], [-1] * 3, [-1] * 3, [0, 1, 2], [0, 3], [0.0], 2)
    assert orc.gbdt_tpot(inst, f2, [0.0] * 5, [0] * 5).tolist() == [np.float32(1e-6)] * 5
    f3 = orc.Forest([-1, -1, -1], [1e8, -1e8, 1.0], [-1] * 3, [-1] * 3, [0, 1, 2], [0, 3], [0.0], 2)
    assert orc.gbdt_tpot(inst, f3, [0.0] * 5, [0] * 5).tolist() == [1.0] * 5


def _linear_as_forest(orc, inst, bmax):
    fd, leaf_index = synth.lookup_forest(inst.M, inst.dec, inst.slope, bmax)
    for t in range(inst.M):
        for b in range(bmax + 1):
            a = np.float32(inst.slope[t] * np.float32(b))
            a = np.float32(np.float32(1.0) + a)
            fd["node_value"][leaf_index[t][b]] = float(np.float32(inst.dec[t] * a))
    return orc.Forest(**fd)


def test_dispatch_with_a_forest_that_tabulates_the_linear_head_equals_the_linear_head(orc):
    """latency_mode 2 differs from the pinned mode 0 only in where tpot comes from; with one tree per tier whose leaf
    for running batch b holds dec*(1+slope*b), base 0, the two must agree bit for bit -- scores, assignment, state,
    and the between-batch drain."""
    rng = np.random.default_rng(12)
    for _ in range(15):
        inst, d, b, Q, L, ell = _rand_case(orc, rng, B=9, I=7, M=3)
        forest = _linear_as_forest(orc, inst, int(inst.cap.max()) + 1)
        w = rng.dirichlet([1, 1, 1]).astype(np.float32)
        bud = None if rng.uniform() < 0.5 else rng.uniform(50, 3000, 9).astype(np.float32)
        ref = orc.dispatch(inst, d, b, Q, L, ell, w, budget=bud)
        out = orc.dispatch(inst, d, b, Q, L, ell, w, budget=bud, latency_mode=2, forest=forest)
        for key in ("assignment", "scores", "scores0", "order", "queued", "running", "max_tokens"):
            np.testing.assert_array_equal(out[key], ref[key], err_msg=key)
        a0 = orc.advance_state(inst, d, b, 37.5)
        a1 = orc.advance_state_gbdt(inst, forest, d, b, 37.5)
        np.testing.assert_array_equal(a0[0], a1[0])
        np.testing.assert_array_equal(a0[1], a1[1])


def test_forest_head_reacts_to_dead_reckoned_state(orc):
    """The head is re-evaluated after every dispatch: with a forest whose TPOT jumps once an instance runs
    2 sequences, two equal instances alternate instead of herding."""
    inst = orc.Instances(tier=[0, 0], cap=[8, 8], price_in=[1], price_out=[1], pre=[0], dec=[1], slope=[0])
    forest = orc.Forest([0, -1, -1], [1.5, 10.0, 50.0], [1, -1, -1], [2, -1, -1], [0], [0, 1], [0.0], 2)
    Q = np.full((4, 1), 0.5, np.float32)
    L = np.full((4, 1), 100.0, np.float32)
    out = orc.dispatch(inst, [0.0, 0.0], [0, 0], Q, L, [10] * 4, [0.0, 1.0, 0.0], latency_mode=2, forest=forest)
    assert sorted(out["assignment"].tolist()) == [0, 0, 1, 1]
    assert out["running"].tolist() == [2, 2]
    with pytest.raises(ValueError):
        orc.dispatch(inst, [0.0, 0.0], [0, 0], Q, L, [10] * 4, [0.0, 1.0, 0.0], latency_mode=2)


def test_make_forest_is_well_formed():
    f = synth.make_forest(4, [10.2, 19.6, 13.9, 41.6], n_trees=16, depth=4, Fa=2, seed=1, I=13)
    n = len(f["node_feature"])
    for i in range(n):
        if f["node_feature"][i] >= 0:
            assert i < f["node_left"][i] < n and i < f["node_right"][i] < n and f["node_feature"][i] < f["n_features"]
    assert f["tier_tree_begin"] == [0, 16, 32, 48, 64] and f["aux"].shape == (13, 2)
