"""Pins for the oracle's score / LPT dispatch / dead-reckoning stages.  No GPU."""
import itertools

import numpy as np
import pytest

from conftest import read_golden


def _rand_case(orc, rng, B, I, M, cap_lo=1, cap_hi=6):
    tier = rng.integers(0, M, I)
    tier[:M] = np.arange(M)[: min(M, I)] if I >= M else tier[:M]
    inst = orc.Instances(tier=tier, cap=rng.integers(cap_lo, cap_hi + 1, I),
                         price_in=rng.uniform(0.05, 2, M), price_out=rng.uniform(0.05, 2, M),
                         pre=rng.uniform(0, 0.3, M), dec=rng.uniform(5, 50, M), slope=rng.uniform(0, 0.05, M))
    queued = rng.integers(0, 3000, I).astype(np.float32)
    running = rng.integers(0, cap_hi + 1, I).astype(np.int32)
    running = np.minimum(running, inst.cap)
    quality = rng.uniform(0, 1, (B, M)).astype(np.float32)
    outlen = rng.lognormal(5.5, 0.6, (B, M)).astype(np.float32)
    plen = rng.integers(1, 3000, B).astype(np.int32)
    return inst, queued, running, quality, outlen, plen


def _score_row_f64(inst, d, b, Q, L, ell, w):
    """Independent fp64 statement of Eq. 1 / Eq. 2 / the latency formula for one request."""
    t = inst.tier
    C = ell * inst.price_in[t].astype(np.float64) + L[t].astype(np.float64) * inst.price_out[t]
    tpot = inst.dec[t].astype(np.float64) * (1 + inst.slope[t].astype(np.float64) * b)
    wait = np.where(b < inst.cap, 0.0, d / np.maximum(b, 1))
    T = inst.pre[t].astype(np.float64) * ell + tpot * (wait + L[t])
    ct = 1 - C / C.max() if C.max() > 0 else np.zeros_like(C)
    lt = 1 - T / T.max() if T.max() > 0 else np.zeros_like(T)
    return w[0] * Q[t] + w[2] * ct + w[1] * lt, C, T


def test_w1_table1_scores(orc):
    g = read_golden("W1_table1_scores.txt")
    inst = orc.Instances(tier=[0, 1, 2, 3], cap=[256] * 4, price_in=g["price_in"], price_out=g["price_out"],
                         pre=[0] * 4, dec=g["dec"], slope=[0] * 4)
    zero = np.zeros(4, np.float32)
    Q = np.array([g["quality"]], np.float32)
    L = np.array([g["outlen"]], np.float32)
    for j in range(7):
        out = orc.decide_from_predictions(inst, zero, zero.astype(np.int32), Q, L, [int(g["prompt_len"][0])],
                                          g["w%d" % j])
        np.testing.assert_allclose(out["scores"][0], g["S%d" % j], atol=2e-7, err_msg="row %d" % j)
        assert out["assignment"][0] == int(g["win%d" % j][0])
        np.testing.assert_array_equal(out["scores"], out["scores0"])


def test_w2_lpt_dead_reckoning_trace(orc):
    g = read_golden("W2_lpt_dead_reckoning.txt")
    inst = orc.Instances(tier=g["tier"], cap=g["cap"], price_in=g["price"], price_out=g["price"], pre=g["pre"],
                         dec=g["dec"], slope=g["slope"])
    Q = np.array(g["quality"], np.float32).reshape(3, 2)
    L = np.array(g["outlen"], np.float32).reshape(3, 2)
    w = [1 / 3, 1 / 3, 1 / 3]
    out = orc.decide_from_predictions(inst, g["d"], g["b"], Q, L, g["prompt_len"], w)
    assert out["order"].tolist() == [int(x) for x in g["order"]]
    assert out["assignment"].tolist() == [int(x) for x in g["assignment"]]
    for step, r in enumerate(out["order"]):
        np.testing.assert_allclose(out["scores"][r], g["step%d_S" % step], atol=2e-7)
    np.testing.assert_array_equal(out["queued"], np.array(g["d_after"], np.float32))
    assert out["running"].tolist() == [int(x) for x in g["b_after"]]
    off = orc.decide_from_predictions(inst, g["d"], g["b"], Q, L, g["prompt_len"], w, update_enabled=0)
    assert off["assignment"].tolist() == [int(x) for x in g["assignment_no_update"]]
    np.testing.assert_allclose(off["scores"][out["order"], 1], g["S_i1_no_update"], atol=2e-7)
    np.testing.assert_array_equal(off["queued"], np.array(g["d"], np.float32))


def test_six_times_cheaper_candidate(orc):
    """'a 6x-cheaper candidate contributes proportionally rather than 0/1': cost term 1 - 1/6."""
    inst = orc.Instances(tier=[0, 1], cap=[8, 8], price_in=[1.0, 6.0], price_out=[1.0, 6.0], pre=[0, 0],
                         dec=[10, 10], slope=[0, 0])
    out = orc.decide_from_predictions(inst, [0, 0], [0, 0], [[0.5, 0.5]], [[100.0, 100.0]], [200], [0, 0, 1])
    np.testing.assert_allclose(out["scores"][0], [1 - 1 / 6, 0.0], rtol=1e-6, atol=1e-7)
    assert out["assignment"][0] == 0


def test_simplex_corners(orc):
    """(1,0,0) -> S = Q^ exactly, argmax Q^; (0,1,0) -> min T^; (0,0,1) -> min C^."""
    rng = np.random.default_rng(10)
    for trial in range(20):
        inst, dq, bq, Q, L, plen = _rand_case(orc, rng, B=6, I=7, M=3)
        out = orc.decide_from_predictions(inst, dq, bq, Q, L, plen, [1, 0, 0], update_enabled=0)
        np.testing.assert_array_equal(out["scores"], Q[:, inst.tier])
        for r in range(6):
            assert Q[r, inst.tier[out["assignment"][r]]] == Q[r, inst.tier].max()
        for corner, which in [([0, 1, 0], 2), ([0, 0, 1], 1)]:
            out = orc.decide_from_predictions(inst, dq, bq, Q, L, plen, corner, update_enabled=0)
            for r in range(6):
                S64, C, T = _score_row_f64(inst, dq, bq, Q[r], L[r], int(plen[r]), corner)
                v = (C, T)[which - 1]
                a = out["assignment"][r]
                assert out["scores"][r, a] == out["scores"][r].max()
                assert v[a] <= v.min() * (1 + 2.0 ** -21)


def test_scores_match_fp64_formula_and_lie_in_unit_interval(orc):
    rng = np.random.default_rng(11)
    for trial in range(20):
        inst, dq, bq, Q, L, plen = _rand_case(orc, rng, B=5, I=9, M=4)
        w = rng.dirichlet([1, 1, 1])
        out = orc.decide_from_predictions(inst, dq, bq, Q, L, plen, w, update_enabled=0)
        for r in range(5):
            S64, _, _ = _score_row_f64(inst, dq, bq, Q[r], L[r], int(plen[r]), w.astype(np.float32))
            np.testing.assert_allclose(out["scores"][r], S64, atol=5e-7)
        assert out["scores"].min() >= 0 and out["scores"].max() <= 1 + 1e-6


def test_static_prior_and_saturated_latency(orc):
    """pre=0, slope=0, free slot: T = dec*L^ (static prior, P:L227 arm 4); saturated: T = dec*(d/b + L^)."""
    inst = orc.Instances(tier=[0, 0], cap=[4, 4], price_in=[1], price_out=[1], pre=[0], dec=[20.0], slope=[0])
    # i0 free (b=1<4), i1 saturated (b=4) with d=800 -> wait 200
    out = orc.decide_from_predictions(inst, [800, 800], [1, 4], [[0.5]], [[100.0]], [10], [0, 1, 0])
    T = np.array([20.0 * 100, 20.0 * (800 / 4 + 100)])
    np.testing.assert_allclose(out["scores"][0], 1 - T / T.max(), atol=1e-7)


def test_single_instance_cluster(orc):
    rng = np.random.default_rng(12)
    inst, dq, bq, Q, L, plen = _rand_case(orc, rng, B=8, I=1, M=1)
    w = np.array([0.5, 0.25, 0.25], np.float32)
    out = orc.decide_from_predictions(inst, dq, bq, Q, L, plen, w)
    assert out["assignment"].tolist() == [0] * 8
    np.testing.assert_array_equal(out["scores"][:, 0], w[0] * Q[:, 0])


def test_scale_invariance_prices_and_latency(orc):
    """rescaling all prices leaves orderings invariant; same for the latency heads.  A power of two
    scales every intermediate exactly, so scores are bit-identical; other factors agree to rounding."""
    rng = np.random.default_rng(13)
    inst, dq, bq, Q, L, plen = _rand_case(orc, rng, B=12, I=8, M=3)
    w = [0.2, 0.5, 0.3]
    base = orc.decide_from_predictions(inst, dq, bq, Q, L, plen, w)
    for a, exact in [(4.0, True), (3.7, False)]:
        sc = orc.Instances(inst.tier, inst.cap, inst.price_in * a, inst.price_out * a, inst.pre * a,
                           inst.dec * a, inst.slope)
        out = orc.decide_from_predictions(sc, dq, bq, Q, L, plen, w)
        if exact:
            np.testing.assert_array_equal(out["scores"], base["scores"])
            np.testing.assert_array_equal(out["assignment"], base["assignment"])
        else:
            np.testing.assert_allclose(out["scores0"], base["scores0"], atol=1e-6)


def test_tier_loss_equals_dropping_its_instances(orc):
    """P:L327 graceful tier loss: removing a tier's instances renormalises cost/latency over the rest;
    quality is never renormalised.  With tier 3 gone its labels must not influence anything."""
    rng = np.random.default_rng(14)
    inst, dq, bq, Q, L, plen = _rand_case(orc, rng, B=10, I=9, M=4)
    keep = inst.tier != 3
    sub = orc.Instances(inst.tier[keep], inst.cap[keep], inst.price_in, inst.price_out, inst.pre, inst.dec,
                        inst.slope)
    w = [0.4, 0.3, 0.3]
    a = orc.decide_from_predictions(sub, dq[keep], bq[keep], Q, L, plen, w)
    L2, Q2 = L.copy(), Q.copy()
    L2[:, 3] = 1e6     # absurd labels on the lost tier: LPT key and maxima must ignore them
    Q2[:, 3] = 1.0
    b = orc.decide_from_predictions(sub, dq[keep], bq[keep], Q2, L2, plen, w)
    np.testing.assert_array_equal(a["assignment"], b["assignment"])
    np.testing.assert_array_equal(a["scores"], b["scores"])
    np.testing.assert_array_equal(a["order"], b["order"])


def test_scores0_vs_scores(orc):
    rng = np.random.default_rng(15)
    inst, dq, bq, Q, L, plen = _rand_case(orc, rng, B=16, I=6, M=3)
    w = [1 / 3, 1 / 3, 1 / 3]
    out = orc.decide_from_predictions(inst, dq, bq, Q, L, plen, w)
    first = out["order"][0]
    np.testing.assert_array_equal(out["scores"][first], out["scores0"][first])
    assert not np.array_equal(out["scores"], out["scores0"])
    off = orc.decide_from_predictions(inst, dq, bq, Q, L, plen, w, update_enabled=0)
    np.testing.assert_array_equal(off["scores"], off["scores0"])
    np.testing.assert_array_equal(off["scores0"], out["scores0"])


def test_lpt_order_invariants(orc):
    rng = np.random.default_rng(16)
    inst, dq, bq, Q, L, plen = _rand_case(orc, rng, B=40, I=5, M=3)
    L[7] = L[3]                                     # equal keys -> smaller request index first
    w = [0.3, 0.4, 0.3]
    out = orc.decide_from_predictions(inst, dq, bq, Q, L, plen, w)
    present = np.unique(inst.tier)
    key = L[:, present].max(1)
    ok = key[out["order"]]
    assert np.all(ok[:-1] >= ok[1:])
    pos = {r: j for j, r in enumerate(out["order"])}
    assert pos[3] < pos[7]
    assert sorted(out["order"].tolist()) == list(range(40))
    # LPT off: input order
    off = orc.decide_from_predictions(inst, dq, bq, Q, L, plen, w, lpt_enabled=0)
    assert off["order"].tolist() == list(range(40))
    # permuting the batch permutes the outputs (keys distinct apart from the planted tie -> drop it)
    L[7] = L[7] * 1.01
    base = orc.decide_from_predictions(inst, dq, bq, Q, L, plen, w)
    perm = rng.permutation(40)
    p = orc.decide_from_predictions(inst, dq, bq, Q[perm], L[perm], plen[perm], w)
    np.testing.assert_array_equal(p["assignment"], base["assignment"][perm])
    np.testing.assert_array_equal(p["scores"], base["scores"][perm])
    np.testing.assert_array_equal(p["queued"], base["queued"])


def test_update_rule_and_state_out(orc):
    """d[i*] += L^[r, m(i*)]; b grows by one while a slot is free (reading 18)."""
    inst = orc.Instances(tier=[0, 1], cap=[2, 2], price_in=[1, 1], price_out=[1, 1], pre=[0, 0], dec=[10, 10],
                         slope=[0, 0])
    Q = np.array([[0.9, 0.1]] * 3, np.float32)
    L = np.array([[30.0, 70.0], [20.0, 70.0], [10.0, 70.0]], np.float32)
    out = orc.decide_from_predictions(inst, [5, 5], [0, 0], Q, L, [1, 1, 1], [1, 0, 0])
    assert out["assignment"].tolist() == [0, 0, 0]
    assert out["queued"].tolist() == [65.0, 5.0] and out["running"].tolist() == [2, 0]


def test_argmax_tiebreak_spreads_replicas(orc):
    """Reading 17: with w_lat = 0 all replicas of a tier tie exactly; (S desc, d asc, i asc) + the update
    spreads them instead of herding (the reactive shortest-queue tiebreak of P:L227 arm 2)."""
    inst = orc.Instances(tier=[0, 0, 0], cap=[8] * 3, price_in=[1], price_out=[1], pre=[0], dec=[10], slope=[0])
    Q = np.full((6, 1), 0.5, np.float32)
    L = np.full((6, 1), 100.0, np.float32)
    out = orc.decide_from_predictions(inst, [50, 0, 50], [0, 0, 0], Q, L, [10] * 6, [1, 0, 0])
    assert out["assignment"].tolist() == [1, 0, 2, 1, 0, 2]


def test_greedy_equals_exhaustive_when_updates_off(orc):
    """P:L80 'the objective decomposes per request': without state updates greedy attains the exhaustive
    maximum of sum_r S[r, a_r] over all I^B assignments."""
    rng = np.random.default_rng(17)
    for trial in range(10):
        B, I = 5, 4
        inst, dq, bq, Q, L, plen = _rand_case(orc, rng, B=B, I=I, M=3)
        w = rng.dirichlet([1, 1, 1])
        out = orc.decide_from_predictions(inst, dq, bq, Q, L, plen, w, update_enabled=0)
        S = out["scores0"].astype(np.float64)
        best = max(sum(S[r, a[r]] for r in range(B)) for a in itertools.product(range(I), repeat=B))
        got = sum(S[r, out["assignment"][r]] for r in range(B))
        assert got == pytest.approx(best, abs=1e-12)


def test_greedy_vs_exhaustive_sequential_upper_bound(orc):
    """With updates the exhaustive search over sequential-state assignments (same LPT order) upper-bounds
    greedy's sum of scores; greedy is a heuristic (15.6 % of assignments differ from a batch-level
    matching), so only the bound is asserted."""
    rng = np.random.default_rng(18)
    B, I = 4, 3
    inst, dq, bq, Q, L, plen = _rand_case(orc, rng, B=B, I=I, M=2)
    w = np.array([0.2, 0.6, 0.2], np.float32)
    out = orc.decide_from_predictions(inst, dq, bq, Q, L, plen, w)
    order = out["order"]
    greedy = sum(float(out["scores"][r, out["assignment"][r]]) for r in range(B))

    def total(assign):
        d, b, tot = dq.astype(np.float64).copy(), bq.copy(), 0.0
        for j, r in enumerate(order):
            S, _, _ = _score_row_f64(inst, d, b, Q[r], L[r], int(plen[r]), w)
            i = assign[j]
            tot += S[i]
            d[i] += L[r, inst.tier[i]]
            if b[i] < inst.cap[i]:
                b[i] += 1
        return tot
    best = max(total(a) for a in itertools.product(range(I), repeat=B))
    assert best >= greedy - 1e-5


def test_advance_state_closed_form(orc):
    """d' = max(0, d - b*dt/tpot), tpot = dec*(1+slope*b); b -> 0 when drained; idle instances untouched."""
    inst = orc.Instances(tier=[0, 1, 0, 1], cap=[8] * 4, price_in=[1, 1], price_out=[1, 1], pre=[0, 0],
                         dec=[10.0, 20.0], slope=[0.0, 0.05])
    d0 = np.array([1000, 1000, 7, 50], np.float32)
    b0 = np.array([4, 2, 0, 2], np.int32)
    d1, b1 = orc.advance_state(inst, d0, b0, 500.0)
    # i0: 4*500/10 = 200 done; i1: tpot=20*1.1=22 -> 2*500/22 = 45.4545; i2 idle; i3: 45.45 < 50 -> 4.5455 left
    np.testing.assert_allclose(d1, [800, 1000 - 2 * 500 / 22, 7, 50 - 2 * 500 / 22], rtol=1e-6)
    assert b1.tolist() == [4, 2, 0, 2]
    d2, b2 = orc.advance_state(inst, d0, b0, 0.0)
    np.testing.assert_array_equal(d2, d0)
    assert b2.tolist() == b0.tolist()
    d3, b3 = orc.advance_state(inst, d0, b0, 1e6)
    assert d3.tolist() == [0, 0, 7, 0] and b3.tolist() == [0, 0, 0, 0]
    da, ba = orc.advance_state(inst, d0, b0, 100.0)
    db, bb = orc.advance_state(inst, da, ba, 150.0)
    dc, bc = orc.advance_state(inst, d0, b0, 250.0)
    np.testing.assert_allclose(db, dc, rtol=1e-6)


def test_paper_cluster_cost_vs_latency_disagree(orc):
    """'14B on V100x4 has lower TPOT than 7B on A30x1 despite a higher price -- cost-minimizing
    and latency-minimizing routing disagree'.  Restricted to those two tiers of Table 1."""
    inst = orc.Instances(tier=[0, 1], cap=[16, 16], price_in=[0.07, 0.15], price_out=[0.07, 0.15], pre=[0, 0],
                         dec=[19.6, 13.9], slope=[0, 0])
    Q, L = [[0.4, 0.4]], [[300.0, 300.0]]
    assert orc.decide_from_predictions(inst, [0, 0], [0, 0], Q, L, [500], [0, 0, 1])["assignment"][0] == 0
    assert orc.decide_from_predictions(inst, [0, 0], [0, 0], Q, L, [500], [0, 1, 0])["assignment"][0] == 1


def test_whole_decision_runs_on_C1(orc):
    from paper_2606_17949_b200 import synth
    cfg = synth.CONFIGS["C1"]
    bank = synth.make_bank(cfg)
    it = synth.make_instances(cfg.I, cfg.M)
    inst = orc.Instances(**it)
    queued, running = synth.make_state(cfg.I, it["cap"], cfg.seed)
    out = orc.decide(bank["emb"].numpy(), bank["quality"].numpy(), bank["outlen"].numpy(), inst, queued.numpy(),
                     running.numpy(), synth.make_queries(cfg).numpy(), synth.make_prompt_len(cfg).numpy(),
                     synth.PRESETS["balanced"], cfg.k, store_dtype="f32")
    assert out["assignment"].shape == (16,) and out["assignment"].min() >= 0 and out["assignment"].max() < 13
    # all k neighbours come from the query's own mixture component (generator sanity)
    assert out["nn_sim"].min() > 0.8
    assert 0 <= out["pred_quality"].min() and out["pred_quality"].max() <= 1
