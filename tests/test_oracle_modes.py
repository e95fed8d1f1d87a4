"""Pins for the oracle's optional pieces: the budget admission filter of Eq. 2 and the
isolation-arm / ablation modes.  Each new behaviour is tied to something other than itself: the
hand-worked W3, closed forms, and -- the strongest pin -- equivalence with the already-pinned default mechanism on a
suitably reduced or modified cluster.  No GPU."""
import numpy as np
import pytest

from conftest import read_golden
from test_oracle_score import _rand_case, _score_row_f64

INT32_MAX = 2**31 - 1


def _inf(x):
    return [float(v) for v in x]


def test_w3_budget_filter_table1(orc):
    g1 = read_golden("W1_table1_scores.txt")
    g = read_golden("W3_budget_table1.txt")
    inst = orc.Instances(tier=[0, 1, 2, 3], cap=[256] * 4, price_in=g1["price_in"], price_out=g1["price_out"],
                         pre=[0] * 4, dec=g1["dec"], slope=[0] * 4)
    zero = np.zeros(4, np.float32)
    Q, L = np.array([g1["quality"]], np.float32), np.array([g1["outlen"]], np.float32)
    for case in "abc":
        bud = np.array(g["budget_" + case], np.float32)
        for wname, w in (("u", [1 / 3] * 3), ("q", [0.8, 0.1, 0.1]), ("corner", [1, 0, 0])):
            out = orc.dispatch(inst, zero, zero.astype(np.int32), Q, L, [500], w, budget=bud)
            assert out["assignment"][0] == int(g["win_%s_%s" % (wname, case)][0]), (case, wname)
            if wname != "corner":
                exp = np.array(g["S%s_%s" % (wname, case)])
                fin = np.isfinite(exp)
                np.testing.assert_allclose(out["scores"][0][fin], exp[fin], atol=2e-7)
                assert np.all(out["scores"][0][~fin] == -np.inf)
                np.testing.assert_array_equal(out["scores"], out["scores0"])
            if wname != "q":
                assert out["max_tokens"][0] == int(g["maxtok_%s_%s" % (wname, case)][0]), (case, wname)


def test_no_budget_and_infinite_budget_equal_the_default_mechanism(orc):
    rng = np.random.default_rng(5)
    for _ in range(20):
        inst, d, b, Q, L, ell = _rand_case(orc, rng, B=int(rng.integers(1, 12)), I=int(rng.integers(1, 9)), M=3)
        w = rng.dirichlet([1, 1, 1]).astype(np.float32)
        ref = orc.decide_from_predictions(inst, d, b, Q, L, ell, w)
        for bud in (None, np.full(len(ell), np.inf, np.float32)):
            out = orc.dispatch(inst, d, b, Q, L, ell, w, budget=bud)
            for key in ("assignment", "scores", "scores0", "order", "queued", "running"):
                np.testing.assert_array_equal(out[key], ref[key], err_msg=key)
            assert np.all(out["max_tokens"] == INT32_MAX)


def _costs_f32(inst, L_row, ell):
    t = inst.tier
    c1 = np.float32(ell) * inst.price_in[t]
    c2 = L_row[t] * inst.price_out[t]
    return (c1 + c2).astype(np.float32)


def test_budget_filter_equals_default_mechanism_on_the_admitted_subcluster(orc):
    """Eq. 2 is a PRE-scoring filter: dispatching r under a budget must equal dispatching r, alone, on the cluster
    reduced to the admitted instances (the pinned default mechanism), from the same running state, request by
    request in the batch's LPT order.  Budgets are drawn away from every cost so that admission is unambiguous."""
    rng = np.random.default_rng(6)
    n_fallback = n_partial = 0
    for _ in range(40):
        B, I, M = int(rng.integers(1, 10)), int(rng.integers(2, 10)), 3
        inst, d, b, Q, L, ell = _rand_case(orc, rng, B, I, M)
        w = rng.dirichlet([1, 1, 1]).astype(np.float32)
        bud = np.empty(B, np.float32)
        for r in range(B):
            C = np.unique(_costs_f32(inst, L[r], ell[r]))
            pick = rng.integers(0, len(C) + 1)   # below everything (fallback) ... above everything
            bud[r] = C[0] * 0.5 if pick == 0 else (C[pick - 1] * 1.01 if pick == len(C) else 0.5 * (C[pick - 1] + C[pick]))
        out = orc.dispatch(inst, d, b, Q, L, ell, w, budget=bud)
        order = orc.decide_from_predictions(inst, d, b, Q, L, ell, w)["order"]
        np.testing.assert_array_equal(out["order"], order)      # the LPT key does not depend on budgets
        dq, bq = d.copy(), b.copy()
        for r in order:
            C = _costs_f32(inst, L[r], ell[r])
            J = np.flatnonzero(C <= bud[r])
            if len(J) == 0:
                J = np.flatnonzero(C == C.min())
                n_fallback += 1
            elif len(J) < I:
                n_partial += 1
            # sub-cluster keeps all M tiers' coefficients; only the instance list shrinks
            sub = orc.Instances(tier=inst.tier[J], cap=inst.cap[J], price_in=inst.price_in, price_out=inst.price_out,
                                pre=inst.pre, dec=inst.dec, slope=inst.slope)
            ref = orc.decide_from_predictions(sub, dq[J], bq[J], Q[r:r + 1], L[r:r + 1], ell[r:r + 1], w)
            assert out["assignment"][r] == J[ref["assignment"][0]]
            np.testing.assert_array_equal(out["scores"][r][J], ref["scores"][0])
            mask = np.ones(I, bool)
            mask[J] = False
            assert np.all(out["scores"][r][mask] == -np.inf)
            dq[J], bq[J] = ref["queued"], ref["running"]
            if len(np.flatnonzero(C <= bud[r])):
                assert C[out["assignment"][r]] <= bud[r]          # Eq. 2 holds for the chosen instance
        np.testing.assert_array_equal(out["queued"], dq)
        np.testing.assert_array_equal(out["running"], bq)
    assert n_fallback > 5 and n_partial > 20


def test_max_tokens_closed_form(orc):
    """remaining budget after the prompt, in output tokens at the chosen model's price, rounded down."""
    inst = orc.Instances(tier=[0], cap=[4], price_in=[1.0], price_out=[2.0], pre=[0.0], dec=[10.0], slope=[0.0])
    Q, L = np.array([[0.5]], np.float32), np.array([[50.0]], np.float32)
    for bud, exp in ((500.0, 200), (501.0, 200), (503.9, 201), (100.0, 0), (99.0, 0), (np.inf, INT32_MAX), (1e30, 2147483520)):
        out = orc.dispatch(inst, [0.0], [0], Q, L, [100], [1 / 3] * 3, budget=[bud])
        assert out["max_tokens"][0] == exp, bud
        assert out["assignment"][0] == 0
    free = orc.Instances(tier=[0], cap=[4], price_in=[1.0], price_out=[0.0], pre=[0.0], dec=[10.0], slope=[0.0])
    assert orc.dispatch(free, [0.0], [0], Q, L, [100], [1 / 3] * 3, budget=[150.0])["max_tokens"][0] == INT32_MAX
    assert orc.dispatch(free, [0.0], [0], Q, L, [100], [1 / 3] * 3, budget=[50.0])["max_tokens"][0] == 0


def test_tiebreak_modes_pick_by_queue_or_by_predicted_latency(orc):
    """P:L227 arms 2/3: with w_lat = 0 all replicas of the winning tier tie on S; mode 0 takes the shortest queue d,
    mode 1 the smallest T^ (checked against an independent fp64 T)."""
    rng = np.random.default_rng(8)
    differ = 0
    for _ in range(60):
        inst, d, b, Q, L, ell = _rand_case(orc, rng, B=1, I=int(rng.integers(3, 12)), M=2)
        wq = float(rng.uniform(0, 1))
        w = np.array([wq, 0.0, 1.0 - wq], np.float32)
        o0 = orc.dispatch(inst, d, b, Q, L, ell, w, tiebreak_mode=0)
        o1 = orc.dispatch(inst, d, b, Q, L, ell, w, tiebreak_mode=1)
        np.testing.assert_array_equal(o0["scores"], o1["scores"])
        S = o0["scores"][0]
        top = np.flatnonzero(S == S.max())
        _, _, T = _score_row_f64(inst, d, b, Q[0], L[0], float(ell[0]), w.astype(np.float64))
        i0, i1 = int(o0["assignment"][0]), int(o1["assignment"][0])
        assert i0 in top and i1 in top
        assert d[i0] == d[top].min() and i0 == top[d[top] == d[top].min()][0]
        assert T[i1] <= T[top].min() * (1 + 1e-6)
        differ += int(i0 != i1)
    assert differ > 5   # the two arms do make different choices


def test_tiebreak_mode_is_irrelevant_without_score_ties(orc):
    rng = np.random.default_rng(9)
    for _ in range(20):
        inst, d, b, Q, L, ell = _rand_case(orc, rng, B=6, I=7, M=3)
        w = rng.dirichlet([1, 1, 1]).astype(np.float32)
        o0 = orc.dispatch(inst, d, b, Q, L, ell, w, tiebreak_mode=0)
        if any(len(np.unique(row)) < len(row) for row in o0["scores"]):
            continue
        o1 = orc.dispatch(inst, d, b, Q, L, ell, w, tiebreak_mode=1)
        for key in ("assignment", "scores", "queued", "running"):
            np.testing.assert_array_equal(o0[key], o1[key])


def test_static_prior_equals_live_head_without_prefill_slope_and_queueing(orc):
    """P:L227 arm 4: T^ = nominal TPOT x predicted length, zero telemetry.  The pinned live formula reduces to exactly
    that when pre = 0, slope = 0 and every instance always has a free slot (test_oracle_score pins T = dec*L there)."""
    rng = np.random.default_rng(10)
    for _ in range(20):
        inst, d, b, Q, L, ell = _rand_case(orc, rng, B=8, I=6, M=3)
        w = rng.dirichlet([1, 1, 1]).astype(np.float32)
        out = orc.dispatch(inst, d, b, Q, L, ell, w, latency_mode=1)
        sur = orc.Instances(tier=inst.tier, cap=np.full(inst.I, 10**6), price_in=inst.price_in, price_out=inst.price_out,
                            pre=np.zeros(inst.M), dec=inst.dec, slope=np.zeros(inst.M))
        ref = orc.decide_from_predictions(sur, d, b, Q, L, ell, w)
        for key in ("assignment", "scores", "scores0", "order", "queued"):
            np.testing.assert_array_equal(out[key], ref[key], err_msg=key)
        # zero telemetry: another state changes no score
        d2 = rng.integers(0, 5000, inst.I).astype(np.float32)
        out2 = orc.dispatch(inst, d2, np.minimum(b + 1, inst.cap), Q, L, ell, w, latency_mode=1)
        np.testing.assert_array_equal(out2["scores0"], out["scores0"])
        np.testing.assert_array_equal(out["scores"], out["scores0"])


def test_update_mode_d_only(orc):
    """P:L121 literally: only d grows.  (i) b is untouched and d grows by the chosen L^; (ii) when every instance is
    saturated the b-update of mode 1 is a no-op, so both modes agree bit for bit; (iii) when every instance keeps a
    free slot the wait term stays off, so every request sees its batch-start scores."""
    rng = np.random.default_rng(11)
    for _ in range(20):
        inst, d, b, Q, L, ell = _rand_case(orc, rng, B=7, I=5, M=2)
        w = rng.dirichlet([1, 1, 1]).astype(np.float32)
        o2 = orc.dispatch(inst, d, b, Q, L, ell, w, update_mode=2)
        np.testing.assert_array_equal(o2["running"], b)
        grow = np.zeros(inst.I, np.float64)
        dd = d.copy()
        for r in o2["order"]:
            i = o2["assignment"][r]
            dd[i] = np.float32(dd[i] + L[r, inst.tier[i]])
        np.testing.assert_array_equal(o2["queued"], dd)
        sat = orc.dispatch(inst, d, inst.cap, Q, L, ell, w, update_mode=2)
        ref = orc.dispatch(inst, d, inst.cap, Q, L, ell, w, update_mode=1)
        for key in ("assignment", "scores", "queued", "running"):
            np.testing.assert_array_equal(sat[key], ref[key])
        free = orc.dispatch(inst, d, np.zeros(inst.I, np.int32), Q, L, ell, w, update_mode=2)
        np.testing.assert_array_equal(free["scores"], free["scores0"])
        o0 = orc.dispatch(inst, d, b, Q, L, ell, w, update_mode=0)
        np.testing.assert_array_equal(o0["queued"], d)
        np.testing.assert_array_equal(o0["scores"], o0["scores0"])
