"""Pins of the adaptive batch-size rule (oracle orc_batch_target, reading 27) and of the
stream driver's window logic (paper_2606_17949_b200/stream.py, host logic) run over the oracle."""
import dataclasses

import numpy as np
import pytest

from paper_2606_17949_b200 import stream, synth
from stream_backends import OracleBackend


def _inst(orc, I=13, M=4, cap=16):
    return orc.Instances(**synth.make_instances(I, M, cap=cap))


def test_rule_limits_closed_form_and_monotonicity(orc):
    """All idle -> bs_min; all busy -> bs_max; in between bs_min + floor((bs_max - bs_min) * n_busy / I), non-decreasing
    in the number of busy instances ("larger when more instances are busy, smaller when idle")."""
    inst = _inst(orc)
    I = inst.I
    cap = inst.cap
    assert orc.batch_target(inst, np.zeros(I, np.int32), 4, 64) == (4, 0)
    assert orc.batch_target(inst, cap.copy(), 4, 64) == (64, I)
    assert orc.batch_target(inst, cap + 7, 4, 64) == (64, I)          # beyond cap is still just "busy"
    prev = 0
    for nb in range(I + 1):
        running = np.where(np.arange(I) < nb, cap, cap - 1).astype(np.int32)   # one slot short of busy elsewhere
        t, b = orc.batch_target(inst, running, 4, 64)
        assert b == nb and t == 4 + (60 * nb) // I and t >= prev
        prev = t
    # which instances are busy does not matter, only how many
    rng = np.random.default_rng(0)
    for _ in range(50):
        running = rng.integers(0, 20, I).astype(np.int32)
        nb = int((running >= cap).sum())
        assert orc.batch_target(inst, running, 1, 32) == (1 + (31 * nb) // I, nb)


def test_rule_off_switch_and_bad_arguments(orc):
    """bs_min = bs_max is the fixed batch size of the paper's ablation (bs = 1, 16, 32), whatever the state."""
    inst = _inst(orc)
    rng = np.random.default_rng(1)
    for bs in (1, 16, 32):
        for _ in range(10):
            assert orc.batch_target(inst, rng.integers(0, 40, inst.I).astype(np.int32), bs, bs)[0] == bs
    for lo, hi in ((0, 4), (5, 4), (-1, -1)):
        with pytest.raises(ValueError):
            orc.batch_target(inst, np.zeros(inst.I, np.int32), lo, hi)


def test_busy_means_the_wait_term_applies(orc):
    """The rule's notion of a busy instance is the one the pinned latency head uses ("if the instance has a free
    decode slot only the second term applies"): instance i counts as busy exactly when its queued tokens d_i enter its
    predicted latency -- observed through the pinned dispatch stage: raising d_i alone changes the batch-start score
    matrix iff the rule counted i."""
    rng = np.random.default_rng(2)
    inst = _inst(orc, cap=6)
    I, M = inst.I, inst.M
    Q = rng.uniform(0, 1, (5, M)).astype(np.float32)
    L = rng.lognormal(5.5, 0.5, (5, M)).astype(np.float32)
    plen = rng.integers(10, 2000, 5).astype(np.int32)
    w = (0.2, 0.6, 0.2)
    for trial in range(8):
        running = rng.integers(0, 12, I).astype(np.int32)
        running[rng.integers(0, I)] = inst.cap[0]                       # exactly at cap: busy
        queued = rng.integers(100, 5000, I).astype(np.float32)
        base = orc.decide_from_predictions(inst, queued, running, Q, L, plen, w)["scores0"]
        enters = 0
        for i in range(I):
            q2 = queued.copy()
            q2[i] += 4000.0
            s2 = orc.decide_from_predictions(inst, q2, running, Q, L, plen, w)["scores0"]
            enters += int(not np.array_equal(base, s2))
        assert orc.batch_target(inst, running, 4, 64)[1] == enters


def _small_world(orc, seed=5, N=1500, n_req=400, rate=30.0):
    cfg = dataclasses.replace(synth.CONFIGS["C2"], N=N, d=32, Kc=8, seed=seed)
    bank = synth.make_bank(cfg)
    it = synth.make_instances(cfg.I, cfg.M, cap=4)
    queued, running = synth.make_state(cfg.I, it["cap"], cfg.seed)
    q = synth.make_queries(cfg, B=n_req).numpy()
    p = synth.make_prompt_len(cfg, B=n_req).numpy()
    arrivals = synth.poisson_arrivals_ms(rate, n_req, seed=cfg.seed)
    from parity import bank_to_numpy
    ob = lambda: OracleBackend(orc, bank_to_numpy(bank["emb"]), bank["quality"].numpy(), bank["outlen"].numpy(),
                               orc.Instances(**it), queued.numpy(), running.numpy(), q, p, cfg.k)
    return ob, arrivals, n_req


def test_driver_window_invariants_over_the_oracle(orc):
    """Every request is dispatched exactly once, in arrival order; a window holds between 1 and `target` requests, all
    arrived by the time it fires; it fires when full or when its first request has waited max_wait_ms (never earlier
    than the previous window); the dead-reckoning steps add up to the last fire time."""
    ob, arrivals, n = _small_world(orc)
    be = ob()
    res = stream.drive(be, arrivals, lambda j: synth.PRESETS["balanced"], bs_min=2, bs_max=24, max_wait_ms=80.0)
    assert res.lo[0] == 0 and res.hi[-1] == n and res.lo[1:] == res.hi[:-1]
    assert (be.assignment >= 0).all() and (be.assignment < 13).all()
    last = 0.0
    for lo, hi, fire, tgt in zip(res.lo, res.hi, res.fire_ms, res.target):
        assert 1 <= hi - lo <= tgt and 2 <= tgt <= 24
        assert arrivals[hi - 1] <= fire and fire >= last
        full = hi - lo == min(tgt, n - lo)
        assert full or fire == max(last, arrivals[lo] + 80.0)           # not full: it timed out
        if hi < n and not full:
            assert arrivals[hi] > fire                                  # nobody who had arrived was left behind
        last = fire
    assert abs(sum(res.elapsed_ms) - res.fire_ms[-1]) < 1e-3 * len(res.lo)
    assert (res.batch_wait_ms(arrivals) >= 0).all()


def test_adaptive_windows_grow_with_busyness_and_fixed_size_is_fixed(orc):
    """The same arrivals over a saturated and over an idle cluster: the saturated one forms larger batches;
    with bs_min = bs_max every window that does not time out holds exactly that many requests."""
    ob, arrivals, n = _small_world(orc, rate=200.0)
    busy, idle = ob(), ob()
    busy.bq[:] = 50
    busy.dq[:] = 1e9            # never drains within the stream
    idle.bq[:] = 0
    idle.dq[:] = 0
    rb_ = stream.drive(busy, arrivals, lambda j: synth.PRESETS["balanced"], bs_min=2, bs_max=32, max_wait_ms=1e9, max_windows=6)
    ri = stream.drive(idle, arrivals, lambda j: synth.PRESETS["balanced"], bs_min=2, bs_max=32, max_wait_ms=1e9, max_windows=6)
    assert rb_.target[0] == 32 and ri.target[0] == 2
    assert all(t == 32 for t in rb_.target) and np.mean(ri.target) < 32
    fx = ob()
    rf = stream.drive(fx, arrivals, lambda j: synth.PRESETS["balanced"], bs_min=16, bs_max=16, max_wait_ms=1e9)
    sizes = [h - l for l, h in zip(rf.lo, rf.hi)]
    assert all(s == 16 for s in sizes[:-1]) and 1 <= sizes[-1] <= 16
