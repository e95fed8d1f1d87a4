"""rb_decide_from_predictions_static: the score + dispatch stages with their scratch in a fixed __device__ array of the
library (no allocation of any kind), against the existing rb_decide_from_predictions path.

Collected last (file name): the run uses `pytest -x`, a failure here must not hide another test.  Passes alone in
a fresh process and after the other tests (the array is per GPU, keeps the last call's contents and needs no clearing)."""
import numpy as np
import pytest
import torch

from paper_2606_17949_b200 import synth

pytestmark = pytest.mark.gpu


def _routers(I, M, max_batch, **modes):
    from paper_2606_17949_b200.router import Router
    emb = torch.randn(64, 16).cuda()
    ql, ol = torch.rand(64, M).cuda(), torch.rand(64, M).cuda() * 100 + 1
    it = synth.make_instances(I, M, cap=4)
    rts = []
    for _ in range(2):
        rt = Router(emb, ql, ol, 4, store="f32", max_batch=max_batch, **modes)
        rt.set_instances(**it)
        rts.append(rt)
    return rts, it


@pytest.mark.parametrize("I,M,B", [(13, 4, 24), (200, 8, 700), (33, 3, 1024)])
def test_static_scratch_path_equals_the_existing_path_on_two_calls_in_a_row(I, M, B):
    """Two committed decisions in a row with an advance in between, different batches: assignment and dead-reckoned state
    after each call equal the existing path's bit for bit (the tolerance of every dispatch test: none)."""
    (ref_rt, rt), it = _routers(I, M, B)
    rng = np.random.default_rng(900 + I + B)
    queued = torch.from_numpy(rng.integers(0, 20001, I).astype(np.float32))
    running = torch.from_numpy(np.minimum(rng.integers(0, 6, I), it["cap"]).astype(np.int32))
    ref_rt.set_state(queued, running)
    rt.set_state(queued, running)
    out = torch.full((B,), -7, dtype=torch.int32, device="cuda")
    for call, w in enumerate([(0.2, 0.5, 0.3), (0.0, 1.0, 0.0)]):
        Bc = B if call == 0 else max(1, B // 2)          # the second call leaves stale words of the first in the array
        Q = torch.from_numpy(rng.uniform(0, 1, (Bc, M)).astype(np.float32)).cuda()
        L = torch.from_numpy(rng.lognormal(5.5, 0.7, (Bc, M)).astype(np.float32)).cuda()
        plen = torch.from_numpy(rng.integers(1, 4000, Bc).astype(np.int32)).cuda()
        ref_rt.advance_state(3.0 + call)
        rt.advance_state(3.0 + call)
        ref = ref_rt.decide_from_predictions(Q, L, plen, w, commit=1)
        got = rt.decide_from_predictions_static(Q, L, plen, w, commit=1, assignment=out[:Bc])
        ref_rt.sync()
        rt.sync()
        assert torch.equal(got.cpu(), ref["assignment"].cpu()), (call, "assignment")
        s_ref, s = ref_rt.get_state(), rt.get_state()
        assert torch.equal(s[0], s_ref[0]) and torch.equal(s[1], s_ref[1]), (call, "state")
    # commit = 0 leaves the state alone and gives the same assignment as the existing path
    before = rt.get_state()
    ref = ref_rt.decide_from_predictions(Q, L, plen, (1.0, 0.0, 0.0), commit=0)
    got = rt.decide_from_predictions_static(Q, L, plen, (1.0, 0.0, 0.0), commit=0)
    rt.sync()
    assert torch.equal(got.cpu(), ref["assignment"].cpu())
    after = rt.get_state()
    assert torch.equal(before[0], after[0]) and torch.equal(before[1], after[1])
    ref_rt.close()
    rt.close()


def test_static_scratch_path_rejects_what_it_cannot_hold():
    """Sizes beyond the array (B > 1024, or B * M > 8192) and host buffers are refused with a clear error before anything
    is launched; the state is untouched and the next valid call works."""
    from paper_2606_17949_b200 import binding as rb
    (ref_rt, rt), it = _routers(20, 16, 2048)
    I, M = 20, 16
    rng = np.random.default_rng(5)
    queued = torch.from_numpy(rng.integers(0, 20001, I).astype(np.float32))
    running = torch.from_numpy(np.minimum(rng.integers(0, 6, I), it["cap"]).astype(np.int32))
    for r in (ref_rt, rt):
        r.set_state(queued, running)

    def batch(B):
        return (torch.rand(B, M, device="cuda"), torch.rand(B, M, device="cuda") * 300 + 1,
                torch.randint(1, 4000, (B,), dtype=torch.int32, device="cuda"))

    w = (0.3, 0.4, 0.3)
    for B in (1025, 513):                                  # B > 1024;  513 * 16 = 8208 > 8192
        Q, L, plen = batch(B)
        with pytest.raises(rb.RbError) as e:
            rt.decide_from_predictions_static(Q, L, plen, w, commit=1)
        assert "exceeds the static scratch" in str(e.value)
    Q, L, plen = batch(8)
    with pytest.raises(rb.RbError) as e:                   # a host buffer
        rt.decide_from_predictions_static(Q.cpu(), L, plen, w, commit=1, assignment=torch.empty(8, dtype=torch.int32, device="cuda"))
    assert "device memory" in str(e.value)
    s = rt.get_state()
    assert torch.equal(s[0], queued) and torch.equal(s[1], running)
    Q, L, plen = batch(512)                                # 512 * 16 = 8192: the largest batch at M = 16
    ref = ref_rt.decide_from_predictions(Q, L, plen, w, commit=1)
    got = rt.decide_from_predictions_static(Q, L, plen, w, commit=1)
    rt.sync()
    ref_rt.sync()
    assert torch.equal(got.cpu(), ref["assignment"].cpu())
    s_ref, s = ref_rt.get_state(), rt.get_state()
    assert torch.equal(s[0], s_ref[0]) and torch.equal(s[1], s_ref[1])
    ref_rt.close()
    rt.close()
