"""Parity tests proper: the CUDA path (through the C ABI) against the oracle, element by element on the same
seeded inputs.  Run with -m gpu on a B200."""
import dataclasses

import numpy as np
import pytest
import torch

import parity
from paper_2606_17949_b200 import synth

pytestmark = pytest.mark.gpu


def _router(bank, cfg, **kw):
    from paper_2606_17949_b200.router import Router
    return Router(bank["emb"], bank["quality"], bank["outlen"], cfg.k, store=cfg.store, **kw)


def _setup(cfg, device="cuda", B=None, sort_bank=False, **kw):
    bank = synth.make_bank(cfg, device=device)
    if sort_bank:   # rows of one mixture component become contiguous: a query's neighbours share one CTA's slab
        order = torch.argsort(bank["comp"], stable=True)
        bank = {k_: v[order].contiguous() for k_, v in bank.items()}
    it = synth.make_instances(cfg.I, cfg.M)
    queued, running = synth.make_state(cfg.I, it["cap"], cfg.seed)
    query = synth.make_queries(cfg, B=B, device=device)
    plen = synth.make_prompt_len(cfg, B=B, device=device)
    torch.cuda.synchronize()
    rt = _router(bank, cfg, **kw)
    rt.set_instances(**it)
    rt.set_state(queued, running)
    return bank, it, queued, running, query, plen, rt


def _np(out):
    torch.cuda.synchronize()
    return {k: v.detach().cpu().numpy() for k, v in out.items()}


def _full_parity(orc, cfg, w, B=None, sim_tol=0.0, **kw):
    bank, it, queued, running, query, plen, rt = _setup(cfg, B=B, **kw)
    out = rt.decide(query, plen, w)
    rt.sync()
    g = _np(out)
    bank_np = parity.bank_to_numpy(bank["emb"])
    qn, ln = bank["quality"].cpu().numpy(), bank["outlen"].cpu().numpy()
    query_np, plen_np = query.cpu().numpy(), plen.cpu().numpy()
    log = []
    oi, os_, near = parity.check_topk(orc, bank_np, query_np, cfg.store, cfg.k, g["nn_idx"], g["nn_sim"], sim_tol, log)
    parity.check_predictions(orc, g["pred_quality"], g["pred_outlen"], g["nn_idx"], g["nn_sim"], oi, os_, near, qn, ln,
                             weight_mode=kw.get("weight_mode", 0), raw_sums=sim_tol > 0)
    inst = orc.Instances(**it)
    state = rt.get_state()
    parity.check_dispatch(orc, inst, queued.numpy(), running.numpy(), g["pred_quality"], g["pred_outlen"], plen_np, w, g,
                          state_after=(state[0].numpy(), state[1].numpy()))
    rt.close()
    return g, near, log


def test_c1_tiny_full_parity(orc):
    """BASELINE.json configs[0]: N=4096, d=384 fp32 bank, B=16, I=13, k=10, w=(1/3,1/3,1/3), seed 0.
    fp32 storage: similarities, neighbour order and predictions are bit-identical to the oracle."""
    cfg = synth.CONFIGS["C1"]
    g, near, _ = _full_parity(orc, cfg, synth.PRESETS["balanced"])
    assert near == []


@pytest.mark.parametrize("slack", [6, 0])
@pytest.mark.parametrize("N,d,B", [(5000, 384, 16), (20011, 128, 300), (777, 64, 5), (64 * 148 * 2 + 3, 256, 128)])
def test_bf16_scan_parity_ragged(orc, N, d, B, slack):
    """tcgen05 scan + merge + aggregate on sizes spanning several tiles, a ragged tail (N not a multiple of
    64), several m-tiles (B > 128) and fewer slabs than SMs (N = 777)."""
    cfg = dataclasses.replace(synth.CONFIGS["C2"], N=N, d=d, B=B, Kc=16, seed=11)
    tol = 0.0 if slack > 0 else 4e-6   # re-ranked similarities are exact; raw tensor-core sums are not
    g, near, log = _full_parity(orc, cfg, synth.PRESETS["balanced"], sim_tol=tol, rerank_slack=slack, max_batch=512)
    assert len(near) <= max(1, B // 20), log


@pytest.mark.parametrize("scan_list", [4, 8, 16])
@pytest.mark.parametrize("N,B,k,slack", [(20000, 24, 10, 6), (3000, 7, 10, 0), (150000, 130, 32, 8)])
def test_short_scan_lists_rescan_clustered_bank(orc, scan_list, N, B, k, slack):
    """The scan keeps only scan_list entries per (CTA, query); with the bank sorted by mixture component all of a
    query's neighbours sit in one or two slabs, so the finishing kernel must search those slabs again
    (exactly) to stay correct.  Also run on the unsorted bank, where the rescan is (almost) never taken."""
    cfg = dataclasses.replace(synth.CONFIGS["C2"], N=N, d=128, B=B, k=k, Kc=8, seed=21)
    tol = 0.0 if slack > 0 else 4e-6
    for sort_bank in (True, False):
        g, near, log = _full_parity(orc, cfg, synth.PRESETS["balanced"], sim_tol=tol, rerank_slack=slack, max_batch=256,
                                    scan_list=scan_list, sort_bank=sort_bank)
        assert len(near) <= max(1, B // 20), log


@pytest.mark.parametrize("N,d,B,k,slack", [(40000, 128, 129, 10, 6), (300, 64, 256, 10, 6), (25000, 192, 600, 10, 0),
                                            (19001, 64, 1030, 32, 8), (256 * 74 * 3 + 100, 64, 257, 5, 3)])
def test_bf16_pair_scan_large_batches(orc, N, d, B, k, slack):
    """B > 128 runs the CTA-pair scan (tcgen05 cta_group::2, 256-query m-tiles): one and several m-pairs, a
    half-empty last pair, fewer 256-row tiles than clusters (N = 300), a ragged last tile, K tails (d = 192)."""
    cfg = dataclasses.replace(synth.CONFIGS["C2"], N=N, d=d, B=B, k=k, Kc=16, seed=31)
    tol = 0.0 if slack > 0 else 4e-6
    for sort_bank in (False, True):
        g, near, log = _full_parity(orc, cfg, synth.PRESETS["balanced"], sim_tol=tol, rerank_slack=slack, max_batch=1100,
                                    sort_bank=sort_bank)
        assert len(near) <= max(1, B // 20), log


@pytest.mark.parametrize("k,slack", [(32, 8), (10, 6)])
@pytest.mark.parametrize("sort_bank", [False, True])
def test_bf16_pair_scan_long_slabs_all_queries(orc, k, slack, sort_bank):
    """The CTA-pair scan in its long-slab regime, every query checked: N = 256 * 74 * 41 + 77 rows (41-42 tiles of 256
    rows per cluster), B = 700 (three 256-query m-pairs, the last one ragged), k = 32 with slack 8 (candidate lists of
    40 against the scan's 32-entry global lists: pooled cross-slab admission bounds, list caps and the finishing
    kernel's re-search of a popped-out slab all take part) and k = 10; on the bank as drawn and on the bank sorted by
    mixture component (all of a query's neighbours in one or two clusters' slabs -- the re-search is certain)."""
    cfg = dataclasses.replace(synth.CONFIGS["C2"], N=256 * 74 * 41 + 77, d=64, B=700, k=k, Kc=24, seed=41)
    g, near, log = _full_parity(orc, cfg, synth.PRESETS["balanced"], rerank_slack=slack, max_batch=768, sort_bank=sort_bank)
    assert len(near) <= 700 // 20, log


@pytest.mark.parametrize("B", [8, 40, 130, 300])
def test_k32_full_length_scan_lists(orc, B):
    """k = 32 with slack 8 keeps 64-entry lists in the scan when slabs are long (C4: 67k rows per CTA); forced here
    with scan_list = 64 on a small bank.  The finishing kernel's shared memory bounds the query replicas."""
    cfg = dataclasses.replace(synth.CONFIGS["C2"], N=30000, d=128, B=B, k=32, Kc=16, seed=32)
    _full_parity(orc, cfg, synth.PRESETS["balanced"], rerank_slack=8, max_batch=512, scan_list=64)


def test_bf16_k32_and_uniform_weights(orc):
    cfg = dataclasses.replace(synth.CONFIGS["C2"], N=30000, d=384, B=40, k=32, Kc=16, seed=12)
    _full_parity(orc, cfg, synth.PRESETS["quality"], rerank_slack=8, max_batch=64)
    _full_parity(orc, cfg, synth.PRESETS["cost"], rerank_slack=0, sim_tol=4e-6, max_batch=64, weight_mode=1)


def test_k_equals_one_and_batch_of_one(orc):
    cfg = dataclasses.replace(synth.CONFIGS["C2"], N=4100, d=64, B=1, k=1, Kc=8, seed=13)
    _full_parity(orc, cfg, synth.PRESETS["latency"], max_batch=1)


def test_tiny_bank_k_equals_N(orc):
    cfg = dataclasses.replace(synth.CONFIGS["C1"], N=12, d=16, B=3, k=12, Kc=2, seed=14)
    _full_parity(orc, cfg, synth.PRESETS["balanced"], max_batch=4)
    cfg = dataclasses.replace(cfg, store="bf16")
    _full_parity(orc, cfg, synth.PRESETS["balanced"], max_batch=4, rerank_slack=0, sim_tol=4e-6)


def test_host_buffers_equal_device_buffers(orc):
    cfg = dataclasses.replace(synth.CONFIGS["C2"], N=9000, d=128, B=33, Kc=16, seed=15)
    bank, it, queued, running, query, plen, rt = _setup(cfg, max_batch=64)
    dev = _np(rt.decide(query, plen, synth.PRESETS["balanced"]))
    rt.set_state(queued, running)
    host = rt.decide(query.cpu(), plen.cpu(), synth.PRESETS["balanced"])   # host in, host out: complete on return
    for key in dev:
        assert np.array_equal(dev[key], host[key].numpy()), key
    rt.close()


def test_router_is_ordered_against_the_callers_stream():
    """Router's stream contract: inputs produced on torch's current stream just before the call (behind several
    milliseconds of queued work) and outputs consumed on it just after, with no host synchronisation anywhere, give the
    results of a fully synchronised run."""
    cfg = dataclasses.replace(synth.CONFIGS["C2"], N=9000, d=128, B=33, Kc=16, seed=16)
    bank, it, queued, running, query, plen, rt = _setup(cfg, max_batch=64)
    w = synth.PRESETS["balanced"]
    ref = _np(rt.decide(query, plen, w))
    torch.cuda.synchronize()
    big = torch.randn(6144, 6144, device="cuda")
    for trial in range(3):
        rt.set_state(queued, running)
        torch.cuda.synchronize()
        x = big
        for _ in range(6):
            x = (x @ big) * 1e-3                      # keeps the current stream busy for a few milliseconds
        q = query + 0.0 * x[0, 0]                     # the inputs exist only once that work has run
        p = plen + (0 * x[0, 0]).to(torch.int32)
        out = rt.decide(q, p, w)
        got = {k_: v.clone() for k_, v in out.items()}   # consumed on the current stream, no synchronisation in between
        del out, q, p
        junk = [torch.full((33, 128), float(trial), device="cuda") for _ in range(8)]   # reuses freed blocks, if any were freed early
        torch.cuda.synchronize()
        for key in ref:
            assert np.array_equal(ref[key], got[key].cpu().numpy()), (trial, key)
        del junk
    rt.close()


@pytest.mark.parametrize("I,M,B", [(13, 4, 16), (64, 4, 200), (256, 8, 1024), (1, 1, 7), (33, 3, 50), (1024, 16, 64)])
@pytest.mark.parametrize("lpt,upd", [(1, 1), (0, 1), (1, 0)])
def test_dispatch_from_predictions_bit_exact(orc, I, M, B, lpt, upd):
    """Score + LPT dispatch given identical predictions: scores bit-equal (bar: 1e-5 rel), assignment, order
    and post-batch state bit-exact; single-warp (I <= 32) and multi-warp kernels; commit on/off."""
    from paper_2606_17949_b200.router import Router
    rng = np.random.default_rng(100 + I + B)
    it = synth.make_instances(I, M, cap=int(rng.integers(1, 9)))
    bank = dict(emb=torch.randn(64, 16), quality=torch.rand(64, M), outlen=torch.rand(64, M) * 100 + 1)
    rt = Router(bank["emb"].cuda(), bank["quality"].cuda(), bank["outlen"].cuda(), 4, store="f32", max_batch=B,
                lpt_enabled=lpt, update_enabled=upd)
    rt.set_instances(**it)
    queued = torch.from_numpy(rng.integers(0, 20001, I).astype(np.float32))
    running = torch.from_numpy(np.minimum(rng.integers(0, 12, I), it["cap"]).astype(np.int32))
    rt.set_state(queued, running)
    Q = torch.from_numpy(rng.uniform(0, 1, (B, M)).astype(np.float32))
    L = torch.from_numpy(rng.lognormal(5.5, 0.7, (B, M)).astype(np.float32))
    if B > 8:
        L[5] = L[2]                      # equal LPT keys -> request index decides
    plen = torch.from_numpy(rng.integers(1, 4000, B).astype(np.int32))
    inst = orc.Instances(**it)
    for w in [synth.PRESETS["balanced"], (1.0, 0.0, 0.0), (0.0, 1.0, 0.0), (0.0, 0.0, 1.0), (0.2, 0.5, 0.3)]:
        out = rt.decide_from_predictions(Q.cuda(), L.cuda(), plen.cuda(), w, commit=0)
        g = _np(out)
        ref = parity.check_dispatch(orc, inst, queued.numpy(), running.numpy(), Q.numpy(), L.numpy(), plen.numpy(), w, g,
                                    lpt_enabled=lpt, update_enabled=upd)
        assert np.array_equal(g["scores"], ref["scores"]) and np.array_equal(g["scores0"], ref["scores0"])
        s = rt.get_state()
        assert np.array_equal(s[0].numpy(), queued.numpy()) and np.array_equal(s[1].numpy(), running.numpy())
    out = rt.decide_from_predictions(Q, L, plen, (0.2, 0.5, 0.3), commit=1)      # host buffers, committed
    s = rt.get_state()
    parity.check_dispatch(orc, inst, queued.numpy(), running.numpy(), Q.numpy(), L.numpy(), plen.numpy(), (0.2, 0.5, 0.3),
                          {k: v.numpy() for k, v in out.items()}, lpt_enabled=lpt, update_enabled=upd,
                          state_after=(s[0].numpy(), s[1].numpy()))
    rt.close()


def test_advance_state_and_stream_lockstep(orc):
    """C2-shaped stream in miniature: Poisson windows, rb_advance_state between batches, all four presets;
    the dead-reckoned state stays bit-identical to the oracle's over the whole stream."""
    cfg = dataclasses.replace(synth.CONFIGS["C2"], N=6000, d=128, Kc=16, seed=16)
    bank, it, queued, running, _, _, rt = _setup(cfg, max_batch=64)
    inst = orc.Instances(**it)
    sizes, elapsed = synth.poisson_windows(30.0, 60, seed=16)
    allq = synth.make_queries(cfg, B=sum(sizes), device="cuda")
    allp = synth.make_prompt_len(cfg, B=sum(sizes), device="cuda")
    torch.cuda.synchronize()
    dq, bq = queued.numpy(), running.numpy()
    presets = list(synth.PRESETS.values())
    off = 0
    for j, (B, dt) in enumerate(zip(sizes, elapsed)):
        rt.advance_state(dt)
        dq, bq = orc.advance_state(inst, dq, bq, np.float32(dt))
        w = presets[j % 4]
        out = _np(rt.decide(allq[off:off + B], allp[off:off + B], w, want=("scores", "pred")))
        s = rt.get_state()
        ref = parity.check_dispatch(orc, inst, dq, bq, out["pred_quality"], out["pred_outlen"],
                                    allp[off:off + B].cpu().numpy(), w, out, state_after=(s[0].numpy(), s[1].numpy()))
        dq, bq = ref["queued"], ref["running"]
        off += B
    assert 4 <= min(sizes) and max(sizes) <= 64
    rt.close()


def test_graph_replay_equals_direct_launch(orc):
    cfg = dataclasses.replace(synth.CONFIGS["C2"], N=8000, d=256, B=24, Kc=16, seed=17)
    bank, it, queued, running, query, plen, rt = _setup(cfg, max_batch=32, use_graph=1)
    a = _np(rt.decide(query, plen, synth.PRESETS["balanced"]))
    rt.set_state(queued, running)
    b = _np(rt.decide(query, plen, synth.PRESETS["balanced"]))    # replay of the captured graph
    rt.close()
    bank2, _, _, _, _, _, rt2 = _setup(cfg, max_batch=32, use_graph=0)
    c = _np(rt2.decide(query, plen, synth.PRESETS["balanced"]))
    rt2.close()
    for key in a:
        assert np.array_equal(a[key], b[key]) and np.array_equal(a[key], c[key]), key


def test_error_codes_and_call_order():
    from paper_2606_17949_b200 import binding as rb
    from paper_2606_17949_b200.router import Router
    emb = torch.randn(100, 16).cuda()
    lab = torch.rand(100, 2).cuda()
    with pytest.raises(rb.RbError) as e:
        Router(emb, lab, lab, 101, store="f32")          # k > N
    assert e.value.status == rb.RB_EINVAL
    with pytest.raises(rb.RbError):
        Router(torch.randn(100, 12).cuda(), lab, lab, 4)   # d % 8 != 0
    rt = Router(emb, lab, lab, 4, store="f32", max_batch=8)
    q = torch.randn(4, 16).cuda()
    pl = torch.ones(4, dtype=torch.int32).cuda()
    with pytest.raises(rb.RbError) as e:
        rt.decide(q, pl, (1 / 3, 1 / 3, 1 / 3))
    assert e.value.status == rb.RB_ESTATE
    it = synth.make_instances(3, 2)
    rt.set_instances(**it)
    for bad_w in [(0.5, 0.5, 0.5), (-0.1, 0.6, 0.5), (float("nan"), 0.5, 0.5)]:
        with pytest.raises(rb.RbError) as e:
            rt.decide(q, pl, bad_w)
        assert e.value.status == rb.RB_EINVAL
    with pytest.raises(rb.RbError):
        rt.decide(torch.randn(9, 16).cuda(), torch.ones(9, dtype=torch.int32).cuda(), (1, 0, 0))   # B > max_batch
    with pytest.raises(rb.RbError):
        rt.advance_state(-1.0)
    bad = dict(it)
    bad["tier"] = [0, 1, 2]
    with pytest.raises(rb.RbError):
        rt.set_instances(**bad)
    out = rt.decide(q, pl, (1 / 3, 1 / 3, 1 / 3))
    rt.sync()
    assert rt.launch_count() > 0
    assert int(out["assignment"].min()) >= 0 and int(out["assignment"].max()) < 3
    rt.close()


def test_c2_full_size_parity(orc):
    """BASELINE.json configs[1] at full size (N=100k, d=768 bf16, B=64, I=13), in the launch configuration
    bench.py times (graph replay, re-rank slack 6): every query checked against the oracle."""
    cfg = synth.CONFIGS["C2"]
    g, near, log = _full_parity(orc, cfg, synth.PRESETS["balanced"], max_batch=64)
    assert len(near) <= 3, log


def test_c4_bank_scan_all_64_queries_parity(orc):
    """BASELINE.json configs[3] (N=10M, d=384 bf16 = 7.68 GB), B=64 launch shape (single-CTA scan, 16-entry lists over
    67k-row slabs): ALL 64 queries checked against the oracle's brute-force scan of the whole bank (BASELINE.md section 3:
    full verification for C4 with B <= 64)."""
    cfg = synth.CONFIGS["C4"]
    bank, it, queued, running, query, plen, rt = _setup(cfg, max_batch=64)
    out = _np(rt.estimate(query))
    rt.close()
    bank_np = parity.bank_to_numpy(bank["emb"])
    qn, ln = bank["quality"].cpu().numpy(), bank["outlen"].cpu().numpy()
    del bank
    torch.cuda.empty_cache()
    log = []
    oi, os_, near = parity.check_topk(orc, bank_np, query.cpu().numpy(), "bf16", cfg.k, out["nn_idx"], out["nn_sim"], 0.0, log)
    parity.check_predictions(orc, out["pred_quality"], out["pred_outlen"], out["nn_idx"], out["nn_sim"], oi, os_, near, qn, ln)
    assert len(near) <= 4, log


def _sampled_estimate_parity(orc, cfg, bank, query, out, rows, max_near):
    bank_np = parity.bank_to_numpy(bank["emb"])
    qn, ln = bank["quality"].cpu().numpy(), bank["outlen"].cpu().numpy()
    log = []
    oi, os_, near = parity.check_topk(orc, bank_np, query.cpu().numpy()[rows], "bf16", cfg.k, out["nn_idx"][rows],
                                      out["nn_sim"][rows], 0.0, log)
    parity.check_predictions(orc, out["pred_quality"][rows], out["pred_outlen"][rows], out["nn_idx"][rows],
                             out["nn_sim"][rows], oi, os_, near, qn, ln)
    assert len(near) <= max_near, log


def test_c3_full_size_sampled_parity(orc):
    """BASELINE.json configs[2] at full size (N=1M, d=1024 bf16, M=8, I=256, B=1024, Zipf-skewed topics) through
    rb_decide in the launch shape bench.py's scan_c3 leg times (CTA-pair scan, 4 m-pairs x ~53 tiles per cluster):
    ALL 1024 queries against the oracle's brute-force scan (about 100 s of oracle time on 16 host threads), and the whole
    dispatch (B=1024 x I=256) against the oracle from the GPU's predictions."""
    cfg = synth.CONFIGS["C3"]
    bank, it, queued, running, query, plen, rt = _setup(cfg, max_batch=cfg.B)
    w = synth.PRESETS["balanced"]
    g = _np(rt.decide(query, plen, w))
    state = rt.get_state()
    rt.close()
    _sampled_estimate_parity(orc, cfg, bank, query, g, list(range(cfg.B)), 40)
    parity.check_dispatch(orc, orc.Instances(**it), queued.numpy(), running.numpy(), g["pred_quality"], g["pred_outlen"],
                          plen.cpu().numpy(), w, g, state_after=(state[0].numpy(), state[1].numpy()))
    # properties that hold at any size: neighbours distinct and in range, similarities sorted, predictions in the labels' range
    assert (g["nn_idx"] >= 0).all() and (g["nn_idx"] < cfg.N).all()
    assert (np.diff(g["nn_sim"], axis=1) <= 0).all()
    assert (g["pred_quality"] >= 0).all() and (g["pred_quality"] <= 1).all()
    assert (g["pred_outlen"] >= 1).all() and (g["pred_outlen"] <= 8192).all()


@pytest.mark.parametrize("B,k,slack", [(4096, 32, 8), (512, 10, 6), (1, 32, 8)])
def test_c4_large_batch_sampled_parity(orc, B, k, slack):
    """BASELINE.json configs[3] sweep ends: N=10M x d=384 bf16 with B=4096 / k=32 (tensor-bound, CTA-pair scan),
    B=512 / k=10 and B=1 / k=32: a seeded 64-query subset (first and last row of the batch always
    included, every 256-query m-pair represented) against the oracle's brute-force scan of the whole bank."""
    cfg = dataclasses.replace(synth.CONFIGS["C4"], k=k)
    bank = synth.make_bank(cfg, device="cuda")
    query = synth.make_queries(cfg, B=B, device="cuda")
    torch.cuda.synchronize()
    rt = _router(bank, cfg, max_batch=B, rerank_slack=slack)
    out = _np(rt.estimate(query))
    rt.close()
    # stratified: one seeded row out of each of 64 equal strata of the batch (every 256-query m-pair and every lane
    # quarter is hit), plus the first and the last row
    rng = np.random.default_rng(1000 + B)
    n = min(B, 64)
    rows = sorted(set([0, B - 1]) | {j * B // n + int(rng.integers(0, max(1, B // n))) for j in range(n)})
    _sampled_estimate_parity(orc, cfg, bank, query, out, rows, 4)
    assert (out["nn_idx"] >= 0).all() and (out["nn_idx"] < cfg.N).all()
    assert (np.diff(out["nn_sim"], axis=1) <= 0).all()


def test_c5_weight_sweep_all_66_points_bit_exact(orc):
    """BASELINE.json configs[4]: N=1M x d=768, B=1024, I=256, M=8.  One estimate, then every point of the 3-simplex at
    step 0.1 through rb_decide_from_predictions(commit=0) from the same state: assignment, order, scores and scores0
    against the oracle for all 66 points; the state must be untouched afterwards."""
    cfg = synth.CONFIGS["C5"]
    bank, it, queued, running, query, plen, rt = _setup(cfg, max_batch=cfg.B)
    est = rt.estimate(query)
    rt.sync()
    # ALL 1024 queries against the brute-force oracle (about 40 s of oracle time)
    _sampled_estimate_parity(orc, cfg, bank, query, _np(est), list(range(cfg.B)), 40)
    inst = orc.Instances(**it)
    pq, pl = est["pred_quality"].cpu().numpy(), est["pred_outlen"].cpu().numpy()
    pts = synth.simplex_points(0.1)
    assert len(pts) == 66
    for w in pts:
        g = _np(rt.decide_from_predictions(est["pred_quality"], est["pred_outlen"], plen, w, commit=0))
        ref = parity.check_dispatch(orc, inst, queued.numpy(), running.numpy(), pq, pl, plen.cpu().numpy(), w, g)
        assert np.array_equal(g["scores"], ref["scores"]) and np.array_equal(g["scores0"], ref["scores0"])
    s = rt.get_state()
    assert np.array_equal(s[0].numpy(), queued.numpy()) and np.array_equal(s[1].numpy(), running.numpy())
    rt.close()


def _random_budgets(rng, it, L, plen, frac_inf=0.25):
    """Budgets around each request's own tier costs (below the cheapest -> fallback, between tiers, above all),
    kept 1 % away from every cost so that fp32 admission is unambiguous; a share unconstrained (+inf)."""
    pin, pout = np.asarray(it["price_in"], np.float32), np.asarray(it["price_out"], np.float32)
    tiers = sorted(set(it["tier"]))
    bud = np.empty(len(plen), np.float32)
    for r in range(len(plen)):
        C = np.unique((np.float32(plen[r]) * pin[tiers] + L[r, tiers] * pout[tiers]).astype(np.float32))
        pick = rng.integers(0, len(C) + 1)
        bud[r] = C[0] * 0.5 if pick == 0 else (C[-1] * 1.01 if pick == len(C) else 0.5 * (C[pick - 1] + C[pick]))
        if rng.uniform() < frac_inf:
            bud[r] = np.inf
    return bud


@pytest.mark.parametrize("I,M,B", [(13, 4, 16), (64, 4, 200), (256, 8, 1024), (33, 3, 50)])
@pytest.mark.parametrize("upd,tb,lat", [(1, 0, 0), (2, 0, 0), (1, 1, 0), (1, 0, 1), (2, 1, 1), (0, 1, 0)])
def test_budget_filter_and_dispatch_modes_bit_exact(orc, I, M, B, upd, tb, lat):
    """SURVEY 8(f) #1 + #2: Eq. 2 admission filter (per-request budgets incl. the nothing-fits fallback and +inf),
    max_tokens clamp, tie-break / latency / update modes: everything bit-exact against orc_dispatch."""
    from paper_2606_17949_b200.router import Router
    rng = np.random.default_rng(7 * I + B + 100 * upd + 10 * tb + lat)
    it = synth.make_instances(I, M, cap=int(rng.integers(1, 9)))
    bank = dict(emb=torch.randn(64, 16), quality=torch.rand(64, M), outlen=torch.rand(64, M) * 100 + 1)
    rt = Router(bank["emb"].cuda(), bank["quality"].cuda(), bank["outlen"].cuda(), 4, store="f32", max_batch=B,
                update_enabled=upd, tiebreak_mode=tb, latency_mode=lat)
    rt.set_instances(**it)
    queued = rng.integers(0, 20001, I).astype(np.float32)
    queued[: I // 3] = queued[0]         # equal queues -> the index decides
    running = np.minimum(rng.integers(0, 12, I), it["cap"]).astype(np.int32)
    Q = rng.uniform(0, 1, (B, M)).astype(np.float32)
    L = rng.lognormal(5.5, 0.7, (B, M)).astype(np.float32)
    plen = rng.integers(1, 4000, B).astype(np.int32)
    bud = _random_budgets(rng, it, L, plen)
    inst = orc.Instances(**it)
    for w in [synth.PRESETS["balanced"], (1.0, 0.0, 0.0), (0.5, 0.0, 0.5), (0.0, 1.0, 0.0), (0.0, 0.0, 1.0)]:
        for budget in (bud, None):
            rt.set_state(torch.from_numpy(queued), torch.from_numpy(running))
            out = rt.decide_from_predictions(torch.from_numpy(Q).cuda(), torch.from_numpy(L).cuda(),
                                             torch.from_numpy(plen).cuda(), w, commit=1,
                                             budget=None if budget is None else torch.from_numpy(budget).cuda())
            g = _np(out)
            ref = orc.dispatch(inst, queued, running, Q, L, plen, w, budget=budget, update_mode=upd, tiebreak_mode=tb,
                               latency_mode=lat)
            for key in ("assignment", "order", "scores", "scores0"):
                assert np.array_equal(g[key], ref[key]), (key, w, budget is None)
            if budget is not None:
                assert np.array_equal(g["max_tokens"], ref["max_tokens"])
                fits = (g["scores"] > -np.inf).any(axis=1)
                assert fits.all()
            s = rt.get_state()
            assert np.array_equal(s[0].numpy(), ref["queued"]) and np.array_equal(s[1].numpy(), ref["running"])
    rt.close()


def test_decide_budgeted_full_path(orc):
    """rb_decide_budgeted end to end (bf16 scan -> finish kernel's terms with the filter -> dispatch), device and host
    buffers, graph replay: predictions against the oracle, then the dispatch against orc_dispatch from the GPU's own
    predictions."""
    cfg = dataclasses.replace(synth.CONFIGS["C2"], N=20000, d=128, B=48, Kc=16, seed=21)
    bank, it, queued, running, query, plen, rt = _setup(cfg, max_batch=64)
    rng = np.random.default_rng(3)
    w = synth.PRESETS["quality"]
    est = _np(rt.estimate(query))
    bud = torch.from_numpy(_random_budgets(rng, it, est["pred_outlen"], plen.cpu().numpy()))
    inst = orc.Instances(**it)
    for host in (False, True):
        rt.set_state(queued, running)
        q, p, b = (query.cpu(), plen.cpu(), bud) if host else (query, plen, bud.cuda())
        for _ in range(2):                    # second call replays the captured graph
            rt.set_state(queued, running)
            g = _np(rt.decide(q, p, w, budget=b))
        assert np.array_equal(g["pred_outlen"], est["pred_outlen"]) and np.array_equal(g["pred_quality"], est["pred_quality"])
        ref = orc.dispatch(inst, queued.numpy(), running.numpy(), g["pred_quality"], g["pred_outlen"], plen.cpu().numpy(), w,
                           budget=bud.numpy())
        for key in ("assignment", "scores", "max_tokens"):
            assert np.array_equal(g[key], ref[key]), key
        s = rt.get_state()
        assert np.array_equal(s[0].numpy(), ref["queued"]) and np.array_equal(s[1].numpy(), ref["running"])
    # no budget through the same entry point == rb_decide
    rt.set_state(queued, running)
    g0 = _np(rt.decide(query, plen, w))
    rt.set_state(queued, running)
    g1 = _np(rt.decide(query, plen, w, budget=torch.full((cfg.B,), float("inf"), device="cuda")))
    assert np.array_equal(g0["assignment"], g1["assignment"]) and np.array_equal(g0["scores"], g1["scores"])
    assert (g1["max_tokens"] == 2**31 - 1).all()
    rt.close()


def _forest_pair(orc, it, I, M, n_trees, depth, Fa, seed):
    fd = synth.make_forest(M, it["dec"], n_trees=n_trees, depth=depth, Fa=Fa, seed=seed, I=I)
    aux = fd.pop("aux")
    of = orc.Forest(aux=None if aux is None else aux.numpy(), **fd)
    return fd, aux, of


@pytest.mark.parametrize("I,M,B,n_trees,depth,Fa", [(13, 4, 16, 32, 4, 2), (64, 4, 200, 100, 5, 3), (256, 8, 1024, 16, 3, 0),
                                                    (33, 3, 50, 256, 2, 6), (5, 2, 9, 1, 0, 1),
                                                    # the packed forest does not fit shared memory as a whole (one tier at a
                                                    # time: 4 x ~80 KB) / not even one tier does (walk in global memory)
                                                    (64, 4, 200, 256, 5, 3), (40, 2, 30, 200, 9, 2),
                                                    # ... and fits with ~200 KB of dynamic shared memory
                                                    (90, 6, 50, 256, 4, 2)])
@pytest.mark.parametrize("upd,tb", [(1, 0), (2, 1)])
def test_boosted_tpot_head_bit_exact(orc, I, M, B, n_trees, depth, Fa, upd, tb):
    """latency_mode 2 -- per-tier gradient-boosted TPOT head over (running, queued, aux telemetry),
    re-evaluated for the chosen instance after every dispatch; scores0/scores/assignment/state and the between-batch
    drain bit-exact against orc_dispatch_gbdt / orc_advance_state_gbdt, with and without budgets."""
    from paper_2606_17949_b200.router import Router
    rng = np.random.default_rng(11 * I + B + upd)
    it = synth.make_instances(I, M, cap=int(rng.integers(2, 9)))
    fd, aux, of = _forest_pair(orc, it, I, M, n_trees, depth, Fa, seed=I + B)
    bank = dict(emb=torch.randn(64, 16), quality=torch.rand(64, M), outlen=torch.rand(64, M) * 100 + 1)
    rt = Router(bank["emb"].cuda(), bank["quality"].cuda(), bank["outlen"].cuda(), 4, store="f32", max_batch=B,
                update_enabled=upd, tiebreak_mode=tb, latency_mode=2)
    rt.set_instances(**it)
    with pytest.raises(Exception):
        rt.decide_from_predictions(torch.rand(B, M).cuda(), torch.rand(B, M).cuda(), torch.ones(B, dtype=torch.int32).cuda(),
                                   synth.PRESETS["balanced"])       # RB_ESTATE: no forest yet
    rt.set_tpot_forest(aux=None if aux is None else aux.cuda(), **fd)
    queued = rng.integers(0, 20001, I).astype(np.float32)
    running = np.minimum(rng.integers(0, 12, I), it["cap"]).astype(np.int32)
    Q = rng.uniform(0, 1, (B, M)).astype(np.float32)
    L = rng.lognormal(5.5, 0.7, (B, M)).astype(np.float32)
    plen = rng.integers(1, 4000, B).astype(np.int32)
    bud = _random_budgets(rng, it, L, plen)
    inst = orc.Instances(**it)
    for w in [synth.PRESETS["balanced"], synth.PRESETS["latency"], (0.0, 1.0, 0.0)]:
        for budget in (None, bud):
            rt.set_state(torch.from_numpy(queued), torch.from_numpy(running))
            rt.advance_state(41.5)
            dq, bq = orc.advance_state_gbdt(inst, of, queued, running, np.float32(41.5))
            g = _np(rt.decide_from_predictions(torch.from_numpy(Q).cuda(), torch.from_numpy(L).cuda(),
                                               torch.from_numpy(plen).cuda(), w, commit=1,
                                               budget=None if budget is None else torch.from_numpy(budget).cuda()))
            ref = orc.dispatch(inst, dq, bq, Q, L, plen, w, budget=budget, update_mode=upd, tiebreak_mode=tb,
                               latency_mode=2, forest=of)
            for key in ("assignment", "order", "scores", "scores0"):
                assert np.array_equal(g[key], ref[key]), (key, w, budget is None)
            s = rt.get_state()
            assert np.array_equal(s[0].numpy(), ref["queued"]) and np.array_equal(s[1].numpy(), ref["running"])
    rt.close()


def test_boosted_head_full_decide_path(orc):
    """rb_decide under latency_mode 2 (graph replay: tpot kernel -> stage -> scan -> finish -> dispatch)."""
    cfg = dataclasses.replace(synth.CONFIGS["C2"], N=20000, d=128, B=40, Kc=16, seed=22)
    bank, it, queued, running, query, plen, rt = _setup(cfg, max_batch=64, latency_mode=2)
    fd, aux, of = _forest_pair(orc, it, cfg.I, cfg.M, 48, 4, 2, seed=5)
    rt.set_tpot_forest(aux=aux.cuda(), **fd)
    inst = orc.Instances(**it)
    w = synth.PRESETS["latency"]
    for _ in range(2):
        rt.set_state(queued, running)
        g = _np(rt.decide(query, plen, w))
    ref = orc.dispatch(inst, queued.numpy(), running.numpy(), g["pred_quality"], g["pred_outlen"], plen.cpu().numpy(), w,
                       latency_mode=2, forest=of)
    assert np.array_equal(g["assignment"], ref["assignment"]) and np.array_equal(g["scores"], ref["scores"])
    s = rt.get_state()
    assert np.array_equal(s[0].numpy(), ref["queued"]) and np.array_equal(s[1].numpy(), ref["running"])
    rt.close()


def test_dispatch_fast_division_is_ieee_exact():
    """The dispatch loop divides with a branch-free reciprocal-refinement sequence inside a safe exponent window
    (IEEE __fdiv_rn outside it): 2^31 pseudo-random in-window operand pairs, bit for bit against the IEEE division."""
    from paper_2606_17949_b200 import binding as rb
    from paper_2606_17949_b200.router import Router
    rt = Router(torch.randn(64, 16).cuda(), torch.rand(64, 2).cuda(), torch.rand(64, 2).cuda() + 1, 4, store="f32", max_batch=4)
    for seed in (0, 12345):
        assert rb.rb_selftest_division(rt.ctx, 1 << 30, seed) == 0
    rt.close()


@pytest.mark.parametrize("I,M,B", [(13, 4, 24), (200, 5, 150)])
@pytest.mark.parametrize("case", ["tiny_lengths", "huge_queue", "denormal_length", "huge_lengths", "in_window"])
def test_dispatch_operand_ranges_pick_the_division(orc, I, M, B, case):
    """The greedy loop runs without any division fallback when the batch's operand ranges (binary exponents of the
    lengths, prefill terms, queues, decode constants, batch slopes) keep every quotient inside the exact window of the
    reciprocal-refinement sequence, and with the IEEE division otherwise.  Batches on both sides of the test, single- and
    multi-warp kernels: assignment, scores and the committed state equal the oracle's bit for bit."""
    from paper_2606_17949_b200.router import Router
    rng = np.random.default_rng(7000 + I + len(case))
    it = synth.make_instances(I, M, cap=3)
    rt = Router(torch.randn(64, 16).cuda(), torch.rand(64, M).cuda(), torch.rand(64, M).cuda() + 1, 4, store="f32", max_batch=B)
    rt.set_instances(**it)
    queued = rng.integers(0, 20001, I).astype(np.float32)
    running = np.minimum(rng.integers(0, 6, I), it["cap"]).astype(np.int32)
    L = rng.lognormal(5.5, 0.7, (B, M)).astype(np.float32)
    if case == "tiny_lengths":
        L *= np.float32(1e-30)                 # T^ far below 2^-34
        queued[:] = 0
    elif case == "huge_queue":
        queued *= np.float32(1e22)             # d / b and T^ above 2^62
    elif case == "denormal_length":
        L[3, 1] = np.float32(1e-41)
    elif case == "huge_lengths":
        L *= np.float32(1e16)
    Q = rng.uniform(0, 1, (B, M)).astype(np.float32)
    plen = rng.integers(1, 4000, B).astype(np.int32)
    inst = orc.Instances(**it)
    rt.set_state(torch.from_numpy(queued), torch.from_numpy(running))
    dq, bq = queued, running
    for w in [(0.2, 0.5, 0.3), (0.0, 1.0, 0.0)]:
        g = _np(rt.decide_from_predictions(torch.from_numpy(Q).cuda(), torch.from_numpy(L).cuda(), torch.from_numpy(plen).cuda(),
                                           w, commit=1))
        ref = orc.dispatch(inst, dq, bq, Q, L, plen, np.asarray(w, dtype=np.float32))
        for key in ("assignment", "order", "scores"):
            assert np.array_equal(g[key], ref[key], equal_nan=True), (case, key, w)
        dq, bq = ref["queued"], ref["running"]
        s = rt.get_state()
        assert np.array_equal(s[0].numpy(), dq) and np.array_equal(s[1].numpy(), bq), (case, "state", w)
    rt.close()


def test_deferred_advance_is_applied_in_call_order(orc):
    """rb_advance_state is deferred into the next rb_decide's first kernel; every other reader or writer of the state
    must see it applied (or, for an overwrite, dropped): sequences of advances, reads, overwrites and both decision
    entry points against the oracle's advance + dispatch, bit for bit."""
    cfg = dataclasses.replace(synth.CONFIGS["C2"], N=6000, d=64, B=9, Kc=8, seed=31)
    bank, it, queued, running, query, plen, rt = _setup(cfg, max_batch=16)
    inst = orc.Instances(**it)
    w = synth.PRESETS["balanced"]
    dq, bq = queued.numpy().copy(), running.numpy().copy()
    # six advances (more than a decision absorbs) then a read
    for dt in (5.0, 17.5, 0.0, 250.0, 3.25, 40.0):
        rt.advance_state(dt)
        dq, bq = orc.advance_state(inst, dq, bq, np.float32(dt))
    s = rt.get_state()
    assert np.array_equal(s[0].numpy(), dq) and np.array_equal(s[1].numpy(), bq)
    # advances, then a full decision: folded into the staging kernel
    for dt in (12.0, 33.0, 8.5):
        rt.advance_state(dt)
        dq, bq = orc.advance_state(inst, dq, bq, np.float32(dt))
    g = _np(rt.decide(query, plen, w))
    ref = orc.dispatch(inst, dq, bq, g["pred_quality"], g["pred_outlen"], plen.cpu().numpy(), w)
    assert np.array_equal(g["assignment"], ref["assignment"]) and np.array_equal(g["scores"], ref["scores"])
    dq, bq = ref["queued"], ref["running"]
    # an advance before decide_from_predictions is applied first
    rt.advance_state(77.0)
    dq, bq = orc.advance_state(inst, dq, bq, np.float32(77.0))
    g2 = _np(rt.decide_from_predictions(torch.from_numpy(g["pred_quality"]).cuda(), torch.from_numpy(g["pred_outlen"]).cuda(),
                                        plen, w, commit=1))
    ref2 = orc.dispatch(inst, dq, bq, g["pred_quality"], g["pred_outlen"], plen.cpu().numpy(), w)
    assert np.array_equal(g2["assignment"], ref2["assignment"]) and np.array_equal(g2["scores0"], ref2["scores0"])
    # an advance followed by an overwrite of the state is dropped; an estimate in between leaves it pending
    rt.advance_state(1000.0)
    rt.estimate(query)
    rt.set_state(queued, running)
    s = rt.get_state()
    assert np.array_equal(s[0].numpy(), queued.numpy()) and np.array_equal(s[1].numpy(), running.numpy())
    rt.close()


@pytest.mark.parametrize("B,I,qmax", [(1, 1, 1), (6, 3, 3), (16, 13, 2), (64, 13, 8), (200, 64, 5), (1024, 256, 6), (300, 7, 60)])
def test_match_replay_reaches_the_oracle_optimum(orc, B, I, qmax):
    """quota-constrained optimum of the batch-start score matrix.  Several optimal assignments may
    exist, so what is compared is what is unique -- the objective (fp64 sum of the chosen fp32 scores) -- and the rest
    is checked for validity: quotas respected, no filtered (-inf) pair chosen, divergence count consistent."""
    from paper_2606_17949_b200.router import Router
    rng = np.random.default_rng(1000 + B + I)
    M = min(4, I)
    it = synth.make_instances(I, M)
    rt = Router(torch.randn(64, 16).cuda(), torch.rand(64, M).cuda(), torch.rand(64, M).cuda() + 1, 4, store="f32", max_batch=8)
    rt.set_instances(**it)
    for trial in range(3):
        S = rng.uniform(0, 1, (B, I)).astype(np.float32)
        if trial == 1:
            S = np.round(S * 8) / 8                                  # many exact ties
        if trial == 2 and I > 1:
            S[rng.uniform(size=S.shape) < 0.3] = -np.inf             # budget-filtered pairs
            S[np.arange(B), rng.integers(0, I, B)] = rng.uniform(0, 1, B).astype(np.float32)   # every request keeps one
        quota = rng.integers(0, qmax + 1, I)
        while quota.sum() < B + I:
            quota[rng.integers(0, I)] += 1
        greedy = np.where(np.isfinite(S), S, -2).argmax(axis=1).astype(np.int32)
        try:
            ref = orc.matching_replay(S, quota, greedy)
        except ValueError:
            with pytest.raises(Exception):
                rt.match_replay(torch.from_numpy(S).cuda(), torch.from_numpy(quota.astype(np.int32)).cuda())
            continue
        for host in (False, True):
            St, qt, gt = torch.from_numpy(S), torch.from_numpy(quota.astype(np.int32)), torch.from_numpy(greedy)
            if not host:
                St, qt, gt = St.cuda(), qt.cuda(), gt.cuda()
            match, obj, div = rt.match_replay(St, qt, gt)
            m = match.cpu().numpy()
            assert abs(obj - ref["objective"]) <= 1e-9 * B, (obj, ref["objective"])
            assert abs(float(S.astype(np.float64)[np.arange(B), m].sum()) - obj) <= 1e-9 * B
            assert (np.bincount(m, minlength=I) <= quota).all() and np.isfinite(S[np.arange(B), m]).all()
            assert div == int((m != greedy).sum())
    # loose quotas: the objective decomposes per request -> row-wise argmax, nothing diverges
    S = rng.uniform(0, 1, (B, I)).astype(np.float32)
    g = S.argmax(axis=1).astype(np.int32)
    match, obj, div = rt.match_replay(torch.from_numpy(S).cuda(), torch.full((I,), B, dtype=torch.int32).cuda(), torch.from_numpy(g).cuda())
    assert np.array_equal(match.cpu().numpy(), g) and div == 0
    with pytest.raises(Exception):
        rt.match_replay(torch.from_numpy(S).cuda(), torch.zeros(I, dtype=torch.int32).cuda())
    rt.close()


def test_match_replay_on_a_real_score_matrix(orc):
    """The replay the paper describes: scores0 of a C5-shaped batch (B=1024, I=256) from the library itself, quota = 6
    requests per instance; objective against the oracle, and the greedy-vs-matching divergence is reported."""
    cfg = dataclasses.replace(synth.CONFIGS["C5"], N=50000, d=128)
    bank, it, queued, running, query, plen, rt = _setup(cfg, max_batch=cfg.B)
    est = rt.estimate(query)
    w = synth.PRESETS["balanced"]
    out = rt.decide_from_predictions(est["pred_quality"], est["pred_outlen"], plen, w, commit=0)
    quota = torch.full((cfg.I,), 6, dtype=torch.int32, device="cuda")
    match, obj, div = rt.match_replay(out["scores0"], quota, out["assignment"])
    ref = orc.matching_replay(out["scores0"].cpu().numpy(), np.full(cfg.I, 6), out["assignment"].cpu().numpy())
    assert abs(obj - ref["objective"]) <= 1e-9 * cfg.B
    m = match.cpu().numpy()
    assert (np.bincount(m, minlength=cfg.I) <= 6).all()
    assert 0 <= div <= cfg.B
    rt.close()


@pytest.mark.parametrize("k,slack", [(5, 6), (20, 6), (50, 6), (50, 14)])
@pytest.mark.parametrize("store", ["bf16", "f32"])
def test_paper_shape_k_sweep(orc, k, slack, store):
    """P0: the paper's own shape (bank of 14,919 prompts x 384, 13 instances of Table 1) over its k
    sweep {5, 20, 50} at its fixed batch size 32, both storage modes, full parity."""
    cfg = dataclasses.replace(synth.CONFIGS["P0"], k=k, store=store)
    bank = synth.make_bank(cfg, device="cuda")
    it = synth.paper_cluster()
    queued, running = synth.make_state(cfg.I, it["cap"], cfg.seed)
    query = synth.make_queries(cfg, device="cuda")
    plen = synth.make_prompt_len(cfg, device="cuda")
    torch.cuda.synchronize()
    rt = _router(bank, cfg, max_batch=32, rerank_slack=slack if store == "bf16" else 0)
    rt.set_instances(**it)
    rt.set_state(queued, running)
    w = synth.PRESETS["balanced"]
    g = _np(rt.decide(query, plen, w))
    bank_np = parity.bank_to_numpy(bank["emb"])
    qn, ln = bank["quality"].cpu().numpy(), bank["outlen"].cpu().numpy()
    log = []
    oi, os_, near = parity.check_topk(orc, bank_np, query.cpu().numpy(), store, k, g["nn_idx"], g["nn_sim"], 0.0, log)
    parity.check_predictions(orc, g["pred_quality"], g["pred_outlen"], g["nn_idx"], g["nn_sim"], oi, os_, near, qn, ln)
    s = rt.get_state()
    parity.check_dispatch(orc, orc.Instances(**it), queued.numpy(), running.numpy(), g["pred_quality"], g["pred_outlen"],
                          plen.cpu().numpy(), w, g, state_after=(s[0].numpy(), s[1].numpy()))
    assert len(near) <= 2, log
    rt.close()


@pytest.mark.parametrize("I,M,B", [(64, 4, 4096), (1024, 16, 4096), (256, 8, 3000)])
def test_dispatch_at_maximum_batch(orc, I, M, B):
    """Largest shapes the ABI admits (max_batch 4096, I 1024, M 16): the per-(request, tier) terms no longer fit shared
    memory (global-memory path of the dispatch loop), the sort runs 4096 keys; with budgets; bit-exact."""
    from paper_2606_17949_b200.router import Router
    rng = np.random.default_rng(I + B)
    it = synth.make_instances(I, M, cap=4)
    rt = Router(torch.randn(64, 16).cuda(), torch.rand(64, M).cuda(), torch.rand(64, M).cuda() + 1, 4, store="f32", max_batch=B)
    rt.set_instances(**it)
    queued = rng.integers(0, 20001, I).astype(np.float32)
    running = np.minimum(rng.integers(0, 12, I), it["cap"]).astype(np.int32)
    Q = rng.uniform(0, 1, (B, M)).astype(np.float32)
    L = rng.lognormal(5.5, 0.7, (B, M)).astype(np.float32)
    L[B // 2] = L[3]
    plen = rng.integers(1, 4000, B).astype(np.int32)
    bud = _random_budgets(rng, it, L, plen)
    inst = orc.Instances(**it)
    for w, budget in ((synth.PRESETS["balanced"], None), (synth.PRESETS["cost"], bud)):
        rt.set_state(torch.from_numpy(queued), torch.from_numpy(running))
        g = _np(rt.decide_from_predictions(torch.from_numpy(Q).cuda(), torch.from_numpy(L).cuda(), torch.from_numpy(plen).cuda(),
                                           w, commit=1, budget=None if budget is None else torch.from_numpy(budget).cuda()))
        ref = orc.dispatch(inst, queued, running, Q, L, plen, w, budget=budget)
        for key in ("assignment", "order", "scores", "scores0"):
            assert np.array_equal(g[key], ref[key]), key
        if budget is not None:
            assert np.array_equal(g["max_tokens"], ref["max_tokens"])
        s = rt.get_state()
        assert np.array_equal(s[0].numpy(), ref["queued"]) and np.array_equal(s[1].numpy(), ref["running"])
    rt.close()


def test_deferred_advance_on_a_bank_that_does_not_fill_the_gpu(orc):
    """On a small bank the scan occupies few SMs, so with programmatic dependent launch every kernel of a decision can be
    resident at once: the dispatch kernel must still see the state advance its own decision's staging kernel applies.
    300 advance + decide steps in lock-step with the oracle (state compared after every step)."""
    cfg = dataclasses.replace(synth.CONFIGS["C2"], N=500, d=64, B=5, Kc=4, seed=41)
    bank, it, queued, running, query, plen, rt = _setup(cfg, max_batch=8)
    inst = orc.Instances(**it)
    bank_np = parity.bank_to_numpy(bank["emb"])
    qn, ln = bank["quality"].cpu().numpy(), bank["outlen"].cpu().numpy()
    ref = orc.decide(bank_np, qn, ln, inst, queued.numpy(), running.numpy(), query.cpu().numpy(), plen.cpu().numpy(),
                     synth.PRESETS["balanced"], cfg.k, store_dtype="bf16")
    pq, pl = ref["pred_quality"], ref["pred_outlen"]
    dq, bq = queued.numpy().copy(), running.numpy().copy()
    rng = np.random.default_rng(2)
    a = torch.empty(cfg.B, dtype=torch.int32, device="cuda")
    from paper_2606_17949_b200 import binding as rb
    for step in range(300):
        dt = float(rng.choice([0.0, 3.0, 40.0, 900.0]))
        w = list(synth.PRESETS.values())[step % 4]
        rb.rb_advance_state(rt.ctx, dt)
        rb.rb_decide(rt.ctx, query, plen, cfg.B, w, a)
        dq, bq = orc.advance_state(inst, dq, bq, np.float32(dt))
        r = orc.dispatch(inst, dq, bq, pq, pl, plen.cpu().numpy(), w)
        dq, bq = r["queued"], r["running"]
        if step % 25 == 24 or step < 5:
            s = rt.get_state()
            assert np.array_equal(a.cpu().numpy(), r["assignment"]), step
            assert np.array_equal(s[0].numpy(), dq) and np.array_equal(s[1].numpy(), bq), step
    rt.close()


@pytest.mark.parametrize("I,M,B", [(13, 4, 16), (64, 4, 200), (256, 8, 1024), (6, 3, 9)])
@pytest.mark.parametrize("policy", [0, 1, 2])
def test_pipeline_mode_dispatchers(orc, I, M, B, policy):
    """P:L135 pipeline mode: round-robin / shortest-queue / random placement inside the chosen model's replica pool, three
    consecutive batches (cursors, draw counter and dead-reckoned state persist), bit-exact against the oracle; commit=0
    leaves everything untouched; a tier without instances places nothing."""
    from paper_2606_17949_b200.router import Router
    rng = np.random.default_rng(50 + I + policy)
    it = synth.make_instances(I, M, cap=4)
    if I == 6:
        it["tier"] = [0, 1, 0, 1, 0, 1]          # tier 2 has no instance
    rt = Router(torch.randn(64, 16).cuda(), torch.rand(64, M).cuda(), torch.rand(64, M).cuda() + 1, 4, store="f32", max_batch=B)
    rt.set_instances(**it)
    inst = orc.Instances(**it)
    dq = rng.integers(0, 5000, I).astype(np.float32)
    dq[: I // 2] = dq[0]
    bq = np.minimum(rng.integers(0, 6, I), it["cap"]).astype(np.int32)
    rt.set_state(torch.from_numpy(dq), torch.from_numpy(bq))
    counter, cursor = 0, None
    for batch in range(3):
        model = rng.integers(0, M, B).astype(np.int32)
        L = rng.lognormal(5.0, 0.5, (B, M)).astype(np.float32)
        use_len = batch != 1
        dry = _np({"a": rt.dispatch_pipeline(torch.from_numpy(model).cuda(), torch.from_numpy(L).cuda(), policy, seed=9, commit=0)})
        ref = orc.pipeline_dispatch(inst, dq, bq, model, L if use_len else None, policy, seed=9, counter=counter, cursor=cursor)
        a = rt.dispatch_pipeline(torch.from_numpy(model) if batch == 2 else torch.from_numpy(model).cuda(),
                                 (torch.from_numpy(L) if batch == 2 else torch.from_numpy(L).cuda()) if use_len else None, policy, seed=9)
        rt.sync()   # the library works on its own stream
        assert np.array_equal(a.cpu().numpy(), ref["assignment"]), (batch, policy)
        if use_len:
            assert np.array_equal(dry["a"], ref["assignment"])      # commit=0 had changed nothing
        if I == 6:
            assert ((a.cpu().numpy() == -1) == (model == 2)).all()
        dq, bq, counter, cursor = ref["queued"], ref["running"], ref["counter"], ref["cursor"]
        s = rt.get_state()
        assert np.array_equal(s[0].numpy(), dq) and np.array_equal(s[1].numpy(), bq)
    rt.close()


@pytest.mark.parametrize("k,slack,M,I,B,d", [(40, 8, 16, 40, 20, 128), (58, 6, 16, 7, 3, 64), (10, 6, 16, 100, 70, 8), (64, 0, 2, 5, 9, 72)])
def test_full_path_at_the_limits_of_k_and_M(orc, k, slack, M, I, B, d):
    """Largest neighbour counts (k + slack = 64), most tiers (M = 16: 32 label columns per candidate), smallest and odd
    embedding widths (d = 8, 72), through the whole rb_decide path against the oracle."""
    cfg = dataclasses.replace(synth.CONFIGS["C2"], N=9000, d=d, M=M, I=I, B=B, k=k, Kc=8, seed=61)
    tol = 0.0 if slack > 0 else 4e-6
    g, near, log = _full_parity(orc, cfg, synth.PRESETS["balanced"], sim_tol=tol, rerank_slack=slack, max_batch=128)
    assert len(near) <= max(1, B // 10), log


def test_contexts_release_their_memory():
    """rb_destroy frees everything a context owns (device, pinned host, graphs): 30 create / decide / destroy cycles leave
    the device's free memory where it was."""
    from paper_2606_17949_b200.router import Router
    cfg = dataclasses.replace(synth.CONFIGS["C2"], N=20000, d=128, B=16, Kc=8, seed=71)
    bank = synth.make_bank(cfg, device="cuda")
    it = synth.make_instances(cfg.I, cfg.M)
    query = synth.make_queries(cfg, device="cuda")
    plen = synth.make_prompt_len(cfg, device="cuda")

    def cycle():
        rt = Router(bank["emb"], bank["quality"], bank["outlen"], cfg.k, store="bf16", max_batch=64)
        rt.set_instances(**it)
        rt.decide(query, plen, synth.PRESETS["balanced"])
        rt.decide(query.cpu(), plen.cpu(), synth.PRESETS["cost"])
        rt.estimate(query[:3])
        rt.sync()
        rt.close()

    cycle()
    torch.cuda.synchronize()
    free0, _ = torch.cuda.mem_get_info()
    for _ in range(30):
        cycle()
    torch.cuda.synchronize()
    free1, _ = torch.cuda.mem_get_info()
    assert free0 - free1 < 32 * 1024 * 1024, (free0, free1)


@pytest.mark.parametrize("I,M,B,P,modes", [(13, 4, 16, 66, {}), (256, 8, 1024, 66, {}), (64, 4, 200, 231, {}),
                                            (40, 4, 70, 21, dict(update_enabled=2, tiebreak_mode=1)),
                                            (13, 4, 33, 6, dict(latency_mode=1, lpt_enabled=0)), (300, 16, 5, 300, {})])
def test_weight_sweep_equals_one_pass_per_point(orc, I, M, B, P, modes):
    """rb_sweep_weights (the weight sweep behind the frontier): P simplex points over the same predictions and
    state in one call, one CTA per point; every row equals the oracle's uncommitted pass under that row's weights, with
    and without budgets, device and host buffers; the state is left untouched and a pending advance is applied first."""
    from paper_2606_17949_b200.router import Router
    rng = np.random.default_rng(1000 + I + B)
    it = synth.make_instances(I, M, cap=int(rng.integers(2, 9)))
    rt = Router(torch.randn(64, 16).cuda(), torch.rand(64, M).cuda(), torch.rand(64, M).cuda() + 1, 4, store="f32", max_batch=B,
                **modes)
    rt.set_instances(**it)
    inst = orc.Instances(**it)
    queued = rng.integers(0, 20001, I).astype(np.float32)
    queued[: I // 3] = queued[0]                       # replicas with equal state: exact ties
    running = np.minimum(rng.integers(0, 12, I), it["cap"]).astype(np.int32)
    Q = rng.uniform(0, 1, (B, M)).astype(np.float32)
    L = rng.lognormal(5.5, 0.7, (B, M)).astype(np.float32)
    plen = rng.integers(1, 4000, B).astype(np.int32)
    bud = _random_budgets(rng, it, L, plen)
    if P in (66, 231, 21, 6):
        step = {66: 0.1, 231: 0.05, 21: 0.2, 6: 0.5}[P]
        W = np.asarray(synth.simplex_points(step), dtype=np.float32)
    else:
        W = rng.dirichlet((1.0, 1.0, 1.0), P).astype(np.float32)
        W[:, 2] = 1.0 - W[:, 0] - W[:, 1]
        W = np.clip(W, 0.0, 1.0)
    assert W.shape == (P, 3)
    rt.set_state(torch.from_numpy(queued), torch.from_numpy(running))
    rt.advance_state(23.0)
    dq, bq = orc.advance_state(inst, queued, running, np.float32(23.0))
    omodes = dict(lpt_enabled=modes.get("lpt_enabled", 1), update_mode=modes.get("update_enabled", 1),
                  tiebreak_mode=modes.get("tiebreak_mode", 0), latency_mode=modes.get("latency_mode", 0))
    for budget, host in ((None, False), (bud, False), (bud, True)):
        dev = (lambda a: torch.from_numpy(a)) if host else (lambda a: torch.from_numpy(a).cuda())
        a = rt.sweep_weights(dev(Q), dev(L), dev(plen), W, budget=None if budget is None else dev(budget))
        rt.sync()
        a = a.cpu().numpy()
        for p in range(P):
            ref = orc.dispatch(inst, dq, bq, Q, L, plen, W[p], budget=budget, **omodes)
            assert np.array_equal(a[p], ref["assignment"]), (p, W[p], budget is None, host)
        s = rt.get_state()
        assert np.array_equal(s[0].numpy(), dq) and np.array_equal(s[1].numpy(), bq)
    # the same context still takes ordinary decisions afterwards (graphs, scratch untouched)
    g = _np(rt.decide_from_predictions(torch.from_numpy(Q).cuda(), torch.from_numpy(L).cuda(), torch.from_numpy(plen).cuda(),
                                       tuple(W[P // 2]), commit=1))
    ref = orc.dispatch(inst, dq, bq, Q, L, plen, W[P // 2], **omodes)
    assert np.array_equal(g["assignment"], ref["assignment"])
    with pytest.raises(Exception):
        rt.sweep_weights(torch.from_numpy(Q).cuda(), torch.from_numpy(L).cuda(), torch.from_numpy(plen).cuda(),
                         np.array([[0.5, 0.6, 0.1]], dtype=np.float32))        # not on the simplex
    rt.close()


def test_c2_stream_10k_decisions_lockstep(orc):
    """SURVEY 8(d), C2 as specified: 10,000 consecutive decisions of the paper-shaped stream at full size (N=100k, d=768
    bf16, I=13; Poisson windows at 12 then 30 req/s, rb_advance_state between them, the four presets in turn) in the
    launch configuration bench.py times.  Score / LPT / dead-reckoned state are checked in lock-step on ALL decisions
    (bit-exact, given the GPU's predictions); neighbours and predictions against the brute-force oracle on every 10th."""
    import bench
    cfg = synth.CONFIGS["C2"]
    n_dec = 10000
    sizes, elapsed, weights = bench.c2_stream(cfg, n_dec)
    n_req = sum(sizes)
    bank, it, queued, running, _, _, rt = _setup(cfg, B=1, max_batch=64)
    allq = synth.make_queries(cfg, B=n_req, device="cuda")
    allp = synth.make_prompt_len(cfg, B=n_req, device="cuda")
    torch.cuda.synchronize()
    allp_np = allp.cpu().numpy()
    bank_np = parity.bank_to_numpy(bank["emb"])
    qn, ln = bank["quality"].cpu().numpy(), bank["outlen"].cpu().numpy()
    inst = orc.Instances(**it)
    dq, bq = queued.numpy().copy(), running.numpy().copy()
    off, near_rows, knn_rows, log = 0, 0, 0, []
    for j, (B, dt, w) in enumerate(zip(sizes, elapsed, weights)):
        rt.advance_state(dt)
        dq, bq = orc.advance_state(inst, dq, bq, np.float32(dt))
        g = _np(rt.decide(allq[off:off + B], allp[off:off + B], w, want=("pred", "nn")))
        if j % 10 == 0:
            q_np = allq[off:off + B].cpu().numpy()
            oi, os_, near = parity.check_topk(orc, bank_np, q_np, cfg.store, cfg.k, g["nn_idx"], g["nn_sim"], 0.0, log)
            parity.check_predictions(orc, g["pred_quality"], g["pred_outlen"], g["nn_idx"], g["nn_sim"], oi, os_, near, qn, ln)
            near_rows += len(near)
            knn_rows += B
        s = rt.get_state()
        ref = parity.check_dispatch(orc, inst, dq, bq, g["pred_quality"], g["pred_outlen"], allp_np[off:off + B], w, g,
                                    state_after=(s[0].numpy(), s[1].numpy()))
        dq, bq = ref["queued"], ref["running"]
        off += B
    assert off == n_req and 4 <= min(sizes) and max(sizes) <= 64
    assert near_rows <= max(3, knn_rows // 200), (near_rows, knn_rows, log[:5])   # documented near-ties only, and rare
    rt.close()


def test_adaptive_batch_rule_and_stream_driver_lockstep(orc):
    """SURVEY 8(f) #4, second half: the adaptive batch-size rule (rb_batch_target; reading 27) and the
    stream driver (stream.py) that forms its windows with it.  A Poisson stream of 1500 requests at 30 req/s over a
    cluster whose instances saturate and drain (cap = 4): the rule's target and busy count, every assignment and the state
    after every decision equal the oracle's, window by window; the targets really move with the load; and the
    fixed-batch-size off-switch (bs_min = bs_max) gives windows of that size."""
    from paper_2606_17949_b200 import binding as rb, stream
    from stream_backends import LockstepBackend
    cfg = dataclasses.replace(synth.CONFIGS["C2"], N=20000, d=128, Kc=16, seed=51)
    n_req = 1500
    bank = synth.make_bank(cfg, device="cuda")
    it = synth.make_instances(cfg.I, cfg.M, cap=4)
    queued, running = synth.make_state(cfg.I, it["cap"], cfg.seed)
    q = synth.make_queries(cfg, B=n_req, device="cuda")
    p = synth.make_prompt_len(cfg, B=n_req, device="cuda")
    arrivals = synth.poisson_arrivals_ms(30.0, n_req, seed=cfg.seed)
    torch.cuda.synchronize()
    rt = _router(bank, cfg, max_batch=64)
    rt.set_instances(**it)
    inst = orc.Instances(**it)
    presets = list(synth.PRESETS.values())
    for bs_min, bs_max in ((4, 64), (16, 16)):
        rt.set_state(queued, running)
        gpu = stream.RouterBackend(rt, q, p, want_predictions=True)
        both = LockstepBackend(orc, gpu, inst, queued.numpy(), running.numpy(), p.cpu().numpy())
        res = stream.drive(both, arrivals, lambda j: presets[j % 4], bs_min=bs_min, bs_max=bs_max, max_wait_ms=500.0)
        assert res.hi[-1] == n_req and both.windows == len(res.lo)
        if bs_min != bs_max:
            assert min(res.target) < max(res.target), "the load never moved the batch size"
            assert min(res.n_busy) < max(res.n_busy)
        else:
            assert set(res.target) == {16}
    # device outputs, and argument checking
    out = torch.zeros(2, dtype=torch.int32, device="cuda")
    assert rb._lib.rb_batch_target(rt.ctx, 4, 64, out.data_ptr(), out.data_ptr() + 4) == rb.RB_OK
    rt.sync()
    assert tuple(out.tolist()) == rt.batch_target(4, 64)
    for lo, hi in ((0, 4), (8, 4)):
        with pytest.raises(rb.RbError):
            rt.batch_target(lo, hi)
    rt.close()


def test_pipelined_decisions_above_128_requests():
    """Throughput mode with batches on both sides of 128 requests (CTA-pair scan above: its finishing kernel gets the GPU
    before the next scan starts, the dispatch CTA runs beside that scan): 50 decisions of 60..400 requests give the outputs
    and the final state of an unpipelined context, bit for bit."""
    cfg = dataclasses.replace(synth.CONFIGS["C2"], N=40000, d=256, Kc=16, seed=67)
    bank = synth.make_bank(cfg, device="cuda")
    it = synth.make_instances(40, cfg.M, cap=6)
    queued, running = synth.make_state(40, it["cap"], cfg.seed)
    rng = np.random.default_rng(67)
    sizes = [int(x) for x in rng.integers(60, 401, 50)]
    q = synth.make_queries(cfg, B=sum(sizes), device="cuda")
    p = synth.make_prompt_len(cfg, B=sum(sizes), device="cuda")
    torch.cuda.synchronize()
    presets = list(synth.PRESETS.values())
    outs = []
    for pipeline in (0, 1):
        rt = _router(bank, cfg, max_batch=512, pipeline=pipeline)
        rt.set_instances(**it)
        rt.set_state(queued, running)
        rec, off = [], 0
        for j, B in enumerate(sizes):
            rt.advance_state(float(3.0 + (j % 7)))
            o = rt.decide(q[off:off + B], p[off:off + B], presets[j % 4])
            rec.append({k_: v.clone() for k_, v in o.items()})
            off += B
        rt.sync()
        s = rt.get_state()
        rec.append({"dq": s[0].clone(), "bq": s[1].clone()})
        outs.append(rec)
        rt.close()
    for a, b in zip(*outs):
        for key in a:
            assert torch.equal(a[key].cpu(), b[key].cpu()), key


def test_pipelined_decisions_under_fp32_storage():
    """Throughput mode under fp32 storage (the staging kernel leaves the fp32 query rows of every buffer set for the exact
    re-rank): 90 decisions of varying size through rb_decide with device buffers and through rb_decide_submit /
    rb_decide_collect give the assignments and the final state of an unpipelined context, bit for bit."""
    from paper_2606_17949_b200 import binding as rb
    cfg = dataclasses.replace(synth.CONFIGS["C1"], N=9000, d=192, Kc=16, seed=63)
    assert cfg.store == "f32"
    bank = synth.make_bank(cfg, device="cuda")
    it = synth.make_instances(cfg.I, cfg.M, cap=5)
    queued, running = synth.make_state(cfg.I, it["cap"], cfg.seed)
    rng = np.random.default_rng(63)
    sizes = [int(x) for x in rng.integers(1, 97, 90)]
    offs = np.concatenate([[0], np.cumsum(sizes)])
    q = synth.make_queries(cfg, B=int(offs[-1]), device="cuda")
    p = synth.make_prompt_len(cfg, B=int(offs[-1]), device="cuda")
    qh, ph = q.cpu().pin_memory(), p.cpu().pin_memory()
    torch.cuda.synchronize()
    presets = list(synth.PRESETS.values())
    res = []
    for mode in ("plain", "device", "host"):
        rt = _router(bank, cfg, max_batch=128, pipeline=0 if mode == "plain" else 1)
        rt.set_instances(**it)
        rt.set_state(queued, running)
        got = torch.empty(int(offs[-1]), dtype=torch.int32, device="cpu" if mode == "host" else "cuda")
        pending = []
        for j, B in enumerate(sizes):
            rt.advance_state(float(2.0 + j % 5))
            sl = slice(int(offs[j]), int(offs[j + 1]))
            if mode == "host":
                rb.rb_decide_submit(rt.ctx, qh[sl], ph[sl], B, presets[j % 4])
                pending.append(j)
                while len(pending) >= 3:
                    c = pending.pop(0)
                    rb.rb_decide_collect(rt.ctx, got[int(offs[c]):int(offs[c + 1])], sizes[c])
            else:
                rb.rb_decide(rt.ctx, q[sl], p[sl], B, presets[j % 4], got[sl])
        for c in pending:
            rb.rb_decide_collect(rt.ctx, got[int(offs[c]):int(offs[c + 1])], sizes[c])
        rt.sync()
        s = rt.get_state()
        res.append((got.cpu().clone(), s[0].clone(), s[1].clone()))
        rt.close()
    for got, dq, bq in res[1:]:
        assert torch.equal(got, res[0][0]) and torch.equal(dq, res[0][1]) and torch.equal(bq, res[0][2])


def test_pipelined_decisions_equal_unpipelined_ones(orc):
    """rb_options.pipeline (throughput mode: the bank scan of a decision overlaps the finishing and dispatch stages of the
    one before it, three buffer sets rotating, consecutive scans on two streams): a stream of 300 decisions of varying size with rb_advance_state between
    them, estimate-only calls, state reads and a budgeted call mixed in, gives bit for bit the outputs and the final state
    of the same calls on an unpipelined context; and the first 40 decisions are checked against the oracle in lock-step."""
    cfg = dataclasses.replace(synth.CONFIGS["C2"], N=30000, d=256, Kc=16, seed=61)
    bank = synth.make_bank(cfg, device="cuda")
    it = synth.make_instances(cfg.I, cfg.M, cap=6)
    queued, running = synth.make_state(cfg.I, it["cap"], cfg.seed)
    rng = np.random.default_rng(61)
    sizes = [int(x) for x in rng.integers(1, 129, 300)]
    q = synth.make_queries(cfg, B=sum(sizes), device="cuda")
    p = synth.make_prompt_len(cfg, B=sum(sizes), device="cuda")
    torch.cuda.synchronize()
    presets = list(synth.PRESETS.values())
    outs = []
    for pipeline in (0, 1):
        rt = _router(bank, cfg, max_batch=128, pipeline=pipeline)
        rt.set_instances(**it)
        rt.set_state(queued, running)
        rec, off = [], 0
        for j, B in enumerate(sizes):
            rt.advance_state(float(3.0 + (j % 7)))
            if j % 5 == 4:
                rt.advance_state(1.5)                      # two pending advances folded into one decision
            qq, pp = q[off:off + B], p[off:off + B]
            if j % 37 == 36:
                bud = torch.full((B,), 1e9, device="cuda")
                o = rt.decide(qq, pp, presets[j % 4], budget=bud)
            else:
                o = rt.decide(qq, pp, presets[j % 4])
            rec.append({k_: v.clone() for k_, v in o.items()})
            if j % 23 == 22:
                e = rt.estimate(qq[:min(B, 9)])            # an unpipelined call in between
                rec.append({k_: v.clone() for k_, v in e.items()})
            if j % 41 == 40:
                s = rt.get_state()
                rec.append({"dq": s[0].clone(), "bq": s[1].clone()})
            if j % 29 == 28:                               # other readers and writers of the state between pipelined calls
                tgt, busy = rt.batch_target(4, 64)
                rec.append({"target": torch.tensor([int(tgt), int(busy)])})
            if j % 31 == 30:                               # the allocation-free score + dispatch entry point, committing
                a2 = rt.decide_from_predictions_static(o["pred_quality"], o["pred_outlen"], pp, presets[(j + 1) % 4], commit=1)
                rec.append({"static": a2.clone()})
            off += B
        rt.sync()
        s = rt.get_state()
        rec.append({"dq": s[0].clone(), "bq": s[1].clone()})
        outs.append(rec)
        rt.close()
    assert len(outs[0]) == len(outs[1])
    for a, b in zip(*outs):
        assert a.keys() == b.keys()
        for key in a:
            assert torch.equal(a[key].cpu(), b[key].cpu()), key
    # lock-step against the oracle (predictions from the GPU, DESIGN.md parity protocol), pipelined context
    rt = _router(bank, cfg, max_batch=128, pipeline=1)
    rt.set_instances(**it)
    rt.set_state(queued, running)
    inst = orc.Instances(**it)
    dq, bq = queued.numpy().copy(), running.numpy().copy()
    off, res = 0, []
    for j, B in enumerate(sizes[:40]):
        rt.advance_state(float(3.0 + (j % 7)))
        res.append(rt.decide(q[off:off + B], p[off:off + B], presets[j % 4]))   # no synchronisation: calls pile up
        off += B
    rt.sync()
    off = 0
    for j, B in enumerate(sizes[:40]):
        g = {k_: v.cpu().numpy() for k_, v in res[j].items()}
        dq, bq = orc.advance_state(inst, dq, bq, np.float32(3.0 + (j % 7)))
        ref = parity.check_dispatch(orc, inst, dq, bq, g["pred_quality"], g["pred_outlen"], p[off:off + B].cpu().numpy(),
                                    presets[j % 4], g)
        dq, bq = ref["queued"], ref["running"]
        off += B
    s = rt.get_state()
    assert np.array_equal(s[0].numpy(), dq) and np.array_equal(s[1].numpy(), bq)
    rt.close()


def test_submit_collect_equals_synchronous_decisions(orc):
    """rb_decide_submit / rb_decide_collect (up to three decisions in flight from host buffers): the assignments and the final
    state of 200 decisions with rb_advance_state in between equal those of synchronous rb_decide calls on an unpipelined
    context; call-order errors are reported (fourth submission, collect with nothing in flight, wrong batch size)."""
    from paper_2606_17949_b200 import binding as rb
    cfg = dataclasses.replace(synth.CONFIGS["C2"], N=30000, d=256, Kc=16, seed=71)
    bank = synth.make_bank(cfg, device="cuda")
    it = synth.make_instances(cfg.I, cfg.M, cap=6)
    queued, running = synth.make_state(cfg.I, it["cap"], cfg.seed)
    rng = np.random.default_rng(71)
    sizes = [int(x) for x in rng.integers(1, 65, 200)]
    offs = np.concatenate([[0], np.cumsum(sizes)])
    q = synth.make_queries(cfg, B=int(offs[-1]), device="cpu").pin_memory()
    p = synth.make_prompt_len(cfg, B=int(offs[-1]), device="cpu").pin_memory()
    torch.cuda.synchronize()
    presets = list(synth.PRESETS.values())
    ref_rt = _router(bank, cfg, max_batch=64)
    ref_rt.set_instances(**it)
    ref_rt.set_state(queued, running)
    ref = torch.empty(int(offs[-1]), dtype=torch.int32)
    for j, B in enumerate(sizes):
        ref_rt.advance_state(float(2.0 + j % 5))
        rb.rb_decide(ref_rt.ctx, q[offs[j]:offs[j + 1]], p[offs[j]:offs[j + 1]], B, presets[j % 4], ref[offs[j]:offs[j + 1]])
    ref_state = ref_rt.get_state()
    ref_rt.close()
    rt = _router(bank, cfg, max_batch=64, pipeline=1)
    rt.set_instances(**it)
    rt.set_state(queued, running)
    got = torch.empty(int(offs[-1]), dtype=torch.int32)
    with pytest.raises(rb.RbError):
        rb.rb_decide_collect(rt.ctx, got[:1], 1)                       # nothing in flight
    pending = []
    for j, B in enumerate(sizes):
        rt.advance_state(float(2.0 + j % 5))
        rb.rb_decide_submit(rt.ctx, q[offs[j]:offs[j + 1]], p[offs[j]:offs[j + 1]], B, presets[j % 4])
        pending.append(j)
        if j == 2:
            with pytest.raises(rb.RbError):                            # three in flight: a fourth is refused, nothing changes
                rb.rb_decide_submit(rt.ctx, q[:1], p[:1], 1, presets[0])
            with pytest.raises(rb.RbError):
                rb.rb_decide_collect(rt.ctx, got[:sizes[0] + 1], sizes[0] + 1)   # not the submitted batch size
        depth = 3 if (j // 10) % 3 == 0 else (2 if (j // 10) % 3 == 1 else 1)    # every depth of the loop
        while len(pending) >= depth:
            c = pending.pop(0)
            rb.rb_decide_collect(rt.ctx, got[offs[c]:offs[c + 1]], sizes[c])
    for c in pending:
        rb.rb_decide_collect(rt.ctx, got[offs[c]:offs[c + 1]], sizes[c])
    assert torch.equal(got, ref)
    s = rt.get_state()
    assert torch.equal(s[0], ref_state[0]) and torch.equal(s[1], ref_state[1])
    rt.close()
