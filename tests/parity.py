"""Parity protocol GPU path vs oracle, shared by the -m gpu tests, smoke() and
bench.py's self-check.  Inputs are the same seeded arrays on both sides; nothing here computes an expected
value by any means other than calling oracle/."""
import numpy as np


def bank_to_numpy(emb):
    """torch bank tensor (float32 or bfloat16, any device) -> numpy float32 or raw-bf16 uint16 array."""
    import torch
    e = emb.detach().cpu()
    if e.dtype == torch.bfloat16:
        return e.view(torch.int16).numpy().view(np.uint16)
    return e.numpy()


def check_topk(orc, bank_np, query_np, store, k, gpu_idx, gpu_sim, sim_tol=0.0, log=None):
    """Top-k sets identical except at documented near-ties (every index in the symmetric difference has an
    oracle similarity within 1e-5 of the oracle's k-th similarity).  Returns (orc_idx, orc_sim, near_tie_rows).
    sim_tol: allowed |gpu_sim - oracle_sim| on common neighbours (0 = bit-equal)."""
    orc_idx, orc_sim = orc.knn(bank_np, query_np, k, store_dtype=store)
    near = []
    for r in range(query_np.shape[0]):
        g, o = set(gpu_idx[r].tolist()), set(orc_idx[r].tolist())
        assert len(g) == k, "row %d: GPU neighbours not distinct: %s" % (r, gpu_idx[r])
        if g != o:
            kth = float(orc_sim[r, k - 1])
            for n in sorted(g ^ o):
                _, s = orc.knn(bank_np[n:n + 1], query_np[r:r + 1], 1, store_dtype=store)
                gap = abs(float(s[0, 0]) - kth)
                assert gap <= 1e-5, "row %d: index %d differs and is no near-tie (gap %.3g)" % (r, n, gap)
                if log is not None:
                    log.append((r, n, float(s[0, 0]), kth))
            near.append(r)
        # similarities of the neighbours the GPU reports
        pos = {n: j for j, n in enumerate(orc_idx[r].tolist())}
        for j, n in enumerate(gpu_idx[r].tolist()):
            if n in pos:
                assert abs(float(gpu_sim[r, j]) - float(orc_sim[r, pos[n]])) <= sim_tol, \
                    "row %d neighbour %d: sim %r vs oracle %r" % (r, n, gpu_sim[r, j], orc_sim[r, pos[n]])
        # order: (sim desc, idx asc) in the GPU's own list
        for j in range(k - 1):
            a, b = (float(gpu_sim[r, j]), int(gpu_idx[r, j])), (float(gpu_sim[r, j + 1]), int(gpu_idx[r, j + 1]))
            assert a[0] > b[0] or (a[0] == b[0] and a[1] < b[1]), "row %d: neighbours out of order at %d" % (r, j)
    return orc_idx, orc_sim, near


def check_predictions(orc, gpu_q, gpu_l, gpu_idx, gpu_sim, orc_idx, orc_sim, near, quality_np, outlen_np,
                      weight_mode=0, eps=1e-6, rtol=1e-3, raw_sums=False):
    """Predicted quality / output length within 1e-3 relative (north_star).  Near-tie rows are compared with
    the oracle's aggregation re-run on the GPU's own neighbour set.  raw_sums (rerank_slack = 0: the similarities are
    the tensor core's own sums, within 4e-6 of the oracle's): the inverse-distance weight 1/(sqrt(2 - 2s) + eps)
    amplifies that deviation without bound as s -> 1: a weight moves by ds / (2 - 2s) relative, which stays within the
    1e-3 bound while 2 - 2s >= 4e-3, i.e. up to s = 0.998; rows with a neighbour closer than that are compared the same
    way as near-tie rows (parity protocol).  The default re-ranked path has bit-equal similarities and needs
    none of it."""
    oq, ol = orc.aggregate(orc_idx, orc_sim, quality_np, outlen_np, weight_mode, eps)
    near = list(near)
    if raw_sums and weight_mode == 0:
        near = sorted(set(near) | set(np.nonzero(gpu_sim.max(axis=1) > 0.998)[0].tolist()))
    if near:
        nq, nl = orc.aggregate(gpu_idx[near], gpu_sim[near], quality_np, outlen_np, weight_mode, eps)
        oq[near], ol[near] = nq, nl
    np.testing.assert_allclose(gpu_q, oq, rtol=rtol, atol=0)
    np.testing.assert_allclose(gpu_l, ol, rtol=rtol, atol=0)
    return oq, ol


def check_dispatch(orc, inst, queued, running, pred_q, pred_l, prompt_len, w, gpu, lpt_enabled=1, update_enabled=1,
                   state_after=None):
    """Given identical predictions: scores within 1e-5 relative, assignment / order / post-decision state
    bit-exact (north_star).  gpu: dict with assignment and optionally scores, scores0, order."""
    ref = orc.decide_from_predictions(inst, queued, running, pred_q, pred_l, prompt_len, w, lpt_enabled, update_enabled)
    assert np.array_equal(gpu["assignment"], ref["assignment"]), "assignment differs from the oracle"
    for key in ("scores", "scores0"):
        if gpu.get(key) is not None:
            np.testing.assert_allclose(gpu[key], ref[key], rtol=1e-5, atol=1e-7, err_msg=key)
    if gpu.get("order") is not None:
        assert np.array_equal(gpu["order"], ref["order"]), "dispatch order differs"
    if state_after is not None:
        assert np.array_equal(state_after[0], ref["queued"]), "queued_tokens after the batch differ"
        assert np.array_equal(state_after[1], ref["running"]), "running after the batch differ"
    return ref
