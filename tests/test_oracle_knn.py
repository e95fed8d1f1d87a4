"""Pins for the oracle's estimate stage (orc_knn, orc_aggregate, orc_round_bf16): closed forms, special
cases that reduce to library routines, invariants and brute force.  No GPU."""
import dataclasses
import math

import numpy as np
import pytest
import torch

from conftest import read_golden


def _unit_circle(deg):
    a = np.deg2rad(np.asarray(deg, dtype=np.float64))
    return np.stack([np.cos(a), np.sin(a)], 1).astype(np.float32)


def test_w0_closed_form(orc):
    """W0: similarity = cos(angle), dist = 2 sin(angle/2) (closed form, not sqrt(2-2s)), weights 1/(dist+eps)."""
    g = read_golden("W0_knn_unit_circle.txt")
    bank = _unit_circle(g["bank_deg"])
    query = _unit_circle(g["query_deg"])
    quality = np.array(g["quality"], np.float32).reshape(4, 2)
    outlen = np.array(g["outlen"], np.float32).reshape(4, 2)
    idx, sim = orc.knn(bank, query, 4, store_dtype="f32")
    assert idx.tolist() == [[0, 1, 2, 3]]
    np.testing.assert_allclose(sim[0], g["sims"], atol=2e-7)
    # closed-form distances from the angles themselves
    ang = np.abs(np.array(g["bank_deg"]) - g["query_deg"][0])
    dist = 2 * np.sin(np.deg2rad(ang) / 2)
    np.testing.assert_allclose(dist, g["dist"], rtol=1e-6)
    for k, mode, tag in [(1, 0, "k1"), (2, 0, "k2"), (2, 1, "k2_uniform"), (4, 0, "k4"), (4, 1, "k4_uniform")]:
        i, s = orc.knn(bank, query, k, store_dtype="f32")
        q, l = orc.aggregate(i, s, quality, outlen, weight_mode=mode)
        np.testing.assert_allclose(q[0], g[tag + "_quality"], rtol=2e-6, err_msg=tag)
        np.testing.assert_allclose(l[0], g[tag + "_outlen"], rtol=2e-6, err_msg=tag)
        # and against the closed-form weights in fp64
        w = np.ones(k) if mode else 1.0 / (dist[:k] + 1e-6)
        np.testing.assert_allclose(q[0], (w[:, None] * quality[:k]).sum(0) / w.sum(), rtol=3e-6)


def test_bf16_rounding_matches_torch_and_known_bits(orc):
    """RNE fp32->bf16: known bit patterns and torch's conversion (library routine)."""
    known = {1.0: 0x3F80, -2.0: 0xC000, 0.0: 0x0000, 1.0 + 2.0 ** -8: 0x3F80,  # tie -> even (down)
             1.0 + 3 * 2.0 ** -8: 0x3F82,                                    # tie -> even (up)
             1.0 + 2.0 ** -8 + 2.0 ** -20: 0x3F81, 3.0e38: 0x7F62}
    x = np.array(list(known.keys()), np.float32)
    assert orc.round_bf16(x).tolist() == list(known.values())
    rng = np.random.default_rng(0)
    x = (rng.standard_normal(100000) * np.exp(rng.uniform(-20, 20, 100000))).astype(np.float32)
    ref = torch.from_numpy(x).to(torch.bfloat16).view(torch.int16).numpy().view(np.uint16)
    assert np.array_equal(orc.round_bf16(x), ref)
    np.testing.assert_array_equal(orc.bf16_bits_to_f32(ref), torch.from_numpy(x).to(torch.bfloat16).float().numpy())


@pytest.mark.parametrize("store", ["f32", "bf16"])
def test_similarity_and_topk_vs_numpy(orc, store):
    """s = fl32(fp64 dot of the stored values); order (s desc, n asc): numpy float64 matmul + lexsort."""
    rng = np.random.default_rng(1)
    N, d, B, k = 700, 72, 9, 13
    bank = rng.standard_normal((N, d)).astype(np.float32)
    bank /= np.linalg.norm(bank, axis=1, keepdims=True)
    query = bank[rng.integers(0, N, B)] + 0.05 * rng.standard_normal((B, d)).astype(np.float32)
    idx, sim = orc.knn(bank, query, k, store_dtype=store)
    if store == "bf16":
        bs = orc.bf16_bits_to_f32(orc.round_bf16(bank)).astype(np.float64)
        qs = orc.bf16_bits_to_f32(orc.round_bf16(query)).astype(np.float64)
    else:
        bs, qs = bank.astype(np.float64), query.astype(np.float64)
    s = (qs @ bs.T).astype(np.float32)
    for r in range(B):
        ref = np.lexsort((np.arange(N), -s[r].astype(np.float64)))[:k]
        assert idx[r].tolist() == ref.tolist()
        np.testing.assert_allclose(sim[r], s[r][ref], rtol=0, atol=1.2e-7)


def test_bf16_bank_passed_as_bits_equals_fp32_bank_rounded(orc):
    rng = np.random.default_rng(2)
    bank = rng.standard_normal((300, 40)).astype(np.float32)
    query = rng.standard_normal((4, 40)).astype(np.float32)
    i1, s1 = orc.knn(bank, query, 7, store_dtype="bf16")
    i2, s2 = orc.knn(orc.round_bf16(bank), query, 7, store_dtype="bf16")
    assert np.array_equal(i1, i2) and np.array_equal(s1, s2)


def test_ties_lower_index_first_and_k1_exact_labels(orc):
    rng = np.random.default_rng(3)
    bank = rng.standard_normal((50, 16)).astype(np.float32)
    bank /= np.linalg.norm(bank, axis=1, keepdims=True)
    bank[31] = bank[7]          # exact duplicates
    bank[44] = bank[7]
    quality = rng.uniform(0, 1, (50, 3)).astype(np.float32)
    outlen = rng.uniform(1, 900, (50, 3)).astype(np.float32)
    idx, sim = orc.knn(bank, bank[7:8], 4, store_dtype="f32")
    assert idx[0, :3].tolist() == [7, 31, 44]
    assert sim[0, 0] == sim[0, 1] == sim[0, 2]
    i1, s1 = orc.knn(bank, bank[20:21], 1, store_dtype="f32")
    q, l = orc.aggregate(i1, s1, quality, outlen)
    assert i1[0, 0] == 20
    np.testing.assert_array_equal(q[0], quality[20])
    np.testing.assert_array_equal(l[0], outlen[20])


def test_k_equals_N_uniform_is_bank_mean(orc):
    """BASELINE.json pin: k = N with uniform weights reduces the KNN head to the per-model bank mean."""
    rng = np.random.default_rng(4)
    N, M = 200, 4
    bank = rng.standard_normal((N, 24)).astype(np.float32)
    quality = rng.uniform(0, 1, (N, M)).astype(np.float32)
    outlen = rng.lognormal(5.5, 0.6, (N, M)).astype(np.float32)
    query = rng.standard_normal((3, 24)).astype(np.float32)
    idx, sim = orc.knn(bank, query, N, store_dtype="f32")
    assert sorted(idx[0].tolist()) == list(range(N))
    q, l = orc.aggregate(idx, sim, quality, outlen, weight_mode=1)
    np.testing.assert_allclose(q, np.tile(quality.astype(np.float64).mean(0), (3, 1)), rtol=2e-6)
    np.testing.assert_allclose(l, np.tile(outlen.astype(np.float64).mean(0), (3, 1)), rtol=2e-6)


def test_permuting_bank_rows_permutes_indices_only(orc):
    rng = np.random.default_rng(5)
    N = 400
    bank = rng.standard_normal((N, 32)).astype(np.float32)
    query = rng.standard_normal((5, 32)).astype(np.float32)
    perm = rng.permutation(N)
    i0, s0 = orc.knn(bank, query, 10, store_dtype="bf16")
    i1, s1 = orc.knn(bank[perm], query, 10, store_dtype="bf16")
    assert np.array_equal(perm[i1], i0) and np.array_equal(s0, s1)


def test_sklearn_distance_weighted_regressor_on_C1(orc):
    """Library cross-check: scikit-learn's brute-force distance-weighted KNN regressor on the Tiny config
    (F32 storage).  Differences: eps=1e-6 in the weight and fp32 vs fp64 arithmetic."""
    from sklearn.neighbors import KNeighborsRegressor

    from paper_2606_17949_b200 import synth
    cfg = synth.CONFIGS["C1"]
    bank = synth.make_bank(cfg)
    emb = bank["emb"].numpy()
    query = synth.make_queries(cfg).numpy()
    quality, outlen = bank["quality"].numpy(), bank["outlen"].numpy()
    idx, sim = orc.knn(emb, query, cfg.k, store_dtype="f32")
    q, l = orc.aggregate(idx, sim, quality, outlen)
    reg = KNeighborsRegressor(n_neighbors=cfg.k, weights="distance", algorithm="brute")
    reg.fit(emb.astype(np.float64), np.concatenate([quality, outlen], 1).astype(np.float64))
    pred = reg.predict(query.astype(np.float64))
    nb = reg.kneighbors(query.astype(np.float64), return_distance=False)
    assert np.array_equal(np.sort(nb, 1), np.sort(idx, 1))
    # dist is recovered from an fp32 similarity: |d dist| ~ 6e-8/dist ~ 2e-7 at dist ~ 0.28 -> weights to ~1e-6
    np.testing.assert_allclose(q, pred[:, :cfg.M], rtol=2e-5)
    np.testing.assert_allclose(l, pred[:, cfg.M:], rtol=2e-5)


def test_query_equal_to_bank_row_is_dominated_by_it(orc):
    """F32 mode, query == bank row: weight 1/eps = 1e6 on that row, so the prediction is its labels up to
    (sum of other weights)/(total weight) * label range."""
    rng = np.random.default_rng(6)
    bank = rng.standard_normal((300, 48)).astype(np.float32)
    bank /= np.linalg.norm(bank, axis=1, keepdims=True)
    quality = rng.uniform(0, 1, (300, 2)).astype(np.float32)
    outlen = rng.uniform(1, 1000, (300, 2)).astype(np.float32)
    idx, sim = orc.knn(bank, bank[5:6], 10, store_dtype="f32")
    assert idx[0, 0] == 5
    q, l = orc.aggregate(idx, sim, quality, outlen)
    # self-similarity of a normalised fp32 row is 1 within ~1e-7 -> dist <= ~5e-4, others ~1.3
    assert np.abs(q[0] - quality[5]).max() < 1e-2
    assert np.abs(l[0] - outlen[5]).max() < 10.0


def test_bad_k_rejected(orc):
    bank = np.zeros((5, 8), np.float32)
    with pytest.raises(ValueError):
        orc.knn(bank, bank[:1], 6)
    assert math.isfinite(1.0)


def test_fast_fp32_scan_finds_the_nearest_row(orc):
    """orc_scan_fast_f32 (the separately labelled fp32-accumulator scan that bench.py's cpu_baseline.split times; never
    used for parity) is pinned to the exact search: on a seeded mixture bank its argmax equals orc_knn(k = 1) for every
    query whose two best similarities are further apart than fp32 accumulation noise (1e-5: nearly all of them), and a
    planted exact copy of the query is found wherever it sits (first, middle, last row)."""
    from paper_2606_17949_b200 import synth
    cfg = dataclasses.replace(synth.CONFIGS["C1"], N=3000, d=96, Kc=12, seed=17)
    bank = synth.make_bank(cfg)["emb"].numpy()
    query = synth.make_queries(cfg, B=40).numpy()
    idx, sim = orc.knn(bank, query, 2, store_dtype="f32")
    clear = sim[:, 0] - sim[:, 1] > 1e-5
    assert clear.sum() >= 30
    assert np.array_equal(orc.scan_fast_f32(bank, query)[clear], idx[clear, 0])
    for pos in (0, 1501, 2999):
        planted = bank.copy()
        planted[pos] = query[7]
        assert orc.scan_fast_f32(planted, query[7:8])[0] == pos
