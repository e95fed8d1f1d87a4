"""ORACLE binding -- test infrastructure, not product code.

ctypes wrapper over oracle/orc.cpp (the slow CPU statement of the paper's per-batch decision).  Only
tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may import this.
It imports nothing from paper_2606_17949_b200 and the product imports nothing from here.
"""
import ctypes
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "orc.cpp")
_LIB = os.path.join(_HERE, "liborc.so")
_lib = None


def build(force=False):
    """Compiles orc.cpp -> liborc.so.  -ffp-contract=off: no fused multiply-add, so every fp32 line of the
    oracle is one IEEE operation."""
    if not force and os.path.exists(_LIB) and os.path.getmtime(_LIB) >= os.path.getmtime(_SRC):
        return _LIB
    cmd = ["g++", "-std=c++17", "-O2", "-fopenmp", "-ffp-contract=off", "-fno-fast-math", "-shared",
           "-fPIC", "-o", _LIB, _SRC]
    subprocess.run(cmd, check=True)
    return _LIB


def lib():
    global _lib
    if _lib is None:
        build()
        _lib = ctypes.CDLL(_LIB)
    return _lib


def _p(a):
    return None if a is None else a.ctypes.data_as(ctypes.c_void_p)


def _f32(a):
    return np.ascontiguousarray(a, dtype=np.float32)


def _i32(a):
    return np.ascontiguousarray(a, dtype=np.int32)


def num_threads():
    """Threads the oracle's neighbour search runs on (OpenMP default: all host cores)."""
    return int(lib().orc_num_threads())


def set_num_threads(n):
    lib().orc_set_num_threads(int(n))


def round_bf16(x):
    """fp32 array -> raw bf16 bit patterns (uint16), round-to-nearest-even."""
    x = _f32(x)
    out = np.empty(x.shape, dtype=np.uint16)
    lib().orc_round_bf16(_p(x), _p(out), ctypes.c_int64(x.size))
    return out


def bf16_bits_to_f32(bits):
    return (np.ascontiguousarray(bits, dtype=np.uint16).astype(np.uint32) << 16).view(np.float32)


def knn(bank, query, k, store_dtype="bf16"):
    """bank: N x d float32, or uint16 (raw bf16).  Returns (nn_idx [B,k] int32, nn_sim [B,k] float32)."""
    if bank.dtype == np.uint16:
        bank = np.ascontiguousarray(bank)
        bank_dtype = 1
    else:
        bank = _f32(bank)
        bank_dtype = 0
    query = _f32(query)
    N, d = bank.shape
    B = query.shape[0]
    assert query.shape[1] == d
    store = {"f32": 0, "bf16": 1}[store_dtype]
    idx = np.empty((B, k), dtype=np.int32)
    sim = np.empty((B, k), dtype=np.float32)
    rc = lib().orc_knn(_p(bank), bank_dtype, store, _p(query), ctypes.c_int64(N), d, B, k, _p(idx), _p(sim))
    if rc != 0:
        raise ValueError("orc_knn: bad arguments")
    return idx, sim


def aggregate(nn_idx, nn_sim, bank_quality, bank_outlen, weight_mode=0, eps=1e-6):
    nn_idx = _i32(nn_idx)
    nn_sim = _f32(nn_sim)
    bank_quality = _f32(bank_quality)
    bank_outlen = _f32(bank_outlen)
    B, k = nn_idx.shape
    M = bank_quality.shape[1]
    q = np.empty((B, M), dtype=np.float32)
    l = np.empty((B, M), dtype=np.float32)
    lib().orc_aggregate(_p(nn_idx), _p(nn_sim), _p(bank_quality), _p(bank_outlen), B, k, M, weight_mode,
                        ctypes.c_float(eps), _p(q), _p(l))
    return q, l


class Instances:
    """Plain record of the instance table: tier[I], cap[I]; per tier price_in, price_out, pre, dec, slope."""

    def __init__(self, tier, cap, price_in, price_out, pre, dec, slope):
        self.tier = _i32(tier)
        self.cap = _i32(cap)
        self.price_in = _f32(price_in)
        self.price_out = _f32(price_out)
        self.pre = _f32(pre)
        self.dec = _f32(dec)
        self.slope = _f32(slope)
        self.I = self.tier.shape[0]
        self.M = self.price_in.shape[0]


def decide_from_predictions(inst, queued, running, quality, outlen, prompt_len, w, lpt_enabled=1,
                            update_enabled=1):
    """Returns dict(assignment, scores, scores0, order, queued, running) -- the state after the batch."""
    quality = _f32(quality)
    outlen = _f32(outlen)
    prompt_len = _i32(prompt_len)
    queued = _f32(queued)
    running = _i32(running)
    w = _f32(w)
    B, M = quality.shape
    assert M == inst.M
    I = inst.I
    assignment = np.empty(B, dtype=np.int32)
    scores = np.empty((B, I), dtype=np.float32)
    scores0 = np.empty((B, I), dtype=np.float32)
    order = np.empty(B, dtype=np.int32)
    dq = np.empty(I, dtype=np.float32)
    bq = np.empty(I, dtype=np.int32)
    lib().orc_decide_from_predictions(I, M, _p(inst.tier), _p(inst.cap), _p(inst.price_in), _p(inst.price_out),
                                      _p(inst.pre), _p(inst.dec), _p(inst.slope), _p(queued), _p(running),
                                      _p(quality), _p(outlen), _p(prompt_len), B, _p(w), int(lpt_enabled),
                                      int(update_enabled), _p(assignment), _p(scores), _p(scores0), _p(order),
                                      _p(dq), _p(bq))
    return dict(assignment=assignment, scores=scores, scores0=scores0, order=order, queued=dq, running=bq)


class _CForest(ctypes.Structure):
    _fields_ = [("node_feature", ctypes.c_void_p), ("node_value", ctypes.c_void_p), ("node_left", ctypes.c_void_p),
                ("node_right", ctypes.c_void_p), ("tree_root", ctypes.c_void_p), ("tier_tree_begin", ctypes.c_void_p),
                ("base", ctypes.c_void_p), ("n_features", ctypes.c_int32), ("aux", ctypes.c_void_p)]


class Forest:
    """Plain record of a boosted TPOT head: node arrays (feature, value, left, right), tree_root [n_trees],
    tier_tree_begin [M+1], base [M], n_features = 2 + Fa and the per-instance auxiliary telemetry aux [I, Fa]."""

    def __init__(self, node_feature, node_value, node_left, node_right, tree_root, tier_tree_begin, base, n_features,
                 aux=None):
        self.node_feature = _i32(node_feature)
        self.node_value = _f32(node_value)
        self.node_left = _i32(node_left)
        self.node_right = _i32(node_right)
        self.tree_root = _i32(tree_root)
        self.tier_tree_begin = _i32(tier_tree_begin)
        self.base = _f32(base)
        self.n_features = int(n_features)
        self.aux = None if aux is None else _f32(aux)

    def c(self):
        return _CForest(_p(self.node_feature), _p(self.node_value), _p(self.node_left), _p(self.node_right),
                        _p(self.tree_root), _p(self.tier_tree_begin), _p(self.base), self.n_features, _p(self.aux))


def gbdt_tpot(inst, forest, queued, running):
    queued, running = _f32(queued), _i32(running)
    out = np.empty(inst.I, dtype=np.float32)
    cf = forest.c()
    lib().orc_gbdt_tpot(inst.I, _p(inst.tier), ctypes.byref(cf), _p(queued), _p(running), _p(out))
    return out


def advance_state_gbdt(inst, forest, queued, running, elapsed_ms):
    dq = _f32(queued).copy()
    bq = _i32(running).copy()
    cf = forest.c()
    lib().orc_advance_state_gbdt(inst.I, _p(inst.tier), ctypes.byref(cf), ctypes.c_float(elapsed_ms), _p(dq), _p(bq))
    return dq, bq


def dispatch(inst, queued, running, quality, outlen, prompt_len, w, budget=None, lpt_enabled=1, update_mode=1,
             tiebreak_mode=0, latency_mode=0, forest=None):
    """orc_dispatch: the score + LPT greedy stage with the optional budget admission filter (Eq. 2) and the
    isolation-arm modes.  Returns dict(assignment, scores, scores0, order, max_tokens, queued, running)."""
    quality = _f32(quality)
    outlen = _f32(outlen)
    prompt_len = _i32(prompt_len)
    queued = _f32(queued)
    running = _i32(running)
    w = _f32(w)
    bud = None if budget is None else _f32(budget)
    B, M = quality.shape
    assert M == inst.M
    I = inst.I
    assignment = np.empty(B, dtype=np.int32)
    scores = np.empty((B, I), dtype=np.float32)
    scores0 = np.empty((B, I), dtype=np.float32)
    order = np.empty(B, dtype=np.int32)
    max_tokens = np.empty(B, dtype=np.int32)
    dq = np.empty(I, dtype=np.float32)
    bq = np.empty(I, dtype=np.int32)
    cf = forest.c() if forest is not None else None
    rc = lib().orc_dispatch_gbdt(I, M, _p(inst.tier), _p(inst.cap), _p(inst.price_in), _p(inst.price_out), _p(inst.pre),
                                 _p(inst.dec), _p(inst.slope), _p(queued), _p(running), _p(quality), _p(outlen),
                                 _p(prompt_len), B, _p(w), _p(bud), int(lpt_enabled), int(update_mode),
                                 int(tiebreak_mode), int(latency_mode), ctypes.byref(cf) if cf is not None else None,
                                 _p(assignment), _p(scores), _p(scores0), _p(order), _p(max_tokens), _p(dq), _p(bq))
    if rc != 0:
        raise ValueError("orc_dispatch_gbdt: latency_mode 2 needs a forest")
    return dict(assignment=assignment, scores=scores, scores0=scores0, order=order, max_tokens=max_tokens, queued=dq,
                running=bq)


def advance_state(inst, queued, running, elapsed_ms):
    dq = _f32(queued).copy()
    bq = _i32(running).copy()
    lib().orc_advance_state(inst.I, _p(inst.tier), _p(inst.dec), _p(inst.slope), ctypes.c_float(elapsed_ms),
                            _p(dq), _p(bq))
    return dq, bq


def batch_target(inst, running, bs_min, bs_max):
    """Adaptive batch size (reading 27): returns (target, n_busy)."""
    running = _i32(running)
    target = ctypes.c_int32(0)
    busy = ctypes.c_int32(0)
    rc = lib().orc_batch_target(inst.I, _p(inst.cap), _p(running), int(bs_min), int(bs_max), ctypes.byref(target),
                                ctypes.byref(busy))
    if rc != 0:
        raise ValueError("orc_batch_target: need I >= 1 and 1 <= bs_min <= bs_max")
    return int(target.value), int(busy.value)


def decide(bank, bank_quality, bank_outlen, inst, queued, running, query, prompt_len, w, k,
           store_dtype="bf16", weight_mode=0, eps=1e-6, lpt_enabled=1, update_enabled=1):
    """The whole per-batch decision: KNN -> aggregate -> score -> LPT greedy dispatch."""
    nn_idx, nn_sim = knn(bank, query, k, store_dtype)
    q, l = aggregate(nn_idx, nn_sim, bank_quality, bank_outlen, weight_mode, eps)
    out = decide_from_predictions(inst, queued, running, q, l, prompt_len, w, lpt_enabled, update_enabled)
    out.update(nn_idx=nn_idx, nn_sim=nn_sim, pred_quality=q, pred_outlen=l)
    return out


def scan_fast_f32(bank, query):
    bank = _f32(bank)
    query = _f32(query)
    best = np.empty(query.shape[0], dtype=np.int32)
    lib().orc_scan_fast_f32(_p(bank), _p(query), ctypes.c_int64(bank.shape[0]), bank.shape[1],
                            query.shape[0], _p(best))
    return best


def matching_replay(scores0, quota, greedy=None):
    """Batch-level matching replay ("A batch-level matching (e.g. Hungarian) ... an offline replay over the logged
    score matrices"; reading 26): the assignment a of the B requests to instances that maximises
    sum_r S0[r, a(r)] over the batch-start score matrix, with at most quota[i] requests on instance i and no request on
    an instance filtered out for it (S0 = -inf).  The definition written out: every instance becomes min(quota, B)
    identical slots and the one-to-one assignment problem on requests x slots is solved by the library routine
    (scipy.optimize.linear_sum_assignment = the Hungarian/Jonker-Volgenant method the paper names).
    Returns dict(match [B] int32, objective float (fp64 sum of the chosen fp32 scores), diverged int or None)."""
    from scipy.optimize import linear_sum_assignment
    S = np.asarray(scores0, dtype=np.float32)
    B, I = S.shape
    quota = np.asarray(quota, dtype=np.int64)
    if quota.shape != (I,) or (quota < 0).any() or quota.sum() < B:
        raise ValueError("quota must be I non-negative counts summing to at least B")
    owner = np.repeat(np.arange(I), np.minimum(quota, B))
    cost = S.astype(np.float64)[:, owner]
    rows, cols = linear_sum_assignment(cost, maximize=True)     # raises when no feasible assignment exists
    match = np.empty(B, dtype=np.int32)
    match[rows] = owner[cols]
    objective = float(S.astype(np.float64)[np.arange(B), match].sum())
    diverged = None if greedy is None else int((match != np.asarray(greedy)).sum())
    return dict(match=match, objective=objective, diverged=diverged)


def splitmix64(x):
    lib().orc_splitmix64.restype = ctypes.c_uint64
    return int(lib().orc_splitmix64(ctypes.c_uint64(x)))


def pipeline_dispatch(inst, queued, running, model, outlen, policy, seed=0, counter=0, cursor=None):
    """Pipeline-mode dispatchers.  Returns dict(assignment, queued, running, counter, cursor)."""
    queued, running, model = _f32(queued), _i32(running), _i32(model)
    B = model.shape[0]
    ol = None if outlen is None else _f32(outlen)
    cur = np.zeros(inst.M, dtype=np.int32) if cursor is None else _i32(cursor).copy()
    cnt = ctypes.c_uint64(counter)
    a = np.empty(B, dtype=np.int32)
    dq = np.empty(inst.I, dtype=np.float32)
    bq = np.empty(inst.I, dtype=np.int32)
    lib().orc_pipeline_dispatch(inst.I, inst.M, _p(inst.tier), _p(inst.cap), _p(queued), _p(running), _p(model), _p(ol), B,
                                int(policy), ctypes.c_uint64(seed), ctypes.byref(cnt), _p(cur), _p(a), _p(dq), _p(bq))
    return dict(assignment=a, queued=dq, running=bq, counter=int(cnt.value), cursor=cur)
