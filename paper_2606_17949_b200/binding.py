"""Thin ctypes binding over the C ABI of include/routebalance.h (argument marshalling only -- every step of the
path runs in the CUDA kernels of librouteb.so).  The function names are the C names.  Array arguments may be
torch tensors (CPU or CUDA) or numpy arrays; they must be contiguous and of the stated dtype.

There is no fallback: importing this module fails if the library has not been built
(`python paper_2606_17949_b200/build.py`), and every call raises RbError on a non-RB_OK status.
"""
import ctypes
import os

import numpy as np

try:
    import torch
except ImportError:  # pragma: no cover
    torch = None

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "librouteb.so")
if not os.path.exists(LIB_PATH):
    raise ImportError("librouteb.so is not built (run `python paper_2606_17949_b200/build.py`); "
                      "there is no CPU fallback for the RouteBalance decision path")
_lib = ctypes.CDLL(LIB_PATH)

RB_OK, RB_EINVAL, RB_ECUDA, RB_ENOMEM, RB_ESTATE, RB_EUNSUPPORTED = range(6)
RB_F32, RB_BF16 = 0, 1
_STATUS = {0: "RB_OK", 1: "RB_EINVAL", 2: "RB_ECUDA", 3: "RB_ENOMEM", 4: "RB_ESTATE", 5: "RB_EUNSUPPORTED"}
EXPORTS = ["rb_options_default", "rb_create", "rb_set_instances", "rb_set_tpot_forest", "rb_set_telemetry", "rb_set_state", "rb_get_state", "rb_advance_state",
           "rb_batch_target", "rb_decide", "rb_decide_submit", "rb_decide_collect", "rb_decide_budgeted", "rb_decide_from_predictions", "rb_decide_from_predictions_budgeted", "rb_decide_from_predictions_static", "rb_sweep_weights", "rb_estimate", "rb_dispatch_pipeline", "rb_match_replay", "rb_set_stage_timing", "rb_last_stage_us", "rb_last_scan_device_us", "rb_selftest_division", "rb_testing_read_bandwidth",
           "rb_launch_count", "rb_sync", "rb_last_error", "rb_destroy"]


class rb_options(ctypes.Structure):
    _fields_ = [("bank_dtype", ctypes.c_int32), ("store_dtype", ctypes.c_int32), ("weight_mode", ctypes.c_int32),
                ("dist_eps", ctypes.c_float), ("rerank_slack", ctypes.c_int32), ("lpt_enabled", ctypes.c_int32),
                ("update_enabled", ctypes.c_int32), ("max_batch", ctypes.c_int32), ("use_graph", ctypes.c_int32),
                ("scan_list", ctypes.c_int32), ("tiebreak_mode", ctypes.c_int32), ("latency_mode", ctypes.c_int32),
                ("pipeline", ctypes.c_int32), ("stream", ctypes.c_void_p)]


class rb_lat_head(ctypes.Structure):
    _fields_ = [("prefill_ms_per_tok", ctypes.c_float), ("decode_ms_per_tok", ctypes.c_float),
                ("batch_slope", ctypes.c_float)]


class rb_tree_node(ctypes.Structure):
    _fields_ = [("feature", ctypes.c_int32), ("value", ctypes.c_float), ("left", ctypes.c_int32), ("right", ctypes.c_int32)]


class RbError(RuntimeError):
    def __init__(self, status, msg):
        super().__init__("%s: %s" % (_STATUS.get(status, status), msg))
        self.status = status


_vp, _i32, _i64, _f = ctypes.c_void_p, ctypes.c_int32, ctypes.c_int64, ctypes.c_float
_lib.rb_options_default.argtypes = [ctypes.POINTER(rb_options)]
_lib.rb_options_default.restype = None
_lib.rb_create.argtypes = [ctypes.POINTER(_vp), _vp, _vp, _vp, _i64, _i32, _i32, _i32, ctypes.POINTER(rb_options)]
_lib.rb_set_instances.argtypes = [_vp, _i32, _vp, _vp, _vp, _vp, ctypes.POINTER(rb_lat_head)]
_lib.rb_set_tpot_forest.argtypes = [_vp, _vp, _i32, _vp, _i32, _vp, _vp, _i32]
_lib.rb_set_telemetry.argtypes = [_vp, _vp]
_lib.rb_set_state.argtypes = [_vp, _vp, _vp]
_lib.rb_get_state.argtypes = [_vp, _vp, _vp]
_lib.rb_advance_state.argtypes = [_vp, _f]
_lib.rb_batch_target.argtypes = [_vp, _i32, _i32, _vp, _vp]
_lib.rb_decide_submit.argtypes = [_vp, _vp, _vp, _i32, ctypes.POINTER(_f * 3)]
_lib.rb_decide_collect.argtypes = [_vp, _vp, _i32]
_lib.rb_decide.argtypes = [_vp, _vp, _vp, _i32, ctypes.POINTER(_f * 3), _vp, _vp, _vp, _vp, _vp, _vp]
_lib.rb_decide_from_predictions.argtypes = [_vp, _vp, _vp, _vp, _i32, ctypes.POINTER(_f * 3), _i32, _vp, _vp, _vp, _vp]
_lib.rb_decide_budgeted.argtypes = [_vp, _vp, _vp, _vp, _i32, ctypes.POINTER(_f * 3), _vp, _vp, _vp, _vp, _vp, _vp, _vp]
_lib.rb_decide_from_predictions_static.argtypes = [_vp, _vp, _vp, _vp, _i32, ctypes.POINTER(_f * 3), _i32, _vp]
_lib.rb_decide_from_predictions_budgeted.argtypes = [_vp, _vp, _vp, _vp, _vp, _i32, ctypes.POINTER(_f * 3), _i32, _vp, _vp,
                                                     _vp, _vp, _vp]
_lib.rb_sweep_weights.argtypes = [_vp, _vp, _vp, _vp, _vp, _i32, _vp, _i32, _vp]
_lib.rb_dispatch_pipeline.argtypes = [_vp, _vp, _vp, _i32, _i32, ctypes.c_uint64, _i32, _vp]
_lib.rb_match_replay.argtypes = [_vp, _vp, _i32, _vp, _vp, _vp, ctypes.POINTER(ctypes.c_double), ctypes.POINTER(_i32)]
_lib.rb_estimate.argtypes = [_vp, _vp, _i32, _vp, _vp, _vp, _vp]
_lib.rb_set_stage_timing.argtypes = [_vp, _i32]
_lib.rb_last_stage_us.argtypes = [_vp, ctypes.POINTER(_f * 6)]
_lib.rb_last_scan_device_us.argtypes = [_vp, ctypes.POINTER(_f)]
_lib.rb_selftest_division.argtypes = [_vp, ctypes.c_uint64, ctypes.c_uint64, ctypes.POINTER(ctypes.c_uint64)]
_lib.rb_testing_read_bandwidth.argtypes = [_vp, ctypes.c_uint64, _i32, ctypes.POINTER(ctypes.c_double)]
_lib.rb_launch_count.argtypes = [_vp]
_lib.rb_launch_count.restype = _i64
_lib.rb_sync.argtypes = [_vp]
_lib.rb_last_error.argtypes = [_vp]
_lib.rb_last_error.restype = ctypes.c_char_p
_lib.rb_destroy.argtypes = [_vp]
_lib.rb_destroy.restype = None


def _ptr(a, dtype=None):
    """Raw address of a contiguous torch tensor / numpy array (None -> NULL)."""
    if a is None:
        return None
    if torch is not None and isinstance(a, torch.Tensor):
        if not a.is_contiguous():
            raise ValueError("tensor must be contiguous")
        if dtype is not None and a.dtype != dtype:
            raise ValueError("expected %s, got %s" % (dtype, a.dtype))
        return a.data_ptr()
    a_np = np.asarray(a)
    if not a_np.flags["C_CONTIGUOUS"]:
        raise ValueError("array must be contiguous")
    if dtype is not None:
        want = {torch.float32: np.float32, torch.int32: np.int32, torch.bfloat16: np.uint16}[dtype] if torch else dtype
        if a_np.dtype != want:
            raise ValueError("expected %s, got %s" % (want, a_np.dtype))
    return a_np.ctypes.data


def _check(ctx, st):
    if st != RB_OK:
        msg = _lib.rb_last_error(ctx).decode() if ctx else ""
        raise RbError(st, msg)


def rb_options_default():
    o = rb_options()
    _lib.rb_options_default(ctypes.byref(o))
    return o


def rb_create(bank_emb, bank_quality, bank_outlen, N, d, M, k, opt=None):
    """Returns the opaque context handle.  bank_emb: float32 [N,d], or bfloat16 (torch) / uint16 (numpy)."""
    ctx = _vp()
    if opt is None:
        opt = rb_options_default()
    f32 = torch.float32 if torch else np.float32
    st = _lib.rb_create(ctypes.byref(ctx), _ptr(bank_emb), _ptr(bank_quality, f32), _ptr(bank_outlen, f32), N, d, M, k,
                        ctypes.byref(opt))
    if st != RB_OK:
        msg = _lib.rb_last_error(ctx).decode() if ctx else ""
        if ctx:
            _lib.rb_destroy(ctx)
        raise RbError(st, msg)
    return ctx


def rb_set_instances(ctx, tier, cap, price_in, price_out, heads):
    """tier, cap: int sequences [I]; price_in/out: float sequences [M]; heads: M (prefill, decode, slope) triples."""
    tier = np.ascontiguousarray(tier, dtype=np.int32)
    cap = np.ascontiguousarray(cap, dtype=np.int32)
    pin = np.ascontiguousarray(price_in, dtype=np.float32)
    pout = np.ascontiguousarray(price_out, dtype=np.float32)
    h = (rb_lat_head * len(heads))(*[rb_lat_head(*map(float, x)) for x in heads])
    _check(ctx, _lib.rb_set_instances(ctx, len(tier), tier.ctypes.data, cap.ctypes.data, pin.ctypes.data,
                                      pout.ctypes.data, h))


def rb_set_tpot_forest(ctx, node_feature, node_value, node_left, node_right, tree_root, tier_tree_begin, base, n_features):
    """Node arrays (four parallel sequences) are packed into rb_tree_node records."""
    n = len(node_feature)
    nodes = np.zeros(n, dtype=[("feature", np.int32), ("value", np.float32), ("left", np.int32), ("right", np.int32)])
    nodes["feature"], nodes["value"], nodes["left"], nodes["right"] = node_feature, node_value, node_left, node_right
    root = np.ascontiguousarray(tree_root, dtype=np.int32)
    begin = np.ascontiguousarray(tier_tree_begin, dtype=np.int32)
    b = np.ascontiguousarray(base, dtype=np.float32)
    _check(ctx, _lib.rb_set_tpot_forest(ctx, nodes.ctypes.data, n, root.ctypes.data, len(root), begin.ctypes.data,
                                        b.ctypes.data, int(n_features)))


def rb_set_telemetry(ctx, aux):
    f32 = torch.float32 if torch else np.float32
    _check(ctx, _lib.rb_set_telemetry(ctx, _ptr(aux, f32)))


def rb_set_state(ctx, queued_tokens, running):
    f32, i32 = (torch.float32, torch.int32) if torch else (np.float32, np.int32)
    _check(ctx, _lib.rb_set_state(ctx, _ptr(queued_tokens, f32), _ptr(running, i32)))


def rb_get_state(ctx, queued_tokens, running):
    f32, i32 = (torch.float32, torch.int32) if torch else (np.float32, np.int32)
    _check(ctx, _lib.rb_get_state(ctx, _ptr(queued_tokens, f32), _ptr(running, i32)))


def rb_advance_state(ctx, elapsed_ms):
    _check(ctx, _lib.rb_advance_state(ctx, float(elapsed_ms)))


def rb_batch_target(ctx, bs_min, bs_max):
    """Adaptive batch size on the current state (reading 27): returns (target, n_busy) as Python ints
    (host outputs: the call synchronises the context's stream)."""
    out = (ctypes.c_int32 * 2)()
    _check(ctx, _lib.rb_batch_target(ctx, int(bs_min), int(bs_max), ctypes.addressof(out), ctypes.addressof(out) + 4))
    return int(out[0]), int(out[1])


_W3_CACHE = {}


def _w3(w):
    """(w_qual, w_lat, w_cost) as a C float[3]; the handful of weight vectors a caller uses are marshalled once."""
    key = tuple(w)
    arr = _W3_CACHE.get(key)
    if arr is None:
        if len(_W3_CACHE) > 4096:
            _W3_CACHE.clear()
        arr = _W3_CACHE[key] = (_f * 3)(*[float(x) for x in key])
    return ctypes.byref(arr)


def rb_decide(ctx, query_emb, prompt_len, B, w, assignment, scores=None, pred_quality=None, pred_outlen=None,
              nn_idx=None, nn_sim=None):
    f32, i32 = (torch.float32, torch.int32) if torch else (np.float32, np.int32)
    _check(ctx, _lib.rb_decide(ctx, _ptr(query_emb, f32), _ptr(prompt_len, i32), B, _w3(w), _ptr(assignment, i32),
                               _ptr(scores, f32), _ptr(pred_quality, f32), _ptr(pred_outlen, f32), _ptr(nn_idx, i32),
                               _ptr(nn_sim, f32)))


def rb_decide_submit(ctx, query_emb, prompt_len, B, w):
    """Enqueues a decision from HOST buffers and returns at once (rb_options.pipeline = 1; at most three in flight)."""
    f32, i32 = (torch.float32, torch.int32) if torch else (np.float32, np.int32)
    _check(ctx, _lib.rb_decide_submit(ctx, _ptr(query_emb, f32), _ptr(prompt_len, i32), B, _w3(w)))


def rb_decide_collect(ctx, assignment, B):
    """Waits for the oldest submitted decision and copies its assignment into the HOST buffer `assignment`."""
    i32 = torch.int32 if torch else np.int32
    _check(ctx, _lib.rb_decide_collect(ctx, _ptr(assignment, i32), B))


def rb_decide_from_predictions(ctx, quality, outlen, prompt_len, B, w, commit, assignment, scores=None, scores0=None,
                               order=None):
    f32, i32 = (torch.float32, torch.int32) if torch else (np.float32, np.int32)
    _check(ctx, _lib.rb_decide_from_predictions(ctx, _ptr(quality, f32), _ptr(outlen, f32), _ptr(prompt_len, i32), B,
                                                _w3(w), int(commit), _ptr(assignment, i32), _ptr(scores, f32),
                                                _ptr(scores0, f32), _ptr(order, i32)))


def rb_decide_from_predictions_static(ctx, quality, outlen, prompt_len, B, w, commit, assignment):
    """rb_decide_from_predictions without any allocation (device buffers only; B <= 1024, B * M <= 8192)."""
    f32, i32 = (torch.float32, torch.int32) if torch else (np.float32, np.int32)
    _check(ctx, _lib.rb_decide_from_predictions_static(ctx, _ptr(quality, f32), _ptr(outlen, f32), _ptr(prompt_len, i32), B,
                                                       _w3(w), int(commit), _ptr(assignment, i32)))


def rb_decide_budgeted(ctx, query_emb, prompt_len, budget, B, w, assignment, max_tokens=None, scores=None,
                       pred_quality=None, pred_outlen=None, nn_idx=None, nn_sim=None):
    f32, i32 = (torch.float32, torch.int32) if torch else (np.float32, np.int32)
    _check(ctx, _lib.rb_decide_budgeted(ctx, _ptr(query_emb, f32), _ptr(prompt_len, i32), _ptr(budget, f32), B, _w3(w),
                                        _ptr(assignment, i32), _ptr(max_tokens, i32), _ptr(scores, f32),
                                        _ptr(pred_quality, f32), _ptr(pred_outlen, f32), _ptr(nn_idx, i32),
                                        _ptr(nn_sim, f32)))


def rb_decide_from_predictions_budgeted(ctx, quality, outlen, prompt_len, budget, B, w, commit, assignment,
                                        max_tokens=None, scores=None, scores0=None, order=None):
    f32, i32 = (torch.float32, torch.int32) if torch else (np.float32, np.int32)
    _check(ctx, _lib.rb_decide_from_predictions_budgeted(ctx, _ptr(quality, f32), _ptr(outlen, f32),
                                                         _ptr(prompt_len, i32), _ptr(budget, f32), B, _w3(w),
                                                         int(commit), _ptr(assignment, i32), _ptr(max_tokens, i32),
                                                         _ptr(scores, f32), _ptr(scores0, f32), _ptr(order, i32)))


def rb_sweep_weights(ctx, quality, outlen, prompt_len, budget, B, w, P, assignment):
    """w: host float32 array [P, 3] (numpy or CPU tensor); assignment: int32 [P, B]."""
    f32, i32 = (torch.float32, torch.int32) if torch else (np.float32, np.int32)
    _check(ctx, _lib.rb_sweep_weights(ctx, _ptr(quality, f32), _ptr(outlen, f32), _ptr(prompt_len, i32), _ptr(budget, f32), B,
                                      _ptr(w, f32), int(P), _ptr(assignment, i32)))


def rb_dispatch_pipeline(ctx, model, outlen, B, policy, seed, commit, assignment):
    f32, i32 = (torch.float32, torch.int32) if torch else (np.float32, np.int32)
    _check(ctx, _lib.rb_dispatch_pipeline(ctx, _ptr(model, i32), _ptr(outlen, f32), B, int(policy), int(seed), int(commit),
                                          _ptr(assignment, i32)))


def rb_match_replay(ctx, scores0, B, quota, greedy, match):
    """Returns (objective, n_diverged); match is filled in place."""
    f32, i32 = (torch.float32, torch.int32) if torch else (np.float32, np.int32)
    obj, div = ctypes.c_double(0.0), _i32(0)
    _check(ctx, _lib.rb_match_replay(ctx, _ptr(scores0, f32), B, _ptr(quota, i32), _ptr(greedy, i32), _ptr(match, i32),
                                     ctypes.byref(obj), ctypes.byref(div)))
    return float(obj.value), int(div.value)


def rb_estimate(ctx, query_emb, B, pred_quality=None, pred_outlen=None, nn_idx=None, nn_sim=None):
    f32, i32 = (torch.float32, torch.int32) if torch else (np.float32, np.int32)
    _check(ctx, _lib.rb_estimate(ctx, _ptr(query_emb, f32), B, _ptr(pred_quality, f32), _ptr(pred_outlen, f32),
                                 _ptr(nn_idx, i32), _ptr(nn_sim, f32)))


def rb_set_stage_timing(ctx, enabled):
    _check(ctx, _lib.rb_set_stage_timing(ctx, int(enabled)))


def rb_last_stage_us(ctx):
    us = (_f * 6)()
    _check(ctx, _lib.rb_last_stage_us(ctx, ctypes.byref(us)))
    return dict(zip(["stage", "scan", "merge", "aggregate", "score", "dispatch"], list(us)))


def rb_last_scan_device_us(ctx):
    us = _f(0.0)
    _check(ctx, _lib.rb_last_scan_device_us(ctx, ctypes.byref(us)))
    return float(us.value)


def rb_selftest_division(ctx, n_pairs, seed=0):
    bad = ctypes.c_uint64(0)
    _check(ctx, _lib.rb_selftest_division(ctx, int(n_pairs), int(seed), ctypes.byref(bad)))
    return int(bad.value)


def rb_testing_read_bandwidth(ctx, nbytes, repeats=10):
    """GB/s of a plain streaming-read kernel over nbytes of scratch (routebalance_testing.h)."""
    out = ctypes.c_double(0.0)
    _check(ctx, _lib.rb_testing_read_bandwidth(ctx, int(nbytes), int(repeats), ctypes.byref(out)))
    return float(out.value)


def rb_launch_count(ctx):
    return int(_lib.rb_launch_count(ctx))


def rb_sync(ctx):
    _check(ctx, _lib.rb_sync(ctx))


def rb_last_error(ctx):
    return _lib.rb_last_error(ctx).decode()


def rb_destroy(ctx):
    _lib.rb_destroy(ctx)
