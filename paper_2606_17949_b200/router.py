"""Convenience wrapper: owns an rb_ctx and torch output buffers; every method is one C-ABI call plus
marshalling.  No arithmetic of the method lives here.

Stream contract.  The context runs on a private stream (`Router.stream`).  Every method that consumes or produces
device tensors orders that stream against torch's current stream on both sides: the library's kernels start after
everything already queued on the current stream (the caller's inputs are complete), and the current stream waits for
the library's kernels before anything queued after the call (the outputs can be consumed like those of any torch op).
Both are event waits on the device, not host synchronisations.  Device tensors are also recorded on the private stream,
so the caching allocator does not hand their memory out while the library still reads or writes it.  Host tensors are
complete when the call returns (C-ABI convention)."""
import contextlib

import torch

from . import binding as rb


class Router:
    def __init__(self, bank_emb, bank_quality, bank_outlen, k, *, store="bf16", rerank_slack=None, weight_mode=0,
                 dist_eps=1e-6, lpt_enabled=1, update_enabled=1, max_batch=4096, use_graph=1, scan_list=0, tiebreak_mode=0,
                 latency_mode=0, pipeline=0, device="cuda"):
        N, d = bank_emb.shape
        M = bank_quality.shape[1]
        opt = rb.rb_options_default()
        opt.bank_dtype = rb.RB_BF16 if bank_emb.dtype == torch.bfloat16 else rb.RB_F32
        opt.store_dtype = rb.RB_BF16 if store == "bf16" else rb.RB_F32
        if rerank_slack is not None:
            opt.rerank_slack = rerank_slack
        opt.weight_mode = weight_mode
        opt.dist_eps = dist_eps
        opt.lpt_enabled = lpt_enabled
        opt.update_enabled = update_enabled
        opt.max_batch = max_batch
        opt.use_graph = use_graph
        opt.scan_list = scan_list
        opt.tiebreak_mode = tiebreak_mode
        opt.latency_mode = latency_mode
        opt.pipeline = pipeline
        self.device = torch.device(device)
        self.stream = torch.cuda.Stream(device=self.device)
        opt.stream = self.stream.cuda_stream
        self.N, self.d, self.M, self.k, self.max_batch = N, d, M, k, max_batch
        self.I = 0
        if torch.cuda.is_available():
            torch.cuda.synchronize()   # the bank may have been produced on another stream
        self.ctx = rb.rb_create(bank_emb.contiguous(), bank_quality.contiguous().float(),
                                bank_outlen.contiguous().float(), N, d, M, k, opt)

    def close(self):
        if self.ctx is not None:
            rb.rb_destroy(self.ctx)
            self.ctx = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    @contextlib.contextmanager
    def _ordered(self, *tensors):
        """Stream ordering of one call (module docstring): private stream after the current one, current one after the
        private one; device tensors recorded on the private stream."""
        cur = torch.cuda.current_stream(self.device)
        self.stream.wait_stream(cur)
        try:
            yield
        finally:
            cur.wait_stream(self.stream)
            for x in tensors:
                if isinstance(x, torch.Tensor) and x.is_cuda:
                    x.record_stream(self.stream)

    def set_instances(self, tier, cap, price_in, price_out, pre, dec, slope):
        rb.rb_set_instances(self.ctx, tier, cap, price_in, price_out, list(zip(pre, dec, slope)))
        self.I = len(tier)

    def set_tpot_forest(self, node_feature, node_value, node_left, node_right, tree_root, tier_tree_begin, base,
                        n_features, aux=None):
        rb.rb_set_tpot_forest(self.ctx, node_feature, node_value, node_left, node_right, tree_root, tier_tree_begin, base,
                              n_features)
        if aux is not None:
            aux = aux.contiguous().float()
            with self._ordered(aux):
                rb.rb_set_telemetry(self.ctx, aux)

    def set_state(self, queued, running):
        q, b = queued.contiguous().float(), running.contiguous().to(torch.int32)
        with self._ordered(q, b):
            rb.rb_set_state(self.ctx, q, b)

    def get_state(self):
        q = torch.empty(self.I, dtype=torch.float32)
        b = torch.empty(self.I, dtype=torch.int32)
        rb.rb_get_state(self.ctx, q, b)
        return q, b

    def advance_state(self, elapsed_ms):
        rb.rb_advance_state(self.ctx, elapsed_ms)

    def batch_target(self, bs_min, bs_max):
        """Adaptive batch size: (target, n_busy) from the current dead-reckoned state."""
        return rb.rb_batch_target(self.ctx, bs_min, bs_max)

    def _buf(self, shape, dtype, device):
        return torch.empty(shape, dtype=dtype, device=device)

    def decide(self, query, prompt_len, w, want=("scores", "pred", "nn"), out_device=None, budget=None):
        """query [B,d] float32, prompt_len [B] int32 (host or device).  Outputs land on out_device
        (default: where the query lives).  budget [B] float32: per-request cost budgets (Eq. 2); adds max_tokens.
        Returns a dict of tensors."""
        B = query.shape[0]
        dev = out_device if out_device is not None else query.device
        out = {"assignment": self._buf((B,), torch.int32, dev)}
        if "scores" in want:
            out["scores"] = self._buf((B, self.I), torch.float32, dev)
        if "pred" in want:
            out["pred_quality"] = self._buf((B, self.M), torch.float32, dev)
            out["pred_outlen"] = self._buf((B, self.M), torch.float32, dev)
        if "nn" in want:
            out["nn_idx"] = self._buf((B, self.k), torch.int32, dev)
            out["nn_sim"] = self._buf((B, self.k), torch.float32, dev)
        if budget is not None:
            out["max_tokens"] = self._buf((B,), torch.int32, dev)
            with self._ordered(query, prompt_len, budget, *out.values()):
                rb.rb_decide_budgeted(self.ctx, query, prompt_len, budget, B, w, out["assignment"], out["max_tokens"],
                                      out.get("scores"), out.get("pred_quality"), out.get("pred_outlen"), out.get("nn_idx"),
                                      out.get("nn_sim"))
            return out
        with self._ordered(query, prompt_len, *out.values()):
            rb.rb_decide(self.ctx, query, prompt_len, B, w, out["assignment"], out.get("scores"), out.get("pred_quality"),
                         out.get("pred_outlen"), out.get("nn_idx"), out.get("nn_sim"))
        return out

    def estimate(self, query, out_device=None):
        B = query.shape[0]
        dev = out_device if out_device is not None else query.device
        out = {"pred_quality": self._buf((B, self.M), torch.float32, dev),
               "pred_outlen": self._buf((B, self.M), torch.float32, dev),
               "nn_idx": self._buf((B, self.k), torch.int32, dev), "nn_sim": self._buf((B, self.k), torch.float32, dev)}
        with self._ordered(query, *out.values()):
            rb.rb_estimate(self.ctx, query, B, out["pred_quality"], out["pred_outlen"], out["nn_idx"], out["nn_sim"])
        return out

    def decide_from_predictions(self, quality, outlen, prompt_len, w, commit=0, out_device=None, budget=None):
        B = quality.shape[0]
        dev = out_device if out_device is not None else quality.device
        out = {"assignment": self._buf((B,), torch.int32, dev), "scores": self._buf((B, self.I), torch.float32, dev),
               "scores0": self._buf((B, self.I), torch.float32, dev), "order": self._buf((B,), torch.int32, dev)}
        if budget is not None:
            out["max_tokens"] = self._buf((B,), torch.int32, dev)
            with self._ordered(quality, outlen, prompt_len, budget, *out.values()):
                rb.rb_decide_from_predictions_budgeted(self.ctx, quality, outlen, prompt_len, budget, B, w, commit,
                                                       out["assignment"], out["max_tokens"], out["scores"], out["scores0"],
                                                       out["order"])
            return out
        with self._ordered(quality, outlen, prompt_len, *out.values()):
            rb.rb_decide_from_predictions(self.ctx, quality, outlen, prompt_len, B, w, commit, out["assignment"],
                                          out["scores"], out["scores0"], out["order"])
        return out

    def decide_from_predictions_static(self, quality, outlen, prompt_len, w, commit=0, assignment=None):
        """The allocation-free entry point (rb_decide_from_predictions_static): device tensors only; `assignment` may be a
        caller-owned int32 device tensor (then nothing is allocated on the Python side either).  Returns the assignment."""
        B = quality.shape[0]
        if assignment is None:
            assignment = self._buf((B,), torch.int32, quality.device)
        with self._ordered(quality, outlen, prompt_len, assignment):
            rb.rb_decide_from_predictions_static(self.ctx, quality, outlen, prompt_len, B, w, commit, assignment)
        return assignment

    def sweep_weights(self, quality, outlen, prompt_len, weights, budget=None, out_device=None):
        """P weight vectors over the same predictions and state, none committed: assignment [P, B]."""
        B = quality.shape[0]
        w = torch.as_tensor(weights, dtype=torch.float32, device="cpu").reshape(-1, 3).contiguous()
        dev = out_device if out_device is not None else quality.device
        a = torch.empty((w.shape[0], B), dtype=torch.int32, device=dev)
        with self._ordered(quality, outlen, prompt_len, budget, a):
            rb.rb_sweep_weights(self.ctx, quality, outlen, prompt_len, budget, B, w, w.shape[0], a)
        return a

    def dispatch_pipeline(self, model, outlen, policy, seed=0, commit=1):
        """Pipeline-mode dispatchers: model [B] int32 tiers, outlen [B,M] or None; returns assignment [B]."""
        B = model.shape[0]
        a = torch.empty(B, dtype=torch.int32, device=model.device)
        model = model.contiguous().to(torch.int32)
        outlen = None if outlen is None else outlen.contiguous().float()
        with self._ordered(model, outlen, a):
            rb.rb_dispatch_pipeline(self.ctx, model, outlen, B, policy, seed, commit, a)
        return a

    def match_replay(self, scores0, quota, greedy=None):
        """Quota-constrained optimum of the batch-start score matrix; returns (match, objective, n_diverged)."""
        B = scores0.shape[0]
        match = torch.empty(B, dtype=torch.int32, device=scores0.device)
        scores0, quota = scores0.contiguous(), quota.contiguous().to(torch.int32)
        greedy = None if greedy is None else greedy.contiguous().to(torch.int32)
        with self._ordered(scores0, quota, greedy, match):
            obj, div = rb.rb_match_replay(self.ctx, scores0, B, quota, greedy, match)
        return match, obj, div

    def sync(self):
        rb.rb_sync(self.ctx)

    def launch_count(self):
        return rb.rb_launch_count(self.ctx)

    def stage_us(self):
        return rb.rb_last_stage_us(self.ctx)

    def scan_device_us(self):
        return rb.rb_last_scan_device_us(self.ctx)

    def set_stage_timing(self, on):
        rb.rb_set_stage_timing(self.ctx, on)
