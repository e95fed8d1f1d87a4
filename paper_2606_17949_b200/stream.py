"""Stream driver: forms batches from an arrival stream with the adaptive batch-size rule and runs one decision per
batch (§4.1 "each batch is the set of requests waiting when the scheduler fires ... Batch size is adaptive --
larger when more instances are busy, smaller when idle"; §6.3, the batch bubble; §6.5, the adaptive-off and
fixed-batch-size ablations).

Host logic only: when a window closes and which requests it holds.  Every step of a decision, and the batch-size rule
itself (rb_batch_target), runs in the CUDA library; the driver talks to a *backend* with three methods so that the tests can
run the same window logic over the oracle:

    backend.batch_target(bs_min, bs_max) -> (target, n_busy)      the rule on the backend's current state
    backend.advance(elapsed_ms)                                   dead reckoning between batches
    backend.decide(lo, hi, w)                                     one decision over requests lo..hi-1 (arrival order)

Window rule (reading 27).  After a decision the rule gives the next batch's target size from the state that
decision left.  The scheduler fires when `target` requests are waiting, or when the first waiting request has waited
max_wait_ms, whichever comes first -- never before the previous decision (decisions take microseconds, arrivals are
milliseconds apart: a decision is treated as instantaneous); the batch is the requests that have arrived by then, at
most `target`.  bs_min = bs_max switches the adaptation off (fixed batch size).
"""
from dataclasses import dataclass, field

import numpy as np


@dataclass
class StreamResult:
    lo: list = field(default_factory=list)          # first request of each window
    hi: list = field(default_factory=list)          # one past its last request
    fire_ms: list = field(default_factory=list)     # when the scheduler fired
    target: list = field(default_factory=list)      # the rule's target size for the window
    n_busy: list = field(default_factory=list)      # busy instances the rule saw
    elapsed_ms: list = field(default_factory=list)  # dead-reckoning step handed to the backend

    def batch_wait_ms(self, arrivals_ms):
        """Per-request wait for its batch to fire (the 'batch wait' column of the paper's Table 4)."""
        a = np.asarray(arrivals_ms, dtype=np.float64)
        out = np.empty(self.hi[-1] if self.hi else 0, dtype=np.float64)
        for lo, hi, f in zip(self.lo, self.hi, self.fire_ms):
            out[lo:hi] = f - a[lo:hi]
        return out


def drive(backend, arrivals_ms, weights, bs_min=4, bs_max=64, max_wait_ms=500.0, max_windows=None):
    """Runs the stream arrivals_ms (non-decreasing arrival times in ms, request k = k-th arrival) through `backend`.
    weights: callable window index -> (w_qual, w_lat, w_cost).  Returns a StreamResult."""
    a = np.asarray(arrivals_ms, dtype=np.float64)
    n = a.shape[0]
    res = StreamResult()
    i, last_fire = 0, 0.0
    while i < n and (max_windows is None or len(res.lo) < max_windows):
        target, n_busy = backend.batch_target(bs_min, bs_max)
        tgt = min(int(target), n - i)
        t_full = a[i + tgt - 1]                       # the target-th waiting request arrives
        deadline = a[i] + max_wait_ms                 # the first waiting request has waited long enough
        fire = max(last_fire, min(t_full, deadline))
        hi = i + int(np.searchsorted(a[i:i + tgt], fire, side="right"))   # arrived by then (>= 1: a[i] <= fire)
        elapsed = np.float32(fire - last_fire)
        backend.advance(float(elapsed))
        backend.decide(i, hi, weights(len(res.lo)))
        res.lo.append(i), res.hi.append(hi), res.fire_ms.append(fire), res.target.append(int(target))
        res.n_busy.append(int(n_busy)), res.elapsed_ms.append(float(elapsed))
        i, last_fire = hi, fire
    return res


class RouterBackend:
    """The CUDA library as a stream backend: device-resident query embeddings and prompt lengths of the whole stream,
    one rb_advance_state + rb_decide per window, assignments collected in a device buffer (no synchronisation except the
    batch-size read-back, which the window logic needs on the host)."""

    def __init__(self, router, queries, prompt_len, want_predictions=False):
        import torch
        from . import binding as rb
        self._rb, self.rt = rb, router
        self.q, self.p = queries, prompt_len
        n = queries.shape[0]
        self.assignment = torch.empty(n, dtype=torch.int32, device=queries.device)
        self.pred_q = torch.empty(n, router.M, dtype=torch.float32, device=queries.device) if want_predictions else None
        self.pred_l = torch.empty(n, router.M, dtype=torch.float32, device=queries.device) if want_predictions else None

    def batch_target(self, bs_min, bs_max):
        return self._rb.rb_batch_target(self.rt.ctx, bs_min, bs_max)

    def advance(self, elapsed_ms):
        self._rb.rb_advance_state(self.rt.ctx, elapsed_ms)

    def decide(self, lo, hi, w):
        pq = None if self.pred_q is None else self.pred_q[lo:hi]
        pl = None if self.pred_l is None else self.pred_l[lo:hi]
        self._rb.rb_decide(self.rt.ctx, self.q[lo:hi], self.p[lo:hi], hi - lo, w, self.assignment[lo:hi], None, pq, pl)
