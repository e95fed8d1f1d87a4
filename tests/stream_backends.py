"""Stream backends for the tests of paper_2606_17949_b200/stream.py (test infrastructure: imports the oracle).

OracleBackend     the whole decision in oracle/ (brute-force KNN -> aggregate -> dispatch), state kept on the host.
LockstepBackend   the CUDA library and the oracle side by side on the same windows: the rule's output, every assignment
                  and the state after every decision are compared as the stream runs (the oracle's dispatch is fed the
                  GPU's own predictions, DESIGN.md parity protocol)."""
import numpy as np


class OracleBackend:
    def __init__(self, orc, bank_np, quality_np, outlen_np, inst, queued, running, queries_np, plen_np, k, store="bf16"):
        self.orc, self.bank, self.qn, self.ln, self.inst = orc, bank_np, quality_np, outlen_np, inst
        self.dq, self.bq = np.asarray(queued, np.float32).copy(), np.asarray(running, np.int32).copy()
        self.q, self.p, self.k, self.store = queries_np, plen_np, k, store
        self.assignment = np.full(queries_np.shape[0], -1, np.int32)

    def batch_target(self, bs_min, bs_max):
        return self.orc.batch_target(self.inst, self.bq, bs_min, bs_max)

    def advance(self, elapsed_ms):
        self.dq, self.bq = self.orc.advance_state(self.inst, self.dq, self.bq, np.float32(elapsed_ms))

    def decide(self, lo, hi, w):
        ref = self.orc.decide(self.bank, self.qn, self.ln, self.inst, self.dq, self.bq, self.q[lo:hi], self.p[lo:hi], w,
                              self.k, store_dtype=self.store)
        self.assignment[lo:hi] = ref["assignment"]
        self.dq, self.bq = ref["queued"], ref["running"]


class LockstepBackend:
    def __init__(self, orc, gpu_backend, inst, queued, running, plen_np):
        self.orc, self.gpu, self.inst = orc, gpu_backend, inst
        self.dq, self.bq = np.asarray(queued, np.float32).copy(), np.asarray(running, np.int32).copy()
        self.p = plen_np
        self.windows = 0

    def batch_target(self, bs_min, bs_max):
        g = self.gpu.batch_target(bs_min, bs_max)
        o = self.orc.batch_target(self.inst, self.bq, bs_min, bs_max)
        assert g == o, "window %d: rule differs: gpu %s oracle %s" % (self.windows, g, o)
        return g

    def advance(self, elapsed_ms):
        self.gpu.advance(elapsed_ms)
        self.dq, self.bq = self.orc.advance_state(self.inst, self.dq, self.bq, np.float32(elapsed_ms))

    def decide(self, lo, hi, w):
        self.gpu.decide(lo, hi, w)
        self.gpu.rt.sync()
        pq, pl = self.gpu.pred_q[lo:hi].cpu().numpy(), self.gpu.pred_l[lo:hi].cpu().numpy()
        ref = self.orc.decide_from_predictions(self.inst, self.dq, self.bq, pq, pl, self.p[lo:hi], w)
        got = self.gpu.assignment[lo:hi].cpu().numpy()
        assert np.array_equal(got, ref["assignment"]), "window %d: assignment differs" % self.windows
        self.dq, self.bq = ref["queued"], ref["running"]
        s = self.gpu.rt.get_state()
        assert np.array_equal(s[0].numpy(), self.dq) and np.array_equal(s[1].numpy(), self.bq), \
            "window %d: state differs" % self.windows
        self.windows += 1
