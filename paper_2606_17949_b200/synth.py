"""Seeded synthetic inputs shaped like the paper's workload.

This module only *draws inputs*; it contains none of the method's arithmetic and is the one module both the
CUDA path's tests/bench and the oracle's tests are fed from.  The paper's own dataset (18,608 prompts with
DeepEval labels) is not available; these generators stand in for it: unit-norm sentence-embedding-like
clusters, quality labels in [0,1] rising slightly with model size, heavy-tailed output lengths that shorten
with model size, 13 instances in 4 tiers with Table 1-like TPOTs and prices, Poisson
arrivals at 12-30 req/s.
"""
import math
from dataclasses import dataclass, field

import torch

# ---- configurations of BASELINE.json (C1..C5) plus the paper-exact shape P0 ------------------------------


@dataclass
class Config:
    name: str
    N: int
    d: int
    M: int
    I: int
    B: int
    k: int = 10
    Kc: int = 32
    store: str = "bf16"          # storage dtype of the bank: "bf16" | "f32"
    zipf_s: float = 0.0          # 0 = uniform component choice
    len_mu: float = math.log(500.0)
    len_sigma: float = 0.8
    seed: int = 0
    extra: dict = field(default_factory=dict)


CONFIGS = {
    "C1": Config("C1", N=4096, d=384, M=4, I=13, B=16, Kc=32, store="f32", seed=0),
    "P0": Config("P0", N=14919, d=384, M=4, I=13, B=32, Kc=64, store="f32", seed=7),
    "C2": Config("C2", N=100_000, d=768, M=4, I=13, B=64, Kc=64, seed=2),
    "C3": Config("C3", N=1_000_000, d=1024, M=8, I=256, B=1024, Kc=256, zipf_s=1.1,
                 len_mu=math.log(800.0), len_sigma=1.0, seed=3),
    "C4": Config("C4", N=10_000_000, d=384, M=4, I=64, B=64, Kc=256, seed=4),
    "C5": Config("C5", N=1_000_000, d=768, M=8, I=256, B=1024, Kc=256, seed=5),
}


def _gen(seed, stream, device):
    g = torch.Generator(device=device)
    g.manual_seed(int(seed) * 1000 + int(stream))
    return g


def centres(Kc, d, seed, device="cpu"):
    """Kc unit vectors = normalise(N(0, I_d))."""
    c = torch.randn(Kc, d, generator=_gen(seed, 0, device), device=device, dtype=torch.float32)
    return c / c.norm(dim=1, keepdim=True)


def _components(n, Kc, zipf_s, g, device):
    if zipf_s and zipf_s > 0:
        p = torch.arange(1, Kc + 1, device=device, dtype=torch.float64).pow(-zipf_s)
        p = (p / p.sum()).float()
        return torch.multinomial(p, n, replacement=True, generator=g)
    return torch.randint(0, Kc, (n,), generator=g, device=device)


def _points(cent, comp, sigma, g, chunk, out_dtype):
    """normalise(centre_c + sigma * g / sqrt(d)): sigma is the expected NORM of the noise."""
    n = comp.shape[0]
    d = cent.shape[1]
    out = torch.empty(n, d, device=cent.device, dtype=out_dtype)
    for s in range(0, n, chunk):
        e = min(n, s + chunk)
        x = torch.randn(e - s, d, generator=g, device=cent.device, dtype=torch.float32)
        x = cent[comp[s:e]] + x * (sigma / math.sqrt(d))
        x = x / x.norm(dim=1, keepdim=True)
        out[s:e] = x.to(out_dtype)
    return out


def make_bank(cfg, device="cpu", chunk=1 << 18):
    """Reference bank: embeddings [N,d] (float32, or bfloat16 when cfg.store == 'bf16'), quality [N,M] in
    [0,1], outlen [N,M] >= 1, comp [N]."""
    cent = centres(cfg.Kc, cfg.d, cfg.seed, device)
    g = _gen(cfg.seed, 1, device)
    comp = _components(cfg.N, cfg.Kc, cfg.zipf_s, g, device)
    dt = torch.bfloat16 if cfg.store == "bf16" else torch.float32
    emb = _points(cent, comp, 0.3, g, chunk, dt)
    gl = _gen(cfg.seed, 2, device)
    base = torch.rand(cfg.Kc, generator=gl, device=device) * 0.6 + 0.2
    bonus = 0.03 * torch.arange(cfg.M, device=device, dtype=torch.float32)
    quality = base[comp][:, None] + bonus[None, :] + 0.05 * torch.randn(cfg.N, cfg.M, generator=gl, device=device)
    quality = quality.clamp_(0.0, 1.0).contiguous()
    mu = math.log(300.0) - 0.1 * torch.arange(cfg.M, device=device, dtype=torch.float32)
    outlen = torch.exp(mu[None, :] + 0.6 * torch.randn(cfg.N, cfg.M, generator=gl, device=device))
    outlen = outlen.clamp_(1.0, 8192.0).contiguous()
    return dict(emb=emb, quality=quality, outlen=outlen, comp=comp)


def make_queries(cfg, B=None, device="cpu", stream=3):
    """B query embeddings [B,d] float32 from the same mixture, noise norm 0.1."""
    B = cfg.B if B is None else B
    cent = centres(cfg.Kc, cfg.d, cfg.seed, device)
    g = _gen(cfg.seed, stream, device)
    comp = _components(B, cfg.Kc, cfg.zipf_s, g, device)
    return _points(cent, comp, 0.1, g, 1 << 16, torch.float32)


def make_prompt_len(cfg, B=None, device="cpu", stream=4):
    B = cfg.B if B is None else B
    g = _gen(cfg.seed, stream, device)
    x = torch.exp(cfg.len_mu + cfg.len_sigma * torch.randn(B, generator=g, device=device))
    return x.round().clamp_(1, 32768).to(torch.int32)


_TIER_COUNTS = {(13, 4): [5, 4, 2, 2], (64, 4): [25, 20, 10, 9], (256, 8): [64, 48, 40, 32, 24, 24, 12, 12]}


def make_instances(I, M, cap=16):
    """Instance table: tier 0 = smallest/cheapest model.  Returns plain python lists."""
    counts = _TIER_COUNTS.get((I, M))
    if counts is None:  # spread evenly, cheap tiers first
        counts = [I // M + (1 if m < I % M else 0) for m in range(M)]
    tier = [m for m, c in enumerate(counts) for _ in range(c)]
    if M == 4:
        price = [0.1, 0.3, 0.8, 2.0]
        dec = [10.2, 19.6, 13.9, 41.6]     # Table 1 TPOTs in 3B/7B/14B/72B order
        pre = [0.05, 0.10, 0.08, 0.25]
    else:
        price = [0.1 * 1.55 ** m for m in range(M)]
        dec = [10.0 * 1.22 ** m for m in range(M)]
        pre = [0.04 * 1.3 ** m for m in range(M)]
    return dict(tier=tier, cap=[cap] * I, price_in=list(price), price_out=list(price), pre=pre, dec=dec,
                slope=[0.02] * M)


def paper_cluster():
    """Table 1: 3B x3, 7B x5, 14B x3, 72B x2 with the measured TPOTs and public prices."""
    counts = [3, 5, 3, 2]
    tier = [m for m, c in enumerate(counts) for _ in range(c)]
    return dict(tier=tier, cap=[16] * 13, price_in=[0.06, 0.07, 0.15, 0.38], price_out=[0.06, 0.07, 0.15, 0.40],
                pre=[0.0] * 4, dec=[10.2, 19.6, 13.9, 41.6], slope=[0.0] * 4)


def make_state(I, cap, seed, stream=5):
    """queued ~ U{0..20000}, running = min(U{0..32}, cap)."""
    g = _gen(seed, stream, "cpu")
    queued = torch.randint(0, 20001, (I,), generator=g).float()
    running = torch.minimum(torch.randint(0, 33, (I,), generator=g), torch.tensor(cap)).to(torch.int32)
    return queued, running


def poisson_arrivals_ms(rate, n_req, seed, stream=9):
    """Arrival times (ms, float64, non-decreasing) of n_req requests of a Poisson stream at `rate` requests per second
    (Poisson arrivals at 6-30 req/s) -- the input of the stream driver (stream.py)."""
    import numpy as np
    g = _gen(seed, stream, "cpu")
    gaps = torch.empty(n_req).exponential_(rate, generator=g).double()
    return (torch.cumsum(gaps, 0) * 1000.0).numpy().astype(np.float64)


def poisson_windows(rate, n_decisions, seed, max_b=64, min_b=4, max_age=0.5, stream=6):
    """Batch windows of a Poisson arrival stream: a batch closes when it holds max_b requests or
    (>= min_b requests and age >= max_age seconds).  Returns lists (B_j, elapsed_ms_j)."""
    g = _gen(seed, stream, "cpu")
    n_req = int(n_decisions * max(min_b, rate * max_age) * 2 + 64)
    gaps = torch.empty(n_req).exponential_(rate, generator=g).double()
    t = torch.cumsum(gaps, 0).tolist()
    sizes, elapsed = [], []
    i = 0
    last_close = 0.0
    while len(sizes) < n_decisions and i < len(t):
        start = t[i]
        j = i
        while True:
            j += 1
            n_in = j - i
            if n_in >= max_b:
                close = t[j - 1]
                break
            if j >= len(t):
                close = t[-1]
                break
            if n_in >= min_b and t[j] - start >= max_age:
                close = max(t[j - 1], start + max_age)
                break
        sizes.append(j - i)
        elapsed.append((close - last_close) * 1000.0)
        last_close = close
        i = j
    return sizes, elapsed


PRESETS = {"quality": (0.8, 0.1, 0.1), "latency": (0.1, 0.8, 0.1), "cost": (0.1, 0.1, 0.8),
           "balanced": (1.0 / 3, 1.0 / 3, 1.0 / 3)}


def simplex_points(step=0.1):
    """All weight vectors (w_qual, w_lat, w_cost) on the 3-simplex at the given step (66 points at 0.1)."""
    n = round(1.0 / step)
    return [(a / n, b / n, (n - a - b) / n) for a in range(n + 1) for b in range(n + 1 - a)]


# ---- gradient-boosted TPOT heads: the paper's trained boosters are unavailable, so forests are drawn ----
def make_forest(M, dec, n_trees=32, depth=4, Fa=2, seed=0, stream=8, I=None):
    """A random regression forest per tier in the node format of include/routebalance.h (rb_tree_node): features
    x[0] = running b, x[1] = queued tokens d, x[2..] = auxiliary telemetry in [0,1].  Leaves are small corrections
    around base[t] = dec[t], rising with b, so that the predicted TPOT stays positive and load-dependent.
    Returns dict(node_feature, node_value, node_left, node_right, tree_root, tier_tree_begin, base, n_features, aux)."""
    g = _gen(seed, stream, "cpu")
    F = 2 + Fa
    feat, val, left, right, roots, begin = [], [], [], [], [], [0]

    def rnd():
        return float(torch.rand((), generator=g))

    def grow(t, level, lo_b, hi_b):
        n = len(feat)
        feat.append(-1), val.append(0.0), left.append(-1), right.append(-1)
        if level == depth or (level >= 1 and rnd() < 0.15):
            mid = 0.5 * (lo_b + hi_b) / 32.0
            val[n] = dec[t] * 0.04 * (mid - 0.5 + 0.5 * (rnd() - 0.5))
            return n
        u = rnd()
        c = 0 if u < 0.5 else (1 if u < 0.75 or Fa == 0 else 2 + int(rnd() * Fa) % Fa)
        feat[n] = c
        if c == 0:
            thr = float(int(lo_b + rnd() * max(1.0, hi_b - lo_b))) + 0.5
            val[n] = thr
            left[n] = grow(t, level + 1, lo_b, min(hi_b, thr))
            right[n] = grow(t, level + 1, max(lo_b, thr), hi_b)
        else:
            val[n] = rnd() * (20000.0 if c == 1 else 1.0)
            left[n] = grow(t, level + 1, lo_b, hi_b)
            right[n] = grow(t, level + 1, lo_b, hi_b)
        return n

    for t in range(M):
        for _ in range(n_trees):
            roots.append(grow(t, 0, 0.0, 32.0))
        begin.append(len(roots))
    aux = None
    if I is not None and Fa > 0:
        aux = torch.rand(I, Fa, generator=g)
    return dict(node_feature=feat, node_value=val, node_left=left, node_right=right, tree_root=roots,
                tier_tree_begin=begin, base=[float(x) for x in dec], n_features=F, aux=aux)


def lookup_forest(M, dec, slope, bmax):
    """One tree per tier that tabulates a function of the running batch b = 0..bmax (a chain of splits at b + 0.5);
    the leaf of b holds the caller-supplied value table[t][b].  Used with table = the linear head's tpot to check that
    the boosted-head path reproduces the linear one.  Returns (forest dict without leaf values filled, leaf_index[t][b])."""
    feat, val, left, right, roots, begin, leaf_index = [], [], [], [], [], [0], []
    for t in range(M):
        roots.append(len(feat))
        idx = []
        for b in range(bmax):
            n = len(feat)
            feat.append(0), val.append(b + 0.5), left.append(n + 1), right.append(n + 2)
            idx.append(len(feat))
            feat.append(-1), val.append(0.0), left.append(-1), right.append(-1)
        idx.append(len(feat))
        feat.append(-1), val.append(0.0), left.append(-1), right.append(-1)
        leaf_index.append(idx)
        begin.append(len(roots))
    return dict(node_feature=feat, node_value=val, node_left=left, node_right=right, tree_root=roots,
                tier_tree_begin=begin, base=[0.0] * M, n_features=2, aux=None), leaf_index
