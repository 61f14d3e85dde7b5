"""Seeded synthetic inputs shaped like the paper's workloads (BASELINE.json configs[0..4]).

This module is input plumbing only: it holds none of the method's arithmetic (no
attention, no acceptance rule, no entropy, no projection, no paging) and imports
neither `oracle/` nor the CUDA binding.  It is the one module both the oracle-side
tests and the CUDA-side tests/bench may import, so both see identical bits.

The datasets of PAPER.md:131 are not available; these inputs take their shapes
(batch 1 in the paper; block 16 / gamma 15 for the diffusion drafter,
PAPER.md:318; acceptance lengths swinging between 1 and 6) and stand in
for them.  The recipe is stated in DESIGN.md §"Input recipe".

Small tensors come from numpy's counter-based Philox generator keyed by
(seed, stream id); benchmark-scale device tensors come from a seeded
torch.Generator on the device (bench.py / full-size parity tests copy the sampled
pieces back to the host for the oracle).
"""

from dataclasses import dataclass, field

import numpy as np

SEED_BASE = 0x5EED0000


@dataclass(frozen=True)
class Shapes:
    name: str
    hidden: int
    n_q_heads: int
    n_kv_heads: int
    head_dim: int
    n_layers: int
    vocab: int
    page_size: int = 16
    logit_sigma: float = 3.0
    drafter_layers: tuple = (1, 5)      # drafter A (autoregressive) and D (configs[1])
    rope_theta: float = 1e6
    tau: float = 2.0

    @property
    def group(self):
        return self.n_q_heads // self.n_kv_heads

    @property
    def ffn(self):
        """MLP width of the drafter layer of the final-token path (reading F5): 3 x hidden (12288 at 8B-class shapes)."""
        return 3 * self.hidden


TINY = Shapes("tiny", hidden=256, n_q_heads=4, n_kv_heads=2, head_dim=64, n_layers=1,
              vocab=4096, logit_sigma=2.0, drafter_layers=(1,))
LLM8B = Shapes("8b-class", hidden=4096, n_q_heads=32, n_kv_heads=8, head_dim=128, n_layers=36,
               vocab=151936, logit_sigma=3.0, drafter_layers=(1, 5))


@dataclass(frozen=True)
class Workload:
    """One BASELINE.json config: shapes + batch / context / gamma recipe."""
    index: int
    name: str
    shapes: Shapes
    batch: int
    ctx: object            # int, or (lo, hi) for log-uniform
    gammas: tuple          # allowed gamma values; route 1 (AR) -> gammas[0], route 0 (diffusion) -> gammas[-1]
    backlog_cap: int = 32
    switch_prob: float = 0.3
    mean_accept: float = 3.5
    shuffled_pages: bool = False
    extra: dict = field(default_factory=dict)

    @property
    def seed(self):
        return SEED_BASE + self.index


WORKLOADS = [
    Workload(0, "cfg1-tiny", TINY, batch=1, ctx=512, gammas=(7,)),
    Workload(1, "cfg2-8b-b1-ctx4096", LLM8B, batch=1, ctx=4096, gammas=(15,)),
    Workload(2, "cfg3-8b-b16-ctx8192", LLM8B, batch=16, ctx=8192, gammas=(7, 15), backlog_cap=32),
    Workload(3, "cfg4-8b-b4-ctx32768", LLM8B, batch=4, ctx=32768, gammas=(15,), backlog_cap=64),
    Workload(4, "cfg5-8b-b64-serving-mix", LLM8B, batch=64, ctx=(512, 16384), gammas=(7, 15),
             backlog_cap=32, shuffled_pages=True),
]


# ---------------------------------------------------------------------------
# host-side generators (numpy, Philox)
# ---------------------------------------------------------------------------
def rng(seed, stream):
    """Counter-based generator: independent stream per (seed, stream id)."""
    return np.random.Generator(np.random.Philox(key=[int(seed) & (2**64 - 1), int(stream)]))


def f32_to_bf16_bits(x):
    """fp32 -> bf16 bit patterns (uint16), round-to-nearest-even.  Input conversion only."""
    x = np.ascontiguousarray(x, dtype=np.float32)
    u = x.view(np.uint32)
    bias = ((u >> np.uint32(16)) & np.uint32(1)) + np.uint32(0x7FFF)
    return ((u + bias) >> np.uint32(16)).astype(np.uint16)


def bf16_bits_to_f32(bits):
    bits = np.ascontiguousarray(bits, dtype=np.uint16)
    return (bits.astype(np.uint32) << np.uint32(16)).view(np.float32)


def normal_f32(g, shape, std):
    return (g.standard_normal(size=shape, dtype=np.float32) * np.float32(std)).astype(np.float32)


def normal_bf16(g, shape, std):
    return f32_to_bf16_bits(normal_f32(g, shape, std))


def draw_contexts(wl: Workload, g):
    """Context length per sequence: fixed, or floor(exp(U[ln lo, ln hi])) (configs[4])."""
    if isinstance(wl.ctx, tuple):
        lo, hi = wl.ctx
        return np.floor(np.exp(g.uniform(np.log(lo), np.log(hi), size=wl.batch))).astype(np.int32)
    return np.full(wl.batch, wl.ctx, dtype=np.int32)


def draw_free_list(num_pages, g, shuffled):
    """Ordered free list handed to both sides' block tables (a seeded permutation if shuffled)."""
    if shuffled:
        return g.permutation(num_pages).astype(np.int32)
    return np.arange(num_pages, dtype=np.int32)


def draw_route_trace(g, n_slots, batch, switch_prob):
    """Planned router output per (round slot, sequence): a per-sequence Markov chain that flips with probability
    switch_prob per round (BASELINE.json configs[4]: "switch probability 0.3 per round"; PAPER.md:59 the preferable
    drafter swings within a sequence).  The schedule is replayed cyclically, so the last slot's flip is the one that
    closes the cycle (an even number of flips per sequence); with 16 slots the realised flip rate is about
    (15 * p + 0.5) / 16.  route[k][b] in {0 = diffusion, 1 = AR}."""
    route = np.zeros((n_slots, batch), dtype=np.int32)
    state = (g.random(batch) < 0.5).astype(np.int32)                 # output of the slot before slot 0 = of slot n-1
    first = state.copy()
    for k in range(n_slots):
        if k < n_slots - 1:
            flip = (g.random(batch) < switch_prob).astype(np.int32)
            state = state ^ flip
        else:
            state = first                                            # closes the cycle
        route[k] = state
    return route


def draw_accept_prefix(g, gammas, mean_accept=None):
    """Planned accepted-prefix length u_b per sequence.

    mean_accept None -> uniform 0..gamma (configs[0]); else geometric with that
    mean (support 0,1,2,...), truncated to gamma (configs[4]).
    """
    gammas = np.asarray(gammas)
    if mean_accept is None:
        return np.array([g.integers(0, gm + 1) for gm in gammas], dtype=np.int32)
    p = 1.0 / (1.0 + mean_accept)
    u = g.geometric(p, size=len(gammas)) - 1
    return np.minimum(u, gammas).astype(np.int32)


def make_logits_block(g, q_lens, vocab, sigma, accept_prefix, spike):
    """Target logits + draft tokens for one round with a planted outcome.

    logits fp32 [sum_q][vocab] ~ N(0, sigma).  Each row i gets a planted unique
    winner token w_i: logits[i, w_i] = (largest other entry) + gap_i, gap ~ U[0.05, 1].
    Sequence b (rows r0 .. r0+gamma): slot 0 is the already-committed token (ignored
    by the method), drafts 1..u_b equal the winners of rows 0..u_b-1, draft u_b+1
    (if any) is a different token, the rest are random.  `spike[b]` is added to the
    winner of row u_b, which moves that row's entropy (large spike -> low entropy).

    Returns logits, draft_tokens (int32 [sum_q]), q_indptr (int32 [B+1]), winners.
    """
    q_lens = np.asarray(q_lens, dtype=np.int64)
    B = len(q_lens)
    q_indptr = np.zeros(B + 1, dtype=np.int32)
    q_indptr[1:] = np.cumsum(q_lens)
    n = int(q_indptr[-1])
    logits = normal_f32(g, (n, vocab), sigma)
    winners = g.integers(0, vocab, size=n).astype(np.int32)
    gaps = g.uniform(0.05, 1.0, size=n).astype(np.float32)
    rows = np.arange(n)
    logits[rows, winners] = -np.inf
    logits[rows, winners] = logits.max(axis=1) + gaps
    drafts = g.integers(0, vocab, size=n).astype(np.int32)
    for b in range(B):
        r0 = int(q_indptr[b])
        gamma = int(q_lens[b]) - 1
        if gamma < 0:
            continue
        u = int(min(accept_prefix[b], gamma))
        for j in range(1, u + 1):
            drafts[r0 + j] = winners[r0 + j - 1]
        if u < gamma:
            wrong = int(drafts[r0 + u + 1])
            if wrong == int(winners[r0 + u]):
                wrong = (wrong + 1) % vocab
            drafts[r0 + u + 1] = wrong
        logits[r0 + u, winners[r0 + u]] += np.float32(spike[b])
    return logits, drafts, q_indptr, winners


def draw_tree(g, n_nodes, max_depth=8, top_k=10):
    """Draft-tree shape like the AR drafter's (depth 8, top-k 10, 60 draft tokens): parent int32
    [n_nodes], parent[0] = -1 (the root = last committed token), nodes in topological order.  Node i >= 1 hangs
    under a uniformly drawn earlier node that is above the depth limit and has fewer than top_k children."""
    parent = np.full(n_nodes, -1, dtype=np.int32)
    depth = np.zeros(n_nodes, dtype=np.int32)
    kids = np.zeros(n_nodes, dtype=np.int32)
    for i in range(1, n_nodes):
        ok = [j for j in range(i) if depth[j] < max_depth and kids[j] < top_k]
        j = int(ok[g.integers(0, len(ok))])
        parent[i] = j
        depth[i] = depth[j] + 1
        kids[j] += 1
    return parent


def chain_parent(n_nodes):
    """The chain block as a tree: parent[i] = i - 1."""
    return np.arange(-1, n_nodes - 1, dtype=np.int32)


def make_tree_logits_block(g, parents, vocab, sigma, accept_depth, spike):
    """Target logits + node tokens for one tree round with a planted outcome.

    parents: list of per-sequence parent arrays.  Rows get planted unique winners as in make_logits_block.
    For sequence b a downward walk of at most accept_depth[b] steps is drawn from the root; each node on it
    carries its parent's winner, every other child of a walked node carries a different token (siblings get
    distinct tokens), and `spike[b]` is added to the winner of the walk's last node.

    Returns logits, tokens (int32 [sum_q]), parent (int32 [sum_q], concatenated), q_indptr, planned paths.
    """
    B = len(parents)
    q_lens = np.array([len(p) for p in parents], dtype=np.int64)
    q_indptr = np.zeros(B + 1, dtype=np.int32)
    q_indptr[1:] = np.cumsum(q_lens)
    n = int(q_indptr[-1])
    logits = normal_f32(g, (n, vocab), sigma)
    winners = g.integers(0, vocab, size=n).astype(np.int32)
    gaps = g.uniform(0.05, 1.0, size=n).astype(np.float32)
    rows = np.arange(n)
    logits[rows, winners] = -np.inf
    logits[rows, winners] = logits.max(axis=1) + gaps
    tokens = g.integers(0, vocab, size=n).astype(np.int32)
    paths = []
    for b in range(B):
        r0, par = int(q_indptr[b]), parents[b]
        m = len(par)
        if m == 0:
            paths.append([])
            continue
        children = [[c for c in range(m) if par[c] == j] for j in range(m)]
        for j in range(m):                                   # siblings: distinct tokens, none equal to the winner
            used = {int(winners[r0 + j])}
            for c in children[j]:
                t = int(tokens[r0 + c])
                while t in used:
                    t = (t + 1) % vocab
                tokens[r0 + c] = t
                used.add(t)
        cur, path = 0, [0]
        while len(path) - 1 < int(accept_depth[b]) and children[cur]:
            c = int(children[cur][g.integers(0, len(children[cur]))])
            tokens[r0 + c] = winners[r0 + cur]
            cur = c
            path.append(cur)
        logits[r0 + cur, winners[r0 + cur]] += np.float32(spike[b])
        paths.append(path)
    parent = np.concatenate([np.asarray(p, dtype=np.int32) for p in parents]) if n else np.zeros(0, np.int32)
    return logits, tokens, parent, q_indptr, paths


# ---------------------------------------------------------------------------
# device-side generators (torch; benchmark-scale tensors)
# ---------------------------------------------------------------------------
def device_normal_bf16(shape, std, seed, stream, device="cuda", chunk_elems=1 << 28):
    """bf16 tensor ~ N(0, std) generated on the device from a seeded torch.Generator."""
    import torch
    gen = torch.Generator(device=device)
    gen.manual_seed((int(seed) * 1000003 + int(stream)) & (2**63 - 1))
    out = torch.empty(shape, dtype=torch.bfloat16, device=device)
    flat = out.view(-1)
    n = flat.numel()
    for s in range(0, n, chunk_elems):
        e = min(n, s + chunk_elems)
        flat[s:e] = (torch.randn(e - s, dtype=torch.float32, device=device, generator=gen) * std).to(torch.bfloat16)
    return out


def device_normal_f32(shape, std, seed, stream, device="cuda"):
    import torch
    gen = torch.Generator(device=device)
    gen.manual_seed((int(seed) * 1000003 + int(stream)) & (2**63 - 1))
    out = torch.empty(shape, dtype=torch.float32, device=device)
    out.normal_(0.0, std, generator=gen)
    return out
