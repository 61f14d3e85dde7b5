"""O7 — tree verification (oracle; test infrastructure, see oracle/__init__.py).  SURVEY.md §8(f) f2.

PAPER.md:65   "drafting proceeds through either an autoregressive drafter which produces a tree of candidate
              tokens, or a diffusion-based parallel drafter which predicts a parallel block of tokens.  This
              sequence of candidate tokens is then returned to the target model for parallel verification.
              Finally, the process repeats, continuing from the last accepted token."
PAPER.md:39   "autoregressive (AR) methods ... introduce dynamic, context-aware draft trees."
PAPER.md:317, :327  EAGLE-3: draft-tree depth 8, top-k 10, 60 total draft tokens.

The paper gives the tree's shape but not the verification rule; readings T1-T5 fix it as the
standard greedy tree verification its AR drafter (EAGLE-3) uses:

  Block layout (T1, extends C9): row 0 of a sequence's block is the previous round's bonus token (committed,
  the ROOT); rows 1..n-1 are draft-tree nodes in topological order, parent[i] in [0, i); parent[0] = -1.
  The block's K/V sit in the cache at positions ctx .. ctx+n-1 (node i at ctx+i), as in C11.
  A chain block is the tree parent[i] = i-1.

  anc(i)   = {i} U anc(parent[i]),  anc(0) = {0}                                      (T2)
  tree attention: row i sees keys 0..ctx-1 and ctx+j for j in anc(i); softmax over exactly those keys  (T2)
  g_i      = argmax_v z_i[v]      (lowest index on ties, C7)
  walk     : cur = 0; while cur has a child c with token[c] == g_cur: cur = that child
             (the lowest-index one if several children carry the same token, T3)
  path     = the nodes visited (path[0] = 0), a = len(path) - 1, bonus = g_cur, n_commit = a + 1   (T3)
  H, route : entropy of softmax(z_cur) and the C1 threshold rule, at the LAST ACCEPTED node          (T4)
  compact  : for every layer, the K/V rows of path[k] move from position ctx+path[k] to ctx+k, k = 1..a;
             then seq_len += a + 1.  Afterwards the cache is exactly what chain decoding of the accepted
             tokens would have left (T5).
"""

import numpy as np

from . import bf16
from .accept_route import ROUTE_AR, ROUTE_DIFFUSION, entropy_direct


def ancestors(parent):
    """parent int [n], parent[0] = -1, 0 <= parent[i] < i  ->  list of sorted ancestor lists (self included)."""
    parent = [int(x) for x in parent]
    n = len(parent)
    anc = []
    for i in range(n):
        if i == 0:
            assert parent[0] == -1, "T1: row 0 is the root"
            anc.append([0])
        else:
            assert 0 <= parent[i] < i, "T1: nodes are in topological order"
            anc.append(anc[parent[i]] + [i])
    return anc


def ancestor_masks(parent):
    """The same sets as 64-bit masks (bit j of mask[i] <=> j in anc(i)); n <= 64."""
    assert len(parent) <= 64
    return np.array([sum(1 << j for j in a) for a in ancestors(parent)], dtype=np.uint64)


def tree_attn(kv, layer, q_bits, q_indptr, parent, n_q_heads, sm_scale):
    """q_bits uint16 [sum_q][Hq][D]; parent int32 [sum_q] (per-sequence node indices); returns fp64 [sum_q][Hq][D].

    Row i of sequence b: keys 0..ctx_b-1 and ctx_b + anc(i), written out key by key (T2).
    """
    q_bits = np.asarray(q_bits, dtype=np.uint16)
    B = len(q_indptr) - 1
    group = n_q_heads // kv.Hkv
    out = np.zeros(q_bits.shape, dtype=np.float64)
    for b in range(B):
        r0, r1 = int(q_indptr[b]), int(q_indptr[b + 1])
        n = r1 - r0
        if n == 0:
            continue
        ctx = int(kv.seq_len[b])
        Kb, Vb = kv.gather(layer, b, ctx + n)
        K, V = bf16.to_f64(Kb), bf16.to_f64(Vb)
        anc = ancestors(parent[r0:r1])
        for i in range(n):
            keys = list(range(ctx)) + [ctx + j for j in anc[i]]
            q = bf16.to_f64(q_bits[r0 + i])
            for h in range(n_q_heads):
                g = h // group
                s = (K[keys, g, :] @ q[h]) * sm_scale
                e = np.exp(s - s.max())
                out[r0 + i, h] = (e / e.sum()) @ V[keys, g, :]
    return out


def tree_accept_entropy_route(logits, tokens, parent, q_indptr, tau, kv=None, max_path=None):
    """logits fp32 [sum_q][V]; tokens, parent int32 [sum_q]; tau scalar or [B].

    Returns accept_len, bonus_token, n_commit, route (int32 [B]), entropy (fp64 [B]) and
    path int32 [B][max_path] (path[b][0..a] = accepted nodes, -1 beyond).  kv.seq_len is NOT advanced here:
    compaction (compact_path) does that, after moving the rows (T5).
    """
    logits = np.asarray(logits)
    B = len(q_indptr) - 1
    tau = np.broadcast_to(np.asarray(tau, dtype=np.float64), (B,))
    if max_path is None:
        max_path = max([int(q_indptr[b + 1] - q_indptr[b]) for b in range(B)] + [1])
    res = dict(accept_len=np.zeros(B, np.int32), bonus_token=np.zeros(B, np.int32), n_commit=np.zeros(B, np.int32),
               route=np.zeros(B, np.int32), entropy=np.zeros(B, np.float64),
               path=np.full((B, max_path), -1, np.int32))
    for b in range(B):
        r0, r1 = int(q_indptr[b]), int(q_indptr[b + 1])
        n = r1 - r0
        if n == 0:
            continue
        par = [int(x) for x in parent[r0:r1]]
        ancestors(par)                                      # validates the layout (T1)
        cur, path = 0, [0]
        while True:
            g = int(np.argmax(logits[r0 + cur]))            # first max = lowest id (C7)
            nxt = -1
            for c in range(cur + 1, n):                     # ascending: the lowest-index matching child (T3)
                if par[c] == cur and int(tokens[r0 + c]) == g:
                    nxt = c
                    break
            if nxt < 0:
                break
            cur = nxt
            path.append(cur)
        a = len(path) - 1
        res["accept_len"][b] = a
        res["bonus_token"][b] = g
        res["n_commit"][b] = a + 1
        res["entropy"][b] = entropy_direct(logits[r0 + cur])
        res["route"][b] = ROUTE_AR if res["entropy"][b] > tau[b] else ROUTE_DIFFUSION
        res["path"][b, :a + 1] = path
    return res


def compact_path(kv, path, n_commit):
    """T5: move the accepted nodes' K/V rows to consecutive positions, every layer, then advance seq_len."""
    for b in range(len(n_commit)):
        nc = int(n_commit[b])
        if nc == 0:
            continue
        ctx = int(kv.seq_len[b])
        for layer in range(kv.L):
            rows = []
            for k in range(nc):                              # read every source row first
                pg, slot = kv.locate(b, ctx + int(path[b][k]))
                rows.append((kv.k_pool[layer, pg, :, slot, :].copy(), kv.v_pool[layer, pg, :, slot, :].copy()))
            for k in range(nc):
                kv.write(layer, b, ctx + k, rows[k][0], rows[k][1])
        kv.seq_len[b] = ctx + nc
