"""O9 — the final backlog token run through the drafter layer in full (oracle).

Test infrastructure; see oracle/__init__.py.

PAPER.md:119 (§3.4 "KV-only Prefill"): "we compute only the attention layer on tokens
accepted by another drafter, processing only the final token in full, so that its
post-MLP hidden state can feed the next draft round."  PAPER.md:206: "The KV-only
prefill of Section 3.4 computes attention over the backlog tokens and continues
processing only the final token in full.  This avoids invoking the transformer MLP
layer and LM head for tokens that have already been accepted".  SURVEY.md §8(f) f3.

The paper names its drafters but not their layer; readings F1-F6 fix it as the
layer oracle O5 (kv_prefill.full_drafter_prefill) already commits to, minus the LM head:

  F1  the final backlog token of sequence b is the last row its catch-up prefill
      appended: position p = cache_len[b] - 1 AFTER the flush; its K/V (bf16) are in
      the cache already, written by the KV-only prefill (O3).
  F2  one layer, no norms, no biases (C16), residual form:
        q   = RoPE(x W_Q, p)                          [Hq][D]   (rotate-half, C17)
        att = softmax(q K^T / sqrt(D)) V  over cache positions 0..p   (GQA map C11)
        y   = x + att W_O                             [hidden]
        h   = y + GELU(y W_up) W_down                 [hidden]  (two-matrix MLP)
      GELU is the tanh form 0.5 u (1 + tanh(sqrt(2/pi) (u + 0.044715 u^3))), the one O5
      was pinned with.  The LM head is NOT run: the post-MLP state is what "feeds the
      next draft round"; the head belongs to drafting.
  F3  a multi-layer drafter (C14: every layer takes the same externally supplied row x)
      yields one post-MLP state per layer: h [L][hidden].
  F4  weights are bf16 (widened exactly); everything else is fp64 and unrounded here.
      The bf16 roundings of the CUDA path (q, att, the operand copies of y and GELU(u),
      the stored h) are its error, covered by the tolerance (rel-L2 5e-3, as for K/V).

Orientation (C18): W_Q [hidden][Hq*D], W_O [Hq*D][hidden], W_up [hidden][F],
W_down [F][hidden]; a row vector multiplies from the left.
"""

import numpy as np

from . import bf16
from .kv_prefill import Drafter, rope_rotate_half


class FullLayer:
    """The weights KV-only prefill skips: per layer W_Q, W_O, W_up, W_down as bf16 bits."""

    def __init__(self, w_q, w_o, w_up, w_down, n_q_heads):
        self.w_q = [np.asarray(w, dtype=np.uint16) for w in w_q]
        self.w_o = [np.asarray(w, dtype=np.uint16) for w in w_o]
        self.w_up = [np.asarray(w, dtype=np.uint16) for w in w_up]
        self.w_down = [np.asarray(w, dtype=np.uint16) for w in w_down]
        self.n_q_heads = int(n_q_heads)


def gelu_tanh(u):
    return 0.5 * u * (1.0 + np.tanh(np.sqrt(2.0 / np.pi) * (u + 0.044715 * u ** 3)))


def layer_forward(x, p, Kc, Vc, w_q, w_o, w_up, w_down, n_q_heads, theta):
    """F2 for one token.  x fp64 [hidden]; p its position; Kc, Vc fp64 [p+1][Hkv][D] = the
    layer's cache at positions 0..p (the token's own K/V at p).  Returns (h, y, att, q)."""
    n, Hkv, D = Kc.shape
    assert n == p + 1
    group = n_q_heads // Hkv
    q = rope_rotate_half((x @ w_q).reshape(n_q_heads, D), p, theta)
    att = np.zeros((n_q_heads, D), dtype=np.float64)
    for h in range(n_q_heads):
        g = h // group                                        # C11
        s = (Kc[:, g, :] @ q[h]) / np.sqrt(D)                 # scores over positions 0..p
        w = np.exp(s - s.max())
        att[h] = (w / w.sum()) @ Vc[:, g, :]
    y = x + att.reshape(-1) @ w_o
    h_out = y + gelu_tanh(y @ w_up) @ w_down
    return h_out, y, att, q


def final_token_full(drafter: Drafter, full: FullLayer, x_bits, b):
    """h fp64 [L][hidden] for the last cached token of sequence b (F1), whose hidden row is x_bits."""
    kv = drafter.kv
    p = int(kv.seq_len[b]) - 1
    assert p >= 0, "final_token_full: the sequence has no cached token"
    x = bf16.to_f64(np.asarray(x_bits, dtype=np.uint16))
    out = np.zeros((kv.L, drafter.hidden), dtype=np.float64)
    for l in range(kv.L):
        Kb, Vb = kv.gather(l, b, p + 1)
        out[l] = layer_forward(x, p, bf16.to_f64(Kb), bf16.to_f64(Vb), bf16.to_f64(full.w_q[l]),
                               bf16.to_f64(full.w_o[l]), bf16.to_f64(full.w_up[l]), bf16.to_f64(full.w_down[l]),
                               full.n_q_heads, drafter.theta)[0]
    return out


def final_tokens_full(drafter: Drafter, full: FullLayer, hidden_bits, q_indptr, n_rows, select):
    """The batch form the switch uses, AFTER the catch-up prefill of this round (C21): for every sequence with
    select[b] (it switched to this drafter) and n_rows[b] > 0, the final token is row n_rows[b]-1 of its block (F1).
    Returns {b: h [L][hidden]}."""
    out = {}
    for b in range(len(q_indptr) - 1):
        n = int(n_rows[b])
        if not select[b] or n == 0:
            continue
        out[b] = final_token_full(drafter, full, hidden_bits[int(q_indptr[b]) + n - 1], b)
    return out
