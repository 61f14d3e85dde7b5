"""O3 — KV-only Prefill, and O5 — the full drafter prefill it is checked against (oracle).

Test infrastructure; see oracle/__init__.py.

PAPER.md:119 (§3.4): "A full forward pass on each token computes self-attention,
the MLP, and the LM head ... for catch-up, only the KV cache is required since the
drafter does not need predictions for tokens that the target has already
accepted."  BASELINE.json north_star (c): the accepted tokens' hidden states go
through the idle drafter's per-layer W_K/W_V with RoPE and are appended to its
paged cache, without running its attention or MLP.

DESIGN.md readings: C14 every drafter layer projects the same externally supplied
hidden rows X; C15 X = rows 0..a of the block; C16 no bias / QK-norm; C17 RoPE
rotate-half pairing (r, r + D/2), position = drafter cache length at append time
+ row offset, angles phi = pos * theta^(-2r/D); C18 W is [hidden][Hkv*D], K = X W,
output column c -> head c // D, lane c % D; C13 bf16 stores are RNE.
"""

import numpy as np

from . import bf16
from .paged_kv import PagedKV


class Drafter:
    """Weights are uint16 bf16 bits, W_K[l], W_V[l] : [hidden][Hkv*D] (C18)."""

    def __init__(self, w_k, w_v, kv: PagedKV, rope_theta):
        assert len(w_k) == len(w_v) == kv.L
        self.w_k = [np.asarray(w, dtype=np.uint16) for w in w_k]
        self.w_v = [np.asarray(w, dtype=np.uint16) for w in w_v]
        self.kv = kv
        self.theta = float(rope_theta)
        self.hidden = self.w_k[0].shape[0]


def rope_rotate_half(x, pos, theta):
    """x fp64 [..., D]; rotate pairs (r, r + D/2) by phi = pos * theta^(-2r/D)  (C17)."""
    D = x.shape[-1]
    half = D // 2
    r = np.arange(half, dtype=np.float64)
    phi = float(pos) * theta ** (-2.0 * r / D)
    c, s = np.cos(phi), np.sin(phi)
    lo, hi = x[..., :half], x[..., half:]
    return np.concatenate([lo * c - hi * s, hi * c + lo * s], axis=-1)


def project_rows(drafter, x_bits, p0):
    """K/V for rows x_bits (uint16 [n][hidden]) appended at positions p0 .. p0+n-1.

    Returns (K, V): fp64 [L][n][Hkv][D], unrounded.
    """
    kv = drafter.kv
    X = bf16.to_f64(x_bits)
    n = X.shape[0]
    K = np.zeros((kv.L, n, kv.Hkv, kv.D), dtype=np.float64)
    V = np.zeros((kv.L, n, kv.Hkv, kv.D), dtype=np.float64)
    for l in range(kv.L):
        k = (X @ bf16.to_f64(drafter.w_k[l])).reshape(n, kv.Hkv, kv.D)
        v = (X @ bf16.to_f64(drafter.w_v[l])).reshape(n, kv.Hkv, kv.D)
        for t in range(n):
            K[l, t] = rope_rotate_half(k[t], p0 + t, drafter.theta)
        V[l] = v
    return K, V


def append_rows(drafter, rows_per_seq):
    """rows_per_seq[b] = uint16 [n_b][hidden] (n_b may be 0).  One reserve call for
    the whole batch (ascending b, C24), then K/V of every layer are written at
    p0_b + t and seq_len[b] += n_b.  Returns {b: (K, V) fp64 unrounded}.
    """
    kv = drafter.kv
    kv.reserve([len(r) for r in rows_per_seq])
    unrounded = {}
    for b, rows in enumerate(rows_per_seq):
        n = len(rows)
        if n == 0:
            continue
        p0 = int(kv.seq_len[b])
        K, V = project_rows(drafter, rows, p0)
        Kb, Vb = bf16.from_f64(K), bf16.from_f64(V)
        for l in range(kv.L):
            for t in range(n):
                kv.write(l, b, p0 + t, Kb[l, t], Vb[l, t])
        kv.seq_len[b] += n
        unrounded[b] = (K, V)
    return unrounded


def kv_only_prefill(drafter, hidden_bits, q_indptr, n_rows):
    """O3.  hidden_bits uint16 [sum_q][hidden]; rows 0..n_rows[b]-1 of each block."""
    hidden_bits = np.asarray(hidden_bits, dtype=np.uint16)
    B = len(q_indptr) - 1
    rows = [hidden_bits[int(q_indptr[b]): int(q_indptr[b]) + int(n_rows[b])] for b in range(B)]
    return append_rows(drafter, rows)


# --------------------------------------------------------------------------
# O5: the comparison.  A complete (single-input, C14) drafter layer stack for the
# same rows: Q/K/V projections, RoPE, causal attention over the drafter cache,
# output projection, a two-matrix GELU MLP and an LM head.  Only the K/V it writes
# on the way are kept; pin O3.i says that cache equals O3's bit for bit.
# Written separately from project_rows on purpose (token by token, einsum).
# --------------------------------------------------------------------------
def full_drafter_prefill(drafter, extra, hidden_bits, q_indptr, n_rows, n_q_heads):
    """extra: dict of fp64 weights w_q[l] [hidden][Hq*D], w_o[l] [Hq*D][hidden],
    w_up[l] [hidden][F], w_down[l] [F][hidden], lm_head [hidden][V]."""
    kv = drafter.kv
    B = len(q_indptr) - 1
    kv.reserve([int(n) for n in n_rows])
    D, Hkv = kv.D, kv.Hkv
    group = n_q_heads // Hkv
    logits_out = []
    for b in range(B):
        n = int(n_rows[b])
        p0 = int(kv.seq_len[b])
        for t in range(n):
            x = bf16.to_f64(hidden_bits[int(q_indptr[b]) + t])           # [hidden]
            pos = p0 + t
            h_out = x
            for l in range(kv.L):
                wk = bf16.to_f64(drafter.w_k[l]).reshape(-1, Hkv, D)
                wv = bf16.to_f64(drafter.w_v[l]).reshape(-1, Hkv, D)
                k = np.einsum("i,ihd->hd", x, wk)
                v = np.einsum("i,ihd->hd", x, wv)
                q = (x @ extra["w_q"][l]).reshape(n_q_heads, D)
                k = rope_rotate_half(k, pos, drafter.theta)
                q = rope_rotate_half(q, pos, drafter.theta)
                kv.write(l, b, pos, bf16.from_f64(k), bf16.from_f64(v))
                # causal self-attention over the drafter cache, positions 0..pos
                Kc, Vc = kv.gather(l, b, pos + 1)
                Kc, Vc = bf16.to_f64(Kc), bf16.to_f64(Vc)
                att = np.zeros((n_q_heads, D))
                for h in range(n_q_heads):
                    s = Kc[:, h // group, :] @ q[h] / np.sqrt(D)
                    p = np.exp(s - s.max())
                    att[h] = (p / p.sum()) @ Vc[:, h // group, :]
                y = x + att.reshape(-1) @ extra["w_o"][l]
                u = y @ extra["w_up"][l]
                gelu = 0.5 * u * (1.0 + np.tanh(np.sqrt(2.0 / np.pi) * (u + 0.044715 * u ** 3)))
                h_out = y + gelu @ extra["w_down"][l]
            logits_out.append(h_out @ extra["lm_head"])                    # discarded by the caller
        kv.seq_len[b] += n
    return logits_out
