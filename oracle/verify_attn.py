"""O1 — target-model verification attention (oracle; test infrastructure).

PAPER.md:65 (§3.2): "This sequence of candidate tokens is then returned to the
target model for parallel verification."  BASELINE.json north_star (a): a block
of gamma+1 draft query tokens per sequence, causal within the block, attends over
a paged bf16 GQA KV cache.

Definition written out (readings C10-C12):
  for sequence b with ctx_b = kv.seq_len[b] tokens already final, query row
  i in [0, q_b), query head h, kv head g = h // (Hq // Hkv):
      s_j = <Q[i,h,:], K[b,j,g,:]> * sm_scale          j = 0 .. ctx_b + i
      p   = softmax(s)                                  (fp64, max-subtracted)
      O[i,h,:] = sum_j p_j * V[b,j,g,:]
  The block's own K/V are already in the cache at positions ctx_b .. ctx_b+q_b-1.
Output stays fp64 (the bf16 rounding of the GPU path is covered by the tolerance).
"""

import numpy as np

from . import bf16


def _attend(q, K, V, n_keys, n_q_heads, n_kv_heads, sm_scale, heads):
    """q fp64 [Hq][D]; K, V fp64 [>=n_keys][Hkv][D]; keys 0..n_keys-1 are visible."""
    group = n_q_heads // n_kv_heads
    out = np.zeros((len(heads), q.shape[-1]), dtype=np.float64)
    for n, h in enumerate(heads):
        g = h // group
        s = (K[:n_keys, g, :] @ q[h]) * sm_scale
        m = s.max()
        e = np.exp(s - m)
        p = e / e.sum()
        out[n] = p @ V[:n_keys, g, :]
    return out


def verify_attn_row(kv, layer, b, q_row_bits, i, n_q_heads, sm_scale, heads=None):
    """One query row i of sequence b: fp64 [Hq][D] (or only the listed heads)."""
    n_keys = int(kv.seq_len[b]) + i + 1        # keys 0 .. ctx+i are visible to row i
    Kb, Vb = kv.gather(layer, b, n_keys)
    heads = list(range(n_q_heads)) if heads is None else list(heads)
    return _attend(bf16.to_f64(q_row_bits), bf16.to_f64(Kb), bf16.to_f64(Vb),
                   n_keys, n_q_heads, kv.Hkv, sm_scale, heads)


def verify_attn(kv, layer, q_bits, q_indptr, n_q_heads, sm_scale):
    """All rows.  q_bits uint16 [sum_q][Hq][D]; returns fp64 [sum_q][Hq][D]."""
    q_bits = np.asarray(q_bits, dtype=np.uint16)
    B = len(q_indptr) - 1
    out = np.zeros(q_bits.shape, dtype=np.float64)
    heads = list(range(n_q_heads))
    for b in range(B):
        r0, r1 = int(q_indptr[b]), int(q_indptr[b + 1])
        q_b = r1 - r0
        if q_b == 0:
            continue
        ctx = int(kv.seq_len[b])
        Kb, Vb = kv.gather(layer, b, ctx + q_b)
        K, V = bf16.to_f64(Kb), bf16.to_f64(Vb)
        for i in range(q_b):
            out[r0 + i] = _attend(bf16.to_f64(q_bits[r0 + i]), K, V, ctx + i + 1,
                                  n_q_heads, kv.Hkv, sm_scale, heads)
    return out
