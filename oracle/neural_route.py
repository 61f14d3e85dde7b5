"""O6 — WhiFlash-Neural routing policy (oracle).  SURVEY.md §8(f) row f1.

Test infrastructure; see oracle/__init__.py.

PAPER.md:87   "our policy takes the final-layer hidden states of the target model at the
              current decoding step t, h_t in R^d ... the network directly predicts a
              continuous scalar, Delta AL_t = f_theta(h_t) ... a lightweight multilayer
              perceptron (MLP) regressor, consisting primarily of two linear layers."
PAPER.md:325  "the router first projects h_t to an intermediate dimension m = d/8.  This
              intermediary representation is then supplied to a Gaussian Error Linear Unit
              (GELU) activation (Hendrycks and Gimpel, 2016), followed by dropout.  Finally,
              the intermediary representation is projected to a scalar output y_t".
PAPER.md:103-107  pi(h_t, tau_neural) = m_a if Delta AL_t > tau_neural, m_d otherwise.

Readings (N1-N6): the two linear layers carry biases (the parameter counts of
PAPER.md Table 5, 0.82 M at d = 2560 and 2.10 M at d = 4096, fit d*m + m + m + 1); GELU is the
exact form x * Phi(x) = 0.5 x (1 + erf(x / sqrt 2)) of the cited paper; dropout is the identity at
inference; h_t is the final hidden row of the last accepted position (row a of the block, the
position whose logits give the bonus token: the same position the entropy policy reads);
strict '>' selects the autoregressive drafter, everything else (ties included) the diffusion
drafter.

  z      = W1 h + b1        W1 in R^{m x d} (one row per hidden unit, bf16), b1 in R^m (fp32)
  u      = GELU(z)
  dAL    = <w2, u> + b2     w2 in R^m (bf16), b2 scalar (fp32)
  route  = 1 (AR) if dAL > tau_neural else 0 (diffusion)
"""

import math

import numpy as np

from . import bf16

ROUTE_DIFFUSION = 0
ROUTE_AR = 1

_erf = np.vectorize(math.erf, otypes=[np.float64])


def gelu(x):
    """Exact GELU, x * Phi(x), fp64 (Hendrycks and Gimpel, 2016)."""
    x = np.asarray(x, dtype=np.float64)
    return 0.5 * x * (1.0 + _erf(x / math.sqrt(2.0)))


def delta_al(h_bits, w1_bits, b1, w2_bits, b2):
    """f_theta(h) for each row of h.  h_bits [B, d], w1_bits [m, d], w2_bits [m] are bf16 bit
    patterns (uint16), b1 [m] and b2 are fp32; everything is widened exactly and evaluated in fp64."""
    h = bf16.to_f64(h_bits)
    w1 = bf16.to_f64(w1_bits)
    w2 = bf16.to_f64(w2_bits)
    b1 = np.asarray(b1, dtype=np.float32).astype(np.float64)
    b2 = float(np.float32(b2))
    assert h.ndim == 2 and w1.ndim == 2 and w1.shape[1] == h.shape[1] and w2.shape == (w1.shape[0],) == b1.shape
    z = h @ w1.T + b1[None, :]
    return gelu(z) @ w2 + b2


def neural_route(hidden_bits, q_indptr, accept_len, w1_bits, b1, w2_bits, b2, tau):
    """Route every sequence of a verified block.  hidden_bits [sum_q, d]: the target's final hidden
    rows of the block; the router reads row q_indptr[b] + accept_len[b] (reading N4).  tau: scalar
    or [B].  Returns (dAL fp64 [B], route int32 [B]); a sequence with an empty block gets (0, 0)."""
    q_indptr = np.asarray(q_indptr, dtype=np.int64)
    B = len(q_indptr) - 1
    tau = np.broadcast_to(np.asarray(tau, dtype=np.float64), (B,))
    out = np.zeros(B, dtype=np.float64)
    route = np.zeros(B, dtype=np.int32)
    for b in range(B):
        if q_indptr[b + 1] == q_indptr[b]:
            continue
        a = int(accept_len[b])
        assert 0 <= a < q_indptr[b + 1] - q_indptr[b]
        row = hidden_bits[q_indptr[b] + a][None, :]
        out[b] = delta_al(row, w1_bits, b1, w2_bits, b2)[0]
        route[b] = ROUTE_AR if out[b] > tau[b] else ROUTE_DIFFUSION
    return out, route
