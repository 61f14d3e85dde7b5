"""O8 — stochastic acceptance: speculative sampling with temperature (oracle; test infrastructure, see
oracle/__init__.py).  SURVEY.md §8(f) f4.

PAPER.md:19   "speculative decoding (SD) (Leviathan et al., 2023; Chen et al., 2023) ... SD utilises a smaller draft
              model to propose tokens, which are subsequently verified in parallel by the target LLM."
PAPER.md:79-81 the entropy is "an O(|V|) reduction over the target next-token probabilities at a single position,
              adding a softmax only when greedy decoding is used": under sampling the softmax already exists, and the
              router reads the entropy of that same distribution.

The paper evaluates greedily and does not restate the sampling rule; readings S1-S5 take the rule of the two
papers it cites for SD (the standard speculative-sampling rule), in the chain block layout of reading C9:

  p_i      = softmax(z_i / T), T > 0                                                        (S1)
  q_i      = the drafter's distribution at row i (full rows, optional); absent = a deterministic drafter,
             q_i = one-hot at the token it proposed                                          (S2)
  accept   : for j = 1, 2, ..: x = draft token j, accepted iff u_accept[r0+j] < min(1, p_{j-1}(x) / q_{j-1}(x))
             (q = 0 counts as ratio 1); a = number accepted before the first rejection       (S3)
  emit     : if a < gamma the token after the accepted prefix is drawn from the residual
             r ∝ max(0, p_a - q_a) (all of p_a if the residual is empty); if a = gamma it is the bonus token drawn
             from p_a.  The draw is the inverse CDF in vocabulary order at u_sample[b]: the smallest v with
             sum_{w<=v} r_w > u * sum_w r_w                                                  (S4)
  H, route : entropy (nats) of p_a — the distribution the sampler already has, at temperature T — and the
             C1 threshold rule                                                               (S5)
The uniforms are inputs (one per draft row, one per sequence), so both sides of a parity test see the same draws.
"""

import numpy as np

from .accept_route import ROUTE_AR, ROUTE_DIFFUSION


def softmax_t(z, temperature):
    """softmax(z / T) in fp64; -inf entries get probability 0 (C23)."""
    z = np.asarray(z, dtype=np.float64) / float(temperature)
    m = z.max()
    assert np.isfinite(m), "C23: a row of all -inf has no distribution"
    e = np.exp(z - m)
    return e / e.sum()


def entropy_of(p):
    nz = p > 0
    return float(-(p[nz] * np.log(p[nz])).sum())


def inverse_cdf(r, u):
    """Smallest v with cumsum(r)[v] > u * sum(r) (S4); r >= 0 with positive total, 0 <= u < 1."""
    c = np.cumsum(np.asarray(r, dtype=np.float64))
    v = int(np.searchsorted(c, float(u) * c[-1], side="right"))
    return min(v, len(c) - 1)


def spec_sample_entropy_route(logits, draft_tokens, q_indptr, temperature, u_accept, u_sample, tau, draft_q=None, kv=None):
    """logits fp32 [sum_q][V]; draft_tokens int32 [sum_q]; u_accept [sum_q], u_sample [B] in [0, 1);
    draft_q None or fp32 [sum_q][V] (row i = the drafter's distribution for the token after row i).

    Returns accept_len, token (the resampled / bonus token), n_commit, route (int32 [B]), entropy (fp64 [B]) and
    margin (fp64 [B]): how far, in units of total mass, u_sample sits from the nearest CDF boundary of the draw —
    parity tests skip the token comparison when a draw is closer to a boundary than the kernel's fp32 softmax resolves.
    """
    logits = np.asarray(logits)
    B = len(q_indptr) - 1
    tau = np.broadcast_to(np.asarray(tau, dtype=np.float64), (B,))
    res = dict(accept_len=np.zeros(B, np.int32), token=np.zeros(B, np.int32), n_commit=np.zeros(B, np.int32),
               route=np.zeros(B, np.int32), entropy=np.zeros(B, np.float64), margin=np.ones(B, np.float64),
               accept_margin=np.ones(B, np.float64))
    for b in range(B):
        r0, r1 = int(q_indptr[b]), int(q_indptr[b + 1])
        gamma = r1 - r0 - 1
        if gamma < 0:
            continue
        a = 0
        p = softmax_t(logits[r0], temperature)
        while a < gamma:
            x = int(draft_tokens[r0 + a + 1])
            qx = 1.0 if draft_q is None else float(draft_q[r0 + a][x])
            ratio = 1.0 if qx <= 0.0 else min(1.0, p[x] / qx)
            u = float(u_accept[r0 + a + 1])
            res["accept_margin"][b] = min(res["accept_margin"][b], abs(u - ratio))
            if not (u < ratio):
                break
            a += 1
            p = softmax_t(logits[r0 + a], temperature)
        if a < gamma:
            x = int(draft_tokens[r0 + a + 1])
            if draft_q is None:
                q = np.zeros_like(p)
                q[x] = 1.0
            else:
                q = np.asarray(draft_q[r0 + a], dtype=np.float64)
            r = np.maximum(0.0, p - q)
            if not (r.sum() > 0.0):
                r = p
        else:
            r = p
        tok = inverse_cdf(r, u_sample[b])
        c = np.cumsum(r) / r.sum()
        res["margin"][b] = float(np.abs(c - float(u_sample[b])).min())
        res["accept_len"][b] = a
        res["token"][b] = tok
        res["n_commit"][b] = a + 1
        res["entropy"][b] = entropy_of(p)
        res["route"][b] = ROUTE_AR if res["entropy"][b] > tau[b] else ROUTE_DIFFUSION
        if kv is not None:
            kv.seq_len[b] += a + 1
    return res
