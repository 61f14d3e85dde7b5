"""O2 — greedy acceptance, bonus token, token-level entropy and route (oracle).

Test infrastructure; see oracle/__init__.py.

PAPER.md:65  "the process repeats, continuing from the last accepted token".
PAPER.md:77  "the target model verifies the tokens proposed by the current drafter
             and produces a next-token distribution p(x_t | x_<t) over the
             vocabulary V for the final accepted position.  The router computes
             the entropy H_t = - sum_x p(x|x_<t) log p(x|x_<t)".
PAPER.md:75  low entropy -> diffusion drafter, high entropy -> autoregressive.
PAPER.md:79-81 the entropy is an O(|V|) reduction at a single position, with a
             softmax added when decoding greedily.
The routing equation itself is lost in the extracted text (between PAPER.md:77
and :79); reading C1 reconstructs it from PAPER.md:75 and the neural
rule at PAPER.md:103-107:   pi(H_t, tau) = m_a if H_t > tau_entropy, else m_d.

Block layout (reading C9): row 0 of a sequence's block is the previous round's
bonus token (already committed), rows 1..gamma are draft tokens t_1..t_gamma;
logits row i is the target's distribution for the token after t_i.

  g_i     = argmax_v z_i[v]           (lowest index on ties, C7)
  a       = max{k in [0,gamma] : t_j == g_{j-1} for all 1<=j<=k}     (C6)
  bonus   = g_a ; n_commit = a + 1 ; ctx' = ctx + a + 1              (C8)
  H       = entropy of softmax(z_a) at T = 1, natural log            (C3-C5)
  route   = 1 (AR) if H > tau else 0 (diffusion)                     (C1, C2)
"""

import numpy as np

ROUTE_DIFFUSION = 0
ROUTE_AR = 1


def entropy_direct(z):
    """Shannon entropy (nats) of softmax(z), fp64.  -inf entries contribute 0 (C23)."""
    z = np.asarray(z, dtype=np.float64)
    assert not np.isnan(z).any() and not np.isposinf(z).any(), "C23: NaN/+inf logits undefined"
    m = z.max()
    assert np.isfinite(m), "C23: a row of all -inf has no distribution"
    d = z - m
    e = np.exp(d)
    Z = e.sum()
    fin = np.isfinite(d)
    S = (e[fin] * d[fin]).sum()              # sum e^{z-m} (z-m); 0 * (-inf) := 0
    return np.log(Z) - S / Z


def entropy_chunked(z, chunk):
    """Same entropy from per-chunk (m_c, Z_c, S_c) triples (the form a split sweep needs).

    m = max m_c ; Z = sum Z_c e^{m_c-m} ; S = sum e^{m_c-m} (S_c + (m_c-m) Z_c).
    Used only to cross-check entropy_direct (pin O2.viii).
    """
    z = np.asarray(z, dtype=np.float64)
    parts = []
    for c0 in range(0, len(z), chunk):
        zc = z[c0:c0 + chunk]
        mc = zc.max()
        if not np.isfinite(mc):
            continue                          # an all -inf chunk carries no mass
        d = zc - mc
        e = np.exp(d)
        fin = np.isfinite(d)
        parts.append((mc, e.sum(), (e[fin] * d[fin]).sum()))
    m = max(p[0] for p in parts)
    Z = sum(Zc * np.exp(mc - m) for mc, Zc, _ in parts)
    S = sum(np.exp(mc - m) * (Sc + (mc - m) * Zc) for mc, Zc, Sc in parts)
    return np.log(Z) - S / Z


def accept_entropy_route(logits, draft_tokens, q_indptr, tau, kv=None):
    """logits fp32 [sum_q][V]; draft_tokens int32 [sum_q]; tau scalar or [B].

    Returns dict of accept_len, bonus_token, n_commit, route (int32 [B]) and
    entropy (fp64 [B]).  If kv is given, kv.seq_len[b] += n_commit[b].
    """
    logits = np.asarray(logits)
    draft_tokens = np.asarray(draft_tokens)
    B = len(q_indptr) - 1
    tau = np.broadcast_to(np.asarray(tau, dtype=np.float64), (B,))
    accept_len = np.zeros(B, dtype=np.int32)
    bonus = np.zeros(B, dtype=np.int32)
    n_commit = np.zeros(B, dtype=np.int32)
    route = np.zeros(B, dtype=np.int32)
    entropy = np.zeros(B, dtype=np.float64)
    for b in range(B):
        r0, r1 = int(q_indptr[b]), int(q_indptr[b + 1])
        gamma = r1 - r0 - 1
        if gamma < 0:                          # empty block: nothing verified, nothing committed
            continue
        g = [int(np.argmax(logits[r0 + i])) for i in range(gamma + 1)]  # first max = lowest id
        a = 0
        while a < gamma and int(draft_tokens[r0 + a + 1]) == g[a]:
            a += 1
        accept_len[b] = a
        bonus[b] = g[a]
        n_commit[b] = a + 1
        entropy[b] = entropy_direct(logits[r0 + a])
        route[b] = ROUTE_AR if entropy[b] > tau[b] else ROUTE_DIFFUSION
        if kv is not None:
            kv.seq_len[b] += a + 1
    return dict(accept_len=accept_len, bonus_token=bonus, n_commit=n_commit,
                route=route, entropy=entropy)
