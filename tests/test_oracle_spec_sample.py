"""Pins for oracle O8 (stochastic acceptance: speculative sampling with temperature), CPU only.

PAPER.md:19, :79-81; readings S1-S5.  Each test fixes the oracle to something other than itself: the
theorem the rule exists for (the emitted token is distributed exactly as the target's p, whatever the drafter's q:
checked by quadrature over the uniforms), hand-computed thresholds and CDF boundaries on a four-token vocabulary, the
p = q and one-hot special cases, the greedy limit against the already-pinned O2, and the temperature identities.
"""

import math

import numpy as np

from oracle import accept_route, spec_sample
from paper_2606_07710_b200 import synth

P4 = np.array([0.1, 0.2, 0.3, 0.4])


def _one(logits_row_list, drafts, u_acc, u_s, T=1.0, q=None, tau=1.0):
    logits = np.asarray(logits_row_list, dtype=np.float32)
    n = len(logits)
    return spec_sample.spec_sample_entropy_route(logits, np.asarray(drafts, np.int32), np.array([0, n], np.int32), T,
                                                 np.asarray(u_acc, np.float64), np.asarray([u_s], np.float64), tau,
                                                 draft_q=None if q is None else np.asarray(q, np.float32))


def test_accept_threshold_one_hot_drafter():
    """Deterministic drafter (q = one-hot): draft x is accepted iff u < p(x) = 0.3."""
    z = np.log(P4)
    for u, want in ((0.0, 1), (0.2999, 1), (0.3001, 0), (0.99, 0)):
        r = _one([z, z], [0, 2], [0.0, u], 0.5)
        assert r["accept_len"][0] == want and r["n_commit"][0] == want + 1


def test_residual_excludes_the_rejected_token_and_cdf_boundaries():
    """Rejected x = 2 with one-hot q: residual = p without x, renormalised: [0.1, 0.2, 0, 0.4] / 0.7.  Boundaries of the
    inverse CDF at 1/7 and 3/7; token 2 can never be emitted."""
    z = np.log(P4)
    for u_s, want in ((0.0, 0), (1 / 7 - 1e-9, 0), (1 / 7 + 1e-9, 1), (3 / 7 - 1e-9, 1), (3 / 7 + 1e-9, 3), (0.999999, 3)):
        r = _one([z, z], [0, 2], [0.0, 0.9], u_s)
        assert r["accept_len"][0] == 0 and r["token"][0] == want


def test_bonus_token_drawn_from_p_when_all_accepted():
    """gamma = 1, draft accepted: the emitted token is the bonus, inverse CDF of p of ROW 1 (a different row)."""
    z0, z1 = np.log(P4), np.log(P4[::-1])                   # row 1: p = [0.4, 0.3, 0.2, 0.1]
    for u_s, want in ((0.39, 0), (0.41, 1), (0.69, 1), (0.71, 2), (0.91, 3)):
        r = _one([z0, z1], [0, 3], [0.0, 0.39], u_s)        # p0(3) = 0.4 > u = 0.39: accepted
        assert r["accept_len"][0] == 1 and r["token"][0] == want and r["n_commit"][0] == 2


def test_full_q_ratio_and_residual():
    """q = [0.4, 0.3, 0.2, 0.1], x = 0: ratio p/q = 0.25; residual max(0, p - q) = [0, 0, 0.1, 0.3] / 0.4."""
    z = np.log(P4)
    q = np.array([[0.4, 0.3, 0.2, 0.1]] * 2)
    assert _one([z, z], [0, 0], [0.0, 0.2499], 0.5, q=q)["accept_len"][0] == 1
    assert _one([z, z], [0, 0], [0.0, 0.2501], 0.5, q=q)["accept_len"][0] == 0
    for u_s, want in ((0.0, 2), (0.2499, 2), (0.2501, 3), (0.99, 3)):
        assert _one([z, z], [0, 0], [0.0, 0.9], u_s, q=q)["token"][0] == want
    # x = 3: p/q = 4 -> min(1, .) = 1: accepted for every u < 1
    assert _one([z, z], [0, 3], [0.0, 0.999999], 0.5, q=q)["accept_len"][0] == 1


def test_p_equals_q_always_accepts():
    z = np.log(P4)
    q = np.array([P4, P4, P4])
    for x in range(4):
        r = _one([z, z, z], [0, x, (x + 1) % 4], [0.0, 0.999, 0.999], 0.3, q=q)
        assert r["accept_len"][0] == 2


def test_first_rejection_stops_the_chain():
    """Draft 2 would pass, but draft 1 fails: a = 0, and the emitted token comes from row 0's residual."""
    z = np.log(P4)
    r = _one([z, z, z], [0, 0, 3], [0.0, 0.5, 0.0], 0.0)    # p(0) = 0.1 < 0.5: rejected at once
    assert r["accept_len"][0] == 0 and r["token"][0] == 1   # residual [0, .2, .3, .4]: u = 0 -> first token with mass


def test_emitted_token_is_distributed_as_the_target_p():
    """The theorem behind the rule (Leviathan et al. 2023, Thm 1; cited at PAPER.md:19): for ANY drafter q, drawing
    x ~ q and applying accept / resample yields a token distributed exactly as p.  Midpoint quadrature over
    (u_accept, u_sample) on a 4-token vocabulary, for a full q and for each one-hot q weighted by a proposal law."""
    z = np.log(P4)
    q = np.array([0.55, 0.05, 0.25, 0.15])
    N = 120
    grid = (np.arange(N) + 0.5) / N
    out = np.zeros(4)
    for x in range(4):
        for ua in grid:
            acc = _one([z, z], [0, x], [0.0, ua], 0.5, q=[q, q])["accept_len"][0]
            if acc:
                out[x] += q[x] / N
            else:
                for us in grid:
                    out[_one([z, z], [0, x], [0.0, ua], us, q=[q, q])["token"][0]] += q[x] / (N * N)
    np.testing.assert_allclose(out, P4, atol=1.5 / N)


def test_greedy_limit_matches_o2():
    """Near-deterministic rows (the winner holds all but 1e-12 of the mass), one-hot drafter: a draft is accepted iff it
    is the argmax, and the emitted token is the argmax of row a: exactly O2's accept_len / bonus (pinned elsewhere)."""
    g = synth.rng(8, 8)
    q_lens = [8, 16, 4, 1]
    prefix = [3, 15, 0, 0]
    logits, drafts, ip, _ = synth.make_logits_block(g, q_lens, 97, 1.0, prefix, [60.0] * 4)
    rows = np.arange(len(logits))
    logits[rows, logits.argmax(axis=1)] += 60.0
    want = accept_route.accept_entropy_route(logits, drafts, ip, 2.0)
    u_acc = g.uniform(0.0, 1.0 - 1e-9, size=len(logits))
    got = spec_sample.spec_sample_entropy_route(logits, drafts, ip, 1.0, u_acc, g.uniform(0, 1 - 1e-9, size=4), 2.0)
    assert list(got["accept_len"]) == list(want["accept_len"]) == prefix
    assert list(got["token"]) == list(want["bonus_token"])
    np.testing.assert_allclose(got["entropy"], want["entropy"], atol=1e-9)


def test_temperature_identities():
    """T scales the logits: (z, T) == (z / T, 1); the entropy is that of softmax(z / T) (O2's entropy_direct on z / T);
    T -> large flattens towards ln V, T -> small sharpens towards 0."""
    g = synth.rng(9, 9)
    logits = synth.normal_f32(g, (6, 50), 2.0)
    drafts = g.integers(0, 50, size=6).astype(np.int32)
    ip = np.array([0, 6], np.int32)
    ua, us = g.uniform(size=6), g.uniform(size=1)
    a = spec_sample.spec_sample_entropy_route(logits, drafts, ip, 2.0, ua, us, 1.0)
    half = (logits.astype(np.float64) / 2.0)
    b = spec_sample.spec_sample_entropy_route(half, drafts, ip, 1.0, ua, us, 1.0)
    for k in ("accept_len", "token", "route"):
        assert list(a[k]) == list(b[k])
    row = int(a["accept_len"][0])
    assert abs(a["entropy"][0] - accept_route.entropy_direct(half[row])) < 1e-12
    hot = spec_sample.spec_sample_entropy_route(logits, drafts, ip, 1e3, ua, us, 1.0)["entropy"][0]
    cold = spec_sample.spec_sample_entropy_route(logits, drafts, ip, 1e-3, ua, us, 1.0)["entropy"][0]
    assert abs(hot - math.log(50)) < 1e-3 and cold < 1e-6


def test_inverse_cdf_skips_zero_mass_and_handles_minus_inf():
    """-inf logits have p = 0 and can never be emitted, even at u = 0 or next to a boundary."""
    z = np.array([-np.inf, math.log(0.5), -np.inf, math.log(0.5)], np.float32)
    for u_s, want in ((0.0, 1), (0.4999, 1), (0.5001, 3), (0.999999, 3)):
        assert _one([z], [0], [0.0], u_s)["token"][0] == want
    r = _one([z], [0], [0.0], 0.25)
    assert r["accept_len"][0] == 0 and r["n_commit"][0] == 1 and abs(r["entropy"][0] - math.log(2)) < 1e-12


def test_empty_block_and_margins():
    logits = np.zeros((2, 4), np.float32)
    r = spec_sample.spec_sample_entropy_route(logits, np.zeros(2, np.int32), np.array([0, 0, 2], np.int32), 1.0,
                                              np.array([0.0, 0.3]), np.array([0.0, 0.6]), 1.0)
    assert list(r["n_commit"]) == [0, 1] and r["token"][0] == 0
    # uniform p = 1/4, one-hot q: ratio 0.25 vs u = 0.3 -> rejected; accept margin 0.05; residual thirds, u = 0.6 -> margin 1/15
    assert r["accept_len"][1] == 0 and abs(r["accept_margin"][1] - 0.05) < 1e-12
    assert abs(r["margin"][1] - (2 / 3 - 0.6)) < 1e-12
