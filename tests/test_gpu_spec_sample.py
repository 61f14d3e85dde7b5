"""GPU parity (through the C-ABI) for stochastic acceptance against oracle O8 on the same seeded
logits, drafter distributions and uniforms.

accept_len, n_commit and the emitted token are compared bit-exact except where the oracle reports that a uniform sits
within MARGIN of its threshold (acceptance) or CDF boundary (draw): the kernel evaluates p in fp32.  Those cases are
counted and must stay rare.  Entropy 1e-3 absolute; route exact outside |H - tau| < 1e-4.
"""

import numpy as np
import pytest

from oracle import spec_sample
from paper_2606_07710_b200 import synth

pytestmark = pytest.mark.gpu

MARGIN = 1e-5
ENTROPY_ABS = 1e-3
ROUTE_BAND = 1e-4


@pytest.fixture(scope="module")
def wf():
    import torch
    assert torch.cuda.is_available(), "gpu tests need a CUDA device"
    from paper_2606_07710_b200 import binding
    ctx = binding.Ctx(0)
    yield binding, ctx
    ctx.close()


def _run(binding, ctx, logits, drafts, ip, T, u_acc, u_s, tau, draft_q=None, max_q=None, kv=None):
    import torch
    import gpu_harness as H
    B, V = len(ip) - 1, logits.shape[1]
    max_q = max_q or max(int(ip[b + 1] - ip[b]) for b in range(B))
    outs = {k: torch.full((B,), -7, dtype=torch.int32, device="cuda") for k in ("accept_len", "token", "route", "n_commit")}
    ent = torch.full((B,), -7.0, dtype=torch.float32, device="cuda")
    tau_arr = np.atleast_1d(np.asarray(tau, dtype=np.float32))
    ws = torch.empty(binding.wf_accept_workspace_bytes(B * max(max_q, 1), V), dtype=torch.uint8, device="cuda")
    binding.wf_accept_sample_entropy_route(ctx, H.f32(logits), V, H.i32(drafts), H.i32(ip), B, max_q, float(T),
                                           None if draft_q is None else H.f32(draft_q), H.f32(u_acc), H.f32(u_s),
                                           H.f32(tau_arr), len(tau_arr) == 1, outs["accept_len"], outs["token"], ent,
                                           outs["route"], outs["n_commit"], kv, ws)
    torch.cuda.synchronize()
    res = {k: v.cpu().numpy() for k, v in outs.items()}
    res["entropy"] = ent.cpu().numpy()
    return res


def _check(res, want, tau):
    """Returns the number of sequences skipped because a uniform sat on a decision boundary."""
    B = len(want["accept_len"])
    tau = np.broadcast_to(np.asarray(tau, dtype=np.float64), (B,))
    skipped = 0
    for b in range(B):
        if want["accept_margin"][b] < MARGIN:
            skipped += 1
            continue
        assert res["accept_len"][b] == want["accept_len"][b] and res["n_commit"][b] == want["n_commit"][b], b
        assert abs(float(res["entropy"][b]) - want["entropy"][b]) <= ENTROPY_ABS, b
        if abs(want["entropy"][b] - tau[b]) >= ROUTE_BAND:
            assert res["route"][b] == want["route"][b], b
        if want["margin"][b] < MARGIN:
            skipped += 1
            continue
        assert res["token"][b] == want["token"][b], (b, res["token"][b], want["token"][b], want["margin"][b])
    return skipped


def _uniforms(g, n, B):
    # fp32 uniforms (what the kernel reads); the oracle gets the same fp32 values widened
    return g.random(n, dtype=np.float32), g.random(B, dtype=np.float32)


def _soft_q(g, logits, T, sharpen):
    """A drafter distribution correlated with the target's: softmax of (logits / T * sharpen + noise), fp32 rows."""
    z = logits.astype(np.float64) / T * sharpen + g.standard_normal(logits.shape)
    z -= z.max(axis=1, keepdims=True)
    e = np.exp(z)
    return (e / e.sum(axis=1, keepdims=True)).astype(np.float32)


@pytest.mark.parametrize("seed", range(8))
def test_sample_tiny_one_hot_drafter(wf, seed):
    """vocab 4096, gamma 7, deterministic drafter: drafts are the target's argmax for a planted prefix, then wrong."""
    binding, ctx = wf
    g = synth.rng(61, seed)
    q_lens = [8, 8, 1, 0, 8, 5]
    prefix = [int(x) for x in g.integers(0, 8, size=6)]
    spike = g.uniform(0.0, 8.0, size=6)
    logits, drafts, ip, _ = synth.make_logits_block(g, q_lens, 4096, 2.0, prefix, spike)
    rows = np.arange(len(logits))
    logits[rows, logits.argmax(axis=1)] += np.float32(3.0)      # winners hold a sizeable share: some drafts are accepted
    u_acc, u_s = _uniforms(g, len(logits), 6)
    T = [1.0, 0.7, 1.5, 1.0, 0.3, 2.0, 1.0, 1.0][seed]
    want = spec_sample.spec_sample_entropy_route(logits, drafts, ip, T, u_acc, u_s, 2.0)
    res = _run(binding, ctx, logits, drafts, ip, T, u_acc, u_s, 2.0, max_q=8)
    assert _check(res, want, 2.0) <= 1
    assert res["n_commit"][3] == 0 and res["accept_len"][3] == 0           # empty block


def test_sample_with_full_drafter_distributions(wf):
    """Full q rows correlated with p (drafts drawn from q): acceptance ratios p/q on both sides of 1, residual draws."""
    binding, ctx = wf
    g = synth.rng(63, 1)
    V, T = 4096, 0.8
    q_lens = [16, 8, 16, 8, 16, 1, 12]
    ip = np.zeros(len(q_lens) + 1, np.int32)
    ip[1:] = np.cumsum(q_lens)
    n = int(ip[-1])
    logits = synth.normal_f32(g, (n, V), 2.5)
    q = _soft_q(g, logits, T, 0.9)
    drafts = np.zeros(n, np.int32)
    for b in range(len(q_lens)):
        for j in range(1, q_lens[b]):
            r = int(ip[b]) + j
            drafts[r] = spec_sample.inverse_cdf(q[r - 1], g.random())      # x_j ~ q_{j-1} (input construction)
    u_acc, u_s = _uniforms(g, n, len(q_lens))
    tau = g.uniform(3.0, 7.0, size=len(q_lens)).astype(np.float32)
    want = spec_sample.spec_sample_entropy_route(logits, drafts, ip, T, u_acc, u_s, tau, draft_q=q)
    res = _run(binding, ctx, logits, drafts, ip, T, u_acc, u_s, tau, draft_q=q, max_q=16)
    assert _check(res, want, tau) <= 1
    assert want["accept_len"].max() >= 2 and (want["accept_len"] < np.array(q_lens) - 1).any()


def test_sample_8b_vocab_and_cache_length(wf):
    """vocab 151936 (19 slices, ragged last one; the draw's segments are 594 tokens wide), mixed gamma, an empty block,
    -inf logits (masked vocabulary) that must never be drawn; seq_len advances by n_commit."""
    import torch
    import gpu_harness as H
    binding, ctx = wf
    g = synth.rng(65, 1)
    V = 151936
    q_lens = [16, 8, 0, 16, 8, 1]
    prefix = [15, 2, 0, 0, 7, 0]
    logits, drafts, ip, _ = synth.make_logits_block(g, q_lens, V, 3.0, prefix, [0.0, 5.0, 0.0, 9.0, 2.0, 4.0])
    rows = np.arange(len(logits))
    logits[:, 1000:3000] = -np.inf                                           # a masked vocabulary range
    logits[rows, logits.argmax(axis=1)] += np.float32(6.0)
    u_acc, u_s = _uniforms(g, len(logits), 6)
    pair = H.make_kv_pair(ctx, [100, 200, 300, 400, 500, 600], q_lens, 1, 2, 64, seed=65, fill=False)
    want = spec_sample.spec_sample_entropy_route(logits, drafts, ip, 1.0, u_acc, u_s, 2.0, kv=pair.oracle)
    res = _run(binding, ctx, logits, drafts, ip, 1.0, u_acc, u_s, 2.0, max_q=16, kv=pair.gpu)
    assert _check(res, want, 2.0) <= 1
    assert not ((res["token"] >= 1000) & (res["token"] < 3000)).any()
    np.testing.assert_array_equal(pair.seq_len.cpu().numpy()[:6][want["accept_margin"] >= MARGIN],
                                  pair.oracle.seq_len[:6][want["accept_margin"] >= MARGIN])
    assert want["accept_len"].max() >= 3
    pair.close()


def test_sample_full_q_at_8b_vocab(wf):
    """Full drafter rows at the real vocabulary (V = 151936: 19 slices, ragged last one, two warp levels over 2 x 600 KB per
    sequence): drafts drawn from q, ratios p/q on both sides of 1, residual draws max(0, p - q), a masked range in both p
    and q, mixed gamma and an empty block."""
    binding, ctx = wf
    g = synth.rng(69, 1)
    V, T = 151936, 0.8
    q_lens = [16, 8, 0, 16, 4]
    ip = np.zeros(len(q_lens) + 1, np.int32)
    ip[1:] = np.cumsum(q_lens)
    n = int(ip[-1])
    logits = synth.normal_f32(g, (n, V), 3.0)
    rows = np.arange(n)
    logits[rows, logits.argmax(axis=1)] += np.float32(7.0)      # a winner with a real share of the mass: some drafts pass
    logits[:, 5000:9000] = -np.inf
    q = _soft_q(g, np.where(np.isfinite(logits), logits, -1e9), T, 0.9)
    drafts = np.zeros(n, np.int32)
    for b in range(len(q_lens)):
        for j in range(1, q_lens[b]):
            r = int(ip[b]) + j
            drafts[r] = spec_sample.inverse_cdf(q[r - 1], g.random())
    u_acc, u_s = _uniforms(g, n, len(q_lens))
    want = spec_sample.spec_sample_entropy_route(logits, drafts, ip, T, u_acc, u_s, 2.0, draft_q=q)
    res = _run(binding, ctx, logits, drafts, ip, T, u_acc, u_s, 2.0, draft_q=q, max_q=16)
    assert _check(res, want, 2.0) <= 1
    assert not ((res["token"] >= 5000) & (res["token"] < 9000)).any()
    assert want["accept_len"].max() >= 1 and (want["accept_len"] < np.maximum(np.array(q_lens) - 1, 0)).any()
    assert res["n_commit"][2] == 0


def test_sample_distribution_of_draws(wf):
    """1024 sequences share one logits row pattern (gamma = 0: pure bonus draws) with stratified uniforms: the
    histogram of emitted tokens must follow p (a wrong CDF order or a dropped segment shows up at once)."""
    binding, ctx = wf
    g = synth.rng(67, 1)
    V, B = 1000, 1024
    row = synth.normal_f32(g, (1, V), 2.0)
    logits = np.repeat(row, B, axis=0)
    ip = np.arange(B + 1, dtype=np.int32)
    u_s = ((np.arange(B) + 0.5) / B).astype(np.float32)
    u_acc = np.zeros(B, np.float32)
    res = _run(binding, ctx, logits, np.zeros(B, np.int32), ip, 1.0, u_acc, u_s, 2.0, max_q=1)
    want = spec_sample.spec_sample_entropy_route(logits, np.zeros(B, np.int32), ip, 1.0, u_acc, u_s, 2.0)
    ok = want["margin"] >= MARGIN
    np.testing.assert_array_equal(res["token"][ok], want["token"][ok])
    assert ok.mean() > 0.98
    assert (np.diff(res["token"]) >= 0).all()                  # the inverse CDF is monotone in u
    p = spec_sample.softmax_t(row[0], 1.0)
    top = int(p.argmax())
    assert abs((res["token"] == top).mean() - p[top]) < 2.0 / B + 1e-3


def test_sample_argument_errors(wf):
    import torch
    binding, ctx = wf
    z = torch.zeros((2, 64), dtype=torch.float32, device="cuda")
    i = torch.zeros(2, dtype=torch.int32, device="cuda")
    ip = torch.tensor([0, 2], dtype=torch.int32, device="cuda")
    f = torch.zeros(2, dtype=torch.float32, device="cuda")
    ws = torch.empty(binding.wf_accept_workspace_bytes(2, 64), dtype=torch.uint8, device="cuda")
    with pytest.raises(binding.WhiFlashError):
        binding.wf_accept_sample_entropy_route(ctx, z, 64, i, ip, 1, 2, 0.0, None, f, f, f, True, i, i, f, i, i, None, ws)
    with pytest.raises(binding.WhiFlashError):
        binding.wf_accept_sample_entropy_route(ctx, z, 64, i, ip, 1, 2, 1.0, None, None, f, f, True, i, i, f, i, i, None, ws)
