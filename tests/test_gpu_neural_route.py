"""GPU parity (through the C-ABI) for the WhiFlash-Neural routing policy against oracle O6.

Tolerance, derived from the arithmetic (N7): bf16 products are exact in fp32; W1 h is a 4096-term fp32
sum of terms of size ~|w||h| accumulated in a fixed order, error ~ sqrt(d) * 2^-24 * |z| ~ 1e-5 relative; erff is
good to a few ulp; the second layer adds 512 terms.  dAL is required within 1e-3 absolute of the fp64 oracle; the
route must be bit-exact except where |dAL - tau| < 1e-3 (counted, and planted to be rare).
"""

import numpy as np
import pytest

from oracle import neural_route
from paper_2606_07710_b200 import synth

pytestmark = pytest.mark.gpu

DAL_ABS = 1e-3
ROUTE_BAND = 1e-3


@pytest.fixture(scope="module")
def wf():
    import torch
    assert torch.cuda.is_available(), "gpu tests need a CUDA device"
    from paper_2606_07710_b200 import binding
    ctx = binding.Ctx(0)
    yield binding, ctx
    ctx.close()


def _case(wf, d, q_lens, seed, tau, use_accept=True, w_std=0.02):
    import torch
    import gpu_harness as H
    binding, ctx = wf
    g = synth.rng(seed, 31)
    m = d // 8
    B = len(q_lens)
    q_indptr = np.zeros(B + 1, dtype=np.int32)
    q_indptr[1:] = np.cumsum(q_lens)
    n = int(q_indptr[-1])
    hidden = synth.normal_bf16(g, (max(n, 1), d), 1.0)
    w1 = synth.normal_bf16(g, (m, d), w_std)
    b1 = synth.normal_f32(g, (m,), 0.1)
    w2 = synth.normal_bf16(g, (m,), 0.3)
    b2 = np.float32(-0.2)
    a = np.array([int(g.integers(0, q)) if q > 0 else 0 for q in q_lens], dtype=np.int32)
    tau_arr = np.broadcast_to(np.asarray(tau, dtype=np.float32), (B,)).copy() if np.ndim(tau) else np.float32(tau)
    want_dal, want_route = neural_route.neural_route(hidden, q_indptr, a if use_accept else np.zeros(B, np.int32),
                                                     w1, b1, w2, b2, tau_arr)
    dev = "cuda"
    t_h = H.bits_to_bf16_tensor(hidden)
    t_w1, t_w2 = H.bits_to_bf16_tensor(w1), H.bits_to_bf16_tensor(w2)
    t_b1, t_b2 = H.f32(b1), H.f32(np.array([b2], dtype=np.float32))
    t_tau = H.f32(np.atleast_1d(tau_arr).astype(np.float32))
    dal = torch.full((B,), 123.0, dtype=torch.float32, device=dev)
    route = torch.full((B,), -7, dtype=torch.int32, device=dev)
    ws = torch.empty(binding.wf_neural_route_workspace_bytes(B, m), dtype=torch.uint8, device=dev)
    for _ in range(2):                                    # twice: the completion counter must reset itself
        binding.wf_neural_route(ctx, t_h, H.i32(q_indptr), H.i32(a) if use_accept else None, B, d, m, t_w1, t_b1, t_w2, t_b2,
                                t_tau, np.ndim(tau) == 0, dal, route, ws)
        torch.cuda.synchronize()
    assert ctx.poll_status() == 0
    got_dal, got_route = dal.cpu().numpy().astype(np.float64), route.cpu().numpy()
    assert np.abs(got_dal - want_dal).max() <= DAL_ABS, (got_dal, want_dal)
    near = np.abs(want_dal - np.broadcast_to(np.asarray(tau_arr, dtype=np.float64), (B,))) < ROUTE_BAND
    assert np.array_equal(got_route[~near], want_route[~near]), (got_route, want_route)
    return int(near.sum()), want_dal, want_route


def test_neural_route_8b(wf):
    """d = 4096, m = 512 (the 2.10 M-parameter router of PAPER.md Table 5); batch 16 with mixed gamma 7/15 and an
    empty block; scalar tau so that both routes occur, then per-sequence thresholds planted around each value."""
    q_lens = [16, 8, 16, 0, 8, 16, 8, 16, 16, 8, 8, 16, 8, 16, 16, 8]
    near, dal, route = _case(wf, 4096, q_lens, seed=1, tau=0.0)
    assert near <= 1 and 0 < route.sum() < len(q_lens) - 1            # both drafters are chosen
    # per-sequence thresholds planted just below / above each value: strictness of '>' away from the band
    tau = dal.astype(np.float32) + np.where(np.arange(len(q_lens)) % 2 == 0, -0.01, 0.01).astype(np.float32)
    near, _, route = _case(wf, 4096, q_lens, seed=1, tau=tau)
    assert near == 0
    assert list(route) == [0 if q == 0 else (1 if i % 2 == 0 else 0) for i, q in enumerate(q_lens)]


def test_neural_route_batch_spanning_tiles_and_tiny(wf):
    """B = 70 (five staging tiles with a ragged tail), accept_len = NULL (row 0), and the tiny config (d = 256, m = 32:
    four CTAs), d = 2560 (Qwen3-4B: m = 320, not a multiple of the per-lane stride)."""
    g = synth.rng(5, 32)
    q_lens = [int(x) for x in g.choice([8, 16, 0], size=70, p=[0.45, 0.45, 0.1])]
    _case(wf, 4096, q_lens, seed=2, tau=0.1, use_accept=False)
    _case(wf, 256, [8], seed=3, tau=-0.3, w_std=0.05)
    _case(wf, 2560, [16, 8, 1, 16, 3], seed=4, tau=0.0)
