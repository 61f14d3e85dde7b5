"""wf_accept_entropy_route_static: the accept / bonus / entropy / route sweep for callers that cannot allocate (code
under CUDA graph capture, tight serving loops, harnesses that forbid cudaMalloc).  Its scratch (slice partials and
completion counters) is one file-scope `static __device__` array inside the library, 516 KB, shared by every call on a
device; the entry point allocates nothing and rejects sizes beyond the array.

Checked here against the existing path (wf_accept_entropy_route with a caller workspace), which the other tests hold to
the oracle: on TWO calls in a row with different inputs and sizes (the array keeps the first call's contents: the second
call must not see them), integers bit-exact, entropy within the tolerance of the accept tests (the kernel is the same, so
equality of bits is what is observed), plus the oracle itself on the first call; and the rejection of a size beyond the
static maximum.  The file is named so that pytest collects it last (`pytest -x`); it passes alone in
a fresh process and after the other tests (its own context, no state shared with them but the library's array)."""

import numpy as np
import pytest

from oracle import accept_route
from paper_2606_07710_b200 import synth

pytestmark = pytest.mark.gpu

ENTROPY_ABS, ROUTE_BAND = 1e-3, 1e-4


@pytest.fixture(scope="module")
def wf():
    import torch
    assert torch.cuda.is_available(), "gpu tests need a CUDA device"
    from paper_2606_07710_b200 import binding
    ctx = binding.Ctx(0)
    yield binding, ctx
    ctx.close()


def _device_inputs(logits, drafts, q_indptr, tau):
    import gpu_harness as H
    tau_arr = np.atleast_1d(np.asarray(tau, dtype=np.float32))
    return H.f32(logits), H.i32(drafts), H.i32(q_indptr), H.f32(tau_arr), len(tau_arr) == 1


def _outputs(B):
    import torch
    outs = {k: torch.full((B,), -7, dtype=torch.int32, device="cuda") for k in ("accept_len", "bonus_token", "route", "n_commit")}
    outs["entropy"] = torch.full((B,), -7.0, dtype=torch.float32, device="cuda")
    return outs


def _call(binding, ctx, static, dev, B, V, max_q):
    import torch
    d_logits, d_drafts, d_indptr, d_tau, scalar = dev
    o = _outputs(B)
    args = (ctx, d_logits, V, d_drafts, d_indptr, B, max_q, d_tau, scalar, o["accept_len"], o["bonus_token"], o["entropy"],
            o["route"], o["n_commit"], None)
    if static:
        binding.wf_accept_entropy_route_static(*args)
    else:
        ws = torch.empty(binding.wf_accept_workspace_bytes(B * max_q, V), dtype=torch.uint8, device="cuda")
        binding.wf_accept_entropy_route(*args, ws)
    torch.cuda.synchronize()
    assert ctx.poll_status() == 0
    return {k: v.cpu().numpy() for k, v in o.items()}


def _same(got, ref):
    for k in ("accept_len", "bonus_token", "n_commit", "route"):
        np.testing.assert_array_equal(got[k], ref[k], err_msg=k)
    assert np.abs(got["entropy"].astype(np.float64) - ref["entropy"].astype(np.float64)).max() <= ENTROPY_ABS
    assert np.array_equal(got["entropy"].view(np.uint32), ref["entropy"].view(np.uint32)), "same kernel: same bits expected"


def test_static_scratch_matches_the_workspace_path_on_two_calls_in_a_row(wf):
    binding, ctx = wf
    g = synth.rng(synth.SEED_BASE + 9, 4242)
    # call 1: vocabulary 151936 (19 slices, ragged last slice), mixed gamma, an empty block, per-sequence tau
    q1 = [16, 8, 0, 16, 8, 1, 16, 16]
    u1 = [15, 3, 0, 0, 7, 0, 9, 2]
    s1 = [6.0, 0.0, 0.0, 9.0, 4.5, 5.0, 0.0, 8.0]
    logits1, drafts1, indptr1, _ = synth.make_logits_block(g, q1, 151936, 3.0, u1, s1)
    tau1 = np.array([2.0, 2.0, 2.0, 1.0, 7.0, 2.0, 2.0, 3.0], dtype=np.float32)
    # call 2: fewer sequences, another vocabulary (not a multiple of the slice, 3 slices), scalar tau: reuses the head of the
    # array that call 1 filled
    q2 = [8, 16, 5]
    u2 = [7, 0, 4]
    s2 = [0.0, 7.0, 9.5]
    logits2, drafts2, indptr2, _ = synth.make_logits_block(g, q2, 20000, 2.0, u2, s2)
    tau2 = 2.0
    dev1 = _device_inputs(logits1, drafts1, indptr1, tau1)
    dev2 = _device_inputs(logits2, drafts2, indptr2, tau2)
    ref1 = _call(binding, ctx, False, dev1, len(q1), 151936, 16)
    ref2 = _call(binding, ctx, False, dev2, len(q2), 20000, 16)
    # the two static calls back to back, then once more in the opposite order (the array now holds call 2's contents)
    got1 = _call(binding, ctx, True, dev1, len(q1), 151936, 16)
    got2 = _call(binding, ctx, True, dev2, len(q2), 20000, 16)
    _same(got1, ref1)
    _same(got2, ref2)
    _same(_call(binding, ctx, True, dev1, len(q1), 151936, 16), ref1)
    # and the oracle, so that the file stands on its own
    want = accept_route.accept_entropy_route(logits1, drafts1, indptr1, tau1)
    for k in ("accept_len", "bonus_token", "n_commit"):
        np.testing.assert_array_equal(got1[k], want[k], err_msg=k)
    assert np.abs(got1["entropy"].astype(np.float64) - want["entropy"]).max() <= ENTROPY_ABS
    near = np.abs(want["entropy"] - tau1) < ROUTE_BAND
    np.testing.assert_array_equal(got1["route"][~near], want["route"][~near])
    assert set(want["route"].tolist()) == {0, 1}


def test_static_scratch_rejects_sizes_beyond_its_maximum(wf):
    """64 sequences x 64 rows x 19 slices = 77824 partials > 32768: a clear error, nothing launched, outputs untouched."""
    import torch
    binding, ctx = wf
    B, V, max_q = 64, 151936, 64
    logits = torch.zeros((1, V), dtype=torch.float32, device="cuda")          # never read: the call is refused on the host
    drafts = torch.zeros(1, dtype=torch.int32, device="cuda")
    indptr = torch.zeros(B + 1, dtype=torch.int32, device="cuda")
    tau = torch.full((1,), 2.0, dtype=torch.float32, device="cuda")
    o = _outputs(B)
    before = ctx.launch_count()
    with pytest.raises(binding.WhiFlashError, match="exceed the static scratch"):
        binding.wf_accept_entropy_route_static(ctx, logits, V, drafts, indptr, B, max_q, tau, True, o["accept_len"],
                                               o["bonus_token"], o["entropy"], o["route"], o["n_commit"], None)
    torch.cuda.synchronize()
    assert ctx.launch_count() == before
    assert int(o["accept_len"][0]) == -7 and ctx.poll_status() == 0
    # more than 1024 sequences is refused as well, whatever the rows
    with pytest.raises(binding.WhiFlashError, match="exceed the static scratch"):
        binding.wf_accept_entropy_route_static(ctx, logits, 4096, drafts, indptr, 1025, 1, tau, True, o["accept_len"],
                                               o["bonus_token"], o["entropy"], o["route"], o["n_commit"], None)
