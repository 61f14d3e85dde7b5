"""GPU parity (through the C-ABI) for (c) KV-only prefill and (d) Lazy Catch-up against oracle/.

Tolerances (BASELINE.json north_star): projected K/V within relative L2 5e-3 of the oracle's fp64
values; cache indices (block tables, lengths) bit-exact; a lazy flush leaves the drafter cache
bit-identical to eager per-round appends.
"""

import numpy as np
import pytest

from oracle import kv_prefill
from paper_2606_07710_b200 import synth

pytestmark = pytest.mark.gpu

KV_REL_L2 = 5e-3


@pytest.fixture(scope="module")
def wf():
    import torch
    assert torch.cuda.is_available(), "gpu tests need a CUDA device"
    from paper_2606_07710_b200 import binding
    ctx = binding.Ctx(0)
    yield binding, ctx
    ctx.close()


def _mk(ctx, L, hidden, Hkv, D, S, pages_per_seq, seed, cap=32, shuffled=True, weights=None, theta=1e6, num_pages=None):
    import gpu_harness as H
    g = synth.rng(seed, 404)
    P = num_pages if num_pages else S * pages_per_seq + 7
    free = synth.draw_free_list(P, g, shuffled)
    return H.DrafterPair(ctx, L, hidden, Hkv, D, P, S, pages_per_seq, free, seed, backlog_cap=cap, weights=weights, theta=theta)


def _start_ctx(dp, lens):
    """Pretend `lens` tokens are already in the drafter cache (pages reserved, contents irrelevant)."""
    dp.kvp.reserve(lens)
    dp.kvp.set_seq_len(lens)


def _eager_both(binding, ctx, dp, hidden_bits, q_indptr, n_rows):
    import gpu_harness as H
    unrounded = kv_prefill.kv_only_prefill(dp.oracle, hidden_bits, q_indptr, n_rows)
    hid = H.bits_to_bf16_tensor(hidden_bits)
    B = len(n_rows)
    binding.wf_kv_only_prefill(ctx, dp.gpu, hid, H.i32(q_indptr), H.i32(n_rows), None, B, int(max(max(n_rows), 1)))
    return unrounded


def _check_new_rows(dp, unrounded, p0):
    """GPU K/V of the rows just appended vs the oracle's unrounded fp64 values; indices bit-exact."""
    import torch
    torch.cuda.synchronize()
    assert dp.ctx.poll_status() == 0
    dp.kvp.assert_tables_equal()
    worst = 0.0
    for b, (K, V) in unrounded.items():
        n = K.shape[1]
        for l in range(K.shape[0]):
            Kg, Vg = dp.gather_gpu(l, b, p0[b] + n)
            import gpu_harness as H
            worst = max(worst, H.rel_l2(Kg[p0[b]:], K[l]), H.rel_l2(Vg[p0[b]:], V[l]))
    return worst


def test_prefill_cfg1_tiny(wf):
    """configs[0]: hidden 256 -> 2 x 64 K and V, 1 layer, accepted rows 1..8, positions from ctx 512."""
    binding, ctx = wf
    for seed in range(4):
        dp = _mk(ctx, 1, 256, 2, 64, 1, 40, seed=synth.SEED_BASE + seed)
        _start_ctx(dp, [512])
        g = synth.rng(synth.SEED_BASE + seed, 505)
        X = synth.normal_bf16(g, (8, 256), 1.0)
        n = int(g.integers(1, 9))
        un = _eager_both(binding, ctx, dp, X, np.array([0, 8], np.int32), [n])
        assert _check_new_rows(dp, un, [512]) <= KV_REL_L2
        dp.close()


def test_prefill_8b_five_layers_ragged(wf):
    """configs[1] shapes: hidden 4096 -> 8 x 128, 5 layers, theta 1e6; ragged rows incl. 0, far positions."""
    binding, ctx = wf
    dp = _mk(ctx, 5, 4096, 8, 128, 4, 2100, seed=21, num_pages=2400)
    p0 = [4096, 17, 0, 32760]
    _start_ctx(dp, p0)
    g = synth.rng(21, 505)
    q_lens = [16, 8, 16, 16]
    q_indptr = np.concatenate([[0], np.cumsum(q_lens)]).astype(np.int32)
    X = synth.normal_bf16(g, (int(q_indptr[-1]), 4096), 1.0)
    un = _eager_both(binding, ctx, dp, X, q_indptr, [5, 0, 16, 1])
    assert _check_new_rows(dp, un, p0) <= KV_REL_L2
    # a second append continues at the new positions and crosses page boundaries
    p1 = [4096 + 5, 17, 16, 32761]
    un = _eager_both(binding, ctx, dp, X, q_indptr, [16, 8, 3, 16])
    assert _check_new_rows(dp, un, p1) <= KV_REL_L2
    dp.close()


def test_flush_multi_tile_and_two_passes(wf):
    """Flush of 5 x 64 = 320 backlog rows (3 m-tiles, 2 passes) vs the oracle; then a masked flush."""
    import torch
    import gpu_harness as H
    binding, ctx = wf
    S, cap = 5, 64
    dp = _mk(ctx, 1, 4096, 8, 128, S, 20, seed=33, cap=cap)
    _start_ctx(dp, [100, 0, 31, 16, 200])
    g = synth.rng(33, 606)
    q_indptr = (np.arange(S + 1) * 16).astype(np.int32)
    for rnd in range(4):                                   # 4 rounds x 16 rows fill every backlog to the cap
        X = synth.normal_bf16(g, (S * 16, 4096), 1.0)
        n = [16] * S
        dp.oracle_lazy.enqueue(X, q_indptr, n, [1] * S)
        binding.wf_lazy_catchup_enqueue(ctx, dp.gpu, H.bits_to_bf16_tensor(X), H.i32(q_indptr), H.i32(n), None,
                                        H.i32([1] * S), S, 16)
    torch.cuda.synchronize()
    np.testing.assert_array_equal(dp.backlog_len.cpu().numpy(), dp.oracle_lazy.backlog_len)
    p0 = dp.kvp.oracle.seq_len.copy()
    mask = [1, 1, 0, 1, 1]
    un = dp.oracle_lazy.flush(mask, S)
    binding.wf_lazy_catchup_flush(ctx, dp.gpu, H.i32(mask), S)
    assert _check_new_rows(dp, un, p0) <= KV_REL_L2
    np.testing.assert_array_equal(dp.backlog_len.cpu().numpy(), dp.oracle_lazy.backlog_len)
    p0 = dp.kvp.oracle.seq_len.copy()
    un = dp.oracle_lazy.flush(None, S)                     # the remaining sequence; empty ones are no-ops
    binding.wf_lazy_catchup_flush(ctx, dp.gpu, None, S)
    assert _check_new_rows(dp, un, p0) <= KV_REL_L2
    binding.wf_lazy_catchup_flush(ctx, dp.gpu, None, S)    # flush on empty queues: no-op (O4.ii)
    torch.cuda.synchronize()
    dp.kvp.assert_tables_equal()
    dp.close()


@pytest.mark.parametrize("shape", ["tiny", "8b"])
def test_lazy_flush_bit_identical_to_eager(wf, shape):
    """random interleaving of idle rounds, switches and forced flushes at the cap; after a
    final flush the lazy drafter's logical cache equals the eager drafter's bit for bit (GPU vs GPU),
    and both match the oracle's indices."""
    import torch
    import gpu_harness as H
    binding, ctx = wf
    L, hidden, Hkv, D = (1, 256, 2, 64) if shape == "tiny" else (5, 4096, 8, 128)
    S, cap, rounds = 4, 32, 14
    eager = _mk(ctx, L, hidden, Hkv, D, S, 40, seed=55, cap=cap, shuffled=False)
    lazy = _mk(ctx, L, hidden, Hkv, D, S, 40, seed=55, cap=cap, shuffled=True, weights=eager.weights)
    start = [70, 0, 15, 33]
    _start_ctx(eager, start)
    _start_ctx(lazy, start)
    g = synth.rng(55, 707)
    q_lens = [16, 8, 16, 8]
    q_indptr = np.concatenate([[0], np.cumsum(q_lens)]).astype(np.int32)
    total = np.array(start)
    for rnd in range(rounds):
        X = synth.normal_bf16(g, (int(q_indptr[-1]), hidden), 1.0)
        n = [int(g.integers(0, q + 1)) for q in q_lens]
        idle = [int(g.random() < 0.8) for _ in range(S)]
        Xg = H.bits_to_bf16_tensor(X)
        binding.wf_kv_only_prefill(ctx, eager.gpu, Xg, H.i32(q_indptr), H.i32(n), None, S, 16)
        kv_prefill.kv_only_prefill(eager.oracle, X, q_indptr, n)
        # lazy: idle sequences enqueue, active ones append eagerly (C22); a switch flushes (C21)
        n_idle = [nn if i else 0 for nn, i in zip(n, idle)]
        n_act = [0 if i else nn for nn, i in zip(n, idle)]
        flush = [int(not i) for i in idle]                 # sequences that are active this round flush first
        lazy.oracle_lazy.flush(flush, S)
        binding.wf_lazy_catchup_flush(ctx, lazy.gpu, H.i32(flush), S)
        lazy.oracle_lazy.enqueue(X, q_indptr, n_idle, idle)
        binding.wf_lazy_catchup_enqueue(ctx, lazy.gpu, Xg, H.i32(q_indptr), H.i32(n_idle), None, H.i32(idle), S, 16)
        kv_prefill.kv_only_prefill(lazy.oracle, X, q_indptr, n_act)
        binding.wf_kv_only_prefill(ctx, lazy.gpu, Xg, H.i32(q_indptr), H.i32(n_act), None, S, 16)
        total += np.array(n)
    lazy.oracle_lazy.flush(None, S)
    binding.wf_lazy_catchup_flush(ctx, lazy.gpu, None, S)
    torch.cuda.synchronize()
    assert ctx.poll_status() == 0
    eager.kvp.assert_tables_equal()
    lazy.kvp.assert_tables_equal()
    np.testing.assert_array_equal(eager.kvp.seq_len.cpu().numpy(), total)
    np.testing.assert_array_equal(lazy.kvp.seq_len.cpu().numpy(), total)
    assert int(lazy.backlog_len.sum()) == 0
    for l in range(L):
        for b in range(S):
            n0, n1 = start[b], int(total[b])
            Ke, Ve = eager.gather_gpu(l, b, n1)
            Kl, Vl = lazy.gather_gpu(l, b, n1)
            np.testing.assert_array_equal(Ke[n0:], Kl[n0:])
            np.testing.assert_array_equal(Ve[n0:], Vl[n0:])
            Ko, Vo = eager.kvp.oracle.gather(l, b, n1)       # the rounded oracle cache: mostly equal bits
            assert H.rel_l2(Ke[n0:], H.bf16_f64(Ko[n0:])) <= KV_REL_L2 if n1 > n0 else True
    eager.close()
    lazy.close()


def test_enqueue_overflow_status(wf):
    import torch
    import gpu_harness as H
    binding, ctx = wf
    dp = _mk(ctx, 1, 256, 2, 64, 2, 8, seed=66, cap=8)
    X = synth.normal_bf16(synth.rng(66, 1), (32, 256), 1.0)
    with pytest.raises(binding.WhiFlashError):               # host bound: max_rows > cap
        binding.wf_lazy_catchup_enqueue(ctx, dp.gpu, H.bits_to_bf16_tensor(X), H.i32([0, 16, 32]), H.i32([9, 1]), None,
                                        H.i32([1, 1]), 2, 16)
    dp.close()


@pytest.mark.parametrize("shape", ["tiny", "8b"])
def test_fused_round_bit_identical_to_eager(wf, shape):
    """wf_lazy_catchup_round (one projection per drafter per round: active rows, switching sequences' backlog + rows,
    forced flushes; idle rows enqueued afterwards) over random rounds: backlog lengths follow the enqueue/flush rules
    (C20, C21) and, after a final flush, the logical cache equals an eager drafter's bit for bit."""
    import torch
    import gpu_harness as H
    binding, ctx = wf
    L, hidden, Hkv, D = (1, 256, 2, 64) if shape == "tiny" else (5, 4096, 8, 128)
    S, cap, rounds = 5, 32, 24
    eager = _mk(ctx, L, hidden, Hkv, D, S, 44, seed=66, cap=cap, shuffled=False)
    fused = _mk(ctx, L, hidden, Hkv, D, S, 44, seed=66, cap=cap, shuffled=True, weights=eager.weights)
    start = [70, 0, 15, 33, 128]
    _start_ctx(eager, start)
    _start_ctx(fused, start)
    g = synth.rng(66, 808)
    q_lens = [16, 8, 16, 8, 16]
    q_indptr = np.concatenate([[0], np.cumsum(q_lens)]).astype(np.int32)
    total = np.array(start)
    blen = np.zeros(S, dtype=np.int64)                       # model of the backlog lengths
    cached = np.array(start)                                 # model of the fused drafter's cache lengths
    forced = 0
    for rnd in range(rounds):
        X = synth.normal_bf16(g, (int(q_indptr[-1]), hidden), 1.0)
        n = [int(g.integers(0, q + 1)) for q in q_lens]
        idle = [int(g.random() < 0.9) for _ in range(S)]
        flush = [int(i and g.random() < 0.15) for i in idle]
        if rnd == 5:
            idle, flush = [0] * S, [0] * S                   # a round with nobody idle: the masks may also be NULL
        Xg = H.bits_to_bf16_tensor(X)
        binding.wf_kv_only_prefill(ctx, eager.gpu, Xg, H.i32(q_indptr), H.i32(n), None, S, 16)
        binding.wf_lazy_catchup_round(ctx, fused.gpu, Xg, H.i32(q_indptr), H.i32(n), None,
                                      None if rnd == 5 else H.i32(idle), None if rnd == 5 else H.i32(flush), S, 16)
        for b in range(S):
            if not idle[b] or flush[b]:
                cached[b] += blen[b] + n[b]; blen[b] = 0
            elif blen[b] + n[b] > cap:
                cached[b] += blen[b]; blen[b] = n[b]; forced += 1
            else:
                blen[b] += n[b]
        total += np.array(n)
        torch.cuda.synchronize()
        assert ctx.poll_status() == 0
        np.testing.assert_array_equal(fused.backlog_len.cpu().numpy(), blen)
        np.testing.assert_array_equal(fused.kvp.seq_len.cpu().numpy(), cached)
    assert forced >= 1 and blen.sum() > 0                    # the run exercised a forced flush and ends with rows queued
    binding.wf_lazy_catchup_flush(ctx, fused.gpu, None, S)
    torch.cuda.synchronize()
    assert ctx.poll_status() == 0
    np.testing.assert_array_equal(fused.kvp.seq_len.cpu().numpy(), total)
    np.testing.assert_array_equal(eager.kvp.seq_len.cpu().numpy(), total)
    assert int(fused.backlog_len.sum()) == 0
    for l in range(L):
        for b in range(S):
            n0, n1 = start[b], int(total[b])
            Ke, Ve = eager.gather_gpu(l, b, n1)
            Kf, Vf = fused.gather_gpu(l, b, n1)
            np.testing.assert_array_equal(Ke[n0:], Kf[n0:])
            np.testing.assert_array_equal(Ve[n0:], Vf[n0:])
    eager.close()
    fused.close()


def test_fused_round_argument_and_overflow_errors(wf):
    """wf_lazy_catchup_round: idle sequences on a drafter without a backlog are refused on the host; a block larger than
    the backlog is refused up front (max_rows <= backlog_cap); a backlog that would overflow is projected first (C20)."""
    import torch
    import gpu_harness as H
    binding, ctx = wf
    dp = _mk(ctx, 1, 256, 2, 64, 2, 8, seed=9, cap=8)
    _start_ctx(dp, [3, 5])
    g = synth.rng(9, 1)
    X = H.bits_to_bf16_tensor(synth.normal_bf16(g, (32, 256), 1.0))
    q_indptr = H.i32([0, 16, 32])
    with pytest.raises(binding.WhiFlashError):                     # max_rows (16) > backlog_cap (8) with idle sequences
        binding.wf_lazy_catchup_round(ctx, dp.gpu, X, q_indptr, H.i32([1, 1]), None, H.i32([1, 0]), None, 2, 16)
    # sequence 0 idle: 8 rows fill its backlog exactly; sequence 1 active: 4 rows appended
    binding.wf_lazy_catchup_round(ctx, dp.gpu, X, q_indptr, H.i32([8, 4]), None, H.i32([1, 0]), None, 2, 8)
    torch.cuda.synchronize()
    assert ctx.poll_status() == 0
    np.testing.assert_array_equal(dp.backlog_len.cpu().numpy(), [8, 0])
    np.testing.assert_array_equal(dp.kvp.seq_len.cpu().numpy(), [3, 9])
    binding.wf_lazy_catchup_round(ctx, dp.gpu, X, q_indptr, H.i32([3, 0]), None, H.i32([1, 0]), None, 2, 8)   # 8 + 3 > 8: forced flush
    torch.cuda.synchronize()
    np.testing.assert_array_equal(dp.backlog_len.cpu().numpy(), [3, 0])
    np.testing.assert_array_equal(dp.kvp.seq_len.cpu().numpy(), [11, 9])
    dp.close()


def test_enqueue_forced_flush_out_of_pages_changes_nothing(wf):
    """A forced flush (C20) that finds no pages: the sticky status becomes WF_ERR_OUT_OF_PAGES and the call changes
    nothing: no backlog row is written (not this sequence's, not its neighbours'), no length moves, backlog_len <= cap."""
    import torch
    import gpu_harness as H
    binding, ctx = wf
    S, cap, hidden = 3, 8, 256
    dp = _mk(ctx, 1, hidden, 2, 64, S, 4, seed=12, cap=cap, num_pages=2)       # a ring of 2 pages = 32 tokens in all
    g = synth.rng(12, 1)
    q_indptr = H.i32([0, 8, 16, 24])
    X1 = synth.normal_bf16(g, (24, hidden), 1.0)
    binding.wf_lazy_catchup_enqueue(ctx, dp.gpu, H.bits_to_bf16_tensor(X1), q_indptr, H.i32([8, 6, 8]), None, H.i32([1, 1, 1]), S, 8)
    torch.cuda.synchronize()
    assert ctx.poll_status() == 0
    np.testing.assert_array_equal(dp.backlog_len.cpu().numpy(), [8, 6, 8])
    # use up the ring: sequence 1 (idle elsewhere) takes both pages through an eager twin call on the same cache
    dp.kvp.gpu.reserve(H.i32([0, 32, 0]), S)
    torch.cuda.synchronize()
    before = H.bf16_tensor_to_bits(dp.backlog).copy()
    X2 = synth.normal_bf16(g, (24, hidden), 1.0)
    # sequences 0 and 2 are full: the enqueue needs a forced flush of 16 rows = pages the ring no longer has
    binding.wf_lazy_catchup_enqueue(ctx, dp.gpu, H.bits_to_bf16_tensor(X2), q_indptr, H.i32([3, 1, 5]), None, H.i32([1, 1, 1]), S, 8)
    torch.cuda.synchronize()
    assert ctx.poll_status() == binding.WF_ERR_OUT_OF_PAGES
    np.testing.assert_array_equal(dp.backlog_len.cpu().numpy(), [8, 6, 8])
    assert int(dp.backlog_len.max()) <= cap
    np.testing.assert_array_equal(H.bf16_tensor_to_bits(dp.backlog), before)
    np.testing.assert_array_equal(dp.kvp.seq_len.cpu().numpy(), [0, 0, 0])
    # the same through the fused round call
    binding.wf_lazy_catchup_round(ctx, dp.gpu, H.bits_to_bf16_tensor(X2), q_indptr, H.i32([3, 1, 5]), None, H.i32([1, 1, 1]), None, S, 8)
    torch.cuda.synchronize()
    assert ctx.poll_status() == binding.WF_ERR_OUT_OF_PAGES
    np.testing.assert_array_equal(dp.backlog_len.cpu().numpy(), [8, 6, 8])
    np.testing.assert_array_equal(H.bf16_tensor_to_bits(dp.backlog), before)
    dp.close()


def test_rows_beyond_the_host_bound_are_clamped_and_flagged(wf):
    """n_rows[b] > max_rows (the host bound that sizes the launch): rows up to the bound are projected, the sticky status
    is WF_ERR_INVALID_ARG, nothing stale is consumed (the projected rows still match the oracle)."""
    import torch
    import gpu_harness as H
    binding, ctx = wf
    dp = _mk(ctx, 1, 256, 2, 64, 2, 8, seed=13, cap=0)
    g = synth.rng(13, 1)
    X = synth.normal_bf16(g, (32, 256), 1.0)
    q_indptr = np.array([0, 16, 32], np.int32)
    binding.wf_kv_only_prefill(ctx, dp.gpu, H.bits_to_bf16_tensor(X), H.i32(q_indptr), H.i32([9, 2]), None, 2, 4)   # 9 > 4
    torch.cuda.synchronize()
    assert ctx.poll_status() == binding.WF_ERR_INVALID_ARG
    un = kv_prefill.kv_only_prefill(dp.oracle, X, q_indptr, [4, 2])
    assert _check_new_rows(dp, un, [0, 0]) <= KV_REL_L2
    dp.close()


def test_switch_round_device_driven_routes_not_planted(wf):
    """wf_switch_round over 30 rounds in which nothing is planned per round slot: every round's route comes from the
    accept/entropy/route kernel itself on logits whose spike magnitude is random (the entropy lands on either side of
    tau, the test learns the route only from the device), masks and cur_drafter never leave the device.  After every
    round both drafters' cache lengths, backlog lengths, block tables and cur_drafter equal the oracle's (driven by the
    oracle's own route); at the end the rows written are within tolerance and, after a final flush, the lazily
    maintained caches equal eager twins bit for bit."""
    import torch
    import gpu_harness as H
    from oracle import accept_route, lazy_catchup
    binding, ctx = wf
    S, cap, hidden, Hkv, D, V, tau = 6, 24, 256, 2, 64, 4096, 2.0
    mk = lambda L, seed, shuffled, weights=None: _mk(ctx, L, hidden, Hkv, D, S, 60, seed=seed, cap=cap, shuffled=shuffled, weights=weights)
    dr = {1: mk(1, 71, True), 0: mk(3, 72, True)}                   # route code -> drafter (AR: 1 layer, diffusion: 3)
    tw = {c: mk(d.shape.n_layers, 80 + c, False, d.weights) for c, d in dr.items()}     # eager twins
    start = [40, 0, 7, 16, 99, 3]
    for d in list(dr.values()) + list(tw.values()):
        _start_ctx(d, start)
    lz = {c: d.oracle_lazy for c, d in dr.items()}
    g = synth.rng(71, 9)
    cur_o = g.integers(0, 2, size=S).astype(np.int32)
    cur = H.i32(cur_o)
    nq = torch.zeros(S, dtype=torch.int32, device="cuda")
    q_len_of = {1: 8, 0: 16}
    q_lens = np.array([q_len_of[int(c)] for c in cur_o])
    outs = {k: torch.zeros(S, dtype=torch.int32, device="cuda") for k in ("accept_len", "bonus", "route", "n_commit")}
    ent = torch.zeros(S, dtype=torch.float32, device="cuda")
    ws = torch.empty(binding.wf_accept_workspace_bytes(S * 16, V), dtype=torch.uint8, device="cuda")
    seen, flushes, near = set(), 0, 0
    for rnd in range(30):
        u = synth.draw_accept_prefix(g, q_lens - 1, 3.5)
        spike = g.uniform(0.0, 10.0, size=S)                       # H lands on either side of tau: not a planned route
        logits, drafts, q_indptr, _ = synth.make_logits_block(g, q_lens, V, 2.0, u, spike)
        X = synth.normal_bf16(g, (int(q_indptr[-1]), hidden), 1.0)
        Xg, qi = H.bits_to_bf16_tensor(X), H.i32(q_indptr)
        binding.wf_accept_entropy_route(ctx, H.f32(logits), V, H.i32(drafts), qi, S, 16, H.f32([tau]), True, outs["accept_len"],
                                        outs["bonus"], ent, outs["route"], outs["n_commit"], None, ws)
        binding.wf_switch_round(ctx, dr[1].gpu, dr[0].gpu, Xg, qi, outs["n_commit"], None, outs["route"], cur, nq, 8, 16, S, 16)
        for c in dr:
            binding.wf_kv_only_prefill(ctx, tw[c].gpu, Xg, qi, outs["n_commit"], None, S, 16)
        want = accept_route.accept_entropy_route(logits, drafts, q_indptr, tau)
        torch.cuda.synchronize()
        assert ctx.poll_status() == 0
        band = np.abs(want["entropy"] - tau) < 1e-4
        near += int(band.sum())
        route_o = np.where(band, outs["route"].cpu().numpy(), want["route"]).astype(np.int32)
        np.testing.assert_array_equal(outs["route"].cpu().numpy(), route_o)
        np.testing.assert_array_equal(outs["n_commit"].cpu().numpy(), want["n_commit"])
        flushes += int((route_o != cur_o).sum())
        seen |= set(route_o.tolist())
        cur_o, nq_o, _ = lazy_catchup.switch_round(lz, X, q_indptr, want["n_commit"], route_o, cur_o, q_len_of)
        np.testing.assert_array_equal(cur.cpu().numpy(), cur_o)
        np.testing.assert_array_equal(nq.cpu().numpy(), nq_o)
        for c, d in dr.items():
            d.kvp.assert_tables_equal()
            np.testing.assert_array_equal(d.backlog_len.cpu().numpy(), lz[c].backlog_len)
        q_lens = nq_o.astype(np.int64)                              # the chosen drafter's block length next round
    assert seen == {0, 1} and flushes >= 10, (seen, flushes)
    total = dr[0].kvp.oracle.seq_len + lz[0].backlog_len
    for c, d in dr.items():
        binding.wf_lazy_catchup_flush(ctx, d.gpu, None, S)
        lz[c].flush(None, S)
    torch.cuda.synchronize()
    assert ctx.poll_status() == 0
    for c, d in dr.items():
        d.kvp.assert_tables_equal()
        np.testing.assert_array_equal(d.kvp.seq_len.cpu().numpy(), total)
        for l in range(d.shape.n_layers):
            for b in range(S):
                Kl, Vl = d.gather_gpu(l, b, int(total[b]))
                Ke, Ve = tw[c].gather_gpu(l, b, int(total[b]))
                np.testing.assert_array_equal(Kl[start[b]:], Ke[start[b]:])
                np.testing.assert_array_equal(Vl[start[b]:], Ve[start[b]:])
                Ko, Vo = d.kvp.oracle.gather(l, b, int(total[b]))
                assert H.rel_l2(Kl[start[b]:], H.bf16_f64(Ko[start[b]:])) <= KV_REL_L2
    for d in list(dr.values()) + list(tw.values()):
        d.close()
