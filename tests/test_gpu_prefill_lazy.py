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
