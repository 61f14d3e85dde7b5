"""Pins for oracle O3 (KV-only prefill), O4 (lazy catch-up), O5 (full prefill) and the
paged block table D1, CPU only.  PAPER.md:117-119, :204; readings C13-C24.
"""

import math

import numpy as np
import pytest

from oracle import bf16, kv_prefill, lazy_catchup
from oracle.paged_kv import OutOfPages, PagedKV
from paper_2606_07710_b200 import synth


def _drafter(L=2, hidden=32, Hkv=2, D=8, page=4, num_pages=64, max_seqs=3, theta=1e6, seed=0,
             shuffled=True, w_std=0.2):
    g = synth.rng(seed, 7)
    free = synth.draw_free_list(num_pages, g, shuffled)
    kv = PagedKV(L, Hkv, D, page, num_pages, max_seqs, num_pages // max_seqs, free)
    wk = [synth.normal_bf16(g, (hidden, Hkv * D), w_std) for _ in range(L)]
    wv = [synth.normal_bf16(g, (hidden, Hkv * D), w_std) for _ in range(L)]
    return kv_prefill.Drafter(wk, wv, kv, theta)


def _logical(kv):
    return [[kv.gather(l, b) for b in range(kv.max_seqs)] for l in range(kv.L)]


def _same_cache(a, b):
    assert np.array_equal(a.seq_len, b.seq_len)
    for l in range(a.L):
        for s in range(a.max_seqs):
            Ka, Va = a.gather(l, s)
            Kb, Vb = b.gather(l, s)
            assert np.array_equal(Ka, Kb) and np.array_equal(Va, Vb)


# ------------------------------------------------------------------ bf16 + RoPE
def test_bf16_rounding_matches_torch_and_is_rne():
    import torch
    g = synth.rng(1, 1)
    x = synth.normal_f32(g, 200000, 1.0)
    ref = torch.from_numpy(x).to(torch.bfloat16).view(torch.int16).numpy().view(np.uint16)
    assert np.array_equal(bf16.from_f64(x.astype(np.float64)), ref)
    # exact halfway cases round to even: 1 + 2^-8 -> 1.0 ; 1 + 3*2^-8 -> 1 + 2^-6
    assert bf16.from_f64(np.array([1.0 + 2.0 ** -8]))[0] == 0x3F80
    assert bf16.from_f64(np.array([1.0 + 3 * 2.0 ** -8]))[0] == 0x3F82
    # a value that double rounding (fp64 -> fp32 -> bf16) gets wrong: just above halfway
    v = 1.0 + 2.0 ** -8 + 2.0 ** -40
    assert bf16.from_f64(np.array([v]))[0] == 0x3F81
    assert np.array_equal(bf16.to_f64(np.array([0x3F80, 0xC000], np.uint16)), [1.0, -2.0])


def test_rope_properties():
    """(ii) position 0 is the identity; (iii) pair norms are preserved; (iv) <RoPE(x,m),RoPE(y,n)>
    depends only on m-n; plus the explicit pairing (r, r+D/2) and angle pos*theta^(-2r/D)."""
    g = synth.rng(2, 1)
    D = 16
    x, y = g.standard_normal(D), g.standard_normal(D)
    assert np.array_equal(kv_prefill.rope_rotate_half(x, 0, 1e6), x)
    rx = kv_prefill.rope_rotate_half(x, 12345, 1e6)
    h = D // 2
    np.testing.assert_allclose(rx[:h] ** 2 + rx[h:] ** 2, x[:h] ** 2 + x[h:] ** 2, rtol=1e-12)
    d1 = kv_prefill.rope_rotate_half(x, 1000, 1e4) @ kv_prefill.rope_rotate_half(y, 990, 1e4)
    d2 = kv_prefill.rope_rotate_half(x, 40, 1e4) @ kv_prefill.rope_rotate_half(y, 30, 1e4)
    assert abs(d1 - d2) < 1e-9
    # explicit formula for one pair
    r, pos, theta = 3, 77, 1e6
    phi = pos * theta ** (-2.0 * r / D)
    out = kv_prefill.rope_rotate_half(x, pos, theta)
    assert abs(out[r] - (x[r] * math.cos(phi) - x[r + h] * math.sin(phi))) < 1e-14
    assert abs(out[r + h] - (x[r + h] * math.cos(phi) + x[r] * math.sin(phi))) < 1e-14


# ------------------------------------------------------------------ O3 pins
def test_o3_bruteforce_projection():
    """Pure-Python K = RoPE(x W_K), V = x W_V for a tiny drafter; checks orientation (C18),
    head/lane split, position offset p0 = cache length, and RNE stores."""
    dr = _drafter(L=2, hidden=6, Hkv=2, D=4, page=4, num_pages=12, max_seqs=2, seed=3)
    g = synth.rng(3, 1)
    X = synth.normal_bf16(g, (5, 6), 1.0)
    dr.kv.reserve([3, 0])
    dr.kv.seq_len[0] = 3                       # three tokens already cached -> p0 = 3
    ip = np.array([0, 3, 5], np.int32)
    kv_prefill.kv_only_prefill(dr, X, ip, [2, 2])
    xf = bf16.to_f64(X)
    for l in range(2):
        wk, wv = bf16.to_f64(dr.w_k[l]), bf16.to_f64(dr.w_v[l])
        for b, (r0, p0) in enumerate(((0, 3), (3, 0))):
            Kc, Vc = dr.kv.gather(l, b)
            for t in range(2):
                for hd in range(2):
                    k = [sum(xf[r0 + t, i] * wk[i, hd * 4 + c] for i in range(6)) for c in range(4)]
                    v = [sum(xf[r0 + t, i] * wv[i, hd * 4 + c] for i in range(6)) for c in range(4)]
                    rot = list(k)
                    for r in range(2):
                        phi = (p0 + t) * 1e6 ** (-2.0 * r / 4)
                        rot[r] = k[r] * math.cos(phi) - k[r + 2] * math.sin(phi)
                        rot[r + 2] = k[r + 2] * math.cos(phi) + k[r] * math.sin(phi)
                    np.testing.assert_allclose(bf16.to_f64(Kc[p0 + t, hd]), rot, rtol=2.0 ** -8)
                    np.testing.assert_allclose(bf16.to_f64(Vc[p0 + t, hd]), v, rtol=2.0 ** -8)
                    assert np.array_equal(Kc[p0 + t, hd], bf16.from_f64(np.array(rot)))
    assert list(dr.kv.seq_len[:2]) == [5, 2]


def test_o3_identity_weights_zero_input_linearity():
    """(v) W = identity slice -> K = RoPE(X); (vi) X = 0 -> zeros; (vii) linear in X before rounding."""
    hidden, Hkv, D = 16, 2, 8
    dr = _drafter(L=1, hidden=hidden, Hkv=Hkv, D=D, seed=4)
    eye = synth.f32_to_bf16_bits(np.eye(hidden, dtype=np.float32))
    dr.w_k[0] = eye
    dr.w_v[0] = eye
    g = synth.rng(4, 1)
    X = synth.normal_bf16(g, (3, hidden), 1.0)
    K, V = kv_prefill.project_rows(dr, X, 10)
    xf = bf16.to_f64(X).reshape(3, Hkv, D)
    for t in range(3):
        np.testing.assert_allclose(K[0, t], kv_prefill.rope_rotate_half(xf[t], 10 + t, dr.theta), atol=1e-15)
    assert np.array_equal(V[0], xf)
    K0, V0 = kv_prefill.project_rows(dr, np.zeros((2, hidden), np.uint16), 5)
    assert not K0.any() and not V0.any()
    dr2 = _drafter(L=1, hidden=hidden, Hkv=Hkv, D=D, seed=5)
    A, Bm = synth.normal_bf16(g, (1, hidden), 1.0), synth.normal_bf16(g, (1, hidden), 1.0)
    S = bf16.from_f64(2.0 * bf16.to_f64(A))           # 2A is exact in bf16
    KA, VA = kv_prefill.project_rows(dr2, A, 9)
    KS, VS = kv_prefill.project_rows(dr2, S, 9)
    np.testing.assert_allclose(KS, 2 * KA, rtol=1e-13)
    np.testing.assert_allclose(VS, 2 * VA, rtol=1e-13)


def test_o3_one_at_a_time_equals_batch():
    """(viii) n rows appended one by one == n rows at once, bit-exact."""
    a, b = _drafter(seed=6), _drafter(seed=6)
    g = synth.rng(6, 1)
    X = synth.normal_bf16(g, (7, 32), 1.0)
    ip = np.array([0, 4, 4, 7], np.int32)
    kv_prefill.kv_only_prefill(a, X, ip, [4, 0, 3])
    for t in range(4):
        n = [1, 0, 1 if t < 3 else 0]
        ipt = np.array([t, t + 1, t + 1, 0], np.int32)
        rows = [X[t:t + 1], X[0:0], X[4 + t:5 + t] if t < 3 else X[0:0]]
        kv_prefill.append_rows(b, rows)
    _same_cache(a.kv, b.kv)


def test_o3_equals_full_drafter_prefill_cache():
    """(i) BASELINE invariant: KV-only prefill yields the same K/V cache as a full drafter
    prefill (Q proj, attention, O proj, MLP, LM head run and discarded), bit for bit."""
    a, b = _drafter(L=2, hidden=32, Hkv=2, D=8, seed=7), _drafter(L=2, hidden=32, Hkv=2, D=8, seed=7)
    g = synth.rng(7, 1)
    Hq = 4
    extra = dict(
        w_q=[g.standard_normal((32, Hq * 8)) * 0.2 for _ in range(2)],
        w_o=[g.standard_normal((Hq * 8, 32)) * 0.2 for _ in range(2)],
        w_up=[g.standard_normal((32, 48)) * 0.2 for _ in range(2)],
        w_down=[g.standard_normal((48, 32)) * 0.2 for _ in range(2)],
        lm_head=g.standard_normal((32, 50)) * 0.2,
    )
    X = synth.normal_bf16(g, (9, 32), 1.0)
    ip = np.array([0, 5, 9, 9], np.int32)
    for rnd in range(2):                                   # two rounds: second one has p0 > 0
        kv_prefill.kv_only_prefill(a, X, ip, [3, 4, 0])
        out = kv_prefill.full_drafter_prefill(b, extra, X, ip, [3, 4, 0], Hq)
        assert len(out) == 7 and all(np.isfinite(o).all() for o in out)
    _same_cache(a.kv, b.kv)
    assert np.array_equal(a.kv.block_table, b.kv.block_table)


# ------------------------------------------------------------------ O4 pins
def test_o4_flush_equals_eager_random_interleavings():
    """(i) flush == eager bit-identical logical cache and lengths; (iii) backlog_len = sum of
    n_commit while idle; (iv) forced flush at the cap keeps order and drops nothing;
    (v) >= 1000 seeded rounds of random enqueue / flush / switch."""
    g = synth.rng(8, 1)
    hidden, S, cap = 16, 3, 10
    eager = _drafter(L=2, hidden=hidden, Hkv=1, D=8, page=4, num_pages=3 * 1200, max_seqs=S, seed=8)
    lazy_d = _drafter(L=2, hidden=hidden, Hkv=1, D=8, page=4, num_pages=3 * 1200, max_seqs=S, seed=8)
    lazy = lazy_catchup.LazyCatchup(lazy_d, cap)
    expected_backlog = np.zeros(S, np.int64)
    forced = 0
    for rnd in range(1000):
        q_lens = g.integers(1, 5, size=S)
        ip = np.zeros(S + 1, np.int32)
        ip[1:] = np.cumsum(q_lens)
        X = synth.normal_bf16(g, (int(ip[-1]), hidden), 1.0)
        n_rows = np.array([g.integers(0, ql + 1) for ql in q_lens])
        kv_prefill.kv_only_prefill(eager, X, ip, n_rows)                 # reference = eager, every round
        idle = np.ones(S, dtype=bool)
        before = lazy.backlog_len.copy()
        lazy.enqueue(X, ip, n_rows, idle)
        for b in range(S):
            if before[b] + n_rows[b] > cap:
                forced += 1
                expected_backlog[b] = n_rows[b]
            else:
                expected_backlog[b] += n_rows[b]
        assert np.array_equal(lazy.backlog_len, expected_backlog)
        switch = g.random(S) < 0.3
        if switch.any():
            lazy.flush(switch, S)
            expected_backlog[switch] = 0
        for b in range(S):                                              # invariant at every round
            assert lazy_d.kv.seq_len[b] + lazy.backlog_len[b] == eager.kv.seq_len[b]
    assert forced > 10
    lazy.flush(None, S)
    assert not lazy.backlog_len.any()
    _same_cache(eager.kv, lazy_d.kv)


def test_o4_empty_flush_is_noop_and_idle_mask():
    dr = _drafter(seed=9)
    lazy = lazy_catchup.LazyCatchup(dr, 8)
    before = (dr.kv.k_pool.copy(), dr.kv.block_table.copy(), dr.kv.free_count)
    lazy.flush(None, 3)
    assert np.array_equal(before[0], dr.kv.k_pool) and np.array_equal(before[1], dr.kv.block_table)
    assert before[2] == dr.kv.free_count and not dr.kv.seq_len.any()
    g = synth.rng(9, 1)
    X = synth.normal_bf16(g, (6, 32), 1.0)
    ip = np.array([0, 2, 4, 6], np.int32)
    lazy.enqueue(X, ip, [2, 2, 1], [True, False, True])
    assert list(lazy.backlog_len) == [2, 0, 1]
    assert np.array_equal(lazy.backlog[2, 0], X[4])


# ------------------------------------------------------------------ D1 pins
def test_paged_kv_allocation_order_and_release():
    """C24: ascending sequences take consecutive free-list entries; release appends to the tail;
    a failed reserve allocates nothing."""
    free = np.array([5, 2, 7, 0, 1, 3, 6, 4], np.int32)
    kv = PagedKV(1, 1, 4, 4, 8, 3, 4, free)
    kv.reserve([5, 0, 4])                      # seq0: 2 pages, seq2: 1 page
    assert list(kv.block_table[0, :2]) == [5, 2] and kv.block_table[2, 0] == 7 and kv.free_count == 5
    kv.seq_len[:] = [5, 0, 4]
    kv.reserve([3, 1, 0])                      # seq0 holds 8 slots already -> 0 new; seq1: 1 page
    assert kv.pages_held[0] == 2 and kv.block_table[1, 0] == 0
    kv.seq_len[1] = 1
    with pytest.raises(OutOfPages):
        kv.reserve([0, 100, 0])
    assert kv.free_count == 4 and kv.pages_held[1] == 1
    kv.release_seq(0)
    assert kv.free_count == 6 and kv.seq_len[0] == 0
    kv.reserve([0, 15, 0])                     # 16 tokens = 4 pages, holds 1 -> takes 1,3,6
    assert list(kv.block_table[1, :4]) == [0, 1, 3, 6]
    kv.seq_len[1] = 16
    kv.reserve([12, 0, 0])
    assert list(kv.block_table[0, :3]) == [4, 5, 2]
    assert kv.locate(0, 9) == (2, 1)


# ------------------------------------------------------------------ the switch (reading C21)
def test_switch_masks_truth_table():
    """the inactive drafter gets no work until the router switches to it.  All four (cur, route) cases,
    for both route codes; exactly one drafter is active per sequence and at most one is flushed."""
    cur = np.array([0, 0, 1, 1])
    route = np.array([0, 1, 0, 1])
    idle_d, fl_d = lazy_catchup.switch_masks(route, cur, 0)        # the diffusion drafter (code 0)
    idle_a, fl_a = lazy_catchup.switch_masks(route, cur, 1)        # the autoregressive drafter (code 1)
    assert idle_d.tolist() == [0, 0, 1, 1] and fl_d.tolist() == [0, 0, 1, 0]
    assert idle_a.tolist() == [1, 1, 0, 0] and fl_a.tolist() == [0, 1, 0, 0]
    assert ((1 - idle_d) + (1 - idle_a)).tolist() == [1, 1, 1, 1]
    assert (fl_d + fl_a).tolist() == [0, 1, 1, 0]                  # a flush exactly where route != cur


def test_o4_round_equals_separate_calls_and_eager():
    """LazyCatchup.round (one batched prefill per round) leaves the logical cache, the cache length and the backlog
    identical to the three separate calls it stands for (kv_only_prefill for the active sequences, enqueue, flush), and
    after a final flush identical to eager appends: 300 random rounds with a route that follows a random walk, cap 8
    (forced flushes happen), rows 0..5 per round."""
    g = synth.rng(21, 3)
    S, cap, hidden = 3, 8, 32
    fused = lazy_catchup.LazyCatchup(_drafter(seed=5, max_seqs=S, num_pages=1200), cap)
    sep = lazy_catchup.LazyCatchup(_drafter(seed=5, max_seqs=S, num_pages=1200), cap)
    eager = _drafter(seed=5, max_seqs=S, num_pages=1200)
    code = 1
    cur = g.integers(0, 2, size=S)
    q_indptr = (np.arange(S + 1) * 6).astype(np.int32)
    forced = 0
    for rnd in range(300):
        X = synth.normal_bf16(g, (S * 6, hidden), 1.0)
        n = g.integers(0, 6, size=S)
        route = np.where(g.random(S) < 0.3, 1 - cur, cur)
        idle, fl = lazy_catchup.switch_masks(route, cur, code)
        forced += int(((sep.backlog_len[:S] + n > cap) & (idle == 1) & (fl == 0)).sum())
        fused.round(X, q_indptr, n, idle, fl)
        kv_prefill.kv_only_prefill(sep.drafter, X, q_indptr, n * (1 - idle))
        sep.enqueue(X, q_indptr, n, idle)
        sep.flush(fl, S)
        kv_prefill.kv_only_prefill(eager, X, q_indptr, n)
        _same_cache(fused.drafter.kv, sep.drafter.kv)
        assert np.array_equal(fused.backlog_len, sep.backlog_len)
        for b in range(S):
            assert np.array_equal(fused.backlog[b, :fused.backlog_len[b]], sep.backlog[b, :sep.backlog_len[b]])
        cur = route
    assert forced > 5, "the run must exercise forced flushes"
    fused.flush(None, S)
    _same_cache(fused.drafter.kv, eager.kv)


def test_switch_round_drives_both_drafters():
    """switch_round: per round exactly the active drafter's cache grows by n_rows, the other one's backlog does (or it
    is flushed on a switch); cur' = route; the next block length follows the route."""
    g = synth.rng(22, 3)
    S, cap = 3, 16
    lz = {0: lazy_catchup.LazyCatchup(_drafter(seed=6, L=2, max_seqs=S, num_pages=600), cap),
          1: lazy_catchup.LazyCatchup(_drafter(seed=7, L=1, max_seqs=S, num_pages=600), cap)}
    cur = np.array([0, 1, 0])
    q_indptr = (np.arange(S + 1) * 4).astype(np.int32)
    total = np.zeros(S, dtype=np.int64)
    for rnd in range(40):
        X = synth.normal_bf16(g, (S * 4, 32), 1.0)
        n = g.integers(1, 5, size=S)
        route = g.integers(0, 2, size=S)
        before = {c: (l.drafter.kv.seq_len.copy(), l.backlog_len.copy()) for c, l in lz.items()}
        cur2, nq, _ = lazy_catchup.switch_round(lz, X, q_indptr, n, route, cur, {0: 16, 1: 8})
        total += n
        for b in range(S):
            act, oth = int(cur[b]), 1 - int(cur[b])
            assert lz[act].drafter.kv.seq_len[b] == before[act][0][b] + n[b] and lz[act].backlog_len[b] == 0
            if route[b] != cur[b]:                                  # the other drafter catches up completely
                assert lz[oth].backlog_len[b] == 0 and lz[oth].drafter.kv.seq_len[b] == total[b]
            else:
                assert lz[oth].drafter.kv.seq_len[b] + lz[oth].backlog_len[b] == total[b]
        assert np.array_equal(cur2, route) and nq.tolist() == [16 if r == 0 else 8 for r in route]
        cur = cur2
