"""Whole rounds at each BASELINE.json config's OWN parameters, through paper_2606_07710_b200.rounds (reserve ->
verify attention -> accept/entropy/route -> wf_switch_round -> wf_final_token_full), against the oracle driven by the ORACLE's
own route.

north_star: "all five configs match the CPU oracle within the stated tolerances".  configs[0] (tiny) is covered by
test_gpu_attn_accept.py / test_gpu_prefill_lazy.py (64 seeds) and smoke(); here are configs[1..4]:
  cfg2  B = 1, ctx 4096, gamma 15, 5-layer + 1-layer drafters
  cfg3  B = 16, ctx 8192, gamma 7 / 15 by route, backlog cap 32
  cfg4  B = 4, ctx 32768, gamma 15, cap 64; plus configs[3] verbatim: a 64-row backlog per sequence built over idle
        rounds at positions >= 32768, ONE flush across the 5 drafter layers, bit-identical to an eager twin
  cfg5  B = 64, contexts log-uniform 512..16384, shuffled block tables, mixed gamma, geometric accepts, switch prob 0.3
One target layer carries the attention check (the 36 layers run the same kernel on distinct pools; the full-depth,
every-SM-busy launch shape is test_gpu_fullsize.py's); every drafter layer is checked.

Compared per round: attention rows of sampled (sequence, query head) pairs (max-abs 2e-2, rel-L2 5e-3 per pair);
accept_len / bonus / n_commit bit-exact, entropy 1e-3, route bit-exact outside |H - tau| < 1e-4; target and drafter
block tables, cache lengths and backlog lengths bit-exact; the K/V rows each drafter wrote this round within rel-L2
5e-3 of the oracle's unrounded fp64; backlog rows bit-exact; cur_drafter, who switched and the next block lengths bit-exact;
the post-MLP state of the final backlog token (f3, oracle O9) of up to two sequences per round that switched to the AR drafter
within rel-L2 5e-3.
"""

import math

import numpy as np
import pytest

from oracle import accept_route, final_token, kv_prefill, lazy_catchup, verify_attn
from oracle.paged_kv import PagedKV as OraclePagedKV
from paper_2606_07710_b200 import synth

pytestmark = pytest.mark.gpu

ATTN_MAX_ABS, ATTN_REL_L2, ENTROPY_ABS, ROUTE_BAND, KV_REL_L2, H_REL_L2 = 2e-2, 5e-3, 1e-3, 1e-4, 5e-3, 5e-3
ROUTE_AR, ROUTE_DIFFUSION = 1, 0


@pytest.fixture(scope="module")
def wf():
    import torch
    assert torch.cuda.is_available(), "gpu tests need a CUDA device"
    from paper_2606_07710_b200 import binding
    ctx = binding.Ctx(0)
    # the launch mode bench.py times: rounds.py keeps the promise of wf_ctx_set_attn_early_kv (no kernel that precedes an
    # attention launch writes lengths, old block-table entries or rows below the cached length)
    ctx.set_attn_early_kv(1)
    yield binding, ctx
    ctx.close()


def _bits(t):
    import torch
    return t.detach().contiguous().view(torch.int16).cpu().numpy().view(np.uint16)


def _mirror_drafter(rs, d):
    """Oracle twin of a RoundState drafter: same free list, same weights, same starting lengths."""
    sh, B = rs.sh, rs.B
    okv = OraclePagedKV(d.n_layers, sh.n_kv_heads, sh.head_dim, sh.page_size, d.kv.shape.num_pages, B,
                        d.kv.shape.max_pages_per_seq, d.free)
    okv.reserve(rs.ctx0)
    okv.seq_len[:B] = rs.ctx0
    od = kv_prefill.Drafter([_bits(w) for w in d.w_k], [_bits(w) for w in d.w_v], okv, sh.rope_theta)
    return lazy_catchup.LazyCatchup(od, d.cap)


def _gather_rows(d, layer, b, p0, n, sh):
    """K/V bits [n][Hkv][D] at logical positions p0..p0+n-1 of sequence b, read from the GPU pools via its block table."""
    import torch
    pos = torch.arange(p0, p0 + n, device="cuda")
    pages = d.block_table[b][(pos // sh.page_size).long()].long()
    slots = (pos % sh.page_size).long()
    K = d.k_pool[layer][pages, :, slots, :]
    V = d.v_pool[layer][pages, :, slots, :]
    return _bits(K), _bits(V)


def _rel_l2(bits, want):
    got = (np.asarray(bits, dtype=np.uint16).astype(np.uint32) << 16).view(np.float32).astype(np.float64)
    return float(np.sqrt(((got - want) ** 2).sum() / max((want ** 2).sum(), 1e-300)))


def _round_parity(wf, index, n_rounds, sample_seqs, sample_heads, sample_rows=None):
    import torch
    from paper_2606_07710_b200.rounds import RoundState
    binding, ctx = wf
    wl = synth.WORKLOADS[index]
    sh = wl.shapes
    rs = RoundState(ctx, wl, n_slots=n_rounds, n_rounds_max=n_rounds + 2, layers=1)
    B = rs.B
    # ---- oracle state: target block table / lengths, both drafters with their lazy queues, the current drafter ----
    okv_t = OraclePagedKV(1, sh.n_kv_heads, sh.head_dim, sh.page_size, rs.kv_shape.num_pages, B, rs.max_pages_per_seq, rs.free)
    okv_t.reserve(rs.ctx0)
    okv_t.seq_len[:B] = rs.ctx0
    lz = {ROUTE_DIFFUSION: _mirror_drafter(rs, rs.drafters["D"]), ROUTE_AR: _mirror_drafter(rs, rs.drafters["A"])}
    gd = {ROUTE_DIFFUSION: rs.drafters["D"], ROUTE_AR: rs.drafters["A"]}
    cur = rs.slots[0].cur.copy()
    full = final_token.FullLayer(*[[_bits(w) for w in ws] for ws in rs.ft.weights], sh.n_q_heads)     # (f3) the AR drafter's layer
    worst_h, n_final = 0.0, 0
    near_tau = worst_attn = worst_kv = 0
    routes_seen, flushes = set(), 0
    for rnd in range(n_rounds):
        s = rs.slots[rnd]
        # sampled sequences' K/V and block inputs as the attention of this round sees them (before the round)
        okv_t.reserve(s.q_lens)
        samples = {}
        for b in sample_seqs(B):
            ctx_b = int(okv_t.seq_len[b])
            r0, r1 = int(s.q_indptr_host[b]), int(s.q_indptr_host[b + 1])
            n_tok = ctx_b + (r1 - r0)
            pages = torch.from_numpy(okv_t.block_table[b, : -(-n_tok // sh.page_size)].astype(np.int64)).cuda()
            K = _bits(rs.k_pool[0][pages].permute(0, 2, 1, 3).reshape(-1, sh.n_kv_heads, sh.head_dim)[:n_tok])
            V = _bits(rs.v_pool[0][pages].permute(0, 2, 1, 3).reshape(-1, sh.n_kv_heads, sh.head_dim)[:n_tok])
            samples[b] = (ctx_b, K, V, _bits(s.q[r0:r1]))
        before = {c: (l.drafter.kv.seq_len.copy(), l.backlog_len.copy()) for c, l in lz.items()}
        rs.run_round()
        torch.cuda.synchronize()
        assert ctx.poll_status() == 0
        # ---- (a) attention, per sampled (sequence, query head) pair ----
        for b, (ctx_b, K, V, Qb) in samples.items():
            one = OraclePagedKV(1, sh.n_kv_heads, sh.head_dim, sh.page_size, -(-len(K) // sh.page_size), 1, -(-len(K) // sh.page_size))
            one.reserve([len(K)])
            for pg in range(-(-len(K) // sh.page_size)):
                cnt = min(sh.page_size, len(K) - pg * sh.page_size)
                one.k_pool[0, pg, :, :cnt, :] = K[pg * sh.page_size: pg * sh.page_size + cnt].transpose(1, 0, 2)
                one.v_pool[0, pg, :, :cnt, :] = V[pg * sh.page_size: pg * sh.page_size + cnt].transpose(1, 0, 2)
            one.seq_len[0] = ctx_b
            r0 = int(s.q_indptr_host[b])
            rows = range(len(Qb)) if sample_rows is None else [i for i in sample_rows if i < len(Qb)]
            got_all = s.attn_out[r0:r0 + len(Qb)].float().cpu().numpy().astype(np.float64)
            for h in sample_heads:
                want = np.stack([verify_attn.verify_attn_row(one, 0, 0, Qb[i], i, sh.n_q_heads, rs.sm_scale, heads=[h])[0] for i in rows])
                got = got_all[list(rows), h, :]
                rel = float(np.sqrt(((got - want) ** 2).sum() / (want ** 2).sum()))
                assert np.abs(got - want).max() <= ATTN_MAX_ABS and rel <= ATTN_REL_L2, (wl.name, rnd, b, h, rel)
                worst_attn = max(worst_attn, rel)
        # ---- (b) accept / bonus / entropy / route, every sequence ----
        want = accept_route.accept_entropy_route(s.logits.cpu().numpy(), s.drafts.cpu().numpy(), s.q_indptr_host, sh.tau, kv=okv_t)
        got = {k: v.cpu().numpy() for k, v in rs.out.items()}
        for k in ("accept_len", "bonus_token", "n_commit"):
            np.testing.assert_array_equal(got[k], want[k], err_msg=f"{wl.name} round {rnd} {k}")
        assert np.abs(rs.entropy.cpu().numpy().astype(np.float64) - want["entropy"]).max() <= ENTROPY_ABS
        near = np.abs(want["entropy"] - sh.tau) < ROUTE_BAND
        np.testing.assert_array_equal(got["route"][~near], want["route"][~near])
        near_tau += int(near.sum())
        route = np.where(near, got["route"], want["route"]).astype(np.int32)   # inside the band either side is right
        routes_seen |= set(route.tolist())
        np.testing.assert_array_equal(rs.seq_len.cpu().numpy(), okv_t.seq_len[:B])
        np.testing.assert_array_equal(rs.block_table.cpu().numpy(), okv_t.block_table)
        # ---- (c) + (d) the switch, driven by the oracle's route ----
        hid = _bits(s.hidden)
        flushes += int((route != cur).sum())
        switched_to_ar = (cur != ROUTE_AR) & (route == ROUTE_AR) & (want["n_commit"] > 0)
        np.testing.assert_array_equal(rs.switched.cpu().numpy(), np.where(route != cur, route, -1))
        cur, nq, outs = lazy_catchup.switch_round(lz, hid, s.q_indptr_host, want["n_commit"], route, cur, rs.q_len_of)
        # ---- (f3) the final backlog token in full, for (at most two of) the sequences that switched to the AR drafter ----
        h_gpu = rs.ft.h_out.float().cpu().numpy().astype(np.float64)
        for b in np.nonzero(switched_to_ar)[0][:2]:
            x_last = hid[int(s.q_indptr_host[b]) + int(want["n_commit"][b]) - 1]
            h_want = final_token.final_token_full(lz[ROUTE_AR].drafter, full, x_last, int(b))
            for layer in range(h_want.shape[0]):
                rel = float(np.sqrt(((h_gpu[b, layer] - h_want[layer]) ** 2).sum() / (h_want[layer] ** 2).sum()))
                assert rel <= H_REL_L2, (wl.name, rnd, int(b), layer, rel)
                worst_h = max(worst_h, rel)
            n_final += 1
        np.testing.assert_array_equal(rs.cur_drafter.cpu().numpy(), cur)
        np.testing.assert_array_equal(rs.next_q_len.cpu().numpy(), nq)
        for code, l in lz.items():
            d = gd[code]
            np.testing.assert_array_equal(d.seq_len.cpu().numpy(), l.drafter.kv.seq_len[:B], err_msg=f"{wl.name} drafter {code} cache length")
            np.testing.assert_array_equal(d.backlog_len.cpu().numpy(), l.backlog_len[:B], err_msg=f"{wl.name} drafter {code} backlog length")
            np.testing.assert_array_equal(d.block_table.cpu().numpy(), l.drafter.kv.block_table, err_msg=f"{wl.name} drafter {code} block table")
            for b, (Ko, Vo) in outs[code].items():                  # rows written this round: [L][n][Hkv][D] fp64 unrounded
                p0, n = int(before[code][0][b]), Ko.shape[1]
                for layer in range(Ko.shape[0]):
                    Kg, Vg = _gather_rows(d, layer, b, p0, n, sh)
                    rk, rv = _rel_l2(Kg, Ko[layer]), _rel_l2(Vg, Vo[layer])
                    assert rk <= KV_REL_L2 and rv <= KV_REL_L2, (wl.name, rnd, code, b, layer, rk, rv)
                    worst_kv = max(worst_kv, rk, rv)
            bl = _bits(d.backlog)
            for b in range(B):
                nb = int(l.backlog_len[b])
                assert np.array_equal(bl[b, :nb], l.backlog[b, :nb]), (wl.name, rnd, code, b, "backlog rows")
    rs.close()
    return dict(near_tau=near_tau, worst_attn=worst_attn, worst_kv=worst_kv, routes=routes_seen, flushes=flushes, worst_h=worst_h,
                n_final=n_final)


def test_cfg2_whole_rounds(wf):
    """configs[1]: batch 1, context 4096, gamma 15, vocabulary 151936; every query head of the one sequence."""
    r = _round_parity(wf, 1, 10, lambda B: [0], range(32))
    assert r["routes"] == {0, 1} and r["flushes"] > 0, r          # the one sequence switches drafters within the run
    print("cfg2", r)


def test_cfg3_whole_rounds(wf):
    """configs[2]: batch 16, context 8192, gamma 7 / 15 by route, cap 32."""
    r = _round_parity(wf, 2, 4, lambda B: [0, 7, 15], [0, 9, 18, 31])
    assert r["routes"] == {0, 1} and r["flushes"] > 0 and r["n_final"] > 0, r
    print("cfg3", r)


def test_cfg4_whole_rounds(wf):
    """configs[3]: batch 4, context 32768, gamma 15, cap 64."""
    r = _round_parity(wf, 3, 3, lambda B: [1, 3], [3, 28], sample_rows=[0, 7, 15])
    print("cfg4", r)


def test_cfg5_whole_rounds(wf):
    """configs[4]: batch 64, log-uniform contexts, shuffled pages, mixed gamma, geometric accepts, switch prob 0.3."""
    r = _round_parity(wf, 4, 3, lambda B: [0, 21, 42, 63], [2, 13, 27], sample_rows=[0, 3, 7, 15])
    assert r["routes"] == {0, 1} and r["flushes"] > 0 and r["n_final"] > 0, r
    print("cfg5", r)


@pytest.mark.parametrize("index,layers,n_rounds", [(1, 36, 12), (2, 3, 6), (4, 2, 5)])
def test_early_kv_rounds_bit_identical_to_waiting_rounds(index, layers, n_rounds):
    """wf_ctx_set_attn_early_kv changes WHEN an attention launch reads the cache (ahead of its dependency wait), never what
    it computes: whole rounds launched back to back without a host synchronisation (every launch overlaps the tail of the
    previous one: reserve -> layers x attention -> accept -> switch -> final token -> reserve ...) leave the same bits in
    every output as the same rounds with the mode off.  Both contexts fold split pairs in a fixed order (deterministic mode)
    so that equality of bits is the expectation.  cfg2 takes the cluster shape at full depth, cfg3 / cfg5 stream-K ranges."""
    import torch
    from paper_2606_07710_b200 import binding
    from paper_2606_07710_b200.rounds import RoundState
    wl = synth.WORKLOADS[index]
    runs = []
    for early in (0, 1):
        ctx = binding.Ctx(0)
        ctx.set_deterministic(1)
        ctx.set_attn_early_kv(early)
        rs = RoundState(ctx, wl, n_slots=n_rounds, n_rounds_max=n_rounds + 2, layers=layers)
        outs = []
        for _ in range(n_rounds):
            s = rs.run_round()
            outs.append((s.attn_out.clone(), {k: v.clone() for k, v in rs.out.items()}, rs.ft.h_out.clone()))
        torch.cuda.synchronize()
        assert ctx.poll_status() == 0
        runs.append((ctx, rs, outs))
    (ctx0, rs0, outs0), (ctx1, rs1, outs1) = runs
    try:
        assert torch.equal(rs0.seq_len, rs1.seq_len)
        for rnd, ((a0, o0, h0), (a1, o1, h1)) in enumerate(zip(outs0, outs1)):
            diff = int((a0.view(torch.int16) != a1.view(torch.int16)).sum())
            assert diff == 0, (wl.name, rnd, "attention output bits", diff)
            for k in o0:
                assert torch.equal(o0[k], o1[k]), (wl.name, rnd, k)
            assert torch.equal(h0.view(torch.int16), h1.view(torch.int16)), (wl.name, rnd, "final-token state bits")
        for n in rs0.drafters:
            d0, d1 = rs0.drafters[n], rs1.drafters[n]
            assert torch.equal(d0.seq_len, d1.seq_len) and torch.equal(d0.backlog_len, d1.backlog_len), (wl.name, n)
            assert torch.equal(d0.k_pool.view(torch.int16), d1.k_pool.view(torch.int16)), (wl.name, n, "K pool")
            assert torch.equal(d0.v_pool.view(torch.int16), d1.v_pool.view(torch.int16)), (wl.name, n, "V pool")
    finally:
        for ctx, rs, _ in runs:
            rs.close()
            ctx.close()


def test_cfg4_flush_of_64_deferred_tokens_bit_identical_to_eager(wf):
    """configs[3] verbatim: "Lazy Catch-up flush of 64 deferred tokens across the 5 drafter layers, checked
    bit-identical against eager per-round KV-only prefill".  B = 4, positions from 32768, cap 64: four idle rounds of 16
    committed rows each (enqueued by wf_switch_round with cur = route = AR, i.e. by the device-side masks), then ONE
    wf_lazy_catchup_flush (M = 256 rows, all 5 layers); an eager twin with the same weights gets wf_kv_only_prefill every
    round.  All 5 x 2 x 4 x 64 x 1024 bf16 values, lengths and backlog lengths must be equal bit for bit (GPU vs GPU),
    the values within rel-L2 5e-3 of the oracle's, the indices equal to the oracle's."""
    import torch
    import gpu_harness as H
    binding, ctx = wf
    B, L, hidden, Hkv, D, cap, p0 = 4, 5, 4096, 8, 128, 64, 32768
    g = synth.rng(synth.SEED_BASE + 3, 909)
    pages_per_seq = (p0 + 5 * 16) // 16 + 2
    P = B * pages_per_seq + 9
    free = synth.draw_free_list(P, g, True)
    lazy = H.DrafterPair(ctx, L, hidden, Hkv, D, P, B, pages_per_seq, free, seed=91, backlog_cap=cap, max_pos=p0 + 200)
    eager = H.DrafterPair(ctx, L, hidden, Hkv, D, P, B, pages_per_seq, free, seed=91, backlog_cap=cap, max_pos=p0 + 200,
                          weights=lazy.weights)
    free_a = synth.draw_free_list(P, g, True)
    ar = H.DrafterPair(ctx, 1, hidden, Hkv, D, P, B, pages_per_seq, free_a, seed=92, backlog_cap=cap, max_pos=p0 + 200)
    for dp in (lazy, eager, ar):
        dp.kvp.reserve([p0] * B)
        dp.kvp.set_seq_len([p0] * B)
    q_indptr = (np.arange(B + 1) * 16).astype(np.int32)
    n = np.full(B, 16, dtype=np.int32)
    cur = H.i32([ROUTE_AR] * B)
    route = H.i32([ROUTE_AR] * B)                                  # the router keeps the AR drafter: D stays idle
    nq = torch.zeros(B, dtype=torch.int32, device="cuda")
    for rnd in range(4):
        X = synth.normal_bf16(g, (B * 16, hidden), 1.0)
        Xd = H.bits_to_bf16_tensor(X)
        binding.wf_switch_round(ctx, ar.gpu, lazy.gpu, Xd, H.i32(q_indptr), H.i32(n), None, route, cur, nq, 16, 16, B, 16)
        lazy.oracle_lazy.round(X, q_indptr, n, [1] * B, [0] * B)
        binding.wf_kv_only_prefill(ctx, eager.gpu, Xd, H.i32(q_indptr), H.i32(n), None, B, 16)
        kv_prefill.kv_only_prefill(eager.oracle, X, q_indptr, n)
    torch.cuda.synchronize()
    assert ctx.poll_status() == 0
    np.testing.assert_array_equal(lazy.backlog_len.cpu().numpy(), [64] * B)
    np.testing.assert_array_equal(lazy.kvp.seq_len.cpu().numpy(), [p0] * B)           # nothing projected yet
    assert np.array_equal(H.bf16_tensor_to_bits(lazy.backlog), lazy.oracle_lazy.backlog)
    un = lazy.oracle_lazy.flush(None, B)
    binding.wf_lazy_catchup_flush(ctx, lazy.gpu, None, B)
    torch.cuda.synchronize()
    assert ctx.poll_status() == 0
    lazy.kvp.assert_tables_equal()
    eager.kvp.assert_tables_equal()
    np.testing.assert_array_equal(lazy.backlog_len.cpu().numpy(), [0] * B)
    np.testing.assert_array_equal(lazy.kvp.seq_len.cpu().numpy(), [p0 + 64] * B)
    n_vals = 0
    for layer in range(L):
        for b in range(B):
            Kl, Vl = lazy.gather_gpu(layer, b, p0 + 64)
            Ke, Ve = eager.gather_gpu(layer, b, p0 + 64)
            assert np.array_equal(Kl[p0:], Ke[p0:]) and np.array_equal(Vl[p0:], Ve[p0:]), (layer, b)
            n_vals += 2 * Kl[p0:].size
            Ko, Vo = un[b]
            assert H.rel_l2(Kl[p0:], Ko[layer]) <= KV_REL_L2 and H.rel_l2(Vl[p0:], Vo[layer]) <= KV_REL_L2
            Kol, Vol = lazy.kvp.oracle.gather(layer, b, p0 + 64)                       # oracle lazy == oracle eager (O4.i)
            Koe, Voe = eager.kvp.oracle.gather(layer, b, p0 + 64)
            assert np.array_equal(Kol[p0:], Koe[p0:]) and np.array_equal(Vol[p0:], Voe[p0:])
    assert n_vals == 5 * 2 * 4 * 64 * 1024
    for dp in (lazy, eager, ar):
        dp.close()
