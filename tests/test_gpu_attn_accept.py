"""GPU parity (through the C-ABI) for the paged-KV block table, (b) accept/entropy/route and
(a) verification attention, element by element against oracle/ on the same seeded inputs.

Tolerances (BASELINE.json north_star): integers bit-exact (route exempt only when |H - tau| < 1e-4,
counted separately); entropy 1e-3 absolute; attention max-abs 2e-2 and relative L2 5e-3.
"""

import math

import numpy as np
import pytest

from oracle import accept_route, verify_attn
from paper_2606_07710_b200 import synth

pytestmark = pytest.mark.gpu

ATTN_MAX_ABS = 2e-2
ATTN_REL_L2 = 5e-3
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


# ------------------------------------------------------------------------------------ block table
def test_block_table_matches_oracle(wf):
    import torch
    import gpu_harness as H
    binding, ctx = wf
    g = synth.rng(7, 1)
    P, S = 300, 6
    free = synth.draw_free_list(P, g, True)
    pair = H.KvPair(ctx, 1, 2, 64, P, S, 40, free)
    pair.reserve([100, 0, 17, 16, 1, 250])
    pair.assert_tables_equal()
    pair.set_seq_len([100, 0, 17, 16, 1, 250])
    pair.reserve([5, 3, 0, 1, 15, 16])                     # grows only where a page boundary is crossed
    pair.assert_tables_equal()
    # release and reuse: pages go to the ring tail in block-table order (C24)
    pair.oracle.release_seq(0)
    pair.gpu.release_seq(0)
    pair.oracle.release_seq(5)
    pair.gpu.release_seq(5)
    pair.assert_tables_equal()
    pair.reserve([300, 10, 0, 0, 0, 40])
    pair.assert_tables_equal()
    assert ctx.poll_status() == 0
    # exhaustion: nothing allocated, sticky status (oracle raises)
    before = pair.block_table.clone()
    pair.gpu.reserve(H.i32([16 * 39] * 6), 6)              # 6 x 39 pages > 300 pages in the pool
    torch.cuda.synchronize()
    assert torch.equal(before, pair.block_table)
    st = ctx.poll_status()
    assert st == binding.WF_ERR_OUT_OF_PAGES
    assert ctx.poll_status() == 0
    pair.close()


# ------------------------------------------------------------------------------ accept / route
def _run_accept(binding, ctx, logits, drafts, q_indptr, tau, max_q):
    import torch
    import gpu_harness as H
    B = len(q_indptr) - 1
    V = logits.shape[1]
    d_logits = H.f32(logits)
    outs = {k: torch.full((B,), -7, dtype=torch.int32, device="cuda") for k in ("accept_len", "bonus_token", "route", "n_commit")}
    ent = torch.full((B,), -7.0, dtype=torch.float32, device="cuda")
    tau_arr = np.atleast_1d(np.asarray(tau, dtype=np.float32))
    ws = torch.empty(binding.wf_accept_workspace_bytes(B * max_q, V), dtype=torch.uint8, device="cuda")
    binding.wf_accept_entropy_route(ctx, d_logits, V, H.i32(drafts), H.i32(q_indptr), B, max_q, H.f32(tau_arr),
                                    len(tau_arr) == 1, outs["accept_len"], outs["bonus_token"], ent, outs["route"],
                                    outs["n_commit"], None, ws)
    torch.cuda.synchronize()
    res = {k: v.cpu().numpy() for k, v in outs.items()}
    res["entropy"] = ent.cpu().numpy()
    return res


def _check_accept(res, want, tau):
    B = len(want["accept_len"])
    tau = np.broadcast_to(np.asarray(tau, dtype=np.float64), (B,))
    for k in ("accept_len", "bonus_token", "n_commit"):
        np.testing.assert_array_equal(res[k], want[k], err_msg=k)
    assert np.abs(res["entropy"].astype(np.float64) - want["entropy"]).max() <= ENTROPY_ABS
    near = np.abs(want["entropy"] - tau) < ROUTE_BAND
    np.testing.assert_array_equal(res["route"][~near], want["route"][~near])
    return int(near.sum())


@pytest.mark.parametrize("seed", range(64))
def test_accept_cfg1_tiny(wf, seed):
    """configs[0]: vocab 4096, gamma 7, planted prefix uniform 0..7, spike puts H on both sides of tau."""
    binding, ctx = wf
    wl = synth.WORKLOADS[0]
    g = synth.rng(wl.seed, 1000 + seed)
    u = synth.draw_accept_prefix(g, [7])
    spike = g.uniform(0.0, 10.0, size=1)
    logits, drafts, q_indptr, _ = synth.make_logits_block(g, [8], wl.shapes.vocab, wl.shapes.logit_sigma, u, spike)
    want = accept_route.accept_entropy_route(logits, drafts, q_indptr, wl.shapes.tau)
    assert want["accept_len"][0] == u[0]
    res = _run_accept(binding, ctx, logits, drafts, q_indptr, wl.shapes.tau, 8)
    _check_accept(res, want, wl.shapes.tau)


def test_accept_8b_vocab_mixed_gamma(wf):
    """vocab 151936 (19 slices, ragged last slice), mixed gamma 7/15, an empty block, per-sequence tau."""
    binding, ctx = wf
    g = synth.rng(synth.SEED_BASE + 1, 77)
    q_lens = [16, 8, 0, 16, 8, 1]
    u = [15, 3, 0, 0, 7, 0]
    spike = [6.0, 0.0, 0.0, 9.0, 4.5, 5.0]
    logits, drafts, q_indptr, _ = synth.make_logits_block(g, q_lens, 151936, 3.0, u, spike)
    tau = np.array([2.0, 2.0, 2.0, 1.0, 7.0, 2.0], dtype=np.float32)
    want = accept_route.accept_entropy_route(logits, drafts, q_indptr, tau)
    res = _run_accept(binding, ctx, logits, drafts, q_indptr, tau, 16)
    _check_accept(res, want, tau)
    assert set(want["route"].tolist()) == {0, 1}, "the case must exercise both routes"
    assert res["n_commit"][2] == 0 and res["accept_len"][2] == 0


def test_accept_block_longer_than_the_host_bound_is_flagged(wf):
    """q_b > max_q_len (the host bound that sizes the grid): the sticky status says so, the block is verified up to the
    bound, and the context's completion counter still resets: the next, valid call is correct."""
    binding, ctx = wf
    g = synth.rng(5, 5)
    logits, drafts, q_indptr, _ = synth.make_logits_block(g, [16, 8], 4096, 2.0, [15, 2], [0.0, 9.0])
    res = _run_accept(binding, ctx, logits, drafts, q_indptr, 2.0, 8)          # sequence 0 has 16 rows, the bound says 8
    assert ctx.poll_status() == binding.WF_ERR_INVALID_ARG
    assert res["accept_len"][0] == 7 and res["accept_len"][1] == 2              # verified up to the bound
    want = accept_route.accept_entropy_route(logits, drafts, q_indptr, 2.0)
    res = _run_accept(binding, ctx, logits, drafts, q_indptr, 2.0, 16)
    assert ctx.poll_status() == 0
    _check_accept(res, want, 2.0)


def test_accept_edge_rows(wf):
    """-inf (masked vocabulary), exact ties (lowest id wins), V % 4 != 0 (scalar path), closed forms."""
    binding, ctx = wf
    V = 1003
    logits = np.full((4, V), -np.inf, dtype=np.float32)
    logits[0, [5, 900]] = 1.5                      # two equal maxima, rest -inf: H = ln 2, argmax = 5
    logits[1, :] = 0.25                            # constant row: H = ln V, argmax = 0
    logits[2, 77] = 3.0                            # one-hot: H = 0
    logits[3, :] = np.linspace(-3, 3, V, dtype=np.float32)
    drafts = np.array([0, 5, 0, 77], dtype=np.int32)   # row1 draft = g_0 = 5, row2 draft 0 = g_1, row3 draft 77 = g_2
    q_indptr = np.array([0, 4], dtype=np.int32)
    want = accept_route.accept_entropy_route(logits, drafts, q_indptr, 2.0)
    assert want["accept_len"][0] == 3
    res = _run_accept(binding, ctx, logits, drafts, q_indptr, 2.0, 4)
    _check_accept(res, want, 2.0)
    for rows, H_want in (([0], math.log(2.0)), ([1], math.log(V)), ([2], 0.0)):
        r = _run_accept(binding, ctx, logits[rows], np.zeros(1, np.int32), np.array([0, 1], np.int32), 2.0, 1)
        assert abs(float(r["entropy"][0]) - H_want) <= ENTROPY_ABS


def test_accept_advances_target_len(wf):
    import torch
    import gpu_harness as H
    binding, ctx = wf
    pair = H.make_kv_pair(ctx, [100, 37], [8, 8], 1, 2, 64, seed=5, fill=False)
    g = synth.rng(11, 3)
    logits, drafts, q_indptr, _ = synth.make_logits_block(g, [8, 8], 4096, 2.0, [4, 7], [0.0, 8.0])
    want = accept_route.accept_entropy_route(logits, drafts, q_indptr, 2.0, kv=pair.oracle)
    B, V = 2, 4096
    o = [torch.zeros(B, dtype=torch.int32, device="cuda") for _ in range(4)]
    ent = torch.zeros(B, dtype=torch.float32, device="cuda")
    ws = torch.empty(binding.wf_accept_workspace_bytes(16, V), dtype=torch.uint8, device="cuda")
    for _ in range(2):                                  # second call checks the self-resetting counters
        pair.set_seq_len([100, 37])
        binding.wf_accept_entropy_route(ctx, H.f32(logits), V, H.i32(drafts), H.i32(q_indptr), B, 8, H.f32([2.0]), True,
                                        o[0], o[1], ent, o[2], o[3], pair.gpu, ws)
        torch.cuda.synchronize()
        np.testing.assert_array_equal(pair.seq_len.cpu().numpy()[:2], [100 + 5, 37 + 8])
        np.testing.assert_array_equal(o[0].cpu().numpy(), want["accept_len"])
    pair.close()


# ------------------------------------------------------------------------------------ attention
def _run_attn(binding, ctx, pair, layer, Q_bits, q_indptr, Hq, max_q, scale):
    import torch
    import gpu_harness as H
    B = len(q_indptr) - 1
    q = H.bits_to_bf16_tensor(Q_bits)
    out = torch.zeros_like(q)
    ws = torch.empty(binding.wf_verify_attn_workspace_bytes(pair.shape, B, Hq, max_q), dtype=torch.uint8, device="cuda")
    binding.wf_verify_attn(ctx, pair.gpu, layer, q, H.i32(q_indptr), B, Hq, max_q, scale, out, ws)
    torch.cuda.synchronize()
    return H.bf16_tensor_to_bits(out)


def _attn_case(wf, ctx_lens, q_lens, Hq, Hkv, D, seed, n_layers=1, layer=0, q_std=1.0, kv_std=None, poison=False):
    import gpu_harness as H
    binding, ctx = wf
    pair = H.make_kv_pair(ctx, ctx_lens, q_lens, n_layers, Hkv, D, seed, kv_std=kv_std)
    if poison:   # NaN in every slot at or beyond ctx+q of each sequence and in unreferenced pages (pin O1.vi)
        ref = np.zeros(pair.oracle.k_pool.shape[1:], dtype=bool)       # [page][head][slot][d] referenced?
        for b, (c, qn) in enumerate(zip(ctx_lens, q_lens)):
            for j in range(c + qn):
                pg, slot = pair.oracle.locate(b, j)
                ref[pg, :, slot, :] = True
        pair.oracle.k_pool[:, ~ref] = 0x7FC0
        pair.oracle.v_pool[:, ~ref] = 0x7FC0
        pair.upload_pools()
    g = synth.rng(seed, 202)
    q_indptr = np.zeros(len(q_lens) + 1, dtype=np.int32)
    q_indptr[1:] = np.cumsum(q_lens)
    Q = synth.normal_bf16(g, (int(q_indptr[-1]), Hq, D), q_std)
    scale = 1.0 / math.sqrt(D)
    want = verify_attn.verify_attn(pair.oracle, layer, Q, q_indptr, Hq, scale)
    got = _run_attn(binding, ctx, pair, layer, Q, q_indptr, Hq, max(q_lens), scale)
    pair.close()
    assert not np.isnan(H.attn_errors(got, want)[0])
    return H.attn_errors(got, want)


def test_attn_cfg1_tiny(wf):
    """configs[0]: 4 q / 2 kv heads, D 64, ctx 512, gamma 7; 64 seeds."""
    for seed in range(64):
        max_abs, rel = _attn_case(wf, [512], [8], 4, 2, 64, seed=synth.SEED_BASE + seed)
        assert max_abs <= ATTN_MAX_ABS and rel <= ATTN_REL_L2, (max_abs, rel)


def test_attn_8b_shapes_ragged_split(wf):
    """8B-class heads (32/8, D 128), ragged contexts spanning several split chunks and a ragged tail,
    mixed gamma 7/15, an empty block, shuffled pages, layer 1 of 2, NaN beyond the visible range."""
    max_abs, rel = _attn_case(wf, [3000, 17, 1, 1500, 640, 255], [16, 8, 16, 0, 8, 16], 32, 8, 128, seed=9,
                              n_layers=2, layer=1, poison=True)
    assert max_abs <= ATTN_MAX_ABS and rel <= ATTN_REL_L2, (max_abs, rel)


def test_attn_peaked_scores(wf):
    """Stress the online-softmax rescaling: Q and K scaled so that the score std is about 4 (SURVEY.md §8(c) tolerance
    note asks for this case to be reported separately).  Here the attention weights concentrate on a few keys, P has
    entries near 1 whose bf16 rounding (2^-9 relative) is no longer averaged over thousands of keys: the measured rel-L2
    is printed, and the assertion is north_star's 5e-3 like everywhere else."""
    max_abs, rel = _attn_case(wf, [2100, 300], [16, 8], 32, 8, 128, seed=10, q_std=4.0, kv_std=1.0)
    print(f"peaked scores: max-abs {max_abs:.3e}, rel-L2 {rel:.3e}")
    assert max_abs <= ATTN_MAX_ABS and rel <= ATTN_REL_L2, (max_abs, rel)


def test_attn_single_query_and_zero_context(wf):
    """q = 1 (plain decode) and ctx = 0 (the block is the whole sequence)."""
    max_abs, rel = _attn_case(wf, [0, 0, 700], [16, 1, 1], 8, 2, 64, seed=12)
    assert max_abs <= ATTN_MAX_ABS and rel <= ATTN_REL_L2, (max_abs, rel)


def test_attn_group_shapes(wf):
    """GQA group sizes 1 (MHA: 16 rows per kv head), 8 (q = 8 -> 64 rows) and 2, with D = 64 and D = 128."""
    for (Hq, Hkv, D, q_lens, ctx) in [(4, 4, 64, [16, 3], [300, 77]), (64, 8, 128, [8, 8], [700, 129]),
                                      (8, 4, 128, [16, 16, 5], [1000, 15, 260])]:
        max_abs, rel = _attn_case(wf, ctx, q_lens, Hq, Hkv, D, seed=21 + Hq)
        assert max_abs <= ATTN_MAX_ABS and rel <= ATTN_REL_L2, (Hq, Hkv, D, max_abs, rel)


def test_attn_blocks_wider_than_64_rows_per_kv_head(wf):
    """max_q_len * group > 64 (gamma = 15 at a GQA group of 8 or 16; blocks of up to 64 tokens at group 4): wf_verify_attn
    runs these as degenerate trees on the tree kernel's 128-row tiles; same definition, same tolerance.  Ragged tails, an
    empty block, a block of one token, zero context, several 128-row tiles per block, NaN beyond the visible range."""
    for (Hq, Hkv, D, q_lens, ctx, poison) in [(64, 8, 128, [16, 9, 16, 0, 1], [700, 129, 2050, 33, 5], True),
                                              (8, 2, 64, [64, 33, 17], [300, 0, 1000], False),
                                              (16, 1, 128, [16, 5, 12], [515, 64, 4100], True)]:
        max_abs, rel = _attn_case(wf, ctx, q_lens, Hq, Hkv, D, seed=61 + Hq, poison=poison)
        assert max_abs <= ATTN_MAX_ABS and rel <= ATTN_REL_L2, (Hq, Hkv, D, max_abs, rel)


def test_attn_wide_blocks_and_plain_blocks_in_early_kv_mode():
    """The same definition with wf_ctx_set_attn_early_kv on (a context of its own): a wide block (its mask kernel is the
    launch's predecessor), 8B-class ragged shapes with NaN poison, and a cluster-shaped batch-1 call."""
    import torch
    from paper_2606_07710_b200 import binding
    ctx = binding.Ctx(0)
    ctx.set_attn_early_kv(1)
    try:
        for (Hq, Hkv, D, q_lens, ctx_lens) in [(64, 8, 128, [16, 9, 0, 1], [700, 2050, 33, 5]),
                                               (32, 8, 128, [16, 8, 16, 0, 8], [3000, 17, 1500, 640, 255]),
                                               (32, 8, 128, [16], [4096])]:
            max_abs, rel = _attn_case((binding, ctx), ctx_lens, q_lens, Hq, Hkv, D, seed=91 + len(q_lens), poison=True)
            assert max_abs <= ATTN_MAX_ABS and rel <= ATTN_REL_L2, (Hq, Hkv, D, max_abs, rel)
        torch.cuda.synchronize()
        assert ctx.poll_status() == 0
    finally:
        ctx.close()


def test_attn_many_short_sequences_with_empty_blocks(wf):
    """200 sequences with contexts 0..40 and blocks of 0, 1, 8 or 16 rows: far more (sequence, kv head) pairs than CTAs,
    every range holds many one-tile segments, empty blocks in between (the weighted walker must skip them)."""
    g = synth.rng(77, 5)
    ctx = [int(x) for x in g.integers(0, 41, size=200)]
    q_lens = [int(x) for x in g.choice([0, 1, 8, 16], size=200)]
    max_abs, rel = _attn_case(wf, ctx, q_lens, 32, 8, 128, seed=31)
    assert max_abs <= ATTN_MAX_ABS and rel <= ATTN_REL_L2, (max_abs, rel)


def test_attn_all_blocks_empty(wf):
    """B > 0 but nothing to verify: the launch must be a no-op (outputs untouched, no fault, status clean)."""
    import torch
    import gpu_harness as H
    binding, ctx = wf
    pair = H.make_kv_pair(ctx, [50, 9], [0, 0], 1, 2, 64, seed=3)
    q = torch.zeros((1, 4, 64), dtype=torch.bfloat16, device="cuda")
    out = torch.full_like(q, 3.0)
    ws = torch.empty(binding.wf_verify_attn_workspace_bytes(pair.shape, 2, 4, 1), dtype=torch.uint8, device="cuda")
    binding.wf_verify_attn(ctx, pair.gpu, 0, q, H.i32([0, 0, 0]), 2, 4, 1, 0.125, out, ws)
    torch.cuda.synchronize()
    assert ctx.poll_status() == 0 and float(out.float().min()) == 3.0
    pair.close()


def test_attn_long_single_sequence_many_partials(wf):
    """One sequence of 70 000 tokens, 2 kv heads: 547 tiles per pair, so a pair is cut into the maximum number of
    ranges the merge allows (the min-range rule caps the partials per pair)."""
    max_abs, rel = _attn_case(wf, [70000], [16], 8, 2, 128, seed=41)
    assert max_abs <= ATTN_MAX_ABS and rel <= ATTN_REL_L2, (max_abs, rel)


def test_attn_cluster_mode_sizes_and_reproducibility(wf):
    """The cluster launch shape (one thread-block cluster per (sequence, kv head) pair, partials folded through distributed
    shared memory in rank order): forced cluster sizes 2..16 incl. ones that do not divide the 64 rows, pairs with fewer
    tiles than CTAs (CTAs without tiles), gamma 7 (32 live rows), an empty block, D = 64; every size within tolerance of the
    oracle, and five repeated launches of the same size give IDENTICAL bits (the fold order is fixed).  Size 0 = stream-K."""
    import gpu_harness as H
    binding, ctx = wf
    cases = [([4096], [16], 32, 8, 128), ([700, 130], [8, 16], 8, 2, 128), ([300, 0, 40], [16, 0, 8], 4, 2, 64),
             ([5, 2000], [16, 1], 32, 8, 128)]
    try:
        for ci, (ctx_lens, q_lens, Hq, Hkv, D) in enumerate(cases):
            pair = H.make_kv_pair(ctx, ctx_lens, q_lens, 1, Hkv, D, 500 + ci)
            g = synth.rng(500 + ci, 202)
            q_indptr = np.zeros(len(q_lens) + 1, dtype=np.int32)
            q_indptr[1:] = np.cumsum(q_lens)
            Q = synth.normal_bf16(g, (int(q_indptr[-1]), Hq, D), 1.0)
            scale = 1.0 / math.sqrt(D)
            want = verify_attn.verify_attn(pair.oracle, 0, Q, q_indptr, Hq, scale)
            for size in (0, 1, 2, 3, 5, 7, 10, 16, -1):
                ctx.set_attn_cluster(size)
                first = _run_attn(binding, ctx, pair, 0, Q, q_indptr, Hq, max(q_lens), scale)
                max_abs, rel = H.attn_errors(first, want)
                assert max_abs <= ATTN_MAX_ABS and rel <= ATTN_REL_L2, (ci, size, max_abs, rel)
                if size > 0 and len(ctx_lens) * Hkv <= 7:            # the cluster shape is what ran: bits must repeat
                    for _ in range(4):
                        assert np.array_equal(first, _run_attn(binding, ctx, pair, 0, Q, q_indptr, Hq, max(q_lens), scale)), (ci, size)
            assert ctx.poll_status() == 0
            pair.close()
    finally:
        ctx.set_attn_cluster(-1)


def test_two_contexts_in_one_process(wf):
    """Per-context bookkeeping (dynamic shared-memory opt-in, merge counters, cluster tables): a second wf_ctx created in the
    same process runs every large-shared-memory kernel on its own (a process-global `configured` flag broke this)."""
    import gpu_harness as H
    binding, ctx = wf
    ctx2 = binding.Ctx(0)
    try:
        for c in (ctx2, ctx, ctx2):
            max_abs, rel = _attn_case((binding, c), [900, 40], [16, 8], 32, 8, 128, seed=77)
            assert max_abs <= ATTN_MAX_ABS and rel <= ATTN_REL_L2
            max_abs, rel = _attn_case((binding, c), [2500] * 18, [16] * 18, 32, 8, 128, seed=78)     # stream-K shape
            assert max_abs <= ATTN_MAX_ABS and rel <= ATTN_REL_L2
            assert c.poll_status() == 0
    finally:
        ctx2.close()


def test_attn_maximum_batch(wf):
    """B = 1024 sequences (the kernel's table limit), contexts 0..70, blocks of 0..16 rows, 8 kv heads: 8192 (sequence, kv head)
    pairs, ranges of many one-tile segments; B = 1025 is refused on the host."""
    import torch
    import gpu_harness as H
    binding, ctx = wf
    g = synth.rng(91, 5)
    ctx_lens = [int(x) for x in g.integers(0, 71, size=1024)]
    q_lens = [int(x) for x in g.choice([0, 1, 4, 8, 16], size=1024)]
    max_abs, rel = _attn_case(wf, ctx_lens, q_lens, 32, 8, 128, seed=92)
    assert max_abs <= ATTN_MAX_ABS and rel <= ATTN_REL_L2, (max_abs, rel)
    pair = H.make_kv_pair(ctx, [4] * 1025, [1] * 1025, 1, 2, 64, seed=93, fill=False)
    q = torch.zeros((1025, 4, 64), dtype=torch.bfloat16, device="cuda")
    ws = torch.empty(binding.wf_verify_attn_workspace_bytes(pair.shape, 1025, 4, 1), dtype=torch.uint8, device="cuda")
    with pytest.raises(binding.WhiFlashError):
        binding.wf_verify_attn(ctx, pair.gpu, 0, q, H.i32(np.arange(1026)), 1025, 4, 1, 0.125, torch.zeros_like(q), ws)
    pair.close()


def test_accept_large_batch_small_vocab(wf):
    """B = 3000 sequences x up to 8 rows, V = 1000 (one ragged slice per row, V % 4 == 0): every output against the oracle."""
    import torch
    import gpu_harness as H
    binding, ctx = wf
    g = synth.rng(94, 1)
    B, V = 3000, 1000
    q_lens = [int(x) for x in g.integers(0, 9, size=B)]
    prefix = [int(g.integers(0, max(q, 1))) for q in q_lens]
    logits, drafts, ip, _ = synth.make_logits_block(g, q_lens, V, 2.0, prefix, g.uniform(0.0, 8.0, size=B))
    want = accept_route.accept_entropy_route(logits, drafts, ip, 2.0)
    o = [torch.zeros(B, dtype=torch.int32, device="cuda") for _ in range(4)]
    ent = torch.zeros(B, dtype=torch.float32, device="cuda")
    ws = torch.empty(binding.wf_accept_workspace_bytes(B * 8, V), dtype=torch.uint8, device="cuda")
    binding.wf_accept_entropy_route(ctx, H.f32(logits), V, H.i32(drafts), H.i32(ip), B, 8, H.f32([2.0]), True, o[0], o[1], ent, o[2], o[3], None, ws)
    torch.cuda.synchronize()
    assert ctx.poll_status() == 0
    np.testing.assert_array_equal(o[0].cpu().numpy(), want["accept_len"])
    np.testing.assert_array_equal(o[1].cpu().numpy(), want["bonus_token"])
    np.testing.assert_array_equal(o[3].cpu().numpy(), want["n_commit"])
    assert np.abs(ent.cpu().numpy().astype(np.float64) - want["entropy"]).max() <= 1e-3
    far = np.abs(want["entropy"] - 2.0) >= 1e-4
    np.testing.assert_array_equal(o[2].cpu().numpy()[far], want["route"][far])
