"""GPU parity (through the C-ABI) for tree verification: ancestor masks, tree attention,
the acceptance walk and path compaction, element by element against oracle O7 on the same seeded inputs.

Tolerances as for the chain path: masks, accept_len, bonus, n_commit, path and every moved K/V bit exact; entropy
1e-3 absolute; route exact outside |H - tau| < 1e-4; attention max-abs 2e-2 and relative L2 5e-3.
"""

import math

import numpy as np
import pytest

from oracle import tree_verify, verify_attn
from paper_2606_07710_b200 import synth

pytestmark = pytest.mark.gpu

ATTN_MAX_ABS = 2e-2
ATTN_REL_L2 = 5e-3
ENTROPY_ABS = 1e-3
ROUTE_BAND = 1e-4


@pytest.fixture(scope="module", params=[0, 1], ids=["wait", "early_kv"])
def wf(request):
    """Every test runs twice: attention launches wait for the previous kernel before anything else (default), or stream the
    cached K/V ahead of that wait (wf_ctx_set_attn_early_kv; in these tests the caches and lengths are set up by uploads and by
    library calls that are followed by other work before the attention launch, which is the promise that mode asks for)."""
    import torch
    assert torch.cuda.is_available(), "gpu tests need a CUDA device"
    from paper_2606_07710_b200 import binding
    ctx = binding.Ctx(0)
    ctx.set_attn_early_kv(request.param)
    yield binding, ctx
    ctx.close()


def _u64(t):
    return t.cpu().numpy().view(np.uint64)


def _masks(binding, ctx, parent, q_indptr, max_nodes=64):
    import torch
    import gpu_harness as H
    n = int(q_indptr[-1])
    out = torch.zeros(max(n, 1), dtype=torch.int64, device="cuda")
    binding.wf_tree_masks(ctx, H.i32(parent) if n else out, H.i32(q_indptr), len(q_indptr) - 1, max_nodes, out)
    torch.cuda.synchronize()
    return out


def _tree_attn(binding, ctx, pair, layer, Q, q_indptr, parent, Hq, scale, max_nodes):
    import torch
    import gpu_harness as H
    B = len(q_indptr) - 1
    masks = _masks(binding, ctx, parent, q_indptr)
    d_q = H.bits_to_bf16_tensor(Q)
    out = torch.zeros_like(d_q)
    ws = torch.empty(binding.wf_verify_attn_workspace_bytes(pair.shape, B, Hq, max_nodes), dtype=torch.uint8, device="cuda")
    binding.wf_verify_attn_tree(ctx, pair.gpu, layer, d_q, H.i32(q_indptr), masks, B, Hq, max_nodes, scale, out, ws)
    torch.cuda.synchronize()
    return H.bf16_tensor_to_bits(out)


def _trees(g, sizes, depth=8, top_k=10):
    parents = [synth.draw_tree(g, n, depth, top_k) if n else np.zeros(0, np.int32) for n in sizes]
    ip = np.zeros(len(sizes) + 1, np.int32)
    ip[1:] = np.cumsum(sizes)
    parent = np.concatenate(parents) if sum(sizes) else np.zeros(0, np.int32)
    return parents, parent, ip


# ------------------------------------------------------------------------------------ masks
def test_masks_bit_exact_and_bad_parent_flagged(wf):
    import gpu_harness as H
    binding, ctx = wf
    g = synth.rng(31, 1)
    sizes = [60, 1, 0, 64, 17, 16]
    parents, parent, ip = _trees(g, sizes)
    got = _u64(_masks(binding, ctx, parent, ip))[: int(ip[-1])]
    want = np.concatenate([tree_verify.ancestor_masks(p) for p in parents if len(p)])
    np.testing.assert_array_equal(got, want)
    assert ctx.poll_status() == 0
    bad = parent.copy()
    bad[int(ip[3]) + 5] = 7                                  # parent above the node: breaks T1
    got = _u64(_masks(binding, ctx, bad, ip))
    assert ctx.poll_status() == binding.WF_ERR_INVALID_ARG
    assert got[int(ip[3]) + 5] == np.uint64(1 << 5)
    assert ctx.poll_status() == 0


# ------------------------------------------------------------------------------------ attention
@pytest.mark.parametrize("name,Hq,Hkv,D,ctx_lens,sizes", [
    ("tiny-d64-group2", 4, 2, 64, [512, 37, 0, 130], [60, 33, 9, 1]),          # 2 sub-blocks of 32 nodes; ctx 0; 1 node
    ("8b-group4-60nodes", 32, 8, 128, [700, 2049, 90], [60, 60, 16]),          # 4 sub-blocks, a chain-sized block
    ("8b-64nodes-tail", 32, 8, 128, [8192 - 64, 100], [64, 61]),                # tree keys fill the last tile exactly; ragged
    ("group8", 16, 2, 64, [300, 5], [60, 20]),                                  # 8 nodes per tile: 8 sub-blocks
    ("group1", 4, 4, 64, [257], [64]),                                          # one sub-block of 64 rows
])
def test_tree_attn_parity(wf, name, Hq, Hkv, D, ctx_lens, sizes):
    import gpu_harness as H
    binding, ctx = wf
    g = synth.rng(41, sum(map(ord, name)))
    parents, parent, ip = _trees(g, sizes)
    pair = H.make_kv_pair(ctx, ctx_lens, sizes, 2, Hkv, D, seed=len(name))
    Q = synth.normal_bf16(g, (int(ip[-1]), Hq, D), 1.0)
    scale = 1.0 / math.sqrt(D)
    for layer in (0, 1):
        got = _tree_attn(binding, ctx, pair, layer, Q, ip, parent, Hq, scale, max(sizes))
        want = tree_verify.tree_attn(pair.oracle, layer, Q, ip, parent, Hq, scale)
        max_abs, rel_l2 = H.attn_errors(got, want)
        assert max_abs <= ATTN_MAX_ABS and rel_l2 <= ATTN_REL_L2, (name, layer, max_abs, rel_l2)
        # per sequence too: a wrong sub-block offset would hide in the aggregate of a large batch
        for b in range(len(sizes)):
            r0, r1 = int(ip[b]), int(ip[b + 1])
            if r1 > r0:
                ma, rl = H.attn_errors(got[r0:r1], want[r0:r1])
                assert ma <= ATTN_MAX_ABS and rl <= ATTN_REL_L2, (name, layer, b, ma, rl)
    assert ctx.poll_status() == 0
    pair.close()


def test_chain_as_tree_matches_chain_kernel(wf):
    """parent[i] = i - 1 through the tree kernel gives the chain kernel's output up to the last bf16 bit or two (the
    tree kernel keeps one running softmax per row over all tiles, the chain kernel merges two that alternate over the
    tiles), and the oracle's within tolerance."""
    import torch
    import gpu_harness as H
    binding, ctx = wf
    Hq, Hkv, D = 32, 8, 128
    ctx_lens, sizes = [1000, 4096, 33], [16, 8, 16]
    g = synth.rng(43, 1)
    ip = np.array([0, 16, 24, 40], np.int32)
    parent = np.concatenate([synth.chain_parent(n) for n in sizes])
    pair = H.make_kv_pair(ctx, ctx_lens, sizes, 1, Hkv, D, seed=43)
    Q = synth.normal_bf16(g, (40, Hq, D), 1.0)
    scale = 1.0 / math.sqrt(D)
    tree = _tree_attn(binding, ctx, pair, 0, Q, ip, parent, Hq, scale, 16)
    d_q = H.bits_to_bf16_tensor(Q)
    out = torch.zeros_like(d_q)
    ws = torch.empty(binding.wf_verify_attn_workspace_bytes(pair.shape, 3, Hq, 16), dtype=torch.uint8, device="cuda")
    binding.wf_verify_attn(ctx, pair.gpu, 0, d_q, H.i32(ip), 3, Hq, 16, scale, out, ws)
    torch.cuda.synchronize()
    chain = H.bf16_tensor_to_bits(out)
    ma, rl = H.attn_errors(tree, (chain.astype(np.uint32) << 16).view(np.float32).astype(np.float64))
    assert ma <= 2e-3 and rl <= 3e-3, (ma, rl)
    want = verify_attn.verify_attn(pair.oracle, 0, Q, ip, Hq, scale)
    max_abs, rel_l2 = H.attn_errors(tree, want)
    assert max_abs <= ATTN_MAX_ABS and rel_l2 <= ATTN_REL_L2
    pair.close()


def test_tree_attn_batch_of_trees_with_split_pairs(wf):
    """Batch 8 of 60-node trees at mixed contexts (pairs cut across CTAs, partial merges per sub-block).  A repeated launch
    must again be within tolerance (the merge counters reset themselves); with wf_ctx_set_deterministic(1) the merges fold
    in key-range order and three launches give IDENTICAL bits."""
    import gpu_harness as H
    binding, ctx = wf
    Hq, Hkv, D = 32, 8, 128
    g = synth.rng(47, 1)
    ctx_lens = [int(x) for x in g.integers(100, 6000, size=8)]
    sizes = [60] * 6 + [16, 8]
    parents, parent, ip = _trees(g, sizes)
    parent[int(ip[6]):int(ip[7])] = synth.chain_parent(16)   # mixed batch: two chain blocks (diffusion-routed)
    parent[int(ip[7]):int(ip[8])] = synth.chain_parent(8)
    pair = H.make_kv_pair(ctx, ctx_lens, sizes, 1, Hkv, D, seed=47)
    Q = synth.normal_bf16(g, (int(ip[-1]), Hq, D), 1.0)
    scale = 1.0 / math.sqrt(D)
    got = _tree_attn(binding, ctx, pair, 0, Q, ip, parent, Hq, scale, 60)
    again = _tree_attn(binding, ctx, pair, 0, Q, ip, parent, Hq, scale, 60)
    want = tree_verify.tree_attn(pair.oracle, 0, Q, ip, parent, Hq, scale)
    for b in range(8):
        r0, r1 = int(ip[b]), int(ip[b + 1])
        ma, rl = H.attn_errors(got[r0:r1], want[r0:r1])
        assert ma <= ATTN_MAX_ABS and rl <= ATTN_REL_L2, (b, ma, rl)
        ma, rl = H.attn_errors(again[r0:r1], want[r0:r1])
        assert ma <= ATTN_MAX_ABS and rl <= ATTN_REL_L2, (b, ma, rl)
    ctx.set_deterministic(True)
    try:
        d0 = _tree_attn(binding, ctx, pair, 0, Q, ip, parent, Hq, scale, 60)
        for _ in range(2):
            assert np.array_equal(d0, _tree_attn(binding, ctx, pair, 0, Q, ip, parent, Hq, scale, 60))
        ma, rl = H.attn_errors(d0, want)
        assert ma <= ATTN_MAX_ABS and rl <= ATTN_REL_L2
    finally:
        ctx.set_deterministic(False)
    pair.close()


def test_tree_attn_argument_errors(wf):
    import torch
    import gpu_harness as H
    binding, ctx = wf
    pair = H.make_kv_pair(ctx, [10], [4], 1, 2, 64, seed=1)
    q = torch.zeros((4, 4, 64), dtype=torch.bfloat16, device="cuda")
    m = torch.zeros(4, dtype=torch.int64, device="cuda")
    ws = torch.empty(binding.wf_verify_attn_workspace_bytes(pair.shape, 1, 4, 64), dtype=torch.uint8, device="cuda")
    ip = H.i32([0, 4])
    with pytest.raises(binding.WhiFlashError):
        binding.wf_verify_attn_tree(ctx, pair.gpu, 0, q, ip, m, 1, 4, 65, 0.1, q, ws)          # more than 64 nodes
    with pytest.raises(binding.WhiFlashError):
        binding.wf_verify_attn_tree(ctx, pair.gpu, 0, q, ip, None, 1, 4, 4, 0.1, q, ws)        # no masks
    with pytest.raises(binding.WhiFlashError):
        binding.wf_verify_attn_tree(ctx, pair.gpu, 3, q, ip, m, 1, 4, 4, 0.1, q, ws)           # bad layer
    pair.close()


# ------------------------------------------------------------------------------------ acceptance walk
def _run_tree_accept(binding, ctx, logits, tokens, parent, ip, tau, max_nodes):
    import torch
    import gpu_harness as H
    B, V = len(ip) - 1, logits.shape[1]
    outs = {k: torch.full((B,), -7, dtype=torch.int32, device="cuda") for k in ("accept_len", "bonus_token", "route", "n_commit")}
    ent = torch.full((B,), -7.0, dtype=torch.float32, device="cuda")
    path = torch.full((B, max_nodes), -9, dtype=torch.int32, device="cuda")
    tau_arr = np.atleast_1d(np.asarray(tau, dtype=np.float32))
    ws = torch.empty(binding.wf_accept_workspace_bytes(B * max_nodes, V), dtype=torch.uint8, device="cuda")
    binding.wf_accept_tree_entropy_route(ctx, H.f32(logits), V, H.i32(tokens), H.i32(parent), H.i32(ip), B, max_nodes,
                                         H.f32(tau_arr), len(tau_arr) == 1, outs["accept_len"], outs["bonus_token"], ent,
                                         outs["route"], outs["n_commit"], path, max_nodes, ws)
    torch.cuda.synchronize()
    res = {k: v.cpu().numpy() for k, v in outs.items()}
    res["entropy"] = ent.cpu().numpy()
    res["path"] = path.cpu().numpy()
    return res, path, outs["n_commit"]


def _check_tree_accept(res, want, tau):
    B = len(want["accept_len"])
    tau = np.broadcast_to(np.asarray(tau, dtype=np.float64), (B,))
    for k in ("accept_len", "bonus_token", "n_commit", "path"):
        np.testing.assert_array_equal(res[k], want[k], err_msg=k)
    assert np.abs(res["entropy"].astype(np.float64) - want["entropy"]).max() <= ENTROPY_ABS
    near = np.abs(want["entropy"] - tau) < ROUTE_BAND
    np.testing.assert_array_equal(res["route"][~near], want["route"][~near])


@pytest.mark.parametrize("seed", range(6))
def test_tree_accept_tiny(wf, seed):
    binding, ctx = wf
    g = synth.rng(51, seed)
    sizes = [int(x) for x in g.integers(1, 61, size=5)] + [0, 60]
    parents, parent, ip = _trees(g, sizes, depth=8, top_k=4)
    depth = g.integers(0, 9, size=len(sizes))
    spike = g.uniform(0.0, 10.0, size=len(sizes))
    logits, tokens, parent, ip, planned = synth.make_tree_logits_block(g, parents, 4096, 2.0, depth, spike)
    if seed == 0:                                             # duplicate sibling tokens under the root: lowest index wins
        kids = [c for c in range(sizes[6]) if parents[6][c] == 0]
        if len(kids) >= 2:
            tokens[int(ip[6]) + kids[1]] = tokens[int(ip[6]) + kids[0]]
    want = tree_verify.tree_accept_entropy_route(logits, tokens, parent, ip, 2.0, max_path=60)
    res, _, _ = _run_tree_accept(binding, ctx, logits, tokens, parent, ip, 2.0, 60)
    _check_tree_accept(res, want, 2.0)
    assert want["accept_len"].max() >= 1


def test_tree_accept_8b_vocab_and_chain_equivalence(wf):
    """vocab 151936 with 60-node trees; then chain parents through the tree call equal the chain call's outputs."""
    import torch
    import gpu_harness as H
    binding, ctx = wf
    g = synth.rng(53, 1)
    sizes = [60, 60, 16, 0, 60]
    parents, parent, ip = _trees(g, sizes)
    parents[2] = synth.chain_parent(16)
    tau = np.array([1.0, 2.0, 3.0, 2.0, 0.5], np.float32)
    logits, tokens, parent, ip, planned = synth.make_tree_logits_block(g, parents, 151936, 3.0, [8, 3, 16, 0, 0], [2.0, 7.0, 0.0, 0.0, 11.0])
    want = tree_verify.tree_accept_entropy_route(logits, tokens, parent, ip, tau, max_path=60)
    res, _, _ = _run_tree_accept(binding, ctx, logits, tokens, parent, ip, tau, 60)
    _check_tree_accept(res, want, tau)
    assert [int(x) for x in want["accept_len"]] == [len(p) - 1 if p else 0 for p in planned]
    # the chain block through the chain call
    r0, r1 = int(ip[2]), int(ip[3])
    B, V = 1, 151936
    outs = {k: torch.full((B,), -7, dtype=torch.int32, device="cuda") for k in ("accept_len", "bonus_token", "route", "n_commit")}
    ent = torch.full((B,), -7.0, dtype=torch.float32, device="cuda")
    ws = torch.empty(binding.wf_accept_workspace_bytes(16, V), dtype=torch.uint8, device="cuda")
    binding.wf_accept_entropy_route(ctx, H.f32(logits[r0:r1]), V, H.i32(tokens[r0:r1]), H.i32([0, 16]), 1, 16, H.f32(tau[2:3]), True,
                                    outs["accept_len"], outs["bonus_token"], ent, outs["route"], outs["n_commit"], None, ws)
    torch.cuda.synchronize()
    for k in outs:
        assert int(outs[k][0]) == int(res[k][2]), k
    assert float(ent[0]) == float(res["entropy"][2])


# ------------------------------------------------------------------------------------ compaction, end to end
def test_tree_round_end_to_end(wf):
    """masks -> tree attention (2 layers) -> walk -> compaction.  After compaction the GPU cache equals the oracle's
    bit for bit on every live position, seq_len advanced by n_commit, and the chain kernel over the compacted cache
    reproduces the tree outputs of the accepted nodes."""
    import torch
    import gpu_harness as H
    binding, ctx = wf
    Hq, Hkv, D, L = 32, 8, 128, 2
    g = synth.rng(57, 1)
    ctx_lens = [500, 31, 2048, 77]
    sizes = [60, 60, 16, 60]
    parents, parent, ip = _trees(g, sizes)
    parents[2] = synth.chain_parent(16)
    logits, tokens, parent, ip, planned = synth.make_tree_logits_block(g, parents, 4096, 2.0, [8, 2, 9, 0], np.zeros(4))
    pair = H.make_kv_pair(ctx, ctx_lens, sizes, L, Hkv, D, seed=57)
    Q = synth.normal_bf16(g, (int(ip[-1]), Hq, D), 1.0)
    scale = 1.0 / math.sqrt(D)
    tree_out = [_tree_attn(binding, ctx, pair, l, Q, ip, parent, Hq, scale, 60) for l in range(L)]
    res, d_path, d_nc = _run_tree_accept(binding, ctx, logits, tokens, parent, ip, 2.0, 60)
    want = tree_verify.tree_accept_entropy_route(logits, tokens, parent, ip, 2.0, max_path=60)
    _check_tree_accept(res, want, 2.0)
    assert max(len(p) for p in planned) >= 4
    binding.wf_kv_compact_path(ctx, pair.gpu, d_path, 60, d_nc, 4)
    torch.cuda.synchronize()
    tree_verify.compact_path(pair.oracle, want["path"], want["n_commit"])
    assert ctx.poll_status() == 0
    np.testing.assert_array_equal(pair.seq_len.cpu().numpy()[:4], pair.oracle.seq_len[:4])
    assert list(pair.oracle.seq_len[:4]) == [c + len(p) for c, p in zip(ctx_lens, planned)]
    k_bits, v_bits = H.bf16_tensor_to_bits(pair.k_pool), H.bf16_tensor_to_bits(pair.v_pool)
    for b in range(4):
        n = int(pair.oracle.seq_len[b])
        for j0 in range(0, n, 16):
            pg = int(pair.oracle.block_table[b, j0 // 16])
            cnt = min(16, n - j0)
            np.testing.assert_array_equal(k_bits[:, pg, :, :cnt, :], pair.oracle.k_pool[:, pg, :, :cnt, :])
            np.testing.assert_array_equal(v_bits[:, pg, :, :cnt, :], pair.oracle.v_pool[:, pg, :, :cnt, :])
    # chain verification of the accepted queries over the compacted cache == tree outputs of those nodes
    rows = [int(ip[b]) + p for b in range(4) for p in planned[b]]
    ip2 = np.zeros(5, np.int32)
    ip2[1:] = np.cumsum([len(p) for p in planned])
    pair.set_seq_len(ctx_lens)
    d_q = H.bits_to_bf16_tensor(Q[rows])
    ws = torch.empty(binding.wf_verify_attn_workspace_bytes(pair.shape, 4, Hq, 16), dtype=torch.uint8, device="cuda")
    for l in range(L):
        out = torch.zeros_like(d_q)
        binding.wf_verify_attn(ctx, pair.gpu, l, d_q, H.i32(ip2), 4, Hq, 16, scale, out, ws)
        torch.cuda.synchronize()
        chain = H.bf16_tensor_to_bits(out)
        a = (chain.astype(np.uint32) << 16).view(np.float32).astype(np.float64)
        ma, rl = H.attn_errors(tree_out[l][rows], a)
        assert ma <= ATTN_MAX_ABS and rl <= ATTN_REL_L2, (l, ma, rl)
    pair.close()


def test_compact_bad_path_flagged(wf):
    import torch
    import gpu_harness as H
    binding, ctx = wf
    pair = H.make_kv_pair(ctx, [20], [8], 1, 2, 64, seed=3)
    before = pair.k_pool.clone()
    path = H.i32(np.array([[0, 3, 2, -1, -1, -1, -1, -1]], np.int32))      # path[2] = 2 is fine, path[1] = 3 fine; make one bad
    path[0, 2] = 1                                                          # below its step index: not a topological path
    binding.wf_kv_compact_path(ctx, pair.gpu, path, 8, H.i32([3]), 1)
    torch.cuda.synchronize()
    assert ctx.poll_status() == binding.WF_ERR_INVALID_ARG
    assert int(pair.seq_len[0]) == 23
    pair.close()


def test_tree_attn_ignores_everything_outside_the_visible_keys(wf):
    """Every K/V slot that no row may read (beyond ctx + n in the last page, and all unused pages) holds NaN bits: the
    outputs stay finite and equal to the oracle's.  Non-ancestor tree nodes keep finite K/V (they are masked, and a
    masked key must contribute exactly 0, also on the polynomial exp2 path)."""
    import gpu_harness as H
    binding, ctx = wf
    Hq, Hkv, D = 32, 8, 128
    g = synth.rng(71, 1)
    ctx_lens, sizes = [300, 1027, 60], [60, 45, 33]          # ragged tails inside the last tile and the last page
    parents, parent, ip = _trees(g, sizes)
    pair = H.make_kv_pair(ctx, ctx_lens, sizes, 1, Hkv, D, seed=71)
    live_k, live_v = pair.oracle.k_pool.copy(), pair.oracle.v_pool.copy()
    pair.oracle.k_pool[:] = 0x7FC0                           # bf16 NaN everywhere ...
    pair.oracle.v_pool[:] = 0x7FC0
    for b in range(3):                                       # ... except the positions a row may see
        for j in range(ctx_lens[b] + sizes[b]):
            pg, slot = pair.oracle.locate(b, j)
            pair.oracle.k_pool[0, pg, :, slot, :] = live_k[0, pg, :, slot, :]
            pair.oracle.v_pool[0, pg, :, slot, :] = live_v[0, pg, :, slot, :]
    pair.upload_pools()
    Q = synth.normal_bf16(g, (int(ip[-1]), Hq, D), 1.0)
    scale = 1.0 / math.sqrt(D)
    got = _tree_attn(binding, ctx, pair, 0, Q, ip, parent, Hq, scale, 60)
    want = tree_verify.tree_attn(pair.oracle, 0, Q, ip, parent, Hq, scale)
    gf = (got.astype(np.uint32) << 16).view(np.float32)
    assert np.isfinite(gf).all() and np.isfinite(want).all()
    for b in range(3):
        r0, r1 = int(ip[b]), int(ip[b + 1])
        ma, rl = H.attn_errors(got[r0:r1], want[r0:r1])
        assert ma <= ATTN_MAX_ABS and rl <= ATTN_REL_L2, (b, ma, rl)
    pair.close()


def test_compact_long_overlapping_path(wf):
    """A 21-step path [0, 2, 4, .., 40] (a comb tree: every accepted node has a rejected sibling before it): three
    batches of eight moves per column, and every even destination is an earlier step's source.  Two layers, two
    sequences (the second keeps its rows: path[k] = k), bit-exact against the oracle, rows below ctx untouched."""
    import torch
    import gpu_harness as H
    binding, ctx = wf
    ctx_lens, sizes = [37, 100], [41, 12]
    pair = H.make_kv_pair(ctx, ctx_lens, sizes, 2, 8, 128, seed=73)
    path = np.full((2, 64), -1, np.int32)
    path[0, :21] = np.arange(0, 42, 2)
    path[1, :12] = np.arange(12)
    n_commit = np.array([21, 12], np.int32)
    binding.wf_kv_compact_path(ctx, pair.gpu, H.i32(path), 64, H.i32(n_commit), 2)
    torch.cuda.synchronize()
    assert ctx.poll_status() == 0
    tree_verify.compact_path(pair.oracle, path, n_commit)
    np.testing.assert_array_equal(pair.seq_len.cpu().numpy()[:2], pair.oracle.seq_len[:2])
    k_bits, v_bits = H.bf16_tensor_to_bits(pair.k_pool), H.bf16_tensor_to_bits(pair.v_pool)
    for b in range(2):
        n = int(pair.oracle.seq_len[b])
        for j0 in range(0, n, 16):
            pg, cnt = int(pair.oracle.block_table[b, j0 // 16]), min(16, n - j0)
            np.testing.assert_array_equal(k_bits[:, pg, :, :cnt, :], pair.oracle.k_pool[:, pg, :, :cnt, :])
            np.testing.assert_array_equal(v_bits[:, pg, :, :cnt, :], pair.oracle.v_pool[:, pg, :, :cnt, :])
    pair.close()
