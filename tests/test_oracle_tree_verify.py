"""Pins for oracle O7 (tree verification: attention, acceptance walk, path compaction), CPU only.

PAPER.md:65, :39, :317, :327; readings T1-T5.  Each test fixes the oracle to something other than
itself: the already-pinned chain oracles (O1, O2) on the chain special case, the library routine (torch fp64
scaled_dot_product_attention with an explicit mask), closed forms, brute force over all root-to-node paths, and
the invariants that tell ancestors from descendants and siblings.
"""

import math

import numpy as np

from oracle import accept_route, bf16, tree_verify, verify_attn
from oracle.paged_kv import PagedKV
from paper_2606_07710_b200 import synth


def _bits(x):
    return synth.f32_to_bf16_bits(np.asarray(x, dtype=np.float32))


def _make_kv(ctx, q, Hkv, D, page=16, L=1, seed=0, fill="normal"):
    g = synth.rng(seed, 1)
    B = len(ctx)
    P = sum(-(-(c + qq) // page) for c, qq in zip(ctx, q)) + 3
    kv = PagedKV(L, Hkv, D, page, P, B, max(-(-(c + qq) // page) for c, qq in zip(ctx, q)) + 1,
                 synth.draw_free_list(P, g, True))
    kv.reserve([c + qq for c, qq in zip(ctx, q)])
    if fill == "normal":
        kv.k_pool[:] = synth.normal_bf16(g, kv.k_pool.shape, 1.0 / math.sqrt(D))
        kv.v_pool[:] = synth.normal_bf16(g, kv.v_pool.shape, 1.0 / math.sqrt(D))
    kv.seq_len[:B] = ctx
    return kv


# ------------------------------------------------------------------ ancestors
def test_ancestors_worked_example():
    """A tree drawn by hand:  0 -> {1, 2}; 1 -> {3}; 2 -> {4, 5}; 4 -> {6}."""
    parent = [-1, 0, 0, 1, 2, 2, 4]
    assert tree_verify.ancestors(parent) == [[0], [0, 1], [0, 2], [0, 1, 3], [0, 2, 4], [0, 2, 5], [0, 2, 4, 6]]
    assert list(tree_verify.ancestor_masks(parent)) == [0b1, 0b11, 0b101, 0b1011, 0b10101, 0b100101, 0b1010101]


def test_ancestors_chain_and_star():
    n = 9
    assert tree_verify.ancestors(synth.chain_parent(n)) == [list(range(i + 1)) for i in range(n)]
    star = [-1] + [0] * (n - 1)
    assert tree_verify.ancestors(star) == [[0]] + [[0, i] for i in range(1, n)]


# ------------------------------------------------------------------ attention
def test_chain_tree_is_causal_verify():
    """parent[i] = i - 1 reduces tree attention to O1 (pinned in test_oracle_attn_accept.py), two sequences."""
    Hq, Hkv, D = 4, 2, 16
    ctx, q = [37, 130], [5, 8]
    kv = _make_kv(ctx, q, Hkv, D, seed=2)
    Q = synth.normal_bf16(synth.rng(2, 2), (sum(q), Hq, D), 1.0)
    ip = np.array([0, 5, 13], np.int32)
    parent = np.concatenate([synth.chain_parent(5), synth.chain_parent(8)])
    got = tree_verify.tree_attn(kv, 0, Q, ip, parent, Hq, 0.25)
    want = verify_attn.verify_attn(kv, 0, Q, ip, Hq, 0.25)
    np.testing.assert_allclose(got, want, rtol=0, atol=1e-13)


def test_matches_library_sdpa_with_explicit_mask():
    """torch fp64 scaled_dot_product_attention over the sequence's whole key range with a boolean mask built here
    from parent pointers by walking up (not from oracle.ancestors)."""
    import torch
    Hq, Hkv, D, n, ctx = 4, 2, 16, 20, 45
    g = synth.rng(7, 3)
    parent = synth.draw_tree(g, n, max_depth=4, top_k=3)
    kv = _make_kv([ctx], [n], Hkv, D, seed=7)
    Q = synth.normal_bf16(g, (n, Hq, D), 1.0)
    got = tree_verify.tree_attn(kv, 0, Q, np.array([0, n], np.int32), parent, Hq, 0.3)
    Kb, Vb = kv.gather(0, 0, ctx + n)
    mask = np.zeros((n, ctx + n), dtype=bool)
    mask[:, :ctx] = True
    for i in range(n):
        j = i
        while j >= 0:
            mask[i, ctx + j] = True
            j = int(parent[j])
    t = lambda a: torch.from_numpy(np.ascontiguousarray(a, dtype=np.float64))
    q = t(bf16.to_f64(Q)).permute(1, 0, 2)                                  # [Hq][n][D]
    k = t(bf16.to_f64(Kb)).permute(1, 0, 2).repeat_interleave(Hq // Hkv, 0)  # [Hq][keys][D]
    v = t(bf16.to_f64(Vb)).permute(1, 0, 2).repeat_interleave(Hq // Hkv, 0)
    want = torch.nn.functional.scaled_dot_product_attention(q, k, v, attn_mask=torch.from_numpy(mask), scale=0.3)
    np.testing.assert_allclose(got, want.permute(1, 0, 2).numpy(), rtol=0, atol=1e-12)


def test_star_tree_closed_form():
    """ctx = 0, every node a child of the root, K = 0: node i > 0 sees exactly {root, itself} with equal weights,
    so O[i] = (V[0] + V[i]) / 2; the root sees only itself.  V[j,:] = j."""
    Hq, Hkv, D, n = 2, 1, 16, 12
    kv = _make_kv([0], [n], Hkv, D, fill="zero")
    for j in range(n):
        pg, slot = kv.locate(0, j)
        kv.v_pool[0, pg, :, slot, :] = _bits(np.full((Hkv, D), float(j)))
    Q = synth.normal_bf16(synth.rng(1, 1), (n, Hq, D), 1.0)
    parent = np.array([-1] + [0] * (n - 1), np.int32)
    out = tree_verify.tree_attn(kv, 0, Q, np.array([0, n], np.int32), parent, Hq, 0.25)
    np.testing.assert_allclose(out[0], 0.0, atol=1e-13)
    for i in range(1, n):
        np.testing.assert_allclose(out[i], i / 2.0, rtol=0, atol=1e-13)


def test_only_ancestors_matter():
    """Changing K/V of a node changes exactly the rows of that node and its descendants (a mask read the wrong
    way round — descendants instead of ancestors — or a causal mask fails this)."""
    Hq, Hkv, D, ctx = 2, 1, 16, 21
    parent = np.array([-1, 0, 0, 1, 2, 2, 4, 1], np.int32)
    n = len(parent)
    kv = _make_kv([ctx], [n], Hkv, D, seed=4)
    Q = synth.normal_bf16(synth.rng(4, 2), (n, Hq, D), 1.0)
    ip = np.array([0, n], np.int32)
    base = tree_verify.tree_attn(kv, 0, Q, ip, parent, Hq, 0.25)
    for node, affected in ((2, {2, 4, 5, 6}), (1, {1, 3, 7}), (6, {6}), (0, set(range(n)))):
        kv2 = _make_kv([ctx], [n], Hkv, D, seed=4)
        pg, slot = kv2.locate(0, ctx + node)
        kv2.k_pool[0, pg, :, slot, :] = _bits(np.full((Hkv, D), 0.5))
        kv2.v_pool[0, pg, :, slot, :] = _bits(np.full((Hkv, D), 3.0))
        out = tree_verify.tree_attn(kv2, 0, Q, ip, parent, Hq, 0.25)
        changed = {i for i in range(n) if np.abs(out[i] - base[i]).max() > 1e-9}
        assert changed == affected


def test_relabelling_siblings_permutes_rows():
    """The same tree in two topological orders (two sibling subtrees swapped): outputs are the same rows permuted."""
    Hq, Hkv, D, ctx = 2, 2, 8, 10
    par_a = np.array([-1, 0, 0, 1, 2], np.int32)          # 0 -> {1 -> {3}, 2 -> {4}}
    perm = [0, 2, 1, 4, 3]                                 # node i of A is node perm[i] of B
    par_b = np.array([-1, 0, 0, 1, 2], np.int32)          # same shape after the swap (symmetric tree)
    n = 5
    kv_a = _make_kv([ctx], [n], Hkv, D, seed=6)
    kv_b = _make_kv([ctx], [n], Hkv, D, seed=6)
    g = synth.rng(6, 5)
    Qa = synth.normal_bf16(g, (n, Hq, D), 1.0)
    Qb = np.empty_like(Qa)
    for i in range(n):
        Qb[perm[i]] = Qa[i]
        pa, sa = kv_a.locate(0, ctx + i)
        pb, sb = kv_b.locate(0, ctx + perm[i])
        kv_b.k_pool[0, pb, :, sb, :] = kv_a.k_pool[0, pa, :, sa, :]
        kv_b.v_pool[0, pb, :, sb, :] = kv_a.v_pool[0, pa, :, sa, :]
    ip = np.array([0, n], np.int32)
    oa = tree_verify.tree_attn(kv_a, 0, Qa, ip, par_a, Hq, 0.35)
    ob = tree_verify.tree_attn(kv_b, 0, Qb, ip, par_b, Hq, 0.35)
    for i in range(n):
        np.testing.assert_allclose(ob[perm[i]], oa[i], rtol=0, atol=1e-13)


# ------------------------------------------------------------------ acceptance walk
def _brute_force_accept(logits, tokens, parent):
    """Every node whose whole root path is 'valid' (each step's token equals the argmax of its parent's row, and no
    lower-index sibling carries that same token) is reachable; the walk ends at the deepest reachable node."""
    n = len(parent)
    g = [int(np.argmax(logits[i])) for i in range(n)]
    best = [0]
    for leaf in range(n):
        path, j = [], leaf
        while j >= 0:
            path.append(j)
            j = int(parent[j])
        path.reverse()
        ok = True
        for u, v in zip(path[:-1], path[1:]):
            if int(tokens[v]) != g[u]:
                ok = False
            if any(int(parent[c]) == u and int(tokens[c]) == g[u] for c in range(v)):
                ok = False
        if ok and len(path) > len(best):
            best = path
    return best, g[best[-1]]


def test_accept_walk_against_brute_force():
    V = 97
    for seed in range(12):
        g = synth.rng(100 + seed, 1)
        parents = [synth.draw_tree(g, int(g.integers(1, 40)), max_depth=6, top_k=4) for _ in range(3)]
        depth = g.integers(0, 7, size=3)
        logits, tokens, parent, ip, planned = synth.make_tree_logits_block(g, parents, V, 2.0, depth, np.zeros(3))
        if seed % 3 == 0:                                   # duplicate sibling tokens: the lowest index wins (T3)
            for b in range(3):
                r0, m = int(ip[b]), len(parents[b])
                kids = [c for c in range(m) if parents[b][c] == 0]
                if len(kids) >= 2:
                    tokens[r0 + kids[1]] = tokens[r0 + kids[0]]
        res = tree_verify.tree_accept_entropy_route(logits, tokens, parent, ip, 2.0)
        for b in range(3):
            r0, r1 = int(ip[b]), int(ip[b + 1])
            path, bonus = _brute_force_accept(logits[r0:r1], tokens[r0:r1], parent[r0:r1])
            a = len(path) - 1
            assert res["accept_len"][b] == a and res["n_commit"][b] == a + 1 and res["bonus_token"][b] == bonus
            assert list(res["path"][b][:a + 1]) == path and (res["path"][b][a + 1:] == -1).all()
            if seed % 3:
                assert path == planned[b]                    # the generator's planted walk is what is accepted
            assert abs(res["entropy"][b] - accept_route.entropy_direct(logits[r0 + path[-1]])) < 1e-12


def test_chain_tree_accept_is_chain_accept():
    """parent[i] = i - 1: same accept_len / bonus / entropy / route as O2 on inputs with planted prefixes."""
    g = synth.rng(5, 5)
    q_lens = [8, 16, 1, 0, 8]
    prefix = [3, 15, 0, 0, 0]
    spike = [0.0, 6.0, 0.0, 0.0, 12.0]
    logits, drafts, ip, _ = synth.make_logits_block(g, q_lens, 211, 2.0, prefix, spike)
    parent = np.concatenate([synth.chain_parent(n) for n in q_lens])
    want = accept_route.accept_entropy_route(logits, drafts, ip, 1.5)
    got = tree_verify.tree_accept_entropy_route(logits, drafts, parent, ip, 1.5)
    for k in ("accept_len", "bonus_token", "n_commit", "route"):
        assert list(got[k]) == list(want[k]), k
    np.testing.assert_allclose(got["entropy"], want["entropy"], rtol=0, atol=0)
    for b, n in enumerate(q_lens):
        a = int(got["accept_len"][b])
        assert list(got["path"][b][:a + 1]) == (list(range(a + 1)) if n else [-1])     # empty block: no path
    assert list(got["accept_len"]) == [3, 15, 0, 0, 0]


def test_entropy_is_read_at_the_last_accepted_node():
    """Two branches with very different entropies: the reported H follows the accepted branch (T4)."""
    V = 64
    logits = np.zeros((3, V), np.float32)
    logits[0, 5] = 4.0                                     # root: argmax 5
    logits[1, 9] = 30.0                                    # node 1: near-deterministic -> H ~ 0
    logits[2, 3] = 0.01                                    # node 2: near-uniform -> H ~ ln V
    parent = np.array([-1, 0, 0], np.int32)
    ip = np.array([0, 3], np.int32)
    r1 = tree_verify.tree_accept_entropy_route(logits, np.array([0, 5, 7], np.int32), parent, ip, 1.0)
    r2 = tree_verify.tree_accept_entropy_route(logits, np.array([0, 7, 5], np.int32), parent, ip, 1.0)
    assert list(r1["path"][0][:2]) == [0, 1] and r1["entropy"][0] < 1e-6 and r1["route"][0] == 0 and r1["bonus_token"][0] == 9
    assert list(r2["path"][0][:2]) == [0, 2] and abs(r2["entropy"][0] - math.log(V)) < 1e-3 and r2["route"][0] == 1
    assert r2["bonus_token"][0] == 3


# ------------------------------------------------------------------ compaction
def test_compaction_leaves_the_chain_cache():
    """After compact_path the cache is what chain decoding of the accepted tokens would have produced: causal O1
    attention of the path's queries over the compacted cache equals the tree attention of those nodes (T5), and
    positions below ctx are untouched."""
    Hq, Hkv, D, L = 4, 2, 16, 2
    ctx = [29, 64]
    g = synth.rng(9, 1)
    parents = [synth.draw_tree(g, 24, max_depth=5, top_k=3), synth.draw_tree(g, 17, max_depth=5, top_k=3)]
    logits, tokens, parent, ip, planned = synth.make_tree_logits_block(g, parents, 101, 2.0, [4, 2], [0, 0])
    kv = _make_kv(ctx, [24, 17], Hkv, D, L=L, seed=9)
    before = [kv.gather(l, b, ctx[b]) for l in range(L) for b in range(2)]
    Q = synth.normal_bf16(g, (int(ip[-1]), Hq, D), 1.0)
    res = tree_verify.tree_accept_entropy_route(logits, tokens, parent, ip, 2.0)
    assert [list(res["path"][b][:res["n_commit"][b]]) for b in range(2)] == planned and len(planned[0]) >= 4
    tree_out = [tree_verify.tree_attn(kv, l, Q, ip, parent, Hq, 0.25) for l in range(L)]
    tree_verify.compact_path(kv, res["path"], res["n_commit"])
    assert list(kv.seq_len[:2]) == [ctx[b] + len(planned[b]) for b in range(2)]
    # chain attention of the accepted queries over the compacted cache
    rows = [int(ip[b]) + p for b in range(2) for p in planned[b]]
    ip2 = np.array([0, len(planned[0]), len(planned[0]) + len(planned[1])], np.int32)
    kv.seq_len[:2] = ctx                                   # O1 convention: the block's rows sit above seq_len
    for l in range(L):
        chain = verify_attn.verify_attn(kv, l, Q[rows], ip2, Hq, 0.25)
        np.testing.assert_allclose(chain, tree_out[l][rows], rtol=0, atol=1e-13)
        for b in range(2):
            Kb, Vb = kv.gather(l, b, ctx[b])
            assert (Kb == before[l * 2 + b][0]).all() and (Vb == before[l * 2 + b][1]).all()


def test_compaction_overlapping_moves():
    """path = [0, 2, 3]: position ctx+2 is both a destination (of node 3) and a source (for slot 1); reading every
    source before writing keeps both rows right."""
    Hkv, D, ctx = 1, 8, 5
    kv = _make_kv([ctx], [4], Hkv, D, fill="zero")
    for j in range(ctx + 4):
        pg, slot = kv.locate(0, j)
        kv.k_pool[0, pg, :, slot, :] = _bits(np.full((Hkv, D), float(j)))
        kv.v_pool[0, pg, :, slot, :] = _bits(np.full((Hkv, D), float(100 + j)))
    tree_verify.compact_path(kv, np.array([[0, 2, 3, -1]], np.int32), np.array([3], np.int32))
    Kb, Vb = kv.gather(0, 0, ctx + 3)
    assert list(bf16.to_f64(Kb)[:, 0, 0]) == [0, 1, 2, 3, 4, 5, 7, 8]
    assert list(bf16.to_f64(Vb)[:, 0, 0]) == [100, 101, 102, 103, 104, 105, 107, 108]
    assert kv.seq_len[0] == ctx + 3
