"""Pins for oracle O1 (verify attention) and O2 (accept / entropy / route), CPU only.

Each test fixes the oracle to something other than itself: a closed form, an
invariant, a textbook special case, or a pure-Python brute force written here from
the definition (readings C1-C12).
"""

import math

import numpy as np
import pytest

from oracle import accept_route, bf16, verify_attn
from oracle.paged_kv import PagedKV
from paper_2606_07710_b200 import synth


def _bits(x):
    return synth.f32_to_bf16_bits(np.asarray(x, dtype=np.float32))


def _make_kv(ctx, q, Hkv, D, page=16, L=1, shuffled=True, seed=0, fill="normal", extra_pages=3):
    g = synth.rng(seed, 1)
    B = len(ctx)
    need = sum(-(-(c + q) // page) for c in ctx)
    P = need + extra_pages
    free = synth.draw_free_list(P, g, shuffled)
    kv = PagedKV(L, Hkv, D, page, P, B, max(-(-(c + q) // page) for c in ctx) + 1, free)
    kv.reserve([c + q for c in ctx])
    if fill == "normal":
        kv.k_pool[:] = synth.normal_bf16(g, kv.k_pool.shape, 1.0 / math.sqrt(D))
        kv.v_pool[:] = synth.normal_bf16(g, kv.v_pool.shape, 1.0 / math.sqrt(D))
    kv.seq_len[:B] = ctx
    return kv


# ------------------------------------------------------------------ O1 pins
def test_o1_brute_force_tiny():
    """(viii) triple loop without any vectorisation, D=8, ctx<=40, two sequences, GQA 4/2."""
    Hq, Hkv, D, q = 4, 2, 8, 3
    ctx = [37, 5]
    kv = _make_kv(ctx, q, Hkv, D, page=4, seed=3)
    g = synth.rng(3, 2)
    Q = synth.normal_bf16(g, (2 * q, Hq, D), 1.0)
    q_indptr = np.array([0, q, 2 * q], dtype=np.int32)
    scale = 1.0 / math.sqrt(D)
    out = verify_attn.verify_attn(kv, 0, Q, q_indptr, Hq, scale)
    kf, vf, qf = bf16.to_f64(kv.k_pool), bf16.to_f64(kv.v_pool), bf16.to_f64(Q)
    for b in range(2):
        for i in range(q):
            for h in range(Hq):
                gk = h // (Hq // Hkv)
                scores = []
                for j in range(ctx[b] + i + 1):
                    pg = kv.block_table[b, j // 4]
                    s = 0.0
                    for d in range(D):
                        s += qf[b * q + i, h, d] * kf[0, pg, gk, j % 4, d]
                    scores.append(s * scale)
                den = sum(math.exp(s) for s in scores)          # naive softmax, no max-shift
                for d in range(D):
                    acc = 0.0
                    for j, s in enumerate(scores):
                        pg = kv.block_table[b, j // 4]
                        acc += math.exp(s) / den * vf[0, pg, gk, j % 4, d]
                    assert abs(out[b * q + i, h, d] - acc) < 1e-12


def test_o1_causal_off_by_one_closed_form():
    """(ii) K == 0 -> uniform weights; V[j,:] = j -> O[i] = (ctx+i)/2 exactly."""
    Hq, Hkv, D, q, ctx = 2, 1, 16, 8, 100
    kv = _make_kv([ctx], q, Hkv, D, fill="zero")
    for j in range(ctx + q):
        pg, slot = kv.locate(0, j)
        kv.v_pool[0, pg, :, slot, :] = _bits(np.full((Hkv, D), float(j)))   # j <= 255 exact in bf16
    Q = synth.normal_bf16(synth.rng(1, 1), (q, Hq, D), 1.0)
    out = verify_attn.verify_attn(kv, 0, Q, np.array([0, q], np.int32), Hq, 0.25)
    for i in range(q):
        np.testing.assert_allclose(out[i], (ctx + i) / 2.0, rtol=0, atol=1e-12)


def test_o1_constant_v_and_dominant_key():
    """(iii) all V rows equal -> O = that row.  (iv) one huge score -> O = its V row."""
    Hq, Hkv, D, q, ctx = 4, 2, 16, 4, 50
    kv = _make_kv([ctx], q, Hkv, D, seed=5)
    row = synth.normal_bf16(synth.rng(5, 9), (Hkv, D), 1.0)
    saved_v = kv.v_pool.copy()
    kv.v_pool[:] = row[None, None, :, None, :]
    Q = synth.normal_bf16(synth.rng(5, 3), (q, Hq, D), 1.0)
    ip = np.array([0, q], np.int32)
    out = verify_attn.verify_attn(kv, 0, Q, ip, Hq, 0.25)
    for h in range(Hq):
        np.testing.assert_allclose(out[:, h], np.broadcast_to(bf16.to_f64(row[h // 2]), (q, D)), atol=1e-14)
    # dominant key at position 7: K[7] = 64 * sign pattern, Q = same pattern -> score ~ 64*D*scale
    kv.v_pool[:] = saved_v
    pat = np.where(np.arange(D) % 2 == 0, 1.0, -1.0)
    pg, slot = kv.locate(0, 7)
    kv.k_pool[0, pg, :, slot, :] = _bits(np.broadcast_to(64.0 * pat, (Hkv, D)))
    Qd = _bits(np.broadcast_to(8.0 * pat, (q, Hq, D)))
    out = verify_attn.verify_attn(kv, 0, Qd, ip, Hq, 0.25)
    for h in range(Hq):
        np.testing.assert_allclose(out[:, h], np.broadcast_to(bf16.to_f64(kv.v_pool[0, pg, h // 2, slot]), (q, D)),
                                   atol=1e-12)


def test_o1_page_permutation_and_garbage_invariance():
    """(v) physical page order does not matter (bit-exact); (vi) NaN in unreferenced pages and in
    slots beyond ctx+q is never read."""
    Hq, Hkv, D, q = 4, 2, 16, 5
    ctx = [33, 18]
    a = _make_kv(ctx, q, Hkv, D, shuffled=False, seed=11)
    b = _make_kv(ctx, q, Hkv, D, shuffled=True, seed=11)
    # same logical content in b as in a
    for s in range(2):
        Ka, Va = a.gather(0, s, ctx[s] + q)
        for j in range(ctx[s] + q):
            b.write(0, s, j, Ka[j], Va[j])
    # garbage: NaN (0x7FC0) everywhere not logically visible
    nan = np.uint16(0x7FC0)
    used = np.zeros(b.k_pool.shape[1:4:2], dtype=bool)   # [pages][slots]
    for s in range(2):
        for j in range(ctx[s] + q):
            pg, slot = b.locate(s, j)
            used[pg, slot] = True
    for pg in range(b.num_pages):
        for slot in range(b.page):
            if not used[pg, slot]:
                b.k_pool[:, pg, :, slot, :] = nan
                b.v_pool[:, pg, :, slot, :] = nan
    Q = synth.normal_bf16(synth.rng(11, 3), (2 * q, Hq, D), 1.0)
    ip = np.array([0, q, 2 * q], np.int32)
    oa = verify_attn.verify_attn(a, 0, Q, ip, Hq, 0.25)
    ob = verify_attn.verify_attn(b, 0, Q, ip, Hq, 0.25)
    assert np.array_equal(oa, ob)
    assert np.isfinite(ob).all()


def test_o1_single_query_textbook_and_group_sharing():
    """(i) q=1, Hq=Hkv is textbook single-query softmax attention (scipy softmax).
    (vii) two heads of one GQA group with equal Q give equal O; heads of different groups do not."""
    from scipy.special import softmax
    Hq, Hkv, D, ctx = 2, 2, 32, 70
    kv = _make_kv([ctx], 1, Hkv, D, seed=21)
    Q = synth.normal_bf16(synth.rng(21, 3), (1, Hq, D), 1.0)
    out = verify_attn.verify_attn(kv, 0, Q, np.array([0, 1], np.int32), Hq, 1 / math.sqrt(D))
    K, V = kv.gather(0, 0, ctx + 1)
    K, V = bf16.to_f64(K), bf16.to_f64(V)
    for h in range(Hq):
        p = softmax(K[:, h] @ bf16.to_f64(Q[0, h]) / math.sqrt(D))
        np.testing.assert_allclose(out[0, h], p @ V[:, h], rtol=1e-12, atol=1e-14)
    # group sharing
    Hq, Hkv = 4, 2
    kv = _make_kv([ctx], 2, Hkv, D, seed=22)
    Q = synth.normal_bf16(synth.rng(22, 3), (2, Hq, D), 1.0)
    Q[:, 1] = Q[:, 0]
    Q[:, 3] = Q[:, 0]
    out = verify_attn.verify_attn(kv, 0, Q, np.array([0, 2], np.int32), Hq, 0.2)
    assert np.array_equal(out[:, 0], out[:, 1])
    assert not np.allclose(out[:, 0], out[:, 3])


def test_o1_row_function_matches_full_and_empty_block():
    Hq, Hkv, D, q = 4, 2, 16, 6
    kv = _make_kv([20, 0, 9], q, Hkv, D, seed=31)
    Q = synth.normal_bf16(synth.rng(31, 3), (q + 0 + 3, Hq, D), 1.0)
    ip = np.array([0, q, q, q + 3], np.int32)            # middle sequence has an empty block
    out = verify_attn.verify_attn(kv, 0, Q, ip, Hq, 0.25)
    r = verify_attn.verify_attn_row(kv, 0, 2, Q[q + 1], 1, Hq, 0.25, heads=[3])
    assert np.array_equal(r[0], out[q + 1, 3])
    r = verify_attn.verify_attn_row(kv, 0, 0, Q[4], 4, Hq, 0.25)
    assert np.array_equal(r, out[4])


# ------------------------------------------------------------------ O2 pins
def _naive_entropy(z):
    ps = [math.exp(v) for v in z]
    t = sum(ps)
    return -sum((p / t) * math.log(p / t) for p in ps if p > 0)


def test_o2_entropy_closed_forms():
    """(iv) constant row -> ln V; (v) two equal maxima, rest -inf -> ln 2; (vi) one-hot -> 0;
    (vii) shift invariance."""
    for V in (4096, 151936):
        assert abs(accept_route.entropy_direct(np.full(V, 1.25, np.float32)) - math.log(V)) < 1e-10
    assert abs(math.log(4096) - 8.3178) < 1e-4 and abs(math.log(151936) - 11.9312) < 1e-4
    z = np.full(1000, -np.inf, np.float32)
    z[3] = z[977] = 0.5
    assert abs(accept_route.entropy_direct(z) - math.log(2)) < 1e-14
    z = np.full(1000, -np.inf, np.float32)
    z[5] = 3.0
    assert accept_route.entropy_direct(z) == 0.0
    g = synth.rng(7, 1)
    z = synth.normal_f32(g, 5000, 2.0).astype(np.float64)
    assert abs(accept_route.entropy_direct(z) - accept_route.entropy_direct(z + 123.456)) < 1e-9


def test_o2_entropy_bruteforce_and_chunked():
    """(ix) brute force on V<=16 vs a naive softmax; (viii) chunked combine == direct."""
    g = synth.rng(8, 1)
    for V in (2, 3, 7, 16):
        z = synth.normal_f32(g, V, 2.0)
        assert abs(accept_route.entropy_direct(z) - _naive_entropy([float(v) for v in z])) < 1e-12
    z = synth.normal_f32(g, 151936, 3.0)
    z[100:300] = -np.inf
    d = accept_route.entropy_direct(z)
    for chunk in (64, 200, 4096, 151936):                # chunk 200 makes an all -inf chunk
        assert abs(accept_route.entropy_chunked(z, chunk) - d) < 1e-10


def test_o2_gaussian_entropy_statistic():
    """(x) Gaussian rows: H ~ ln V - sigma^2/2 (large-V approximation)."""
    g = synth.rng(9, 1)
    hs = [accept_route.entropy_direct(synth.normal_f32(g, 4096, 2.0)) for _ in range(32)]
    assert abs(np.mean(hs) - (math.log(4096) - 2.0)) < 0.15
    # at sigma = 3 the finite-V sum is dominated by a few large terms: only a band holds
    h = accept_route.entropy_direct(synth.normal_f32(g, 151936, 3.0))
    assert 5.0 < h < math.log(151936) - 3.0


def _bruteforce_accept(logits, drafts, tau):
    """Definition straight from C6/C7: first mismatch between draft j and argmax of row j-1."""
    gamma = len(logits) - 1
    am = []
    for row in logits:
        best, bi = -math.inf, -1
        for i, v in enumerate(row):
            if v > best:                                   # strict > keeps the lowest index on ties
                best, bi = float(v), i
        am.append(bi)
    a = gamma
    for j in range(1, gamma + 1):
        if drafts[j] != am[j - 1]:
            a = j - 1
            break
    h = _naive_entropy([float(v) for v in logits[a]])
    return a, am[a], a + 1, (1 if h > tau else 0), h


def test_o2_accept_special_cases():
    """(i) drafts == target argmax -> a = gamma; (ii) first draft wrong -> a = 0, bonus = g_0;
    (iii) a <= gamma; ties take the lowest token id (C7)."""
    g = synth.rng(10, 1)
    gamma, V = 7, 64
    logits = synth.normal_f32(g, (gamma + 1, V), 2.0)
    am = logits.argmax(axis=1)
    drafts = np.zeros(gamma + 1, np.int32)
    drafts[1:] = am[:-1]
    ip = np.array([0, gamma + 1], np.int32)
    r = accept_route.accept_entropy_route(logits, drafts, ip, 2.0)
    assert r["accept_len"][0] == gamma and r["bonus_token"][0] == am[gamma] and r["n_commit"][0] == gamma + 1
    drafts2 = drafts.copy()
    drafts2[1] = (am[0] + 1) % V
    r = accept_route.accept_entropy_route(logits, drafts2, ip, 2.0)
    assert r["accept_len"][0] == 0 and r["bonus_token"][0] == am[0] and r["n_commit"][0] == 1
    # ties: rows with duplicated maxima
    logits[2, 40] = logits[2, 11] = 50.0
    drafts3 = drafts.copy()
    drafts3[3] = 11
    r = accept_route.accept_entropy_route(logits, drafts3, ip, 2.0)
    assert r["accept_len"][0] == gamma
    drafts3[3] = 40
    r = accept_route.accept_entropy_route(logits, drafts3, ip, 2.0)
    assert r["accept_len"][0] == 2 and r["bonus_token"][0] == 11


def test_o2_bruteforce_batches_and_route_direction():
    """Random small batches vs the brute force; route: H > tau -> AR(1), else diffusion(0) (C1, C2);
    entropy is taken at row a (C3); seq_len advances by a+1."""
    g = synth.rng(11, 1)
    for trial in range(40):
        B = int(g.integers(1, 5))
        q_lens = g.integers(0, 6, size=B)
        V = 12
        u = [int(g.integers(0, max(1, ql))) for ql in q_lens]
        logits, drafts, ip, _ = synth.make_logits_block(g, q_lens, V, 2.0, u, g.uniform(0, 6, size=B))
        tau = g.uniform(0.5, 2.4, size=B)
        kv = PagedKV(1, 1, 8, 16, 4, B, 2)
        kv.seq_len[:] = 10
        r = accept_route.accept_entropy_route(logits, drafts, ip, tau, kv)
        for b in range(B):
            if q_lens[b] == 0:
                assert r["n_commit"][b] == 0 and kv.seq_len[b] == 10
                continue
            a, bonus, nc, route, h = _bruteforce_accept(logits[ip[b]:ip[b + 1]], drafts[ip[b]:ip[b + 1]], tau[b])
            assert (r["accept_len"][b], r["bonus_token"][b], r["n_commit"][b], r["route"][b]) == (a, bonus, nc, route)
            assert a == min(u[b], q_lens[b] - 1)            # the generator's planted outcome
            assert abs(r["entropy"][b] - h) < 1e-12
            assert kv.seq_len[b] == 10 + a + 1
            assert 0 <= a <= q_lens[b] - 1
    # direction and tie: H == tau -> diffusion
    z = np.zeros((1, 8), np.float32)
    r = accept_route.accept_entropy_route(z, np.zeros(1, np.int32), np.array([0, 1], np.int32), math.log(8))
    assert r["route"][0] == 0
    r = accept_route.accept_entropy_route(z, np.zeros(1, np.int32), np.array([0, 1], np.int32), math.log(8) - 1e-9)
    assert r["route"][0] == 1


def test_o2_spike_moves_entropy_both_sides():
    """The generator's spike puts H on both sides of tau = 2.0 at the configs' (V, sigma)."""
    g = synth.rng(12, 1)
    for V, sigma in ((4096, 2.0), (151936, 3.0)):
        hs = []
        for spike in (0.0, 12.0):
            logits, drafts, ip, _ = synth.make_logits_block(g, [4], V, sigma, [2], [spike])
            hs.append(accept_route.accept_entropy_route(logits, drafts, ip, 2.0)["entropy"][0])
        assert hs[0] > 2.0 > hs[1]
