"""Pins for oracle O9 (the final backlog token through the drafter layer in full), CPU only.
PAPER.md:119, :206; readings F1-F6.

Each pin is something other than the oracle's own code: pure-Python scalar loops, torch fp64 library routines,
closed forms of degenerate weights, and the separately written (and separately pinned) layer inside O5.
"""

import math

import numpy as np
import pytest

from oracle import bf16, final_token, kv_prefill
from oracle.paged_kv import PagedKV
from paper_2606_07710_b200 import synth


def _setup(L=1, hidden=32, Hq=4, Hkv=2, D=8, F=24, page=4, num_pages=64, max_seqs=2, seed=0, w_std=0.3, theta=1e6):
    g = synth.rng(seed, 11)
    free = synth.draw_free_list(num_pages, g, True)
    kv = PagedKV(L, Hkv, D, page, num_pages, max_seqs, num_pages // max_seqs, free)
    wk = [synth.normal_bf16(g, (hidden, Hkv * D), w_std) for _ in range(L)]
    wv = [synth.normal_bf16(g, (hidden, Hkv * D), w_std) for _ in range(L)]
    dr = kv_prefill.Drafter(wk, wv, kv, theta)
    full = final_token.FullLayer([synth.normal_bf16(g, (hidden, Hq * D), w_std) for _ in range(L)],
                                 [synth.normal_bf16(g, (Hq * D, hidden), w_std) for _ in range(L)],
                                 [synth.normal_bf16(g, (hidden, F), w_std) for _ in range(L)],
                                 [synth.normal_bf16(g, (F, hidden), w_std) for _ in range(L)], Hq)
    return dr, full, g


def _prefill(dr, g, n_rows, hidden):
    """KV-only prefill (O3, pinned elsewhere) of n_rows[b] random rows per sequence; returns the rows."""
    q_indptr = np.concatenate([[0], np.cumsum(n_rows)]).astype(np.int32)
    X = synth.normal_bf16(g, (int(q_indptr[-1]), hidden), 1.0)
    kv_prefill.kv_only_prefill(dr, X, q_indptr, n_rows)
    return X, q_indptr


def test_o9_bruteforce_scalar_loops():
    """Pure-Python loops, no max-shift, explicit RoPE pair formula, explicit GQA map and orientation."""
    hidden, Hq, Hkv, D, F = 6, 2, 1, 4, 5
    dr, full, g = _setup(L=2, hidden=hidden, Hq=Hq, Hkv=Hkv, D=D, F=F, num_pages=16, seed=1)
    X, qi = _prefill(dr, g, [5, 3], hidden)
    b = 1
    got = final_token.final_token_full(dr, full, X[qi[b] + 2], b)
    p = 2
    x = [float(v) for v in bf16.to_f64(X[qi[b] + 2])]
    for l in range(2):
        wq, wo = bf16.to_f64(full.w_q[l]), bf16.to_f64(full.w_o[l])
        wu, wd = bf16.to_f64(full.w_up[l]), bf16.to_f64(full.w_down[l])
        q = [[sum(x[i] * wq[i, h * D + d] for i in range(hidden)) for d in range(D)] for h in range(Hq)]
        for h in range(Hq):
            for r in range(D // 2):
                phi = p * 1e6 ** (-2.0 * r / D)
                a, c = q[h][r], q[h][r + D // 2]
                q[h][r] = a * math.cos(phi) - c * math.sin(phi)
                q[h][r + D // 2] = c * math.cos(phi) + a * math.sin(phi)
        att = []
        for h in range(Hq):
            gk = h // (Hq // Hkv)
            e, acc = [], [0.0] * D
            for j in range(p + 1):
                pg, slot = dr.kv.locate(b, j)
                kj = bf16.to_f64(dr.kv.k_pool[l, pg, gk, slot])
                e.append(math.exp(sum(q[h][d] * kj[d] for d in range(D)) / math.sqrt(D)))
            for j in range(p + 1):
                pg, slot = dr.kv.locate(b, j)
                vj = bf16.to_f64(dr.kv.v_pool[l, pg, gk, slot])
                for d in range(D):
                    acc[d] += e[j] / sum(e) * vj[d]
            att += acc
        y = [x[c] + sum(att[i] * wo[i, c] for i in range(Hq * D)) for c in range(hidden)]
        u = [sum(y[i] * wu[i, f] for i in range(hidden)) for f in range(F)]
        ge = [0.5 * v * (1.0 + math.tanh(math.sqrt(2.0 / math.pi) * (v + 0.044715 * v ** 3))) for v in u]
        h_out = [y[c] + sum(ge[f] * wd[f, c] for f in range(F)) for c in range(hidden)]
        np.testing.assert_allclose(got[l], h_out, rtol=1e-11, atol=1e-12)


def test_o9_against_torch_fp64():
    """torch library routines: linear, scaled_dot_product_attention with GQA, gelu(approximate='tanh')."""
    import torch
    import torch.nn.functional as Fn
    hidden, Hq, Hkv, D, F = 32, 4, 2, 8, 24
    dr, full, g = _setup(L=2, hidden=hidden, Hq=Hq, Hkv=Hkv, D=D, F=F, seed=2)
    X, qi = _prefill(dr, g, [9, 6], hidden)
    for b, n in ((0, 9), (1, 6)):
        got = final_token.final_token_full(dr, full, X[qi[b] + n - 1], b)
        p = n - 1
        x = torch.from_numpy(bf16.to_f64(X[qi[b] + n - 1]))
        for l in range(2):
            Kb, Vb = dr.kv.gather(l, b, n)
            K = torch.from_numpy(bf16.to_f64(Kb)).permute(1, 0, 2)[None]         # [1][Hkv][n][D]
            V = torch.from_numpy(bf16.to_f64(Vb)).permute(1, 0, 2)[None]
            q = Fn.linear(x, torch.from_numpy(bf16.to_f64(full.w_q[l])).T).reshape(Hq, D)
            # rotate-half with torch ops: [lo, hi] -> [lo c - hi s, hi c + lo s]
            inv = 1e6 ** (-torch.arange(0, D, 2, dtype=torch.float64) / D)
            ang = p * inv
            cos, sin = torch.cat([ang.cos(), ang.cos()]), torch.cat([ang.sin(), ang.sin()])
            rot = torch.cat([-q[:, D // 2:], q[:, :D // 2]], dim=1)
            q = q * cos + rot * sin
            att = Fn.scaled_dot_product_attention(q[None, :, None, :], K, V, enable_gqa=True)[0, :, 0, :]
            y = x + Fn.linear(att.reshape(-1), torch.from_numpy(bf16.to_f64(full.w_o[l])).T)
            u = Fn.linear(y, torch.from_numpy(bf16.to_f64(full.w_up[l])).T)
            h = y + Fn.linear(Fn.gelu(u, approximate="tanh"), torch.from_numpy(bf16.to_f64(full.w_down[l])).T)
            np.testing.assert_allclose(got[l], h.numpy(), rtol=1e-10, atol=1e-11)


def test_o9_equals_the_layer_inside_o5():
    """O5 (full_drafter_prefill, written token by token with einsum and pinned through O3) runs the same layer on
    every row; with an identity LM head its discarded 'logits' are the last layer's post-MLP state."""
    hidden, Hq, Hkv, D, F = 16, 4, 2, 4, 12
    for L in (1, 2):
        dr, full, g = _setup(L=L, hidden=hidden, Hq=Hq, Hkv=Hkv, D=D, F=F, num_pages=32, seed=3 + L)
        dr5, _, _ = _setup(L=L, hidden=hidden, Hq=Hq, Hkv=Hkv, D=D, F=F, num_pages=32, seed=3 + L)
        n_rows = [4, 7]
        X, qi = _prefill(dr, g, n_rows, hidden)
        extra = {"w_q": [bf16.to_f64(w) for w in full.w_q], "w_o": [bf16.to_f64(w) for w in full.w_o],
                 "w_up": [bf16.to_f64(w) for w in full.w_up], "w_down": [bf16.to_f64(w) for w in full.w_down],
                 "lm_head": np.eye(hidden)}
        outs = kv_prefill.full_drafter_prefill(dr5, extra, X, qi, n_rows, Hq)
        got = final_token.final_tokens_full(dr, full, X, qi, n_rows, [1, 1])
        np.testing.assert_allclose(got[0][L - 1], outs[n_rows[0] - 1], rtol=1e-11, atol=1e-12)
        np.testing.assert_allclose(got[1][L - 1], outs[-1], rtol=1e-11, atol=1e-12)


def test_o9_degenerate_weights_closed_forms():
    import torch
    import torch.nn.functional as Fn
    hidden, Hq, Hkv, D, F = 32, 4, 2, 8, 24
    dr, full, g = _setup(hidden=hidden, Hq=Hq, Hkv=Hkv, D=D, F=F, seed=6)
    X, qi = _prefill(dr, g, [7, 1], hidden)
    x = bf16.to_f64(X[6])
    zero = lambda w: [np.zeros_like(w[0])]
    # W_O = 0: the attention is irrelevant, h = x + MLP(x)
    f0 = final_token.FullLayer(full.w_q, zero(full.w_o), full.w_up, full.w_down, Hq)
    xt = torch.from_numpy(x)
    mlp = Fn.gelu(xt @ torch.from_numpy(bf16.to_f64(full.w_up[0])), approximate="tanh") @ torch.from_numpy(bf16.to_f64(full.w_down[0]))
    np.testing.assert_allclose(final_token.final_token_full(dr, f0, X[6], 0)[0], (xt + mlp).numpy(), rtol=1e-11)
    # W_down = 0 and W_up = 0 (GELU(0) = 0): h = y = x + att W_O, the same for both
    f1 = final_token.FullLayer(full.w_q, full.w_o, full.w_up, zero(full.w_down), Hq)
    f2 = final_token.FullLayer(full.w_q, full.w_o, zero(full.w_up), full.w_down, Hq)
    h1 = final_token.final_token_full(dr, f1, X[6], 0)[0]
    np.testing.assert_array_equal(h1, final_token.final_token_full(dr, f2, X[6], 0)[0])
    assert np.abs(h1 - x).max() > 1e-3                                   # the attention branch is live
    # a single cached key (sequence 1 holds one token): every head returns that token's V of its group (C11)
    pg, slot = dr.kv.locate(1, 0)
    v = bf16.to_f64(dr.kv.v_pool[0, pg, :, slot, :])                      # [Hkv][D]
    att = np.repeat(v, Hq // Hkv, axis=0).reshape(-1)
    x1 = bf16.to_f64(X[qi[1]])
    np.testing.assert_allclose(final_token.final_token_full(dr, f1, X[qi[1]], 1)[0],
                               x1 + att @ bf16.to_f64(full.w_o[0]), rtol=1e-12)


def test_o9_reads_exactly_positions_0_to_p():
    """The token's own K/V (position p) count; nothing behind p does; the pages may be anywhere."""
    hidden, Hq, Hkv, D, F = 32, 4, 2, 8, 24
    dr, full, g = _setup(hidden=hidden, Hq=Hq, Hkv=Hkv, D=D, F=F, seed=7)
    X, qi = _prefill(dr, g, [6, 0], hidden)
    base = final_token.final_token_full(dr, full, X[5], 0)
    kv = dr.kv
    # garbage in the rest of the last page (positions 6, 7) and in every unreferenced page
    held = set(kv.block_table[0, :kv.pages_held[0]].tolist())
    for pg in range(kv.num_pages):
        if pg not in held:
            kv.k_pool[:, pg] = 0x7FC0
            kv.v_pool[:, pg] = 0x7FC0
    pg, _ = kv.locate(0, 4)
    kv.k_pool[:, pg, :, 2:, :] = 0x7FC0                                   # slots 2, 3 of the page holding 4, 5
    kv.v_pool[:, pg, :, 2:, :] = 0x7FC0
    np.testing.assert_array_equal(final_token.final_token_full(dr, full, X[5], 0), base)
    # the own key is inside the window: changing V at p changes the result; changing position 0 does too
    for pos in (5, 0):
        pg, slot = kv.locate(0, pos)
        keep = kv.v_pool[0, pg, :, slot, :].copy()
        kv.v_pool[0, pg, :, slot, :] = bf16.from_f64(np.full((Hkv, D), 3.0))
        assert np.abs(final_token.final_token_full(dr, full, X[5], 0) - base).max() > 1e-4
        kv.v_pool[0, pg, :, slot, :] = keep


def test_o9_batch_form_selects_last_committed_row():
    """F1: the final token is row n_rows[b]-1 of the block, at position cache_len-1; unselected and empty sequences
    produce nothing; a multi-layer drafter gives one state per layer (F3), each from its own cache and weights."""
    hidden, Hq, Hkv, D, F = 16, 2, 1, 8, 8
    dr, full, g = _setup(L=3, hidden=hidden, Hq=Hq, Hkv=Hkv, D=D, F=F, max_seqs=3, num_pages=48, seed=8)
    X, qi = _prefill(dr, g, [3, 0, 5], hidden)
    out = final_token.final_tokens_full(dr, full, X, qi, [3, 0, 5], [1, 1, 0])
    assert sorted(out) == [0]
    out = final_token.final_tokens_full(dr, full, X, qi, [3, 0, 5], [1, 1, 1])
    assert sorted(out) == [0, 2] and out[2].shape == (3, hidden)
    np.testing.assert_array_equal(out[2], final_token.final_token_full(dr, full, X[qi[2] + 4], 2))
    # layers are independent branches over the same x: swapping two layers' weights and caches swaps the states
    assert np.abs(out[2][0] - out[2][1]).max() > 1e-3
    l0 = final_token.layer_forward(bf16.to_f64(X[qi[2] + 4]), 4, *[bf16.to_f64(a) for a in dr.kv.gather(1, 2, 5)],
                                   bf16.to_f64(full.w_q[1]), bf16.to_f64(full.w_o[1]), bf16.to_f64(full.w_up[1]),
                                   bf16.to_f64(full.w_down[1]), Hq, dr.theta)[0]
    np.testing.assert_array_equal(l0, out[2][1])


def test_o9_gelu_tanh_reference_values():
    """The tanh form against torch, its limits, and its distance from the erf form (they are different functions)."""
    import torch
    u = np.linspace(-6, 6, 1001)
    np.testing.assert_allclose(final_token.gelu_tanh(u), torch.nn.functional.gelu(torch.from_numpy(u), approximate="tanh").numpy(),
                               rtol=1e-12, atol=1e-15)
    assert final_token.gelu_tanh(np.array([0.0]))[0] == 0.0
    assert abs(final_token.gelu_tanh(np.array([10.0]))[0] - 10.0) < 1e-12
    erf_form = torch.nn.functional.gelu(torch.from_numpy(u)).numpy()
    d = np.abs(final_token.gelu_tanh(u) - erf_form).max()
    assert 1e-4 < d < 1e-3
