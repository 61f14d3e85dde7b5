"""Shared helpers for the `-m gpu` parity tests: mirror oracle-side state (numpy) onto the GPU.

Test infrastructure.  The CUDA path is reached only through paper_2606_07710_b200.binding
(the C-ABI); expected values come only from oracle/.
"""

import math

import numpy as np

from oracle.paged_kv import PagedKV as OraclePagedKV
from paper_2606_07710_b200 import synth


def torch_mod():
    import torch
    return torch


def bits_to_bf16_tensor(bits, device="cuda"):
    torch = torch_mod()
    a = np.ascontiguousarray(bits, dtype=np.uint16).view(np.int16)
    return torch.from_numpy(a).to(device).view(torch.bfloat16)


def bf16_tensor_to_bits(t):
    torch = torch_mod()
    return t.detach().contiguous().view(torch.int16).cpu().numpy().view(np.uint16)


def i32(a, device="cuda"):
    torch = torch_mod()
    return torch.from_numpy(np.ascontiguousarray(a, dtype=np.int32)).to(device)


def f32(a, device="cuda"):
    torch = torch_mod()
    return torch.from_numpy(np.ascontiguousarray(a, dtype=np.float32)).to(device)


class KvPair:
    """An oracle PagedKV and its GPU twin created from the same free list."""

    def __init__(self, ctx, n_layers, n_kv_heads, head_dim, num_pages, max_seqs, max_pages_per_seq,
                 free_pages, page_size=16):
        from paper_2606_07710_b200 import binding
        torch = torch_mod()
        self.oracle = OraclePagedKV(n_layers, n_kv_heads, head_dim, page_size, num_pages, max_seqs,
                                    max_pages_per_seq, free_pages)
        self.shape = binding.KvShape(n_layers, n_kv_heads, head_dim, page_size, num_pages, max_seqs,
                                     max_pages_per_seq)
        pool_shape = (n_layers, num_pages, n_kv_heads, page_size, head_dim)
        self.k_pool = torch.zeros(pool_shape, dtype=torch.bfloat16, device="cuda")
        self.v_pool = torch.zeros(pool_shape, dtype=torch.bfloat16, device="cuda")
        self.block_table = torch.full((max_seqs, max_pages_per_seq), -1, dtype=torch.int32, device="cuda")
        self.seq_len = torch.zeros(max_seqs, dtype=torch.int32, device="cuda")
        self.gpu = binding.PagedKV(ctx, self.shape, self.k_pool, self.v_pool, self.block_table, self.seq_len,
                                   np.asarray(free_pages, dtype=np.int32))
        self.ctx = ctx

    def reserve(self, add_tokens):
        add = np.asarray(add_tokens, dtype=np.int32)
        self.oracle.reserve(add)
        self.gpu.reserve(i32(add), len(add))

    def set_seq_len(self, lens):
        lens = np.asarray(lens, dtype=np.int32)
        self.oracle.seq_len[: len(lens)] = lens
        self.seq_len[: len(lens)] = i32(lens)

    def fill_random(self, g, std):
        self.oracle.k_pool[:] = synth.normal_bf16(g, self.oracle.k_pool.shape, std)
        self.oracle.v_pool[:] = synth.normal_bf16(g, self.oracle.v_pool.shape, std)
        self.upload_pools()

    def upload_pools(self):
        self.k_pool.copy_(bits_to_bf16_tensor(self.oracle.k_pool))
        self.v_pool.copy_(bits_to_bf16_tensor(self.oracle.v_pool))

    def assert_tables_equal(self):
        torch_mod().cuda.synchronize()
        np.testing.assert_array_equal(self.block_table.cpu().numpy(), self.oracle.block_table)
        np.testing.assert_array_equal(self.seq_len.cpu().numpy(), self.oracle.seq_len)

    def close(self):
        self.gpu.close()


def make_kv_pair(ctx, ctx_lens, q_lens, n_layers, n_kv_heads, head_dim, seed, shuffled=True, extra_pages=5,
                 kv_std=None, fill=True):
    """Paged cache holding ctx_lens[b] final tokens plus the block's q_lens[b] tokens (reading C10)."""
    g = synth.rng(seed, 101)
    B = len(ctx_lens)
    tot = [int(c) + int(q) for c, q in zip(ctx_lens, q_lens)]
    need = sum(-(-t // 16) for t in tot)
    P = need + extra_pages
    free = synth.draw_free_list(P, g, shuffled)
    pair = KvPair(ctx, n_layers, n_kv_heads, head_dim, P, B, max(-(-t // 16) for t in tot) + 2, free)
    pair.reserve(tot)
    if fill:
        pair.fill_random(g, kv_std if kv_std is not None else 1.0 / math.sqrt(head_dim))
    pair.set_seq_len(ctx_lens)
    return pair


def attn_errors(got_bits, want_f64):
    got = (np.asarray(got_bits, dtype=np.uint16).astype(np.uint32) << 16).view(np.float32).astype(np.float64)
    diff = got - want_f64
    max_abs = float(np.abs(diff).max()) if diff.size else 0.0
    rel_l2 = float(np.sqrt((diff ** 2).sum() / max((want_f64 ** 2).sum(), 1e-300)))
    return max_abs, rel_l2


class DrafterPair:
    """An oracle drafter (+ LazyCatchup) and its GPU twin with identical weights and free list."""

    def __init__(self, ctx, n_layers, hidden, n_kv_heads, head_dim, num_pages, max_seqs, max_pages_per_seq,
                 free_pages, seed, backlog_cap=32, theta=1e6, max_pos=40000, w_std=0.02, weights=None):
        from oracle.kv_prefill import Drafter as OracleDrafter
        from oracle.lazy_catchup import LazyCatchup
        from paper_2606_07710_b200 import binding
        torch = torch_mod()
        self.kvp = KvPair(ctx, n_layers, n_kv_heads, head_dim, num_pages, max_seqs, max_pages_per_seq, free_pages)
        N = n_kv_heads * head_dim
        if weights is None:
            g = synth.rng(seed, 303)
            weights = ([synth.normal_bf16(g, (hidden, N), w_std) for _ in range(n_layers)],
                       [synth.normal_bf16(g, (hidden, N), w_std) for _ in range(n_layers)])
        self.weights = weights
        self.oracle = OracleDrafter(weights[0], weights[1], self.kvp.oracle, theta)
        self.oracle_lazy = LazyCatchup(self.oracle, backlog_cap)
        self.w_k = [bits_to_bf16_tensor(w) for w in weights[0]]
        self.w_v = [bits_to_bf16_tensor(w) for w in weights[1]]
        self.backlog = torch.zeros((max_seqs, max(backlog_cap, 1), hidden), dtype=torch.bfloat16, device="cuda")
        self.backlog_len = torch.zeros(max_seqs, dtype=torch.int32, device="cuda")
        self.shape = binding.DrafterShape(n_layers, hidden, n_kv_heads, head_dim, theta, max_pos, backlog_cap)
        self.gpu = binding.Drafter(ctx, self.shape, self.w_k, self.w_v, self.kvp.gpu, self.backlog, self.backlog_len)
        self.ctx = ctx

    def gather_gpu(self, layer, b, n):
        """Logical (K, V) bits [n][Hkv][D] of sequence b read back from the GPU pools through its block table."""
        kv = self.kvp
        if n == 0:
            z = np.empty((0, kv.oracle.Hkv, kv.oracle.D), dtype=np.uint16)
            return z, z.copy()
        pages = kv.block_table[b, : -(-n // 16)].long()
        K = bf16_tensor_to_bits(kv.k_pool[layer][pages].permute(0, 2, 1, 3).reshape(-1, kv.oracle.Hkv, kv.oracle.D)[:n])
        V = bf16_tensor_to_bits(kv.v_pool[layer][pages].permute(0, 2, 1, 3).reshape(-1, kv.oracle.Hkv, kv.oracle.D)[:n])
        return K, V

    def close(self):
        self.gpu.close()
        self.kvp.close()


def rel_l2(got_bits, want_f64):
    got = (np.asarray(got_bits, dtype=np.uint16).astype(np.uint32) << 16).view(np.float32).astype(np.float64)
    return float(np.sqrt(((got - want_f64) ** 2).sum() / max((want_f64 ** 2).sum(), 1e-300)))


def bf16_f64(bits):
    return (np.asarray(bits, dtype=np.uint16).astype(np.uint32) << 16).view(np.float32).astype(np.float64)
