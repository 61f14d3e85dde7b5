"""Paged KV cache with an explicit block table (oracle; test infrastructure).

The paper uses the Hugging Face cache; paging with 16-token pages
and a shuffled block table is BASELINE.json's extension (north_star "plus a
paged-KV block table", configs[4]).  The allocation order is DESIGN.md reading
C24: the free list is an explicit ordered ring; one reserve call serves sequences
in ascending index, each taking consecutive entries from the head of the ring;
released pages go to the tail.

Pools are uint16 arrays of bf16 bits, [n_layers][num_pages][n_kv_heads][page][head_dim].
"""

import numpy as np


class OutOfPages(Exception):
    pass


class PagedKV:
    def __init__(self, n_layers, n_kv_heads, head_dim, page_size, num_pages, max_seqs,
                 max_pages_per_seq, free_pages=None):
        self.L, self.Hkv, self.D = n_layers, n_kv_heads, head_dim
        self.page, self.num_pages = page_size, num_pages
        self.max_seqs, self.max_pages_per_seq = max_seqs, max_pages_per_seq
        shape = (n_layers, num_pages, n_kv_heads, page_size, head_dim)
        self.k_pool = np.zeros(shape, dtype=np.uint16)
        self.v_pool = np.zeros(shape, dtype=np.uint16)
        self.block_table = np.full((max_seqs, max_pages_per_seq), -1, dtype=np.int32)
        self.seq_len = np.zeros(max_seqs, dtype=np.int32)
        self.pages_held = np.zeros(max_seqs, dtype=np.int32)
        if free_pages is None:
            free_pages = np.arange(num_pages, dtype=np.int32)
        free_pages = np.asarray(free_pages, dtype=np.int32)
        assert len(set(free_pages.tolist())) == len(free_pages)
        # ring buffer of page ids: entries [head, head+count) modulo num_pages are free
        self.free_ring = np.full(num_pages, -1, dtype=np.int32)
        self.free_ring[: len(free_pages)] = free_pages
        self.free_head = 0
        self.free_count = len(free_pages)

    # -- allocation ---------------------------------------------------------
    def reserve(self, add_tokens):
        """Grow block tables so sequence b can hold seq_len[b] + add_tokens[b] tokens.

        Ascending b, consecutive entries from the ring head (C24).  If the ring
        cannot serve the whole call nothing is allocated and OutOfPages is raised.
        """
        add_tokens = np.asarray(add_tokens, dtype=np.int64)
        B = len(add_tokens)
        need = np.zeros(B, dtype=np.int64)
        for b in range(B):
            want = -(-(int(self.seq_len[b]) + int(add_tokens[b])) // self.page)  # ceil
            if want > self.max_pages_per_seq:
                raise OutOfPages(f"seq {b} needs {want} pages > max_pages_per_seq")
            need[b] = max(0, want - int(self.pages_held[b]))
        if need.sum() > self.free_count:
            raise OutOfPages(f"need {need.sum()} pages, {self.free_count} free")
        for b in range(B):
            for _ in range(int(need[b])):
                pg = self.free_ring[self.free_head]
                self.free_head = (self.free_head + 1) % self.num_pages
                self.free_count -= 1
                self.block_table[b, self.pages_held[b]] = pg
                self.pages_held[b] += 1

    def release_seq(self, b):
        """Return sequence b's pages to the ring tail, in block-table order."""
        for i in range(int(self.pages_held[b])):
            tail = (self.free_head + self.free_count) % self.num_pages
            self.free_ring[tail] = self.block_table[b, i]
            self.free_count += 1
            self.block_table[b, i] = -1
        self.pages_held[b] = 0
        self.seq_len[b] = 0

    # -- addressing ---------------------------------------------------------
    def locate(self, b, pos):
        """Logical position -> (physical page, slot) through the block table."""
        pg = int(self.block_table[b, pos // self.page])
        assert pg >= 0, f"seq {b} pos {pos}: no page"
        return pg, pos % self.page

    def write(self, layer, b, pos, k_bits, v_bits):
        """k_bits, v_bits: uint16 [n_kv_heads][head_dim] for one token."""
        pg, slot = self.locate(b, pos)
        self.k_pool[layer, pg, :, slot, :] = k_bits
        self.v_pool[layer, pg, :, slot, :] = v_bits

    def gather(self, layer, b, n=None):
        """Logical view of sequence b: (K, V) uint16 [n][n_kv_heads][head_dim]."""
        if n is None:
            n = int(self.seq_len[b])
        K = np.empty((n, self.Hkv, self.D), dtype=np.uint16)
        V = np.empty((n, self.Hkv, self.D), dtype=np.uint16)
        for j0 in range(0, n, self.page):  # one page at a time: tokens j0 .. j0+cnt-1
            pg, _ = self.locate(b, j0)
            cnt = min(self.page, n - j0)
            K[j0:j0 + cnt] = self.k_pool[layer, pg, :, :cnt, :].transpose(1, 0, 2)
            V[j0:j0 + cnt] = self.v_pool[layer, pg, :, :cnt, :].transpose(1, 0, 2)
        return K, V
