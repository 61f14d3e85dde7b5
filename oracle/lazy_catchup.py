"""O4 — Lazy Catch-up (oracle; test infrastructure, see oracle/__init__.py).

PAPER.md:117 (§3.4): "we defer the updates for the inactive drafter entirely: no
work is performed for the inactive drafter until a switch is committed.  Upon
preparing for a switch, the incoming drafter prefills its KV cache over all tokens
accepted during its inactivity as a single batched operation.  We refer to these
tokens ... as backlog tokens.  Their quantity defines the size of the catch-up
prefill at each switch."  PAPER.md:204: "the tokens accepted by the target are
identical under both schemes" -> a flush leaves the cache identical to eager
per-round appends.

DESIGN.md readings: C20 the backlog cap is a parameter; an enqueue that would
exceed it flushes that sequence first and never drops a row.  C21 the flush runs
in the round whose route differs from the sequence's current drafter, after that
round's own rows were enqueued.  Backlog row j of sequence b has position
cache_len[b] + j (FIFO).
"""

import numpy as np

from .kv_prefill import Drafter, append_rows


class LazyCatchup:
    def __init__(self, drafter: Drafter, backlog_cap):
        self.drafter = drafter
        self.cap = int(backlog_cap)
        S = drafter.kv.max_seqs
        self.backlog = np.zeros((S, self.cap, drafter.hidden), dtype=np.uint16)
        self.backlog_len = np.zeros(S, dtype=np.int32)

    def flush(self, flush_mask=None, B=None):
        """KV-only prefill (O3) of every flagged sequence's whole backlog, FIFO order."""
        if B is None:
            B = self.drafter.kv.max_seqs
        rows = []
        for b in range(B):
            on = True if flush_mask is None else bool(flush_mask[b])
            n = int(self.backlog_len[b]) if on else 0
            rows.append(self.backlog[b, :n].copy())
        out = append_rows(self.drafter, rows)
        for b in range(B):
            if len(rows[b]):
                self.backlog_len[b] = 0
        return out

    def enqueue(self, hidden_bits, q_indptr, n_rows, idle_mask):
        """Append rows 0..n_rows[b]-1 of each flagged sequence's block to its backlog.

        If that would exceed the cap, the sequence is flushed first (C20); the
        forced flushes of one call are one batched prefill.
        """
        B = len(q_indptr) - 1
        over = np.zeros(B, dtype=bool)
        for b in range(B):
            if idle_mask[b] and int(self.backlog_len[b]) + int(n_rows[b]) > self.cap:
                over[b] = True
        if over.any():
            self.flush(over, B)
        for b in range(B):
            if not idle_mask[b]:
                continue
            n = int(n_rows[b])
            assert n <= self.cap, "a single round's rows must fit the backlog"
            r0 = int(q_indptr[b])
            l0 = int(self.backlog_len[b])
            self.backlog[b, l0:l0 + n] = hidden_bits[r0:r0 + n]
            self.backlog_len[b] = l0 + n
