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

    def round(self, hidden_bits, q_indptr, n_rows, idle_mask, flush_mask):
        """Everything one round asks of this drafter (readings C21, C22), as ONE batched prefill:

          not idle        the drafter is active for b: its backlog (normally empty), then rows 0..n_rows[b]-1;
          idle and flush  b switches to this drafter: its backlog, then this round's rows ("enqueue, then flush", C21);
          idle, no flush  the rows are enqueued; a backlog they would overflow is prefilled first (C20).

        The rows that are prefilled go through ONE append_rows call (one reserve, ascending b, C24), so the cache
        CONTENTS equal those of the separate calls (kv_only_prefill for the active sequences, enqueue, flush) and only
        the physical page order can differ from theirs; the enqueues follow.
        """
        B = len(q_indptr) - 1
        rows, enq = [], []
        for b in range(B):
            n, r0, l0 = int(n_rows[b]), int(q_indptr[b]), int(self.backlog_len[b])
            idle = bool(idle_mask[b]) if idle_mask is not None else False
            fl = bool(flush_mask[b]) if flush_mask is not None else False
            blk = np.asarray(hidden_bits[r0:r0 + n], dtype=np.uint16)
            if not idle or fl:
                rows.append(np.concatenate([self.backlog[b, :l0], blk], axis=0))
                enq.append(None)
            else:
                assert n <= self.cap, "a single round's rows must fit the backlog"
                rows.append(self.backlog[b, :l0].copy() if l0 + n > self.cap else blk[:0])
                enq.append(blk)
        out = append_rows(self.drafter, rows)
        for b in range(B):
            if len(rows[b]) and (enq[b] is None or int(self.backlog_len[b]) + len(enq[b]) > self.cap):
                self.backlog_len[b] = 0
            if enq[b] is not None:
                l0 = int(self.backlog_len[b])
                self.backlog[b, l0:l0 + len(enq[b])] = enq[b]
                self.backlog_len[b] = l0 + len(enq[b])
        return out


def switch_masks(route, cur, code):
    """Who is idle for the drafter with route code `code`, and who switches to it this round (reading C21).

    PAPER.md:117: "no work is performed for the inactive drafter until a switch is committed.  Upon preparing for a
    switch, the incoming drafter prefills its KV cache over all tokens accepted during its inactivity".  cur[b] is the
    drafter that drafted this round's block, route[b] the router's choice for the next round:
        idle[b]  = cur[b] != code                   (the drafter did not draft this round: its rows are deferred)
        flush[b] = idle[b] and route[b] == code     (the router switches b to this drafter: catch up now)
    """
    route, cur = np.asarray(route), np.asarray(cur)
    idle = (cur != code)
    flush = idle & (route == code)
    return idle.astype(np.int32), flush.astype(np.int32)


def switch_round(lazy_by_code, hidden_bits, q_indptr, n_rows, route, cur, q_len_by_code):
    """One round's switch for all drafters: lazy_by_code = {route code: LazyCatchup}.  Returns (cur', next_q_len):
    cur' = route (the chosen drafter drafts the next round) and the block length it will bring."""
    outs = {}
    for code, lz in lazy_by_code.items():
        idle, flush = switch_masks(route, cur, code)
        outs[code] = lz.round(hidden_bits, q_indptr, n_rows, idle, flush)
    nxt = np.asarray(route, dtype=np.int32).copy()
    return nxt, np.array([q_len_by_code[int(r)] for r in nxt], dtype=np.int32), outs
