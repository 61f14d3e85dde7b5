"""Round driver: one verify-and-switch round of the hot path on synthetic, device-resident inputs.

    reserve target pages -> 36 x wf_verify_attn -> wf_accept_entropy_route
      -> ONE wf_switch_round for both drafters, driven on the device by this round's `route` and the `cur_drafter`
         array: the drafter that is active for a sequence gets a KV-only prefill of its rows (stands in for its own
         forward, reading C22), the idle one has them enqueued, a sequence that the router switches is flushed
         together with this round's rows (C21); cur_drafter <- route.  No mask crosses the host.

Everything is launched on one stream with no host synchronisation inside the round.
The route trace is a seeded per-sequence Markov chain (flip with probability Workload.switch_prob per
round, BASELINE.json configs[4]) planted in the logits (spike on the row of the last accepted token), so
the host knows every round's block lengths in advance and can lay out the ragged inputs; the device still
computes every output, derives every mask from its own route, and `check_plan` compares outputs and
cur_drafter with the plan afterwards.  This module holds no method arithmetic: it
only builds inputs (synth) and calls the C-ABI binding.  It never imports oracle/.
"""

import math

import numpy as np

from . import binding as wf
from . import synth

SPIKE_LOW_ENTROPY = 9.0      # added to the planted winner: H well below tau = 2.0 -> diffusion
SPIKE_HIGH_ENTROPY = 0.0     # Gaussian row: H ~ ln V - sigma^2/2 (about 7.4 nats at V = 151936) -> AR


def _i32(a, device):
    import torch
    return torch.from_numpy(np.ascontiguousarray(a, dtype=np.int32)).to(device)


class Slot:
    """Inputs and plan of one round of the cyclic schedule."""
    pass


class RoundState:
    def __init__(self, ctx, wl: synth.Workload, n_slots=16, n_rounds_max=64, device="cuda", layers=None,
                 host_copies=False, final_token=True):
        import torch
        self.torch, self.ctx, self.wl, self.device = torch, ctx, wl, device
        sh = wl.shapes
        self.sh = sh
        self.L = layers if layers is not None else sh.n_layers
        self.B = B = wl.batch
        g = synth.rng(wl.seed, 1)
        self.gmax = max(wl.gammas)
        self.qmax = self.gmax + 1
        # ---- target cache: contexts, pages for n_rounds_max rounds of growth, shuffled or not ----
        self.ctx0 = synth.draw_contexts(wl, g)
        grow = n_rounds_max * self.qmax + self.qmax
        self.max_pages_per_seq = int(-(-(int(self.ctx0.max()) + grow) // sh.page_size)) + 1
        num_pages = int(sum(-(-(int(c) + grow) // sh.page_size) for c in self.ctx0)) + 8
        free = synth.draw_free_list(num_pages, g, wl.shuffled_pages)
        self.free = free
        self.kv_shape = wf.KvShape(self.L, sh.n_kv_heads, sh.head_dim, sh.page_size, num_pages, B, self.max_pages_per_seq)
        pool = (self.L, num_pages, sh.n_kv_heads, sh.page_size, sh.head_dim)
        kv_std = 1.0 / math.sqrt(sh.head_dim)
        # The block's own K/V (reading C10) are whatever the pool already holds at those slots: every
        # page is pre-filled with N(0, 1/sqrt(D)) values, which is what the target's QKV projection
        # would have written there.
        self.k_pool = synth.device_normal_bf16(pool, kv_std, wl.seed, 11, device)
        self.v_pool = synth.device_normal_bf16(pool, kv_std, wl.seed, 12, device)
        self.block_table = torch.full((B, self.max_pages_per_seq), -1, dtype=torch.int32, device=device)
        self.seq_len = torch.zeros(B, dtype=torch.int32, device=device)
        self.target_kv = wf.PagedKV(ctx, self.kv_shape, self.k_pool, self.v_pool, self.block_table, self.seq_len, free)
        self.target_kv.reserve(_i32(self.ctx0, device), B)
        self.seq_len.copy_(_i32(self.ctx0, device))
        # ---- drafters: A = autoregressive (1 layer), D = diffusion (5 layers, configs[1]) ----
        self.drafters = {}
        for name, n_layers in zip(("A", "D"), sh.drafter_layers if len(sh.drafter_layers) == 2 else (sh.drafter_layers[0],) * 2):
            self.drafters[name] = self._make_drafter(name, n_layers, grow, g)
        # ---- cyclic schedule of n_slots rounds: route OUTPUT of slot k (1 = AR) ----
        self.n_slots = n_slots
        route = synth.draw_route_trace(g, n_slots, B, wl.switch_prob)
        if len(wl.gammas) == 1:
            gam_of = lambda r: wl.gammas[0]
        else:
            gam_of = lambda r: wl.gammas[0] if r == wf.ROUTE_AR else wl.gammas[-1]
        self.slots = []
        for k in range(n_slots):
            s = Slot()
            s.cur = route[(k - 1) % n_slots]                                 # drafter that drafted slot k's block
            s.next = route[k]
            s.q_lens = np.array([gam_of(r) + 1 for r in s.cur], dtype=np.int64)
            s.u = synth.draw_accept_prefix(g, s.q_lens - 1, wl.mean_accept)
            s.spike = np.where(s.next == wf.ROUTE_AR, SPIKE_HIGH_ENTROPY, SPIKE_LOW_ENTROPY)
            self._make_slot_inputs(s, k, host_copies)
            self.slots.append(s)
        # the drafter that drafted the block of the next round to run (device state, advanced by wf_switch_round)
        self.cur_drafter = _i32(self.slots[0].cur, device)
        self.next_q_len = torch.zeros(B, dtype=torch.int32, device=device)
        self.q_len_of = {wf.ROUTE_AR: gam_of(wf.ROUTE_AR) + 1, wf.ROUTE_DIFFUSION: gam_of(wf.ROUTE_DIFFUSION) + 1}
        self.tau = torch.full((1,), sh.tau, dtype=torch.float32, device=device)
        # the round's five result vectors are rows of ONE buffer: a caller reads them back with a single copy
        self.out_all = torch.zeros((5, B), dtype=torch.int32, device=device)
        self.out = {n: self.out_all[i] for i, n in enumerate(("accept_len", "bonus_token", "route", "n_commit"))}
        self.entropy = self.out_all[4].view(torch.float32)
        self.attn_ws = torch.empty(wf.wf_verify_attn_workspace_bytes(self.kv_shape, B, sh.n_q_heads, self.qmax),
                                   dtype=torch.uint8, device=device)
        self.acc_ws = torch.empty(wf.wf_accept_workspace_bytes(B * self.qmax, sh.vocab), dtype=torch.uint8, device=device)
        self.sm_scale = 1.0 / math.sqrt(sh.head_dim)
        # ---- WhiFlash-Neural router: d -> d/8 -> 1, seeded random weights ----
        d, m = sh.hidden, sh.hidden // 8
        self.nr = Slot()
        self.nr.d, self.nr.m = d, m
        self.nr.w1 = synth.device_normal_bf16((m, d), 0.02, wl.seed, 60, device)
        self.nr.b1 = synth.device_normal_f32((m,), 0.1, wl.seed, 61, device)
        self.nr.w2 = synth.device_normal_bf16((m,), 0.3, wl.seed, 62, device)
        self.nr.b2 = torch.full((1,), -0.2, dtype=torch.float32, device=device)
        self.nr.tau = torch.zeros(1, dtype=torch.float32, device=device)
        self.nr.delta_al = torch.zeros(B, dtype=torch.float32, device=device)
        self.nr.route = torch.zeros(B, dtype=torch.int32, device=device)
        self.nr.ws = torch.empty(wf.wf_neural_route_workspace_bytes(B, m), dtype=torch.uint8, device=device)
        # ---- (f3) the final backlog token in full, for the AR drafter (the drafter whose catch-up the paper profiles,
        #      PAPER.md:206; a single transformer layer): W_Q, W_O and a two-matrix MLP of width `ffn` ----
        self.switched = torch.full((B,), -1, dtype=torch.int32, device=device)
        self.ft = None
        if final_token:
            ft = Slot()
            dA = self.drafters["A"]
            qd, ffn = sh.n_q_heads * sh.head_dim, sh.ffn
            ft.ffn = ffn
            mk = lambda shape, stream: [synth.device_normal_bf16(shape, 0.02, wl.seed, stream + l, device) for l in range(dA.n_layers)]
            ws_ = (mk((sh.hidden, qd), 70), mk((qd, sh.hidden), 75), mk((sh.hidden, ffn), 80), mk((ffn, sh.hidden), 85))
            dA.handle.set_full_layer(sh.n_q_heads, ffn, min(B, 256), *ws_)       # the library keeps its own repacked copy
            ft.weights = ws_                                   # (W_Q, W_O, W_up, W_down) per layer: the tests hand them to the oracle
            ft.weight_bytes = dA.n_layers * 2 * (2 * sh.hidden * qd + 2 * sh.hidden * ffn)
            ft.h_out = torch.zeros((B, dA.n_layers, sh.hidden), dtype=torch.bfloat16, device=device)
            ft.ws = torch.empty(wf.wf_final_token_workspace_bytes(dA.handle, B), dtype=torch.uint8, device=device)
            self.ft = ft
        self.rounds_done = 0
        torch.cuda.synchronize()

    def run_final_token(self, s, select, code, stream=None):
        """(f3) the last committed row of every selected sequence through the AR drafter's layer in full."""
        wf.wf_final_token_full(self.ctx, self.drafters["A"].handle, s.hidden, s.q_indptr, self.out["n_commit"], select, code,
                               self.B, self.ft.h_out, self.ft.ws, stream)

    # ------------------------------------------------------------------------------------------
    def _make_drafter(self, name, n_layers, grow, g):
        torch, sh, B, wl = self.torch, self.sh, self.B, self.wl
        N = sh.n_kv_heads * sh.head_dim
        per_seq = int(-(-(int(self.ctx0.max()) + grow) // sh.page_size)) + 1
        # drafter caches start EMPTY of history the bench never reads: positions continue from ctx0
        num_pages = int(sum(-(-(int(c) + grow) // sh.page_size) for c in self.ctx0)) + 8
        free = synth.draw_free_list(num_pages, g, wl.shuffled_pages)
        shape = wf.KvShape(n_layers, sh.n_kv_heads, sh.head_dim, sh.page_size, num_pages, B, per_seq)
        pool = (n_layers, num_pages, sh.n_kv_heads, sh.page_size, sh.head_dim)
        d = Slot()
        d.free, d.n_layers = free, n_layers
        d.k_pool = torch.zeros(pool, dtype=torch.bfloat16, device=self.device)
        d.v_pool = torch.zeros(pool, dtype=torch.bfloat16, device=self.device)
        d.block_table = torch.full((B, per_seq), -1, dtype=torch.int32, device=self.device)
        d.seq_len = torch.zeros(B, dtype=torch.int32, device=self.device)
        d.kv = wf.PagedKV(self.ctx, shape, d.k_pool, d.v_pool, d.block_table, d.seq_len, free)
        d.kv.reserve(_i32(self.ctx0, self.device), B)
        d.seq_len.copy_(_i32(self.ctx0, self.device))
        sid = 20 if name == "A" else 40
        d.w_k = [synth.device_normal_bf16((sh.hidden, N), 0.02, wl.seed, sid + 2 * l, self.device) for l in range(n_layers)]
        d.w_v = [synth.device_normal_bf16((sh.hidden, N), 0.02, wl.seed, sid + 2 * l + 1, self.device) for l in range(n_layers)]
        cap = max(wl.backlog_cap, self.qmax)
        d.backlog = torch.zeros((B, cap, sh.hidden), dtype=torch.bfloat16, device=self.device)
        d.backlog_len = torch.zeros(B, dtype=torch.int32, device=self.device)
        max_pos = int(self.ctx0.max()) + grow + 64
        d.shape = wf.DrafterShape(n_layers, sh.hidden, sh.n_kv_heads, sh.head_dim, sh.rope_theta, max_pos, cap)
        d.handle = wf.Drafter(self.ctx, d.shape, d.w_k, d.w_v, d.kv, d.backlog, d.backlog_len)
        d.cap = cap
        return d

    def _make_slot_inputs(self, s, k, host_copies):
        """Device-resident inputs of slot k: Q, hidden rows, logits with planted winners, draft tokens, masks."""
        torch, sh, wl, dev = self.torch, self.sh, self.wl, self.device
        B = self.B
        s.q_indptr_host = np.zeros(B + 1, dtype=np.int32)
        s.q_indptr_host[1:] = np.cumsum(s.q_lens)
        n = int(s.q_indptr_host[-1])
        s.sum_q = n
        s.q = synth.device_normal_bf16((n, sh.n_q_heads, sh.head_dim), 1.0, wl.seed, 1000 + 10 * k, dev)
        s.attn_out = torch.zeros_like(s.q)
        s.hidden = synth.device_normal_bf16((n, sh.hidden), 1.0, wl.seed, 1001 + 10 * k, dev)
        s.logits = synth.device_normal_f32((n, sh.vocab), sh.logit_sigma, wl.seed, 1002 + 10 * k, dev)
        g = synth.rng(wl.seed, 2000 + k)
        winners = g.integers(0, sh.vocab, size=n).astype(np.int64)
        gaps = g.uniform(0.05, 1.0, size=n).astype(np.float32)
        spike_rows = np.zeros(n, dtype=np.float32)
        drafts = g.integers(0, sh.vocab, size=n).astype(np.int32)
        for b in range(B):
            r0, gamma = int(s.q_indptr_host[b]), int(s.q_lens[b]) - 1
            u = int(s.u[b])
            for j in range(1, u + 1):
                drafts[r0 + j] = winners[r0 + j - 1]
            if u < gamma and drafts[r0 + u + 1] == winners[r0 + u]:
                drafts[r0 + u + 1] = (drafts[r0 + u + 1] + 1) % sh.vocab
            spike_rows[r0 + u] = s.spike[b]
        # planted unique winner per row: logits[row, w] = (largest other entry) + gap (+ spike on row u_b)
        rows = torch.arange(n, device=dev)
        w_t = torch.from_numpy(winners).to(dev)
        s.logits[rows, w_t] = -float("inf")
        s.logits[rows, w_t] = s.logits.amax(dim=1) + torch.from_numpy(gaps + spike_rows).to(dev)
        s.winners = winners
        s.drafts = _i32(drafts, dev)
        s.q_indptr = _i32(s.q_indptr_host, dev)
        s.add_tokens = _i32(s.q_lens, dev)
        # per-drafter masks (host-planned): who is active, idle, and who switches in after this round
        s.masks = {}
        for name, code in (("A", wf.ROUTE_AR), ("D", wf.ROUTE_DIFFUSION)):
            active = (s.cur == code).astype(np.int32)
            m = Slot()
            m.active_host, m.idle_host = active, 1 - active
            m.flush_host = ((s.next == code) & (s.cur != code)).astype(np.int32)
            m.active, m.idle, m.flush = _i32(active, dev), _i32(1 - active, dev), _i32(m.flush_host, dev)
            m.n_rows = torch.zeros(B, dtype=torch.int32, device=dev)
            s.masks[name] = m
        if host_copies:
            s.host = {k2: getattr(s, k2).cpu().pin_memory() for k2 in ("q", "hidden", "logits", "drafts")}

    # ------------------------------------------------------------------------------------------
    def attn_bytes(self, slot, ctx_lens):
        """Algorithmic KV bytes one attention launch reads: K and V once per kv head."""
        sh = self.sh
        return int(sum(int(c) + int(q) for c, q in zip(ctx_lens, slot.q_lens))) * sh.n_kv_heads * sh.head_dim * 2 * 2

    def run_attention(self, s, stream=None):
        sh = self.sh
        for l in range(self.L):
            wf.wf_verify_attn(self.ctx, self.target_kv, l, s.q, s.q_indptr, self.B, sh.n_q_heads, self.qmax,
                              self.sm_scale, s.attn_out, self.attn_ws, stream)

    def run_accept(self, s, stream=None):
        o = self.out
        wf.wf_accept_entropy_route(self.ctx, s.logits, self.sh.vocab, s.drafts, s.q_indptr, self.B, self.qmax, self.tau, True,
                                   o["accept_len"], o["bonus_token"], self.entropy, o["route"], o["n_commit"],
                                   self.target_kv, self.acc_ws, stream)

    def run_neural_route(self, s, stream=None):
        """The learned policy on the final hidden row of the last accepted position (the block's hidden rows stand in
        for the target's final hidden states); reads accept_len left on the device by run_accept."""
        n = self.nr
        wf.wf_neural_route(self.ctx, s.hidden, s.q_indptr, self.out["accept_len"], self.B, n.d, n.m, n.w1, n.b1, n.w2, n.b2,
                           n.tau, True, n.delta_al, n.route, n.ws, stream)

    def sync_cur(self):
        """cur_drafter <- the plan's value for the next round to run (after legs that do not drive the switch)."""
        self.cur_drafter.copy_(_i32(self.slots[self.rounds_done % self.n_slots].cur, self.device))

    def run_catchup(self, s, stream=None, lazy=True, fused=True, mode=None, events=None):
        """Drafter-cache maintenance after the accept.
        mode "switch" (default): ONE wf_switch_round for both drafters, masks derived on the device from route and
             cur_drafter (the paper's scheme: Lazy Catch-up + KV-only prefill at the switch);
        mode "round": one wf_lazy_catchup_round per drafter with host-planned masks;
        mode "separate": the three separate calls a round is equivalent to;
        mode "eager": the paper's baseline, a KV-only prefill into both drafters every round;
        mode "active": only the active drafter's own append (reading C22), nothing for the idle one."""
        torch, B = self.torch, self.B
        n_commit = self.out["n_commit"]
        if mode is None:
            mode = "eager" if not lazy else ("switch" if fused else "separate")
        if mode == "switch":
            wf.wf_switch_round(self.ctx, self.drafters["A"].handle, self.drafters["D"].handle, s.hidden, s.q_indptr, n_commit,
                               None, self.out["route"], self.cur_drafter, self.next_q_len, self.q_len_of[wf.ROUTE_AR],
                               self.q_len_of[wf.ROUTE_DIFFUSION], B, self.qmax, stream, switched=self.switched)
            if self.ft is not None:                            # the switch as the paper defines it ends with the final token
                if events:
                    events["final"][0].record()
                self.run_final_token(s, self.switched, wf.ROUTE_AR, stream)
                if events:
                    events["final"][1].record()
            return
        for name, d in self.drafters.items():
            m = s.masks[name]
            if mode == "round":
                wf.wf_lazy_catchup_round(self.ctx, d.handle, s.hidden, s.q_indptr, n_commit, None,
                                         m.idle if m.idle_host.any() else None, m.flush if m.flush_host.any() else None,
                                         B, self.qmax, stream)
            elif mode == "active":
                if m.active_host.any():
                    torch.mul(n_commit, m.active, out=m.n_rows)            # argument marshalling, not the path
                    wf.wf_kv_only_prefill(self.ctx, d.handle, s.hidden, s.q_indptr, m.n_rows, None, B, self.qmax, stream)
            elif mode == "separate":
                if m.active_host.any():
                    torch.mul(n_commit, m.active, out=m.n_rows)            # argument marshalling, not the path
                    wf.wf_kv_only_prefill(self.ctx, d.handle, s.hidden, s.q_indptr, m.n_rows, None, B, self.qmax, stream)
                if m.idle_host.any():
                    wf.wf_lazy_catchup_enqueue(self.ctx, d.handle, s.hidden, s.q_indptr, n_commit, None, m.idle, B, self.qmax, stream)
                if m.flush_host.any():
                    wf.wf_lazy_catchup_flush(self.ctx, d.handle, m.flush, B, stream)
            else:
                wf.wf_kv_only_prefill(self.ctx, d.handle, s.hidden, s.q_indptr, n_commit, None, B, self.qmax, stream)
        if self.ft is not None and mode != "active":             # every round, as in the device-driven mode (empty calls included)
            if events:
                events["final"][0].record()
            self.run_final_token(s, s.masks["A"].flush, 1, stream)
            if events:
                events["final"][1].record()

    def run_round(self, stream=None, lazy=True, events=None, fused=True, mode=None):
        """One whole round.  events: optional dict of (start, end) CUDA event pairs to record around parts."""
        s = self.slots[self.rounds_done % self.n_slots]
        self.target_kv.reserve(s.add_tokens, self.B, stream)
        if events:
            events["attn"][0].record()
        self.run_attention(s, stream)
        if events:
            events["attn"][1].record()
        self.run_accept(s, stream)
        if events:
            events["catchup"][0].record()
        self.run_catchup(s, stream, lazy, fused, mode, events if events and "final" in events else None)
        if events:
            events["catchup"][1].record()
        self.rounds_done += 1
        return s

    # ------------------------------------------------------------------------------------------
    # Tree verification round: every sequence is AR-routed and brings a draft tree of
    # `n_nodes` rows (depth 8, top-k 10, 60 draft tokens).  Inputs and calls only.
    def make_tree_slot(self, n_nodes=60, depth=8, top_k=10):
        torch, sh, wl, dev, B = self.torch, self.sh, self.wl, self.device, self.B
        g = synth.rng(wl.seed, 3000)
        t = Slot()
        t.n_nodes = n_nodes
        parents = [synth.draw_tree(g, n_nodes, depth, top_k) for _ in range(B)]
        n = B * n_nodes
        t.q_indptr_host = np.arange(0, n + 1, n_nodes, dtype=np.int32)
        t.q = synth.device_normal_bf16((n, sh.n_q_heads, sh.head_dim), 1.0, wl.seed, 3001, dev)
        t.attn_out = torch.zeros_like(t.q)
        t.logits = synth.device_normal_f32((n, sh.vocab), sh.logit_sigma, wl.seed, 3002, dev)
        winners = g.integers(0, sh.vocab, size=n).astype(np.int64)
        gaps = g.uniform(0.05, 1.0, size=n).astype(np.float32)
        tokens = g.integers(0, sh.vocab, size=n).astype(np.int32)
        want = synth.draw_accept_prefix(g, np.full(B, depth), wl.mean_accept)
        t.paths = []
        for b in range(B):
            r0, par = b * n_nodes, parents[b]
            kids = [[c for c in range(n_nodes) if par[c] == j] for j in range(n_nodes)]
            for j in range(n_nodes):                         # siblings carry distinct tokens, none the winner
                used = {int(winners[r0 + j])}
                for c in kids[j]:
                    while int(tokens[r0 + c]) in used:
                        tokens[r0 + c] = (tokens[r0 + c] + 1) % sh.vocab
                    used.add(int(tokens[r0 + c]))
            cur, path = 0, [0]
            while len(path) - 1 < int(want[b]) and kids[cur]:
                c = int(kids[cur][g.integers(0, len(kids[cur]))])
                tokens[r0 + c] = winners[r0 + cur]
                cur = c
                path.append(cur)
            t.paths.append(path)
        rows = torch.arange(n, device=dev)
        w_t = torch.from_numpy(winners).to(dev)
        t.logits[rows, w_t] = -float("inf")
        t.logits[rows, w_t] = t.logits.amax(dim=1) + torch.from_numpy(gaps).to(dev)
        t.tokens = _i32(tokens, dev)
        t.parent = _i32(np.concatenate(parents), dev)
        t.q_indptr = _i32(t.q_indptr_host, dev)
        t.add_tokens = _i32(np.full(B, n_nodes), dev)
        t.masks = torch.zeros(n, dtype=torch.int64, device=dev)
        t.path = torch.full((B, n_nodes), -1, dtype=torch.int32, device=dev)
        t.attn_ws = torch.empty(wf.wf_verify_attn_workspace_bytes(self.kv_shape, B, sh.n_q_heads, n_nodes),
                                dtype=torch.uint8, device=dev)
        t.acc_ws = torch.empty(wf.wf_accept_workspace_bytes(n, sh.vocab), dtype=torch.uint8, device=dev)
        return t

    def run_tree_round(self, t, stream=None, events=None):
        """reserve -> ancestor masks (once) -> L x tree attention -> acceptance walk -> path compaction."""
        sh, B, o = self.sh, self.B, self.out
        self.target_kv.reserve(t.add_tokens, B, stream)
        wf.wf_tree_masks(self.ctx, t.parent, t.q_indptr, B, t.n_nodes, t.masks, stream)
        if events:
            events["attn"][0].record()
        for l in range(self.L):
            wf.wf_verify_attn_tree(self.ctx, self.target_kv, l, t.q, t.q_indptr, t.masks, B, sh.n_q_heads, t.n_nodes,
                                   self.sm_scale, t.attn_out, t.attn_ws, stream)
        if events:
            events["attn"][1].record()
        wf.wf_accept_tree_entropy_route(self.ctx, t.logits, sh.vocab, t.tokens, t.parent, t.q_indptr, B, t.n_nodes, self.tau,
                                        True, o["accept_len"], o["bonus_token"], self.entropy, o["route"], o["n_commit"],
                                        t.path, t.n_nodes, t.acc_ws, stream)
        wf.wf_kv_compact_path(self.ctx, self.target_kv, t.path, t.n_nodes, o["n_commit"], B, stream)

    def check_tree_plan(self, t):
        self.torch.cuda.synchronize()
        st = self.ctx.poll_status()
        if st != 0:
            raise RuntimeError(f"device status {st}")
        a = self.out["accept_len"].cpu().numpy()
        path = t.path.cpu().numpy()
        for b, want in enumerate(t.paths):
            if int(a[b]) != len(want) - 1 or list(path[b][:len(want)]) != want:
                raise RuntimeError(f"tree round: sequence {b} accepted {list(path[b][:int(a[b]) + 1])}, planted {want}")

    def check_plan(self, s, switched=True):
        """After a sync: the device's outputs of the last round must equal the planted plan (and, when the round went
        through wf_switch_round, so must the device-side drafter state and the next block lengths)."""
        self.torch.cuda.synchronize()
        st = self.ctx.poll_status()
        if st != 0:
            raise RuntimeError(f"device status {st}")
        a = self.out["accept_len"].cpu().numpy()
        r = self.out["route"].cpu().numpy()
        if not (np.array_equal(a, s.u) and np.array_equal(r, s.next)):
            raise RuntimeError(f"device outputs differ from the planted plan: accept {a} vs {s.u}; route {r} vs {s.next}")
        if switched:
            c = self.cur_drafter.cpu().numpy()
            nq = self.next_q_len.cpu().numpy()
            want_q = np.array([self.q_len_of[int(x)] for x in s.next])
            if not (np.array_equal(c, s.next) and np.array_equal(nq, want_q)):
                raise RuntimeError(f"device-driven switch: cur_drafter {c} vs {s.next}; next block lengths {nq} vs {want_q}")

    def close(self):
        for d in self.drafters.values():
            d.handle.close()
            d.kv.close()
        self.target_kv.close()
