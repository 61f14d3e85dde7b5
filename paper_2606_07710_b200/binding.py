"""Thin ctypes binding of include/whiflash.h: same names, argument marshalling only.

Every step runs in libwhiflash's CUDA kernels.  There is no CPU path: importing this module
raises if the library has not been built (python -m paper_2606_07710_b200.build).
torch is used by callers for device memory and streams; this module only needs `.data_ptr()`.
"""

import ctypes as C
import os

_LIB_PATH = os.path.join(os.path.dirname(os.path.abspath(__file__)), "libwhiflash.so")
if not os.path.exists(_LIB_PATH):
    raise ImportError(
        f"{_LIB_PATH} is missing: build it with `python -m paper_2606_07710_b200.build` "
        "(the hot path is CUDA-only; there is no fallback)")
lib = C.CDLL(_LIB_PATH)

WF_OK = 0
WF_ERR_INVALID_ARG = -1
WF_ERR_UNSUPPORTED_SHAPE = -2
WF_ERR_OUT_OF_PAGES = -3
WF_ERR_QUEUE_OVERFLOW = -4
WF_ERR_CUDA = -5
ROUTE_DIFFUSION = 0
ROUTE_AR = 1

EXPORTS = [
    "wf_ctx_create", "wf_ctx_destroy", "wf_last_error", "wf_poll_status", "wf_launch_count",
    "wf_kv_create", "wf_kv_destroy", "wf_kv_reserve", "wf_kv_release_seq", "wf_kv_pages_held",
    "wf_verify_attn", "wf_verify_attn_workspace_bytes",
    "wf_accept_entropy_route", "wf_accept_workspace_bytes", "wf_accept_entropy_route_static",
    "wf_drafter_create", "wf_drafter_destroy", "wf_kv_only_prefill",
    "wf_lazy_catchup_enqueue", "wf_lazy_catchup_flush",
    "wf_neural_route", "wf_neural_route_workspace_bytes", "wf_lazy_catchup_round",
    "wf_tree_masks", "wf_verify_attn_tree", "wf_accept_tree_entropy_route", "wf_kv_compact_path",
    "wf_accept_sample_entropy_route", "wf_switch_round",
    "wf_drafter_set_full_layer", "wf_final_token_workspace_bytes", "wf_final_token_full", "wf_ctx_set_attn_cluster", "wf_ctx_set_deterministic",
    "wf_ctx_set_attn_early_kv",
]


class KvShape(C.Structure):
    _fields_ = [(n, C.c_int) for n in ("n_layers", "n_kv_heads", "head_dim", "page_size", "num_pages",
                                       "max_seqs", "max_pages_per_seq")]


class DrafterShape(C.Structure):
    _fields_ = [("n_layers", C.c_int), ("hidden", C.c_int), ("n_kv_heads", C.c_int), ("head_dim", C.c_int),
                ("rope_theta", C.c_float), ("max_pos", C.c_int), ("backlog_cap", C.c_int)]


_vp, _i, _sz = C.c_void_p, C.c_int, C.c_size_t
_SIG = {
    "wf_ctx_create": (_i, [C.POINTER(_vp), _i]),
    "wf_ctx_destroy": (_i, [_vp]),
    "wf_last_error": (C.c_char_p, [_vp]),
    "wf_poll_status": (_i, [_vp, _vp, C.POINTER(_i)]),
    "wf_launch_count": (C.c_int64, [_vp]),
    "wf_kv_create": (_i, [_vp, C.POINTER(KvShape), _vp, _vp, _vp, _vp, _vp, _i, C.POINTER(_vp)]),
    "wf_kv_destroy": (_i, [_vp]),
    "wf_kv_reserve": (_i, [_vp, _vp, _i, _vp]),
    "wf_kv_release_seq": (_i, [_vp, _i, _vp]),
    "wf_kv_pages_held": (_vp, [_vp]),
    "wf_verify_attn": (_i, [_vp, _vp, _i, _vp, _vp, _i, _i, _i, C.c_float, _vp, _vp, _sz, _vp]),
    "wf_verify_attn_workspace_bytes": (_sz, [C.POINTER(KvShape), _i, _i, _i]),
    "wf_accept_entropy_route": (_i, [_vp, _vp, _i, _vp, _vp, _i, _i, _vp, _i, _vp, _vp, _vp, _vp, _vp, _vp, _vp, _sz, _vp]),
    "wf_accept_entropy_route_static": (_i, [_vp, _vp, _i, _vp, _vp, _i, _i, _vp, _i, _vp, _vp, _vp, _vp, _vp, _vp, _vp]),
    "wf_accept_workspace_bytes": (_sz, [_i, _i]),
    "wf_drafter_create": (_i, [_vp, C.POINTER(DrafterShape), C.POINTER(_vp), C.POINTER(_vp), _vp, _vp, _vp, C.POINTER(_vp)]),
    "wf_drafter_destroy": (_i, [_vp]),
    "wf_kv_only_prefill": (_i, [_vp, _vp, _vp, _vp, _vp, _vp, _i, _i, _vp]),
    "wf_lazy_catchup_enqueue": (_i, [_vp, _vp, _vp, _vp, _vp, _vp, _vp, _i, _i, _vp]),
    "wf_lazy_catchup_flush": (_i, [_vp, _vp, _vp, _i, _vp]),
    "wf_lazy_catchup_round": (_i, [_vp, _vp, _vp, _vp, _vp, _vp, _vp, _vp, _i, _i, _vp]),
    "wf_switch_round": (_i, [_vp, _vp, _vp, _vp, _vp, _vp, _vp, _vp, _vp, _vp, _vp, _i, _i, _i, _i, _vp]),
    "wf_drafter_set_full_layer": (_i, [_vp, _vp, _i, _i, _i, C.POINTER(_vp), C.POINTER(_vp), C.POINTER(_vp), C.POINTER(_vp)]),
    "wf_final_token_workspace_bytes": (_sz, [_vp, _i]),
    "wf_ctx_set_attn_cluster": (_i, [_vp, _i]),
    "wf_ctx_set_deterministic": (_i, [_vp, _i]),
    "wf_ctx_set_attn_early_kv": (_i, [_vp, _i]),
    "wf_final_token_full": (_i, [_vp, _vp, _vp, _vp, _vp, _vp, _i, _i, _vp, _vp, _sz, _vp]),
    "wf_neural_route_workspace_bytes": (_sz, [_i, _i]),
    "wf_neural_route": (_i, [_vp, _vp, _vp, _vp, _i, _i, _i, _vp, _vp, _vp, _vp, _vp, _i, _vp, _vp, _vp, _sz, _vp]),
    "wf_tree_masks": (_i, [_vp, _vp, _vp, _i, _i, _vp, _vp]),
    "wf_verify_attn_tree": (_i, [_vp, _vp, _i, _vp, _vp, _vp, _i, _i, _i, C.c_float, _vp, _vp, _sz, _vp]),
    "wf_accept_tree_entropy_route": (_i, [_vp, _vp, _i, _vp, _vp, _vp, _i, _i, _vp, _i, _vp, _vp, _vp, _vp, _vp, _vp, _i,
                                          _vp, _sz, _vp]),
    "wf_kv_compact_path": (_i, [_vp, _vp, _i, _vp, _i, _vp]),
    "wf_accept_sample_entropy_route": (_i, [_vp, _vp, _i, _vp, _vp, _i, _i, C.c_float, _vp, _vp, _vp, _vp, _i, _vp, _vp, _vp,
                                            _vp, _vp, _vp, _vp, _sz, _vp]),
}
for _name, (_res, _args) in _SIG.items():
    _f = getattr(lib, _name)
    _f.restype, _f.argtypes = _res, _args


class WhiFlashError(RuntimeError):
    pass


def _ptr(t):
    """torch tensor / int / None -> void*."""
    if t is None:
        return None
    if isinstance(t, int):
        return t
    return t.data_ptr()


def _stream(stream):
    if stream is None:
        import torch
        return torch.cuda.current_stream().cuda_stream
    return stream if isinstance(stream, int) else stream.cuda_stream


class Ctx:
    def __init__(self, device=0):
        h = _vp()
        rc = lib.wf_ctx_create(C.byref(h), int(device))
        if rc != WF_OK:
            raise WhiFlashError(f"wf_ctx_create failed: {rc} (needs an sm_100 GPU; no CPU fallback)")
        self.h = h

    def check(self, rc):
        if rc != WF_OK:
            raise WhiFlashError(f"rc={rc}: {lib.wf_last_error(self.h).decode()}")

    def poll_status(self, stream=None):
        s = _i(0)
        self.check(lib.wf_poll_status(self.h, _stream(stream), C.byref(s)))
        return s.value

    def launch_count(self):
        return int(lib.wf_launch_count(self.h))

    def set_deterministic(self, on):
        """Attention merges fold a pair's partials in key-range order (bit-reproducible) instead of last-arriver order."""
        self.check(lib.wf_ctx_set_deterministic(self.h, 1 if on else 0))

    def set_attn_early_kv(self, on):
        """Attention launches read lengths, page ids and the K/V below the cached length ahead of the dependency wait
        (the caller promises the preceding kernel of the stream writes none of them; see whiflash.h)."""
        self.check(lib.wf_ctx_set_attn_early_kv(self.h, 1 if on else 0))

    def set_attn_cluster(self, cluster_size):
        """Launch shape of wf_verify_attn: -1 automatic, 0 never clusters, 1..16 force that many CTAs per pair (1 = no merge)."""
        self.check(lib.wf_ctx_set_attn_cluster(self.h, int(cluster_size)))

    def close(self):
        if self.h:
            lib.wf_ctx_destroy(self.h)
            self.h = None


class PagedKV:
    """wf_paged_kv handle; pools/block_table/seq_len are caller-owned torch tensors kept alive here."""

    def __init__(self, ctx, shape: KvShape, k_pool, v_pool, block_table, seq_len, free_pages):
        import numpy as np
        self.ctx, self.shape = ctx, shape
        self.k_pool, self.v_pool, self.block_table, self.seq_len = k_pool, v_pool, block_table, seq_len
        fp = np.ascontiguousarray(free_pages, dtype=np.int32)
        h = _vp()
        ctx.check(lib.wf_kv_create(ctx.h, C.byref(shape), _ptr(k_pool), _ptr(v_pool), _ptr(block_table),
                                   _ptr(seq_len), fp.ctypes.data, len(fp), C.byref(h)))
        self.h = h

    def reserve(self, add_tokens, B, stream=None):
        self.ctx.check(lib.wf_kv_reserve(self.h, _ptr(add_tokens), B, _stream(stream)))

    def release_seq(self, seq, stream=None):
        self.ctx.check(lib.wf_kv_release_seq(self.h, seq, _stream(stream)))

    def pages_held_ptr(self):
        return lib.wf_kv_pages_held(self.h)

    def close(self):
        if self.h:
            lib.wf_kv_destroy(self.h)
            self.h = None


def wf_verify_attn_workspace_bytes(shape, B, n_q_heads, max_q_len):
    return int(lib.wf_verify_attn_workspace_bytes(C.byref(shape), B, n_q_heads, max_q_len))


def wf_verify_attn(ctx, kv, layer, q, q_indptr, B, n_q_heads, max_q_len, sm_scale, out, workspace, stream=None):
    ctx.check(lib.wf_verify_attn(ctx.h, kv.h, layer, _ptr(q), _ptr(q_indptr), B, n_q_heads, max_q_len,
                                 C.c_float(sm_scale), _ptr(out), _ptr(workspace),
                                 workspace.numel() * workspace.element_size(), _stream(stream)))


def wf_accept_workspace_bytes(sum_q, V):
    return int(lib.wf_accept_workspace_bytes(sum_q, V))


def wf_accept_entropy_route(ctx, logits, V, draft_tokens, q_indptr, B, max_q_len, tau, tau_is_scalar,
                            accept_len, bonus_token, entropy, route, n_commit, target_kv, workspace, stream=None):
    ctx.check(lib.wf_accept_entropy_route(
        ctx.h, _ptr(logits), V, _ptr(draft_tokens), _ptr(q_indptr), B, max_q_len, _ptr(tau), int(tau_is_scalar),
        _ptr(accept_len), _ptr(bonus_token), _ptr(entropy), _ptr(route), _ptr(n_commit),
        target_kv.h if target_kv is not None else None, _ptr(workspace),
        workspace.numel() * workspace.element_size(), _stream(stream)))


def wf_accept_entropy_route_static(ctx, logits, V, draft_tokens, q_indptr, B, max_q_len, tau, tau_is_scalar,
                                   accept_len, bonus_token, entropy, route, n_commit, target_kv, stream=None):
    """wf_accept_entropy_route without a workspace and without any allocation: scratch in the library's static device array
    (limits and the sharing rule: include/whiflash.h)."""
    ctx.check(lib.wf_accept_entropy_route_static(
        ctx.h, _ptr(logits), V, _ptr(draft_tokens), _ptr(q_indptr), B, max_q_len, _ptr(tau), int(tau_is_scalar),
        _ptr(accept_len), _ptr(bonus_token), _ptr(entropy), _ptr(route), _ptr(n_commit),
        target_kv.h if target_kv is not None else None, _stream(stream)))


class Drafter:
    def __init__(self, ctx, shape: DrafterShape, w_k, w_v, kv: PagedKV, backlog, backlog_len):
        self.ctx, self.shape, self.kv = ctx, shape, kv
        self.w_k, self.w_v, self.backlog, self.backlog_len = list(w_k), list(w_v), backlog, backlog_len
        L = shape.n_layers
        assert len(self.w_k) == L and len(self.w_v) == L
        wk = (_vp * L)(*[_ptr(w) for w in self.w_k])
        wv = (_vp * L)(*[_ptr(w) for w in self.w_v])
        h = _vp()
        ctx.check(lib.wf_drafter_create(ctx.h, C.byref(shape), wk, wv, kv.h, _ptr(backlog), _ptr(backlog_len), C.byref(h)))
        self.h = h

    def set_full_layer(self, n_q_heads, ffn, max_tokens, w_q, w_o, w_up, w_down):
        """(f3) the weights of the drafter layer that KV-only prefill skips; the library repacks its own copy."""
        L = self.shape.n_layers
        arrs = [(_vp * L)(*[_ptr(w) for w in ws]) for ws in (w_q, w_o, w_up, w_down)]
        self.ctx.check(lib.wf_drafter_set_full_layer(self.ctx.h, self.h, n_q_heads, ffn, max_tokens, *arrs))

    def close(self):
        if self.h:
            lib.wf_drafter_destroy(self.h)
            self.h = None


def wf_kv_only_prefill(ctx, drafter, hidden, q_indptr, n_rows, seq_ids, B, max_rows, stream=None):
    ctx.check(lib.wf_kv_only_prefill(ctx.h, drafter.h, _ptr(hidden), _ptr(q_indptr), _ptr(n_rows), _ptr(seq_ids),
                                     B, max_rows, _stream(stream)))


def wf_lazy_catchup_enqueue(ctx, drafter, hidden, q_indptr, n_rows, seq_ids, idle_mask, B, max_rows, stream=None):
    ctx.check(lib.wf_lazy_catchup_enqueue(ctx.h, drafter.h, _ptr(hidden), _ptr(q_indptr), _ptr(n_rows), _ptr(seq_ids),
                                          _ptr(idle_mask), B, max_rows, _stream(stream)))


def wf_lazy_catchup_flush(ctx, drafter, flush_mask, B, stream=None):
    ctx.check(lib.wf_lazy_catchup_flush(ctx.h, drafter.h, _ptr(flush_mask), B, _stream(stream)))


def wf_neural_route_workspace_bytes(B, m):
    return int(lib.wf_neural_route_workspace_bytes(B, m))


def wf_neural_route(ctx, hidden_final, q_indptr, accept_len, B, d, m, w1, b1, w2, b2, tau, tau_is_scalar,
                    delta_al, route, workspace, stream=None):
    ctx.check(lib.wf_neural_route(ctx.h, _ptr(hidden_final), _ptr(q_indptr), _ptr(accept_len), B, d, m, _ptr(w1), _ptr(b1),
                                  _ptr(w2), _ptr(b2), _ptr(tau), int(tau_is_scalar), _ptr(delta_al), _ptr(route),
                                  _ptr(workspace), workspace.numel() * workspace.element_size(), _stream(stream)))


def wf_lazy_catchup_round(ctx, drafter, hidden, q_indptr, n_rows, seq_ids, idle_mask, flush_mask, B, max_rows, stream=None):
    ctx.check(lib.wf_lazy_catchup_round(ctx.h, drafter.h, _ptr(hidden), _ptr(q_indptr), _ptr(n_rows), _ptr(seq_ids),
                                        _ptr(idle_mask), _ptr(flush_mask), B, max_rows, _stream(stream)))


def wf_switch_round(ctx, drafter_ar, drafter_diffusion, hidden, q_indptr, n_rows, seq_ids, route, cur_drafter, next_q_len,
                    q_len_ar, q_len_diffusion, B, max_rows, stream=None, switched=None):
    ctx.check(lib.wf_switch_round(ctx.h, drafter_ar.h, drafter_diffusion.h, _ptr(hidden), _ptr(q_indptr), _ptr(n_rows),
                                  _ptr(seq_ids), _ptr(route), _ptr(cur_drafter), _ptr(next_q_len), _ptr(switched),
                                  q_len_ar, q_len_diffusion, B, max_rows, _stream(stream)))


def wf_final_token_workspace_bytes(drafter, B):
    return int(lib.wf_final_token_workspace_bytes(drafter.h, B))


def wf_final_token_full(ctx, drafter, hidden, q_indptr, n_rows, select, select_code, B, h_out, workspace, stream=None):
    ctx.check(lib.wf_final_token_full(ctx.h, drafter.h, _ptr(hidden), _ptr(q_indptr), _ptr(n_rows), _ptr(select),
                                      select_code, B, _ptr(h_out), _ptr(workspace),
                                      workspace.numel() * workspace.element_size(), _stream(stream)))


def wf_tree_masks(ctx, parent, q_indptr, B, max_nodes, tree_mask, stream=None):
    ctx.check(lib.wf_tree_masks(ctx.h, _ptr(parent), _ptr(q_indptr), B, max_nodes, _ptr(tree_mask), _stream(stream)))


def wf_verify_attn_tree(ctx, kv, layer, q, q_indptr, tree_mask, B, n_q_heads, max_nodes, sm_scale, out, workspace,
                        stream=None):
    ctx.check(lib.wf_verify_attn_tree(ctx.h, kv.h, layer, _ptr(q), _ptr(q_indptr), _ptr(tree_mask), B, n_q_heads, max_nodes,
                                      C.c_float(sm_scale), _ptr(out), _ptr(workspace),
                                      workspace.numel() * workspace.element_size(), _stream(stream)))


def wf_accept_tree_entropy_route(ctx, logits, V, node_tokens, parent, q_indptr, B, max_nodes, tau, tau_is_scalar,
                                 accept_len, bonus_token, entropy, route, n_commit, path, path_stride, workspace,
                                 stream=None):
    ctx.check(lib.wf_accept_tree_entropy_route(
        ctx.h, _ptr(logits), V, _ptr(node_tokens), _ptr(parent), _ptr(q_indptr), B, max_nodes, _ptr(tau),
        int(tau_is_scalar), _ptr(accept_len), _ptr(bonus_token), _ptr(entropy), _ptr(route), _ptr(n_commit), _ptr(path),
        path_stride, _ptr(workspace), workspace.numel() * workspace.element_size(), _stream(stream)))


def wf_kv_compact_path(ctx, kv, path, path_stride, n_commit, B, stream=None):
    ctx.check(lib.wf_kv_compact_path(kv.h, _ptr(path), path_stride, _ptr(n_commit), B, _stream(stream)))


def wf_accept_sample_entropy_route(ctx, logits, V, draft_tokens, q_indptr, B, max_q_len, temperature, draft_q, u_accept,
                                   u_sample, tau, tau_is_scalar, accept_len, token, entropy, route, n_commit, target_kv,
                                   workspace, stream=None):
    ctx.check(lib.wf_accept_sample_entropy_route(
        ctx.h, _ptr(logits), V, _ptr(draft_tokens), _ptr(q_indptr), B, max_q_len, C.c_float(temperature), _ptr(draft_q),
        _ptr(u_accept), _ptr(u_sample), _ptr(tau), int(tau_is_scalar), _ptr(accept_len), _ptr(token), _ptr(entropy),
        _ptr(route), _ptr(n_commit), target_kv.h if target_kv is not None else None, _ptr(workspace),
        workspace.numel() * workspace.element_size(), _stream(stream)))
