"""CPU oracle for the WhiFlash verify-and-switch hot path (arxiv/paper_2606_07710).

THIS PACKAGE IS TEST INFRASTRUCTURE, NOT PRODUCT.  Only `tests/`,
`__graft_entry__.smoke()` and `bench.py`'s `cpu_baseline` / `--impl reference`
legs may import it.  It shares no code with the CUDA path under
`paper_2606_07710_b200/` and never imports it; the product path never imports
this package and has no CPU fallback.

Everything here is plain numpy in fp64 (bf16 / fp32 inputs are widened exactly),
written in the paper's order and notation so it can be checked against
`/root/reference/PAPER.md` by eye:

  O1  verify_attn.verify_attn            PAPER.md:65  (§3.2 "parallel verification")
  O2  accept_route.accept_entropy_route  PAPER.md:75-81 (§3.3.1), :65, :135
  O3  kv_prefill.kv_only_prefill         PAPER.md:119 (§3.4 "KV-only Prefill")
  O4  lazy_catchup.LazyCatchup           PAPER.md:117 (§3.4 "Lazy Catch-up"), :204
  O5  kv_prefill.full_drafter_prefill    PAPER.md:119 ("A full forward pass ...")
  D1  paged_kv.PagedKV                   BASELINE.json north_star (paged-KV block table)
  O6  neural_route.neural_route          PAPER.md:87, :103-107, :325 (WhiFlash-Neural policy)
  O7  tree_verify.tree_attn / tree_accept_entropy_route / compact_path
                                         PAPER.md:65, :39, :317, :327 (tree verification)
  O8  spec_sample.spec_sample_entropy_route  PAPER.md:19, :79-81 (stochastic acceptance with temperature)
  O9  final_token.final_tokens_full      PAPER.md:119, :206 (the final backlog token through the drafter layer in full;
                                         SURVEY.md §8(f) f3)

Pins (tests/test_oracle_*.py, `-m "not gpu"`): closed forms, invariants,
textbook special cases and pure-Python brute force; see DESIGN.md §"Oracle pins".
Parity status: every function is pinned except the whole-round composition, for
which the paper prints no worked numeric example ("parity unpinned" for the
end-to-end round values only; each part is pinned separately).
"""

from . import bf16, paged_kv, verify_attn, accept_route, kv_prefill, lazy_catchup, neural_route, tree_verify, spec_sample, final_token  # noqa: F401
