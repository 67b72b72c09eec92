"""CPU oracle for the Moebius TP<->EP reshard (arXiv 2606.26607) -- TEST INFRASTRUCTURE ONLY.

Plain, slow, obviously-correct numpy: it BUILDS each layout directly from the logical tensors
(PAPER.md:100 §3.1, :116-126 §3.2); it never converts one layout into the other and it shares no
code, table, header or helper with the CUDA path under `paper_2606_26607_b200/`.

Only `tests/`, `__graft_entry__.smoke()` and `bench.py`'s cpu_baseline / `--impl reference` legs
may import this package.  The product path never does (it fails loudly without its CUDA library).

Parity status: every function here is pinned by `tests/test_oracle_*.py` (`-m "not gpu"`) against
brute force, closed forms, invariants, the FFN equivalence the paper states and the
hand-worked fixtures under `tests/golden/`.  No function is "parity unpinned".
"""
from .weights import (  # noqa: F401
    ep_weight_view, tp_weight_view, tp_scale_blocks, tp_scale_view, ep_scale_view, tp_w13_view, tp_w2_view,
)
from .kv import (  # noqa: F401
    CapacityError, canonical_block_tables, ep_pool_image, kv_heads_of_rank, pages_needed,
    partition_requests, tp_pool_image, tp_source_rank, gather_request_from_tp, gather_request_from_ep,
)
from .accounting import kv_bytes, scale_bytes, weight_bytes  # noqa: F401
from .ffn import moe_ffn_dense, moe_ffn_ep, moe_ffn_tp, route_top2  # noqa: F401
from .ffn import moe_ffn_dense_w13, moe_ffn_ep_w13, moe_ffn_tp_w13  # noqa: F401
from .attention import (  # noqa: F401
    ATTN_KINDS, attn_bytes, attn_ep_view, attn_forward_dense, attn_forward_ep, attn_forward_tp, attn_shape, attn_tp_view,
    q_heads_of_rank,
)
from .image import OracleLayout, State, np_view, target_request_state  # noqa: F401,E402
