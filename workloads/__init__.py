"""Seeded synthetic workloads shared by the oracle-side tests and the CUDA-side tests.

This module holds NO arithmetic of the method (no layout math, no partitioning, no page
allocation): only the five BASELINE.json configurations as plain data and seeded random
draws (weights, KV values, request lengths, page permutations).  Both `oracle/` and the
CUDA path are fed from here; neither imports the other.
"""
from .configs import CONFIGS, Config, get_config  # noqa: F401
from .gen import (  # noqa: F401
    bf16_bits_from_f32,
    draw_seq_lens,
    gen_kv_request,
    gen_logical_weight,
    gen_logical_scale,
    random_page_tables,
    kv_pool_bytes,
    tag_fill_u16,
    tag_fill_u16_torch,
    tag_salt_offset,
    weight_tag_salt,
    weight_shape,
    kv_tag_salt,
    attn_weight_shape,
    attn_tag_salt,
    gen_attn_weight,
)
