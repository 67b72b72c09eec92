"""The five BASELINE.json configurations, as plain data (shapes, dtypes, length recipes, seeds).

Stand-ins: the paper's workloads are Qwen3-235B-A22B weights and DeepMath / ShareGPT request
lengths; none is available, only their shapes and length statistics
are reproduced here (reading A18).
"""
from __future__ import annotations

from dataclasses import dataclass, field, replace


@dataclass(frozen=True)
class Config:
    name: str
    R: int            # logical ranks (P in PAPER.md:100)
    L: int            # layers
    E: int            # experts
    H: int            # hidden
    I: int            # moe_intermediate
    w_dtype: str      # "bf16" | "fp32" | "fp8_e4m3_b128"
    kv_heads: int
    head_dim: int
    page: int         # tokens per page
    n_req: int
    len_dist: tuple   # ("uniform", lo, hi) | ("lognormal", median, sigma, cap) | ("geometric", mean, cap)
    seed: int
    pool_policy: str = "roomy"   # roomy = 1.1 x (TP need + max EP live)
    w_orient: int = 0            # 0: gate,up [E,H,I], down [E,I,H] (BASELINE.json); 1: W13 [E,2I,H], W2 [E,H,I]
    n_q_heads: int = 0           # query heads (attention projections); 0 = no attention tensors
    w_inplace: int = 0           # 1: force the fully in-place weight path (EP and TP views alias the same bytes)
    attn_mode: int = 0           # 0 none, 1 both layouts resident (pointer swap), 2 memory-saving (All-Gather rebuild)
    extra: dict = field(default_factory=dict)

    @property
    def w_elem_bytes(self) -> int:
        return {"bf16": 2, "fp32": 4, "fp8_e4m3_b128": 1}[self.w_dtype]

    @property
    def kv_elem_bytes(self) -> int:
        return 2  # bf16 in every config (reading A14)

    @property
    def w_kinds(self) -> tuple:
        return ("gate", "up", "down") if self.w_orient == 0 else ("w13", "w2")

    def with_(self, **kw) -> "Config":
        return replace(self, **kw)


# sigma of the lognormal: ln(p99/median)/2.326 with the paper's median 1,510 / p99 10,386
# -> 0.83 (reading A18)
_SIGMA = 0.83

CONFIGS = {
    "tiny": Config("tiny", R=2, L=1, E=8, H=64, I=32, w_dtype="bf16", kv_heads=2, head_dim=16,
                   page=16, n_req=4, len_dist=("uniform", 1, 64), seed=1001),
    "small": Config("small", R=4, L=4, E=16, H=1024, I=512, w_dtype="bf16", kv_heads=8,
                    head_dim=128, page=16, n_req=64, len_dist=("uniform", 128, 2048), seed=1002),
    "qwen3_30b": Config("qwen3_30b", R=8, L=24, E=128, H=2048, I=768, w_dtype="bf16", kv_heads=4,
                        head_dim=128, page=16, n_req=256,
                        len_dist=("lognormal", 1024, _SIGMA, 8192), seed=1003),
    "qwen3_235b": Config("qwen3_235b", R=8, L=12, E=128, H=4096, I=1536, w_dtype="bf16",
                         kv_heads=4, head_dim=128, page=16, n_req=512,
                         len_dist=("lognormal", 1500, _SIGMA, 8192), seed=1004),
    "fp8_graph": Config("fp8_graph", R=8, L=4, E=128, H=4096, I=1536, w_dtype="fp8_e4m3_b128",
                        kv_heads=4, head_dim=128, page=16, n_req=2048,
                        len_dist=("geometric", 600, 16384), seed=1005),
}


def get_config(name: str) -> Config:
    return CONFIGS[name]
