"""Plumbing around the C ABI: torch owns the device bytes and the stream, nothing else.

`Session` allocates the four caller-owned buffers once (one unified allocation),
binds them, and hands out torch tensors that alias the fixed views.  All arithmetic of the method
(planning, relayout) happens inside libmoebius.so.
"""
from __future__ import annotations

import numpy as np

from . import _binding as B

_W_DT = {"bf16": B.MOEBIUS_BF16, "fp32": B.MOEBIUS_FP32, "fp8_e4m3_b128": B.MOEBIUS_FP8_E4M3_B128}


def make_config(*, R, L, E, H, I, w_dtype="bf16", kv_heads, head_dim, page_tokens,
                kv_pool_bytes_per_rank_layer, max_requests, max_pages_per_request,
                staging_cap_bytes=0, kv_dtype="bf16", w_orient=0, n_q_heads=0, attn_mode=0,
                w_inplace=0) -> B.moebius_config_t:
    c = B.moebius_config_t()
    c.R, c.L, c.E, c.H, c.I = R, L, E, H, I
    c.w_dtype = _W_DT[w_dtype]
    c.w_orient = w_orient
    c.kv_heads, c.head_dim, c.page_tokens = kv_heads, head_dim, page_tokens
    c.kv_dtype = _W_DT[kv_dtype]
    c.kv_pool_bytes_per_rank_layer = int(kv_pool_bytes_per_rank_layer)
    c.max_requests, c.max_pages_per_request = max_requests, max_pages_per_request
    c.staging_cap_bytes = int(staging_cap_bytes)
    c.n_q_heads, c.attn_mode = n_q_heads, attn_mode
    c.w_inplace = w_inplace
    return c


class _RawCuda:
    """A device byte range that torch did not allocate, exposed through __cuda_array_interface__."""

    def __init__(self, ptr: int, nbytes: int):
        self.__cuda_array_interface__ = {"shape": (nbytes,), "typestr": "|u1", "data": (ptr, False), "version": 2}


class Session:
    """One context + its torch-owned device buffers.  `device=None` keeps it host-only (planner)."""

    def __init__(self, cfg: B.moebius_config_t, device=None, initial_mode: int = B.MOEBIUS_TP,
                 guard_bytes: int = 0, vmm: bool = False):
        """vmm=True: the unified buffer is a moebius_arena -- one virtual range, one physical allocation
        per rank (the address layout of a multi-GPU deployment, here with every rank on `device`)."""
        self.cfg = cfg
        self.ctx = B.moebius_create(cfg)
        self.layout = B.moebius_layout(self.ctx)
        self.device = device
        self.guard_bytes = guard_bytes
        self._plans = []
        self.vmm_arena = None
        if device is not None:
            import torch
            if not torch.cuda.is_available():
                raise RuntimeError("Session(device=...) needs a CUDA device; there is no CPU fallback")
            lay = self.layout
            g = guard_bytes
            al = lambda n: (int(n) + 255) // 256 * 256  # noqa: E731
            sizes = [0 if vmm else al(lay.base_bytes), al(max(lay.staging_bytes, 256)), al(lay.desc_bytes),
                     al(lay.table_bytes)]
            total = sum(s + g for s in sizes) + g
            self.arena = torch.empty(total, dtype=torch.uint8, device=device)
            assert self.arena.data_ptr() % 256 == 0
            offs, o = [], g
            for s in sizes:
                offs.append(o)
                o += s + g
            self._offs, self._sizes = offs, sizes
            if vmm:
                dev_index = torch.device(device).index or 0
                self.vmm_arena = B.moebius_arena_create(self.ctx, dev_index, 0, cfg.R)
                assert B.moebius_arena_ready(self.vmm_arena)
                self.base = torch.as_tensor(_RawCuda(B.moebius_arena_base(self.vmm_arena), int(lay.base_bytes)),
                                            device=device)
            else:
                self.base = self.arena[offs[0]:offs[0] + sizes[0]]
            self.staging = self.arena[offs[1]:offs[1] + sizes[1]]
            self.desc = self.arena[offs[2]:offs[2] + sizes[2]]
            self.tables = self.arena[offs[3]:offs[3] + sizes[3]].view(torch.int32)
            B.moebius_bind(self.ctx, self.base.data_ptr(), self.staging.data_ptr(), self.desc.data_ptr(),
                           self.tables.data_ptr(), initial_mode)

    def w_staging_offset(self) -> int:
        """Where the weight part of the staging buffer starts (its tail; S2 parks blocks there)."""
        return int(self.layout.staging_bytes - self.layout.w_staging_bytes)

    # -- views ------------------------------------------------------------------------------------
    def view_desc(self, mode, rank, layer, tensor_id) -> B.moebius_view_t:
        return B.moebius_view(self.ctx, mode, rank, layer, tensor_id)

    def view(self, mode, rank, layer, tensor_id):
        """torch tensor aliasing the fixed view (raw storage dtype: int16 / uint8 / float32)."""
        import torch
        v = self.view_desc(mode, rank, layer, tensor_id)
        shape = [v.shape[i] for i in range(v.ndim)]
        stride = [v.stride[i] for i in range(v.ndim)]
        dt = {1: torch.uint8, 2: torch.int16, 4: torch.float32}[v.elem_bytes]
        span = (sum((n - 1) * st for n, st in zip(shape, stride)) + 1) * v.elem_bytes   # a strided view spans more than its elements
        return self.base[v.offset:v.offset + span].view(dt).as_strided(shape, stride)

    def guards(self):
        """The guard strips between / around the buffers (for canary checks)."""
        g = self.guard_bytes
        if not g:
            return []
        out = [self.arena[0:g]]
        for o, s in zip(self._offs, self._sizes):
            out.append(self.arena[o + s:o + s + g])
        return out

    # -- the three calls --------------------------------------------------------------------------
    def plan(self, to_mode, seq_lens=None, src_owner=None, src_block_tables=None, from_mode=None):
        frm = B.moebius_active_mode(self.ctx) if from_mode is None else from_mode
        if frm < 0:
            frm = B.MOEBIUS_EP if to_mode == B.MOEBIUS_TP else B.MOEBIUS_TP
        p = B.moebius_plan(self.ctx, frm, to_mode, seq_lens, src_owner, src_block_tables)
        self._plans.append(p)
        return p

    def block_tables(self, plan, n_req):
        return B.moebius_block_tables(plan, n_req, self.cfg.max_pages_per_request)

    def reshard(self, plan, stream=None):
        import torch
        s = torch.cuda.current_stream(self.device) if stream is None else stream
        B.moebius_reshard(self.ctx, plan, s.cuda_stream)

    def stage(self, plan):
        """Copies the plan into the fixed pinned mailbox (host side of a graph-captured switch)."""
        B.moebius_stage_plan(self.ctx, plan)

    def reshard_staged(self, stream=None):
        """Plan-independent enqueue of the staged switch; legal under CUDA-graph capture."""
        import torch
        s = torch.cuda.current_stream(self.device) if stream is None else stream
        B.moebius_reshard_staged(self.ctx, s.cuda_stream)

    def free_plan(self, plan):
        self._plans = [p for p in self._plans if p.value != plan.value]
        B.moebius_plan_destroy(plan)

    def close(self):
        for p in self._plans:
            B.moebius_plan_destroy(p)
        self._plans = []
        if self.vmm_arena is not None:
            import torch
            torch.cuda.synchronize()
            self.base = None
            B.moebius_arena_destroy(self.vmm_arena)
            self.vmm_arena = None
        if self.ctx:
            B.moebius_destroy(self.ctx)
            self.ctx = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass
