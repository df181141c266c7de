"""Thin Python binding of the C ABI in include/sp.h (argument marshalling only).

Every step of the path runs in the library's CUDA kernels; torch is used for device memory and the
current stream.  There is no CPU fallback: if libsp.so is missing or cannot be loaded this module
raises.  Function names and argument meaning are those of include/sp.h.
"""
from __future__ import annotations

import ctypes as C
import math
import os
from dataclasses import dataclass
from typing import Optional, Sequence

import torch

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libsp.so")

SP_OK, SP_ERR_INVALID_ARG, SP_ERR_UNSUPPORTED, SP_ERR_WORKSPACE, SP_ERR_CUDA, SP_ERR_TOO_LARGE = 0, -1, -2, -3, -4, -5
SP_MODE_ORACLE, SP_MODE_INDEXER = 0, 1
SP_F_RELU, SP_F_KEY_LN, SP_F_ROPE = 1, 2, 4   # sp_params.flags: the served scorer of PAPER.md:270-274
SP_F_GROUP_SUPPORT = 8                        # idx is [Hkv, n_rows, k]: one list per KV group
SP_F_HEAD_SUPPORT = 16                        # idx is [Hq, n_rows, k]: one list per query head
(SP_STAGE_INDEXER_SCORES, SP_STAGE_ORACLE_MASS, SP_STAGE_TOPK, SP_STAGE_SPARSE_ATTN, SP_STAGE_DENSE_ATTN,
 SP_STAGE_LAYER_ORACLE, SP_STAGE_LAYER_INDEXER) = range(7)

EXPORTS = (
    "sp_num_rows", "sp_workspace_bytes", "sp_indexer_scores", "sp_oracle_mass", "sp_topk_support",
    "sp_sparse_gqa_attn", "sp_dense_gqa_attn", "sp_prefill_layer", "sp_layer_host_arena_bytes",
    "sp_prefill_layer_host", "sp_strerror", "sp_launch_count", "sp_sparse_gqa_attn_static", "sp_support_overlap", "sp_row_kl",
    "sp_oracle_mass_group", "sp_gather_probe", "sp_kv_append", "sp_kv_gather", "sp_chunk_workspace_bytes",
    "sp_prefill_chunk", "sp_oracle_mass_head",
)


class SpParams(C.Structure):
    _fields_ = [
        ("batch", C.c_int32), ("L", C.c_int32),
        ("cu_seqlens", C.c_void_p), ("cu_seqlens_host", C.c_void_p),
        ("Hq", C.c_int32), ("Hkv", C.c_int32), ("d", C.c_int32),
        ("k", C.c_int32), ("b_sel", C.c_int32), ("hidden", C.c_int32), ("d_idx", C.c_int32),
        ("scale", C.c_float), ("idx_scale", C.c_float),
        ("local_window", C.c_int32), ("local_bias", C.c_float), ("flags", C.c_uint32),
    ]


class SpKvPages(C.Structure):
    _fields_ = [
        ("k_pages", C.c_void_p), ("v_pages", C.c_void_p), ("kidx_pages", C.c_void_p), ("block_table", C.c_void_p),
        ("n_blocks", C.c_int32), ("page_size", C.c_int32), ("n_pages", C.c_int32),
    ]


class SpError(RuntimeError):
    def __init__(self, code: int, text: str):
        super().__init__(f"sp error {code}: {text}")
        self.code = code


_lib = None


def lib() -> C.CDLL:
    """Load libsp.so (in-tree).  Fails loudly when the CUDA extension has not been built."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise RuntimeError(f"{LIB_PATH} is missing: run `python -m paper_2606_07703_b200.build` "
                               "(there is no fallback path)")
        _lib = C.CDLL(LIB_PATH)
        _lib.sp_strerror.restype = C.c_char_p
        _lib.sp_num_rows.restype = C.c_int64
        _lib.sp_launch_count.restype = C.c_int64
    return _lib


def _check(rc: int):
    if rc != SP_OK:
        raise SpError(rc, lib().sp_strerror(C.c_int(rc)).decode())


@dataclass
class Problem:
    """Host-side mirror of sp_params; owns the cu_seqlens copies."""
    L: int
    Hq: int
    Hkv: int
    d: int
    k: int
    b_sel: int = 1
    hidden: int = 0
    d_idx: int = 0
    scale: float = 0.0
    idx_scale: float = 0.0
    local_window: int = 0
    local_bias: float = 0.0
    cu_seqlens: Optional[Sequence[int]] = None
    flags: int = 0
    device: str = "cuda"

    def __post_init__(self):
        self._cu_host = None
        self._cu_dev = None
        if self.cu_seqlens is not None:
            self._cu_host = torch.tensor(list(self.cu_seqlens), dtype=torch.int32)
            self._cu_dev = self._cu_host.to(self.device)

    @property
    def batch(self) -> int:
        return 1 if self.cu_seqlens is None else len(self.cu_seqlens) - 1

    def c(self) -> SpParams:
        return SpParams(
            self.batch, self.L,
            self._cu_dev.data_ptr() if self._cu_dev is not None else None,
            self._cu_host.data_ptr() if self._cu_host is not None else None,
            self.Hq, self.Hkv, self.d, self.k, self.b_sel, self.hidden, self.d_idx,
            self.scale, self.idx_scale, self.local_window, self.local_bias, self.flags)

    @property
    def num_rows(self) -> int:
        p = self.c()
        n = lib().sp_num_rows(C.byref(p))
        if n < 0:
            _check(int(n))
        return int(n)

    @property
    def max_seqlen(self) -> int:
        if self.cu_seqlens is None:
            return self.L
        cu = list(self.cu_seqlens)
        return max(b - a for a, b in zip(cu[:-1], cu[1:]))

    @classmethod
    def from_config(cls, cfg, device="cuda", **over):
        kw = dict(L=cfg.L, Hq=cfg.Hq, Hkv=cfg.Hkv, d=cfg.d, k=cfg.k, b_sel=cfg.b_sel, hidden=cfg.hidden,
                  d_idx=cfg.d_idx, local_window=cfg.local_window, local_bias=cfg.local_bias,
                  cu_seqlens=cfg.cu_seqlens, flags=getattr(cfg, "flags", 0), device=device)
        kw.update(over)
        return cls(**kw)


def _ptr(t: Optional[torch.Tensor]):
    if t is None:
        return None
    assert t.is_contiguous(), "tensors crossing the ABI must be contiguous"
    return C.c_void_p(t.data_ptr())


def _stream() -> C.c_void_p:
    return C.c_void_p(torch.cuda.current_stream().cuda_stream)


def workspace_bytes(pb: Problem, stage: int) -> int:
    p = pb.c()
    out = C.c_size_t(0)
    _check(lib().sp_workspace_bytes(C.byref(p), C.c_int(stage), C.byref(out)))
    return int(out.value)


def alloc_workspace(pb: Problem, stage: int) -> torch.Tensor:
    return torch.empty(max(workspace_bytes(pb, stage), 256), dtype=torch.uint8, device=pb.device)


def _ws_args(ws: Optional[torch.Tensor]):
    if ws is None:
        return None, C.c_size_t(0)
    return C.c_void_p(ws.data_ptr()), C.c_size_t(ws.numel() * ws.element_size())


def sp_indexer_scores(pb: Problem, X, Wqi, Wki, q_idx, k_idx, preprojected: bool, row_begin: int, row_count: int,
                      scores: torch.Tensor, ws: Optional[torch.Tensor] = None):
    p = pb.c()
    wp, wb = _ws_args(ws)
    _check(lib().sp_indexer_scores(C.byref(p), _ptr(X), _ptr(Wqi), _ptr(Wki), _ptr(q_idx), _ptr(k_idx),
                                   C.c_int32(1 if preprojected else 0), C.c_int32(row_begin), C.c_int32(row_count),
                                   _ptr(scores), C.c_int64(scores.stride(0)), wp, wb, _stream()))


def sp_oracle_mass(pb: Problem, Q, K, lse: Optional[torch.Tensor], lse_ready: bool, row_begin: int, row_count: int,
                   mass: torch.Tensor, ws: Optional[torch.Tensor] = None):
    p = pb.c()
    wp, wb = _ws_args(ws)
    _check(lib().sp_oracle_mass(C.byref(p), _ptr(Q), _ptr(K), _ptr(lse), C.c_int32(1 if lse_ready else 0),
                                C.c_int32(row_begin), C.c_int32(row_count), _ptr(mass), C.c_int64(mass.stride(0)),
                                wp, wb, _stream()))


def sp_oracle_mass_group(pb: Problem, Q, K, lse: Optional[torch.Tensor], lse_ready: bool, group: int, row_begin: int,
                         row_count: int, mass: torch.Tensor, ws: Optional[torch.Tensor] = None):
    p = pb.c()
    wp, wb = _ws_args(ws)
    _check(lib().sp_oracle_mass_group(C.byref(p), _ptr(Q), _ptr(K), _ptr(lse), C.c_int32(1 if lse_ready else 0),
                                      C.c_int32(group), C.c_int32(row_begin), C.c_int32(row_count), _ptr(mass),
                                      C.c_int64(mass.stride(0)), wp, wb, _stream()))


def sp_oracle_mass_head(pb: Problem, Q, K, lse: Optional[torch.Tensor], lse_ready: bool, head: int, row_begin: int,
                        row_count: int, mass: torch.Tensor, ws: Optional[torch.Tensor] = None):
    p = pb.c()
    wp, wb = _ws_args(ws)
    _check(lib().sp_oracle_mass_head(C.byref(p), _ptr(Q), _ptr(K), _ptr(lse), C.c_int32(1 if lse_ready else 0),
                                     C.c_int32(head), C.c_int32(row_begin), C.c_int32(row_count), _ptr(mass),
                                     C.c_int64(mass.stride(0)), wp, wb, _stream()))


def sp_topk_support(pb: Problem, scores: torch.Tensor, row_begin: int, row_count: int, idx: torch.Tensor,
                    cnt: Optional[torch.Tensor] = None, ws: Optional[torch.Tensor] = None):
    p = pb.c()
    wp, wb = _ws_args(ws)
    _check(lib().sp_topk_support(C.byref(p), _ptr(scores), C.c_int64(scores.stride(0)), C.c_int32(row_begin),
                                 C.c_int32(row_count), _ptr(idx), _ptr(cnt), wp, wb, _stream()))


def sp_sparse_gqa_attn(pb: Problem, Q, K, V, idx, O, lse: Optional[torch.Tensor] = None,
                       ws: Optional[torch.Tensor] = None):
    p = pb.c()
    if idx.dim() == 3:   # one support list per KV group [Hkv, n_rows, k] or per head [Hq, n_rows, k]
        assert idx.is_contiguous(), "index tensors crossing the ABI must be contiguous"
        p.flags &= ~(SP_F_GROUP_SUPPORT | SP_F_HEAD_SUPPORT)
        if pb.flags & SP_F_HEAD_SUPPORT or (idx.shape[0] == pb.Hq and pb.Hq != pb.Hkv):
            assert idx.shape[0] == pb.Hq, idx.shape
            p.flags |= SP_F_HEAD_SUPPORT
        else:
            assert idx.shape[0] == pb.Hkv, idx.shape
            p.flags |= SP_F_GROUP_SUPPORT
    wp, wb = _ws_args(ws)
    _check(lib().sp_sparse_gqa_attn(C.byref(p), _ptr(Q), _ptr(K), _ptr(V), _ptr(idx), _ptr(O), _ptr(lse), wp, wb,
                                    _stream()))


def sp_sparse_gqa_attn_static(pb: Problem, Q, K, V, idx, O, lse: Optional[torch.Tensor] = None):
    """The no-allocation entry point: per-query lists through the masked tile loop, bitmap in the library's fixed array."""
    p = pb.c()
    _check(lib().sp_sparse_gqa_attn_static(C.byref(p), _ptr(Q), _ptr(K), _ptr(V), _ptr(idx), _ptr(O), _ptr(lse), _stream()))


def sp_dense_gqa_attn(pb: Problem, Q, K, V, O, lse: Optional[torch.Tensor] = None,
                      ws: Optional[torch.Tensor] = None):
    p = pb.c()
    wp, wb = _ws_args(ws)
    _check(lib().sp_dense_gqa_attn(C.byref(p), _ptr(Q), _ptr(K), _ptr(V), _ptr(O), _ptr(lse), wp, wb, _stream()))


def sp_prefill_layer(pb: Problem, mode: int, X, Wqi, Wki, Q, K, V, O, idx_out: Optional[torch.Tensor],
                     ws: torch.Tensor):
    p = pb.c()
    wp, wb = _ws_args(ws)
    _check(lib().sp_prefill_layer(C.byref(p), C.c_int32(mode), _ptr(X), _ptr(Wqi), _ptr(Wki), _ptr(Q), _ptr(K),
                                  _ptr(V), _ptr(O), _ptr(idx_out), wp, wb, _stream()))


def layer_host_arena_bytes(pb: Problem, mode: int) -> int:
    p = pb.c()
    out = C.c_size_t(0)
    _check(lib().sp_layer_host_arena_bytes(C.byref(p), C.c_int32(mode), C.byref(out)))
    return int(out.value)


def sp_prefill_layer_host(pb: Problem, mode: int, X, Wqi, Wki, Q, K, V, O, arena: torch.Tensor):
    """X..O are HOST (pinned) tensors; arena is device scratch."""
    p = pb.c()
    wp, wb = _ws_args(arena)
    _check(lib().sp_prefill_layer_host(C.byref(p), C.c_int32(mode), _ptr(X), _ptr(Wqi), _ptr(Wki), _ptr(Q), _ptr(K),
                                       _ptr(V), _ptr(O), wp, wb, _stream()))


def sp_support_overlap(pb: Problem, idx_a: torch.Tensor, idx_b: torch.Tensor, inter: torch.Tensor):
    p = pb.c()
    _check(lib().sp_support_overlap(C.byref(p), _ptr(idx_a), _ptr(idx_b), _ptr(inter), _stream()))


def sp_row_kl(pb: Problem, mass: torch.Tensor, scores: torch.Tensor, row_begin: int, row_count: int, kl: torch.Tensor):
    p = pb.c()
    _check(lib().sp_row_kl(C.byref(p), _ptr(mass), C.c_int64(mass.stride(0)), _ptr(scores), C.c_int64(scores.stride(0)),
                           C.c_int32(row_begin), C.c_int32(row_count), _ptr(kl), _stream()))


def sp_gather_probe(base: torch.Tensor, row_bytes: int, row_pitch_bytes: int, idx: torch.Tensor, sink: torch.Tensor):
    """Plain gather of idx.numel() rows of row_bytes bytes (measurement aid, see include/sp.h)."""
    _check(lib().sp_gather_probe(_ptr(base), C.c_int32(row_bytes), C.c_int64(row_pitch_bytes), _ptr(idx),
                                 C.c_int64(idx.numel()), _ptr(sink), C.c_size_t(sink.numel() * sink.element_size()),
                                 _stream()))


@dataclass
class KvPages:
    """Host-side mirror of sp_kv_pages: torch tensors of one sequence's paged cache (include/sp.h)."""
    k_pages: torch.Tensor                 # [n_pages, page_size, Hkv, d] bf16
    v_pages: torch.Tensor
    kidx_pages: Optional[torch.Tensor]    # [n_pages, page_size, d_idx] bf16
    block_table: torch.Tensor             # [n_blocks] int32, device

    def c(self) -> SpKvPages:
        return SpKvPages(self.k_pages.data_ptr(), self.v_pages.data_ptr(),
                         self.kidx_pages.data_ptr() if self.kidx_pages is not None else None,
                         self.block_table.data_ptr(), int(self.block_table.numel()), int(self.k_pages.shape[1]),
                         int(self.k_pages.shape[0]))


def sp_kv_append(pb: Problem, kv: KvPages, t_begin: int, t_count: int, K_new, V_new, kidx_new=None):
    p, c = pb.c(), kv.c()
    _check(lib().sp_kv_append(C.byref(p), C.byref(c), C.c_int32(t_begin), C.c_int32(t_count), _ptr(K_new), _ptr(V_new),
                              _ptr(kidx_new), _stream()))


def sp_kv_gather(pb: Problem, kv: KvPages, t_begin: int, t_count: int, K_out, V_out, kidx_out=None):
    p, c = pb.c(), kv.c()
    _check(lib().sp_kv_gather(C.byref(p), C.byref(c), C.c_int32(t_begin), C.c_int32(t_count), _ptr(K_out), _ptr(V_out),
                              _ptr(kidx_out), _stream()))


def chunk_workspace_bytes(pb: Problem, q_begin: int, q_count: int) -> int:
    p = pb.c()
    out = C.c_size_t(0)
    _check(lib().sp_chunk_workspace_bytes(C.byref(p), C.c_int32(q_begin), C.c_int32(q_count), C.byref(out)))
    return int(out.value)


def sp_prefill_chunk(pb: Problem, q_begin: int, q_count: int, X, Wqi, Wki, Q, K_new, V_new, kv: KvPages, O,
                     idx_out: Optional[torch.Tensor], ws: torch.Tensor):
    """pb.L must be q_begin + q_count (the context length after the chunk)."""
    p, c = pb.c(), kv.c()
    wp, wb = _ws_args(ws)
    _check(lib().sp_prefill_chunk(C.byref(p), C.c_int32(q_begin), C.c_int32(q_count), _ptr(X), _ptr(Wqi), _ptr(Wki),
                                  _ptr(Q), _ptr(K_new), _ptr(V_new), C.byref(c), _ptr(O), _ptr(idx_out), wp, wb,
                                  _stream()))


def launch_count() -> int:
    return int(lib().sp_launch_count())


def bf16_tensor(u16, device="cuda") -> torch.Tensor:
    """uint16 bit patterns (numpy) -> torch.bfloat16 tensor on `device` with the same bytes."""
    t = torch.from_numpy(u16.view("int16")).view(torch.bfloat16)
    return t.to(device) if device != "cpu" else t
