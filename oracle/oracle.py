"""ctypes binding and step composition for the CPU fp64 ORACLE (oracle/sp_oracle.c).

TEST INFRASTRUCTURE, NOT THE PRODUCT: only tests/, __graft_entry__.smoke() and bench.py's
cpu_baseline / --impl reference legs may import this module.  It imports nothing from the CUDA
package and never receives a value the CUDA path produced.

All tensors are numpy arrays; bf16 tensors are uint16 bit patterns.  Step names O1..O7 and the
PAPER.md citations are in sp_oracle.c's header.  This file only marshals arguments and chains the
steps in the paper's order (Alg.1 steps 2-5; Alg.2 steps 2,4,5).
"""
from __future__ import annotations

import ctypes as C
import math
import os
import subprocess
from dataclasses import dataclass
from typing import Optional, Sequence

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "sp_oracle.c")
_LIB = os.path.join(_HERE, "libsp_oracle.so")

MODE_ORACLE = 0
MODE_INDEXER = 1


def build(force: bool = False) -> str:
    """Compile sp_oracle.c with gcc (fp64, OpenMP, no fast-math, no FMA contraction)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        cmd = ["gcc", "-O2", "-ffp-contract=off", "-fopenmp", "-shared", "-fPIC", "-o", _LIB, _SRC, "-lm"]
        subprocess.run(cmd, check=True)
    return _LIB


class _Params(C.Structure):
    _fields_ = [
        ("batch", C.c_int32), ("L", C.c_int32), ("cu_seqlens", C.POINTER(C.c_int32)),
        ("Hq", C.c_int32), ("Hkv", C.c_int32), ("d", C.c_int32), ("k", C.c_int32),
        ("b_sel", C.c_int32), ("hidden", C.c_int32), ("d_idx", C.c_int32),
        ("scale", C.c_double), ("idx_scale", C.c_double),
        ("local_window", C.c_int32), ("local_bias", C.c_double), ("flags", C.c_int32),
    ]


@dataclass
class Problem:
    """The paper's problem statement for one layer."""
    L: int
    Hq: int
    Hkv: int
    d: int
    k: int
    b_sel: int = 1
    hidden: int = 0
    d_idx: int = 0
    scale: Optional[float] = None        # None -> 1/sqrt(d)
    idx_scale: Optional[float] = None    # None -> 1/sqrt(d_idx)
    local_window: int = 0
    local_bias: float = 0.0
    cu_seqlens: Optional[Sequence[int]] = None
    flags: int = 0                       # F_RELU | F_KEY_LN | F_ROPE: the served scorer

    def c_params(self):
        cu = None
        batch = 1
        keep = None
        if self.cu_seqlens is not None:
            keep = np.ascontiguousarray(np.asarray(self.cu_seqlens, dtype=np.int32))
            cu = keep.ctypes.data_as(C.POINTER(C.c_int32))
            batch = len(keep) - 1
        p = _Params(
            batch, self.L, cu, self.Hq, self.Hkv, self.d, self.k, self.b_sel, self.hidden, self.d_idx,
            self.scale if self.scale is not None else 1.0 / math.sqrt(self.d),
            self.idx_scale if self.idx_scale is not None else (1.0 / math.sqrt(self.d_idx) if self.d_idx else 0.0),
            self.local_window, self.local_bias, self.flags,
        )
        p._keep = keep
        return p


_lib = None


def lib():
    global _lib
    if _lib is None:
        _lib = C.CDLL(build())
        _lib.orc_num_rows.restype = C.c_int32
        _lib.orc_row_info.restype = C.c_int32
        _lib.orc_row_of_pos.restype = C.c_int32
        _lib.orc_max_threads.restype = C.c_int32
    return _lib


def _u16(a):
    a = np.ascontiguousarray(a)
    assert a.dtype == np.uint16, a.dtype
    return a


def _i32(a):
    return np.ascontiguousarray(np.asarray(a, dtype=np.int32))


def _ptr(a, ty):
    return a.ctypes.data_as(C.POINTER(ty))


def max_threads() -> int:
    return int(lib().orc_max_threads())


def f64_to_bf16(x) -> np.ndarray:
    x = np.ascontiguousarray(np.asarray(x, dtype=np.float64))
    out = np.empty(x.shape, dtype=np.uint16)
    lib().orc_f64_to_bf16(_ptr(x, C.c_double), C.c_int64(x.size), _ptr(out, C.c_uint16))
    return out


def bf16_to_f64(b) -> np.ndarray:
    b = np.ascontiguousarray(b, dtype=np.uint16)
    return (b.astype(np.uint32) << 16).view(np.float32).astype(np.float64)


def num_rows(pb: Problem) -> int:
    p = pb.c_params()
    return int(lib().orc_num_rows(C.byref(p)))


def row_info(pb: Problem, row: int):
    """(seq_start, first local position, last local position) of a support row (A8)."""
    p = pb.c_params()
    a, b, c = C.c_int32(), C.c_int32(), C.c_int32()
    rc = lib().orc_row_info(C.byref(p), C.c_int32(row), C.byref(a), C.byref(b), C.byref(c))
    if rc != 0:
        raise IndexError(row)
    return a.value, b.value, c.value


def row_of_pos(pb: Problem, pos: int) -> int:
    p = pb.c_params()
    return int(lib().orc_row_of_pos(C.byref(p), C.c_int32(pos)))


F_RELU, F_KEY_LN, F_ROPE = 1, 2, 4


def project(pb: Problem, X, W, rows=None, key: bool = False) -> np.ndarray:
    """O3' projection: bf16_rne(T(X[rows] @ W)) with an fp64 sum (A14); T = key LayerNorm
    (key side only) and RoPE when pb.flags asks for them (A27, A28), else the identity."""
    X, W = _u16(X), _u16(W)
    rows = _i32(np.arange(X.shape[0]) if rows is None else rows)
    out = np.empty((len(rows), pb.d_idx), dtype=np.uint16)
    cp = pb.c_params()
    lib().orc_project(C.byref(cp), _ptr(X, C.c_uint16), _ptr(W, C.c_uint16), C.c_int32(1 if key else 0),
                      _ptr(rows, C.c_int32), C.c_int32(len(rows)), _ptr(out, C.c_uint16))
    return out


def transform(y, pos_local: int, flags: int, key: bool) -> np.ndarray:
    """The fp64 core of the served scorer's per-token transform (LayerNorm then RoPE), for the pins."""
    y = np.ascontiguousarray(np.asarray(y, dtype=np.float64)).copy()
    lib().orc_transform(y.ctypes.data_as(C.POINTER(C.c_double)), C.c_int32(y.shape[0]), C.c_int32(pos_local),
                        C.c_int32(flags), C.c_int32(1 if key else 0))
    return y


def query_scores(pb: Problem, mode: int, A, B, pos, ld: Optional[int] = None) -> np.ndarray:
    """Per-query score rows: mass P_t (mode ORACLE; A=Q, B=K) or indexer logits
    (mode INDEXER; A=q_idx, B=k_idx).  Returns [len(pos), ld] fp64, -inf beyond t."""
    A, B = _u16(A), _u16(B)
    pos = _i32(pos)
    ld = int(ld or pb.L)
    out = np.empty((len(pos), ld), dtype=np.float64)
    p = pb.c_params()
    lib().orc_query_scores(C.byref(p), C.c_int32(mode), _ptr(A, C.c_uint16), _ptr(B, C.c_uint16),
                           _ptr(pos, C.c_int32), C.c_int32(len(pos)), _ptr(out, C.c_double), C.c_int64(ld))
    return out


def support_scores(pb: Problem, mode: int, A, B, rows, ld: Optional[int] = None):
    """O4: support-row scores R. Returns (R [len(rows), ld] fp64, n_valid int32)."""
    A, B = _u16(A), _u16(B)
    rows = _i32(rows)
    ld = int(ld or pb.L)
    out = np.empty((len(rows), ld), dtype=np.float64)
    nv = np.empty(len(rows), dtype=np.int32)
    p = pb.c_params()
    lib().orc_support_scores(C.byref(p), C.c_int32(mode), _ptr(A, C.c_uint16), _ptr(B, C.c_uint16),
                             _ptr(rows, C.c_int32), C.c_int32(len(rows)), _ptr(out, C.c_double),
                             C.c_int64(ld), _ptr(nv, C.c_int32))
    return out, nv


def topk(scores, n_valid, k: int, seq_start=None):
    """O5: per row the first min(k,n) of (score desc, index asc), ascending, -1 padded."""
    scores = np.ascontiguousarray(np.asarray(scores, dtype=np.float64))
    if scores.ndim == 1:
        scores = scores[None, :]
    n_valid = _i32(n_valid)
    nrows, ld = scores.shape
    idx = np.empty((nrows, k), dtype=np.int32)
    cnt = np.empty(nrows, dtype=np.int32)
    ss = _i32(seq_start) if seq_start is not None else None
    lib().orc_topk(_ptr(scores, C.c_double), C.c_int64(ld), _ptr(n_valid, C.c_int32),
                   _ptr(ss, C.c_int32) if ss is not None else None,
                   C.c_int32(nrows), C.c_int32(k), _ptr(idx, C.c_int32), _ptr(cnt, C.c_int32))
    return idx, cnt


def sparse_attn(pb: Problem, Q, K, V, pos, sup, want_lse: bool = False):
    """O6: attention recomputed on the support. sup: [len(pos), k] packed idx."""
    Q, K, V = _u16(Q), _u16(K), _u16(V)
    pos = _i32(pos)
    sup = _i32(sup)
    assert sup.shape == (len(pos), pb.k), (sup.shape, len(pos), pb.k)
    o = np.empty((len(pos), pb.Hq, pb.d), dtype=np.float64)
    lse = np.empty((len(pos), pb.Hq), dtype=np.float64)
    p = pb.c_params()
    lib().orc_sparse_attn(C.byref(p), _ptr(Q, C.c_uint16), _ptr(K, C.c_uint16), _ptr(V, C.c_uint16),
                          _ptr(pos, C.c_int32), C.c_int32(len(pos)), _ptr(sup, C.c_int32),
                          _ptr(o, C.c_double), _ptr(lse, C.c_double))
    return (o, lse) if want_lse else o


def dense_attn(pb: Problem, Q, K, V, pos, want_lse: bool = False):
    """O7: dense causal GQA attention by brute force."""
    Q, K, V = _u16(Q), _u16(K), _u16(V)
    pos = _i32(pos)
    o = np.empty((len(pos), pb.Hq, pb.d), dtype=np.float64)
    lse = np.empty((len(pos), pb.Hq), dtype=np.float64)
    p = pb.c_params()
    lib().orc_dense_attn(C.byref(p), _ptr(Q, C.c_uint16), _ptr(K, C.c_uint16), _ptr(V, C.c_uint16),
                         _ptr(pos, C.c_int32), C.c_int32(len(pos)), _ptr(o, C.c_double), _ptr(lse, C.c_double))
    return (o, lse) if want_lse else o


# ---------------------------------------------------------------------------------------------
# Composition in the paper's order
# ---------------------------------------------------------------------------------------------

@dataclass
class LayerResult:
    rows: np.ndarray        # support rows evaluated
    scores: np.ndarray      # R [len(rows), ld] fp64
    n_valid: np.ndarray     # [len(rows)]
    idx: np.ndarray         # [len(rows), k] packed positions, ascending, -1 padded
    cnt: np.ndarray         # [len(rows)]
    pos: np.ndarray         # query positions whose outputs were computed
    out: np.ndarray         # [len(pos), Hq, d] fp64
    q_idx: Optional[np.ndarray] = None
    k_idx: Optional[np.ndarray] = None


def select_support(pb: Problem, mode: int, A, B, rows):
    """Alg.1 steps 2-4 / Alg.2 steps 4-5 (first half): scores -> causal top-k for the given rows."""
    rows = _i32(rows)
    R, nv = support_scores(pb, mode, A, B, rows)
    starts = np.array([row_info(pb, int(r))[0] for r in rows], dtype=np.int32)
    idx, cnt = topk(R, nv, pb.k, starts)
    return R, nv, idx, cnt


def prefill_layer(pb: Problem, mode: int, Q, K, V, X=None, Wqi=None, Wki=None,
                  rows=None, pos=None, q_idx=None, k_idx=None) -> LayerResult:
    """One patched layer on a subset of support rows (all when rows is None).

    ORACLE mode: Alg.1 steps 2-5. INDEXER mode: Alg.2 steps 2,4,5.
    `pos` (query positions whose output is computed) defaults to every query of the chosen rows.
    """
    rows = _i32(np.arange(num_rows(pb)) if rows is None else rows)
    if mode == MODE_INDEXER:
        if q_idx is None:
            q_idx = project(pb, X, Wqi)
        if k_idx is None:
            k_idx = project(pb, X, Wki, key=True)
        A, B = q_idx, k_idx
    else:
        A, B = Q, K
    R, nv, idx, cnt = select_support(pb, mode, A, B, rows)
    if pos is None:
        pos = []
        for r in rows:
            s0, t0, t1 = row_info(pb, int(r))
            pos.extend(range(s0 + t0, s0 + t1 + 1))
    pos = _i32(pos)
    row_index = {int(r): i for i, r in enumerate(rows)}
    sup = np.stack([idx[row_index[row_of_pos(pb, int(t))]] for t in pos]) if len(pos) else np.empty((0, pb.k), np.int32)
    out = sparse_attn(pb, Q, K, V, pos, sup)
    return LayerResult(rows, R, nv, idx, cnt, pos, out, q_idx, k_idx)


# ---------------------------------------------------------------- per-KV-group support
# ORACLE GROUNDWORK FOR SURVEY.md 8(f) f4: no CUDA path yet.  The paper names the variant -- one support
# S_{l,t,r} shared by the query heads with g(h) = r (:100) -- and says it does not evaluate it (:133, :137);
# the reading taken here (A29): the mass of group r is the mean over ITS G = Hq/Hkv query heads,
# P_r[t,s] = (1/G) sum_{h: g(h)=r} A[t,h,s], everything else (block max, top-k, tie rule, recompute) as for the
# head-averaged support.  That is literally the head-averaged definition applied to the sub-problem
# (Q[:, rG:(r+1)G], K[:, r], V[:, r]) with Hq' = G, Hkv' = 1, which is how it is written out below.

def _group_problem(pb: Problem) -> Problem:
    G = pb.Hq // pb.Hkv
    return Problem(L=pb.L, Hq=G, Hkv=1, d=pb.d, k=pb.k, b_sel=pb.b_sel, scale=pb.scale,
                   local_window=pb.local_window, local_bias=pb.local_bias, cu_seqlens=pb.cu_seqlens)


def _group_slices(pb: Problem, Q, K, V, r: int):
    G = pb.Hq // pb.Hkv
    Q = _u16(Q).reshape(pb.L, pb.Hq, pb.d)
    K = _u16(K).reshape(pb.L, pb.Hkv, pb.d)
    V = _u16(V).reshape(pb.L, pb.Hkv, pb.d) if V is not None else None
    return (np.ascontiguousarray(Q[:, r * G:(r + 1) * G]), np.ascontiguousarray(K[:, r:r + 1]),
            np.ascontiguousarray(V[:, r:r + 1]) if V is not None else None)


def select_support_per_group(pb: Problem, Q, K, rows):
    """Oracle-mode supports per KV group: idx [Hkv, len(rows), k], cnt [Hkv, len(rows)]."""
    gp = _group_problem(pb)
    idx, cnt = [], []
    for r in range(pb.Hkv):
        Qr, Kr, _ = _group_slices(pb, Q, K, None, r)
        _, _, i, c = select_support(gp, MODE_ORACLE, Qr, Kr, rows)
        idx.append(i)
        cnt.append(c)
    return np.stack(idx), np.stack(cnt)


def sparse_attn_per_group(pb: Problem, Q, K, V, pos, sup):
    """O6 with one support per KV group: sup [Hkv, len(pos), k]; head h attends S_{r(t), g(h)}."""
    gp = _group_problem(pb)
    G = pb.Hq // pb.Hkv
    pos = _i32(pos)
    out = np.empty((len(pos), pb.Hq, pb.d), dtype=np.float64)
    for r in range(pb.Hkv):
        Qr, Kr, Vr = _group_slices(pb, Q, K, V, r)
        out[:, r * G:(r + 1) * G] = sparse_attn(gp, Qr, Kr, Vr, pos, sup[r])
    return out


# ---------------------------------------------------------------- per-head support ("separately per query head")
# S_{l,t,h}: head h's own attention distribution A[t,h,.] is its mass (the head "mean" over one head); block max, top-k,
# tie rule and recompute as for the head-averaged support -- the head-averaged definition on the sub-problem
# (Q[:, h], K[:, g(h)], V[:, g(h)]) with Hq' = Hkv' = 1.  The paper names the variant and evaluates none (:133, :137).

def _head_problem(pb: Problem) -> Problem:
    return Problem(L=pb.L, Hq=1, Hkv=1, d=pb.d, k=pb.k, b_sel=pb.b_sel, scale=pb.scale,
                   local_window=pb.local_window, local_bias=pb.local_bias, cu_seqlens=pb.cu_seqlens)


def _head_slices(pb: Problem, Q, K, V, h: int):
    G = pb.Hq // pb.Hkv
    Q = _u16(Q).reshape(pb.L, pb.Hq, pb.d)
    K = _u16(K).reshape(pb.L, pb.Hkv, pb.d)
    V = _u16(V).reshape(pb.L, pb.Hkv, pb.d) if V is not None else None
    r = h // G                                                   # g(h), A5
    return (np.ascontiguousarray(Q[:, h:h + 1]), np.ascontiguousarray(K[:, r:r + 1]),
            np.ascontiguousarray(V[:, r:r + 1]) if V is not None else None)


def select_support_per_head(pb: Problem, Q, K, rows):
    """Oracle-mode supports per query head: idx [Hq, len(rows), k], cnt [Hq, len(rows)]."""
    hp = _head_problem(pb)
    idx, cnt = [], []
    for h in range(pb.Hq):
        Qh, Kh, _ = _head_slices(pb, Q, K, None, h)
        _, _, i, c = select_support(hp, MODE_ORACLE, Qh, Kh, rows)
        idx.append(i)
        cnt.append(c)
    return np.stack(idx), np.stack(cnt)


def sparse_attn_per_head(pb: Problem, Q, K, V, pos, sup):
    """O6 with one support per head: sup [Hq, len(pos), k]; head h attends S_{r(t), h}."""
    hp = _head_problem(pb)
    pos = _i32(pos)
    out = np.empty((len(pos), pb.Hq, pb.d), dtype=np.float64)
    for h in range(pb.Hq):
        Qh, Kh, Vh = _head_slices(pb, Q, K, V, h)
        out[:, h:h + 1] = sparse_attn(hp, Qh, Kh, Vh, pos, sup[h])
    return out


# ---------------------------------------------------------------- chunked prefill against a paged KV cache
# PAPER.md:292 (five-stage serving path, stage 4 "reconstruct K/V from the paged KV cache when the chunked path requires
# contiguous tensors"), :331 and :428 (chunks of max_num_batched_tokens = 4K / 8K queries against the whole prefix).
# Reading (A30): a chunk is the queries [q_begin, q_begin + q_count) of ONE sequence whose first q_begin
# tokens are already cached; the chunk first writes its own K, V (and indexer keys) into the cache, then every stage
# of the layer runs for the chunk's support rows against the cache's first q_begin + q_count tokens.  Selection blocks
# stay aligned to the sequence start, so q_begin must be a multiple of b_sel.  The oracle does literally what the
# paper's stage 4 says: it reconstructs contiguous tensors from the pages (pure indexing) and runs the SAME functions
# as for a full prefill -- the result for the chunk's queries must equal the full-prefill result bit for bit.

@dataclass
class PagedCache:
    """K / V / indexer-key pages: [n_pages, page_size, row_elems] uint16 each; block_table[i] = physical page of logical block i."""
    page_size: int
    block_table: np.ndarray
    k: np.ndarray
    v: np.ndarray
    kidx: Optional[np.ndarray] = None


def paged_scatter(cache: np.ndarray, block_table, page_size: int, t_begin: int, rows: np.ndarray):
    rows = _u16(rows).reshape(rows.shape[0], -1)
    bt = _i32(block_table)
    assert cache.dtype == np.uint16 and cache.flags.c_contiguous
    lib().orc_paged_scatter(_ptr(cache, C.c_uint16), _ptr(bt, C.c_int32), C.c_int32(page_size),
                            C.c_int64(rows.shape[1]), C.c_int32(t_begin), C.c_int32(t_begin + rows.shape[0]),
                            _ptr(rows, C.c_uint16))


def paged_gather(cache: np.ndarray, block_table, page_size: int, t_begin: int, t_end: int) -> np.ndarray:
    bt = _i32(block_table)
    assert cache.dtype == np.uint16 and cache.flags.c_contiguous
    row_elems = int(np.prod(cache.shape[2:]))
    out = np.empty((t_end - t_begin, row_elems), dtype=np.uint16)
    lib().orc_paged_gather(_ptr(cache, C.c_uint16), _ptr(bt, C.c_int32), C.c_int32(page_size), C.c_int64(row_elems),
                           C.c_int32(t_begin), C.c_int32(t_end), _ptr(out, C.c_uint16))
    return out


def prefill_chunk(pb: Problem, mode: int, q_begin: int, q_count: int, Q_chunk, K_chunk, V_chunk, cache: PagedCache,
                  X_chunk=None, Wqi=None, Wki=None, rows=None, pos=None) -> LayerResult:
    """One prefill chunk of one sequence against the paged cache (see the block comment above).  pb.L must be the
    context length q_begin + q_count.  The cache is UPDATED with the chunk's K, V (and k_idx).  `rows` / `pos` restrict
    the evaluation to some of the chunk's support rows / queries (absolute row numbers and positions)."""
    n_ctx = q_begin + q_count
    assert pb.cu_seqlens is None and pb.L == n_ctx and q_begin % pb.b_sel == 0
    ps, bt = cache.page_size, cache.block_table
    k_idx_chunk = None
    if mode == MODE_INDEXER:
        # projections of the chunk's tokens at their absolute positions (RoPE, A28)
        Xf = np.zeros((n_ctx, pb.hidden), np.uint16)
        Xf[q_begin:] = _u16(X_chunk).reshape(q_count, pb.hidden)
        chunk_pos = np.arange(q_begin, n_ctx)
        q_idx_chunk = project(pb, Xf, Wqi, rows=chunk_pos)
        k_idx_chunk = project(pb, Xf, Wki, rows=chunk_pos, key=True)
        paged_scatter(cache.kidx, bt, ps, q_begin, k_idx_chunk)
    paged_scatter(cache.k, bt, ps, q_begin, K_chunk)
    paged_scatter(cache.v, bt, ps, q_begin, V_chunk)
    # stage 4: contiguous K, V (k_idx) of the whole context from the pages
    K = paged_gather(cache.k, bt, ps, 0, n_ctx)
    V = paged_gather(cache.v, bt, ps, 0, n_ctx)
    Q = np.zeros((n_ctx, pb.Hq * pb.d), np.uint16)
    Q[q_begin:] = _u16(Q_chunk).reshape(q_count, -1)
    r0, r1 = q_begin // pb.b_sel, num_rows(pb)
    rows = _i32(np.arange(r0, r1) if rows is None else rows)
    assert rows.min() >= r0 and rows.max() < r1
    kw = {}
    if mode == MODE_INDEXER:
        qi = np.zeros((n_ctx, pb.d_idx), np.uint16)
        qi[q_begin:] = q_idx_chunk
        kw = dict(q_idx=qi, k_idx=paged_gather(cache.kidx, bt, ps, 0, n_ctx))
    return prefill_layer(pb, mode, Q, K, V, rows=rows, pos=pos, **kw)


# ---------------------------------------------------------------- support-level diagnostics

def support_overlap(idx_a, idx_b) -> np.ndarray:
    """|S_a(r) & S_b(r)| per support row: how much of one support (e.g. the oracle's) the other
    (e.g. the indexer's, :300) recovers -- the "support-level diagnostic" of :478.  Entries < 0 are padding."""
    idx_a, idx_b = np.asarray(idx_a), np.asarray(idx_b)
    out = np.zeros(idx_a.shape[0], dtype=np.int32)
    for r in range(idx_a.shape[0]):
        a = idx_a[r][idx_a[r] >= 0]
        b = idx_b[r][idx_b[r] >= 0]
        out[r] = len(set(a.tolist()) & set(b.tolist()))
    return out


def row_kl(P, z, n_valid) -> np.ndarray:
    """KL(P_t || softmax(z_t)) over the valid causal keys s < n_valid[t] of each per-query row:
    sum_s P[s] (log P[s] - log softmax(z)[s]), terms with P[s] = 0 contribute 0.  fp64, log-sum-exp form."""
    P, z = np.asarray(P, dtype=np.float64), np.asarray(z, dtype=np.float64)
    out = np.zeros(P.shape[0])
    for r in range(P.shape[0]):
        n = int(n_valid[r])
        p, x = P[r, :n], z[r, :n]
        m = x.max()
        lse = m + math.log(np.exp(x - m).sum())
        nz = p > 0
        out[r] = float((p[nz] * (np.log(p[nz]) - (x[nz] - lse))).sum())
    return out
