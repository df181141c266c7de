"""A second, independent, vectorised numpy fp64 implementation of the paper's definitions, for TINY
inputs only.  It exists to pin oracle/sp_oracle.c (brute force on tiny inputs); it is written with
dense [L, L] masks and library routines (einsum, scipy softmax, stable argsort) instead of the
oracle's row loops.  Single sequence only.  PAPER.md:94 (attention), :123 (mass), :154 (block max),
:127 (top-k), :107/:156 (sparse attention with per-query causal re-mask)."""
import numpy as np
from scipy.special import softmax


def bf16_to_f64(b):
    return (np.asarray(b, dtype=np.uint16).astype(np.uint32) << 16).view(np.float32).astype(np.float64)


def logits(Q, K, scale, G, local_window=0, local_bias=0.0):
    """[Hq, L, L] scaled logits with -inf above the diagonal."""
    q = bf16_to_f64(Q)  # [L, Hq, d]
    k = np.repeat(bf16_to_f64(K), G, axis=1)  # [L, Hq, d]: head h uses kv head h // G
    z = np.einsum("thc,shc->hts", q, k) * scale
    L = q.shape[0]
    t = np.arange(L)[:, None]
    s = np.arange(L)[None, :]
    if local_window > 0:
        z = z + np.where((t - s >= 0) & (t - s < local_window), local_bias, 0.0)[None]
    return np.where((s <= t)[None], z, -np.inf)


def mass(Q, K, scale, G, **kw):
    """P [L, L] (zeros above the diagonal)."""
    return softmax(logits(Q, K, scale, G, **kw), axis=-1).mean(axis=0)


def indexer_logits(q_idx, k_idx, idx_scale, local_window=0, local_bias=0.0):
    z = bf16_to_f64(q_idx) @ bf16_to_f64(k_idx).T * idx_scale
    L = z.shape[0]
    t = np.arange(L)[:, None]
    s = np.arange(L)[None, :]
    if local_window > 0:
        z = z + np.where((t - s >= 0) & (t - s < local_window), local_bias, 0.0)
    return np.where(s <= t, z, -np.inf)


def support_rows(score, b):
    """score [L, L] with invalid entries masked to -inf -> (R [rows, L], n_valid)."""
    L = score.shape[0]
    sc = np.where(np.arange(L)[None, :] <= np.arange(L)[:, None], score, -np.inf)
    rows = (L + b - 1) // b
    R = np.full((rows, L), -np.inf)
    nv = np.zeros(rows, dtype=np.int64)
    for j in range(rows):
        R[j] = sc[j * b:min(L, (j + 1) * b)].max(axis=0)
        nv[j] = min(L, (j + 1) * b)
    return R, nv


def topk_rows(R, nv, k):
    out = np.full((R.shape[0], k), -1, dtype=np.int64)
    for j in range(R.shape[0]):
        n = int(nv[j])
        sel = np.sort(np.argsort(-R[j, :n], kind="stable")[:k])
        out[j, :len(sel)] = sel
    return out


def sparse_attention(Q, K, V, scale, G, idx, b, **kw):
    """o [L, Hq, d] with the support of row t // b, re-masked per query."""
    z = logits(Q, K, scale, G, **kw)  # [Hq, L, L]
    Hq, L, _ = z.shape
    keep = np.zeros((L, L), dtype=bool)
    for t in range(L):
        s = idx[t // b]
        s = s[(s >= 0) & (s <= t)]
        keep[t, s] = True
    z = np.where(keep[None], z, -np.inf)
    v = np.repeat(bf16_to_f64(V), G, axis=1)  # [L, Hq, d]
    with np.errstate(invalid="ignore"):
        a = softmax(z, axis=-1)
    a = np.nan_to_num(a, nan=0.0)
    return np.einsum("hts,shc->thc", a, v)
