"""Comparison rules of BASELINE.json's north_star, written out once for all GPU parity tests.

Support indices (readings A16/A17):
  * a row is STRICT when n_valid <= k (the whole prefix is kept) or when the oracle's fp64 gap between
    the k-th and (k+1)-th largest support-row score exceeds 1e-3 relative,
        gap = (v_k - v_{k+1}) / max(|v_k|, |v_{k+1}|)        (0/0 := 0);
    strict rows must match bit-exactly (index arrays are ascending, -1 padded);
  * on the remaining (fuzzy) rows the pooled overlap sum|S_gpu & S_orc| / sum|S_orc| must be >= 0.999.
Attention outputs: rel-L2 <= 1e-2 and max-abs <= 3e-2 (bf16 in / fp32 accumulate).
"""
import numpy as np

GAP_REL = 1e-3
OVERLAP_MIN = 0.999
ATT_REL_L2 = 1e-2
ATT_MAX_ABS = 3e-2


def row_gap(R_row, n, k):
    if n <= k:
        return np.inf
    v = R_row[:n]
    part = np.partition(v, n - k - 1)          # ascending: part[n-k-1] is the (k+1)-th largest
    vk1 = part[n - k - 1]
    vk = part[n - k:].min()
    den = max(abs(vk), abs(vk1))
    return 0.0 if den == 0 else (vk - vk1) / den


def compare_supports(idx_gpu, idx_orc, R_orc, n_valid, k):
    """Returns a dict with the counts; raises AssertionError when the rule is violated."""
    idx_gpu = np.asarray(idx_gpu)
    idx_orc = np.asarray(idx_orc)
    assert idx_gpu.shape == idx_orc.shape, (idx_gpu.shape, idx_orc.shape)
    strict = fuzzy = 0
    inter = total = 0
    worst = 1.0
    bad_strict = []
    for r in range(idx_orc.shape[0]):
        gap = row_gap(R_orc[r], int(n_valid[r]), k)
        if gap > GAP_REL:
            strict += 1
            if not np.array_equal(idx_gpu[r], idx_orc[r]):
                bad_strict.append(r)
        else:
            fuzzy += 1
            a = idx_gpu[r][idx_gpu[r] >= 0]
            b = idx_orc[r][idx_orc[r] >= 0]
            # structural validity still holds on fuzzy rows
            assert len(a) == len(b), (r, len(a), len(b))
            assert np.all(np.diff(a) > 0), r
            c = len(np.intersect1d(a, b, assume_unique=True))
            inter += c
            total += len(b)
            worst = min(worst, c / max(1, len(b)))
    assert not bad_strict, f"strict rows differ: {bad_strict[:10]} ({len(bad_strict)} of {strict})"
    overlap = inter / total if total else 1.0
    assert overlap >= OVERLAP_MIN, f"pooled fuzzy overlap {overlap:.5f} < {OVERLAP_MIN} (worst row {worst:.4f})"
    return dict(strict=strict, fuzzy=fuzzy, overlap=overlap, worst=worst)


def compare_attention(o_gpu, o_orc):
    o_gpu = np.asarray(o_gpu, dtype=np.float64)
    o_orc = np.asarray(o_orc, dtype=np.float64)
    assert o_gpu.shape == o_orc.shape
    assert np.isfinite(o_gpu).all()
    num = np.linalg.norm((o_gpu - o_orc).ravel())
    den = np.linalg.norm(o_orc.ravel())
    rel = num / den if den > 0 else num
    mx = np.abs(o_gpu - o_orc).max() if o_orc.size else 0.0
    assert rel <= ATT_REL_L2, f"rel-L2 {rel:.3e} > {ATT_REL_L2}"
    assert mx <= ATT_MAX_ABS, f"max-abs {mx:.3e} > {ATT_MAX_ABS}"
    return dict(rel_l2=rel, max_abs=mx)
