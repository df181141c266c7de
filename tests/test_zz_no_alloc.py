"""sp_sparse_gqa_attn_static: the entry point that allocates nothing (bitmap scratch in a fixed device array inside the
library, include/sp.h).  Collected last on purpose (file name): the suite runs with pytest -x.

Checked against the existing path (sp_sparse_gqa_attn given the SPARSE_ATTN workspace) and against the oracle
(PAPER.md:107, :156), on two calls in a row whose supports differ -- the second call's lists are a strict subset of the
first's for half the queries, so anything the first call left in the shared array would show."""
import numpy as np
import pytest
import torch

import parity
from oracle import oracle as orc
from paper_2606_07703_b200 import binding as B

pytestmark = pytest.mark.gpu
DEV = "cuda"


def _dev(u16):
    return torch.from_numpy(np.ascontiguousarray(u16).view(np.int16)).to(DEV).view(torch.bfloat16)


def _f64(t):
    return t.float().cpu().numpy().astype(np.float64)


def _supports(L, k, rng, thin):
    """Random per-query subsets of the causal prefix, unsorted, -1 padded; thin=True keeps at most k/4 per query."""
    idx = np.full((L, k), -1, dtype=np.int32)
    for t in range(L):
        if t % 41 == 7:
            continue                                                  # empty rows: O = 0, lse = -inf
        cap = max(1, k // 4) if thin else k
        m = int(rng.integers(1, min(t + 1, cap) + 1))
        idx[t, :m] = rng.choice(t + 1, size=m, replace=False)
        rng.shuffle(idx[t])
    return idx


def test_static_scratch_entry_point_matches_workspace_path_twice():
    L, Hq, Hkv, d, k = 777, 8, 2, 128, 96
    rng = np.random.Generator(np.random.Philox(4242))
    Qb = orc.f64_to_bf16(rng.standard_normal((L, Hq, d)))
    Kb = orc.f64_to_bf16(rng.standard_normal((L, Hkv, d)))
    Vb = orc.f64_to_bf16(rng.standard_normal((L, Hkv, d)))
    kw = dict(L=L, Hq=Hq, Hkv=Hkv, d=d, k=k, b_sel=1)
    pbo, pbg = orc.Problem(**kw), B.Problem(**kw)
    Q, K, V = _dev(Qb), _dev(Kb), _dev(Vb)
    nb = B.workspace_bytes(pbg, B.SP_STAGE_SPARSE_ATTN)
    assert nb > 0
    ws = torch.empty(nb, dtype=torch.uint8, device=DEV)
    for call, thin in enumerate((False, True)):                       # dense lists first, then sparser ones
        idx = _supports(L, k, rng, thin)
        idx_d = torch.from_numpy(idx).to(DEV)
        O_ref = torch.full((L, Hq, d), float("nan"), dtype=torch.bfloat16, device=DEV)
        lse_ref = torch.full((L, Hq), float("nan"), dtype=torch.float32, device=DEV)
        B.sp_sparse_gqa_attn(pbg, Q, K, V, idx_d, O_ref, lse_ref, ws)
        O = torch.full_like(O_ref, float("nan"))
        lse = torch.full_like(lse_ref, float("nan"))
        torch.cuda.synchronize()
        mem0 = torch.cuda.mem_get_info()[0]
        n0 = B.launch_count()
        B.sp_sparse_gqa_attn_static(pbg, Q, K, V, idx_d, O, lse)
        torch.cuda.synchronize()
        assert B.launch_count() - n0 == 2, call                       # bitmap builder + attention
        assert torch.cuda.mem_get_info()[0] >= mem0 - (1 << 20), call   # the call took no device memory
        # existing path: the attention tolerance of the other tests (the two run the same kernels: in fact identical)
        parity.compare_attention(_f64(O), _f64(O_ref))
        assert torch.equal(O.view(torch.int16), O_ref.view(torch.int16)), call
        fin = torch.isfinite(lse_ref)
        assert torch.equal(torch.isfinite(lse), fin), call
        assert torch.allclose(lse[fin], lse_ref[fin], rtol=0, atol=2e-5), call
        # oracle
        want, lse_o = orc.sparse_attn(pbo, Qb, Kb, Vb, np.arange(L), idx, want_lse=True)
        parity.compare_attention(_f64(O), want)
        got = _f64(lse)
        fo = np.isfinite(lse_o)
        assert (~fo).sum() > 0 and np.array_equal(np.isfinite(got), fo), call
        assert np.allclose(got[fo], lse_o[fo], rtol=0, atol=2e-5), call


def test_static_scratch_entry_point_rejects_what_it_cannot_hold():
    """Beyond the fixed array: SP_ERR_TOO_LARGE and nothing launched; outside the masked loop's shapes: UNSUPPORTED."""
    def call(**over):
        kw = dict(dict(L=512, Hq=8, Hkv=2, d=128, k=64, b_sel=1), **over)
        pb = B.Problem(**kw)
        L = kw["L"]
        Q = torch.zeros(L, kw["Hq"], kw["d"], dtype=torch.bfloat16, device=DEV)
        K = torch.zeros(L, kw["Hkv"], kw["d"], dtype=torch.bfloat16, device=DEV)
        idx = torch.zeros(pb.num_rows, kw["k"], dtype=torch.int32, device=DEV)
        n0 = B.launch_count()
        with pytest.raises(B.SpError) as e:
            B.sp_sparse_gqa_attn_static(pb, Q, K, K, idx, torch.empty_like(Q))
        assert B.launch_count() == n0
        return e.value
    e = call(L=8193, k=2048)
    assert e.code == B.SP_ERR_TOO_LARGE and "8192" in str(e)
    assert call(L=16384, k=2048).code == B.SP_ERR_TOO_LARGE
    assert call(b_sel=64).code == B.SP_ERR_UNSUPPORTED
    assert call(Hkv=8).code == B.SP_ERR_UNSUPPORTED                   # G = 1: the gather kernel's shape
    assert call(local_window=16, local_bias=0.5).code == B.SP_ERR_UNSUPPORTED
    # the largest pack the array holds is accepted (zeros in, finite out)
    pb = B.Problem(L=8192, Hq=8, Hkv=2, d=64, k=1024, b_sel=1)
    Q = torch.zeros(8192, 8, 64, dtype=torch.bfloat16, device=DEV)
    K = torch.zeros(8192, 2, 64, dtype=torch.bfloat16, device=DEV)
    idx = torch.arange(1024, dtype=torch.int32, device=DEV).repeat(8192, 1)
    O = torch.full_like(Q, float("nan"))
    B.sp_sparse_gqa_attn_static(pb, Q, K, K, idx, O)
    torch.cuda.synchronize()
    assert torch.isfinite(O.float()).all()
