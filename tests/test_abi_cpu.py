"""CPU-only checks of the C-ABI boundary: libsp.so loads without a GPU, exports every symbol that
include/sp.h declares, and rejects bad arguments with the documented codes before launching anything."""
import ctypes as C
import os
import re

import pytest

from paper_2606_07703_b200 import binding as B
from paper_2606_07703_b200 import build as sp_build

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    sp_build.build()
    return B.lib()


def declared_functions():
    src = open(os.path.join(ROOT, "include", "sp.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(sp_[a-z_]+)\s*\(", src)))


def test_every_declared_symbol_is_exported(lib):
    names = declared_functions()
    assert set(names) == set(B.EXPORTS), (names, B.EXPORTS)
    for n in names:
        assert getattr(lib, n) is not None


def test_struct_size_matches_header(lib):
    # 2 int32 + 2 pointers + 7 int32 + 2 float + int32 + float + uint32 = 8 + 16 + 28 + 8 + 12 = 72 bytes
    assert C.sizeof(B.SpParams) == 72


def P(**kw):
    base = dict(L=256, Hq=8, Hkv=2, d=64, k=16, b_sel=1, hidden=128, d_idx=64, device="cpu")
    base.update(kw)
    return B.Problem(**base)


def test_num_rows_and_workspace_are_host_arithmetic(lib):
    assert P().num_rows == 256
    assert P(b_sel=64, L=300).num_rows == 5
    assert P(L=40, b_sel=8, cu_seqlens=[0, 19, 27, 40]).num_rows == 3 + 1 + 2
    for st in range(7):
        assert B.workspace_bytes(P(), st) >= 0
    big = P(L=65536, Hq=32, Hkv=8, d=128, k=2048, hidden=4096, d_idx=128)
    need = B.workspace_bytes(big, B.SP_STAGE_LAYER_INDEXER)
    assert 1 << 30 < need < 3 << 30          # 1 GiB score panel + 537 MB of indices + projections


@pytest.mark.parametrize("kw,code", [
    (dict(L=0), B.SP_ERR_INVALID_ARG),
    (dict(k=0), B.SP_ERR_INVALID_ARG),
    (dict(b_sel=0), B.SP_ERR_INVALID_ARG),
    (dict(Hq=6, Hkv=4), B.SP_ERR_INVALID_ARG),
    (dict(d=96), B.SP_ERR_UNSUPPORTED),
    (dict(Hq=32, Hkv=2), B.SP_ERR_UNSUPPORTED),
    (dict(flags=8), B.SP_ERR_UNSUPPORTED),               # SP_F_GROUP_SUPPORT: oracle-mode layer / sp_sparse_gqa_attn only
    (dict(flags=16), B.SP_ERR_UNSUPPORTED),              # SP_F_HEAD_SUPPORT: likewise (this is the INDEXER layer stage)
    (dict(flags=32), B.SP_ERR_UNSUPPORTED),              # unknown flag bit
    (dict(flags=1, b_sel=16), B.SP_ERR_UNSUPPORTED),     # served-scorer flags need a tcgen05 score path
    (dict(d_idx=32), B.SP_ERR_UNSUPPORTED),
    (dict(hidden=100), B.SP_ERR_UNSUPPORTED),
    (dict(local_window=-1), B.SP_ERR_INVALID_ARG),
    (dict(L=40, cu_seqlens=[0, 19, 19, 40]), B.SP_ERR_INVALID_ARG),
    (dict(L=40, cu_seqlens=[0, 19, 41]), B.SP_ERR_INVALID_ARG),
])
def test_bad_params_are_rejected(lib, kw, code):
    with pytest.raises(B.SpError) as ei:
        B.workspace_bytes(P(**kw), B.SP_STAGE_LAYER_INDEXER)
    assert ei.value.code == code


def test_null_and_misaligned_pointers_and_panels(lib):
    pb = P()
    p = pb.c()
    fake = C.c_void_p(0x1000)   # never dereferenced: validation fails first
    odd = C.c_void_p(0x1008)
    n = None
    f = lib.sp_topk_support
    assert f(C.byref(p), n, C.c_int64(256), 0, 4, fake, n, n, C.c_size_t(0), n) == B.SP_ERR_INVALID_ARG
    assert f(C.byref(p), odd, C.c_int64(256), 0, 4, fake, n, n, C.c_size_t(0), n) == B.SP_ERR_INVALID_ARG
    assert f(C.byref(p), fake, C.c_int64(256), 250, 10, fake, n, n, C.c_size_t(0), n) == B.SP_ERR_INVALID_ARG  # panel past the end
    assert f(C.byref(p), fake, C.c_int64(100), 0, 256, fake, n, n, C.c_size_t(0), n) == B.SP_ERR_INVALID_ARG   # ld < n_valid
    g = lib.sp_sparse_gqa_attn
    assert g(C.byref(p), fake, fake, fake, n, fake, n, n, C.c_size_t(0), n) == B.SP_ERR_INVALID_ARG
    h = lib.sp_prefill_layer
    assert h(C.byref(p), 7, n, n, n, fake, fake, fake, fake, n, fake, C.c_size_t(1 << 40), n) == B.SP_ERR_INVALID_ARG
    assert h(C.byref(p), B.SP_MODE_ORACLE, n, n, n, fake, fake, fake, fake, n, fake, C.c_size_t(16), n) == B.SP_ERR_WORKSPACE
    assert h(C.byref(p), B.SP_MODE_INDEXER, n, n, n, fake, fake, fake, fake, n, fake, C.c_size_t(1 << 40), n) == B.SP_ERR_INVALID_ARG
    assert b"SP_ERR_WORKSPACE" in lib.sp_strerror(B.SP_ERR_WORKSPACE)
    assert lib.sp_launch_count() == 0


def test_head_axis_flags_in_the_oracle_layer_workspace(lib):
    base = B.workspace_bytes(P(), B.SP_STAGE_LAYER_ORACLE)
    grp = B.workspace_bytes(P(flags=B.SP_F_GROUP_SUPPORT), B.SP_STAGE_LAYER_ORACLE)
    head = B.workspace_bytes(P(flags=B.SP_F_HEAD_SUPPORT), B.SP_STAGE_LAYER_ORACLE)
    idx_bytes = 256 * 16 * 4                                  # n_rows * k * int32
    assert grp - base == (2 - 1) * idx_bytes and head - base == (8 - 1) * idx_bytes
    with pytest.raises(B.SpError) as ei:
        B.workspace_bytes(P(flags=B.SP_F_GROUP_SUPPORT | B.SP_F_HEAD_SUPPORT), B.SP_STAGE_LAYER_ORACLE)
    assert ei.value.code == B.SP_ERR_INVALID_ARG


def test_chunk_api_validates_before_launching(lib):
    """sp_prefill_chunk / sp_kv_append / sp_chunk_workspace_bytes (PAPER.md:292 stage 4, :331): documented codes, no launch."""
    assert C.sizeof(B.SpKvPages) == 48            # 4 pointers + 3 int32 (+ 4 bytes of tail padding)
    fake = C.c_void_p(0x1000)
    n = None
    def pages(**kw):
        base = dict(k_pages=0x1000, v_pages=0x2000, kidx_pages=0x3000, block_table=0x4000, n_blocks=16, page_size=16, n_pages=32)
        base.update(kw)
        return B.SpKvPages(**base)
    def chunk(pb, q0, qc, kv, ws_bytes=1 << 40, X=fake):
        p = pb.c()
        return lib.sp_prefill_chunk(C.byref(p), q0, qc, X, fake, fake, fake, fake, fake, C.byref(kv), fake, n, fake,
                                    C.c_size_t(ws_bytes), n)
    pb = P(L=256, b_sel=32)
    assert B.chunk_workspace_bytes(pb, 128, 128) > 0
    assert chunk(pb, 128, 128, pages(), ws_bytes=16) == B.SP_ERR_WORKSPACE
    assert chunk(pb, 128, 100, pages()) == B.SP_ERR_INVALID_ARG            # q_begin + q_count != L
    assert chunk(pb, 130, 126, pages()) == B.SP_ERR_INVALID_ARG            # q_begin not a multiple of b_sel
    assert chunk(pb, 128, 128, pages(page_size=24)) == B.SP_ERR_UNSUPPORTED  # not a power of two
    assert chunk(pb, 128, 128, pages(n_blocks=8)) == B.SP_ERR_INVALID_ARG  # table does not cover the context
    assert chunk(pb, 128, 128, pages(kidx_pages=0)) == B.SP_ERR_INVALID_ARG
    assert chunk(pb, 128, 128, pages(), X=n) == B.SP_ERR_INVALID_ARG
    assert chunk(P(L=256, b_sel=16), 128, 128, pages()) == B.SP_ERR_UNSUPPORTED      # no paged reader for this block size
    assert chunk(P(L=40, b_sel=8, cu_seqlens=[0, 19, 40]), 8, 32, pages()) == B.SP_ERR_UNSUPPORTED   # one sequence per call
    p = pb.c()
    kv = pages()
    assert lib.sp_kv_append(C.byref(p), C.byref(kv), 250, 10, fake, fake, n, n) == B.SP_ERR_INVALID_ARG   # past the table
    assert lib.sp_kv_append(C.byref(p), C.byref(kv), 0, 10, n, n, n, n) == B.SP_ERR_INVALID_ARG
    assert lib.sp_launch_count() == 0


def test_missing_library_fails_loudly(monkeypatch):
    monkeypatch.setattr(B, "_lib", None)
    monkeypatch.setattr(B, "LIB_PATH", "/nonexistent/libsp.so")
    with pytest.raises(RuntimeError):
        B.lib()
