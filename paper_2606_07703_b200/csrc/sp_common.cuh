// sp_common.cuh -- shared device/host helpers of the sm_100a sparse-prefill kernels.
// Geometry of support rows follows include/sp.h ("Support rows"), i.e. PAPER.md:101-103, :152.
#pragma once
#include <cuda_bf16.h>
#include <cuda_runtime.h>
#include <stdint.h>

#include "../../include/sp.h"

#define SP_LOG2E 1.4426950408889634f
#define SP_LN2 0.6931471805599453f

// Device-visible description of the pack and of the selection granularity.
struct SpGeom {
  int batch;
  int L;
  const int* cu;  // device cu_seqlens or nullptr
  int b_sel;
  long long idx_grp;  // SP_F_GROUP_SUPPORT: elements between two KV groups' index lists ([Hkv, n_rows, k]); 0 = one shared list
  // ---- chunked prefill against a paged KV cache (sp_prefill_chunk; PAPER.md:292 stage 4, :331); all zero otherwise ----
  int q_off;       // packed position of row 0 of the QUERY-side tensors (Q, O, lse, q_idx): they hold the chunk only
  int q_rows;      // rows of those tensors (0 = L)
  int row_off;     // support row of row 0 of the index tensor
  int pos_off;     // projection only: position of row 0 of X (rotary embedding of a chunk)
  const int* bt;   // DEVICE block table of the KEY-side tensors (K, V, k_idx pages), nullptr = contiguous [L, ...]
  int page_shift;  // log2(tokens per page)
  int n_blocks;    // entries of bt
  long long kv_rows;  // rows of the page pool (n_pages * page_size)
};

// row of packed key position p in the key-side tensors: p itself, or its slot in the paged cache
__device__ __forceinline__ long long sp_kv_row(const SpGeom& g, int p) {
  if (g.bt == nullptr) return p;
  const int blk = min(p >> g.page_shift, g.n_blocks - 1);
  return ((long long)__ldg(g.bt + blk) << g.page_shift) | (long long)(p & ((1 << g.page_shift) - 1));
}

struct SpRow {
  int seq_start;  // packed position of the sequence's first token
  int t_first;    // first local query position of the row
  int t_last;     // last local query position of the row (n_valid = t_last + 1)
  int seq_len;
};

__device__ __forceinline__ SpRow sp_row_info(const SpGeom& g, int row) {
  const int b = g.b_sel;
  if (g.cu == nullptr) {
    const int t0 = row * b;
    return SpRow{0, t0, min(t0 + b - 1, g.L - 1), g.L};
  }
  int r0 = 0;
  for (int i = 0; i < g.batch; ++i) {
    const int s = g.cu[i], n = g.cu[i + 1] - s;
    const int nr = (n + b - 1) / b;
    if (row < r0 + nr) {
      const int j = row - r0;
      return SpRow{s, j * b, min(j * b + b - 1, n - 1), n};
    }
    r0 += nr;
  }
  return SpRow{0, 0, -1, 0};
}

struct SpPos {
  int seq_start;
  int seq_len;
  int row;  // support row of this packed position
};

__device__ __forceinline__ SpPos sp_pos_info(const SpGeom& g, int pos) {
  const int b = g.b_sel;
  if (g.cu == nullptr) return SpPos{0, g.L, pos / b};
  int r0 = 0;
  for (int i = 0; i < g.batch; ++i) {
    const int s = g.cu[i], n = g.cu[i + 1] - s;
    if (pos < s + n) return SpPos{s, n, r0 + (pos - s) / b};
    r0 += (n + b - 1) / b;
  }
  return SpPos{0, 0, 0};
}

__device__ __forceinline__ float sp_bf16lo(uint32_t w) { return __uint_as_float(w << 16); }
__device__ __forceinline__ float sp_bf16hi(uint32_t w) { return __uint_as_float(w & 0xffff0000u); }

__device__ __forceinline__ uint32_t sp_pack_bf16(float lo, float hi) {
  __nv_bfloat162 v = __floats2bfloat162_rn(lo, hi);
  return *reinterpret_cast<uint32_t*>(&v);
}

__device__ __forceinline__ float sp_warp_max(float v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v = fmaxf(v, __shfl_xor_sync(0xffffffffu, v, o));
  return v;
}
__device__ __forceinline__ float sp_warp_sum(float v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
  return v;
}

// ---- host-side launch helpers implemented in the individual .cu files ----
struct SpLaunch {
  cudaStream_t stream;
};

cudaError_t sp_launch_topk(const SpGeom& g, const float* scores, int64_t ld, int row_begin, int row_count, int k,
                           int max_n_valid, int32_t* idx, int32_t* cnt, cudaStream_t st);

cudaError_t sp_launch_indexer_scores(const SpGeom& g, const void* q_idx, const void* k_idx, int d_idx,
                                     float idx_scale, int local_window, float local_bias, int row_begin,
                                     int row_count, int max_n_valid, float* scores, int64_t ld, cudaStream_t st);

cudaError_t sp_launch_mass(const SpGeom& g, const void* Q, const void* K, const float* lse, int Hq, int Hkv, int d,
                           float scale, int local_window, float local_bias, int row_begin, int row_count,
                           int max_n_valid, float* mass, int64_t ld, cudaStream_t st);

// idx == nullptr -> dense causal attention.  O may be nullptr (lse only); lse may be nullptr.
// [q_begin, q_begin+q_count) is the packed query range to process.
cudaError_t sp_launch_attn(const SpGeom& g, const void* Q, const void* K, const void* V, const int32_t* idx, int k,
                           int Hq, int Hkv, int d, float scale, int local_window, float local_bias, int q_begin,
                           int q_count, void* O, float* lse, cudaStream_t st);

// tcgen05 paths (sp_tc_gemm.cu, sp_tc_attn.cu)
cudaError_t sp_launch_project_tc(const SpGeom& g, uint32_t flags, const void* X, const void* Wq, const void* Wk,
                                 void* q_idx, void* k_idx, int L, int hidden, int d_idx, cudaStream_t st);
bool sp_tc_scores_supported(int b_sel);
cudaError_t sp_launch_indexer_scores_tc(const SpGeom& g, const int32_t* cu_host, const void* q_idx, const void* k_idx,
                                        int d_idx, float idx_scale, int local_window, float local_bias, int relu,
                                        int row_begin, int row_count, int max_n_valid, float* scores, int64_t ld,
                                        cudaStream_t st);

bool sp_tc_mass_supported(int b_sel, int d);
cudaError_t sp_launch_mass_tc(const SpGeom& g, const int32_t* cu_host, const void* Q, const void* K, const float* lse,
                              int Hq, int Hkv, int d, float scale, int local_window, float local_bias, int row_begin,
                              int row_count, float* mass, int64_t ld, cudaStream_t st, int grp = -1,
                              int head = -1);  // grp >= 0: that KV group's heads only; head >= 0: that one head only

bool sp_tc_attn_supported(int b_sel, int G, bool sparse, int k, int d, bool paged = false);
cudaError_t sp_launch_attn_tc(const SpGeom& g, long long n_rows, long long n_chunks_dense, long long chunk_base,
                              const void* Q, const void* K, const void* V, const int32_t* idx, int k, int Hq, int Hkv,
                              int d, float scale, int local_window, float local_bias, void* O, float* lse,
                              cudaStream_t st);
// device address and size of the library's fixed scratch array (sp_tc_attn.cu; no allocation, once per device)
cudaError_t sp_static_scratch_ptr(uint32_t** ptr, size_t* bytes);
// per-query supports as membership-masked dense attention (sp_tc_attn.cu)
bool sp_tc_attn_masked_supported(int G, int d);
void sp_support_bits_shape(long long L, long long* pitch, long long* rows);
cudaError_t sp_launch_support_bits(const SpGeom& g, const int32_t* idx, int k, long long n_rows, uint32_t* bits,
                                   cudaStream_t st);
cudaError_t sp_launch_attn_tc_masked(const SpGeom& g, long long n_chunks, const void* Q, const void* K, const void* V,
                                     const uint32_t* bits, int Hq, int Hkv, int d, float scale, void* O, float* lse,
                                     cudaStream_t st);

// per-query gather-sparse attention on mma.sync (sp_mma_attn.cu)
cudaError_t sp_launch_attn_pq(const SpGeom& g, const void* Q, const void* K, const void* V, const int32_t* idx, int k,
                              int Hq, int Hkv, int d, float scale, int local_window, float local_bias, int q_begin,
                              int q_count, void* O, float* lse, cudaStream_t st, bool per_head = false);

// diagnostics (sp_diag.cu)
cudaError_t sp_launch_overlap(const int32_t* a, const int32_t* b, long long n_rows, int k, int32_t* inter,
                              cudaStream_t st);
cudaError_t sp_launch_row_kl(const SpGeom& g, const float* P, int64_t ldp, const float* z, int64_t ldz, int row_begin,
                             int row_count, float* kl, cudaStream_t st);

// paged KV cache plumbing (sp_paged.cu): rows <-> page slots through the block table
cudaError_t sp_launch_paged_copy(bool to_pages, void* pool, void* rows, const int32_t* bt, int page_shift,
                                 long long row_bytes, int t_begin, int t_count, cudaStream_t st);

cudaError_t sp_launch_gather_probe(const void* base, int row_bytes, long long row_pitch_bytes, const int32_t* idx,
                                   long long n_idx, uint32_t* sink, int blocks, cudaStream_t st);

void sp_count_launch(int n = 1);

// Per-DEVICE host-side caches: a process may drive several GPUs through the library (cudaFuncSetAttribute and the SM
// count belong to the current device).  Races between threads are benign (the same value is written twice).
constexpr int SP_MAX_DEVICES = 64;
int sp_current_device();              // cudaGetDevice, clamped to [0, SP_MAX_DEVICES)
int sp_sm_count();                    // multiprocessors of the current device
inline bool sp_first_use_on_device(unsigned char (&seen)[SP_MAX_DEVICES]) {
  const int d = sp_current_device();
  if (seen[d]) return false;
  seen[d] = 1;
  return true;
}
