// sp_tc_gemm.cu -- tcgen05/TMEM/TMA kernels for the two indexer contractions:
//   * sp_tc_project_kernel : q_idx = bf16(X Wqi), k_idx = bf16(X Wki)
//   * sp_tc_score_kernel   : z[t,s] = idx_scale <q_idx[t], k_idx[s]> (+ local term), s <= t,
//                            R_B(s) = max_{t in B, t >= s} z[t,s] fused in the epilogue
// Both are one-output-tile-per-CTA kernels: TMA (SWIZZLE_128B) -> shared memory -> tcgen05.mma with the fp32
// accumulator in TMEM -> tcgen05.ld epilogue.  In the score kernel the KEY index is the MMA M dimension
// (TMEM lane = key, column = query), so the max over a selection block's queries is a per-thread running
// max over columns and global writes are coalesced along s.
#include "sp_common.cuh"
#include "sp_tc.cuh"

using namespace sptc;

// ---------------------------------------------------------------------------------------------------
// host: tensor maps
// ---------------------------------------------------------------------------------------------------
typedef CUresult (*sp_encode_tiled_fn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*,
                                       const cuuint64_t*, const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave,
                                       CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

static sp_encode_tiled_fn sp_get_encode() {
  static sp_encode_tiled_fn fn = nullptr;
  if (!fn) {
    void* p = nullptr;
    cudaDriverEntryPointQueryResult q;
    if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &q) == cudaSuccess &&
        q == cudaDriverEntryPointSuccess)
      fn = (sp_encode_tiled_fn)p;
  }
  return fn;
}

cudaError_t sp_make_tmap_bf16(CUtensorMap* out, const void* base, uint64_t rows, uint64_t cols, uint64_t pitch_elems,
                              uint32_t box_rows) {
  sp_encode_tiled_fn enc = sp_get_encode();
  if (!enc) return cudaErrorNotSupported;
  const cuuint64_t dims[2] = {cols, rows};
  const cuuint64_t strides[1] = {pitch_elems * 2};
  const cuuint32_t box[2] = {64, box_rows};
  const cuuint32_t estr[2] = {1, 1};
  const CUresult r = enc(out, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 2, const_cast<void*>(base), dims, strides, box, estr,
                         CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                         CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
  return r == CUDA_SUCCESS ? cudaSuccess : cudaErrorInvalidValue;
}

namespace {

__device__ __forceinline__ uint8_t* align1024(uint8_t* p) {
  return reinterpret_cast<uint8_t*>((reinterpret_cast<uintptr_t>(p) + 1023) & ~(uintptr_t)1023);
}

// ===================================================================================================
// Projection: C[m, 0:DI] = X[m,:] Wq, C[m, DI:2DI] = X[m,:] Wk.   M tile 128, N = 2*DI, K pipelined by 64.
// ===================================================================================================
constexpr int PJ_STAGES = 4;

template <int DI>
__global__ void __launch_bounds__(128, 1)
sp_tc_project_kernel(const __grid_constant__ CUtensorMap tmX, const __grid_constant__ CUtensorMap tmWq,
                     const __grid_constant__ CUtensorMap tmWk, __nv_bfloat16* __restrict__ q_idx,
                     __nv_bfloat16* __restrict__ k_idx, int L, int hidden) {
  constexpr int N = 2 * DI;
  constexpr int NG = N / 64;                  // 64-column groups of B
  constexpr uint32_t A_BYTES = 128 * 128;     // 128 rows x 64 k
  constexpr uint32_t B_BYTES = NG * 64 * 128; // NG groups of [64 k-rows x 128 B]
  constexpr uint32_t STAGE = A_BYTES + B_BYTES;
  extern __shared__ uint8_t smem_raw[];
  uint8_t* smem = align1024(smem_raw);
  __shared__ uint64_t full[PJ_STAGES], empty[PJ_STAGES], done;
  __shared__ uint32_t tmem_slot;
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int m0 = blockIdx.x * 128;
  const int nkb = hidden / 64;

  if (threadIdx.x == 0) {
    for (int i = 0; i < PJ_STAGES; ++i) {
      mbar_init(&full[i], 1);
      mbar_init(&empty[i], 1);
    }
    mbar_init(&done, 1);
    fence_barrier_init();
    tma_prefetch_desc(&tmX);
    tma_prefetch_desc(&tmWq);
    tma_prefetch_desc(&tmWk);
  }
  if (warp == 1) tmem_alloc<N>(&tmem_slot);
  tc_fence_before_sync();
  __syncthreads();
  tc_fence_after_sync();
  const uint32_t tmem = tmem_slot;

  if (warp == 0 && lane == 0) {
    for (int kb = 0; kb < nkb; ++kb) {
      const int s = kb % PJ_STAGES;
      if (kb >= PJ_STAGES) mbar_wait(&empty[s], ((kb / PJ_STAGES) - 1) & 1);
      uint8_t* a = smem + (size_t)s * STAGE;
      uint8_t* b = a + A_BYTES;
      mbar_expect_tx(&full[s], STAGE);
      tma_load_2d(a, &tmX, &full[s], kb * 64, m0);
#pragma unroll
      for (int g = 0; g < DI / 64; ++g) {
        tma_load_2d(b + g * 8192, &tmWq, &full[s], g * 64, kb * 64);
        tma_load_2d(b + (DI / 64 + g) * 8192, &tmWk, &full[s], g * 64, kb * 64);
      }
    }
  } else if (warp == 1 && lane == 0) {
    constexpr uint32_t idesc = umma_idesc_bf16(128, N, 0, 1);  // A K-major, B MN-major
    for (int kb = 0; kb < nkb; ++kb) {
      const int s = kb % PJ_STAGES;
      mbar_wait(&full[s], (kb / PJ_STAGES) & 1);
      tc_fence_after_sync();
      const uint32_t a = smem_u32(smem + (size_t)s * STAGE);
      const uint32_t b = a + A_BYTES;
#pragma unroll
      for (int k = 0; k < 4; ++k) {
        const uint64_t ad = umma_desc_sw128(a + k * 32, 16, 1024);
        const uint64_t bd = umma_desc_sw128(b + k * 2048, 8192, 1024);
        umma_ss(tmem, ad, bd, idesc, (kb | k) != 0);
      }
      umma_commit(&empty[s]);
    }
    umma_commit(&done);
  }
  __syncwarp();
  mbar_wait(&done, 0);
  tc_fence_after_sync();

  // epilogue: thread = output row
  const int m = m0 + warp * 32 + lane;
  const uint32_t trow = tmem + ((uint32_t)(warp * 32) << 16);
#pragma unroll
  for (int c0 = 0; c0 < N; c0 += 32) {
    uint32_t v[32];
    tmem_ld_x32(trow + c0, v);
    tmem_ld_wait();
    if (m < L) {
      __nv_bfloat16* dst = (c0 < DI ? q_idx + (size_t)m * DI + c0 : k_idx + (size_t)m * DI + (c0 - DI));
#pragma unroll
      for (int j = 0; j < 32; j += 8) {
        uint4 o;
        o.x = sp_pack_bf16(__uint_as_float(v[j]), __uint_as_float(v[j + 1]));
        o.y = sp_pack_bf16(__uint_as_float(v[j + 2]), __uint_as_float(v[j + 3]));
        o.z = sp_pack_bf16(__uint_as_float(v[j + 4]), __uint_as_float(v[j + 5]));
        o.w = sp_pack_bf16(__uint_as_float(v[j + 6]), __uint_as_float(v[j + 7]));
        *reinterpret_cast<uint4*>(dst + j) = o;
      }
    }
  }
  tc_fence_before_sync();
  __syncthreads();
  if (warp == 1) tmem_dealloc<N>(tmem);
}

// ===================================================================================================
// Indexer scores.  CTA tile = 128 keys (MMA M, TMEM lanes) x 256 queries (MMA N, TMEM columns), K = DI.
// A query tile is 256 consecutive LOCAL positions of one sequence; selection blocks (b_sel in
// {16,32,64,128,256}) never straddle query tiles.  b_sel == 1 writes every causal (t, s).
// ===================================================================================================
constexpr int SC_NQ = 256;

struct ScTile {
  int seq_start, n, q0;  // sequence start (packed), sequence length, first LOCAL query of the tile
  int row0;              // support row of the tile's first query
};

__device__ __forceinline__ ScTile sc_tile_info(const SpGeom& g, int qy) {
  const int b = g.b_sel;
  if (g.cu == nullptr) return ScTile{0, g.L, qy * SC_NQ, qy * SC_NQ / b};
  int t0 = 0, r0 = 0;
  for (int i = 0; i < g.batch; ++i) {
    const int s = g.cu[i], n = g.cu[i + 1] - s;
    const int nt = (n + SC_NQ - 1) / SC_NQ;
    if (qy < t0 + nt) {
      const int q0 = (qy - t0) * SC_NQ;
      return ScTile{s, n, q0, r0 + q0 / b};
    }
    t0 += nt;
    r0 += (n + b - 1) / b;
  }
  return ScTile{0, 0, 0, 0};
}

template <int DI>
__global__ void __launch_bounds__(128)
sp_tc_score_kernel(const __grid_constant__ CUtensorMap tmQ, const __grid_constant__ CUtensorMap tmK, SpGeom g,
                   float idx_scale, int local_window, float local_bias, int row_begin, int row_count, int qy_begin,
                   float* __restrict__ scores, int64_t ld) {
  constexpr int KB = DI / 64;
  constexpr uint32_t A_BYTES = 128 * 128;    // per 64-wide K block: 128 keys
  constexpr uint32_t B_BYTES = SC_NQ * 128;  // per K block: 256 queries
  extern __shared__ uint8_t smem_raw[];
  __shared__ uint64_t full, done;
  __shared__ uint32_t tmem_slot;
  const ScTile ti = sc_tile_info(g, qy_begin + blockIdx.y);
  const int s0 = blockIdx.x * 128;  // local key position of lane 0
  const int q_last = min(ti.q0 + SC_NQ, ti.n) - 1;
  if (ti.n == 0 || s0 > q_last) return;
  const int b = g.b_sel;
  const int nblk = (q_last - ti.q0) / b + 1;  // support rows in this tile (b == 1: queries)
  if (ti.row0 >= row_begin + row_count || ti.row0 + nblk <= row_begin) return;

  uint8_t* smem = align1024(smem_raw);
  uint8_t* sA = smem;
  uint8_t* sB = smem + KB * A_BYTES;
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  if (threadIdx.x == 0) {
    mbar_init(&full, 1);
    mbar_init(&done, 1);
    fence_barrier_init();
  }
  if (warp == 0) tmem_alloc<SC_NQ>(&tmem_slot);
  tc_fence_before_sync();
  __syncthreads();
  tc_fence_after_sync();
  const uint32_t tmem = tmem_slot;

  if (threadIdx.x == 0) {
    mbar_expect_tx(&full, KB * (A_BYTES + B_BYTES));
#pragma unroll
    for (int kb = 0; kb < KB; ++kb) {
      tma_load_2d(sA + kb * A_BYTES, &tmK, &full, kb * 64, ti.seq_start + s0);
      tma_load_2d(sB + kb * B_BYTES, &tmQ, &full, kb * 64, ti.seq_start + ti.q0);
    }
    mbar_wait(&full, 0);
    tc_fence_after_sync();
    constexpr uint32_t idesc = umma_idesc_bf16(128, SC_NQ, 0, 0);
#pragma unroll
    for (int k = 0; k < DI / 16; ++k) {
      const uint64_t ad = umma_desc_sw128(smem_u32(sA + (k / 4) * A_BYTES) + (k % 4) * 32, 16, 1024);
      const uint64_t bd = umma_desc_sw128(smem_u32(sB + (k / 4) * B_BYTES) + (k % 4) * 32, 16, 1024);
      umma_ss(tmem, ad, bd, idesc, k != 0);
    }
    umma_commit(&done);
  }
  __syncwarp();
  mbar_wait(&done, 0);
  tc_fence_after_sync();

  const int s = s0 + warp * 32 + lane;  // this thread's local key
  const int s_lo = s0 + warp * 32;      // warp-uniform: smallest / largest key of the warp
  const int s_hi = s_lo + 31;
  const uint32_t trow = tmem + ((uint32_t)(warp * 32) << 16);
  float best = -INFINITY;
  for (int c0 = 0; c0 < SC_NQ; c0 += 32) {
    const int t0 = ti.q0 + c0;  // local query of column c0
    if (t0 > q_last) break;
    const int t1 = min(t0 + 31, q_last);
    if (s_lo <= t1) {  // warp-uniform: some (t, s) of this chunk is causal
      uint32_t v[32];
      tmem_ld_x32(trow + c0, v);
      tmem_ld_wait();
      if (b == 1) {
#pragma unroll
        for (int j = 0; j < 32; ++j) {
          const int t = t0 + j;
          const int row = ti.row0 + c0 + j;
          if (t <= q_last && s <= t && row >= row_begin && row < row_begin + row_count) {
            float z = __uint_as_float(v[j]) * idx_scale;
            if (local_window > 0 && t - s < local_window) z += local_bias;
            scores[(size_t)(row - row_begin) * ld + s] = z;
          }
        }
      } else if (s_hi <= t0 && t0 + 31 <= q_last && idx_scale > 0.f && (local_window == 0 || t0 - s_hi >= local_window)) {
        // interior chunk: every pair is causal and outside the local window; max commutes with the positive scale
        float m = __uint_as_float(v[0]);
#pragma unroll
        for (int j = 1; j < 32; ++j) m = fmaxf(m, __uint_as_float(v[j]));
        best = fmaxf(best, m * idx_scale);
      } else {
#pragma unroll
        for (int j = 0; j < 32; ++j) {
          const int t = t0 + j;
          if (t <= q_last && s <= t) {
            float z = __uint_as_float(v[j]) * idx_scale;
            if (local_window > 0 && t - s < local_window) z += local_bias;
            best = fmaxf(best, z);
          }
        }
      }
    }
    if (b > 1 && ((c0 + 32) % b == 0 || t1 == q_last)) {  // last chunk of a selection block: flush
      const int blk = c0 / b;
      const int row = ti.row0 + blk;
      const int blk_last = min(ti.q0 + blk * b + b - 1, q_last);  // n_valid - 1 of the block
      if (row >= row_begin && row < row_begin + row_count && s <= blk_last)
        scores[(size_t)(row - row_begin) * ld + s] = best;
      best = -INFINITY;
    }
  }
  tc_fence_before_sync();
  __syncthreads();
  if (warp == 0) tmem_dealloc<SC_NQ>(tmem);
}

}  // namespace

// ---------------------------------------------------------------------------------------------------
// launchers
// ---------------------------------------------------------------------------------------------------
template <int DI>
static cudaError_t launch_project_tc(const void* X, const void* Wq, const void* Wk, void* q_idx, void* k_idx, int L,
                                     int hidden, cudaStream_t st) {
  CUtensorMap tmX, tmWq, tmWk;
  cudaError_t e;
  if ((e = sp_make_tmap_bf16(&tmX, X, L, hidden, hidden, 128)) != cudaSuccess) return e;
  if ((e = sp_make_tmap_bf16(&tmWq, Wq, hidden, DI, DI, 64)) != cudaSuccess) return e;
  if ((e = sp_make_tmap_bf16(&tmWk, Wk, hidden, DI, DI, 64)) != cudaSuccess) return e;
  constexpr size_t smem = (size_t)PJ_STAGES * (128 * 128 + (2 * DI / 64) * 8192) + 1024;
  static bool attr_done = false;
  if (!attr_done) {
    e = cudaFuncSetAttribute(sp_tc_project_kernel<DI>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    attr_done = true;
  }
  sp_tc_project_kernel<DI><<<(L + 127) / 128, 128, smem, st>>>(tmX, tmWq, tmWk, (__nv_bfloat16*)q_idx,
                                                               (__nv_bfloat16*)k_idx, L, hidden);
  sp_count_launch();
  return cudaGetLastError();
}

cudaError_t sp_launch_project_tc(const void* X, const void* Wq, const void* Wk, void* q_idx, void* k_idx, int L,
                                 int hidden, int d_idx, cudaStream_t st) {
  return d_idx == 128 ? launch_project_tc<128>(X, Wq, Wk, q_idx, k_idx, L, hidden, st)
                      : launch_project_tc<64>(X, Wq, Wk, q_idx, k_idx, L, hidden, st);
}

bool sp_tc_scores_supported(int b_sel) { return b_sel == 1 || b_sel == 32 || b_sel == 64 || b_sel == 128 || b_sel == 256; }

template <int DI>
static cudaError_t launch_scores_tc(const SpGeom& g, const void* q_idx, const void* k_idx, float idx_scale, int lw,
                                    float lb, int row_begin, int row_count, int max_n_valid, int qy_begin, int qy_count,
                                    float* scores, int64_t ld, cudaStream_t st) {
  CUtensorMap tmQ, tmK;
  cudaError_t e;
  if ((e = sp_make_tmap_bf16(&tmQ, q_idx, g.L, DI, DI, SC_NQ)) != cudaSuccess) return e;
  if ((e = sp_make_tmap_bf16(&tmK, k_idx, g.L, DI, DI, 128)) != cudaSuccess) return e;
  constexpr size_t smem = (size_t)(DI / 64) * (128 * 128 + SC_NQ * 128) + 1024;
  static bool attr_done = false;
  if (!attr_done) {
    e = cudaFuncSetAttribute(sp_tc_score_kernel<DI>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    attr_done = true;
  }
  dim3 grid((max_n_valid + 127) / 128, qy_count);
  sp_tc_score_kernel<DI><<<grid, 128, smem, st>>>(tmQ, tmK, g, idx_scale, lw, lb, row_begin, row_count, qy_begin, scores, ld);
  sp_count_launch();
  return cudaGetLastError();
}

// cu_host: HOST copy of cu_seqlens (nullptr = one sequence).
cudaError_t sp_launch_indexer_scores_tc(const SpGeom& g, const int32_t* cu_host, const void* q_idx, const void* k_idx,
                                        int d_idx, float idx_scale, int local_window, float local_bias, int row_begin,
                                        int row_count, int max_n_valid, float* scores, int64_t ld, cudaStream_t st) {
  if (row_count <= 0) return cudaSuccess;
  // query tiles (256 local positions of one sequence) that intersect the panel
  const int b = g.b_sel;
  long long t0 = 0, r0 = 0;
  long long qlo = -1, qhi = -1;
  for (int i = 0; i < g.batch; ++i) {
    const int n = cu_host ? cu_host[i + 1] - cu_host[i] : g.L;
    const long long nr = (n + b - 1) / b, nt = (n + SC_NQ - 1) / SC_NQ;
    const long long lo = row_begin > r0 ? row_begin : r0;
    const long long hi = ((long long)row_begin + row_count < r0 + nr ? (long long)row_begin + row_count : r0 + nr) - 1;
    if (lo <= hi) {
      const long long a = t0 + (lo - r0) * b / SC_NQ;
      long long last_q = (hi - r0 + 1) * b - 1;
      if (last_q > n - 1) last_q = n - 1;
      const long long z = t0 + last_q / SC_NQ;
      if (qlo < 0) qlo = a;
      qhi = z;
    }
    t0 += nt;
    r0 += nr;
  }
  if (qlo < 0) return cudaSuccess;
  const int cnt = (int)(qhi - qlo + 1);
  return d_idx == 128 ? launch_scores_tc<128>(g, q_idx, k_idx, idx_scale, local_window, local_bias, row_begin, row_count,
                                              max_n_valid, (int)qlo, cnt, scores, ld, st)
                      : launch_scores_tc<64>(g, q_idx, k_idx, idx_scale, local_window, local_bias, row_begin, row_count,
                                             max_n_valid, (int)qlo, cnt, scores, ld, st);
}
