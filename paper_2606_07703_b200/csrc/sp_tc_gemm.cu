// sp_tc_gemm.cu -- tcgen05/TMEM/TMA kernel for the indexer projection (the score GEMM lives in sp_tc_score.cu):
//   * sp_tc_project_kernel : q_idx = bf16(X Wqi), k_idx = bf16(X Wki)
// One output tile per CTA: TMA (SWIZZLE_128B) -> shared memory -> tcgen05.mma with the fp32 accumulator in
// TMEM -> tcgen05.ld epilogue.  Also holds the host-side tensor-map helper shared by the TMA kernels.
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

// bf16 tensor [d2][d1][d0] (d0 contiguous) with byte strides s1, s2; box = [b2 x b1 x 64 elements], SWIZZLE_128B.
cudaError_t sp_make_tmap_bf16_3d(CUtensorMap* out, const void* base, uint64_t d0, uint64_t d1, uint64_t d2, uint64_t s1,
                                 uint64_t s2, uint32_t b1, uint32_t b2) {
  sp_encode_tiled_fn enc = sp_get_encode();
  if (!enc) return cudaErrorNotSupported;
  const cuuint64_t dims[3] = {d0, d1, d2};
  const cuuint64_t strides[2] = {s1, s2};
  const cuuint32_t box[3] = {64, b1, b2};
  const cuuint32_t estr[3] = {1, 1, 1};
  const CUresult r = enc(out, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 3, const_cast<void*>(base), dims, strides, box, estr,
                         CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                         CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
  return r == CUDA_SUCCESS ? cudaSuccess : cudaErrorInvalidValue;
}

namespace {

__device__ __forceinline__ uint8_t* align1024(uint8_t* p) {
  return reinterpret_cast<uint8_t*>((reinterpret_cast<uintptr_t>(p) + 1023) & ~(uintptr_t)1023);
}

// ===================================================================================================
// Projection: C[m, 0:DI] = X[m,:] Wq, C[m, DI:2DI] = X[m,:] Wk.   M tile 128 or 256 (`halves`: two 128-row halves, two accumulators
// sharing every B stage: the weights are re-read from L2 once per 256 rows, which is what bounds the kernel on the
// per-SM L2 bandwidth), N = 2*DI, K pipelined by 64.
// ===================================================================================================
constexpr int PJ_STAGES = 4;  // ring slots with 128-token tiles (48 KB each at d_idx 128); 3 with 256-token tiles (64 KB)

template <int DI>
__global__ void __launch_bounds__(128, 1)
sp_tc_project_kernel(const __grid_constant__ CUtensorMap tmX, const __grid_constant__ CUtensorMap tmWq,
                     const __grid_constant__ CUtensorMap tmWk, __nv_bfloat16* __restrict__ q_idx,
                     __nv_bfloat16* __restrict__ k_idx, int L, int hidden, SpGeom g, uint32_t flags,
                     int halves) {
  constexpr int N = 2 * DI;
  constexpr int NG = N / 64;                  // 64-column groups of B
  constexpr uint32_t A_HALF = 128 * 128;      // 128 rows x 64 k
  constexpr uint32_t B_BYTES = NG * 64 * 128; // NG groups of [64 k-rows x 128 B]
  extern __shared__ uint8_t smem_raw[];
  uint8_t* smem = align1024(smem_raw);
  __shared__ uint64_t full[PJ_STAGES], empty[PJ_STAGES], done;
  __shared__ uint32_t tmem_slot;
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int m0 = blockIdx.x * 128 * halves;
  const int nh = (halves == 2 && m0 + 128 < L) ? 2 : 1;  // the last tile may hold one half only
  const int nkb = hidden / 64;
  const int NS = halves == 2 ? PJ_STAGES - 1 : PJ_STAGES;
  const uint32_t A_BYTES = A_HALF * halves, STAGE = A_BYTES + B_BYTES;

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
  if (warp == 1) tmem_alloc<2 * N>(&tmem_slot);
  tc_fence_before_sync();
  __syncthreads();
  tc_fence_after_sync();
  const uint32_t tmem = tmem_slot;

  if (warp == 0 && lane == 0) {
    int s = 0;
    uint32_t ph = 1;  // ring slot and the parity of its previous release (NS is a run-time value: no modulo here)
    for (int kb = 0; kb < nkb; ++kb, ++s) {
      if (s == NS) { s = 0; ph ^= 1; }
      if (kb >= NS) mbar_wait(&empty[s], ph);
      uint8_t* a = smem + (size_t)s * STAGE;
      uint8_t* b = a + A_BYTES;
      mbar_expect_tx(&full[s], A_HALF * nh + B_BYTES);
      tma_load_2d(a, &tmX, &full[s], kb * 64, m0);
      if (nh == 2) tma_load_2d(a + A_HALF, &tmX, &full[s], kb * 64, m0 + 128);
#pragma unroll
      for (int g = 0; g < DI / 64; ++g) {
        tma_load_2d(b + g * 8192, &tmWq, &full[s], g * 64, kb * 64);
        tma_load_2d(b + (DI / 64 + g) * 8192, &tmWk, &full[s], g * 64, kb * 64);
      }
    }
  } else if (warp == 1 && lane == 0) {
    constexpr uint32_t idesc = umma_idesc_bf16(128, N, 0, 1);  // A K-major, B MN-major
    // descriptors of ring slot 0, advanced by adding (byte offset >> 4) to the 14-bit address field (all of shared
    // memory is below 2^18 B, so the sum cannot carry out of the field): no descriptor arithmetic inside the loop
    const uint64_t ad0 = umma_desc_sw128(smem_u32(smem), 16, 1024);
    const uint64_t bd0 = umma_desc_sw128(smem_u32(smem) + A_BYTES, 8192, 1024);
    const uint64_t st16 = STAGE >> 4;
    int s = 0;
    uint32_t ph = 0;
    uint64_t so = 0;
    for (int kb = 0; kb < nkb; ++kb, ++s, so += st16) {
      if (s == NS) { s = 0; ph ^= 1; so = 0; }
      mbar_wait(&full[s], ph);
      tc_fence_after_sync();
      const uint64_t ad = ad0 + so, bd = bd0 + so;
      if (nh == 2) {
#pragma unroll
        for (int k = 0; k < 4; ++k) {
          umma_ss(tmem, ad + k * 2, bd + k * 128, idesc, (kb | k) != 0);
          umma_ss(tmem + N, ad + (A_HALF >> 4) + k * 2, bd + k * 128, idesc, (kb | k) != 0);
        }
      } else {
#pragma unroll
        for (int k = 0; k < 4; ++k) umma_ss(tmem, ad + k * 2, bd + k * 128, idesc, (kb | k) != 0);
      }
      umma_commit(&empty[s]);
    }
    umma_commit(&done);
  }
  __syncwarp();
  mbar_wait(&done, 0);
  tc_fence_after_sync();

  // epilogue: thread = output row of each half
  for (int h = 0; h < nh; ++h) {
  const int m = m0 + h * 128 + warp * 32 + lane;
  const uint32_t trow = tmem + h * N + ((uint32_t)(warp * 32) << 16);
  if ((flags & (SP_F_KEY_LN | SP_F_ROPE)) == 0) {
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
  } else {
    // The served scorer (readings A27/A28): LayerNorm of the KEY row over its DI channels (no
    // affine, biased variance, eps 1e-6), then RoPE of both rows in the rotate-half pairing (i, i + DI/2) at the
    // token's LOCAL position; everything in fp32 on the fp32 accumulator, ONE rounding to bf16.
    const int mm = min(m, L - 1);
    const int pos = g.pos_off + mm - sp_pos_info(g, mm).seq_start;
    float mean = 0.f, rstd = 1.f;
    if (flags & SP_F_KEY_LN) {
      float sum = 0.f;
#pragma unroll
      for (int c0 = 0; c0 < DI; c0 += 32) {
        uint32_t v[32];
        tmem_ld_x32(trow + DI + c0, v);
        tmem_ld_wait();
#pragma unroll
        for (int j = 0; j < 32; ++j) sum += __uint_as_float(v[j]);
      }
      mean = sum * (1.f / DI);
      float ss = 0.f;
#pragma unroll
      for (int c0 = 0; c0 < DI; c0 += 32) {
        uint32_t v[32];
        tmem_ld_x32(trow + DI + c0, v);
        tmem_ld_wait();
#pragma unroll
        for (int j = 0; j < 32; ++j) {
          const float dlt = __uint_as_float(v[j]) - mean;
          ss = fmaf(dlt, dlt, ss);
        }
      }
      rstd = rsqrtf(ss * (1.f / DI) + 1e-6f);
    }
    constexpr int H = DI / 2;
#pragma unroll
    for (int c0 = 0; c0 < H; c0 += 32) {
      float cs[32], sn[32];
      if (flags & SP_F_ROPE) {
#pragma unroll
        for (int j = 0; j < 32; ++j) {
          // theta = pos * 10000^(-2i/DI), reduced to [-pi, pi] in double before the fp32 sin / cos
          const double inv_freq = exp2(-(double)(2 * (c0 + j)) / DI * 13.287712379549449);  // log2(10000)
          const double th = (double)pos * inv_freq;
          const float r = (float)(th - 6.283185307179586 * rint(th * 0.15915494309189535));
          cs[j] = cosf(r);
          sn[j] = sinf(r);
        }
      } else {
#pragma unroll
        for (int j = 0; j < 32; ++j) {
          cs[j] = 1.f;
          sn[j] = 0.f;
        }
      }
#pragma unroll
      for (int side = 0; side < 2; ++side) {
        uint32_t a[32], b2[32];
        tmem_ld_x32(trow + side * DI + c0, a);
        tmem_ld_x32(trow + side * DI + H + c0, b2);
        tmem_ld_wait();
        const float mu = side ? mean : 0.f, rs = side ? rstd : 1.f;
        float lo[32], hi[32];
#pragma unroll
        for (int j = 0; j < 32; ++j) {
          const float x = (__uint_as_float(a[j]) - mu) * rs, y = (__uint_as_float(b2[j]) - mu) * rs;
          lo[j] = x * cs[j] - y * sn[j];
          hi[j] = y * cs[j] + x * sn[j];
        }
        if (m < L) {
          __nv_bfloat16* dst = (side ? k_idx : q_idx) + (size_t)m * DI;
#pragma unroll
          for (int j = 0; j < 32; j += 8) {
            uint4 o;
            o.x = sp_pack_bf16(lo[j], lo[j + 1]);
            o.y = sp_pack_bf16(lo[j + 2], lo[j + 3]);
            o.z = sp_pack_bf16(lo[j + 4], lo[j + 5]);
            o.w = sp_pack_bf16(lo[j + 6], lo[j + 7]);
            *reinterpret_cast<uint4*>(dst + c0 + j) = o;
            o.x = sp_pack_bf16(hi[j], hi[j + 1]);
            o.y = sp_pack_bf16(hi[j + 2], hi[j + 3]);
            o.z = sp_pack_bf16(hi[j + 4], hi[j + 5]);
            o.w = sp_pack_bf16(hi[j + 6], hi[j + 7]);
            *reinterpret_cast<uint4*>(dst + H + c0 + j) = o;
          }
        }
      }
    }
  }
  }
  tc_fence_before_sync();
  __syncthreads();
  if (warp == 1) tmem_dealloc<2 * N>(tmem);
}

}  // namespace

// ---------------------------------------------------------------------------------------------------
// launchers
// ---------------------------------------------------------------------------------------------------
static int pj_sm_count() { return sp_sm_count(); }

template <int DI>
static cudaError_t launch_project_tc(const SpGeom& g, uint32_t flags, const void* X, const void* Wq, const void* Wk,
                                     void* q_idx, void* k_idx, int L, int hidden, cudaStream_t st) {
  CUtensorMap tmX, tmWq, tmWk;
  cudaError_t e;
  if ((e = sp_make_tmap_bf16(&tmX, X, L, hidden, hidden, 128)) != cudaSuccess) return e;
  if ((e = sp_make_tmap_bf16(&tmWq, Wq, hidden, DI, DI, 64)) != cudaSuccess) return e;
  if ((e = sp_make_tmap_bf16(&tmWk, Wk, hidden, DI, DI, 64)) != cudaSuccess) return e;
  constexpr size_t s1 = (size_t)PJ_STAGES * (128 * 128 + (2 * DI / 64) * 8192);
  constexpr size_t s2 = (size_t)(PJ_STAGES - 1) * (2 * 128 * 128 + (2 * DI / 64) * 8192);
  constexpr size_t smem = (s1 > s2 ? s1 : s2) + 1024;
  static unsigned char attr_seen[SP_MAX_DEVICES];
  if (sp_first_use_on_device(attr_seen)) {
    e = cudaFuncSetAttribute(sp_tc_project_kernel<DI>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
  }
  // 128- or 256-token CTAs (one CTA per SM): whichever needs less time by waves x tile cost, a 256-token tile costing
  // 1.45-1.85x a 128-token one (measured at 32K-128K tokens: the weights are read once per tile; 1.7 is used).
  // Short inputs keep the finer grid.
  const int sms = pj_sm_count();
  const int t1 = (L + 127) / 128, t2 = (L + 255) / 256;
  const double c1 = (double)((t1 + sms - 1) / sms), c2 = 1.7 * (double)((t2 + sms - 1) / sms);
  const int halves = (t1 > sms && c2 <= c1) ? 2 : 1;
  const int tile = 128 * halves;
  sp_tc_project_kernel<DI><<<(L + tile - 1) / tile, 128, smem, st>>>(tmX, tmWq, tmWk, (__nv_bfloat16*)q_idx,
                                                               (__nv_bfloat16*)k_idx, L, hidden, g, flags, halves);
  sp_count_launch();
  return cudaGetLastError();
}

cudaError_t sp_launch_project_tc(const SpGeom& g, uint32_t flags, const void* X, const void* Wq, const void* Wk,
                                 void* q_idx, void* k_idx, int L, int hidden, int d_idx, cudaStream_t st) {
  return d_idx == 128 ? launch_project_tc<128>(g, flags, X, Wq, Wk, q_idx, k_idx, L, hidden, st)
                      : launch_project_tc<64>(g, flags, X, Wq, Wk, q_idx, k_idx, L, hidden, st);
}
