// sp_tc_attn.cu -- GQA attention with online softmax on tcgen05 / TMEM (PAPER.md:94 dense, :107 + :156 sparse).
//
// One CTA = one chunk of up to 256/G consecutive queries of ONE support row x one KV head: the G query heads of
// the KV group are stacked along the MMA M dimension (row R = query * G + head), so one gathered K/V tile is
// shared by 256 rows (two M = 128 tiles).  Key tiles hold 64 keys.
//   SPARSE: the keys are the support row's index list (gathered rows, cp.async 16-byte vectors, 128-byte swizzle
//           written by hand so the tile has the image TMA SWIZZLE_128B would have produced);
//   DENSE : the keys are the causal prefix of the sequence (same loader, consecutive rows).
// Warp roles: warps 0-3 / 4-7 softmax of M tile 0 / 1 (thread = row, TMEM lane = row), warp 8 MMA issuer
// (one elected thread), warps 9-12 K/V/Q loaders.  Per key tile and M tile:
//   S = Q K^T (tcgen05.mma, fp32 in TMEM, double buffered) -> tcgen05.ld -> scale, mask by KEY POSITION VALUE,
//   online softmax with lazy rescaling of the TMEM-resident O accumulator -> P (bf16) to shared memory ->
//   O += P V (tcgen05.mma, V read MN-major from the same row-major tile).
// Only tiles that can contain a masked or locally-biased element take the per-element path (flags computed
// once per CTA from the index list).
#include "sp_common.cuh"
#include "sp_tc.cuh"

using namespace sptc;

namespace {

constexpr int AT_KT = 64;        // keys per tile
constexpr int AT_STAGES = 3;     // K/V ring
constexpr int AT_THREADS = 416;  // 8 softmax warps + 1 MMA warp + 4 loader warps
constexpr int AT_MMA_WARP = 8;
constexpr int AT_LOAD_WARP0 = 9;
constexpr float AT_RESCALE_THRESHOLD = 8.0f;  // log2 units: O is rescaled only when the row max grew by > 2^8

__device__ __forceinline__ void cp_async_arrive_noinc(uint64_t* bar) {
  asm volatile("cp.async.mbarrier.arrive.noinc.shared::cta.b64 [%0];" ::"r"(smem_u32(bar)) : "memory");
}

struct AtBarriers {
  uint64_t qfull;
  uint64_t kfull[AT_STAGES], kempty[AT_STAGES], vfull[AT_STAGES], vempty[AT_STAGES];
  uint64_t sfull[2][2], sempty[2][2];
  uint64_t pfull[2], pempty[2];
};

template <int D, int G, bool SPARSE, bool WITH_O>
__global__ void __launch_bounds__(AT_THREADS, 1)
sp_tc_attn_kernel(SpGeom g, const __nv_bfloat16* __restrict__ Q, const __nv_bfloat16* __restrict__ K,
                  const __nv_bfloat16* __restrict__ V, const int32_t* __restrict__ idx, int k, int Hkv, float scale,
                  int local_window, float local_bias, int chunks_per_row, __nv_bfloat16* __restrict__ O,
                  float* __restrict__ lse) {
  constexpr int QT = 256 / G;             // queries per CTA
  constexpr int KB = D / 64;              // 64-wide column blocks of a row
  constexpr int CPR = D / 8;              // 16-byte chunks per row
  constexpr uint32_t Q_BLK = 256 * 128;   // bytes of one column block of the Q tile (256 rows)
  constexpr uint32_t KV_BLK = AT_KT * 128;
  constexpr uint32_t KV_TILE = KB * KV_BLK;
  constexpr uint32_t P_TILE = 128 * 128;  // 128 rows x 64 keys bf16
  constexpr uint32_t TM_O = 0, TM_S = 256;

  extern __shared__ uint8_t smem_raw[];
  __shared__ AtBarriers bar;
  __shared__ uint32_t tmem_slot;
  __shared__ int n_eff_sh;

  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int kvh = blockIdx.y;
  const int Hq = Hkv * G;

  // ---- which queries ----
  int seq_start, t0, t1, row = 0;
  if (SPARSE) {
    row = blockIdx.x / chunks_per_row;
    const int ci = blockIdx.x % chunks_per_row;
    const SpRow ri = sp_row_info(g, row);
    seq_start = ri.seq_start;
    t0 = ri.t_first + ci * QT;
    t1 = min(t0 + QT - 1, ri.t_last);
    if (t0 > ri.t_last) return;
  } else {
    SpGeom g2 = g;
    g2.b_sel = QT;
    const SpRow ri = sp_row_info(g2, (int)(gridDim.x - 1 - blockIdx.x));  // heavy (late) chunks first
    seq_start = ri.seq_start;
    t0 = ri.t_first;
    t1 = ri.t_last;
    if (t1 < t0) return;
  }
  const int nq = t1 - t0 + 1;
  const int n_mt = (nq * G > 128) ? 2 : 1;
  const int32_t* sup = SPARSE ? idx + (size_t)row * k : nullptr;

  uint8_t* smem = reinterpret_cast<uint8_t*>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~(uintptr_t)1023);
  uint8_t* sQ = smem;
  uint8_t* sK = sQ + KB * Q_BLK;
  uint8_t* sV = sK + AT_STAGES * KV_TILE;
  uint8_t* sP = sV + AT_STAGES * KV_TILE;
  uint32_t* flags = reinterpret_cast<uint32_t*>(sP + 2 * P_TILE);  // SPARSE: one word per key tile

  // first query (packed) of each M tile and the position threshold below which a key needs no per-element work
  const int win = local_window > 0 ? local_window : 0;
  const int qa0 = seq_start + t0, qa1 = seq_start + t0 + 128 / G;

  // ---- prologue: tile count and per-tile flags ----
  int nt;
  int nt_mt[2];
  if (SPARSE) {
    const int nt_max = (k + AT_KT - 1) / AT_KT;
    if (threadIdx.x == 0) n_eff_sh = 0;
    for (int i = threadIdx.x; i < nt_max; i += AT_THREADS) flags[i] = (i * AT_KT + AT_KT > k) ? 3u : 0u;
    __syncthreads();
    int my_last = 0;
    for (int i = threadIdx.x; i < k; i += AT_THREADS) {
      const int p = __ldg(sup + i);
      if (p >= 0) my_last = i + 1;
      uint32_t f = 0;
      if (p < seq_start || p > qa0 - win) f |= 1u;
      if (p < seq_start || p > qa1 - win) f |= 2u;
      if (f) atomicOr(&flags[i / AT_KT], f);
    }
    if (my_last) atomicMax(&n_eff_sh, my_last);
    __syncthreads();
    nt = (n_eff_sh + AT_KT - 1) / AT_KT;
    nt_mt[0] = nt_mt[1] = nt;
  } else {
    nt = t1 / AT_KT + 1;
    nt_mt[0] = min(t0 + 128 / G - 1, t1) / AT_KT + 1;
    nt_mt[1] = nt;
  }
  const bool scale_pos = scale > 0.f;
  const float sl2 = scale * SP_LOG2E, lb2 = local_bias * SP_LOG2E;

  if (nt == 0) {  // empty support: O = 0, lse = -inf (reading A9)
    if (warp < 8) {
      const int R = warp * 32 + lane;
      const int ql = R / G, h = R % G;
      if (ql < nq) {
        const size_t orow = ((size_t)(seq_start + t0 + ql) * Hq + kvh * G + h);
        if (WITH_O) {
          uint4 z = make_uint4(0, 0, 0, 0);
          for (int c = 0; c < CPR; ++c) reinterpret_cast<uint4*>(O + orow * D)[c] = z;
        }
        if (lse) lse[orow] = -INFINITY;
      }
    }
    return;
  }

  // ---- barriers, TMEM ----
  if (threadIdx.x == 0) {
    mbar_init(&bar.qfull, 128);
    for (int s = 0; s < AT_STAGES; ++s) {
      mbar_init(&bar.kfull[s], 128);
      mbar_init(&bar.vfull[s], 128);
      mbar_init(&bar.kempty[s], 1);
      mbar_init(&bar.vempty[s], 1);
    }
    for (int m = 0; m < 2; ++m) {
      for (int b = 0; b < 2; ++b) {
        mbar_init(&bar.sfull[m][b], 1);
        mbar_init(&bar.sempty[m][b], 128);
      }
      mbar_init(&bar.pfull[m], 128);
      mbar_init(&bar.pempty[m], 1);
    }
    fence_barrier_init();
  }
  if (warp == AT_MMA_WARP) tmem_alloc<512>(&tmem_slot);
  tc_fence_before_sync();
  __syncthreads();
  tc_fence_after_sync();
  const uint32_t tmem = tmem_slot;

  if (warp >= AT_LOAD_WARP0) {
    // =========================================== loaders ===========================================
    const int ptid = threadIdx.x - AT_LOAD_WARP0 * 32;  // 0..127
    {  // Q tile: row R = query * G + head; rows past the chunk repeat its last query (outputs never written)
      for (int e = ptid; e < 256 * CPR; e += 128) {
        const int R = e / CPR, c = e % CPR;
        if (R >= n_mt * 128) break;
        const int ql = min(R / G, nq - 1), h = R % G;
        const __nv_bfloat16* src = Q + ((size_t)(seq_start + t0 + ql) * Hq + kvh * G + h) * D + c * 8;
        cp_async16(smem_u32(sQ + (c / 8) * Q_BLK) + sw128_offset(R, c % 8), src);
      }
      cp_async_arrive_noinc(&bar.qfull);
    }
    constexpr int KPP = 128 / CPR;       // keys per pass of the 128 loader threads
    constexpr int PASSES = AT_KT / KPP;  // passes per tile
    const int c = ptid % CPR;
    const int key0 = ptid / CPR;
    for (int j = 0; j < nt; ++j) {
      const int s = j % AT_STAGES, u = j / AT_STAGES;
      int pos[PASSES];
#pragma unroll
      for (int i = 0; i < PASSES; ++i) {
        const int col = j * AT_KT + key0 + i * KPP;
        int p;
        if (SPARSE) {
          p = col < k ? __ldg(sup + col) : -1;
          if (p < seq_start || p > seq_start + t1) p = seq_start;  // masked later; any valid row will do
        } else {
          p = seq_start + min(col, t1);
        }
        pos[i] = p;
      }
      if (u > 0) mbar_wait(&bar.kempty[s], (u - 1) & 1);
#pragma unroll
      for (int i = 0; i < PASSES; ++i) {
        const int key = key0 + i * KPP;
        cp_async16(smem_u32(sK + s * KV_TILE + (c / 8) * KV_BLK) + sw128_offset(key, c % 8),
                   K + ((size_t)pos[i] * Hkv + kvh) * D + c * 8);
      }
      cp_async_arrive_noinc(&bar.kfull[s]);
      if (WITH_O) {
        if (u > 0) mbar_wait(&bar.vempty[s], (u - 1) & 1);
#pragma unroll
        for (int i = 0; i < PASSES; ++i) {
          const int key = key0 + i * KPP;
          cp_async16(smem_u32(sV + s * KV_TILE + (c / 8) * KV_BLK) + sw128_offset(key, c % 8),
                     V + ((size_t)pos[i] * Hkv + kvh) * D + c * 8);
        }
        cp_async_arrive_noinc(&bar.vfull[s]);
      }
    }
    cp_async_wait<0>();
  } else if (warp == AT_MMA_WARP) {
    // =========================================== MMA issuer ===========================================
    if (lane == 0) {
      constexpr uint32_t idesc_s = umma_idesc_bf16(128, AT_KT, 0, 0);  // S = Q K^T : both K-major
      constexpr uint32_t idesc_o = umma_idesc_bf16(128, D, 0, 1);      // O += P V : V is MN-major
      mbar_wait(&bar.qfull, 0);
      tc_fence_after_sync();
      const uint32_t q_addr = smem_u32(sQ), k_addr = smem_u32(sK), v_addr = smem_u32(sV), p_addr = smem_u32(sP);
      auto issue_s = [&](int j) {
        const int s = j % AT_STAGES;
        mbar_wait(&bar.kfull[s], (j / AT_STAGES) & 1);
        tc_fence_after_sync();
        for (int mt = 0; mt < n_mt; ++mt) {
          if (j >= nt_mt[mt]) continue;
          const int b = j & 1, n = j >> 1;
          if (n > 0) {
            mbar_wait(&bar.sempty[mt][b], (n - 1) & 1);
            tc_fence_after_sync();
          }
#pragma unroll
          for (int kk = 0; kk < D / 16; ++kk) {
            const uint64_t ad = umma_desc_sw128(q_addr + (kk / 4) * Q_BLK + mt * 16384 + (kk % 4) * 32, 16, 1024);
            const uint64_t bd = umma_desc_sw128(k_addr + s * KV_TILE + (kk / 4) * KV_BLK + (kk % 4) * 32, 16, 1024);
            umma_ss(tmem + TM_S + mt * 128 + b * 64, ad, bd, idesc_s, kk != 0);
          }
          umma_commit(&bar.sfull[mt][b]);
        }
        umma_commit(&bar.kempty[s]);
      };
      auto issue_pv = [&](int j) {
        const int s = j % AT_STAGES;
        mbar_wait(&bar.vfull[s], (j / AT_STAGES) & 1);
        for (int mt = 0; mt < n_mt; ++mt) {
          if (j >= nt_mt[mt]) continue;
          mbar_wait(&bar.pfull[mt], j & 1);
          tc_fence_after_sync();
#pragma unroll
          for (int kk = 0; kk < AT_KT / 16; ++kk) {
            const uint64_t ad = umma_desc_sw128(p_addr + mt * P_TILE + kk * 32, 16, 1024);
            const uint64_t bd = umma_desc_sw128(v_addr + s * KV_TILE + kk * 2048, KV_BLK, 1024);
            umma_ss(tmem + TM_O + mt * 128, ad, bd, idesc_o, (j | kk) != 0);
          }
          umma_commit(&bar.pempty[mt]);
        }
        umma_commit(&bar.vempty[s]);
      };
      issue_s(0);
      for (int j = 0; j < nt; ++j) {
        if (j + 1 < nt) issue_s(j + 1);
        if (WITH_O) issue_pv(j);
      }
    }
    __syncwarp();
  } else if (warp / 4 < n_mt) {
    // =========================================== softmax ===========================================
    const int mt = warp / 4;
    const int r = (warp % 4) * 32 + lane;  // row inside the M tile == TMEM lane
    const int R = mt * 128 + r;
    const int ql = R / G, h = R % G;
    const bool row_valid = ql < nq;
    const int tl = t0 + min(ql, nq - 1);  // local query position of this row
    const int tp = seq_start + tl;        // packed
    const uint32_t lane_base = (uint32_t)((warp % 4) * 32) << 16;
    const uint32_t t_s = tmem + lane_base + TM_S + mt * 128;
    const uint32_t t_o = tmem + lane_base + TM_O + mt * 128;
    const int qa_local = t0 + mt * (128 / G);
    float m_run = -INFINITY, l_run = 0.f;
    const int my_nt = nt_mt[mt];
    for (int j = 0; j < my_nt; ++j) {
      const int b = j & 1;
      mbar_wait(&bar.sfull[mt][b], (j >> 1) & 1);
      tc_fence_after_sync();
      uint32_t v[AT_KT];
      tmem_ld_x32(t_s + b * 64, v);
      tmem_ld_x32(t_s + b * 64 + 32, v + 32);
      tmem_ld_wait();
      tc_fence_before_sync();
      mbar_arrive(&bar.sempty[mt][b]);

      bool flagged;
      if (SPARSE) flagged = ((flags[j] >> mt) & 1u) != 0;
      else flagged = (j * AT_KT + AT_KT - 1 > qa_local - win);
      flagged = flagged || !scale_pos;
      float mx;
      if (!flagged) {
        float a = __uint_as_float(v[0]);
#pragma unroll
        for (int cc = 1; cc < AT_KT; ++cc) a = fmaxf(a, __uint_as_float(v[cc]));
        mx = a * sl2;
      } else {
        mx = -INFINITY;
#pragma unroll
        for (int cc = 0; cc < AT_KT; ++cc) {
          const int col = j * AT_KT + cc;
          bool ok;
          int dist;
          if (SPARSE) {
            const int p = col < k ? __ldg(sup + col) : -1;
            ok = p >= seq_start && p <= tp;
            dist = tp - p;
          } else {
            ok = col <= tl;
            dist = tl - col;
          }
          float x = -INFINITY;
          if (ok) x = fmaf(__uint_as_float(v[cc]), sl2, (win > 0 && dist < win) ? lb2 : 0.f);
          v[cc] = __float_as_uint(x);  // already scaled
          mx = fmaxf(mx, x);
        }
      }
      // ---- running max with lazy rescale of the TMEM accumulator ----
      const float m_new = fmaxf(m_run, mx);
      const bool need = m_new > m_run + AT_RESCALE_THRESHOLD;  // also true for the first finite max
      bool waited_pv = false;
      if (__any_sync(0xffffffffu, need)) {
        const float f = need ? exp2f(m_run - m_new) : 1.f;  // m_run = -inf -> 0
        if (WITH_O && j > 0) {
          mbar_wait(&bar.pempty[mt], (j - 1) & 1);  // PV(j-1) has finished updating O
          tc_fence_after_sync();
          waited_pv = true;
#pragma unroll
          for (int c0 = 0; c0 < D; c0 += 32) {
            uint32_t o[32];
            tmem_ld_x32(t_o + c0, o);
            tmem_ld_wait();
#pragma unroll
            for (int i = 0; i < 32; ++i) o[i] = __float_as_uint(__uint_as_float(o[i]) * f);
            tmem_st_x32(t_o + c0, o);
          }
          tmem_st_wait();
        }
        l_run *= f;
        if (need) m_run = m_new;
      }
      const float m_off = (m_run == -INFINITY) ? 0.f : m_run;
      float sum = 0.f;
      uint32_t pk[AT_KT / 2];
      if (!flagged) {
#pragma unroll
        for (int cc = 0; cc < AT_KT; cc += 2) {
          const float p0 = exp2f(fmaf(__uint_as_float(v[cc]), sl2, -m_off));
          const float p1 = exp2f(fmaf(__uint_as_float(v[cc + 1]), sl2, -m_off));
          sum += p0 + p1;
          pk[cc / 2] = sp_pack_bf16(p0, p1);
        }
      } else {
#pragma unroll
        for (int cc = 0; cc < AT_KT; cc += 2) {
          const float p0 = exp2f(__uint_as_float(v[cc]) - m_off);
          const float p1 = exp2f(__uint_as_float(v[cc + 1]) - m_off);
          sum += p0 + p1;
          pk[cc / 2] = sp_pack_bf16(p0, p1);
        }
      }
      l_run += sum;
      if (WITH_O) {
        if (j > 0 && !waited_pv) mbar_wait(&bar.pempty[mt], (j - 1) & 1);  // PV(j-1) no longer reads P
        uint8_t* prow = sP + mt * P_TILE;
#pragma unroll
        for (int c8 = 0; c8 < 8; ++c8) {
          const uint4 w = make_uint4(pk[4 * c8], pk[4 * c8 + 1], pk[4 * c8 + 2], pk[4 * c8 + 3]);
          *reinterpret_cast<uint4*>(prow + sw128_offset(r, c8)) = w;
        }
        fence_proxy_async_smem();
        tc_fence_before_sync();
        mbar_arrive(&bar.pfull[mt]);
      }
    }
    // ---- epilogue ----
    const size_t orow = ((size_t)tp * Hq + kvh * G + h);
    if (WITH_O) {
      mbar_wait(&bar.pempty[mt], (my_nt - 1) & 1);
      tc_fence_after_sync();
      const float inv = l_run > 0.f ? 1.f / l_run : 0.f;
#pragma unroll
      for (int c0 = 0; c0 < D; c0 += 32) {
        uint32_t o[32];
        tmem_ld_x32(t_o + c0, o);
        tmem_ld_wait();
        if (row_valid) {
#pragma unroll
          for (int i = 0; i < 32; i += 8) {
            uint4 w;
            w.x = sp_pack_bf16(__uint_as_float(o[i]) * inv, __uint_as_float(o[i + 1]) * inv);
            w.y = sp_pack_bf16(__uint_as_float(o[i + 2]) * inv, __uint_as_float(o[i + 3]) * inv);
            w.z = sp_pack_bf16(__uint_as_float(o[i + 4]) * inv, __uint_as_float(o[i + 5]) * inv);
            w.w = sp_pack_bf16(__uint_as_float(o[i + 6]) * inv, __uint_as_float(o[i + 7]) * inv);
            *reinterpret_cast<uint4*>(O + orow * D + c0 + i) = w;
          }
        }
      }
    }
    if (lse != nullptr && row_valid) lse[orow] = l_run > 0.f ? (m_run + log2f(l_run)) * SP_LN2 : -INFINITY;
  }
  tc_fence_before_sync();
  __syncthreads();
  if (warp == AT_MMA_WARP) tmem_dealloc<512>(tmem);
}

template <int D>
size_t attn_smem_bytes(int k, bool sparse) {
  const size_t kb = D / 64;
  return kb * 256 * 128 + 2 * AT_STAGES * kb * AT_KT * 128 + 2 * 128 * 128 + (sparse ? 4 * (size_t)((k + AT_KT - 1) / AT_KT) : 0) +
         16 + 1024;
}

template <int D, int G, bool SPARSE, bool WITH_O>
cudaError_t launch_one(const SpGeom& g, dim3 grid, size_t smem, cudaStream_t st, const void* Q, const void* K,
                       const void* V, const int32_t* idx, int k, int Hkv, float scale, int lw, float lb, int cpr, void* O,
                       float* lse) {
  static size_t attr_smem = 0;
  if (smem > attr_smem) {
    cudaError_t e = cudaFuncSetAttribute(sp_tc_attn_kernel<D, G, SPARSE, WITH_O>,
                                         cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    attr_smem = smem;
  }
  sp_tc_attn_kernel<D, G, SPARSE, WITH_O><<<grid, AT_THREADS, smem, st>>>(
      g, (const __nv_bfloat16*)Q, (const __nv_bfloat16*)K, (const __nv_bfloat16*)V, idx, k, Hkv, scale, lw, lb, cpr,
      (__nv_bfloat16*)O, lse);
  return cudaGetLastError();
}

template <int D, int G>
cudaError_t launch_dg(const SpGeom& g, dim3 grid, cudaStream_t st, const void* Q, const void* K, const void* V,
                      const int32_t* idx, int k, int Hkv, float scale, int lw, float lb, int cpr, void* O, float* lse) {
  const bool sparse = idx != nullptr;
  const size_t smem = attn_smem_bytes<D>(k, sparse);
  if (smem > 227 * 1024) return cudaErrorInvalidValue;
  if (sparse) {
    if (O) return launch_one<D, G, true, true>(g, grid, smem, st, Q, K, V, idx, k, Hkv, scale, lw, lb, cpr, O, lse);
    return launch_one<D, G, true, false>(g, grid, smem, st, Q, K, V, idx, k, Hkv, scale, lw, lb, cpr, O, lse);
  }
  if (O) return launch_one<D, G, false, true>(g, grid, smem, st, Q, K, V, idx, k, Hkv, scale, lw, lb, cpr, O, lse);
  return launch_one<D, G, false, false>(g, grid, smem, st, Q, K, V, idx, k, Hkv, scale, lw, lb, cpr, O, lse);
}

template <int D>
cudaError_t launch_d(int G, const SpGeom& g, dim3 grid, cudaStream_t st, const void* Q, const void* K, const void* V,
                     const int32_t* idx, int k, int Hkv, float scale, int lw, float lb, int cpr, void* O, float* lse) {
  switch (G) {
    case 1: return launch_dg<D, 1>(g, grid, st, Q, K, V, idx, k, Hkv, scale, lw, lb, cpr, O, lse);
    case 2: return launch_dg<D, 2>(g, grid, st, Q, K, V, idx, k, Hkv, scale, lw, lb, cpr, O, lse);
    case 4: return launch_dg<D, 4>(g, grid, st, Q, K, V, idx, k, Hkv, scale, lw, lb, cpr, O, lse);
    case 8: return launch_dg<D, 8>(g, grid, st, Q, K, V, idx, k, Hkv, scale, lw, lb, cpr, O, lse);
  }
  return cudaErrorInvalidValue;
}

}  // namespace

// The tcgen05 attention covers dense attention always and sparse attention when a support row's queries fill a
// useful part of an M tile; per-query (b_sel == 1) supports are gather-bound and stay on the CUDA-core kernel.
bool sp_tc_attn_supported(int b_sel, int G, bool sparse, int k) {
  if (!sparse) return true;
  if (b_sel * G < 32) return false;
  return 4 * (size_t)((k + AT_KT - 1) / AT_KT) <= 16 * 1024;
}

// idx == nullptr -> dense causal attention over the whole pack.  n_chunks_dense = sum_i ceil(n_i / (256/G)).
cudaError_t sp_launch_attn_tc(const SpGeom& g, long long n_rows, long long n_chunks_dense, const void* Q, const void* K,
                              const void* V, const int32_t* idx, int k, int Hq, int Hkv, int d, float scale,
                              int local_window, float local_bias, void* O, float* lse, cudaStream_t st) {
  const int G = Hq / Hkv;
  const int QT = 256 / G;
  const bool sparse = idx != nullptr;
  const int cpr = sparse ? (g.b_sel + QT - 1) / QT : 1;
  const long long nx = sparse ? n_rows * cpr : n_chunks_dense;
  if (nx <= 0) return cudaSuccess;
  dim3 grid((unsigned)nx, (unsigned)Hkv);
  cudaError_t e = d == 128 ? launch_d<128>(G, g, grid, st, Q, K, V, idx, k, Hkv, scale, local_window, local_bias, cpr, O, lse)
                           : launch_d<64>(G, g, grid, st, Q, K, V, idx, k, Hkv, scale, local_window, local_bias, cpr, O, lse);
  sp_count_launch();
  return e;
}
