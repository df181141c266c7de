// sp_mma_attn.cu -- per-query (b_sel == 1 or small blocks) gather-sparse GQA attention.
//
// Every query has its own support, so a gathered K/V row serves only the G heads of one KV group: there is no M
// dimension worth a tcgen05 tile and the stage is bound by the gather (north_star).  One WARP per (query, KV head):
//   * the support's K and V rows are gathered 32 keys at a time with cp.async 16-byte vectors into a swizzled
//     shared-memory tile (the only bulk traffic; everything else stays in registers),
//   * S = Q_g K^T and O += P V run on warp-level mma.sync m16n8k16 (bf16 in, fp32 accumulate) with the G heads in
//     rows 0..G-1 of the 16-row tile -- 1/4 of the rows are useful at G = 4, which is still ~6x fewer issue slots
//     than the CUDA-core formulation and leaves the gather as the bound,
//   * online softmax per head row with the accumulator -> A-fragment register reuse (no shared-memory round trip).
// Masking is by INDEX VALUE (entries < 0, outside the sequence or above the query are dropped).
#include "sp_common.cuh"

namespace {

constexpr int PQ_WARPS = 4;    // warps per CTA; 16 KB of shared memory per warp at d = 128
constexpr int PQ_KEYS = 32;    // keys per gathered tile

__device__ __forceinline__ uint32_t pq_smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void pq_cp_async16(uint32_t dst, const void* src) {
  asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(dst), "l"(src) : "memory");
}
__device__ __forceinline__ void pq_cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
template <int N>
__device__ __forceinline__ void pq_cp_async_wait_group() { asm volatile("cp.async.wait_group %0;" ::"n"(N) : "memory"); }
__device__ __forceinline__ void pq_ldsm_x4(uint32_t addr, uint32_t& r0, uint32_t& r1, uint32_t& r2, uint32_t& r3) {
  asm volatile("ldmatrix.sync.aligned.m8n8.x4.shared.b16 {%0, %1, %2, %3}, [%4];"
               : "=r"(r0), "=r"(r1), "=r"(r2), "=r"(r3)
               : "r"(addr));
}
__device__ __forceinline__ void pq_ldsm_x4_t(uint32_t addr, uint32_t& r0, uint32_t& r1, uint32_t& r2, uint32_t& r3) {
  asm volatile("ldmatrix.sync.aligned.m8n8.x4.trans.shared.b16 {%0, %1, %2, %3}, [%4];"
               : "=r"(r0), "=r"(r1), "=r"(r2), "=r"(r3)
               : "r"(addr));
}
// D (16x8 fp32) += A (16x16 bf16, row) * B (16x8 bf16, col)
__device__ __forceinline__ void pq_mma(float* c, uint32_t a0, uint32_t a1, uint32_t a2, uint32_t a3, uint32_t b0,
                                       uint32_t b1) {
  asm volatile(
      "mma.sync.aligned.m16n8k16.row.col.f32.bf16.bf16.f32 {%0, %1, %2, %3}, {%4, %5, %6, %7}, {%8, %9}, "
      "{%0, %1, %2, %3};"
      : "+f"(c[0]), "+f"(c[1]), "+f"(c[2]), "+f"(c[3])
      : "r"(a0), "r"(a1), "r"(a2), "r"(a3), "r"(b0), "r"(b1));
}
// byte offset of 16-byte chunk c of row r in a [rows x D] bf16 tile: chunks are XOR-swizzled inside groups of 8 so
// that the 8 row addresses of one ldmatrix 8x8 block fall into distinct banks
template <int D>
__device__ __forceinline__ uint32_t pq_off(int r, int c) {
  return (uint32_t)(r * (D * 2) + ((((c & 7) ^ (r & 7)) | (c & ~7)) << 4));
}

template <int D, int G>
__global__ void __launch_bounds__(PQ_WARPS * 32, 3)  // 3 CTAs per SM (the shared-memory limit at d = 128): <= 168 registers; at 180 only 2 fit
sp_attn_pq_kernel(SpGeom g, const __nv_bfloat16* __restrict__ Q, const __nv_bfloat16* __restrict__ K,
                  const __nv_bfloat16* __restrict__ V, const int32_t* __restrict__ idx, int k, int Hkv, float scale,
                  int local_window, float local_bias, int q_begin, int q_count, int kv_div,
                  __nv_bfloat16* __restrict__ O, float* __restrict__ lse) {
  constexpr int KS = D / 16;   // k-slices of the QK^T contraction
  constexpr int NT = D / 8;    // 8-channel n tiles of O
  constexpr int CPR = D / 8;   // 16-byte chunks per row
  extern __shared__ __align__(128) uint8_t pq_smem[];
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const long long wid = (long long)blockIdx.x * PQ_WARPS + warp;
  // units per query: the Hkv KV groups (G heads each share the gathered rows), or -- one support list per HEAD
  // (PAPER.md:100 S_{l,t,h}; G == 1 instantiation, kv_div = heads per KV group) -- the Hq heads, each gathering its own rows
  const int NU = Hkv * kv_div;
  if (wid >= (long long)q_count * NU) return;
  const int t = q_begin + (int)(wid / NU);
  const int unit = (int)(wid % NU);
  const int kvh = unit / kv_div;  // KV head whose rows are gathered
  const int Hq = NU * G;
  const SpPos pi = sp_pos_info(g, t);
  const int gq = lane >> 2, tq = lane & 3;  // fragment coordinates: row group, column pair
  uint8_t* sK = pq_smem + (size_t)warp * (2 * PQ_KEYS * D * 2);
  uint8_t* sV = sK + PQ_KEYS * D * 2;
  const uint32_t sK_u = pq_smem_u32(sK), sV_u = pq_smem_u32(sV);

  // ---- A fragments of Q: head h = row gq (< G), channels ks*16 + 2 tq (+1) and + 8 ----
  uint32_t qa[KS][2];
  {
    const __nv_bfloat16* qr = Q + ((size_t)(t - g.q_off) * Hq + unit * G + min(gq, G - 1)) * D;
#pragma unroll
    for (int ks = 0; ks < KS; ++ks) {
      qa[ks][0] = gq < G ? *reinterpret_cast<const uint32_t*>(qr + ks * 16 + 2 * tq) : 0u;
      qa[ks][1] = gq < G ? *reinterpret_cast<const uint32_t*>(qr + ks * 16 + 2 * tq + 8) : 0u;
    }
  }
  const float sl2 = scale * SP_LOG2E, lb2 = local_bias * SP_LOG2E;
  float m_run = -INFINITY, l_run = 0.f;  // of head row gq (lanes with gq >= G carry harmless junk rows)
  float o[NT][4];
#pragma unroll
  for (int n = 0; n < NT; ++n) o[n][0] = o[n][1] = o[n][2] = o[n][3] = 0.f;
  const int32_t* sup = idx + (size_t)unit * (size_t)g.idx_grp + (size_t)(pi.row - g.row_off) * k;

  int e_next = lane < k ? __ldg(sup + lane) : -1;  // index entries are fetched ONE TILE AHEAD (their L2 latency used to
                                                   // sit in front of every tile's gathers)
  for (int c0 = 0; c0 < k; c0 += PQ_KEYS) {
    // ---- this lane's key of the tile ----
    int sp = -1;
    if (e_next >= pi.seq_start && e_next <= t) sp = e_next;
    e_next = c0 + PQ_KEYS + lane < k ? __ldg(sup + c0 + PQ_KEYS + lane) : -1;
    if (__ballot_sync(0xffffffffu, sp >= 0) == 0) continue;
    const long long sp_row = sp_kv_row(g, sp >= 0 ? sp : t);  // row of this lane's key in the K / V tensors (paged or not)
    // ---- gather the 32 K rows and V rows (invalid keys: row of the query itself, masked below) ----
    __syncwarp();  // the previous tile's ldmatrix reads are done
#pragma unroll
    for (int i = 0; i < (PQ_KEYS * CPR) / 32; ++i) {
      const int e = i * 32 + lane, r = e / CPR, c = e % CPR;
      const long long pr = __shfl_sync(0xffffffffu, sp_row, r);
      const size_t goff = ((size_t)pr * Hkv + kvh) * D + c * 8;
      pq_cp_async16(sK_u + pq_off<D>(r, c), K + goff);
    }
    pq_cp_async_commit();
    if (O != nullptr) {
#pragma unroll
      for (int i = 0; i < (PQ_KEYS * CPR) / 32; ++i) {
        const int e = i * 32 + lane, r = e / CPR, c = e % CPR;
        const long long pr = __shfl_sync(0xffffffffu, sp_row, r);
        const size_t goff = ((size_t)pr * Hkv + kvh) * D + c * 8;
        pq_cp_async16(sV_u + pq_off<D>(r, c), V + goff);
      }
    }
    pq_cp_async_commit();
    pq_cp_async_wait_group<1>();  // K has landed; V keeps arriving under S = Q K^T and the softmax
    __syncwarp();

    // ---- S = Q K^T: 4 n tiles of 8 keys ----
    float s[4][4];
#pragma unroll
    for (int nt = 0; nt < 4; ++nt) {
      s[nt][0] = s[nt][1] = s[nt][2] = s[nt][3] = 0.f;
#pragma unroll
      for (int ks = 0; ks < KS; ks += 2) {
        // matrices: (keys nt*8.., chunk 2ks), (.., 2ks+1), (.., 2ks+2), (.., 2ks+3); lane supplies row lane%8 of matrix lane/8
        uint32_t b0, b1, b2, b3;
        pq_ldsm_x4(sK_u + pq_off<D>(nt * 8 + (lane & 7), 2 * ks + (lane >> 3)), b0, b1, b2, b3);
        pq_mma(s[nt], qa[ks][0], 0u, qa[ks][1], 0u, b0, b1);
        pq_mma(s[nt], qa[ks + 1][0], 0u, qa[ks + 1][1], 0u, b2, b3);
      }
    }
    // ---- scale, mask by index value, online softmax of row gq (columns nt*8 + 2 tq + {0,1}) ----
    float mx = -INFINITY;
#pragma unroll
    for (int nt = 0; nt < 4; ++nt) {
#pragma unroll
      for (int j = 0; j < 2; ++j) {
        const int pk = __shfl_sync(0xffffffffu, sp, nt * 8 + 2 * tq + j);
        float z = -INFINITY;
        if (pk >= 0) {
          z = s[nt][j] * sl2;
          if (local_window > 0 && t - pk < local_window) z += lb2;
        }
        s[nt][j] = z;
        mx = fmaxf(mx, z);
      }
    }
    mx = fmaxf(mx, __shfl_xor_sync(0xffffffffu, mx, 1));
    mx = fmaxf(mx, __shfl_xor_sync(0xffffffffu, mx, 2));
    const float m_new = fmaxf(m_run, mx);  // finite: the tile has a valid key, valid for every head
    const float corr = exp2f(m_run - m_new);
    float psum = 0.f;
    uint32_t pa[2][2];  // A fragments of P for the two 16-key slices: [slice][cols 2tq / 2tq+8]
#pragma unroll
    for (int nt = 0; nt < 4; ++nt) {
      const float p0 = exp2f(s[nt][0] - m_new), p1 = exp2f(s[nt][1] - m_new);
      psum += p0 + p1;
      pa[nt >> 1][nt & 1] = sp_pack_bf16(p0, p1);
    }
    psum += __shfl_xor_sync(0xffffffffu, psum, 1);
    psum += __shfl_xor_sync(0xffffffffu, psum, 2);
    l_run = l_run * corr + psum;
    m_run = m_new;
    if (O != nullptr) {
      pq_cp_async_wait_group<0>();
      __syncwarp();
#pragma unroll
      for (int n = 0; n < NT; ++n) {
        o[n][0] *= corr;
        o[n][1] *= corr;
      }
      // ---- O += P V: per 16-key slice, pairs of 8-channel n tiles ----
#pragma unroll
      for (int kt = 0; kt < 2; ++kt) {
#pragma unroll
        for (int n = 0; n < NT; n += 2) {
          // matrices: (keys kt*16+0..7, chunk n), (keys kt*16+8..15, chunk n), (.., chunk n+1) x 2; transposed loads
          uint32_t b0, b1, b2, b3;
          pq_ldsm_x4_t(sV_u + pq_off<D>(kt * 16 + (lane & 7) + ((lane >> 3) & 1) * 8, n + (lane >> 4)), b0, b1, b2, b3);
          pq_mma(o[n], pa[kt][0], 0u, pa[kt][1], 0u, b0, b1);
          pq_mma(o[n + 1], pa[kt][0], 0u, pa[kt][1], 0u, b2, b3);
        }
      }
    }
  }
  // ---- epilogue: rows gq < G ----
  if (gq < G) {
    const size_t orow = (size_t)(t - g.q_off) * Hq + unit * G + gq;
    if (O != nullptr) {
      const float inv = l_run > 0.f ? 1.f / l_run : 0.f;
      __nv_bfloat16* dst = O + orow * D + 2 * tq;
#pragma unroll
      for (int n = 0; n < NT; ++n)
        *reinterpret_cast<uint32_t*>(dst + n * 8) = sp_pack_bf16(o[n][0] * inv, o[n][1] * inv);
    }
    if (lse != nullptr && tq == 0) lse[orow] = l_run > 0.f ? (m_run + log2f(l_run)) * SP_LN2 : -INFINITY;
  }
}

template <int D, int G>
cudaError_t launch_pq(const SpGeom& g, const void* Q, const void* K, const void* V, const int32_t* idx, int k, int Hkv,
                      float scale, int lw, float lb, int q_begin, int q_count, int kv_div, void* O, float* lse,
                      cudaStream_t st) {
  const size_t smem = (size_t)PQ_WARPS * 2 * PQ_KEYS * D * 2;
  static unsigned char attr_seen[SP_MAX_DEVICES];
  if (sp_first_use_on_device(attr_seen)) {
    cudaError_t e = cudaFuncSetAttribute(sp_attn_pq_kernel<D, G>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
  }
  const long long warps = (long long)q_count * Hkv * kv_div;
  sp_attn_pq_kernel<D, G><<<(unsigned)((warps + PQ_WARPS - 1) / PQ_WARPS), PQ_WARPS * 32, smem, st>>>(
      g, (const __nv_bfloat16*)Q, (const __nv_bfloat16*)K, (const __nv_bfloat16*)V, idx, k, Hkv, scale, lw, lb, q_begin,
      q_count, kv_div, (__nv_bfloat16*)O, lse);
  return cudaGetLastError();
}

template <int D>
cudaError_t launch_pq_d(int G, const SpGeom& g, const void* Q, const void* K, const void* V, const int32_t* idx, int k,
                        int Hkv, float scale, int lw, float lb, int q_begin, int q_count, bool per_head, void* O,
                        float* lse, cudaStream_t st) {
  if (per_head) return launch_pq<D, 1>(g, Q, K, V, idx, k, Hkv, scale, lw, lb, q_begin, q_count, G, O, lse, st);
  switch (G) {
    case 1: return launch_pq<D, 1>(g, Q, K, V, idx, k, Hkv, scale, lw, lb, q_begin, q_count, 1, O, lse, st);
    case 2: return launch_pq<D, 2>(g, Q, K, V, idx, k, Hkv, scale, lw, lb, q_begin, q_count, 1, O, lse, st);
    case 4: return launch_pq<D, 4>(g, Q, K, V, idx, k, Hkv, scale, lw, lb, q_begin, q_count, 1, O, lse, st);
    case 8: return launch_pq<D, 8>(g, Q, K, V, idx, k, Hkv, scale, lw, lb, q_begin, q_count, 1, O, lse, st);
  }
  return cudaErrorInvalidValue;
}

}  // namespace

// Sparse attention of the packed queries [q_begin, q_begin + q_count) with one support row per sp_pos_info(g, t).row.
cudaError_t sp_launch_attn_pq(const SpGeom& g, const void* Q, const void* K, const void* V, const int32_t* idx, int k,
                              int Hq, int Hkv, int d, float scale, int local_window, float local_bias, int q_begin,
                              int q_count, void* O, float* lse, cudaStream_t st, bool per_head) {
  if (q_count <= 0) return cudaSuccess;
  const int G = Hq / Hkv;
  cudaError_t e = d == 128 ? launch_pq_d<128>(G, g, Q, K, V, idx, k, Hkv, scale, local_window, local_bias, q_begin,
                                              q_count, per_head, O, lse, st)
                           : launch_pq_d<64>(G, g, Q, K, V, idx, k, Hkv, scale, local_window, local_bias, q_begin,
                                             q_count, per_head, O, lse, st);
  sp_count_launch();
  return e;
}
