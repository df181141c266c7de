// sp_simt.cu -- CUDA-core kernels of the sparse-prefill path, used only OUTSIDE the tcgen05 kernels' built set
// (selection blocks b_sel not in {1,32,64,128}; dense attention over a query sub-range):
//   * indexer scoring + block max   z = idx_scale <q_idx[t],k_idx[s]>, R_B = max_t
//   * attention mass pass 2         P_t(s) = (1/Hq) sum_h exp(z - lse), R_B = max_t PAPER.md:123, :154
//   * warp-per-(query, KV head) attention with online softmax over a key list that is either the
//     causal prefix (dense) or the gathered support (sparse).
// Scoring/mass kernels give one thread one KEY (lane = key position) so that the max over a
// selection block's queries is a per-thread running max and global writes are coalesced along s.
#include "sp_common.cuh"

namespace {

// =============================================================================================
// Score / mass kernels: thread = key, block = (128-key tile, group of query rows).
// A "group" is the b_sel queries of one support row (b_sel > 1) or 64 consecutive packed
// positions (b_sel == 1, support row == packed position).
// =============================================================================================
constexpr int SC_KEYS = 128;  // keys (threads) per block
constexpr int SC_QSUB = 64;   // queries staged in shared memory at a time

struct SpGroup {
  int q_first;  // first packed query position of the group
  int q_count;  // number of queries
  int row0;     // support row of the first query
};

__device__ __forceinline__ SpGroup sp_group(const SpGeom& g, int row_begin, int row_count, int gi) {
  if (g.b_sel > 1) {
    const SpRow r = sp_row_info(g, row_begin + gi);
    return SpGroup{r.seq_start + r.t_first, r.t_last - r.t_first + 1, row_begin + gi};
  }
  const int q0 = row_begin + gi * SC_QSUB;
  return SpGroup{q0, min(SC_QSUB, row_begin + row_count - q0), q0};
}

template <int DI>
__global__ void __launch_bounds__(SC_KEYS)
sp_indexer_score_kernel(SpGeom g, const __nv_bfloat16* __restrict__ q_idx, const __nv_bfloat16* __restrict__ k_idx,
                        float idx_scale, int local_window, float local_bias, int row_begin, int row_count,
                        float* __restrict__ scores, int64_t ld) {
  __shared__ float qs[SC_QSUB][DI];
  __shared__ int q_seq_start[SC_QSUB];
  const SpGroup grp = sp_group(g, row_begin, row_count, blockIdx.y);
  const int s = blockIdx.x * SC_KEYS + threadIdx.x;  // local key position
  // skip tiles entirely above the diagonal of the group's last query (cheap upper bound: packed distance)
  const SpPos last = sp_pos_info(g, grp.q_first + grp.q_count - 1);
  {  // tiles entirely above the diagonal of every query of the group have nothing to do
    const int q_last = grp.q_first + grp.q_count - 1;
    const int tl_bound = g.b_sel > 1 ? q_last - last.seq_start : q_last;
    if ((int)(blockIdx.x * SC_KEYS) > tl_bound) return;
  }

  uint32_t kreg[DI / 2];
  int k_seq_start = -1;
  float best = -INFINITY;
  for (int sub = 0; sub < grp.q_count; sub += SC_QSUB) {
    const int nq = min(SC_QSUB, grp.q_count - sub);
    __syncthreads();
    for (int e = threadIdx.x; e < nq * (DI / 2); e += SC_KEYS) {
      const int qi = e / (DI / 2), c = e % (DI / 2);
      const uint32_t w =
          reinterpret_cast<const uint32_t*>(q_idx + (size_t)(grp.q_first + sub + qi) * DI)[c];
      qs[qi][2 * c] = sp_bf16lo(w);
      qs[qi][2 * c + 1] = sp_bf16hi(w);
    }
    if (threadIdx.x < nq) q_seq_start[threadIdx.x] = sp_pos_info(g, grp.q_first + sub + threadIdx.x).seq_start;
    __syncthreads();
    for (int qi = 0; qi < nq; ++qi) {
      const int t = grp.q_first + sub + qi;
      const int ss = q_seq_start[qi];
      const int tl = t - ss;
      if (blockIdx.x * SC_KEYS > tl) continue;  // uniform
      if (ss != k_seq_start) {                  // uniform: (re)load this thread's key row
        k_seq_start = ss;
        const int kp = min(ss + s, g.L - 1);
        const uint4* src = reinterpret_cast<const uint4*>(k_idx + (size_t)kp * DI);
#pragma unroll
        for (int c = 0; c < DI / 8; ++c) {
          const uint4 v = __ldg(src + c);
          kreg[4 * c] = v.x; kreg[4 * c + 1] = v.y; kreg[4 * c + 2] = v.z; kreg[4 * c + 3] = v.w;
        }
      }
      float acc0 = 0.f, acc1 = 0.f;
#pragma unroll
      for (int c = 0; c < DI / 2; ++c) {
        const float2 qv = *reinterpret_cast<const float2*>(&qs[qi][2 * c]);
        acc0 = fmaf(qv.x, sp_bf16lo(kreg[c]), acc0);
        acc1 = fmaf(qv.y, sp_bf16hi(kreg[c]), acc1);
      }
      if (s <= tl) {
        float z = (acc0 + acc1) * idx_scale;
        if (local_window > 0 && tl - s < local_window) z += local_bias;
        if (g.b_sel > 1) best = fmaxf(best, z);
        else scores[(size_t)(t - row_begin) * ld + s] = z;
      }
    }
  }
  if (g.b_sel > 1) {
    const int n_valid = grp.q_first + grp.q_count - last.seq_start;
    if (s < n_valid) scores[(size_t)(grp.row0 - row_begin) * ld + s] = best;
  }
}

constexpr int MS_QSUB = 32;  // queries per pass of the mass kernel (accumulators live in shared memory)

template <int D>
__global__ void __launch_bounds__(SC_KEYS)
sp_mass_kernel(SpGeom g, const __nv_bfloat16* __restrict__ Q, const __nv_bfloat16* __restrict__ K,
               const float* __restrict__ lse, int Hq, int Hkv, float scale, int local_window, float local_bias,
               int row_begin, int row_count, float* __restrict__ mass, int64_t ld) {
  __shared__ float qs[MS_QSUB][D];
  __shared__ float accs[MS_QSUB][SC_KEYS];  // [query][key thread]: conflict-free column per thread
  __shared__ float lse2[MS_QSUB];
  __shared__ int q_seq_start[MS_QSUB];
  const SpGroup grp = sp_group(g, row_begin, row_count, blockIdx.y);
  const int s = blockIdx.x * SC_KEYS + threadIdx.x;
  const SpPos last = sp_pos_info(g, grp.q_first + grp.q_count - 1);
  {  // tiles entirely above the diagonal of every query of the group have nothing to do
    const int q_last = grp.q_first + grp.q_count - 1;
    const int tl_bound = g.b_sel > 1 ? q_last - last.seq_start : q_last;
    if ((int)(blockIdx.x * SC_KEYS) > tl_bound) return;
  }
  const int G = Hq / Hkv;
  const float sl2 = scale * SP_LOG2E, lb2 = local_bias * SP_LOG2E;
  const float inv_hq = 1.f / (float)Hq;

  uint32_t kreg[D / 2];
  int k_seq_start = -1;
  float best = -INFINITY;
  for (int sub = 0; sub < grp.q_count; sub += MS_QSUB) {
    const int nq = min(MS_QSUB, grp.q_count - sub);
    for (int qi = 0; qi < MS_QSUB; ++qi) accs[qi][threadIdx.x] = 0.f;
    __syncthreads();
    if (threadIdx.x < nq) q_seq_start[threadIdx.x] = sp_pos_info(g, grp.q_first + sub + threadIdx.x).seq_start;
    for (int h = 0; h < Hq; ++h) {
      __syncthreads();
      for (int e = threadIdx.x; e < nq * (D / 2); e += SC_KEYS) {
        const int qi = e / (D / 2), c = e % (D / 2);
        const uint32_t w =
            reinterpret_cast<const uint32_t*>(Q + ((size_t)(grp.q_first + sub + qi) * Hq + h) * D)[c];
        qs[qi][2 * c] = sp_bf16lo(w);
        qs[qi][2 * c + 1] = sp_bf16hi(w);
      }
      if (threadIdx.x < nq) lse2[threadIdx.x] = lse[(size_t)(grp.q_first + sub + threadIdx.x) * Hq + h] * SP_LOG2E;
      __syncthreads();
      const int kvh = h / G;
      if (h % G == 0) k_seq_start = -1;  // new KV head: this thread's key row must be reloaded
#pragma unroll 1
      for (int qi = 0; qi < nq; ++qi) {
        const int t = grp.q_first + sub + qi;
        const int ss = q_seq_start[qi];
        const int tl = t - ss;
        if ((int)(blockIdx.x * SC_KEYS) > tl) continue;  // uniform
        if (ss != k_seq_start) {
          k_seq_start = ss;
          const int kp = min(ss + s, g.L - 1);
          const uint4* src = reinterpret_cast<const uint4*>(K + ((size_t)kp * Hkv + kvh) * D);
#pragma unroll
          for (int c = 0; c < D / 8; ++c) {
            const uint4 v = __ldg(src + c);
            kreg[4 * c] = v.x; kreg[4 * c + 1] = v.y; kreg[4 * c + 2] = v.z; kreg[4 * c + 3] = v.w;
          }
        }
        float a0 = 0.f, a1 = 0.f;
#pragma unroll
        for (int c = 0; c < D / 2; ++c) {
          const float2 qv = *reinterpret_cast<const float2*>(&qs[qi][2 * c]);
          a0 = fmaf(qv.x, sp_bf16lo(kreg[c]), a0);
          a1 = fmaf(qv.y, sp_bf16hi(kreg[c]), a1);
        }
        if (s <= tl) {
          float z2 = (a0 + a1) * sl2;
          if (local_window > 0 && tl - s < local_window) z2 += lb2;
          accs[qi][threadIdx.x] += exp2f(z2 - lse2[qi]);
        }
      }
    }
    for (int qi = 0; qi < nq; ++qi) {
      const int t = grp.q_first + sub + qi;
      const int tl = t - q_seq_start[qi];
      if (s <= tl) {
        const float p = accs[qi][threadIdx.x] * inv_hq;
        if (g.b_sel > 1) best = fmaxf(best, p);
        else mass[(size_t)(t - row_begin) * ld + s] = p;
      }
    }
    __syncthreads();
  }
  if (g.b_sel > 1) {
    const int n_valid = grp.q_first + grp.q_count - last.seq_start;
    if (s < n_valid) mass[(size_t)(grp.row0 - row_begin) * ld + s] = best;
  }
}

// =============================================================================================
// Attention: one warp per (query t, KV head).  Lanes own keys for QK^T, own channels for PV.
// =============================================================================================
template <int D, int G, bool SPARSE>
__global__ void __launch_bounds__(256)
sp_attn_warp_kernel(SpGeom g, const __nv_bfloat16* __restrict__ Q, const __nv_bfloat16* __restrict__ K,
                    const __nv_bfloat16* __restrict__ V, const int32_t* __restrict__ idx, int k, int Hkv, float scale,
                    int local_window, float local_bias, int q_begin, int q_count, __nv_bfloat16* __restrict__ O,
                    float* __restrict__ lse) {
  constexpr int WARPS = 8;
  constexpr int EPL = D / 32;  // channels per lane in the PV phase
  __shared__ float qsm[WARPS][G][D];
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const long long wid = (long long)blockIdx.x * WARPS + warp;
  if (wid >= (long long)q_count * Hkv) return;
  const int t = q_begin + (int)(wid / Hkv);
  const int kvh = (int)(wid % Hkv);
  const int Hq = Hkv * G;
  const SpPos pi = sp_pos_info(g, t);

  // stage the G query heads of this KV group as fp32
  for (int e = lane; e < G * D / 2; e += 32) {
    const int h = e / (D / 2), c = e % (D / 2);
    const uint32_t w = reinterpret_cast<const uint32_t*>(Q + ((size_t)t * Hq + kvh * G + h) * D)[c];
    qsm[warp][h][2 * c] = sp_bf16lo(w);
    qsm[warp][h][2 * c + 1] = sp_bf16hi(w);
  }
  __syncwarp();

  const float sl2 = scale * SP_LOG2E, lb2 = local_bias * SP_LOG2E;
  float m[G], l[G], o[G][EPL];
#pragma unroll
  for (int h = 0; h < G; ++h) {
    m[h] = -INFINITY;
    l[h] = 0.f;
#pragma unroll
    for (int e = 0; e < EPL; ++e) o[h][e] = 0.f;
  }
  const int n_keys = SPARSE ? k : (t - pi.seq_start + 1);
  const int32_t* sup = SPARSE ? idx + (size_t)kvh * (size_t)g.idx_grp + (size_t)pi.row * k : nullptr;

  for (int c0 = 0; c0 < n_keys; c0 += 32) {
    int sp = -1;  // packed key position of this lane, -1 = none
    if (c0 + lane < n_keys) {
      if (SPARSE) {
        const int e = __ldg(sup + c0 + lane);
        if (e >= pi.seq_start && e <= t) sp = e;
      } else {
        sp = pi.seq_start + c0 + lane;
      }
    }
    const uint32_t vmask = __ballot_sync(0xffffffffu, sp >= 0);
    if (vmask == 0) {
      if (SPARSE) continue;
      break;
    }
    float z[G];
#pragma unroll
    for (int h = 0; h < G; ++h) z[h] = 0.f;
    if (sp >= 0) {
      const uint4* kr = reinterpret_cast<const uint4*>(K + ((size_t)sp * Hkv + kvh) * D);
#pragma unroll
      for (int c = 0; c < D / 8; ++c) {
        const uint4 v = __ldg(kr + c);
        const float kf[8] = {sp_bf16lo(v.x), sp_bf16hi(v.x), sp_bf16lo(v.y), sp_bf16hi(v.y),
                             sp_bf16lo(v.z), sp_bf16hi(v.z), sp_bf16lo(v.w), sp_bf16hi(v.w)};
#pragma unroll
        for (int h = 0; h < G; ++h) {
          const float4 q0 = *reinterpret_cast<const float4*>(&qsm[warp][h][8 * c]);
          const float4 q1 = *reinterpret_cast<const float4*>(&qsm[warp][h][8 * c + 4]);
          z[h] = fmaf(q0.x, kf[0], z[h]); z[h] = fmaf(q0.y, kf[1], z[h]);
          z[h] = fmaf(q0.z, kf[2], z[h]); z[h] = fmaf(q0.w, kf[3], z[h]);
          z[h] = fmaf(q1.x, kf[4], z[h]); z[h] = fmaf(q1.y, kf[5], z[h]);
          z[h] = fmaf(q1.z, kf[6], z[h]); z[h] = fmaf(q1.w, kf[7], z[h]);
        }
      }
    }
    float p[G];
#pragma unroll
    for (int h = 0; h < G; ++h) {
      float z2 = -INFINITY;
      if (sp >= 0) {
        z2 = z[h] * sl2;
        if (local_window > 0 && t - sp < local_window) z2 += lb2;
      }
      const float mn = fmaxf(m[h], sp_warp_max(z2));  // finite: vmask != 0
      const float corr = exp2f(m[h] - mn);            // m = -inf -> 0
      p[h] = exp2f(z2 - mn);                          // invalid lane -> 0
      l[h] = l[h] * corr + sp_warp_sum(p[h]);
      m[h] = mn;
#pragma unroll
      for (int e = 0; e < EPL; ++e) o[h][e] *= corr;
    }
    if (O != nullptr) {
      uint32_t rem = vmask;
      while (rem) {
        const int j = __ffs(rem) - 1;
        rem &= rem - 1;
        const int sj = __shfl_sync(0xffffffffu, sp, j);
        const __nv_bfloat16* vr = V + ((size_t)sj * Hkv + kvh) * D + lane * EPL;
        float vf[EPL];
        if (EPL == 4) {
          const uint2 v = __ldg(reinterpret_cast<const uint2*>(vr));
          vf[0] = sp_bf16lo(v.x); vf[1] = sp_bf16hi(v.x); vf[EPL - 2] = sp_bf16lo(v.y); vf[EPL - 1] = sp_bf16hi(v.y);
        } else {
          const uint32_t v = __ldg(reinterpret_cast<const uint32_t*>(vr));
          vf[0] = sp_bf16lo(v); vf[1] = sp_bf16hi(v);
        }
#pragma unroll
        for (int h = 0; h < G; ++h) {
          const float pj = __shfl_sync(0xffffffffu, p[h], j);
#pragma unroll
          for (int e = 0; e < EPL; ++e) o[h][e] = fmaf(pj, vf[e], o[h][e]);
        }
      }
    }
  }
#pragma unroll
  for (int h = 0; h < G; ++h) {
    const int hq = kvh * G + h;
    if (O != nullptr) {
      const float inv = l[h] > 0.f ? 1.f / l[h] : 0.f;
      __nv_bfloat16* orow = O + ((size_t)t * Hq + hq) * D + lane * EPL;
      if (EPL == 4) {
        uint2 w;
        w.x = sp_pack_bf16(o[h][0] * inv, o[h][1] * inv);
        w.y = sp_pack_bf16(o[h][EPL - 2] * inv, o[h][EPL - 1] * inv);
        *reinterpret_cast<uint2*>(orow) = w;
      } else {
        *reinterpret_cast<uint32_t*>(orow) = sp_pack_bf16(o[h][0] * inv, o[h][1] * inv);
      }
    }
    if (lse != nullptr && lane == 0)
      lse[(size_t)t * Hq + hq] = l[h] > 0.f ? (m[h] + log2f(l[h])) * SP_LN2 : -INFINITY;
  }
}

template <int D, int G>
cudaError_t launch_attn_dg(bool sparse, dim3 grid, cudaStream_t st, const SpGeom& g, const void* Q, const void* K,
                           const void* V, const int32_t* idx, int k, int Hkv, float scale, int lw, float lb,
                           int q_begin, int q_count, void* O, float* lse) {
  auto q = (const __nv_bfloat16*)Q;
  auto kk = (const __nv_bfloat16*)K;
  auto v = (const __nv_bfloat16*)V;
  auto o = (__nv_bfloat16*)O;
  if (sparse)
    sp_attn_warp_kernel<D, G, true><<<grid, 256, 0, st>>>(g, q, kk, v, idx, k, Hkv, scale, lw, lb, q_begin, q_count, o, lse);
  else
    sp_attn_warp_kernel<D, G, false><<<grid, 256, 0, st>>>(g, q, kk, v, idx, k, Hkv, scale, lw, lb, q_begin, q_count, o, lse);
  return cudaGetLastError();
}

template <int D>
cudaError_t launch_attn_d(int G, bool sparse, dim3 grid, cudaStream_t st, const SpGeom& g, const void* Q,
                          const void* K, const void* V, const int32_t* idx, int k, int Hkv, float scale, int lw,
                          float lb, int q_begin, int q_count, void* O, float* lse) {
  switch (G) {
    case 1: return launch_attn_dg<D, 1>(sparse, grid, st, g, Q, K, V, idx, k, Hkv, scale, lw, lb, q_begin, q_count, O, lse);
    case 2: return launch_attn_dg<D, 2>(sparse, grid, st, g, Q, K, V, idx, k, Hkv, scale, lw, lb, q_begin, q_count, O, lse);
    case 4: return launch_attn_dg<D, 4>(sparse, grid, st, g, Q, K, V, idx, k, Hkv, scale, lw, lb, q_begin, q_count, O, lse);
    case 8: return launch_attn_dg<D, 8>(sparse, grid, st, g, Q, K, V, idx, k, Hkv, scale, lw, lb, q_begin, q_count, O, lse);
  }
  return cudaErrorInvalidValue;
}

int sp_num_groups(const SpGeom& g, int row_count) {
  return g.b_sel > 1 ? row_count : (row_count + SC_QSUB - 1) / SC_QSUB;
}

}  // namespace

cudaError_t sp_launch_indexer_scores(const SpGeom& g, const void* q_idx, const void* k_idx, int d_idx,
                                     float idx_scale, int local_window, float local_bias, int row_begin,
                                     int row_count, int max_n_valid, float* scores, int64_t ld, cudaStream_t st) {
  if (row_count <= 0) return cudaSuccess;
  dim3 grid((max_n_valid + SC_KEYS - 1) / SC_KEYS, sp_num_groups(g, row_count));
  auto q = (const __nv_bfloat16*)q_idx;
  auto k = (const __nv_bfloat16*)k_idx;
  if (d_idx == 128)
    sp_indexer_score_kernel<128><<<grid, SC_KEYS, 0, st>>>(g, q, k, idx_scale, local_window, local_bias, row_begin,
                                                           row_count, scores, ld);
  else
    sp_indexer_score_kernel<64><<<grid, SC_KEYS, 0, st>>>(g, q, k, idx_scale, local_window, local_bias, row_begin,
                                                          row_count, scores, ld);
  sp_count_launch();
  return cudaGetLastError();
}

cudaError_t sp_launch_mass(const SpGeom& g, const void* Q, const void* K, const float* lse, int Hq, int Hkv, int d,
                           float scale, int local_window, float local_bias, int row_begin, int row_count,
                           int max_n_valid, float* mass, int64_t ld, cudaStream_t st) {
  if (row_count <= 0) return cudaSuccess;
  dim3 grid((max_n_valid + SC_KEYS - 1) / SC_KEYS, sp_num_groups(g, row_count));
  auto q = (const __nv_bfloat16*)Q;
  auto k = (const __nv_bfloat16*)K;
  if (d == 128)
    sp_mass_kernel<128><<<grid, SC_KEYS, 0, st>>>(g, q, k, lse, Hq, Hkv, scale, local_window, local_bias, row_begin,
                                                  row_count, mass, ld);
  else
    sp_mass_kernel<64><<<grid, SC_KEYS, 0, st>>>(g, q, k, lse, Hq, Hkv, scale, local_window, local_bias, row_begin,
                                                 row_count, mass, ld);
  sp_count_launch();
  return cudaGetLastError();
}

cudaError_t sp_launch_attn(const SpGeom& g, const void* Q, const void* K, const void* V, const int32_t* idx, int k,
                           int Hq, int Hkv, int d, float scale, int local_window, float local_bias, int q_begin,
                           int q_count, void* O, float* lse, cudaStream_t st) {
  if (q_count <= 0) return cudaSuccess;
  const long long warps = (long long)q_count * Hkv;
  dim3 grid((unsigned)((warps + 7) / 8));
  const int G = Hq / Hkv;
  const bool sparse = idx != nullptr;
  cudaError_t e = d == 128
      ? launch_attn_d<128>(G, sparse, grid, st, g, Q, K, V, idx, k, Hkv, scale, local_window, local_bias, q_begin, q_count, O, lse)
      : launch_attn_d<64>(G, sparse, grid, st, g, Q, K, V, idx, k, Hkv, scale, local_window, local_bias, q_begin, q_count, O, lse);
  sp_count_launch();
  return e;
}
