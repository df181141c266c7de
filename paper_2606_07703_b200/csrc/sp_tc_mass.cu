// sp_tc_mass.cu -- oracle attention mass, pass 2, on tcgen05 / TMEM / TMA (Alg.1 step 3 :143):
//   P[t,s] = (1/Hq) sum_h exp(z[t,h,s] - lse[t,h]),  z = scale <q_{t,h}, k_{s,g(h)}> (+ local term),  s <= t
// and, for block-shared rows (b_sel in {32, 64, 128}), R_B(s) = max over the block's queries.
//
// Persistent, warp specialised.  A work item = 128 consecutive queries of one sequence (MMA M, TMEM lane =
// query, so lse[t,h] is a per-thread scalar) x 256 consecutive keys (MMA N); only lower-triangular items exist.
// For each of the Hq heads: TMA brings the head's Q tile (ring) and, once per KV group, the K tile (double
// buffered); S_h = Q_h K_g^T lands in one of two 256-column TMEM accumulators; two epilogue warpgroups (128
// key columns each) read it back, form exp2(sl2 * s - lse2) with packed fp32 FMAs + MUFU.EX2 and add into
// 128 register accumulators per thread, so the head sum never leaves the register file; after the last head
// the mean is written.  The exponential unit, not the tensor pipe, bounds this kernel (one ex2 per 2d flops).
// Items go to the CTAs round robin or in contiguous ranges (see ms_cta_range).
#include "sp_common.cuh"
#include "sp_tc.cuh"

using namespace sptc;

namespace {

constexpr int MS_MQ = 128;        // queries per item (MMA M)
constexpr int MS_NK = 256;        // keys per item (MMA N)
constexpr int MS_THREADS = 384;   // warps 0-3 / 4-7: epilogue of key columns 0-127 / 128-255; 8: TMA; 9: MMA; 10-11 idle
constexpr int MS_QSTAGES = 2;

__device__ __forceinline__ uint8_t* ms_align1024(uint8_t* p) {
  return reinterpret_cast<uint8_t*>((reinterpret_cast<uintptr_t>(p) + 1023) & ~(uintptr_t)1023);
}
__device__ __forceinline__ bool ms_elect_one() {
  uint32_t pred;
  asm volatile("{\n\t.reg .pred p;\n\telect.sync _|p, 0xffffffff;\n\tselp.u32 %0, 1, 0, p;\n\t}" : "=r"(pred));
  return pred != 0;
}
__device__ __forceinline__ uint64_t ms_pack(float lo, float hi) {
  uint64_t r;
  asm("mov.b64 %0, {%1, %2};" : "=l"(r) : "f"(lo), "f"(hi));
  return r;
}
__device__ __forceinline__ void ms_unpack(uint64_t v, float& lo, float& hi) {
  asm("mov.b64 {%0, %1}, %2;" : "=f"(lo), "=f"(hi) : "l"(v));
}
__device__ __forceinline__ uint64_t ms_fma2(uint64_t a, uint64_t b, uint64_t c) {
  uint64_t d;
  asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(d) : "l"(a), "l"(b), "l"(c));
  return d;
}
__device__ __forceinline__ uint64_t ms_add2(uint64_t a, uint64_t b) {
  uint64_t d;
  asm("add.rn.f32x2 %0, %1, %2;" : "=l"(d) : "l"(a), "l"(b));
  return d;
}
__device__ __forceinline__ float ms_ex2(float x) {
  float y;
  asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
  return y;
}
// exp2 of two fp32 values on the FMA / ALU pipes (the exponential unit bounds this kernel: one ex2 per 2 d flops, XU at
// 60-65 % of its peak against 10 % for the FMA pipe in profiles/r2_mass_pq.md): round-to-nearest split x = n + f
// (magic-number add), degree-4 minimax polynomial for 2^f on [-0.5, 0.5] (max relative error 2.7e-6 in fp32 Horner
// form, far inside the 1e-4 mass tolerance), exponent patched in with an integer add.  Inputs are clamped to >= -125.
#ifndef MS_POLY_EVERY
#define MS_POLY_EVERY 0  // one pair in MS_POLY_EVERY takes the polynomial path (0 = never: measured SLOWER here, 7.9 -> 9.3 ms at 1 in 2)
#endif
__device__ __forceinline__ void ms_ex2_poly2(uint64_t x2, float& p0, float& p1) {
  float x0, x1;
  ms_unpack(x2, x0, x1);
  x0 = fmaxf(x0, -125.f);
  x1 = fmaxf(x1, -125.f);
  const uint64_t xc = ms_pack(x0, x1);
  const uint64_t t = ms_add2(xc, ms_pack(12582912.f, 12582912.f));  // 1.5 * 2^23
  const uint64_t nf = ms_add2(t, ms_pack(-12582912.f, -12582912.f));
  const uint64_t f = ms_fma2(nf, ms_pack(-1.f, -1.f), xc);
  uint64_t q = ms_fma2(f, ms_pack(0.009570099413394928f, 0.009570099413394928f), ms_pack(0.05591785907745361f, 0.05591785907745361f));
  q = ms_fma2(q, f, ms_pack(0.240247443318367f, 0.240247443318367f));
  q = ms_fma2(q, f, ms_pack(0.6931217908859253f, 0.6931217908859253f));
  q = ms_fma2(q, f, ms_pack(0.9999992847442627f, 0.9999992847442627f));
  float q0, q1, t0, t1;
  ms_unpack(q, q0, q1);
  ms_unpack(t, t0, t1);
  p0 = __int_as_float(__float_as_int(q0) + (__float_as_int(t0) << 23));
  p1 = __int_as_float(__float_as_int(q1) + (__float_as_int(t1) << 23));
}

struct MsTile {
  int seq_start, n, q0;  // sequence start (packed), sequence length, first LOCAL query of the 128-query tile
  int row0;              // support row of the tile's first query
};

// linear query-tile index over the pack -> geometry
__device__ __forceinline__ MsTile ms_tile_info(const SpGeom& g, int qt) {
  const int b = g.b_sel;
  if (g.cu == nullptr) return MsTile{0, g.L, qt * MS_MQ, qt * MS_MQ / b};
  int t0 = 0, r0 = 0;
  for (int i = 0; i < g.batch; ++i) {
    const int s = g.cu[i], n = g.cu[i + 1] - s;
    const int nt = (n + MS_MQ - 1) / MS_MQ;
    if (qt < t0 + nt) return MsTile{s, n, (qt - t0) * MS_MQ, r0 + (qt - t0) * MS_MQ / b};
    t0 += nt;
    r0 += (n + b - 1) / b;
  }
  return MsTile{0, 0, 0, 0};
}
// key tiles of a query tile: every 256-key tile that starts at or below the tile's last query
__device__ __forceinline__ int ms_nkt(const MsTile& t) { return (min(t.q0 + MS_MQ, t.n) - 1) / MS_NK + 1; }

// Work distribution over the (query tile, key tile) units of the launch, numbered query tile by query tile.
//  * ROUND ROBIN (unit u -> CTA u mod P) for block-shared rows: the CTAs that run together then work on the same two or
//    three query tiles, whose Q (1 MB per query tile over the Hq heads, re-read by every key tile) stays in L2.  With
//    contiguous ranges the 148 CTAs walked 148 different query tiles at once -- 148 MB of Q -- and the all-rows launch
//    at 32K re-read Q from DRAM (21 GB per launch, L2 hit rate 33 %): 10.7 -> 7.9 ms; one KV group: 1.51 -> 1.31 ms.
//  * CONTIGUOUS equal ranges per CTA for per-query rows, whose launches are row panels of at most a few dozen query
//    tiles (Q fits L2 either way) and whose units each write 128 KB of P: a CTA that stays on one query tile writes
//    whole rows progressively, and measured 12 % faster than round robin there (profiles/r2_mass_pq.md).
struct MsRange {
  long long lo, hi;  // contiguous mode: this CTA's units [lo, hi)
  int rr;            // 1 = round robin
};
__device__ __forceinline__ MsRange ms_cta_range(const SpGeom& g, int qt_begin, int qt_count, int cta, int P, int rr) {
  MsRange r;
  r.rr = rr;
  r.lo = r.hi = 0;
  if (rr) return r;
  long long U = 0;
  for (int i = 0; i < qt_count; ++i) U += ms_nkt(ms_tile_info(g, qt_begin + i));
  r.lo = (U * cta + P - 1) / P;
  r.hi = (U * (cta + 1) + P - 1) / P;
  return r;
}
// key tiles [kt_lo, kt_hi) step kt_step of a query tile with nkt key tiles whose first unit is number B
__device__ __forceinline__ void ms_units(int nkt, long long B, const MsRange& r, int cta, int P, int& kt_lo, int& kt_hi,
                                         int& kt_step) {
  if (r.rr) {
    const int m = (int)(B % P);
    kt_lo = cta >= m ? cta - m : cta - m + P;
    kt_hi = nkt;
    kt_step = P;
  } else {
    const long long a = r.lo > B ? r.lo - B : 0, z = r.hi < B + nkt ? r.hi - B : nkt;
    kt_lo = (int)a;
    kt_hi = z > a ? (int)z : (int)a;
    kt_step = 1;
  }
}

// Max over the 32 lanes of a warp for 32 columns at once (reduce-scatter butterfly, 31 shuffles): on return lane l
// holds the maximum of column l.
__device__ __forceinline__ float ms_warp_colmax32(const float* x, int lane) {
  float y16[16], y8[8], y4[4], y2[2];
  const bool b16 = lane & 16, b8 = lane & 8, b4 = lane & 4, b2 = lane & 2, b1 = lane & 1;
#pragma unroll
  for (int i = 0; i < 16; ++i) {
    const float mine = b16 ? x[16 + i] : x[i], other = b16 ? x[i] : x[16 + i];
    y16[i] = fmaxf(mine, __shfl_xor_sync(0xffffffffu, other, 16));
  }
#pragma unroll
  for (int i = 0; i < 8; ++i) {
    const float mine = b8 ? y16[8 + i] : y16[i], other = b8 ? y16[i] : y16[8 + i];
    y8[i] = fmaxf(mine, __shfl_xor_sync(0xffffffffu, other, 8));
  }
#pragma unroll
  for (int i = 0; i < 4; ++i) {
    const float mine = b4 ? y8[4 + i] : y8[i], other = b4 ? y8[i] : y8[4 + i];
    y4[i] = fmaxf(mine, __shfl_xor_sync(0xffffffffu, other, 4));
  }
#pragma unroll
  for (int i = 0; i < 2; ++i) {
    const float mine = b2 ? y4[2 + i] : y4[i], other = b2 ? y4[i] : y4[2 + i];
    y2[i] = fmaxf(mine, __shfl_xor_sync(0xffffffffu, other, 2));
  }
  const float mine = b1 ? y2[1] : y2[0], other = b1 ? y2[0] : y2[1];
  return fmaxf(mine, __shfl_xor_sync(0xffffffffu, other, 1));
}

struct MsBarriers {
  uint64_t qfull[MS_QSTAGES], qempty[MS_QSTAGES];
  uint64_t kfull[2], kempty[2];
  uint64_t accfull[2], accempty[2];
};

template <int D>
__global__ void __launch_bounds__(MS_THREADS, 1)
sp_tc_mass_kernel(const __grid_constant__ CUtensorMap tmQ, const __grid_constant__ CUtensorMap tmK, SpGeom g,
                  const float* __restrict__ lse, int lse_stride, int Hq, int Hkv, float scale, int local_window,
                  float local_bias,
                  int row_begin, int row_count, int qt_begin, int qt_count, int round_robin, float* __restrict__ mass,
                  int64_t ld) {
  constexpr int KB = D / 64;
  constexpr uint32_t A_BYTES = MS_MQ * 128;  // per 64-wide K block: 128 queries
  constexpr uint32_t B_BYTES = MS_NK * 128;  // per 64-wide K block: 256 keys
  constexpr uint32_t Q_STAGE = KB * A_BYTES, K_BUF = KB * B_BYTES;
  extern __shared__ uint8_t smem_raw[];
  __shared__ MsBarriers bar;
  __shared__ uint32_t tmem_slot;
  __shared__ float ms_x[2][4][128];  // block-shared rows: per-warp column maxima of one warpgroup's 128 key columns
  uint8_t* smem = ms_align1024(smem_raw);
  uint8_t* sQ = smem;                         // [stage][kb] boxes of 128 rows x 128 B
  uint8_t* sK = smem + MS_QSTAGES * Q_STAGE;  // [buf][kb] boxes of 256 rows x 128 B
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int G = Hq / Hkv;
  const int b_sel = g.b_sel;

  if (threadIdx.x == 0) {
    for (int s = 0; s < MS_QSTAGES; ++s) {
      mbar_init(&bar.qfull[s], 1);
      mbar_init(&bar.qempty[s], 1);
    }
    for (int b = 0; b < 2; ++b) {
      mbar_init(&bar.kfull[b], 1);
      mbar_init(&bar.kempty[b], 1);
      mbar_init(&bar.accfull[b], 1);
      mbar_init(&bar.accempty[b], 256);
    }
    fence_barrier_init();
    tma_prefetch_desc(&tmQ);
    tma_prefetch_desc(&tmK);
  }
  if (warp == 9) tmem_alloc<512>(&tmem_slot);
  tc_fence_before_sync();
  __syncthreads();
  tc_fence_after_sync();
  const uint32_t tmem = tmem_slot;
  const MsRange rg = ms_cta_range(g, qt_begin, qt_count, blockIdx.x, gridDim.x, round_robin);

  if (warp >= 10) {
    asm volatile("setmaxnreg.dec.sync.aligned.u32 56;");
  } else if (warp == 8) {
    // =========================================== TMA producer ===========================================
    asm volatile("setmaxnreg.dec.sync.aligned.u32 56;");
    if (lane == 0) {
      uint32_t q_s = 0, q_ph = 0, k_n = 0;  // Q ring position; K tiles loaded so far
      long long B = 0;
      for (int i = 0; i < qt_count; ++i) {
        const MsTile ti = ms_tile_info(g, qt_begin + i);
        const int nkt = ms_nkt(ti);
        int kt_lo, kt_hi, kt_step;
        ms_units(nkt, B, rg, (int)blockIdx.x, (int)gridDim.x, kt_lo, kt_hi, kt_step);
        B += nkt;
        for (int kt = kt_lo; kt < kt_hi; kt += kt_step) {
          for (int h = 0; h < Hq; ++h) {
            if (h % G == 0) {
              const uint32_t kb_i = k_n & 1;
              mbar_wait(&bar.kempty[kb_i], ((k_n >> 1) & 1) ^ 1);
              mbar_expect_tx(&bar.kfull[kb_i], K_BUF);
#pragma unroll
              for (int kb = 0; kb < KB; ++kb)
                tma_load_2d(sK + kb_i * K_BUF + kb * B_BYTES, &tmK, &bar.kfull[kb_i], (h / G) * D + kb * 64,
                            ti.seq_start + kt * MS_NK);
              ++k_n;
            }
            mbar_wait(&bar.qempty[q_s], q_ph ^ 1);
            mbar_expect_tx(&bar.qfull[q_s], Q_STAGE);
#pragma unroll
            for (int kb = 0; kb < KB; ++kb)
              tma_load_2d(sQ + q_s * Q_STAGE + kb * A_BYTES, &tmQ, &bar.qfull[q_s], h * D + kb * 64,
                          ti.seq_start + ti.q0);
            if (++q_s == MS_QSTAGES) {
              q_s = 0;
              q_ph ^= 1;
            }
          }
        }
      }
    }
  } else if (warp == 9) {
    // =========================================== MMA issuer ===========================================
    asm volatile("setmaxnreg.dec.sync.aligned.u32 56;");
    const bool leader = ms_elect_one();
    constexpr uint32_t idesc = umma_idesc_bf16(MS_MQ, MS_NK, 0, 0);
    const uint64_t qdesc0 = umma_desc_sw128(smem_u32(sQ), 16, 1024);
    const uint64_t kdesc0 = umma_desc_sw128(smem_u32(sK), 16, 1024);
    uint32_t q_s = 0, q_ph = 0, k_n = 0, hc = 0;  // hc: heads issued so far (accumulator = hc & 1)
    long long B = 0;
    for (int i = 0; i < qt_count; ++i) {
      const MsTile ti = ms_tile_info(g, qt_begin + i);
      const int nkt = ms_nkt(ti);
      int kt_lo, kt_hi, kt_step;
      ms_units(nkt, B, rg, (int)blockIdx.x, (int)gridDim.x, kt_lo, kt_hi, kt_step);
      B += nkt;
      for (int kt = kt_lo; kt < kt_hi; kt += kt_step) {
        for (int h = 0; h < Hq; ++h, ++hc) {
          if (h % G == 0) {
            mbar_wait(&bar.kfull[k_n & 1], (k_n >> 1) & 1);
            ++k_n;
          }
          const uint32_t kb_i = (k_n - 1) & 1;
          mbar_wait(&bar.qfull[q_s], q_ph);
          const uint32_t ab = hc & 1, an = hc >> 1;
          if (an > 0) mbar_wait(&bar.accempty[ab], (an - 1) & 1);
          tc_fence_after_sync();
          if (leader) {
            const uint64_t qd = qdesc0 + (uint64_t)((q_s * Q_STAGE) >> 4);
            const uint64_t kd = kdesc0 + (uint64_t)((kb_i * K_BUF) >> 4);
#pragma unroll
            for (int k = 0; k < D / 16; ++k)
              umma_ss(tmem + ab * MS_NK, qd + (uint64_t)(((k / 4) * A_BYTES + (k % 4) * 32) >> 4),
                      kd + (uint64_t)(((k / 4) * B_BYTES + (k % 4) * 32) >> 4), idesc, k != 0);
            umma_commit(&bar.accfull[ab]);
            umma_commit(&bar.qempty[q_s]);
            if (h % G == G - 1) umma_commit(&bar.kempty[kb_i]);
          }
          if (++q_s == MS_QSTAGES) {
            q_s = 0;
            q_ph ^= 1;
          }
        }
      }
    }
    __syncwarp();
  } else {
    // =========================================== epilogue ===========================================
    asm volatile("setmaxnreg.inc.sync.aligned.u32 200;");
    const int e = warp >> 2;   // key columns [128 e, 128 e + 128)
    const int wq = warp & 3;   // TMEM lane quarter
    const int r = wq * 32 + lane;  // query row inside the tile
    const uint32_t tbase = tmem + ((uint32_t)(wq * 32) << 16) + e * 128;
    const int win = local_window > 0 ? local_window : 0;
    const float sl2 = scale * SP_LOG2E, lb2 = local_bias * SP_LOG2E;
    const uint64_t sl2_2 = ms_pack(sl2, sl2);
    const float inv_hq = 1.f / (float)Hq;
    const bool vec_ok = (ld & 3) == 0 && (reinterpret_cast<uintptr_t>(mass) & 15u) == 0;
    uint32_t hc = 0;
    long long B = 0;
    for (int i = 0; i < qt_count; ++i) {
      const MsTile ti = ms_tile_info(g, qt_begin + i);
      const int nkt = ms_nkt(ti);
      int kt_lo, kt_hi, kt_step;
      ms_units(nkt, B, rg, (int)blockIdx.x, (int)gridDim.x, kt_lo, kt_hi, kt_step);
      B += nkt;
      const int tl = ti.q0 + r;                      // local query of this thread
      const bool t_ok = tl < ti.n;
      const int tw0 = ti.q0 + wq * 32;               // warp-uniform: first / last valid query of the warp
      const int tw1 = min(tw0 + 31, ti.n - 1);
      const float* lse_row = lse + (size_t)(ti.seq_start + min(tl, ti.n - 1)) * lse_stride;
      for (int kt = kt_lo; kt < kt_hi; kt += kt_step) {
        const int sc0 = kt * MS_NK + e * 128;  // local key of this warpgroup's column 0
        uint64_t acc[64];
#pragma unroll
        for (int c = 0; c < 64; ++c) acc[c] = 0ull;
        float lse2_next = __ldg(lse_row) * SP_LOG2E;
        for (int h = 0; h < Hq; ++h, ++hc) {
          const float lse2 = lse2_next;
          if (h + 1 < Hq) lse2_next = __ldg(lse_row + h + 1) * SP_LOG2E;
          const uint32_t ab = hc & 1;
          mbar_wait(&bar.accfull[ab], (hc >> 1) & 1);
          tc_fence_after_sync();
          const uint64_t nl2 = ms_pack(-lse2, -lse2);
#pragma unroll
          for (int c0 = 0; c0 < 128; c0 += 32) {
            const int s_lo = sc0 + c0, s_hi = s_lo + 31;
            uint32_t v[32];
            const bool any = s_lo <= tw1;  // warp-uniform: some (t, s) of this chunk is causal
            if (any) {
              tmem_ld_x32(tbase + ab * MS_NK + c0, v);
              tmem_ld_wait();
            }
            if (c0 == 96) {  // the accumulator is in registers (or not needed): the next head's MMA may overwrite it
              tc_fence_before_sync();
              mbar_arrive(&bar.accempty[ab]);
            }
            if (!any) continue;
            if (s_hi <= tw0 - win && tw0 + 31 < ti.n) {
              // interior chunk: every pair causal, outside the local window, every query valid
#pragma unroll
              for (int j = 0; j < 32; j += 2) {
                const uint64_t x2 = ms_fma2(ms_pack(__uint_as_float(v[j]), __uint_as_float(v[j + 1])), sl2_2, nl2);
                float p0, p1;
                if (MS_POLY_EVERY > 0 && (j / 2) % MS_POLY_EVERY == MS_POLY_EVERY - 1) {
                  ms_ex2_poly2(x2, p0, p1);
                } else {
                  float x0, x1;
                  ms_unpack(x2, x0, x1);
                  p0 = ms_ex2(x0);
                  p1 = ms_ex2(x1);
                }
                acc[(c0 + j) >> 1] = ms_add2(acc[(c0 + j) >> 1], ms_pack(p0, p1));
              }
            } else {
#pragma unroll
              for (int j = 0; j < 32; j += 2) {
                float p[2];
#pragma unroll
                for (int u = 0; u < 2; ++u) {
                  const int s = s_lo + j + u;
                  float x = fmaf(__uint_as_float(v[j + u]), sl2, -lse2);
                  if (win > 0 && tl - s < win) x += lb2;
                  p[u] = (t_ok && s <= tl) ? ms_ex2(x) : 0.f;
                }
                acc[(c0 + j) >> 1] = ms_add2(acc[(c0 + j) >> 1], ms_pack(p[0], p[1]));
              }
            }
          }
        }
        if (b_sel == 1) {
          // ---- mean over heads, write this thread's row segment ----
          const int row = ti.seq_start + tl;  // b_sel == 1: support row == packed position
          if (t_ok && row >= row_begin && row < row_begin + row_count && sc0 <= tl) {
            float* dst = mass + (size_t)(row - row_begin) * ld + sc0;
            if (vec_ok && sc0 + 127 <= tl) {
#pragma unroll
              for (int c = 0; c < 64; c += 2) {
                float a0, a1, a2, a3;
                ms_unpack(acc[c], a0, a1);
                ms_unpack(acc[c + 1], a2, a3);
                reinterpret_cast<float4*>(dst)[c >> 1] = make_float4(a0 * inv_hq, a1 * inv_hq, a2 * inv_hq, a3 * inv_hq);
              }
            } else {
#pragma unroll
              for (int c = 0; c < 64; ++c) {
                float a0, a1;
                ms_unpack(acc[c], a0, a1);
                if (sc0 + 2 * c <= tl) dst[2 * c] = a0 * inv_hq;
                if (sc0 + 2 * c + 1 <= tl) dst[2 * c + 1] = a1 * inv_hq;
              }
            }
          }
        } else {
          // ---- block-shared rows: R_B(s) = max over the block's queries of the head mean.  Masked
          // (s > t) and out-of-sequence pairs contributed exactly 0, below every valid mass.  Lanes of a warp are 32
          // consecutive queries: reduce-scatter over the lanes, then over the warps of the block through shared memory.
          float red[4];
#pragma unroll
          for (int gq = 0; gq < 4; ++gq) {
            float x[32];
#pragma unroll
            for (int c = 0; c < 16; ++c) {
              float a0, a1;
              ms_unpack(acc[16 * gq + c], a0, a1);
              x[2 * c] = a0 * inv_hq;
              x[2 * c + 1] = a1 * inv_hq;
            }
            red[gq] = ms_warp_colmax32(x, lane);
          }
          const int wpb = b_sel >> 5;  // warps per block: 1, 2 or 4
          if (wpb > 1) {
            asm volatile("bar.sync %0, 128;" ::"r"(1 + e) : "memory");  // previous item's readers are done
#pragma unroll
            for (int gq = 0; gq < 4; ++gq) ms_x[e][wq][32 * gq + lane] = red[gq];
            asm volatile("bar.sync %0, 128;" ::"r"(1 + e) : "memory");
          }
          if ((wq & (wpb - 1)) == 0) {  // first warp of its block writes
            const int bq0 = ti.q0 + 32 * wq;
            if (bq0 < ti.n) {
              const int blk_last = min(bq0 + b_sel - 1, ti.n - 1);
              const int row = ti.row0 + (32 * wq) / b_sel;
              if (row >= row_begin && row < row_begin + row_count) {
#pragma unroll
                for (int gq = 0; gq < 4; ++gq) {
                  float v = red[gq];
                  for (int w = 1; w < wpb; ++w) v = fmaxf(v, ms_x[e][wq + w][32 * gq + lane]);
                  const int s = sc0 + 32 * gq + lane;
                  if (s <= blk_last) mass[(size_t)(row - row_begin) * ld + s] = v;
                }
              }
            }
          }
        }
      }
    }
  }
  tc_fence_before_sync();
  __syncthreads();
  if (warp == 9) tmem_dealloc<512>(tmem);
}

int ms_sm_count() { return sp_sm_count(); }

template <int D>
cudaError_t launch_mass_tc(const SpGeom& g, const void* Q, const void* K, const float* lse, int Hq, int Hkv, int grp,
                           int head, float scale, int lw, float lb, int row_begin, int row_count, int qt_begin, int qt_count,
                           long long items, float* mass, int64_t ld, cudaStream_t st) {
  CUtensorMap tmQ, tmK;
  cudaError_t e;
  // grp >= 0 (per-KV-group mass): the kernel sees the sub-problem of that group -- G heads over one KV
  // head -- through offset base pointers; the row pitches of Q, K and lse stay those of the full tensors.
  const int lse_stride = Hq, G = Hq / Hkv;
  const uint64_t q_pitch = (uint64_t)Hq * D, k_pitch = (uint64_t)Hkv * D;
  if (head >= 0) {  // per-HEAD mass (PAPER.md:100 S_{l,t,h}): one head over its KV head
    Q = (const __nv_bfloat16*)Q + (size_t)head * D;
    K = (const __nv_bfloat16*)K + (size_t)(head / G) * D;
    lse += (size_t)head;
    Hq = 1;
    Hkv = 1;
  } else if (grp >= 0) {
    Q = (const __nv_bfloat16*)Q + (size_t)grp * G * D;
    K = (const __nv_bfloat16*)K + (size_t)grp * D;
    lse += (size_t)grp * G;
    Hq = G;
    Hkv = 1;
  }
  if ((e = sp_make_tmap_bf16(&tmQ, Q, g.L, (uint64_t)Hq * D, q_pitch, MS_MQ)) != cudaSuccess) return e;
  if ((e = sp_make_tmap_bf16(&tmK, K, g.L, (uint64_t)Hkv * D, k_pitch, MS_NK)) != cudaSuccess) return e;
  constexpr size_t smem = (size_t)(D / 64) * (MS_QSTAGES * MS_MQ * 128 + 2 * MS_NK * 128) + 1024;
  static unsigned char attr_seen[SP_MAX_DEVICES];
  if (sp_first_use_on_device(attr_seen)) {
    e = cudaFuncSetAttribute(sp_tc_mass_kernel<D>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
  }
  long long grid = items < ms_sm_count() ? items : ms_sm_count();
  if (grid < 1) grid = 1;
  const int rr = g.b_sel > 1 ? 1 : 0;
  sp_tc_mass_kernel<D><<<(unsigned)grid, MS_THREADS, smem, st>>>(tmQ, tmK, g, lse, lse_stride, Hq, Hkv, scale, lw, lb,
                                                                row_begin,
                                                                row_count, qt_begin, qt_count, rr, mass, ld);
  sp_count_launch();
  return cudaGetLastError();
}

}  // namespace

bool sp_tc_mass_supported(int b_sel, int d) {
  return (b_sel == 1 || b_sel == 32 || b_sel == 64 || b_sel == 128) && (d == 64 || d == 128);
}

// cu_host: HOST copy of cu_seqlens (nullptr = one sequence).
cudaError_t sp_launch_mass_tc(const SpGeom& g, const int32_t* cu_host, const void* Q, const void* K, const float* lse,
                              int Hq, int Hkv, int d, float scale, int local_window, float local_bias, int row_begin,
                              int row_count, float* mass, int64_t ld, cudaStream_t st, int grp, int head) {
  if (row_count <= 0) return cudaSuccess;
  // 128-query tiles (per sequence) that intersect the support-row panel [row_begin, row_begin + row_count)
  const int b = g.b_sel;
  long long t0 = 0, r0 = 0, items = 0;
  long long qlo = -1, qhi = -1;
  for (int i = 0; i < g.batch; ++i) {
    const int n = cu_host ? cu_host[i + 1] - cu_host[i] : g.L;
    const long long nr = (n + b - 1) / b, nt = (n + MS_MQ - 1) / MS_MQ;
    const long long lo = row_begin > r0 ? row_begin : r0;
    const long long hi = ((long long)row_begin + row_count < r0 + nr ? (long long)row_begin + row_count : r0 + nr) - 1;
    if (lo <= hi) {
      const long long a = (lo - r0) * b / MS_MQ;
      long long last_q = (hi - r0 + 1) * b - 1;
      if (last_q > n - 1) last_q = n - 1;
      const long long z = last_q / MS_MQ;
      if (qlo < 0) qlo = t0 + a;
      qhi = t0 + z;
      for (long long j = a; j <= z; ++j) {
        const long long q_last = (j + 1) * MS_MQ < n ? (j + 1) * MS_MQ - 1 : n - 1;
        items += q_last / MS_NK + 1;
      }
    }
    t0 += nt;
    r0 += nr;
  }
  if (qlo < 0) return cudaSuccess;
  const int cnt = (int)(qhi - qlo + 1);
  return d == 128 ? launch_mass_tc<128>(g, Q, K, lse, Hq, Hkv, grp, head, scale, local_window, local_bias, row_begin,
                                        row_count, (int)qlo, cnt, items, mass, ld, st)
                  : launch_mass_tc<64>(g, Q, K, lse, Hq, Hkv, grp, head, scale, local_window, local_bias, row_begin,
                                       row_count, (int)qlo, cnt, items, mass, ld, st);
}
