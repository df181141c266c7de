// sp_tc_score.cu -- indexer score GEMM on tcgen05 / TMEM / TMA, persistent and warp specialised:
//   z[t,s] = idx_scale <q_idx[t], k_idx[s]> (+ local term), s <= t
//   R_B(s) = max_{t in B, t >= s} z[t,s] fused in the epilogue (b_sel > 1)
// The KEY index is the MMA M dimension (TMEM lane = key, column = query), so the max over a selection block's
// queries is a per-thread running max over columns and global writes are coalesced along s.
//
// One CTA per SM.  A query SUPER TILE (512 consecutive local positions of one sequence = four MMA N = 128
// parts) stays resident in shared memory while 128-key tiles stream through a TMA ring; each part owns one
// 128-column TMEM accumulator and one epilogue warpgroup (tcgen05.ld -> block max -> coalesced stores); a
// part's accumulator is reused only after the other three parts' MMAs, so the epilogues hide behind the
// tensor pipe.  Only lower-triangular (key tile, part) pairs are computed.  The
// linear sequence of key-tile steps (weight = active parts) is cut into equal contiguous ranges, one per
// CTA, so a CTA reloads Q only when its range crosses a super-tile boundary.
#include "sp_common.cuh"
#include "sp_tc.cuh"

using namespace sptc;

namespace {

constexpr int SC_NQ = 128;     // queries per part (MMA N); a super tile has SC_PARTS parts
constexpr int SC_PARTS = 4;
constexpr int SC_SUPER = 512;  // queries per resident super tile
constexpr int SC_KT = 128;     // keys per tile (MMA M)
constexpr int SC_THREADS = 576;  // warp 0: TMA, warp 1: MMA, warps 2-17: one epilogue warpgroup per part
constexpr int SC_MAX_STAGES = 4;

__device__ __forceinline__ uint8_t* sc_align1024(uint8_t* p) {
  return reinterpret_cast<uint8_t*>((reinterpret_cast<uintptr_t>(p) + 1023) & ~(uintptr_t)1023);
}
__device__ __forceinline__ bool sc_elect_one() {
  uint32_t pred;
  asm volatile("{\n\t.reg .pred p;\n\telect.sync _|p, 0xffffffff;\n\tselp.u32 %0, 1, 0, p;\n\t}" : "=r"(pred));
  return pred != 0;
}

struct ScSuper {
  int seq_start, n, q0;  // sequence start (packed), sequence length, first LOCAL query of the super tile
  int row0;              // support row of the super tile's first query
};

// linear super-tile index over the pack -> geometry
__device__ __forceinline__ ScSuper sc_super_info(const SpGeom& g, int st) {
  const int b = g.b_sel;
  if (g.cu == nullptr) return ScSuper{0, g.L, st * SC_SUPER, st * SC_SUPER / b};
  int t0 = 0, r0 = 0;
  for (int i = 0; i < g.batch; ++i) {
    const int s = g.cu[i], n = g.cu[i + 1] - s;
    const int nt = (n + SC_SUPER - 1) / SC_SUPER;
    if (st < t0 + nt) {
      const int q0 = (st - t0) * SC_SUPER;
      return ScSuper{s, n, q0, r0 + q0 / b};
    }
    t0 += nt;
    r0 += (n + b - 1) / b;
  }
  return ScSuper{0, 0, 0, 0};
}

// Key-tile steps of one super tile: kt in [0, nkt).  Part p (queries q0 + 128 p ...) needs key tile kt iff
// kt * 128 <= its last query: steps kt < jfull feed every existing part (weight np), step jfull + m (m >= 0)
// only parts p > m (weight np - 1 - m).
constexpr int SC_FIXED_W = 8;  // weight units (one unit = one 128 x 128 x d_idx MMA tile) charged per super tile
                               // for draining the pipeline and reloading the resident Q tile
struct ScSteps {
  int nkt, jfull, np;
  __device__ __forceinline__ int w_steps(int kt) const {  // MMA weight of steps [0, kt)
    if (kt <= jfull) return np * kt;
    const int m = kt - jfull;  // tail steps taken: weights np-1, np-2, ...
    return np * jfull + m * np - m * (m + 1) / 2;
  }
  __device__ __forceinline__ int w_before(int kt) const { return kt == 0 ? 0 : SC_FIXED_W + w_steps(kt); }
  __device__ __forceinline__ int weight() const { return w_before(nkt); }
  __device__ __forceinline__ int first_at(int x) const {  // smallest kt with w_before(kt) >= x
    if (x <= 0) return 0;
    const int y = x - SC_FIXED_W;
    if (y <= np) return 1;
    if (y <= np * jfull) return (y + np - 1) / np;
    int kt = jfull;
    while (kt < nkt && w_steps(kt) < y) ++kt;
    return kt;
  }
};

__device__ __forceinline__ ScSteps sc_steps(const ScSuper& su) {
  const int q_last = min(su.q0 + SC_SUPER, su.n) - 1;
  ScSteps s;
  s.nkt = q_last / SC_KT + 1;
  s.np = (q_last - su.q0) / SC_NQ + 1;
  s.jfull = min(su.q0 / SC_KT + 1, s.nkt);
  return s;
}

// is (kt, part p) a computed pair?  (identical in the MMA and the epilogue role)
__device__ __forceinline__ bool sc_part_active(const ScSuper& su, int kt, int p) {
  const int qp0 = su.q0 + p * SC_NQ;
  if (qp0 >= su.n) return false;
  const int qp_last = min(qp0 + SC_NQ, su.n) - 1;
  return kt * SC_KT <= qp_last;
}

// This CTA's contiguous range [lo, hi) of the global weight axis.
struct ScRange {
  long long lo, hi;
  int i_first;        // first super tile (relative to st_begin) that intersects [lo, hi)
  long long b_first;  // its weight base
};
__device__ __forceinline__ ScRange sc_cta_range(const SpGeom& g, int st_begin, int st_count, int cta, int P) {
  long long U = 0;
  for (int i = 0; i < st_count; ++i) U += sc_steps(sc_super_info(g, st_begin + i)).weight();
  ScRange r;
  r.lo = (U * cta + P - 1) / P;
  r.hi = (U * (cta + 1) + P - 1) / P;
  r.i_first = st_count;
  r.b_first = U;
  long long B = 0;
  for (int i = 0; i < st_count; ++i) {
    const long long W = sc_steps(sc_super_info(g, st_begin + i)).weight();
    if (B + W > r.lo) {
      r.i_first = i;
      r.b_first = B;
      break;
    }
    B += W;
  }
  return r;
}
// key-tile segment [kt_lo, kt_hi) of super tile with weight base B that falls into range r
__device__ __forceinline__ void sc_segment(const ScSteps& s, long long B, const ScRange& r, int& kt_lo, int& kt_hi) {
  const long long W = s.weight();
  if (r.hi <= B || r.lo >= B + W) {
    kt_lo = kt_hi = 0;
    return;
  }
  kt_lo = r.lo <= B ? 0 : s.first_at((int)(r.lo - B));
  kt_hi = r.hi >= B + W ? s.nkt : s.first_at((int)(r.hi - B));
  if (kt_hi > s.nkt) kt_hi = s.nkt;
  if (kt_lo > kt_hi) kt_lo = kt_hi;
}

struct ScBarriers {
  uint64_t qfull, qempty;
  uint64_t kfull[SC_MAX_STAGES], kempty[SC_MAX_STAGES];
  uint64_t accfull[SC_PARTS], accempty[SC_PARTS];
};

__device__ __forceinline__ float sc_max32(const uint32_t* v) {
  float m0 = fmaxf(__uint_as_float(v[0]), __uint_as_float(v[1]));
  float m1 = fmaxf(__uint_as_float(v[2]), __uint_as_float(v[3]));
  float m2 = fmaxf(__uint_as_float(v[4]), __uint_as_float(v[5]));
  float m3 = fmaxf(__uint_as_float(v[6]), __uint_as_float(v[7]));
#pragma unroll
  for (int j = 8; j < 32; j += 8) {
    m0 = fmaxf(m0, fmaxf(__uint_as_float(v[j]), __uint_as_float(v[j + 1])));
    m1 = fmaxf(m1, fmaxf(__uint_as_float(v[j + 2]), __uint_as_float(v[j + 3])));
    m2 = fmaxf(m2, fmaxf(__uint_as_float(v[j + 4]), __uint_as_float(v[j + 5])));
    m3 = fmaxf(m3, fmaxf(__uint_as_float(v[j + 6]), __uint_as_float(v[j + 7])));
  }
  return fmaxf(fmaxf(m0, m1), fmaxf(m2, m3));
}

// Epilogue of one (key tile, part): thread = key (TMEM lane), columns = the part's 128 queries.
// b == 1 writes every causal (t, s); b > 1 (a power of two, 2^lb) keeps the max of each selection block.
__device__ __forceinline__ void sc_epilogue(uint32_t trow, int warp_q, int lane, int s0, int hq0, int hrow0, int q_last,
                                            int b, int lb, float idx_scale, int local_window, float local_bias, bool relu,
                                            int row_begin, int row_count, float* __restrict__ scores, int64_t ld) {
  const int s = s0 + warp_q * 32 + lane;  // this thread's local key
  const int s_lo = s0 + warp_q * 32;      // warp-uniform: smallest / largest key of the warp
  const int s_hi = s_lo + 31;
  if (b == 1) {
    for (int c0 = 0; c0 < SC_NQ; c0 += 32) {
      const int t0 = hq0 + c0;  // local query of column c0
      if (t0 > q_last) break;
      const int t1 = min(t0 + 31, q_last);
      if (s_lo > t1) continue;  // warp-uniform: no causal pair in this chunk
      uint32_t v[32];
      tmem_ld_x32(trow + c0, v);
      tmem_ld_wait();
      // interior chunk (the bulk of a per-query panel): all 32 x 32 pairs are causal, inside the sequence, inside the row
      // panel and outside the local window -> multiply, store, step the pointer: no per-element tests (the kernel is
      // bound by the instructions of this loop, not by the 2 GB it writes: ncu has ALU at 62 %, DRAM at 0.4 of the
      // write rate a plain fill reaches)
      const int rowc = hrow0 + c0;
      if (s_hi <= t0 && t0 + 31 <= q_last && rowc >= row_begin && rowc + 31 < row_begin + row_count &&
          (local_window <= 0 || t0 - s_hi >= local_window)) {
        float* dst = scores + (size_t)(rowc - row_begin) * ld + s;
        if (relu) {
#pragma unroll
          for (int j = 0; j < 32; ++j) {
            *dst = fmaxf(__uint_as_float(v[j]) * idx_scale, 0.f);
            dst += ld;
          }
        } else {
#pragma unroll
          for (int j = 0; j < 32; ++j) {
            *dst = __uint_as_float(v[j]) * idx_scale;
            dst += ld;
          }
        }
        continue;
      }
#pragma unroll
      for (int j = 0; j < 32; ++j) {
        const int t = t0 + j;
        const int row = hrow0 + c0 + j;
        if (t <= q_last && s <= t && row >= row_begin && row < row_begin + row_count) {
          float z = __uint_as_float(v[j]) * idx_scale;
          if (local_window > 0 && t - s < local_window) z += local_bias;
          if (relu) z = fmaxf(z, 0.f);  // PAPER.md:274 (A26): ReLU on the final logit
          scores[(size_t)(row - row_begin) * ld + s] = z;
        }
      }
    }
    return;
  }
  const bool fast_ok = idx_scale > 0.f;  // max commutes with a positive scale
  const int nblk = SC_NQ >> lb;
  if (fast_ok && hq0 + SC_NQ - 1 <= q_last && hq0 - s_hi >= (local_window > 0 ? local_window : 0)) {
    // interior (key warp, part): all 32 x 128 pairs are causal, inside the sequence and outside the local
    // window -> no per-element work, no inner branches: chunk maxima, then one store per selection block
    float cm[4];
#pragma unroll
    for (int hh = 0; hh < 2; ++hh) {
      uint32_t v0[32], v1[32];
      tmem_ld_x32(trow + hh * 64, v0);
      tmem_ld_x32(trow + hh * 64 + 32, v1);
      tmem_ld_wait();
      cm[2 * hh] = sc_max32(v0);
      cm[2 * hh + 1] = sc_max32(v1);
    }
    if (lb == 6) {
      cm[0] = fmaxf(cm[0], cm[1]);
      cm[1] = fmaxf(cm[2], cm[3]);
    } else if (lb == 7) {
      cm[0] = fmaxf(fmaxf(cm[0], cm[1]), fmaxf(cm[2], cm[3]));
    }
#pragma unroll
    for (int blk = 0; blk < 4; ++blk) {
      const int row = hrow0 + blk;
      if (blk < nblk && row >= row_begin && row < row_begin + row_count)
        scores[(size_t)(row - row_begin) * ld + s] = relu ? fmaxf(cm[blk] * idx_scale, 0.f) : cm[blk] * idx_scale;
    }
    return;
  }
  for (int blk = 0; blk < nblk; ++blk) {
    const int bq0 = hq0 + (blk << lb);  // first local query of the selection block
    if (bq0 > q_last) break;
    const int blk_last = min(bq0 + b - 1, q_last);  // n_valid - 1 of the block
    if (s_lo > blk_last) continue;                  // warp-uniform: every key of the warp is above the block
    float best = -INFINITY;
    for (int c0 = blk << lb; c0 < ((blk + 1) << lb); c0 += 32) {
      const int t0 = hq0 + c0;
      if (t0 > q_last) break;
      const int t1 = min(t0 + 31, q_last);
      if (s_lo > t1) continue;
      uint32_t v[32];
      tmem_ld_x32(trow + c0, v);
      tmem_ld_wait();
      if (fast_ok && s_hi <= t0 && t0 + 31 <= q_last && (local_window == 0 || t0 - s_hi >= local_window)) {
        // interior chunk: every pair is causal and outside the local window
        float m0 = fmaxf(__uint_as_float(v[0]), __uint_as_float(v[1]));
        float m1 = fmaxf(__uint_as_float(v[2]), __uint_as_float(v[3]));
        float m2 = fmaxf(__uint_as_float(v[4]), __uint_as_float(v[5]));
        float m3 = fmaxf(__uint_as_float(v[6]), __uint_as_float(v[7]));
#pragma unroll
        for (int j = 8; j < 32; j += 8) {
          m0 = fmaxf(m0, fmaxf(__uint_as_float(v[j]), __uint_as_float(v[j + 1])));
          m1 = fmaxf(m1, fmaxf(__uint_as_float(v[j + 2]), __uint_as_float(v[j + 3])));
          m2 = fmaxf(m2, fmaxf(__uint_as_float(v[j + 4]), __uint_as_float(v[j + 5])));
          m3 = fmaxf(m3, fmaxf(__uint_as_float(v[j + 6]), __uint_as_float(v[j + 7])));
        }
        best = fmaxf(best, fmaxf(fmaxf(m0, m1), fmaxf(m2, m3)) * idx_scale);
      } else {
        // diagonal / local-window chunk: branch-free per element, four independent max chains
        const int d0 = t0 - s;          // t - s of column j is d0 + j
        const int jmax = q_last - t0;   // warp-uniform: columns j > jmax lie beyond the sequence end
        float m4[4] = {-INFINITY, -INFINITY, -INFINITY, -INFINITY};
#pragma unroll
        for (int j = 0; j < 32; ++j) {
          float z = __uint_as_float(v[j]) * idx_scale;
          if (local_window > 0) z = (d0 + j < local_window) ? z + local_bias : z;
          z = (d0 + j >= 0 && j <= jmax) ? z : -INFINITY;
          m4[j & 3] = fmaxf(m4[j & 3], z);
        }
        best = fmaxf(best, fmaxf(fmaxf(m4[0], m4[1]), fmaxf(m4[2], m4[3])));
      }
    }
    const int row = hrow0 + blk;
    if (relu) best = fmaxf(best, 0.f);  // max and ReLU commute; a block row always has a valid (t >= s) pair here
    if (row >= row_begin && row < row_begin + row_count && s <= blk_last)
      scores[(size_t)(row - row_begin) * ld + s] = best;
  }
}

template <int DI>
__global__ void __launch_bounds__(SC_THREADS, 1)
sp_tc_score_kernel(const __grid_constant__ CUtensorMap tmQ, const __grid_constant__ CUtensorMap tmK, SpGeom g,
                   float idx_scale, int local_window, float local_bias, int relu, int row_begin, int row_count,
                   int st_begin, int st_count, int n_stages, float* __restrict__ scores, int64_t ld) {
  constexpr int KB = DI / 64;
  constexpr uint32_t A_BYTES = SC_KT * 128;  // per 64-wide K block: 128 keys
  constexpr uint32_t B_BYTES = SC_NQ * 128;  // per 64-wide K block: the 128 queries of one part
  constexpr uint32_t K_STAGE = KB * A_BYTES;
  extern __shared__ uint8_t smem_raw[];
  __shared__ ScBarriers bar;
  __shared__ uint32_t tmem_slot;
  uint8_t* smem = sc_align1024(smem_raw);
  uint8_t* sQ = smem;                             // [part][kb] boxes of 128 rows x 128 B
  uint8_t* sK = smem + SC_PARTS * KB * B_BYTES;   // [stage][kb] boxes of 128 rows x 128 B
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int NS = n_stages;
  const int b = g.b_sel;

  if (threadIdx.x == 0) {
    mbar_init(&bar.qfull, 1);
    mbar_init(&bar.qempty, 1);
    for (int s = 0; s < SC_MAX_STAGES; ++s) {
      mbar_init(&bar.kfull[s], 1);
      mbar_init(&bar.kempty[s], 1);
    }
    for (int h = 0; h < SC_PARTS; ++h) {
      mbar_init(&bar.accfull[h], 1);
      mbar_init(&bar.accempty[h], 128);
    }
    fence_barrier_init();
    tma_prefetch_desc(&tmQ);
    tma_prefetch_desc(&tmK);
  }
  if (warp == 1) tmem_alloc<512>(&tmem_slot);
  tc_fence_before_sync();
  __syncthreads();
  tc_fence_after_sync();
  const uint32_t tmem = tmem_slot;
  const ScRange rg = sc_cta_range(g, st_begin, st_count, blockIdx.x, gridDim.x);

  if (warp == 0) {
    // =========================================== TMA producer ===========================================
    if (lane == 0) {
      uint32_t k_s = 0, k_ph = 0, n_seg = 0;
      long long B = rg.b_first;
      for (int i = rg.i_first; i < st_count && B < rg.hi; ++i) {
        const ScSuper su = sc_super_info(g, st_begin + i);
        const ScSteps ss = sc_steps(su);
        int kt_lo, kt_hi;
        sc_segment(ss, B, rg, kt_lo, kt_hi);
        B += ss.weight();
        if (kt_lo >= kt_hi) continue;
        if (n_seg > 0) mbar_wait(&bar.qempty, (n_seg - 1) & 1);
        const int nh = ss.np;
        mbar_expect_tx(&bar.qfull, nh * KB * B_BYTES);
        for (int h = 0; h < nh; ++h)
#pragma unroll
          for (int kb = 0; kb < KB; ++kb)
            tma_load_2d(sQ + (h * KB + kb) * B_BYTES, &tmQ, &bar.qfull, kb * 64,
                        su.seq_start + su.q0 + h * SC_NQ - g.q_off);  // chunked prefill: q_idx holds the chunk's rows only
                                                                       // (rows before it: negative coordinate -> zero fill)
        ++n_seg;
        for (int kt = kt_lo; kt < kt_hi; ++kt) {
          mbar_wait(&bar.kempty[k_s], k_ph ^ 1);  // first pass over the ring: parity 1 of a fresh barrier passes
          mbar_expect_tx(&bar.kfull[k_s], K_STAGE);
          if (g.bt == nullptr) {
#pragma unroll
            for (int kb = 0; kb < KB; ++kb)
              tma_load_2d(sK + k_s * K_STAGE + kb * A_BYTES, &tmK, &bar.kfull[k_s], kb * 64, su.seq_start + kt * SC_KT);
          } else {
            // paged indexer keys: the 128-key tile is one box inside a page (pages >= 128 tokens) or 128 / page_size
            // boxes of one page each, landing at their row offsets of the same SWIZZLE_128B image
            const int ps = 1 << g.page_shift;
            const int rows = ps < SC_KT ? ps : SC_KT;
            for (int r0 = 0; r0 < SC_KT; r0 += rows) {
              const int y = (int)sp_kv_row(g, su.seq_start + kt * SC_KT + r0);
#pragma unroll
              for (int kb = 0; kb < KB; ++kb)
                tma_load_2d(sK + k_s * K_STAGE + kb * A_BYTES + r0 * 128, &tmK, &bar.kfull[k_s], kb * 64, y);
            }
          }
          if (++k_s == (uint32_t)NS) {
            k_s = 0;
            k_ph ^= 1;
          }
        }
      }
    }
  } else if (warp == 1) {
    // =========================================== MMA issuer ===========================================
    const bool leader = sc_elect_one();
    constexpr uint32_t idesc = umma_idesc_bf16(SC_KT, SC_NQ, 0, 0);
    const uint64_t qdesc0 = umma_desc_sw128(smem_u32(sQ), 16, 1024);
    const uint64_t kdesc0 = umma_desc_sw128(smem_u32(sK), 16, 1024);
    uint32_t k_s = 0, k_ph = 0, n_seg = 0;
    uint32_t use[SC_PARTS] = {0, 0, 0, 0};  // accumulator uses so far
    long long B = rg.b_first;
    for (int i = rg.i_first; i < st_count && B < rg.hi; ++i) {
      const ScSuper su = sc_super_info(g, st_begin + i);
      const ScSteps ss = sc_steps(su);
      int kt_lo, kt_hi;
      sc_segment(ss, B, rg, kt_lo, kt_hi);
      B += ss.weight();
      if (kt_lo >= kt_hi) continue;
      mbar_wait(&bar.qfull, n_seg & 1);
      tc_fence_after_sync();
      for (int kt = kt_lo; kt < kt_hi; ++kt) {
        mbar_wait(&bar.kfull[k_s], k_ph);
        tc_fence_after_sync();
        const uint64_t kd = kdesc0 + (uint64_t)((k_s * K_STAGE) >> 4);
#pragma unroll
        for (int h = 0; h < SC_PARTS; ++h) {
          if (!sc_part_active(su, kt, h)) continue;
          if (use[h] > 0) {
            mbar_wait(&bar.accempty[h], (use[h] - 1) & 1);
            tc_fence_after_sync();
          }
          if (leader) {
#pragma unroll
            for (int k = 0; k < DI / 16; ++k)
              umma_ss(tmem + h * SC_NQ, kd + (uint64_t)(((k / 4) * A_BYTES + (k % 4) * 32) >> 4),
                      qdesc0 + (uint64_t)(((h * KB + k / 4) * B_BYTES + (k % 4) * 32) >> 4), idesc, k != 0);
            umma_commit(&bar.accfull[h]);
          }
          ++use[h];
        }
        if (leader) umma_commit(&bar.kempty[k_s]);
        if (++k_s == (uint32_t)NS) {
          k_s = 0;
          k_ph ^= 1;
        }
      }
      if (leader) umma_commit(&bar.qempty);
      ++n_seg;
    }
    __syncwarp();
  } else {
    // =========================================== epilogue ===========================================
    // one epilogue warpgroup per part (warps 2-5, 6-9, 10-13, 14-17).  A part's accumulator is needed again
    // only after the MMAs of the other three parts, so each epilogue has ~3x its MMA time of slack.
    const int p = (warp - 2) >> 2;
    const int wq = warp & 3;  // TMEM lane quarter this warp may access
    const uint32_t trow = tmem + ((uint32_t)(wq * 32) << 16) + p * SC_NQ;
    const int lb = 31 - __clz(b);
    uint32_t use = 0;
    long long B = rg.b_first;
    for (int i = rg.i_first; i < st_count && B < rg.hi; ++i) {
      const ScSuper su = sc_super_info(g, st_begin + i);
      const ScSteps ss = sc_steps(su);
      int kt_lo, kt_hi;
      sc_segment(ss, B, rg, kt_lo, kt_hi);
      B += ss.weight();
      const int pq0 = su.q0 + p * SC_NQ;
      const int q_last = min(pq0 + SC_NQ, su.n) - 1;
      const int prow0 = su.row0 + ((p * SC_NQ) >> lb);
      for (int kt = kt_lo; kt < kt_hi; ++kt) {
        if (!sc_part_active(su, kt, p)) continue;
        mbar_wait(&bar.accfull[p], use & 1);
        tc_fence_after_sync();
        sc_epilogue(trow, wq, lane, kt * SC_KT, pq0, prow0, q_last, b, lb, idx_scale, local_window, local_bias,
                    relu != 0, row_begin, row_count, scores, ld);
        tc_fence_before_sync();
        mbar_arrive(&bar.accempty[p]);
        ++use;
      }
    }
  }
  tc_fence_before_sync();
  __syncthreads();
  if (warp == 1) tmem_dealloc<512>(tmem);
}

}  // namespace

// ---------------------------------------------------------------------------------------------------
// launchers
// ---------------------------------------------------------------------------------------------------
bool sp_tc_scores_supported(int b_sel) { return b_sel == 1 || b_sel == 32 || b_sel == 64 || b_sel == 128; }

static int sc_sm_count() { return sp_sm_count(); }

template <int DI>
static cudaError_t launch_scores_tc(const SpGeom& g, const void* q_idx, const void* k_idx, float idx_scale, int lw,
                                    float lb, int relu, int row_begin, int row_count, int st_begin, int st_count, long long units,
                                    float* scores, int64_t ld, cudaStream_t st) {
  CUtensorMap tmQ, tmK;
  cudaError_t e;
  if ((e = sp_make_tmap_bf16(&tmQ, q_idx, g.q_rows ? g.q_rows : g.L, DI, DI, SC_NQ)) != cudaSuccess) return e;
  if (g.bt == nullptr) {
    e = sp_make_tmap_bf16(&tmK, k_idx, g.L, DI, DI, SC_KT);
  } else {  // k_idx = the page pool [n_pages * page_size, DI]; box = one page, at most one 128-key tile
    const uint64_t ps = 1ull << g.page_shift;
    e = sp_make_tmap_bf16(&tmK, k_idx, (uint64_t)g.kv_rows, DI, DI, (uint32_t)(ps < SC_KT ? ps : SC_KT));
  }
  if (e != cudaSuccess) return e;
  constexpr int stages = DI == 128 ? 3 : 4;
  constexpr size_t smem = (size_t)(DI / 64) * (SC_PARTS * SC_NQ * 128 + stages * SC_KT * 128) + 1024;
  static unsigned char attr_seen[SP_MAX_DEVICES];
  if (sp_first_use_on_device(attr_seen)) {
    e = cudaFuncSetAttribute(sp_tc_score_kernel<DI>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
  }
  long long grid = units < sc_sm_count() ? units : sc_sm_count();
  if (grid < 1) grid = 1;
  sp_tc_score_kernel<DI><<<(unsigned)grid, SC_THREADS, smem, st>>>(tmQ, tmK, g, idx_scale, lw, lb, relu, row_begin, row_count,
                                                                  st_begin, st_count, stages, scores, ld);
  sp_count_launch();
  return cudaGetLastError();
}

// cu_host: HOST copy of cu_seqlens (nullptr = one sequence).
cudaError_t sp_launch_indexer_scores_tc(const SpGeom& g, const int32_t* cu_host, const void* q_idx, const void* k_idx,
                                        int d_idx, float idx_scale, int local_window, float local_bias, int relu,
                                        int row_begin, int row_count, int max_n_valid, float* scores, int64_t ld,
                                        cudaStream_t st) {
  (void)max_n_valid;
  if (row_count <= 0) return cudaSuccess;
  // query super tiles (512 local positions of one sequence) that intersect the row panel, and their step count
  const int b = g.b_sel;
  long long t0 = 0, r0 = 0;
  long long qlo = -1, qhi = -1, units = 0;
  for (int i = 0; i < g.batch; ++i) {
    const int n = cu_host ? cu_host[i + 1] - cu_host[i] : g.L;
    const long long nr = (n + b - 1) / b, nt = (n + SC_SUPER - 1) / SC_SUPER;
    const long long lo = row_begin > r0 ? row_begin : r0;
    const long long hi = ((long long)row_begin + row_count < r0 + nr ? (long long)row_begin + row_count : r0 + nr) - 1;
    if (lo <= hi) {
      const long long a = (lo - r0) * b / SC_SUPER;
      long long last_q = (hi - r0 + 1) * b - 1;
      if (last_q > n - 1) last_q = n - 1;
      const long long z = last_q / SC_SUPER;
      if (qlo < 0) qlo = t0 + a;
      qhi = t0 + z;
    }
    t0 += nt;
    r0 += nr;
  }
  if (qlo < 0) return cudaSuccess;
  // super tiles between two intersecting sequences all intersect (a panel is a contiguous row range); count steps
  {
    long long tt = 0;
    for (int i = 0; i < g.batch; ++i) {
      const int n = cu_host ? cu_host[i + 1] - cu_host[i] : g.L;
      const long long nt = (n + SC_SUPER - 1) / SC_SUPER;
      for (long long j = 0; j < nt; ++j) {
        const long long stx = tt + j;
        if (stx < qlo || stx > qhi) continue;
        long long q_last = (j + 1) * SC_SUPER < n ? (j + 1) * SC_SUPER - 1 : n - 1;
        units += q_last / SC_KT + 1;
      }
      tt += nt;
    }
  }
  const int cnt = (int)(qhi - qlo + 1);
  return d_idx == 128 ? launch_scores_tc<128>(g, q_idx, k_idx, idx_scale, local_window, local_bias, relu, row_begin, row_count,
                                              (int)qlo, cnt, units, scores, ld, st)
                      : launch_scores_tc<64>(g, q_idx, k_idx, idx_scale, local_window, local_bias, relu, row_begin, row_count,
                                             (int)qlo, cnt, units, scores, ld, st);
}
