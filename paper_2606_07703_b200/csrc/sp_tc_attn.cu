// sp_tc_attn.cu -- GQA attention with online softmax on tcgen05 / TMEM (PAPER.md:94 dense, :107 + :156 sparse).
//
// PERSISTENT kernel, one CTA per SM.  A work item = one chunk of up to 256/G consecutive queries of ONE support
// row x one KV head: the G query heads of the KV group are stacked along the MMA M dimension (row R = query * G +
// head), so one gathered K/V tile is shared by 256 rows (two M = 128 tiles).  Key tiles hold 64 keys.
//   SPARSE: the keys are the support row's index list, staged once per item in shared memory; K/V rows are
//           gathered with cp.async 16-byte vectors written in the SWIZZLE_128B image TMA would have produced;
//   DENSE : the keys are the causal prefix of the sequence (same loader, consecutive rows), heavy chunks first.
// Warp roles: warps 0-3 / 4-7 softmax of M tile 0 / 1 (thread = row = TMEM lane), warps 9-12 index staging +
// Q/K/V loaders, warp 8 / warp 13 issue ALL MMAs of M tile 0 / 1 (PV(j) then S(j+2) from one elected lane, so the
// tensor pipe orders them), warps 14, 15 idle.  Rings (K, V stages; S double buffered per M tile in TMEM) run ACROSS
// items, so the loaders prefetch the next item's index list, K and V while the current one finishes.
// Per key tile and M tile:
//   S = Q K^T (tcgen05.mma SS, fp32 in TMEM) -> tcgen05.ld -> scale, mask by KEY POSITION VALUE, online softmax
//   with lazy rescaling of the TMEM-resident O accumulator -> P (bf16x2) written back over S with tcgen05.st ->
//   O += P V (tcgen05.mma with A = P from TMEM, B = V read MN-major from the row-major tile).
// Softmax arithmetic is SPECULATIVE: the exponentials of a tile are taken against the running max as it stood before
// the tile; unflagged tiles never reduce their max at all -- a logit more than 2^8 above the running max shows in the
// tile's SUM of exponentials (all p >= 0), and only then is the max taken from a fresh read of S, the accumulator
// rescaled and the tile redone (the softmax warps are issue-bound at ~2 busy warps per scheduler: instructions per
// element are what the kernel's time is made of, profiles/r2_attn.md).
// Only tiles that can contain a masked or locally-biased element take the per-element path (flags computed by
// the loaders while staging the index list).
//   MASKED: per-query supports (b_sel = 1) as the DENSE tile loop with a membership mask: a one-hot query selector and a
//           mask tile the loaders expand from a [L/32, L] bitmap are multiplied on the tensor core into S (two extra K
//           steps per tile), so the softmax warps run their unmasked path; chosen by sp_api.cu when the causal pairs are
//           few enough against the kept ones (k a sizeable part of the prefix).  Also holds the bitmap builder and the
//           fixed scratch array of the no-allocation entry point.
// Barrier rule (profiles/r2_final.md): a parity wait is only safe for a warp whose arrival the barrier's next phase
// needs; the one wait that was not (the loaders' wait for the Q buffer) is followed by a named barrier.
#include "sp_common.cuh"
#include "sp_tc.cuh"

using namespace sptc;

namespace {

constexpr int AT_KT = 64;          // keys per tile
#ifndef AT_MAX_STAGES_DEF
#define AT_MAX_STAGES_DEF 6
#endif
#ifndef AT_STORE_V8
#define AT_STORE_V8 1  // O rows leave in 32-byte stores (one whole sector per lane and instruction: half the LSU wavefronts)
#endif
constexpr int AT_MAX_STAGES = AT_MAX_STAGES_DEF;   // K/V ring depth is chosen at launch from the shared-memory budget
constexpr int AT_THREADS = 512;    // 8 softmax warps + 4 loader warps + 4 MMA-issuing warps (whole warpgroups for setmaxnreg)
constexpr int AT_LOAD_WARPS = 4;
constexpr int AT_MMA_WARP = 8;
constexpr int AT_LOAD_WARP0 = 9;
// (Measured and not kept: MMA issuers on warps 8, 9 and the loaders on warps 10, 11, 14, 15, i.e. two loaders on each of
// schedulers 2 and 3 instead of issuer + loader on schedulers 0 and 1: +2.5 % slower.)
constexpr uint32_t AT_AX_BYTES = 128 * 128;  // membership-masked mode: query selector tile
constexpr uint32_t AT_BX_BYTES = 64 * 128;   // ... and one mask tile per ring stage
constexpr float AT_NO_KEY = -1e30f;          // a raw logit below this is a masked one (the mask adds -2^127)
constexpr float AT_RESCALE_THRESHOLD = 8.0f;  // log2 units: O is rescaled only when the row max grew by > 2^8

__device__ __forceinline__ void cp_async_arrive_noinc(uint64_t* bar) {
  asm volatile("cp.async.mbarrier.arrive.noinc.shared::cta.b64 [%0];" ::"r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ bool elect_one() {
  uint32_t pred;
  asm volatile("{\n\t.reg .pred p;\n\telect.sync _|p, 0xffffffff;\n\tselp.u32 %0, 1, 0, p;\n\t}" : "=r"(pred));
  return pred != 0;
}
__device__ __forceinline__ void mbar_wait_addr(uint32_t addr, uint32_t parity) {
  uint32_t ok;
  do {
    asm volatile(
        "{\n\t.reg .pred p;\n\t"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\t"
        "selp.u32 %0, 1, 0, p;\n\t}"
        : "=r"(ok)
        : "r"(addr), "r"(parity)
        : "memory");
  } while (!ok);
}
__device__ __forceinline__ void mbar_arrive_addr(uint32_t addr) {
  asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(addr) : "memory");
}
__device__ __forceinline__ void loader_bar_sync() { asm volatile("bar.sync 1, 128;" ::: "memory"); }

// D[tmem] (+)= A[tmem] * B[smem]: A = 128 lanes x (K/2) 32-bit columns of packed bf16 pairs (K-major).
__device__ __forceinline__ void umma_ts(uint32_t d_tmem, uint32_t a_tmem, uint64_t b_desc, uint32_t idesc,
                                        uint32_t accumulate) {
  asm volatile(
      "{\n\t.reg .pred p;\n\t"
      "setp.ne.b32 p, %4, 0;\n\t"
      "tcgen05.mma.cta_group::1.kind::f16 [%0], [%1], %2, %3, p;\n\t}"
      ::"r"(d_tmem), "r"(a_tmem), "l"(b_desc), "r"(idesc), "r"(accumulate)
      : "memory");
}

// packed fp32 pairs (sm_100 FFMA2 / FADD2)
__device__ __forceinline__ uint64_t f2_pack(float lo, float hi) {
  uint64_t r;
  asm("mov.b64 %0, {%1, %2};" : "=l"(r) : "f"(lo), "f"(hi));
  return r;
}
__device__ __forceinline__ void f2_unpack(uint64_t v, float& lo, float& hi) {
  asm("mov.b64 {%0, %1}, %2;" : "=f"(lo), "=f"(hi) : "l"(v));
}
__device__ __forceinline__ uint64_t f2_fma(uint64_t a, uint64_t b, uint64_t c) {
  uint64_t d;
  asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(d) : "l"(a), "l"(b), "l"(c));
  return d;
}
__device__ __forceinline__ uint64_t f2_add(uint64_t a, uint64_t b) {
  uint64_t d;
  asm("add.rn.f32x2 %0, %1, %2;" : "=l"(d) : "l"(a), "l"(b));
  return d;
}
__device__ __forceinline__ float ex2_approx(float x) {
  float y;
  asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
  return y;
}
// exp2 of two fp32 values on the FMA / ALU pipes: round-to-nearest split x = n + f (magic-number add), degree-4
// minimax polynomial for 2^f on [-0.5, 0.5] (max relative error 2.7e-6 in fp32 Horner form), exponent patched
// in with an integer add.  Inputs are clamped to >= -125 (result ~2^-125, i.e. 0 for every use here).
#ifndef AT_POLY_EVERY_LSE
#define AT_POLY_EVERY_LSE 4  // the same for LSE-only launches (no P, no PV: the exponential unit alone paces them)
#endif
#ifndef AT_POLY_EVERY
#define AT_POLY_EVERY 4  // one pair in AT_POLY_EVERY takes the polynomial path (0 = never)
#endif
// fast-path overflow guard: a tile whose exponentials (taken against the running max as it stood before the tile) sum
// to more than this is redone after the running max has been moved; every p of an accepted tile is therefore <= 2^8,
// the bound the lazy-rescale threshold gives
#define AT_SUM_LIMIT 256.0f
__device__ __forceinline__ void ex2_poly2(uint64_t x2, float& p0, float& p1) {
  float x0, x1;
  f2_unpack(x2, x0, x1);
  x0 = fmaxf(x0, -125.f);
  x1 = fmaxf(x1, -125.f);
  const uint64_t xc = f2_pack(x0, x1);
  const uint64_t magic = f2_pack(12582912.f, 12582912.f);  // 1.5 * 2^23
  const uint64_t t = f2_add(xc, magic);
  const uint64_t nf = f2_add(t, f2_pack(-12582912.f, -12582912.f));
  const uint64_t f = f2_fma(nf, f2_pack(-1.f, -1.f), xc);
  uint64_t q = f2_fma(f, f2_pack(0.009570099413394928f, 0.009570099413394928f), f2_pack(0.05591785907745361f, 0.05591785907745361f));
  q = f2_fma(q, f, f2_pack(0.240247443318367f, 0.240247443318367f));
  q = f2_fma(q, f, f2_pack(0.6931217908859253f, 0.6931217908859253f));
  q = f2_fma(q, f, f2_pack(0.9999992847442627f, 0.9999992847442627f));
  float q0, q1, t0, t1;
  f2_unpack(q, q0, q1);
  f2_unpack(t, t0, t1);
  p0 = __int_as_float(__float_as_int(q0) + (__float_as_int(t0) << 23));
  p1 = __int_as_float(__float_as_int(q1) + (__float_as_int(t1) << 23));
}
__device__ __forceinline__ uint32_t bf16x2_rn(float lo, float hi) {
  uint32_t r;
  asm("cvt.rn.bf16x2.f32 %0, %1, %2;" : "=r"(r) : "f"(hi), "f"(lo));
  return r;
}

struct AtBarriers {
  uint64_t qfull, qempty;
  uint64_t kfull[AT_MAX_STAGES], kempty[AT_MAX_STAGES], vfull[AT_MAX_STAGES], vempty[AT_MAX_STAGES];
  uint64_t sfull[2][2];  // MMA -> softmax: S tile (M tile, buffer) is in TMEM
  uint64_t sdone[2][2];  // softmax -> MMA: S has been read (and P written over it)
  uint64_t ofull[2];     // MMA -> softmax: one completion per PV of that M tile (lazy-rescale path)
  uint64_t ofin[2];      // MMA -> softmax: one completion per ITEM, after its last PV (epilogue).  A parity wait on
                         // ofull could alias here: the softmax may be two PVs ahead of the tensor pipe.
  uint64_t oempty[2];    // softmax -> MMA: the item's O accumulator has been read out
  uint64_t idxfull[2], idxempty[2];
};

// byte offset of packed key position p's row in a PAGED K / V pool (deliberately not inlined, see the loaders)
__device__ __noinline__ unsigned long long at_paged_row_bytes(const SpGeom& g, int p, uint32_t row_bytes) {
  return (unsigned long long)sp_kv_row(g, p) * row_bytes;
}

struct AtItem {
  int seq_start, t0, t1, kvh, row;
};

// Work item `id` -> queries and KV head.  Identical in every warp role.
template <int G, bool SPARSE>
__device__ __forceinline__ bool at_item(const SpGeom& g, int id, int Hkv, int cpr, int n_chunks, int chunk_base, AtItem& it) {
  constexpr int QT = 256 / G;
  it.kvh = id % Hkv;
  const int x = id / Hkv;
  if (SPARSE) {
    it.row = g.row_off + x / cpr;
    const SpRow ri = sp_row_info(g, it.row);
    it.seq_start = ri.seq_start;
    it.t0 = ri.t_first + (x % cpr) * QT;
    it.t1 = min(it.t0 + QT - 1, ri.t_last);
    return it.t0 <= ri.t_last;
  } else {
    SpGeom g2 = g;
    g2.b_sel = QT;
    it.row = chunk_base + n_chunks - 1 - x;  // heavy (late) chunks first
    const SpRow ri = sp_row_info(g2, it.row);
    it.seq_start = ri.seq_start;
    it.t0 = ri.t_first;
    it.t1 = ri.t_last;
    return it.t1 >= it.t0;
  }
}

// The i-th item of CTA c out of P: boustrophedon over rounds so that per-CTA totals balance when the cost falls
// monotonically with the item id (dense causal chunks).  Returns -1 when the round has no item for this CTA.
__device__ __forceinline__ int at_item_id(int i, int c, int P, int n_items) {
  const int id = i * P + ((i & 1) ? P - 1 - c : c);
  return id < n_items ? id : -1;
}

template <int D, int G, bool SPARSE, bool WITH_O, bool MASKED = false>
__global__ void __launch_bounds__(AT_THREADS, 1)
sp_tc_attn_kernel(const __grid_constant__ CUtensorMap tmQ, SpGeom g, const __nv_bfloat16* __restrict__ Q,
                  const __nv_bfloat16* __restrict__ K,
                  const __nv_bfloat16* __restrict__ V, const int32_t* __restrict__ idx, int k, int Hkv, float scale,
                  int local_window, float local_bias, int chunks_per_row, int n_chunks, int chunk_base, int n_items,
                  int n_stages, int kpad, __nv_bfloat16* __restrict__ O, float* __restrict__ lse,
                  const uint32_t* __restrict__ mbits = nullptr, long long mbits_pitch = 0) {
  static_assert(!MASKED || (!SPARSE && WITH_O && (G == 4 || G == 8)), "membership-masked mode: dense key tiles, G in {4, 8}");
  constexpr int QM = 128 / G;             // queries per M tile (MASKED: K extent of the mask product)
  constexpr int KB = D / 64;              // 64-wide column blocks of a row
  constexpr int CPR = D / 8;              // 16-byte chunks per row
  constexpr uint32_t Q_BLK = 256 * 128;   // bytes of one column block of the Q tile (256 rows)
  constexpr uint32_t KV_BLK = AT_KT * 128;
  constexpr uint32_t KV_TILE = KB * KV_BLK;
  constexpr uint32_t TM_O = 0, TM_S = 256;  // O: M tile mt at columns [mt*D, mt*D+D); S: (mt, b) at 256 + mt*128 + b*64

  extern __shared__ uint8_t smem_raw[];
  __shared__ AtBarriers bar;
  __shared__ uint32_t tmem_slot;
  __shared__ int n_eff_sh[2];

  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int Hq = Hkv * G;
  const int NS = n_stages;
  const int P = gridDim.x, cta = blockIdx.x;

  // 1024-byte alignment as an OFFSET from the shared array, so the compiler keeps the shared address space
  // (LDS / STS instead of generic loads) for everything carved from it
  uint8_t* smem = smem_raw + ((1024u - (smem_u32(smem_raw) & 1023u)) & 1023u);
  uint8_t* sQ = smem;
  uint8_t* sK = sQ + KB * Q_BLK;
  uint8_t* sV = sK + NS * KV_TILE;
  // MASKED: sAx = the one-hot query selector [128 rows x 64 columns] (constant), sBx = per ring stage the mask tile
  // [64 keys x 2 * QM queries] (0 / -2^127), both K-major SWIZZLE_128B like Q and K
  uint8_t* sAx = sV + (WITH_O ? NS * KV_TILE : 0);
  uint8_t* sBx = sAx + (MASKED ? AT_AX_BYTES : 0);
  int* sIdx = reinterpret_cast<int*>(sBx + (MASKED ? NS * AT_BX_BYTES : 0));  // SPARSE: [2][kpad]
  uint32_t* sFlag = reinterpret_cast<uint32_t*>(sIdx + 2 * kpad);          // SPARSE: [2][kpad / 64]
  // SPARSE over a PAGED cache: the pool row of every staged entry, [2][kpad] (translated ONCE per entry while staging;
  // the loaders then gather exactly as from contiguous tensors.  Translating per 16-byte chunk and key tile -- 16 threads
  // repeat one key's lookup -- made the loaders pace the kernel: 400 us for a 4K-query chunk at 128K, 3x the item time)
  int* sRow = reinterpret_cast<int*>(sFlag + 2 * (kpad / AT_KT));
  const int ntmax = kpad / AT_KT;

  const int win = local_window > 0 ? local_window : 0;
  const bool scale_pos = scale > 0.f;
  const float sl2 = scale * SP_LOG2E, lb2 = local_bias * SP_LOG2E;

  // ---- barriers, TMEM ----
  if (threadIdx.x == 0) {
    mbar_init(&bar.qfull, 1);
    tma_prefetch_desc(&tmQ);
    mbar_init(&bar.qempty, 2);
    for (int s = 0; s < AT_MAX_STAGES; ++s) {
      mbar_init(&bar.kfull[s], MASKED ? 256 : 128);  // MASKED: + one plain arrive per loader thread (mask tile stores)
      mbar_init(&bar.vfull[s], 128);
      mbar_init(&bar.kempty[s], 2);
      mbar_init(&bar.vempty[s], 2);
    }
    for (int m = 0; m < 2; ++m) {
      for (int b = 0; b < 2; ++b) {
        mbar_init(&bar.sfull[m][b], 1);
        mbar_init(&bar.sdone[m][b], 128);
      }
      mbar_init(&bar.ofull[m], 1);
      mbar_init(&bar.ofin[m], 1);
      mbar_init(&bar.oempty[m], 128);
      mbar_init(&bar.idxfull[m], 128);
      mbar_init(&bar.idxempty[m], 256 + 2);  // every softmax thread + the two MMA issuers
    }
    fence_barrier_init();
  }
  if (MASKED) {
    // selector tile: row R of an M tile (query R / G of the tile) has a single 1.0 in column R / G, so that
    // (selector x mask tile^T)[R, key] = mask tile[key, query of R]: the membership mask is ADDED to S by the tensor
    // core (QM / 16 extra K steps per S tile) and the softmax warps run the plain unmasked path
    for (int ch = threadIdx.x; ch < 128 * 8; ch += AT_THREADS) {
      const int row = ch >> 3, c8 = ch & 7, q = row / G;
      uint32_t w[4] = {0u, 0u, 0u, 0u};
      if ((q >> 3) == c8) w[(q & 7) >> 1] = (q & 1) ? 0x3F800000u : 0x00003F80u;  // bf16 1.0
      *reinterpret_cast<uint4*>(sAx + sw128_offset(row, c8)) = make_uint4(w[0], w[1], w[2], w[3]);
    }
    fence_proxy_async_smem();
  }
  if (warp == AT_MMA_WARP) tmem_alloc<512>(&tmem_slot);
  tc_fence_before_sync();
  __syncthreads();
  tc_fence_after_sync();
  const uint32_t tmem = tmem_slot;

  // register budget: 512 x 128 at launch -> softmax warpgroups 192, the other two warpgroups 64
  // (each role's code is dominated by its own setmaxnreg so ptxas allocates per role)
  if (warp >= AT_LOAD_WARP0 && warp < AT_LOAD_WARP0 + AT_LOAD_WARPS) {
    asm volatile("setmaxnreg.dec.sync.aligned.u32 64;");
    // =========================================== loaders ===========================================
    const int ptid = threadIdx.x - AT_LOAD_WARP0 * 32;  // 0..127
    constexpr int KPP = 128 / CPR;       // keys per pass of the 128 loader threads
    constexpr int PASSES = AT_KT / KPP;  // passes per tile
    const int c = ptid % CPR;
    const int key0 = ptid / CPR;
    const uint32_t kv_off = (uint32_t)(c / 8) * KV_BLK;
    uint32_t n_q = 0, n_it = 0;
    uint32_t ld_s = 0, ld_ph = 0;  // K / V ring slot of the next tile, and the parity of its use count
    bool ld_wrapped = false;       // the ring has been filled once: slots must be waited for
    // ---- index-list staging runs ONE ITEM AHEAD of the K/V loads (its global loads have L2 / DRAM latency and would
    // otherwise sit between two items): `is` / n_st walk the same item sequence as `i` / n_it ----
    int is = 0;
    uint32_t n_st = 0;
    int nt_buf[2] = {0, 0};
    auto stage_next = [&]() {  // stage the next valid item's support row into buffer n_st & 1 (SPARSE only)
      AtItem its;
      for (;; ++is) {
        if (is * P >= n_items) return;
        const int ids = at_item_id(is, cta, P, n_items);
        if (ids >= 0 && at_item<G, SPARSE>(g, ids, Hkv, chunks_per_row, n_chunks, chunk_base, its)) break;
      }
      ++is;
      const int ib = n_st & 1, iu = n_st >> 1;
      if (iu > 0) mbar_wait(&bar.idxempty[ib], (iu - 1) & 1);  // the softmax warps are done with item n_st - 2
      int* siw = sIdx + ib * kpad;
      uint32_t* fl = sFlag + ib * ntmax;
      for (int t = ptid; t < ntmax; t += 128) fl[t] = 0u;
      if (ptid == 0) n_eff_sh[ib] = 0;
      loader_bar_sync();
      const int32_t* sup = idx + (size_t)its.kvh * (size_t)g.idx_grp + (size_t)(its.row - g.row_off) * k;
      const int qa0 = its.seq_start + its.t0, qa1 = qa0 + 128 / G, plast = its.seq_start + its.t1;
      int my_last = 0;
      for (int e0 = ptid; e0 < kpad; e0 += 128 * 8) {  // 8 independent loads in flight per thread
        int pv[8];
#pragma unroll
        for (int u = 0; u < 8; ++u) {
          const int e = e0 + u * 128;
          pv[u] = e < k ? __ldg(sup + e) : -1;
        }
#pragma unroll
        for (int u = 0; u < 8; ++u) {
          const int e = e0 + u * 128;
          if (e < kpad) {
            const int p = pv[u];
            const bool ok = p >= its.seq_start && p <= plast;
            siw[e] = ok ? p : -1;
            uint32_t f = 0;
            if (!ok || p > qa0 - win) f |= 1u;
            if (!ok || p > qa1 - win) f |= 2u;
            if (ok) my_last = e + 1;
            // the 32 entries of a warp lie in ONE tile (e0 and 128 u are multiples of 32): one atomic per warp
            f = __reduce_or_sync(0xffffffffu, f);
            if (f && (ptid & 31) == 0) atomicOr(&fl[e / AT_KT], f);
          }
        }
      }
      my_last = __reduce_max_sync(0xffffffffu, my_last);
      if (my_last && (ptid & 31) == 0) atomicMax(&n_eff_sh[ib], my_last);
      if (g.bt != nullptr) {  // paged cache: the pool row of every entry, in a loop of its own (the contiguous path pays one branch)
        // (an ignored entry still gathers a row: a written one, so that 0 x garbage cannot make a NaN)
        for (int e = ptid; e < kpad; e += 128) {
          const int p = siw[e];  // written by this very thread above
          sRow[ib * kpad + e] = (int)sp_kv_row(g, p >= 0 ? p : its.seq_start);
        }
      }
      loader_bar_sync();
      nt_buf[ib] = (n_eff_sh[ib] + AT_KT - 1) / AT_KT;
      mbar_arrive(&bar.idxfull[ib]);
      ++n_st;
    };
    if (SPARSE) stage_next();
    for (int i = 0; i * P < n_items; ++i) {
      const int id = at_item_id(i, cta, P, n_items);
      AtItem it;
      if (id < 0 || !at_item<G, SPARSE>(g, id, Hkv, chunks_per_row, n_chunks, chunk_base, it)) continue;
      const int nq = it.t1 - it.t0 + 1;
      const int n_mt = (nq * G > 128) ? 2 : 1;
      int nt;
      const int* si = nullptr;
      bool staged_ahead = false;
      if (SPARSE) {
        nt = nt_buf[n_it & 1];
        si = (g.bt != nullptr ? sRow : sIdx) + (n_it & 1) * kpad;  // what the loaders gather by: pool rows / positions
        if (nt == 0) stage_next();  // nothing to load for this item: keep the one-item lookahead
      } else {
        nt = it.t1 / AT_KT + 1;
      }
      ++n_it;
      if (nt == 0) continue;
      // Per 16-byte chunk the loaders spend an LDS (the key's position), one 32 x 32 -> 64-bit multiply-add (row
      // address) and the cp.async itself: everything else is hoisted -- a loader warp shares its scheduler with two
      // softmax warps, and at ~280 instructions per tile (run-time ring modulo, 64-bit offset multiplies and the
      // swizzle recomputed per pass) the loaders took a fifth of the kernel's issue slots (profiles/r2_attn.md).
      const char* Kb = reinterpret_cast<const char*>(K) + ((size_t)it.kvh * D + c * 8) * 2;
      const long long v_minus_k = reinterpret_cast<const char*>(V) - reinterpret_cast<const char*>(K);
      const uint32_t row_bytes = (uint32_t)Hkv * D * 2;
      // destination of pass pi: row key0 + pi * KPP keeps the row's low three bits (KPP % 8 == 0), so its swizzled
      // offset is that of row key0 plus pi * KPP * 128
      static_assert(KPP % 8 == 0, "a loader pass must step whole swizzle atoms");
      const uint32_t dst_row0 = sw128_offset(key0, c % 8) + kv_off;
      // MASKED: thread -> (key mkey of the tile, M tile mmt): one 32-bit word of the membership bitmap
      // mbits[query / 32][key] holds the tile's QM queries for that key
      constexpr int NCH = QM / 8;  // 16-byte chunks (8 bf16 mask values) per key and M tile
      const int mkey = ptid & 63, mmt = ptid >> 6;
      const int mq0 = it.seq_start + it.t0 + mmt * QM;  // first query of the M tile (packed; a multiple of QM)
      const uint32_t* mrow = MASKED ? mbits + (size_t)(mq0 >> 5) * (size_t)mbits_pitch + it.seq_start : nullptr;
      const int msh = mq0 & 31;
      auto load_tile = [&](int j) {
        uint32_t mw = 0u;
        if (MASKED) {
          const int keyl = j * AT_KT + mkey;
          if (keyl <= it.t1) mw = __ldg(mrow + keyl);
        }
        const char* src[PASSES];
        int pos[PASSES];
#pragma unroll
        for (int pi = 0; pi < PASSES; ++pi) {
          int p;
          if (SPARSE) {
            p = si[j * AT_KT + key0 + pi * KPP];
            if (p < 0) p = it.seq_start;  // masked later; any valid row will do
          } else {
            p = it.seq_start + min(j * AT_KT + key0 + pi * KPP, it.t1);
          }
          src[pi] = Kb + (unsigned long long)(uint32_t)p * row_bytes;
          pos[pi] = p;
        }
        if (!SPARSE && g.bt != nullptr) {  // paged cache, dense: rows through the block table.  A CALL, so that the contiguous path above
                                // carries none of it as predicated-off instructions (64 issue slots per tile otherwise)
#pragma unroll
          for (int pi = 0; pi < PASSES; ++pi) src[pi] = Kb + at_paged_row_bytes(g, pos[pi], row_bytes);
        }
        if (ld_wrapped) mbar_wait(&bar.kempty[ld_s], ld_ph ^ 1);
        const uint32_t kdst = smem_u32(sK) + ld_s * KV_TILE + dst_row0;
#pragma unroll
        for (int pi = 0; pi < PASSES; ++pi) cp_async16(kdst + pi * (KPP * 128), src[pi]);
        cp_async_arrive_noinc(&bar.kfull[ld_s]);
        if (MASKED) {
          // 1 bit -> one bf16: 0x0000 (member) or 0xFF00 = -2^127 (not a member; finite, so 0 x mask stays 0).  Four
          // inverted bits times 0x10204080 put bit a into the sign of byte a (no two partial products share a bit
          // position); PRMT's sign-replicate mode turns each into the 0x00 / 0xFF high byte of a bf16.
          const uint32_t nw = ~(mw >> msh);
          uint8_t* xdst = sBx + ld_s * AT_BX_BYTES;
#pragma unroll
          for (int i = 0; i < NCH; ++i) {
            uint32_t o[4];
#pragma unroll
            for (int h2 = 0; h2 < 2; ++h2) {
              const uint32_t X = ((nw >> (8 * i + 4 * h2)) & 0xFu) * 0x10204080u;
              asm("prmt.b32 %0, %1, %2, %3;" : "=r"(o[2 * h2]) : "r"(X), "r"(0u), "r"(0x9484u));
              asm("prmt.b32 %0, %1, %2, %3;" : "=r"(o[2 * h2 + 1]) : "r"(X), "r"(0u), "r"(0xB4A4u));
            }
            *reinterpret_cast<uint4*>(xdst + sw128_offset(mkey, mmt * NCH + i)) = make_uint4(o[0], o[1], o[2], o[3]);
          }
          mbar_arrive(&bar.kfull[ld_s]);  // release: the stores above are visible to whoever sees the phase complete
        }
        if (WITH_O) {
          if (ld_wrapped) mbar_wait(&bar.vempty[ld_s], ld_ph ^ 1);
          const uint32_t vdst = smem_u32(sV) + ld_s * KV_TILE + dst_row0;
#pragma unroll
          for (int pi = 0; pi < PASSES; ++pi) cp_async16(vdst + pi * (KPP * 128), src[pi] + v_minus_k);
          cp_async_arrive_noinc(&bar.vfull[ld_s]);
        }
        if (++ld_s == (uint32_t)NS) {  // ring position and phase of the next tile
          ld_s = 0;
          ld_ph ^= 1;
          ld_wrapped = true;
        }
      };
      // The first tiles only need ring slots whose MMAs were issued before the previous item's last S MMA, so they
      // are prefetched BEFORE waiting for the Q buffer (released by that last S MMA).
      const int pre = min(nt, NS - 2);
      for (int j = 0; j < pre; ++j) load_tile(j);
      {  // Q tile: ONE 3-D TMA box per 64-column block: [256/G queries] x [G heads] x [64 channels] lands as rows
         // R = query * G + head of 128 bytes, SWIZZLE_128B (rows past the chunk are later queries or zero fill: their
         // outputs are never written).  The cp.async version cost ~800 address instructions per loader warp per item.
        // Every loader thread waits for the buffer (holding the loaders here, instead of letting three of the four warps
        // run ahead into the next ring slots, measured 3 % faster), and they meet at a named barrier BEFORE the one thread
        // issues the load.  The barrier is what makes the parity wait safe: without it a loader warp that is not needed
        // for progress could be lapped -- an item whose tiles were all prefetched above (nt <= NS - 2) can finish, and
        // complete the Q barrier's NEXT phase, before a slow warp gets here, and a parity wait on a lapped barrier never
        // returns (seen under ncu's SASS instrumentation: dense launches with several items per CTA hung on exactly
        // that).  Now the next phase cannot start before all 128 threads have passed this wait.
        if (n_q > 0) {
          mbar_wait(&bar.qempty, (n_q - 1) & 1);
          loader_bar_sync();
        }
        if (ptid == 0) {
          mbar_expect_tx(&bar.qfull, KB * Q_BLK);
#pragma unroll
          for (int kb = 0; kb < KB; ++kb)
            tma_load_3d(sQ + kb * Q_BLK, &tmQ, &bar.qfull, kb * 64, it.kvh * G, it.seq_start + it.t0 - g.q_off);
        }
        ++n_q;
      }
      for (int j = pre; j < nt; ++j) {
        load_tile(j);
        if (SPARSE && !staged_ahead && (j >= 3 || j == nt - 1)) {  // a few tiles are in flight: now fetch the NEXT item's list
          stage_next();
          staged_ahead = true;
        }
      }
      if (SPARSE && !staged_ahead) stage_next();
    }
    cp_async_wait<0>();
  } else if (warp == AT_MMA_WARP || warp >= AT_LOAD_WARP0 + AT_LOAD_WARPS) {
    // =========================================== MMA issuers ===========================================
    // One issuing warp per M tile (warps 8 and 13; 14, 15 idle).  Per key tile j it waits for softmax(j), issues
    // O += P V (j) and then S(j+2) = Q K^T into the S buffer that PV(j) just consumed: both come from the same
    // thread, so the tensor pipe orders them and no completion round trip sits between "P(j) written" and
    // "S(j+2) ready".  A single warp issuing for BOTH M tiles (~200 dependent uniform-datapath instructions per
    // tile) paced the whole CTA; split per M tile it stays under the ~1000 cycles a tile occupies the tensor pipe.
    // The whole warp runs the (warp-uniform) control flow and the mbarrier waits; one elected lane issues
    // tcgen05.mma / tcgen05.commit.  K / V stages and the Q buffer are released by BOTH M tiles (barrier count 2;
    // an M tile without work for a tile arrives without MMAs).
    asm volatile("setmaxnreg.dec.sync.aligned.u32 64;");
    const bool leader = elect_one();
    const int mt = warp == AT_MMA_WARP ? 0 : 1;
    if (warp == AT_MMA_WARP || warp == AT_LOAD_WARP0 + AT_LOAD_WARPS) {
      constexpr uint32_t idesc_s = umma_idesc_bf16(128, AT_KT, 0, 0);  // S = Q K^T : both K-major
      constexpr uint32_t idesc_o = umma_idesc_bf16(128, D, 0, 1);      // O += P V : P from TMEM, V MN-major
      const uint64_t qdesc0 = umma_desc_sw128(smem_u32(sQ) + mt * 16384, 16, 1024);
      const uint64_t kdesc0 = umma_desc_sw128(smem_u32(sK), 16, 1024);
      const uint64_t vdesc0 = umma_desc_sw128(smem_u32(sV), KV_BLK, 1024);
      const uint64_t axdesc0 = umma_desc_sw128(smem_u32(sAx), 16, 1024);
      const uint64_t bxdesc0 = umma_desc_sw128(smem_u32(sBx) + mt * (QM * 2), 16, 1024);  // this M tile's query columns
      uint32_t k_s = 0, k_ph = 0, v_s = 0, v_ph = 0;  // K / V ring positions of the next tile this warp consumes
      uint32_t n_q = 0, n_it = 0, n_o = 0;            // items with work / items seen / items this M tile was active in
      uint32_t cs = 0, cp = 0;                        // S tiles issued / PV tiles issued by this warp (buffer = & 1)
      for (int i = 0; i * P < n_items; ++i) {
        const int id = at_item_id(i, cta, P, n_items);
        AtItem it;
        if (id < 0 || !at_item<G, SPARSE>(g, id, Hkv, chunks_per_row, n_chunks, chunk_base, it)) continue;
        const int nq = it.t1 - it.t0 + 1;
        const int n_mt = (nq * G > 128) ? 2 : 1;
        int nt, my_nt;
        if (SPARSE) {
          const int ib = n_it & 1, iu = n_it >> 1;
          mbar_wait(&bar.idxfull[ib], iu & 1);
          nt = (n_eff_sh[ib] + AT_KT - 1) / AT_KT;
          my_nt = nt;
          // the issuers release the index buffer too: an item with an empty support needs no MMA, so without this the
          // loaders could restage the buffer (n_eff_sh, and the barrier's next phase) before a slow issuer got here
          __syncwarp();
          if (leader) mbar_arrive(&bar.idxempty[ib]);
        } else {
          nt = it.t1 / AT_KT + 1;
          my_nt = mt == 0 ? min(it.t0 + 128 / G - 1, it.t1) / AT_KT + 1 : nt;
        }
        if (mt >= n_mt) my_nt = 0;
        ++n_it;
        if (nt == 0) continue;
        auto adv_k = [&]() {
          if (++k_s == (uint32_t)NS) {
            k_s = 0;
            k_ph ^= 1;
          }
        };
        auto adv_v = [&]() {
          if (++v_s == (uint32_t)NS) {
            v_s = 0;
            v_ph ^= 1;
          }
        };
        auto issue_s = [&](int j) {  // S(j) into buffer cs & 1 (free: its previous tile's PV was issued by this thread)
          mbar_wait(&bar.kfull[k_s], k_ph);
          fence_proxy_async_smem();
          tc_fence_after_sync();
          if (leader) {
            const uint32_t d_s = tmem + TM_S + mt * 128 + (cs & 1) * 64;
            const uint64_t kd = kdesc0 + (uint64_t)((k_s * KV_TILE) >> 4);
#pragma unroll
            for (int kk = 0; kk < D / 16; ++kk) {
              umma_ss(d_s, qdesc0 + (uint64_t)(((kk / 4) * Q_BLK + (kk % 4) * 32) >> 4),
                      kd + (uint64_t)(((kk / 4) * KV_BLK + (kk % 4) * 32) >> 4), idesc_s, kk != 0);
            }
            if (MASKED) {  // S += selector x mask tile^T
              const uint64_t bx = bxdesc0 + (uint64_t)((k_s * AT_BX_BYTES) >> 4);
#pragma unroll
              for (int kk = 0; kk < QM / 16; ++kk) umma_ss(d_s, axdesc0 + (uint64_t)(kk * 2), bx + (uint64_t)(kk * 2), idesc_s, 1);
            }
            umma_commit(&bar.sfull[mt][cs & 1]);
            umma_commit(&bar.kempty[k_s]);
            if (j == my_nt - 1) umma_commit(&bar.qempty);  // every S MMA of the item is issued: Q is free when they finish
          }
          ++cs;
          adv_k();
        };
        mbar_wait(&bar.qfull, n_q & 1);
        fence_proxy_async_smem();
        tc_fence_after_sync();
        if (my_nt == 0 && leader) mbar_arrive(&bar.qempty);
        for (int j = 0; j < 2 && j < my_nt; ++j) issue_s(j);
        for (int j = 0; j < my_nt; ++j) {
          const uint32_t b = cp & 1, n = cp >> 1;
          if (WITH_O) {
            mbar_wait(&bar.vfull[v_s], v_ph);
            fence_proxy_async_smem();
          }
          mbar_wait(&bar.sdone[mt][b], n & 1);  // softmax(j) has read S (and written P over it)
          if (WITH_O) {
            if (j == 0 && n_o > 0) mbar_wait(&bar.oempty[mt], (n_o - 1) & 1);
            tc_fence_after_sync();
            if (leader) {
              const uint64_t vd = vdesc0 + (uint64_t)((v_s * KV_TILE) >> 4);
              const uint32_t d_o = tmem + TM_O + mt * D, a_p = tmem + TM_S + mt * 128 + b * 64;
#pragma unroll
              for (int kk = 0; kk < AT_KT / 16; ++kk)
                umma_ts(d_o, a_p + kk * 8, vd + (uint64_t)((kk * 2048) >> 4), idesc_o, (j | kk) != 0);
              umma_commit(&bar.ofull[mt]);
              if (j == my_nt - 1) umma_commit(&bar.ofin[mt]);
              umma_commit(&bar.vempty[v_s]);
            }
            adv_v();
          }
          ++cp;
          if (j + 2 < my_nt) issue_s(j + 2);
        }
        for (int j = my_nt; j < nt; ++j) {  // tiles only the other M tile reads: keep the ring counts in step
          mbar_wait(&bar.kfull[k_s], k_ph);
          if (leader) mbar_arrive(&bar.kempty[k_s]);
          adv_k();
          if (WITH_O) {
            mbar_wait(&bar.vfull[v_s], v_ph);
            if (leader) mbar_arrive(&bar.vempty[v_s]);
            adv_v();
          }
        }
        if (WITH_O && my_nt > 0) ++n_o;
        ++n_q;
      }
    }
    __syncwarp();
  } else {
    // =========================================== softmax ===========================================
    asm volatile("setmaxnreg.inc.sync.aligned.u32 192;");
    const int mt = warp / 4;
    const int r = (warp % 4) * 32 + lane;  // row inside the M tile == TMEM lane
    const int R = mt * 128 + r;
    const int ql = R / G, h = R % G;
    const uint32_t lane_base = (uint32_t)((warp % 4) * 32) << 16;
    uint32_t t_o = tmem + lane_base + TM_O + mt * D;
    const uint64_t sl2_2 = f2_pack(sl2, sl2);
    uint32_t t_s0 = tmem + lane_base + TM_S + mt * 128;
    uint32_t a_sfull = smem_u32(&bar.sfull[mt][0]), a_sdone = smem_u32(&bar.sdone[mt][0]);  // 32-bit barrier addresses
    // Loop invariants of the key-tile loop are made opaque to the compiler: left visible, ptxas re-derives them from
    // %tid / %cluster_ctaid in EVERY tile (S2R has tens of cycles of latency; ~60 instructions per tile went there).
    asm volatile("" : "+r"(t_o), "+r"(t_s0), "+r"(a_sfull), "+r"(a_sdone));
    uint32_t cs = 0, n_it = 0, n_ep = 0;  // S tiles consumed by this M tile (== PVs issued for it), items seen, epilogues
    for (int i = 0; i * P < n_items; ++i) {
      const int id = at_item_id(i, cta, P, n_items);
      AtItem it;
      if (id < 0 || !at_item<G, SPARSE>(g, id, Hkv, chunks_per_row, n_chunks, chunk_base, it)) continue;
      const int nq = it.t1 - it.t0 + 1;
      const int n_mt = (nq * G > 128) ? 2 : 1;
      int my_nt;
      const int ib = n_it & 1;
      const int* si = sIdx + ib * kpad;
      const uint32_t* fl = sFlag + ib * ntmax;
      if (SPARSE) {
        mbar_wait(&bar.idxfull[ib], (n_it >> 1) & 1);
        my_nt = (n_eff_sh[ib] + AT_KT - 1) / AT_KT;
      } else {
        my_nt = (mt == 0 ? min(it.t0 + 128 / G - 1, it.t1) : it.t1) / AT_KT + 1;
      }
      ++n_it;
      const bool row_valid = ql < nq;
      const int tl = it.t0 + min(ql, nq - 1);  // local query position of this row
      const int tp = it.seq_start + tl;        // packed
      const size_t orow = ((size_t)(tp - g.q_off) * Hq + it.kvh * G + h);
      const int qa_local = it.t0 + mt * (128 / G);
      // masked tiles: reference position of this row (packed for index lists, local for the dense kernel) and the last
      // position OUTSIDE its local window (no window: nothing is inside)
      int t_ref = SPARSE ? tp : tl;
      int near_lo = win > 0 ? t_ref - win : 0x7fffffff;
      asm volatile("" : "+r"(t_ref), "+r"(near_lo));

      if (mt < n_mt && my_nt > 0) {
        float m_run = -INFINITY, l_run = 0.f;
        // SPECULATIVE OFFSET: the exponentials of tile j are taken against the running max as it stood BEFORE the tile,
        // while the tile's own max is reduced beside them (independent instruction chains: FMNMX3 on the ALU pipe under
        // the MUFU / FMA work), so the row max is off the critical path of the softmax warps.  Only when the tile's max
        // exceeds the running max by more than the lazy-rescale threshold (always on the first finite tile of a row) is
        // the running max moved, O rescaled, S re-read from TMEM (P has not been stored over it yet) and the tile
        // redone: at most once per tile, p <= 2^AT_RESCALE_THRESHOLD otherwise, exactly as with the max taken first.
        for (int j = 0; j < my_nt; ++j, ++cs) {
          const uint32_t b = cs & 1;
          const uint32_t t_s = t_s0 + b * 64;
          mbar_wait_addr(a_sfull + b * 8, (cs >> 1) & 1);
          tc_fence_after_sync();
          bool flagged;
          if (SPARSE) flagged = ((fl[j] >> mt) & 1u) != 0;
          else flagged = (j * AT_KT + AT_KT - 1 > qa_local - win);
          flagged = flagged || !scale_pos;
          if (MASKED) flagged = false;  // causal order and membership both come with the mask product (host: scale > 0, no window)
          uint32_t pk[AT_KT / 2];
          float tsum;
          if (j == 0 && !flagged) {  // first tile: its max IS the running max (saves the certain second pass)
            uint32_t v[AT_KT];
            tmem_ld_x32(t_s, v);
            tmem_ld_x32(t_s + 32, v + 32);
            tmem_ld_wait();
            float a0 = fmaxf(__uint_as_float(v[0]), __uint_as_float(v[1]));
            float a1 = fmaxf(__uint_as_float(v[2]), __uint_as_float(v[3]));
#pragma unroll
            for (int cc = 4; cc < AT_KT; cc += 4) {
              a0 = fmaxf(a0, fmaxf(__uint_as_float(v[cc]), __uint_as_float(v[cc + 1])));
              a1 = fmaxf(a1, fmaxf(__uint_as_float(v[cc + 2]), __uint_as_float(v[cc + 3])));
            }
            const float a = fmaxf(a0, a1);
            m_run = (MASKED && a < AT_NO_KEY) ? -INFINITY : a * sl2;
          }
          bool redone = false;
#pragma unroll 1
          for (;;) {
            uint32_t v[AT_KT];
            tmem_ld_x32(t_s, v);
            tmem_ld_x32(t_s + 32, v + 32);
            tmem_ld_wait();
            const float m_off = (m_run == -INFINITY) ? 0.f : m_run;
            uint64_t sum2 = 0ull;
            float mx = -INFINITY;
            if (!flagged) {
              const uint64_t nm2 = f2_pack(-m_off, -m_off);
#pragma unroll
              for (int cc = 0; cc < AT_KT; cc += 2) {
                const uint64_t x2 = f2_fma(f2_pack(__uint_as_float(v[cc]), __uint_as_float(v[cc + 1])), sl2_2, nm2);
                float p0, p1;
                if ((WITH_O ? AT_POLY_EVERY : AT_POLY_EVERY_LSE) > 0 &&
                    (cc / 2) % (WITH_O ? AT_POLY_EVERY : AT_POLY_EVERY_LSE) == (WITH_O ? AT_POLY_EVERY : AT_POLY_EVERY_LSE) - 1) {
                  ex2_poly2(x2, p0, p1);  // FMA-pipe exp2 for a fraction of the pairs: MUFU.EX2 co-limits the tensor pipe
                } else {
                  float x0, x1;
                  f2_unpack(x2, x0, x1);
                  p0 = ex2_approx(x0);
                  p1 = ex2_approx(x1);
                }
                sum2 = f2_add(sum2, f2_pack(p0, p1));
                pk[cc / 2] = bf16x2_rn(p0, p1);
              }
            } else {
              // masked tile: the position tests of PAPER.md eq. (2) (causal, p <= t) and of the local window
              // (t - p < W gets the bias), folded into ONE additive term per element: -inf, or the bias, or 0, each
              // already less the running max, so that x - m comes out of a single FFMA.  One unsigned compare covers
              // "-1 (no entry)" and "p > t"; positions are read four at a time (same address in all lanes: broadcast).
              const float nm = -m_off, nb = lb2 - m_off;
              float mxr = -INFINITY;
#pragma unroll
              for (int cc = 0; cc < AT_KT; cc += 4) {
                int pp[4];
                if (SPARSE) {
                  const int4 p4 = *reinterpret_cast<const int4*>(si + j * AT_KT + cc);
                  pp[0] = p4.x, pp[1] = p4.y, pp[2] = p4.z, pp[3] = p4.w;
                } else {
#pragma unroll
                  for (int u = 0; u < 4; ++u) pp[u] = j * AT_KT + cc + u;
                }
                float xr[4];
#pragma unroll
                for (int u = 0; u < 4; ++u) {
                  const bool ok = (uint32_t)pp[u] <= (uint32_t)t_ref;
                  const float b = pp[u] > near_lo ? nb : nm;
                  xr[u] = fmaf(__uint_as_float(v[cc + u]), sl2, ok ? b : -INFINITY);
                }
                mxr = fmaxf(mxr, fmaxf(fmaxf(xr[0], xr[1]), fmaxf(xr[2], xr[3])));
#pragma unroll
                for (int u = 0; u < 4; u += 2) {
                  const float p0 = ex2_approx(xr[u]);
                  const float p1 = ex2_approx(xr[u + 1]);
                  sum2 = f2_add(sum2, f2_pack(p0, p1));
                  pk[(cc + u) / 2] = bf16x2_rn(p0, p1);
                }
              }
              mx = mxr + m_off;  // -inf stays -inf (m_off is finite)
            }
            {
              float s0, s1;
              f2_unpack(sum2, s0, s1);
              tsum = s0 + s1;
            }
            // ---- did the running max hold?  Unflagged tiles never reduce their max: every p >= 0, so a logit more than
            // 2^8 above the running max (or an overflow to inf) shows in the tile's SUM; only then is the max taken, from
            // a fresh read of S.  Flagged tiles have their max from the masking pass. ----
            bool need;
            if (!flagged) {
              // (a row with no finite running max yet -- only possible here after fully masked tiles of a list that is
              // not ascending -- has no reference to speculate against and takes its max the classic way)
              // (MASKED: a row none of whose keys so far was a member stays at -inf; one redo per tile at most)
              need = !(tsum <= AT_SUM_LIMIT) || (m_run == -INFINITY && !(MASKED && redone));
              if (!__any_sync(0xffffffffu, need)) break;
              redone = true;
              uint32_t w[AT_KT];
              tmem_ld_x32(t_s, w);
              tmem_ld_x32(t_s + 32, w + 32);
              tmem_ld_wait();
              float a0 = fmaxf(__uint_as_float(w[0]), __uint_as_float(w[1]));
              float a1 = fmaxf(__uint_as_float(w[2]), __uint_as_float(w[3]));
#pragma unroll
              for (int cc = 4; cc < AT_KT; cc += 4) {
                a0 = fmaxf(a0, fmaxf(__uint_as_float(w[cc]), __uint_as_float(w[cc + 1])));
                a1 = fmaxf(a1, fmaxf(__uint_as_float(w[cc + 2]), __uint_as_float(w[cc + 3])));
              }
              const float a = fmaxf(a0, a1);
              mx = (MASKED && a < AT_NO_KEY) ? -INFINITY : a * sl2;
            }
            // ---- running max with lazy rescale of the TMEM accumulator ----
            const float m_new = fmaxf(m_run, mx);
            if (flagged) {
              need = m_new > m_run + AT_RESCALE_THRESHOLD;  // also true for the first finite max
              if (!__any_sync(0xffffffffu, need)) break;
            }
            const float f = (need && m_new > m_run) ? ex2_approx(m_run - m_new) : 1.f;  // m_run = -inf -> 0
            if (WITH_O && j > 0) {
              mbar_wait(&bar.ofull[mt], (cs - 1) & 1);  // PV(j-1) has finished updating O
              tc_fence_after_sync();
#pragma unroll
              for (int c0 = 0; c0 < D; c0 += 32) {
                uint32_t o[32];
                tmem_ld_x32(t_o + c0, o);
                tmem_ld_wait();
#pragma unroll
                for (int q = 0; q < 32; ++q) o[q] = __float_as_uint(__uint_as_float(o[q]) * f);
                tmem_st_x32(t_o + c0, o);
              }
              tmem_st_wait();
            }
            l_run *= f;
            if (need) m_run = m_new;
          }
          l_run += tsum;
          if (WITH_O) {
            tmem_st_x32(t_s, pk);  // P (64 keys as 32 bf16x2 columns) over the first half of S
            tmem_st_wait();
          }
          tc_fence_before_sync();
          mbar_arrive_addr(a_sdone + b * 8);
        }
        // ---- epilogue ----
        if (WITH_O) {
          mbar_wait(&bar.ofin[mt], n_ep & 1);
          ++n_ep;
          tc_fence_after_sync();
          // (MASKED: a row without any member key has m_run = -inf; its l_run may hold the polynomial path's 2^-125s)
          const float inv = (l_run > 0.f && !(MASKED && m_run == -INFINITY)) ? 1.f / l_run : 0.f;
#pragma unroll
          for (int c0 = 0; c0 < D; c0 += 32) {
            uint32_t o[32];
            tmem_ld_x32(t_o + c0, o);
            tmem_ld_wait();
            if (c0 + 32 == D) {  // O is in registers: the next item's first PV may overwrite the accumulator
              tc_fence_before_sync();
              mbar_arrive(&bar.oempty[mt]);
            }
            if (row_valid) {
#if AT_STORE_V8
#pragma unroll
              for (int q = 0; q < 32; q += 16) {  // 32-byte stores: one whole sector per lane and instruction
                uint32_t w[8];
#pragma unroll
                for (int e = 0; e < 8; ++e)
                  w[e] = bf16x2_rn(__uint_as_float(o[q + 2 * e]) * inv, __uint_as_float(o[q + 2 * e + 1]) * inv);
                asm volatile("st.global.v8.b32 [%0], {%1, %2, %3, %4, %5, %6, %7, %8};" ::"l"(O + orow * D + c0 + q),
                             "r"(w[0]), "r"(w[1]), "r"(w[2]), "r"(w[3]), "r"(w[4]), "r"(w[5]), "r"(w[6]), "r"(w[7])
                             : "memory");
              }
#else
#pragma unroll
              for (int q = 0; q < 32; q += 8) {
                uint4 w;
                w.x = bf16x2_rn(__uint_as_float(o[q]) * inv, __uint_as_float(o[q + 1]) * inv);
                w.y = bf16x2_rn(__uint_as_float(o[q + 2]) * inv, __uint_as_float(o[q + 3]) * inv);
                w.z = bf16x2_rn(__uint_as_float(o[q + 4]) * inv, __uint_as_float(o[q + 5]) * inv);
                w.w = bf16x2_rn(__uint_as_float(o[q + 6]) * inv, __uint_as_float(o[q + 7]) * inv);
                *reinterpret_cast<uint4*>(O + orow * D + c0 + q) = w;
              }
#endif
            }
          }
        }
        if (lse != nullptr && row_valid)
          lse[orow] = (l_run > 0.f && !(MASKED && m_run == -INFINITY)) ? (m_run + log2f(l_run)) * SP_LN2 : -INFINITY;
      } else if (my_nt == 0 && row_valid) {  // empty support: O = 0, lse = -inf (reading A9)
        if (WITH_O) {
          const uint4 z = make_uint4(0, 0, 0, 0);
          for (int cc = 0; cc < CPR; ++cc) reinterpret_cast<uint4*>(O + orow * D)[cc] = z;
        }
        if (lse) lse[orow] = -INFINITY;
      }
      if (SPARSE) mbar_arrive(&bar.idxempty[ib]);
    }
  }
  tc_fence_before_sync();
  __syncthreads();
  if (warp == AT_MMA_WARP) tmem_dealloc<512>(tmem);
}

template <int D>
size_t attn_smem_bytes(int kpad, bool sparse, bool with_o, int stages, bool masked = false, bool paged = false) {
  const size_t kb = D / 64;
  return 1024 + kb * 256 * 128 + (size_t)stages * (with_o ? 2 : 1) * kb * AT_KT * 128 +
         (sparse ? (size_t)2 * kpad * 4 + (size_t)2 * (kpad / AT_KT) * 4 : 0) + (sparse && paged ? (size_t)2 * kpad * 4 : 0) +
         (masked ? (size_t)AT_AX_BYTES + (size_t)stages * AT_BX_BYTES : 0);
}

constexpr size_t AT_SMEM_LIMIT = 227 * 1024 - 512;  // dynamic limit minus the static barriers / slots

template <int D>
int attn_pick_stages(int kpad, bool sparse, bool with_o, bool masked = false, bool paged = false) {
  int s = AT_MAX_STAGES;
  while (s >= 2 && attn_smem_bytes<D>(kpad, sparse, with_o, s, masked, paged) > AT_SMEM_LIMIT) --s;
  return s;  // < 2 -> unsupported
}

int at_sm_count() { return sp_sm_count(); }

template <int D, int G, bool SPARSE, bool WITH_O, bool MASKED = false>
cudaError_t launch_one(const SpGeom& g, cudaStream_t st, const void* Q, const void* K, const void* V,
                       const int32_t* idx, int k, int Hkv, float scale, int lw, float lb, int cpr, int n_chunks,
                       int chunk_base, int n_items, void* O, float* lse, const uint32_t* mbits = nullptr,
                       long long mbits_pitch = 0) {
  const int kpad = SPARSE ? (k + AT_KT - 1) / AT_KT * AT_KT : 0;
  const bool paged = g.bt != nullptr;
  const int stages = attn_pick_stages<D>(kpad, SPARSE, WITH_O, MASKED, paged);
  if (stages < 2) return cudaErrorInvalidValue;
  const size_t smem = attn_smem_bytes<D>(kpad, SPARSE, WITH_O, stages, MASKED, paged);
  static size_t attr_smem_dev[SP_MAX_DEVICES];
  size_t& attr_smem = attr_smem_dev[sp_current_device()];
  if (smem > attr_smem) {
    cudaError_t e = cudaFuncSetAttribute(sp_tc_attn_kernel<D, G, SPARSE, WITH_O, MASKED>,
                                         cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    attr_smem = smem;
  }
  const int grid = n_items < at_sm_count() ? n_items : at_sm_count();
  CUtensorMap tmQ;  // Q viewed as [L][Hq][D]: box = 256/G queries x G heads x 64 channels
  {
    cudaError_t e = sp_make_tmap_bf16_3d(&tmQ, Q, D, (uint64_t)Hkv * G, (uint64_t)(g.q_rows ? g.q_rows : g.L), (uint64_t)D * 2,
                                         (uint64_t)Hkv * G * D * 2, G, 256 / G);
    if (e != cudaSuccess) return e;
  }
  sp_tc_attn_kernel<D, G, SPARSE, WITH_O, MASKED><<<grid, AT_THREADS, smem, st>>>(
      tmQ, g, (const __nv_bfloat16*)Q, (const __nv_bfloat16*)K, (const __nv_bfloat16*)V, idx, k, Hkv, scale, lw, lb, cpr,
      n_chunks, chunk_base, n_items, stages, kpad, (__nv_bfloat16*)O, lse, mbits, mbits_pitch);
  return cudaGetLastError();
}

template <int D, int G>
cudaError_t launch_dg(const SpGeom& g, cudaStream_t st, const void* Q, const void* K, const void* V, const int32_t* idx,
                      int k, int Hkv, float scale, int lw, float lb, int cpr, int n_chunks, int chunk_base, int n_items, void* O,
                      float* lse) {
  if (idx != nullptr) {
    if (O) return launch_one<D, G, true, true>(g, st, Q, K, V, idx, k, Hkv, scale, lw, lb, cpr, n_chunks, chunk_base, n_items, O, lse);
    return launch_one<D, G, true, false>(g, st, Q, K, V, idx, k, Hkv, scale, lw, lb, cpr, n_chunks, chunk_base, n_items, O, lse);
  }
  if (O) return launch_one<D, G, false, true>(g, st, Q, K, V, idx, k, Hkv, scale, lw, lb, cpr, n_chunks, chunk_base, n_items, O, lse);
  return launch_one<D, G, false, false>(g, st, Q, K, V, idx, k, Hkv, scale, lw, lb, cpr, n_chunks, chunk_base, n_items, O, lse);
}

template <int D>
cudaError_t launch_d(int G, const SpGeom& g, cudaStream_t st, const void* Q, const void* K, const void* V,
                     const int32_t* idx, int k, int Hkv, float scale, int lw, float lb, int cpr, int n_chunks,
                     int chunk_base, int n_items, void* O, float* lse) {
  switch (G) {
    case 1: return launch_dg<D, 1>(g, st, Q, K, V, idx, k, Hkv, scale, lw, lb, cpr, n_chunks, chunk_base, n_items, O, lse);
    case 2: return launch_dg<D, 2>(g, st, Q, K, V, idx, k, Hkv, scale, lw, lb, cpr, n_chunks, chunk_base, n_items, O, lse);
    case 4: return launch_dg<D, 4>(g, st, Q, K, V, idx, k, Hkv, scale, lw, lb, cpr, n_chunks, chunk_base, n_items, O, lse);
    case 8: return launch_dg<D, 8>(g, st, Q, K, V, idx, k, Hkv, scale, lw, lb, cpr, n_chunks, chunk_base, n_items, O, lse);
  }
  return cudaErrorInvalidValue;
}

// Membership bitmap of per-query supports (b_sel == 1): bit (t & 31) of bits[(t >> 5) * pitch + p] is set iff packed key
// position p is in query t's list AND causally valid for it (same sequence, p <= t).  One CTA per row.
__global__ void __launch_bounds__(256)
sp_support_bits_kernel(SpGeom g, const int32_t* __restrict__ idx, int k, uint32_t* __restrict__ bits, long long pitch) {
  const long long r = blockIdx.x;
  const SpRow ri = sp_row_info(g, (int)r);
  const int t = ri.seq_start + ri.t_last;
  uint32_t* row = bits + (size_t)(t >> 5) * (size_t)pitch;
  const uint32_t bit = 1u << (t & 31);
  const int32_t* sup = idx + (size_t)r * k;
  for (int e = threadIdx.x; e < k; e += 256) {
    const int p = __ldg(sup + e);
    if (p >= ri.seq_start && p <= t) atomicOr(row + p, bit);
  }
}

template <int D>
cudaError_t launch_masked_d(int G, const SpGeom& g, cudaStream_t st, const void* Q, const void* K, const void* V, int Hkv,
                            float scale, int n_chunks, int n_items, void* O, float* lse, const uint32_t* bits,
                            long long pitch) {
  switch (G) {
    case 4:
      return launch_one<D, 4, false, true, true>(g, st, Q, K, V, nullptr, 0, Hkv, scale, 0, 0.f, 1, n_chunks, 0, n_items, O,
                                                 lse, bits, pitch);
    case 8:
      return launch_one<D, 8, false, true, true>(g, st, Q, K, V, nullptr, 0, Hkv, scale, 0, 0.f, 1, n_chunks, 0, n_items, O,
                                                 lse, bits, pitch);
  }
  return cudaErrorInvalidValue;
}

}  // namespace

// ---- per-query supports as MASKED DENSE attention (PAPER.md:107 + :156; :315-317 names the per-query realization as
// the one that is "harder to fuse and amortize") ----
// When k is a sizeable fraction of the prefix, gathering k rows per query and KV head (4 flop per gathered byte) costs
// more than running the dense tcgen05 tile loop over the whole prefix and masking by membership: the mask reaches S
// as a rank-(128/G) product on the tensor core, so the softmax warps run their unmasked path and the kernel keeps
// the dense kernel's rate.  The caller (sp_api.cu) chooses between this and the gather kernel from the pair counts.
bool sp_tc_attn_masked_supported(int G, int d) {
  if (G != 4 && G != 8) return false;
  if (d != 64 && d != 128) return false;
  return (d == 128 ? attn_pick_stages<128>(0, false, true, true) : attn_pick_stages<64>(0, false, true, true)) >= 2;
}

// words per bitmap row and rows of the bitmap for a pack of L tokens
void sp_support_bits_shape(long long L, long long* pitch, long long* rows) {
  *pitch = (L + 3) / 4 * 4;
  *rows = (L + 31) / 32 + 8;  // + the query blocks a last, partly filled M tile names
}

cudaError_t sp_launch_support_bits(const SpGeom& g, const int32_t* idx, int k, long long n_rows, uint32_t* bits,
                                   cudaStream_t st) {
  long long pitch, rows;
  sp_support_bits_shape(g.L, &pitch, &rows);
  cudaError_t e = cudaMemsetAsync(bits, 0, (size_t)pitch * rows * sizeof(uint32_t), st);
  if (e != cudaSuccess) return e;
  if (n_rows <= 0) return cudaSuccess;
  sp_support_bits_kernel<<<(unsigned)n_rows, 256, 0, st>>>(g, idx, k, bits, pitch);
  sp_count_launch();
  return cudaGetLastError();
}

cudaError_t sp_launch_attn_tc_masked(const SpGeom& g, long long n_chunks, const void* Q, const void* K, const void* V,
                                     const uint32_t* bits, int Hq, int Hkv, int d, float scale, void* O, float* lse,
                                     cudaStream_t st) {
  const int G = Hq / Hkv;
  if (n_chunks <= 0) return cudaSuccess;
  if (n_chunks * Hkv > 0x7fffffffLL) return cudaErrorInvalidValue;
  long long pitch, rows;
  sp_support_bits_shape(g.L, &pitch, &rows);
  const int n_items = (int)(n_chunks * Hkv);
  cudaError_t e = d == 128 ? launch_masked_d<128>(G, g, st, Q, K, V, Hkv, scale, (int)n_chunks, n_items, O, lse, bits, pitch)
                           : launch_masked_d<64>(G, g, st, Q, K, V, Hkv, scale, (int)n_chunks, n_items, O, lse, bits, pitch);
  sp_count_launch();
  return e;
}

// ---- fixed scratch of the no-allocation entry point (sp_sparse_gqa_attn_static, include/sp.h) ----
// The membership bitmap of the masked tile loop for packs of up to SP_STATIC_MAX_TOKENS tokens lives in this file-scope
// array: every GPU that loads the library holds these 8.25 MiB until exit.  In HOST code the array's name is a host-side
// stand-in, not a device address: the address a kernel may use comes from cudaGetSymbolAddress, taken once per device
// with that device current.  Every call shares the array (contents are the last call's; the bitmap builder clears
// what it uses first), so calls that overlap on the GPU race.
constexpr size_t SP_STATIC_SCRATCH_WORDS = SP_STATIC_SCRATCH_BYTES / 4;  // pitch x rows of sp_support_bits_shape(8192)
static_assert(SP_STATIC_SCRATCH_WORDS == (size_t)SP_STATIC_MAX_TOKENS * (SP_STATIC_MAX_TOKENS / 32 + 8), "include/sp.h");
static __device__ __align__(256) uint32_t sp_static_scratch[SP_STATIC_SCRATCH_WORDS];

cudaError_t sp_static_scratch_ptr(uint32_t** ptr, size_t* bytes) {
  static uint32_t* dev_ptr[SP_MAX_DEVICES];
  const int dev = sp_current_device();
  if (dev_ptr[dev] == nullptr) {
    uint32_t* q = nullptr;
    cudaError_t e = cudaGetSymbolAddress((void**)&q, sp_static_scratch);
    if (e != cudaSuccess) return e;
    if (q == nullptr) return cudaErrorInvalidSymbol;
    dev_ptr[dev] = q;
  }
  *ptr = dev_ptr[dev];
  *bytes = SP_STATIC_SCRATCH_WORDS * sizeof(uint32_t);
  return cudaSuccess;
}

// The tcgen05 attention covers dense attention always and sparse attention when a support row's queries fill a
// useful part of an M tile; per-query (b_sel == 1) supports are gather-bound and stay on the CUDA-core kernel.
bool sp_tc_attn_supported(int b_sel, int G, bool sparse, int k, int d, bool paged) {
  if (!sparse) return true;
  if (b_sel * G < 32) return false;
  const int kpad = (k + AT_KT - 1) / AT_KT * AT_KT;
  return (d == 128 ? attn_pick_stages<128>(kpad, true, true, false, paged)
                   : attn_pick_stages<64>(kpad, true, true, false, paged)) >= 2;
}

// idx == nullptr -> dense causal attention over the query chunks [chunk_base, chunk_base + n_chunks_dense) of the
// pack (a chunk = 256/G consecutive queries of one sequence; the whole pack has sum_i ceil(n_i / (256/G)) chunks).
cudaError_t sp_launch_attn_tc(const SpGeom& g, long long n_rows, long long n_chunks_dense, long long chunk_base,
                              const void* Q, const void* K, const void* V, const int32_t* idx, int k, int Hq, int Hkv,
                              int d, float scale, int local_window, float local_bias, void* O, float* lse,
                              cudaStream_t st) {
  const int G = Hq / Hkv;
  const int QT = 256 / G;
  const bool sparse = idx != nullptr;
  const int cpr = sparse ? (g.b_sel + QT - 1) / QT : 1;
  const long long nx = sparse ? n_rows * cpr : n_chunks_dense;
  if (nx <= 0) return cudaSuccess;
  if (nx * Hkv > 0x7fffffffLL) return cudaErrorInvalidValue;
  const int n_items = (int)(nx * Hkv);
  cudaError_t e = d == 128 ? launch_d<128>(G, g, st, Q, K, V, idx, k, Hkv, scale, local_window, local_bias, cpr,
                                           (int)nx, sparse ? 0 : (int)chunk_base, n_items, O, lse)
                           : launch_d<64>(G, g, st, Q, K, V, idx, k, Hkv, scale, local_window, local_bias, cpr,
                                          (int)nx, sparse ? 0 : (int)chunk_base, n_items, O, lse);
  sp_count_launch();
  return e;
}
