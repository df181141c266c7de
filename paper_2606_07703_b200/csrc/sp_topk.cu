// sp_topk.cu -- causal top-k of support-row scores (PAPER.md:127 TopK_s(P,k); :145 sentinel padding;
// :156 invalid positions masked before selection).  Exact: compare/integer work only.
//
// One CTA (1024 threads) per support row.  The kept set is the first min(k, n) elements of the total order
// (score descending, index ascending), emitted in ascending index order, tail padded with -1.  With
// key = order-preserving uint32 image of the fp32 score, the kept set is { key > T } plus the first `need_eq`
// elements with key == T in index order, T = key of the k-th largest element.  Finding (T, need_eq):
//   1. a 1024-element pseudo-random sample of the row is sorted (bitonic: shuffles inside a warp, shared memory
//      across warps); two of its order statistics bracket T with high probability: klo <= T <= khi;
//   2. ONE pass over the row (staged in shared memory when it fits, else re-read from L2): every warp owns a
//      contiguous segment, counts its elements above khi and appends those inside [klo, khi] to its private
//      candidate list (no atomics);
//   3. if the bracket holds (count(>khi) < k <= count(>khi) + candidates, no list overflowed) T is found by a
//      bit-by-bit bisection over the few candidates (register resident; only the bits below the common prefix
//      of klo and khi are undecided); otherwise an exact 4-pass radix select over the whole row takes over
//      (always correct; only slower).
//   4. one index-ordered compaction pass; the per-warp output bases come from the candidate lists (or from a
//      counting pass in the fallback).  Ties go to the lower index and the output is ascending by construction.
#include "sp_common.cuh"

namespace {

constexpr int TK_THREADS = 1024;
constexpr int TK_WARPS = TK_THREADS / 32;
constexpr int TK_CACHE = 40 * 1024;       // keys staged in shared memory (160 KB)
constexpr int TK_CAND_PER_WARP = 256;     // private candidate list per warp (32 x 256 x 4 B = 32 KB)
constexpr int TK_SAMPLE = 1024;

__device__ __forceinline__ uint32_t order_key(float x) {
  uint32_t u = __float_as_uint(x);
  if (u == 0x80000000u) u = 0u;  // -0 ranks equal to +0
  return (u & 0x80000000u) ? ~u : (u | 0x80000000u);
}

template <bool CACHED>
__device__ __forceinline__ uint32_t load_key(const float* __restrict__ x, const uint32_t* keys, int i) {
  if (CACHED) return keys[i];
  return order_key(__ldg(x + i));
}

struct TkShared {
  uint32_t hist[256];
  uint32_t wgt[TK_WARPS], weq[TK_WARPS];  // per-warp totals (elements above khi / T; equal to T)
  uint32_t wcand[TK_WARPS];               // per-warp candidate counts
  uint32_t bis[34];                       // [32]: candidates above T
  uint32_t part[2][TK_WARPS];             // bisection: per-warp partial counts, double buffered by step parity
  uint32_t sel[2];                        // radix select scratch
  uint32_t T, need_eq, ok;
};

// ---- exact fallback: 4-pass MSB-first radix select (8 bits per pass) -> sh.T, sh.need_eq ----
template <bool CACHED>
__device__ void radix_select(const float* __restrict__ x, const uint32_t* keys, int n, int k, TkShared& sh) {
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  uint32_t prefix = 0, need = (uint32_t)k;
  for (int pass = 0; pass < 4; ++pass) {
    const int shift = 24 - 8 * pass;
    if (tid < 256) sh.hist[tid] = 0;
    __syncthreads();
    const uint32_t hi_mask = pass == 0 ? 0u : (0xffffffffu << (shift + 8));
    for (int i0 = 0; i0 < n; i0 += TK_THREADS) {
      const int i = i0 + tid;
      bool act = false;
      uint32_t bin = 0;
      if (i < n) {
        const uint32_t key = load_key<CACHED>(x, keys, i);
        act = ((key & hi_mask) == prefix);
        bin = (key >> shift) & 255u;
      }
      const uint32_t amask = __ballot_sync(0xffffffffu, act);
      if (act) {
        const uint32_t peers = __match_any_sync(amask, bin);
        if (lane == __ffs(peers) - 1) atomicAdd(&sh.hist[bin], (uint32_t)__popc(peers));
      }
    }
    __syncthreads();
    if (warp == 0) {  // locate the bin holding rank `need` counting from the top: 8 bins per lane
      uint32_t c[8];
      uint32_t tot = 0;
#pragma unroll
      for (int j = 0; j < 8; ++j) {
        c[j] = sh.hist[255 - (lane * 8 + j)];
        tot += c[j];
      }
      uint32_t incl = tot;
#pragma unroll
      for (int o = 1; o < 32; o <<= 1) {
        const uint32_t v = __shfl_up_sync(0xffffffffu, incl, o);
        if (lane >= o) incl += v;
      }
      uint32_t before = incl - tot;
      if (before < need && need <= incl) {
#pragma unroll
        for (int j = 0; j < 8; ++j) {
          if (need <= before + c[j]) {
            sh.sel[0] = 255u - (uint32_t)(lane * 8 + j);
            sh.sel[1] = need - before;
            break;
          }
          before += c[j];
        }
      }
    }
    __syncthreads();
    prefix |= sh.sel[0] << shift;
    need = sh.sel[1];
    __syncthreads();
  }
  if (tid == 0) {
    sh.T = prefix;
    sh.need_eq = need;
  }
  __syncthreads();
}

template <bool CACHED>
__device__ void topk_row(const float* __restrict__ x, uint32_t* keys, uint32_t* cand, int n, int k, int seq_start,
                         int32_t* __restrict__ out, TkShared& sh) {
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const uint32_t lt = (1u << lane) - 1u;

  if (CACHED) {  // stage the row once: 8 independent loads in flight per thread
    int i = tid;
    for (; i + 7 * TK_THREADS < n; i += 8 * TK_THREADS) {
      float v[8];
#pragma unroll
      for (int j = 0; j < 8; ++j) v[j] = __ldg(x + i + j * TK_THREADS);
#pragma unroll
      for (int j = 0; j < 8; ++j) keys[i + j * TK_THREADS] = order_key(v[j]);
    }
    for (; i < n; i += TK_THREADS) keys[i] = order_key(__ldg(x + i));
  }
  if (tid < 34) sh.bis[tid] = 0;
  // warp segments: contiguous, a multiple of 32 elements
  const int seg = ((n + TK_WARPS - 1) / TK_WARPS + 31) & ~31;
  const int seg0 = min(warp * seg, n), seg1 = min(seg0 + seg, n);
  uint32_t* my_cand = cand + warp * TK_CAND_PER_WARP;

  // ---- 1. bracket [klo, khi] from a sorted sample (short rows: everything is a candidate) ----
  uint32_t klo = 0u, khi = 0xffffffffu;
  if (n > TK_WARPS * TK_CAND_PER_WARP) {
    const int stride = n / TK_SAMPLE;  // >= 8
    uint32_t v;
    {
      const uint32_t h = ((uint32_t)tid * 2654435761u) >> 12;
      const int i = tid * stride + (int)(h % (uint32_t)stride);
      __syncthreads();  // keys staged
      v = load_key<CACHED>(x, keys, i);
    }
    // bitonic sort, descending; partners closer than a warp exchange by shuffle, the others through `cand`
    for (int size = 2; size <= TK_SAMPLE; size <<= 1) {
      const bool desc = (tid & size) == 0;
      for (int st = size >> 1; st > 0; st >>= 1) {
        uint32_t pv;
        if (st >= 32) {
          cand[tid] = v;
          __syncthreads();
          pv = cand[tid ^ st];
          __syncthreads();
        } else {
          pv = __shfl_xor_sync(0xffffffffu, v, st);
        }
        const bool keep_max = desc == ((tid & st) == 0);
        v = keep_max ? max(v, pv) : min(v, pv);
      }
    }
    cand[tid] = v;
    __syncthreads();
    const float frac = (float)k / (float)n;
    const float r = frac * TK_SAMPLE;  // expected sample rank (from the top) of T
    const int margin = (int)ceilf(3.5f * sqrtf(r * (1.f - frac))) + 4;
    const int ih = (int)floorf(r) - margin, il = (int)ceilf(r) + margin;
    if (ih > 0) khi = cand[ih];
    if (il < TK_SAMPLE - 1) klo = cand[il];
  }
  __syncthreads();  // sample reads done before the candidate lists reuse the buffer; keys staged

  // ---- 2. one pass: count above khi, collect candidates per warp ----
  uint32_t my_gt = 0, ncand = 0;  // ncand is warp-uniform
  for (int i0 = seg0; i0 < seg1; i0 += 32) {
    const int i = i0 + lane;
    bool c = false;
    uint32_t key = 0u;
    if (i < seg1) {
      key = load_key<CACHED>(x, keys, i);
      my_gt += key > khi;
      c = key >= klo && key <= khi;
    }
    const uint32_t m = __ballot_sync(0xffffffffu, c);
    if (c) {
      const uint32_t slot = ncand + __popc(m & lt);
      if (slot < TK_CAND_PER_WARP) my_cand[slot] = key;
    }
    ncand += __popc(m);
  }
  const uint32_t warp_gt = __reduce_add_sync(0xffffffffu, my_gt);
  if (lane == 0) {
    sh.wgt[warp] = warp_gt;
    sh.wcand[warp] = ncand;
  }
  __syncthreads();
  if (warp == 0) {
    const uint32_t tg = __reduce_add_sync(0xffffffffu, sh.wgt[lane]);
    const uint32_t tc = __reduce_add_sync(0xffffffffu, sh.wcand[lane]);
    const uint32_t mx = __reduce_max_sync(0xffffffffu, sh.wcand[lane]);
    if (lane == 0) {
      sh.ok = (mx <= TK_CAND_PER_WARP && tg < (uint32_t)k && (uint32_t)k <= tg + tc) ? 1u : 0u;
      sh.sel[0] = tg;
    }
  }
  __syncthreads();
  uint32_t T, need_eq;
  uint32_t base_gt, base_eq;  // selected-before counts at the start of this warp's segment
  if (sh.ok) {
    // ---- 3. bisection over the candidates: T = need-th largest candidate key ----
    const uint32_t need = (uint32_t)k - sh.sel[0];
    uint32_t ck[TK_CAND_PER_WARP / 32];
#pragma unroll
    for (int j = 0; j < TK_CAND_PER_WARP / 32; ++j) {
      const uint32_t e = lane + 32 * j;
      ck[j] = e < ncand ? my_cand[e] : 0u;  // key 0 never counts: thresholds below are >= 1 ... see note
    }
    // note: a padding key of 0 is only counted by the threshold 0 itself, which is never tested (bit steps OR in
    // at least one bit)
    // T lies in [klo, khi]: the bits above their highest differing bit are already known
    const uint32_t diff = klo ^ khi;
    const int top = diff ? 31 - __clz(diff) : -1;  // highest undecided bit
    uint32_t t = top < 0 ? khi : (top >= 31 ? 0u : (khi & ~((2u << top) - 1u)));
    for (int bit = top; bit >= 0; --bit) {
      const uint32_t c0 = t | (1u << bit);
      uint32_t cnt = 0;
#pragma unroll
      for (int j = 0; j < TK_CAND_PER_WARP / 32; ++j) cnt += ck[j] >= c0;
      cnt = __reduce_add_sync(0xffffffffu, cnt);
      uint32_t* part = sh.part[bit & 1];
      if (lane == 0) part[warp] = cnt;
      __syncthreads();
      if (__reduce_add_sync(0xffffffffu, part[lane]) >= need) t = c0;
    }
    T = t;
    {
      uint32_t g = 0, e = 0;
#pragma unroll
      for (int j = 0; j < TK_CAND_PER_WARP / 32; ++j) {
        g += ck[j] > T;
        e += (ck[j] == T) && (lane + 32 * j < ncand);
      }
      g = __reduce_add_sync(0xffffffffu, g);
      e = __reduce_add_sync(0xffffffffu, e);
      if (lane == 0) {
        if (g) atomicAdd(&sh.bis[32], g);
        sh.wgt[warp] = warp_gt + g;  // elements of this segment with key > T
        sh.weq[warp] = e;
      }
    }
    __syncthreads();
    need_eq = need - sh.bis[32];
  } else {
    radix_select<CACHED>(x, keys, n, k, sh);
    T = sh.T;
    need_eq = sh.need_eq;
    uint32_t g = 0, e = 0;
    for (int i = seg0 + lane; i < seg1; i += 32) {
      const uint32_t key = load_key<CACHED>(x, keys, i);
      g += key > T;
      e += key == T;
    }
    g = __reduce_add_sync(0xffffffffu, g);
    e = __reduce_add_sync(0xffffffffu, e);
    if (lane == 0) {
      sh.wgt[warp] = g;
      sh.weq[warp] = e;
    }
    __syncthreads();
  }
  {
    const uint32_t g = lane < warp ? sh.wgt[lane] : 0u, e = lane < warp ? sh.weq[lane] : 0u;
    base_gt = __reduce_add_sync(0xffffffffu, g);
    base_eq = __reduce_add_sync(0xffffffffu, e);
  }

  // ---- 4. index-ordered compaction of this warp's segment ----
  uint32_t run_gt = base_gt, run_eq = base_eq;
  for (int i0 = seg0; i0 < seg1; i0 += 32) {
    const int i = i0 + lane;
    bool gt = false, eq = false;
    if (i < seg1) {
      const uint32_t key = load_key<CACHED>(x, keys, i);
      gt = key > T;
      eq = key == T;
    }
    const uint32_t mg = __ballot_sync(0xffffffffu, gt), me = __ballot_sync(0xffffffffu, eq);
    const uint32_t pg = run_gt + __popc(mg & lt);
    const uint32_t pe = run_eq + __popc(me & lt);
    if (gt || (eq && pe < need_eq)) out[pg + min(pe, need_eq)] = seq_start + i;
    run_gt += __popc(mg);
    run_eq += __popc(me);
  }
}

__global__ void __launch_bounds__(TK_THREADS, 1)
sp_topk_kernel(SpGeom g, const float* __restrict__ scores, int64_t ld, int row_begin, int row_count, int k,
               int n_lo, int32_t* __restrict__ idx, int32_t* __restrict__ cnt) {
  extern __shared__ uint32_t tk_smem[];
  __shared__ TkShared sh;
  uint32_t* keys = tk_smem;
  uint32_t* cand = tk_smem + TK_CACHE;
  // long rows first: the row count is rarely a multiple of the SM count and the tail should be short rows
  const int r = row_count - 1 - (int)blockIdx.x;
  const SpRow ri = sp_row_info(g, row_begin + r);
  const int n = ri.t_last + 1;
  if (n <= n_lo) return;  // a short row: sp_topk_small_kernel's
  int32_t* out = idx + (size_t)r * k;
  const int keep = min(n, k);
  if (threadIdx.x == 0 && cnt) cnt[r] = keep;
  for (int j = keep + threadIdx.x; j < k; j += TK_THREADS) out[j] = -1;
  if (n <= k) {
    for (int j = threadIdx.x; j < n; j += TK_THREADS) out[j] = ri.seq_start + j;
    return;
  }
  const float* x = scores + (size_t)r * ld;
  if (n <= TK_CACHE) topk_row<true>(x, keys, cand, n, k, ri.seq_start, out, sh);
  else topk_row<false>(x, keys, cand, n, k, ri.seq_start, out, sh);
}

// ---- rows up to 16384 keys: W = 1, 2, ... 16 warps per support row (class W takes n <= 1024 W), the whole row in
// registers.
// Warp w owns the contiguous segment [w * seg, (w + 1) * seg) of the row (seg a multiple of 32, element
// i = w * seg + slot * 32 + lane, at most 32 slots).  32-step bisection on the order-preserving keys with
// `redux.sync` counts (W > 1: combined through a double-buffered shared array, one named barrier of the row's W
// warps per step), then an
// index-ordered compaction by ballots from per-warp bases.  The 1024-thread kernel above spends ~9 us per row on
// block barriers whatever n is; this one costs O(n) issue slots.  A row is processed iff n_lo < n <= n_hi, so that
// a panel with mixed row lengths can be covered by one launch per class. ----
constexpr int TKS_WARPS = 8;   // warps per CTA for W <= 8; W = 16 and 32 use one CTA of W warps per row
constexpr int TKS_WMAX = 16;   // the largest class: n <= 16384, two rows fill the register file of an SM (W = 32, one
                               // row per SM with nothing to overlap its barriers, measured SLOWER than sp_topk_kernel)
constexpr int TKS_NW = 1024;  // class W holds rows with n <= TKS_NW * W
template <int W>
__global__ void __launch_bounds__((W > TKS_WARPS ? W : TKS_WARPS) * 32, W <= 8 ? 3 : 2)
sp_topk_small_kernel(SpGeom g, const float* __restrict__ scores, int64_t ld, int row_begin, int row_count, int k,
                     int n_lo, int n_hi, int32_t* __restrict__ idx, int32_t* __restrict__ cnt) {
  constexpr int CTA_WARPS = W > TKS_WARPS ? W : TKS_WARPS;
  constexpr int RPC = CTA_WARPS / W;  // rows per CTA
  __shared__ int sh_cnt[2][TKS_WMAX];
  __shared__ int sh_fin[2][TKS_WMAX];
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const int w = warp % W;
  const int r = blockIdx.x * RPC + warp / W;
  if (r >= row_count) return;  // uniform over the W warps of a row, which are the only ones that synchronise
  const SpRow ri = sp_row_info(g, row_begin + r);
  const int n = ri.t_last + 1;
  if (n <= n_lo || n > n_hi) return;
  int32_t* out = idx + (size_t)r * k;
  const int keep = min(n, k);
  const int tr = w * 32 + lane;  // thread index within the row's W warps
  if (tr == 0 && cnt) cnt[r] = keep;
  for (int j = keep + tr; j < k; j += W * 32) out[j] = -1;
  if (n <= k) {
    for (int j = tr; j < n; j += W * 32) out[j] = ri.seq_start + j;
    return;
  }
  const float* x = scores + (size_t)r * ld;
  const int seg = (((n + W - 1) / W) + 31) & ~31;  // <= 1024
  const int ns = seg >> 5;
  const int i0 = w * seg + lane;
  uint32_t key[32];
#pragma unroll
  for (int s = 0; s < 32; ++s) {
    const int i = i0 + s * 32;
    key[s] = (s < ns && i < n) ? order_key(__ldg(x + i)) : 0u;  // padding key 0 is below every tested threshold
  }
  auto row_bar = [&]() { asm volatile("bar.sync %0, %1;" ::"r"(1 + warp / W), "n"(W * 32) : "memory"); };
  auto row_sum = [&](int c, int (*buf)[TKS_WMAX], int step) -> int {
    c = __reduce_add_sync(0xffffffffu, c);
    if (W == 1) return c;
    if (lane == 0) buf[step & 1][warp] = c;
    row_bar();  // the double buffer saves the second barrier
    int v = lane < W ? buf[step & 1][warp - w + lane] : 0;
    return __reduce_add_sync(0xffffffffu, v);
  };
  uint32_t t = 0;
  for (int bit = 31; bit >= 0; --bit) {  // T = the largest value with count(key >= T) >= k = the k-th largest key
    const uint32_t c0 = t | (1u << bit);
    // key >= c0  <=>  key + (2^32 - c0) carries out (c0 >= 1): two instructions per key, four chains; slots past
    // ns hold the padding key 0 < c0, no guard needed
    const uint32_t nc0 = 0u - c0;
    int c[4] = {0, 0, 0, 0};
#pragma unroll
    for (int s = 0; s < 32; ++s)
      asm("{\n\t.reg .u32 d;\n\tadd.cc.u32 d, %1, %2;\n\taddc.u32 %0, %0, 0;\n\t}" : "+r"(c[s & 3]) : "r"(key[s]), "r"(nc0));
    const int tot = row_sum((c[0] + c[1]) + (c[2] + c[3]), sh_cnt, bit);
    if (tot >= k) t = c0;
    if (tot == k) break;  // exactly k keys >= c0: they are the support, whatever the lower bits of the k-th key are
  }
  int cg = 0, ce = 0;
#pragma unroll
  for (int s = 0; s < 32; ++s) {
    cg += key[s] > t;  // padding keys are 0 < T
    ce += key[s] == t;
  }
  cg = __reduce_add_sync(0xffffffffu, cg);
  ce = __reduce_add_sync(0xffffffffu, ce);
  uint32_t run_gt = 0, run_eq = 0, total_gt = (uint32_t)cg;
  if (W > 1) {
    if (lane == 0) { sh_fin[0][warp] = cg; sh_fin[1][warp] = ce; }
    row_bar();
    total_gt = 0;
    for (int j = 0; j < W; ++j) {
      const uint32_t a = (uint32_t)sh_fin[0][warp - w + j], b = (uint32_t)sh_fin[1][warp - w + j];
      total_gt += a;
      if (j < w) { run_gt += a; run_eq += b; }
    }
  }
  const uint32_t need_eq = (uint32_t)k - total_gt;
  const uint32_t lt = (1u << lane) - 1u;
#pragma unroll
  for (int s = 0; s < 32; ++s) {
    if (s >= ns) break;
    const int i = i0 + s * 32;
    const bool gt = i < n && key[s] > t, eq = i < n && key[s] == t;
    const uint32_t mg = __ballot_sync(0xffffffffu, gt), me = __ballot_sync(0xffffffffu, eq);
    const uint32_t pg = run_gt + __popc(mg & lt), pe = run_eq + __popc(me & lt);
    if (gt || (eq && pe < need_eq)) out[pg + min(pe, need_eq)] = ri.seq_start + i;
    run_gt += __popc(mg);
    run_eq += __popc(me);
  }
}

int g_sm_count() { return sp_sm_count(); }

}  // namespace

cudaError_t sp_launch_topk(const SpGeom& g, const float* scores, int64_t ld, int row_begin, int row_count, int k,
                           int max_n_valid, int32_t* idx, int32_t* cnt, cudaStream_t st) {
  if (row_count <= 0) return cudaSuccess;
  static unsigned char attr_seen[SP_MAX_DEVICES];
  const size_t smem = (size_t)(TK_CACHE + TK_WARPS * TK_CAND_PER_WARP) * sizeof(uint32_t);
  if (sp_first_use_on_device(attr_seen)) {
    cudaError_t e = cudaFuncSetAttribute(sp_topk_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
  }
  // Row classes by n = n_valid: W = 1, 2, 4, 8 warps per row for n <= 1024 W, the 1024-thread kernel for longer rows.
  // One sequence (cu == nullptr): n(r) = min(L, (r + 1) b_sel) is monotone, each class is a contiguous row range and
  // gets a launch over exactly that range (the bound (r + 1) b_sel is conservative, so no class filter is needed).
  // Packed varlen: every class that can occur is launched over the whole panel and filters its rows by n.
  const int end = row_begin + row_count;
  const bool contiguous = g.cu == nullptr || max_n_valid <= TKS_NW;
  auto launch_small = [&](int W, int rb, int rc, int nlo) {
    const float* sc = scores + (size_t)(rb - row_begin) * ld;
    int32_t* ix = idx + (size_t)(rb - row_begin) * k;
    int32_t* cn = cnt ? cnt + (rb - row_begin) : nullptr;
    const int cw = W > TKS_WARPS ? W : TKS_WARPS, rpc = cw / W;
    const int grid = (rc + rpc - 1) / rpc, nhi = TKS_NW * W;
    switch (W) {
      case 1: sp_topk_small_kernel<1><<<grid, cw * 32, 0, st>>>(g, sc, ld, rb, rc, k, nlo, nhi, ix, cn); break;
      case 2: sp_topk_small_kernel<2><<<grid, cw * 32, 0, st>>>(g, sc, ld, rb, rc, k, nlo, nhi, ix, cn); break;
      case 4: sp_topk_small_kernel<4><<<grid, cw * 32, 0, st>>>(g, sc, ld, rb, rc, k, nlo, nhi, ix, cn); break;
      case 8: sp_topk_small_kernel<8><<<grid, cw * 32, 0, st>>>(g, sc, ld, rb, rc, k, nlo, nhi, ix, cn); break;
      default: sp_topk_small_kernel<16><<<grid, cw * 32, 0, st>>>(g, sc, ld, rb, rc, k, nlo, nhi, ix, cn); break;
    }
    sp_count_launch();
  };
  auto launch_big = [&](int rb, int rc, int nlo) {
    sp_topk_kernel<<<rc, TK_THREADS, smem, st>>>(g, scores + (size_t)(rb - row_begin) * ld, ld, rb, rc, k, nlo,
                                                 idx + (size_t)(rb - row_begin) * k,
                                                 cnt ? cnt + (rb - row_begin) : nullptr);
    sp_count_launch();
  };
  // A class is launched only when it fills the machine (rows * W >= one 8-warp CTA per SM) or when it is the last
  // one the panel needs; otherwise its rows are merged into the next larger class (which handles shorter rows too,
  // less efficiently) and finally into the 1024-thread kernel: a near-empty extra launch costs more than it saves
  // (c3 has 128 rows with n <= 8192: four extra launches made its top-k 0.068 -> 0.094 ms).
  const int fill = g_sm_count() * TKS_WARPS;
  if (contiguous) {
    // first row (absolute) whose bound (r + 1) b_sel exceeds the class limit; every row when the panel's longest fits
    auto first_above = [&](int nmax) {
      return max_n_valid <= nmax ? end : min(end, max(row_begin, nmax / g.b_sel));
    };
    int cls_w[6], cls_lo[6], cls_hi[6], ncls = 0;
    int pending = row_begin;
    for (int W = 1; W <= TKS_WMAX; W <<= 1) {
      const int hi = first_above(TKS_NW * W);
      const int rows = hi - pending;
      if (rows > 0 && ((long long)rows * W >= fill || hi == end)) {
        cls_w[ncls] = W; cls_lo[ncls] = pending; cls_hi[ncls] = hi; ++ncls;
        pending = hi;
      }
      if (hi == end) break;
    }
    if (pending < end) launch_big(pending, end - pending, -1);  // the longest rows first
    for (int i = ncls - 1; i >= 0; --i) launch_small(cls_w[i], cls_lo[i], cls_hi[i] - cls_lo[i], -1);
  } else if ((long long)row_count < fill) {  // packed, few rows: one launch
    if (max_n_valid > TKS_NW * TKS_WMAX) {
      launch_big(row_begin, row_count, -1);
    } else {
      int W = 2;
      while (TKS_NW * W < max_n_valid) W <<= 1;
      launch_small(W, row_begin, row_count, -1);
    }
  } else {
    if (max_n_valid > TKS_NW * TKS_WMAX) launch_big(row_begin, row_count, TKS_NW * TKS_WMAX);
    for (int W = TKS_WMAX; W >= 1; W >>= 1)
      if (W == 1 || max_n_valid > TKS_NW * (W / 2)) launch_small(W, row_begin, row_count, W == 1 ? -1 : TKS_NW * (W / 2));
  }
  return cudaGetLastError();
}
