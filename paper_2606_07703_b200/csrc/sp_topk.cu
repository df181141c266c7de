// sp_topk.cu -- causal top-k of support-row scores (PAPER.md:127 TopK_s(P,k); :145 sentinel padding;
// :156 invalid positions masked before selection).  Exact: compare/integer work only.
//
// The kept set is the first min(k, n) elements of the total order (score descending, index ascending), emitted in
// ascending index order, tail padded with -1.  With key = order-preserving uint32 image of the fp32 score, the kept
// set is { key > T } plus the first `need_eq` elements with key == T in index order, T = key of the k-th largest
// element.  Two kernels find (T, need_eq) and compact:
//   sp_topk_small_kernel<W>  rows up to 1024 W keys (W = 1 .. 8 warps per row), the row in registers, bit-by-bit
//                            bisection with redux.sync counts;
//   sp_topk_stream_kernel<W> longer rows (W = 8 warps per row, three rows per SM; W = 32 for panels of fewer long rows than
//                            SMs, e.g. a prefill chunk's): sampled bracket, ONE streaming pass that lists what can still be selected,
//                            radix select over the candidates, compaction from the list; exact radix-select fallback
//                            over the whole row when the bracket does not hold (always correct, only slower).
#include "sp_common.cuh"

namespace {

constexpr int TK_WARPS = 32;  // sizes the per-warp scratch arrays of TkShared (any CTA up to 1024 threads)

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
  uint32_t hist2[256];
  uint32_t wgt[TK_WARPS], weq[TK_WARPS];  // per-warp totals (elements above khi / T; equal to T)
  uint32_t wcand[TK_WARPS];               // per-warp candidate counts
  uint32_t bis[34];                       // [32]: candidates above T
  uint32_t part[2][TK_WARPS];             // bisection: per-warp partial counts, double buffered by step parity
  uint32_t sel[2];                        // radix select scratch
  uint32_t T, need_eq, ok, tg;
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
    for (int i0 = 0; i0 < n; i0 += (int)blockDim.x) {
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

// ---- rows beyond the register-resident classes: ONE streaming pass ----
// 256 threads per row, three rows per SM.  (1) 512 pseudo-random keys of the row are sorted (bitonic, shared memory);
// two order statistics bracket the k-th largest key T: klo <= T <= khi with high probability.  (2) The row is read
// ONCE, 16 bytes per lane and load: every warp owns a contiguous segment, counts its keys above khi and appends every
// key >= klo, with its index, to a private list in shared memory -- in index order (ballots), so the concatenation of
// the eight lists is the index-ordered list of everything that can still be selected (~k + 10 % of n entries).
// (3) If the bracket held (count(> khi) < k <= entries, no list overflowed) T is found by bit-by-bit bisection over the
// register-resident list entries (only the bits below the common prefix of klo and khi are undecided), and (4) the
// output is compacted from the lists: ties to the lower index and ascending order fall out of the list order.
// Otherwise the exact radix select over the row (from L2 / HBM) and two more passes take over: always correct, only
// slower.  (Round 1's kernel, 1024 threads per row, staged the row in shared memory and walked it three times with a
// block-wide barrier between the phases of the single row an SM held: ~45 K cycles per 24 K-key row, 0.09 of the HBM
// rate.)
// list entries per warp (8 B each).  8 warps per row: 1024 (64 KB, three rows per SM) or, when the panel's longest row is
// expected to list well under 640 entries per warp, 768 (48 KB and 64 registers: FOUR rows per SM, 9 % faster at c4 @ 32K;
// at 64K the lists outgrow it and rows fall to the exact fallback, 5.4 against 4.3 ms; there 16 warps per row with 512
// entries each -- the same 64 KB, two rows = 32 warps per SM -- give 4.0 ms).  32 warps per row: 512 (128 KB).
constexpr int TX_LIST_16 = 512, TX_LIST_WIDE = 512, TX_LIST_8 = 1024, TX_LIST_8_SMALL = 768;  // list entries per warp (8 B each): 64 KB / 128 KB per row
constexpr int TX_SAMPLE = 1024;
constexpr int TX_UNROLL = 4;     // 16-byte loads in flight per lane
constexpr int TX_WIDE_MIN_N = 16384;  // the 32-warp form pays from here (a warp's segment still spans several load steps)

// rank-th largest (rank >= 1) of the keys the CTA's threads hold in registers: slot j of a thread counts iff bit j of
// `valid` is set.  MSB-first radix select in digits of up to 8 bits starting at bit `top`: every valid key agrees with
// `known` above that bit.  At most `max_passes` digits are resolved; the result has the unresolved low bits zero and
// *rest = how many keys share its resolved prefix down to the rank (the number of ties to take when all bits are
// resolved).  *low = mask of the unresolved bits.
template <int NK>
__device__ __forceinline__ uint32_t tx_select(const uint32_t (&key)[NK], uint32_t valid, int nk_used, uint32_t rank, int top,
                                              uint32_t known, int max_passes, TkShared& sh, uint32_t* rest, uint32_t* low) {
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  uint32_t hi_mask = top >= 31 ? 0u : (0xffffffffu << (top + 1));  // bits already decided
  uint32_t prefix = known & hi_mask, need = rank;
  int hi = top;
  for (int pass = 0; pass < max_passes && hi >= 0; ++pass) {
    const int lo = hi >= 7 ? hi - 7 : 0;
    const uint32_t dmask = (2u << (hi - lo)) - 1u;
    if (tid < 256) sh.hist[tid] = 0;
    __syncthreads();
#pragma unroll
    for (int j = 0; j < NK; ++j) {
      if (j >= nk_used) break;  // warp-uniform
      if (((valid >> j) & 1u) && ((key[j] & hi_mask) == prefix)) atomicAdd(&sh.hist[(key[j] >> lo) & dmask], 1u);
    }
    __syncthreads();
    if (warp == 0) {  // the bin holding rank `need` counting from the top: 8 bins per lane
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
    prefix |= sh.sel[0] << lo;
    need = sh.sel[1];
    hi_mask |= dmask << lo;
    hi = lo - 1;
  }
  *rest = need;
  *low = ~hi_mask;
  return prefix;
}

// Bracket of the sample: the keys of sample ranks r_hi < r_lo (0-based from the top), each resolved to the two 8-bit
// digits below bit `top` (above it all sample keys agree with `known`) and rounded outwards -- an approximate bracket
// is as good as an exact one, it only has to contain T.  Two passes; the first histogram serves both ranks.
template <int NK>
__device__ __forceinline__ void tx_bracket(const uint32_t (&key)[NK], int r_hi, int r_lo, bool want_hi, bool want_lo, int top,
                                           uint32_t known, TkShared& sh, uint32_t* khi, uint32_t* klo) {
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  uint32_t hi_mask = top >= 31 ? 0u : (0xffffffffu << (top + 1));
  uint32_t pre_h = known & hi_mask, pre_l = pre_h;
  uint32_t need_h = (uint32_t)r_hi + 1u, need_l = (uint32_t)r_lo + 1u;
  int hi = top;
  for (int pass = 0; pass < 2 && hi >= 0; ++pass) {
    const int lo = hi >= 7 ? hi - 7 : 0;
    const uint32_t dmask = (2u << (hi - lo)) - 1u;
    if (tid < 256) {
      sh.hist[tid] = 0;
      sh.hist2[tid] = 0;
    }
    __syncthreads();
#pragma unroll
    for (int j = 0; j < NK; ++j) {
      const uint32_t bin = (key[j] >> lo) & dmask, top_bits = key[j] & hi_mask;
      if (top_bits == pre_h) atomicAdd(&sh.hist[bin], 1u);
      if (top_bits == pre_l) atomicAdd(&sh.hist2[bin], 1u);
    }
    __syncthreads();
    if (warp < 2) {  // warp 0: rank r_hi in hist, warp 1: rank r_lo in hist2
      const uint32_t* hh = warp == 0 ? sh.hist : sh.hist2;
      const uint32_t need = warp == 0 ? need_h : need_l;
      uint32_t c[8];
      uint32_t tot = 0;
#pragma unroll
      for (int j = 0; j < 8; ++j) {
        c[j] = hh[255 - (lane * 8 + j)];
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
            sh.part[warp][0] = 255u - (uint32_t)(lane * 8 + j);
            sh.part[warp][1] = need - before;
            break;
          }
          before += c[j];
        }
      }
    }
    __syncthreads();
    pre_h |= sh.part[0][0] << lo;
    need_h = sh.part[0][1];
    pre_l |= sh.part[1][0] << lo;
    need_l = sh.part[1][1];
    hi_mask |= dmask << lo;
    hi = lo - 1;
  }
  if (want_hi) *khi = pre_h | ~hi_mask;
  if (want_lo) *klo = pre_l;
}

__device__ __forceinline__ float key_to_float(uint32_t key) {
  return __uint_as_float((key & 0x80000000u) ? (key ^ 0x80000000u) : ~key);
}

// TXW = warps per row: 8 (three rows per SM) when the panel has rows enough to fill the machine, 32 (one row per SM, the
// row's passes spread over four times the warps) for panels of few long rows -- a prefill CHUNK has q_count / b_sel of them.
template <int TXW, int TX_LIST>
__global__ void __launch_bounds__(TXW * 32, TXW == 8 ? (TX_LIST <= TX_LIST_8_SMALL ? 4 : 3) : (TXW == 16 ? 2 : 1))
sp_topk_stream_kernel(SpGeom g, const float* __restrict__ scores, int64_t ld, int row_begin, int row_count, int k,
                      int n_lo, int32_t* __restrict__ idx, int32_t* __restrict__ cnt) {
  constexpr int TX_THREADS = TXW * 32, TX_WARPS = TXW;
  extern __shared__ uint32_t tx_smem[];  // [TX_WARPS][TX_LIST] pairs (score bits, index)
  __shared__ TkShared sh;
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const uint32_t lt = (1u << lane) - 1u;
  const int r = row_count - 1 - (int)blockIdx.x;  // long rows first
  const SpRow ri = sp_row_info(g, row_begin + r);
  const int n = ri.t_last + 1;
  if (n <= n_lo) return;
  int32_t* out = idx + (size_t)r * k;
  const int keep = min(n, k);
  if (tid == 0 && cnt) cnt[r] = keep;
  for (int j = keep + tid; j < k; j += TX_THREADS) out[j] = -1;
  if (n <= k) {
    for (int j = tid; j < n; j += TX_THREADS) out[j] = ri.seq_start + j;
    return;
  }
  const float* x = scores + (size_t)r * ld;

  // ---- 1. bracket from a sample (rows too short to sample: everything is a candidate).  Two order statistics of the
  // sample, each resolved to the 16 bits below the sample's highest differing bit and rounded outwards ----
  uint32_t klo = 0u, khi = 0xffffffffu;
  if (n >= 4 * TX_SAMPLE) {
    const int stride = n / TX_SAMPLE;
    uint32_t sk[TX_SAMPLE / TX_THREADS];
    uint32_t dif = 0;
#pragma unroll
    for (int j = 0; j < TX_SAMPLE / TX_THREADS; ++j) {
      const int e = tid + j * TX_THREADS;
      const uint32_t h = ((uint32_t)e * 2654435761u) >> 16;  // 16 pseudo-random bits -> an offset below stride
      sk[j] = order_key(__ldg(x + e * stride + (int)((h * (uint32_t)stride) >> 16)));
    }
    if (tid == 0) sh.T = sk[0];
    __syncthreads();
    const uint32_t ref = sh.T;
#pragma unroll
    for (int j = 0; j < TX_SAMPLE / TX_THREADS; ++j) dif |= sk[j] ^ ref;
    dif = __reduce_or_sync(0xffffffffu, dif);
    if (lane == 0) sh.part[0][warp] = dif;
    __syncthreads();
    dif = 0;
    for (int w = 0; w < TX_WARPS; ++w) dif |= sh.part[0][w];
    const int stop = dif ? 31 - __clz(dif) : -1;
    const float frac = (float)k / (float)n;
    const float rr = frac * TX_SAMPLE;  // expected sample rank (from the top) of T
    const int margin = (int)ceilf(3.5f * sqrtf(rr * (1.f - frac))) + 4;
    const int ih = (int)floorf(rr) - margin, il = (int)ceilf(rr) + margin;  // 0-based ranks from the top
    if (stop < 0) {
      klo = khi = ref;
    } else {
      // a rank outside the sample leaves that side of the bracket open; the helper still needs a valid rank to walk
      const bool want_hi = ih > 0, want_lo = il < TX_SAMPLE - 1;
      tx_bracket<TX_SAMPLE / TX_THREADS>(sk, want_hi ? ih : 0, want_lo ? il : TX_SAMPLE - 1, want_hi, want_lo, stop, ref, sh,
                                         &khi, &klo);
    }
  }
  // float images of the bracket for the streaming compare (-0 == +0 and the order of non-NaN values are those of the
  // keys; under flush-to-zero a denormal may pass as 0: the filter is a superset, the exact counts come from the keys)
  const float klo_f = klo == 0u ? -INFINITY : key_to_float(klo);

  // ---- 2. one pass over the row: every warp lists the elements >= klo of its segment, in index order ----
  const int seg = ((n + TX_WARPS - 1) / TX_WARPS + 127) & ~127;
  const int seg0 = min(warp * seg, n), seg1 = min(seg0 + seg, n);
  uint32_t* lst = tx_smem + warp * (2 * TX_LIST);
  const uint32_t lst_addr = (uint32_t)__cvta_generic_to_shared(lst);
  const bool vec_ok = (ld & 3) == 0;  // rows start 16-byte aligned
  uint32_t nl = 0;                     // warp-uniform
  bool over = false;
  for (int i0 = seg0; i0 < seg1; i0 += 128 * TX_UNROLL) {
    float v[TX_UNROLL][4];
#pragma unroll
    for (int u = 0; u < TX_UNROLL; ++u) {
      const int i = i0 + u * 128 + lane * 4;
      if (vec_ok && i + 3 < seg1) {
        const float4 q = __ldg(reinterpret_cast<const float4*>(x + i));
        v[u][0] = q.x, v[u][1] = q.y, v[u][2] = q.z, v[u][3] = q.w;
      } else {
#pragma unroll
        for (int c = 0; c < 4; ++c) v[u][c] = (i + c < seg1) ? __ldg(x + i + c) : __uint_as_float(0x7fc00000u);  // NaN: never listed
      }
    }
#pragma unroll
    for (int u = 0; u < TX_UNROLL; ++u) {
      const int i = i0 + u * 128 + lane * 4;
      bool f[4];
      uint32_t bal[4];
#pragma unroll
      for (int c = 0; c < 4; ++c) {
        f[c] = v[u][c] >= klo_f;
        bal[c] = __ballot_sync(0xffffffffu, f[c]);
      }
      if (bal[0] | bal[1] | bal[2] | bal[3]) {
        if (nl + 128u <= (uint32_t)TX_LIST) {  // room for a whole step
          // list order = index order: lane-major, then the lane's four elements
          uint32_t a = lst_addr + 8u * (nl + __popc(bal[0] & lt) + __popc(bal[1] & lt) + __popc(bal[2] & lt) + __popc(bal[3] & lt));
#pragma unroll
          for (int c = 0; c < 4; ++c) {
            if (f[c]) {
              asm volatile("st.shared.v2.b32 [%0], {%1, %2};" ::"r"(a), "r"(__float_as_uint(v[u][c])), "r"(i + c) : "memory");
              a += 8u;
            }
          }
        } else {
          over = true;
        }
        nl += __popc(bal[0]) + __popc(bal[1]) + __popc(bal[2]) + __popc(bal[3]);
      }
    }
  }
  __syncwarp();
  // ---- the warp's list in registers as keys; exact counts above / inside the bracket ----
  uint32_t ck[TX_LIST / 32];
  uint32_t cmask = 0, my_gt = 0, my_c = 0;
  const int slots = over ? 0 : (int)((nl + 31u) >> 5);
  // (no early exit from this loop: it WRITES the register array, and a break makes ptxas zero the remaining registers on
  // every one of the 32 exit paths -- ~290 moves per warp; slots are tested in groups of four instead)
#pragma unroll
  for (int j0 = 0; j0 < TX_LIST / 32; j0 += 4) {
#pragma unroll
    for (int j = j0; j < j0 + 4; ++j) ck[j] = 0u;
    if (j0 < slots) {  // warp-uniform
#pragma unroll
      for (int j = j0; j < j0 + 4; ++j) {
        const uint32_t e = lane + 32 * j;
        uint32_t bits;
        asm volatile("ld.shared.b32 %0, [%1];" : "=r"(bits) : "r"(lst_addr + 8u * e));
        const uint32_t key = order_key(__uint_as_float(bits));
        const bool in = e < nl, gt = in && key > khi, cd = in && key <= khi && key >= klo;
        my_gt += gt;
        my_c += cd;
        cmask |= (cd ? 1u : 0u) << j;
        ck[j] = (gt || cd) ? key : 0u;  // (flush-to-zero extras and padding: key 0)
      }
    }
  }
  my_gt = __reduce_add_sync(0xffffffffu, my_gt);
  my_c = __reduce_add_sync(0xffffffffu, my_c);
  if (lane == 0) {
    sh.wgt[warp] = my_gt;
    sh.wcand[warp] = my_c;
    sh.weq[warp] = over ? 1u : 0u;
  }
  __syncthreads();
  if (warp == 0) {
    const uint32_t a = lane < TX_WARPS ? sh.wgt[lane] : 0u, b = lane < TX_WARPS ? sh.wcand[lane] : 0u;
    const uint32_t c = lane < TX_WARPS ? sh.weq[lane] : 0u;
    const uint32_t tg0 = __reduce_add_sync(0xffffffffu, a), tc0 = __reduce_add_sync(0xffffffffu, b);
    const uint32_t ov0 = __reduce_or_sync(0xffffffffu, c);
    if (lane == 0) {
      sh.tg = tg0;
      sh.ok = (!ov0 && tg0 < (uint32_t)k && (uint32_t)k <= tg0 + tc0) ? 1u : 0u;
    }
  }
  __syncthreads();
  const uint32_t tg = sh.tg;
  const bool ok = sh.ok != 0u;
  uint32_t T, need_eq, base_gt, base_eq;
  if (ok) {
    // ---- 3. T = the (k - tg)-th largest of the candidates klo <= key <= khi ----
    const uint32_t diff = klo ^ khi;
    const int top = diff ? 31 - __clz(diff) : -1;  // highest bit the candidates can differ in
    if (top < 0) {
      T = khi;
      need_eq = (uint32_t)k - tg;
    } else {
      uint32_t low;
      T = tx_select<TX_LIST / 32>(ck, cmask, slots, (uint32_t)k - tg, top, khi, 4, sh, &need_eq, &low);
    }
    uint32_t gg = 0, ee = 0;
#pragma unroll
    for (int j = 0; j < TX_LIST / 32; ++j) {
      if (j >= slots) break;
      gg += ck[j] > T;
      ee += ck[j] == T;  // T >= klo >= 1 whenever a padding 0 could be met ... see below
    }
    // (a padding / dropped slot holds key 0; T == 0 only if klo == 0 and then nothing was dropped, and padding slots
    // lie past nl: they are excluded in the compaction by e < nl and here by the count below)
    if (T == 0u) {
      ee = 0;
#pragma unroll
      for (int j = 0; j < TX_LIST / 32; ++j) ee += (j < slots) && (lane + 32 * j < (int)nl) && ck[j] == 0u;
    }
    gg = __reduce_add_sync(0xffffffffu, gg);
    ee = __reduce_add_sync(0xffffffffu, ee);
    if (lane == 0) {
      sh.wgt[warp] = gg;
      sh.weq[warp] = ee;
    }
    __syncthreads();
    base_gt = base_eq = 0;
    for (int w = 0; w < warp; ++w) {
      base_gt += sh.wgt[w];
      base_eq += sh.weq[w];
    }
    // ---- 4. compaction from the list (index order) ----
    uint32_t run_gt = base_gt, run_eq = base_eq;
#pragma unroll
    for (int j = 0; j < TX_LIST / 32; ++j) {
      if (j >= slots) break;
      const uint32_t e = lane + 32 * j;
      const bool in = e < nl;
      const bool gt = in && ck[j] > T, eq = in && ck[j] == T;
      const uint32_t mg = __ballot_sync(0xffffffffu, gt), me = __ballot_sync(0xffffffffu, eq);
      const uint32_t pg = run_gt + __popc(mg & lt), pe = run_eq + __popc(me & lt);
      if (gt || (eq && pe < need_eq)) {
        uint32_t ix;
        asm volatile("ld.shared.b32 %0, [%1];" : "=r"(ix) : "r"(lst_addr + 8u * e + 4u));
        out[pg + min(pe, need_eq)] = ri.seq_start + (int)ix;
      }
      run_gt += __popc(mg);
      run_eq += __popc(me);
    }
    return;
  }
  // ---- exact fallback: radix select over the row, then a counting and a compaction pass ----
  radix_select<false>(x, nullptr, n, k, sh);
  T = sh.T;
  need_eq = sh.need_eq;
  {
    uint32_t gg = 0, ee = 0;
    for (int i = seg0 + lane; i < seg1; i += 32) {
      const uint32_t key = order_key(__ldg(x + i));
      gg += key > T;
      ee += key == T;
    }
    gg = __reduce_add_sync(0xffffffffu, gg);
    ee = __reduce_add_sync(0xffffffffu, ee);
    if (lane == 0) {
      sh.wgt[warp] = gg;
      sh.weq[warp] = ee;
    }
    __syncthreads();
    base_gt = base_eq = 0;
    for (int w = 0; w < warp; ++w) {
      base_gt += sh.wgt[w];
      base_eq += sh.weq[w];
    }
  }
  uint32_t run_gt = base_gt, run_eq = base_eq;
  for (int i0 = seg0; i0 < seg1; i0 += 32) {
    const int i = i0 + lane;
    bool gt = false, eq = false;
    if (i < seg1) {
      const uint32_t key = order_key(__ldg(x + i));
      gt = key > T;
      eq = key == T;
    }
    const uint32_t mg = __ballot_sync(0xffffffffu, gt), me = __ballot_sync(0xffffffffu, eq);
    const uint32_t pg = run_gt + __popc(mg & lt), pe = run_eq + __popc(me & lt);
    if (gt || (eq && pe < need_eq)) out[pg + min(pe, need_eq)] = ri.seq_start + i;
    run_gt += __popc(mg);
    run_eq += __popc(me);
  }
}

// ---- rows up to 16384 keys: W = 1, 2, ... 16 warps per support row (class W takes n <= 1024 W), the whole row in
// registers.
// Warp w owns the contiguous segment [w * seg, (w + 1) * seg) of the row (seg a multiple of 32, element
// i = w * seg + slot * 32 + lane, at most 32 slots).  32-step bisection on the order-preserving keys with
// `redux.sync` counts (W > 1: combined through a double-buffered shared array, one named barrier of the row's W
// warps per step), then an
// index-ordered compaction by ballots from per-warp bases.  (A 1024-thread kernel per row spends ~9 us per row on
// block barriers whatever n is; this one costs O(n) issue slots.)  A row is processed iff n_lo < n <= n_hi, so that
// a panel with mixed row lengths can be covered by one launch per class. ----
constexpr int TKS_WARPS = 8;   // warps per CTA for W <= 8; W = 16 and 32 use one CTA of W warps per row
#ifndef TKS_WMAX_DEF
#define TKS_WMAX_DEF 8
#endif
constexpr int TKS_WMAX = TKS_WMAX_DEF;  // the largest class: n <= 8192 (W = 16, rows up to 16384, measured slower than
                                        // the streaming kernel: c4 @ 32K 1.97 vs 1.79 ms; W = 4: 1.82)
constexpr int TKS_NW = 1024;  // class W holds rows with n <= TKS_NW * W
template <int W>
__global__ void __launch_bounds__((W > TKS_WARPS ? W : TKS_WARPS) * 32, W <= 8 ? 3 : 2)
sp_topk_small_kernel(SpGeom g, const float* __restrict__ scores, int64_t ld, int row_begin, int row_count, int k,
                     int n_lo, int n_hi, int32_t* __restrict__ idx, int32_t* __restrict__ cnt) {
  constexpr int CTA_WARPS = W > TKS_WARPS ? W : TKS_WARPS;
  constexpr int RPC = CTA_WARPS / W;  // rows per CTA
  __shared__ int sh_cnt[2][16];
  __shared__ int sh_fin[2][16];
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
  auto row_sum = [&](int c, int (*buf)[16], int step) -> int {
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
  // Row classes by n = n_valid: W = 1, 2, 4, 8 warps per row for n <= 1024 W, the streaming kernel for longer rows.
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
  const size_t smem_x = (size_t)2 * 8 * TX_LIST_8 * sizeof(uint32_t), smem_s = (size_t)2 * 8 * TX_LIST_8_SMALL * sizeof(uint32_t);
  const size_t smem_w = (size_t)2 * 32 * TX_LIST_WIDE * sizeof(uint32_t);
  static unsigned char attr_seen_x[SP_MAX_DEVICES];
  if (sp_first_use_on_device(attr_seen_x)) {
    cudaError_t e = cudaFuncSetAttribute(sp_topk_stream_kernel<8, TX_LIST_8>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_x);
    if (e != cudaSuccess) return e;
    e = cudaFuncSetAttribute(sp_topk_stream_kernel<8, TX_LIST_8_SMALL>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_s);
    if (e != cudaSuccess) return e;
    e = cudaFuncSetAttribute(sp_topk_stream_kernel<32, TX_LIST_WIDE>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_w);
    if (e != cudaSuccess) return e;
    e = cudaFuncSetAttribute(sp_topk_stream_kernel<16, TX_LIST_16>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_x);
    if (e != cudaSuccess) return e;
  }
  // entries per warp the longest row of the panel is expected to list: the bracket's floor is the sample rank
  // ceil(r) + margin of TX_SAMPLE, r = k / n * TX_SAMPLE (the kernel's own formula), spread over 8 warps
  auto expected_list8 = [&](int n) {
    const float frac = (float)k / (float)n, r = frac * TX_SAMPLE;
    const float il = ceilf(r) + ceilf(3.5f * sqrtf(r * (1.f - frac))) + 4.f;
    return (double)n * (il / TX_SAMPLE) / 8.0;
  };
  auto launch_big = [&](int rb, int rc, int nlo) {
    const float* sc = scores + (size_t)(rb - row_begin) * ld;
    int32_t* ix = idx + (size_t)(rb - row_begin) * k;
    int32_t* cn = cnt ? cnt + (rb - row_begin) : nullptr;
    // fewer rows than SMs: one 32-warp CTA per row instead of an 8-warp one (the SMs would idle otherwise)
    if (rc <= g_sm_count() && max_n_valid >= TX_WIDE_MIN_N)
      sp_topk_stream_kernel<32, TX_LIST_WIDE><<<rc, 32 * 32, smem_w, st>>>(g, sc, ld, rb, rc, k, nlo, ix, cn);
    else if (max_n_valid > k && expected_list8(max_n_valid) <= 400.0)
      sp_topk_stream_kernel<8, TX_LIST_8_SMALL><<<rc, 8 * 32, smem_s, st>>>(g, sc, ld, rb, rc, k, nlo, ix, cn);
    else if (expected_list8(max_n_valid) * 0.5 <= 240.0)  // 16 warps per row, two rows per SM: 32 instead of 24 warps per SM
      sp_topk_stream_kernel<16, TX_LIST_16><<<rc, 16 * 32, smem_x, st>>>(g, sc, ld, rb, rc, k, nlo, ix, cn);
    else
      sp_topk_stream_kernel<8, TX_LIST_8><<<rc, 8 * 32, smem_x, st>>>(g, sc, ld, rb, rc, k, nlo, ix, cn);
    sp_count_launch();
  };
  // A class is launched only when it fills the machine (rows * W >= one 8-warp CTA per SM) or when it is the last
  // one the panel needs; otherwise its rows are merged into the next larger class (which handles shorter rows too,
  // less efficiently) and finally into the streaming kernel: a near-empty extra launch costs more than it saves
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
