// sp_topk.cu -- causal top-k of support-row scores (PAPER.md:127 TopK_s(P,k); :145 sentinel padding;
// :156 invalid positions masked before selection).  Exact: compare/integer work only.
//
// One CTA per support row.  The kept set is the first min(k, n) elements of the total order
// (score descending, index ascending), emitted in ascending index order, tail padded with -1:
//   1. 4-pass MSB-first radix select (8 bits per pass) on an order-preserving uint32 image of the
//      fp32 score finds the exact key T of the k-th largest element and how many elements equal
//      to T must still be taken (`need_eq`).
//   2. One index-ordered compaction pass keeps every element with key > T and the first `need_eq`
//      elements with key == T  ->  ties go to the lower index, output is ascending.
// The row is staged in shared memory when it fits (one global read), else re-read (L2 resident).
#include "sp_common.cuh"

namespace {

constexpr int TOPK_THREADS = 512;
constexpr int TOPK_WARPS = TOPK_THREADS / 32;
constexpr int TOPK_SMEM_FLOATS = 48 * 1024;  // 192 KB row cache

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

template <bool CACHED>
__device__ void topk_row(const float* __restrict__ x, uint32_t* keys, int n, int k, int seq_start,
                         int32_t* __restrict__ out, uint32_t* hist, uint32_t* sh) {
  const int tid = threadIdx.x;
  const int lane = tid & 31, warp = tid >> 5;

  if (CACHED) {
    for (int i = tid; i < n; i += TOPK_THREADS) keys[i] = order_key(__ldg(x + i));
  }
  // ---- radix select ----
  uint32_t prefix = 0;       // high bits of T decided so far
  uint32_t need = (uint32_t)k;  // rank still to be located inside the current prefix bucket
  for (int pass = 0; pass < 4; ++pass) {
    const int shift = 24 - 8 * pass;
    if (tid < 256) hist[tid] = 0;
    __syncthreads();
    const uint32_t hi_mask = pass == 0 ? 0u : (0xffffffffu << (shift + 8));
    for (int i0 = 0; i0 < n; i0 += TOPK_THREADS) {
      const int i = i0 + tid;
      bool act = false;
      uint32_t bin = 0;
      if (i < n) {
        const uint32_t key = load_key<CACHED>(x, keys, i);
        act = ((key & hi_mask) == prefix);
        bin = (key >> shift) & 255u;
      }
      // warp-aggregated histogram update: scores cluster in a few high-byte bins
      const uint32_t amask = __ballot_sync(0xffffffffu, act);
      if (act) {
        const uint32_t peers = __match_any_sync(amask, bin);
        if (lane == __ffs(peers) - 1) atomicAdd(&hist[bin], (uint32_t)__popc(peers));
      }
    }
    __syncthreads();
    // locate the bin holding rank `need` counting from the top: warp 0 scans 256 bins, 8 per lane
    if (warp == 0) {
      uint32_t c[8];
      uint32_t tot = 0;
#pragma unroll
      for (int j = 0; j < 8; ++j) {
        c[j] = hist[255 - (lane * 8 + j)];  // descending bin order
        tot += c[j];
      }
      uint32_t incl = tot;
#pragma unroll
      for (int o = 1; o < 32; o <<= 1) {
        const uint32_t v = __shfl_up_sync(0xffffffffu, incl, o);
        if (lane >= o) incl += v;
      }
      uint32_t before = incl - tot;  // elements in bins above this lane's 8 bins
      if (before < need && need <= incl) {
#pragma unroll
        for (int j = 0; j < 8; ++j) {
          if (need <= before + c[j]) {
            sh[0] = 255u - (uint32_t)(lane * 8 + j);
            sh[1] = need - before;
            break;
          }
          before += c[j];
        }
      }
    }
    __syncthreads();
    prefix |= sh[0] << shift;
    need = sh[1];
    __syncthreads();
  }
  const uint32_t T = prefix;
  const uint32_t need_eq = need;  // >= 1

  // ---- index-ordered compaction ----
  uint32_t run_gt = 0, run_eq = 0;  // totals of earlier chunks
  uint32_t* wsum = sh + 2;          // [2 * TOPK_WARPS]
  for (int i0 = 0; i0 < n; i0 += TOPK_THREADS) {
    const int i = i0 + tid;
    bool gt = false, eq = false;
    if (i < n) {
      const uint32_t key = load_key<CACHED>(x, keys, i);
      gt = key > T;
      eq = key == T;
    }
    const uint32_t mg = __ballot_sync(0xffffffffu, gt), me = __ballot_sync(0xffffffffu, eq);
    const uint32_t lt = (1u << lane) - 1u;
    if (lane == 0) {
      wsum[warp] = __popc(mg);
      wsum[TOPK_WARPS + warp] = __popc(me);
    }
    __syncthreads();
    uint32_t bg = run_gt, be = run_eq, tg = 0, te = 0;
#pragma unroll
    for (int w = 0; w < TOPK_WARPS; ++w) {
      const uint32_t a = wsum[w], b = wsum[TOPK_WARPS + w];
      if (w < warp) { bg += a; be += b; }
      tg += a;
      te += b;
    }
    const uint32_t my_gt = bg + __popc(mg & lt);
    const uint32_t my_eq = be + __popc(me & lt);
    if (gt || (eq && my_eq < need_eq)) out[my_gt + min(my_eq, need_eq)] = seq_start + i;
    run_gt += tg;
    run_eq += te;
    __syncthreads();
    if (run_eq >= need_eq && run_gt + need_eq >= (uint32_t)k) break;  // uniform: all k slots written
  }
}

__global__ void __launch_bounds__(TOPK_THREADS)
sp_topk_kernel(SpGeom g, const float* __restrict__ scores, int64_t ld, int row_begin, int k,
               int32_t* __restrict__ idx, int32_t* __restrict__ cnt) {
  extern __shared__ uint32_t keys[];
  __shared__ uint32_t hist[256];
  __shared__ uint32_t sh[2 + 2 * TOPK_WARPS];
  const int r = blockIdx.x;
  const SpRow ri = sp_row_info(g, row_begin + r);
  const int n = ri.t_last + 1;
  int32_t* out = idx + (size_t)r * k;
  const int keep = min(n, k);
  if (threadIdx.x == 0 && cnt) cnt[r] = keep;
  for (int j = keep + threadIdx.x; j < k; j += TOPK_THREADS) out[j] = -1;
  if (n <= k) {
    for (int j = threadIdx.x; j < n; j += TOPK_THREADS) out[j] = ri.seq_start + j;
    return;
  }
  const float* x = scores + (size_t)r * ld;
  if (n <= TOPK_SMEM_FLOATS) topk_row<true>(x, keys, n, k, ri.seq_start, out, hist, sh);
  else topk_row<false>(x, keys, n, k, ri.seq_start, out, hist, sh);
}

}  // namespace

cudaError_t sp_launch_topk(const SpGeom& g, const float* scores, int64_t ld, int row_begin, int row_count, int k,
                           int32_t* idx, int32_t* cnt, cudaStream_t st) {
  static bool attr_done = false;
  const size_t smem = (size_t)TOPK_SMEM_FLOATS * sizeof(uint32_t);
  if (!attr_done) {
    cudaError_t e = cudaFuncSetAttribute(sp_topk_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    attr_done = true;
  }
  if (row_count <= 0) return cudaSuccess;
  sp_topk_kernel<<<row_count, TOPK_THREADS, smem, st>>>(g, scores, ld, row_begin, k, idx, cnt);
  sp_count_launch();
  return cudaGetLastError();
}
