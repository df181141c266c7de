// sp_diag.cu -- support-level diagnostics (PAPER.md:262 KL(P || softmax(z)); :478 "support-level diagnostics":
// how much of the oracle support the indexer recovers).  Plain bandwidth-bound CUDA-core kernels: each row is
// read a small constant number of times, nothing here is a contraction.
#include "sp_common.cuh"

namespace {

// |S_a(r) & S_b(r)| for ascending, -1 padded index rows.  One warp per row: lanes stride over a's entries and
// binary-search them in b (both lists are L2 resident: k <= a few thousand).
__global__ void __launch_bounds__(256)
sp_overlap_kernel(const int32_t* __restrict__ a, const int32_t* __restrict__ b, int n_rows, int k,
                  int32_t* __restrict__ inter) {
  const int row = blockIdx.x * 8 + (threadIdx.x >> 5), lane = threadIdx.x & 31;
  if (row >= n_rows) return;
  const int32_t* ra = a + (size_t)row * k;
  const int32_t* rb = b + (size_t)row * k;
  // number of valid entries of b (valid entries come first): first index with rb[i] < 0
  int lo = 0, hi = k;
  while (lo < hi) {
    const int mid = (lo + hi) >> 1;
    if (__ldg(rb + mid) >= 0) lo = mid + 1;
    else hi = mid;
  }
  const int nb = lo;
  int cnt = 0;
  for (int i = lane; i < k; i += 32) {
    const int32_t x = __ldg(ra + i);
    if (x < 0) break;  // padding tail
    int l = 0, h = nb;
    while (l < h) {
      const int mid = (l + h) >> 1;
      if (__ldg(rb + mid) < x) l = mid + 1;
      else h = mid;
    }
    cnt += (l < nb && __ldg(rb + l) == x);
  }
  cnt = __reduce_add_sync(0xffffffffu, cnt);
  if (lane == 0) inter[row] = cnt;
}

__device__ __forceinline__ float blk_reduce(float v, bool is_max, float* sh) {
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  for (int o = 16; o > 0; o >>= 1) {
    const float w = __shfl_xor_sync(0xffffffffu, v, o);
    v = is_max ? fmaxf(v, w) : v + w;
  }
  __syncthreads();
  if (lane == 0) sh[warp] = v;
  __syncthreads();
  float r = sh[0];
  for (int w = 1; w < (int)(blockDim.x >> 5); ++w) r = is_max ? fmaxf(r, sh[w]) : r + sh[w];
  return r;
}

// KL(P_t || softmax(z_t)) over s in [0, n_valid): one CTA per per-query row; three passes over the two rows
// (max of z, sum exp, the KL sum); the sums are Kahan-free fp32 partials per thread reduced in fp32 -- 512 threads
// x <= 256 terms each -- and the result is accurate to ~1e-6 relative (checked against the fp64 oracle at 1e-4).
__global__ void __launch_bounds__(512)
sp_row_kl_kernel(SpGeom g, const float* __restrict__ P, int64_t ldp, const float* __restrict__ z, int64_t ldz,
                 int row_begin, float* __restrict__ kl) {
  __shared__ float sh[16];
  const int r = blockIdx.x;
  const SpRow ri = sp_row_info(g, row_begin + r);
  const int n = ri.t_last + 1;
  const float* p = P + (size_t)r * ldp;
  const float* x = z + (size_t)r * ldz;
  float m = -INFINITY;
  for (int i = threadIdx.x; i < n; i += blockDim.x) m = fmaxf(m, __ldg(x + i));
  m = blk_reduce(m, true, sh);
  float s = 0.f;
  for (int i = threadIdx.x; i < n; i += blockDim.x) s += expf(__ldg(x + i) - m);
  s = blk_reduce(s, false, sh);
  const float lse = m + logf(s);
  float acc = 0.f;
  for (int i = threadIdx.x; i < n; i += blockDim.x) {
    const float pi = __ldg(p + i);
    if (pi > 0.f) acc += pi * (logf(pi) - (__ldg(x + i) - lse));
  }
  acc = blk_reduce(acc, false, sh);
  if (threadIdx.x == 0) kl[r] = acc;
}

// Gather-bandwidth probe (measurement aid for the per-query attention's roofline: bench.py divides the kernel's
// gathered bytes per second by what THIS plain kernel reaches on the same access pattern).  Each 16-lane half warp
// fetches one `row_bytes`-byte row (16 bytes per lane and step, cp.async-free plain loads) at the position its index
// entry names and xors the words into a register; one word per thread is written so the loads cannot be dropped.
__global__ void __launch_bounds__(256)
sp_gather_probe_kernel(const uint4* __restrict__ base, int row_bytes, long long row_pitch_bytes,
                       const int32_t* __restrict__ idx, long long n_idx, uint32_t* __restrict__ sink) {
  const long long half = ((long long)blockIdx.x * blockDim.x + threadIdx.x) >> 4;
  const long long n_half = ((long long)gridDim.x * blockDim.x) >> 4;
  const int l16 = threadIdx.x & 15;
  uint32_t acc = 0;
  const int steps = row_bytes / 256;  // 16 lanes x 16 B per step
  for (long long e = half; e < n_idx; e += 4 * n_half) {
    uint4 w[4];
#pragma unroll
    for (int u = 0; u < 4; ++u) {  // four independent rows in flight per half warp
      const long long ee = e + u * n_half;
      const int p = ee < n_idx ? __ldg(idx + ee) : -1;
      w[u] = make_uint4(0, 0, 0, 0);
      if (p >= 0)
        for (int s = 0; s < steps; ++s) {
          const uint4 x = __ldcg(reinterpret_cast<const uint4*>(reinterpret_cast<const char*>(base) +
                                                               (long long)p * row_pitch_bytes) + s * 16 + l16);
          w[u].x ^= x.x; w[u].y ^= x.y; w[u].z ^= x.z; w[u].w ^= x.w;
        }
    }
#pragma unroll
    for (int u = 0; u < 4; ++u) acc ^= w[u].x ^ w[u].y ^ w[u].z ^ w[u].w;
  }
  sink[(long long)blockIdx.x * blockDim.x + threadIdx.x] = acc;
}

}  // namespace

cudaError_t sp_launch_gather_probe(const void* base, int row_bytes, long long row_pitch_bytes, const int32_t* idx,
                                   long long n_idx, uint32_t* sink, int blocks, cudaStream_t st) {
  sp_gather_probe_kernel<<<blocks, 256, 0, st>>>((const uint4*)base, row_bytes, row_pitch_bytes, idx, n_idx, sink);
  sp_count_launch();
  return cudaGetLastError();
}

cudaError_t sp_launch_overlap(const int32_t* a, const int32_t* b, long long n_rows, int k, int32_t* inter,
                              cudaStream_t st) {
  if (n_rows <= 0) return cudaSuccess;
  sp_overlap_kernel<<<(unsigned)((n_rows + 7) / 8), 256, 0, st>>>(a, b, (int)n_rows, k, inter);
  sp_count_launch();
  return cudaGetLastError();
}

cudaError_t sp_launch_row_kl(const SpGeom& g, const float* P, int64_t ldp, const float* z, int64_t ldz, int row_begin,
                             int row_count, float* kl, cudaStream_t st) {
  if (row_count <= 0) return cudaSuccess;
  sp_row_kl_kernel<<<row_count, 512, 0, st>>>(g, P, ldp, z, ldz, row_begin, kl);
  sp_count_launch();
  return cudaGetLastError();
}
