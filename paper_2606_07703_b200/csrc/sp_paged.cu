// sp_paged.cu -- paged KV cache plumbing of the chunked-prefill path (stage 4 of the five-stage serving
// path: "reconstruct K/V from the paged KV cache when the chunked path requires contiguous tensors"; :331, :428
// chunks of max_num_batched_tokens queries against the cached prefix).
//   append : a chunk writes its own K, V and indexer keys into the pages its block table names;
//   gather : pages -> contiguous rows (the paper's reconstruction; the attention / scoring kernels of this library
//            read the pages THROUGH the block table instead and never need it -- kept as the stated stage and for tests).
// Pure data movement, 16 bytes per thread and step, grid sized to the machine: HBM-bound by construction.
#include "sp_common.cuh"

namespace {

// rows[t - t_begin, :] <-> pool[bt[t / ps] * ps + t % ps, :], row_chunks = 16-byte chunks per row
template <bool TO_PAGES>
__global__ void __launch_bounds__(256)
sp_paged_copy_kernel(uint4* __restrict__ pool, uint4* __restrict__ rows, const int32_t* __restrict__ bt,
                     int page_shift, int row_chunks, int t_begin, long long n_chunks) {
  const long long stride = (long long)gridDim.x * blockDim.x;
  for (long long e = (long long)blockIdx.x * blockDim.x + threadIdx.x; e < n_chunks; e += stride) {
    const int r = (int)(e / row_chunks), c = (int)(e % row_chunks);
    const int t = t_begin + r;
    const long long slot = ((long long)__ldg(bt + (t >> page_shift)) << page_shift) | (t & ((1 << page_shift) - 1));
    if (TO_PAGES) pool[slot * row_chunks + c] = rows[(long long)r * row_chunks + c];
    else rows[(long long)r * row_chunks + c] = pool[slot * row_chunks + c];
  }
}

}  // namespace

cudaError_t sp_launch_paged_copy(bool to_pages, void* pool, void* rows, const int32_t* bt, int page_shift,
                                 long long row_bytes, int t_begin, int t_count, cudaStream_t st) {
  if (t_count <= 0) return cudaSuccess;
  const int row_chunks = (int)(row_bytes / 16);
  const long long n = (long long)t_count * row_chunks;
  long long blocks = (n + 255) / 256;
  const long long cap = (long long)sp_sm_count() * 8;
  if (blocks > cap) blocks = cap;
  if (to_pages)
    sp_paged_copy_kernel<true><<<(unsigned)blocks, 256, 0, st>>>((uint4*)pool, (uint4*)rows, bt, page_shift, row_chunks,
                                                                t_begin, n);
  else
    sp_paged_copy_kernel<false><<<(unsigned)blocks, 256, 0, st>>>((uint4*)pool, (uint4*)rows, bt, page_shift, row_chunks,
                                                                 t_begin, n);
  sp_count_launch();
  return cudaGetLastError();
}
