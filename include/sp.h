/*
 * sp.h -- C ABI of the B200 (sm_100a) sparse-prefill library: one causal GQA layer of
 * "oracle-guided sparse prefill" (arxiv/paper_2606_07703; citations are /root/reference/PAPER.md lines).
 *
 *   score -> causal top-k -> (optional) query-block-shared support -> gather-sparse GQA attention
 *
 * Conventions that hold for EVERY entry point
 *  - Pointers are DEVICE pointers unless the comment says HOST.  The caller owns every buffer, the
 *    workspace and the stream.  The library allocates no device memory, never synchronises the device
 *    and enqueues all work on `stream` (a cudaStream_t passed as void*).  Inputs are read-only.
 *  - sp_params is read on the host at call time.
 *  - Layouts (row-major, base pointers 16-byte aligned, bf16 = IEEE bfloat16 bit patterns):
 *      Q [L,Hq,d]   K,V [L,Hkv,d]   O [L,Hq,d]   X [L,hidden]   Wqi,Wki [hidden,d_idx]
 *      q_idx,k_idx [L,d_idx]   lse [L,Hq] fp32 (natural log)
 *    Query head h reads KV head g(h) = h / (Hq/Hkv)  (contiguous groups).
 *  - Positions are 0-based; query t may attend keys s <= t of ITS OWN sequence.
 *    With cu_seqlens the L tokens are a pack of `batch` sequences; every s, t, block and n_valid below is
 *    local to its sequence, while emitted indices are PACKED positions (local + cu_seqlens[i]).
 *  - Support rows: per sequence of length n, b_sel==1 gives n rows (row = query);
 *    b_sel>1 gives ceil(n/b_sel) rows, block j = local positions [j*b_sel, min((j+1)*b_sel, n)) (blocks
 *    never straddle sequences; the last may be ragged).  Rows of all sequences are concatenated in order.
 *    n_valid(row) = last local position of the row + 1.
 *  - Score matrices (`scores`, `mass`) are fp32, one row per support row of the requested panel
 *    [row_begin, row_begin+row_count), leading dimension ld >= max n_valid of the panel, column = key
 *    position local to the row's sequence.  Columns >= n_valid(row) are NOT written and never read.
 *  - Optional banded logit term (reading A20): when local_window > 0, local_bias is added to the
 *    scaled logit wherever 0 <= t-s < local_window, in every stage that forms a causal logit.
 *  - One library instance may be used on several devices of a process (the caller selects the device with
 *    cudaSetDevice before the call, as for any stream-ordered work); per-device function attributes and SM counts are
 *    cached per device.  There are no environment-variable switches.
 *  - Return value: SP_OK (0) or a negative sp_status.  On any error nothing has been launched.  No
 *    exceptions cross this ABI and nothing aborts.  There is no CPU fallback.
 */
#ifndef SP_H_
#define SP_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef enum sp_status {
  SP_OK = 0,
  SP_ERR_INVALID_ARG = -1, /* null / misaligned pointer, nonpositive size, Hq % Hkv, bad cu_seqlens, bad panel */
  SP_ERR_UNSUPPORTED = -2, /* shape outside the built set (d not in {64,128}: the Qwen3.5 head dim 256 / d_idx 256 rows of
                              PAPER.md:280 are NOT built; Hq/Hkv not in {1,2,4,8}; unknown flag bits ...)              */
  SP_ERR_WORKSPACE = -3,   /* workspace too small (see sp_workspace_bytes)                                      */
  SP_ERR_CUDA = -4,        /* a CUDA launch / API error; text via sp_strerror                                   */
  SP_ERR_TOO_LARGE = -5    /* the problem needs more scratch than a no-allocation entry point's fixed array holds */
} sp_status;

typedef enum sp_mode {
  SP_MODE_ORACLE = 0, /* support from dense attention mass  (Alg.1)  */
  SP_MODE_INDEXER = 1 /* support from the head-collapsed indexer (Alg.2) */
} sp_mode;

typedef enum sp_stage {
  SP_STAGE_INDEXER_SCORES = 0,
  SP_STAGE_ORACLE_MASS = 1,
  SP_STAGE_TOPK = 2,
  SP_STAGE_SPARSE_ATTN = 3,
  SP_STAGE_DENSE_ATTN = 4,
  SP_STAGE_LAYER_ORACLE = 5,
  SP_STAGE_LAYER_INDEXER = 6
} sp_stage;

/* The paper's problem statement for one layer call (PAPER.md:90-107 S,Hq,Hkv,g,d_h,k; :101-103,:178 b_sel;
 * :270-274 d_idx). */
typedef struct sp_params {
  int32_t batch;                  /* sequences in the pack; 1 when cu_seqlens == NULL                     */
  int32_t L;                      /* total packed tokens, >= 1                                            */
  const int32_t *cu_seqlens;      /* DEVICE ptr [batch+1], cu[0]=0, cu[batch]=L; NULL = one sequence      */
  const int32_t *cu_seqlens_host; /* HOST copy of the same array (needed iff cu_seqlens != NULL)          */
  int32_t Hq, Hkv, d;             /* Hq % Hkv == 0, Hq/Hkv in {1,2,4,8}; d in {64,128}                    */
  int32_t k;                      /* budget per support row, >= 1 */
  int32_t b_sel;                  /* 1 = per-query support; >1 = one support per b_sel queries            */
  int32_t hidden, d_idx;          /* indexer sizes; d_idx in {64,128}, hidden % 64 == 0 (indexer mode)    */
  float scale;                    /* attention scale; 0 -> 1/sqrt(d) */
  float idx_scale;                /* indexer scale;   0 -> 1/sqrt(d_idx) */
  int32_t local_window;           /* 0 = off                                                              */
  float local_bias;               /* added to the scaled logit when 0 <= t-s < local_window               */
  uint32_t flags;                 /* SP_F_* below; 0 = the plain scorer BASELINE.json configs 2-5 define       */
} sp_params;

/* The served scorer of PAPER.md:268-274 / Alg.2 steps 3-4 (indexer mode only; needs the tcgen05 paths, i.e.
 * b_sel in {1,32,64,128}, else SP_ERR_UNSUPPORTED).  Readings where the paper is silent: DESIGN.md A26-A28.
 *   SP_F_KEY_LN : k_idx = LayerNorm(X Wki) over the d_idx channels of a token (no affine, biased variance, eps 1e-6)
 *   SP_F_ROPE   : rotary embedding of q_idx and (after the LayerNorm) k_idx, rotate-half pairing (i, i + d_idx/2),
 *                 theta_i = pos * 10000^(-2i/d_idx), pos local to the sequence
 *   SP_F_RELU   : z = max(idx_scale <q_idx, k_idx> + local term, 0)
 * KEY_LN and ROPE act in the projection (q_idx / k_idx come out transformed, rounded once to bf16; with
 * preprojected = 1 the caller's tensors are taken as already transformed); RELU acts in the score epilogue. */
enum { SP_F_RELU = 1u, SP_F_KEY_LN = 2u, SP_F_ROPE = 4u, SP_F_GROUP_SUPPORT = 8u, SP_F_HEAD_SUPPORT = 16u };
/* Support granularity on the HEAD axis ("shared within each KV group S_{l,t,r}" / "separately per query
 * head S_{l,t,h}"; the paper evaluates neither, :133, :137; A29).  Default (neither bit): ONE head-averaged list
 * per support row.
 *   SP_F_GROUP_SUPPORT: one list per KV group; index tensors are [Hkv, n_rows, k]; group r's mass is the mean over ITS
 *     G = Hq/Hkv query heads, P_r[t,s] = (1/G) sum_{g(h)=r} A[t,h,s].
 *   SP_F_HEAD_SUPPORT : one list per query head; index tensors are [Hq, n_rows, k]; head h's mass is A[t,h,s] itself.
 * Everything else (block max, top-k, tie rule, recompute) is the head-averaged definition on the sub-problem.  The bits
 * are read by sp_sparse_gqa_attn (layout of idx) and by sp_prefill_layer in SP_MODE_ORACLE (which then selects Hkv or Hq
 * lists from ONE pass 1 and attends with them); every other entry point returns SP_ERR_UNSUPPORTED when one is set, and
 * both together are SP_ERR_INVALID_ARG.  Per-head lists leave no two heads a shared gathered row, so the attention runs
 * on the per-query kernel's tile shape for every b_sel. */

/* Number of support rows of the whole pack (host arithmetic only). Returns < 0 on invalid params. */
int64_t sp_num_rows(const sp_params *p);

/* Bytes of workspace `stage` (an sp_stage) needs for these params; written to *bytes_out.
 * For the two LAYER stages the figure includes the score panel and the index buffer. */
int sp_workspace_bytes(const sp_params *p, int stage, size_t *bytes_out);

/* Indexer support-row scores (PAPER.md:270 projections, :274 scaled similarity -- plain when flags == 0, with the
 * key LayerNorm / RoPE / ReLU of the served scorer when the SP_F_* flags ask for them --, :299 max-aggregate over
 * each b_sel block; Alg.2 steps 2-4).
 *   preprojected == 0: q_idx = bf16(X Wqi), k_idx = bf16(X Wki) are computed for ALL L tokens (fp32
 *     accumulate, one round-to-nearest-even to bf16) and written to q_idx / k_idx (outputs, [L,d_idx]).
 *   preprojected != 0: X, Wqi, Wki are ignored (may be NULL); q_idx / k_idx are inputs.
 *   scores[r - row_begin, s] = max over queries t of support row r with s <= t of
 *       idx_scale * <q_idx[t], k_idx[s]> (+ local term),  s in [0, n_valid(r)).       fp32, never rounded to bf16. */
int sp_indexer_scores(const sp_params *p, const void *X, const void *Wqi, const void *Wki,
                      void *q_idx, void *k_idx, int32_t preprojected,
                      int32_t row_begin, int32_t row_count, float *scores, int64_t ld_scores,
                      void *ws, size_t ws_bytes, void *stream);

/* Attention-mass support-row scores (PAPER.md:123 P_t(s) = (1/Hq) sum_h A[t,h,s]; :154 block max; Alg.1
 * steps 2-3).  Pass 1 computes the per-(t,h) softmax normaliser as a log-sum-exp over s <= t; pass 2
 * rebuilds the probabilities and averages them over ALL Hq query heads.
 *   lse: [L,Hq] fp32.  lse_ready == 0: pass 1 runs for every query of the panel and writes lse (output;
 *        may be NULL, then it lives in the workspace).  lse_ready != 0: lse is an input (e.g. from
 *        sp_dense_gqa_attn) and pass 1 is skipped.
 *   mass[r - row_begin, s] = max over queries t of row r with s <= t of P_t(s),  s in [0, n_valid(r)). */
int sp_oracle_mass(const sp_params *p, const void *Q, const void *K, float *lse, int32_t lse_ready,
                   int32_t row_begin, int32_t row_count, float *mass, int64_t ld_mass,
                   void *ws, size_t ws_bytes, void *stream);

/* The same for ONE KV group ("shared within each KV group S_{l,t,r}"; A29): pass 2
 * averages over the G = Hq/Hkv query heads h with g(h) = group only, P_r[t,s] = (1/G) sum_{g(h)=r} A[t,h,s].
 * Every other argument as for sp_oracle_mass; lse is still the [L,Hq] array of ALL heads, so one pass 1
 * (lse_ready == 0 on the first group) serves the Hkv calls.  Followed by sp_topk_support on the panel this
 * gives group r's list, and Hkv such lists, stacked as idx [Hkv, n_rows, k], are what sp_sparse_gqa_attn
 * reads under SP_F_GROUP_SUPPORT.  group outside [0,Hkv) -> SP_ERR_INVALID_ARG; shapes outside the tcgen05
 * mass kernel's set (b_sel in {1,32,64,128}, d in {64,128}) -> SP_ERR_UNSUPPORTED. */
int sp_oracle_mass_group(const sp_params *p, const void *Q, const void *K, float *lse, int32_t lse_ready,
                         int32_t group, int32_t row_begin, int32_t row_count, float *mass, int64_t ld_mass,
                         void *ws, size_t ws_bytes, void *stream);
/* The same for ONE query head ("separately per query head S_{l,t,h}"): mass = A[t,head,s] (block max for
 * b_sel > 1).  head outside [0,Hq) -> SP_ERR_INVALID_ARG. */
int sp_oracle_mass_head(const sp_params *p, const void *Q, const void *K, float *lse, int32_t lse_ready,
                        int32_t head, int32_t row_begin, int32_t row_count, float *mass, int64_t ld_mass,
                        void *ws, size_t ws_bytes, void *stream);

/* Causal top-k of each support row of the panel (PAPER.md:127 TopK_s(P,k); :145 sentinel padding; :156
 * causally invalid positions masked before selection).  Row r ranks columns [0, n_valid(r)) of
 * scores[r - row_begin, :]; the kept set is the first min(k, n_valid) elements of the order
 * (score descending, index ascending) -- ties go to the lower index.
 *   idx: [row_count, k] int32 packed positions, ascending, tail padded with -1.
 *   cnt: [row_count] int32 = min(k, n_valid(r)); may be NULL. */
int sp_topk_support(const sp_params *p, const float *scores, int64_t ld_scores,
                    int32_t row_begin, int32_t row_count, int32_t *idx, int32_t *cnt,
                    void *ws, size_t ws_bytes, void *stream);

/* GQA attention recomputed only over the selected KV positions, online softmax (PAPER.md:107; :156 each
 * query re-applies its own causal mask; Alg.1 step 5).
 *   idx: [sp_num_rows(p), k] as produced by sp_topk_support for the WHOLE pack (row of query t =
 *        its support row).  Entries < 0 or > t (or outside t's sequence) are ignored for query t, in any order;
 *        the valid entries of a row are a SET (distinct positions, as a top-k gives them).
 *   O: [L,Hq,d] bf16 (fp32 accumulate).  Empty effective support -> O row = 0, lse = -inf.
 *   lse: [L,Hq] fp32 or NULL.
 *   ws: optional.  For per-query lists (b_sel == 1) whose k is a sizeable part of the prefix the layer is cheaper as
 *        the dense tile loop over the whole causal prefix with a membership mask than as k gathered rows per query
 *        and KV head (the per-query realization is "harder to fuse and amortize").
 *        sp_workspace_bytes(SP_STAGE_SPARSE_ATTN) is non-zero exactly when that plan applies to p (Hq/Hkv in {4,8},
 *        d in {64,128}, scale > 0, no local bias, every sequence starting at a multiple of 32, causal pairs at most
 *        ~22x the kept pairs); with a workspace of that size the call takes it (device scratch, overwritten: a
 *        [L/32, L] bitmap), with ws == NULL or a smaller one it gathers.  Same result up to summation order. */
int sp_sparse_gqa_attn(const sp_params *p, const void *Q, const void *K, const void *V,
                       const int32_t *idx, void *O, float *lse, void *ws, size_t ws_bytes, void *stream);

/* sp_sparse_gqa_attn for callers that cannot allocate or pass scratch (CUDA graph capture, tight serving loops,
 * harnesses that forbid cudaMalloc): per-query lists (b_sel == 1) through the membership-masked tile loop (PAPER.md:107,
 * :156, :315-317) with its [L/32 + 8, L] bitmap in a FIXED device array inside the library, SP_STATIC_SCRATCH_BYTES
 * (8.25 MiB: every GPU that loads the library holds it until exit).  The call allocates nothing -- no cudaMalloc,
 * cudaFree or allocating library routine; it launches the bitmap builder (which first clears the part of the array it
 * uses) and the attention kernel on `stream`.
 *   Arguments as for sp_sparse_gqa_attn (device pointers; idx [sp_num_rows(p), k]; O [L,Hq,d] bf16; lse or NULL).
 *   L > SP_STATIC_MAX_TOKENS (8192)            -> SP_ERR_TOO_LARGE, nothing launched.
 *   p outside the masked tile loop's shape set (sp_workspace_bytes(p, SP_STAGE_SPARSE_ATTN) == 0), or a support-
 *   granularity flag set                        -> SP_ERR_UNSUPPORTED.
 *   Result: identical to sp_sparse_gqa_attn given the SPARSE_ATTN workspace.
 *   EVERY call on a device shares the one array, which keeps the last call's contents: two calls whose kernels
 *   overlap on the GPU (different streams, no dependency between them) race.  Calls on one stream are safe. */
#define SP_STATIC_MAX_TOKENS 8192
#define SP_STATIC_SCRATCH_BYTES (8192u * (8192u / 32u + 8u) * 4u)
int sp_sparse_gqa_attn_static(const sp_params *p, const void *Q, const void *K, const void *V,
                              const int32_t *idx, void *O, float *lse, void *stream);

/* Dense causal GQA attention of the same layer: the same-library baseline and pass 1 of
 * the attention mass.  O may be NULL (only lse is produced); lse may be NULL. */
int sp_dense_gqa_attn(const sp_params *p, const void *Q, const void *K, const void *V, void *O, float *lse,
                      void *ws, size_t ws_bytes, void *stream);

/* Support-level diagnostics (PAPER.md:478: "which part of the oracle support the indexer recovers"; :262 the
 * distillation objective evaluated forward only).  Not on the serving path; both are single bandwidth-bound passes.
 *   sp_support_overlap: inter[r] = |S_a(r) & S_b(r)| for two index tensors [sp_num_rows(p), k] in the layout
 *     sp_topk_support emits (ascending, -1 padded), e.g. the oracle-mode and the indexer-mode supports.
 *   sp_row_kl: kl[r - row_begin] = KL(P_t || softmax(z_t)) over the valid causal keys of per-query row r
 *     (b_sel must be 1: a block-max row is not a distribution); P = a mass panel, z = an indexer score panel of the
 *     SAME rows, fp32 with their own leading dimensions; terms with P = 0 contribute 0. */
int sp_support_overlap(const sp_params *p, const int32_t *idx_a, const int32_t *idx_b, int32_t *inter, void *stream);
int sp_row_kl(const sp_params *p, const float *mass, int64_t ld_mass, const float *scores, int64_t ld_scores,
              int32_t row_begin, int32_t row_count, float *kl, void *stream);

/* Measurement aid, not a step of the path: a plain gather of n_idx rows of row_bytes bytes (a multiple of 256) at
 * base + idx[e] * row_pitch_bytes (idx < 0 = skip), 16 bytes per lane, four rows in flight per half warp.  bench.py times
 * it on the per-query attention's own index stream to obtain the L2 / HBM gather bandwidth that path can be held
 * against (a per-query support row is used by only Hq/Hkv query rows: "harder to fuse and amortize").
 * sink: DEVICE scratch of >= 148 * 8 * 256 * 4 bytes (one word per probe thread). */
int sp_gather_probe(const void *base, int32_t row_bytes, int64_t row_pitch_bytes, const int32_t *idx, int64_t n_idx,
                    void *sink, size_t sink_bytes, void *stream);

/* One patched layer on one stream (PAPER.md:292 five-stage path without the paged-cache stage; Alg.1 steps
 * 2-5 in SP_MODE_ORACLE, Alg.2 steps 2,4,5 in SP_MODE_INDEXER).  Support rows are processed in panels so the
 * score workspace stays bounded.
 *   X, Wqi, Wki: indexer mode only (ignored in oracle mode).  O: [L,Hq,d] bf16.
 *   idx_out: [sp_num_rows(p), k] int32 or NULL (then the indices live in the workspace); with SP_F_GROUP_SUPPORT /
 *   SP_F_HEAD_SUPPORT (oracle mode) [Hkv or Hq, sp_num_rows(p), k], and sp_workspace_bytes(SP_STAGE_LAYER_ORACLE)
 *   accounts for those lists when the same flags are set in the params it is given. */
int sp_prefill_layer(const sp_params *p, int32_t mode, const void *X, const void *Wqi, const void *Wki,
                     const void *Q, const void *K, const void *V, void *O, int32_t *idx_out,
                     void *ws, size_t ws_bytes, void *stream);

/* ------------------------------------------------------------------------------------------------------------------
 * Chunked prefill against a paged KV cache (stage 4 of the five-stage serving path: "reconstruct K/V from
 * the paged KV cache when the chunked path requires contiguous tensors"; :331 and :428: the GPU TTFT rows run with
 * max_num_batched_tokens = 4K / 8K query chunks against the whole cached prefix).  DESIGN.md reading A30.
 *
 * The cache of ONE sequence: three page pools and a block table.  Logical token t lives in page block_table[t / page_size]
 * at slot t % page_size; a pool row is one token ([Hkv, d] bf16 for K and V, [d_idx] bf16 for the indexer keys).
 * Pools and table are caller-owned DEVICE memory; the library writes only the slots of the tokens it is asked to append. */
typedef struct sp_kv_pages {
  void *k_pages;              /* [n_pages, page_size, Hkv, d] bf16                                              */
  void *v_pages;              /* [n_pages, page_size, Hkv, d] bf16                                              */
  void *kidx_pages;           /* [n_pages, page_size, d_idx]  bf16 (transformed indexer keys, A14/A27/A28)      */
  const int32_t *block_table; /* [n_blocks] physical page of logical block i; n_blocks * page_size >= p->L      */
  int32_t n_blocks;
  int32_t page_size;          /* a power of two in [16, 4096]                                                   */
  int32_t n_pages;
} sp_kv_pages;

/* Append / reconstruct: rows of tokens [t_begin, t_begin + t_count) <-> their page slots.  K / V rows are [Hkv, d], kidx
 * rows [d_idx]; any of the three row pointers may be NULL (skipped).  sp_kv_gather is the paper's stage 4 as stated;
 * sp_prefill_chunk itself never needs it -- its kernels read the pages through the block table. */
int sp_kv_append(const sp_params *p, const sp_kv_pages *kv, int32_t t_begin, int32_t t_count, const void *K_new,
                 const void *V_new, const void *kidx_new, void *stream);
int sp_kv_gather(const sp_params *p, const sp_kv_pages *kv, int32_t t_begin, int32_t t_count, void *K_out, void *V_out,
                 void *kidx_out, void *stream);

/* One prefill CHUNK of one sequence, indexer mode (Alg.2 steps 2,4,5 for the queries [q_begin, q_begin + q_count)):
 *   p->L = q_begin + q_count is the context length after the chunk; p->batch = 1, no cu_seqlens; q_begin must be a
 *   multiple of b_sel (selection blocks stay aligned to the sequence start); b_sel in {1,32,64,128}.
 *   X [q_count, hidden], Q [q_count, Hq, d], K_new / V_new [q_count, Hkv, d], O [q_count, Hq, d]: the CHUNK's rows only.
 *   The first q_begin tokens must already be in the cache (earlier chunks).  The call (1) projects the chunk (rotary
 *   positions q_begin ...), (2) appends K_new, V_new and the chunk's indexer keys to the cache, (3) scores the chunk's
 *   support rows against all p->L cached indexer keys, (4) selects top-k, (5) runs the gather-sparse attention over the
 *   paged K / V.  Results equal sp_prefill_layer on the whole sequence, bit for bit, for the chunk's queries.
 *   idx_out: [ceil(q_count / b_sel), k] (the chunk's support rows) or NULL.  Workspace: sp_chunk_workspace_bytes. */
int sp_chunk_workspace_bytes(const sp_params *p, int32_t q_begin, int32_t q_count, size_t *bytes_out);
int sp_prefill_chunk(const sp_params *p, int32_t q_begin, int32_t q_count, const void *X, const void *Wqi,
                     const void *Wki, const void *Q, const void *K_new, const void *V_new, const sp_kv_pages *kv,
                     void *O, int32_t *idx_out, void *ws, size_t ws_bytes, void *stream);

/* Same as sp_prefill_layer but X, Wqi, Wki, Q, K, V and O are HOST pointers (pinned memory recommended).
 * `dev_arena` is DEVICE scratch of at least sp_layer_host_arena_bytes() bytes that receives the inputs, the
 * output and the workspace.  Copies are enqueued on `stream` (cudaMemcpyAsync); O_host is valid once the
 * stream has been synchronised by the caller. */
int sp_layer_host_arena_bytes(const sp_params *p, int32_t mode, size_t *bytes_out);
int sp_prefill_layer_host(const sp_params *p, int32_t mode, const void *X_host, const void *Wqi_host,
                          const void *Wki_host, const void *Q_host, const void *K_host, const void *V_host,
                          void *O_host, void *dev_arena, size_t arena_bytes, void *stream);

/* Text for a status code; for SP_ERR_CUDA it includes the last CUDA error string seen by this library. */
const char *sp_strerror(int code);

/* Number of kernel launches this library has enqueued since load (for bench.py's gpu_launches). */
int64_t sp_launch_count(void);

#ifdef __cplusplus
}
#endif
#endif /* SP_H_ */
