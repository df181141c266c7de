// sp_api.cu -- the C ABI declared in include/sp.h: argument validation, workspace carving, panel
// loops and stage chaining.  No device memory is allocated here and the device is never synchronised.
#include <atomic>
#include <cmath>
#include <cstdio>
#include <cstring>
#include <mutex>

#include <cstdlib>

#include "sp_common.cuh"

namespace {

std::atomic<long long> g_launches{0};
std::mutex g_err_mu;
char g_err_text[512] = "no CUDA error recorded";

int cuda_fail(cudaError_t e, const char* where) {
  std::lock_guard<std::mutex> lk(g_err_mu);
  snprintf(g_err_text, sizeof(g_err_text), "SP_ERR_CUDA: %s: %s (%s)", where, cudaGetErrorName(e),
           cudaGetErrorString(e));
  return SP_ERR_CUDA;
}
#define SP_CUDA(call, where)                         \
  do {                                               \
    cudaError_t e__ = (call);                        \
    if (e__ != cudaSuccess) return cuda_fail(e__, where); \
  } while (0)

inline size_t align_up(size_t x, size_t a = 256) { return (x + a - 1) / a * a; }
inline bool aligned16(const void* p) { return (reinterpret_cast<uintptr_t>(p) & 15u) == 0; }

struct HostGeom {
  int batch, L, b;
  const int32_t* cu;  // host or nullptr
  int seq_start(int i) const { return cu ? cu[i] : 0; }
  int seq_len(int i) const { return cu ? cu[i + 1] - cu[i] : L; }
  int rows_of(int n) const { return (n + b - 1) / b; }
  long long num_rows() const {
    long long r = 0;
    for (int i = 0; i < batch; ++i) r += rows_of(seq_len(i));
    return r;
  }
  int max_seqlen() const {
    int m = 0;
    for (int i = 0; i < batch; ++i) m = seq_len(i) > m ? seq_len(i) : m;
    return m;
  }
  // max n_valid over support rows [row_begin, row_begin + row_count)
  int max_n_valid(long long row_begin, long long row_count) const {
    long long r0 = 0;
    int best = 0;
    for (int i = 0; i < batch; ++i) {
      const int n = seq_len(i);
      const long long nr = rows_of(n);
      const long long lo = row_begin > r0 ? row_begin : r0;
      const long long hi = (row_begin + row_count < r0 + nr ? row_begin + row_count : r0 + nr) - 1;
      if (lo <= hi) {
        const long long j = hi - r0;  // last intersecting row of this sequence
        const long long nv = (j + 1) * b < n ? (j + 1) * b : n;
        if (nv > best) best = (int)nv;
      }
      r0 += nr;
    }
    return best;
  }
};

int validate_common(const sp_params* p, bool need_attn, bool need_indexer) {
  if (!p) return SP_ERR_INVALID_ARG;
  if (p->L < 1 || p->batch < 1 || p->k < 1 || p->b_sel < 1) return SP_ERR_INVALID_ARG;
  if (p->cu_seqlens) {
    if (!p->cu_seqlens_host) return SP_ERR_INVALID_ARG;
    const int32_t* cu = p->cu_seqlens_host;
    if (cu[0] != 0 || cu[p->batch] != p->L) return SP_ERR_INVALID_ARG;
    for (int i = 0; i < p->batch; ++i)
      if (cu[i + 1] <= cu[i]) return SP_ERR_INVALID_ARG;
  } else if (p->batch != 1) {
    return SP_ERR_INVALID_ARG;
  }
  if (p->flags & ~(uint32_t)(SP_F_RELU | SP_F_KEY_LN | SP_F_ROPE)) return SP_ERR_UNSUPPORTED;
  if (p->flags != 0 && !sp_tc_scores_supported(p->b_sel)) return SP_ERR_UNSUPPORTED;
  if (p->local_window < 0) return SP_ERR_INVALID_ARG;
  if (need_attn) {
    if (p->Hq < 1 || p->Hkv < 1 || p->d < 1 || p->Hq % p->Hkv != 0) return SP_ERR_INVALID_ARG;
    const int G = p->Hq / p->Hkv;
    if (!(p->d == 64 || p->d == 128)) return SP_ERR_UNSUPPORTED;
    if (!(G == 1 || G == 2 || G == 4 || G == 8)) return SP_ERR_UNSUPPORTED;
  }
  if (need_indexer) {
    if (p->hidden < 1 || p->d_idx < 1) return SP_ERR_INVALID_ARG;
    if (!(p->d_idx == 64 || p->d_idx == 128) || p->hidden % 64 != 0) return SP_ERR_UNSUPPORTED;
  }
  return SP_OK;
}

HostGeom host_geom(const sp_params* p) {
  return HostGeom{p->batch, p->L, p->b_sel, p->cu_seqlens ? p->cu_seqlens_host : nullptr};
}
SpGeom dev_geom(const sp_params* p) { return SpGeom{p->batch, p->L, p->cu_seqlens, p->b_sel, 0}; }
float attn_scale(const sp_params* p) { return p->scale != 0.f ? p->scale : 1.0f / sqrtf((float)p->d); }
float index_scale(const sp_params* p) { return p->idx_scale != 0.f ? p->idx_scale : 1.0f / sqrtf((float)p->d_idx); }

int validate_panel(const sp_params* p, int32_t row_begin, int32_t row_count, int64_t ld, int* max_nv) {
  const HostGeom hg = host_geom(p);
  const long long nr = hg.num_rows();
  if (row_begin < 0 || row_count < 0 || (long long)row_begin + row_count > nr) return SP_ERR_INVALID_ARG;
  *max_nv = hg.max_n_valid(row_begin, row_count);
  if (ld < *max_nv) return SP_ERR_INVALID_ARG;
  return SP_OK;
}

// ---- stage dispatch: tcgen05 kernels where the shape is in their built set; the CUDA-core kernels of sp_simt.cu
// only for selection blocks outside it (b_sel not in {1,32,64,128}) and for dense attention over a query sub-range ----
cudaError_t run_project(const sp_params* p, const void* X, const void* Wq, const void* Wk, void* q_idx, void* k_idx,
                        void* ws, cudaStream_t st) {
  (void)ws;
  return sp_launch_project_tc(dev_geom(p), p->flags, X, Wq, Wk, q_idx, k_idx, p->L, p->hidden, p->d_idx, st);
}

cudaError_t run_indexer_scores(const sp_params* p, const void* q_idx, const void* k_idx, int row_begin, int row_count,
                               int max_nv, float* scores, int64_t ld, cudaStream_t st) {
  const SpGeom g = dev_geom(p);
  if (sp_tc_scores_supported(p->b_sel))
    return sp_launch_indexer_scores_tc(g, p->cu_seqlens ? p->cu_seqlens_host : nullptr, q_idx, k_idx, p->d_idx,
                                       index_scale(p), p->local_window, p->local_bias, (p->flags & SP_F_RELU) ? 1 : 0,
                                       row_begin, row_count, max_nv, scores, ld, st);
  return sp_launch_indexer_scores(g, q_idx, k_idx, p->d_idx, index_scale(p), p->local_window, p->local_bias, row_begin,
                                  row_count, max_nv, scores, ld, st);
}

cudaError_t run_mass(const sp_params* p, const void* Q, const void* K, const float* lse, int row_begin, int row_count,
                     int max_nv, float* mass, int64_t ld, cudaStream_t st, int grp = -1, int head = -1) {
  const SpGeom g = dev_geom(p);
  if (sp_tc_mass_supported(p->b_sel, p->d))
    return sp_launch_mass_tc(g, p->cu_seqlens ? p->cu_seqlens_host : nullptr, Q, K, lse, p->Hq, p->Hkv, p->d,
                             attn_scale(p), p->local_window, p->local_bias, row_begin, row_count, mass, ld, st, grp, head);
  if (grp >= 0 || head >= 0) return cudaErrorNotSupported;  // callers check sp_tc_mass_supported first
  return sp_launch_mass(g, Q, K, lse, p->Hq, p->Hkv, p->d, attn_scale(p), p->local_window, p->local_bias, row_begin,
                        row_count, max_nv, mass, ld, st);
}

// ---- per-query supports: gather kernel or membership-masked dense tiles (sp_tc_attn.cu) ----
// The gather kernel moves k rows per query and KV head; the masked tile loop touches every (query, key <= query) pair
// once on the tensor core.  Measured on a B200 (c4: d = 128, G = 4, k = L/16 up to 2048): the gather kernel costs
// 350-405 ps per kept pair, the masked loop 14-15.5 ps per causal pair (L = 16K: 5.83 vs 1.88 ms; 32K: 23.0 vs 7.6 ms;
// 64K: 53.5 vs 33.2 ms), i.e. the masked loop wins while the causal pairs are fewer than ~25x the kept ones; at
// k = 2048 that is L below ~100K.  The threshold leaves a margin for the long runs' power cap.
constexpr double MASKED_PAIR_RATIO = 22.0;
constexpr size_t MASKED_MAX_BYTES = (size_t)3 << 30;

struct MaskedPlan {
  bool use;
  size_t bytes;
  long long chunks;
};

MaskedPlan masked_plan(const sp_params* p) {
  MaskedPlan m{false, 0, 0};
  if (p->b_sel != 1 || p->k < 1 || p->Hkv < 1) return m;
  const int G = p->Hq / p->Hkv;
  if (!sp_tc_attn_masked_supported(G, p->d)) return m;
  if (!(attn_scale(p) > 0.f)) return m;
  if (p->local_window > 0 && p->local_bias != 0.f) return m;  // the local bias needs the per-element path
  const HostGeom hg = host_geom(p);
  const int QT = 256 / G;
  double dense = 0.0, kept = 0.0;
  long long chunks = 0;
  for (int i = 0; i < hg.batch; ++i) {
    const long long s0 = hg.seq_start(i), n = hg.seq_len(i);
    if (s0 % 32 != 0) return m;  // a bitmap word holds 32 consecutive queries of ONE sequence
    const double nn = (double)n, kk = (double)(n < p->k ? n : p->k);
    dense += nn * (nn + 1.0) / 2.0;
    kept += kk * (kk + 1.0) / 2.0 + (nn - kk) * kk;
    chunks += (n + QT - 1) / QT;
  }
  if (dense > MASKED_PAIR_RATIO * kept) return m;
  long long pitch, rows;
  sp_support_bits_shape(p->L, &pitch, &rows);
  m.bytes = align_up((size_t)pitch * rows * sizeof(uint32_t));
  if (m.bytes > MASKED_MAX_BYTES) return m;
  m.chunks = chunks;
  m.use = true;
  return m;
}

// idx == nullptr -> dense.  The tcgen05 kernel covers the whole pack, or -- dense and LSE-only (O == nullptr,
// the oracle's pass 1 of a row panel) -- the query chunks that intersect [q_begin, q_begin + q_count): rows of a
// boundary chunk outside the range get their lse too, which is harmless.
cudaError_t run_attn(const sp_params* p, const void* Q, const void* K, const void* V, const int32_t* idx, int q_begin,
                     int q_count, void* O, float* lse, cudaStream_t st, long long idx_grp = 0, bool per_head = false,
                     void* ws = nullptr, size_t ws_bytes = 0) {
  SpGeom g = dev_geom(p);
  g.idx_grp = idx_grp;
  if (idx != nullptr && O != nullptr && !per_head && idx_grp == 0 && q_begin == 0 && q_count == p->L && ws != nullptr) {
    const MaskedPlan mp = masked_plan(p);
    if (mp.use && ws_bytes >= mp.bytes) {
      cudaError_t e = sp_launch_support_bits(g, idx, p->k, host_geom(p).num_rows(), (uint32_t*)ws, st);
      if (e != cudaSuccess) return e;
      return sp_launch_attn_tc_masked(g, mp.chunks, Q, K, V, (const uint32_t*)ws, p->Hq, p->Hkv, p->d, attn_scale(p), O, lse,
                                      st);
    }
  }
  if (per_head)  // one list per HEAD: no two heads share gathered rows, the per-query kernel's tile shape (G = 1 rows per warp)
    return sp_launch_attn_pq(g, Q, K, V, idx, p->k, p->Hq, p->Hkv, p->d, attn_scale(p), p->local_window, p->local_bias,
                             q_begin, q_count, O, lse, st, true);
  const int G = p->Hq / p->Hkv;
  const bool whole = q_begin == 0 && q_count == p->L;
  const bool dense_lse_range = idx == nullptr && O == nullptr && q_count > 0;
  if ((whole || dense_lse_range) && sp_tc_attn_supported(p->b_sel, G, idx != nullptr, p->k, p->d)) {
    const HostGeom hg = host_geom(p);
    const int QT = 256 / G;
    long long chunks = 0, c_lo = -1, c_hi = -1;
    const long long q_lo = q_begin, q_hi = (long long)q_begin + q_count - 1;
    for (int i = 0; i < hg.batch; ++i) {
      const long long s0 = hg.seq_start(i), n = hg.seq_len(i);
      const long long lo = q_lo > s0 ? q_lo : s0, hi = q_hi < s0 + n - 1 ? q_hi : s0 + n - 1;
      if (lo <= hi) {
        if (c_lo < 0) c_lo = chunks + (lo - s0) / QT;
        c_hi = chunks + (hi - s0) / QT;
      }
      chunks += (n + QT - 1) / QT;
    }
    if (idx != nullptr || whole) {
      c_lo = 0;
      c_hi = chunks - 1;
    }
    if (c_lo < 0) return cudaSuccess;
    return sp_launch_attn_tc(g, hg.num_rows(), c_hi - c_lo + 1, c_lo, Q, K, V, idx, p->k, p->Hq, p->Hkv, p->d,
                             attn_scale(p), p->local_window, p->local_bias, O, lse, st);
  }
  if (idx != nullptr)  // per-query / small-block supports: warp-level mma.sync + cp.async gathers
    return sp_launch_attn_pq(g, Q, K, V, idx, p->k, p->Hq, p->Hkv, p->d, attn_scale(p), p->local_window, p->local_bias,
                             q_begin, q_count, O, lse, st);
  return sp_launch_attn(g, Q, K, V, idx, p->k, p->Hq, p->Hkv, p->d, attn_scale(p), p->local_window, p->local_bias,
                        q_begin, q_count, O, lse, st);
}

// ---- workspace sizes ----
size_t ws_indexer(const sp_params* p) { return align_up((size_t)2 * p->hidden * p->d_idx * 2); }
size_t ws_mass(const sp_params* p) { return align_up((size_t)p->L * p->Hq * sizeof(float)); }

constexpr size_t PANEL_BYTES = (size_t)1 << 30;  // score panel budget inside sp_prefill_layer

struct LayerPlan {
  int64_t ld;
  long long n_rows, panel_rows;
  size_t off_qidx, off_kidx, off_lse, off_scores, off_idx, off_stage, total, scores_bytes;
};

LayerPlan plan_layer(const sp_params* p, int mode, bool idx_in_ws, int units = 1) {
  LayerPlan pl{};
  const HostGeom hg = host_geom(p);
  pl.n_rows = hg.num_rows();
  pl.ld = (int64_t)align_up((size_t)hg.max_seqlen(), 4);
  long long pr = (long long)(PANEL_BYTES / ((size_t)pl.ld * sizeof(float)));
  if (pr < 1) pr = 1;
  if (p->b_sel == 1 && pr >= 64) pr = pr / 64 * 64;
  if (pr > pl.n_rows) pr = pl.n_rows;
  pl.panel_rows = pr;
  size_t off = 0;
  if (mode == SP_MODE_INDEXER) {
    pl.off_qidx = off; off += align_up((size_t)p->L * p->d_idx * 2);
    pl.off_kidx = off; off += align_up((size_t)p->L * p->d_idx * 2);
    pl.off_stage = off; off += ws_indexer(p);
  } else {
    pl.off_lse = off; off += ws_mass(p);
  }
  pl.off_scores = off;
  {
    // the membership bitmap of the masked per-query attention (masked_plan) reuses the score panel, free by then
    size_t panel = align_up((size_t)pl.panel_rows * pl.ld * sizeof(float));
    if (units == 1) {
      const MaskedPlan mp = masked_plan(p);
      if (mp.use && mp.bytes > panel) panel = mp.bytes;
    }
    pl.scores_bytes = panel;
    off += panel;
  }
  pl.off_idx = off;
  if (idx_in_ws) off += align_up((size_t)units * pl.n_rows * p->k * sizeof(int32_t));
  pl.total = off;
  return pl;
}

// number of support lists per support row the layer call selects: 1, Hkv (SP_F_GROUP_SUPPORT) or Hq (SP_F_HEAD_SUPPORT);
// negative = an sp_status
int layer_units(const sp_params* p, int mode) {
  const uint32_t gf = p->flags & (SP_F_GROUP_SUPPORT | SP_F_HEAD_SUPPORT);
  if (gf == 0) return 1;
  if (gf == (SP_F_GROUP_SUPPORT | SP_F_HEAD_SUPPORT)) return SP_ERR_INVALID_ARG;
  if (mode != SP_MODE_ORACLE) return SP_ERR_UNSUPPORTED;
  if (p->Hq < 1 || p->Hkv < 1) return SP_ERR_INVALID_ARG;
  return gf == SP_F_GROUP_SUPPORT ? p->Hkv : p->Hq;
}

}  // namespace

void sp_count_launch(int n) { g_launches.fetch_add(n, std::memory_order_relaxed); }

int sp_current_device() {
  int dev = 0;
  if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= SP_MAX_DEVICES) dev = 0;
  return dev;
}

int sp_sm_count() {
  static int n[SP_MAX_DEVICES];
  const int dev = sp_current_device();
  if (n[dev] == 0) {
    int v = 0;
    if (cudaDeviceGetAttribute(&v, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess || v <= 0) v = 148;
    n[dev] = v;
  }
  return n[dev];
}

extern "C" {

int64_t sp_launch_count(void) { return g_launches.load(); }

const char* sp_strerror(int code) {
  switch (code) {
    case SP_OK: return "SP_OK";
    case SP_ERR_INVALID_ARG: return "SP_ERR_INVALID_ARG: null/misaligned pointer, bad size, bad cu_seqlens or bad panel";
    case SP_ERR_UNSUPPORTED: return "SP_ERR_UNSUPPORTED: shape outside the built set (d in {64,128}, Hq/Hkv in {1,2,4,8}, d_idx in {64,128}, hidden % 64 == 0, known flags; flags need b_sel in {1,32,64,128})";
    case SP_ERR_WORKSPACE: return "SP_ERR_WORKSPACE: workspace too small, see sp_workspace_bytes";
    case SP_ERR_TOO_LARGE:
      return "SP_ERR_TOO_LARGE: the problem needs more scratch than the library's fixed array holds (sp_sparse_gqa_attn_static: L <= 8192)";
    case SP_ERR_CUDA: return g_err_text;
  }
  return "unknown sp_status";
}

int64_t sp_num_rows(const sp_params* p) {
  const int rc = validate_common(p, false, false);
  if (rc != SP_OK) return rc;
  return host_geom(p).num_rows();
}

int sp_workspace_bytes(const sp_params* p, int stage, size_t* bytes_out) {
  if (!bytes_out) return SP_ERR_INVALID_ARG;
  const bool idxr = stage == SP_STAGE_INDEXER_SCORES || stage == SP_STAGE_LAYER_INDEXER;
  const bool attn = stage != SP_STAGE_INDEXER_SCORES && stage != SP_STAGE_TOPK;
  int units = 1;
  sp_params pq;
  if (p && stage == SP_STAGE_LAYER_ORACLE && (p->flags & (SP_F_GROUP_SUPPORT | SP_F_HEAD_SUPPORT))) {
    units = layer_units(p, SP_MODE_ORACLE);
    if (units < 0) return units;
    pq = *p;
    pq.flags &= ~(uint32_t)(SP_F_GROUP_SUPPORT | SP_F_HEAD_SUPPORT);
    p = &pq;
  }
  const int rc = validate_common(p, attn, idxr);
  if (rc != SP_OK) return rc;
  switch (stage) {
    case SP_STAGE_INDEXER_SCORES: *bytes_out = ws_indexer(p); return SP_OK;
    case SP_STAGE_ORACLE_MASS: *bytes_out = ws_mass(p); return SP_OK;
    case SP_STAGE_SPARSE_ATTN: {
      const MaskedPlan mp = masked_plan(p);
      *bytes_out = mp.use ? mp.bytes : 0;
      return SP_OK;
    }
    case SP_STAGE_TOPK:
    case SP_STAGE_DENSE_ATTN: *bytes_out = 0; return SP_OK;
    case SP_STAGE_LAYER_ORACLE: *bytes_out = plan_layer(p, SP_MODE_ORACLE, true, units).total; return SP_OK;
    case SP_STAGE_LAYER_INDEXER: *bytes_out = plan_layer(p, SP_MODE_INDEXER, true).total; return SP_OK;
  }
  return SP_ERR_INVALID_ARG;
}

int sp_indexer_scores(const sp_params* p, const void* X, const void* Wqi, const void* Wki, void* q_idx, void* k_idx,
                      int32_t preprojected, int32_t row_begin, int32_t row_count, float* scores, int64_t ld_scores,
                      void* ws, size_t ws_bytes, void* stream) {
  int rc = validate_common(p, false, true);
  if (rc != SP_OK) return rc;
  if (!q_idx || !k_idx || !scores || !aligned16(q_idx) || !aligned16(k_idx) || !aligned16(scores))
    return SP_ERR_INVALID_ARG;
  if (!preprojected && (!X || !Wqi || !Wki || !aligned16(X) || !aligned16(Wqi) || !aligned16(Wki)))
    return SP_ERR_INVALID_ARG;
  int max_nv = 0;
  rc = validate_panel(p, row_begin, row_count, ld_scores, &max_nv);
  if (rc != SP_OK) return rc;
  if (!preprojected && (ws_bytes < ws_indexer(p) || !ws)) return SP_ERR_WORKSPACE;
  cudaStream_t st = (cudaStream_t)stream;
  if (!preprojected) SP_CUDA(run_project(p, X, Wqi, Wki, q_idx, k_idx, ws, st), "projection");
  SP_CUDA(run_indexer_scores(p, q_idx, k_idx, row_begin, row_count, max_nv, scores, ld_scores, st), "indexer scores");
  return SP_OK;
}

static int oracle_mass_impl(const sp_params* p, const void* Q, const void* K, float* lse, int32_t lse_ready, int grp,
                            int head, int32_t row_begin, int32_t row_count, float* mass, int64_t ld_mass, void* ws,
                            size_t ws_bytes, void* stream) {
  int rc = validate_common(p, true, false);
  if (rc != SP_OK) return rc;
  if (grp >= p->Hkv || head >= p->Hq) return SP_ERR_INVALID_ARG;
  if ((grp >= 0 || head >= 0) && !sp_tc_mass_supported(p->b_sel, p->d)) return SP_ERR_UNSUPPORTED;
  if (!Q || !K || !mass || !aligned16(Q) || !aligned16(K) || !aligned16(mass)) return SP_ERR_INVALID_ARG;
  if (lse_ready && !lse) return SP_ERR_INVALID_ARG;
  int max_nv = 0;
  rc = validate_panel(p, row_begin, row_count, ld_mass, &max_nv);
  if (rc != SP_OK) return rc;
  if (!lse) {
    if (!ws || ws_bytes < ws_mass(p)) return SP_ERR_WORKSPACE;
    lse = (float*)ws;
  }
  cudaStream_t st = (cudaStream_t)stream;
  const SpGeom g = dev_geom(p);
  if (!lse_ready && row_count > 0) {
    // pass 1 (Alg.1 step 2): softmax normalisers of the panel's queries.  The panel's queries are a
    // contiguous packed range: from the first query of row_begin to the last query of the last row.
    const HostGeom hg = host_geom(p);
    long long r0 = 0;
    int q_lo = -1, q_hi = -1;
    for (int i = 0; i < hg.batch; ++i) {
      const int n = hg.seq_len(i);
      const long long nr = hg.rows_of(n);
      const long long lo = row_begin > r0 ? row_begin : r0;
      const long long hi = ((long long)row_begin + row_count < r0 + nr ? (long long)row_begin + row_count : r0 + nr) - 1;
      if (lo <= hi) {
        const int a = hg.seq_start(i) + (int)((lo - r0) * hg.b);
        long long e = (hi - r0 + 1) * hg.b;
        if (e > n) e = n;
        const int b = hg.seq_start(i) + (int)e - 1;
        if (q_lo < 0) q_lo = a;
        q_hi = b;
      }
      r0 += nr;
    }
    SP_CUDA(run_attn(p, Q, K, nullptr, nullptr, q_lo, q_hi - q_lo + 1, nullptr, lse, st), "mass pass 1 (lse)");
  }
  SP_CUDA(run_mass(p, Q, K, lse, row_begin, row_count, max_nv, mass, ld_mass, st, grp, head), "mass pass 2");
  return SP_OK;
}

int sp_oracle_mass(const sp_params* p, const void* Q, const void* K, float* lse, int32_t lse_ready, int32_t row_begin,
                   int32_t row_count, float* mass, int64_t ld_mass, void* ws, size_t ws_bytes, void* stream) {
  return oracle_mass_impl(p, Q, K, lse, lse_ready, -1, -1, row_begin, row_count, mass, ld_mass, ws, ws_bytes, stream);
}

int sp_oracle_mass_group(const sp_params* p, const void* Q, const void* K, float* lse, int32_t lse_ready, int32_t group,
                         int32_t row_begin, int32_t row_count, float* mass, int64_t ld_mass, void* ws, size_t ws_bytes,
                         void* stream) {
  if (group < 0) return SP_ERR_INVALID_ARG;
  return oracle_mass_impl(p, Q, K, lse, lse_ready, group, -1, row_begin, row_count, mass, ld_mass, ws, ws_bytes, stream);
}

int sp_oracle_mass_head(const sp_params* p, const void* Q, const void* K, float* lse, int32_t lse_ready, int32_t head,
                        int32_t row_begin, int32_t row_count, float* mass, int64_t ld_mass, void* ws, size_t ws_bytes,
                        void* stream) {
  if (head < 0) return SP_ERR_INVALID_ARG;
  return oracle_mass_impl(p, Q, K, lse, lse_ready, -1, head, row_begin, row_count, mass, ld_mass, ws, ws_bytes, stream);
}

int sp_topk_support(const sp_params* p, const float* scores, int64_t ld_scores, int32_t row_begin, int32_t row_count,
                    int32_t* idx, int32_t* cnt, void* /*ws*/, size_t /*ws_bytes*/, void* stream) {
  int rc = validate_common(p, false, false);
  if (rc != SP_OK) return rc;
  if (!scores || !idx || !aligned16(scores)) return SP_ERR_INVALID_ARG;
  int max_nv = 0;
  rc = validate_panel(p, row_begin, row_count, ld_scores, &max_nv);
  if (rc != SP_OK) return rc;
  SP_CUDA(sp_launch_topk(dev_geom(p), scores, ld_scores, row_begin, row_count, p->k, max_nv, idx, cnt, (cudaStream_t)stream),
          "top-k");
  return SP_OK;
}

int sp_support_overlap(const sp_params* p, const int32_t* idx_a, const int32_t* idx_b, int32_t* inter, void* stream) {
  const int rc = validate_common(p, false, false);
  if (rc != SP_OK) return rc;
  if (!idx_a || !idx_b || !inter) return SP_ERR_INVALID_ARG;
  SP_CUDA(sp_launch_overlap(idx_a, idx_b, host_geom(p).num_rows(), p->k, inter, (cudaStream_t)stream), "support overlap");
  return SP_OK;
}

int sp_row_kl(const sp_params* p, const float* mass, int64_t ld_mass, const float* scores, int64_t ld_scores,
              int32_t row_begin, int32_t row_count, float* kl, void* stream) {
  int rc = validate_common(p, false, false);
  if (rc != SP_OK) return rc;
  if (p->b_sel != 1) return SP_ERR_UNSUPPORTED;
  if (!mass || !scores || !kl) return SP_ERR_INVALID_ARG;
  int max_nv = 0;
  rc = validate_panel(p, row_begin, row_count, ld_mass, &max_nv);
  if (rc != SP_OK) return rc;
  if (ld_scores < max_nv) return SP_ERR_INVALID_ARG;
  SP_CUDA(sp_launch_row_kl(dev_geom(p), mass, ld_mass, scores, ld_scores, row_begin, row_count, kl, (cudaStream_t)stream),
          "row KL");
  return SP_OK;
}

int sp_gather_probe(const void* base, int32_t row_bytes, int64_t row_pitch_bytes, const int32_t* idx, int64_t n_idx,
                    void* sink, size_t sink_bytes, void* stream) {
  if (!base || !idx || !sink || !aligned16(base) || n_idx < 1) return SP_ERR_INVALID_ARG;
  if (row_bytes < 256 || row_bytes % 256 != 0 || row_pitch_bytes < row_bytes || row_pitch_bytes % 16 != 0)
    return SP_ERR_INVALID_ARG;
  const int blocks = 148 * 8;
  if (sink_bytes < (size_t)blocks * 256 * sizeof(uint32_t)) return SP_ERR_WORKSPACE;
  SP_CUDA(sp_launch_gather_probe(base, row_bytes, row_pitch_bytes, idx, n_idx, (uint32_t*)sink, blocks,
                                 (cudaStream_t)stream), "gather probe");
  return SP_OK;
}

int sp_sparse_gqa_attn(const sp_params* p, const void* Q, const void* K, const void* V, const int32_t* idx, void* O,
                       float* lse, void* ws, size_t ws_bytes, void* stream) {
  if (!p) return SP_ERR_INVALID_ARG;
  if (ws && !aligned16(ws)) return SP_ERR_INVALID_ARG;
  sp_params q = *p;  // the support-granularity flags belong to this entry point and to sp_prefill_layer's oracle mode
  q.flags &= ~(uint32_t)(SP_F_GROUP_SUPPORT | SP_F_HEAD_SUPPORT);
  if ((p->flags & SP_F_GROUP_SUPPORT) && (p->flags & SP_F_HEAD_SUPPORT)) return SP_ERR_INVALID_ARG;
  const int rc = validate_common(&q, true, false);
  if (rc != SP_OK) return rc;
  if (!Q || !K || !V || !idx || !O || !aligned16(Q) || !aligned16(K) || !aligned16(V) || !aligned16(O))
    return SP_ERR_INVALID_ARG;
  const bool per_head = (p->flags & SP_F_HEAD_SUPPORT) != 0;
  const long long idx_grp =
      (p->flags & (SP_F_GROUP_SUPPORT | SP_F_HEAD_SUPPORT)) ? host_geom(&q).num_rows() * (long long)q.k : 0;
  SP_CUDA(run_attn(&q, Q, K, V, idx, 0, q.L, O, lse, (cudaStream_t)stream, idx_grp, per_head, ws, ws_bytes), "sparse attention");
  return SP_OK;
}

int sp_sparse_gqa_attn_static(const sp_params* p, const void* Q, const void* K, const void* V, const int32_t* idx,
                              void* O, float* lse, void* stream) {
  if (!p) return SP_ERR_INVALID_ARG;
  if (p->flags & (SP_F_GROUP_SUPPORT | SP_F_HEAD_SUPPORT)) return SP_ERR_UNSUPPORTED;
  const int rc = validate_common(p, true, false);
  if (rc != SP_OK) return rc;
  if (!Q || !K || !V || !idx || !O || !aligned16(Q) || !aligned16(K) || !aligned16(V) || !aligned16(O))
    return SP_ERR_INVALID_ARG;
  long long pitch, rows;
  sp_support_bits_shape(p->L, &pitch, &rows);
  uint32_t* scratch = nullptr;
  size_t scratch_bytes = 0;
  SP_CUDA(sp_static_scratch_ptr(&scratch, &scratch_bytes), "static scratch address");
  if ((size_t)pitch * (size_t)rows * sizeof(uint32_t) > scratch_bytes) return SP_ERR_TOO_LARGE;
  const MaskedPlan mp = masked_plan(p);
  if (!mp.use) return SP_ERR_UNSUPPORTED;  // the masked tile loop's shape set; sp_sparse_gqa_attn covers the rest
  const SpGeom g = dev_geom(p);
  cudaStream_t st = (cudaStream_t)stream;
  SP_CUDA(sp_launch_support_bits(g, idx, p->k, host_geom(p).num_rows(), scratch, st), "support bitmap (static scratch)");
  SP_CUDA(sp_launch_attn_tc_masked(g, mp.chunks, Q, K, V, scratch, p->Hq, p->Hkv, p->d, attn_scale(p), O, lse, st),
          "sparse attention (static scratch)");
  return SP_OK;
}

int sp_dense_gqa_attn(const sp_params* p, const void* Q, const void* K, const void* V, void* O, float* lse,
                      void* /*ws*/, size_t /*ws_bytes*/, void* stream) {
  const int rc = validate_common(p, true, false);
  if (rc != SP_OK) return rc;
  if (!Q || !K || (!V && O) || (!O && !lse) || !aligned16(Q) || !aligned16(K) || !aligned16(V) || !aligned16(O))
    return SP_ERR_INVALID_ARG;
  SP_CUDA(run_attn(p, Q, K, V, nullptr, 0, p->L, O, lse, (cudaStream_t)stream), "dense attention");
  return SP_OK;
}

int sp_prefill_layer(const sp_params* p, int32_t mode, const void* X, const void* Wqi, const void* Wki, const void* Q,
                     const void* K, const void* V, void* O, int32_t* idx_out, void* ws, size_t ws_bytes,
                     void* stream) {
  if (mode != SP_MODE_ORACLE && mode != SP_MODE_INDEXER || !p) return SP_ERR_INVALID_ARG;
  // support granularity on the head axis: oracle mode only (the indexer is head-collapsed by construction)
  const int units = layer_units(p, mode);
  if (units < 0) return units;
  sp_params pq = *p;
  pq.flags &= ~(uint32_t)(SP_F_GROUP_SUPPORT | SP_F_HEAD_SUPPORT);
  const bool per_head = (p->flags & SP_F_HEAD_SUPPORT) != 0, per_group = (p->flags & SP_F_GROUP_SUPPORT) != 0;
  p = &pq;
  const int rc = validate_common(p, true, mode == SP_MODE_INDEXER);
  if (rc != SP_OK) return rc;
  if ((per_head || per_group) && !sp_tc_mass_supported(p->b_sel, p->d)) return SP_ERR_UNSUPPORTED;
  if (!Q || !K || !V || !O || !aligned16(Q) || !aligned16(K) || !aligned16(V) || !aligned16(O)) return SP_ERR_INVALID_ARG;
  if (mode == SP_MODE_INDEXER && (!X || !Wqi || !Wki || !aligned16(X) || !aligned16(Wqi) || !aligned16(Wki)))
    return SP_ERR_INVALID_ARG;
  const LayerPlan pl = plan_layer(p, mode, idx_out == nullptr, units);
  if (!ws || !aligned16(ws) || ws_bytes < pl.total) return SP_ERR_WORKSPACE;
  char* base = (char*)ws;
  cudaStream_t st = (cudaStream_t)stream;
  const SpGeom g = dev_geom(p);
  const HostGeom hg = host_geom(p);
  float* scores = (float*)(base + pl.off_scores);
  int32_t* idx = idx_out ? idx_out : (int32_t*)(base + pl.off_idx);
  void* q_idx = base + pl.off_qidx;
  void* k_idx = base + pl.off_kidx;
  float* lse = (float*)(base + pl.off_lse);

  if (mode == SP_MODE_INDEXER) {
    SP_CUDA(run_project(p, X, Wqi, Wki, q_idx, k_idx, base + pl.off_stage, st), "projection");
  } else {
    SP_CUDA(run_attn(p, Q, K, nullptr, nullptr, 0, p->L, nullptr, lse, st), "mass pass 1 (lse)");
  }
  // one selection per unit: the whole layer (head-averaged support), each KV group, or each head -- all from ONE pass 1
  for (int u = 0; u < units; ++u) {
    int32_t* idx_u = idx + (size_t)u * pl.n_rows * p->k;
    for (long long r0 = 0; r0 < pl.n_rows; r0 += pl.panel_rows) {
      const int rcnt = (int)(pl.n_rows - r0 < pl.panel_rows ? pl.n_rows - r0 : pl.panel_rows);
      const int max_nv = hg.max_n_valid(r0, rcnt);
      if (mode == SP_MODE_INDEXER) {
        SP_CUDA(run_indexer_scores(p, q_idx, k_idx, (int)r0, rcnt, max_nv, scores, pl.ld, st), "indexer scores");
      } else {
        SP_CUDA(run_mass(p, Q, K, lse, (int)r0, rcnt, max_nv, scores, pl.ld, st, per_group ? u : -1, per_head ? u : -1),
                "mass pass 2");
      }
      SP_CUDA(sp_launch_topk(g, scores, pl.ld, (int)r0, rcnt, p->k, max_nv, idx_u + (size_t)r0 * p->k, nullptr, st), "top-k");
    }
  }
  SP_CUDA(run_attn(p, Q, K, V, idx, 0, p->L, O, nullptr, st, units > 1 || per_group || per_head ? pl.n_rows * (long long)p->k : 0,
                   per_head, base + pl.off_scores, pl.scores_bytes),
          "sparse attention");
  return SP_OK;
}

}  // extern "C"

// ---------------------------------------------------------------------------------------------------------------
// Chunked prefill against a paged KV cache (PAPER.md:292 stage 4, :331, :428; reading A30)
// ---------------------------------------------------------------------------------------------------------------
namespace {

int page_shift_of(int32_t page_size) {
  for (int s = 4; s <= 12; ++s)
    if (page_size == (1 << s)) return s;
  return -1;
}

int validate_pages(const sp_params* p, const sp_kv_pages* kv, bool need_kidx) {
  if (!kv || !kv->k_pages || !kv->v_pages || !kv->block_table) return SP_ERR_INVALID_ARG;
  if (need_kidx && !kv->kidx_pages) return SP_ERR_INVALID_ARG;
  if (!aligned16(kv->k_pages) || !aligned16(kv->v_pages) || !aligned16(kv->kidx_pages)) return SP_ERR_INVALID_ARG;
  if (page_shift_of(kv->page_size) < 0) return SP_ERR_UNSUPPORTED;  // powers of two, 16 ... 4096 tokens
  if (kv->n_pages < 1 || kv->n_blocks < 1) return SP_ERR_INVALID_ARG;
  if ((long long)kv->n_blocks * kv->page_size < p->L) return SP_ERR_INVALID_ARG;  // the table must cover the context
  return SP_OK;
}

struct ChunkPlan {
  int64_t ld;
  long long row0, n_rows, panel_rows;
  size_t off_qidx, off_kidx, off_scores, off_idx, total;
};

ChunkPlan plan_chunk(const sp_params* p, int32_t q_begin, int32_t q_count, bool idx_in_ws) {
  ChunkPlan pl{};
  pl.row0 = q_begin / p->b_sel;
  pl.n_rows = (q_count + p->b_sel - 1) / p->b_sel;
  pl.ld = (int64_t)align_up((size_t)p->L, 4);
  long long pr = (long long)(PANEL_BYTES / ((size_t)pl.ld * sizeof(float)));
  if (pr < 1) pr = 1;
  if (p->b_sel == 1 && pr >= 64) pr = pr / 64 * 64;
  if (pr > pl.n_rows) pr = pl.n_rows;
  pl.panel_rows = pr;
  size_t off = 0;
  pl.off_qidx = off; off += align_up((size_t)q_count * p->d_idx * 2);
  pl.off_kidx = off; off += align_up((size_t)q_count * p->d_idx * 2);
  pl.off_scores = off; off += align_up((size_t)pl.panel_rows * pl.ld * sizeof(float));
  pl.off_idx = off;
  if (idx_in_ws) off += align_up((size_t)pl.n_rows * p->k * sizeof(int32_t));
  pl.total = off;
  return pl;
}

int validate_chunk(const sp_params* p, int32_t q_begin, int32_t q_count) {
  const int rc = validate_common(p, true, true);
  if (rc != SP_OK) return rc;
  if (p->cu_seqlens || p->batch != 1) return SP_ERR_UNSUPPORTED;  // one sequence per chunk call
  if (q_begin < 0 || q_count < 1 || (long long)q_begin + q_count != p->L) return SP_ERR_INVALID_ARG;
  if (q_begin % p->b_sel != 0) return SP_ERR_INVALID_ARG;         // selection blocks stay aligned to the sequence start
  if (!sp_tc_scores_supported(p->b_sel)) return SP_ERR_UNSUPPORTED;  // the paged readers are the tcgen05 / mma.sync kernels
  return SP_OK;
}

}  // namespace

extern "C" int sp_chunk_workspace_bytes(const sp_params* p, int32_t q_begin, int32_t q_count, size_t* bytes_out) {
  if (!bytes_out) return SP_ERR_INVALID_ARG;
  const int rc = validate_chunk(p, q_begin, q_count);
  if (rc != SP_OK) return rc;
  *bytes_out = plan_chunk(p, q_begin, q_count, true).total;
  return SP_OK;
}

static int kv_copy_impl(bool to_pages, const sp_params* p, const sp_kv_pages* kv, int32_t t_begin, int32_t t_count,
                        void* Kc, void* Vc, void* kidx_c, void* stream) {
  int rc = validate_common(p, true, kidx_c != nullptr);
  if (rc != SP_OK) return rc;
  rc = validate_pages(p, kv, kidx_c != nullptr);
  if (rc != SP_OK) return rc;
  if (t_begin < 0 || t_count < 0 || (long long)t_begin + t_count > (long long)kv->n_blocks * kv->page_size)
    return SP_ERR_INVALID_ARG;
  if ((!Kc && !Vc && !kidx_c) || !aligned16(Kc) || !aligned16(Vc) || !aligned16(kidx_c)) return SP_ERR_INVALID_ARG;
  const int sh = page_shift_of(kv->page_size);
  cudaStream_t st = (cudaStream_t)stream;
  const long long kvb = (long long)p->Hkv * p->d * 2;
  if (Kc) SP_CUDA(sp_launch_paged_copy(to_pages, kv->k_pages, Kc, kv->block_table, sh, kvb, t_begin, t_count, st), "paged K copy");
  if (Vc) SP_CUDA(sp_launch_paged_copy(to_pages, kv->v_pages, Vc, kv->block_table, sh, kvb, t_begin, t_count, st), "paged V copy");
  if (kidx_c)
    SP_CUDA(sp_launch_paged_copy(to_pages, kv->kidx_pages, kidx_c, kv->block_table, sh, (long long)p->d_idx * 2, t_begin,
                                 t_count, st), "paged k_idx copy");
  return SP_OK;
}

extern "C" int sp_kv_append(const sp_params* p, const sp_kv_pages* kv, int32_t t_begin, int32_t t_count, const void* K_new,
                            const void* V_new, const void* kidx_new, void* stream) {
  return kv_copy_impl(true, p, kv, t_begin, t_count, const_cast<void*>(K_new), const_cast<void*>(V_new),
                      const_cast<void*>(kidx_new), stream);
}

extern "C" int sp_kv_gather(const sp_params* p, const sp_kv_pages* kv, int32_t t_begin, int32_t t_count, void* K_out,
                            void* V_out, void* kidx_out, void* stream) {
  return kv_copy_impl(false, p, kv, t_begin, t_count, K_out, V_out, kidx_out, stream);
}

extern "C" int sp_prefill_chunk(const sp_params* p, int32_t q_begin, int32_t q_count, const void* X, const void* Wqi,
                                const void* Wki, const void* Q, const void* K_new, const void* V_new,
                                const sp_kv_pages* kv, void* O, int32_t* idx_out, void* ws, size_t ws_bytes,
                                void* stream) {
  int rc = validate_chunk(p, q_begin, q_count);
  if (rc != SP_OK) return rc;
  rc = validate_pages(p, kv, true);
  if (rc != SP_OK) return rc;
  if (!X || !Wqi || !Wki || !Q || !K_new || !V_new || !O) return SP_ERR_INVALID_ARG;
  if (!aligned16(X) || !aligned16(Wqi) || !aligned16(Wki) || !aligned16(Q) || !aligned16(K_new) || !aligned16(V_new) ||
      !aligned16(O))
    return SP_ERR_INVALID_ARG;
  const ChunkPlan pl = plan_chunk(p, q_begin, q_count, idx_out == nullptr);
  if (!ws || !aligned16(ws) || ws_bytes < pl.total) return SP_ERR_WORKSPACE;
  char* base = (char*)ws;
  cudaStream_t st = (cudaStream_t)stream;
  void* q_idx = base + pl.off_qidx;
  void* k_idx = base + pl.off_kidx;
  float* scores = (float*)(base + pl.off_scores);
  int32_t* idx = idx_out ? idx_out : (int32_t*)(base + pl.off_idx);
  const int sh = page_shift_of(kv->page_size);

  // stage 1: indexer projections of the chunk's tokens at their absolute positions
  SpGeom gp{1, q_count, nullptr, p->b_sel, 0};
  gp.pos_off = q_begin;
  SP_CUDA(sp_launch_project_tc(gp, p->flags, X, Wqi, Wki, q_idx, k_idx, q_count, p->hidden, p->d_idx, st), "chunk projection");
  // the chunk's own K, V and indexer keys go into the cache before anything reads it
  SP_CUDA(sp_launch_paged_copy(true, kv->k_pages, const_cast<void*>(K_new), kv->block_table, sh, (long long)p->Hkv * p->d * 2,
                               q_begin, q_count, st), "append K");
  SP_CUDA(sp_launch_paged_copy(true, kv->v_pages, const_cast<void*>(V_new), kv->block_table, sh, (long long)p->Hkv * p->d * 2,
                               q_begin, q_count, st), "append V");
  SP_CUDA(sp_launch_paged_copy(true, kv->kidx_pages, k_idx, kv->block_table, sh, (long long)p->d_idx * 2, q_begin, q_count, st),
          "append k_idx");
  // stages 2, 3, 5: every reader goes through the block table (no reconstruction of contiguous K / V)
  SpGeom g = dev_geom(p);
  g.q_off = q_begin;
  g.q_rows = q_count;
  g.row_off = (int)pl.row0;
  g.bt = kv->block_table;
  g.page_shift = sh;
  g.n_blocks = kv->n_blocks;
  g.kv_rows = (long long)kv->n_pages * kv->page_size;
  const HostGeom hg = host_geom(p);
  for (long long r = 0; r < pl.n_rows; r += pl.panel_rows) {
    const int rcnt = (int)(pl.n_rows - r < pl.panel_rows ? pl.n_rows - r : pl.panel_rows);
    const int rb = (int)(pl.row0 + r);
    const int max_nv = hg.max_n_valid(rb, rcnt);
    SP_CUDA(sp_launch_indexer_scores_tc(g, nullptr, q_idx, kv->kidx_pages, p->d_idx, index_scale(p), p->local_window,
                                        p->local_bias, (p->flags & SP_F_RELU) ? 1 : 0, rb, rcnt, max_nv, scores, pl.ld, st),
            "chunk indexer scores");
    SP_CUDA(sp_launch_topk(g, scores, pl.ld, rb, rcnt, p->k, max_nv, idx + (size_t)r * p->k, nullptr, st), "chunk top-k");
  }
  const int G = p->Hq / p->Hkv;
  if (sp_tc_attn_supported(p->b_sel, G, true, p->k, p->d, true)) {
    SP_CUDA(sp_launch_attn_tc(g, pl.n_rows, 0, 0, Q, kv->k_pages, kv->v_pages, idx, p->k, p->Hq, p->Hkv, p->d, attn_scale(p),
                              p->local_window, p->local_bias, O, nullptr, st), "chunk sparse attention");
  } else {
    SP_CUDA(sp_launch_attn_pq(g, Q, kv->k_pages, kv->v_pages, idx, p->k, p->Hq, p->Hkv, p->d, attn_scale(p), p->local_window,
                              p->local_bias, q_begin, q_count, O, nullptr, st), "chunk sparse attention (per query)");
  }
  return SP_OK;
}

extern "C" {

int sp_layer_host_arena_bytes(const sp_params* p, int32_t mode, size_t* bytes_out) {
  if (!bytes_out || (mode != SP_MODE_ORACLE && mode != SP_MODE_INDEXER)) return SP_ERR_INVALID_ARG;
  const int rc = validate_common(p, true, mode == SP_MODE_INDEXER);
  if (rc != SP_OK) return rc;
  size_t b = 0;
  b += align_up((size_t)p->L * p->Hq * p->d * 2) * 2;   // Q, O
  b += align_up((size_t)p->L * p->Hkv * p->d * 2) * 2;  // K, V
  if (mode == SP_MODE_INDEXER) {
    b += align_up((size_t)p->L * p->hidden * 2);
    b += align_up((size_t)p->hidden * p->d_idx * 2) * 2;
  }
  b += plan_layer(p, mode, true).total;
  *bytes_out = b;
  return SP_OK;
}

int sp_prefill_layer_host(const sp_params* p, int32_t mode, const void* X_host, const void* Wqi_host,
                          const void* Wki_host, const void* Q_host, const void* K_host, const void* V_host,
                          void* O_host, void* dev_arena, size_t arena_bytes, void* stream) {
  size_t need = 0;
  const int rc = sp_layer_host_arena_bytes(p, mode, &need);
  if (rc != SP_OK) return rc;
  if (!Q_host || !K_host || !V_host || !O_host) return SP_ERR_INVALID_ARG;
  if (mode == SP_MODE_INDEXER && (!X_host || !Wqi_host || !Wki_host)) return SP_ERR_INVALID_ARG;
  if (!dev_arena || !aligned16(dev_arena) || arena_bytes < need) return SP_ERR_WORKSPACE;
  cudaStream_t st = (cudaStream_t)stream;
  char* a = (char*)dev_arena;
  const size_t qb = (size_t)p->L * p->Hq * p->d * 2, kb = (size_t)p->L * p->Hkv * p->d * 2;
  void* dQ = a; a += align_up(qb);
  void* dO = a; a += align_up(qb);
  void* dK = a; a += align_up(kb);
  void* dV = a; a += align_up(kb);
  void *dX = nullptr, *dWq = nullptr, *dWk = nullptr;
  SP_CUDA(cudaMemcpyAsync(dQ, Q_host, qb, cudaMemcpyHostToDevice, st), "H2D Q");
  SP_CUDA(cudaMemcpyAsync(dK, K_host, kb, cudaMemcpyHostToDevice, st), "H2D K");
  SP_CUDA(cudaMemcpyAsync(dV, V_host, kb, cudaMemcpyHostToDevice, st), "H2D V");
  if (mode == SP_MODE_INDEXER) {
    const size_t xb = (size_t)p->L * p->hidden * 2, wb = (size_t)p->hidden * p->d_idx * 2;
    dX = a; a += align_up(xb);
    dWq = a; a += align_up(wb);
    dWk = a; a += align_up(wb);
    SP_CUDA(cudaMemcpyAsync(dX, X_host, xb, cudaMemcpyHostToDevice, st), "H2D X");
    SP_CUDA(cudaMemcpyAsync(dWq, Wqi_host, wb, cudaMemcpyHostToDevice, st), "H2D Wqi");
    SP_CUDA(cudaMemcpyAsync(dWk, Wki_host, wb, cudaMemcpyHostToDevice, st), "H2D Wki");
  }
  const size_t ws_bytes = arena_bytes - (size_t)(a - (char*)dev_arena);
  const int rc2 = sp_prefill_layer(p, mode, dX, dWq, dWk, dQ, dK, dV, dO, nullptr, a, ws_bytes, stream);
  if (rc2 != SP_OK) return rc2;
  SP_CUDA(cudaMemcpyAsync(O_host, dO, qb, cudaMemcpyDeviceToHost, st), "D2H O");
  return SP_OK;
}

}  // extern "C"
