// api.cu -- the C ABI of include/gcore.h: argument validation, workspace carving, and the
// host-side plan (row compaction, chunk loop of the backward).  No allocation, no sync.
#include "common.cuh"
#include <math.h>

using namespace gc;

namespace gc {
static thread_local cudaError_t t_last_cuda_error = cudaSuccess;
void note_cuda_error(cudaError_t e) {
  t_last_cuda_error = e;
  (void)cudaGetLastError();        // clear the runtime's non-sticky error state
}
}  // namespace gc

namespace {

bool aligned16(const void* p) { return (reinterpret_cast<uintptr_t>(p) & 15) == 0; }

int check_arch() {
  int dev = 0, major = 0;
  if (cudaGetDevice(&dev) != cudaSuccess) return GC_ERR_CUDA;
  if (cudaDeviceGetAttribute(&major, cudaDevAttrComputeCapabilityMajor, dev) != cudaSuccess)
    return GC_ERR_CUDA;
  return major == 10 ? GC_OK : GC_ERR_ARCH;
}

int elem_bytes(int dtype) { return dtype == GC_F32 ? 4 : 2; }

int check_head_args(const void* H, int64_t ldH, const void* W, int64_t ldW, int dtype,
                    const int32_t* targets, int64_t T, int64_t D, int64_t V, float tau) {
  if (dtype != GC_F32 && dtype != GC_BF16 && dtype != GC_BF16_SIMT) return GC_ERR_DTYPE;
  if (T < 0 || D <= 0 || V <= 0 || T >= (1ll << 31) || V >= (1ll << 31)) return GC_ERR_SHAPE;
  if (!(tau > 0.f)) return GC_ERR_ARG;
  if (!W || (T > 0 && (!H || !targets))) return GC_ERR_NULL;
  if (ldH < D || ldW < D) return GC_ERR_SHAPE;
  if (dtype == GC_BF16) {
    if (D % 8 != 0) return GC_ERR_SHAPE;
    if (ldH % 8 != 0 || ldW % 8 != 0 || !aligned16(H) || !aligned16(W)) return GC_ERR_ALIGN;
  }
  return GC_OK;
}

// ---- backward chunk size: rows of the dS buffer (multiple of 256) -----------------------------
// Minimises the number of dH tile waves -- the coarsest-grained of the three chunk kernels: 256 x 512
// dual-N tiles over the 74 CTA pairs, a last wave that is at most half full costing half a wave
// (tc_gemm.cuh) -- with a small charge per chunk (one more fp32 accumulate pass over dW); larger
// chunks win ties.  Capped at 8192 rows / 6 GB (measured: 8192, 12288 and 16384 rows run cfg2 within
// 1 % of each other) and at T/2, so the [T,V] matrix never exists whole.
int64_t pick_chunk(int64_t T, int64_t D, int64_t V) {
  const int64_t Tr = ceil_div(T > 0 ? T : 1, 256) * 256;
  if (Tr <= 256) return 256;
  const int64_t half = ceil_div(Tr / 2, 256) * 256;          // at least two chunks
  int64_t best = 256;
  double best_cost = 1e300;
  for (int64_t tc = 256; tc <= 8192 && tc <= half; tc += 256) {
    if (tc > 256 && (double)tc * (double)V * 2.0 > 6.0e9) break;   // dS buffer <= 6 GB
    double waves = 0;
    for (int64_t r0 = 0; r0 < Tr; r0 += tc) waves += tc_dh_waves((Tr - r0 < tc) ? Tr - r0 : tc, D);
    const double cost = waves * (1.0 + 0.01 * (double)ceil_div(Tr, tc));
    if (cost <= best_cost) { best_cost = cost; best = tc; }
  }
  return best;
}

int64_t resolve_chunk(int64_t T, int64_t D, int64_t V, int64_t chunk_tokens) {
  if (chunk_tokens <= 0) return pick_chunk(T, D, V);
  return ceil_div(chunk_tokens, 256) * 256;
}

int64_t ld_ds(int64_t V) { return ceil_div(V, 64) * 64; }

// Workspace layouts (mirrored by gc_workspace_bytes).
struct FwdWs {
  uint32_t* counters; RowStat* partials; int32_t* rows; int32_t* n_rows; int32_t* targets_c; void* Hs; void* compact;
};
size_t carve_fwd(Carver& c, int64_t T, int64_t D, int64_t V, int dtype, FwdWs* w) {
  const int64_t cap = ceil_div(T > 0 ? T : 1, 256) * 256;
  if (dtype == GC_BF16) {
    uint32_t* ctr = c.take<uint32_t>(kTcCounters);
    RowStat* p = c.take<RowStat>(tc_fwd_partials_bytes(T, D, V) / sizeof(RowStat));
    int32_t* rows = c.take<int32_t>((size_t)cap);
    int32_t* n_rows = c.take<int32_t>(64);
    int32_t* tc_ = c.take<int32_t>((size_t)cap);
    void* Hs = c.take<uint8_t>((size_t)cap * (size_t)D * 2);
    void* cw = c.take<uint8_t>(compact_ws_bytes(T));
    if (w) { w->counters = ctr; w->partials = p; w->rows = rows; w->n_rows = n_rows; w->targets_c = tc_; w->Hs = Hs; w->compact = cw; }
  }
  return c.off;
}

struct BwdWs {
  uint32_t* counters; void* loss; float* out5; float* g; int32_t* rows; int32_t* n_rows; int32_t* targets_c;
  float* lse_c; float* g_c; void* Hs; void* compact; void* dS; float* dW_acc;
};
// dW_dtype == GC_BF16: the chunks accumulate in an fp32 [V, D] staging buffer at the end of the
// workspace and are rounded to bf16 once, after the last chunk (SURVEY.md sec 8(c) reading 13)
size_t carve_bwd(Carver& c, int64_t T, int64_t D, int64_t V, int dtype, int64_t chunk, int32_t R,
                 int dW_dtype, BwdWs* w) {
  const int64_t cap = ceil_div(T > 0 ? T : 1, 256) * 256;
  void* loss = c.take<uint8_t>(loss_ws_bytes(T, R));
  float* out5 = c.take<float>(64);
  float* g = c.take<float>((size_t)cap);
  if (w) { w->loss = loss; w->out5 = out5; w->g = g; }
  if (dtype == GC_BF16) {
    uint32_t* ctr = c.take<uint32_t>(kTcCounters);
    if (w) w->counters = ctr;
    int32_t* rows = c.take<int32_t>((size_t)cap);
    int32_t* n_rows = c.take<int32_t>(64);
    int32_t* tcx = c.take<int32_t>((size_t)cap);
    float* lse_c = c.take<float>((size_t)cap);
    float* g_c = c.take<float>((size_t)cap);
    void* Hs = c.take<uint8_t>((size_t)cap * (size_t)D * 2);
    void* cw = c.take<uint8_t>(compact_ws_bytes(T));
    void* dS = c.take<uint8_t>((size_t)chunk * (size_t)ld_ds(V) * 2);
    if (w) { w->rows = rows; w->n_rows = n_rows; w->targets_c = tcx; w->lse_c = lse_c; w->g_c = g_c;
             w->Hs = Hs; w->compact = cw; w->dS = dS; }
  }
  float* acc = dW_dtype == GC_BF16 ? c.take<float>((size_t)V * (size_t)D) : nullptr;
  if (w) w->dW_acc = acc;
  return c.off;
}

// gc_workspace_bytes has no R argument: the loss scratch inside the fwd / bwd workspaces is
// sized for R <= T + 1 responses (one count per response), which the fwd / bwd entry points
// enforce.  gc_grpo_token_loss takes any R with gc_loss_workspace_bytes(T, R).
int32_t loss_rcap(int64_t T) { return (int32_t)((T + 1 < (1ll << 31) - 1) ? T + 1 : (1ll << 31) - 1); }

}  // namespace

extern "C" {

const char* gc_status_string(int status) {
  switch (status) {
    case GC_OK: return "GC_OK";
    case GC_ERR_NULL: return "GC_ERR_NULL: required pointer is NULL";
    case GC_ERR_SHAPE: return "GC_ERR_SHAPE: bad shape or leading dimension";
    case GC_ERR_DTYPE: return "GC_ERR_DTYPE: unknown dtype";
    case GC_ERR_ALIGN: return "GC_ERR_ALIGN: pointer or leading dimension not aligned";
    case GC_ERR_WORKSPACE: return "GC_ERR_WORKSPACE: workspace missing or too small";
    case GC_ERR_ARG: return "GC_ERR_ARG: bad scalar argument";
    case GC_ERR_ARCH: return "GC_ERR_ARCH: device is not compute capability 10.x";
    case GC_ERR_CUDA: return "GC_ERR_CUDA: CUDA call failed";
    default: return "GC_ERR_UNKNOWN";
  }
}

const char* gc_last_cuda_error(void) { return cudaGetErrorName(gc::t_last_cuda_error); }

int gc_version(void) { return 200; }

size_t gc_workspace_bytes(int op, int64_t T, int64_t D, int64_t V, int dtype, int64_t chunk_tokens) {
  if (T < 0 || D <= 0 || V <= 0) return 0;
  if (dtype != GC_F32 && dtype != GC_BF16 && dtype != GC_BF16_SIMT) return 0;
  Carver c(nullptr);
  const int32_t Rcap = loss_rcap(T);
  switch (op) {
    case GC_OP_LOGPROBS:
      carve_fwd(c, T, D, V, dtype, nullptr);
      break;
    case GC_OP_LOSS_FWD:
      carve_fwd(c, T, D, V, dtype, nullptr);
      c.take<uint8_t>(loss_ws_bytes(T, Rcap));
      break;
    case GC_OP_LOSS_BWD:
      carve_bwd(c, T, D, V, dtype, resolve_chunk(T, D, V, chunk_tokens), Rcap, GC_F32, nullptr);
      break;
    default:
      return 0;
  }
  return c.off + 256;
}

size_t gc_bwd_workspace_bytes(int64_t T, int64_t D, int64_t V, int dtype, int64_t chunk_tokens,
                              int dW_dtype) {
  if (T < 0 || D <= 0 || V <= 0) return 0;
  if (dtype != GC_F32 && dtype != GC_BF16 && dtype != GC_BF16_SIMT) return 0;
  if (dW_dtype != GC_F32 && dW_dtype != GC_BF16) return 0;
  Carver c(nullptr);
  carve_bwd(c, T, D, V, dtype, resolve_chunk(T, D, V, chunk_tokens), loss_rcap(T), dW_dtype, nullptr);
  return c.off + 256;
}

int gc_token_logprobs(const void* H, int64_t ldH, const void* W, int64_t ldW, int dtype,
                      const int32_t* targets, const uint8_t* mask, int64_t T, int64_t D, int64_t V,
                      float temperature, float* logp, float* entropy, float* lse, void* workspace,
                      size_t workspace_bytes, void* cuda_stream) {
  GC_TRY(check_head_args(H, ldH, W, ldW, dtype, targets, T, D, V, temperature));
  if (T > 0 && !logp) return GC_ERR_NULL;
  if (T == 0) return GC_OK;
  GC_TRY(check_arch());
  cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
  if (dtype != GC_BF16)
    return simt_logprobs(H, ldH, W, ldW, dtype == GC_BF16_SIMT, targets, mask, T, D, V, temperature,
                         logp, entropy, lse, st);
  if (!workspace || workspace_bytes < gc_workspace_bytes(GC_OP_LOGPROBS, T, D, V, dtype, 0))
    return GC_ERR_WORKSPACE;
  if (reinterpret_cast<uintptr_t>(workspace) & 255) return GC_ERR_ALIGN;
  Carver c(workspace);
  FwdWs w;
  carve_fwd(c, T, D, V, dtype, &w);
  const TcPlan pl = tc_plan_forward(T, D, V);
  const int64_t cap = ceil_div(T, 256) * 256;
  GC_CUDA_TRY(cudaMemsetAsync(w.counters, 0, sizeof(uint32_t) * kTcCounters, st));
  if (!mask) {
    // dense mode: every row goes through the contraction; rows with target < 0 come out as 0
    GC_TRY(tc_forward_stats(H, ldH, W, ldW, T, D, V, temperature, targets, nullptr, w.partials, w.counters, st));
    return launch_combine(w.partials, pl.n_split, cap, nullptr, nullptr, T, logp, entropy, lse, st);
  }
  // compaction mode (a1): only scored rows reach the tensor cores
  GC_TRY(launch_compact_rows(targets, mask, T, w.rows, w.n_rows, w.compact, st));
  GC_TRY(launch_gather_rows(H, ldH, 2, D, T, w.rows, w.n_rows, w.Hs, cap, st));
  GC_TRY(launch_gather_i32(targets, w.rows, w.n_rows, T, w.targets_c, st));
  GC_TRY(launch_zero_unscored(targets, mask, T, logp, entropy, lse, st));
  GC_TRY(tc_forward_stats(w.Hs, D, W, ldW, T, D, V, temperature, w.targets_c, w.n_rows, w.partials,
                          w.counters, st));
  return launch_combine(w.partials, pl.n_split, cap, w.rows, w.n_rows, T, logp, entropy, lse, st);
}

size_t gc_multi_workspace_bytes(int64_t T, int64_t D, int64_t V, int32_t K) {
  if (T < 0 || D <= 0 || V <= 0 || K < 1 || K > 8) return 0;
  const size_t cap = (size_t)ceil_div(T > 0 ? T : 1, 256) * 256;
  return align_up(sizeof(uint32_t) * kTcCounters, 256) + tc_fwd_partials_bytes(T, D, V) +
         align_up(cap * (size_t)K * sizeof(float), 256) + 256;
}

int gc_token_logprobs_multi(const void* H, int64_t ldH, const void* W, int64_t ldW, int dtype,
                            const int32_t* targets, int32_t K, int64_t T, int64_t D, int64_t V,
                            float temperature, float* logp, float* entropy, float* lse,
                            void* workspace, size_t workspace_bytes, void* cuda_stream) {
  if (dtype != GC_BF16) return GC_ERR_DTYPE;
  if (K < 1 || K > 8) return GC_ERR_ARG;
  GC_TRY(check_head_args(H, ldH, W, ldW, dtype, targets, T, D, V, temperature));
  if (T > 0 && !logp) return GC_ERR_NULL;
  if (T == 0) return GC_OK;
  if (!workspace || workspace_bytes < gc_multi_workspace_bytes(T, D, V, K)) return GC_ERR_WORKSPACE;
  if (reinterpret_cast<uintptr_t>(workspace) & 255) return GC_ERR_ALIGN;
  GC_TRY(check_arch());
  cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
  const size_t cap = (size_t)ceil_div(T, 256) * 256;
  Carver c(workspace);
  uint32_t* counters = c.take<uint32_t>(kTcCounters);
  RowStat* partials = c.take<RowStat>(tc_fwd_partials_bytes(T, D, V) / sizeof(RowStat));
  float* ay = c.take<float>(cap * (size_t)K);
  GC_CUDA_TRY(cudaMemsetAsync(counters, 0, sizeof(uint32_t) * kTcCounters, st));
  GC_TRY(launch_fill_f32(ay, -INFINITY, (int64_t)T * K, st));     // "target not met"
  GC_TRY(tc_forward_stats_multi(H, ldH, W, ldW, T, D, V, temperature, targets, K, ay, partials,
                                counters, st));
  const TcPlan pl = tc_plan_forward(T, D, V);
  return launch_combine_multi(partials, pl.n_split, (int64_t)cap, ay, K, T, logp, entropy, lse, st);
}

int gc_grpo_advantages(const float* rewards, const int32_t* group_offsets, int32_t G, float eps,
                       int unbiased_std, int drop_constant_groups, float* adv, uint8_t* keep,
                       void* cuda_stream) {
  if (G < 0) return GC_ERR_SHAPE;
  if (!(eps >= 0.f)) return GC_ERR_ARG;
  if (G == 0) return GC_OK;
  if (!rewards || !group_offsets || !adv) return GC_ERR_NULL;
  GC_TRY(check_arch());
  return launch_advantages(rewards, group_offsets, G, eps, unbiased_std != 0,
                           drop_constant_groups != 0, adv, keep, static_cast<cudaStream_t>(cuda_stream));
}

// bound_R: the fwd / bwd entry points size their loss scratch for R <= T + 1 (empty responses are
// fine, a batch with more responses than tokens + 1 is refused there; gc_grpo_token_loss takes it)
static int check_loss_args(const int32_t* cu_seqlens, int32_t R, const float* adv,
                           const float* old_logp, const float* ref_logp, float clip_lo,
                           float clip_hi, float beta, int agg, int64_t T, bool bound_R = true) {
  if (R < 0 || (T > 0 && R < 1) || (bound_R && (int64_t)R > T + 1)) return GC_ERR_SHAPE;
  if (agg != GC_AGG_TOKEN_MEAN && agg != GC_AGG_SEQ_MEAN) return GC_ERR_ARG;
  if (!(clip_lo >= 0.f) || !(clip_hi >= 0.f) || !(beta >= 0.f)) return GC_ERR_ARG;
  if (!cu_seqlens || (T > 0 && (!adv || !old_logp))) return GC_ERR_NULL;
  if (beta != 0.f && T > 0 && !ref_logp) return GC_ERR_NULL;
  return GC_OK;
}

size_t gc_loss_workspace_bytes(int64_t T, int32_t R) {
  return (T < 0 || R < 0) ? 0 : loss_ws_bytes(T, R) + 256;
}

int gc_grpo_token_loss(const float* logp, const float* old_logp, const float* ref_logp,
                       const int32_t* targets, const uint8_t* mask, int64_t T,
                       const int32_t* cu_seqlens, int32_t R, const float* adv, float clip_lo,
                       float clip_hi, float beta, int agg, float grad_loss, float* out5, float* g,
                       void* workspace, size_t workspace_bytes, void* cuda_stream) {
  if (T < 0 || T >= (1ll << 31)) return GC_ERR_SHAPE;
  GC_TRY(check_loss_args(cu_seqlens, R, adv, old_logp, ref_logp, clip_lo, clip_hi, beta, agg, T,
                         false));
  if (!out5 || (T > 0 && (!logp || !targets))) return GC_ERR_NULL;
  if (!aligned16(logp) || !aligned16(old_logp) || !aligned16(ref_logp) || !aligned16(targets) ||
      !aligned16(g) || (reinterpret_cast<uintptr_t>(mask) & 3))
    return GC_ERR_ALIGN;
  if (!workspace || workspace_bytes < loss_ws_bytes(T, R)) return GC_ERR_WORKSPACE;
  if (reinterpret_cast<uintptr_t>(workspace) & 255) return GC_ERR_ALIGN;
  GC_TRY(check_arch());
  return launch_token_loss(logp, old_logp, ref_logp, targets, mask, T, cu_seqlens, R, adv, clip_lo,
                           clip_hi, beta, agg, grad_loss, out5, g, workspace,
                           static_cast<cudaStream_t>(cuda_stream));
}

int gc_grpo_loss_fwd(const void* H, int64_t ldH, const void* W, int64_t ldW, int dtype,
                     const int32_t* targets, const uint8_t* mask, int64_t T, int64_t D, int64_t V,
                     float temperature, const int32_t* cu_seqlens, int32_t R, const float* adv,
                     const float* old_logp, const float* ref_logp, float clip_lo, float clip_hi,
                     float beta, int agg, float* out5, float* logp, float* entropy, float* lse,
                     void* workspace, size_t workspace_bytes, void* cuda_stream) {
  GC_TRY(check_head_args(H, ldH, W, ldW, dtype, targets, T, D, V, temperature));
  GC_TRY(check_loss_args(cu_seqlens, R, adv, old_logp, ref_logp, clip_lo, clip_hi, beta, agg, T));
  if (!out5 || (T > 0 && (!logp || !lse))) return GC_ERR_NULL;
  const size_t need = gc_workspace_bytes(GC_OP_LOSS_FWD, T, D, V, dtype, 0);
  if (!workspace || workspace_bytes < need) return GC_ERR_WORKSPACE;
  if (reinterpret_cast<uintptr_t>(workspace) & 255) return GC_ERR_ALIGN;
  const size_t fwd_bytes = gc_workspace_bytes(GC_OP_LOGPROBS, T, D, V, dtype, 0);
  GC_TRY(gc_token_logprobs(H, ldH, W, ldW, dtype, targets, mask, T, D, V, temperature, logp, entropy,
                           lse, workspace, fwd_bytes, cuda_stream));
  void* loss_ws = static_cast<char*>(workspace) + align_up(fwd_bytes, 256);
  return gc_grpo_token_loss(logp, old_logp, ref_logp, targets, mask, T, cu_seqlens, R, adv, clip_lo,
                            clip_hi, beta, agg, 1.0f, out5, nullptr, loss_ws,
                            workspace_bytes - align_up(fwd_bytes, 256), cuda_stream);
}

}  // extern "C"

namespace {
// where dW goes: a local [V, D] buffer, or (shards != NULL) the per-rank shards of a fused
// reduce-scatter (tc_dw_reduce_scatter)
struct DwSink {
  void* dW; int64_t lddW; int accumulate;
  float* const* shards; int world; int64_t shard_rows;
  int dW_dtype;             // GC_F32 / GC_BF16 (local dW only)
  const void* fwd_state;    // the forward's workspace (row list + compacted H reused), or NULL
  // host_api.cu only: an event recorded right after the dH launch of the last NON-EMPTY chunk (dH is
  // complete from there on: gc_grpo_step_host starts its device -> host copy of dH under the last dW
  // contraction); dh_rows = scored rows of the batch (chunks past them are empty)
  cudaEvent_t dh_done = nullptr;
  int64_t dh_rows = 0;
};

int loss_bwd_impl(const void* H, int64_t ldH, const void* W, int64_t ldW, int dtype,
                  const int32_t* targets, const uint8_t* mask, int64_t T, int64_t D, int64_t V,
                  float temperature, const int32_t* cu_seqlens, int32_t R, const float* adv,
                  const float* old_logp, const float* ref_logp, float clip_lo, float clip_hi,
                  float beta, int agg, const float* logp, const float* lse, float grad_loss,
                  void* dH, int64_t lddH, const DwSink& sink, int64_t chunk_tokens, void* workspace,
                  size_t workspace_bytes, void* cuda_stream) {
  void* dW = sink.dW;
  int64_t lddW = sink.lddW;
  int accumulate_dW = sink.accumulate;
  const bool dW_bf16 = !sink.shards && sink.dW_dtype == GC_BF16;
  GC_TRY(check_head_args(H, ldH, W, ldW, dtype, targets, T, D, V, temperature));
  GC_TRY(check_loss_args(cu_seqlens, R, adv, old_logp, ref_logp, clip_lo, clip_hi, beta, agg, T));
  if (sink.shards) {
    if (dtype != GC_BF16) return GC_ERR_DTYPE;
    if (sink.world < 1 || sink.world > 8 || sink.shard_rows <= 0 || sink.shard_rows % 32 != 0)
      return GC_ERR_ARG;
    if (sink.shard_rows * sink.world < V || lddW < D || lddW % 4 != 0) return GC_ERR_SHAPE;
    for (int r = 0; r < sink.world; ++r) {
      if (!sink.shards[r]) return GC_ERR_NULL;
      if (!aligned16(sink.shards[r])) return GC_ERR_ALIGN;
    }
  } else {
    if (!dW) return GC_ERR_NULL;
    if (lddW < D) return GC_ERR_SHAPE;
    if (dW_bf16) {
      if (dtype == GC_BF16 && (lddW % 8 != 0 || !aligned16(dW))) return GC_ERR_ALIGN;
    } else if (dtype == GC_BF16 && (lddW % 4 != 0 || !aligned16(dW))) {
      return GC_ERR_ALIGN;
    }
  }
  if (T > 0 && (!dH || !logp || !lse)) return GC_ERR_NULL;
  if (lddH < D) return GC_ERR_SHAPE;
  if (dtype == GC_BF16 && (lddH % 8 != 0 || !aligned16(dH))) return GC_ERR_ALIGN;
  if (!aligned16(logp) || !aligned16(old_logp) || !aligned16(ref_logp) || !aligned16(targets) ||
      (reinterpret_cast<uintptr_t>(mask) & 3))
    return GC_ERR_ALIGN;
  const size_t need = gc_bwd_workspace_bytes(T, D, V, dtype, chunk_tokens, dW_bf16 ? GC_BF16 : GC_F32);
  if (!workspace || workspace_bytes < need) return GC_ERR_WORKSPACE;
  if (reinterpret_cast<uintptr_t>(workspace) & 255) return GC_ERR_ALIGN;
  if (sink.fwd_state && (reinterpret_cast<uintptr_t>(sink.fwd_state) & 255)) return GC_ERR_ALIGN;
  if (sink.fwd_state) {          // the forward's workspace must not overlap this call's scratch
    const uintptr_t f0 = reinterpret_cast<uintptr_t>(sink.fwd_state);
    const uintptr_t f1 = f0 + gc_workspace_bytes(GC_OP_LOSS_FWD, T, D, V, dtype, 0);
    const uintptr_t w0 = reinterpret_cast<uintptr_t>(workspace), w1 = w0 + need;
    if (f0 < w1 && w0 < f1) return GC_ERR_ARG;
  }
  GC_TRY(check_arch());
  cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
  if (T == 0) {
    const size_t eb = dW_bf16 ? 2 : 4;
    if (!sink.shards && !accumulate_dW)
      GC_CUDA_TRY(cudaMemset2DAsync(dW, (size_t)lddW * eb, 0, (size_t)D * eb, (size_t)V, st));
    return GC_OK;
  }
  const int64_t chunk = resolve_chunk(T, D, V, chunk_tokens);
  const int32_t Rcap = loss_rcap(T);
  Carver c(workspace);
  BwdWs w;
  carve_bwd(c, T, D, V, dtype, chunk, Rcap, dW_bf16 ? GC_BF16 : GC_F32, &w);
  // bf16 dW: the chunk loop writes the fp32 staging buffer; one rounding pass at the end
  void* const dW_out = dW;
  const int64_t lddW_out = lddW;
  const int accumulate_out = accumulate_dW;
  if (dW_bf16) { dW = w.dW_acc; lddW = D; accumulate_dW = 0; }

  // a9: g_t = grad_loss * d loss / d logp_t for every token (0 at unscored tokens)
  GC_TRY(launch_token_loss(logp, old_logp, ref_logp, targets, mask, T, cu_seqlens, R, adv, clip_lo,
                           clip_hi, beta, agg, grad_loss, w.out5, w.g, w.loss, st));

  if (dtype != GC_BF16) {
    GC_TRY(simt_backward(H, ldH, W, ldW, dtype == GC_BF16_SIMT, targets, mask, T, D, V, temperature,
                         lse, w.g, dH, lddH, static_cast<float*>(dW), lddW, accumulate_dW, st));
    if (dW_bf16) GC_TRY(launch_cast_f32_bf16(w.dW_acc, D, dW_out, lddW_out, V, D, accumulate_out, st));
    return GC_OK;
  }

  const int64_t cap = ceil_div(T > 0 ? T : 1, 256) * 256;
  const int64_t ldS = ld_ds(V);
  const bool compact = mask != nullptr;
  const void* Hs = H;
  int64_t ldHs = ldH;
  const int32_t* targets_c = targets;
  const float* lse_c = lse;
  const float* g_c = w.g;
  const int32_t* rows = nullptr;
  const int32_t* n_rows = nullptr;
  if (compact) {
    if (sink.fwd_state) {
      // a1 was done by the forward on the same inputs: reuse its row list, compacted targets and
      // compacted H instead of recomputing them (the caller keeps that workspace untouched)
      Carver cf(const_cast<void*>(sink.fwd_state));
      FwdWs fw;
      carve_fwd(cf, T, D, V, dtype, &fw);
      w.rows = fw.rows; w.n_rows = fw.n_rows; w.targets_c = fw.targets_c; w.Hs = fw.Hs;
    } else {
      GC_TRY(launch_compact_rows(targets, mask, T, w.rows, w.n_rows, w.compact, st));
      GC_TRY(launch_gather_rows(H, ldH, 2, D, T, w.rows, w.n_rows, w.Hs, cap, st));
      GC_TRY(launch_gather_i32(targets, w.rows, w.n_rows, T, w.targets_c, st));
    }
    GC_TRY(launch_gather_f32(lse, w.rows, w.n_rows, T, w.lse_c, st));
    GC_TRY(launch_gather_f32(w.g, w.rows, w.n_rows, T, w.g_c, st));
    GC_TRY(launch_zero_rows_unscored(targets, mask, T, dH, lddH, 2, D, st));
    Hs = w.Hs; ldHs = D; targets_c = w.targets_c; lse_c = w.lse_c; g_c = w.g_c;
    rows = w.rows; n_rows = w.n_rows;
  }
  GC_CUDA_TRY(cudaMemsetAsync(w.counters, 0, sizeof(uint32_t) * kTcCounters, st));
  cudaEvent_t dh_done = sink.dh_done;
  const int64_t dh_rows = compact ? sink.dh_rows : T;         // rows that reach the contractions
  int ci = 0;
  for (int64_t row0 = 0; row0 < T; row0 += chunk) {
    if (ci + kCountersPerChunk > kTcCounters) {
      GC_CUDA_TRY(cudaMemsetAsync(w.counters, 0, sizeof(uint32_t) * kTcCounters, st));
      ci = 0;
    }
    const int64_t n_static = compact ? 0 : ((T - row0 < chunk) ? T - row0 : chunk);
    const int64_t rows_cap = compact ? ((cap - row0 < chunk) ? cap - row0 : chunk) : chunk;
    const char* Hc = static_cast<const char*>(Hs) + (size_t)row0 * (size_t)ldHs * 2;
    // a10: recompute the logit chunk, dS = (g/tau)(onehot - p) in bf16
    GC_TRY(tc_recompute_ds(Hc, ldHs, W, ldW, rows_cap, n_static, D, V, temperature,
                           targets_c + row0, lse_c + row0, g_c + row0, n_rows, row0, w.dS, ldS,
                           w.counters + ci, st));
    // a11: dH rows of this chunk
    GC_TRY(tc_dh(w.dS, ldS, rows_cap, n_static, W, ldW, D, V, rows ? rows + row0 : nullptr, n_rows,
                 row0, dH, lddH, w.counters + ci + 2, st));
    if (dh_done && row0 < (dh_rows > 0 ? dh_rows : 1) && row0 + chunk >= dh_rows)
      GC_CUDA_TRY(cudaEventRecord(dh_done, st));     // the last non-empty chunk: dH is complete
    // a12: dW accumulates over chunks in fp32
    if (sink.shards)
      GC_TRY(tc_dw_reduce_scatter(w.dS, ldS, rows_cap, n_static, Hc, ldHs, D, V, n_rows, row0,
                                  sink.shards, sink.world, sink.shard_rows, lddW,
                                  w.counters + ci + 1, st));
    else
      GC_TRY(tc_dw(w.dS, ldS, rows_cap, n_static, Hc, ldHs, D, V, n_rows, row0,
                   static_cast<float*>(dW), lddW, (accumulate_dW || row0 > 0) ? 1 : 0,
                   w.counters + ci + 1, st));
    ci += kCountersPerChunk;
  }
  if (dW_bf16) GC_TRY(launch_cast_f32_bf16(w.dW_acc, D, dW_out, lddW_out, V, D, accumulate_out, st));
  return GC_OK;
}

}  // namespace

namespace gc {
// gc_grpo_loss_bwd with the dH-done event of gc_grpo_step_host (host_api.cu); not exported
int grpo_loss_bwd_dh_event(const void* H, int64_t ldH, const void* W, int64_t ldW, int dtype,
                           const int32_t* targets, const uint8_t* mask, int64_t T, int64_t D,
                           int64_t V, float temperature, const int32_t* cu_seqlens, int32_t R,
                           const float* adv, const float* old_logp, const float* ref_logp,
                           float clip_lo, float clip_hi, float beta, int agg, const float* logp,
                           const float* lse, float grad_loss, void* dH, int64_t lddH, void* dW,
                           int64_t lddW, int dW_dtype, int accumulate_dW, void* workspace,
                           size_t workspace_bytes, void* cuda_stream, cudaEvent_t dh_done,
                           int64_t dh_rows) {
  if (dW_dtype != GC_F32 && dW_dtype != GC_BF16) return GC_ERR_DTYPE;
  DwSink sink{dW, lddW, accumulate_dW, nullptr, 0, 0, dW_dtype, nullptr};
  sink.dh_done = dh_done;
  sink.dh_rows = dh_rows;
  return loss_bwd_impl(H, ldH, W, ldW, dtype, targets, mask, T, D, V, temperature, cu_seqlens, R, adv,
                       old_logp, ref_logp, clip_lo, clip_hi, beta, agg, logp, lse, grad_loss, dH, lddH,
                       sink, 0, workspace, workspace_bytes, cuda_stream);
}
}  // namespace gc

extern "C" {

int gc_grpo_loss_bwd(const void* H, int64_t ldH, const void* W, int64_t ldW, int dtype,
                     const int32_t* targets, const uint8_t* mask, int64_t T, int64_t D, int64_t V,
                     float temperature, const int32_t* cu_seqlens, int32_t R, const float* adv,
                     const float* old_logp, const float* ref_logp, float clip_lo, float clip_hi,
                     float beta, int agg, const float* logp, const float* lse, float grad_loss,
                     void* dH, int64_t lddH, void* dW, int64_t lddW, int dW_dtype,
                     int accumulate_dW, int64_t chunk_tokens, const void* fwd_state,
                     void* workspace, size_t workspace_bytes, void* cuda_stream) {
  if (dW_dtype != GC_F32 && dW_dtype != GC_BF16) return GC_ERR_DTYPE;
  const DwSink sink{dW, lddW, accumulate_dW, nullptr, 0, 0, dW_dtype, fwd_state};
  return loss_bwd_impl(H, ldH, W, ldW, dtype, targets, mask, T, D, V, temperature, cu_seqlens, R, adv,
                       old_logp, ref_logp, clip_lo, clip_hi, beta, agg, logp, lse, grad_loss, dH, lddH,
                       sink, chunk_tokens, workspace, workspace_bytes, cuda_stream);
}

int gc_grpo_loss_bwd_reduce_scatter(
    const void* H, int64_t ldH, const void* W, int64_t ldW, int dtype, const int32_t* targets,
    const uint8_t* mask, int64_t T, int64_t D, int64_t V, float temperature,
    const int32_t* cu_seqlens, int32_t R, const float* adv, const float* old_logp,
    const float* ref_logp, float clip_lo, float clip_hi, float beta, int agg, const float* logp,
    const float* lse, float grad_loss, void* dH, int64_t lddH, float* const* dW_shards_host,
    int32_t world, int64_t shard_rows, int64_t ld_shard, int64_t chunk_tokens,
    const void* fwd_state, void* workspace, size_t workspace_bytes, void* cuda_stream) {
  if (!dW_shards_host) return GC_ERR_NULL;
  const DwSink sink{nullptr, ld_shard, 1, dW_shards_host, world, shard_rows, GC_F32, fwd_state};
  return loss_bwd_impl(H, ldH, W, ldW, dtype, targets, mask, T, D, V, temperature, cu_seqlens, R, adv,
                       old_logp, ref_logp, clip_lo, clip_hi, beta, agg, logp, lse, grad_loss, dH, lddH,
                       sink, chunk_tokens, workspace, workspace_bytes, cuda_stream);
}

int gc_validate_targets(const int32_t* targets, const uint8_t* mask, int64_t T, int64_t V,
                        int64_t* n_bad_host, void* cuda_stream) {
  if (!n_bad_host) return GC_ERR_NULL;
  *n_bad_host = 0;
  if (T == 0) return GC_OK;
  if (!targets) return GC_ERR_NULL;
  cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
  unsigned long long* d = nullptr;
  // debug helper: the one entry point that allocates and synchronises
  GC_CUDA_TRY(cudaMalloc(&d, sizeof(unsigned long long)));
  cudaMemsetAsync(d, 0, sizeof(unsigned long long), st);
  int s = launch_validate_targets(targets, mask, T, V, d, st);
  unsigned long long h = 0;
  if (s == GC_OK && cudaMemcpyAsync(&h, d, sizeof(h), cudaMemcpyDeviceToHost, st) != cudaSuccess)
    s = GC_ERR_CUDA;
  if (s == GC_OK && cudaStreamSynchronize(st) != cudaSuccess) s = GC_ERR_CUDA;
  cudaFree(d);
  *n_bad_host = (int64_t)h;
  return s;
}

int gc_compact_rows(const void* H, int64_t ldH, int dtype, const int32_t* targets,
                    const uint8_t* mask, int64_t T, int64_t D, int32_t* rows, int32_t* n_rows,
                    void* Hs, void* workspace, size_t workspace_bytes, void* cuda_stream) {
  if (T < 0 || T >= (1ll << 31) || D <= 0) return GC_ERR_SHAPE;
  if (!rows || !n_rows || (T > 0 && !targets)) return GC_ERR_NULL;
  if (!workspace || workspace_bytes < compact_ws_bytes(T)) return GC_ERR_WORKSPACE;
  cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
  GC_TRY(launch_compact_rows(targets, mask, T, rows, n_rows, workspace, st));
  if (Hs) {
    if (!H) return GC_ERR_NULL;
    if (ldH < D) return GC_ERR_SHAPE;
    GC_TRY(launch_gather_rows(H, ldH, elem_bytes(dtype), D, T, rows, n_rows, Hs, T, st));
  }
  return GC_OK;
}

static int check_value_args(const void* H, int64_t ldH, int dtype, const void* w, int64_t T,
                            int64_t D) {
  if (dtype != GC_F32 && dtype != GC_BF16) return GC_ERR_DTYPE;
  if (T < 0 || D <= 0 || D % 8 != 0 || ldH < D || T >= (1ll << 31)) return GC_ERR_SHAPE;
  if (!w || (T > 0 && !H)) return GC_ERR_NULL;
  if (!aligned16(H) || !aligned16(w) || (ldH * elem_bytes(dtype)) % 16 != 0) return GC_ERR_ALIGN;
  return GC_OK;
}

int gc_value_head_fwd(const void* H, int64_t ldH, int dtype, const void* w, float bias, int64_t T,
                      int64_t D, float* values, void* cuda_stream) {
  GC_TRY(check_value_args(H, ldH, dtype, w, T, D));
  if (T == 0) return GC_OK;
  if (!values) return GC_ERR_NULL;
  return launch_value_fwd(H, ldH, dtype == GC_BF16, w, bias, T, D, values,
                          static_cast<cudaStream_t>(cuda_stream));
}

int gc_gae(const float* rewards, const float* values, const uint8_t* mask,
           const int32_t* cu_seqlens, int32_t R, int64_t T, float gamma, float lambda, float* adv,
           float* returns, void* cuda_stream) {
  if (R < 0 || T < 0) return GC_ERR_SHAPE;
  if (!(gamma >= 0.f) || !(lambda >= 0.f)) return GC_ERR_ARG;
  if (R == 0 || T == 0) return GC_OK;
  if (!rewards || !values || !cu_seqlens || !adv || !returns) return GC_ERR_NULL;
  return launch_gae(rewards, values, mask, cu_seqlens, R, gamma, lambda, adv, returns,
                    static_cast<cudaStream_t>(cuda_stream));
}

size_t gc_critic_workspace_bytes(int64_t T, int64_t D) {
  if (T < 0 || D <= 0) return 0;
  const size_t a = value_loss_ws_bytes(T), b = value_bwd_ws_bytes(T, D);
  return (a > b ? a : b) + 256;
}

int gc_value_loss(const float* values, const float* old_values, const float* returns,
                  const uint8_t* mask, int64_t T, float clip_v, float grad_loss, float* out3,
                  float* g, void* workspace, size_t workspace_bytes, void* cuda_stream) {
  if (T < 0) return GC_ERR_SHAPE;
  if (!(clip_v >= 0.f)) return GC_ERR_ARG;
  if (!out3) return GC_ERR_NULL;
  cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
  if (T == 0) {
    GC_CUDA_TRY(cudaMemsetAsync(out3, 0, 3 * sizeof(float), st));
    return GC_OK;
  }
  if (!values || !old_values || !returns) return GC_ERR_NULL;
  if (!workspace || workspace_bytes < value_loss_ws_bytes(T)) return GC_ERR_WORKSPACE;
  if (reinterpret_cast<uintptr_t>(workspace) & 255) return GC_ERR_ALIGN;
  return launch_value_loss(values, old_values, returns, mask, T, clip_v, grad_loss, out3, g,
                           workspace, st);
}

int gc_value_head_bwd(const void* H, int64_t ldH, int dtype, const void* w, const float* g,
                      int64_t T, int64_t D, void* dH, int64_t lddH, float* dw, float* dbias,
                      void* workspace, size_t workspace_bytes, void* cuda_stream) {
  GC_TRY(check_value_args(H, ldH, dtype, w, T, D));
  if (!dw) return GC_ERR_NULL;
  cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
  if (T == 0) {
    GC_CUDA_TRY(cudaMemsetAsync(dw, 0, (size_t)D * sizeof(float), st));
    if (dbias) GC_CUDA_TRY(cudaMemsetAsync(dbias, 0, sizeof(float), st));
    return GC_OK;
  }
  if (!g || !dH) return GC_ERR_NULL;
  if (lddH < D || !aligned16(dH) || (lddH * elem_bytes(dtype)) % 16 != 0) return GC_ERR_ALIGN;
  if (!workspace || workspace_bytes < value_bwd_ws_bytes(T, D)) return GC_ERR_WORKSPACE;
  if (reinterpret_cast<uintptr_t>(workspace) & 255) return GC_ERR_ALIGN;
  return launch_value_bwd(H, ldH, dtype == GC_BF16, w, g, T, D, dH, lddH, dw, dbias, workspace, st);
}

size_t gc_balance_workspace_bytes(int32_t R) { return R < 0 ? 0 : balance_ws_bytes(R); }

int gc_balance_plan(const int32_t* cu_seqlens, int32_t R, const int32_t* group_offsets,
                    const uint8_t* keep, int32_t G, uint64_t w_lin, uint64_t w_quad,
                    int32_t bucket_size, uint64_t seed, int shuffle, int32_t* order,
                    int32_t* n_kept, int32_t* cu_out, int32_t* src_token, int32_t* n_tokens,
                    void* workspace, size_t workspace_bytes, void* cuda_stream) {
  if (R < 0 || G < 0) return GC_ERR_SHAPE;
  if (bucket_size < 1) return GC_ERR_ARG;
  if (!n_kept || !n_tokens || !cu_out) return GC_ERR_NULL;
  cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
  if (R == 0) {
    GC_CUDA_TRY(cudaMemsetAsync(n_kept, 0, sizeof(int32_t), st));
    GC_CUDA_TRY(cudaMemsetAsync(n_tokens, 0, sizeof(int32_t), st));
    GC_CUDA_TRY(cudaMemsetAsync(cu_out, 0, sizeof(int32_t), st));
    return GC_OK;
  }
  if (!cu_seqlens || !order || !src_token) return GC_ERR_NULL;
  if (keep && !group_offsets) return GC_ERR_NULL;
  if (!workspace || workspace_bytes < balance_ws_bytes(R)) return GC_ERR_WORKSPACE;
  if (reinterpret_cast<uintptr_t>(workspace) & 255) return GC_ERR_ALIGN;
  GC_TRY(check_arch());
  return launch_balance_plan(cu_seqlens, R, group_offsets, keep, G, w_lin, w_quad, bucket_size, seed,
                             shuffle, order, n_kept, cu_out, src_token, n_tokens, workspace, st);
}

int gc_gather_rows(const void* X, int64_t ldX, int dtype, int64_t D, const int32_t* rows,
                   const int32_t* n_rows, int64_t y_rows, void* Y, void* cuda_stream) {
  if (dtype != GC_F32 && dtype != GC_BF16) return GC_ERR_DTYPE;
  if (D <= 0 || ldX < D || y_rows < 0) return GC_ERR_SHAPE;
  if (y_rows == 0) return GC_OK;
  if (!X || !rows || !n_rows || !Y) return GC_ERR_NULL;
  if (!aligned16(X) || !aligned16(Y)) return GC_ERR_ALIGN;
  return launch_gather_rows(X, ldX, elem_bytes(dtype), D, y_rows, rows, n_rows, Y, y_rows,
                            static_cast<cudaStream_t>(cuda_stream));
}

int gc_gather_1d(const void* x, const int32_t* rows, const int32_t* n_rows, int64_t max_rows,
                 void* y, void* cuda_stream) {
  if (max_rows < 0) return GC_ERR_SHAPE;
  if (max_rows == 0) return GC_OK;
  if (!x || !rows || !n_rows || !y) return GC_ERR_NULL;
  return launch_gather_i32(static_cast<const int32_t*>(x), rows, n_rows, max_rows,
                           static_cast<int32_t*>(y), static_cast<cudaStream_t>(cuda_stream));
}

int gc_debug_gemm_bf16(const void* A, int64_t lda, int a_mn_major, const void* B, int64_t ldb,
                       int b_mn_major, float* C, int64_t ldc, int64_t M, int64_t N, int64_t K,
                       int accumulate, int cta_group, int dynamic_schedule, int dual_n,
                       int cluster4, int c_major, int m_band, int chunk_ntiles, int n_band,
                       void* cuda_stream) {
  if (!A || !B || !C) return GC_ERR_NULL;
  if (M <= 0 || N <= 0 || K <= 0) return GC_ERR_SHAPE;
  GC_TRY(check_arch());
  return tc_debug_gemm(A, lda, a_mn_major, B, ldb, b_mn_major, C, ldc, M, N, K, accumulate,
                       cta_group, dynamic_schedule, dual_n, cluster4, c_major, m_band, chunk_ntiles,
                       n_band, static_cast<cudaStream_t>(cuda_stream));
}

}  // extern "C"
