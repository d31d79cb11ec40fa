// host_api.cu -- the entry points that take the per-step inputs and outputs in HOST memory
// (gc_token_logprobs_host, gc_grpo_step_host): the end-to-end path a caller without device
// buffers uses, and what bench.py's `e2e` figure times.  They only marshal: host -> device copies,
// the device entry points of api.cu, device -> host copies.  The H copy is overlapped with the
// forward contraction: H is copied band by band (the forward's own M bands) on a side stream and
// each band is scored as soon as it has arrived, so only the first, small band is exposed.
#include <mutex>

#include "common.cuh"

using namespace gc;

namespace {

constexpr int kHostEvents = 68;        // fork + small inputs + up to 64 H bands + dH done / copied

// Side stream + events, per device, created on first use and kept (process-global state (iv) of
// gcore.h): creating them per call would cost more than the copy they hide.
struct HostCtx {
  cudaStream_t cs = nullptr;
  cudaEvent_t ev[kHostEvents] = {};
  bool ok = false;
  std::mutex use;      // held for the whole enqueue of one *_host call (events are re-recorded per call)
};
std::mutex g_ctx_mu;
HostCtx g_ctx[64];

int get_ctx(HostCtx** out) {
  int dev = 0;
  GC_CUDA_TRY(cudaGetDevice(&dev));
  if (dev < 0 || dev >= 64) return GC_ERR_CUDA;
  std::lock_guard<std::mutex> lk(g_ctx_mu);
  HostCtx& c = g_ctx[dev];
  if (!c.ok) {
    GC_CUDA_TRY(cudaStreamCreateWithFlags(&c.cs, cudaStreamNonBlocking));
    for (int i = 0; i < kHostEvents; ++i)
      GC_CUDA_TRY(cudaEventCreateWithFlags(&c.ev[i], cudaEventDisableTiming));
    c.ok = true;
  }
  *out = &c;
  return GC_OK;
}

int elem_bytes(int dtype) { return dtype == GC_F32 ? 4 : 2; }

// Bands of H rows: a short first band (its copy is the only exposed one), then the forward
// schedule's own M bands (whole multiples of 256 rows), at most 64.
int plan_bands(int64_t T, int64_t D, int64_t V, int dtype, int64_t* start /*[65]*/) {
  int64_t band = dtype == GC_BF16 ? tc_forward_band_rows(T, D, V) : 4096;
  if (band < 256) band = 256;
  while (ceil_div(T, band) > 62) band *= 2;
  int n = 0;
  start[0] = 0;
  int64_t r = T < 512 ? T : 512;
  if (T > 2 * band) { start[++n] = r; } else { r = 0; }
  while (r < T) {
    r = r + band < T ? r + band : T;
    start[++n] = r;
  }
  return n;     // bands are [start[i], start[i+1])
}

// Workspace the band-by-band forward needs: every band is its own gc_token_logprobs call and is
// planned on its own (vocab splits, partial statistics), and that plan is not monotonic in the row
// count -- a band can need more than the whole batch would.  So: the largest query over the bands.
size_t banded_inner_bytes(int64_t T, int64_t D, int64_t V, int dtype) {
  size_t need = gc_workspace_bytes(GC_OP_LOGPROBS, T, D, V, dtype, 0);
  if (T <= 0) return need;
  int64_t start[65];
  const int nb = plan_bands(T, D, V, dtype, start);
  for (int b = 0; b < nb; ++b) {
    const size_t n = gc_workspace_bytes(GC_OP_LOGPROBS, start[b + 1] - start[b], D, V, dtype, 0);
    if (n > need) need = n;
  }
  return need;
}

struct Staging {
  void* H; int32_t* y; uint8_t* m; float* logp; float* ent; float* lse;
};
size_t carve_staging(Carver& c, int64_t T, int64_t D, int dtype, Staging* s) {
  const size_t t = (size_t)(T > 0 ? T : 1);
  void* H = c.take<uint8_t>(t * (size_t)D * elem_bytes(dtype));
  int32_t* y = c.take<int32_t>(t);
  uint8_t* m = c.take<uint8_t>(t);
  float* lp = c.take<float>(t);
  float* en = c.take<float>(t);
  float* ls = c.take<float>(t);
  if (s) { s->H = H; s->y = y; s->m = m; s->logp = lp; s->ent = en; s->lse = ls; }
  return c.off;
}

// H2D of targets / mask / H on the side stream, band events; on the main stream each band is
// scored as it arrives.  loss == false: plain log-probs.
int banded_forward(HostCtx* cx, const void* H_host, const void* W, int64_t ldW, int dtype,
                   const int32_t* targets_host, const uint8_t* mask_host, int64_t T, int64_t D,
                   int64_t V, float tau, const Staging& sg, bool want_entropy, bool want_lse,
                   void* inner_ws, size_t inner_bytes, cudaStream_t st, int first_event) {
  int64_t start[65];
  const int nb = plan_bands(T, D, V, dtype, start);
  const size_t row_bytes = (size_t)D * elem_bytes(dtype);
  GC_CUDA_TRY(cudaMemcpyAsync(sg.y, targets_host, (size_t)T * 4, cudaMemcpyHostToDevice, cx->cs));
  if (mask_host) GC_CUDA_TRY(cudaMemcpyAsync(sg.m, mask_host, (size_t)T, cudaMemcpyHostToDevice, cx->cs));
  for (int b = 0; b < nb; ++b) {
    const int64_t r0 = start[b], r1 = start[b + 1];
    GC_CUDA_TRY(cudaMemcpyAsync(static_cast<char*>(sg.H) + (size_t)r0 * row_bytes,
                                static_cast<const char*>(H_host) + (size_t)r0 * row_bytes,
                                (size_t)(r1 - r0) * row_bytes, cudaMemcpyHostToDevice, cx->cs));
    GC_CUDA_TRY(cudaEventRecord(cx->ev[first_event + b], cx->cs));
  }
  for (int b = 0; b < nb; ++b) {
    const int64_t r0 = start[b], r1 = start[b + 1];
    GC_CUDA_TRY(cudaStreamWaitEvent(st, cx->ev[first_event + b], 0));
    GC_TRY(gc_token_logprobs(static_cast<char*>(sg.H) + (size_t)r0 * row_bytes, D, W, ldW, dtype,
                             sg.y + r0, mask_host ? sg.m + r0 : nullptr, r1 - r0, D, V, tau,
                             sg.logp + r0, want_entropy ? sg.ent + r0 : nullptr,
                             want_lse ? sg.lse + r0 : nullptr, inner_ws, inner_bytes, st));
  }
  return GC_OK;
}

}  // namespace

extern "C" {

int32_t gc_host_band_plan(int64_t T, int64_t D, int64_t V, int dtype, int64_t* starts_host) {
  if (T <= 0 || D <= 0 || V <= 0 || !starts_host) return 0;
  if (dtype != GC_F32 && dtype != GC_BF16 && dtype != GC_BF16_SIMT) return 0;
  return plan_bands(T, D, V, dtype, starts_host);
}

size_t gc_logprobs_host_workspace_bytes(int64_t T, int64_t D, int64_t V, int dtype) {
  if (T < 0 || D <= 0 || V <= 0) return 0;
  if (dtype != GC_F32 && dtype != GC_BF16 && dtype != GC_BF16_SIMT) return 0;
  return align_up(banded_inner_bytes(T, D, V, dtype), 256) + gc_host_staging_bytes(T, D, dtype);
}

size_t gc_host_staging_bytes(int64_t T, int64_t D, int dtype) {
  if (T < 0 || D <= 0) return 0;
  Carver c(nullptr);
  return carve_staging(c, T, D, dtype, nullptr) + 256;
}

int gc_token_logprobs_host(const void* H_host, const void* W, int64_t ldW, int dtype,
                           const int32_t* targets_host, const uint8_t* mask_host, int64_t T,
                           int64_t D, int64_t V, float temperature, float* logp_host,
                           float* entropy_host, void* workspace, size_t workspace_bytes,
                           void* cuda_stream) {
  if (T < 0 || D <= 0 || V <= 0) return GC_ERR_SHAPE;
  if (dtype != GC_F32 && dtype != GC_BF16 && dtype != GC_BF16_SIMT) return GC_ERR_DTYPE;
  if (T == 0) return GC_OK;
  if (!H_host || !targets_host || !logp_host || !W) return GC_ERR_NULL;
  const size_t inner = banded_inner_bytes(T, D, V, dtype);
  if (!workspace || workspace_bytes < align_up(inner, 256) + gc_host_staging_bytes(T, D, dtype))
    return GC_ERR_WORKSPACE;
  if (reinterpret_cast<uintptr_t>(workspace) & 255) return GC_ERR_ALIGN;
  cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
  HostCtx* cx = nullptr;
  GC_TRY(get_ctx(&cx));
  // one enqueue at a time per device: a second host thread on another stream would re-record the
  // events between this call's record and the wait that is meant to see it
  std::lock_guard<std::mutex> use_lock(cx->use);
  Carver c(static_cast<char*>(workspace) + align_up(inner, 256));
  Staging sg;
  carve_staging(c, T, D, dtype, &sg);
  // fork: the copies may start once earlier work on `st` (a previous call's kernels reading the
  // staging buffers) is done
  GC_CUDA_TRY(cudaEventRecord(cx->ev[0], st));
  GC_CUDA_TRY(cudaStreamWaitEvent(cx->cs, cx->ev[0], 0));
  GC_TRY(banded_forward(cx, H_host, W, ldW, dtype, targets_host, mask_host, T, D, V, temperature, sg,
                        entropy_host != nullptr, false, workspace, inner, st, 2));
  GC_CUDA_TRY(cudaMemcpyAsync(logp_host, sg.logp, (size_t)T * 4, cudaMemcpyDeviceToHost, st));
  if (entropy_host)
    GC_CUDA_TRY(cudaMemcpyAsync(entropy_host, sg.ent, (size_t)T * 4, cudaMemcpyDeviceToHost, st));
  return GC_OK;
}

// ---- one whole training step of the loss head from host buffers ---------------------------------
namespace {
struct StepWs {
  void* fwd; size_t fwd_bytes; void* bwd; size_t bwd_bytes; Staging sg;
  int32_t* cu; float* rewards; int32_t* go; float* adv; float* old_lp; float* ref_lp; float* out5;
  void* dH;
};
size_t carve_step(Carver& c, int64_t T, int64_t D, int64_t V, int dtype, int32_t R, int32_t G,
                  int dW_dtype, StepWs* w) {
  // forward workspace: the banded forward's need (max over bands), then the loss scratch -- the
  // part of the GC_OP_LOSS_FWD query that lies behind its GC_OP_LOGPROBS part
  const size_t lp = align_up(gc_workspace_bytes(GC_OP_LOGPROBS, T, D, V, dtype, 0), 256);
  const size_t lf = align_up(gc_workspace_bytes(GC_OP_LOSS_FWD, T, D, V, dtype, 0), 256);
  const size_t fb = align_up(banded_inner_bytes(T, D, V, dtype), 256) + (lf > lp ? lf - lp : 0) + 256;
  const size_t bb = align_up(gc_bwd_workspace_bytes(T, D, V, dtype, 0, dW_dtype), 256);
  void* f = c.take<uint8_t>(fb);
  void* b = c.take<uint8_t>(bb);
  Staging sg;
  carve_staging(c, T, D, dtype, &sg);
  const size_t t = (size_t)(T > 0 ? T : 1);
  int32_t* cu = c.take<int32_t>((size_t)R + 1);
  float* rw = c.take<float>((size_t)(R > 0 ? R : 1));
  int32_t* go = c.take<int32_t>((size_t)G + 1);
  float* adv = c.take<float>((size_t)(R > 0 ? R : 1));
  float* ol = c.take<float>(t);
  float* rf = c.take<float>(t);
  float* o5 = c.take<float>(64);
  void* dH = c.take<uint8_t>(t * (size_t)D * elem_bytes(dtype));
  if (w) {
    w->fwd = f; w->fwd_bytes = fb; w->bwd = b; w->bwd_bytes = bb; w->sg = sg; w->cu = cu;
    w->rewards = rw; w->go = go; w->adv = adv; w->old_lp = ol; w->ref_lp = rf; w->out5 = o5; w->dH = dH;
  }
  return c.off;
}
}  // namespace

size_t gc_step_host_workspace_bytes(int64_t T, int64_t D, int64_t V, int dtype, int32_t R, int32_t G,
                                    int dW_dtype) {
  if (T < 0 || D <= 0 || V <= 0 || R < 0 || G < 0) return 0;
  Carver c(nullptr);
  return carve_step(c, T, D, V, dtype, R, G, dW_dtype, nullptr) + 256;
}

int gc_grpo_step_host(const void* H_host, const void* W, int64_t ldW, int dtype,
                      const int32_t* targets_host, const uint8_t* mask_host, int64_t T, int64_t D,
                      int64_t V, float temperature, const int32_t* cu_seqlens_host, int32_t R,
                      const float* rewards_host, const int32_t* group_offsets_host, int32_t G,
                      float adv_eps, const float* old_logp_host, const float* ref_logp_host,
                      float clip_lo, float clip_hi, float beta, int agg, float grad_loss,
                      float* out5_host, float* logp_host, void* dH_host, void* dW, int64_t lddW,
                      int dW_dtype, int accumulate_dW, void* workspace, size_t workspace_bytes,
                      void* cuda_stream) {
  if (T <= 0 || D <= 0 || V <= 0 || R < 1 || G < 1) return GC_ERR_SHAPE;
  if (dtype != GC_F32 && dtype != GC_BF16 && dtype != GC_BF16_SIMT) return GC_ERR_DTYPE;
  if (!H_host || !W || !targets_host || !cu_seqlens_host || !rewards_host || !group_offsets_host ||
      !old_logp_host || !out5_host || !dH_host || !dW)
    return GC_ERR_NULL;
  if (beta != 0.f && !ref_logp_host) return GC_ERR_NULL;
  if (!workspace || workspace_bytes < gc_step_host_workspace_bytes(T, D, V, dtype, R, G, dW_dtype))
    return GC_ERR_WORKSPACE;
  if (reinterpret_cast<uintptr_t>(workspace) & 255) return GC_ERR_ALIGN;
  cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
  HostCtx* cx = nullptr;
  GC_TRY(get_ctx(&cx));
  // one enqueue at a time per device: a second host thread on another stream would re-record the
  // events between this call's record and the wait that is meant to see it
  std::lock_guard<std::mutex> use_lock(cx->use);
  Carver c(workspace);
  StepWs w;
  carve_step(c, T, D, V, dtype, R, G, dW_dtype, &w);
  GC_CUDA_TRY(cudaEventRecord(cx->ev[0], st));
  GC_CUDA_TRY(cudaStreamWaitEvent(cx->cs, cx->ev[0], 0));
  // small inputs first (side stream), then H band by band inside banded_forward
  GC_CUDA_TRY(cudaMemcpyAsync(w.cu, cu_seqlens_host, ((size_t)R + 1) * 4, cudaMemcpyHostToDevice, cx->cs));
  GC_CUDA_TRY(cudaMemcpyAsync(w.rewards, rewards_host, (size_t)R * 4, cudaMemcpyHostToDevice, cx->cs));
  GC_CUDA_TRY(cudaMemcpyAsync(w.go, group_offsets_host, ((size_t)G + 1) * 4, cudaMemcpyHostToDevice, cx->cs));
  GC_CUDA_TRY(cudaMemcpyAsync(w.old_lp, old_logp_host, (size_t)T * 4, cudaMemcpyHostToDevice, cx->cs));
  if (ref_logp_host)
    GC_CUDA_TRY(cudaMemcpyAsync(w.ref_lp, ref_logp_host, (size_t)T * 4, cudaMemcpyHostToDevice, cx->cs));
  GC_CUDA_TRY(cudaEventRecord(cx->ev[1], cx->cs));
  // forward, band by band as H arrives (logp, lse kept for the backward)
  const size_t fwd_inner = banded_inner_bytes(T, D, V, dtype);
  GC_TRY(banded_forward(cx, H_host, W, ldW, dtype, targets_host, mask_host, T, D, V, temperature,
                        w.sg, false, true, w.fwd, fwd_inner, st, 2));
  GC_CUDA_TRY(cudaStreamWaitEvent(st, cx->ev[1], 0));
  GC_TRY(gc_grpo_advantages(w.rewards, w.go, G, adv_eps, 0, 0, w.adv, nullptr, st));
  const uint8_t* m = mask_host ? w.sg.m : nullptr;
  const float* rf = ref_logp_host ? w.ref_lp : nullptr;
  void* loss_ws = static_cast<char*>(w.fwd) + align_up(fwd_inner, 256);
  GC_TRY(gc_grpo_token_loss(w.sg.logp, w.old_lp, rf, w.sg.y, m, T, w.cu, R, w.adv, clip_lo, clip_hi,
                            beta, agg, 1.0f, w.out5, nullptr, loss_ws,
                            w.fwd_bytes - align_up(fwd_inner, 256), st));
  GC_CUDA_TRY(cudaMemcpyAsync(out5_host, w.out5, 5 * sizeof(float), cudaMemcpyDeviceToHost, st));
  if (logp_host)
    GC_CUDA_TRY(cudaMemcpyAsync(logp_host, w.sg.logp, (size_t)T * 4, cudaMemcpyDeviceToHost, st));
  // dH is complete after the last chunk's dH contraction: its copy back to the host runs on the
  // side stream under the last dW contraction (bf16 tcgen05 path; the SIMT path copies at the end)
  const bool overlap_dh = dtype == GC_BF16;
  int64_t n_scored = 0;            // host-side count: which chunk is the last non-empty one
  if (overlap_dh)
    for (int64_t t = 0; t < T; ++t)
      n_scored += (targets_host[t] >= 0 && (!mask_host || mask_host[t] != 0)) ? 1 : 0;
  GC_TRY(gc::grpo_loss_bwd_dh_event(w.sg.H, D, W, ldW, dtype, w.sg.y, m, T, D, V, temperature, w.cu, R,
                                    w.adv, w.old_lp, rf, clip_lo, clip_hi, beta, agg, w.sg.logp,
                                    w.sg.lse, grad_loss, w.dH, D, dW, lddW, dW_dtype, accumulate_dW,
                                    w.bwd, w.bwd_bytes, st,
                                    overlap_dh ? cx->ev[kHostEvents - 1] : nullptr, n_scored));
  const size_t dh_bytes = (size_t)T * (size_t)D * elem_bytes(dtype);
  if (overlap_dh) {
    GC_CUDA_TRY(cudaStreamWaitEvent(cx->cs, cx->ev[kHostEvents - 1], 0));
    GC_CUDA_TRY(cudaMemcpyAsync(dH_host, w.dH, dh_bytes, cudaMemcpyDeviceToHost, cx->cs));
    GC_CUDA_TRY(cudaEventRecord(cx->ev[kHostEvents - 2], cx->cs));
    GC_CUDA_TRY(cudaStreamWaitEvent(st, cx->ev[kHostEvents - 2], 0));     // join: ordered on `st`
  } else {
    GC_CUDA_TRY(cudaMemcpyAsync(dH_host, w.dH, dh_bytes, cudaMemcpyDeviceToHost, st));
  }
  return GC_OK;
}

}  // extern "C"
