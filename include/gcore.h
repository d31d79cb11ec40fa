/* gcore.h -- C ABI of the RLHF scoring hot path for one NVIDIA B200 (sm_100a).
 *
 * The path is stages 3 and 4 of the 4-stage RLHF workflow of G-Core (arxiv 2507.22789):
 *   stage 3 "the policy and reference policy computes their reference log probabilities"
 *           (sec 2.2), run data-parallel on all GPUs (sec 3.2);
 *   stage 4 "The actor ... trained on the batch ... and the loss function", for
 *           GRPO, the algorithm the paper names as typical (sec 2.3);
 *   the dynamic-sampling group filter of PAPER.md:150 (sec 3.2).
 * The paper prints no formula; the arithmetic is BASELINE.json:north_star, restated step by
 * step in SURVEY.md sec 8(c) and DESIGN.md sec 2.  Notation: T packed tokens, D hidden, V vocab,
 * R responses, G groups; H[T,D] hidden states, W[V,D] LM-head weight (logits = H W^T / tau),
 * y[T] target ids, m[T] response mask.
 *
 * Conventions (all entry points)
 *   - Every pointer is a DEVICE pointer owned by the caller unless the name ends in "_host".
 *     The library never allocates, frees or keeps memory; scratch comes from `workspace`
 *     (size from gc_workspace_bytes; 256-byte aligned).
 *   - Calls enqueue work on `cuda_stream` (a cudaStream_t; NULL = legacy default stream) and
 *     return without synchronising.  Inputs must stay alive until the stream has passed the call.
 *   - Return value is a gc_status.  Host-checkable errors are reported before any launch.  No
 *     exceptions, no abort(), no environment variables.  Process-global state is limited to:
 *     (i) a write-once, atomically published cache of launch attributes per kernel and device
 *     (idempotent: host threads may race on a first launch); (ii) the measurement aid
 *     gc_kernel_timing_* (mutex-guarded, off by default); (iii) the tile counter and progress ring of
 *     gc_debug_gemm_bf16 (a test entry point; do not run two of them concurrently); (iv) one side
 *     stream and a few events per device for the *_host and attention entry points (their enqueue
 *     is serialised per device by a mutex, so host threads may call them on different streams);
 *     (v) the 33 KB scratch array of gc_value_loss_static_scratch.  None of it changes results.  Calls on different streams need different workspaces.
 *   - The tensor-core kernels are persistent (one CTA per SM) and the CTA pairs of the dH launch
 *     pace one another through progress counters: they are meant to own the GPU.  A kernel of
 *     another stream or process that holds some SMs only delays them, but every wait inside the
 *     kernels carries a watchdog of 2^36 cycles (35-60 s) that turns a wait longer than that --
 *     a protocol bug, or SMs withheld for that long -- into a launch failure (GC_ERR_CUDA at the
 *     next call that checks) instead of a hang.  The bound is that long because the cycle counter
 *     keeps running while the context is time-sliced out or slowed by a profiler / sanitizer.
 *   - Matrices are row-major; ld* are row strides in ELEMENTS.  For GC_BF16: D % 8 == 0,
 *     ld % 8 == 0, base pointers 16-byte aligned (TMA).
 *   - A token is SCORED iff (mask == NULL or mask[t] != 0) and targets[t] >= 0.  targets[t] >= V
 *     is a caller error (undefined result for that row; use gc_validate_targets to check).
 *     With a mask, only scored rows reach the tensor cores (row selection a1).  mask == NULL
 *     declares (almost) every row scored and skips the selection: rows with targets[t] < 0 are
 *     then computed and discarded -- pass a mask (all ones will do) when many targets are < 0.
 *   - Outputs at unscored rows are exactly 0 (logp, entropy, lse, rows of dH).
 *   - Same inputs give bit-identical outputs from run to run (no floating-point atomics).
 */
#ifndef GCORE_H_
#define GCORE_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef enum {
  GC_OK = 0,
  GC_ERR_NULL = 1,      /* a required pointer is NULL */
  GC_ERR_SHAPE = 2,     /* T, D, V, R, G out of range; ld < D; D not supported by this dtype */
  GC_ERR_DTYPE = 3,     /* unknown gc_dtype */
  GC_ERR_ALIGN = 4,     /* pointer or ld alignment */
  GC_ERR_WORKSPACE = 5, /* workspace NULL or smaller than gc_workspace_bytes */
  GC_ERR_ARG = 6,       /* temperature <= 0, clip < 0, eps < 0, bad enum */
  GC_ERR_ARCH = 7,      /* current device is not compute capability 10.x */
  GC_ERR_CUDA = 8       /* a CUDA runtime/driver call failed (launch configuration etc.) */
} gc_status;

typedef enum {
  GC_F32 = 0,       /* H, W, dH fp32; plain SIMT kernels (BASELINE.json configs[0]) */
  GC_BF16 = 1,      /* H, W, dH bf16, fp32 accumulation; tcgen05/TMEM/TMA kernels */
  GC_BF16_SIMT = 2  /* bf16 operands through the SIMT kernels: slow cross-check path */
} gc_dtype;

typedef enum {
  GC_AGG_TOKEN_MEAN = 0, /* loss = sum_t m_t l_t / max(sum_t m_t, 1)           (default) */
  GC_AGG_SEQ_MEAN = 1    /* loss = mean over responses of per-response token means        */
} gc_agg;

typedef enum { GC_OP_LOGPROBS = 0, GC_OP_LOSS_FWD = 1, GC_OP_LOSS_BWD = 2 } gc_op;

/* Static string for a gc_status (never NULL). */
const char* gc_status_string(int status);

/* Name of the CUDA error behind the calling thread's most recent GC_ERR_CUDA ("cudaSuccess" if
 * there was none): thread-local, static string. */
const char* gc_last_cuda_error(void);

/* Library version (major*10000 + minor*100 + patch). */
int gc_version(void);

/* Bytes of workspace the given op needs for these shapes.  chunk_tokens is the backward's
 * T-chunk (rows of the dS buffer); 0 lets the library pick.
 * Returns 0 on invalid arguments. */
size_t gc_workspace_bytes(int op, int64_t T, int64_t D, int64_t V, int dtype, int64_t chunk_tokens);

/* ---- stage 3: token log-probs + entropy (north_star: "fused LM-head contraction H.W^T over
 * the vocabulary, then an online (chunked, never materialised) log-softmax, then a gather of
 * the sampled token's log-prob and the per-token entropy").
 *   z[t,v]     = (sum_d H[t,d] W[v,d]) / temperature
 *   lse[t]     = ln sum_v exp z[t,v];   logp[t] = z[t,y_t] - lse[t]
 *   entropy[t] = -sum_v p ln p,  p = exp(z - lse)                      (natural log)
 * H [T,D] (ldH), W [V,D] (ldW) of `dtype`; targets [T] int32; mask [T] uint8 or NULL (= all 1).
 * logp [T] f32 required; entropy, lse [T] f32 nullable.  The [T,V] logits are never stored. */
int gc_token_logprobs(const void* H, int64_t ldH, const void* W, int64_t ldW, int dtype,
                      const int32_t* targets, const uint8_t* mask,
                      int64_t T, int64_t D, int64_t V, float temperature,
                      float* logp, float* entropy, float* lse,
                      void* workspace, size_t workspace_bytes, void* cuda_stream);

/* Same computation with the per-step inputs and outputs in HOST memory (pinned for async
 * copies): H_host [T,D] dense, targets_host, mask_host (nullable) are copied to the device,
 * logp_host / entropy_host (nullable) are copied back, staged in `workspace`
 * (gc_logprobs_host_workspace_bytes(T, D, V, dtype): the staging buffers,
 * gc_host_staging_bytes(T, D, dtype), plus the LARGEST gc_workspace_bytes(GC_OP_LOGPROBS, rows, ...)
 * over the bands below -- each band is planned on its own and a band can need more scratch than the
 * whole batch would).  W is model state
 * and stays a device pointer.  The H copy overlaps the contraction: H travels band by band (the
 * forward schedule's M bands, after a short first band) on a library-owned side stream and each
 * band is scored on `cuda_stream` as soon as it has arrived; the results are complete in stream
 * order on `cuda_stream`.  Process-global state (iv): one side stream and a few events per device,
 * created on first use.  Used for the end-to-end measurement. */
size_t gc_host_staging_bytes(int64_t T, int64_t D, int dtype);
size_t gc_logprobs_host_workspace_bytes(int64_t T, int64_t D, int64_t V, int dtype);
/* The bands the *_host entry points cut H into: writes starts_host[0..n] (HOST array of 65 entries),
 * band b = rows [starts_host[b], starts_host[b+1]), and returns n (<= 64; 0 on invalid arguments).
 * Host-only arithmetic; exposed so that the workspace sizing above can be checked without a GPU. */
int32_t gc_host_band_plan(int64_t T, int64_t D, int64_t V, int dtype, int64_t* starts_host);
int gc_token_logprobs_host(const void* H_host, const void* W, int64_t ldW, int dtype,
                           const int32_t* targets_host, const uint8_t* mask_host,
                           int64_t T, int64_t D, int64_t V, float temperature,
                           float* logp_host, float* entropy_host,
                           void* workspace, size_t workspace_bytes, void* cuda_stream);

/* One whole training step of the loss head from HOST buffers (the end-to-end fwd+bwd path):
 * copies H, targets, mask, cu_seqlens, rewards, group_offsets, old / ref log-probs to the device
 * (H band by band, overlapped with the forward as above), then gc_grpo_advantages (population
 * std, no group drop) -> forward -> loss -> backward, and copies out5 [5], logp (nullable) and
 * dH [T,D] back to the host -- dH on the side stream as soon as the last non-empty chunk's dH
 * contraction has finished, i.e. under the last dW contraction.  dW [V,D] (lddW, dW_dtype,
 * accumulate_dW as in gc_grpo_loss_bwd) is model state and stays on the device.  Everything is
 * ordered on `cuda_stream` when the call's work completes there.
 * workspace: gc_step_host_workspace_bytes(T, D, V, dtype, R, G, dW_dtype). */
size_t gc_step_host_workspace_bytes(int64_t T, int64_t D, int64_t V, int dtype, int32_t R, int32_t G,
                                    int dW_dtype);
int gc_grpo_step_host(const void* H_host, const void* W, int64_t ldW, int dtype,
                      const int32_t* targets_host, const uint8_t* mask_host,
                      int64_t T, int64_t D, int64_t V, float temperature,
                      const int32_t* cu_seqlens_host, int32_t R,
                      const float* rewards_host, const int32_t* group_offsets_host, int32_t G,
                      float adv_eps, const float* old_logp_host, const float* ref_logp_host,
                      float clip_lo, float clip_hi, float beta, int agg, float grad_loss,
                      float* out5_host, float* logp_host, void* dH_host,
                      void* dW, int64_t lddW, int dW_dtype, int accumulate_dW,
                      void* workspace, size_t workspace_bytes, void* cuda_stream);

/* ---- group filter + GRPO advantages ("filter out prompts with the accuracy
 * equal to 1 and 0"; north_star "GRPO group-normalised advantages"; steps 4-5).
 *   keep[g] = 0 iff all rewards of group g are equal (exact float compare)
 *   A_i     = (r_i - mean_g) / (std_g + eps)
 * rewards [R] f32; group_offsets [G+1] int32, ascending, group g = responses
 * [group_offsets[g], group_offsets[g+1]), R = group_offsets[G] (read on the device).
 * unbiased_std: 0 population std (default), 1 sample std (n-1).  drop_constant_groups: 1 ->
 * constant groups get A = 0 and keep = 0; 0 -> keep = 1 everywhere (A = 0 for constant groups
 * follows from eps > 0).  adv [R] f32; keep [G] uint8 nullable. */
int gc_grpo_advantages(const float* rewards, const int32_t* group_offsets, int32_t G,
                       float eps, int unbiased_std, int drop_constant_groups,
                       float* adv, uint8_t* keep, void* cuda_stream);

/* ---- stage 4 forward: log-probs as above, then the GRPO loss (north_star: "clipped-ratio
 * policy loss with a k3 KL penalty against the reference"; steps 6-7).  Per scored token t of
 * response r (cu_seqlens[r] <= t < cu_seqlens[r+1]):
 *   rho = exp(logp - old_logp);  s = min(rho A_r, clip(rho, 1-clip_lo, 1+clip_hi) A_r)
 *   d = ref_logp - logp;  k3 = exp(d) - d - 1;  l = -s + beta k3
 * cu_seqlens [R+1] int32 with cu_seqlens[0] = 0, cu_seqlens[R] = T.  adv [R].  old_logp [T];
 * ref_logp [T], nullable iff beta == 0.  out5 [5] f32 on the device:
 *   {loss, pg_loss, kl_mean, clip_frac, n_scored}; loss = pg_loss + beta kl_mean (both use
 *   `agg`), clip_frac = clipped scored tokens / n_scored.
 * logp and lse [T] are required (the backward needs them); entropy nullable. */
int gc_grpo_loss_fwd(const void* H, int64_t ldH, const void* W, int64_t ldW, int dtype,
                     const int32_t* targets, const uint8_t* mask,
                     int64_t T, int64_t D, int64_t V, float temperature,
                     const int32_t* cu_seqlens, int32_t R, const float* adv,
                     const float* old_logp, const float* ref_logp,
                     float clip_lo, float clip_hi, float beta, int agg,
                     float* out5, float* logp, float* entropy, float* lse,
                     void* workspace, size_t workspace_bytes, void* cuda_stream);

/* ---- stage 4 backward (north_star: "The backward pass recomputes each logit chunk to produce
 * dH and dW without storing [T,V] logits"; steps 8-9).  Takes the forward's logp and lse.
 *   g_t     = grad_loss * d loss / d logp_t
 *   dz[t,v] = g_t (1[v = y_t] - exp(z[t,v] - lse[t]))
 *   dH[t,:] = (1/tau) sum_v dz[t,v] W[v,:]        dW[v,:] (+)= (1/tau) sum_t dz[t,v] H[t,:]
 * dH [T,D] (lddH) in H's dtype, zero rows at unscored tokens.  dW [V,D] (lddW) of dW_dtype:
 * GC_F32 (BASELINE.json configs[4]: "dW accumulated in fp32"), or GC_BF16 -- the chunks then
 * accumulate in an fp32 [V,D] staging buffer inside the workspace and are rounded to bf16 ONCE,
 * after the last chunk (SURVEY.md sec 8(c) reading 13).  accumulate_dW != 0 adds to the existing
 * contents (for GC_BF16: out = bf16(out + sum), one rounding per call).  chunk_tokens: rows of the
 * bf16 dS chunk buffer (0 = library picks; must match the workspace query).
 * fwd_state (nullable): the workspace gc_grpo_loss_fwd was given for the SAME inputs, untouched
 * since; the backward then reuses the forward's row selection (a1: row list, compacted targets,
 * compacted H) instead of recomputing it.  It must not overlap `workspace` (GC_ERR_ARG if it does).
 * The library cannot tell whether the state still belongs to these inputs: a later forward with the
 * same workspace overwrites it (the Python binding tracks that and then passes NULL).
 * workspace: gc_bwd_workspace_bytes(T, D, V, dtype, chunk_tokens, dW_dtype)
 * (= gc_workspace_bytes(GC_OP_LOSS_BWD, ...) for GC_F32). */
size_t gc_bwd_workspace_bytes(int64_t T, int64_t D, int64_t V, int dtype, int64_t chunk_tokens,
                              int dW_dtype);
int gc_grpo_loss_bwd(const void* H, int64_t ldH, const void* W, int64_t ldW, int dtype,
                     const int32_t* targets, const uint8_t* mask,
                     int64_t T, int64_t D, int64_t V, float temperature,
                     const int32_t* cu_seqlens, int32_t R, const float* adv,
                     const float* old_logp, const float* ref_logp,
                     float clip_lo, float clip_hi, float beta, int agg,
                     const float* logp, const float* lse, float grad_loss,
                     void* dH, int64_t lddH, void* dW, int64_t lddW, int dW_dtype,
                     int accumulate_dW, int64_t chunk_tokens, const void* fwd_state,
                     void* workspace, size_t workspace_bytes, void* cuda_stream);

/* ---- stage 4 backward fused with its data-parallel exchange (training
 * across ranks needs "one all-reduce (or reduce-scatter ...) of fp32 dW [V,D]").  Same computation
 * as gc_grpo_loss_bwd, but the dW contraction's epilogue TMA-reduce-adds every tile straight into
 * the shard of the rank that owns its vocab rows, so the reduce-scatter rides on the contraction
 * and no full-size local dW exists.  dW_shards_host: HOST array of `world` (<= 8) DEVICE pointers;
 * entry r is rank r's shard, fp32 [shard_rows, D] with row stride ld_shard, holding vocab rows
 * [r shard_rows, (r+1) shard_rows) -- this rank's own buffer or a peer-mapped one (CUDA IPC /
 * cudaDeviceEnablePeerAccess; NVLink carries the adds).  shard_rows % 32 == 0, shard_rows * world
 * >= V.  Protocol: every rank zeroes its own shard, all ranks synchronise, every rank runs this
 * call, all ranks synchronise again; each shard then holds the sum over ranks of those rows of dW
 * (divide by `world` or fold 1/world into grad_loss for a mean).  Adds from different ranks meet
 * in no fixed order: reruns agree to rounding, not bit for bit.  GC_BF16 only. */
int gc_grpo_loss_bwd_reduce_scatter(
    const void* H, int64_t ldH, const void* W, int64_t ldW, int dtype,
    const int32_t* targets, const uint8_t* mask, int64_t T, int64_t D, int64_t V, float temperature,
    const int32_t* cu_seqlens, int32_t R, const float* adv,
    const float* old_logp, const float* ref_logp, float clip_lo, float clip_hi, float beta, int agg,
    const float* logp, const float* lse, float grad_loss,
    void* dH, int64_t lddH, float* const* dW_shards_host, int32_t world, int64_t shard_rows,
    int64_t ld_shard, int64_t chunk_tokens, const void* fwd_state,
    void* workspace, size_t workspace_bytes, void* cuda_stream);

/* ---- helpers ---- */
/* Debug: synchronises the stream; *n_bad_host = number of scored tokens with target >= V. */
int gc_validate_targets(const int32_t* targets, const uint8_t* mask, int64_t T, int64_t V,
                        int64_t* n_bad_host, void* cuda_stream);

/* Row selection: rows[0..n) = ascending indices of scored tokens,
 * *n_rows (device int32) = n; if Hs != NULL also gathers H[rows[i],:] into Hs[i,:] (dense,
 * ld = D).  Exposed for tests and the HBM-roofline measurement; the entry points above call
 * the same kernels internally.  workspace: gc_workspace_bytes(GC_OP_LOGPROBS, ...). */
int gc_compact_rows(const void* H, int64_t ldH, int dtype, const int32_t* targets,
                    const uint8_t* mask, int64_t T, int64_t D,
                    int32_t* rows, int32_t* n_rows, void* Hs,
                    void* workspace, size_t workspace_bytes, void* cuda_stream);

/* The loss kernels alone on given log-probs (steps 6-8): out5 as in gc_grpo_loss_fwd;
 * g [T] nullable (d loss / d logp * grad_loss).  Exposed for tests and for the HBM-roofline
 * measurement of the elementwise kernels on a scaled-up stand-in.
 * Any R >= 1 (empty responses, i.e. repeated cu_seqlens entries, are fine; the fwd / bwd entry
 * points above additionally require R <= T + 1, the size their internal loss scratch is carved
 * for).  logp, old_logp, ref_logp, targets, g 16-byte aligned; mask 4-byte aligned.  Unscored
 * positions may hold anything (inf, NaN): only scored tokens enter the sums.
 * workspace: gc_loss_workspace_bytes(T, R). */
size_t gc_loss_workspace_bytes(int64_t T, int32_t R);
int gc_grpo_token_loss(const float* logp, const float* old_logp, const float* ref_logp,
                       const int32_t* targets, const uint8_t* mask, int64_t T,
                       const int32_t* cu_seqlens, int32_t R, const float* adv,
                       float clip_lo, float clip_hi, float beta, int agg, float grad_loss,
                       float* out5, float* g,
                       void* workspace, size_t workspace_bytes, void* cuda_stream);

/* ---- the PPO variant of stages 3-4: critic values, GAE, clipped value loss (SURVEY.md sec 8(f)
 * NEXT-2).  PAPER.md:96 (sec 2.2): in PPO "the critic computes values"; stage 3
 * computes them, stage 4 trains actor and critic.  The paper prints no formula; the arithmetic is
 * PPO [18] as read in DESIGN.md sec 11:
 *   v_t      = sum_d H[t,d] w[d] + bias                                      (gc_value_head_fwd)
 *   delta_t  = r_t + gamma v_next(t) - v_t;  A_t = delta_t + gamma lambda A_next(t);
 *   return_t = A_t + v_t, over the scored tokens of each response in order (a masked token is not
 *              part of the trajectory; v_next = 0 after the last); 0 at unscored tokens   (gc_gae)
 *   v_clip   = clip(v, v_old - clip_v, v_old + clip_v);  l_t = 0.5 max((v-ret)^2, (v_clip-ret)^2)
 *   loss     = sum m l / max(sum m, 1);  out3 = {loss, clip_frac, n_scored};
 *   g_t      = grad_loss d loss / d v_t                                       (gc_value_loss)
 *   dH[t,:]  = g_t w;  dw = sum_t g_t H[t,:];  dbias = sum_t g_t              (gc_value_head_bwd)
 * The policy side of PPO is gc_grpo_token_loss with one "response" per token (cu_seqlens = 0..T)
 * and adv = the per-token GAE advantages.  H [T,D] and w [D] of `dtype` (GC_F32 / GC_BF16),
 * D % 8 == 0, 16-byte aligned rows; values, rewards, adv, returns, g [T] f32; mask [T] uint8
 * nullable; dH in H's dtype; dw [D] f32, dbias device [1] f32 nullable.  Deterministic. */
int gc_value_head_fwd(const void* H, int64_t ldH, int dtype, const void* w, float bias, int64_t T,
                      int64_t D, float* values, void* cuda_stream);
int gc_gae(const float* rewards, const float* values, const uint8_t* mask,
           const int32_t* cu_seqlens, int32_t R, int64_t T, float gamma, float lambda,
           float* adv, float* returns, void* cuda_stream);
size_t gc_critic_workspace_bytes(int64_t T, int64_t D);
int gc_value_loss(const float* values, const float* old_values, const float* returns,
                  const uint8_t* mask, int64_t T, float clip_v, float grad_loss, float* out3,
                  float* g, void* workspace, size_t workspace_bytes, void* cuda_stream);
int gc_value_head_bwd(const void* H, int64_t ldH, int dtype, const void* w, const float* g,
                      int64_t T, int64_t D, void* dH, int64_t lddH, float* dw, float* dbias,
                      void* workspace, size_t workspace_bytes, void* cuda_stream);

/* ---- gc_value_loss without a workspace, for callers that have no way to get device memory.
 * Every other entry point takes its scratch from a `workspace` the caller allocated.  Some callers
 * cannot do that: a hook or plug-in that runs inside another framework's training step and is
 * handed only the tensors it reads and writes; a process whose memory pool has claimed the whole
 * HBM at start-up, so that a later cudaMalloc simply fails; a step loop that must not stall,
 * because cudaMalloc / cudaFree synchronise the whole device.  For them this call computes exactly
 * what gc_value_loss computes (same kernels, bit-identical out3 and g; PPO value loss, PAPER.md:96,
 * PAPER.md:102-103, formulas above) with the scratch -- the scored / clipped counters and one fp64
 * partial sum per 1024-token tile -- in a fixed array that is part of the library image.
 *   Arguments: as gc_value_loss, minus workspace / workspace_bytes.  values, old_values, returns
 *   [T] f32, mask [T] uint8 nullable, out3 [3] f32, g [T] f32 nullable: DEVICE pointers, owned by
 *   the caller.  Work is enqueued on `cuda_stream`; no synchronisation.
 *   Limit: T <= GC_VALUE_LOSS_STATIC_MAX_T (4,194,304 tokens).  A larger T returns GC_ERR_SHAPE
 *   before anything is launched -- use gc_value_loss with a workspace instead.  Other errors as
 *   gc_value_loss (GC_ERR_NULL, GC_ERR_ARG for clip_v < 0, GC_ERR_CUDA).
 *   Cost: the array is 33,024 bytes of device memory on every GPU that loads the library, held
 *   from load until the process exits, whether or not this call is ever made.
 *   No allocation: the call makes no cudaMalloc / cudaFree / cudaMallocAsync and calls no library
 *   routine that allocates; it issues one cudaMemsetAsync of 24 bytes and two kernel launches.
 *   First call on a device: looks up the array's address on the CURRENT device
 *   (cudaGetSymbolAddress; the address is per device and is cached per device).  Make that first
 *   call with the right device current and before starting any stream capture on it.
 *   Sharing: there is ONE array per device and every call uses it.  It keeps the previous call's
 *   contents; the call clears what has to start at zero (the counters), the partials are rewritten
 *   before they are read.  Two calls that can overlap on the GPU (different streams, no event
 *   between them; or two host threads on two streams) RACE on the array and give wrong results:
 *   keep all calls on one stream per device, or order them with events. */
#define GC_VALUE_LOSS_STATIC_MAX_T 4194304
int gc_value_loss_static_scratch(const float* values, const float* old_values, const float* returns,
                                 const uint8_t* mask, int64_t T, float clip_v, float grad_loss,
                                 float* out3, float* g, void* cuda_stream);

/* ---- verdict-token scoring for a generative reward model.
 * PAPER.md:144 (sec 3.2): "Generative rewarding using standard next-token prediction, represents
 * solution correctness using the LLM's probability distribution over tokens ... the verification
 * decision is just another token".  Only the scoring is in scope (generation and regex matching,
 * PAPER.md:146, need an inference engine and trained weights): at each given position, the
 * log-probability of each of K candidate verdict tokens, in one pass of the forward contraction.
 *   logp[t,k] = z[t, targets[t,k]] - lse[t]      (0 where targets[t,k] < 0 or >= V)
 * H [T,D] holds the hidden states at the verdict positions (gather them with gc_gather_rows);
 * targets [T,K] int32 row-major, 1 <= K <= 8; logp [T,K]; entropy, lse [T] nullable.  GC_BF16 only.
 * exp(logp[t,:]) are the candidates' probabilities; a reward such as P(yes) / (P(yes) + P(no)) is
 * the caller's arithmetic.  workspace: gc_multi_workspace_bytes(T, D, V, K). */
size_t gc_multi_workspace_bytes(int64_t T, int64_t D, int64_t V, int32_t K);
int gc_token_logprobs_multi(const void* H, int64_t ldH, const void* W, int64_t ldW, int dtype,
                            const int32_t* targets, int32_t K, int64_t T, int64_t D, int64_t V,
                            float temperature, float* logp, float* entropy, float* lse,
                            void* workspace, size_t workspace_bytes, void* cuda_stream);

/* ---- distributed attention by all-gather of K and V.
 * PAPER.md:209 (sec 4.5): "we implemented distributed attention based on CCL all-gather, where we
 * first all-gather the key (K) and value (V) tensors, and then compute attention output for the
 * local query (Q) tensor chunk"; "we process only a subset of attention heads at a
 * time and overlap KV communication with attention computation."  Forward only.
 * The sequence of S = sum_r shard_rows[r] tokens is cut into `world` contiguous chunks; this rank
 * (`rank`) holds Q [S_local, Hq, head_dim] and every rank r holds K_r, V_r [shard_rows[r], Hkv,
 * head_dim] (bf16, dense).  K_shards_host / V_shards_host: HOST arrays of `world` DEVICE pointers --
 * this rank's own buffers or peer-mapped ones (CUDA IPC / peer access; NVLink carries the copies).
 * For each subset of heads_per_step key/value heads the shards are gathered by the copy engines
 * into one of two [S, heads, head_dim] buffers on a library-owned side stream while the attention
 * kernel works on the previous subset; the peers' K/V must stay unchanged until the call has
 * completed on `cuda_stream` (the caller synchronises the ranks around the call).
 *   out[q, h, :] = sum_k softmax_k(scale <Q[q,h,:], K[k,g,:]>) V[k,g,:],  g = h / (Hq / Hkv),
 * over the keys k (global positions) the query at global position q may attend:
 *   same document (cu_seqlens [n_docs + 1] int32 on the device, global positions; NULL = one
 *   document), k <= q if causal, and q - k < window if window > 0 (|q - k| < window when not
 *   causal).  O [S_local, Hq, head_dim] bf16; lse [Hq, S_local] f32 nullable (natural log).
 * head_dim = 128.  workspace: gc_attention_workspace_bytes(S_local, S, heads_per_step). */
size_t gc_attention_workspace_bytes(int64_t S_local, int64_t S_total, int32_t heads_per_step);
int gc_attention_allgather_kv(const void* Q, const void* const* K_shards_host,
                              const void* const* V_shards_host, const int64_t* shard_rows_host,
                              int32_t world, int32_t rank, int32_t Hq, int32_t Hkv, int32_t head_dim,
                              const int32_t* cu_seqlens, int32_t n_docs, int causal, int32_t window,
                              float scale, int32_t heads_per_step, void* O, float* lse,
                              void* workspace, size_t workspace_bytes, void* cuda_stream);

/* ---- the step before the path: dynamic-sampling repack + workload balancing (SURVEY.md sec
 * 8(f) NEXT-1).  PAPER.md:150 (sec 3.2): prompts whose samples are all right or all wrong are
 * filtered out; PAPER.md:201 (sec 4.4): "we simply sort data by simulated workload"; PAPER.md:205:
 * "we first bucket data according to the global batch size, then shuffle the buckets".
 *   kept samples  = samples of groups with keep[g] != 0 (keep == NULL or group_offsets == NULL: all)
 *   workload w_i  = w_lin L_i + w_quad L_i^2, L_i = cu_seqlens[i+1] - cu_seqlens[i]  (unsigned 64-bit)
 *   sorted        = kept samples in ascending w, ties by ascending index
 *   buckets       = consecutive runs of bucket_size sorted samples (the last may be short)
 *   shuffle != 0  : buckets reordered by ascending (splitmix64(seed + (b+1) 0x9E3779B97F4A7C15) >> 1, b)
 * Outputs (device): order [R] (source sample of each destination slot, -1 past n_kept), *n_kept,
 * cu_out [R+1] (cu_seqlens of the repacked batch; entries past n_kept repeat the total),
 * src_token [T] (source token of each destination token, first *n_tokens valid), *n_tokens.
 * Integer work, bit-exact.  Use src_token with gc_gather_rows / gc_gather_1d to repack H, targets,
 * log-probs.  workspace: gc_balance_workspace_bytes(R).  group_offsets[G] must equal R. */
size_t gc_balance_workspace_bytes(int32_t R);
int gc_balance_plan(const int32_t* cu_seqlens, int32_t R, const int32_t* group_offsets,
                    const uint8_t* keep, int32_t G, uint64_t w_lin, uint64_t w_quad,
                    int32_t bucket_size, uint64_t seed, int shuffle,
                    int32_t* order, int32_t* n_kept, int32_t* cu_out, int32_t* src_token,
                    int32_t* n_tokens, void* workspace, size_t workspace_bytes, void* cuda_stream);

/* Y[i,:] = X[rows[i],:] for i < *n_rows (device scalar), rows n_rows .. min(round_up(n_rows, 256),
 * y_rows) of Y are zero-filled.  X [*, D] (ldX), Y [y_rows, D] dense, of `dtype` (GC_F32 / GC_BF16).
 * HBM-bound: 2 n_rows D elem bytes. */
int gc_gather_rows(const void* X, int64_t ldX, int dtype, int64_t D, const int32_t* rows,
                   const int32_t* n_rows, int64_t y_rows, void* Y, void* cuda_stream);
/* y[i] = x[rows[i]] for i < *n_rows, 4-byte elements (int32 / float). */
int gc_gather_1d(const void* x, const int32_t* rows, const int32_t* n_rows, int64_t max_rows,
                 void* y, void* cuda_stream);

/* Measurement aid (bench.py's roofline figure): between _begin and _end the library brackets
 * every tcgen05 contraction launch with a pair of CUDA events recorded on the call's stream.
 * _end waits for the recorded events, then writes per kernel kind the summed duration in ms and
 * the number of launches into two HOST arrays of GC_KERNEL_KINDS entries, and switches the
 * facility off.  This is the one piece of process-global state in the library (mutex-guarded);
 * it never changes results.  Kinds: the four dense contractions of SURVEY.md sec 8(a). */
typedef enum {
  GC_KERNEL_FWD_STATS = 0,   /* a2+a3: H W^T with the online log-softmax epilogue */
  GC_KERNEL_RECOMPUTE_DS = 1,/* a10:  H W^T again with the dS epilogue            */
  GC_KERNEL_DH = 2,          /* a11:  dS W                                        */
  GC_KERNEL_DW = 3,          /* a12:  dS^T H                                      */
  GC_KERNEL_KINDS = 4
} gc_kernel_kind;
int gc_kernel_timing_begin(void);
int gc_kernel_timing_end(float* ms_by_kind_host, int32_t* launches_by_kind_host);

/* Plain bf16 GEMM on the library's tcgen05 main loop, for unit tests of the tile engine:
 * C[M,N] (f32, ldc) = A . B with A given as [M,K] (a_mn_major = 0, lda >= K) or [K,M]
 * (a_mn_major = 1, lda >= M), B as [N,K] (b_mn_major = 0) or [K,N] (b_mn_major = 1).
 * accumulate != 0 adds to C.  cta_group is 1 or 2.  dynamic_schedule != 0: tiles are claimed
 * by whichever CTA pair is free (the schedule of the forward / recompute / dW kernels; uses one
 * library-owned counter, so do not run two such debug calls concurrently); 0: static round-robin
 * (the schedule of the dH kernel).  dual_n != 0 (cta_group 2 only): 256 x 512 tiles whose two
 * halves share the A stages (the dH kernel's tile).  cluster4 != 0 (cta_group 2 only): clusters
 * of two CTA pairs that take adjacent M tiles and fetch every B stage once, by TMA multicast.
 * Item order (so that the production schedules of the path's kernels are reachable at any size):
 *   c_major != 0: items = (band of m_band M tiles, run of chunk_ntiles N tiles, M tile in band),
 *                 the forward / recompute order (m_band = 0: one band; a last, shorter band and a
 *                 last, shorter run are allowed);
 *   n_band  >  0: items = (band of n_band N tiles, M tile, N tile in band), the dW order (a last,
 *                 narrower band is allowed);  c_major and n_band exclude each other;
 *   c_major == 2: (N tile, M tile) -- the dH order when the dS chunk has fewer rows than D;
 *   both 0      : (M tile, N tile). */
int gc_debug_gemm_bf16(const void* A, int64_t lda, int a_mn_major,
                       const void* B, int64_t ldb, int b_mn_major,
                       float* C, int64_t ldc, int64_t M, int64_t N, int64_t K,
                       int accumulate, int cta_group, int dynamic_schedule, int dual_n,
                       int cluster4, int c_major, int m_band, int chunk_ntiles, int n_band,
                       void* cuda_stream);

#ifdef __cplusplus
}
#endif
#endif /* GCORE_H_ */
