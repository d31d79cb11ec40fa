// common.cuh -- shared declarations of the gcore CUDA library (sm_100a only).
#pragma once
#include <cuda_runtime.h>
#include <cuda_bf16.h>
#include <stdint.h>
#include <stddef.h>
#include "../../include/gcore.h"

// the CUDA error behind the calling thread's last GC_ERR_CUDA (api.cu; gc_last_cuda_error)
namespace gc {
void note_cuda_error(cudaError_t e);
// api.cu: gc_grpo_loss_bwd that records `dh_done` after the dH launch of the last non-empty chunk
int grpo_loss_bwd_dh_event(const void* H, int64_t ldH, const void* W, int64_t ldW, int dtype,
                           const int32_t* targets, const uint8_t* mask, int64_t T, int64_t D,
                           int64_t V, float temperature, const int32_t* cu_seqlens, int32_t R,
                           const float* adv, const float* old_logp, const float* ref_logp,
                           float clip_lo, float clip_hi, float beta, int agg, const float* logp,
                           const float* lse, float grad_loss, void* dH, int64_t lddH, void* dW,
                           int64_t lddW, int dW_dtype, int accumulate_dW, void* workspace,
                           size_t workspace_bytes, void* cuda_stream, cudaEvent_t dh_done,
                           int64_t dh_rows);
}

#define GC_CUDA_TRY(expr)                         \
  do {                                            \
    cudaError_t _e = (expr);                      \
    if (_e != cudaSuccess) {                      \
      ::gc::note_cuda_error(_e);                  \
      return GC_ERR_CUDA;                         \
    }                                             \
  } while (0)

#define GC_TRY(expr)                              \
  do {                                            \
    int _s = (expr);                              \
    if (_s != GC_OK) return _s;                   \
  } while (0)

namespace gc {

constexpr int kNumSMs = 148;          // B200: 2 dies x 74 SMs
constexpr float kLog2e = 1.4426950408889634f;
constexpr float kLn2 = 0.6931471805599453f;

static inline size_t align_up(size_t x, size_t a) { return (x + a - 1) / a * a; }
static inline int64_t ceil_div(int64_t a, int64_t b) { return (a + b - 1) / b; }

// Workspace carving: a bump allocator over the caller's buffer (256-byte granules).
struct Carver {
  char* base;
  size_t off = 0;
  explicit Carver(void* p) : base(static_cast<char*>(p)) {}
  template <typename T>
  T* take(size_t n) {
    T* p = reinterpret_cast<T*>(base + off);
    off += align_up(n * sizeof(T), 256);
    return p;
  }
};

// Partial (per row, per vocab chunk) online-softmax statistics, in log2-scaled units
// a = z * log2(e):  m = max a, s = sum 2^(a-m), u = sum 2^(a-m) (a-m), ay = a at the target
// (-inf if the target is not in this chunk).
struct __align__(16) RowStat { float m, s, u, ay; };

// timing.cu: RAII bracket around one contraction launch (no-op unless gc_kernel_timing_begin ran)
class KernelTimer {
 public:
  KernelTimer(int kind, cudaStream_t st);
  ~KernelTimer();
 private:
  cudaStream_t st_;
  long idx_;
};

// ---- launchers implemented in the .cu files (all enqueue on `st`, no sync) ----------------
// small_kernels.cu
int launch_advantages(const float* rewards, const int32_t* group_offsets, int32_t G, float eps,
                      int unbiased, int drop_const, float* adv, uint8_t* keep, cudaStream_t st);
size_t loss_ws_bytes(int64_t T, int32_t R);
int launch_token_loss(const float* logp, const float* old_logp, const float* ref_logp,
                      const int32_t* targets, const uint8_t* mask, int64_t T,
                      const int32_t* cu_seqlens, int32_t R, const float* adv,
                      float clip_lo, float clip_hi, float beta, int agg, float grad_loss,
                      float* out5, float* g, void* ws, cudaStream_t st);
int launch_combine(const RowStat* partials, int n_split, int64_t split_stride,
                   const int32_t* rows, const int32_t* n_rows_dev, int64_t n_rows_max,
                   float* logp, float* entropy, float* lse, cudaStream_t st);
int launch_combine_multi(const RowStat* partials, int n_split, int64_t split_stride,
                         const float* ay, int K, int64_t T, float* logp, float* entropy,
                         float* lse, cudaStream_t st);
int launch_fill_f32(float* p, float v, int64_t n, cudaStream_t st);
int launch_zero_unscored(const int32_t* targets, const uint8_t* mask, int64_t T,
                         float* logp, float* entropy, float* lse, cudaStream_t st);
size_t compact_ws_bytes(int64_t T);
int launch_compact_rows(const int32_t* targets, const uint8_t* mask, int64_t T, int32_t* rows,
                        int32_t* n_rows, void* ws, cudaStream_t st);
int launch_gather_rows(const void* H, int64_t ldH, int elem_bytes, int64_t D, int64_t T,
                       const int32_t* rows, const int32_t* n_rows, void* Hs, int64_t pad_rows,
                       cudaStream_t st);
int launch_gather_f32(const float* src, const int32_t* rows, const int32_t* n_rows,
                      int64_t T, float* dst, cudaStream_t st);
int launch_gather_i32(const int32_t* src, const int32_t* rows, const int32_t* n_rows,
                      int64_t T, int32_t* dst, cudaStream_t st);
int launch_zero_rows_unscored(const int32_t* targets, const uint8_t* mask, int64_t T, void* dH,
                              int64_t lddH, int elem_bytes, int64_t D, cudaStream_t st);
int launch_cast_f32_bf16(const float* acc, int64_t ld_acc, void* out, int64_t ld_out, int64_t V,
                         int64_t D, int accumulate, cudaStream_t st);
int launch_validate_targets(const int32_t* targets, const uint8_t* mask, int64_t T, int64_t V,
                            unsigned long long* n_bad_dev, cudaStream_t st);

// balance.cu (NEXT-1: dynamic-sampling repack + workload balancing)
size_t balance_ws_bytes(int32_t R);
int launch_balance_plan(const int32_t* cu, int32_t R, const int32_t* group_offsets,
                        const uint8_t* keep, int32_t G, uint64_t w_lin, uint64_t w_quad,
                        int32_t bucket_size, uint64_t seed, int shuffle, int32_t* order,
                        int32_t* n_kept, int32_t* cu_out, int32_t* src_token, int32_t* n_tokens,
                        void* ws, cudaStream_t st);

// critic.cu (NEXT-2: PPO critic path)
int launch_value_fwd(const void* H, int64_t ldH, bool bf16, const void* w, float bias, int64_t T,
                     int64_t D, float* values, cudaStream_t st);
int launch_gae(const float* rewards, const float* values, const uint8_t* mask, const int32_t* cu,
               int32_t R, float gamma, float lam, float* adv, float* ret, cudaStream_t st);
size_t value_loss_ws_bytes(int64_t T);
int launch_value_loss(const float* values, const float* old_values, const float* returns,
                      const uint8_t* mask, int64_t T, float clip_v, float grad_loss, float* out3,
                      float* g, void* ws, cudaStream_t st);
size_t value_bwd_ws_bytes(int64_t T, int64_t D);
int launch_value_bwd(const void* H, int64_t ldH, bool bf16, const void* w, const float* g, int64_t T,
                     int64_t D, void* dH, int64_t lddH, float* dw, float* dbias, void* ws,
                     cudaStream_t st);

// simt_head.cu
int simt_logprobs(const void* H, int64_t ldH, const void* W, int64_t ldW, bool bf16,
                  const int32_t* targets, const uint8_t* mask, int64_t T, int64_t D, int64_t V,
                  float tau, float* logp, float* entropy, float* lse, cudaStream_t st);
int simt_backward(const void* H, int64_t ldH, const void* W, int64_t ldW, bool bf16,
                  const int32_t* targets, const uint8_t* mask, int64_t T, int64_t D, int64_t V,
                  float tau, const float* lse, const float* g, void* dH, int64_t lddH,
                  float* dW, int64_t lddW, int accumulate, cudaStream_t st);

// tc_head.cu (tcgen05 engine).  `counter`: a zeroed device word per launch (dynamic item
// schedule, tc_gemm.cuh) -- for tc_dh kDhLockWords of them (the K-lockstep progress ring); the API
// zeroes kTcCounters words once per call (again when a long chunk loop runs out of them).
constexpr int kTcCounters = 1024;
constexpr int kDhLockWords = 32;                       // == tc::kLockRing
constexpr int kCountersPerChunk = 2 + kDhLockWords;    // recompute, dW, dH ring
struct TcPlan {            // forward / recompute schedule: items = (vocab chunk c, M tile)
  int n_vtiles;            // ceil(V / 256)
  int chunk_vtiles;        // vocab tiles per item
  int n_split;             // number of vocab chunks = partial slots per row
};
TcPlan tc_plan_forward(int64_t T, int64_t D, int64_t V);
size_t tc_fwd_partials_bytes(int64_t T, int64_t D, int64_t V);
int64_t tc_forward_band_rows(int64_t T, int64_t D, int64_t V);
int tc_forward_stats(const void* H, int64_t ldH, const void* W, int64_t ldW, int64_t T,
                     int64_t D, int64_t V, float tau, const int32_t* targets_c,
                     const int32_t* n_rows_dev, RowStat* partials, uint32_t* counter,
                     cudaStream_t st);
int tc_forward_stats_multi(const void* H, int64_t ldH, const void* W, int64_t ldW, int64_t T,
                           int64_t D, int64_t V, float tau, const int32_t* targets, int K,
                           float* ay, RowStat* partials, uint32_t* counter, cudaStream_t st);
// Backward chunk kernels.  rows_cap = rows of the dS chunk buffer (multiple of 256); the valid
// rows of the chunk are clamp(*n_rows_dev - row0, 0, rows_cap), or n_static if n_rows_dev == NULL.
int tc_recompute_ds(const void* H, int64_t ldH, const void* W, int64_t ldW, int64_t rows_cap,
                    int64_t n_static, int64_t D, int64_t V, float tau, const int32_t* targets_c,
                    const float* lse_c, const float* g_c, const int32_t* n_rows_dev,
                    int64_t row0, void* dS, int64_t ldS, uint32_t* counter, cudaStream_t st);
int tc_dh(const void* dS, int64_t ldS, int64_t rows_cap, int64_t n_static, const void* W,
          int64_t ldW, int64_t D, int64_t V, const int32_t* rows, const int32_t* n_rows_dev,
          int64_t row0, void* dH, int64_t lddH, uint32_t* counter, cudaStream_t st);
int tc_dw(const void* dS, int64_t ldS, int64_t rows_cap, int64_t n_static, const void* Hs,
          int64_t ldH, int64_t D, int64_t V, const int32_t* n_rows_dev, int64_t row0, float* dW,
          int64_t lddW, int accumulate, uint32_t* counter, cudaStream_t st);
int tc_dw_reduce_scatter(const void* dS, int64_t ldS, int64_t rows_cap, int64_t n_static,
                         const void* Hs, int64_t ldH, int64_t D, int64_t V,
                         const int32_t* n_rows_dev, int64_t row0, float* const* shards, int world,
                         int64_t shard_rows, int64_t ld_shard, uint32_t* counter, cudaStream_t st);
int tc_debug_gemm(const void* A, int64_t lda, int a_mn, const void* B, int64_t ldb, int b_mn,
                  float* C, int64_t ldc, int64_t M, int64_t N, int64_t K, int accumulate,
                  int cta_group, int dynamic_schedule, int dual_n, int cluster4, int c_major,
                  int m_band, int chunk_ntiles, int n_band, cudaStream_t st);
double tc_dh_waves(int64_t rows, int64_t D);

}  // namespace gc
