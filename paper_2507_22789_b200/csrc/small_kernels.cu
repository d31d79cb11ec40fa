// small_kernels.cu -- the HBM/latency-bound steps of the path (SURVEY.md sec 8(a) rows a1, a4,
// a6, a7): row selection/compaction, partial-stat combine, group filter + GRPO advantages.
// (a8 + a9, the per-token loss and its gradient w.r.t. logp, live in loss.cu.)
// All floating-point reductions are fixed-order (no float atomics): reruns are bit-identical.
#include "common.cuh"

namespace gc {

__device__ __forceinline__ bool is_scored(const int32_t* targets, const uint8_t* mask, int64_t t) {
  return targets[t] >= 0 && (mask == nullptr || mask[t] != 0);
}

template <typename T>
__device__ __forceinline__ T warp_sum(T v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
  return v;
}

// =============================================================================================
// a6 + a7: group filter and advantages.  One warp per group; fp64 accumulation (R is tiny).
//   keep[g] = 0 iff all rewards equal;  A_i = (r_i - mu_g) / (sigma_g + eps)
// =============================================================================================
__global__ void k_advantages(const float* __restrict__ rewards,
                             const int32_t* __restrict__ group_offsets, int32_t G, float eps,
                             int unbiased, int drop_const, float* __restrict__ adv,
                             uint8_t* __restrict__ keep) {
  const int g = (blockIdx.x * blockDim.x + threadIdx.x) >> 5;
  const int lane = threadIdx.x & 31;
  if (g >= G) return;
  const int a = group_offsets[g], b = group_offsets[g + 1];
  const int n = b - a;
  if (n <= 0) {
    if (keep && lane == 0) keep[g] = drop_const ? 0 : 1;
    return;
  }
  const float r0 = rewards[a];
  double sum = 0.0;
  int all_eq = 1;
  for (int i = a + lane; i < b; i += 32) {
    const float r = rewards[i];
    sum += (double)r;
    all_eq &= (r == r0);
  }
  sum = warp_sum(sum);
  all_eq = __all_sync(0xffffffffu, all_eq);
  const double mu = sum / (double)n;
  double ss = 0.0;
  for (int i = a + lane; i < b; i += 32) {
    const double d = (double)rewards[i] - mu;
    ss += d * d;
  }
  ss = warp_sum(ss);
  double sigma;
  if (unbiased) sigma = n > 1 ? sqrt(ss / (double)(n - 1)) : 0.0;
  else sigma = sqrt(ss / (double)n);
  const bool dropped = drop_const && all_eq;
  const double inv = 1.0 / (sigma + (double)eps);
  for (int i = a + lane; i < b; i += 32)
    adv[i] = dropped ? 0.0f : (float)(((double)rewards[i] - mu) * inv);
  if (keep && lane == 0) keep[g] = dropped ? 0 : 1;
}

int launch_advantages(const float* rewards, const int32_t* group_offsets, int32_t G, float eps,
                      int unbiased, int drop_const, float* adv, uint8_t* keep, cudaStream_t st) {
  if (G == 0) return GC_OK;
  const int threads = 128;
  const int64_t blocks = ceil_div((int64_t)G * 32, threads);
  k_advantages<<<(unsigned)blocks, threads, 0, st>>>(rewards, group_offsets, G, eps, unbiased,
                                                     drop_const, adv, keep);
  GC_CUDA_TRY(cudaGetLastError());
  return GC_OK;
}

// =============================================================================================
// a4: combine split-V partials (fixed order) and finish:
//   lse = ln2 (M + log2 S);  logp = ln2 a_y - lse;  entropy = lse - ln2 U / S
// partials[c * split_stride + i] for compact row i; output row = rows ? rows[i] : i.
// =============================================================================================
__global__ void k_combine(const RowStat* __restrict__ partials, int n_split, int64_t split_stride,
                          const int32_t* __restrict__ rows, const int32_t* __restrict__ n_rows_dev,
                          int64_t n_rows_max, float* __restrict__ logp,
                          float* __restrict__ entropy, float* __restrict__ lse) {
  const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  const int64_t n_rows = n_rows_dev ? (int64_t)*n_rows_dev : n_rows_max;
  if (i >= n_rows) return;
  float M = -INFINITY;
  for (int c = 0; c < n_split; ++c) M = fmaxf(M, partials[(int64_t)c * split_stride + i].m);
  float S = 0.f, U = 0.f, ay = -INFINITY;
  for (int c = 0; c < n_split; ++c) {
    const RowStat p = partials[(int64_t)c * split_stride + i];
    const float sc = exp2f(p.m - M);
    S += p.s * sc;
    U += (p.u + p.m * p.s) * sc;         // sum 2^(a-M) a
    ay = fmaxf(ay, p.ay);
  }
  const float l = kLn2 * (M + log2f(S));
  const int64_t o = rows ? (int64_t)rows[i] : i;
  const bool ok = ay > -INFINITY;        // dense mode: target < 0 -> never found -> outputs 0
  logp[o] = ok ? kLn2 * ay - l : 0.f;
  if (entropy) entropy[o] = ok ? l - kLn2 * (U / S) : 0.f;
  if (lse) lse[o] = ok ? l : 0.f;
}

int launch_combine(const RowStat* partials, int n_split, int64_t split_stride,
                   const int32_t* rows, const int32_t* n_rows_dev, int64_t n_rows_max,
                   float* logp, float* entropy, float* lse, cudaStream_t st) {
  if (n_rows_max <= 0) return GC_OK;
  const int threads = 128;
  k_combine<<<(unsigned)ceil_div(n_rows_max, threads), threads, 0, st>>>(
      partials, n_split, split_stride, rows, n_rows_dev, n_rows_max, logp, entropy, lse);
  GC_CUDA_TRY(cudaGetLastError());
  return GC_OK;
}

__global__ void k_fill_f32(float* __restrict__ p, float v, int64_t n) {
  for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n;
       i += (int64_t)gridDim.x * blockDim.x)
    p[i] = v;
}
int launch_fill_f32(float* p, float v, int64_t n, cudaStream_t st) {
  if (n <= 0) return GC_OK;
  int64_t blocks = ceil_div(n, 256);
  if (blocks > kNumSMs * 8) blocks = kNumSMs * 8;
  k_fill_f32<<<(unsigned)blocks, 256, 0, st>>>(p, v, n);
  GC_CUDA_TRY(cudaGetLastError());
  return GC_OK;
}

// K targets per row (verdict-token scoring): logp[t,k] = ln2 ay[t,k] - lse[t], 0 where the target
// was absent (id < 0 or >= V: ay still holds its -inf fill).
__global__ void k_combine_multi(const RowStat* __restrict__ partials, int n_split,
                                int64_t split_stride, const float* __restrict__ ay, int K, int64_t T,
                                float* __restrict__ logp, float* __restrict__ entropy,
                                float* __restrict__ lse) {
  const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= T) return;
  float M = -INFINITY;
  for (int c = 0; c < n_split; ++c) M = fmaxf(M, partials[(int64_t)c * split_stride + i].m);
  float S = 0.f, U = 0.f;
  for (int c = 0; c < n_split; ++c) {
    const RowStat p = partials[(int64_t)c * split_stride + i];
    const float sc = exp2f(p.m - M);
    S += p.s * sc;
    U += (p.u + p.m * p.s) * sc;
  }
  const float l = kLn2 * (M + log2f(S));
  for (int k = 0; k < K; ++k) {
    const float a = ay[i * K + k];
    logp[i * K + k] = a > -INFINITY ? kLn2 * a - l : 0.f;
  }
  if (entropy) entropy[i] = l - kLn2 * (U / S);
  if (lse) lse[i] = l;
}

int launch_combine_multi(const RowStat* partials, int n_split, int64_t split_stride,
                         const float* ay, int K, int64_t T, float* logp, float* entropy,
                         float* lse, cudaStream_t st) {
  if (T <= 0) return GC_OK;
  k_combine_multi<<<(unsigned)ceil_div(T, 128), 128, 0, st>>>(partials, n_split, split_stride, ay, K,
                                                              T, logp, entropy, lse);
  GC_CUDA_TRY(cudaGetLastError());
  return GC_OK;
}

// =============================================================================================
// a1: row selection.  rows[] = ascending indices of scored tokens (bit-exact integer work):
// per-block counts -> single-block exclusive scan -> per-block ordered scatter.
// =============================================================================================
constexpr int kCompactThreads = 256;
constexpr int kCompactTile = kCompactThreads * 8;

__global__ void k_compact_count(const int32_t* __restrict__ targets,
                                const uint8_t* __restrict__ mask, int64_t T,
                                int32_t* __restrict__ block_counts) {
  const int64_t base = (int64_t)blockIdx.x * kCompactTile;
  int c = 0;
  for (int k = 0; k < 8; ++k) {
    const int64_t t = base + (int64_t)k * kCompactThreads + threadIdx.x;
    c += (t < T && is_scored(targets, mask, t)) ? 1 : 0;
  }
  c = warp_sum(c);
  __shared__ int sm[kCompactThreads / 32];
  if ((threadIdx.x & 31) == 0) sm[threadIdx.x >> 5] = c;
  __syncthreads();
  if (threadIdx.x == 0) {
    int tot = 0;
    for (int w = 0; w < kCompactThreads / 32; ++w) tot += sm[w];
    block_counts[blockIdx.x] = tot;
  }
}

// exclusive scan of block_counts in place; total -> *n_rows.  One block.
__global__ void k_compact_scan(int32_t* __restrict__ block_counts, int64_t nblocks,
                               int32_t* __restrict__ n_rows) {
  __shared__ int sm[1024];
  __shared__ int carry;
  if (threadIdx.x == 0) carry = 0;
  __syncthreads();
  for (int64_t base = 0; base < nblocks; base += 1024) {
    const int64_t i = base + threadIdx.x;
    const int v = i < nblocks ? block_counts[i] : 0;
    sm[threadIdx.x] = v;
    __syncthreads();
    for (int o = 1; o < 1024; o <<= 1) {            // Hillis-Steele inclusive scan
      const int add = threadIdx.x >= o ? sm[threadIdx.x - o] : 0;
      __syncthreads();
      sm[threadIdx.x] += add;
      __syncthreads();
    }
    if (i < nblocks) block_counts[i] = carry + sm[threadIdx.x] - v;
    __syncthreads();
    if (threadIdx.x == 0) carry += sm[1023];
    __syncthreads();
  }
  if (threadIdx.x == 0) *n_rows = carry;
}

__global__ void k_compact_scatter(const int32_t* __restrict__ targets,
                                  const uint8_t* __restrict__ mask, int64_t T,
                                  const int32_t* __restrict__ block_offsets,
                                  int32_t* __restrict__ rows) {
  const int64_t base = (int64_t)blockIdx.x * kCompactTile;
  __shared__ int warp_off[kCompactThreads / 32];
  __shared__ int running;
  if (threadIdx.x == 0) running = block_offsets[blockIdx.x];
  __syncthreads();
  const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
  for (int k = 0; k < 8; ++k) {
    const int64_t t = base + (int64_t)k * kCompactThreads + threadIdx.x;
    const bool f = t < T && is_scored(targets, mask, t);
    const unsigned int bal = __ballot_sync(0xffffffffu, f);
    if (lane == 0) warp_off[wid] = __popc(bal);
    __syncthreads();
    int off = running;
    for (int w = 0; w < wid; ++w) off += warp_off[w];
    if (f) rows[off + __popc(bal & ((1u << lane) - 1u))] = (int32_t)t;
    __syncthreads();
    if (threadIdx.x == 0) {
      int tot = 0;
      for (int w = 0; w < kCompactThreads / 32; ++w) tot += warp_off[w];
      running += tot;
    }
    __syncthreads();
  }
}

size_t compact_ws_bytes(int64_t T) {
  return align_up((size_t)ceil_div(T > 0 ? T : 1, kCompactTile) * sizeof(int32_t), 256);
}

int launch_compact_rows(const int32_t* targets, const uint8_t* mask, int64_t T, int32_t* rows,
                        int32_t* n_rows, void* ws, cudaStream_t st) {
  const int64_t nblocks = ceil_div(T > 0 ? T : 1, kCompactTile);
  int32_t* block_counts = static_cast<int32_t*>(ws);
  k_compact_count<<<(unsigned)nblocks, kCompactThreads, 0, st>>>(targets, mask, T, block_counts);
  k_compact_scan<<<1, 1024, 0, st>>>(block_counts, nblocks, n_rows);
  k_compact_scatter<<<(unsigned)nblocks, kCompactThreads, 0, st>>>(targets, mask, T, block_counts,
                                                                   rows);
  GC_CUDA_TRY(cudaGetLastError());
  return GC_OK;
}

// Gather H rows: Hs[i,:] = H[rows[i],:] for i < n_rows; zero rows for n_rows <= i < pad_end,
// pad_end = min(round_up(n_rows, 256), pad_rows).  One warp per row, 16-byte vectors,
// 4 loads in flight per lane.  HBM-bound: 2 * n_rows * D * elem_bytes.
__global__ void __launch_bounds__(256)
k_gather_rows(const uint8_t* __restrict__ H, int64_t ld_bytes, int64_t row_bytes, int64_t T,
              const int32_t* __restrict__ rows, const int32_t* __restrict__ n_rows_dev,
              uint8_t* __restrict__ Hs, int64_t pad_rows) {
  const int64_t n_rows = *n_rows_dev;
  int64_t pad_end = (n_rows + 255) / 256 * 256;
  if (pad_end > pad_rows) pad_end = pad_rows;
  const int lane = threadIdx.x & 31;
  const int64_t warps = ((int64_t)gridDim.x * blockDim.x) >> 5;
  const int64_t nvec = row_bytes >> 4;
  for (int64_t i = ((int64_t)blockIdx.x * blockDim.x + threadIdx.x) >> 5; i < pad_end; i += warps) {
    int4* dst = reinterpret_cast<int4*>(Hs + i * row_bytes);
    if (i < n_rows) {
      const int4* src = reinterpret_cast<const int4*>(H + (int64_t)rows[i] * ld_bytes);
      int64_t v = lane;
      for (; v + 96 < nvec; v += 128) {
        const int4 a = __ldg(src + v), b = __ldg(src + v + 32), c = __ldg(src + v + 64),
                   d = __ldg(src + v + 96);
        dst[v] = a; dst[v + 32] = b; dst[v + 64] = c; dst[v + 96] = d;
      }
      for (; v < nvec; v += 32) dst[v] = __ldg(src + v);
    } else {
      for (int64_t v = lane; v < nvec; v += 32) dst[v] = make_int4(0, 0, 0, 0);
    }
  }
}

int launch_gather_rows(const void* H, int64_t ldH, int elem_bytes, int64_t D, int64_t T,
                       const int32_t* rows, const int32_t* n_rows, void* Hs, int64_t pad_rows,
                       cudaStream_t st) {
  if ((D * elem_bytes) % 16 != 0 || (ldH * elem_bytes) % 16 != 0) return GC_ERR_ALIGN;
  int64_t blocks = ceil_div(T > 0 ? T : 1, 8);
  if (blocks > kNumSMs * 8) blocks = kNumSMs * 8;
  k_gather_rows<<<(unsigned)blocks, 256, 0, st>>>(
      static_cast<const uint8_t*>(H), ldH * elem_bytes, D * elem_bytes, T, rows, n_rows,
      static_cast<uint8_t*>(Hs), pad_rows);
  GC_CUDA_TRY(cudaGetLastError());
  return GC_OK;
}

template <typename T>
__global__ void k_gather_1d(const T* __restrict__ src, const int32_t* __restrict__ rows,
                            const int32_t* __restrict__ n_rows_dev, int64_t max_rows,
                            T* __restrict__ dst) {
  int64_t n = *n_rows_dev;
  n = n < max_rows ? n : max_rows;          // never past the caller's allocation
  for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n;
       i += (int64_t)gridDim.x * blockDim.x)
    dst[i] = src[rows[i]];
}

int launch_gather_f32(const float* src, const int32_t* rows, const int32_t* n_rows, int64_t T,
                      float* dst, cudaStream_t st) {
  int64_t blocks = ceil_div(T > 0 ? T : 1, 256);
  if (blocks > kNumSMs * 8) blocks = kNumSMs * 8;
  k_gather_1d<float><<<(unsigned)blocks, 256, 0, st>>>(src, rows, n_rows, T, dst);
  GC_CUDA_TRY(cudaGetLastError());
  return GC_OK;
}

int launch_gather_i32(const int32_t* src, const int32_t* rows, const int32_t* n_rows, int64_t T,
                      int32_t* dst, cudaStream_t st) {
  int64_t blocks = ceil_div(T > 0 ? T : 1, 256);
  if (blocks > kNumSMs * 8) blocks = kNumSMs * 8;
  k_gather_1d<int32_t><<<(unsigned)blocks, 256, 0, st>>>(src, rows, n_rows, T, dst);
  GC_CUDA_TRY(cudaGetLastError());
  return GC_OK;
}

// logp / entropy / lse at unscored rows = 0 (compaction mode writes only scored rows).
__global__ void k_zero_unscored(const int32_t* __restrict__ targets,
                                const uint8_t* __restrict__ mask, int64_t T,
                                float* __restrict__ logp, float* __restrict__ entropy,
                                float* __restrict__ lse) {
  for (int64_t t = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; t < T;
       t += (int64_t)gridDim.x * blockDim.x) {
    if (!is_scored(targets, mask, t)) {
      logp[t] = 0.f;
      if (entropy) entropy[t] = 0.f;
      if (lse) lse[t] = 0.f;
    }
  }
}

int launch_zero_unscored(const int32_t* targets, const uint8_t* mask, int64_t T, float* logp,
                         float* entropy, float* lse, cudaStream_t st) {
  int64_t blocks = ceil_div(T > 0 ? T : 1, 256);
  if (blocks > kNumSMs * 8) blocks = kNumSMs * 8;
  k_zero_unscored<<<(unsigned)blocks, 256, 0, st>>>(targets, mask, T, logp, entropy, lse);
  GC_CUDA_TRY(cudaGetLastError());
  return GC_OK;
}

// dH rows of unscored tokens = 0.  One warp per row.
__global__ void k_zero_rows_unscored(const int32_t* __restrict__ targets,
                                     const uint8_t* __restrict__ mask, int64_t T,
                                     uint8_t* __restrict__ dH, int64_t ld_bytes, int64_t row_bytes) {
  const int lane = threadIdx.x & 31;
  const int64_t warps = ((int64_t)gridDim.x * blockDim.x) >> 5;
  for (int64_t t = ((int64_t)blockIdx.x * blockDim.x + threadIdx.x) >> 5; t < T; t += warps) {
    if (is_scored(targets, mask, t)) continue;
    int4* dst = reinterpret_cast<int4*>(dH + t * ld_bytes);
    for (int64_t v = lane; v < (row_bytes >> 4); v += 32) dst[v] = make_int4(0, 0, 0, 0);
  }
}

int launch_zero_rows_unscored(const int32_t* targets, const uint8_t* mask, int64_t T, void* dH,
                              int64_t lddH, int elem_bytes, int64_t D, cudaStream_t st) {
  if ((D * elem_bytes) % 16 != 0 || (lddH * elem_bytes) % 16 != 0) return GC_ERR_ALIGN;
  int64_t blocks = ceil_div(T > 0 ? T : 1, 8);
  if (blocks > kNumSMs * 8) blocks = kNumSMs * 8;
  k_zero_rows_unscored<<<(unsigned)blocks, 256, 0, st>>>(
      targets, mask, T, static_cast<uint8_t*>(dH), lddH * elem_bytes, D * elem_bytes);
  GC_CUDA_TRY(cudaGetLastError());
  return GC_OK;
}

// dW fp32 -> bf16 ("dW fp32->bf16 cast -- HBM bandwidth"): out[v, :] =
// bf16(acc[v, :] (+ out[v, :])), rounded once.  8 elements per thread when rows are 16-byte
// aligned (D % 8 == 0), else element-wise.
__global__ void __launch_bounds__(256)
k_cast_f32_bf16(const float* __restrict__ acc, int64_t ld_acc, __nv_bfloat16* __restrict__ out,
                int64_t ld_out, int64_t V, int64_t D, int accumulate, int vec) {
  if (vec) {
    const int64_t per_row = D >> 3, n = V * per_row;
    for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n;
         i += (int64_t)gridDim.x * blockDim.x) {
      const int64_t v = i / per_row, d = (i - v * per_row) << 3;
      const float4 a = __ldcs(reinterpret_cast<const float4*>(acc + v * ld_acc + d));
      const float4 b = __ldcs(reinterpret_cast<const float4*>(acc + v * ld_acc + d + 4));
      float x[8] = {a.x, a.y, a.z, a.w, b.x, b.y, b.z, b.w};
      uint4* dst = reinterpret_cast<uint4*>(out + v * ld_out + d);
      if (accumulate) {
        const uint4 o = *dst;
        const __nv_bfloat162* ob = reinterpret_cast<const __nv_bfloat162*>(&o);
#pragma unroll
        for (int j = 0; j < 4; ++j) {
          const float2 f = __bfloat1622float2(ob[j]);
          x[2 * j] += f.x;
          x[2 * j + 1] += f.y;
        }
      }
      uint4 r;
      __nv_bfloat162* rb = reinterpret_cast<__nv_bfloat162*>(&r);
#pragma unroll
      for (int j = 0; j < 4; ++j) rb[j] = __floats2bfloat162_rn(x[2 * j], x[2 * j + 1]);
      *dst = r;
    }
  } else {
    const int64_t n = V * D;
    for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n;
         i += (int64_t)gridDim.x * blockDim.x) {
      const int64_t v = i / D, d = i - v * D;
      float x = acc[v * ld_acc + d];
      if (accumulate) x += __bfloat162float(out[v * ld_out + d]);
      out[v * ld_out + d] = __float2bfloat16_rn(x);
    }
  }
}

int launch_cast_f32_bf16(const float* acc, int64_t ld_acc, void* out, int64_t ld_out, int64_t V,
                         int64_t D, int accumulate, cudaStream_t st) {
  if (V <= 0 || D <= 0) return GC_OK;
  const int vec = (D % 8 == 0 && ld_acc % 4 == 0 && ld_out % 8 == 0 &&
                   (reinterpret_cast<uintptr_t>(acc) & 15) == 0 &&
                   (reinterpret_cast<uintptr_t>(out) & 15) == 0) ? 1 : 0;
  int64_t blocks = ceil_div(V * D / (vec ? 8 : 1), 256);
  if (blocks > kNumSMs * 16) blocks = kNumSMs * 16;
  if (blocks < 1) blocks = 1;
  k_cast_f32_bf16<<<(unsigned)blocks, 256, 0, st>>>(acc, ld_acc, static_cast<__nv_bfloat16*>(out),
                                                    ld_out, V, D, accumulate, vec);
  GC_CUDA_TRY(cudaGetLastError());
  return GC_OK;
}

__global__ void k_validate_targets(const int32_t* __restrict__ targets,
                                   const uint8_t* __restrict__ mask, int64_t T, int64_t V,
                                   unsigned long long* __restrict__ n_bad) {
  unsigned int c = 0;
  for (int64_t t = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; t < T;
       t += (int64_t)gridDim.x * blockDim.x)
    c += (is_scored(targets, mask, t) && (int64_t)targets[t] >= V) ? 1u : 0u;
  c = warp_sum(c);
  if ((threadIdx.x & 31) == 0 && c) atomicAdd(n_bad, (unsigned long long)c);
}

int launch_validate_targets(const int32_t* targets, const uint8_t* mask, int64_t T, int64_t V,
                            unsigned long long* n_bad_dev, cudaStream_t st) {
  int64_t blocks = ceil_div(T > 0 ? T : 1, 256);
  if (blocks > kNumSMs * 8) blocks = kNumSMs * 8;
  k_validate_targets<<<(unsigned)blocks, 256, 0, st>>>(targets, mask, T, V, n_bad_dev);
  GC_CUDA_TRY(cudaGetLastError());
  return GC_OK;
}

}  // namespace gc
