// simt_head.cu -- plain SIMT (CUDA-core) kernels for the LM-head scoring pass and its backward.
// Used for GC_F32 (BASELINE.json configs[0], fp32 everywhere) and as the slow on-device
// cross-check GC_BF16_SIMT.  fp32 FMA dot products, warp-shuffle reductions, online softmax
// statistics (m, s, u) per row; all reductions in fixed order.  Steps 1-3 and 9 of
// SURVEY.md sec 8(c).
#include "common.cuh"

namespace gc {

template <typename TI> __device__ __forceinline__ float ldf(const TI* p);
template <> __device__ __forceinline__ float ldf<float>(const float* p) { return *p; }
template <> __device__ __forceinline__ float ldf<__nv_bfloat16>(const __nv_bfloat16* p) {
  return __bfloat162float(*p);
}
template <typename TI> __device__ __forceinline__ TI stf(float v);
template <> __device__ __forceinline__ float stf<float>(float v) { return v; }
template <> __device__ __forceinline__ __nv_bfloat16 stf<__nv_bfloat16>(float v) {
  return __float2bfloat16_rn(v);
}

__device__ __forceinline__ float wsum(float v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
  return v;
}

constexpr int kFwdRows = 8;
constexpr int kWarps = 8;

// ---------------------------------------------------------------------------------------------
// forward: one block per kFwdRows token rows; warps stride over vocab rows.
// ---------------------------------------------------------------------------------------------
template <typename TI>
__global__ void __launch_bounds__(kWarps * 32)
k_simt_fwd(const TI* __restrict__ H, int64_t ldH, const TI* __restrict__ W, int64_t ldW,
           const int32_t* __restrict__ targets, const uint8_t* __restrict__ mask, int64_t T,
           int D, int64_t V, float inv_tau, float* __restrict__ logp,
           float* __restrict__ entropy, float* __restrict__ lse) {
  extern __shared__ float smem[];
  float* hs = smem;                                   // [kFwdRows][D]
  float* red = smem + (size_t)kFwdRows * D;           // [kWarps][kFwdRows][4]
  const int64_t row0 = (int64_t)blockIdx.x * kFwdRows;
  const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
  for (int i = threadIdx.x; i < kFwdRows * D; i += blockDim.x) {
    const int r = i / D, d = i - r * D;
    hs[i] = (row0 + r < T) ? ldf<TI>(H + (row0 + r) * ldH + d) : 0.f;
  }
  __syncthreads();
  int32_t y[kFwdRows];
  float m[kFwdRows], s[kFwdRows], u[kFwdRows], zy[kFwdRows];
#pragma unroll
  for (int r = 0; r < kFwdRows; ++r) {
    y[r] = (row0 + r < T) ? targets[row0 + r] : -1;
    m[r] = -INFINITY; s[r] = 0.f; u[r] = 0.f; zy[r] = -INFINITY;
  }
  for (int64_t v = wid; v < V; v += kWarps) {
    float acc[kFwdRows];
#pragma unroll
    for (int r = 0; r < kFwdRows; ++r) acc[r] = 0.f;
    const TI* wrow = W + v * ldW;
    for (int d = lane; d < D; d += 32) {
      const float w = ldf<TI>(wrow + d);
#pragma unroll
      for (int r = 0; r < kFwdRows; ++r) acc[r] = fmaf(hs[r * D + d], w, acc[r]);
    }
#pragma unroll
    for (int r = 0; r < kFwdRows; ++r) {
      const float z = wsum(acc[r]) * inv_tau;
      const float mn = fmaxf(m[r], z);
      const float sc = expf(m[r] - mn), e = expf(z - mn);
      s[r] = s[r] * sc + e;
      u[r] = u[r] * sc + e * z;
      m[r] = mn;
      if ((int64_t)y[r] == v) zy[r] = z;
    }
  }
  if (lane == 0) {
#pragma unroll
    for (int r = 0; r < kFwdRows; ++r) {
      float* p = red + ((size_t)wid * kFwdRows + r) * 4;
      p[0] = m[r]; p[1] = s[r]; p[2] = u[r]; p[3] = zy[r];
    }
  }
  __syncthreads();
  if (threadIdx.x < kFwdRows) {
    const int r = threadIdx.x;
    const int64_t t = row0 + r;
    if (t < T) {
      float M = -INFINITY;
      for (int w = 0; w < kWarps; ++w) M = fmaxf(M, red[((size_t)w * kFwdRows + r) * 4]);
      float S = 0.f, U = 0.f, ZY = -INFINITY;
      for (int w = 0; w < kWarps; ++w) {
        const float* p = red + ((size_t)w * kFwdRows + r) * 4;
        if (p[1] > 0.f) {
          const float sc = expf(p[0] - M);
          S += p[1] * sc;
          U += p[2] * sc;
        }
        ZY = fmaxf(ZY, p[3]);
      }
      const float l = M + logf(S);
      const bool sc_row = targets[t] >= 0 && (mask == nullptr || mask[t] != 0);
      logp[t] = sc_row ? ZY - l : 0.f;
      if (entropy) entropy[t] = sc_row ? l - U / S : 0.f;
      if (lse) lse[t] = sc_row ? l : 0.f;
    }
  }
}

// ---------------------------------------------------------------------------------------------
// backward dH: one block per token row.  dH[t,:] = (1/tau) sum_v g_t (1[v=y]-p[t,v]) W[v,:]
// ---------------------------------------------------------------------------------------------
template <typename TI>
__global__ void k_simt_dh(const TI* __restrict__ H, int64_t ldH, const TI* __restrict__ W,
                          int64_t ldW, const int32_t* __restrict__ targets,
                          const uint8_t* __restrict__ mask, int D, int64_t V, float inv_tau,
                          const float* __restrict__ lse, const float* __restrict__ g,
                          TI* __restrict__ dH, int64_t lddH) {
  extern __shared__ float smem[];
  const int nw = blockDim.x >> 5;
  float* hs = smem;                         // [D]
  float* acc = smem + D;                    // [nw][D]
  const int64_t t = blockIdx.x;
  const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
  const bool scored = targets[t] >= 0 && (mask == nullptr || mask[t] != 0);
  const float gt = scored ? g[t] : 0.f;
  if (gt == 0.f) {                          // uniform branch: zero row
    for (int d = threadIdx.x; d < D; d += blockDim.x) dH[t * lddH + d] = stf<TI>(0.f);
    return;
  }
  for (int d = threadIdx.x; d < D; d += blockDim.x) hs[d] = ldf<TI>(H + t * ldH + d);
  for (int d = lane; d < D; d += 32) acc[(size_t)wid * D + d] = 0.f;
  __syncthreads();
  const float l = lse[t];
  const int64_t y = targets[t];
  for (int64_t v = wid; v < V; v += nw) {
    const TI* wrow = W + v * ldW;
    float a = 0.f;
    for (int d = lane; d < D; d += 32) a = fmaf(hs[d], ldf<TI>(wrow + d), a);
    const float z = wsum(a) * inv_tau;
    const float dz = gt * ((v == y ? 1.f : 0.f) - expf(z - l));
    for (int d = lane; d < D; d += 32)
      acc[(size_t)wid * D + d] = fmaf(dz, ldf<TI>(wrow + d), acc[(size_t)wid * D + d]);
  }
  __syncthreads();
  for (int d = threadIdx.x; d < D; d += blockDim.x) {
    float sum = 0.f;
    for (int w = 0; w < nw; ++w) sum += acc[(size_t)w * D + d];
    dH[t * lddH + d] = stf<TI>(sum * inv_tau);
  }
}

// ---------------------------------------------------------------------------------------------
// backward dW: one block per vocab row.  dW[v,:] (+)= (1/tau) sum_t g_t (1[v=y_t]-p[t,v]) H[t,:]
// ---------------------------------------------------------------------------------------------
template <typename TI>
__global__ void k_simt_dw(const TI* __restrict__ H, int64_t ldH, const TI* __restrict__ W,
                          int64_t ldW, const int32_t* __restrict__ targets,
                          const uint8_t* __restrict__ mask, int64_t T, int D, float inv_tau,
                          const float* __restrict__ lse, const float* __restrict__ g,
                          float* __restrict__ dW, int64_t lddW, int accumulate) {
  extern __shared__ float smem[];
  const int nw = blockDim.x >> 5;
  float* ws = smem;                         // [D]
  float* acc = smem + D;                    // [nw][D]
  const int64_t v = blockIdx.x;
  const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
  for (int d = threadIdx.x; d < D; d += blockDim.x) ws[d] = ldf<TI>(W + v * ldW + d);
  for (int d = lane; d < D; d += 32) acc[(size_t)wid * D + d] = 0.f;
  __syncthreads();
  for (int64_t t = wid; t < T; t += nw) {
    const bool scored = targets[t] >= 0 && (mask == nullptr || mask[t] != 0);
    const float gt = scored ? g[t] : 0.f;
    if (gt == 0.f) continue;                // warp-uniform
    const TI* hrow = H + t * ldH;
    float a = 0.f;
    for (int d = lane; d < D; d += 32) a = fmaf(ldf<TI>(hrow + d), ws[d], a);
    const float z = wsum(a) * inv_tau;
    const float dz = gt * (((int64_t)targets[t] == v ? 1.f : 0.f) - expf(z - lse[t]));
    for (int d = lane; d < D; d += 32)
      acc[(size_t)wid * D + d] = fmaf(dz, ldf<TI>(hrow + d), acc[(size_t)wid * D + d]);
  }
  __syncthreads();
  for (int d = threadIdx.x; d < D; d += blockDim.x) {
    float sum = 0.f;
    for (int w = 0; w < nw; ++w) sum += acc[(size_t)w * D + d];
    const float prev = accumulate ? dW[v * lddW + d] : 0.f;
    dW[v * lddW + d] = prev + sum * inv_tau;
  }
}

static int bwd_warps(int64_t D) {
  for (int nw = 8; nw >= 1; nw >>= 1)
    if ((size_t)(nw + 1) * D * sizeof(float) <= 200 * 1024) return nw;
  return 0;
}

template <typename TI>
static int simt_logprobs_t(const void* H, int64_t ldH, const void* W, int64_t ldW,
                           const int32_t* targets, const uint8_t* mask, int64_t T, int64_t D,
                           int64_t V, float tau, float* logp, float* entropy, float* lse,
                           cudaStream_t st) {
  const size_t smem = ((size_t)kFwdRows * D + (size_t)kWarps * kFwdRows * 4) * sizeof(float);
  if (smem > 200 * 1024) return GC_ERR_SHAPE;
  GC_CUDA_TRY(cudaFuncSetAttribute(k_simt_fwd<TI>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                   (int)smem));
  const int64_t blocks = ceil_div(T, kFwdRows);
  k_simt_fwd<TI><<<(unsigned)blocks, kWarps * 32, smem, st>>>(
      static_cast<const TI*>(H), ldH, static_cast<const TI*>(W), ldW, targets, mask, T, (int)D, V,
      1.0f / tau, logp, entropy, lse);
  GC_CUDA_TRY(cudaGetLastError());
  return GC_OK;
}

int simt_logprobs(const void* H, int64_t ldH, const void* W, int64_t ldW, bool bf16,
                  const int32_t* targets, const uint8_t* mask, int64_t T, int64_t D, int64_t V,
                  float tau, float* logp, float* entropy, float* lse, cudaStream_t st) {
  if (T == 0) return GC_OK;
  return bf16 ? simt_logprobs_t<__nv_bfloat16>(H, ldH, W, ldW, targets, mask, T, D, V, tau, logp,
                                               entropy, lse, st)
              : simt_logprobs_t<float>(H, ldH, W, ldW, targets, mask, T, D, V, tau, logp, entropy,
                                       lse, st);
}

template <typename TI>
static int simt_backward_t(const void* H, int64_t ldH, const void* W, int64_t ldW,
                           const int32_t* targets, const uint8_t* mask, int64_t T, int64_t D,
                           int64_t V, float tau, const float* lse, const float* g, void* dH,
                           int64_t lddH, float* dW, int64_t lddW, int accumulate,
                           cudaStream_t st) {
  const int nw = bwd_warps(D);
  if (nw == 0) return GC_ERR_SHAPE;
  const size_t smem = (size_t)(nw + 1) * D * sizeof(float);
  GC_CUDA_TRY(cudaFuncSetAttribute(k_simt_dh<TI>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                   (int)smem));
  GC_CUDA_TRY(cudaFuncSetAttribute(k_simt_dw<TI>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                   (int)smem));
  if (T > 0) {
    k_simt_dh<TI><<<(unsigned)T, nw * 32, smem, st>>>(
        static_cast<const TI*>(H), ldH, static_cast<const TI*>(W), ldW, targets, mask, (int)D, V,
        1.0f / tau, lse, g, static_cast<TI*>(dH), lddH);
    GC_CUDA_TRY(cudaGetLastError());
  }
  k_simt_dw<TI><<<(unsigned)V, nw * 32, smem, st>>>(
      static_cast<const TI*>(H), ldH, static_cast<const TI*>(W), ldW, targets, mask, T, (int)D,
      1.0f / tau, lse, g, dW, lddW, accumulate);
  GC_CUDA_TRY(cudaGetLastError());
  return GC_OK;
}

int simt_backward(const void* H, int64_t ldH, const void* W, int64_t ldW, bool bf16,
                  const int32_t* targets, const uint8_t* mask, int64_t T, int64_t D, int64_t V,
                  float tau, const float* lse, const float* g, void* dH, int64_t lddH,
                  float* dW, int64_t lddW, int accumulate, cudaStream_t st) {
  return bf16 ? simt_backward_t<__nv_bfloat16>(H, ldH, W, ldW, targets, mask, T, D, V, tau, lse, g,
                                               dH, lddH, dW, lddW, accumulate, st)
              : simt_backward_t<float>(H, ldH, W, ldW, targets, mask, T, D, V, tau, lse, g, dH,
                                       lddH, dW, lddW, accumulate, st);
}

}  // namespace gc
