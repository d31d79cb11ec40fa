// critic.cu -- the PPO variant of stages 3-4: value head, generalised
// advantage estimation, clipped value loss and the value head's backward.  PAPER.md:96 (sec 2.2)
// "the critic computes values"; PAPER.md:102-103 stage 3 computes them, stage 4 trains the critic.
// The paper prints no formula; the arithmetic is PPO [18] as read in DESIGN.md
// sec 11 and written out in oracle/critic_oracle.py.  All kernels here are HBM-bound (the value
// head reads H once, its backward reads H once and writes dH once) or latency-bound (GAE, loss).
#include "common.cuh"
#include <atomic>

namespace gc {

namespace {

template <typename T>
__device__ __forceinline__ T wsum(T v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
  return v;
}

__device__ __forceinline__ void bf16x8_to_f32(const int4& v, float (&f)[8]) {
  const __nv_bfloat162* p = reinterpret_cast<const __nv_bfloat162*>(&v);
#pragma unroll
  for (int i = 0; i < 4; ++i) {
    const float2 t = __bfloat1622float2(p[i]);
    f[2 * i] = t.x;
    f[2 * i + 1] = t.y;
  }
}

// ---- step 1: v_t = H[t,:] . w + b.  One warp per row, 16-byte loads, fp32 accumulation. -------
template <bool kBf16>
__global__ void __launch_bounds__(256)
k_value_fwd(const void* __restrict__ H, int64_t ld, const void* __restrict__ w, float bias, int64_t T,
            int64_t D, float* __restrict__ values) {
  const int lane = threadIdx.x & 31;
  const int64_t warps = ((int64_t)gridDim.x * blockDim.x) >> 5;
  for (int64_t t = ((int64_t)blockIdx.x * blockDim.x + threadIdx.x) >> 5; t < T; t += warps) {
    float acc = 0.f;
    if (kBf16) {
      const int4* row = reinterpret_cast<const int4*>(static_cast<const __nv_bfloat16*>(H) + t * ld);
      const int4* wv = reinterpret_cast<const int4*>(w);
      const int64_t nv = D / 8;
      int64_t i = lane;
      for (; i + 96 < nv; i += 128) {                 // 4 row loads in flight per lane
        int4 h4[4];
#pragma unroll
        for (int u = 0; u < 4; ++u) h4[u] = __ldcs(row + i + 32 * u);   // H streams through once
#pragma unroll
        for (int u = 0; u < 4; ++u) {
          float a[8], b[8];
          bf16x8_to_f32(h4[u], a);
          bf16x8_to_f32(__ldg(wv + i + 32 * u), b);
#pragma unroll
          for (int j = 0; j < 8; ++j) acc = fmaf(a[j], b[j], acc);
        }
      }
      for (; i < nv; i += 32) {
        float a[8], b[8];
        bf16x8_to_f32(__ldcs(row + i), a);
        bf16x8_to_f32(__ldg(wv + i), b);
#pragma unroll
        for (int j = 0; j < 8; ++j) acc = fmaf(a[j], b[j], acc);
      }
    } else {
      const float4* row = reinterpret_cast<const float4*>(static_cast<const float*>(H) + t * ld);
      const float4* wv = reinterpret_cast<const float4*>(w);
      for (int64_t i = lane; i < D / 4; i += 32) {
        const float4 a = __ldcs(row + i), b = __ldg(wv + i);
        acc = fmaf(a.x, b.x, fmaf(a.y, b.y, fmaf(a.z, b.z, fmaf(a.w, b.w, acc))));
      }
    }
    acc = wsum(acc);
    if (lane == 0) values[t] = acc + bias;
  }
}

// ---- step 2: GAE.  One warp per response, chunks of 32 tokens from the end backwards.  A token
// is an affine map of what follows it: scored  x -> delta_t + c x (c = gamma lambda), masked  x -> x;
// a reverse warp scan composes the maps.  delta needs the value at the NEXT SCORED token, which is
// a second reverse scan ("nearest scored value to the right"). ---------------------------------
__global__ void __launch_bounds__(256)
k_gae(const float* __restrict__ rewards, const float* __restrict__ values,
      const uint8_t* __restrict__ mask, const int32_t* __restrict__ cu, int32_t R, float gamma,
      float lam, float* __restrict__ adv, float* __restrict__ ret) {
  const int r = (blockIdx.x * blockDim.x + threadIdx.x) >> 5;
  const int lane = threadIdx.x & 31;
  if (r >= R) return;
  const int t_lo = cu[r], t_hi = cu[r + 1];
  const float c = gamma * lam;
  float a_carry = 0.f;       // A at the nearest scored token after the chunk
  float v_carry = 0.f;       // its value (0 past the end of the response)
  for (int base = t_hi - 32; base > t_lo - 32; base -= 32) {
    const int t = base + lane;
    const bool in = t >= t_lo;
    const bool sc = in && (mask == nullptr || mask[t] != 0);
    const float v = in ? values[t] : 0.f;
    const float rw = in ? rewards[t] : 0.f;
    // nearest scored value strictly to the right (inclusive scan of (has, val), then shift)
    int has = sc ? 1 : 0;
    float nv = sc ? v : 0.f;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
      const int h2 = __shfl_down_sync(0xffffffffu, has, o);
      const float n2 = __shfl_down_sync(0xffffffffu, nv, o);
      if (lane + o < 32 && !has) { has = h2; nv = n2; }
    }
    int has_r = __shfl_down_sync(0xffffffffu, has, 1);
    float nv_r = __shfl_down_sync(0xffffffffu, nv, 1);
    if (lane == 31) has_r = 0;
    const float v_next = has_r ? nv_r : v_carry;
    // affine map of this token, then reverse inclusive scan of compositions f_t o f_{t+1} o ...
    float ma = sc ? c : 1.f;
    float mb = sc ? rw + gamma * v_next - v : 0.f;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
      const float a2 = __shfl_down_sync(0xffffffffu, ma, o);
      const float b2 = __shfl_down_sync(0xffffffffu, mb, o);
      if (lane + o < 32) { mb = fmaf(ma, b2, mb); ma *= a2; }
    }
    const float a_t = fmaf(ma, a_carry, mb);
    if (in) {
      adv[t] = sc ? a_t : 0.f;
      ret[t] = sc ? a_t + v : 0.f;
    }
    // carries for the next (earlier) chunk: lane 0 holds the composition of the whole chunk
    a_carry = __shfl_sync(0xffffffffu, a_t, 0);
    const int has0 = __shfl_sync(0xffffffffu, has, 0);
    const float nv0 = __shfl_sync(0xffffffffu, nv, 0);
    if (has0) v_carry = nv0;
  }
}

// ---- steps 3 + 4: clipped value loss and d loss / d v.  Two launches: count, then loss. --------
struct VCounters { unsigned long long n_scored, n_clipped; unsigned int ticket, pad; };
struct VPartial { double loss; };
constexpr int kVThreads = 256;
constexpr int kVTile = kVThreads * 4;

__global__ void k_vloss_count(const uint8_t* __restrict__ mask, int64_t T, VCounters* cnt) {
  unsigned int c = 0;
  for (int64_t t = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; t < T;
       t += (int64_t)gridDim.x * blockDim.x)
    c += mask[t] != 0 ? 1u : 0u;
  c = wsum(c);
  if ((threadIdx.x & 31) == 0 && c) atomicAdd(&cnt->n_scored, (unsigned long long)c);
}

__global__ void __launch_bounds__(kVThreads)
k_vloss(const float* __restrict__ values, const float* __restrict__ old_values,
        const float* __restrict__ returns, const uint8_t* __restrict__ mask, int64_t T, float clip_v,
        float grad_loss, VCounters* __restrict__ cnt, VPartial* __restrict__ partials,
        float* __restrict__ out3, float* __restrict__ g) {
  const double n_scored = mask ? (double)cnt->n_scored : (double)T;
  const float gs = grad_loss / (float)fmax(n_scored, 1.0);
  float acc = 0.f;
  unsigned int ncl = 0;
  const int64_t t0 = (int64_t)blockIdx.x * kVTile;
#pragma unroll
  for (int k = 0; k < 4; ++k) {
    const int64_t t = t0 + (int64_t)k * kVThreads + threadIdx.x;
    if (t >= T) continue;
    const bool sc = mask == nullptr || mask[t] != 0;
    const float v = values[t], vo = old_values[t], rt = returns[t];
    const float vc = fminf(fmaxf(v, vo - clip_v), vo + clip_v);
    const float e1 = v - rt, e2 = vc - rt;
    const float l1 = e1 * e1, l2 = e2 * e2;
    const bool unclipped = l1 >= l2;
    const bool inside = v > vo - clip_v && v < vo + clip_v;
    if (sc) {
      acc += 0.5f * fmaxf(l1, l2);
      ncl += unclipped ? 0u : 1u;
    }
    if (g) g[t] = sc ? gs * (unclipped ? e1 : (inside ? e2 : 0.f)) : 0.f;
  }
  double d = wsum((double)acc);
  ncl = wsum(ncl);
  __shared__ double s_l[kVThreads / 32];
  __shared__ unsigned int s_c[kVThreads / 32];
  __shared__ bool is_last;
  const int wid = threadIdx.x >> 5;
  if ((threadIdx.x & 31) == 0) { s_l[wid] = d; s_c[wid] = ncl; }
  __syncthreads();
  if (threadIdx.x == 0) {
    double a = 0.0;
    unsigned long long c = 0;
    for (int w = 0; w < kVThreads / 32; ++w) { a += s_l[w]; c += s_c[w]; }
    partials[blockIdx.x].loss = a;
    if (c) atomicAdd(&cnt->n_clipped, c);
    __threadfence();
    is_last = atomicAdd(&cnt->ticket, 1u) == gridDim.x - 1;
  }
  __syncthreads();
  if (!is_last) return;
  __threadfence();
  double a = 0.0;
  for (unsigned int i = threadIdx.x; i < gridDim.x; i += kVThreads) a += partials[i].loss;
  a = wsum(a);
  __syncthreads();
  if ((threadIdx.x & 31) == 0) s_l[wid] = a;
  __syncthreads();
  if (threadIdx.x == 0) {
    a = 0.0;
    for (int w = 0; w < kVThreads / 32; ++w) a += s_l[w];
    const double denom = fmax(n_scored, 1.0);
    out3[0] = (float)(a / denom);
    out3[1] = (float)((double)atomicAdd(&cnt->n_clipped, 0ull) / denom);
    out3[2] = (float)n_scored;
  }
}

// ---- step 5: dH[t,:] = g_t w (written once), dw = sum_t g_t H[t,:], db = sum_t g_t.  A block owns
// kBwdRows consecutive rows and a 2048-column slab; thread = 8 columns; per-block partial dw rows
// go to the workspace and a second kernel sums them in block order (deterministic). -------------
constexpr int kBwdThreads = 256;
constexpr int kBwdCols = kBwdThreads * 8;     // columns per block slab
constexpr int kBwdRows = 64;                  // rows per block

template <bool kBf16>
__global__ void __launch_bounds__(kBwdThreads)
k_value_bwd(const void* __restrict__ H, int64_t ld, const void* __restrict__ w,
            const float* __restrict__ g, int64_t T, int64_t D, void* __restrict__ dH, int64_t lddH,
            float* __restrict__ dw_part /*[row blocks, D]*/, float* __restrict__ db_part) {
  const int64_t col = (int64_t)blockIdx.y * kBwdCols + (int64_t)threadIdx.x * 8;
  if (col >= D) return;
  float wv[8], acc[8];
  if (kBf16) {
    bf16x8_to_f32(__ldg(reinterpret_cast<const int4*>(static_cast<const __nv_bfloat16*>(w) + col)), wv);
  } else {
    const float4 a = __ldg(reinterpret_cast<const float4*>(static_cast<const float*>(w) + col));
    const float4 b = __ldg(reinterpret_cast<const float4*>(static_cast<const float*>(w) + col + 4));
    wv[0] = a.x; wv[1] = a.y; wv[2] = a.z; wv[3] = a.w; wv[4] = b.x; wv[5] = b.y; wv[6] = b.z; wv[7] = b.w;
  }
#pragma unroll
  for (int j = 0; j < 8; ++j) acc[j] = 0.f;
  float gsum = 0.f;                              // sum of g over this block's rows (for dbias)
  // persistent over row tiles: tile = blockIdx.x, + gridDim.x, ... (one partial per block)
  for (int64_t r0 = (int64_t)blockIdx.x * kBwdRows; r0 < T; r0 += (int64_t)gridDim.x * kBwdRows) {
  const int64_t r1 = r0 + kBwdRows < T ? r0 + kBwdRows : T;
  // 4 rows per step: the 4 loads of H are issued before anything depends on them
  for (int64_t tb = r0; tb < r1; tb += 4) {
    float gt[4], h[4][8];
#pragma unroll
    for (int u = 0; u < 4; ++u) {
      const int64_t t = tb + u < r1 ? tb + u : r1 - 1;       // clamp: duplicates get gt = 0
      gt[u] = tb + u < r1 ? g[t] : 0.f;
      if (kBf16) {
        bf16x8_to_f32(__ldcs(reinterpret_cast<const int4*>(static_cast<const __nv_bfloat16*>(H) + t * ld + col)),
                      h[u]);
      } else {
        const float* hp = static_cast<const float*>(H) + t * ld + col;
        const float4 a = __ldcs(reinterpret_cast<const float4*>(hp));
        const float4 c = __ldcs(reinterpret_cast<const float4*>(hp + 4));
        h[u][0] = a.x; h[u][1] = a.y; h[u][2] = a.z; h[u][3] = a.w;
        h[u][4] = c.x; h[u][5] = c.y; h[u][6] = c.z; h[u][7] = c.w;
      }
    }
#pragma unroll
    for (int u = 0; u < 4; ++u) {
      if (tb + u >= r1) break;
      const int64_t t = tb + u;
      if (kBf16) {
        __nv_bfloat162 o[4];
#pragma unroll
        for (int j = 0; j < 4; ++j) o[j] = __floats2bfloat162_rn(gt[u] * wv[2 * j], gt[u] * wv[2 * j + 1]);
        __stcs(reinterpret_cast<int4*>(static_cast<__nv_bfloat16*>(dH) + t * lddH + col),
               *reinterpret_cast<const int4*>(o));
      } else {
        float* op = static_cast<float*>(dH) + t * lddH + col;
        __stcs(reinterpret_cast<float4*>(op),
               make_float4(gt[u] * wv[0], gt[u] * wv[1], gt[u] * wv[2], gt[u] * wv[3]));
        __stcs(reinterpret_cast<float4*>(op + 4),
               make_float4(gt[u] * wv[4], gt[u] * wv[5], gt[u] * wv[6], gt[u] * wv[7]));
      }
#pragma unroll
      for (int j = 0; j < 8; ++j) acc[j] = fmaf(gt[u], h[u][j], acc[j]);
      gsum += gt[u];
    }
  }
  }
  if (blockIdx.y == 0 && threadIdx.x == 0) db_part[blockIdx.x] = gsum;
  float* out = dw_part + (int64_t)blockIdx.x * D + col;
  *reinterpret_cast<float4*>(out) = make_float4(acc[0], acc[1], acc[2], acc[3]);
  *reinterpret_cast<float4*>(out + 4) = make_float4(acc[4], acc[5], acc[6], acc[7]);
}

// dw[d] = sum over row blocks in index order (fp64); db = the blocks' row sums in index order
__global__ void k_value_bwd_reduce(const float* __restrict__ dw_part, const float* __restrict__ db_part,
                                   int64_t nblocks, int64_t D, float* __restrict__ dw,
                                   float* __restrict__ dbias) {
  const int64_t d = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (d < D) {
    double a = 0.0;
    for (int64_t b = 0; b < nblocks; ++b) a += (double)dw_part[b * D + d];
    dw[d] = (float)a;
  }
  if (blockIdx.x == 0 && threadIdx.x == 0 && dbias) {
    double a = 0.0;
    for (int64_t b = 0; b < nblocks; ++b) a += (double)db_part[b];
    *dbias = (float)a;
  }
}

}  // namespace

int launch_value_fwd(const void* H, int64_t ldH, bool bf16, const void* w, float bias, int64_t T,
                     int64_t D, float* values, cudaStream_t st) {
  int64_t blocks = ceil_div(T, 8);
  if (blocks > kNumSMs * 16) blocks = kNumSMs * 16;
  if (bf16) k_value_fwd<true><<<(unsigned)blocks, 256, 0, st>>>(H, ldH, w, bias, T, D, values);
  else k_value_fwd<false><<<(unsigned)blocks, 256, 0, st>>>(H, ldH, w, bias, T, D, values);
  GC_CUDA_TRY(cudaGetLastError());
  return GC_OK;
}

int launch_gae(const float* rewards, const float* values, const uint8_t* mask, const int32_t* cu,
               int32_t R, float gamma, float lam, float* adv, float* ret, cudaStream_t st) {
  k_gae<<<(unsigned)ceil_div((int64_t)R * 32, 256), 256, 0, st>>>(rewards, values, mask, cu, R, gamma,
                                                                  lam, adv, ret);
  GC_CUDA_TRY(cudaGetLastError());
  return GC_OK;
}

size_t value_loss_ws_bytes(int64_t T) {
  return 256 + align_up((size_t)ceil_div(T > 0 ? T : 1, kVTile) * sizeof(VPartial), 256);
}

int launch_value_loss(const float* values, const float* old_values, const float* returns,
                      const uint8_t* mask, int64_t T, float clip_v, float grad_loss, float* out3,
                      float* g, void* ws, cudaStream_t st) {
  Carver c(ws);
  VCounters* cnt = c.take<VCounters>(1);
  VPartial* partials = c.take<VPartial>((size_t)ceil_div(T, kVTile));
  GC_CUDA_TRY(cudaMemsetAsync(cnt, 0, sizeof(VCounters), st));
  if (mask) {
    int64_t b = ceil_div(T, 256 * 8);
    if (b > kNumSMs * 8) b = kNumSMs * 8;
    k_vloss_count<<<(unsigned)b, 256, 0, st>>>(mask, T, cnt);
  }
  k_vloss<<<(unsigned)ceil_div(T, kVTile), kVThreads, 0, st>>>(values, old_values, returns, mask, T,
                                                              clip_v, grad_loss, cnt, partials, out3, g);
  GC_CUDA_TRY(cudaGetLastError());
  return GC_OK;
}

static int64_t value_bwd_row_blocks(int64_t T) {
  const int64_t rb = ceil_div(T > 0 ? T : 1, kBwdRows);
  return rb < 2 * kNumSMs ? rb : 2 * kNumSMs;      // a function of T only: reruns are bit-identical
}
size_t value_bwd_ws_bytes(int64_t T, int64_t D) {
  return align_up((size_t)value_bwd_row_blocks(T) * (size_t)D * sizeof(float), 256) +
         align_up((size_t)value_bwd_row_blocks(T) * sizeof(float), 256);
}

int launch_value_bwd(const void* H, int64_t ldH, bool bf16, const void* w, const float* g, int64_t T,
                     int64_t D, void* dH, int64_t lddH, float* dw, float* dbias, void* ws,
                     cudaStream_t st) {
  const int64_t rb = value_bwd_row_blocks(T);
  Carver c(ws);
  float* part = c.take<float>((size_t)rb * (size_t)D);
  float* db_part = c.take<float>((size_t)rb);
  dim3 grid((unsigned)rb, (unsigned)ceil_div(D, kBwdCols));
  if (bf16) k_value_bwd<true><<<grid, kBwdThreads, 0, st>>>(H, ldH, w, g, T, D, dH, lddH, part, db_part);
  else k_value_bwd<false><<<grid, kBwdThreads, 0, st>>>(H, ldH, w, g, T, D, dH, lddH, part, db_part);
  k_value_bwd_reduce<<<(unsigned)ceil_div(D, 256), 256, 0, st>>>(part, db_part, rb, D, dw, dbias);
  GC_CUDA_TRY(cudaGetLastError());
  return GC_OK;
}

}  // namespace gc

// ---- gc_value_loss_static_scratch: the value loss for callers that cannot obtain device memory --
// The scratch of the value loss (the counters block and one fp64 partial per 1024-token tile) lives
// in this file-scope device array instead of a caller workspace.  It is part of the library image:
// every GPU that loads libgcore.so carries these 33,024 bytes from module load until the process
// exits.  Its size fixes the largest T the entry point takes (GC_VALUE_LOSS_STATIC_MAX_T).
namespace gc {
namespace {

constexpr int64_t kStaticMaxT = GC_VALUE_LOSS_STATIC_MAX_T;
constexpr size_t kStaticScratchBytes = 256 + (size_t)(kStaticMaxT / kVTile) * sizeof(VPartial);
static_assert(kStaticMaxT % kVTile == 0, "the limit is a whole number of tiles");
static_assert(sizeof(VCounters) <= 256, "counters fit the first 256-byte granule");

static __device__ __align__(256) unsigned char g_vloss_static_scratch[kStaticScratchBytes];

// On the host `g_vloss_static_scratch` is only a handle for the runtime's symbol table: it is NOT
// the array's device address and must never be handed to a kernel.  The real address differs per
// device (each device has its own copy of the array) and comes from cudaGetSymbolAddress, asked
// once per device with that device current and remembered here.
constexpr int kStaticMaxDevices = 64;
std::atomic<void*> g_vloss_static_addr[kStaticMaxDevices];

int static_scratch_address(void** out) {
  int dev = 0;
  GC_CUDA_TRY(cudaGetDevice(&dev));
  const bool cached = dev >= 0 && dev < kStaticMaxDevices;
  void* p = cached ? g_vloss_static_addr[dev].load(std::memory_order_acquire) : nullptr;
  if (!p) {
    GC_CUDA_TRY(cudaGetSymbolAddress(&p, g_vloss_static_scratch));   // device `dev` is current
    if (!p) return GC_ERR_CUDA;
    // two host threads may both get here on a first call: they publish the same address
    if (cached) g_vloss_static_addr[dev].store(p, std::memory_order_release);
  }
  *out = p;
  return GC_OK;
}

}  // namespace
}  // namespace gc

extern "C" int gc_value_loss_static_scratch(const float* values, const float* old_values,
                                            const float* returns, const uint8_t* mask, int64_t T,
                                            float clip_v, float grad_loss, float* out3, float* g,
                                            void* cuda_stream) {
  using namespace gc;
  if (T < 0) return GC_ERR_SHAPE;
  if (T > kStaticMaxT) return GC_ERR_SHAPE;        // the fixed array has no room for more tiles
  if (!(clip_v >= 0.f)) return GC_ERR_ARG;
  if (!out3) return GC_ERR_NULL;
  cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
  if (T == 0) {
    GC_CUDA_TRY(cudaMemsetAsync(out3, 0, 3 * sizeof(float), st));
    return GC_OK;
  }
  if (!values || !old_values || !returns) return GC_ERR_NULL;
  void* scratch = nullptr;
  GC_TRY(static_scratch_address(&scratch));
  // Same two kernels and the same carving as gc_value_loss, so the results are bit-identical to it.
  // The array still holds the previous call's counters and partials: launch_value_loss clears the
  // counters block on the stream (a memset node, no allocation) and every partial that is read is
  // written first by its own block in this launch.
  return launch_value_loss(values, old_values, returns, mask, T, clip_v, grad_loss, out3, g, scratch,
                           st);
}
