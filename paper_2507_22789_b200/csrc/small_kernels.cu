// small_kernels.cu -- the HBM/latency-bound steps of the path (SURVEY.md sec 8(a) rows a1, a4,
// a6-a9): row selection/compaction, partial-stat combine, group filter + GRPO advantages,
// per-token clipped-ratio loss with k3 KL and its gradient w.r.t. logp.
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
// a8 + a9: per-token loss and d loss / d logp.
//   rho = e^{logp-old}; s = min(rho A, clip(rho) A); d = ref - logp; k3 = e^d - d - 1
//   l = -s + beta k3;   dl/dlogp = -[rho A <= clip(rho) A] rho A + beta (1 - e^d)
// Weights: token-mean w_t = m_t / max(sum m, 1);  seq-mean w_t = m_t / (R_kept max(cnt_r, 1)).
// Pass 1 (k_loss_counts): integer counts (sum m; per-response counts, R_kept) -- integer
// atomics only.  Pass 2 (k_token_loss): each block reduces its tile in fixed order to fp64
// partials; the last block to finish (integer ticket) sums the partials in index order.
// =============================================================================================
struct LossCounters {
  unsigned long long n_scored;   // sum_t m_t
  unsigned long long n_clipped;
  unsigned int n_kept;           // responses with >= 1 scored token
  unsigned int ticket;
};

// e^x as one multiply and one MUFU.EX2 (relative error ~2^-22; exact 1 at x = 0, which keeps the
// identities rho = 1 for logp = old and k3 = 0 for logp = ref exact)
__device__ __forceinline__ float fast_exp(float x) {
  float y;
  asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x * kLog2e));
  return y;
}

constexpr int kLossThreads = 256;
constexpr int kLossTile = kLossThreads * 4 * 2;   // tokens per block (4 per thread, 2 rounds)
constexpr int kCuSmem = kLossTile + 8;            // cu_seqlens entries staged per block

// upper_bound(cu, cu+R+1, t) - 1  : response containing token t (cu[0]=0, cu[R]=T).
template <typename P>
__device__ __forceinline__ int find_response(P cu, int lo, int hi, int32_t t) {
  // invariant: cu[lo] <= t < cu[hi]
  while (hi - lo > 1) {
    const int mid = (lo + hi) >> 1;
    if (cu[mid] <= t) lo = mid; else hi = mid;
  }
  return lo;
}

// Pass 0: first response of every kLossTile-token tile (one thread per tile), so that
// the token kernels stage only their own slice of cu_seqlens in shared memory instead of paying a
// ~22-step dependent global binary search per thread.
__global__ void k_loss_tile_ranges(const int32_t* __restrict__ cu, int32_t R, int64_t T,
                                   int64_t ntiles, int32_t* __restrict__ tile_r) {
  const int64_t b = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (b > ntiles) return;
  // tile b spans responses tile_r[b] .. tile_r[b+1] (the response of the next tile's first token
  // bounds the response of this tile's last token); the sentinel entry is the last response
  tile_r[b] = b < ntiles ? find_response(cu, 0, R, (int32_t)(b * kLossTile)) : (R > 0 ? R - 1 : 0);
}

// The slice cu[r0 .. r1+1] of one tile, in shared memory when it fits.
struct CuSlice {
  const int32_t* g;     // global cu_seqlens
  const int32_t* s;     // shared copy (entry i = cu[r0 + i]) or nullptr
  int r0, r1;
  __device__ __forceinline__ int32_t at(int r) const { return s ? s[r - r0] : g[r]; }
  __device__ __forceinline__ int locate(int32_t t) const {   // response containing token t
    int lo = r0, hi = r1 + 1;
    while (hi - lo > 1) {
      const int mid = (lo + hi) >> 1;
      if (at(mid) <= t) lo = mid; else hi = mid;
    }
    return lo;
  }
};

__device__ __forceinline__ CuSlice load_cu_slice(const int32_t* __restrict__ cu,
                                                 const int32_t* __restrict__ tile_r,
                                                 int32_t* smem) {
  CuSlice c;
  c.g = cu;
  c.r0 = tile_r[blockIdx.x];
  c.r1 = tile_r[blockIdx.x + 1];
  const int n = c.r1 - c.r0 + 2;
  c.s = nullptr;
  if (n <= kCuSmem) {
    for (int i = threadIdx.x; i < n; i += blockDim.x) smem[i] = cu[c.r0 + i];
    c.s = smem;
  }
  __syncthreads();
  return c;
}

// 4 consecutive tokens' targets + mask -> scored flags (vector loads when the group is whole)
__device__ __forceinline__ void load_scored4(const int32_t* __restrict__ targets,
                                             const uint8_t* __restrict__ mask, int64_t t0, int nt,
                                             int32_t (&y)[4], bool (&sc)[4]) {
  uint8_t mk[4] = {1, 1, 1, 1};
  if (nt == 4) {
    const int4 c = *reinterpret_cast<const int4*>(targets + t0);
    y[0] = c.x; y[1] = c.y; y[2] = c.z; y[3] = c.w;
    if (mask) {
      const uchar4 e = *reinterpret_cast<const uchar4*>(mask + t0);
      mk[0] = e.x; mk[1] = e.y; mk[2] = e.z; mk[3] = e.w;
    }
  } else {
    for (int i = 0; i < 4; ++i) {
      y[i] = i < nt ? targets[t0 + i] : -1;
      mk[i] = (i < nt && mask) ? mask[t0 + i] : 1;
    }
  }
#pragma unroll
  for (int i = 0; i < 4; ++i) sc[i] = i < nt && y[i] >= 0 && mk[i] != 0;
}

// Pass 1: integer counts.  n_scored always; for seq-mean also the scored tokens per response
// (run-length per thread, one integer atomicAdd per response a thread touches; the thread that
// finds the old value 0 counts the response as kept).  Integer atomics only: order-independent.
__global__ void __launch_bounds__(kLossThreads)
k_loss_counts(const int32_t* __restrict__ targets, const uint8_t* __restrict__ mask, int64_t T,
              const int32_t* __restrict__ cu, int32_t R, const int32_t* __restrict__ tile_r,
              int per_response,
              int32_t* __restrict__ resp_cnt, LossCounters* __restrict__ cnt) {
  __shared__ int32_t s_cu[kCuSmem];
  CuSlice cs;
  const int64_t tile0 = (int64_t)blockIdx.x * kLossTile;
  if (per_response) cs = load_cu_slice(cu, tile_r, s_cu);
  unsigned int n_sc = 0, n_kept = 0;
#pragma unroll
  for (int round = 0; round < 2; ++round) {
    const int64_t t0 = tile0 + ((int64_t)round * kLossThreads + threadIdx.x) * 4;
    if (t0 >= T) continue;
    const int nt = (int)min((int64_t)4, T - t0);
    int32_t y[4];
    bool sc[4];
    load_scored4(targets, mask, t0, nt, y, sc);
    if (!per_response) {
      n_sc += (unsigned)sc[0] + (unsigned)sc[1] + (unsigned)sc[2] + (unsigned)sc[3];
      continue;
    }
    int r = cs.locate((int32_t)t0);
    int32_t r_end = cs.at(r + 1);
    int run = 0;
#pragma unroll
    for (int i = 0; i < 4; ++i) {
      if (i >= nt) break;
      const int32_t t = (int32_t)(t0 + i);
      if (t >= r_end) {
        if (run) { n_kept += atomicAdd(resp_cnt + r, run) == 0 ? 1u : 0u; n_sc += run; run = 0; }
        while (t >= r_end && r + 1 < R) { ++r; r_end = cs.at(r + 1); }
      }
      run += sc[i] ? 1 : 0;
    }
    if (run) { n_kept += atomicAdd(resp_cnt + r, run) == 0 ? 1u : 0u; n_sc += run; }
  }
  n_sc = warp_sum(n_sc);
  n_kept = warp_sum(n_kept);
  __shared__ unsigned int sm[2][kLossThreads / 32];
  if ((threadIdx.x & 31) == 0) { sm[0][threadIdx.x >> 5] = n_sc; sm[1][threadIdx.x >> 5] = n_kept; }
  __syncthreads();
  if (threadIdx.x == 0) {
    unsigned long long a = 0;
    unsigned int k = 0;
    for (int w = 0; w < kLossThreads / 32; ++w) { a += sm[0][w]; k += sm[1][w]; }
    if (a) atomicAdd(&cnt->n_scored, a);
    if (k) atomicAdd(&cnt->n_kept, k);
  }
}

// seq-mean with long responses (>= 128 tokens on average): one warp per response, coalesced; the
// token-parallel kernel above would put ~L/8 atomics on one counter.
__global__ void k_loss_counts_seq(const int32_t* __restrict__ targets,
                                  const uint8_t* __restrict__ mask,
                                  const int32_t* __restrict__ cu, int32_t R,
                                  int32_t* __restrict__ resp_cnt, LossCounters* __restrict__ cnt) {
  const int r = (blockIdx.x * blockDim.x + threadIdx.x) >> 5;
  const int lane = threadIdx.x & 31;
  if (r >= R) return;
  unsigned int c = 0;
  for (int64_t t = cu[r] + lane; t < cu[r + 1]; t += 32) c += is_scored(targets, mask, t) ? 1u : 0u;
  c = warp_sum(c);
  if (lane == 0) {
    resp_cnt[r] = (int32_t)c;
    if (c) {
      atomicAdd(&cnt->n_scored, (unsigned long long)c);
      atomicAdd(&cnt->n_kept, 1u);
    }
  }
}

struct LossPartial { double loss_pg, loss_kl; };

// Pass 2: per-token loss terms and g.  21 B per token (logp, old, ref, target 4 B each, mask 1 B,
// g 4 B written), 16-byte vector accesses, both rounds' loads issued before the arithmetic.
__global__ void __launch_bounds__(kLossThreads)
k_token_loss(const float* __restrict__ logp, const float* __restrict__ old_logp,
             const float* __restrict__ ref_logp, const int32_t* __restrict__ targets,
             const uint8_t* __restrict__ mask, int64_t T, const int32_t* __restrict__ cu,
             int32_t R, const float* __restrict__ adv, const int32_t* __restrict__ resp_cnt,
             const int32_t* __restrict__ tile_r, float clip_lo, float clip_hi, float beta, int agg, float grad_loss,
             LossCounters* __restrict__ cnt, LossPartial* __restrict__ partials,
             float* __restrict__ out5, float* __restrict__ g) {
  __shared__ int32_t s_cu[kCuSmem];
  const int64_t tile0 = (int64_t)blockIdx.x * kLossTile;
  // Whole tiles: issue this thread's 8 tokens' loads first, so that their DRAM latency overlaps
  // the staging of the cu_seqlens slice (two dependent loads and a block barrier).
  const bool whole = tile0 + kLossTile <= T;
  const int64_t t0f = tile0 + (int64_t)threadIdx.x * 8;
  float4 a0, a1, b0, b1, d0, d1;
  int4 c0, c1;
  unsigned long long mk8 = 0x0101010101010101ull;
  if (whole) {
    a0 = *reinterpret_cast<const float4*>(logp + t0f);
    a1 = *reinterpret_cast<const float4*>(logp + t0f + 4);
    b0 = *reinterpret_cast<const float4*>(old_logp + t0f);
    b1 = *reinterpret_cast<const float4*>(old_logp + t0f + 4);
    c0 = *reinterpret_cast<const int4*>(targets + t0f);
    c1 = *reinterpret_cast<const int4*>(targets + t0f + 4);
    if (ref_logp) {
      d0 = *reinterpret_cast<const float4*>(ref_logp + t0f);
      d1 = *reinterpret_cast<const float4*>(ref_logp + t0f + 4);
    } else {
      d0 = a0;
      d1 = a1;
    }
    if (mask) {
      // t0f is a multiple of 8: the 8-byte load is aligned iff the mask pointer is; a mask view
      // at a 4-byte offset (the API's minimum alignment) takes two 4-byte loads
      if ((reinterpret_cast<uintptr_t>(mask) & 7) == 0) {
        mk8 = *reinterpret_cast<const unsigned long long*>(mask + t0f);
      } else {
        const unsigned int lo4 = *reinterpret_cast<const unsigned int*>(mask + t0f);
        const unsigned int hi4 = *reinterpret_cast<const unsigned int*>(mask + t0f + 4);
        mk8 = (unsigned long long)lo4 | ((unsigned long long)hi4 << 32);
      }
    }
  }
  const CuSlice cs = load_cu_slice(cu, tile_r, s_cu);
  const double n_scored = (double)cnt->n_scored;
  const double n_kept = (double)cnt->n_kept;
  // gradient scale shared by every token of the batch
  const float gscale_tok = grad_loss / (float)fmax(n_scored, 1.0);
  const float gscale_seq = grad_loss / (float)fmax(n_kept, 1.0);
  const float lo_c = 1.0f - clip_lo, hi_c = 1.0f + clip_hi;

  float acc_pg = 0.f, acc_kl = 0.f;     // 8 terms per thread in fp32, fp64 from there on
  unsigned int n_clip = 0;

  if (cs.s != nullptr && whole) {
    // ---- fast path: whole tile, cu slice in shared memory.  8 consecutive tokens per thread,
    // tile-relative 32-bit indices, one binary search per thread then a forward walk. ----
    const int64_t t0 = t0f;
    float lp[8], ol[8], rf[8], gout[8];
    int32_t y[8];
    lp[0] = a0.x; lp[1] = a0.y; lp[2] = a0.z; lp[3] = a0.w;
    lp[4] = a1.x; lp[5] = a1.y; lp[6] = a1.z; lp[7] = a1.w;
    ol[0] = b0.x; ol[1] = b0.y; ol[2] = b0.z; ol[3] = b0.w;
    ol[4] = b1.x; ol[5] = b1.y; ol[6] = b1.z; ol[7] = b1.w;
    rf[0] = d0.x; rf[1] = d0.y; rf[2] = d0.z; rf[3] = d0.w;
    rf[4] = d1.x; rf[5] = d1.y; rf[6] = d1.z; rf[7] = d1.w;
    y[0] = c0.x; y[1] = c0.y; y[2] = c0.z; y[3] = c0.w;
    y[4] = c1.x; y[5] = c1.y; y[6] = c1.z; y[7] = c1.w;
    // slice-relative response index: largest r with cu[r0 + r] <= t0
    const int32_t* sc_ = cs.s;
    const int32_t tq = (int32_t)t0;
    int lo = 0, hi = cs.r1 - cs.r0 + 1;
    while (hi - lo > 1) {
      const int mid = (lo + hi) >> 1;
      if (sc_[mid] <= tq) lo = mid; else hi = mid;
    }
    int r = lo;
    int32_t r_end = sc_[r + 1];
    float A = adv[cs.r0 + r];
    float w = 1.0f, gs = gscale_tok;
    if (agg == GC_AGG_SEQ_MEAN) {
      w = 1.0f / (float)max(resp_cnt[cs.r0 + r], 1);
      gs = gscale_seq * w;
    }
#pragma unroll
    for (int i = 0; i < 8; ++i) {
      const int32_t t = tq + i;
      if (t >= r_end) {
        do { ++r; r_end = sc_[r + 1]; } while (t >= r_end);
        A = adv[cs.r0 + r];
        if (agg == GC_AGG_SEQ_MEAN) {
          w = 1.0f / (float)max(resp_cnt[cs.r0 + r], 1);
          gs = gscale_seq * w;
        }
      }
      const bool scored = y[i] >= 0 && ((mk8 >> (8 * i)) & 0xffull) != 0;
      const float rho = fast_exp(lp[i] - ol[i]);
      const float s1 = rho * A;
      const float s2 = fminf(fmaxf(rho, lo_c), hi_c) * A;
      const bool unclipped = s1 <= s2;
      const float sm = fminf(s1, s2);
      const float d = rf[i] - lp[i];
      const float ed = fast_exp(d);
      const float k3 = ed - d - 1.0f;
      // selects, not zero weights: inf / NaN at an unscored position must not reach the sums
      acc_pg -= scored ? sm * w : 0.0f;
      acc_kl += scored ? k3 * w : 0.0f;
      n_clip += (scored && !unclipped) ? 1u : 0u;
      gout[i] = scored ? gs * ((unclipped ? -s1 : 0.0f) + beta * (1.0f - ed)) : 0.0f;
    }
    if (g) {
      *reinterpret_cast<float4*>(g + t0) = make_float4(gout[0], gout[1], gout[2], gout[3]);
      *reinterpret_cast<float4*>(g + t0 + 4) = make_float4(gout[4], gout[5], gout[6], gout[7]);
    }
  } else {
  // ---- general path (last, partial tile; cu slice too long for shared memory) ----
  // ---- loads of both rounds first (memory-level parallelism) ----
  float lp[2][4], ol[2][4], rf[2][4];
  int32_t y[2][4];
  bool sc[2][4];
  int nts[2];
#pragma unroll
  for (int round = 0; round < 2; ++round) {
    const int64_t t0 = tile0 + ((int64_t)round * kLossThreads + threadIdx.x) * 4;
    const int nt = t0 >= T ? 0 : (int)min((int64_t)4, T - t0);
    nts[round] = nt;
    if (nt == 4) {
      const float4 a = *reinterpret_cast<const float4*>(logp + t0);
      const float4 b = *reinterpret_cast<const float4*>(old_logp + t0);
      lp[round][0] = a.x; lp[round][1] = a.y; lp[round][2] = a.z; lp[round][3] = a.w;
      ol[round][0] = b.x; ol[round][1] = b.y; ol[round][2] = b.z; ol[round][3] = b.w;
      if (ref_logp) {
        const float4 d = *reinterpret_cast<const float4*>(ref_logp + t0);
        rf[round][0] = d.x; rf[round][1] = d.y; rf[round][2] = d.z; rf[round][3] = d.w;
      } else {
#pragma unroll
        for (int i = 0; i < 4; ++i) rf[round][i] = lp[round][i];
      }
    } else {
      for (int i = 0; i < 4; ++i) {
        const bool in = i < nt;
        lp[round][i] = in ? logp[t0 + i] : 0.f;
        ol[round][i] = in ? old_logp[t0 + i] : 0.f;
        rf[round][i] = in ? (ref_logp ? ref_logp[t0 + i] : lp[round][i]) : 0.f;
      }
    }
    if (nt > 0) load_scored4(targets, mask, t0, nt, y[round], sc[round]);
  }

#pragma unroll
  for (int round = 0; round < 2; ++round) {
    const int nt = nts[round];
    if (nt == 0) continue;
    const int64_t t0 = tile0 + ((int64_t)round * kLossThreads + threadIdx.x) * 4;
    // response of the first token by binary search in the staged slice, then walk forward
    int r = cs.locate((int32_t)t0);
    int32_t r_end = cs.at(r + 1);
    float gout[4];
#pragma unroll
    for (int i = 0; i < 4; ++i) {
      gout[i] = 0.f;
      if (i >= nt) continue;
      const int32_t t = (int32_t)(t0 + i);
      while (t >= r_end && r + 1 < R) { ++r; r_end = cs.at(r + 1); }
      if (!(sc[round][i] && t < r_end)) continue;
      const float A = adv[r];
      const float rho = fast_exp(lp[round][i] - ol[round][i]);
      const float s1 = rho * A;
      const float s2 = fminf(fmaxf(rho, lo_c), hi_c) * A;
      const bool unclipped = s1 <= s2;
      const float s = fminf(s1, s2);
      const float d = rf[round][i] - lp[round][i];
      const float ed = fast_exp(d);
      const float k3 = ed - d - 1.0f;
      float w = 1.0f, gs = gscale_tok;
      if (agg == GC_AGG_SEQ_MEAN) {
        w = 1.0f / (float)max(resp_cnt[r], 1);
        gs = gscale_seq * w;
      }
      acc_pg -= s * w;
      acc_kl += k3 * w;
      n_clip += unclipped ? 0u : 1u;
      gout[i] = gs * ((unclipped ? -s1 : 0.0f) + beta * (1.0f - ed));
    }
    if (g) {
      if (nt == 4) *reinterpret_cast<float4*>(g + t0) = make_float4(gout[0], gout[1], gout[2], gout[3]);
      else for (int i = 0; i < nt; ++i) g[t0 + i] = gout[i];
    }
  }
  }
  // block reduction in fixed order
  double d_pg = warp_sum((double)acc_pg);
  double d_kl = warp_sum((double)acc_kl);
  n_clip = warp_sum(n_clip);
  __shared__ double s_pg[kLossThreads / 32], s_kl[kLossThreads / 32];
  __shared__ unsigned int s_cl[kLossThreads / 32];
  __shared__ bool is_last;
  const int wid = threadIdx.x >> 5;
  if ((threadIdx.x & 31) == 0) { s_pg[wid] = d_pg; s_kl[wid] = d_kl; s_cl[wid] = n_clip; }
  __syncthreads();
  if (threadIdx.x == 0) {
    double a = 0.0, b = 0.0;
    unsigned long long c = 0;
    for (int w = 0; w < kLossThreads / 32; ++w) { a += s_pg[w]; b += s_kl[w]; c += s_cl[w]; }
    partials[blockIdx.x].loss_pg = a;
    partials[blockIdx.x].loss_kl = b;
    if (c) atomicAdd(&cnt->n_clipped, c);
    __threadfence();
    const unsigned int ticket = atomicAdd(&cnt->ticket, 1u);
    is_last = (ticket == gridDim.x - 1);
  }
  __syncthreads();
  if (!is_last) return;
  __threadfence();
  // final fixed-order sum over block partials (the last block, strided, then shuffle / smem tree)
  double a = 0.0, b = 0.0;
  for (unsigned int i = threadIdx.x; i < gridDim.x; i += kLossThreads) {
    a += partials[i].loss_pg;
    b += partials[i].loss_kl;
  }
  a = warp_sum(a);
  b = warp_sum(b);
  __syncthreads();
  if ((threadIdx.x & 31) == 0) { s_pg[wid] = a; s_kl[wid] = b; }
  __syncthreads();
  if (threadIdx.x == 0) {
    a = 0.0; b = 0.0;
    for (int w = 0; w < kLossThreads / 32; ++w) { a += s_pg[w]; b += s_kl[w]; }
    const double denom = (agg == GC_AGG_SEQ_MEAN) ? fmax(n_kept, 1.0) : fmax(n_scored, 1.0);
    const double pg = a / denom, kl = b / denom;
    out5[0] = (float)(pg + (double)beta * kl);
    out5[1] = (float)pg;
    out5[2] = (float)kl;
    out5[3] = (float)((double)atomicAdd(&cnt->n_clipped, 0ull) / fmax(n_scored, 1.0));
    out5[4] = (float)n_scored;
  }
}

size_t loss_ws_bytes(int64_t T, int32_t R) {
  const int64_t blocks = ceil_div(T > 0 ? T : 1, kLossTile);
  return align_up(sizeof(LossCounters), 256) + align_up((size_t)blocks * sizeof(LossPartial), 256) +
         align_up((size_t)(blocks + 1) * sizeof(int32_t), 256) +
         align_up((size_t)(R > 0 ? R : 1) * sizeof(int32_t), 256);
}

int launch_token_loss(const float* logp, const float* old_logp, const float* ref_logp,
                      const int32_t* targets, const uint8_t* mask, int64_t T,
                      const int32_t* cu_seqlens, int32_t R, const float* adv,
                      float clip_lo, float clip_hi, float beta, int agg, float grad_loss,
                      float* out5, float* g, void* ws, cudaStream_t st) {
  if (T <= 0) {                  // nothing scored: loss and every statistic are 0
    GC_CUDA_TRY(cudaMemsetAsync(out5, 0, 5 * sizeof(float), st));
    return GC_OK;
  }
  const int64_t blocks = ceil_div(T, kLossTile);
  Carver c(ws);
  LossCounters* cnt = c.take<LossCounters>(1);
  LossPartial* partials = c.take<LossPartial>((size_t)blocks);
  int32_t* tile_r = c.take<int32_t>((size_t)blocks + 1);
  int32_t* resp_cnt = c.take<int32_t>((size_t)(R > 0 ? R : 1));
  const int per_response = agg == GC_AGG_SEQ_MEAN ? 1 : 0;
  GC_CUDA_TRY(cudaMemsetAsync(cnt, 0, sizeof(LossCounters), st));
  if (per_response)
    GC_CUDA_TRY(cudaMemsetAsync(resp_cnt, 0, sizeof(int32_t) * (size_t)(R > 0 ? R : 1), st));
  k_loss_tile_ranges<<<(unsigned)ceil_div(blocks + 1, 256), 256, 0, st>>>(cu_seqlens, R, T, blocks,
                                                                          tile_r);
  if (per_response && T >= (int64_t)R * 128)
    k_loss_counts_seq<<<(unsigned)ceil_div((int64_t)R * 32, 256), 256, 0, st>>>(
        targets, mask, cu_seqlens, R, resp_cnt, cnt);
  else
    k_loss_counts<<<(unsigned)blocks, kLossThreads, 0, st>>>(targets, mask, T, cu_seqlens, R, tile_r,
                                                            per_response, resp_cnt, cnt);
  GC_CUDA_TRY(cudaGetLastError());
  k_token_loss<<<(unsigned)blocks, kLossThreads, 0, st>>>(
      logp, old_logp, ref_logp, targets, mask, T, cu_seqlens, R, adv, resp_cnt, tile_r, clip_lo, clip_hi, beta, agg, grad_loss, cnt, partials, out5, g);
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
