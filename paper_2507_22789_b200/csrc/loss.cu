// loss.cu -- a8 + a9: the per-token clipped-ratio loss with k3 KL, its
// reduction, and g_t = d loss / d logp_t, in ONE cooperative launch (no memsets, no helper
// kernels).
//   rho = e^{logp-old}; s = min(rho A, clip(rho) A); d = ref - logp; k3 = e^d - d - 1
//   l = -s + beta k3;   dl/dlogp = -[rho A <= clip(rho) A] rho A + beta (1 - e^d)
// Weights: token-mean w_t = m_t / max(sum m, 1);  seq-mean w_t = m_t / (R_kept max(cnt_r, 1)).
//
// g_t needs the normaliser before it can be written, so the kernel has phases separated by grid
// barriers (cooperative launch: every block is resident):
//   phase 0  first response of every 1024-token tile (one binary search per tile) and the zeroing
//            of the ticket / the per-response counts
//   phase 1  integer counts: scored tokens, and for seq-mean the scored tokens per response and
//            the number of responses that have any; per-block partials, no float atomics.  The
//            scored flags of each thread's 8 tokens are kept as one byte of a T/8-byte bitmap in
//            the workspace, so that phase 2 does not read targets and mask a second time (21.25
//            bytes of DRAM traffic per token instead of 26; the bitmap mostly stays in L2)
//   phase 2  persistent blocks walk the tiles: a thread takes 8 consecutive tokens (two 16-byte
//            loads per array), the tile's slice of cu_seqlens, advantages and per-response weights
//            is staged in shared memory, fp32 math with e^x as one FMUL + one MUFU.EX2, 8 terms
//            summed in fp32 and everything above that in fp64 in a fixed order; the last block to
//            finish (integer ticket) adds the per-block partials in index order.
// Same inputs give bit-identical outputs on the same device (the grid size is a function of T and
// the device only).
#include <atomic>
#include <cooperative_groups.h>

#include "common.cuh"

namespace cg = cooperative_groups;

namespace gc {

namespace {

constexpr int kLossThreads = 128;
constexpr int kLossBlocksPerSM = 8;
constexpr int kLossBatch = 4;                        // tiles per block iteration of the count phase
constexpr int kLossTok = 8;                          // consecutive tokens per thread
constexpr int kLossTile = kLossThreads * kLossTok;   // tokens per tile
constexpr int kCuSmem = 512 + 8;                     // responses of a tile staged in shared memory
                                                     // (more: the tile reads them from global memory)
constexpr int kLossMaxBlocks = 2048;                 // upper bound of the persistent grid

struct LossHead { unsigned int ticket; unsigned int pad[3]; };
struct LossBlockCnt { unsigned long long n_scored; unsigned int n_kept; unsigned int pad; };
struct LossPartial { double pg, kl; unsigned long long n_clip; unsigned long long pad; };

template <typename T>
__device__ __forceinline__ T warp_sum(T v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
  return v;
}

// e^x as one multiply and one MUFU.EX2 (relative error ~2^-22; exact 1 at x = 0, which keeps the
// identities rho = 1 for logp = old and k3 = 0 for logp = ref exact)
__device__ __forceinline__ float fast_exp(float x) {
  float y;
  asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x * kLog2e));
  return y;
}

// largest r in [lo, hi) with cu[r] <= t, given cu[lo] <= t < cu[hi]
template <typename P>
__device__ __forceinline__ int find_response(P cu, int lo, int hi, int32_t t) {
  while (hi - lo > 1) {
    const int mid = (lo + hi) >> 1;
    if (cu[mid] <= t) lo = mid; else hi = mid;
  }
  return lo;
}

// 8 mask bytes of tokens t0 .. t0+7 (t0 a multiple of 8) as two 32-bit words: one 8-byte load
// when the mask pointer is 8-byte aligned, else two 4-byte loads (the API requires 4-byte alignment)
__device__ __forceinline__ uint2 load_mask8(const uint8_t* __restrict__ mask, int64_t t0) {
  if (mask == nullptr) return make_uint2(0x01010101u, 0x01010101u);
  if ((reinterpret_cast<uintptr_t>(mask) & 7) == 0)
    return *reinterpret_cast<const uint2*>(mask + t0);
  return make_uint2(*reinterpret_cast<const unsigned int*>(mask + t0),
                    *reinterpret_cast<const unsigned int*>(mask + t0 + 4));
}
__device__ __forceinline__ bool mask_byte(uint2 m, int i) {      // i is a compile-time constant
  return (((i < 4) ? m.x : m.y) & (0xffu << (8 * (i & 3)))) != 0u;
}

// scored flags (bit i = token t0 + i) of up to 8 tokens; whole = all 8 inside [0, T)
__device__ __forceinline__ unsigned int scored8(const int32_t* __restrict__ targets,
                                                const uint8_t* __restrict__ mask, int64_t t0,
                                                int64_t T, bool whole) {
  unsigned int bits = 0;
  if (whole) {
    const int4 c0 = *reinterpret_cast<const int4*>(targets + t0);
    const int4 c1 = *reinterpret_cast<const int4*>(targets + t0 + 4);
    const uint2 mk = load_mask8(mask, t0);
    const int32_t y[8] = {c0.x, c0.y, c0.z, c0.w, c1.x, c1.y, c1.z, c1.w};
#pragma unroll
    for (int i = 0; i < 8; ++i) bits |= (y[i] >= 0 && mask_byte(mk, i)) ? (1u << i) : 0u;
  } else {
    for (int i = 0; i < 8; ++i) {
      const int64_t t = t0 + i;
      if (t < T && targets[t] >= 0 && (mask == nullptr || mask[t] != 0)) bits |= 1u << i;
    }
  }
  return bits;
}

// The responses of one tile: slice cu[r0 .. r1+1] with the advantages and (seq-mean) weights of
// responses r0 .. r1, from shared memory when the slice fits, else from global memory.
template <bool SMEM>
struct RespView {
  const int32_t* cu; const float* adv; const int32_t* cnt;     // global arrays
  const int32_t* s_cu; const float* s_adv; const float* s_w;   // staged slice (entry i = r0 + i)
  int r0;
  __device__ __forceinline__ int32_t cu_at(int r) const { return SMEM ? s_cu[r - r0] : cu[r]; }
  __device__ __forceinline__ float adv_at(int r) const { return SMEM ? s_adv[r - r0] : adv[r]; }
  __device__ __forceinline__ float w_at(int r) const {
    return SMEM ? s_w[r - r0] : 1.0f / (float)max(cnt[r], 1);
  }
};

struct Acc { float pg, kl; unsigned int n_clip; };
struct TokConst { float lo_c, hi_c, beta; };

// one token: its terms go to (a_pg, a_kl, n_clip) and g only if it is scored -- by selects, not by
// zero weights: inf / NaN at an unscored position must not reach the sums
template <int AGG>
__device__ __forceinline__ float token_term(float lp, float ol, float rf, bool scored, float A,
                                            float w, float gs, const TokConst& k, float& a_pg,
                                            float& a_kl, unsigned int& n_clip) {
  const float rho = fast_exp(lp - ol);
  const float s1 = rho * A;
  const float s2 = fminf(fmaxf(rho, k.lo_c), k.hi_c) * A;
  const bool unclipped = s1 <= s2;
  const float sm = fminf(s1, s2);
  const float d = rf - lp;
  const float ed = fast_exp(d);
  const float k3 = ed - d - 1.0f;
  if (AGG == GC_AGG_SEQ_MEAN) {
    a_pg -= scored ? sm * w : 0.0f;
    a_kl += scored ? k3 * w : 0.0f;
  } else {
    a_pg -= scored ? sm : 0.0f;
    a_kl += scored ? k3 : 0.0f;
  }
  n_clip += (scored && !unclipped) ? 1u : 0u;
  return scored ? gs * ((unclipped ? -s1 : 0.0f) + fmaf(-k.beta, ed, k.beta)) : 0.0f;
}

// One thread's 8 tokens.  WHOLE: vector loads / stores, every token inside [0, T).
template <int AGG, bool SMEM, bool WHOLE>
__device__ __forceinline__ void tokens8(int64_t T, int32_t R, int64_t t0, const RespView<SMEM>& rv,
                                        int r1, const TokConst& k, float gs_tok, float gs_seq,
                                        float* __restrict__ g, const float (&lp)[8],
                                        const float (&ol)[8], const float (&rf)[8],
                                        unsigned int sc /* bit i: token t0 + i is scored */,
                                        Acc& acc) {
  // response of the first token: binary search in the tile's slice
  const int32_t tq = (int32_t)t0;
  int lo = rv.r0, hi = r1 + 1;
  while (hi - lo > 1) {
    const int mid = (lo + hi) >> 1;
    if (rv.cu_at(mid) <= tq) lo = mid; else hi = mid;
  }
  int r = lo;
  int32_t r_end = rv.cu_at(r + 1);
  float A = rv.adv_at(r);
  float w = 1.0f, gs = gs_tok;
  if (AGG == GC_AGG_SEQ_MEAN) { w = rv.w_at(r); gs = gs_seq * w; }
  float gout[8];
  float a_pg = 0.f, a_kl = 0.f;
  // Boundary handling.  c = index of the first token past this response (>= 8: none inside the 8
  // tokens).  With at most one boundary inside, the tokens take (A, w, gs) of the first or the
  // second response by selects -- no per-token branch; two or more boundaries inside 8 tokens
  // (responses shorter than 8 tokens) and partial tiles take the generic forward walk.
  const int c = r_end - tq;
  bool generic = !WHOLE;
  float A1 = A, w1 = w, gs1 = gs;
  if (WHOLE && c < 8 && r + 1 < R) {
    int r2 = r;
    int32_t e2 = r_end;
    do { ++r2; e2 = rv.cu_at(r2 + 1); } while (tq + c >= e2 && r2 + 1 < R);   // skip empty responses
    generic = tq + 7 >= e2 && r2 + 1 < R;
    A1 = rv.adv_at(r2);
    if (AGG == GC_AGG_SEQ_MEAN) { w1 = rv.w_at(r2); gs1 = gs_seq * w1; }
  }
  if (!generic) {
#pragma unroll
    for (int i = 0; i < 8; ++i) {
      const bool second = i >= c;
      gout[i] = token_term<AGG>(lp[i], ol[i], rf[i], (sc >> i) & 1u, second ? A1 : A,
                                second ? w1 : w, second ? gs1 : gs, k, a_pg, a_kl, acc.n_clip);
    }
  } else {
#pragma unroll
    for (int i = 0; i < 8; ++i) {
      const int32_t t = tq + i;
      if (t >= r_end && r + 1 < R) {
        do { ++r; r_end = rv.cu_at(r + 1); } while (t >= r_end && r + 1 < R);
        A = rv.adv_at(r);
        if (AGG == GC_AGG_SEQ_MEAN) { w = rv.w_at(r); gs = gs_seq * w; }
      }
      const bool scored = ((sc >> i) & 1u) && t < r_end;     // the bits already hold t < T
      gout[i] = token_term<AGG>(lp[i], ol[i], rf[i], scored, A, w, gs, k, a_pg, a_kl, acc.n_clip);
    }
  }
  acc.pg = a_pg;
  acc.kl = a_kl;
  if (g) {
    if (WHOLE) {
      *reinterpret_cast<float4*>(g + t0) = make_float4(gout[0], gout[1], gout[2], gout[3]);
      *reinterpret_cast<float4*>(g + t0 + 4) = make_float4(gout[4], gout[5], gout[6], gout[7]);
    } else {
      for (int i = 0; i < 8; ++i)
        if (t0 + i < T) g[t0 + i] = gout[i];
    }
  }
}

template <int AGG>
__global__ void __launch_bounds__(kLossThreads, kLossBlocksPerSM)
k_grpo_loss(const float* __restrict__ logp, const float* __restrict__ old_logp,
            const float* __restrict__ ref_logp, const int32_t* __restrict__ targets,
            const uint8_t* __restrict__ mask, int64_t T, const int32_t* __restrict__ cu, int32_t R,
            const float* __restrict__ adv, float clip_lo, float clip_hi, float beta,
            float grad_loss, LossHead* __restrict__ head,
            LossBlockCnt* __restrict__ blk_cnt, LossPartial* __restrict__ partials,
            int32_t* __restrict__ tile_r, int32_t* __restrict__ resp_cnt,
            uint8_t* sc_bits /* [tiles * kLossThreads]: written in phase 1, read in phase 2 */,
            float* __restrict__ out5, float* __restrict__ g) {
  cg::grid_group grid = cg::this_grid();
  // the tile's slice, double-buffered so that a tile costs one block barrier (the buffer written
  // for tile k + 2 was last read for tile k, which every thread finished before barrier k + 1)
  __shared__ int32_t s_cu[AGG == GC_AGG_SEQ_MEAN ? kLossBatch : 2][kCuSmem];
  __shared__ float s_adv[2][kCuSmem];
  __shared__ float s_w[2][AGG == GC_AGG_SEQ_MEAN ? kCuSmem : 1];
  __shared__ double s_red[2][kLossThreads / 32];
  __shared__ unsigned long long s_redu[2][kLossThreads / 32];
  __shared__ bool is_last;

  const int tid = threadIdx.x, wid = tid >> 5, lane = tid & 31;
  const int64_t ntiles = (T + kLossTile - 1) / kLossTile;
  const int64_t gtid = (int64_t)blockIdx.x * kLossThreads + tid;
  const int64_t gthreads = (int64_t)gridDim.x * kLossThreads;

  // ---------------- phase 0: tile -> first response; zeroing ----------------
  // tile b spans responses tile_r[b] .. tile_r[b+1] (the response of the next tile's first token
  // bounds the response of this tile's last token); the sentinel entry is the last response
  for (int64_t b = gtid; b <= ntiles; b += gthreads)
    tile_r[b] = b < ntiles ? find_response(cu, 0, R, (int32_t)(b * kLossTile)) : (R > 0 ? R - 1 : 0);
  if (gtid == 0) head->ticket = 0u;
  if constexpr (AGG == GC_AGG_SEQ_MEAN) {
    for (int64_t i = gtid; i < R; i += gthreads) resp_cnt[i] = 0;
    grid.sync();                         // the counts below need tile_r and the zeroed resp_cnt
  }

  // ---------------- phase 1: integer counts ----------------
  // Batches of kLossBatch consecutive tiles per block iteration: the loads, the staging and the
  // searches of the batch's tiles are independent and overlap (a tile alone is one dependent
  // chain tile_r -> cu slice -> search of ~2 us, which 5 bytes per token cannot amortise).
  unsigned long long n_sc = 0;
  unsigned int n_kp = 0;
  for (int64_t tb = (int64_t)blockIdx.x * kLossBatch; tb < ntiles; tb += (int64_t)gridDim.x * kLossBatch) {
    unsigned int bits[kLossBatch];
#pragma unroll
    for (int j = 0; j < kLossBatch; ++j) {
      const int64_t tile0 = (tb + j) * kLossTile;
      const int64_t t0 = tile0 + (int64_t)tid * kLossTok;
      bits[j] = t0 < T ? scored8(targets, mask, t0, T, tile0 + kLossTile <= T) : 0u;
      if (tb + j < ntiles) sc_bits[(tb + j) * kLossThreads + tid] = (uint8_t)bits[j];
    }
    if constexpr (AGG != GC_AGG_SEQ_MEAN) {
#pragma unroll
      for (int j = 0; j < kLossBatch; ++j) n_sc += __popc(bits[j]);
    } else {
      // Scored tokens per response: run lengths per thread over the tile's staged slice of
      // cu_seqlens.  A run that ends inside the thread's 8 tokens is added with an integer
      // atomicAdd; the thread's last run is first summed over the consecutive lanes of the warp
      // that end in the same response (responses are contiguous, so these lanes are too: a
      // segmented sum from one inclusive warp scan), so a long response costs one atomic per
      // warp and 16-token responses one per lane pair.  Integer atomics only (no return value
      // needed): order-independent.  Kept responses are counted from resp_cnt after a barrier.
      int r0[kLossBatch], r1[kLossBatch];
#pragma unroll
      for (int j = 0; j < kLossBatch; ++j) {
        const bool in = tb + j < ntiles;
        r0[j] = in ? tile_r[tb + j] : 0;
        r1[j] = in ? tile_r[tb + j + 1] : -1;
      }
      __syncthreads();                     // the previous batch's readers are done
#pragma unroll
      for (int j = 0; j < kLossBatch; ++j) {
        const int n = r1[j] - r0[j] + 2;
        if (n <= kCuSmem)
          for (int i = tid; i < n; i += kLossThreads) s_cu[j][i] = cu[r0[j] + i];
      }
      __syncthreads();
#pragma unroll
      for (int j = 0; j < kLossBatch; ++j) {
        const int64_t t0 = (tb + j) * kLossTile + (int64_t)tid * kLossTok;
        const bool fits = r1[j] - r0[j] + 2 <= kCuSmem;
        int last_r = -1 - lane;          // lanes past T: each its own (ignored) segment
        unsigned int last_run = 0;
        if (t0 < T) {
          const int32_t* cv = fits ? s_cu[j] - r0[j] : cu;    // cv[r] = cu[r] for r0 <= r <= r1 + 1
          int r = find_response(cv, r0[j], r1[j] + 1, (int32_t)t0);
          int32_t r_end = cv[r + 1];
          if ((int32_t)t0 + 7 < r_end) {
            last_run = __popc(bits[j]);  // all 8 tokens in one response
          } else {
            unsigned int run = 0;
            for (int i = 0; i < kLossTok; ++i) {
              const int32_t t = (int32_t)t0 + i;
              if (t >= r_end && r + 1 < R) {
                if (run) { atomicAdd(resp_cnt + r, (int)run); n_sc += run; run = 0; }
                do { ++r; r_end = cv[r + 1]; } while (t >= r_end && r + 1 < R);
              }
              run += (((bits[j] >> i) & 1u) && t < r_end) ? 1u : 0u;
            }
            last_run = run;
          }
          last_r = r;
        }
        // segmented sum over lanes with equal last_r: inclusive scan, total = P[end] - P[start-1]
        unsigned int P = last_run;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
          const unsigned int v = __shfl_up_sync(0xffffffffu, P, o);
          P += lane >= o ? v : 0u;
        }
        const int prev_r = __shfl_up_sync(0xffffffffu, last_r, 1);
        const unsigned int heads = __ballot_sync(0xffffffffu, lane == 0 || prev_r != last_r);
        const unsigned int above = heads & ~((2u << lane) - 1u);            // heads after this lane
        const int end = above ? __ffs(above) - 2 : 31;                      // last lane of the segment
        const unsigned int p_end = __shfl_sync(0xffffffffu, P, end);
        const bool is_head = (heads >> lane) & 1u;
        const unsigned int tot = p_end - (P - last_run);                    // valid on the head lane
        if (is_head && last_r >= 0 && tot) {
          atomicAdd(resp_cnt + last_r, (int)tot);    // result unused: a fire-and-forget RED
          n_sc += tot;
        }
      }
    }
  }
  if constexpr (AGG == GC_AGG_SEQ_MEAN) {
    grid.sync();                          // every response's count is complete
    for (int64_t i = gtid; i < R; i += gthreads) n_kp += resp_cnt[i] > 0 ? 1u : 0u;
  }
  n_sc = warp_sum(n_sc);
  n_kp = warp_sum(n_kp);
  __syncthreads();
  if (lane == 0) { s_redu[0][wid] = n_sc; s_redu[1][wid] = n_kp; }
  __syncthreads();
  if (tid == 0) {
    unsigned long long a = 0, k = 0;
    for (int w = 0; w < kLossThreads / 32; ++w) { a += s_redu[0][w]; k += s_redu[1][w]; }
    blk_cnt[blockIdx.x].n_scored = a;
    blk_cnt[blockIdx.x].n_kept = (unsigned int)k;
  }
  grid.sync();

  // totals (integers: any order gives the same sum)
  {
    unsigned long long a = 0, k = 0;
    for (unsigned int i = tid; i < gridDim.x; i += kLossThreads) { a += blk_cnt[i].n_scored; k += blk_cnt[i].n_kept; }
    a = warp_sum(a);
    k = warp_sum(k);
    __syncthreads();
    if (lane == 0) { s_redu[0][wid] = a; s_redu[1][wid] = k; }
    __syncthreads();
    a = 0; k = 0;
    for (int w = 0; w < kLossThreads / 32; ++w) { a += s_redu[0][w]; k += s_redu[1][w]; }
    n_sc = a;
    n_kp = (unsigned int)k;
    __syncthreads();
  }
  const double n_scored = (double)n_sc, n_kept = (double)n_kp;
  const float gs_tok = grad_loss / (float)fmax(n_scored, 1.0);
  const float gs_seq = grad_loss / (float)fmax(n_kept, 1.0);
  const TokConst kc{1.0f - clip_lo, 1.0f + clip_hi, beta};

  // ---------------- phase 2: per-token terms and g ----------------
  double d_pg = 0.0, d_kl = 0.0;
  unsigned long long d_clip = 0;
  int buf = 0;
  for (int64_t tile = blockIdx.x; tile < ntiles; tile += gridDim.x, buf ^= 1) {
    const int64_t tile0 = tile * kLossTile;
    const bool whole = tile0 + kLossTile <= T;
    const int64_t t0 = tile0 + (int64_t)tid * kLossTok;
    // this thread's loads first: their DRAM latency overlaps the staging of the slice
    float lp[8], ol[8], rf[8];
    // scored flags from phase 1 (plain global store there, grid barrier in between: read through L2)
    const unsigned int sc = __ldcg(sc_bits + tile * kLossThreads + tid);
    if (whole) {
      const float4 a0 = *reinterpret_cast<const float4*>(logp + t0);
      const float4 a1 = *reinterpret_cast<const float4*>(logp + t0 + 4);
      const float4 b0 = *reinterpret_cast<const float4*>(old_logp + t0);
      const float4 b1 = *reinterpret_cast<const float4*>(old_logp + t0 + 4);
      float4 d0 = a0, d1 = a1;
      if (ref_logp) {
        d0 = *reinterpret_cast<const float4*>(ref_logp + t0);
        d1 = *reinterpret_cast<const float4*>(ref_logp + t0 + 4);
      }
      lp[0] = a0.x; lp[1] = a0.y; lp[2] = a0.z; lp[3] = a0.w;
      lp[4] = a1.x; lp[5] = a1.y; lp[6] = a1.z; lp[7] = a1.w;
      ol[0] = b0.x; ol[1] = b0.y; ol[2] = b0.z; ol[3] = b0.w;
      ol[4] = b1.x; ol[5] = b1.y; ol[6] = b1.z; ol[7] = b1.w;
      rf[0] = d0.x; rf[1] = d0.y; rf[2] = d0.z; rf[3] = d0.w;
      rf[4] = d1.x; rf[5] = d1.y; rf[6] = d1.z; rf[7] = d1.w;
    } else {
      for (int i = 0; i < 8; ++i) {
        const int64_t t = t0 + i;
        const bool in = t < T;
        lp[i] = in ? logp[t] : 0.f;
        ol[i] = in ? old_logp[t] : 0.f;
        rf[i] = in ? (ref_logp ? ref_logp[t] : lp[i]) : 0.f;
      }
    }
    // stage the tile's slice of cu_seqlens / advantages / weights
    const int r0 = tile_r[tile], r1 = tile_r[tile + 1];
    const int n = r1 - r0 + 2;
    const bool fits = n <= kCuSmem;
    if (fits) {
      for (int i = tid; i < n; i += kLossThreads) {
        s_cu[buf][i] = cu[r0 + i];
        if (i < n - 1) {
          s_adv[buf][i] = adv[r0 + i];
          if constexpr (AGG == GC_AGG_SEQ_MEAN) s_w[buf][i] = 1.0f / (float)max(resp_cnt[r0 + i], 1);
        }
      }
    }
    __syncthreads();
    Acc acc{0.f, 0.f, 0u};
    if (t0 < T) {
      if (fits) {
        const RespView<true> rv{cu, adv, resp_cnt, s_cu[buf], s_adv[buf], s_w[buf], r0};
        if (whole)
          tokens8<AGG, true, true>(T, R, t0, rv, r1, kc, gs_tok, gs_seq, g, lp, ol, rf, sc, acc);
        else
          tokens8<AGG, true, false>(T, R, t0, rv, r1, kc, gs_tok, gs_seq, g, lp, ol, rf, sc, acc);
      } else {
        const RespView<false> rv{cu, adv, resp_cnt, nullptr, nullptr, nullptr, r0};
        tokens8<AGG, false, false>(T, R, t0, rv, r1, kc, gs_tok, gs_seq, g, lp, ol, rf, sc, acc);
      }
    }
    d_pg += (double)acc.pg;                // 8 terms in fp32, everything above in fp64
    d_kl += (double)acc.kl;
    d_clip += acc.n_clip;
  }

  // block reduction in fixed order, then the last block adds the block partials in index order
  d_pg = warp_sum(d_pg);
  d_kl = warp_sum(d_kl);
  d_clip = warp_sum(d_clip);
  __syncthreads();
  if (lane == 0) { s_red[0][wid] = d_pg; s_red[1][wid] = d_kl; s_redu[0][wid] = d_clip; }
  __syncthreads();
  if (tid == 0) {
    double a = 0.0, b = 0.0;
    unsigned long long c = 0;
    for (int w = 0; w < kLossThreads / 32; ++w) { a += s_red[0][w]; b += s_red[1][w]; c += s_redu[0][w]; }
    partials[blockIdx.x].pg = a;
    partials[blockIdx.x].kl = b;
    partials[blockIdx.x].n_clip = c;
    __threadfence();
    is_last = atomicAdd(&head->ticket, 1u) == gridDim.x - 1;
  }
  __syncthreads();
  if (!is_last) return;
  __threadfence();
  double a = 0.0, b = 0.0;
  unsigned long long c = 0;
  for (unsigned int i = tid; i < gridDim.x; i += kLossThreads) {
    a += __ldcg(&partials[i].pg);
    b += __ldcg(&partials[i].kl);
    c += __ldcg(&partials[i].n_clip);
  }
  a = warp_sum(a);
  b = warp_sum(b);
  c = warp_sum(c);
  __syncthreads();
  if (lane == 0) { s_red[0][wid] = a; s_red[1][wid] = b; s_redu[0][wid] = c; }
  __syncthreads();
  if (tid == 0) {
    a = 0.0; b = 0.0; c = 0;
    for (int w = 0; w < kLossThreads / 32; ++w) { a += s_red[0][w]; b += s_red[1][w]; c += s_redu[0][w]; }
    const double denom = (AGG == GC_AGG_SEQ_MEAN) ? fmax(n_kept, 1.0) : fmax(n_scored, 1.0);
    const double pg = a / denom, kl = b / denom;
    out5[0] = (float)(pg + (double)beta * kl);
    out5[1] = (float)pg;
    out5[2] = (float)kl;
    out5[3] = (float)((double)c / fmax(n_scored, 1.0));
    out5[4] = (float)n_scored;
  }
}

// resident blocks of the cooperative grid, per device (write-once, idempotent, atomically published)
// (AGG is a template parameter so that each kernel instantiation has its own cache: the two
// function pointers have the same type)
template <int AGG>
int loss_max_blocks(int* out) {
  auto kern = k_grpo_loss<AGG>;
  static std::atomic<int> by_dev[64];
  int dev = 0;
  GC_CUDA_TRY(cudaGetDevice(&dev));
  if (dev < 0 || dev >= 64) return GC_ERR_CUDA;
  int n = by_dev[dev].load(std::memory_order_acquire);
  if (n == 0) {
    int per_sm = 0, sms = 0;
    GC_CUDA_TRY(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, kern, kLossThreads, 0));
    GC_CUDA_TRY(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
    if (per_sm > kLossBlocksPerSM) per_sm = kLossBlocksPerSM;
    n = per_sm * sms;
    if (n < 1) return GC_ERR_CUDA;
    if (n > kLossMaxBlocks) n = kLossMaxBlocks;
    by_dev[dev].store(n, std::memory_order_release);
  }
  *out = n;
  return GC_OK;
}

}  // namespace

size_t loss_ws_bytes(int64_t T, int32_t R) {
  const int64_t tiles = ceil_div(T > 0 ? T : 1, kLossTile);
  return align_up(sizeof(LossHead), 256) + align_up(sizeof(LossBlockCnt) * kLossMaxBlocks, 256) +
         align_up(sizeof(LossPartial) * kLossMaxBlocks, 256) +
         align_up((size_t)(tiles + 1) * sizeof(int32_t), 256) +
         align_up((size_t)(R > 0 ? R : 1) * sizeof(int32_t), 256) +
         align_up((size_t)tiles * kLossThreads, 256);          // scored-bits bitmap, T/8 bytes
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
  const int64_t tiles = ceil_div(T, kLossTile);
  Carver c(ws);
  LossHead* head = c.take<LossHead>(1);
  LossBlockCnt* blk_cnt = c.take<LossBlockCnt>(kLossMaxBlocks);
  LossPartial* partials = c.take<LossPartial>(kLossMaxBlocks);
  int32_t* tile_r = c.take<int32_t>((size_t)tiles + 1);
  int32_t* resp_cnt = c.take<int32_t>((size_t)(R > 0 ? R : 1));
  uint8_t* sc_bits = c.take<uint8_t>((size_t)tiles * kLossThreads);
  void* args[] = {&logp, &old_logp, &ref_logp, &targets, &mask, &T, &cu_seqlens, &R, &adv, &clip_lo,
                  &clip_hi, &beta, &grad_loss, &head, &blk_cnt, &partials, &tile_r,
                  &resp_cnt, &sc_bits, &out5, &g};
  int max_blocks = 0;
  const void* kern = nullptr;
  if (agg == GC_AGG_SEQ_MEAN) {
    GC_TRY(loss_max_blocks<GC_AGG_SEQ_MEAN>(&max_blocks));
    kern = reinterpret_cast<const void*>(k_grpo_loss<GC_AGG_SEQ_MEAN>);
  } else {
    GC_TRY(loss_max_blocks<GC_AGG_TOKEN_MEAN>(&max_blocks));
    kern = reinterpret_cast<const void*>(k_grpo_loss<GC_AGG_TOKEN_MEAN>);
  }
  // grid: a function of T and the device only (reruns are bit-identical)
  const int64_t blocks = tiles < max_blocks ? tiles : max_blocks;
  GC_CUDA_TRY(cudaLaunchCooperativeKernel(kern, dim3((unsigned)blocks), dim3(kLossThreads), args, 0, st));
  return GC_OK;
}

}  // namespace gc
