// attention.cu -- NEXT-4: the distributed attention of G-Core sec 4.5.
// "we first all-gather the key (K) and value (V) tensors, and then compute attention
// output for the local query (Q) tensor chunk"; "we process only a subset of
// attention heads at a time and overlap KV communication with attention computation".
//
// Two parts:
//   * gc_attention_allgather_kv (host): for each subset of key/value heads, the ranks' K/V shards
//     (this rank's own memory or peer-mapped: CUDA IPC / peer access, NVLink carries the bytes) are
//     gathered by the copy engines into one of two [S, heads, d] buffers on a side stream while the
//     attention kernel works on the previous subset out of the other buffer.
//   * k_attn_fwd: a tcgen05 flash-attention forward for one (128-query tile, query head):
//       S_j = Q K_j^T (UMMA 128x128x16, fp32 in TMEM, two buffers), online softmax by a
//       4-warp group (thread = query row; exp2 domain; the whole 128-column score row is read
//       from TMEM in one round trip), P_j -> bf16 -> 128B-swizzled smem, O += P_j V_j accumulated
//       IN TMEM by the second contraction (V is the MN-major B operand).  The reference maximum of
//       a row is raised lazily -- only when the block's maximum exceeds it by more than 2^8 -- and
//       only then is the row of O rescaled in TMEM (tcgen05.ld / st); P stays <= 2^8, exact in the
//       end because l and O share the reference.  The MMA warp issues S_{j+1} before P_j V_j, so
//       the tensor core computes the next scores while the softmax group works.
//     Masks: per query row an allowed key interval [k_lo, k_hi) -- packed
//     documents, causal, sliding window -- computed once by k_attn_rows; blocks outside the
//     tile's interval are skipped, blocks inside every row's interval take no per-element test.
#include <math.h>
#include <mutex>

#include "tc_gemm.cuh"

namespace gc {
namespace attn {

constexpr int kD = 128;            // head dimension
constexpr int kBQ = 128;           // query rows per CTA
#ifndef GC_ATTN_BK
#define GC_ATTN_BK 64
#endif
constexpr int kBK = GC_ATTN_BK;    // keys per block.  64: 112 KB of shared memory and 256 TMEM columns
                                   // per CTA, so TWO CTAs share an SM and one's softmax (MUFU-bound)
                                   // runs under the other's TMEM round trips, barriers and P stores;
                                   // 128: one CTA per SM (224 KB, 384 columns)
static_assert(kBK == 64 || kBK == 128, "key block");
constexpr int kKB = kBK / 64;      // 64-key k-blocks per block (second contraction)
constexpr int kCH = kBK / 32;      // 32-column TMEM chunks of a score row
constexpr int kCtasPerSM = kBK == 64 ? 2 : 1;
constexpr int kTmemCols = kBK == 64 ? 256 : 512;
constexpr int kThreads = 256;
constexpr int kQBytes = kBQ * kD * 2;        // 32 KB: 128 x 128 bf16 (two 64-wide k-blocks of 16 KB)
constexpr int kKSub = kBK * 128;             // one 64-wide k-block of a K tile: kBK rows x 128 B
constexpr int kKVBytes = kBK * kD * 2;       // a K or V stage
constexpr int kKStages = kBK == 64 ? 3 : 2;  // P lives in tensor memory, so shared memory holds only
constexpr int kVStages = 2;                  // Q and the K / V rings
constexpr int kSmemQ = 0;
constexpr int kSmemK = kSmemQ + kQBytes;
constexpr int kSmemV = kSmemK + kKStages * kKVBytes;
constexpr int kSmemBar = kSmemV + kVStages * kKVBytes;     // tiles, then the barriers
constexpr int kSmemBytes = kSmemBar + 256;                 // (the dynamic smem base is 1024-aligned)
static_assert(kSmemBytes <= (kCtasPerSM == 2 ? 113 : 227) * 1024, "attention shared memory budget");

struct TileMeta { int32_t kb_begin, kb_end, lo_max, hi_min; };

struct Params {
  int64_t S_local, q_off, S;
  int32_t n_q_tiles;
  int32_t h_begin;          // first query head of this launch
  int32_t n_q_heads;        // query heads of this launch
  int32_t grp;              // query heads per key/value head
  float scale2;             // scale * log2(e)
  const int32_t* k_lo;      // [S_local] first allowed key of each query row
  const int32_t* k_hi;      // [S_local] one past the last allowed key
  const TileMeta* meta;     // [n_q_tiles]
  __nv_bfloat16* O;         // [S_local, Hq, d]
  int64_t ldO;              // Hq * d
  float* lse;               // [Hq, S_local] or NULL
};

// ---------------------------------------------------------------------------------------------
// Allowed key interval of every local query row, and per 128-row tile the key blocks to visit.
//   doc(q) from cu_seqlens (global positions; NULL = one document [0, S))
//   causal: k <= q;  window W > 0: q - k < W (causal) or |q - k| < W (not causal)
// ---------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(kBQ)
k_attn_rows(int64_t S_local, int64_t q_off, int64_t S, const int32_t* __restrict__ cu, int32_t n_docs,
            int causal, int32_t window, int32_t* __restrict__ k_lo, int32_t* __restrict__ k_hi,
            TileMeta* __restrict__ meta) {
  const int64_t i = (int64_t)blockIdx.x * kBQ + threadIdx.x;
  int32_t lo = 0, hi = 0;
  if (i < S_local) {
    const int32_t q = (int32_t)(q_off + i);
    int32_t d0 = 0, d1 = (int32_t)S;
    if (cu != nullptr) {                        // largest d with cu[d] <= q
      int a = 0, b = n_docs;
      while (b - a > 1) {
        const int mid = (a + b) >> 1;
        if (cu[mid] <= q) a = mid; else b = mid;
      }
      d0 = cu[a];
      d1 = cu[a + 1];
    }
    lo = d0;
    hi = d1;
    if (causal) hi = min(hi, q + 1);
    if (window > 0) {
      lo = max(lo, q - window + 1);
      if (!causal) hi = min(hi, q + window);
    }
    k_lo[i] = lo;
    k_hi[i] = hi;
  }
  // tile reductions: union of the rows' intervals (blocks to visit), intersection (no-mask blocks)
  __shared__ int32_t s[4][kBQ / 32];
  const bool valid = i < S_local;
  int32_t lo_min = valid ? lo : INT32_MAX, hi_max = valid ? hi : 0;
  int32_t lo_max = valid ? lo : 0, hi_min = valid ? hi : INT32_MAX;
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) {
    lo_min = min(lo_min, __shfl_xor_sync(0xffffffffu, lo_min, o));
    hi_max = max(hi_max, __shfl_xor_sync(0xffffffffu, hi_max, o));
    lo_max = max(lo_max, __shfl_xor_sync(0xffffffffu, lo_max, o));
    hi_min = min(hi_min, __shfl_xor_sync(0xffffffffu, hi_min, o));
  }
  const int w = threadIdx.x >> 5;
  if ((threadIdx.x & 31) == 0) { s[0][w] = lo_min; s[1][w] = hi_max; s[2][w] = lo_max; s[3][w] = hi_min; }
  __syncthreads();
  if (threadIdx.x == 0) {
    for (int k = 1; k < kBQ / 32; ++k) {
      s[0][0] = min(s[0][0], s[0][k]); s[1][0] = max(s[1][0], s[1][k]);
      s[2][0] = max(s[2][0], s[2][k]); s[3][0] = min(s[3][0], s[3][k]);
    }
    TileMeta m;
    m.kb_begin = s[0][0] / kBK;
    m.kb_end = (s[1][0] + kBK - 1) / kBK;
    if (m.kb_end < m.kb_begin) m.kb_end = m.kb_begin;
    m.lo_max = s[2][0];
    m.hi_min = s[3][0];
    meta[blockIdx.x] = m;
  }
}

__device__ __forceinline__ uint32_t pack_bf16x2(float lo, float hi) {
  __nv_bfloat162 v = __floats2bfloat162_rn(lo, hi);
  return *reinterpret_cast<uint32_t*>(&v);
}
// packed fp32 pairs (Blackwell FFMA2 / FADD2): one issue slot for two scores
__device__ __forceinline__ uint64_t pack2(float lo, float hi) {
  uint64_t v;
  asm("mov.b64 %0, {%1, %2};" : "=l"(v) : "f"(lo), "f"(hi));
  return v;
}
__device__ __forceinline__ void unpack2(uint64_t v, float& lo, float& hi) {
  asm("mov.b64 {%0, %1}, %2;" : "=f"(lo), "=f"(hi) : "l"(v));
}
__device__ __forceinline__ uint64_t ffma2(uint64_t a, uint64_t b, uint64_t c) {
  uint64_t d;
  asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(d) : "l"(a), "l"(b), "l"(c));
  return d;
}
__device__ __forceinline__ uint64_t fadd2(uint64_t a, uint64_t b) {
  uint64_t d;
  asm("add.rn.f32x2 %0, %1, %2;" : "=l"(d) : "l"(a), "l"(b));
  return d;
}

__device__ __forceinline__ void st_shared_v4_u32(uint32_t addr, uint32_t a, uint32_t b, uint32_t c,
                                                 uint32_t d) {
  asm volatile("st.shared.v4.b32 [%0], {%1, %2, %3, %4};" ::"r"(addr), "r"(a), "r"(b), "r"(c), "r"(d)
               : "memory");
}

// ---------------------------------------------------------------------------------------------
// One CTA = one (query tile, query head).  Warps: 0 TMA producer, 1 MMA issuer, 2 TMEM allocator,
// 4..7 softmax / output group (thread = query row).
// ---------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(kThreads, kCtasPerSM)
k_attn_fwd(const __grid_constant__ CUtensorMap tmQ, const __grid_constant__ CUtensorMap tmK,
           const __grid_constant__ CUtensorMap tmV, const Params p) {
  extern __shared__ __align__(1024) uint8_t smem_raw[];
  const uint32_t base = ptx::smem_u32(smem_raw);
  if (base & 1023u) __trap();              // the swizzled tiles need a 1024-byte aligned base
  const uint32_t sQ = base + kSmemQ, sK = base + kSmemK, sV = base + kSmemV;
  const uint32_t bar = base + kSmemBar;
  // barriers (8 bytes each)
  const uint32_t q_full = bar;
  auto k_full = [&](int i) { return bar + 8u * (1 + i); };
  auto k_empty = [&](int i) { return bar + 8u * (5 + i); };
  auto v_full = [&](int i) { return bar + 8u * (9 + i); };
  auto v_empty = [&](int i) { return bar + 8u * (13 + i); };
  auto s_full = [&](int i) { return bar + 8u * (17 + i); };
  auto p_full = [&](int i) { return bar + 8u * (19 + i); };
  const uint32_t o_done = bar + 8u * 21;    // one phase per key block: P_j V_j has been accumulated
  const uint32_t tmem_slot = bar + 8u * 23;
  static_assert(kKStages <= 4 && kVStages <= 4, "barrier slots");

  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int head_local = (int)(blockIdx.x % (unsigned)p.n_q_heads);
  const int q_tile = p.n_q_tiles - 1 - (int)(blockIdx.x / (unsigned)p.n_q_heads);   // long tiles first
  const int hq = p.h_begin + head_local;
  const int g_local = head_local / p.grp;            // key/value head inside the gathered buffer
  const TileMeta tm = p.meta[q_tile];
  const int nb = tm.kb_end - tm.kb_begin;

  if (warp == 0 && lane == 0) {
    ptx::prefetch_tmap(&tmQ);
    ptx::prefetch_tmap(&tmK);
    ptx::prefetch_tmap(&tmV);
  }
  if (warp == 1 && lane == 0) {
    ptx::mbar_init(q_full, 1);
    for (int i = 0; i < kKStages; ++i) {
      ptx::mbar_init(k_full(i), 1);
      ptx::mbar_init(k_empty(i), 1);
    }
    for (int i = 0; i < kVStages; ++i) {
      ptx::mbar_init(v_full(i), 1);
      ptx::mbar_init(v_empty(i), 1);
    }
    for (int i = 0; i < 2; ++i) {
      ptx::mbar_init(s_full(i), 1);
      ptx::mbar_init(p_full(i), 4);        // one arrive per softmax warp
    }
    ptx::mbar_init(o_done, 1);
    ptx::fence_barrier_init();
  }
  if (warp == 2) {
    ptx::tmem_alloc<1>(tmem_slot, kTmemCols);
    ptx::tmem_relinquish<1>();
  }
  ptx::tc_fence_before();
  __syncthreads();
  ptx::tc_fence_after();
  uint32_t tmem_base;
  asm volatile("ld.shared.u32 %0, [%1];" : "=r"(tmem_base) : "r"(tmem_slot));
  // TMEM columns: S0 [0,kBK) S1 [kBK,2 kBK) O [2 kBK, 2 kBK + 128).  P_j (bf16, two per column)
  // is written IN PLACE over the first kBK / 2 columns of S_j by the rows' owners and read from
  // there as the A operand of the second contraction: no shared-memory round trip, and the two
  // S buffers double-buffer P for free.  Buffer j & 1 is written again by S_{j+2}, which the MMA
  // thread issues after P_j V_j -- the tensor pipe executes in issue order, so no barrier guards it.
  constexpr uint32_t kOCol = 2u * kBK;

  if (warp == 0) {
    // ===================== TMA producer =====================
    if (lane == 0 && nb > 0) {
      const uint64_t pol_q = ptx::make_l2_policy(ptx::kL2Normal);
      const uint64_t pol_kv = ptx::make_l2_policy(ptx::kL2EvictLast);   // K/V are re-read by every query tile
      const int32_t q_row = q_tile * kBQ;
      const int32_t q_col = hq * kD;
      const int32_t kv_col = g_local * kD;
      ptx::mbar_arrive_expect_tx(q_full, kQBytes);
      ptx::tma_load_2d(sQ, &tmQ, q_col, q_row, q_full, pol_q);
      ptx::tma_load_2d(sQ + 16384, &tmQ, q_col + 64, q_row, q_full, pol_q);
      auto load_k = [&](int j) {
        const int st = j % kKStages;
        ptx::mbar_wait(k_empty(st), (((uint32_t)(j / kKStages)) & 1u) ^ 1u);
        ptx::mbar_arrive_expect_tx(k_full(st), kKVBytes);
        const int32_t row = (tm.kb_begin + j) * kBK;
        const uint32_t dst = sK + st * kKVBytes;
        ptx::tma_load_2d(dst, &tmK, kv_col, row, k_full(st), pol_kv);
        ptx::tma_load_2d(dst + kKSub, &tmK, kv_col + 64, row, k_full(st), pol_kv);
      };
      auto load_v = [&](int j) {
        const int st = j % kVStages;
        ptx::mbar_wait(v_empty(st), (((uint32_t)(j / kVStages)) & 1u) ^ 1u);
        ptx::mbar_arrive_expect_tx(v_full(st), kKVBytes);
        const int32_t row = (tm.kb_begin + j) * kBK;
        const uint32_t dst = sV + st * kKVBytes;
        // MN-major B operand: per 64-key k-block two 64(d) x 64(keys) boxes, 8 KB apart
#pragma unroll
        for (int kb = 0; kb < kKB; ++kb)
#pragma unroll
          for (int nbx = 0; nbx < 2; ++nbx)
            ptx::tma_load_2d(dst + kb * 16384 + nbx * 8192, &tmV, kv_col + 64 * nbx, row + 64 * kb,
                             v_full(st), pol_kv);
      };
      for (int j = 0; j < kKStages - 1 && j < nb; ++j) load_k(j);
      for (int j = 0; j < nb; ++j) {
        if (j + kKStages - 1 < nb) load_k(j + kKStages - 1);
        load_v(j);
      }
    }
  } else if (warp == 1) {
    // ===================== MMA issuer =====================
    if (lane == 0 && nb > 0) {
      constexpr uint32_t idesc_qk = ptx::make_idesc_bf16(kBQ, kBK, false, false);
      constexpr uint32_t idesc_pv = ptx::make_idesc_bf16(kBQ, kD, false, true);
      auto issue_s = [&](int j) {
        const int st = j % kKStages;
        ptx::mbar_wait(k_full(st), ((uint32_t)(j / kKStages)) & 1u);
        ptx::tc_fence_after();
        const uint32_t d_tmem = tmem_base + (uint32_t)((j & 1) * kBK);
#pragma unroll
        for (int kb = 0; kb < 2; ++kb) {            // the two 64-wide halves of head_dim
          const uint64_t adesc = ptx::make_smem_desc(sQ + kb * 16384, false);
          const uint64_t bdesc = ptx::make_smem_desc(sK + st * kKVBytes + kb * kKSub, false);
#pragma unroll
          for (int k = 0; k < 4; ++k)
            ptx::umma_bf16<1>(d_tmem, adesc + (uint64_t)(k * 2), bdesc + (uint64_t)(k * 2), idesc_qk,
                              (uint32_t)(kb | k));
        }
        ptx::umma_commit<1>(k_empty(st));      // the K stage is free once these MMAs have read it
        ptx::umma_commit<1>(s_full(j & 1));
      };
      auto issue_pv = [&](int j) {             // O (+)= P_j V_j, P_j read from tensor memory
        const int st = j % kVStages;
        ptx::mbar_wait(v_full(st), ((uint32_t)(j / kVStages)) & 1u);
        ptx::mbar_wait(p_full(j & 1), ((uint32_t)j >> 1) & 1u);   // P_j written, O rescaled if it had to be
        ptx::tc_fence_after();
        const uint32_t d_tmem = tmem_base + kOCol;
        const uint32_t a_tmem = tmem_base + (uint32_t)((j & 1) * kBK);
#pragma unroll
        for (int kb = 0; kb < kKB; ++kb) {
          const uint64_t bdesc = ptx::make_smem_desc(sV + st * kKVBytes + kb * 16384, true);
#pragma unroll
          for (int k = 0; k < 4; ++k)
            ptx::umma_bf16_ts(d_tmem, a_tmem + (uint32_t)((kb * 4 + k) * 8), bdesc + (uint64_t)(k * 128),
                              idesc_pv, (uint32_t)(j | kb | k));
        }
        ptx::umma_commit<1>(v_empty(st));
        ptx::umma_commit<1>(o_done);
      };
      ptx::mbar_wait(q_full, 0);
      issue_s(0);
      for (int j = 0; j < nb; ++j) {
        if (j + 1 < nb) issue_s(j + 1);        // the next scores run under this block's softmax
        issue_pv(j);
      }
    }
  } else if (warp >= 4) {
    // ===================== softmax / output group =====================
    const int q = warp & 3;
    const int row = q * 32 + lane;
    const int64_t i = (int64_t)q_tile * kBQ + row;           // local query row
    const bool valid = i < p.S_local;
    const int32_t lo = valid ? p.k_lo[i] : 0, hi = valid ? p.k_hi[i] : 0;
    const uint32_t lane_base = tmem_base + ((uint32_t)(q * 32) << 16);
    float m_ref = -1e30f;     // the maximum P, l and O are relative to (log2 domain), raised lazily
    float l_run = 0.f;
    constexpr float kLazy = 8.0f;              // P <= 2^8 between raises of the reference

    for (int j = 0; j < nb; ++j) {
      const int st = j & 1;
      const uint32_t ph = ((uint32_t)j >> 1) & 1u;
      const int32_t k0 = (tm.kb_begin + j) * kBK;
      const bool need_mask = k0 < tm.lo_max || k0 + kBK > tm.hi_min;
      ptx::mbar_wait(s_full(st), ph);
      ptx::tc_fence_after();
      // the whole score row in one TMEM round trip
      uint32_t r[kCH][32];
#pragma unroll
      for (int ch = 0; ch < kCH; ++ch) ptx::tmem_ld_32x32(lane_base + (uint32_t)(st * kBK + ch * 32), r[ch]);
      ptx::tmem_wait_ld();
      if (need_mask) {
#pragma unroll
        for (int ch = 0; ch < kCH; ++ch)
#pragma unroll
          for (int c = 0; c < 32; ++c) {
            const int32_t k = k0 + ch * 32 + c;
            r[ch][c] = (k >= lo && k < hi) ? r[ch][c] : 0xff800000u;      // -inf
          }
      }
      float mx0 = -INFINITY, mx1 = -INFINITY;
#pragma unroll
      for (int ch = 0; ch < kCH; ++ch)
#pragma unroll
        for (int c = 0; c < 32; c += 2) {
          mx0 = fmaxf(mx0, __uint_as_float(r[ch][c]));
          mx1 = fmaxf(mx1, __uint_as_float(r[ch][c + 1]));
        }
      const float mx = fmaxf(mx0, mx1) * p.scale2;
      // lazy reference: raise it only when this block's maximum exceeds it by more than 2^kLazy
      const bool raise = mx > m_ref + kLazy;
      const float m_new = raise ? mx : m_ref;
      const float factor = raise ? ptx::ex2(m_ref - m_new) : 1.0f;
      m_ref = m_new;
      l_run *= factor;
      // p = 2^(s * scale2 - m_ref), row sum, P -> bf16 pairs -> tensor memory, over S_j
      const uint64_t scale_2 = pack2(p.scale2, p.scale2), neg_m2 = pack2(-m_new, -m_new);
      uint64_t sum_a = pack2(0.f, 0.f), sum_b = sum_a;
#pragma unroll
      for (int cp = 0; cp < kCH / 2; ++cp) {
        uint32_t pk[32];
#pragma unroll
        for (int h = 0; h < 2; ++h) {
          const int ch = 2 * cp + h;
#pragma unroll
          for (int c = 0; c < 32; c += 2) {
            float x0, x1;
            unpack2(ffma2(pack2(__uint_as_float(r[ch][c]), __uint_as_float(r[ch][c + 1])), scale_2, neg_m2),
                    x0, x1);
            const float e0 = ptx::ex2(x0), e1 = ptx::ex2(x1);
            if (c & 2) sum_b = fadd2(sum_b, pack2(e0, e1)); else sum_a = fadd2(sum_a, pack2(e0, e1));
            pk[16 * h + (c >> 1)] = pack_bf16x2(e0, e1);
          }
        }
        ptx::tmem_st_32x32(lane_base + (uint32_t)(st * kBK + cp * 32), pk);
      }
      float sum0, sum1;
      unpack2(fadd2(sum_a, sum_b), sum0, sum1);
      l_run += sum0 + sum1;
      // O holds blocks 0 .. j-1 relative to the old reference: wait for P_{j-1} V_{j-1} (long done:
      // it ran under the exponentials above), rescale the rows whose reference was raised
      // (the wait is taken every block: it keeps this thread on o_done's current phase)
      if (j > 0) {
        ptx::mbar_wait(o_done, (uint32_t)(j - 1) & 1u);
        if (__any_sync(0xffffffffu, raise)) {
          ptx::tc_fence_after();
#pragma unroll
          for (int ch = 0; ch < 4; ++ch) {
            uint32_t o[32];
            ptx::tmem_ld_32x32(lane_base + kOCol + (uint32_t)(ch * 32), o);
            ptx::tmem_wait_ld();
#pragma unroll
            for (int c = 0; c < 32; ++c) o[c] = __float_as_uint(__uint_as_float(o[c]) * factor);
            ptx::tmem_st_32x32(lane_base + kOCol + (uint32_t)(ch * 32), o);
          }
        }
      }
      ptx::tmem_wait_st();
      ptx::tc_fence_before();
      __syncwarp();
      if (lane == 0) ptx::mbar_arrive(p_full(st));
    }
    // out = O / l; lse = ln2 * (m + log2 l): read O from TMEM 32 columns at a time and store
    if (nb > 0) {
      ptx::mbar_wait(o_done, (uint32_t)(nb - 1) & 1u);
      ptx::tc_fence_after();
    }
    const float inv = (nb > 0 && l_run > 0.f) ? 1.0f / l_run : 0.f;
#pragma unroll
    for (int ch = 0; ch < 4; ++ch) {
      uint32_t o[32];
      if (nb > 0) {
        ptx::tmem_ld_32x32(lane_base + kOCol + (uint32_t)(ch * 32), o);
        ptx::tmem_wait_ld();
      } else {
#pragma unroll
        for (int c = 0; c < 32; ++c) o[c] = 0u;
      }
      if (valid) {
        uint4* dst = reinterpret_cast<uint4*>(p.O + i * p.ldO + (int64_t)hq * kD + ch * 32);
#pragma unroll
        for (int c = 0; c < 32; c += 8)
          dst[c >> 3] = make_uint4(
              pack_bf16x2(__uint_as_float(o[c]) * inv, __uint_as_float(o[c + 1]) * inv),
              pack_bf16x2(__uint_as_float(o[c + 2]) * inv, __uint_as_float(o[c + 3]) * inv),
              pack_bf16x2(__uint_as_float(o[c + 4]) * inv, __uint_as_float(o[c + 5]) * inv),
              pack_bf16x2(__uint_as_float(o[c + 6]) * inv, __uint_as_float(o[c + 7]) * inv));
      }
    }
    if (valid && p.lse)
      p.lse[(int64_t)hq * p.S_local + i] = l_run > 0.f ? kLn2 * (m_ref + log2f(l_run)) : -INFINITY;
  }

  ptx::tc_fence_before();
  __syncthreads();
  if (warp == 2) ptx::tmem_dealloc<1>(tmem_base, kTmemCols);
}

// ---------------------------------------------------------------------------------------------
// host side
// ---------------------------------------------------------------------------------------------
struct SideCtx {
  cudaStream_t cs = nullptr; cudaEvent_t ev[6] = {}; bool ok = false; bool attr = false;
  std::mutex use;      // held for the whole enqueue of one call: the events are re-recorded per call
};
std::mutex g_mu;
SideCtx g_ctx[64];

int get_side(SideCtx** out) {
  int dev = 0;
  GC_CUDA_TRY(cudaGetDevice(&dev));
  if (dev < 0 || dev >= 64) return GC_ERR_CUDA;
  std::lock_guard<std::mutex> lk(g_mu);
  SideCtx& c = g_ctx[dev];
  if (!c.ok) {
    GC_CUDA_TRY(cudaStreamCreateWithFlags(&c.cs, cudaStreamNonBlocking));
    for (auto& e : c.ev) GC_CUDA_TRY(cudaEventCreateWithFlags(&e, cudaEventDisableTiming));
    GC_CUDA_TRY(cudaFuncSetAttribute(k_attn_fwd, cudaFuncAttributeMaxDynamicSharedMemorySize, kSmemBytes));
    c.ok = true;
  }
  *out = &c;
  return GC_OK;
}

struct Ws { int32_t* k_lo; int32_t* k_hi; TileMeta* meta; void* Kg[2]; void* Vg[2]; };
size_t carve(Carver& c, int64_t S_local, int64_t S, int32_t hs, Ws* w) {
  const size_t n_tiles = (size_t)ceil_div(S_local > 0 ? S_local : 1, kBQ);
  int32_t* lo = c.take<int32_t>(n_tiles * kBQ);
  int32_t* hi = c.take<int32_t>(n_tiles * kBQ);
  TileMeta* m = c.take<TileMeta>(n_tiles);
  const size_t buf = (size_t)(S > 0 ? S : 1) * (size_t)hs * kD * 2;
  void* k0 = c.take<uint8_t>(buf);
  void* k1 = c.take<uint8_t>(buf);
  void* v0 = c.take<uint8_t>(buf);
  void* v1 = c.take<uint8_t>(buf);
  if (w) { w->k_lo = lo; w->k_hi = hi; w->meta = m; w->Kg[0] = k0; w->Kg[1] = k1; w->Vg[0] = v0; w->Vg[1] = v1; }
  return c.off;
}

}  // namespace attn
}  // namespace gc

using namespace gc;

extern "C" {

size_t gc_attention_workspace_bytes(int64_t S_local, int64_t S_total, int32_t heads_per_step) {
  if (S_local < 0 || S_total < 0 || heads_per_step < 1) return 0;
  Carver c(nullptr);
  return attn::carve(c, S_local, S_total, heads_per_step, nullptr) + 256;
}

int gc_attention_allgather_kv(const void* Q, const void* const* K_shards_host,
                              const void* const* V_shards_host, const int64_t* shard_rows_host,
                              int32_t world, int32_t rank, int32_t Hq, int32_t Hkv, int32_t head_dim,
                              const int32_t* cu_seqlens, int32_t n_docs, int causal, int32_t window,
                              float scale, int32_t heads_per_step, void* O, float* lse,
                              void* workspace, size_t workspace_bytes, void* cuda_stream) {
  if (head_dim != attn::kD) return GC_ERR_SHAPE;
  if (world < 1 || world > 64 || rank < 0 || rank >= world) return GC_ERR_ARG;
  if (Hq < 1 || Hkv < 1 || Hq % Hkv != 0 || heads_per_step < 1 || window < 0) return GC_ERR_ARG;
  if (!(scale > 0.f)) return GC_ERR_ARG;
  if (!K_shards_host || !V_shards_host || !shard_rows_host) return GC_ERR_NULL;
  int64_t S = 0, q_off = 0;
  for (int r = 0; r < world; ++r) {
    if (shard_rows_host[r] < 0) return GC_ERR_SHAPE;
    if (r < rank) q_off += shard_rows_host[r];
    S += shard_rows_host[r];
  }
  const int64_t S_local = shard_rows_host[rank];
  if (S >= (1ll << 31) - 256) return GC_ERR_SHAPE;
  if (S_local == 0) return GC_OK;
  if (!Q || !O) return GC_ERR_NULL;
  if (cu_seqlens != nullptr && n_docs < 1) return GC_ERR_ARG;
  for (int r = 0; r < world; ++r) {
    if (shard_rows_host[r] > 0 && (!K_shards_host[r] || !V_shards_host[r])) return GC_ERR_NULL;
    if ((reinterpret_cast<uintptr_t>(K_shards_host[r]) & 15) || (reinterpret_cast<uintptr_t>(V_shards_host[r]) & 15))
      return GC_ERR_ALIGN;
  }
  if ((reinterpret_cast<uintptr_t>(Q) & 15) || (reinterpret_cast<uintptr_t>(O) & 15)) return GC_ERR_ALIGN;
  const int32_t hs = heads_per_step < Hkv ? heads_per_step : Hkv;
  if (!workspace || workspace_bytes < gc_attention_workspace_bytes(S_local, S, hs)) return GC_ERR_WORKSPACE;
  if (reinterpret_cast<uintptr_t>(workspace) & 255) return GC_ERR_ALIGN;
  {
    int dev = 0, major = 0;
    GC_CUDA_TRY(cudaGetDevice(&dev));
    GC_CUDA_TRY(cudaDeviceGetAttribute(&major, cudaDevAttrComputeCapabilityMajor, dev));
    if (major != 10) return GC_ERR_ARCH;
  }
  cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
  attn::SideCtx* cx = nullptr;
  GC_TRY(attn::get_side(&cx));
  // one enqueue at a time per device: two host threads on two streams would otherwise re-record
  // each other's events between a record and the wait that is meant to see it
  std::lock_guard<std::mutex> use_lock(cx->use);
  Carver c(workspace);
  attn::Ws w;
  attn::carve(c, S_local, S, hs, &w);
  const int32_t n_q_tiles = (int32_t)ceil_div(S_local, attn::kBQ);
  const int grp = Hq / Hkv;

  attn::k_attn_rows<<<(unsigned)n_q_tiles, attn::kBQ, 0, st>>>(S_local, q_off, S, cu_seqlens, n_docs,
                                                                causal ? 1 : 0, window, w.k_lo, w.k_hi,
                                                                w.meta);
  GC_CUDA_TRY(cudaGetLastError());

  CUtensorMap tmQ;
  GC_TRY(tc::make_tmap_bf16(&tmQ, Q, (int64_t)Hq * attn::kD, S_local, (int64_t)Hq * attn::kD, 64, attn::kBQ));
  // fork: the gathers may start once earlier work on `st` (a previous call reading the buffers) is done
  GC_CUDA_TRY(cudaEventRecord(cx->ev[0], st));
  GC_CUDA_TRY(cudaStreamWaitEvent(cx->cs, cx->ev[0], 0));
  const size_t src_pitch = (size_t)Hkv * attn::kD * 2;
  const int n_steps = (int)ceil_div(Hkv, hs);
  for (int s = 0; s < n_steps; ++s) {
    const int b = s & 1;
    const int h0 = s * hs;
    const int nh = (Hkv - h0) < hs ? (Hkv - h0) : hs;
    const size_t dst_pitch = (size_t)nh * attn::kD * 2;
    // ---- all-gather of this head subset (copy engines, side stream) ----
    if (s >= 2) GC_CUDA_TRY(cudaStreamWaitEvent(cx->cs, cx->ev[3 + b], 0));   // buffer b consumed
    int64_t pos = 0;
    for (int r = 0; r < world; ++r) {
      const int64_t rows = shard_rows_host[r];
      if (rows == 0) continue;
      GC_CUDA_TRY(cudaMemcpy2DAsync(static_cast<char*>(w.Kg[b]) + (size_t)pos * dst_pitch, dst_pitch,
                                    static_cast<const char*>(K_shards_host[r]) + (size_t)h0 * attn::kD * 2,
                                    src_pitch, dst_pitch, (size_t)rows, cudaMemcpyDeviceToDevice, cx->cs));
      GC_CUDA_TRY(cudaMemcpy2DAsync(static_cast<char*>(w.Vg[b]) + (size_t)pos * dst_pitch, dst_pitch,
                                    static_cast<const char*>(V_shards_host[r]) + (size_t)h0 * attn::kD * 2,
                                    src_pitch, dst_pitch, (size_t)rows, cudaMemcpyDeviceToDevice, cx->cs));
      pos += rows;
    }
    GC_CUDA_TRY(cudaEventRecord(cx->ev[1 + b], cx->cs));
    // ---- attention of this subset's query heads (main stream) ----
    GC_CUDA_TRY(cudaStreamWaitEvent(st, cx->ev[1 + b], 0));
    CUtensorMap tmK, tmV;
    GC_TRY(tc::make_tmap_bf16(&tmK, w.Kg[b], (int64_t)nh * attn::kD, S, (int64_t)nh * attn::kD, 64, attn::kBK));
    GC_TRY(tc::make_tmap_bf16(&tmV, w.Vg[b], (int64_t)nh * attn::kD, S, (int64_t)nh * attn::kD, 64, 64));
    attn::Params p;
    p.S_local = S_local; p.q_off = q_off; p.S = S; p.n_q_tiles = n_q_tiles;
    p.h_begin = h0 * grp; p.n_q_heads = nh * grp; p.grp = grp;
    p.scale2 = scale * kLog2e;
    p.k_lo = w.k_lo; p.k_hi = w.k_hi; p.meta = w.meta;
    p.O = static_cast<__nv_bfloat16*>(O); p.ldO = (int64_t)Hq * attn::kD; p.lse = lse;
    attn::k_attn_fwd<<<(unsigned)(n_q_tiles * p.n_q_heads), attn::kThreads, attn::kSmemBytes, st>>>(tmQ, tmK, tmV, p);
    GC_CUDA_TRY(cudaGetLastError());
    GC_CUDA_TRY(cudaEventRecord(cx->ev[3 + b], st));
  }
  return GC_OK;
}

}  // extern "C"
