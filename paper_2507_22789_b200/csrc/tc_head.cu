// tc_head.cu -- the four dense contractions of the path on the tcgen05 tile engine, each with
// its fused epilogue:
//   a2+a3  forward      S = Hs W^T            -> online (m, s, u, a_y) row statistics, split over V
//   a10    recompute    S = Hs W^T again      -> dS = (g/tau)(onehot - exp(S/tau - lse)), bf16
//   a11    dH           dH = dS W             -> bf16 rows scattered to their original positions
//   a12    dW           dW (+)= dS^T Hs       -> fp32
#include "tc_gemm.cuh"

// Production launch shape: CTA pairs (cta_group::2) in clusters of kPpc pairs (tc_gemm.cuh).
// kPpc = 2 (4-CTA clusters, B stages fetched once per cluster by TMA multicast) is built, tested
// (test_engine_gemm_cluster4) and measured, but is not the default: only 33 clusters of 4 are
// co-resident on the 148 SMs, and same-box A/B on cfg2 gave 79.5 ms (kPpc 2: 132 SMs at 1395 MHz)
// against 78.7 ms (kPpc 1: 148 SMs at 1245 MHz) and 81.0 ms (kPpc 1 restricted to 132 SMs): the
// multicast saves ~2 % energy per flop, less than the 16 idle SMs cost.  Build with -DGC_PPC=2 to
// use it.
#ifndef GC_PPC
#define GC_PPC 1
#endif
constexpr int kPpc = GC_PPC;
// scheduling units = co-resident clusters on a B200 (the launcher queries the real number; the
// planners only need it to size waves): 74 pairs, or 33 clusters of two pairs
constexpr int kUnits = kPpc == 2 ? 33 : 74;

namespace gc {

using tc::Sched;

// ---------------------------------------------------------------------------------------------
// Epilogue a3: online log-softmax statistics in log2 units (a = x * log2(e)/tau).
// A thread owns one row; state lives in registers across the N tiles of an item.
// ---------------------------------------------------------------------------------------------
struct EpiStats {
  static constexpr int kWarpSmem = 0;
  struct Params {
    const int32_t* targets;   // [rows] compact targets
    RowStat* partials;        // [n_split][split_stride]
    int64_t split_stride;
    int64_t V;
    float c;                  // log2(e) / tau
  };
  struct State { float m, s0, s1, u0, u1, ay; int32_t y; };
  static __device__ __forceinline__ void setup(State&, const Params&, uint32_t) {}

  static __device__ __forceinline__ void item_begin(State& st, const Params& p, int64_t row,
                                                    bool valid, int64_t) {
    st.y = valid ? p.targets[row] : -1;
    st.m = -1e30f;
    st.s0 = st.s1 = st.u0 = st.u1 = 0.f;
    st.ay = -INFINITY;
  }
  static __device__ __forceinline__ void tile_prefetch(const Params&, int64_t, bool, int64_t) {}
  static __device__ __forceinline__ void chunk(State& st, const Params& p, int64_t, bool,
                                               int64_t col0, const float (&x)[32]) {
    if (col0 >= p.V) return;
    const bool full = col0 + 32 <= p.V;
    const int nvalid = full ? 32 : (int)(p.V - col0);
    float cm = -INFINITY;
#pragma unroll
    for (int j = 0; j < 32; ++j) cm = (full || j < nvalid) ? fmaxf(cm, x[j]) : cm;
    const float mnew = fmaxf(st.m, cm * p.c);
    const float dm = st.m - mnew;
    const float sc = ptx::ex2(dm);
    st.u0 = (st.u0 + dm * st.s0) * sc;
    st.u1 = (st.u1 + dm * st.s1) * sc;
    st.s0 *= sc;
    st.s1 *= sc;
    st.m = mnew;
#pragma unroll
    for (int j = 0; j < 32; j += 2) {
      const float t0 = fmaf(x[j], p.c, -mnew), t1 = fmaf(x[j + 1], p.c, -mnew);
      float e0 = ptx::ex2(t0), e1 = ptx::ex2(t1);
      if (!full) { e0 = j < nvalid ? e0 : 0.f; e1 = j + 1 < nvalid ? e1 : 0.f; }
      st.s0 += e0;
      st.s1 += e1;
      st.u0 = fmaf(e0, t0, st.u0);
      st.u1 = fmaf(e1, t1, st.u1);
    }
    const uint32_t rel = (uint32_t)((int64_t)st.y - col0);
    if (st.y >= 0 && rel < 32u) {
#pragma unroll
      for (int j = 0; j < 32; ++j) st.ay = (rel == (uint32_t)j) ? x[j] * p.c : st.ay;
    }
  }
  static __device__ __forceinline__ void item_end(State& st, const Params& p, int64_t row,
                                                  bool valid, int64_t c) {
    if (!valid) return;
    RowStat o;
    o.m = st.m;
    o.s = st.s0 + st.s1;
    o.u = st.u0 + st.u1;
    o.ay = st.ay;
    p.partials[c * p.split_stride + row] = o;
  }
  static __device__ __forceinline__ void finish(State&, const Params&) {}
};

// ---------------------------------------------------------------------------------------------
// Epilogue of the verdict-token scoring ("Generative
// rewarding ... represents solution correctness using the LLM's probability distribution over
// tokens"): the same online statistics as EpiStats, with K target ids per row.  Every target logit
// lives in exactly one vocab tile, so the thread that meets it stores it straight to ay[row, k]
// (one writer in the whole grid; the buffer is pre-filled with -inf) instead of carrying it in the
// split-V partials.
// ---------------------------------------------------------------------------------------------
constexpr int kMaxTargets = 8;
struct EpiStatsMulti {
  static constexpr int kWarpSmem = 0;
  struct Params {
    const int32_t* targets;   // [rows, K]
    float* ay;                // [rows, K], log2-scaled target logits
    RowStat* partials;
    int64_t split_stride;
    int64_t V;
    float c;
    int K;
  };
  struct State { float m, s0, s1, u0, u1; int32_t y[kMaxTargets]; int64_t row; };
  static __device__ __forceinline__ void setup(State&, const Params&, uint32_t) {}
  static __device__ __forceinline__ void item_begin(State& st, const Params& p, int64_t row,
                                                    bool valid, int64_t) {
#pragma unroll
    for (int k = 0; k < kMaxTargets; ++k)
      st.y[k] = (valid && k < p.K) ? p.targets[row * p.K + k] : -1;
    st.row = row;
    st.m = -1e30f;
    st.s0 = st.s1 = st.u0 = st.u1 = 0.f;
  }
  static __device__ __forceinline__ void tile_prefetch(const Params&, int64_t, bool, int64_t) {}
  static __device__ __forceinline__ void chunk(State& st, const Params& p, int64_t, bool,
                                               int64_t col0, const float (&x)[32]) {
    if (col0 >= p.V) return;
    const bool full = col0 + 32 <= p.V;
    const int nvalid = full ? 32 : (int)(p.V - col0);
    float cm = -INFINITY;
#pragma unroll
    for (int j = 0; j < 32; ++j) cm = (full || j < nvalid) ? fmaxf(cm, x[j]) : cm;
    const float mnew = fmaxf(st.m, cm * p.c);
    const float dm = st.m - mnew;
    const float sc = ptx::ex2(dm);
    st.u0 = (st.u0 + dm * st.s0) * sc;
    st.u1 = (st.u1 + dm * st.s1) * sc;
    st.s0 *= sc;
    st.s1 *= sc;
    st.m = mnew;
#pragma unroll
    for (int j = 0; j < 32; j += 2) {
      const float t0 = fmaf(x[j], p.c, -mnew), t1 = fmaf(x[j + 1], p.c, -mnew);
      float e0 = ptx::ex2(t0), e1 = ptx::ex2(t1);
      if (!full) { e0 = j < nvalid ? e0 : 0.f; e1 = j + 1 < nvalid ? e1 : 0.f; }
      st.s0 += e0;
      st.s1 += e1;
      st.u0 = fmaf(e0, t0, st.u0);
      st.u1 = fmaf(e1, t1, st.u1);
    }
#pragma unroll
    for (int k = 0; k < kMaxTargets; ++k) {
      const uint32_t rel = (uint32_t)((int64_t)st.y[k] - col0);
      if (st.y[k] >= 0 && rel < 32u && (int64_t)st.y[k] < p.V) {
        float v = 0.f;
#pragma unroll
        for (int j = 0; j < 32; ++j) v = (rel == (uint32_t)j) ? x[j] : v;
        p.ay[st.row * p.K + k] = v * p.c;
      }
    }
  }
  static __device__ __forceinline__ void item_end(State& st, const Params& p, int64_t row,
                                                  bool valid, int64_t c) {
    if (!valid) return;
    RowStat o;
    o.m = st.m;
    o.s = st.s0 + st.s1;
    o.u = st.u0 + st.u1;
    o.ay = -INFINITY;
    p.partials[c * p.split_stride + row] = o;
  }
  static __device__ __forceinline__ void finish(State&, const Params&) {}
};

__device__ __forceinline__ uint32_t pack_bf16x2(float lo, float hi) {
  __nv_bfloat162 v = __floats2bfloat162_rn(lo, hi);
  return *reinterpret_cast<uint32_t*>(&v);
}

// ---------------------------------------------------------------------------------------------
// Epilogue a10: dS[r, v] = (g_r/tau) (1[v = y_r] - 2^(a - lse2)) in bf16; zeros for rows past the
// dynamic row count and for columns >= V (the dW contraction runs over those rows).
// ---------------------------------------------------------------------------------------------
struct EpiDS {
  static constexpr int kWarpSmem = 0;
  struct Params {
    const int32_t* targets;   // chunk-local compact arrays
    const float* lse;
    const float* g;
    __nv_bfloat16* dS;        // [rows_cap, ldS]
    int64_t ldS;
    int64_t V;
    float c;                  // log2(e) / tau
    float inv_tau;
    const int32_t* n_dyn;     // device scalar: dynamic row count of the batch (nullable)
    int64_t row0;             // rows of the batch before this chunk
    int64_t n_static;         // rows of this chunk when n_dyn == NULL
    int64_t cap;              // chunk capacity
  };
  struct State { float lse2, gp; int32_t y; int64_t n_eff; };
  static __device__ __forceinline__ void setup(State& st, const Params& p, uint32_t) {
    int64_t n = p.n_static;
    if (p.n_dyn) {
      n = (int64_t)(*p.n_dyn) - p.row0;
      n = n < 0 ? 0 : (n > p.cap ? p.cap : n);
    }
    st.n_eff = n;
  }

  static __device__ __forceinline__ void item_begin(State& st, const Params& p, int64_t row,
                                                    bool valid, int64_t) {
    st.y = -1; st.lse2 = 0.f; st.gp = 0.f;
    if (valid && row < st.n_eff) {
      st.y = p.targets[row];
      st.gp = p.g[row] * p.inv_tau;
      st.lse2 = p.lse[row] * kLog2e;
      if (st.y < 0) st.gp = 0.f;
    }
  }
  static __device__ __forceinline__ void tile_prefetch(const Params&, int64_t, bool, int64_t) {}
  static __device__ __forceinline__ void chunk(State& st, const Params& p, int64_t row, bool valid,
                                               int64_t col0, const float (&x)[32]) {
    if (!valid || col0 >= p.ldS) return;       // !valid: phantom M tile of an odd cluster item
    float v[32];
    if (st.gp == 0.f) {
#pragma unroll
      for (int j = 0; j < 32; ++j) v[j] = 0.f;
    } else {
      const float ng = -st.gp;
#pragma unroll
      for (int j = 0; j < 32; ++j) v[j] = ng * ptx::ex2(fmaf(x[j], p.c, -st.lse2));
      const uint32_t rel = (uint32_t)((int64_t)st.y - col0);
      if (rel < 32u) {
#pragma unroll
        for (int j = 0; j < 32; ++j) v[j] = (rel == (uint32_t)j) ? v[j] + st.gp : v[j];
      }
      if (col0 + 32 > p.V) {
#pragma unroll
        for (int j = 0; j < 32; ++j) v[j] = (col0 + j < p.V) ? v[j] : 0.f;
      }
    }
    uint4* dst = reinterpret_cast<uint4*>(p.dS + row * p.ldS + col0);
#pragma unroll
    for (int q = 0; q < 4; ++q) {
      if (col0 + 8 * q < p.ldS)     // streaming store: 2 GB per chunk must not evict the H band
        __stcs(dst + q,
               make_uint4(pack_bf16x2(v[8 * q], v[8 * q + 1]), pack_bf16x2(v[8 * q + 2], v[8 * q + 3]),
                          pack_bf16x2(v[8 * q + 4], v[8 * q + 5]), pack_bf16x2(v[8 * q + 6], v[8 * q + 7])));
    }
  }
  static __device__ __forceinline__ void item_end(State&, const Params&, int64_t, bool, int64_t) {}
  static __device__ __forceinline__ void finish(State&, const Params&) {}
};

// ---------------------------------------------------------------------------------------------
// Epilogue a11: store bf16 rows, optionally scattered through rows[] (dH of compacted tokens).
// ---------------------------------------------------------------------------------------------
struct EpiStoreBf16 {
  static constexpr int kWarpSmem = 0;
  struct Params {
    __nv_bfloat16* out;
    int64_t ldo;
    const int32_t* rows;      // nullable; chunk-local
    int64_t row_base;         // used when rows == NULL
    int64_t N;
  };
  struct State { int64_t orow; };
  static __device__ __forceinline__ void setup(State&, const Params&, uint32_t) {}
  static __device__ __forceinline__ void item_begin(State& st, const Params& p, int64_t row,
                                                    bool valid, int64_t) {
    st.orow = valid ? (p.rows ? (int64_t)p.rows[row] : p.row_base + row) : -1;
  }
  static __device__ __forceinline__ void tile_prefetch(const Params&, int64_t, bool, int64_t) {}
  static __device__ __forceinline__ void chunk(State& st, const Params& p, int64_t, bool,
                                               int64_t col0, const float (&x)[32]) {
    if (st.orow < 0 || col0 >= p.N) return;
    uint4* dst = reinterpret_cast<uint4*>(p.out + st.orow * p.ldo + col0);
#pragma unroll
    for (int q = 0; q < 4; ++q) {
      if (col0 + 8 * q < p.N)
        dst[q] = make_uint4(pack_bf16x2(x[8 * q], x[8 * q + 1]), pack_bf16x2(x[8 * q + 2], x[8 * q + 3]),
                            pack_bf16x2(x[8 * q + 4], x[8 * q + 5]), pack_bf16x2(x[8 * q + 6], x[8 * q + 7]));
    }
  }
  static __device__ __forceinline__ void item_end(State&, const Params&, int64_t, bool, int64_t) {}
  static __device__ __forceinline__ void finish(State&, const Params&) {}
};

// ---------------------------------------------------------------------------------------------
// Epilogue a12 (and the debug GEMM): fp32 tile store, or accumulate, through TMA.  Each epilogue
// warp stages its 32 rows x 32 columns (4 KB, 128-byte-swizzled, ONE buffer: 16 KB per CTA, which
// leaves room for a 6th operand stage -- dW waits for operands, not for its stores: measured
// -4.5 % at cfg4, -2 % at cfg2 against 4 buffers and 5 stages) in shared memory
// and one lane issues a bulk tensor store -- or, when accumulating, a bulk tensor REDUCE-ADD, so
// the read-modify-write of dW happens at the L2 and the old values never travel to the SM.  Every
// dW element receives exactly one add per launch and launches are stream-ordered, so the result
// is deterministic.  Rows >= M and columns >= N are clipped by the tensor map.
// (A register read-add-store epilogue was latency-bound: cfg4's accumulating dW launch ran at 27 %
// tensor-pipe activity, profiles/.)
// ---------------------------------------------------------------------------------------------
struct EpiStoreF32 {
  static constexpr int kBufs = 1;                // 4 KB staging buffers per warp (see above)
  static constexpr int kWarpSmem = kBufs * 4096;
  struct alignas(64) Params {
    CUtensorMap tm;           // fp32 [M, N] (row stride ldo), box {32 columns, 32 rows}, swizzle 128B
    int64_t N;
    int accumulate;
  };
  struct State { uint32_t smem; uint32_t buf; };
  static __device__ __forceinline__ void setup(State& st, const Params&, uint32_t warp_smem) {
    st.smem = warp_smem;
    st.buf = 0;
  }
  static __device__ __forceinline__ void item_begin(State&, const Params&, int64_t, bool, int64_t) {}
  static __device__ __forceinline__ void tile_prefetch(const Params&, int64_t, bool, int64_t) {}
  static __device__ __forceinline__ void chunk(State& st, const Params& p, int64_t row, bool,
                                               int64_t col0, const float (&x)[32]) {
    if (col0 >= p.N) return;                       // uniform over the warp
    const int lane = threadIdx.x & 31;
    const uint32_t base = st.smem + st.buf * 4096u;
    st.buf = (st.buf + 1u) % (uint32_t)kBufs;
    // the store issued kBufs chunks ago (same buffer) must have finished reading it
    if (lane == 0) ptx::bulk_wait_group_read<kBufs - 1>();
    __syncwarp();
    const uint32_t rbase = base + (uint32_t)lane * 128u;
#pragma unroll
    for (int q = 0; q < 8; ++q)
      ptx::st_shared_v4(rbase + (uint32_t)((q ^ (lane & 7)) << 4), x[4 * q], x[4 * q + 1],
                        x[4 * q + 2], x[4 * q + 3]);
    ptx::fence_proxy_async_smem();
    __syncwarp();
    if (lane == 0) {
      // `row` is this lane's row = first row of the warp's 32-row slab
      if (p.accumulate) ptx::tma_reduce_add_2d(&p.tm, base, (int32_t)col0, (int32_t)row);
      else ptx::tma_store_2d(&p.tm, base, (int32_t)col0, (int32_t)row);
      ptx::bulk_commit_group();
    }
  }
  static __device__ __forceinline__ void item_end(State&, const Params&, int64_t, bool, int64_t) {}
  static __device__ __forceinline__ void finish(State&, const Params&) {
    if ((threadIdx.x & 31) == 0) ptx::bulk_wait_group_read<0>();
  }
};

static int make_f32_out_tmap(CUtensorMap* m, float* out, int64_t rows, int64_t cols, int64_t ld) {
  tc::PFN_encodeTiled fn = tc::get_encode_fn();
  if (!fn) return GC_ERR_CUDA;
  if ((reinterpret_cast<uintptr_t>(out) & 15) || ((ld * 4) & 15)) return GC_ERR_ALIGN;
  cuuint64_t dims[2] = {(cuuint64_t)cols, (cuuint64_t)rows};
  cuuint64_t strides[1] = {(cuuint64_t)ld * 4};
  cuuint32_t box[2] = {32, 32};
  cuuint32_t estr[2] = {1, 1};
  CUresult r = fn(m, CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 2, out, dims, strides, box, estr,
                  CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B,
                  CU_TENSOR_MAP_L2_PROMOTION_NONE, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
  return r == CUDA_SUCCESS ? GC_OK : GC_ERR_CUDA;
}

// ---------------------------------------------------------------------------------------------
// Epilogue a12 fused with its data-parallel exchange ("one all-reduce (or
// reduce-scatter ...) of fp32 dW"): instead of accumulating into a local dW and calling a
// collective afterwards, every tile is TMA-reduce-added straight into the shard of the rank that
// OWNS its vocab rows -- a peer-mapped buffer reached over NVLink (or this rank's own memory) --
// so the reduce-scatter overlaps the contraction tile by tile and no full-size local dW exists.
// Shard r holds vocab rows [r shard_rows, (r+1) shard_rows); shard_rows % 32 == 0 so that a warp's
// 32-row slab never straddles two owners.  All ranks add into zero-initialised shards; after a
// barrier each rank's shard is the sum over ranks.  (Adds from different ranks arrive in no fixed
// order: across ranks the fp32 sum is reproducible only up to rounding, as with any NCCL ring.)
// ---------------------------------------------------------------------------------------------
constexpr int kMaxShards = 8;
struct EpiReduceScatterF32 {
  static constexpr int kBufs = 1;                // as EpiStoreF32
  static constexpr int kWarpSmem = kBufs * 4096;
  struct alignas(64) Params {
    CUtensorMap tm[kMaxShards];   // shard r: fp32 [rows of shard r, N], box {32, 32}, swizzle 128B
    int64_t N;
    int64_t shard_rows;
    int world;
  };
  struct State { uint32_t smem; uint32_t buf; };
  static __device__ __forceinline__ void setup(State& st, const Params&, uint32_t warp_smem) {
    st.smem = warp_smem;
    st.buf = 0;
  }
  static __device__ __forceinline__ void item_begin(State&, const Params&, int64_t, bool, int64_t) {}
  static __device__ __forceinline__ void tile_prefetch(const Params&, int64_t, bool, int64_t) {}
  static __device__ __forceinline__ void chunk(State& st, const Params& p, int64_t row, bool,
                                               int64_t col0, const float (&x)[32]) {
    if (col0 >= p.N) return;
    const int lane = threadIdx.x & 31;
    const uint32_t base = st.smem + st.buf * 4096u;
    st.buf = (st.buf + 1u) % (uint32_t)kBufs;
    if (lane == 0) ptx::bulk_wait_group_read<kBufs - 1>();
    __syncwarp();
    const uint32_t rbase = base + (uint32_t)lane * 128u;
#pragma unroll
    for (int q = 0; q < 8; ++q)
      ptx::st_shared_v4(rbase + (uint32_t)((q ^ (lane & 7)) << 4), x[4 * q], x[4 * q + 1],
                        x[4 * q + 2], x[4 * q + 3]);
    ptx::fence_proxy_async_smem();
    __syncwarp();
    if (lane == 0) {
      const int64_t owner = row / p.shard_rows;            // `row` = first row of the warp's slab
      if (owner < p.world)
        ptx::tma_reduce_add_2d(&p.tm[owner], base, (int32_t)col0,
                               (int32_t)(row - owner * p.shard_rows));
      ptx::bulk_commit_group();
    }
  }
  static __device__ __forceinline__ void item_end(State&, const Params&, int64_t, bool, int64_t) {}
  static __device__ __forceinline__ void finish(State&, const Params&) {
    if ((threadIdx.x & 31) == 0) ptx::bulk_wait_group_read<0>();
  }
};

// L2 budget of the forward / recompute schedule.  Measured (profiles/): an H band plus the W tiles
// in flight stay resident up to ~50 MB, 60 MB and more thrash (DRAM reads x2.5 .. x7) -- about
// half of the 126 MB, consistent with each die's L2 also holding the lines its SMs fetch from the
// other die.  The W tiles alive at a time are about k (vocab tiles per item) panels: the band's
// pairs reach a given W tile spread over a fraction of an item time.
constexpr int64_t kL2BudgetBytes = 52ll << 20;     // H band + W in flight
constexpr int64_t kL2StreamBytes = 16ll << 20;     // of which W in flight (caps k)
constexpr int64_t kL2ResidentBytes = 40ll << 20;   // resident panels of the dW schedule

// ---------------------------------------------------------------------------------------------
// forward plan: vocab tiles per item k.  Among k <= 16 MB / panel (and >= what the cap of 512
// partial slots per row and 512 MB of partials needs) pick the one whose items balance best over
// the CTA pairs (wave quantisation, SURVEY.md sec 7.2 hard part 5); longer items win ties.
// ---------------------------------------------------------------------------------------------
TcPlan tc_plan_forward(int64_t T, int64_t D, int64_t V) {
  const int P = kUnits;
  const int64_t Mt = ceil_div(T > 0 ? T : 1, 256 * kPpc);      // M extent of an item = kPpc tiles
  const int64_t Nt = ceil_div(V, tc::BN);
  const int64_t panel = 512 * D;
  TcPlan best{(int)Nt, 1, (int)Nt};
  double best_cost = 1e300;
  int64_t max_split = (512ll << 20) / (Mt * 256 * kPpc * (int64_t)sizeof(RowStat));
  if (max_split > 512) max_split = 512;
  if (max_split < 1) max_split = 1;
  int64_t kmin = ceil_div(Nt, max_split);
  if (kmin < 1) kmin = 1;
  int64_t kmax = kL2StreamBytes / panel;
  if (kmax < 2) kmax = 2;
  if (kmax < kmin) kmax = kmin;
  for (int64_t k = kmin; k <= kmax && k <= Nt; ++k) {
    const int64_t C = ceil_div(Nt, k);
    // makespan in tiles (upper bound: every item counted as k tiles) + a charge per item flush
    const double cost = (double)(ceil_div(C * Mt, P) * k) * (1.0 + 0.02 / (double)k);
    if (cost <= best_cost) {
      best_cost = cost;
      best.chunk_vtiles = (int)k;
      best.n_split = (int)C;
    }
  }
  best.n_vtiles = (int)Nt;
  return best;
}

// M tiles per band of the forward / recompute schedule: the band's A panels (m_band x 256 rows x
// D bf16) stay in L2 while the N sweep streams W past; W is re-read once per band.
static int pick_m_band(int64_t D, int k) {
  const int64_t panel = 512 * D;
  int64_t mb = (kL2BudgetBytes - (int64_t)k * panel) / panel;
  mb = mb < 4 ? 4 : (mb > 64 ? 64 : mb);
  return (int)(mb / kPpc);                     // in items (kPpc M tiles each)
}
// N tiles per band of the dW schedule: the band's H panels (k_rows x 256 columns bf16).
static int pick_n_band(int64_t k_rows) {
  int64_t nb = kL2ResidentBytes / (512 * (k_rows > 0 ? k_rows : 1));
  return (int)(nb < 1 ? 1 : nb);
}

// rows of one M band of the forward schedule (host-buffer entry points copy and score H band by band)
int64_t tc_forward_band_rows(int64_t T, int64_t D, int64_t V) {
  const TcPlan pl = tc_plan_forward(T, D, V);
  return (int64_t)pick_m_band(D, pl.chunk_vtiles) * kPpc * 256;
}

size_t tc_fwd_partials_bytes(int64_t T, int64_t D, int64_t V) {
  const TcPlan pl = tc_plan_forward(T, D, V);
  const int64_t cap = ceil_div(T > 0 ? T : 1, 256) * 256;
  return align_up((size_t)pl.n_split * (size_t)cap * sizeof(RowStat), 256);
}


// every launch shape of the engine (debug GEMM only; the path's kernels use fixed shapes)
template <class Epi, bool A_MN, bool B_MN>
static int launch_any(int cg, bool dual_n, int ppc, const CUtensorMap& a, const CUtensorMap& b,
                      const Sched& s, const typename Epi::Params& ep, cudaStream_t st) {
  if (cg == 1) {
    if (dual_n || ppc != 1) return GC_ERR_ARG;
    return tc::launch_tc_gemm<1, A_MN, B_MN, Epi>(a, b, s, ep, st);
  }
  if (ppc == 2)
    return dual_n ? tc::launch_tc_gemm<2, A_MN, B_MN, Epi, 2, 2>(a, b, s, ep, st)
                  : tc::launch_tc_gemm<2, A_MN, B_MN, Epi, 1, 2>(a, b, s, ep, st);
  return dual_n ? tc::launch_tc_gemm<2, A_MN, B_MN, Epi, 2, 1>(a, b, s, ep, st)
                : tc::launch_tc_gemm<2, A_MN, B_MN, Epi, 1, 1>(a, b, s, ep, st);
}

// K-major B operand: rows of one TMA box = the share of the 256-row tile one CTA fetches
static int b_box_rows(int cg, int ppc) { return tc::BN / cg / ppc; }

// MN-major operand [K, rows]: the slab form (one TMA box per stage, tc_gemm.cuh) when rows is a
// multiple of 64 -- `padded_rows` >= rows says how far the buffer's rows really extend (zero-filled
// padding, e.g. the dS chunk buffer) -- else one 2-D box per 64-wide slab.  *slab tells which.
static int make_mn_tmap(CUtensorMap* m, const void* base, int64_t rows, int64_t padded_rows, int64_t K,
                        int64_t ld, int slabs, bool allow_slab, int* slab) {
  const int64_t r64 = ceil_div(rows, 64) * 64;
  *slab = (allow_slab && r64 <= padded_rows) ? 1 : 0;
  if (*slab) return tc::make_slab_tmap_bf16(m, base, r64, K, ld, slabs);
  return tc::make_operand_tmap(m, base, rows, K, ld, true, 0);
}

static Sched make_sched(int64_t M, int64_t N, int64_t K) {
  Sched s;
  s.M = M; s.N = N; s.K = K;
  s.n_dyn = nullptr; s.dyn_row0 = 0; s.dyn_cap = 0; s.dyn_dim = 0; s.dyn_round = 1;
  s.chunk_ntiles = 1; s.c_major = 0; s.m_band = 0; s.n_band = 0; s.skip_empty_k = 0; s.n_major = 0;
  s.counter = nullptr; s.lockstep = nullptr; s.a_slab = 0; s.b_slab = 0; s.a_hint = ptx::kL2Normal; s.b_hint = ptx::kL2Normal;
  return s;
}

int tc_forward_stats(const void* H, int64_t ldH, const void* W, int64_t ldW, int64_t T, int64_t D,
                     int64_t V, float tau, const int32_t* targets_c, const int32_t* n_rows_dev,
                     RowStat* partials, uint32_t* counter, cudaStream_t st) {
  CUtensorMap ta, tb;
  GC_TRY(tc::make_operand_tmap(&ta, H, T, D, ldH, false, tc::BM_CTA));
  GC_TRY(tc::make_operand_tmap(&tb, W, V, D, ldW, false, b_box_rows(2, kPpc)));
  const TcPlan pl = tc_plan_forward(T, D, V);
  Sched s = make_sched(T, V, D);
  s.chunk_ntiles = pl.chunk_vtiles;
  s.c_major = 1;
  s.m_band = pick_m_band(D, pl.chunk_vtiles);
  s.counter = counter;
  s.a_hint = ptx::kL2EvictLast;     // the band's H tiles are re-read for every vocab tile
  s.b_hint = ptx::kL2Normal;        // W streams past, shared by the band's pairs a few us apart
  if (n_rows_dev) { s.n_dyn = n_rows_dev; s.dyn_dim = 1; s.dyn_row0 = 0; s.dyn_cap = T; }
  EpiStats::Params ep;
  ep.targets = targets_c;
  ep.partials = partials;
  ep.split_stride = ceil_div(T, 256) * 256;
  ep.V = V;
  ep.c = kLog2e / tau;
  KernelTimer kt(GC_KERNEL_FWD_STATS, st);
  return tc::launch_tc_gemm<2, false, false, EpiStats, 1, kPpc>(ta, tb, s, ep, st);
}

int tc_forward_stats_multi(const void* H, int64_t ldH, const void* W, int64_t ldW, int64_t T,
                           int64_t D, int64_t V, float tau, const int32_t* targets, int K,
                           float* ay, RowStat* partials, uint32_t* counter, cudaStream_t st) {
  if (K < 1 || K > kMaxTargets) return GC_ERR_ARG;
  CUtensorMap ta, tb;
  GC_TRY(tc::make_operand_tmap(&ta, H, T, D, ldH, false, tc::BM_CTA));
  GC_TRY(tc::make_operand_tmap(&tb, W, V, D, ldW, false, b_box_rows(2, kPpc)));
  const TcPlan pl = tc_plan_forward(T, D, V);
  Sched s = make_sched(T, V, D);
  s.chunk_ntiles = pl.chunk_vtiles;
  s.c_major = 1;
  s.m_band = pick_m_band(D, pl.chunk_vtiles);
  s.counter = counter;
  s.a_hint = ptx::kL2EvictLast;
  s.b_hint = ptx::kL2Normal;
  EpiStatsMulti::Params ep;
  ep.targets = targets;
  ep.ay = ay;
  ep.partials = partials;
  ep.split_stride = ceil_div(T, 256) * 256;
  ep.V = V;
  ep.c = kLog2e / tau;
  ep.K = K;
  KernelTimer kt(GC_KERNEL_FWD_STATS, st);
  return tc::launch_tc_gemm<2, false, false, EpiStatsMulti, 1, kPpc>(ta, tb, s, ep, st);
}

int tc_recompute_ds(const void* H, int64_t ldH, const void* W, int64_t ldW, int64_t rows_cap,
                    int64_t n_static, int64_t D, int64_t V, float tau, const int32_t* targets_c,
                    const float* lse_c, const float* g_c, const int32_t* n_rows_dev, int64_t row0,
                    void* dS, int64_t ldS, uint32_t* counter, cudaStream_t st) {
  const int64_t h_rows = n_rows_dev ? rows_cap : n_static;   // rows behind the H pointer
  CUtensorMap ta, tb;
  GC_TRY(tc::make_operand_tmap(&ta, H, h_rows, D, ldH, false, tc::BM_CTA));
  GC_TRY(tc::make_operand_tmap(&tb, W, V, D, ldW, false, b_box_rows(2, kPpc)));
  // rows up to the next multiple of 256 past the valid count are written as zeros: the dW
  // contraction runs over them (rows_cap is a multiple of 256)
  Sched s = make_sched(ceil_div(h_rows, 256) * 256, V, D);
  const TcPlan pl = tc_plan_forward(rows_cap, D, V);
  s.chunk_ntiles = pl.chunk_vtiles;
  s.c_major = 1;
  s.m_band = pick_m_band(D, pl.chunk_vtiles);
  s.counter = counter;
  s.a_hint = ptx::kL2EvictLast;
  s.b_hint = ptx::kL2Normal;
  if (n_rows_dev) {
    s.n_dyn = n_rows_dev; s.dyn_dim = 1; s.dyn_row0 = row0; s.dyn_cap = rows_cap; s.dyn_round = 256;
  }
  EpiDS::Params ep;
  ep.n_dyn = n_rows_dev;
  ep.row0 = row0;
  ep.n_static = n_static;
  ep.cap = rows_cap;
  ep.targets = targets_c;
  ep.lse = lse_c;
  ep.g = g_c;
  ep.dS = static_cast<__nv_bfloat16*>(dS);
  ep.ldS = ldS;
  ep.V = V;
  ep.c = kLog2e / tau;
  ep.inv_tau = 1.0f / tau;
  KernelTimer kt(GC_KERNEL_RECOMPUTE_DS, st);
  return tc::launch_tc_gemm<2, false, false, EpiDS, 1, kPpc>(ta, tb, s, ep, st);
}

int tc_dh(const void* dS, int64_t ldS, int64_t rows_cap, int64_t n_static, const void* W,
          int64_t ldW, int64_t D, int64_t V, const int32_t* rows, const int32_t* n_rows_dev,
          int64_t row0, void* dH, int64_t lddH, uint32_t* counter, cudaStream_t st) {
  CUtensorMap ta, tb;
  GC_TRY(tc::make_operand_tmap(&ta, dS, rows_cap, V, ldS, false, tc::BM_CTA));
  int b_slab = 0;                            // W as 64-wide slabs: one TMA box per B sub-tile and stage
  GC_TRY(make_mn_tmap(&tb, W, D, D, V, ldW, tc::BN / 2 / 64, kPpc == 1, &b_slab));
  Sched s = make_sched(n_rows_dev ? rows_cap : n_static, D, V);
  s.b_slab = b_slab;
  // K-lockstep kernel: all pairs stream V together -- static schedule, paced through `counter`
  // (tc::kLockRing zeroed words; NULL: unpaced)
  static_assert(kDhLockWords == tc::kLockRing, "dH progress ring size");
  s.lockstep = counter;
  // Every wave of 74 tiles streams, over the whole of K = V, the dS rows of the M tiles it covers and
  // the W columns of the N tiles it covers; the operand whose tiles a wave covers COMPLETELY is
  // re-read by every wave.  Order the tiles so that this is the smaller one: dS chunk (rows x V)
  // against W (V x D), i.e. N-major iff rows < D (cfg4: 4096 rows < D = 8192: W, 4.2 GB, is then
  // read once per launch instead of once per wave).
  s.n_major = rows_cap < D ? 1 : 0;
  if (n_rows_dev) { s.n_dyn = n_rows_dev; s.dyn_dim = 1; s.dyn_row0 = row0; s.dyn_cap = rows_cap; }
  EpiStoreBf16::Params ep;
  ep.out = static_cast<__nv_bfloat16*>(dH);
  ep.ldo = lddH;
  ep.rows = rows;
  ep.row_base = row0;
  ep.N = D;
  KernelTimer kt(GC_KERNEL_DH, st);
  // K = V is ~2000 k-blocks per tile: 256 x 512 dual-N tiles (tc_gemm.cuh, Cfg)
  return tc::launch_tc_gemm<2, false, true, EpiStoreBf16, 2, kPpc>(ta, tb, s, ep, st);
}

int tc_dw(const void* dS, int64_t ldS, int64_t rows_cap, int64_t n_static, const void* Hs,
          int64_t ldH, int64_t D, int64_t V, const int32_t* n_rows_dev, int64_t row0, float* dW,
          int64_t lddW, int accumulate, uint32_t* counter, cudaStream_t st) {
  const int64_t k_rows = n_rows_dev ? rows_cap : n_static;
  CUtensorMap ta, tb;
  // both operands MN-major; in slab form (one TMA box per operand and stage instead of two) when
  // their row counts allow: dS is padded with zero columns up to ldS = ceil(V / 64) 64
  int a_slab = 0, b_slab = 0;
  GC_TRY(make_mn_tmap(&ta, dS, V, ldS, rows_cap, ldS, tc::BM_CTA / 64, true, &a_slab));
  GC_TRY(make_mn_tmap(&tb, Hs, D, D, k_rows, ldH, tc::BN / 2 / 64, kPpc == 1, &b_slab));
  Sched s = make_sched(V, D, k_rows);
  s.a_slab = a_slab;
  s.b_slab = b_slab;
  // items (D band, vocab tile, D tile in band): the band's H panels stay in L2, the D tiles of a
  // vocab tile run together and share its dS^T panel, which streams past once per band
  s.counter = counter;
  s.a_hint = ptx::kL2Normal;
  s.b_hint = ptx::kL2EvictLast;
  s.n_band = pick_n_band(k_rows);
  s.skip_empty_k = accumulate ? 1 : 0;
  if (n_rows_dev) { s.n_dyn = n_rows_dev; s.dyn_dim = 2; s.dyn_row0 = row0; s.dyn_cap = rows_cap; }
  EpiStoreF32::Params ep;
  GC_TRY(make_f32_out_tmap(&ep.tm, dW, V, D, lddW));
  ep.N = D;
  ep.accumulate = accumulate;
  KernelTimer kt(GC_KERNEL_DW, st);
  return tc::launch_tc_gemm<2, true, true, EpiStoreF32, 1, kPpc>(ta, tb, s, ep, st);
}

int tc_dw_reduce_scatter(const void* dS, int64_t ldS, int64_t rows_cap, int64_t n_static,
                         const void* Hs, int64_t ldH, int64_t D, int64_t V,
                         const int32_t* n_rows_dev, int64_t row0, float* const* shards, int world,
                         int64_t shard_rows, int64_t ld_shard, uint32_t* counter, cudaStream_t st) {
  if (world < 1 || world > kMaxShards || shard_rows <= 0 || shard_rows % 32 != 0) return GC_ERR_ARG;
  if (shard_rows * world < V) return GC_ERR_SHAPE;
  const int64_t k_rows = n_rows_dev ? rows_cap : n_static;
  CUtensorMap ta, tb;
  int a_slab = 0, b_slab = 0;
  GC_TRY(make_mn_tmap(&ta, dS, V, ldS, rows_cap, ldS, tc::BM_CTA / 64, true, &a_slab));
  GC_TRY(make_mn_tmap(&tb, Hs, D, D, k_rows, ldH, tc::BN / 2 / 64, kPpc == 1, &b_slab));
  Sched s = make_sched(V, D, k_rows);
  s.a_slab = a_slab;
  s.b_slab = b_slab;
  s.counter = counter;
  s.a_hint = ptx::kL2Normal;
  s.b_hint = ptx::kL2EvictLast;
  s.n_band = pick_n_band(k_rows);
  s.skip_empty_k = 1;                               // every launch adds: an empty chunk adds nothing
  if (n_rows_dev) { s.n_dyn = n_rows_dev; s.dyn_dim = 2; s.dyn_row0 = row0; s.dyn_cap = rows_cap; }
  EpiReduceScatterF32::Params ep;
  for (int r = 0; r < kMaxShards; ++r) {
    const int rr = r < world ? r : 0;
    int64_t rows = V - (int64_t)rr * shard_rows;
    rows = rows > shard_rows ? shard_rows : rows;
    if (rows < 1) rows = 1;                         // an owner past the end of V is never addressed
    if (!shards[rr]) return GC_ERR_NULL;
    GC_TRY(make_f32_out_tmap(&ep.tm[r], shards[rr], rows, D, ld_shard));
  }
  ep.N = D;
  ep.shard_rows = shard_rows;
  ep.world = world;
  KernelTimer kt(GC_KERNEL_DW, st);
  return tc::launch_tc_gemm<2, true, true, EpiReduceScatterF32, 1, kPpc>(ta, tb, s, ep, st);
}

// one counter and one K-lockstep progress ring for the debug GEMM (not safe for concurrent debug
// calls on different streams)
__device__ uint32_t g_debug_counter;
__device__ uint32_t g_debug_lockstep[tc::kLockRing];

// dH tile waves of a chunk of `rows` rows (api.cu's chunk picker): items of kPpc x (256 x 512) tiles
// over the scheduling units; a last wave that is at most half full costs half a wave.
double tc_dh_waves(int64_t rows, int64_t D) {
  const int64_t items = ceil_div(rows, 256 * kPpc) * ceil_div(D, 512);
  const int64_t r = items % kUnits;
  return (double)(items / kUnits) + (r == 0 ? 0.0 : (2 * r <= kUnits ? 0.5 : 1.0));
}

int tc_debug_gemm(const void* A, int64_t lda, int a_mn, const void* B, int64_t ldb, int b_mn,
                  float* C, int64_t ldc, int64_t M, int64_t N, int64_t K, int accumulate,
                  int cta_group, int dynamic_schedule, int dual_n, int cluster4, int c_major,
                  int m_band, int chunk_ntiles, int n_band, cudaStream_t st) {
  if (cta_group != 1 && cta_group != 2) return GC_ERR_ARG;
  if (c_major < 0 || c_major > 2 || m_band < 0 || chunk_ntiles < 0 || n_band < 0) return GC_ERR_ARG;
  if (c_major && n_band) return GC_ERR_ARG;          // the item orders exclude each other
  if ((dual_n || cluster4) && cta_group != 2) return GC_ERR_ARG;
  const int ppc = cluster4 ? 2 : 1;
  if (N % 4 != 0) return GC_ERR_SHAPE;
  CUtensorMap ta, tb;
  // MN-major operands take the slab form whenever their extent is a multiple of 64 (as the path's
  // kernels do), the per-slab 2-D boxes otherwise
  int a_slab = 0, b_slab = 0;
  if (a_mn) GC_TRY(make_mn_tmap(&ta, A, M, M, K, lda, tc::BM_CTA / 64, true, &a_slab));
  else GC_TRY(tc::make_operand_tmap(&ta, A, M, K, lda, false, tc::BM_CTA));
  if (b_mn) GC_TRY(make_mn_tmap(&tb, B, N, N, K, ldb, tc::BN / cta_group / 64, ppc == 1, &b_slab));
  else GC_TRY(tc::make_operand_tmap(&tb, B, N, K, ldb, false, b_box_rows(cta_group, ppc)));
  Sched s = make_sched(M, N, K);
  s.a_slab = a_slab;
  s.b_slab = b_slab;
  // the item orders of the path's kernels (forward / recompute: c_major + m_band + chunk_ntiles;
  // dW: n_band), reachable here at any size
  s.c_major = c_major == 1 ? 1 : 0;
  s.n_major = c_major == 2 ? 1 : 0;                  // c_major = 2: plain order, N-major (dH)
  s.m_band = m_band;
  s.chunk_ntiles = chunk_ntiles > 0 ? chunk_ntiles : 1;
  s.n_band = n_band;
  if (dynamic_schedule) {
    void* ctr = nullptr;
    GC_CUDA_TRY(cudaGetSymbolAddress(&ctr, g_debug_counter));
    GC_CUDA_TRY(cudaMemsetAsync(ctr, 0, sizeof(uint32_t), st));
    s.counter = static_cast<uint32_t*>(ctr);
  }
  if (dual_n && !dynamic_schedule && c_major != 1) {
    // the static dual-N launch is dH's: paced like it (K-lockstep window, tc_gemm.cuh)
    void* ls = nullptr;
    GC_CUDA_TRY(cudaGetSymbolAddress(&ls, g_debug_lockstep));
    GC_CUDA_TRY(cudaMemsetAsync(ls, 0, sizeof(uint32_t) * tc::kLockRing, st));
    s.lockstep = static_cast<uint32_t*>(ls);
  }
  EpiStoreF32::Params ep;
  GC_TRY(make_f32_out_tmap(&ep.tm, C, M, N, ldc));
  ep.N = N;
  ep.accumulate = accumulate;
  const bool d2 = dual_n != 0;
  if (!a_mn && !b_mn) return launch_any<EpiStoreF32, false, false>(cta_group, d2, ppc, ta, tb, s, ep, st);
  if (!a_mn && b_mn) return launch_any<EpiStoreF32, false, true>(cta_group, d2, ppc, ta, tb, s, ep, st);
  if (a_mn && !b_mn) return launch_any<EpiStoreF32, true, false>(cta_group, d2, ppc, ta, tb, s, ep, st);
  return launch_any<EpiStoreF32, true, true>(cta_group, d2, ppc, ta, tb, s, ep, st);
}

}  // namespace gc
