// tc_gemm.cuh -- the tcgen05 tile engine: a persistent, warp-specialised bf16 GEMM main loop
// (TMA -> 128B-swizzled smem ring -> tcgen05.mma -> double-buffered TMEM accumulators ->
// tcgen05.ld epilogue) shared by the four dense contractions of the path
// (SURVEY.md sec 8(a) rows a2/a3, a10, a11, a12).  What differs per use is the operand
// major-ness and the epilogue functor (tc_head.cu).
//
// Tile: UMMA 128*CG x 256 x 16, BK = 64 (one 128-byte swizzle row of bf16).  CG = 2 pairs two
// SMs (cta_group::2): each CTA stages its own 128 rows of A and its own 128 of the 256 B rows,
// the leader CTA issues the MMAs for both, each CTA's TMEM holds its 128 accumulator rows.
// Warps: 0 = TMA producer, 1 = MMA issuer (leader CTA only), 2 = TMEM allocator,
// 4..7 = epilogue (thread = one accumulator row, 32 fp32 columns per tcgen05.ld).
#pragma once
#include <atomic>
#include "common.cuh"
#include "tc_ptx.cuh"

namespace gc {
namespace tc {

constexpr int BK = 64;
constexpr int BN = 256;
constexpr int BM_CTA = 128;
constexpr int kThreads = 256;
constexpr int kTmemCols = 512;
constexpr int kABytes = BM_CTA * BK * 2;   // 16 KB

// NSUB = 256-wide N sub-tiles per item step (1 or 2).  NSUB = 2 ("dual-N", CG = 2 only): both TMEM
// accumulators belong to one 256 x 512 output tile whose two halves share every A stage, which
// cuts the L2 -> smem operand traffic per flop by a quarter; the epilogue then cannot overlap
// the next tile's MMAs, so it is for contractions with a very long K (dH: K = V).
// kEpiSmem = staging bytes the epilogue functor wants per CTA; the operand ring takes the stages
// that fit in what is left of the 227 KB (7 x 32 KB with no staging, 6 with the fp32 TMA-store
// epilogue's 16 KB, 4 x 48 KB for dual-N).
template <int CG, int NSUB = 1, int kEpiSmem = 0> struct Cfg {
  static_assert(NSUB == 1 || (NSUB == 2 && CG == 2), "dual-N needs the CTA pair");
  static constexpr int kBRows = BN / CG;                 // B rows of one sub-tile staged by one CTA
  static constexpr int kBBytes = kBRows * BK * 2;
  static constexpr int kStageBytes = kABytes + NSUB * kBBytes;  // 32 / 48 KB (CG=2), 48 KB (CG=1)
  static constexpr int kBarBytes = 1024;   // barriers + item ring (keeps what follows 1024-aligned)
  static constexpr int kFit = (227 * 1024 - 1024 /*align slack*/ - kBarBytes - kEpiSmem) / kStageBytes;
  static constexpr int kStages = kFit > 8 ? 8 : kFit;
  static_assert(kStages >= 2, "operand ring too shallow");
  static constexpr int kSmemBase = kStages * kStageBytes + 1024 + kBarBytes;
  static constexpr int kSmemBytes = kSmemBase + kEpiSmem;
};

// Work schedule.  An item is (M tile, run of N tiles).  Items are handed out in index order to
// whichever CTA pair is free (one atomicAdd per item by the leader CTA's producer lane, published
// to the other roles and the peer CTA through a 4-slot smem ring): per-item time jitter (~4 %,
// measured) otherwise accumulates as a random walk, pairs that share a tile drift rounds apart and
// re-fetch it from DRAM.  With a NULL counter pair p takes items p, p+P, ... (static).
struct Sched {
  int64_t M, N, K;        // static extents of the problem
  const int32_t* n_dyn;   // device scalar: dynamic row count of the whole batch (nullable)
  int64_t dyn_row0;       // rows of the batch that precede this launch's chunk
  int64_t dyn_cap;        // chunk capacity in rows
  int dyn_dim;            // 0: none; 1: M = clamp(*n_dyn - row0, 0, cap); 2: same for K
  int dyn_round;          // the dynamic extent is rounded up to a multiple of this (>= 1)
  uint32_t* counter;      // device word, 0 at launch: items are claimed with atomicAdd in the order
                          // pairs become free (dynamic).  NULL: pair p takes items p, p+P, ... (static)
  int a_hint, b_hint;     // L2 eviction priority of the A / B tile loads (ptx::kL2*)
  int chunk_ntiles;       // N tiles per item
  int c_major;            // 1: items ordered (M band, N chunk, M tile in band); 0: (M tile, N tile)
  int m_band;             // c_major: M tiles per band.  The ~74 items in flight then touch only
                          // m_band A tiles (kept in L2 across the whole N sweep) and 74/m_band
                          // N chunks, instead of every A tile of the problem (L2 thrash).
  int n_band;             // c_major == 0 and n_band > 0: items ordered (N band, M tile, N tile in
                          // band): the band's B panels stay in L2 while the A panels stream past
  int skip_empty_k;       // 1: a launch whose K extent resolves to 0 does nothing (accumulating
                          // epilogues: adding zero)
  int n_major;            // plain order only: 1: items ordered (N tile, M tile) -- a wave of pairs
                          // then covers every M tile and few N tiles, so the A operand is what gets
                          // re-read per wave; 0: (M tile, N tile), B is re-read per wave.  Pick the
                          // order that re-reads the SMALLER operand (K-lockstep kernels: dH).
  int a_slab, b_slab;     // MN-major operand whose tensor map is the 3-D slab form (make_operand_tmap):
                          // the stage's 64-wide slabs come in ONE TMA box instead of one per slab
  uint32_t* lockstep;     // static schedule, NSUB == 2 only (nullable): kLockRing zeroed device words.
                          // The pairs of a wave stream the same K range of both operands; left alone
                          // they drift apart by more k-blocks than the L2 holds and every pair
                          // fetches its operands from DRAM.  With this set, a pair announces every
                          // kLockSeg-th k-block it starts loading and does not start segment g + 1
                          // before EVERY pair has started segment g: the wave's loads stay within
                          // 2 * kLockSeg + ring depth k-blocks of one another.  Measured (cfg4 /
                          // cfg2 dH launch): DRAM reads 27.2 -> 13.4 GB / 12.6 -> 6.5 GB, L2 hit rate
                          // 70 -> 81 %, launch -5 % alone, whole step -1.5 % (same box).
};
constexpr int kLockSeg = 16;    // k-blocks per progress segment (measured, cfg2 / cfg4 dH: 8, 16 and 32
                                // give the same DRAM traffic, 64 starts to leak; 16 and 32 are fastest)
constexpr int kLockSlack = 1;   // a pair starts segment g + kLockSlack only when all have started g
constexpr int kLockRing = 32;   // counter slots (a pair is never more than 2 segments from another)

__device__ __forceinline__ void resolve_dims(const Sched& s, int64_t& M, int64_t& K) {
  M = s.M;
  K = s.K;
  if (s.dyn_dim != 0) {
    int64_t n = (int64_t)(*s.n_dyn) - s.dyn_row0;
    n = n < 0 ? 0 : (n > s.dyn_cap ? s.dyn_cap : n);
    n = (n + s.dyn_round - 1) / s.dyn_round * s.dyn_round;
    if (s.dyn_dim == 1) M = M < n ? M : n;
    else K = K < n ? K : n;
  }
}

struct Item { int64_t m_tile, n0, n1, c; int half; };   // half: dual-N tail, see k_tc_gemm

// Item index -> tile coordinates.  Every role of every CTA calls this once per item -- the MMA
// lane before it can issue the item's first MMA -- so the arithmetic is 32-bit (tile counts and
// item indices are far below 2^31; a 64-bit division is a ~100-instruction subroutine on the GPU,
// and three of them per item were a measurable bubble on short items: dW at K = 4096).
__device__ __forceinline__ Item get_item(const Sched& s, int64_t it64, int64_t Mt64, int64_t Nt64) {
  const uint32_t it = (uint32_t)it64, Mt = (uint32_t)Mt64, Nt = (uint32_t)Nt64;
  const uint32_t ck = (uint32_t)s.chunk_ntiles;
  Item x;
  x.half = -1;
  uint32_t m_tile, n0, n1, c = 0;
  if (s.c_major) {
    const uint32_t C = (Nt + ck - 1) / ck;
    const uint32_t band = s.m_band > 0 ? (uint32_t)s.m_band : Mt;
    const uint32_t full_bands = Mt / band;
    const uint32_t items_full = full_bands * C * band;
    uint32_t rem, mb, m0;
    if (it < items_full) {
      const uint32_t b = it / (C * band);
      rem = it - b * C * band;
      mb = band;
      m0 = b * band;
    } else {
      rem = it - items_full;
      mb = Mt - full_bands * band;
      m0 = full_bands * band;
    }
    c = rem / mb;
    m_tile = m0 + (rem - c * mb);
    n0 = c * ck;
    n1 = n0 + ck < Nt ? n0 + ck : Nt;
  } else if (s.n_band > 0 && (uint32_t)s.n_band < Nt) {
    const uint32_t nbw = (uint32_t)s.n_band;
    const uint32_t per_band = Mt * nbw;
    const uint32_t b = it / per_band;
    const uint32_t n_start = b * nbw;
    const uint32_t w = Nt - n_start < nbw ? Nt - n_start : nbw;   // last band: narrower
    const uint32_t rem = it - b * per_band;
    m_tile = rem / w;
    n0 = n_start + (rem - m_tile * w);
    n1 = n0 + 1;
  } else if (s.n_major) {
    n0 = it / Mt;
    m_tile = it - n0 * Mt;
    n1 = n0 + 1;
  } else {
    m_tile = it / Nt;
    n0 = it - m_tile * Nt;
    n1 = n0 + 1;
  }
  x.m_tile = m_tile; x.n0 = n0; x.n1 = n1; x.c = c;
  return x;
}

// Epilogue functor contract (tc_head.cu): Params (kernel parameter, __grid_constant__ so that it
// may hold a CUtensorMap), State (registers of one epilogue thread), kWarpSmem (bytes of staging
// smem per epilogue warp, 1024-aligned), setup / item_begin / tile_prefetch / chunk / item_end /
// finish.
//
// PPC = CTA pairs per cluster (1 or 2).  PPC = 2 (CG = 2 only): a 4-CTA cluster whose two pairs take
// M tiles 2i and 2i+1 of the same item and walk the same N tiles in lock-step; every B stage is
// fetched from L2 once per cluster -- each CTA loads a quarter of the 256-row B tile and multicasts
// it to the CTA of the other pair that needs the same half -- so the L2 -> SM operand traffic per
// flop drops by a quarter.  Only 33 clusters of 4 are co-resident on the 148 SMs of a B200, which
// is why the path's kernels stay on PPC = 1 (measurements in tc_head.cu).
template <int CG, bool A_MN, bool B_MN, class Epi, int NSUB = 1, int PPC = 1>
__global__ void __launch_bounds__(kThreads, 1)
k_tc_gemm(const __grid_constant__ CUtensorMap tmA, const __grid_constant__ CUtensorMap tmB,
          const Sched s, const __grid_constant__ typename Epi::Params ep) {
  static_assert(PPC == 1 || (PPC == 2 && CG == 2), "pairs per cluster");
  constexpr int CL = CG * PPC;                 // CTAs per cluster
  using C = Cfg<CG, NSUB, 4 * Epi::kWarpSmem>;
  extern __shared__ uint8_t smem_raw[];
  const uint32_t smem_base = (ptx::smem_u32(smem_raw) + 1023u) & ~1023u;
  const uint32_t bar_base = smem_base + C::kStages * C::kStageBytes;
  // barrier layout (8 bytes each): full[kStages], empty[kStages], tmem_full[2], tmem_empty[2]
  auto full_bar = [&](int i) { return bar_base + 8u * i; };
  auto empty_bar = [&](int i) { return bar_base + 8u * (C::kStages + i); };
  auto tfull_bar = [&](int i) { return bar_base + 8u * (2 * C::kStages + i); };
  auto tempty_bar = [&](int i) { return bar_base + 8u * (2 * C::kStages + 2 + i); };
  const uint32_t tmem_slot = bar_base + 8u * (2 * C::kStages + 4);
  // item ring (dynamic schedule), after the pipeline barriers: sfull[4], sempty[4] (the cluster
  // leader's are used), item[4]
  constexpr int kSlots = 4;
  constexpr uint32_t kRing = 8u * (2 * C::kStages + 4) + 8u;
  auto sfull_bar = [&](int i) { return bar_base + kRing + 8u * i; };
  auto sempty_bar = [&](int i) { return bar_base + kRing + 32u + 8u * i; };
  auto sitem = [&](int i) { return bar_base + kRing + 64u + 4u * i; };
  static_assert(kRing + 80u <= (uint32_t)C::kBarBytes, "barrier area overflow");

  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const uint32_t rank = CL > 1 ? ptx::cluster_ctarank() : 0u;   // rank in the cluster
  const uint32_t prank = rank % CG;                             // rank in the CTA pair
  const uint32_t pic = rank / CG;                               // pair in the cluster
  const uint32_t lead = rank - prank;                           // cluster rank of the pair's leader
  // scheduling unit = cluster
  const int64_t pair = blockIdx.x / CL, n_pairs = gridDim.x / CL;

  if (warp == 0 && lane == 0) {
    ptx::prefetch_tmap(&tmA);
    ptx::prefetch_tmap(&tmB);
  }
  if (warp == 1 && lane == 0) {
    for (int i = 0; i < C::kStages; ++i) {
      ptx::mbar_init(full_bar(i), 1);
      ptx::mbar_init(empty_bar(i), PPC);       // every pair that receives this CTA's multicast
    }
    for (int i = 0; i < 2; ++i) {
      ptx::mbar_init(tfull_bar(i), 1);
      ptx::mbar_init(tempty_bar(i), 4 * CG);
    }
    for (int i = 0; i < kSlots; ++i) {
      ptx::mbar_init(sfull_bar(i), 1);
      // consumers of a slot: 4 epilogue warps per CTA, the producer lane of every CTA but the
      // scheduler's, the MMA lane of every pair leader
      ptx::mbar_init(sempty_bar(i), 4 * CL + (CL - 1) + PPC);
    }
    ptx::fence_barrier_init();
  }
  if (warp == 2) {
    ptx::tmem_alloc<CG>(tmem_slot, kTmemCols);
    ptx::tmem_relinquish<CG>();
  }
  ptx::tc_fence_before();
  if constexpr (CL > 1) ptx::cluster_sync(); else __syncthreads();
  ptx::tc_fence_after();
  uint32_t tmem_base;
  asm volatile("ld.shared.u32 %0, [%1];" : "=r"(tmem_base) : "r"(tmem_slot));

  int64_t M_eff, K_eff;
  resolve_dims(s, M_eff, K_eff);
  // M tiles of an item's unit: PPC consecutive 128*CG-row tiles (one per pair of the cluster)
  const int64_t Mt = (M_eff + BM_CTA * CG * PPC - 1) / (BM_CTA * CG * PPC);
  const int64_t Nt = (s.N + BN * NSUB - 1) / (BN * NSUB);   // item tiles along N
  const int64_t n_chunks = s.c_major ? (Nt + s.chunk_ntiles - 1) / s.chunk_ntiles : Nt;
  const int num_kb = (int)((K_eff + BK - 1) / BK);
  // Dual-N tail: 256 x 512 tiles make the waves coarse.  When the last wave would be at most
  // half full, its r tiles are issued as 2r half tiles (one 256 x 256 sub-tile each, `half` = 0/1)
  // spread over twice as many pairs: the tail costs half a wave instead of a whole one.
  int64_t tail_start = Mt * n_chunks, n_total = Mt * n_chunks;
  if constexpr (NSUB == 2) {
    const int64_t full = n_total / n_pairs * n_pairs, r = n_total - full;
    if (s.counter == nullptr && !s.c_major && r > 0 && 2 * r <= n_pairs) {
      tail_start = full;
      n_total = full + 2 * r;
    }
  }
  const int64_t n_items = (s.skip_empty_k && num_kb == 0) ? 0 : n_total;
  auto item_of = [&](int64_t it) -> Item {
    if (NSUB == 2 && it >= tail_start) {
      const int64_t j = it - tail_start;
      Item x = get_item(s, tail_start + (j >> 1), Mt, Nt);
      x.half = (int)(j & 1);
      return x;
    }
    return get_item(s, it, Mt, Nt);
  };

  // ---- item stream -------------------------------------------------------------------------
  const bool dynamic = s.counter != nullptr;
  struct Cursor { int64_t next; int slot; uint32_t phase; };
  Cursor cur{pair, 0, 0u};
  // consumer side: next item index of this pair, or -1 when the work is exhausted
  auto consume = [&](bool warp_wide) -> int64_t {
    if (!dynamic) {
      const int64_t it = cur.next;
      cur.next += n_pairs;
      return it < n_items ? it : -1;
    }
    ptx::mbar_wait_cluster(sfull_bar(cur.slot), cur.phase);
    const int32_t v = (int32_t)ptx::ld_shared_u32(sitem(cur.slot));
    if (warp_wide) __syncwarp();
    if (!warp_wide || lane == 0) {
      if (rank == 0) ptx::mbar_arrive(sempty_bar(cur.slot));
      else ptx::mbar_arrive_cluster(ptx::mapa(sempty_bar(cur.slot), 0));
    }
    if (++cur.slot == kSlots) { cur.slot = 0; cur.phase ^= 1u; }
    return (int64_t)v;
  };
  // scheduler side (leader CTA's producer lane): publish a claimed ticket to both CTAs
  auto publish = [&](uint32_t ticket) -> int64_t {
    const int32_t v = (int64_t)ticket < n_items ? (int32_t)ticket : -1;
    ptx::mbar_wait_cluster(sempty_bar(cur.slot), cur.phase ^ 1u);
    ptx::st_shared_u32(sitem(cur.slot), (uint32_t)v);
    ptx::mbar_arrive(sfull_bar(cur.slot));
#pragma unroll
    for (uint32_t peer = 1; peer < (uint32_t)CL; ++peer) {
      ptx::st_shared_cluster_u32(ptx::mapa(sitem(cur.slot), peer), (uint32_t)v);
      ptx::mbar_arrive_cluster(ptx::mapa(sfull_bar(cur.slot), peer));
    }
    if (++cur.slot == kSlots) { cur.slot = 0; cur.phase ^= 1u; }
    return (int64_t)v;
  };

  if (warp == 0) {
    // ===================== TMA producer (one lane, every CTA) =====================
    if (lane == 0) {
      int stage = 0;
      uint32_t phase = 0;
      const uint64_t polA = ptx::make_l2_policy(s.a_hint), polB = ptx::make_l2_policy(s.b_hint);
      const bool scheduler = dynamic && rank == 0;
      int64_t it = scheduler ? publish(atomicAdd(s.counter, 1u)) : consume(false);
      // K-lockstep window (see Sched::lockstep): the pair leader's producer paces the pair; the
      // peer's loads follow through the shared ring.  G counts segments over the waves.
      bool paced = false;
      uint32_t G = 0;
      if constexpr (NSUB == 2) paced = s.lockstep != nullptr && !dynamic && !s.c_major && rank == 0;
      auto pace = [&]() {
        const uint32_t slot = G % kLockRing;
        ptx::red_add_relaxed_gpu(s.lockstep + slot, 1u);
        if (G >= (uint32_t)kLockSlack) {
          const uint32_t prev = G - (uint32_t)kLockSlack;
          ptx::wait_counter_ge(s.lockstep + prev % kLockRing,
                               (prev / kLockRing + 1u) * (uint32_t)n_pairs);
        }
        ++G;
      };
      while (it >= 0) {
        // claim the following item now (the atomic's latency hides behind this item's loads),
        // publish it after the first N tile of this one
        uint32_t ticket = 0;
        if (scheduler) ticket = atomicAdd(s.counter, 1u);
        int64_t it_next = -1;
        const Item item = item_of(it);
        const int32_t m_coord =
            (int32_t)((item.m_tile * PPC + pic) * BM_CTA * CG + prank * BM_CTA);
        const uint16_t b_mask = (uint16_t)((1u << prank) | (1u << (prank + CG)));   // PPC == 2
        for (int64_t n = item.n0; n < item.n1; ++n) {
          const int nsub = item.half < 0 ? NSUB : 1;    // half tile: one B sub-tile, in slot 0
          const int32_t n_coord = (int32_t)(n * BN * NSUB + (item.half > 0 ? BN : 0) +
                                            prank * C::kBRows);
          const uint32_t stage_tx = (uint32_t)(kABytes + nsub * C::kBBytes);
          for (int kb = 0; kb < num_kb; ++kb) {
            if constexpr (NSUB == 2) {
              if (paced && (kb % kLockSeg) == 0) pace();
            }
            ptx::mbar_wait(empty_bar(stage), phase ^ 1u);
            const uint32_t sa = smem_base + stage * C::kStageBytes;
            const uint32_t sb = sa + kABytes;
            const int32_t k_coord = kb * BK;
            if constexpr (CG == 1) {
              ptx::mbar_arrive_expect_tx(full_bar(stage), stage_tx);
              const uint32_t fb = full_bar(stage);
              if constexpr (!A_MN) ptx::tma_load_2d(sa, &tmA, k_coord, m_coord, fb, polA);
              else if (s.a_slab) ptx::tma_load_3d(sa, &tmA, 0, k_coord, m_coord >> 6, fb, polA);
              else {
                ptx::tma_load_2d(sa, &tmA, m_coord, k_coord, fb, polA);
                ptx::tma_load_2d(sa + 8192, &tmA, m_coord + 64, k_coord, fb, polA);
              }
#pragma unroll
              for (int sub = 0; sub < NSUB; ++sub) {
                if (sub >= nsub) break;
                const uint32_t sbs = sb + sub * C::kBBytes;
                const int32_t nc = n_coord + sub * BN;
                if constexpr (!B_MN) ptx::tma_load_2d(sbs, &tmB, k_coord, nc, fb, polB);
                else if (s.b_slab) ptx::tma_load_3d(sbs, &tmB, 0, k_coord, nc >> 6, fb, polB);
                else {
#pragma unroll
                  for (int b = 0; b < C::kBRows / 64; ++b)
                    ptx::tma_load_2d(sbs + 8192 * b, &tmB, nc + 64 * b, k_coord, fb, polB);
                }
              }
            } else {
              // the leader's barrier collects the bytes of both CTAs
              if (prank == 0) ptx::mbar_arrive_expect_tx(full_bar(stage), stage_tx * 2);
              const uint32_t fb = ptx::mapa(full_bar(stage), lead);
              if constexpr (!A_MN) ptx::tma_load_2d_cg2(sa, &tmA, k_coord, m_coord, fb, polA);
              else if (s.a_slab) ptx::tma_load_3d_cg2(sa, &tmA, 0, k_coord, m_coord >> 6, fb, polA);
              else {
                ptx::tma_load_2d_cg2(sa, &tmA, m_coord, k_coord, fb, polA);
                ptx::tma_load_2d_cg2(sa + 8192, &tmA, m_coord + 64, k_coord, fb, polA);
              }
#pragma unroll
              for (int sub = 0; sub < NSUB; ++sub) {
                if (sub >= nsub) break;
                const uint32_t sbs = sb + sub * C::kBBytes;
                const int32_t nc = n_coord + sub * BN;
                if constexpr (PPC == 2) {
                  // this CTA's quarter (64 B rows) of the tile, multicast to the CTA of the
                  // other pair that stages the same half
                  if constexpr (!B_MN)
                    ptx::tma_load_2d_cg2_mc(sbs + 8192 * pic, &tmB, k_coord, nc + 64 * (int32_t)pic, fb,
                                            b_mask, polB);
                  else
                    ptx::tma_load_2d_cg2_mc(sbs + 8192 * pic, &tmB, nc + 64 * (int32_t)pic, k_coord, fb,
                                            b_mask, polB);
                } else if constexpr (!B_MN) {
                  ptx::tma_load_2d_cg2(sbs, &tmB, k_coord, nc, fb, polB);
                } else if (s.b_slab) {
                  ptx::tma_load_3d_cg2(sbs, &tmB, 0, k_coord, nc >> 6, fb, polB);
                } else {
#pragma unroll
                  for (int b = 0; b < C::kBRows / 64; ++b)
                    ptx::tma_load_2d_cg2(sbs + 8192 * b, &tmB, nc + 64 * b, k_coord, fb, polB);
                }
              }
            }
            if (++stage == C::kStages) { stage = 0; phase ^= 1u; }
          }
          if (scheduler && n == item.n0) it_next = publish(ticket);
        }
        it = scheduler ? it_next : consume(false);
      }
      if constexpr (NSUB == 2) {
        // a pair without a tile in the last wave keeps counting, so that every slot sees n_pairs
        // arrivals per use
        if (paced) {
          const uint32_t segs = (uint32_t)((num_kb + kLockSeg - 1) / kLockSeg);
          const uint32_t waves = (uint32_t)((n_items + n_pairs - 1) / n_pairs);
          while (G < waves * segs) pace();
        }
      }
    }
  } else if (warp == 1) {
    // ===================== MMA issuer (one lane of the leader CTA) =====================
    if (prank == 0 && lane == 0) {
      // commits: a smem slot is released in every CTA of the cluster (each multicasts into it),
      // an accumulator is announced to this pair's two CTAs
      constexpr uint16_t kAllCtas = (uint16_t)((1u << CL) - 1u);
      const uint16_t pair_ctas = (uint16_t)(((1u << CG) - 1u) << lead);
      constexpr uint32_t idesc = ptx::make_idesc_bf16(BM_CTA * CG, BN, A_MN, B_MN);
      constexpr uint32_t a_step = A_MN ? (2048 >> 4) : (32 >> 4);   // per UMMA_K = 16
      constexpr uint32_t b_step = B_MN ? (2048 >> 4) : (32 >> 4);
      int stage = 0;
      uint32_t phase = 0;
      int acc = 0;
      uint32_t acc_phase = 0;
      for (int64_t it = consume(false); it >= 0; it = consume(false)) {
        const Item item = item_of(it);
        for (int64_t n = item.n0; n < item.n1; ++n) {
          // NSUB == 1: the two accumulators alternate between N tiles; NSUB == 2: both belong
          // to this tile (sub-tile `sub` accumulates in buffer `sub`)
          if constexpr (NSUB == 1) {
            ptx::mbar_wait(tempty_bar(acc), acc_phase ^ 1u);
          } else {
            ptx::mbar_wait(tempty_bar(0), acc_phase ^ 1u);
            ptx::mbar_wait(tempty_bar(1), acc_phase ^ 1u);
          }
          ptx::tc_fence_after();
          for (int kb = 0; kb < num_kb; ++kb) {
            ptx::mbar_wait(full_bar(stage), phase);
            ptx::tc_fence_after();
            const uint32_t sa = smem_base + stage * C::kStageBytes;
            const uint64_t adesc = ptx::make_smem_desc(sa, A_MN);
#pragma unroll
            for (int sub = 0; sub < NSUB; ++sub) {
              if (sub > 0 && item.half >= 0) break;      // half tile: accumulator 0 only
              const uint32_t d_tmem = tmem_base + (uint32_t)(NSUB == 1 ? acc : sub) * BN;
              const uint64_t bdesc = ptx::make_smem_desc(sa + kABytes + sub * C::kBBytes, B_MN);
#pragma unroll
              for (int k = 0; k < BK / 16; ++k)
                ptx::umma_bf16<CG>(d_tmem, adesc + (uint64_t)(k * a_step),
                                   bdesc + (uint64_t)(k * b_step), idesc, (uint32_t)(kb | k));
            }
            ptx::umma_commit<CG>(empty_bar(stage), kAllCtas);   // frees the smem slot
            if (++stage == C::kStages) { stage = 0; phase ^= 1u; }
          }
          if constexpr (NSUB == 1) {
            ptx::umma_commit<CG>(tfull_bar(acc), pair_ctas);    // accumulator ready (both CTAs)
            if (++acc == 2) { acc = 0; acc_phase ^= 1u; }
          } else {
            ptx::umma_commit<CG>(tfull_bar(0), pair_ctas);
            ptx::umma_commit<CG>(tfull_bar(1), pair_ctas);
            acc_phase ^= 1u;
          }
        }
      }
    }
  } else if (warp >= 4) {
    // ===================== epilogue warps =====================
    const int q = warp & 3;
    const int row_in_tile = q * 32 + lane;
    const uint32_t lane_base = tmem_base + ((uint32_t)(q * 32) << 16);
    int acc = 0;
    uint32_t acc_phase = 0;
    typename Epi::State st;
    Epi::setup(st, ep, bar_base + C::kBarBytes + (uint32_t)(q * Epi::kWarpSmem));
    for (int64_t it = consume(true); it >= 0; it = consume(true)) {
      const Item item = item_of(it);
      const int64_t grow = (item.m_tile * PPC + pic) * BM_CTA * CG + prank * BM_CTA + row_in_tile;
      const bool valid = grow < M_eff;
      Epi::item_begin(st, ep, grow, valid, item.c);
      for (int64_t nn = item.n0 * NSUB; nn < item.n1 * NSUB; ++nn) {
        // 256-wide tile index along N; a half tile keeps its data in accumulator 0 and only
        // hands accumulator 1 back
        const int64_t n = item.half > 0 ? nn + 1 : nn;
        const bool skip = NSUB == 2 && item.half >= 0 && nn != item.n0 * NSUB;
        Epi::tile_prefetch(ep, grow, valid && !skip, n * BN);
        ptx::mbar_wait(tfull_bar(acc), acc_phase);
        ptx::tc_fence_after();
        if (skip) {
          ptx::tc_fence_before();
          __syncwarp();
          if (lane == 0) {
            if constexpr (CG == 1) ptx::mbar_arrive(tempty_bar(acc));
            else ptx::mbar_arrive_cluster(ptx::mapa(tempty_bar(acc), lead));
          }
          if (++acc == 2) { acc = 0; acc_phase ^= 1u; }
          continue;
        }
#pragma unroll 1
        for (int ch = 0; ch < BN / 32; ++ch) {
          uint32_t r[32];
          __syncwarp();
          if (num_kb > 0) {
            ptx::tmem_ld_32x32(lane_base + (uint32_t)(acc * BN + ch * 32), r);
            ptx::tmem_wait_ld();
          } else {
#pragma unroll
            for (int j = 0; j < 32; ++j) r[j] = 0u;
          }
          if (ch == BN / 32 - 1) {
            // all of this warp's reads of the accumulator are done: hand it back to the MMA
            ptx::tc_fence_before();
            __syncwarp();
            if (lane == 0) {
              if constexpr (CG == 1) ptx::mbar_arrive(tempty_bar(acc));
              else ptx::mbar_arrive_cluster(ptx::mapa(tempty_bar(acc), lead));
            }
          }
          float x[32];
#pragma unroll
          for (int j = 0; j < 32; ++j) x[j] = __uint_as_float(r[j]);
          Epi::chunk(st, ep, grow, valid, n * BN + ch * 32, x);
        }
        if (++acc == 2) { acc = 0; acc_phase ^= 1u; }
      }
      Epi::item_end(st, ep, grow, valid, item.c);
    }
    Epi::finish(st, ep);
  }

  // ---- teardown ----
  ptx::tc_fence_before();
  if constexpr (CL > 1) ptx::cluster_sync(); else __syncthreads();
  if (warp == 2) ptx::tmem_dealloc<CG>(tmem_base, kTmemCols);
}

// ---------------------------------------------------------------------------------------------
// host side
// ---------------------------------------------------------------------------------------------
typedef CUresult (*PFN_encodeTiled)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*,
                                    const cuuint64_t*, const cuuint64_t*, const cuuint32_t*,
                                    const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle,
                                    CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

inline PFN_encodeTiled get_encode_fn() {
  static PFN_encodeTiled fn = [] {
    void* p = nullptr;
    cudaDriverEntryPointQueryResult q;
    if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &q) != cudaSuccess)
      p = nullptr;
    return reinterpret_cast<PFN_encodeTiled>(p);
  }();
  return fn;
}

// bf16 2-D row-major tensor [outer, inner] with row stride ld (elements), 128B-swizzled boxes.
inline int make_tmap_bf16(CUtensorMap* m, const void* base, int64_t inner, int64_t outer,
                          int64_t ld, int box_inner, int box_outer) {
  PFN_encodeTiled fn = get_encode_fn();
  if (!fn) return GC_ERR_CUDA;
  if (inner <= 0 || outer <= 0) return GC_ERR_SHAPE;
  if ((reinterpret_cast<uintptr_t>(base) & 15) || ((ld * 2) & 15)) return GC_ERR_ALIGN;
  cuuint64_t dims[2] = {(cuuint64_t)inner, (cuuint64_t)outer};
  cuuint64_t strides[1] = {(cuuint64_t)ld * 2};
  cuuint32_t box[2] = {(cuuint32_t)box_inner, (cuuint32_t)box_outer};
  cuuint32_t estr[2] = {1, 1};
  CUresult r = fn(m, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 2, const_cast<void*>(base), dims, strides,
                  box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B,
                  CU_TENSOR_MAP_L2_PROMOTION_L2_256B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
  return r == CUDA_SUCCESS ? GC_OK : GC_ERR_CUDA;
}

// Operand X of a GEMM with `rows` along M (or N) and `K` along the contraction:
//   K-major  : memory is [rows, K] (ld >= K)   -> box {64 k, box_rows}
//   MN-major : memory is [K, rows] (ld >= rows) -> box {64 rows, 64 k}
inline int make_operand_tmap(CUtensorMap* m, const void* base, int64_t rows, int64_t K, int64_t ld,
                             bool mn_major, int box_rows) {
  if (!mn_major) return make_tmap_bf16(m, base, K, rows, ld, BK, box_rows);
  return make_tmap_bf16(m, base, rows, K, ld, 64, BK);
}

// MN-major operand in slab form: memory [K, rows] with rows % 64 == 0 seen as the 3-D tensor
// {64 mn in a slab, K, rows / 64 slabs} (strides: ld elements between k, 64 elements between slabs);
// a box of `slabs` slabs x 64 k lands in shared memory as `slabs` consecutive 8 KB [64 k][64 mn]
// tiles -- exactly what `slabs` 2-D boxes would write, in one TMA instruction.  Slabs past the
// extent are zero-filled.  (rows % 64 != 0 cannot take this form: the last slab would run into
// the next k row.)
inline int make_slab_tmap_bf16(CUtensorMap* m, const void* base, int64_t rows, int64_t K, int64_t ld,
                               int slabs) {
  PFN_encodeTiled fn = get_encode_fn();
  if (!fn) return GC_ERR_CUDA;
  if (rows <= 0 || K <= 0 || rows % 64 != 0 || slabs < 1) return GC_ERR_SHAPE;
  if ((reinterpret_cast<uintptr_t>(base) & 15) || ((ld * 2) & 15)) return GC_ERR_ALIGN;
  cuuint64_t dims[3] = {64, (cuuint64_t)K, (cuuint64_t)(rows / 64)};
  cuuint64_t strides[2] = {(cuuint64_t)ld * 2, 128};
  cuuint32_t box[3] = {64, (cuuint32_t)BK, (cuuint32_t)slabs};
  cuuint32_t estr[3] = {1, 1, 1};
  CUresult r = fn(m, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 3, const_cast<void*>(base), dims, strides, box,
                  estr, CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B,
                  CU_TENSOR_MAP_L2_PROMOTION_L2_256B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
  return r == CUDA_SUCCESS ? GC_OK : GC_ERR_CUDA;
}

inline int num_sms() {
  int dev = 0, n = kNumSMs;
  if (cudaGetDevice(&dev) == cudaSuccess)
    cudaDeviceGetAttribute(&n, cudaDevAttrMultiProcessorCount, dev);
  return n;
}

// Clusters of `cl` CTAs that can be co-resident with this kernel's resources (1 CTA per SM): 74 of
// 2, 33 of 4 on a B200 (GPC boundaries).  Queried once per kernel instantiation.
template <class Kern>
inline int max_active_clusters(Kern kern, int cl, int smem_bytes) {
  cudaLaunchConfig_t cfg = {};
  cfg.gridDim = dim3((unsigned)(num_sms() / cl * cl));
  cfg.blockDim = dim3(kThreads);
  cfg.dynamicSmemBytes = (size_t)smem_bytes;
  cudaLaunchAttribute attr[1];
  attr[0].id = cudaLaunchAttributeClusterDimension;
  attr[0].val.clusterDim.x = (unsigned)cl;
  attr[0].val.clusterDim.y = 1;
  attr[0].val.clusterDim.z = 1;
  cfg.attrs = attr;
  cfg.numAttrs = 1;
  int n = 0;
  if (cudaOccupancyMaxActiveClusters(&n, kern, &cfg) != cudaSuccess || n < 1) n = num_sms() / cl;
  return n;
}

template <int CG, bool A_MN, bool B_MN, class Epi, int NSUB = 1, int PPC = 1>
int launch_tc_gemm(const CUtensorMap& tmA, const CUtensorMap& tmB, const Sched& s,
                   const typename Epi::Params& ep, cudaStream_t st) {
  auto kern = k_tc_gemm<CG, A_MN, B_MN, Epi, NSUB, PPC>;
  constexpr int CL = CG * PPC;
  constexpr int kSmemBytes = Cfg<CG, NSUB, 4 * Epi::kWarpSmem>::kSmemBytes;
  static_assert(kSmemBytes <= 227 * 1024, "shared memory budget");
  // Per instantiation and device: the smem opt-in is a per-device function attribute, and the
  // number of co-resident clusters is queried once.  This cache is the library's only launch-path
  // state; it is write-once per slot with an idempotent value (concurrent first calls compute the
  // same number), published with release/acquire so host threads may race on the first launch.
  static std::atomic<int> clusters_by_dev[64];
  int dev = 0;
  GC_CUDA_TRY(cudaGetDevice(&dev));
  if (dev < 0 || dev >= 64) return GC_ERR_CUDA;
  int clusters = clusters_by_dev[dev].load(std::memory_order_acquire);
  if (clusters == 0) {
    GC_CUDA_TRY(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, kSmemBytes));
    clusters = max_active_clusters(kern, CL, kSmemBytes);
    clusters_by_dev[dev].store(clusters, std::memory_order_release);
  }
  cudaLaunchConfig_t cfg = {};
  cfg.gridDim = dim3((unsigned)(clusters * CL));
  cfg.blockDim = dim3(kThreads);
  cfg.dynamicSmemBytes = kSmemBytes;
  cfg.stream = st;
  cudaLaunchAttribute attr[1];
  attr[0].id = cudaLaunchAttributeClusterDimension;
  attr[0].val.clusterDim.x = CL;
  attr[0].val.clusterDim.y = 1;
  attr[0].val.clusterDim.z = 1;
  cfg.attrs = attr;
  cfg.numAttrs = 1;
  GC_CUDA_TRY(cudaLaunchKernelEx(&cfg, kern, tmA, tmB, s, ep));
  return GC_OK;
}

}  // namespace tc
}  // namespace gc
