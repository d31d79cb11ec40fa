// timing.cu -- optional per-kernel timing of the tcgen05 contraction launches with CUDA events
// recorded on the stream the kernel is launched on (gc_kernel_timing_begin / _end in gcore.h).
// Off by default: when off, the launch path costs one relaxed atomic load.
#include <atomic>
#include <mutex>
#include <vector>

#include "common.cuh"

namespace gc {

namespace {
struct Rec { cudaEvent_t e0, e1; int kind; };
std::atomic<int> g_on{0};
std::mutex g_mu;
std::vector<Rec> g_recs;                  // records of the current session
std::vector<cudaEvent_t> g_pool;          // events kept for reuse across sessions
constexpr size_t kMaxRecs = 1 << 16;

cudaEvent_t take_event() {
  if (!g_pool.empty()) {
    cudaEvent_t e = g_pool.back();
    g_pool.pop_back();
    return e;
  }
  cudaEvent_t e = nullptr;
  if (cudaEventCreate(&e) != cudaSuccess) return nullptr;
  return e;
}
}  // namespace

KernelTimer::KernelTimer(int kind, cudaStream_t st) : st_(st), idx_(-1) {
  if (!g_on.load(std::memory_order_relaxed)) return;
  std::lock_guard<std::mutex> lk(g_mu);
  if (!g_on.load() || g_recs.size() >= kMaxRecs) return;
  Rec r{take_event(), take_event(), kind};
  if (!r.e0 || !r.e1) return;
  if (cudaEventRecord(r.e0, st) != cudaSuccess) return;
  g_recs.push_back(r);
  idx_ = (long)g_recs.size() - 1;
}

KernelTimer::~KernelTimer() {
  if (idx_ < 0) return;
  std::lock_guard<std::mutex> lk(g_mu);
  if ((size_t)idx_ < g_recs.size()) cudaEventRecord(g_recs[idx_].e1, st_);
}

}  // namespace gc

extern "C" {

int gc_kernel_timing_begin(void) {
  std::lock_guard<std::mutex> lk(gc::g_mu);
  for (auto& r : gc::g_recs) { gc::g_pool.push_back(r.e0); gc::g_pool.push_back(r.e1); }
  gc::g_recs.clear();
  gc::g_on.store(1);
  return GC_OK;
}

int gc_kernel_timing_end(float* ms_by_kind_host, int32_t* launches_by_kind_host) {
  if (!ms_by_kind_host || !launches_by_kind_host) return GC_ERR_NULL;
  std::lock_guard<std::mutex> lk(gc::g_mu);
  gc::g_on.store(0);
  for (int k = 0; k < GC_KERNEL_KINDS; ++k) { ms_by_kind_host[k] = 0.f; launches_by_kind_host[k] = 0; }
  int status = GC_OK;
  for (auto& r : gc::g_recs) {
    float ms = 0.f;
    if (cudaEventSynchronize(r.e1) != cudaSuccess ||
        cudaEventElapsedTime(&ms, r.e0, r.e1) != cudaSuccess) {
      status = GC_ERR_CUDA;
    } else if (r.kind >= 0 && r.kind < GC_KERNEL_KINDS) {
      ms_by_kind_host[r.kind] += ms;
      launches_by_kind_host[r.kind] += 1;
    }
    gc::g_pool.push_back(r.e0);
    gc::g_pool.push_back(r.e1);
  }
  gc::g_recs.clear();
  return status;
}

}  // extern "C"
