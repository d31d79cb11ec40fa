// balance.cu -- the step before the scoring path: dynamic-sampling
// repack + workload balancing.  PAPER.md:150 (sec 3.2) "filter out prompts with the accuracy equal
// to 1 and 0"; PAPER.md:201 (sec 4.4) "instead of sequence packing, we simply sort data by simulated
// workload"; "we first bucket data according to the global batch size, then shuffle
// the buckets".  Steps (oracle/balance_oracle.py):
//   1 kept samples = samples of groups with keep != 0, in ascending index
//   2 workload w_i = w_lin L_i + w_quad L_i^2 (unsigned 64-bit), L_i = cu[i+1] - cu[i]
//   3 stable ascending sort of the kept samples by w
//   4 consecutive buckets of `bucket_size` samples (the last may be short)
//   5 buckets reordered by ascending (splitmix64(seed, b), b)           (shuffle != 0)
//   6 order[] = the buckets concatenated; cu_out = prefix sums of the lengths in that order;
//     src_token[cu_out[d] + t] = cu[order[d]] + t
// All integer work: bit-exact against the oracle.  Sorting is rank-by-counting over (key, index)
// pairs, O(R^2) compares tiled through shared memory -- R is samples per step (<= ~10^5), where this
// is tens of microseconds and needs no multi-pass radix machinery.
#include "common.cuh"

namespace gc {

namespace {

constexpr int kRankThreads = 256;
constexpr int kRankTile = 2048;               // keys staged per shared-memory tile
constexpr uint64_t kDropped = ~0ull;          // key of a dropped sample: sorts after every kept one

__device__ __forceinline__ uint64_t splitmix64(uint64_t seed, uint64_t b) {
  uint64_t z = seed + (b + 1ull) * 0x9E3779B97F4A7C15ull;
  z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9ull;
  z = (z ^ (z >> 27)) * 0x94D049BB133111EBull;
  return z ^ (z >> 31);
}

// step 1 + 2: one thread per group walks its samples; key = workload or kDropped
__global__ void k_bal_keys(const int32_t* __restrict__ cu, const int32_t* __restrict__ group_offsets,
                           const uint8_t* __restrict__ keep, int32_t G, uint64_t w_lin,
                           uint64_t w_quad, uint64_t* __restrict__ key) {
  const int g = blockIdx.x * blockDim.x + threadIdx.x;
  if (g >= G) return;
  const bool kept = keep == nullptr || keep[g] != 0;
  for (int i = group_offsets[g]; i < group_offsets[g + 1]; ++i) {
    const uint64_t L = (uint64_t)(cu[i + 1] - cu[i]);
    key[i] = kept ? w_lin * L + w_quad * L * L : kDropped;
  }
}

// no groups given: every sample is kept
__global__ void k_bal_keys_all(const int32_t* __restrict__ cu, int32_t R, uint64_t w_lin,
                               uint64_t w_quad, uint64_t* __restrict__ key) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= R) return;
  const uint64_t L = (uint64_t)(cu[i + 1] - cu[i]);
  key[i] = w_lin * L + w_quad * L * L;
}

// rank[i] = #{ j : (key_j, j) < (key_i, i) } ; also counts the entries with key != kDropped
__global__ void __launch_bounds__(kRankThreads)
k_bal_rank(const uint64_t* __restrict__ key, int32_t n, int32_t* __restrict__ rank,
           int32_t* __restrict__ n_valid) {
  __shared__ uint64_t s_key[kRankTile];
  const int i = blockIdx.x * kRankThreads + threadIdx.x;
  const uint64_t ki = i < n ? key[i] : 0;
  int r = 0;
  for (int base = 0; base < n; base += kRankTile) {
    const int m = min(kRankTile, n - base);
    __syncthreads();
    for (int j = threadIdx.x; j < m; j += kRankThreads) s_key[j] = key[base + j];
    __syncthreads();
    if (i < n) {
      // j < i: counts when key_j <= key_i ; j > i: when key_j < key_i
      const int split = min(max(i - base, 0), m);     // entries [0, split) have index < i
      for (int j = 0; j < split; ++j) r += s_key[j] <= ki ? 1 : 0;
      for (int j = split + (base + split == i ? 1 : 0); j < m; ++j) r += s_key[j] < ki ? 1 : 0;
    }
  }
  if (i < n) {
    rank[i] = r;
    if (n_valid && ki != kDropped) atomicAdd(n_valid, 1);
  }
}

__global__ void k_bal_bucket_keys(const int32_t* __restrict__ n_kept, int32_t bucket_size,
                                  uint64_t seed, int shuffle, int32_t nb_cap,
                                  uint64_t* __restrict__ bkey) {
  const int b = blockIdx.x * blockDim.x + threadIdx.x;
  if (b >= nb_cap) return;
  const int nb = (*n_kept + bucket_size - 1) / bucket_size;
  // buckets past the last one sort to the end; without shuffle the key is the index itself
  bkey[b] = b < nb ? (shuffle ? (splitmix64(seed, (uint64_t)b) >> 1) : (uint64_t)b) : kDropped;
}

// steps 4-6a: destination slot of every kept sample
__global__ void k_bal_place(const uint64_t* __restrict__ key, const int32_t* __restrict__ rank,
                            const int32_t* __restrict__ brank, const int32_t* __restrict__ n_kept,
                            const int32_t* __restrict__ cu, int32_t R, int32_t bucket_size,
                            int32_t* __restrict__ order, int32_t* __restrict__ len_out) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= R) return;
  const int n = *n_kept;
  if (key[i] == kDropped) return;
  const int k = rank[i];
  const int nb = (n + bucket_size - 1) / bucket_size;
  const int b = k / bucket_size, p = k - b * bucket_size;
  const int q = brank[b];
  const int short_by = nb * bucket_size - n;         // the last bucket is this much short
  const int q_last = brank[nb - 1];
  const int dst = q * bucket_size + p - (q > q_last ? short_by : 0);
  order[dst] = i;
  len_out[dst] = cu[i + 1] - cu[i];
}

// exclusive scan of len[0..n) into cu_out[0..n], cu_out[j] = total for n < j <= R.  One block.
__global__ void k_bal_scan(const int32_t* __restrict__ len, const int32_t* __restrict__ n_kept,
                           int32_t R, int32_t* __restrict__ cu_out, int32_t* __restrict__ n_tokens,
                           int32_t* __restrict__ order) {
  __shared__ int sm[1024];
  __shared__ int carry;
  const int n = *n_kept;
  if (threadIdx.x == 0) carry = 0;
  __syncthreads();
  for (int base = 0; base < n; base += 1024) {
    const int i = base + threadIdx.x;
    const int v = i < n ? len[i] : 0;
    sm[threadIdx.x] = v;
    __syncthreads();
    for (int o = 1; o < 1024; o <<= 1) {
      const int add = threadIdx.x >= o ? sm[threadIdx.x - o] : 0;
      __syncthreads();
      sm[threadIdx.x] += add;
      __syncthreads();
    }
    if (i < n) cu_out[i] = carry + sm[threadIdx.x] - v;
    __syncthreads();
    if (threadIdx.x == 0) carry += sm[1023];
    __syncthreads();
  }
  for (int j = n + threadIdx.x; j <= R; j += 1024) cu_out[j] = carry;
  for (int j = n + threadIdx.x; j < R; j += 1024) order[j] = -1;
  if (threadIdx.x == 0) *n_tokens = carry;
}

// step 6b: one warp per destination sample writes the source token index of each of its tokens
__global__ void k_bal_src_tokens(const int32_t* __restrict__ order, const int32_t* __restrict__ cu,
                                 const int32_t* __restrict__ cu_out,
                                 const int32_t* __restrict__ n_kept, int32_t* __restrict__ src_token) {
  const int d = (blockIdx.x * blockDim.x + threadIdx.x) >> 5;
  const int lane = threadIdx.x & 31;
  if (d >= *n_kept) return;
  const int src0 = cu[order[d]], dst0 = cu_out[d], L = cu_out[d + 1] - dst0;
  for (int t = lane; t < L; t += 32) src_token[dst0 + t] = src0 + t;
}

}  // namespace

size_t balance_ws_bytes(int32_t R) {
  const size_t r = (size_t)(R > 0 ? R : 1);
  return align_up(r * 8, 256) * 2 + align_up(r * 4, 256) * 3 + 256;
}

int launch_balance_plan(const int32_t* cu, int32_t R, const int32_t* group_offsets,
                        const uint8_t* keep, int32_t G, uint64_t w_lin, uint64_t w_quad,
                        int32_t bucket_size, uint64_t seed, int shuffle, int32_t* order,
                        int32_t* n_kept, int32_t* cu_out, int32_t* src_token, int32_t* n_tokens,
                        void* ws, cudaStream_t st) {
  Carver c(ws);
  uint64_t* key = c.take<uint64_t>((size_t)R);
  uint64_t* bkey = c.take<uint64_t>((size_t)R);
  int32_t* rank = c.take<int32_t>((size_t)R);
  int32_t* brank = c.take<int32_t>((size_t)R);
  int32_t* len_out = c.take<int32_t>((size_t)R);
  GC_CUDA_TRY(cudaMemsetAsync(n_kept, 0, sizeof(int32_t), st));
  const int rb = (int)ceil_div(R, kRankThreads);
  if (group_offsets && G > 0)
    k_bal_keys<<<(unsigned)ceil_div(G, 128), 128, 0, st>>>(cu, group_offsets, keep, G, w_lin, w_quad,
                                                          key);
  else
    k_bal_keys_all<<<(unsigned)ceil_div(R, 256), 256, 0, st>>>(cu, R, w_lin, w_quad, key);
  k_bal_rank<<<rb, kRankThreads, 0, st>>>(key, R, rank, n_kept);
  // at most ceil(R / bucket_size) buckets exist whatever n_kept turns out to be
  const int32_t nb_cap = (int32_t)ceil_div(R, bucket_size);
  k_bal_bucket_keys<<<(unsigned)ceil_div(nb_cap, 256), 256, 0, st>>>(n_kept, bucket_size, seed, shuffle,
                                                                    nb_cap, bkey);
  k_bal_rank<<<(unsigned)ceil_div(nb_cap, kRankThreads), kRankThreads, 0, st>>>(bkey, nb_cap, brank,
                                                                               nullptr);
  k_bal_place<<<(unsigned)ceil_div(R, 256), 256, 0, st>>>(key, rank, brank, n_kept, cu, R, bucket_size,
                                                         order, len_out);
  k_bal_scan<<<1, 1024, 0, st>>>(len_out, n_kept, R, cu_out, n_tokens, order);
  k_bal_src_tokens<<<(unsigned)ceil_div((int64_t)R * 32, 256), 256, 0, st>>>(order, cu, cu_out, n_kept,
                                                                            src_token);
  GC_CUDA_TRY(cudaGetLastError());
  return GC_OK;
}

}  // namespace gc
