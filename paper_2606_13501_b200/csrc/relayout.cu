// relayout.cu — on-device re-layout of a row-sharded artifact between split degrees P -> P' (
// PAPER.md:285-293, §5.3 "Layout-Aware Artifact Migration": intersect every source-owned slice with every
// destination-required slice, every non-empty intersection is a transfer entry (source rank, destination rank, source
// range, destination range, size); each rank packs the ranges, they are exchanged and installed in the destination
// representation).  On one GPU the P source shards and the P' destination shards are buffers in the same HBM, so
// "pack -> exchange -> install" is ONE copy kernel that executes the whole plan: a pure HBM-bound kernel (algorithmic
// bytes = 2 x artifact size), 128-bit accesses, every transfer entry is a grid row.
// Shards follow reading R20: P contiguous row ranges of ceil(n / P) rows, the last ones shorter or empty.
#include <algorithm>

#include "common.cuh"

namespace dit {
namespace {

constexpr int MAX_ENTRIES = 64;   // P + P' - 1 <= 63 for P, P' <= 32

struct CopyPlan {
  const char* src[MAX_ENTRIES];
  char* dst[MAX_ENTRIES];
  int64_t bytes[MAX_ENTRIES];
};

template <typename V>
__global__ void __launch_bounds__(256) relayout_kernel(const __grid_constant__ CopyPlan plan) {
  pdl_trigger();
  pdl_wait();
  const int e = blockIdx.y;
  const V* __restrict__ s = reinterpret_cast<const V*>(plan.src[e]);
  V* __restrict__ d = reinterpret_cast<V*>(plan.dst[e]);
  const int64_t n = plan.bytes[e] / (int64_t)sizeof(V);
  const int64_t stride = (int64_t)gridDim.x * blockDim.x;
  int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  // four independent 16-byte loads in flight per thread before the first store
  for (; i + 3 * stride < n; i += 4 * stride) {
    const V a = s[i], b = s[i + stride], c = s[i + 2 * stride], f = s[i + 3 * stride];
    d[i] = a; d[i + stride] = b; d[i + 2 * stride] = c; d[i + 3 * stride] = f;
  }
  for (; i < n; i += stride) d[i] = s[i];
}

static void shard_range(int64_t n, int P, int p, int64_t* lo, int64_t* hi) {   // R20
  const int64_t sz = (n + P - 1) / P;
  *lo = std::min<int64_t>((int64_t)p * sz, n);
  *hi = std::min<int64_t>((int64_t)(p + 1) * sz, n);
}

}  // namespace
}  // namespace dit

using namespace dit;

extern "C" {

int32_t dit_relayout_plan(int64_t n_rows, int32_t p_src, int32_t p_dst, dit_transfer* entries, int32_t max_entries) {
  if (n_rows < 0 || p_src < 1 || p_dst < 1 || p_src > 32 || p_dst > 32 || (entries == nullptr && max_entries > 0)) {
    set_error("dit_relayout_plan: n_rows %lld, p_src %d, p_dst %d (1..32)", (long long)n_rows, p_src, p_dst);
    return DIT_ERR_INVALID_ARG;
  }
  int32_t n = 0;
  for (int q = 0; q < p_dst; ++q) {          // destination-major: a destination shard is filled front to back
    int64_t dlo, dhi;
    shard_range(n_rows, p_dst, q, &dlo, &dhi);
    for (int p = 0; p < p_src; ++p) {
      int64_t slo, shi;
      shard_range(n_rows, p_src, p, &slo, &shi);
      const int64_t lo = std::max(slo, dlo), hi = std::min(shi, dhi);
      if (lo >= hi) continue;                // empty intersection: no transfer entry
      if (n < max_entries) entries[n] = dit_transfer{p, q, lo - slo, lo - dlo, hi - lo};
      ++n;
    }
  }
  return n;   // the number of entries the plan has (may exceed max_entries: call again with a larger array)
}

dit_status dit_relayout(const dit_transfer* entries, int32_t n_entries, const void* const* src_shards,
                        void* const* dst_shards, int64_t row_bytes, void* stream) {
  DIT_REQUIRE(n_entries >= 0 && n_entries <= MAX_ENTRIES, DIT_ERR_INVALID_ARG, "dit_relayout: %d entries (max %d)", n_entries, MAX_ENTRIES);
  DIT_REQUIRE(n_entries == 0 || (entries && src_shards && dst_shards), DIT_ERR_INVALID_ARG, "dit_relayout: NULL argument");
  DIT_REQUIRE(row_bytes > 0, DIT_ERR_INVALID_ARG, "dit_relayout: row_bytes %lld", (long long)row_bytes);
  if (n_entries == 0) return DIT_OK;
  CopyPlan plan;
  int64_t total = 0, biggest = 0;
  uintptr_t align = 0;
  for (int i = 0; i < n_entries; ++i) {
    const dit_transfer& t = entries[i];
    DIT_REQUIRE(t.src_rank >= 0 && t.src_rank < 32 && t.dst_rank >= 0 && t.dst_rank < 32 && t.src_row >= 0 && t.dst_row >= 0 &&
                    t.n_rows > 0, DIT_ERR_INVALID_ARG, "dit_relayout: entry %d is malformed", i);
    DIT_REQUIRE(src_shards[t.src_rank] && dst_shards[t.dst_rank], DIT_ERR_INVALID_ARG, "dit_relayout: shard pointer of entry %d is NULL", i);
    plan.src[i] = (const char*)src_shards[t.src_rank] + t.src_row * row_bytes;
    plan.dst[i] = (char*)dst_shards[t.dst_rank] + t.dst_row * row_bytes;
    plan.bytes[i] = t.n_rows * row_bytes;
    total += plan.bytes[i];
    biggest = std::max(biggest, plan.bytes[i]);
    align |= (uintptr_t)plan.src[i] | (uintptr_t)plan.dst[i] | (uintptr_t)plan.bytes[i];
  }
  for (int i = n_entries; i < MAX_ENTRIES; ++i) { plan.src[i] = nullptr; plan.dst[i] = nullptr; plan.bytes[i] = 0; }
  cudaStream_t st = (cudaStream_t)stream;
  ProfScope _prof(DIT_KC_MISC, st);
  // grid: one row of CTAs per entry; enough CTAs for the largest entry to keep ~8 x 148 CTAs in flight overall
  const int vec = (align & 15) == 0 ? 16 : ((align & 3) == 0 ? 4 : 1);
  int gx = (int)std::min<int64_t>((biggest / vec + 256 * 4 - 1) / (256 * 4), std::max(1, 8 * 148 / n_entries));
  if (gx < 1) gx = 1;
  dim3 grid(gx, n_entries);
  if (vec == 16) DIT_CUDA_OK(launch_pdl(relayout_kernel<uint4>, grid, dim3(256), 0, st, 1, plan));
  else if (vec == 4) DIT_CUDA_OK(launch_pdl(relayout_kernel<uint32_t>, grid, dim3(256), 0, st, 1, plan));
  else DIT_CUDA_OK(launch_pdl(relayout_kernel<uint8_t>, grid, dim3(256), 0, st, 1, plan));
  DIT_LAUNCH_CHECK();
  (void)total;
  return DIT_OK;
}

}  // extern "C"
