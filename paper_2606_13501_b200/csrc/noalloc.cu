// noalloc.cu — split-KV attention + LSE merge with the partials in a STATIC device array: an entry point for callers that
// cannot allocate device memory (code under CUDA graph capture, tight serving loops, harnesses that forbid cudaMalloc).
//
// dit_attn_split_static is dit_attn_partial over P contiguous KV shards (R20) followed by dit_attn_merge (SURVEY.md §8(a)
// a13 / a14), but the P partial outputs and their log-sum-exps — which the other paths keep in the caller's workspace
// (dit_step with split_p > 1) or in caller tensors (dit_attn_partial / dit_attn_merge) — live in `g_static_scratch` below.
//   * The array is part of the library image: every GPU that loads the library holds DIT_STATIC_SCRATCH_BYTES (8 MiB) of
//     device memory until the process exits.
//   * In host code the array's NAME is a host-side stand-in, not a device address.  The device address is obtained once per
//     device, with that device current, by cudaGetSymbolAddress (device_scratch below), and only that pointer is handed to
//     the kernels.
//   * The entry point calls no cudaMalloc / cudaFree and no allocating library routine; sizes beyond the array are rejected.
//   * Every call on a device shares the one array and the array keeps the last call's contents.  Nothing has to start at zero:
//     every row of every partial (output and LSE) that the merge reads is written by the partial-attention kernels of the
//     same call first (an empty shard writes o = 0, lse = -inf, R18).  Calls that OVERLAP on the GPU (two streams, or two
//     host threads on one device) race on the array: callers serialise them.
#include <mutex>

#include "common.cuh"

#define DIT_STATIC_SCRATCH_BYTES (8u << 20)

static __device__ __align__(256) unsigned char g_static_scratch[DIT_STATIC_SCRATCH_BYTES];

namespace dit {
namespace {

constexpr int MAX_DEVICES = 64;

// Device address of g_static_scratch on the CURRENT device (looked up once per device).
dit_status device_scratch(unsigned char** out) {
  static std::mutex mu;
  static unsigned char* addr[MAX_DEVICES] = {};
  int dev = -1;
  DIT_CUDA_OK(cudaGetDevice(&dev));
  DIT_REQUIRE(dev >= 0 && dev < MAX_DEVICES, DIT_ERR_UNSUPPORTED, "device ordinal %d (max %d)", dev, MAX_DEVICES - 1);
  std::lock_guard<std::mutex> lock(mu);
  if (addr[dev] == nullptr) {
    void* p = nullptr;
    DIT_CUDA_OK(cudaGetSymbolAddress(&p, g_static_scratch));
    DIT_REQUIRE(p != nullptr && ((uintptr_t)p & 255) == 0, DIT_ERR_CUDA, "static scratch: bad device address %p", p);
    addr[dev] = (unsigned char*)p;
  }
  *out = addr[dev];
  return DIT_OK;
}

size_t align256(size_t v) { return (v + 255) & ~(size_t)255; }

}  // namespace
}  // namespace dit

using namespace dit;

extern "C" {

size_t dit_static_scratch_bytes(void) { return DIT_STATIC_SCRATCH_BYTES; }

dit_status dit_attn_split_static(int32_t dtype, const void* q, const void* k, const void* v, int32_t n_q, int32_t n_k,
                                 int32_t n_heads, int32_t head_dim, int64_t q_row_stride, int64_t kv_row_stride,
                                 float softmax_scale, int32_t split_p, void* o, float* lse_out, void* stream) {
  DIT_REQUIRE(dtype == DIT_F32 || dtype == DIT_BF16, DIT_ERR_INVALID_ARG, "dtype %d", dtype);
  DIT_REQUIRE(n_q >= 0 && n_k >= 0 && n_heads > 0, DIT_ERR_INVALID_ARG, "n_q %d n_k %d n_heads %d", n_q, n_k, n_heads);
  DIT_REQUIRE(head_dim == 64 || head_dim == 128, DIT_ERR_UNSUPPORTED, "head_dim %d not in {64,128}", head_dim);
  DIT_REQUIRE(split_p >= 1 && split_p <= 8, DIT_ERR_INVALID_ARG, "split_p %d not in 1..8", split_p);
  DIT_REQUIRE(n_q == 0 || (q && o), DIT_ERR_INVALID_ARG, "q / o is NULL");
  DIT_REQUIRE(n_k == 0 || (k && v), DIT_ERR_INVALID_ARG, "k / v is NULL");
  DIT_REQUIRE(q_row_stride >= (int64_t)n_heads * head_dim && kv_row_stride >= (int64_t)n_heads * head_dim, DIT_ERR_INVALID_ARG,
              "row strides smaller than H*d");
  if (n_q == 0) return DIT_OK;
  const size_t es = dtype == DIT_F32 ? 4 : 2;
  const size_t o_bytes = align256((size_t)n_q * n_heads * head_dim * es);   // one partial output
  const size_t l_bytes = align256((size_t)n_q * n_heads * 4);               // one partial LSE
  const size_t need = (size_t)split_p * (o_bytes + l_bytes);
  DIT_REQUIRE(need <= DIT_STATIC_SCRATCH_BYTES, DIT_ERR_WORKSPACE,
              "dit_attn_split_static: %d partials of %d x %d x %d need %zu bytes of scratch, the static array holds %u "
              "(use dit_attn_partial + dit_attn_merge with caller memory)",
              split_p, n_q, n_heads, head_dim, need, DIT_STATIC_SCRATCH_BYTES);
  unsigned char* base = nullptr;
  dit_status s = device_scratch(&base);
  if (s != DIT_OK) return s;
  cudaStream_t st = (cudaStream_t)stream;
  AttnArgs a;
  a.q = q; a.k = k; a.v = v; a.q_stride = q_row_stride; a.kv_stride = kv_row_stride;
  a.o_stride = (int64_t)n_heads * head_dim;
  a.cu_q = a.cu_k = nullptr; a.cu_q_host = a.cu_k_host = nullptr;
  a.R = 1; a.n_q = n_q; a.n_k = n_k; a.H = n_heads; a.d = head_dim; a.scale = softmax_scale; a.n_shards = split_p;
  const void* op[8];
  const float* lp[8];
  for (int p = 0; p < split_p; ++p) {
    a.o = base + (size_t)p * o_bytes;
    a.lse = (float*)(base + (size_t)split_p * o_bytes + (size_t)p * l_bytes);
    a.shard = p;
    op[p] = a.o; lp[p] = a.lse;
    if (dtype == DIT_BF16) {
      DIT_REQUIRE(attn_tc_supported(a), DIT_ERR_UNSUPPORTED,
                  "dit_attn_split_static (bf16): head_dim 128, strides multiples of 8, 16-byte aligned pointers");
      s = launch_attn_tc(a, st);
    } else {
      s = launch_attn_simt(dtype, a, st);
    }
    if (s != DIT_OK) return s;
  }
  return launch_merge(dtype, op, lp, split_p, (int64_t)n_q * n_heads, head_dim, o, lse_out, st);
}

}  // extern "C"
