// common.cuh — shared device/host helpers of libdit_b200 (CUDA path only; the oracle shares nothing with it).
#pragma once
#include <atomic>
#include <utility>
#include <cuda_bf16.h>
#include <cuda_runtime.h>
#include <stdint.h>

#include "../../include/dit.h"

namespace dit {

typedef __nv_bfloat16 bf16;

// launch accounting (dit_kernel_launches); g_fallback_launches counts bf16 GEMM / attention launches that did NOT take
// the tcgen05 path (dit_fallback_launches): the FFMA kernels are the fp32 path, never a silent substitute for bf16
extern std::atomic<int> g_launches;
extern std::atomic<int> g_fallback_launches;
void set_error(const char* fmt, ...);
const char* get_error();

#define DIT_CUDA_OK(expr)                                                                       \
  do {                                                                                          \
    cudaError_t _e = (expr);                                                                    \
    if (_e != cudaSuccess) {                                                                    \
      dit::set_error("%s failed: %s (%s:%d)", #expr, cudaGetErrorString(_e), __FILE__, __LINE__); \
      return DIT_ERR_CUDA;                                                                      \
    }                                                                                           \
  } while (0)

#define DIT_LAUNCH_CHECK()                                                                  \
  do {                                                                                      \
    dit::g_launches++;                                                                      \
    cudaError_t _e = cudaPeekAtLastError();                                                 \
    if (_e != cudaSuccess) {                                                                \
      (void)cudaGetLastError();                                                             \
      dit::set_error("kernel launch failed: %s (%s:%d)", cudaGetErrorString(_e), __FILE__, __LINE__); \
      return DIT_ERR_CUDA;                                                                  \
    }                                                                                       \
  } while (0)

#define DIT_REQUIRE(cond, status, ...) \
  do {                                 \
    if (!(cond)) {                     \
      dit::set_error(__VA_ARGS__);     \
      return status;                   \
    }                                  \
  } while (0)

static inline int cdiv(int64_t a, int64_t b) { return (int)((a + b - 1) / b); }

// per-class device timing (dit_profile_begin / dit_profile_end): when a class is enabled every launcher of that
// class brackets its launch with a cudaEvent pair on the launching stream.  Off by default (zero overhead).
extern std::atomic<int> g_prof_mask;
extern thread_local int g_prof_class_override;  // >= 0: launchers report this class instead of their own
void prof_record(int cls, cudaStream_t st, bool start);
struct ProfScope {
  int cls;
  cudaStream_t st;
  bool on;
  ProfScope(int c, cudaStream_t s) : cls(g_prof_class_override >= 0 ? g_prof_class_override : c), st(s) {
    on = (g_prof_mask.load(std::memory_order_relaxed) >> cls) & 1;
    if (on) prof_record(cls, st, true);
  }
  ~ProfScope() {
    if (on) prof_record(cls, st, false);
  }
};

// ---------------------------------------------------------------------------------------------
// Programmatic dependent launch (PDL): a kernel launched with the programmatic-stream-serialisation attribute may
// become resident while its predecessor drains; it runs its private prologue (barrier init, TMEM allocation,
// descriptor prefetch) and then blocks in pdl_wait() until the predecessor grid has completed and its writes are
// visible.  Every kernel below calls pdl_trigger() first (lets ITS successor do the same) and pdl_wait() before its
// first access to global data.  Without the launch attribute both are no-ops.  DIT_NO_PDL=1 disables the attribute.
// ---------------------------------------------------------------------------------------------
__device__ __forceinline__ void pdl_trigger() { asm volatile("griddepcontrol.launch_dependents;" ::: "memory"); }
__device__ __forceinline__ void pdl_wait() { asm volatile("griddepcontrol.wait;" ::: "memory"); }
bool pdl_enabled();   // dit.cu

template <typename... KArgs, typename... Args>
inline cudaError_t launch_pdl(void (*kernel)(KArgs...), dim3 grid, dim3 block, size_t smem, cudaStream_t st, int cluster_x,
                              Args&&... args) {
  cudaLaunchConfig_t cfg = {};
  cfg.gridDim = grid;
  cfg.blockDim = block;
  cfg.dynamicSmemBytes = smem;
  cfg.stream = st;
  cudaLaunchAttribute attr[2];
  int n = 0;
  if (cluster_x > 1) {
    attr[n].id = cudaLaunchAttributeClusterDimension;
    attr[n].val.clusterDim.x = cluster_x; attr[n].val.clusterDim.y = 1; attr[n].val.clusterDim.z = 1;
    ++n;
  }
  if (pdl_enabled()) {
    attr[n].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[n].val.programmaticStreamSerializationAllowed = 1;
    ++n;
  }
  cfg.attrs = attr;
  cfg.numAttrs = n;
  return cudaLaunchKernelEx(&cfg, kernel, KArgs(std::forward<Args>(args))...);
}

// ---------------------------------------------------------------------------------------------
// 128-bit vector access: 8 consecutive elements of T <-> 8 floats
// ---------------------------------------------------------------------------------------------
__device__ __forceinline__ float bf16lo(uint32_t u) { return __uint_as_float(u << 16); }
__device__ __forceinline__ float bf16hi(uint32_t u) { return __uint_as_float(u & 0xffff0000u); }
__device__ __forceinline__ uint32_t pack_bf16(float a, float b) {
  __nv_bfloat162 t = __floats2bfloat162_rn(a, b);
  return *reinterpret_cast<uint32_t*>(&t);
}

template <typename T>
__device__ __forceinline__ void ld8(const T* p, float v[8]);
template <>
__device__ __forceinline__ void ld8<float>(const float* p, float v[8]) {
  float4 a = *reinterpret_cast<const float4*>(p), b = *reinterpret_cast<const float4*>(p + 4);
  v[0] = a.x; v[1] = a.y; v[2] = a.z; v[3] = a.w; v[4] = b.x; v[5] = b.y; v[6] = b.z; v[7] = b.w;
}
template <>
__device__ __forceinline__ void ld8<bf16>(const bf16* p, float v[8]) {
  uint4 a = *reinterpret_cast<const uint4*>(p);
  v[0] = bf16lo(a.x); v[1] = bf16hi(a.x); v[2] = bf16lo(a.y); v[3] = bf16hi(a.y);
  v[4] = bf16lo(a.z); v[5] = bf16hi(a.z); v[6] = bf16lo(a.w); v[7] = bf16hi(a.w);
}
// streaming variant for data read exactly once (weights of a GEMV): bypass L1, evict-first in L2
template <typename T>
__device__ __forceinline__ void ld8_stream(const T* p, float v[8]);
template <>
__device__ __forceinline__ void ld8_stream<float>(const float* p, float v[8]) {
  float4 a = __ldcs(reinterpret_cast<const float4*>(p)), b = __ldcs(reinterpret_cast<const float4*>(p + 4));
  v[0] = a.x; v[1] = a.y; v[2] = a.z; v[3] = a.w; v[4] = b.x; v[5] = b.y; v[6] = b.z; v[7] = b.w;
}
template <>
__device__ __forceinline__ void ld8_stream<bf16>(const bf16* p, float v[8]) {
  uint4 a = __ldcs(reinterpret_cast<const uint4*>(p));
  v[0] = bf16lo(a.x); v[1] = bf16hi(a.x); v[2] = bf16lo(a.y); v[3] = bf16hi(a.y);
  v[4] = bf16lo(a.z); v[5] = bf16hi(a.z); v[6] = bf16lo(a.w); v[7] = bf16hi(a.w);
}
template <typename T>
__device__ __forceinline__ void st8(T* p, const float v[8]);
template <>
__device__ __forceinline__ void st8<float>(float* p, const float v[8]) {
  *reinterpret_cast<float4*>(p) = make_float4(v[0], v[1], v[2], v[3]);
  *reinterpret_cast<float4*>(p + 4) = make_float4(v[4], v[5], v[6], v[7]);
}
template <>
__device__ __forceinline__ void st8<bf16>(bf16* p, const float v[8]) {
  uint4 a;
  a.x = pack_bf16(v[0], v[1]); a.y = pack_bf16(v[2], v[3]); a.z = pack_bf16(v[4], v[5]); a.w = pack_bf16(v[6], v[7]);
  *reinterpret_cast<uint4*>(p) = a;
}

template <typename T> __device__ __forceinline__ float to_f(T v);
template <> __device__ __forceinline__ float to_f<float>(float v) { return v; }
template <> __device__ __forceinline__ float to_f<bf16>(bf16 v) { return __bfloat162float(v); }
template <typename T> __device__ __forceinline__ T from_f(float v);
template <> __device__ __forceinline__ float from_f<float>(float v) { return v; }
template <> __device__ __forceinline__ bf16 from_f<bf16>(float v) { return __float2bfloat16_rn(v); }

__device__ __forceinline__ float warp_sum(float v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
  return v;
}

// row -> request through cu_seqlens (R <= 64: linear scan, warp-uniform)
__device__ __forceinline__ int find_request(const int32_t* __restrict__ cu, int R, int row) {
  int r = 0;
  while (r + 1 < R && row >= cu[r + 1]) ++r;
  return r;
}

__device__ __forceinline__ float gelu_tanh_f(float z) {
  // 0.5 z (1 + tanh(0.79788456 (z + 0.044715 z^3)))   (DESIGN.md §3 step 5); accurate tanhf, not the approx one
  float t = tanhf(0.7978845608028654f * (z + 0.044715f * z * z * z));
  return 0.5f * z * (1.0f + t);
}
__device__ __forceinline__ float silu_f(float z) { return z / (1.0f + expf(-z)); }

// ---------------------------------------------------------------------------------------------
// internal launchers (implemented across the .cu files); every one enqueues on `st`
// ---------------------------------------------------------------------------------------------
struct SeqMeta {        // one per request, device resident
  int32_t seq_start;    // first row of the request in the packed sequence
  int32_t n_cond;       // joint-mode cond rows at the head of the segment (0 otherwise)
  int32_t gf, gh, gw;   // token grid (F', H', W')
  int32_t lat_off_lo, lat_off_hi;  // element offset of the request's latent in the packed latents (64-bit split)
  int32_t pad;
};

struct GemvBatch {      // one per weight matrix of a batched GEMV
  const void* W;
  const void* b;
  int32_t N;
  int32_t out_off;      // column offset inside an output row
  int32_t row_begin;    // first flattened row index of this matrix
  int32_t pad;
};

dit_status launch_gemv(int dtype, const float* in, const GemvBatch* batches_dev, const GemvBatch* single, int n_batches,
                       int total_rows, float* out, int64_t out_stride, int R, int K, int silu_input, cudaStream_t st);
// split != 0 (bf16 only): y is [T, 2D] = [hi | lo], y = hi + lo to ~16 bits (the final layer's input, R36)
dit_status launch_adaln(int dtype, float* x, const void* h, const float* gate, const float* shift, const float* scale,
                        int64_t mod_stride, const int32_t* cu, int R, void* y, int T, int D, float eps, cudaStream_t st,
                        int split = 0, int64_t set_off = 0);   // set_off != 0: cu = R row segments, text | image alternating (R37)
dit_status launch_qknorm_rope(int dtype, void* qkv, int64_t row_stride, int T, int H, int d, int n_tensors,
                              const void* gq, const void* gk, float eps, const float* rc, const float* rs,
                              cudaStream_t st);
dit_status launch_rope_table(const SeqMeta* meta, int R, int T, int d, const int32_t rope_dims[3], float theta,
                             float* rc, float* rs, cudaStream_t st);
dit_status launch_silu_split(const float* c, void* out, int R, int D, cudaStream_t st);
dit_status launch_scatter_cond_rows(const float* src, float* x, const int32_t* cu_dev, const int32_t* cu_cond_dev, int R,
                                    int Lc_total, int D, cudaStream_t st);
dit_status launch_patchify_varlen(int dtype, const void* lat, void* patches, const SeqMeta* meta_dev, int R, int64_t max_elems,
                                  int C, const int32_t patch[3], cudaStream_t st);
dit_status launch_unpatchify_varlen(int dtype, const float* tok, void* out, const SeqMeta* meta_dev, int R, int64_t max_elems,
                                    int C, const int32_t patch[3], cudaStream_t st);
dit_status launch_patchify(int dtype, const void* lat, void* patches, int C, int F, int H, int W, const int32_t patch[3],
                           cudaStream_t st);
// Sampler epilogue of the unpatchify kernel (dit_sample).  mode 0: out = v.  mode 1: v_hold = v (fp32, no out).
// mode 2: v' = v_hold ? v_hold + guidance (v - v_hold) : v;  state += dsigma v';  out = state.
struct SampleEpi {
  int mode;
  float* state;
  float* v_hold;
  float dsigma, guidance;
};
dit_status launch_unpatchify(int dtype, const float* tok, void* out, int C, int F, int H, int W, const int32_t patch[3],
                             cudaStream_t st, const SampleEpi* epi = nullptr);
dit_status launch_sample_init(int dtype, const void* lat, float* state, int64_t n, cudaStream_t st);
dit_status launch_sample_final(int dtype, const float* state, void* out, int64_t n, cudaStream_t st);
dit_status launch_merge(int dtype, const void* const* o_parts, const float* const* lses, int P, int64_t n_rows_heads,
                        int d, void* o, float* lse_out, cudaStream_t st);

// GEMM: out[M,N] = epi(A[M,K] W[N,K]^T + bias).  *_simt works for both dtypes; *_tc is the tcgen05 path (bf16).
// epi 3 (DIT_EPI_GATE_RESIDUAL): out fp32 [M, ldo] <- out + gate[req(row)] (.) (A W^T + bias)
dit_status launch_gemm_simt(int dtype, int epi, const void* A, int64_t lda, const void* W, const void* bias, void* out,
                            int64_t ldo, int M, int N, int K, cudaStream_t st, const float* gate = nullptr,
                            int64_t gate_stride = 0, const int32_t* cu = nullptr, int R = 1);
// epi 5 (split): out bf16 [M, 2N] = [hi | lo] of A W^T + bias.  a_split != 0: A is such a [hi | lo] pair, [M, 2K]
dit_status launch_gemm_tc(int epi, const void* A, int64_t lda, const void* W, const void* bias, void* out, int64_t ldo,
                          int M, int N, int K, cudaStream_t st, int a_split = 0);
// epi 3: the gated residual fused in the epilogue (gate nullptr = 1; cu nullptr = one request)
dit_status launch_gemm_tc_ex(int epi, const void* A, int64_t lda, const void* W, const void* bias, void* out, int64_t ldo,
                             const float* gate, int64_t gate_stride, const int32_t* cu, int R, int M, int N, int K,
                             cudaStream_t st, int a_split = 0);
// Projection + QK-RMSNorm + RoPE in one kernel (bf16, head_dim 128): out [M, N] holds normalised, rotated q heads in columns
// [0, q_end), k heads in [q_end, k_end), plain v heads behind them (self-attention: D, 2D, N = 3D)
dit_status launch_gemm_tc_qkv(const void* A, int64_t lda, const void* W, const void* bias, void* out, int64_t ldo,
                              const void* gq, const void* gk, float rms_eps, const float* rc, const float* rs, int q_end,
                              int k_end, int M, int N, int K, cudaStream_t st, int a_split = 0);
// Row-segmented ("grouped") tcgen05 GEMM for the dual-stream blocks (R37): A and out are ONE packed [M, .] buffer whose rows
// fall into segments (a request's text rows, its image rows); a segment uses weight set `which` (0 = image, 1 = text) and
// the gate row of request `req`.  One launch covers every segment: a 256-row tile pair never straddles a segment.
constexpr int GEMM_MAX_SEGS = 128;
struct GemmSegs {
  int n;                              // 0: not segmented
  int tile0[GEMM_MAX_SEGS + 1];       // first row-tile pair of segment i (prefix sum of ceil(rows / 256))
  int row0[GEMM_MAX_SEGS];
  int rows[GEMM_MAX_SEGS];            // > 0
  uint8_t which[GEMM_MAX_SEGS];
  uint8_t req[GEMM_MAX_SEGS];
};
struct SegGemm {
  int kind;                           // 0 bias, 1 bias + GELU, 3 gated residual, 4 QKV (+ norm / RoPE), 6 SwiGLU
  const void* A; int64_t lda; void* out; int64_t ldo; int M, N, K;
  const GemmSegs* segs;
  const void* W[2]; const void* bias[2];        // per weight set
  const void* W3[2]; const void* b3[2];         // SwiGLU
  const void* gq[2]; const void* gk[2]; float rms_eps; const float* rc; const float* rs;   // QKV (rc / rs: [M, 64] of the packed rows)
  const float* gate; int64_t gate_stride; int64_t gate_set_off;   // gated residual: gate row = gate + req * stride + which * set_off
};
dit_status launch_gemm_tc_segs(const SegGemm& g, cudaStream_t st);
// Gated-MLP up-projection (R40): out bf16 [M, ldo] <- SiLU(A W1^T + b1) (.) (A W3^T + b3), one kernel (tcgen05)
dit_status launch_gemm_tc_swiglu(const void* A, int64_t lda, const void* W1, const void* b1, const void* W3, const void* b3,
                                 void* out, int64_t ldo, int M, int N, int K, cudaStream_t st);
// fp8 (e4m3) linear layer with fp32 row scales on both operands (R42)
dit_status launch_gemm_tc_fp8(int epi, const void* Aq, int64_t lda, const float* a_scale, const void* Wq, const float* w_scale,
                              const void* bias, void* out, int64_t ldo, int M, int N, int K, cudaStream_t st);
// block-scaled MXFP8 layer on the pair kernel (R43)
dit_status launch_gemm_tc_mx(int epi, const void* Aq, int64_t lda, const void* sfa, const void* Wq, const void* sfw, const void* bias,
                             void* out, int64_t ldo, int M, int N, int K, cudaStream_t st);
// rows of x [M, K] (ldx elements) -> e4m3 codes [M, ldq bytes] + fp32 row scales (R42: scale = amax / 448, RN-even, saturating)
dit_status launch_quantize_fp8(int dtype, const void* x, int64_t ldx, int M, int K, void* q, int64_t ldq, float* scale, cudaStream_t st);
dit_status launch_silu_mul(int dtype, void* u, const void* u3, int64_t n, cudaStream_t st);   // u <- SiLU(u) (.) u3 (FFMA path)
bool gemm_tc_supported(int epi, const void* A, int64_t lda, const void* W, void* out, int64_t ldo, int M, int N, int K);

// Attention over packed sequences.  q rows [cu_q[r], cu_q[r+1]) attend to k/v rows [cu_k[r], cu_k[r+1])
// restricted to shard `shard` of `n_shards` (contiguous, size ceil(len/n_shards), R20).
struct AttnArgs {
  const void* q; const void* k; const void* v;
  int64_t q_stride, kv_stride;     // row strides in elements
  void* o; int64_t o_stride;
  float* lse;                      // [rows, H] or nullptr
  const int32_t* cu_q; const int32_t* cu_k;   // device, [R+1]; nullptr => single request [0, n_q) x [0, n_k)
  const int32_t* cu_q_host; const int32_t* cu_k_host;
  int R; int n_q; int n_k;         // totals
  int H; int d;
  float scale;
  int shard, n_shards;
};
dit_status launch_attn_simt(int dtype, const AttnArgs& a, cudaStream_t st);
dit_status launch_attn_tc(const AttnArgs& a, cudaStream_t st);
bool attn_tc_supported(const AttnArgs& a);

}  // namespace dit
