// elementwise.cu — the HBM-bound kernels of the DiT step: weight-streaming GEMV (t-MLP, modulation),
// adaLN-Zero modulation (LayerNorm + shift/scale + gated residual), QK-RMSNorm + RoPE, RoPE tables,
// patchify / unpatchify, LSE merge.  All 128-bit coalesced global access, warp-shuffle reductions.
#include <algorithm>
#include <cstdlib>
#include <cstring>

#include "common.cuh"
#include "tc.cuh"   // mbarrier helpers (adaln_stream_kernel)

namespace dit {

// =================================================================================================
// GEMV:  out[r, off_b + n] = sum_k act(in[r,k]) W_b[n,k] + bias_b[n]      (DESIGN.md §3 steps 1-2)
// Roofline: HBM, weights are streamed exactly once (N*K*sizeof(T) bytes); `in` lives in shared memory.
// A warp owns 4 weight rows at a time so every staged input fragment is reused 4x from registers (keeps
// shared-memory traffic at R/2 bytes per weight byte); the K loop is unrolled twice, so a lane has 8 independent
// 16-byte loads in flight and a resident SM (4 CTAs x 8 warps) about 128 KB — HBM latency x bandwidth needs ~45 KB.
// The batch table (one entry per weight matrix) is copied to shared memory once per CTA.
// =================================================================================================
constexpr int GEMV_MAX_BATCHES = 264;   // n_blocks <= 256 (+ final layer)

template <typename T, int RMAX>
__global__ void __launch_bounds__(256) gemv_kernel(const float* __restrict__ in, const GemvBatch* __restrict__ batches,
                                                   const GemvBatch single, int n_batches, int total_rows,
                                                   float* __restrict__ out, int64_t out_stride, int R, int K,
                                                   int silu_input) {
  pdl_trigger();
  pdl_wait();
  extern __shared__ float s_in[];  // [R][K], then the batch table
  GemvBatch* s_b = reinterpret_cast<GemvBatch*>(s_in + (size_t)R * K);
  for (int i = threadIdx.x; i < n_batches; i += blockDim.x) s_b[i] = batches != nullptr ? batches[i] : single;
  for (int i = threadIdx.x; i < R * K; i += blockDim.x) {
    float v = in[i];
    s_in[i] = silu_input ? silu_f(v) : v;
  }
  __syncthreads();
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const int warps_total = gridDim.x * (blockDim.x >> 5);
  // balanced static partition: warp w streams the contiguous rows [w N / W, (w + 1) N / W) — row counts differ by
  // at most one, so the last wave is not a quarter empty as with a strided loop over 4-row groups
  const int wid = blockIdx.x * (blockDim.x >> 5) + warp;
  const int r_begin = (int)((int64_t)wid * total_rows / warps_total);
  const int r_end = (int)((int64_t)(wid + 1) * total_rows / warps_total);
  for (int g0 = r_begin; g0 < r_end; g0 += 4) {
    const T* wrow[4];
    bool valid[4];
    int bidx[4], nloc[4];
#pragma unroll
    for (int j = 0; j < 4; ++j) {
      int row = g0 + j;
      valid[j] = row < r_end;
      if (!valid[j]) row = r_end - 1;
      int b = 0;
      while (b + 1 < n_batches && row >= s_b[b + 1].row_begin) ++b;
      bidx[j] = b;
      nloc[j] = row - s_b[b].row_begin;
      wrow[j] = reinterpret_cast<const T*>(s_b[b].W) + (int64_t)nloc[j] * K;
    }
    float acc[4][RMAX];
#pragma unroll
    for (int j = 0; j < 4; ++j)
#pragma unroll
      for (int r = 0; r < RMAX; ++r) acc[j][r] = 0.f;
#pragma unroll 2
    for (int k0 = lane * 8; k0 < K; k0 += 256) {
      float w[4][8];
#pragma unroll
      for (int j = 0; j < 4; ++j) ld8_stream<T>(wrow[j] + k0, w[j]);
#pragma unroll
      for (int r = 0; r < RMAX; ++r) {
        if (r < R) {
          float xin[8];
          ld8<float>(s_in + r * K + k0, xin);
#pragma unroll
          for (int j = 0; j < 4; ++j)
#pragma unroll
            for (int e = 0; e < 8; ++e) acc[j][r] = fmaf(w[j][e], xin[e], acc[j][r]);
        }
      }
    }
#pragma unroll
    for (int j = 0; j < 4; ++j)
#pragma unroll
      for (int r = 0; r < RMAX; ++r) acc[j][r] = warp_sum(acc[j][r]);
    if (lane == 0) {
#pragma unroll
      for (int j = 0; j < 4; ++j) {
        if (!valid[j]) continue;
        const GemvBatch& B = s_b[bidx[j]];
        float bias = B.b ? to_f<T>(reinterpret_cast<const T*>(B.b)[nloc[j]]) : 0.f;
#pragma unroll
        for (int r = 0; r < RMAX; ++r)
          if (r < R) out[(int64_t)r * out_stride + B.out_off + nloc[j]] = acc[j][r] + bias;
      }
    }
  }
}

template <typename T>
static dit_status launch_gemv_t(const float* in, const GemvBatch* batches, const GemvBatch& single, int n_batches,
                                int total_rows, float* out, int64_t out_stride, int R, int K, int silu_input,
                                cudaStream_t st) {
  DIT_REQUIRE(K % 8 == 0, DIT_ERR_UNSUPPORTED, "gemv: K=%d must be a multiple of 8", K);
  DIT_REQUIRE(n_batches >= 1 && n_batches <= GEMV_MAX_BATCHES, DIT_ERR_UNSUPPORTED, "gemv: %d matrices (max %d)", n_batches,
              GEMV_MAX_BATCHES);
  ProfScope _prof(DIT_KC_GEMV, st);
  int dev = 0, sms = 148;
  cudaGetDevice(&dev);
  cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
  // requests are processed RMAX at a time (weights re-streamed per chunk only when R > 8)
  for (int r0 = 0; r0 < R; r0 += 8) {
    int rc = R - r0 < 8 ? R - r0 : 8;
    size_t smem = (size_t)rc * K * sizeof(float) + (size_t)n_batches * sizeof(GemvBatch);
    int ctas = (total_rows + 63) / 64;   // at least 8 rows per warp
    int per_sm = 1;   // exactly one resident wave: the partition is static, a partial second wave would be idle time
    const float* inr = in + (int64_t)r0 * K;
    float* outr = out + (int64_t)r0 * out_stride;
#define GEMV_LAUNCH(RM)                                                                                         \
  {                                                                                                             \
    DIT_CUDA_OK(cudaFuncSetAttribute(gemv_kernel<T, RM>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem)); \
    DIT_CUDA_OK(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, gemv_kernel<T, RM>, 256, smem));          \
    if (per_sm < 1) per_sm = 1;                                                                                 \
    if (ctas > sms * per_sm) ctas = sms * per_sm;                                                               \
    DIT_CUDA_OK(launch_pdl(gemv_kernel<T, RM>, dim3(ctas), dim3(256), smem, st, 1, inr, batches, single, n_batches,     \
                           total_rows, outr, out_stride, rc, K, silu_input));                                   \
  }
    DIT_REQUIRE(smem <= 200 * 1024, DIT_ERR_UNSUPPORTED, "gemv: R*K too large for shared memory");
    if (rc == 1) GEMV_LAUNCH(1) else if (rc == 2) GEMV_LAUNCH(2) else if (rc <= 4) GEMV_LAUNCH(4) else GEMV_LAUNCH(8)
#undef GEMV_LAUNCH
    DIT_LAUNCH_CHECK();
  }
  return DIT_OK;
}

// batches_dev == nullptr: one matrix, described by `single` (travels as a kernel parameter)
dit_status launch_gemv(int dtype, const float* in, const GemvBatch* batches_dev, const GemvBatch* single, int n_batches,
                       int total_rows, float* out, int64_t out_stride, int R, int K, int silu_input, cudaStream_t st) {
  GemvBatch one = single ? *single : GemvBatch{nullptr, nullptr, 0, 0, 0, 0};
  if (dtype == DIT_F32)
    return launch_gemv_t<float>(in, batches_dev, one, n_batches, total_rows, out, out_stride, R, K, silu_input, st);
  return launch_gemv_t<bf16>(in, batches_dev, one, n_batches, total_rows, out, out_stride, R, K, silu_input, st);
}

// =================================================================================================
// adaLN-Zero modulation (north_star subsystem 2; DESIGN.md §3 step 5):
//   x <- x + gate (.) h   (optional);   y = LN(x) (.) (1 + scale) + shift
// WPR warps per row (1, 2 or 4), the whole row in registers (NCW chunks of 8 elements per lane and warp: at most 48
// data registers, so 8+ CTAs of 128 threads stay resident and a row's 12-20 KB is in flight at once), two-pass
// statistics: warp shuffles, then WPR partial sums through shared memory.  Algorithmic bytes per token: 4D (x) +
// 2D (y) [+ 2D (h) + 4D (x write)].
// =================================================================================================
template <typename T, int NCW, int WPR>
__global__ void __launch_bounds__(128) adaln_kernel(float* __restrict__ x, const T* __restrict__ h,
                                                    const float* __restrict__ gate, const float* __restrict__ shift,
                                                    const float* __restrict__ scale, int64_t mod_stride,
                                                    const int32_t* __restrict__ cu, int R, T* __restrict__ y, int T_rows,
                                                    float eps, int split, int64_t set_off) {
  pdl_trigger();
  pdl_wait();
  constexpr int D = NCW * WPR * 256;
  constexpr int RPB = 4 / WPR;                       // rows per block
  __shared__ float red[2][4];
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const int sub = warp % WPR;                        // which slice of the row this warp owns
  const int row_raw = blockIdx.x * RPB + warp / WPR;
  const bool row_ok = row_raw < T_rows;
  const int row = row_ok ? row_raw : T_rows - 1;     // out-of-range warps redo the last row and store nothing
  // set_off != 0 (dual-stream blocks, R37): `cu` holds the R row SEGMENTS [text of request 0 | image of request 0 | text of
  // request 1 | ...]; an even (text) segment takes the modulation row at + set_off
  const int seg = (cu != nullptr && R > 1) ? find_request(cu, R, row) : 0;
  const int64_t moff = set_off != 0 ? (int64_t)(seg >> 1) * mod_stride + ((seg & 1) ? 0 : set_off) : (int64_t)seg * mod_stride;
  const int col0 = sub * (NCW * 256) + lane * 8;     // chunk c of this lane starts at col0 + c * 256
  float* xr = x + (int64_t)row * D + col0;
  float v[NCW][8];
#pragma unroll
  for (int c = 0; c < NCW; ++c) ld8<float>(xr + c * 256, v[c]);
  if (h != nullptr) {
    const T* hr = h + (int64_t)row * D + col0;
    const float* g = gate ? gate + moff + col0 : nullptr;
#pragma unroll
    for (int c = 0; c < NCW; ++c) {
      float hv[8], gv[8];
      ld8<T>(hr + c * 256, hv);
      if (g) ld8<float>(g + c * 256, gv);
#pragma unroll
      for (int e = 0; e < 8; ++e) v[c][e] = g ? fmaf(gv[e], hv[e], v[c][e]) : v[c][e] + hv[e];
      if (row_ok) st8<float>(xr + c * 256, v[c]);
    }
  }
  float s = 0.f;
#pragma unroll
  for (int c = 0; c < NCW; ++c)
#pragma unroll
    for (int e = 0; e < 8; ++e) s += v[c][e];
  s = warp_sum(s);
  if (WPR > 1) {
    if (lane == 0) red[0][warp] = s;
    __syncthreads();
    s = 0.f;
#pragma unroll
    for (int i = 0; i < WPR; ++i) s += red[0][(warp / WPR) * WPR + i];
  }
  const float mean = s * (1.0f / D);
  float q = 0.f;
#pragma unroll
  for (int c = 0; c < NCW; ++c)
#pragma unroll
    for (int e = 0; e < 8; ++e) {
      float dlt = v[c][e] - mean;
      q = fmaf(dlt, dlt, q);
    }
  q = warp_sum(q);
  if (WPR > 1) {
    if (lane == 0) red[1][warp] = q;
    __syncthreads();
    q = 0.f;
#pragma unroll
    for (int i = 0; i < WPR; ++i) q += red[1][(warp / WPR) * WPR + i];
  }
  const float rstd = rsqrtf(q * (1.0f / D) + eps);
  const float* sh = shift ? shift + moff + col0 : nullptr;
  const float* sc = scale ? scale + moff + col0 : nullptr;
  T* yr = y + (int64_t)row * (split ? 2 * D : D) + col0;   // split: row = [hi (D) | lo (D)]
#pragma unroll
  for (int c = 0; c < NCW; ++c) {
    float o[8], a[8], b[8];
    if (sc) ld8<float>(sc + c * 256, a);
    if (sh) ld8<float>(sh + c * 256, b);
#pragma unroll
    for (int e = 0; e < 8; ++e) {
      float n = (v[c][e] - mean) * rstd;
      if (sc) n = fmaf(n, a[e], n);
      if (sh) n += b[e];
      o[e] = n;
    }
    if (row_ok) st8<T>(yr + c * 256, o);
    if (split && row_ok) {   // lo = y - hi, exact in fp32, rounded to T once more
      float lo[8];
#pragma unroll
      for (int e = 0; e < 8; ++e) lo[e] = o[e] - to_f<T>(from_f<T>(o[e]));
      st8<T>(yr + D + c * 256, lo);
    }
  }
}

// -------------------------------------------------------------------------------------------------
// The same operation (without the h / gate residual) for launches of a few waves: a PERSISTENT grid (resident CTAs only),
// every CTA walks its rows (strided or contiguous, see below) and keeps STAGES rows in flight in shared memory with 1-D bulk copies
// (cp.async.bulk + mbarrier): the bytes in flight per SM no longer depend on registers or on how many CTAs have been
// launched yet, and there is no wave tail — at cfg 2 (4352 rows of 12 KB) the one-row-per-CTA kernel above is 3.3 waves of
// load -> reduce -> load modulation -> store chains.  128 threads per row, NCT = D / 1024 chunks of 8 per thread; the
// modulation rows stay in registers and are reloaded only when the request (segment) changes.
// -------------------------------------------------------------------------------------------------
constexpr int ADALN_STAGES = 3;

__device__ __forceinline__ void bulk_load_1d(uint32_t dst, const void* src, uint32_t bytes, uint32_t bar) {
  asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(dst), "l"(src),
               "r"(bytes), "r"(bar)
               : "memory");
}

template <typename T, int NCT>
__global__ void __launch_bounds__(128) adaln_stream_kernel(const float* __restrict__ x, const float* __restrict__ shift,
                                                           const float* __restrict__ scale, int64_t mod_stride,
                                                           const int32_t* __restrict__ cu, int R, T* __restrict__ y,
                                                           int T_rows, float eps, int split, int64_t set_off) {
  constexpr int D = NCT * 1024;
  extern __shared__ __align__(128) unsigned char adaln_smem[];
  float* stage = reinterpret_cast<float*>(adaln_smem);                       // [STAGES][D]
  __shared__ __align__(8) uint64_t full[ADALN_STAGES];
  __shared__ float red[2][4];
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  // One request: CTA b walks rows b, b + G, b + 2G ... (the CTAs read one moving window of the matrix).  Several requests: CTA b owns
  // the CONTIGUOUS rows [b T / G, (b + 1) T / G) — it crosses a request boundary at most a few times, so the modulation rows are
  // reloaded and the request looked up rarely (the strided walk changed request at every row of a many-request batch: 2.4x slower
  // at 64 requests, 15 % at cfg 4's six)
  const int G = gridDim.x, b = blockIdx.x;
  const bool multi = cu != nullptr && R > 1;
  const int row_begin = multi ? (int)((int64_t)b * T_rows / G) : b;
  const int row_step = multi ? 1 : G;
  const int n_my = multi ? (int)((int64_t)(b + 1) * T_rows / G) - row_begin : (b < T_rows ? (T_rows - b + G - 1) / G : 0);
  if (tid == 0) {
    for (int s = 0; s < ADALN_STAGES; ++s) tc::mbar_init(tc::smem_u32(&full[s]), 1);
    tc::fence_barrier_init();
  }
  pdl_trigger();
  pdl_wait();                                                                 // x and the modulation rows come from earlier kernels
  if (tid == 0) {
    for (int s = 0; s < ADALN_STAGES && s < n_my; ++s) {
      tc::mbar_expect_tx(tc::smem_u32(&full[s]), D * 4);
      bulk_load_1d(tc::smem_u32(stage + (size_t)s * D), x + (int64_t)(row_begin + s * row_step) * D, D * 4, tc::smem_u32(&full[s]));
    }
  }
  __syncthreads();                                                            // barrier init visible to the waiting threads
  const int col0 = tid * 8;                                                   // chunk c of this thread starts at col0 + c * 1024
  float a[NCT][8], sft[NCT][8];
  int64_t cur = -1;
  int seg = multi ? find_request(cu, R, row_begin) : 0;
  for (int i = 0; i < n_my; ++i) {
    const int s = i % ADALN_STAGES;
    const uint32_t ph = (uint32_t)(i / ADALN_STAGES) & 1u;
    const int row = row_begin + i * row_step;
    if (multi)
      while (seg + 1 < R && row >= cu[seg + 1]) ++seg;
    const int64_t moff = set_off != 0 ? (int64_t)(seg >> 1) * mod_stride + ((seg & 1) ? 0 : set_off) : (int64_t)seg * mod_stride;
    if (moff != cur) {                                                        // uniform over the CTA
      cur = moff;
#pragma unroll
      for (int c = 0; c < NCT; ++c) {
        if (scale) ld8<float>(scale + moff + col0 + c * 1024, a[c]);
        if (shift) ld8<float>(shift + moff + col0 + c * 1024, sft[c]);
      }
    }
    tc::mbar_wait(tc::smem_u32(&full[s]), ph);
    const float* xs = stage + (size_t)s * D + col0;
    float v[NCT][8];
#pragma unroll
    for (int c = 0; c < NCT; ++c) {
      const float4 lo = *reinterpret_cast<const float4*>(xs + c * 1024), hi = *reinterpret_cast<const float4*>(xs + c * 1024 + 4);
      v[c][0] = lo.x; v[c][1] = lo.y; v[c][2] = lo.z; v[c][3] = lo.w;
      v[c][4] = hi.x; v[c][5] = hi.y; v[c][6] = hi.z; v[c][7] = hi.w;
    }
    float sum = 0.f;
#pragma unroll
    for (int c = 0; c < NCT; ++c)
#pragma unroll
      for (int e = 0; e < 8; ++e) sum += v[c][e];
    sum = warp_sum(sum);
    if (lane == 0) red[0][warp] = sum;
    __syncthreads();                                                          // also: every thread has read stage s
    if (tid == 0 && i + ADALN_STAGES < n_my) {
      tc::mbar_expect_tx(tc::smem_u32(&full[s]), D * 4);
      bulk_load_1d(tc::smem_u32(stage + (size_t)s * D), x + (int64_t)(row + ADALN_STAGES * row_step) * D, D * 4,
                   tc::smem_u32(&full[s]));
    }
    const float mean = (red[0][0] + red[0][1] + red[0][2] + red[0][3]) * (1.0f / D);
    float q = 0.f;
#pragma unroll
    for (int c = 0; c < NCT; ++c)
#pragma unroll
      for (int e = 0; e < 8; ++e) {
        float dlt = v[c][e] - mean;
        q = fmaf(dlt, dlt, q);
      }
    q = warp_sum(q);
    if (lane == 0) red[1][warp] = q;
    __syncthreads();
    const float rstd = rsqrtf((red[1][0] + red[1][1] + red[1][2] + red[1][3]) * (1.0f / D) + eps);
    T* yr = y + (int64_t)row * (split ? 2 * D : D) + col0;
#pragma unroll
    for (int c = 0; c < NCT; ++c) {
      float o[8];
#pragma unroll
      for (int e = 0; e < 8; ++e) {
        float n = (v[c][e] - mean) * rstd;
        if (scale) n = fmaf(n, a[c][e], n);
        if (shift) n += sft[c][e];
        o[e] = n;
      }
      st8<T>(yr + c * 1024, o);
      if (split) {
        float lo[8];
#pragma unroll
        for (int e = 0; e < 8; ++e) lo[e] = o[e] - to_f<T>(from_f<T>(o[e]));
        st8<T>(yr + D + c * 1024, lo);
      }
    }
  }
}

template <typename T, int NCT>
static cudaError_t launch_adaln_stream(const float* x, const float* shift, const float* scale, int64_t mod_stride,
                                       const int32_t* cu, int R, T* y, int T_rows, float eps, cudaStream_t st, int split,
                                       int64_t set_off) {
  constexpr int smem = ADALN_STAGES * NCT * 1024 * 4;
  // per device: resident CTAs of this instantiation x SMs (0 = not asked yet; racing first calls compute the same value)
  static std::atomic<int> ctas_per_sm[16];
  int dev = 0;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return e;
  if (dev >= 16) return cudaErrorInvalidDevice;
  if (ctas_per_sm[dev].load(std::memory_order_acquire) == 0) {
    e = cudaFuncSetAttribute(adaln_stream_kernel<T, NCT>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem);
    if (e != cudaSuccess) return e;
    int n = 0;
    e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&n, adaln_stream_kernel<T, NCT>, 128, smem);
    if (e != cudaSuccess) return e;
    int sms = 148;
    e = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    if (e != cudaSuccess) return e;
    ctas_per_sm[dev].store((n > 0 ? n : 1) * sms, std::memory_order_release);
  }
  const int grid = std::min(T_rows, ctas_per_sm[dev].load(std::memory_order_relaxed));
  return launch_pdl(adaln_stream_kernel<T, NCT>, dim3(grid), dim3(128), smem, st, 1, x, shift, scale, mod_stride, cu, R, y,
                    T_rows, eps, split, set_off);
}

static bool adaln_stream_enabled() {
  static const bool on = [] {
    const char* e = std::getenv("DIT_ADALN_KERNEL");
    return !(e && std::strcmp(e, "rows") == 0);
  }();
  return on;
}

template <typename T>
static dit_status launch_adaln_t(float* x, const T* h, const float* gate, const float* shift, const float* scale,
                                 int64_t mod_stride, const int32_t* cu, int R, T* y, int T_rows, int D, float eps,
                                 cudaStream_t st, int split, int64_t set_off) {
  if (T_rows == 0) return DIT_OK;
  DIT_REQUIRE(D % 256 == 0 && D <= 6144, DIT_ERR_UNSUPPORTED, "adaln: D=%d must be a multiple of 256 (<= 6144)", D);
  ProfScope _prof(DIT_KC_ADALN, st);
  // few-wave launches without the residual: the persistent bulk-copy kernel (rows of whole KB; x rows 16-byte aligned)
  if (h == nullptr && D % 1024 == 0 && D / 1024 <= 6 && T_rows >= 592 && ((uintptr_t)x & 15) == 0 && adaln_stream_enabled()) {
    cudaError_t e = cudaSuccess;
    switch (D / 1024) {
      case 1: e = launch_adaln_stream<T, 1>(x, shift, scale, mod_stride, cu, R, y, T_rows, eps, st, split, set_off); break;
      case 2: e = launch_adaln_stream<T, 2>(x, shift, scale, mod_stride, cu, R, y, T_rows, eps, st, split, set_off); break;
      case 3: e = launch_adaln_stream<T, 3>(x, shift, scale, mod_stride, cu, R, y, T_rows, eps, st, split, set_off); break;
      case 4: e = launch_adaln_stream<T, 4>(x, shift, scale, mod_stride, cu, R, y, T_rows, eps, st, split, set_off); break;
      case 5: e = launch_adaln_stream<T, 5>(x, shift, scale, mod_stride, cu, R, y, T_rows, eps, st, split, set_off); break;
      default: e = launch_adaln_stream<T, 6>(x, shift, scale, mod_stride, cu, R, y, T_rows, eps, st, split, set_off); break;
    }
    DIT_CUDA_OK(e);
    DIT_LAUNCH_CHECK();
    return DIT_OK;
  }
#define ADALN_CASE(NCV, NCW, WPR)                                                                           \
  case NCV:                                                                                                 \
    DIT_CUDA_OK(launch_pdl(adaln_kernel<T, NCW, WPR>, dim3(cdiv(T_rows, 4 / WPR)), dim3(128), 0, st, 1, x, h, gate, \
                           shift, scale, mod_stride, cu, R, y, T_rows, eps, split, set_off));                \
    break;
  switch (D / 256) {   // D / 256 chunks per row = NCW per warp x WPR warps
    ADALN_CASE(1, 1, 1) ADALN_CASE(2, 2, 1) ADALN_CASE(3, 3, 1) ADALN_CASE(4, 4, 1) ADALN_CASE(5, 5, 1)
    ADALN_CASE(6, 3, 2) ADALN_CASE(8, 4, 2) ADALN_CASE(10, 5, 2) ADALN_CASE(12, 3, 4) ADALN_CASE(16, 4, 4)
    ADALN_CASE(20, 5, 4) ADALN_CASE(24, 6, 4)
    default:
      DIT_REQUIRE(false, DIT_ERR_UNSUPPORTED, "adaln: D=%d has no instantiation", D);
  }
#undef ADALN_CASE
  DIT_LAUNCH_CHECK();
  return DIT_OK;
}

dit_status launch_adaln(int dtype, float* x, const void* h, const float* gate, const float* shift, const float* scale,
                        int64_t mod_stride, const int32_t* cu, int R, void* y, int T, int D, float eps, cudaStream_t st,
                        int split, int64_t set_off) {
  if (dtype == DIT_F32)
    return launch_adaln_t<float>(x, (const float*)h, gate, shift, scale, mod_stride, cu, R, (float*)y, T, D, eps, st, 0, set_off);
  return launch_adaln_t<bf16>(x, (const bf16*)h, gate, shift, scale, mod_stride, cu, R, (bf16*)y, T, D, eps, st, split, set_off);
}

// =================================================================================================
// QK-RMSNorm + RoPE, in place on the q and k thirds of qkv[T, 3D] (R5, R6).  d/8 lanes own one head row.
// =================================================================================================
template <typename T, int HD>
__global__ void __launch_bounds__(256) qknorm_rope_kernel(T* __restrict__ qkv, int64_t row_stride, int T_rows, int H,
                                                          int n_tensors, const T* __restrict__ gq,
                                                          const T* __restrict__ gk, float eps,
                                                          const float* __restrict__ rc, const float* __restrict__ rs) {
  // The q | k part of a row is n_tensors * D contiguous elements.  A warp pass covers UN consecutive 256-element
  // chunks of one row (32 lanes x 8 elements = 256 / HD head rows each); every load of a pass is issued before
  // its first use, so a lane keeps UN x (16 B data + 32 B table) in flight.
  constexpr int LPH = HD / 8;           // lanes per head row
  constexpr int UN = 4;
  const int lane = threadIdx.x & 31;
  const int D = H * HD;
  const int width = n_tensors * D;      // elements per row that are normalised
  const int cpr = (width + 255) / 256;  // chunks per row
  const int ppr = (cpr + UN - 1) / UN;  // passes per row
  const int64_t n_pass = (int64_t)T_rows * ppr;
  const int64_t warp_id = (int64_t)blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5);
  const int64_t n_warps = (int64_t)gridDim.x * (blockDim.x >> 5);
  const int hoff = (lane % LPH) * 8;    // offset inside the head row
  float gqv[8], gkv[8];
  if (gq != nullptr) ld8<T>(gq + hoff, gqv);
  if (gk != nullptr) ld8<T>(gk + hoff, gkv);
  for (int64_t pass = warp_id; pass < n_pass; pass += n_warps) {
    const int row = (int)(pass / ppr);
    const int c0 = (int)(pass % ppr) * UN;
    T* const rowp = qkv + (int64_t)row * row_stride;
    float v[UN][8];
    bool ok[UN];
#pragma unroll
    for (int u = 0; u < UN; ++u) {
      const int col = (c0 + u) * 256 + lane * 8;
      ok[u] = col < width;
      if (ok[u]) ld8<T>(rowp + col, v[u]);
      else {
#pragma unroll
        for (int e = 0; e < 8; ++e) v[u][e] = 0.f;
      }
    }
    float4 cs, sn4;
    if (rc != nullptr) {   // the table row depends on the token only: one load serves all UN chunks
      cs = *reinterpret_cast<const float4*>(rc + (int64_t)row * (HD / 2) + hoff / 2);
      sn4 = *reinterpret_cast<const float4*>(rs + (int64_t)row * (HD / 2) + hoff / 2);
    }
#pragma unroll
    for (int u = 0; u < UN; ++u) {
      const int col = (c0 + u) * 256 + lane * 8;
      const bool is_q = col < D;                       // tensor 0 = q, tensor 1 = k
      if ((is_q ? gq : gk) != nullptr) {
        float ss = 0.f;
#pragma unroll
        for (int e = 0; e < 8; ++e) ss = fmaf(v[u][e], v[u][e], ss);
#pragma unroll
        for (int o = LPH / 2; o > 0; o >>= 1) ss += __shfl_xor_sync(0xffffffffu, ss, o);
        const float r = rsqrtf(ss * (1.0f / HD) + eps);
#pragma unroll
        for (int e = 0; e < 8; ++e) v[u][e] = v[u][e] * r * (is_q ? gqv[e] : gkv[e]);
      }
      if (rc != nullptr) {
        const float cc[4] = {cs.x, cs.y, cs.z, cs.w}, sn[4] = {sn4.x, sn4.y, sn4.z, sn4.w};
#pragma unroll
        for (int j = 0; j < 4; ++j) {
          const float a = v[u][2 * j], b = v[u][2 * j + 1];
          v[u][2 * j] = a * cc[j] - b * sn[j];
          v[u][2 * j + 1] = a * sn[j] + b * cc[j];
        }
      }
      if (ok[u]) st8<T>(rowp + col, v[u]);
    }
  }
}

dit_status launch_qknorm_rope(int dtype, void* qkv, int64_t row_stride, int T, int H, int d, int n_tensors,
                              const void* gq, const void* gk, float eps, const float* rc, const float* rs,
                              cudaStream_t st) {
  if (T == 0 || (gq == nullptr && gk == nullptr && rc == nullptr)) return DIT_OK;
  DIT_REQUIRE(d == 64 || d == 128, DIT_ERR_UNSUPPORTED, "qknorm_rope: head_dim %d not in {64,128}", d);
  ProfScope _prof(DIT_KC_QKNORM, st);
  const int cpr = (n_tensors * H * d + 255) / 256;
  const int64_t passes = (int64_t)T * ((cpr + 3) / 4);
  int grid = (int)((passes + 7) / 8);
  if (grid > 148 * 8) grid = 148 * 8;
  if (grid < 1) grid = 1;
#define QK_LAUNCH(TT, HDV)                                                                                      \
  qknorm_rope_kernel<TT, HDV><<<grid, 256, 0, st>>>((TT*)qkv, row_stride, T, H, n_tensors, (const TT*)gq,       \
                                                    (const TT*)gk, eps, rc, rs)
  if (dtype == DIT_F32) {
    if (d == 64) QK_LAUNCH(float, 64); else QK_LAUNCH(float, 128);
  } else {
    if (d == 64) QK_LAUNCH(bf16, 64); else QK_LAUNCH(bf16, 128);
  }
#undef QK_LAUNCH
  DIT_LAUNCH_CHECK();
  return DIT_OK;
}

// =================================================================================================
// RoPE tables (R6): cos/sin[t, j] for the pair j of token t; angles in double.
// =================================================================================================
__global__ void rope_table_kernel(const SeqMeta* __restrict__ meta, int R, int T_rows, int half, int d0, int d1, int d2,
                                  double log2_theta, float* __restrict__ rc, float* __restrict__ rs) {
  const int64_t idx = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (idx >= (int64_t)T_rows * half) return;
  const int t = (int)(idx / half), j = (int)(idx % half);
  int r = 0;
  while (r + 1 < R && t >= meta[r + 1].seq_start) ++r;
  const SeqMeta m = meta[r];
  const int n = t - m.seq_start - m.n_cond;
  int pos[3] = {0, 0, 0};
  if (n >= 0) {
    pos[2] = n % m.gw;
    pos[1] = (n / m.gw) % m.gh;
    pos[0] = n / (m.gw * m.gh);
  }
  int axis, jj, da;
  if (j < d0 / 2) { axis = 0; jj = j; da = d0; }
  else if (j < (d0 + d1) / 2) { axis = 1; jj = j - d0 / 2; da = d1; }
  else { axis = 2; jj = j - (d0 + d1) / 2; da = d2; }
  const double omega = exp2(-2.0 * (double)jj / (double)da * log2_theta);
  const double ang = (double)pos[axis] * omega;
  double s, c;
  sincos(ang, &s, &c);
  rc[idx] = (float)c;
  rs[idx] = (float)s;
}

dit_status launch_rope_table(const SeqMeta* meta, int R, int T, int d, const int32_t rope_dims[3], float theta,
                             float* rc, float* rs, cudaStream_t st) {
  if (T == 0) return DIT_OK;
  const int half = d / 2;
  ProfScope _prof(DIT_KC_MISC, st);
  const int64_t n = (int64_t)T * half;
  rope_table_kernel<<<cdiv(n, 256), 256, 0, st>>>(meta, R, T, half, rope_dims[0], rope_dims[1], rope_dims[2],
                                                 log2((double)theta), rc, rs);
  DIT_LAUNCH_CHECK();
  return DIT_OK;
}

// =================================================================================================
// patchify (im2col, DESIGN.md §3 step 3 / R11) and unpatchify (step 6)
// =================================================================================================
template <typename T>
__global__ void patchify_kernel(const T* __restrict__ lat, T* __restrict__ patches, int C, int F, int H, int W, int pf,
                                int ph, int pw) {
  const int Fp = F / pf, Hp = H / ph, Wp = W / pw, pv = pf * ph * pw;
  const int64_t total = (int64_t)Fp * Hp * Wp * C * pv;
  const int64_t idx = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (idx >= total) return;
  const int feat = (int)(idx % (C * pv));
  const int n = (int)(idx / (C * pv));
  const int k = feat % pw, j = (feat / pw) % ph, i = (feat / (pw * ph)) % pf, c = feat / pv;
  const int w_ = n % Wp, h_ = (n / Wp) % Hp, f_ = n / (Wp * Hp);
  patches[idx] = lat[(((int64_t)c * F + f_ * pf + i) * H + h_ * ph + j) * W + w_ * pw + k];
}

template <typename T>
__global__ void unpatchify_kernel(const float* __restrict__ tok, T* __restrict__ out, int C, int F, int H, int W,
                                  int pf, int ph, int pw, SampleEpi epi) {
  const int Hp = H / ph, Wp = W / pw, pv = pf * ph * pw;
  const int64_t total = (int64_t)C * F * H * W;
  const int64_t idx = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (idx >= total) return;
  const int w = (int)(idx % W), hh = (int)((idx / W) % H), f = (int)((idx / ((int64_t)W * H)) % F);
  const int c = (int)(idx / ((int64_t)W * H * F));
  const int n = ((f / pf) * Hp + hh / ph) * Wp + w / pw;
  const int feat = ((c * pf + f % pf) * ph + hh % ph) * pw + w % pw;
  float v = tok[(int64_t)n * (C * pv) + feat];
  if (epi.mode == 1) {          // unconditional pass of a guided step: keep v_u in fp32
    epi.v_hold[idx] = v;
    return;
  }
  if (epi.mode == 2) {          // Euler update on the fp32 state (dit_sample)
    if (epi.v_hold != nullptr) {
      const float vu = epi.v_hold[idx];
      v = vu + epi.guidance * (v - vu);
    }
    v = epi.state[idx] + epi.dsigma * v;
    epi.state[idx] = v;
  }
  out[idx] = from_f<T>(v);
}

// Packed forms (R > 1 requests in one step): blockIdx.y = request, its geometry from the device-resident SeqMeta table; rows are
// written to / read from the request's image rows of the packed sequence (seq_start + n_cond).  Same index arithmetic as above.
template <typename T>
__global__ void patchify_varlen_kernel(const T* __restrict__ lat, T* __restrict__ patches, const SeqMeta* __restrict__ meta,
                                       int C, int pf, int ph, int pw) {
  const SeqMeta m = meta[blockIdx.y];
  const int Fp = m.gf, Hp = m.gh, Wp = m.gw, pv = pf * ph * pw;
  const int F = Fp * pf, H = Hp * ph, W = Wp * pw;
  const int64_t total = (int64_t)Fp * Hp * Wp * C * pv;
  const int64_t idx = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (idx >= total) return;
  const int64_t lat_off = ((int64_t)(uint32_t)m.lat_off_lo) | ((int64_t)m.lat_off_hi << 32);
  const int feat = (int)(idx % (C * pv));
  const int n = (int)(idx / (C * pv));
  const int k = feat % pw, j = (feat / pw) % ph, i = (feat / (pw * ph)) % pf, c = feat / pv;
  const int w_ = n % Wp, h_ = (n / Wp) % Hp, f_ = n / (Wp * Hp);
  patches[(int64_t)(m.seq_start + m.n_cond) * (C * pv) + idx] =
      lat[lat_off + (((int64_t)c * F + f_ * pf + i) * H + h_ * ph + j) * W + w_ * pw + k];
}

template <typename T>
__global__ void unpatchify_varlen_kernel(const float* __restrict__ tok, T* __restrict__ out, const SeqMeta* __restrict__ meta,
                                         int C, int pf, int ph, int pw) {
  const SeqMeta m = meta[blockIdx.y];
  const int Hp = m.gh, Wp = m.gw, pv = pf * ph * pw;
  const int F = m.gf * pf, H = Hp * ph, W = Wp * pw;
  const int64_t total = (int64_t)C * F * H * W;
  const int64_t idx = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (idx >= total) return;
  const int64_t lat_off = ((int64_t)(uint32_t)m.lat_off_lo) | ((int64_t)m.lat_off_hi << 32);
  const int w = (int)(idx % W), hh = (int)((idx / W) % H), f = (int)((idx / ((int64_t)W * H)) % F);
  const int c = (int)(idx / ((int64_t)W * H * F));
  const int n = ((f / pf) * Hp + hh / ph) * Wp + w / pw;
  const int feat = ((c * pf + f % pf) * ph + hh % ph) * pw + w % pw;
  out[lat_off + idx] = from_f<T>(tok[(int64_t)(m.seq_start + m.n_cond + n) * (C * pv) + feat]);
}

template <typename T>
__global__ void sample_init_kernel(const T* __restrict__ lat, float* __restrict__ state, int64_t n) {
  const int64_t idx = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (idx < n) state[idx] = to_f(lat[idx]);
}
template <typename T>
__global__ void sample_final_kernel(const float* __restrict__ state, T* __restrict__ out, int64_t n) {
  const int64_t idx = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (idx < n) out[idx] = from_f<T>(state[idx]);
}

dit_status launch_patchify(int dtype, const void* lat, void* patches, int C, int F, int H, int W, const int32_t patch[3],
                           cudaStream_t st) {
  const int64_t total = (int64_t)C * F * H * W;
  if (total == 0) return DIT_OK;
  ProfScope _prof(DIT_KC_MISC, st);
  if (dtype == DIT_F32)
    patchify_kernel<float><<<cdiv(total, 256), 256, 0, st>>>((const float*)lat, (float*)patches, C, F, H, W, patch[0],
                                                            patch[1], patch[2]);
  else
    patchify_kernel<bf16><<<cdiv(total, 256), 256, 0, st>>>((const bf16*)lat, (bf16*)patches, C, F, H, W, patch[0],
                                                           patch[1], patch[2]);
  DIT_LAUNCH_CHECK();
  return DIT_OK;
}

dit_status launch_unpatchify(int dtype, const float* tok, void* out, int C, int F, int H, int W, const int32_t patch[3],
                             cudaStream_t st, const SampleEpi* epi) {
  const int64_t total = (int64_t)C * F * H * W;
  if (total == 0) return DIT_OK;
  const SampleEpi e = epi ? *epi : SampleEpi{0, nullptr, nullptr, 0.f, 0.f};
  ProfScope _prof(DIT_KC_MISC, st);
  if (dtype == DIT_F32)
    unpatchify_kernel<float><<<cdiv(total, 256), 256, 0, st>>>(tok, (float*)out, C, F, H, W, patch[0], patch[1], patch[2], e);
  else
    unpatchify_kernel<bf16><<<cdiv(total, 256), 256, 0, st>>>(tok, (bf16*)out, C, F, H, W, patch[0], patch[1], patch[2], e);
  DIT_LAUNCH_CHECK();
  return DIT_OK;
}

// out[r, 0..D) = bf16(SiLU(c[r, :])), out[r, D..2D) = bf16(SiLU(c) - hi): the [hi | lo] operand (R36) of the modulation GEMMs of a
// packed step with more than 8 requests (dit.cu).  One thread per element.
__global__ void silu_split_kernel(const float* __restrict__ c, bf16* __restrict__ out, int R, int D) {
  pdl_trigger();
  pdl_wait();
  const int idx = blockIdx.x * blockDim.x + threadIdx.x;
  if (idx >= R * D) return;
  const int r = idx / D, k = idx % D;
  const float v = silu_f(c[idx]);
  const bf16 hi = __float2bfloat16_rn(v);
  out[(size_t)r * 2 * D + k] = hi;
  out[(size_t)r * 2 * D + D + k] = __float2bfloat16_rn(v - __bfloat162float(hi));
}

dit_status launch_silu_split(const float* c, void* out, int R, int D, cudaStream_t st) {
  if (R == 0) return DIT_OK;
  ProfScope _prof(DIT_KC_GEMV, st);
  DIT_CUDA_OK(launch_pdl(silu_split_kernel, dim3((unsigned)cdiv(R * D, 256)), dim3(256), 0, st, 1, c, (bf16*)out, R, D));
  DIT_LAUNCH_CHECK();
  return DIT_OK;
}

// Rows of a [Lc_total, D] fp32 matrix packed by request -> the cond rows at the head of every request's segment of x
// (row cu_cond[r] + i -> row cu[r] + i).  One thread per 4 elements.
__global__ void scatter_cond_rows_kernel(const float* __restrict__ src, float* __restrict__ x, const int32_t* __restrict__ cu,
                                         const int32_t* __restrict__ cu_cond, int R, int Lc_total, int D4) {
  pdl_trigger();
  pdl_wait();
  const int64_t idx = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (idx >= (int64_t)Lc_total * D4) return;
  const int row = (int)(idx / D4), col = (int)(idx % D4);
  const int r = find_request(cu_cond, R, row);
  const int dst = cu[r] + (row - cu_cond[r]);
  reinterpret_cast<float4*>(x)[(int64_t)dst * D4 + col] = reinterpret_cast<const float4*>(src)[idx];
}

dit_status launch_scatter_cond_rows(const float* src, float* x, const int32_t* cu_dev, const int32_t* cu_cond_dev, int R,
                                    int Lc_total, int D, cudaStream_t st) {
  if (Lc_total == 0) return DIT_OK;
  ProfScope _prof(DIT_KC_MISC, st);
  const int64_t n = (int64_t)Lc_total * (D / 4);
  DIT_CUDA_OK(launch_pdl(scatter_cond_rows_kernel, dim3((unsigned)cdiv(n, 256)), dim3(256), 0, st, 1, src, x, cu_dev, cu_cond_dev, R,
                         Lc_total, D / 4));
  DIT_LAUNCH_CHECK();
  return DIT_OK;
}

// max_elems = the largest request's C*F*H*W (grid x); lat / out = the PACKED latents, patches / tok = [T, C*pv] in sequence rows
dit_status launch_patchify_varlen(int dtype, const void* lat, void* patches, const SeqMeta* meta_dev, int R, int64_t max_elems,
                                  int C, const int32_t patch[3], cudaStream_t st) {
  if (R == 0 || max_elems == 0) return DIT_OK;
  ProfScope _prof(DIT_KC_MISC, st);
  const dim3 grid((unsigned)cdiv(max_elems, 256), (unsigned)R);
  if (dtype == DIT_F32)
    patchify_varlen_kernel<float><<<grid, 256, 0, st>>>((const float*)lat, (float*)patches, meta_dev, C, patch[0], patch[1], patch[2]);
  else
    patchify_varlen_kernel<bf16><<<grid, 256, 0, st>>>((const bf16*)lat, (bf16*)patches, meta_dev, C, patch[0], patch[1], patch[2]);
  DIT_LAUNCH_CHECK();
  return DIT_OK;
}

dit_status launch_unpatchify_varlen(int dtype, const float* tok, void* out, const SeqMeta* meta_dev, int R, int64_t max_elems,
                                    int C, const int32_t patch[3], cudaStream_t st) {
  if (R == 0 || max_elems == 0) return DIT_OK;
  ProfScope _prof(DIT_KC_MISC, st);
  const dim3 grid((unsigned)cdiv(max_elems, 256), (unsigned)R);
  if (dtype == DIT_F32)
    unpatchify_varlen_kernel<float><<<grid, 256, 0, st>>>(tok, (float*)out, meta_dev, C, patch[0], patch[1], patch[2]);
  else
    unpatchify_varlen_kernel<bf16><<<grid, 256, 0, st>>>(tok, (bf16*)out, meta_dev, C, patch[0], patch[1], patch[2]);
  DIT_LAUNCH_CHECK();
  return DIT_OK;
}

dit_status launch_sample_init(int dtype, const void* lat, float* state, int64_t n, cudaStream_t st) {
  if (n == 0) return DIT_OK;
  ProfScope _prof(DIT_KC_MISC, st);
  if (dtype == DIT_F32) sample_init_kernel<float><<<cdiv(n, 256), 256, 0, st>>>((const float*)lat, state, n);
  else sample_init_kernel<bf16><<<cdiv(n, 256), 256, 0, st>>>((const bf16*)lat, state, n);
  DIT_LAUNCH_CHECK();
  return DIT_OK;
}

dit_status launch_sample_final(int dtype, const float* state, void* out, int64_t n, cudaStream_t st) {
  if (n == 0) return DIT_OK;
  ProfScope _prof(DIT_KC_MISC, st);
  if (dtype == DIT_F32) sample_final_kernel<float><<<cdiv(n, 256), 256, 0, st>>>(state, (float*)out, n);
  else sample_final_kernel<bf16><<<cdiv(n, 256), 256, 0, st>>>(state, (bf16*)out, n);
  DIT_LAUNCH_CHECK();
  return DIT_OK;
}

// =================================================================================================
// LSE merge (north_star subsystem 5; R18):  lse = ln sum_p e^{lse_p};  o = sum_p e^{lse_p - lse} o_p
// One thread per 8 output elements; bytes = P (rows*d*sizeof(T) + rows*4) + rows*d*sizeof(T) (+ rows*4).
// =================================================================================================
struct MergePtrs {
  const void* o[8];
  const float* lse[8];
};

template <typename T, int P>
__global__ void __launch_bounds__(256) merge_kernel(MergePtrs ptrs, int64_t n_rh, int d, T* __restrict__ o,
                                                    float* __restrict__ lse_out) {
  pdl_trigger();
  pdl_wait();
  const int cpr = d / 8;  // 8-element chunks per (row, head)
  const int64_t idx = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (idx >= n_rh * cpr) return;
  const int64_t rh = idx / cpr;
  float l[P], m = -INFINITY;
#pragma unroll
  for (int p = 0; p < P; ++p) {
    l[p] = ptrs.lse[p][rh];
    m = fmaxf(m, l[p]);
  }
  const float ms = (m == -INFINITY) ? 0.f : m;
  float z = 0.f, w[P];
#pragma unroll
  for (int p = 0; p < P; ++p) {
    w[p] = expf(l[p] - ms);
    z += w[p];
  }
  const float inv = z > 0.f ? 1.0f / z : 0.f;
  float acc[8] = {0, 0, 0, 0, 0, 0, 0, 0};
#pragma unroll
  for (int p = 0; p < P; ++p) {
    float v[8];
    ld8<T>(reinterpret_cast<const T*>(ptrs.o[p]) + idx * 8, v);
    const float wp = w[p] * inv;
#pragma unroll
    for (int e = 0; e < 8; ++e) acc[e] = fmaf(wp, v[e], acc[e]);
  }
  st8<T>(o + idx * 8, acc);
  if (lse_out != nullptr && idx % cpr == 0) lse_out[rh] = ms + logf(z);
}

template <typename T>
static dit_status launch_merge_t(const MergePtrs& ptrs, int P, int64_t n_rh, int d, T* o, float* lse_out,
                                 cudaStream_t st) {
  const int64_t n = n_rh * (d / 8);
  const int grid = cdiv(n, 256);
  switch (P) {
    case 1: DIT_CUDA_OK(launch_pdl(merge_kernel<T, 1>, dim3(grid), dim3(256), 0, st, 1, ptrs, n_rh, d, o, lse_out)); break;
    case 2: DIT_CUDA_OK(launch_pdl(merge_kernel<T, 2>, dim3(grid), dim3(256), 0, st, 1, ptrs, n_rh, d, o, lse_out)); break;
    case 3: DIT_CUDA_OK(launch_pdl(merge_kernel<T, 3>, dim3(grid), dim3(256), 0, st, 1, ptrs, n_rh, d, o, lse_out)); break;
    case 4: DIT_CUDA_OK(launch_pdl(merge_kernel<T, 4>, dim3(grid), dim3(256), 0, st, 1, ptrs, n_rh, d, o, lse_out)); break;
    case 5: DIT_CUDA_OK(launch_pdl(merge_kernel<T, 5>, dim3(grid), dim3(256), 0, st, 1, ptrs, n_rh, d, o, lse_out)); break;
    case 6: DIT_CUDA_OK(launch_pdl(merge_kernel<T, 6>, dim3(grid), dim3(256), 0, st, 1, ptrs, n_rh, d, o, lse_out)); break;
    case 7: DIT_CUDA_OK(launch_pdl(merge_kernel<T, 7>, dim3(grid), dim3(256), 0, st, 1, ptrs, n_rh, d, o, lse_out)); break;
    default: DIT_CUDA_OK(launch_pdl(merge_kernel<T, 8>, dim3(grid), dim3(256), 0, st, 1, ptrs, n_rh, d, o, lse_out)); break;
  }
  DIT_LAUNCH_CHECK();
  return DIT_OK;
}

// Gated MLP on the FFMA (fp32) path (R40): u <- SiLU(u) (.) u3, elementwise; the tcgen05 path fuses this in the GEMM.
template <typename T>
__global__ void __launch_bounds__(256) silu_mul_kernel(T* __restrict__ u, const T* __restrict__ u3, int64_t n8) {
  pdl_trigger();
  pdl_wait();
  for (int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; i < n8; i += (int64_t)gridDim.x * blockDim.x) {
    float a[8], b[8];
    ld8<T>(u + i * 8, a);
    ld8<T>(u3 + i * 8, b);
#pragma unroll
    for (int e = 0; e < 8; ++e) a[e] = a[e] / (1.0f + expf(-a[e])) * b[e];
    st8<T>(u + i * 8, a);
  }
}

dit_status launch_silu_mul(int dtype, void* u, const void* u3, int64_t n, cudaStream_t st) {
  if (n == 0) return DIT_OK;
  DIT_REQUIRE(n % 8 == 0, DIT_ERR_UNSUPPORTED, "silu_mul: %lld elements, not a multiple of 8", (long long)n);
  ProfScope _prof(DIT_KC_MISC, st);
  const int64_t n8 = n / 8;
  const int grid = (int)std::min<int64_t>((n8 + 255) / 256, 148 * 8);
  if (dtype == DIT_F32) DIT_CUDA_OK(launch_pdl(silu_mul_kernel<float>, dim3(grid), dim3(256), 0, st, 1, (float*)u, (const float*)u3, n8));
  else DIT_CUDA_OK(launch_pdl(silu_mul_kernel<bf16>, dim3(grid), dim3(256), 0, st, 1, (bf16*)u, (const bf16*)u3, n8));
  DIT_LAUNCH_CHECK();
  return DIT_OK;
}

dit_status launch_merge(int dtype, const void* const* o_parts, const float* const* lses, int P, int64_t n_rh, int d,
                        void* o, float* lse_out, cudaStream_t st) {
  if (n_rh == 0) return DIT_OK;
  DIT_REQUIRE(P >= 1 && P <= 8, DIT_ERR_INVALID_ARG, "merge: P=%d not in 1..8", P);
  DIT_REQUIRE(d % 8 == 0, DIT_ERR_UNSUPPORTED, "merge: head_dim %d must be a multiple of 8", d);
  ProfScope _prof(DIT_KC_MERGE, st);
  MergePtrs ptrs;
  for (int p = 0; p < 8; ++p) {
    ptrs.o[p] = o_parts[p < P ? p : 0];
    ptrs.lse[p] = lses[p < P ? p : 0];
  }
  if (dtype == DIT_F32) return launch_merge_t<float>(ptrs, P, n_rh, d, (float*)o, lse_out, st);
  return launch_merge_t<bf16>(ptrs, P, n_rh, d, (bf16*)o, lse_out, st);
}

}  // namespace dit
