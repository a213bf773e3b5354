// simt.cu — FFMA (CUDA-core) GEMM and attention.  These are the fp32 path (BASELINE.json configs[0]: rel-L2 1e-5
// needs true fp32 products, TF32 tensor cores are 38x outside the bar — SURVEY.md §7.2 item 6) and serve bf16
// only for shapes the tcgen05 kernels do not take (K or strides not 16-byte aligned).
#include "common.cuh"

namespace dit {

// -------------------------------------------------------------------------------------------------
// GEMM: out[M,N] = epi(A[M,K] W[N,K]^T + bias[N]);  64x64x16 tiles, 256 threads, 4x4 micro-tile.
// -------------------------------------------------------------------------------------------------
template <typename T, typename TO, int EPI>
__global__ void __launch_bounds__(256) gemm_simt_kernel(const T* __restrict__ A, int64_t lda, const T* __restrict__ W,
                                                        const T* __restrict__ bias, TO* __restrict__ out, int64_t ldo,
                                                        int M, int N, int K, const float* __restrict__ gate,
                                                        int64_t gate_stride, const int32_t* __restrict__ cu, int R) {
  __shared__ float sA[16][64 + 4];
  __shared__ float sB[16][64 + 4];
  const int tid = threadIdx.x;
  const int m0 = blockIdx.y * 64, n0 = blockIdx.x * 64;
  const int tx = tid % 16, ty = tid / 16;       // micro-tile: rows ty*4.., cols tx*4..
  const int lr = tid / 4, lk = (tid % 4) * 4;   // loader: row lr (0..63), k offset lk (0,4,8,12)
  float acc[4][4] = {};
  for (int k0 = 0; k0 < K; k0 += 16) {
#pragma unroll
    for (int e = 0; e < 4; ++e) {
      const int k = k0 + lk + e;
      const int am = m0 + lr, bn = n0 + lr;
      sA[lk + e][lr] = (am < M && k < K) ? to_f<T>(A[(int64_t)am * lda + k]) : 0.f;
      sB[lk + e][lr] = (bn < N && k < K) ? to_f<T>(W[(int64_t)bn * K + k]) : 0.f;
    }
    __syncthreads();
#pragma unroll
    for (int k = 0; k < 16; ++k) {
      const float4 a = *reinterpret_cast<const float4*>(&sA[k][ty * 4]);
      const float4 b = *reinterpret_cast<const float4*>(&sB[k][tx * 4]);
      const float av[4] = {a.x, a.y, a.z, a.w}, bv[4] = {b.x, b.y, b.z, b.w};
#pragma unroll
      for (int i = 0; i < 4; ++i)
#pragma unroll
        for (int j = 0; j < 4; ++j) acc[i][j] = fmaf(av[i], bv[j], acc[i][j]);
    }
    __syncthreads();
  }
#pragma unroll
  for (int i = 0; i < 4; ++i) {
    const int m = m0 + ty * 4 + i;
    if (m >= M) continue;
    const float* grow = nullptr;
    if (EPI == 3 && gate != nullptr) grow = gate + (int64_t)((cu != nullptr && R > 1) ? find_request(cu, R, m) : 0) * gate_stride;
#pragma unroll
    for (int j = 0; j < 4; ++j) {
      const int n = n0 + tx * 4 + j;
      if (n >= N) continue;
      float v = acc[i][j] + (bias ? to_f<T>(bias[n]) : 0.f);
      if (EPI == DIT_EPI_BIAS_GELU) v = gelu_tanh_f(v);
      if (EPI == 3) {  // x <- x + gate (.) v   (TO = float)
        const float xo = to_f<TO>(out[(int64_t)m * ldo + n]);
        v = grow ? fmaf(grow[n], v, xo) : xo + v;
      }
      out[(int64_t)m * ldo + n] = from_f<TO>(v);
    }
  }
}

dit_status launch_gemm_simt(int dtype, int epi, const void* A, int64_t lda, const void* W, const void* bias, void* out,
                            int64_t ldo, int M, int N, int K, cudaStream_t st, const float* gate, int64_t gate_stride,
                            const int32_t* cu, int R) {
  if (M == 0 || N == 0) return DIT_OK;
  dim3 grid(cdiv(N, 64), cdiv(M, 64));
  ProfScope _prof(DIT_KC_GEMM, st);
#define GS(TT, TOO, E)                                                                                         \
  gemm_simt_kernel<TT, TOO, E><<<grid, 256, 0, st>>>((const TT*)A, lda, (const TT*)W, (const TT*)bias, (TOO*)out, \
                                                     ldo, M, N, K, gate, gate_stride, cu, R)
  if (dtype == DIT_F32) {
    if (epi == DIT_EPI_BIAS_GELU) GS(float, float, DIT_EPI_BIAS_GELU);
    else if (epi == 3) GS(float, float, 3);
    else GS(float, float, DIT_EPI_BIAS);
  } else {
    if (epi == DIT_EPI_BIAS_GELU) GS(bf16, bf16, DIT_EPI_BIAS_GELU);
    else if (epi == 3) GS(bf16, float, 3);
    else if (epi == DIT_EPI_BIAS_F32) GS(bf16, float, DIT_EPI_BIAS_F32);
    else GS(bf16, bf16, DIT_EPI_BIAS);
  }
#undef GS
  DIT_LAUNCH_CHECK();
  return DIT_OK;
}

// -------------------------------------------------------------------------------------------------
// Attention (non-causal, block diagonal over requests, optional KV shard): 32 query rows per CTA, 4 threads
// per row (each owns d/4 of q and o), K/V tiles of 32 keys in shared memory, exact online softmax in fp32
// with expf.  Writes locally-normalised o and lse = m + ln(l)   (R7, R18).
// -------------------------------------------------------------------------------------------------
template <typename T, int HD>
__global__ void __launch_bounds__(128) attn_simt_kernel(const T* __restrict__ q, const T* __restrict__ k,
                                                        const T* __restrict__ v, int64_t q_stride, int64_t kv_stride,
                                                        T* __restrict__ o, int64_t o_stride, float* __restrict__ lse,
                                                        const int32_t* __restrict__ cu_q,
                                                        const int32_t* __restrict__ cu_k, int n_q, int n_k, int H,
                                                        float scale, int shard, int n_shards) {
  constexpr int KT = 32;           // keys per tile
  constexpr int DP = HD / 4;       // dims per thread
  __shared__ float sK[KT][HD];
  __shared__ float sV[KT][HD];
  const int req = blockIdx.z, head = blockIdx.y;
  const int q_lo = cu_q ? cu_q[req] : 0, q_hi = cu_q ? cu_q[req + 1] : n_q;
  const int k_lo0 = cu_k ? cu_k[req] : 0, k_hi0 = cu_k ? cu_k[req + 1] : n_k;
  const int q_base = q_lo + blockIdx.x * 32;
  if (q_base >= q_hi) return;
  const int klen = k_hi0 - k_lo0;
  const int ssz = (klen + n_shards - 1) / n_shards;
  int k_lo = k_lo0 + shard * ssz, k_hi = k_lo0 + (shard + 1) * ssz;
  if (k_lo > k_hi0) k_lo = k_hi0;
  if (k_hi > k_hi0) k_hi = k_hi0;
  const int tid = threadIdx.x;
  const int r = tid / 4, part = tid % 4;
  const int row = q_base + r;
  const bool row_ok = row < q_hi;
  float qv[DP], acc[DP];
  // thread `part` owns dims {part*4 + 16*i + e}: a warp reads 64 contiguous bytes of a smem row (no conflicts)
#pragma unroll
  for (int i = 0; i < DP / 4; ++i)
#pragma unroll
    for (int e = 0; e < 4; ++e) {
      const int dd = part * 4 + 16 * i + e;
      qv[i * 4 + e] = row_ok ? to_f<T>(q[(int64_t)row * q_stride + head * HD + dd]) * scale : 0.f;
      acc[i * 4 + e] = 0.f;
    }
  float m = -INFINITY, l = 0.f;
  for (int kt = k_lo; kt < k_hi; kt += KT) {
    __syncthreads();
    for (int i = tid; i < KT * HD; i += 128) {
      const int kk = i / HD, dd = i % HD;
      const int kr = kt + kk;
      sK[kk][dd] = kr < k_hi ? to_f<T>(k[(int64_t)kr * kv_stride + head * HD + dd]) : 0.f;
      sV[kk][dd] = kr < k_hi ? to_f<T>(v[(int64_t)kr * kv_stride + head * HD + dd]) : 0.f;
    }
    __syncthreads();
    const int nk = min(KT, k_hi - kt);
    for (int kk = 0; kk < nk; ++kk) {
      float s = 0.f;
#pragma unroll
      for (int i = 0; i < DP / 4; ++i) {
        const float4 kv4 = *reinterpret_cast<const float4*>(&sK[kk][part * 4 + 16 * i]);
        s = fmaf(qv[i * 4 + 0], kv4.x, s); s = fmaf(qv[i * 4 + 1], kv4.y, s);
        s = fmaf(qv[i * 4 + 2], kv4.z, s); s = fmaf(qv[i * 4 + 3], kv4.w, s);
      }
      s += __shfl_xor_sync(0xffffffffu, s, 1);
      s += __shfl_xor_sync(0xffffffffu, s, 2);
      const float mn = fmaxf(m, s);
      const float corr = expf(m - mn);       // m = -inf first time: exp(-inf) = 0
      const float p = expf(s - mn);
      l = l * corr + p;
#pragma unroll
      for (int i = 0; i < DP / 4; ++i) {
        const float4 vv = *reinterpret_cast<const float4*>(&sV[kk][part * 4 + 16 * i]);
        acc[i * 4 + 0] = fmaf(p, vv.x, acc[i * 4 + 0] * corr); acc[i * 4 + 1] = fmaf(p, vv.y, acc[i * 4 + 1] * corr);
        acc[i * 4 + 2] = fmaf(p, vv.z, acc[i * 4 + 2] * corr); acc[i * 4 + 3] = fmaf(p, vv.w, acc[i * 4 + 3] * corr);
      }
      m = mn;
    }
  }
  if (!row_ok) return;
  const float inv = l > 0.f ? 1.0f / l : 0.f;
#pragma unroll
  for (int i = 0; i < DP / 4; ++i)
#pragma unroll
    for (int e = 0; e < 4; ++e)
      o[(int64_t)row * o_stride + head * HD + part * 4 + 16 * i + e] = from_f<T>(acc[i * 4 + e] * inv);
  if (lse != nullptr && part == 0) lse[(int64_t)row * H + head] = l > 0.f ? m + logf(l) : -INFINITY;
}

dit_status launch_attn_simt(int dtype, const AttnArgs& a, cudaStream_t st) {
  if (a.n_q == 0) return DIT_OK;
  DIT_REQUIRE(a.d == 64 || a.d == 128, DIT_ERR_UNSUPPORTED, "attention: head_dim %d not in {64,128}", a.d);
  int max_q = a.n_q;
  if (a.cu_q_host) {
    max_q = 0;
    for (int r = 0; r < a.R; ++r) max_q = max(max_q, a.cu_q_host[r + 1] - a.cu_q_host[r]);
  }
  if (max_q == 0) return DIT_OK;
  ProfScope _prof(DIT_KC_ATTN, st);
  dim3 grid(cdiv(max_q, 32), a.H, a.cu_q ? a.R : 1);
#define AS(TT, HDV)                                                                                              \
  attn_simt_kernel<TT, HDV><<<grid, 128, 0, st>>>((const TT*)a.q, (const TT*)a.k, (const TT*)a.v, a.q_stride,    \
                                                  a.kv_stride, (TT*)a.o, a.o_stride, a.lse, a.cu_q, a.cu_k, a.n_q, \
                                                  a.n_k, a.H, a.scale, a.shard, a.n_shards)
  if (dtype == DIT_F32) {
    if (a.d == 64) AS(float, 64); else AS(float, 128);
  } else {
    if (a.d == 64) AS(bf16, 64); else AS(bf16, 128);
  }
#undef AS
  DIT_LAUNCH_CHECK();
  return DIT_OK;
}

}  // namespace dit
