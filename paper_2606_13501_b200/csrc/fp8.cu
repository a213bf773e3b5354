// fp8.cu — the fp8 (e4m3) linear layer: row-wise quantisation kernel + C ABI (SURVEY.md §8(f) item 2 "fp8 GEMMs with the
// same oracle"; reading R42).  The GEMM itself is gemm_tc_kernel<EPI_F8 + e, BN> (gemm_tc.cu): kind::f8f6f4 MMAs.
//
// Quantisation of a row x (R42; the same decisions, in the same precision, as oracle/fp8_oracle.py — written independently):
//   amax = max |x| (fp32);  inv = 448 / amax, scale = amax / 448 (IEEE fp32 divisions; both 1 when amax = 0);
//   code = e4m3(x * inv): one fp32 multiplication, then round-to-nearest-even, saturating (cvt.rn.satfinite.e4m3x2.f32).
// (x / scale per element would be 18 instructions per element on the MUFU + FMA pipes — ncu: issue slots 67 % busy, XU
// 62 %, 3.9 TB/s; the multiplication by the row's reciprocal is the usual rule and keeps the kernel memory bound.)
// HBM-bound: reads the row once (bf16 rows up to 16384 elements live in registers; otherwise the second pass over the row hits
// L1 / L2), writes one byte per element:
// algorithmic bytes = s * M * K + M * K + 4 M  (s = 2 for bf16 input, 4 for fp32).
#include <cuda_fp8.h>

#include "common.cuh"

namespace dit {
namespace {

constexpr int QROWS = 4;   // rows (= warps) per CTA

template <typename T>
__global__ void __launch_bounds__(QROWS * 32) quantize_fp8_kernel(const T* __restrict__ x, int64_t ldx, int M, int K,
                                                                  uint8_t* __restrict__ q, int64_t ldq, float* __restrict__ scale) {
  pdl_trigger();
  pdl_wait();
  const int row = blockIdx.x * QROWS + (threadIdx.x >> 5), lane = threadIdx.x & 31;
  if (row >= M) return;
  const T* xr = x + (int64_t)row * ldx;
  const int n8 = K >> 3;   // K % 8 == 0
  float amax = 0.f;
  for (int i = lane; i < n8; i += 32) {
    float v[8];
    ld8<T>(xr + i * 8, v);
#pragma unroll
    for (int e = 0; e < 8; ++e) amax = fmaxf(amax, fabsf(v[e]));
  }
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) amax = fmaxf(amax, __shfl_xor_sync(0xffffffffu, amax, o));
  const float s = amax > 0.f ? __fdiv_rn(amax, 448.0f) : 1.0f;
  const float inv = amax > 0.f ? __fdiv_rn(448.0f, amax) : 1.0f;
  if (lane == 0) scale[row] = s;
  uint8_t* qr = q + (int64_t)row * ldq;
  for (int i = lane; i < n8; i += 32) {
    float v[8];
    ld8<T>(xr + i * 8, v);
    uint32_t w[2];
#pragma unroll
    for (int h = 0; h < 2; ++h) {
      const __nv_fp8x2_storage_t lo = __nv_cvt_float2_to_fp8x2(make_float2(__fmul_rn(v[4 * h], inv), __fmul_rn(v[4 * h + 1], inv)),
                                                              __NV_SATFINITE, __NV_E4M3);
      const __nv_fp8x2_storage_t hi = __nv_cvt_float2_to_fp8x2(make_float2(__fmul_rn(v[4 * h + 2], inv), __fmul_rn(v[4 * h + 3], inv)),
                                                              __NV_SATFINITE, __NV_E4M3);
      w[h] = (uint32_t)lo | ((uint32_t)hi << 16);
    }
    *reinterpret_cast<uint2*>(qr + i * 8) = make_uint2(w[0], w[1]);
  }
}

// bf16 rows held in registers: a row is read from memory once.  TPR threads per row (32: one warp, 4 rows per CTA; 128: the
// CTA), up to NCH 16-byte chunks per thread, all loads issued before the first use; amax by shuffles (+ 16 bytes of shared
// memory across the 4 warps of a row).
template <int TPR, int NCH>
__global__ void __launch_bounds__(128) quantize_fp8_reg_kernel(const bf16* __restrict__ x, int64_t ldx, int M, int K,
                                                               uint8_t* __restrict__ q, int64_t ldq, float* __restrict__ scale) {
  pdl_trigger();
  pdl_wait();
  __shared__ float s_max[4];
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const int row = TPR == 32 ? blockIdx.x * 4 + warp : blockIdx.x;
  const int t = TPR == 32 ? lane : threadIdx.x;
  const bool row_ok = row < M;
  const int n8 = K >> 3;
  const bf16* xr = x + (int64_t)(row_ok ? row : 0) * ldx;
  uint4 c[NCH];
#pragma unroll
  for (int j = 0; j < NCH; ++j) {
    const int i = t + j * TPR;
    c[j] = (row_ok && i < n8) ? __ldg(reinterpret_cast<const uint4*>(xr) + i) : make_uint4(0, 0, 0, 0);
  }
  float amax = 0.f;
#pragma unroll
  for (int j = 0; j < NCH; ++j) {
    const uint32_t w[4] = {c[j].x, c[j].y, c[j].z, c[j].w};
#pragma unroll
    for (int e = 0; e < 4; ++e)
      amax = fmaxf(amax, fmaxf(fabsf(__uint_as_float(w[e] << 16)), fabsf(__uint_as_float(w[e] & 0xffff0000u))));
  }
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) amax = fmaxf(amax, __shfl_xor_sync(0xffffffffu, amax, o));
  if (TPR == 128) {
    if (lane == 0) s_max[warp] = amax;
    __syncthreads();
    amax = fmaxf(fmaxf(s_max[0], s_max[1]), fmaxf(s_max[2], s_max[3]));
  }
  if (!row_ok) return;
  const float inv = amax > 0.f ? __fdiv_rn(448.0f, amax) : 1.0f;
  if (t == 0) scale[row] = amax > 0.f ? __fdiv_rn(amax, 448.0f) : 1.0f;
  uint8_t* qr = q + (int64_t)row * ldq;
#pragma unroll
  for (int j = 0; j < NCH; ++j) {
    const int i = t + j * TPR;
    if (i >= n8) break;
    const uint32_t w[4] = {c[j].x, c[j].y, c[j].z, c[j].w};
    uint32_t o[2];
#pragma unroll
    for (int h = 0; h < 2; ++h) {
      const float2 a = make_float2(__fmul_rn(__uint_as_float(w[2 * h] << 16), inv), __fmul_rn(__uint_as_float(w[2 * h] & 0xffff0000u), inv));
      const float2 b = make_float2(__fmul_rn(__uint_as_float(w[2 * h + 1] << 16), inv), __fmul_rn(__uint_as_float(w[2 * h + 1] & 0xffff0000u), inv));
      o[h] = (uint32_t)__nv_cvt_float2_to_fp8x2(a, __NV_SATFINITE, __NV_E4M3) |
             ((uint32_t)__nv_cvt_float2_to_fp8x2(b, __NV_SATFINITE, __NV_E4M3) << 16);
    }
    *reinterpret_cast<uint2*>(qr + i * 8) = make_uint2(o[0], o[1]);
  }
}

template <int TPR, int NCH>
cudaError_t launch_quantize_reg(const bf16* x, int64_t ldx, int M, int K, uint8_t* q, int64_t ldq, float* scale, cudaStream_t st) {
  const dim3 grid(TPR == 32 ? (M + 3) / 4 : M);
  return launch_pdl(quantize_fp8_reg_kernel<TPR, NCH>, grid, dim3(128), 0, st, 1, x, ldx, M, K, q, ldq, scale);
}

}  // namespace

dit_status launch_quantize_fp8(int dtype, const void* x, int64_t ldx, int M, int K, void* q, int64_t ldq, float* scale,
                               cudaStream_t st) {
  if (M == 0) return DIT_OK;
  DIT_REQUIRE(K > 0 && K % 8 == 0 && ldx % 8 == 0 && ldq % 8 == 0, DIT_ERR_UNSUPPORTED,
              "quantize_fp8: K (%d), ldx (%lld) and ldq (%lld) must be multiples of 8", K, (long long)ldx, (long long)ldq);
  DIT_REQUIRE(!((uintptr_t)x & 15) && !((uintptr_t)q & 7), DIT_ERR_UNSUPPORTED, "quantize_fp8: x must be 16-byte, q 8-byte aligned");
  ProfScope _prof(DIT_KC_MISC, st);
  if (dtype == DIT_BF16 && K <= 16384) {   // the row fits in the registers of at most 128 threads
    const bf16* xb = (const bf16*)x;
    uint8_t* qb = (uint8_t*)q;
    if (K <= 1024) DIT_CUDA_OK((launch_quantize_reg<32, 4>(xb, ldx, M, K, qb, ldq, scale, st)));
    else if (K <= 4096) DIT_CUDA_OK((launch_quantize_reg<128, 4>(xb, ldx, M, K, qb, ldq, scale, st)));
    else if (K <= 8192) DIT_CUDA_OK((launch_quantize_reg<128, 8>(xb, ldx, M, K, qb, ldq, scale, st)));
    else DIT_CUDA_OK((launch_quantize_reg<128, 16>(xb, ldx, M, K, qb, ldq, scale, st)));
    DIT_LAUNCH_CHECK();
    return DIT_OK;
  }
  const dim3 grid((M + QROWS - 1) / QROWS), block(QROWS * 32);
  if (dtype == DIT_F32)
    DIT_CUDA_OK(launch_pdl(quantize_fp8_kernel<float>, grid, block, 0, st, 1, (const float*)x, ldx, M, K, (uint8_t*)q, ldq, scale));
  else
    DIT_CUDA_OK(launch_pdl(quantize_fp8_kernel<bf16>, grid, block, 0, st, 1, (const bf16*)x, ldx, M, K, (uint8_t*)q, ldq, scale));
  DIT_LAUNCH_CHECK();
  return DIT_OK;
}

}  // namespace dit

using namespace dit;

extern "C" {

dit_status dit_quantize_fp8(int32_t dtype, const void* x, int64_t ldx, int32_t M, int32_t K, void* q, int64_t ldq,
                            float* scale, void* stream) {
  DIT_REQUIRE(dtype == DIT_F32 || dtype == DIT_BF16, DIT_ERR_INVALID_ARG, "dtype %d", dtype);
  DIT_REQUIRE(M >= 0 && K > 0 && ldx >= K && ldq >= K, DIT_ERR_INVALID_ARG, "dit_quantize_fp8: M=%d K=%d ldx=%lld ldq=%lld", M, K,
              (long long)ldx, (long long)ldq);
  DIT_REQUIRE(M == 0 || (x && q && scale), DIT_ERR_INVALID_ARG, "dit_quantize_fp8: NULL argument");
  return launch_quantize_fp8(dtype, x, ldx, M, K, q, ldq, scale, (cudaStream_t)stream);
}

dit_status dit_linear_fp8(int32_t epilogue, const void* Aq, int64_t lda, const float* a_scale, const void* Wq,
                          const float* w_scale, const void* bias, void* out, int64_t ldo, int32_t M, int32_t N, int32_t K,
                          void* stream) {
  DIT_REQUIRE(epilogue >= DIT_EPI_BIAS && epilogue <= DIT_EPI_BIAS_F32, DIT_ERR_INVALID_ARG, "epilogue %d", epilogue);
  DIT_REQUIRE(M >= 0 && N > 0 && K > 0 && lda >= K && ldo >= N, DIT_ERR_INVALID_ARG,
              "dit_linear_fp8: bad shape M=%d N=%d K=%d lda=%lld ldo=%lld", M, N, K, (long long)lda, (long long)ldo);
  DIT_REQUIRE(M == 0 || (Aq && Wq && a_scale && w_scale && out), DIT_ERR_INVALID_ARG, "dit_linear_fp8: NULL argument");
  DIT_REQUIRE(gemm_tc_supported(epilogue, Aq, 16, Wq, out, ldo, M > 0 ? M : 1, N, 16), DIT_ERR_UNSUPPORTED,
              "dit_linear_fp8: tcgen05 path unavailable (no sm_100 driver entry point, or N / ldo not multiples of 8)");
  return launch_gemm_tc_fp8(epilogue, Aq, lda, a_scale, Wq, w_scale, bias, out, ldo, M, N, K, (cudaStream_t)stream);
}

}  // extern "C"
