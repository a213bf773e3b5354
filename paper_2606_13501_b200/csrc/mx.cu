// mx.cu — block-scaled MXFP8 linear layer (SURVEY.md §8(f) item 2 "block-scaled ... mxf8 GEMMs with the same oracle";
// DESIGN.md reading R43): block quantisation kernel, tcgen05 `kind::mxf8f6f4.block_scale` GEMM, C ABI.
//
// Format (OCP MX, restated): a block = 32 consecutive elements along K = 32 E4M3 codes + ONE E8M0 scale X = 2^(code - 127).
// Quantisation (R43; the same decisions as oracle/mx_oracle.py, written independently): amax = max |v| (fp32);
// shared_exp = clamp(exponent_fp32(amax) - 8, -127, 127) (0 for a zero block); code_i = e4m3(v_i * 2^-shared_exp), round to
// nearest even, saturating.  The scaling is an exact multiplication by a power of two.
//
// GEMM: one CTA per 128 x 128 output tile, 192 threads.
//   warp 0      TMA producer: A and W tiles of 128 rows x 128 bytes (= 128 elements = 4 blocks of K) per k-block, 4-stage ring
//   warp 1      one elected thread issues 4 MMAs (M 128, N 128, K 32) per k-block; the instruction reads the E8M0 scales of
//               its 32-element K slice from TENSOR MEMORY: a_sf_id / b_sf_id in the instruction descriptor select byte k of the
//               32-bit scale columns
//   warps 2-5   scale writers, then epilogue.  Scale layout in tensor memory (what `tcgen05.cp ... 32x128b.warpx4` produces
//               from the canonical 32 x 16-byte shared-memory tile; here written with tcgen05.st from registers): lane l of
//               EVERY lane quadrant, column c0 + j (j = 0..3) holds the four scale bytes (k slices 0..3 of the k-block) of
//               row l + 32 j of the tile — for A rows in columns c0.., for W rows in columns c0 + 4...  Each of the four warps
//               writes the same 4 + 4 words into its own quadrant; 4 scale stages follow the smem ring.
// Accumulator: fp32 in tensor memory columns 0..127; epilogue: bias (+ GELU) -> bf16 or fp32.
// Not the peak design (1-CTA tiles, no epilogue overlap): the bf16 / e4m3 block GEMMs of gemm_tc.cu are the tuned ones.
#include <cuda_fp8.h>

#include "common.cuh"
#include "tc.cuh"

namespace dit {

using namespace tc;

namespace {

constexpr int MT = 128, NT = 128, KB = 128;          // tile; k-block in elements (= bytes)
constexpr int MSTAGES = 4;
constexpr int MSTAGE_BYTES = (MT + NT) * KB;         // 32 KB
constexpr int MX_SMEM = MSTAGES * MSTAGE_BYTES + 1024 + 256 + NT * 4;
constexpr uint32_t TM_SF = 128;                      // scale columns: stage s -> A at 128 + 8 s, W at 128 + 8 s + 4

__device__ __forceinline__ void tmem_st4(uint32_t taddr, uint32_t a, uint32_t b, uint32_t c, uint32_t d) {
  asm volatile("tcgen05.st.sync.aligned.32x32b.x4.b32 [%0], {%1, %2, %3, %4};" ::"r"(taddr), "r"(a), "r"(b), "r"(c), "r"(d) : "memory");
}
__device__ __forceinline__ void umma_mx(uint32_t d_tmem, uint64_t adesc, uint64_t bdesc, uint32_t idesc, uint32_t sfa, uint32_t sfb,
                                        uint32_t accumulate) {
  asm volatile(
      "{\n\t.reg .pred p;\n\t"
      "setp.ne.b32 p, %4, 0;\n\t"
      "tcgen05.mma.cta_group::1.kind::mxf8f6f4.block_scale [%0], %1, %2, %3, [%5], [%6], p;\n\t}" ::"r"(d_tmem),
      "l"(adesc), "l"(bdesc), "r"(idesc), "r"(accumulate), "r"(sfa), "r"(sfb)
      : "memory");
}
// block-scaled instruction descriptor: E4M3 x E4M3, E8M0 scales, K-major operands, K = 32; sf: scale byte of this K slice
__device__ __forceinline__ uint32_t idesc_mx(int M, int N, uint32_t sf) {
  return (sf << 4) | ((uint32_t)(N >> 3) << 17) | (1u << 23) | ((uint32_t)(M >> 4) << 24) | (sf << 29);
}

template <int EPI>
__global__ void __launch_bounds__(192, 1)
gemm_mx_kernel(const __grid_constant__ CUtensorMap tmA, const __grid_constant__ CUtensorMap tmB, const uint8_t* __restrict__ sfa,
               const uint8_t* __restrict__ sfw, const bf16* __restrict__ bias, void* __restrict__ out, int64_t ldo, int M, int N, int K) {
  pdl_trigger();
  extern __shared__ uint8_t smem_raw[];
  const uint32_t smem0 = (smem_u32(smem_raw) + 1023u) & ~1023u;
  const uint32_t bar0 = smem0 + MSTAGES * MSTAGE_BYTES;
  auto full_bar = [&](int s) { return bar0 + 8u * s; };
  auto empty_bar = [&](int s) { return bar0 + 8u * (MSTAGES + s); };
  auto sf_full = [&](int s) { return bar0 + 8u * (2 * MSTAGES + s); };
  auto sf_empty = [&](int s) { return bar0 + 8u * (3 * MSTAGES + s); };
  const uint32_t tfull = bar0 + 8u * (4 * MSTAGES);
  const uint32_t tmem_slot = bar0 + 8u * (4 * MSTAGES + 1);
  float* const s_bias = reinterpret_cast<float*>(smem_raw + (bar0 - smem_u32(smem_raw)) + 256);

  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int nt = (N + NT - 1) / NT;
  const int m0 = (blockIdx.x / nt) * MT, n0 = (blockIdx.x % nt) * NT;
  const int nkb = K / KB;
  const int sf_ld = K / 32;                                  // scale bytes per row

  if (warp == 0 && lane == 0) {
    tma_prefetch_desc(&tmA);
    tma_prefetch_desc(&tmB);
  }
  if (warp == 1 && lane == 0) {
    for (int s = 0; s < MSTAGES; ++s) {
      mbar_init(full_bar(s), 1);
      mbar_init(empty_bar(s), 1);
      mbar_init(sf_full(s), 4);        // the four scale-writer warps
      mbar_init(sf_empty(s), 1);
    }
    mbar_init(tfull, 1);
    fence_barrier_init();
  }
  if (warp == 2) tmem_alloc<256>(tmem_slot);
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  pdl_wait();
  uint32_t tmem_base;
  asm volatile("ld.shared.b32 %0, [%1];" : "=r"(tmem_base) : "r"(tmem_slot));

  if (warp == 0) {
    // ===================================================== TMA producer
    for (int kb = 0; kb < nkb; ++kb) {
      const int s = kb % MSTAGES;
      mbar_wait(empty_bar(s), (uint32_t)((kb / MSTAGES) & 1) ^ 1u);
      if (elect_one()) {
        mbar_expect_tx(full_bar(s), MSTAGE_BYTES);
        tma_load_2d(smem0 + s * MSTAGE_BYTES, &tmA, kb * KB, m0, full_bar(s));
        tma_load_2d(smem0 + s * MSTAGE_BYTES + MT * KB, &tmB, kb * KB, n0, full_bar(s));
      }
      __syncwarp();
    }
  } else if (warp == 1) {
    // ===================================================== MMA issuer
    for (int kb = 0; kb < nkb; ++kb) {
      const int s = kb % MSTAGES;
      const uint32_t ph = (uint32_t)(kb / MSTAGES) & 1u;
      mbar_wait(full_bar(s), ph);
      mbar_wait(sf_full(s), ph);
      tc_fence_after();
      if (elect_one()) {
        const uint64_t ad = desc_kmajor_sw128(smem0 + s * MSTAGE_BYTES);
        const uint64_t bd = desc_kmajor_sw128(smem0 + s * MSTAGE_BYTES + MT * KB);
        const uint32_t ta = tmem_base + TM_SF + 8u * s, tb = ta + 4u;
#pragma unroll
        for (int k = 0; k < 4; ++k) umma_mx(tmem_base, ad + 2 * k, bd + 2 * k, idesc_mx(MT, NT, (uint32_t)k), ta, tb, (kb | k) != 0);
        umma_commit(empty_bar(s));
        umma_commit(sf_empty(s));
        if (kb == nkb - 1) umma_commit(tfull);
      }
      __syncwarp();
    }
  } else {
    // ===================================================== scale writers (all four quadrants), then epilogue
    const int quad = warp & 3;
    const uint32_t lane_off = (uint32_t)(quad * 32) << 16;
    for (int i = threadIdx.x - 64; i < NT; i += 128) s_bias[i] = (bias != nullptr && n0 + i < N) ? __bfloat162float(bias[n0 + i]) : 0.f;
    for (int kb = 0; kb < nkb; ++kb) {
      const int s = kb % MSTAGES;
      uint32_t wa[4], wb[4];
#pragma unroll
      for (int j = 0; j < 4; ++j) {     // rows lane + 32 j of the A / W tile; rows past the matrix: scale 1 (their codes are 0)
        const int ra = m0 + lane + 32 * j, rb = n0 + lane + 32 * j;
        wa[j] = ra < M ? __ldg(reinterpret_cast<const uint32_t*>(sfa + (int64_t)ra * sf_ld + kb * 4)) : 0x7f7f7f7fu;
        wb[j] = rb < N ? __ldg(reinterpret_cast<const uint32_t*>(sfw + (int64_t)rb * sf_ld + kb * 4)) : 0x7f7f7f7fu;
      }
      mbar_wait(sf_empty(s), (uint32_t)((kb / MSTAGES) & 1) ^ 1u);
      tc_fence_after();
      const uint32_t ta = tmem_base + TM_SF + 8u * s + lane_off;
      tmem_st4(ta, wa[0], wa[1], wa[2], wa[3]);
      tmem_st4(ta + 4u, wb[0], wb[1], wb[2], wb[3]);
      tmem_st_wait();
      tc_fence_before();
      __syncwarp();
      if (lane == 0) mbar_arrive(sf_full(s));
    }
    asm volatile("bar.sync 1, 128;" ::: "memory");   // s_bias visible
    mbar_wait(tfull, 0);
    tc_fence_after();
    const int row = m0 + quad * 32 + lane;
    const bool row_ok = row < M;
#pragma unroll 1
    for (int c = 0; c < NT / 32; ++c) {
      if (n0 + c * 32 >= N) break;
      uint32_t r[32];
      tmem_ld32(tmem_base + lane_off + c * 32, r);
      tmem_ld_wait();
      if (!row_ok) continue;
#pragma unroll
      for (int g = 0; g < 4; ++g) {
        const int ng = n0 + c * 32 + g * 8;
        if (ng >= N) break;                           // N % 8 == 0
        float v[8];
#pragma unroll
        for (int e = 0; e < 8; ++e) {
          v[e] = __uint_as_float(r[g * 8 + e]) + s_bias[c * 32 + g * 8 + e];
          if (EPI == DIT_EPI_BIAS_GELU) v[e] = gelu_tanh_f(v[e]);
        }
        if (EPI == DIT_EPI_BIAS_F32) st8<float>(reinterpret_cast<float*>(out) + (int64_t)row * ldo + ng, v);
        else st8<bf16>(reinterpret_cast<bf16*>(out) + (int64_t)row * ldo + ng, v);
      }
    }
  }
  tc_fence_before();
  __syncthreads();
  if (warp == 2) {
    tc_fence_after();
    tmem_dealloc<256>(tmem_base);
  }
}

// ---- quantisation: one thread per 32-element block
template <typename T>
__global__ void __launch_bounds__(256) quantize_mx_kernel(const T* __restrict__ x, int64_t ldx, int M, int K, uint8_t* __restrict__ q,
                                                          int64_t ldq, uint8_t* __restrict__ scales) {
  pdl_trigger();
  pdl_wait();
  const int bpr = K / 32;
  const int64_t idx = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (idx >= (int64_t)M * bpr) return;
  const int row = (int)(idx / bpr), b = (int)(idx % bpr);
  const T* xp = x + (int64_t)row * ldx + b * 32;
  float v[32];
#pragma unroll
  for (int i = 0; i < 4; ++i) ld8<T>(xp + 8 * i, v + 8 * i);
  float amax = 0.f;
#pragma unroll
  for (int i = 0; i < 32; ++i) amax = fmaxf(amax, fabsf(v[i]));
  int sh = 0;
  if (amax > 0.f) {
    sh = (int)((__float_as_uint(amax) >> 23) & 0xffu) - 127 - 8;   // exponent of amax (zero / subnormal field: -127) minus 8
    sh = sh < -127 ? -127 : (sh > 127 ? 127 : sh);
  }
  const float mult = __uint_as_float((uint32_t)(127 - sh) << 23);  // 2^-sh: exponent field 0 < 127 - sh <= 254, a normal number
  uint32_t w[8];
#pragma unroll
  for (int i = 0; i < 8; ++i) {
    const uint32_t lo = __nv_cvt_float2_to_fp8x2(make_float2(__fmul_rn(v[4 * i], mult), __fmul_rn(v[4 * i + 1], mult)), __NV_SATFINITE, __NV_E4M3);
    const uint32_t hi = __nv_cvt_float2_to_fp8x2(make_float2(__fmul_rn(v[4 * i + 2], mult), __fmul_rn(v[4 * i + 3], mult)), __NV_SATFINITE, __NV_E4M3);
    w[i] = lo | (hi << 16);
  }
  uint4* qp = reinterpret_cast<uint4*>(q + (int64_t)row * ldq + b * 32);
  qp[0] = make_uint4(w[0], w[1], w[2], w[3]);
  qp[1] = make_uint4(w[4], w[5], w[6], w[7]);
  scales[(int64_t)row * bpr + b] = (uint8_t)(sh + 127);
}

template <int EPI>
dit_status launch_mx_t(const CUtensorMap& ta, const CUtensorMap& tb, const uint8_t* sfa, const uint8_t* sfw, const void* bias, void* out,
                       int64_t ldo, int M, int N, int K, cudaStream_t st) {
  static std::atomic<bool> attr_set{false};
  if (!attr_set) {
    DIT_CUDA_OK(cudaFuncSetAttribute(gemm_mx_kernel<EPI>, cudaFuncAttributeMaxDynamicSharedMemorySize, MX_SMEM));
    attr_set = true;
  }
  const int tiles = cdiv(M, MT) * cdiv(N, NT);
  DIT_CUDA_OK(launch_pdl(gemm_mx_kernel<EPI>, dim3(tiles), dim3(192), MX_SMEM, st, 1, ta, tb, sfa, sfw, (const bf16*)bias, out, ldo, M, N, K));
  DIT_LAUNCH_CHECK();
  return DIT_OK;
}

}  // namespace
}  // namespace dit

using namespace dit;

extern "C" {

dit_status dit_quantize_mxfp8(int32_t dtype, const void* x, int64_t ldx, int32_t M, int32_t K, void* q, int64_t ldq, void* scales,
                              void* stream) {
  DIT_REQUIRE(dtype == DIT_F32 || dtype == DIT_BF16, DIT_ERR_INVALID_ARG, "dtype %d", dtype);
  DIT_REQUIRE(M >= 0 && K > 0 && ldx >= K && ldq >= K, DIT_ERR_INVALID_ARG, "dit_quantize_mxfp8: M=%d K=%d ldx=%lld ldq=%lld", M, K,
              (long long)ldx, (long long)ldq);
  if (M == 0) return DIT_OK;
  DIT_REQUIRE(x && q && scales, DIT_ERR_INVALID_ARG, "dit_quantize_mxfp8: NULL argument");
  DIT_REQUIRE(K % 32 == 0 && ldx % 8 == 0 && ldq % 16 == 0 && !((uintptr_t)x & 15) && !((uintptr_t)q & 15), DIT_ERR_UNSUPPORTED,
              "dit_quantize_mxfp8: K %% 32, ldx %% 8, ldq %% 16, 16-byte aligned x / q (K=%d ldx=%lld ldq=%lld)", K, (long long)ldx,
              (long long)ldq);
  cudaStream_t st = (cudaStream_t)stream;
  ProfScope _prof(DIT_KC_MISC, st);
  const int64_t n = (int64_t)M * (K / 32);
  const dim3 grid((unsigned)((n + 255) / 256));
  if (dtype == DIT_F32)
    DIT_CUDA_OK(launch_pdl(quantize_mx_kernel<float>, grid, dim3(256), 0, st, 1, (const float*)x, ldx, M, K, (uint8_t*)q, ldq, (uint8_t*)scales));
  else
    DIT_CUDA_OK(launch_pdl(quantize_mx_kernel<bf16>, grid, dim3(256), 0, st, 1, (const bf16*)x, ldx, M, K, (uint8_t*)q, ldq, (uint8_t*)scales));
  DIT_LAUNCH_CHECK();
  return DIT_OK;
}

dit_status dit_linear_mxfp8(int32_t epilogue, const void* Aq, int64_t lda, const void* a_scales, const void* Wq, const void* w_scales,
                            const void* bias, void* out, int64_t ldo, int32_t M, int32_t N, int32_t K, void* stream) {
  DIT_REQUIRE(epilogue >= DIT_EPI_BIAS && epilogue <= DIT_EPI_BIAS_F32, DIT_ERR_INVALID_ARG, "epilogue %d", epilogue);
  DIT_REQUIRE(M >= 0 && N > 0 && K > 0 && lda >= K && ldo >= N, DIT_ERR_INVALID_ARG, "dit_linear_mxfp8: bad shape M=%d N=%d K=%d lda=%lld ldo=%lld",
              M, N, K, (long long)lda, (long long)ldo);
  if (M == 0) return DIT_OK;
  DIT_REQUIRE(Aq && Wq && a_scales && w_scales && out, DIT_ERR_INVALID_ARG, "dit_linear_mxfp8: NULL argument");
  DIT_REQUIRE(K % 128 == 0 && lda % 16 == 0 && N % 8 == 0 && ldo % 8 == 0, DIT_ERR_UNSUPPORTED,
              "dit_linear_mxfp8: K (%d) must be a multiple of 128, lda (%lld) of 16, N (%d) and ldo (%lld) of 8", K, (long long)lda, N, (long long)ldo);
  DIT_REQUIRE(!(((uintptr_t)Aq | (uintptr_t)Wq | (uintptr_t)out) & 15) && !(((uintptr_t)a_scales | (uintptr_t)w_scales) & 3), DIT_ERR_UNSUPPORTED,
              "dit_linear_mxfp8: operands 16-byte, scales 4-byte aligned");
  DIT_REQUIRE(encode_tiled_fn() != nullptr, DIT_ERR_UNSUPPORTED, "dit_linear_mxfp8: cuTensorMapEncodeTiled unavailable");
  // default: the persistent CTA-pair kernel of gemm_tc.cu (EPI_MX); DIT_MX_KERNEL=simple selects the 1-CTA kernel of this file
  static const bool simple = []() { const char* e = getenv("DIT_MX_KERNEL"); return e != nullptr && e[0] == 's'; }();
  // (the pair kernel loads the scales of four k-blocks with one 16-byte load: K % 512 == 0 and 16-byte aligned scale rows)
  if (!simple && K % 512 == 0 && !(((uintptr_t)a_scales | (uintptr_t)w_scales) & 15))
    return launch_gemm_tc_mx(epilogue, Aq, lda, a_scales, Wq, w_scales, bias, out, ldo, M, N, K, (cudaStream_t)stream);
  CUtensorMap ta, tb;
  DIT_REQUIRE(make_tmap_2d_u8(&ta, Aq, M, K, lda, MT) && make_tmap_2d_u8(&tb, Wq, N, K, K, NT), DIT_ERR_CUDA,
              "dit_linear_mxfp8: cuTensorMapEncodeTiled failed (M=%d N=%d K=%d)", M, N, K);
  cudaStream_t st = (cudaStream_t)stream;
  ProfScope _prof(DIT_KC_GEMM, st);
  const uint8_t* sa = (const uint8_t*)a_scales;
  const uint8_t* sw = (const uint8_t*)w_scales;
  switch (epilogue) {
    case DIT_EPI_BIAS: return launch_mx_t<DIT_EPI_BIAS>(ta, tb, sa, sw, bias, out, ldo, M, N, K, st);
    case DIT_EPI_BIAS_GELU: return launch_mx_t<DIT_EPI_BIAS_GELU>(ta, tb, sa, sw, bias, out, ldo, M, N, K, st);
    default: return launch_mx_t<DIT_EPI_BIAS_F32>(ta, tb, sa, sw, bias, out, ldo, M, N, K, st);
  }
}

}  // extern "C"
