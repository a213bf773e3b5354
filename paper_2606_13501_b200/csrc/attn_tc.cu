// attn_tc.cu — non-causal flash attention on tcgen05 tensor cores (north_star subsystems 4 and 5), head_dim 128, bf16.
//   for every query row i of a request, over the key rows of this call's KV shard:
//     s_ij = scale * q_i . k_j ;  o_i = sum_j softmax_j(s_ij) v_j ;  lse_i = ln sum_j exp(s_ij)        (R7, R18)
// Design (sm_100a), one CTA = one (request, head, 256 query rows) work item, 384 threads:
//   warp 0      TMA producer: two Q tiles (128 x 128) once, then a K ring and a V ring of 128-key tiles
//               (each tile = two 128 x 64 boxes, 128-byte swizzle);
//   warp 1      MMA issuer (one thread): S_t = Q_t K_j^T (M=128, N=128, K=16 x 8, both operands K-major from
//               shared memory) into TMEM, then O_t += P_t V_j with P read from TMEM (A operand in tensor memory)
//               and V as an MN-major shared-memory operand; the two Q tiles ping-pong so the tensor pipe computes
//               one tile's S / PV while the other tile's softmax runs;
//   warps 4-7   softmax warpgroup of Q tile 0, warps 8-11 of Q tile 1: one thread owns one query row — tcgen05.ld
//               of the whole 128-wide S row, row max, exp2 with the scale folded into one FFMA, bf16 P written back
//               over S in TMEM (tcgen05.st), fp32 row sum.  O is rescaled lazily: only when the running max grows
//               by more than 2^8 (exact: the same max is used for P and for the sum, and divided out at the end);
//   epilogue    the same warpgroups: O / l -> bf16 -> global, lse = ln2 * (m + log2 l).
// TMEM: S0 | S1 | O0 | O1 = 4 x 128 fp32 columns = all 512; P_t aliases the first 64 columns of S_t.
// Roofline: tensor pipe, co-limited by MUFU.EX2 (16 / clk / SM): 2 x 128 x 128 exps per 2048 tensor cycles.
#include "tc.cuh"

namespace dit {
using namespace tc;

namespace {

constexpr int HD = 128;          // head dim
constexpr int TQ = 128;          // query rows per tile (2 tiles per CTA)
constexpr int TK = 128;          // keys per tile
constexpr int KS = 2, VS = 2;    // K / V ring depths
constexpr int TILE_BYTES = 128 * HD * 2;   // 32 KB: two [128 x 64] swizzled boxes
constexpr int HALF_BYTES = TILE_BYTES / 2;
constexpr int ATTN_THREADS = 384;
constexpr int ATTN_SMEM = (2 + KS + VS) * TILE_BYTES + 1024 + 256;
constexpr float RESCALE_THRESHOLD = 8.0f;  // log2 units

struct AttnParams {
  bf16* o; int64_t o_stride;
  float* lse;
  const int32_t* cu_q; const int32_t* cu_k;
  int n_q, n_k, H;
  float scale_log2;   // softmax scale * log2(e)
  int shard, n_shards;
};

__device__ __forceinline__ float ex2(float x) {
  float y;
  asm volatile("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
  return y;
}


__device__ __forceinline__ void mask32(uint32_t (&s)[32], int valid) {
#pragma unroll
  for (int i = 0; i < 32; ++i) s[i] = (i >= valid) ? 0xff800000u : s[i];  // select, not a store: stays in registers
}
__device__ __forceinline__ float max32(const uint32_t (&s)[32]) {
  float m0 = __uint_as_float(s[0]), m1 = __uint_as_float(s[1]), m2 = __uint_as_float(s[2]), m3 = __uint_as_float(s[3]);
#pragma unroll
  for (int i = 4; i < 32; i += 4) {
    m0 = fmaxf(m0, __uint_as_float(s[i]));
    m1 = fmaxf(m1, __uint_as_float(s[i + 1]));
    m2 = fmaxf(m2, __uint_as_float(s[i + 2]));
    m3 = fmaxf(m3, __uint_as_float(s[i + 3]));
  }
  return fmaxf(fmaxf(m0, m1), fmaxf(m2, m3));
}
// p = 2^(s c + nm) for 32 scores -> 16 bf16 pairs into TMEM columns [taddr, taddr + 16); fp32 partial sums
__device__ __forceinline__ void exp_pack_store(const uint32_t (&s)[32], float c, float nm, uint32_t taddr, float& sum0,
                                               float& sum1) {
  uint32_t pk[16];
#pragma unroll
  for (int i = 0; i < 16; ++i) {
    const float a = ex2(fmaf(__uint_as_float(s[2 * i]), c, nm));
    const float b = ex2(fmaf(__uint_as_float(s[2 * i + 1]), c, nm));
    sum0 += a;
    sum1 += b;
    pk[i] = pack_bf16(a, b);
  }
  tmem_st16(taddr, pk);
}

__global__ void __launch_bounds__(ATTN_THREADS, 1)
attn_tc_kernel(const __grid_constant__ CUtensorMap tmQ, const __grid_constant__ CUtensorMap tmK,
               const __grid_constant__ CUtensorMap tmV, AttnParams p) {
  extern __shared__ uint8_t smem_raw[];
  const uint32_t smem0 = (smem_u32(smem_raw) + 1023u) & ~1023u;
  const uint32_t sQ = smem0, sK = sQ + 2 * TILE_BYTES, sV = sK + KS * TILE_BYTES;
  const uint32_t bar0 = sV + VS * TILE_BYTES;
  // barrier map
  auto q_full = [&](int t) { return bar0 + 8u * t; };
  auto k_full = [&](int s) { return bar0 + 8u * (2 + s); };
  auto k_empty = [&](int s) { return bar0 + 8u * (2 + KS + s); };
  auto v_full = [&](int s) { return bar0 + 8u * (2 + 2 * KS + s); };
  auto v_empty = [&](int s) { return bar0 + 8u * (2 + 2 * KS + VS + s); };
  auto s_full = [&](int t) { return bar0 + 8u * (2 + 2 * KS + 2 * VS + t); };
  auto p_full = [&](int t) { return bar0 + 8u * (4 + 2 * KS + 2 * VS + t); };
  auto pv_done = [&](int t) { return bar0 + 8u * (6 + 2 * KS + 2 * VS + t); };
  const uint32_t tmem_slot = bar0 + 8u * (8 + 2 * KS + 2 * VS);

  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int req = blockIdx.z, head = blockIdx.y;
  const int q_lo = p.cu_q ? p.cu_q[req] : 0, q_hi = p.cu_q ? p.cu_q[req + 1] : p.n_q;
  const int q_base = q_lo + blockIdx.x * (2 * TQ);
  if (q_base >= q_hi) return;  // CTA-uniform
  const int k_lo0 = p.cu_k ? p.cu_k[req] : 0, k_hi0 = p.cu_k ? p.cu_k[req + 1] : p.n_k;
  const int klen = k_hi0 - k_lo0;
  const int ssz = (klen + p.n_shards - 1) / p.n_shards;
  int k_lo = k_lo0 + p.shard * ssz, k_hi = k_lo0 + (p.shard + 1) * ssz;
  if (k_lo > k_hi0) k_lo = k_hi0;
  if (k_hi > k_hi0) k_hi = k_hi0;
  const int kv_len = k_hi - k_lo;
  const int n_tiles = (kv_len + TK - 1) / TK;

  if (n_tiles == 0) {  // empty shard: o = 0, lse = -inf (R18)
    if (warp >= 4) {
      const int row = q_base + (warp - 4) * 32 + lane;
      if (row < q_hi) {
        const float z[8] = {0, 0, 0, 0, 0, 0, 0, 0};
        for (int c = 0; c < HD; c += 8) st8<bf16>(p.o + (int64_t)row * p.o_stride + head * HD + c, z);
        if (p.lse) p.lse[(int64_t)row * p.H + head] = -INFINITY;
      }
    }
    return;
  }

  if (warp == 0 && lane == 0) {
    tma_prefetch_desc(&tmQ);
    tma_prefetch_desc(&tmK);
    tma_prefetch_desc(&tmV);
  }
  if (warp == 1 && lane == 0) {
    for (int t = 0; t < 2; ++t) {
      mbar_init(q_full(t), 1);
      mbar_init(s_full(t), 1);
      mbar_init(p_full(t), 128);
      mbar_init(pv_done(t), 1);
    }
    for (int s = 0; s < KS; ++s) { mbar_init(k_full(s), 1); mbar_init(k_empty(s), 1); }
    for (int s = 0; s < VS; ++s) { mbar_init(v_full(s), 1); mbar_init(v_empty(s), 1); }
    fence_barrier_init();
  }
  if (warp == 2) tmem_alloc<512>(tmem_slot);
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  uint32_t tmem_base;
  asm volatile("ld.shared.b32 %0, [%1];" : "=r"(tmem_base) : "r"(tmem_slot));

  // register budget: warpgroup 0 (TMA / MMA / idle warps) gives registers to the two softmax warpgroups
  if (warp < 4) {
    asm volatile("setmaxnreg.dec.sync.aligned.u32 56;");
  if (warp == 0) {
    // ===================================================== TMA producer
    const int c0 = head * HD;
    if (lane == 0) {
      for (int t = 0; t < 2; ++t) {
        mbar_expect_tx(q_full(t), TILE_BYTES);
        tma_load_2d(sQ + t * TILE_BYTES, &tmQ, c0, q_base + t * TQ, q_full(t));
        tma_load_2d(sQ + t * TILE_BYTES + HALF_BYTES, &tmQ, c0 + 64, q_base + t * TQ, q_full(t));
      }
    }
    int sk = 0, sv = 0;
    uint32_t pk = 0, pv = 0;
    for (int j = 0; j < n_tiles; ++j) {
      const int r0 = k_lo + j * TK;
      mbar_wait(k_empty(sk), pk ^ 1);
      if (lane == 0) {
        mbar_expect_tx(k_full(sk), TILE_BYTES);
        tma_load_2d(sK + sk * TILE_BYTES, &tmK, c0, r0, k_full(sk));
        tma_load_2d(sK + sk * TILE_BYTES + HALF_BYTES, &tmK, c0 + 64, r0, k_full(sk));
      }
      if (++sk == KS) { sk = 0; pk ^= 1; }
      mbar_wait(v_empty(sv), pv ^ 1);
      if (lane == 0) {
        mbar_expect_tx(v_full(sv), TILE_BYTES);
        tma_load_2d(sV + sv * TILE_BYTES, &tmV, c0, r0, v_full(sv));
        tma_load_2d(sV + sv * TILE_BYTES + HALF_BYTES, &tmV, c0 + 64, r0, v_full(sv));
      }
      if (++sv == VS) { sv = 0; pv ^= 1; }
      __syncwarp();
    }
  } else if (warp == 1) {
    // ===================================================== MMA issuer
    constexpr uint32_t idesc_s = idesc_bf16(TQ, TK, 0, 0);   // S = Q K^T: A, B K-major
    constexpr uint32_t idesc_o = idesc_bf16(TQ, HD, 0, 1);   // O += P V: A from TMEM, B (V) MN-major
    // V tile: two [128 keys x 64 d] boxes 16 KB apart (LBO), 8-key groups 1 KB apart (SBO); 16 keys = +2 KB
    constexpr uint64_t vdesc_hi = desc_base_sw128(HALF_BYTES >> 4, 64);
    auto issue_s = [&](int t, int sk) {
      const uint32_t d = tmem_base + t * 128;
      const uint32_t qa = sQ + t * TILE_BYTES, ka = sK + sk * TILE_BYTES;
#pragma unroll
      for (int k = 0; k < HD / 16; ++k) {
        const uint32_t off = (k >> 2) * HALF_BYTES + (k & 3) * 32;
        umma_ss(d, desc_kmajor_sw128(qa + off), desc_kmajor_sw128(ka + off), idesc_s, k != 0);
      }
    };
    auto issue_pv = [&](int t, int sv, bool acc) {
      const uint32_t d = tmem_base + 256 + t * 128;
      const uint32_t pa = tmem_base + t * 128;  // P_t: bf16 pairs in the first 64 columns of S_t
      const uint32_t va = sV + sv * TILE_BYTES;
#pragma unroll
      for (int k = 0; k < TK / 16; ++k)
        umma_ts(d, pa + 8 * k, vdesc_hi | (uint64_t)(((va + k * 2048) >> 4) & 0x3fff), idesc_o, acc || k != 0);
    };
    int sk = 0, sv = 0;
    uint32_t pk = 0, pv = 0;
    mbar_wait(q_full(0), 0);
    mbar_wait(k_full(0), 0);
    tc_fence_after();
    if (lane == 0) { issue_s(0, 0); umma_commit(s_full(0)); }
    mbar_wait(q_full(1), 0);
    tc_fence_after();
    if (lane == 0) { issue_s(1, 0); umma_commit(s_full(1)); umma_commit(k_empty(0)); }
    __syncwarp();
    if (++sk == KS) { sk = 0; pk ^= 1; }
    for (int j = 0; j < n_tiles; ++j) {
      for (int t = 0; t < 2; ++t) {
        if (t == 0) mbar_wait(v_full(sv), pv);
        mbar_wait(p_full(t), j & 1);
        tc_fence_after();
        if (lane == 0) {
          issue_pv(t, sv, j > 0);
          umma_commit(pv_done(t));
          if (t == 1) umma_commit(v_empty(sv));
        }
        __syncwarp();
        if (j + 1 < n_tiles) {
          if (t == 0) {
            mbar_wait(k_full(sk), pk);
            tc_fence_after();
          }
          if (lane == 0) {
            issue_s(t, sk);
            umma_commit(s_full(t));
            if (t == 1) umma_commit(k_empty(sk));
          }
          __syncwarp();
        }
      }
      if (++sv == VS) { sv = 0; pv ^= 1; }
      if (j + 1 < n_tiles) { if (++sk == KS) { sk = 0; pk ^= 1; } }
    }
  }
  } else {
    asm volatile("setmaxnreg.inc.sync.aligned.u32 224;");
    // ===================================================== softmax + correction + epilogue warpgroups
    const int t = (warp - 4) >> 2;                 // Q tile of this warpgroup
    const int quad = warp & 3;                     // TMEM lane quadrant of this warp
    const int row = q_base + t * TQ + quad * 32 + lane;
    const uint32_t lane_off = (uint32_t)(quad * 32) << 16;
    const uint32_t s_addr = tmem_base + t * 128 + lane_off;        // S_t (fp32) and P_t (bf16 pairs, 64 columns)
    const uint32_t o_addr = tmem_base + 256 + t * 128 + lane_off;  // O_t
    const float c = p.scale_log2;
    float m_used = -INFINITY;   // running max in log2 units (raw score * c) that P and l are expressed against
    float l = 0.f;
    for (int j = 0; j < n_tiles; ++j) {
      mbar_wait(s_full(t), j & 1);
      tc_fence_after();
      uint32_t s0[32], s1[32], s2[32], s3[32];      // the thread's whole S row (four register arrays of 32)
      tmem_ld32(s_addr + 0, s0);
      tmem_ld32(s_addr + 32, s1);
      tmem_ld32(s_addr + 64, s2);
      tmem_ld32(s_addr + 96, s3);
      tmem_ld_wait();
      const int valid = kv_len - j * TK;           // keys of this tile that exist (warp-uniform)
      if (valid < TK) {                            // -inf before the row max
        mask32(s0, valid);
        mask32(s1, valid - 32);
        mask32(s2, valid - 64);
        mask32(s3, valid - 96);
      }
      const float mx = fmaxf(fmaxf(max32(s0), max32(s1)), fmaxf(max32(s2), max32(s3)));
      const float m_new = fmaxf(m_used, mx * c);   // c > 0
      if (j == 0) {
        m_used = m_new;                            // PV_0 overwrites O: nothing to rescale
      } else {
        const bool need = (m_new - m_used) > RESCALE_THRESHOLD;
        if (__any_sync(0xffffffffu, need)) {       // lazy rescale of O_t (rare): wait for PV_t(j-1), then O *= f
          mbar_wait(pv_done(t), (j - 1) & 1);
          tc_fence_after();
          const float f = need ? ex2(m_used - m_new) : 1.0f;
#pragma unroll 1
          for (int cc = 0; cc < 8; ++cc) {
            uint32_t o[16];
            tmem_ld16(o_addr + cc * 16, o);
            tmem_ld_wait();
#pragma unroll
            for (int i = 0; i < 16; ++i) o[i] = __float_as_uint(__uint_as_float(o[i]) * f);
            tmem_st16(o_addr + cc * 16, o);
          }
          tmem_st_wait();
          l *= f;
          if (need) m_used = m_new;
        }
      }
      // P = 2^(s c - m_used): one FFMA + one EX2 per element; row sum in fp32; bf16 pairs back into TMEM
      const float nm = -m_used;
      float sum0 = 0.f, sum1 = 0.f;
      exp_pack_store(s0, c, nm, s_addr + 0, sum0, sum1);
      exp_pack_store(s1, c, nm, s_addr + 16, sum0, sum1);
      exp_pack_store(s2, c, nm, s_addr + 32, sum0, sum1);
      exp_pack_store(s3, c, nm, s_addr + 48, sum0, sum1);
      l += sum0 + sum1;
      tmem_st_wait();
      tc_fence_before();
      mbar_arrive(p_full(t));
    }
    // ---- epilogue: O_t / l -> bf16 -> global; lse = ln2 (m + log2 l)
    mbar_wait(pv_done(t), (n_tiles - 1) & 1);
    tc_fence_after();
    const float inv = 1.0f / l;                    // l >= 2^-8 > 0: every tile has at least one valid key
    const bool row_ok = row < q_hi;
    bf16* orow = p.o + (int64_t)(row_ok ? row : q_lo) * p.o_stride + head * HD;
#pragma unroll 1
    for (int cc = 0; cc < 4; ++cc) {
      uint32_t o[32];
      tmem_ld32(o_addr + cc * 32, o);
      tmem_ld_wait();
      if (row_ok) {
#pragma unroll
        for (int g = 0; g < 4; ++g) {
          float v[8];
#pragma unroll
          for (int e = 0; e < 8; ++e) v[e] = __uint_as_float(o[g * 8 + e]) * inv;
          st8<bf16>(orow + cc * 32 + g * 8, v);
        }
      }
    }
    if (row_ok && p.lse != nullptr) p.lse[(int64_t)row * p.H + head] = 0.6931471805599453f * (m_used + log2f(l));
  }
  tc_fence_before();
  __syncthreads();
  if (warp == 2) {
    tc_fence_after();
    tmem_dealloc<512>(tmem_base);
  }
}

}  // namespace

bool attn_tc_supported(const AttnArgs& a) {
  if (a.d != HD || a.n_q <= 0) return false;
  if (a.q_stride % 8 || a.kv_stride % 8 || a.o_stride % 8) return false;
  if (((uintptr_t)a.q & 15) || ((uintptr_t)a.o & 15)) return false;
  if (a.n_k > 0 && (((uintptr_t)a.k & 15) || ((uintptr_t)a.v & 15))) return false;
  return encode_tiled_fn() != nullptr;
}

dit_status launch_attn_tc(const AttnArgs& a, cudaStream_t st) {
  if (a.n_q == 0) return DIT_OK;
  int max_q = a.n_q;
  if (a.cu_q_host) {
    max_q = 0;
    for (int r = 0; r < a.R; ++r) max_q = max(max_q, a.cu_q_host[r + 1] - a.cu_q_host[r]);
  }
  if (max_q == 0) return DIT_OK;
  static bool attr_set = false;
  if (!attr_set) {
    DIT_CUDA_OK(cudaFuncSetAttribute(attn_tc_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, ATTN_SMEM));
    attr_set = true;
  }
  // K / V maps need a valid base even when there are no keys (the kernel then never issues a load)
  const void* kb = a.n_k > 0 ? a.k : a.q;
  const void* vb = a.n_k > 0 ? a.v : a.q;
  const uint64_t nk_rows = a.n_k > 0 ? a.n_k : 1;
  const uint64_t kv_ld = a.n_k > 0 ? a.kv_stride : a.q_stride;
  CUtensorMap tq, tk, tv;
  const uint64_t cols = (uint64_t)a.H * HD;
  DIT_REQUIRE(make_tmap_2d_bf16(&tq, a.q, a.n_q, cols, a.q_stride, TQ, 64) &&
                  make_tmap_2d_bf16(&tk, kb, nk_rows, cols, kv_ld, TK, 64) &&
                  make_tmap_2d_bf16(&tv, vb, nk_rows, cols, kv_ld, TK, 64),
              DIT_ERR_CUDA, "attn_tc: cuTensorMapEncodeTiled failed (n_q=%d n_k=%d H=%d)", a.n_q, a.n_k, a.H);
  AttnParams p;
  p.o = (bf16*)a.o; p.o_stride = a.o_stride; p.lse = a.lse;
  p.cu_q = a.cu_q; p.cu_k = a.cu_k;
  p.n_q = a.n_q; p.n_k = a.n_k; p.H = a.H;
  p.scale_log2 = a.scale * 1.4426950408889634f;
  p.shard = a.shard; p.n_shards = a.n_shards;
  ProfScope _prof(DIT_KC_ATTN, st);
  dim3 grid(cdiv(max_q, 2 * TQ), a.H, a.cu_q ? a.R : 1);
  attn_tc_kernel<<<grid, ATTN_THREADS, ATTN_SMEM, st>>>(tq, tk, tv, p);
  DIT_LAUNCH_CHECK();
  return DIT_OK;
}

}  // namespace dit
