// gemm_tc.cu — the block GEMMs of the DiT step on 5th-generation tensor cores (north_star subsystem 3):
//   out[M, N] = epilogue(A[M, K] W[N, K]^T + bias[N]),  bf16 x bf16 -> fp32 accumulate.
// Design (sm_100a):
//   * persistent kernel on CTA PAIRS (cluster of 2, one CTA per SM): the pair walks a static round-robin list of
//     256 x BN output tiles (row-tile pairs fastest, so the pairs of a wave share W tiles through L2); BN is 256,
//     240 or 192, whichever fills the last wave best (pick_bn);
//   * warp 0 of each CTA = TMA producer: its own A rows (128 x 64) and its own HALF of the W tile (BN/2 x 64),
//     128-byte swizzle, 6-stage ring; both CTAs' boxes complete on the leader CTA's full barrier (cta_group::2
//     form of cp.async.bulk.tensor);
//   * warp 1 of the LEADER CTA = MMA issuer: one elected thread issues tcgen05.mma.cta_group::2 M=256 N=BN K=16 —
//     each SM's tensor core reads its own A and its own half of W and the halves are exchanged inside the pair —
//     accumulators (128 rows per CTA) in TMEM; two accumulator stages (2 x 256 columns = all 512) so the epilogue
//     of tile i overlaps the mainloop of i+1; tcgen05.commit.cta_group::2 is multicast to both CTAs' barriers;
//   * warps 2-5 of each CTA = epilogue of its own 128 rows: tcgen05.ld (32 lanes x 32 columns per warp), bias /
//     GELU-tanh / gated-residual / QK-RMSNorm + RoPE in fp32 registers, 16-byte global stores; the peer CTA's
//     epilogue warps release the accumulator stage with a remote mbarrier arrive on the leader's barrier.
// Roofline: tensor pipe.  M=256 (pair), N=256, K=16 takes 128 cycles on both tensor cores = 4096 MAC/cycle/SM
// (measured, clock64 loop).  Per SM a stage is A + W/2 = 32 KB, written once by TMA and read once by the MMAs per
// 512 tensor cycles: 128 B/cycle of shared-memory traffic in total — the port's limit; a 1-CTA 128 x 256 tile needs
// 192 B/cycle and stalled at ~80 % tensor-pipe utilisation.
#include <cstdlib>

#include "tc.cuh"

namespace dit {
namespace tc {

EncodeTiledFn encode_tiled_fn() {
  static EncodeTiledFn fn = []() -> EncodeTiledFn {
    void* p = nullptr;
    cudaDriverEntryPointQueryResult qr;
    if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &qr) != cudaSuccess ||
        qr != cudaDriverEntryPointSuccess) {
      (void)cudaGetLastError();
      return nullptr;
    }
    return (EncodeTiledFn)p;
  }();
  return fn;
}

bool make_tmap_2d_bf16(CUtensorMap* out, const void* base, uint64_t rows, uint64_t cols, uint64_t ld, uint32_t box_rows,
                       uint32_t box_cols) {
  EncodeTiledFn fn = encode_tiled_fn();
  if (!fn) return false;
  cuuint64_t dims[2] = {cols, rows};
  cuuint64_t strides[1] = {ld * 2};
  cuuint32_t box[2] = {box_cols, box_rows};
  cuuint32_t estr[2] = {1, 1};
  return fn(out, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 2, const_cast<void*>(base), dims, strides, box, estr,
            CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
            CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
}

bool make_tmap_2d_u8(CUtensorMap* out, const void* base, uint64_t rows, uint64_t cols, uint64_t ld, uint32_t box_rows) {
  EncodeTiledFn fn = encode_tiled_fn();
  if (!fn) return false;
  cuuint64_t dims[2] = {cols, rows};
  cuuint64_t strides[1] = {ld};
  cuuint32_t box[2] = {128, box_rows};
  cuuint32_t estr[2] = {1, 1};
  return fn(out, CU_TENSOR_MAP_DATA_TYPE_UINT8, 2, const_cast<void*>(base), dims, strides, box, estr,
            CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
            CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
}

bool make_tmap_2d_f32(CUtensorMap* out, const void* base, uint64_t rows, uint64_t cols, uint64_t ld, uint32_t box_rows) {
  EncodeTiledFn fn = encode_tiled_fn();
  if (!fn) return false;
  cuuint64_t dims[2] = {cols, rows};
  cuuint64_t strides[1] = {ld * 4};
  cuuint32_t box[2] = {32, box_rows};
  cuuint32_t estr[2] = {1, 1};
  return fn(out, CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 2, const_cast<void*>(base), dims, strides, box, estr,
            CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
            CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
}

}  // namespace tc

using namespace tc;

namespace {

constexpr int BM = 128, BK = 64;
constexpr int BN_MAX = 256;   // TMEM accumulator stage stride and staging-row size; the tile width BN is a template
                              // parameter (192 / 240 / 256) picked per problem to fill the last wave (see pick_bn)
constexpr int A_BYTES = BM * BK * 2;
constexpr int stage_bytes(int bn) { return A_BYTES + (bn / 2) * BK * 2; }   // own A rows + own HALF of the W tile
constexpr int GEMM_THREADS = 192;
constexpr int EPI_THREADS = 128;
enum { EPI_GATE_RESID = 3, EPI_QKV_NORM_ROPE = 4, EPI_BIAS_SPLIT = 5, EPI_SWIGLU = 6, EPI_F8 = 7 /* + 0 / 1 / 2 */,
       EPI_MX = 10 /* + 0 / 1 / 2 */ };
// EPI_MX + e: block-scaled MXFP8 (R43): e4m3 operands as in EPI_F8, but `kind::mxf8f6f4.block_scale` MMAs read one
// E8M0 scale per row and 32-element K slice from TENSOR MEMORY.  Four extra warps per CTA (6-9, one per TMEM lane quadrant) write
// them there for every k-block, in the layout `tcgen05.cp ... 32x128b.warpx4` would produce: lane l of every quadrant, column
// c0 + j, byte k = scale of row l + 32 j, K slice k.  Each CTA holds the scales of its own 128 A rows and of ALL BN W rows.
// Tile width 224: two accumulator stages (2 x 224 columns) + 4 scale stages of 12 columns fit the 512 TMEM columns.
constexpr int MX_THREADS = 320, MX_SF_STAGES = 4, MX_SF_COLS = 12;
// EPI_F8 + e (e = DIT_EPI_BIAS / _GELU / _F32): both operands are e4m3 bytes (R42), kind::f8f6f4 MMAs with K = 32;
// a k-block is still 128 bytes of every operand row (128 elements instead of 64), so stages, descriptors and the
// instruction count per byte are those of the bf16 kernel at twice the flops.  The epilogue applies the row scales:
// out = e(acc * a_scale[row] * w_scale[col] + bias).
// EPI_SWIGLU (gated MLP, R40): out[row, n] = SiLU(A W1^T + b1)[n] * (A W3^T + b3)[n], n < N.  One 256-wide
// accumulator tile holds 128 columns of each product: the pair's leader CTA stages 128 rows of W1 (tensor map B), its peer
// the same 128 rows of W3 (tensor map X) — each CTA supplies half of the MMA's N extent anyway — so accumulator columns
// [0, 128) are the SiLU branch and [128, 256) the linear branch of output columns 128 nn .. 128 nn + 127.  Neither
// product is ever written to memory.
// EPI_BIAS_SPLIT: out[row, n] = hi = bf16(acc + bias), out[row, N + n] = lo = bf16((acc + bias) - hi): the result as an
// unevaluated sum of two bf16 numbers (~16 significand bits).  A consumer GEMM reads [hi | lo] as ONE A operand of
// width 2N against W wrapped along K (k_wrap): hi W^T + lo W^T in the fp32 accumulator — for the small operands whose
// bf16 rounding would otherwise sit on the critical error path (the cross-attention context, R36).
// The gated-residual epilogue stages its fp32 tile chunks in shared memory for TMA reduce-add (two 32 x 32 fp32
// buffers per epilogue warp = 32 KB) and gives up one ring stage for them.
constexpr int STG_WARP_BYTES = 2 * 32 * 128;
constexpr int stages_for(int epi) { return epi == EPI_GATE_RESID ? 5 : 6; }
constexpr int staging_bytes(int epi) { return epi == EPI_GATE_RESID ? 4 * STG_WARP_BYTES : 0; }
constexpr int smem_bytes(int bn, int epi) {
  return stages_for(epi) * stage_bytes(bn) + staging_bytes(epi) + 1024 /* alignment slack */ + 256 /* barriers */ +
         2 * 2 * BN_MAX * 4 /* bias + gate rows of the tile, fp32, one set per accumulator stage */;
}

struct EpiArgs {
  const bf16* bias;       // [N] or nullptr
  const bf16* bias2;      // EPI_SWIGLU: b3 [N] or nullptr
  void* out;              // bf16 or fp32 [M, ldo]
  int64_t ldo;
  const float* gate;      // EPI_GATE_RESID: fp32 [R, gate_stride], nullptr = 1
  int64_t gate_stride;
  const int32_t* cu;      // row -> request (nullptr: one request)
  int R;
  // EPI_QKV_NORM_ROPE (head_dim 128): columns [0, q_end) = q heads, [q_end, k_end) = k heads, [k_end, N) = v heads
  // (self-attention: q_end = D, k_end = 2D; cross-attention q projection: q_end = k_end = N; cross k | v: q_end = 0,
  // k_end = D)
  const bf16* gq; const bf16* gk;   // RMSNorm gains [128] (nullptr: no norm)
  const float* rc; const float* rs; // RoPE tables [M, 64] (nullptr: no RoPE)
  float rms_eps;
  int q_end, k_end;
  const float* a_scale; const float* w_scale;   // EPI_F8: fp32 row scales of A [M] and W [N]
  // segmented launches (GemmSegs): the second weight set's vectors, and the offset of its gate rows
  const bf16* bias_b; const bf16* bias2_b; const bf16* gq_b; const bf16* gk_b;
  int64_t gate_set_off;
  // EPI_QKV_NORM_ROPE: tiles from this index on (the last, less than half full wave) are HALF tiles of one head (128 columns,
  // N = 128 MMAs, 64 W rows per CTA through tensor map X / X2): the tail wave takes half a tile time.  -1: none.
  int narrow_from;
  const uint8_t* mx_sfa; const uint8_t* mx_sfw;   // EPI_MX: E8M0 block scales [M, K / 32], [N, K / 32]
};

__device__ __forceinline__ float gelu_tanh_fast(float z) {
  // 0.5 z (1 + tanh(u)) = z / (1 + exp(-2u)),  u = 0.79788456 (z + 0.044715 z^3): exact identity, fast exp
  const float u2 = 1.5957691216057308f * fmaf(0.044715f * z * z, z, z);
  return __fdividef(z, 1.0f + __expf(-u2));
}

__device__ __forceinline__ void umma_mx_pair(uint32_t d_tmem, uint64_t adesc, uint64_t bdesc, uint32_t idesc, uint32_t sfa,
                                             uint32_t sfb, uint32_t accumulate) {
  asm volatile(
      "{\n\t.reg .pred p;\n\t"
      "setp.ne.b32 p, %4, 0;\n\t"
      "tcgen05.mma.cta_group::2.kind::mxf8f6f4.block_scale [%0], %1, %2, %3, [%5], [%6], p;\n\t}" ::"r"(d_tmem),
      "l"(adesc), "l"(bdesc), "r"(idesc), "r"(accumulate), "r"(sfa), "r"(sfb)
      : "memory");
}
// block-scaled instruction descriptor: E4M3 x E4M3, E8M0 scales, K-major, K = 32; sf = scale byte (K slice) for A and B
__device__ __forceinline__ uint32_t idesc_mx(int M, int N, uint32_t sf) {
  return (sf << 4) | ((uint32_t)(N >> 3) << 17) | (1u << 23) | ((uint32_t)(M >> 4) << 24) | (sf << 29);
}
__device__ __forceinline__ void tmem_st4(uint32_t taddr, uint32_t a, uint32_t b, uint32_t c, uint32_t d) {
  asm volatile("tcgen05.st.sync.aligned.32x32b.x4.b32 [%0], {%1, %2, %3, %4};" ::"r"(taddr), "r"(a), "r"(b), "r"(c), "r"(d) : "memory");
}

template <int EPI, int BN>
__global__ void __launch_bounds__(EPI >= EPI_MX ? MX_THREADS : GEMM_THREADS, 1)
gemm_tc_kernel(const __grid_constant__ CUtensorMap tmA, const __grid_constant__ CUtensorMap tmB,
               const __grid_constant__ CUtensorMap tmX, const __grid_constant__ CUtensorMap tmB2,
               const __grid_constant__ CUtensorMap tmX2, EpiArgs ep, const __grid_constant__ GemmSegs segs, int M, int N, int K,
               int GM, int k_wrap) {
  pdl_trigger();
  constexpr int STAGES = stages_for(EPI);
  extern __shared__ uint8_t smem_raw[];
  constexpr int BH_BYTES = (BN / 2) * BK * 2, STAGE_BYTES = A_BYTES + BH_BYTES;   // multiples of 1024 (swizzle atom)
  static_assert(BN % 16 == 0 && BN <= BN_MAX && STAGE_BYTES % 1024 == 0, "tile width");
  const uint32_t smem0 = (smem_u32(smem_raw) + 1023u) & ~1023u;
  const uint32_t stg0 = smem0 + STAGES * STAGE_BYTES;          // TMA reduce staging (gated residual only), 1024-aligned
  const uint32_t bar0 = stg0 + staging_bytes(EPI);
  // barriers: full[STAGES], empty[STAGES], tfull[2], tempty[2]; then the TMEM base address word
  auto full_bar = [&](int s) { return bar0 + 8u * s; };
  auto empty_bar = [&](int s) { return bar0 + 8u * (STAGES + s); };
  auto tfull_bar = [&](int s) { return bar0 + 8u * (2 * STAGES + s); };
  auto tempty_bar = [&](int s) { return bar0 + 8u * (2 * STAGES + 2 + s); };
  const uint32_t tmem_slot = bar0 + 8u * (2 * STAGES + 4);
  auto sf_full = [&](int s) { return bar0 + 8u * (2 * STAGES + 5 + s); };                    // EPI_MX (leader only)
  auto sf_empty = [&](int s) { return bar0 + 8u * (2 * STAGES + 5 + MX_SF_STAGES + s); };    // EPI_MX (both CTAs)
  static_assert(8 * (2 * STAGES + 5 + 2 * MX_SF_STAGES) <= 256, "barrier area");

  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  // CTA pairs (cluster of 2, cta_group::2): the pair computes a 256 x BN tile with ONE M = 256 MMA stream issued by
  // the leader CTA (rank 0).  Each CTA holds its own 128 rows of A and HALF of the W tile (rows rank * BN/2 ...) in
  // shared memory and its own 128 accumulator rows in TMEM: per CTA a stage is A + W/2 bytes — written once by TMA
  // and read once by the tensor core — instead of A + W, which is what a 1-CTA tile cannot feed through a
  // 128 B/clk shared-memory port.
  const int rank = (int)cluster_ctarank();
  const int pair = blockIdx.x >> 1, n_pairs = gridDim.x >> 1;
  // EPI_SWIGLU: a 256-wide accumulator tile is 128 output columns
  constexpr int BN_OUT = EPI == EPI_SWIGLU ? BN / 2 : BN;
  constexpr bool F8 = EPI >= EPI_F8;
  constexpr bool MX = EPI >= EPI_MX;
  constexpr int EPB = MX ? EPI - EPI_MX : (F8 ? EPI - EPI_F8 : EPI);   // the epilogue proper
  constexpr int ACC_STRIDE = MX ? BN : BN_MAX;                         // TMEM columns between the two accumulator stages
  constexpr uint32_t TM_SF = 2 * ACC_STRIDE;                           // EPI_MX: first scale column
  static_assert(!MX || (BN % 32 == 0 && BN / 32 <= 8 && 2 * BN + MX_SF_STAGES * MX_SF_COLS <= 512), "MX tile width");
  constexpr int BKE = F8 ? 2 * BK : BK;          // elements per 128-byte k-block
  const int mt = (M + BM - 1) / BM, mt2 = segs.n > 0 ? segs.tile0[segs.n] : (mt + 1) >> 1;
  const int nt = (N + BN_OUT - 1) / BN_OUT, n_wide = mt2 * nt;   // tile PAIRS
  const int narrow_from = (EPI == EPI_QKV_NORM_ROPE && ep.narrow_from >= 0) ? ep.narrow_from : n_wide;
  const int n_tiles = narrow_from + 2 * (n_wide - narrow_from);
  const int nkb = (K + BKE - 1) / BKE;
  // Tile order: groups of GM row-tile pairs; inside a group the column tile is the slow index.  A wave of 74 CTA
  // pairs then covers ~74 / GM column tiles of the same GM row-tile pairs, whose A panels (GM x 256 x K) are sized
  // by the host to stay in L2 while the group sweeps over all column tiles: A is read from DRAM about once instead
  // of once per column tile (cfg 3: 335 MB of A x 60 column tiles = 20 GB per QKV GEMM with the plain order).
  auto tile_mn = [&](int t, int& mp, int& n) {
    const int per_group = GM * nt;
    const int g = t / per_group, r = t - g * per_group;
    const int gsize = (mt2 - g * GM) < GM ? (mt2 - g * GM) : GM;
    n = r / gsize;
    mp = g * GM + (r - n * gsize);
  };

  // tile t -> row-tile pair, column tile, and for the half tiles of the tail wave which half (else -1)
  auto tile_of = [&](int t, int& mp, int& n, int& half) {
    if (t < narrow_from) {
      tile_mn(t, mp, n);
      half = -1;
    } else {
      const int u = t - narrow_from;
      tile_mn(narrow_from + (u >> 1), mp, n);
      half = u & 1;
    }
  };

  // Segmented launch: row-tile pair mp belongs to the last segment whose first pair is <= mp; its rows start at the segment's
  // first row and end at the segment's end (the tile may reach past it: those rows are loaded but never stored).
  auto seg_of = [&](int mp, int& m_base, int& m_end, int& which, int& req) {
    if (segs.n == 0) {
      m_base = mp * 2 * BM; m_end = M; which = 0; req = -1;
      return;
    }
    int lo = 0, hi = segs.n - 1;
    while (lo < hi) {
      const int mid = (lo + hi + 1) >> 1;
      if (segs.tile0[mid] <= mp) lo = mid;
      else hi = mid - 1;
    }
    m_base = segs.row0[lo] + (mp - segs.tile0[lo]) * 2 * BM;
    m_end = segs.row0[lo] + segs.rows[lo];
    which = segs.which[lo];
    req = segs.req[lo];
  };

  if (warp == 0 && lane == 0) {
    tma_prefetch_desc(&tmA);
    tma_prefetch_desc(&tmB);
    if (EPI == EPI_GATE_RESID || EPI == EPI_SWIGLU) tma_prefetch_desc(&tmX);
  }
  if (warp == 1 && lane == 0) {
    for (int s = 0; s < STAGES; ++s) {
      mbar_init(full_bar(s), 1);        // (leader only) the TMA bytes of BOTH CTAs' halves of the stage
      mbar_init(empty_bar(s), 1);       // the leader's commit, multicast to both CTAs
    }
    for (int s = 0; s < 2; ++s) {
      mbar_init(tfull_bar(s), 1);       // the leader's commit, multicast
      mbar_init(tempty_bar(s), 8);      // (leader only) 4 epilogue warps of each CTA
    }
    if (MX)
      for (int s = 0; s < MX_SF_STAGES; ++s) {
        mbar_init(sf_full(s), 8);       // (leader only) 4 scale-writer warps of each CTA
        mbar_init(sf_empty(s), 1);      // the leader's commit, multicast
      }
    fence_barrier_init();
  }
  if (warp == 2) tmem_alloc_pair<512>(tmem_slot);
  tc_fence_before();
  __syncthreads();
  cluster_sync_all();   // the peer's barriers are initialised before anything arrives on them
  tc_fence_after();
  pdl_wait();           // prologue done; from here on global memory written by the previous kernel is read
  uint32_t tmem_base;
  asm volatile("ld.shared.b32 %0, [%1];" : "=r"(tmem_base) : "r"(tmem_slot));

  if (warp == 0) {
    // ===================================================== TMA producer (both CTAs: own A rows, own half of W)
    // Both CTAs' boxes complete on the LEADER's full barrier (cta_group::2 form of the TMA load), which expects the
    // bytes of both stages; a CTA refills a stage when the leader's commit has arrived on its own empty barrier.
    int s = 0;
    uint32_t ph = 0;
    for (int t = pair; t < n_tiles; t += n_pairs) {
      int mp, nn, half;
      tile_of(t, mp, nn, half);
      int m_base, m_end, wset, req;
      seg_of(mp, m_base, m_end, wset, req);
      const bool narrow = EPI == EPI_QKV_NORM_ROPE && half >= 0;
      const int m0 = m_base + rank * BM;
      const int n0 = EPI == EPI_SWIGLU ? nn * (BN / 2) : (narrow ? nn * BN + half * 128 + rank * 64 : nn * BN + rank * (BN / 2));
      const CUtensorMap* const tmW =
          ((EPI == EPI_SWIGLU && rank != 0) || narrow) ? (wset ? &tmX2 : &tmX) : (wset ? &tmB2 : &tmB);
      const uint32_t stage_tx = narrow ? 2 * (A_BYTES + 64 * BK * 2) : 2 * STAGE_BYTES;
      for (int kb = 0; kb < nkb; ++kb) {
        mbar_wait_poll(empty_bar(s), ph ^ 1);
        if (elect_one()) {
          const uint32_t fb = mapa_cluster(full_bar(s), 0);
          if (rank == 0) mbar_expect_tx(full_bar(s), stage_tx);
          tma_load_2d_pair(smem0 + s * STAGE_BYTES, &tmA, kb * BKE, m0, fb);
          // k_wrap > 0: A is [hi | lo] (two bf16 parts side by side) and W repeats along K every k_wrap blocks
          tma_load_2d_pair(smem0 + s * STAGE_BYTES + A_BYTES, tmW, (k_wrap > 0 ? kb % k_wrap : kb) * BKE, n0, fb);
        }
        __syncwarp();
        if (++s == STAGES) { s = 0; ph ^= 1; }
      }
    }
  } else if (warp == 1 && rank != 0) {
    // the peer CTA's warp 1 has nothing to issue: the leader drives both tensor cores
  } else if (warp == 1) {
    // ===================================================== leader CTA: MMA issuer for the pair
    constexpr uint32_t idesc = F8 ? idesc_e4m3(2 * BM, BN) : idesc_bf16(2 * BM, BN, 0, 0);
    int s = 0;
    uint32_t ph = 0;
    int it = 0;
    for (int t = pair; t < n_tiles; t += n_pairs, ++it) {
      const int as = it & 1;
      const uint32_t aph = (it >> 1) & 1;
      mbar_wait_poll(tempty_bar(as), aph ^ 1);
      tc_fence_after();
      const uint32_t d_tmem = tmem_base + as * ACC_STRIDE;
      const uint32_t idesc_t = (EPI == EPI_QKV_NORM_ROPE && t >= narrow_from) ? idesc_bf16(2 * BM, 128, 0, 0) : idesc;
      for (int kb = 0; kb < nkb; ++kb) {
        mbar_wait_poll(full_bar(s), ph);
        const int gk = it * nkb + kb, ss = gk % MX_SF_STAGES;    // EPI_MX: scale stage of this k-block
        if (MX) mbar_wait_poll(sf_full(ss), (uint32_t)(gk / MX_SF_STAGES) & 1u);
        tc_fence_after();
        if (elect_one()) {
          const uint64_t ad = desc_kmajor_sw128(smem0 + s * STAGE_BYTES);
          const uint64_t bd = desc_kmajor_sw128(smem0 + s * STAGE_BYTES + A_BYTES);
#pragma unroll
          for (int k = 0; k < BK / 16; ++k) {   // 32 bytes of K per instruction in both kinds
            if (MX) umma_mx_pair(d_tmem, ad + 2 * k, bd + 2 * k, idesc_mx(2 * BM, BN, (uint32_t)k), tmem_base + TM_SF + ss * MX_SF_COLS,
                                 tmem_base + TM_SF + ss * MX_SF_COLS + 4, (kb | k) != 0);
            else if (F8) umma_ss_pair_f8(d_tmem, ad + 2 * k, bd + 2 * k, idesc, (kb | k) != 0);
            else umma_ss_pair(d_tmem, ad + 2 * k, bd + 2 * k, idesc_t, (kb | k) != 0);
          }
          umma_commit_pair(empty_bar(s), (uint16_t)3);
          if (MX) umma_commit_pair(sf_empty(ss), (uint16_t)3);
          if (kb == nkb - 1) umma_commit_pair(tfull_bar(as), (uint16_t)3);
        }
        __syncwarp();
        if (++s == STAGES) { s = 0; ph ^= 1; }
      }
    }
  } else if (MX && warp >= 6) {
    // ===================================================== EPI_MX: scale writers (TMEM lane quadrant = warp % 4)
    const uint32_t lane_off = (uint32_t)((warp & 3) * 32) << 16;
    const int sf_ld = K / 32;
    const uint32_t a_full = mapa_cluster(sf_full(0), 0);
    int gk = 0;
    for (int t = pair; t < n_tiles; t += n_pairs) {
      int mp, nn, half;
      tile_of(t, mp, nn, half);
      const int m0 = mp * 2 * BM + rank * BM, n0 = nn * BN;
      // One 16-byte load per row covers the scales of FOUR k-blocks; the next group's loads are in flight while this group's
      // words go to tensor memory (a load per k-block put ~700 cycles of L2 latency on every 448-cycle k-block: 0.8 PFLOP/s).
      constexpr int NB = BN / 32;
      auto load_group = [&](int g, uint4 (&ra)[4], uint4 (&rb)[NB]) {
        const uint4 one = make_uint4(0x7f7f7f7fu, 0x7f7f7f7fu, 0x7f7f7f7fu, 0x7f7f7f7fu);   // scale 1: rows past the matrix (codes 0)
#pragma unroll
        for (int j = 0; j < 4; ++j) {
          const int r = m0 + lane + 32 * j;
          ra[j] = r < M ? __ldg(reinterpret_cast<const uint4*>(ep.mx_sfa + (int64_t)r * sf_ld + g * 16)) : one;
        }
#pragma unroll
        for (int j = 0; j < NB; ++j) {
          const int r = n0 + lane + 32 * j;
          rb[j] = r < N ? __ldg(reinterpret_cast<const uint4*>(ep.mx_sfw + (int64_t)r * sf_ld + g * 16)) : one;
        }
      };
      auto word = [](const uint4& v, int q) { return q == 0 ? v.x : (q == 1 ? v.y : (q == 2 ? v.z : v.w)); };
      uint4 ca[4], cb[NB], na[4], nb[NB];
      load_group(0, ca, cb);
      for (int kb0 = 0; kb0 < nkb; kb0 += 4) {
        const bool more = kb0 + 4 < nkb;
        if (more) load_group(kb0 / 4 + 1, na, nb);
#pragma unroll
        for (int q = 0; q < 4; ++q, ++gk) {
          const int ss = gk % MX_SF_STAGES;
          mbar_wait_poll(sf_empty(ss), (uint32_t)((gk / MX_SF_STAGES) & 1) ^ 1u);
          tc_fence_after();
          const uint32_t ta = tmem_base + TM_SF + ss * MX_SF_COLS + lane_off;
          tmem_st4(ta, word(ca[0], q), word(ca[1], q), word(ca[2], q), word(ca[3], q));
          tmem_st4(ta + 4u, word(cb[0], q), word(cb[1], q), word(cb[2], q), word(cb[3], q));
          tmem_st4(ta + 8u, NB > 4 ? word(cb[NB > 4 ? 4 : 0], q) : 0u, NB > 5 ? word(cb[NB > 5 ? 5 : 0], q) : 0u,
                   NB > 6 ? word(cb[NB > 6 ? 6 : 0], q) : 0u, NB > 7 ? word(cb[NB > 7 ? 7 : 0], q) : 0u);
          tmem_st_wait();
          tc_fence_before();
          __syncwarp();
          if (lane == 0)   // tensor-memory writes are ordered by wait::st + the fence: the barrier carries the event only
            asm volatile("mbarrier.arrive.relaxed.cluster.shared::cluster.b64 _, [%0];" ::"r"(a_full + 8u * ss) : "memory");
        }
        if (more) {
#pragma unroll
          for (int j = 0; j < 4; ++j) ca[j] = na[j];
#pragma unroll
          for (int j = 0; j < NB; ++j) cb[j] = nb[j];
        }
      }
    }
  } else {
    // ===================================================== epilogue warps (TMEM lane quadrant = warp % 4)
    // Per tile: the 128 epilogue threads first stage the tile's bias row (and, for the gated residual, the gate
    // row of the tile's first request) in shared memory as fp32 — one global load per thread instead of one
    // dependent global load per 8 columns — then each thread walks its accumulator row in 32-column chunks.
    const int quad = warp & 3;
    const int et = threadIdx.x - 64;  // 0..127
    float* const s_vec = reinterpret_cast<float*>(smem_raw + (bar0 - smem_u32(smem_raw)) + 256);
    int it = 0;
    for (int t = pair; t < n_tiles; t += n_pairs, ++it) {
      const int as = it & 1;
      const uint32_t aph = (it >> 1) & 1;
      int mp, nn, half;
      tile_of(t, mp, nn, half);
      int m_base, m_end, wset, seg_req;
      seg_of(mp, m_base, m_end, wset, seg_req);
      const int m0 = m_base + rank * BM, n0 = nn * BN_OUT + ((EPI == EPI_QKV_NORM_ROPE && half > 0) ? 128 : 0);
      const int heads_in_tile = (EPI == EPI_QKV_NORM_ROPE && half >= 0) ? 1 : BN / 128;
      const int row = m0 + quad * 32 + lane;
      const bool row_ok = row < m_end;
      const bf16* const bias_p = wset ? ep.bias_b : ep.bias;
      const bf16* const bias2_p = wset ? ep.bias2_b : ep.bias2;
      float* const s_bias = s_vec + as * 2 * BN_MAX;
      float* const s_gate = s_bias + BN_MAX;
      bool gate_smem = true;          // this thread's row takes the staged gate row
      const float* gate_row = nullptr;
      if (EPI == EPI_GATE_RESID && ep.gate != nullptr) {
        int req0 = 0, req = 0;
        if (seg_req >= 0) {   // segmented: the whole tile is one request's rows
          req0 = req = seg_req;
        } else if (ep.cu != nullptr && ep.R > 1) {
          req0 = find_request(ep.cu, ep.R, m0);
          req = find_request(ep.cu, ep.R, row_ok ? row : M - 1);
        }
        gate_smem = req == req0;
        const int64_t set_off = wset ? ep.gate_set_off : 0;
        gate_row = ep.gate + (int64_t)req * ep.gate_stride + set_off;
        const float* g0 = ep.gate + (int64_t)req0 * ep.gate_stride + set_off;
#pragma unroll
        for (int i = et; i < BN; i += EPI_THREADS) s_gate[i] = (n0 + i < N) ? g0[n0 + i] : 0.f;
      }
      if (EPI == EPI_QKV_NORM_ROPE) {   // the two gain vectors: s_gate[0..127] = g_q, s_gate[128..255] = g_k
        for (int i = et; i < 256; i += EPI_THREADS) {
          const bf16* g = i < 128 ? (wset ? ep.gq_b : ep.gq) : (wset ? ep.gk_b : ep.gk);
          s_gate[i] = g != nullptr ? __bfloat162float(g[i & 127]) : 1.f;
        }
      }
      float a_scale = 1.0f;
      if (F8 && !MX) {   // s_gate = the tile's W row scales; this thread's A row scale
        for (int i = et; i < BN; i += EPI_THREADS) s_gate[i] = (n0 + i < N) ? ep.w_scale[n0 + i] : 0.f;
        a_scale = row_ok ? ep.a_scale[row] : 0.f;
      }
      if (EPI == EPI_SWIGLU) {   // s_bias[0..127] = b1, [128..255] = b3 of the tile's 128 output columns
        for (int i = et; i < BN; i += EPI_THREADS) {
          const bf16* const bsrc = i < BN / 2 ? bias_p : bias2_p;
          const int n = n0 + (i & (BN / 2 - 1));
          s_bias[i] = (bsrc != nullptr && n < N) ? __bfloat162float(bsrc[n]) : 0.f;
        }
      } else
#pragma unroll
      for (int i = et; i < BN; i += EPI_THREADS)
        s_bias[i] = (bias_p != nullptr && n0 + i < N) ? __bfloat162float(bias_p[n0 + i]) : 0.f;
      asm volatile("bar.sync 1, 128;" ::: "memory");  // staged rows visible to the 4 epilogue warps
      // Gated residual (x <- x + gate (.) (acc + bias)): the thread's 32-column chunk of gate (.) (acc + bias) goes to
      // a swizzled shared-memory buffer of its warp (32 rows x 128 bytes) and ONE TMA reduce-add per warp and chunk
      // adds it to x in L2: x is never read into the SM, and the global traffic is full 128-byte rows instead of
      // 32 scattered 16-byte pieces per load / store instruction (which made this epilogue 40 k cycles per tile).
      const uint32_t stg = stg0 + (uint32_t)quad * STG_WARP_BYTES;
      mbar_wait_poll(tfull_bar(as), aph);
      tc_fence_after();
      const uint32_t t_addr = tmem_base + as * ACC_STRIDE + ((uint32_t)(quad * 32) << 16);
      if (EPI == EPI_QKV_NORM_ROPE) {
        // QKV projection with QK-RMSNorm (R5) and RoPE (R6) applied to the fp32 accumulators before the one and
        // only bf16 rounding: per 128-column head, pass 1 reads the accumulator row for sum(q^2), pass 2 reads it
        // again (TMEM reads are cheap), scales by rsqrt * gain, rotates interleaved pairs, stores.  v heads: bias.
        bf16* const orow = reinterpret_cast<bf16*>(ep.out) + (int64_t)(row_ok ? row : 0) * ep.ldo + n0;
        const float* const rcr = ep.rc != nullptr ? ep.rc + (int64_t)(row_ok ? row : 0) * 64 : nullptr;
        const float* const rsr = ep.rs != nullptr ? ep.rs + (int64_t)(row_ok ? row : 0) * 64 : nullptr;
#pragma unroll 1
        for (int hh = 0; hh < heads_in_tile; ++hh) {
          const int nh = n0 + hh * 128;
          if (nh >= N) break;  // warp-uniform
          const int which = nh < ep.q_end ? 0 : (nh < ep.k_end ? 1 : 2);   // 0 = q, 1 = k, 2 = v
          const bool norm = which < 2 && (which == 0 ? ep.gq : ep.gk) != nullptr;   // both weight sets norm or neither
          const bool rope = which < 2 && rcr != nullptr;
          const float* const sg = s_gate + (which == 1 ? 128 : 0);
          float rinv = 1.0f;
          if (norm) {
            float ss = 0.f;
#pragma unroll 1
            for (int c4 = 0; c4 < 4; ++c4) {
              uint32_t r[32];
              tmem_ld32(t_addr + hh * 128 + c4 * 32, r);
              tmem_ld_wait();
#pragma unroll
              for (int e = 0; e < 32; ++e) {
                const float v = __uint_as_float(r[e]) + s_bias[hh * 128 + c4 * 32 + e];
                ss = fmaf(v, v, ss);
              }
            }
            rinv = rsqrtf(ss * (1.0f / 128.0f) + ep.rms_eps);
          }
#pragma unroll 1
          for (int c4 = 0; c4 < 4; ++c4) {
            uint32_t r[32];
            tmem_ld32(t_addr + hh * 128 + c4 * 32, r);
            float cs[16], sn[16];
            if (rope) {
#pragma unroll
              for (int g = 0; g < 4; ++g) {
                const float4 a = __ldg(reinterpret_cast<const float4*>(rcr + c4 * 16 + g * 4));
                const float4 b = __ldg(reinterpret_cast<const float4*>(rsr + c4 * 16 + g * 4));
                cs[g * 4 + 0] = a.x; cs[g * 4 + 1] = a.y; cs[g * 4 + 2] = a.z; cs[g * 4 + 3] = a.w;
                sn[g * 4 + 0] = b.x; sn[g * 4 + 1] = b.y; sn[g * 4 + 2] = b.z; sn[g * 4 + 3] = b.w;
              }
            }
            tmem_ld_wait();
            float v[32];
#pragma unroll
            for (int e = 0; e < 32; ++e) {
              v[e] = __uint_as_float(r[e]) + s_bias[hh * 128 + c4 * 32 + e];
              if (norm) v[e] = v[e] * rinv * sg[c4 * 32 + e];
            }
            if (rope) {
#pragma unroll
              for (int j = 0; j < 16; ++j) {
                const float a = v[2 * j], b = v[2 * j + 1];
                v[2 * j] = a * cs[j] - b * sn[j];
                v[2 * j + 1] = a * sn[j] + b * cs[j];
              }
            }
            if (row_ok) {
#pragma unroll
              for (int g = 0; g < 4; ++g) st8<bf16>(orow + hh * 128 + c4 * 32 + g * 8, &v[g * 8]);
            }
          }
        }
      } else if (EPI == EPI_SWIGLU) {
        bf16* const orow = reinterpret_cast<bf16*>(ep.out) + (int64_t)(row_ok ? row : 0) * ep.ldo + n0;
#pragma unroll 1
        for (int c = 0; c < BN / 64; ++c) {
          if (n0 + c * 32 >= N) break;  // warp-uniform
          uint32_t r1[32], r3[32];
          tmem_ld32(t_addr + c * 32, r1);
          tmem_ld32(t_addr + BN / 2 + c * 32, r3);
          tmem_ld_wait();
          float v[32];
#pragma unroll
          for (int e = 0; e < 32; ++e) {
            const float a = __uint_as_float(r1[e]) + s_bias[c * 32 + e];
            const float b = __uint_as_float(r3[e]) + s_bias[BN / 2 + c * 32 + e];
            v[e] = __fdividef(a, 1.0f + __expf(-a)) * b;
          }
          if (row_ok) {
#pragma unroll
            for (int g = 0; g < 4; ++g)
              if (n0 + c * 32 + g * 8 < N) st8<bf16>(orow + c * 32 + g * 8, &v[g * 8]);
          }
        }
      } else
#pragma unroll 1
      for (int c = 0; c < (BN + 31) / 32; ++c) {
        const int n = n0 + c * 32;
        if (n >= N) break;  // warp-uniform
        uint32_t r[32];
        tmem_ld32(t_addr + c * 32, r);
        tmem_ld_wait();
        if (EPI == EPI_GATE_RESID) {
          const uint32_t buf = stg + (uint32_t)(c & 1) * (STG_WARP_BYTES / 2);
          if (lane == 0) tma_store_wait_read<1>();   // the reduce issued from this buffer two chunks ago has read it
          __syncwarp();
#pragma unroll
          for (int g = 0; g < 4; ++g) {
            const int ng = n + g * 8;
            float v[8], b[8], gv[8];
            ld8<float>(s_bias + c * 32 + g * 8, b);
            // columns past the tile belong to the next tile, rows past the segment to the next segment: add 0
            const bool live = row_ok && ng < N && c * 32 + g * 8 < BN;
            if (gate_row != nullptr && live) {
              if (gate_smem) ld8<float>(s_gate + c * 32 + g * 8, gv);
              else ld8<float>(gate_row + ng, gv);
            } else {
#pragma unroll
              for (int e = 0; e < 8; ++e) gv[e] = 1.0f;
            }
#pragma unroll
            for (int e = 0; e < 8; ++e) v[e] = live ? gv[e] * (__uint_as_float(r[g * 8 + e]) + b[e]) : 0.f;
            // 128-byte swizzle of the TMA box: 16-byte chunk j of row `lane` sits at chunk j ^ (lane & 7)
            const uint32_t a0 = buf + (uint32_t)lane * 128u + (uint32_t)(((2 * g) ^ (lane & 7)) << 4);
            const uint32_t a1 = buf + (uint32_t)lane * 128u + (uint32_t)(((2 * g + 1) ^ (lane & 7)) << 4);
            asm volatile("st.shared.v4.f32 [%0], {%1, %2, %3, %4};" ::"r"(a0), "f"(v[0]), "f"(v[1]), "f"(v[2]), "f"(v[3]) : "memory");
            asm volatile("st.shared.v4.f32 [%0], {%1, %2, %3, %4};" ::"r"(a1), "f"(v[4]), "f"(v[5]), "f"(v[6]), "f"(v[7]) : "memory");
          }
          fence_proxy_async();   // the generic-proxy stores above are visible to the TMA engine
          __syncwarp();
          if (lane == 0) {
            tma_reduce_add_2d(&tmX, buf, n, m0 + quad * 32);   // rows >= M and columns >= N are clipped by the map
            tma_store_commit();
          }
          continue;
        }
#pragma unroll
        for (int g = 0; g < 4; ++g) {  // groups of 8 columns
          const int ng = n + g * 8;
          if (ng >= N || c * 32 + g * 8 >= BN) break;  // N % 8 == 0, BN % 16 == 0: groups are all-or-nothing
          float v[8], b[8];
          ld8<float>(s_bias + c * 32 + g * 8, b);
#pragma unroll
          for (int e = 0; e < 8; ++e) {
            if (F8 && !MX) v[e] = fmaf(__uint_as_float(r[g * 8 + e]), a_scale * s_gate[c * 32 + g * 8 + e], b[e]);
            else v[e] = __uint_as_float(r[g * 8 + e]) + b[e];
          }
          if (EPB == DIT_EPI_BIAS_GELU) {
#pragma unroll
            for (int e = 0; e < 8; ++e) v[e] = gelu_tanh_fast(v[e]);
          }
          if (!row_ok) continue;
          if (EPI == EPI_BIAS_SPLIT) {
            bf16* const o = reinterpret_cast<bf16*>(ep.out) + (int64_t)row * ep.ldo + ng;
            float lo[8];
#pragma unroll
            for (int e = 0; e < 8; ++e) lo[e] = v[e] - __bfloat162float(__float2bfloat16_rn(v[e]));
            st8<bf16>(o, v);
            st8<bf16>(o + N, lo);
          } else if (EPB == DIT_EPI_BIAS || EPB == DIT_EPI_BIAS_GELU) {
            st8<bf16>(reinterpret_cast<bf16*>(ep.out) + (int64_t)row * ep.ldo + ng, v);
          } else if (EPB == DIT_EPI_BIAS_F32) {
            st8<float>(reinterpret_cast<float*>(ep.out) + (int64_t)row * ep.ldo + ng, v);
          }
        }
      }
      tc_fence_before();
      __syncwarp();
      if (lane == 0) {   // the accumulator stage is drained: tell the leader's MMA warp
        if (rank == 0) mbar_arrive(tempty_bar(as));
        else mbar_arrive_remote(tempty_bar(as), 0);
      }
    }
  }
  if (EPI == EPI_GATE_RESID && warp >= 2 && lane == 0) tma_store_wait<0>();   // every reduce-add has been performed
  tc_fence_before();
  __syncthreads();
  cluster_sync_all();   // no CTA leaves while its peer may still signal its barriers
  if (warp == 2) {
    tc_fence_after();
    tmem_dealloc_pair<512>(tmem_base);
  }
}

// Row-tile pairs per raster group: their A panels (256 rows x K bf16 each) should take about 36 MB of the 126 MB L2 (DRAM reads
// of the cfg 3 QKV GEMM by ncu at 12 / 24 / 36 / 48 / 72 MB: 7.49 / 4.61 / 3.66 / 4.69 / 7.06 GB, 3.58 / 3.41 / 3.31 / 3.39 / 3.56 ms;
// the step times are flat between 30 and 48 MB: profiles/r02_gemm_cfg3_traffic.md).
int group_rows(int M, int K) {
  const int mt2 = cdiv(cdiv(M, BM), 2);
  static const double budget = []() {   // DIT_GEMM_L2_MB overrides the 36 MB default (tuning knob)
    const char* e = getenv("DIT_GEMM_L2_MB");
    return (e != nullptr && atof(e) > 0 ? atof(e) : 36.0) * 1.0e6;
  }();
  int gm = (int)(budget / (512.0 * K) + 0.5);
  if (gm < 4) gm = 4;
  if (gm > mt2) gm = mt2;
  return gm;
}

int sm_count() {
  static int n = []() {
    int dev = 0, v = 148;
    cudaGetDevice(&dev);
    cudaDeviceGetAttribute(&v, cudaDevAttrMultiProcessorCount, dev);
    return v;
  }();
  return n;
}

const GemmSegs& no_segs() {
  static const GemmSegs z = {};
  return z;
}

// segmented launches pass the segment table and the second weight set's tensor maps (tb2: W, tx2: W3 of the SwiGLU form)
struct SegLaunch { const GemmSegs* segs; const CUtensorMap* tb2; const CUtensorMap* tx2; };

// First tile of the tail wave when that wave would be less than half full (then it is run as half-width tiles), else -1
int narrow_tail_from(int n_wide) {
  static const bool off = []() { const char* e = getenv("DIT_GEMM_NO_NARROW_TAIL"); return e != nullptr && e[0] == '1'; }();
  const int max_pairs = sm_count() / 2;
  const int full = (n_wide / max_pairs) * max_pairs, rem = n_wide - full;
  return (!off && rem > 0 && 2 * rem <= max_pairs) ? full : -1;
}

template <int EPI, int BN>
dit_status launch_t(const CUtensorMap& ta, const CUtensorMap& tb, const CUtensorMap& tx, const EpiArgs& ep, int M, int N, int K,
                    cudaStream_t st, int k_wrap = 0, const SegLaunch* sl = nullptr) {
  static std::atomic<bool> attr_set{false};
  if (!attr_set) {
    DIT_CUDA_OK(cudaFuncSetAttribute(gemm_tc_kernel<EPI, BN>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                     smem_bytes(BN, EPI)));
    attr_set = true;
  }
  const int mt2 = sl != nullptr ? sl->segs->tile0[sl->segs->n] : cdiv(cdiv(M, BM), 2);
  const int n_wide = mt2 * cdiv(N, EPI == EPI_SWIGLU ? BN / 2 : BN);
  const int pairs = (EPI == EPI_QKV_NORM_ROPE && ep.narrow_from >= 0) ? ep.narrow_from + 2 * (n_wide - ep.narrow_from) : n_wide;
  const int max_pairs = sm_count() / 2;
  DIT_CUDA_OK(launch_pdl(gemm_tc_kernel<EPI, BN>, dim3(2 * (pairs < max_pairs ? pairs : max_pairs)),
                         dim3(EPI >= EPI_MX ? MX_THREADS : GEMM_THREADS),
                         smem_bytes(BN, EPI), st, 2, ta, tb, tx, sl != nullptr ? *sl->tb2 : tb, sl != nullptr ? *sl->tx2 : tx, ep,
                         sl != nullptr ? *sl->segs : no_segs(), M, N, K, group_rows(mt2 * 2 * BM, K), k_wrap));
  DIT_LAUNCH_CHECK();
  return DIT_OK;
}

// Tile width that minimises waves x width on this many SMs (wave quantisation: M = 4352 gives 34 M-tiles, and
// 34 x {36, 48, 12} tiles of 256 columns leave the last wave 3-27 % full; 240- or 192-wide tiles fill it).
int pick_bn(int M, int N, int mt2 = -1) {
  const int cand[3] = {256, 240, 192};
  int best = 256;
  int64_t best_cost = INT64_MAX;
  if (mt2 < 0) mt2 = cdiv(cdiv(M, BM), 2);
  for (int i = 0; i < 3; ++i) {
    const int bn = cand[i];
    const int64_t tiles = (int64_t)mt2 * cdiv(N, bn);   // tile pairs on CTA pairs
    const int64_t cost = cdiv(tiles, (int64_t)(sm_count() / 2)) * bn;
    if (cost < best_cost - best_cost / 64) {   // a narrower tile must win by > 1.5 %
      best_cost = cost;
      best = bn;
    }
  }
  return best;
}

template <int EPI>
dit_status launch_bn(int bn, const CUtensorMap& ta, const CUtensorMap& tb, const CUtensorMap& tx, const EpiArgs& ep, int M,
                     int N, int K, cudaStream_t st, int k_wrap = 0, const SegLaunch* sl = nullptr) {
  if (bn == 192) return launch_t<EPI, 192>(ta, tb, tx, ep, M, N, K, st, k_wrap, sl);
  if (bn == 240) return launch_t<EPI, 240>(ta, tb, tx, ep, M, N, K, st, k_wrap, sl);
  return launch_t<EPI, 256>(ta, tb, tx, ep, M, N, K, st, k_wrap, sl);
}

}  // namespace

bool gemm_tc_supported(int epi, const void* A, int64_t lda, const void* W, void* out, int64_t ldo, int M, int N, int K) {
  (void)epi;
  if (M <= 0 || N <= 0 || K <= 0) return false;
  if (K % 8 != 0 || lda % 8 != 0 || N % 8 != 0 || ldo % 8 != 0) return false;
  if (((uintptr_t)A & 15) || ((uintptr_t)W & 15) || ((uintptr_t)out & 15)) return false;
  return encode_tiled_fn() != nullptr;
}

dit_status launch_gemm_tc_ex(int epi, const void* A, int64_t lda, const void* W, const void* bias, void* out, int64_t ldo,
                             const float* gate, int64_t gate_stride, const int32_t* cu, int R, int M, int N, int K,
                             cudaStream_t st, int a_split) {
  if (M == 0 || N == 0) return DIT_OK;
  CUtensorMap ta, tb;
  const int bn = pick_bn(M, N);
  // a_split: A is [hi | lo], 2K columns; W [N, K] is walked twice along K (k_wrap blocks of 64)
  DIT_REQUIRE(!a_split || K % BK == 0, DIT_ERR_INVALID_ARG, "gemm_tc: split A needs K %% 64 == 0 (K=%d)", K);
  const int k_wrap = a_split ? K / BK : 0;
  const int Ka = a_split ? 2 * K : K;
  DIT_REQUIRE(make_tmap_2d_bf16(&ta, A, M, Ka, lda, BM, BK) && make_tmap_2d_bf16(&tb, W, N, K, K, bn / 2, BK), DIT_ERR_CUDA,
              "gemm_tc: cuTensorMapEncodeTiled failed (M=%d N=%d K=%d lda=%lld)", M, N, K, (long long)lda);
  EpiArgs ep{(const bf16*)bias, nullptr, out, ldo, gate, gate_stride, cu, R, nullptr, nullptr, nullptr, nullptr, 0.f, 0, 0, nullptr, nullptr, nullptr, nullptr, nullptr, nullptr, 0, -1};
  ProfScope _prof(DIT_KC_GEMM, st);
  switch (epi) {
    case DIT_EPI_BIAS: return launch_bn<DIT_EPI_BIAS>(bn, ta, tb, ta, ep, M, N, Ka, st, k_wrap);
    case DIT_EPI_BIAS_GELU: return launch_bn<DIT_EPI_BIAS_GELU>(bn, ta, tb, ta, ep, M, N, Ka, st, k_wrap);
    case DIT_EPI_BIAS_F32: return launch_bn<DIT_EPI_BIAS_F32>(bn, ta, tb, ta, ep, M, N, Ka, st, k_wrap);
    case EPI_BIAS_SPLIT: return launch_bn<EPI_BIAS_SPLIT>(bn, ta, tb, ta, ep, M, N, Ka, st, k_wrap);
    case EPI_GATE_RESID: {
      CUtensorMap tx;   // the fp32 residual stream as the target of the epilogue's TMA reduce-add
      DIT_REQUIRE(make_tmap_2d_f32(&tx, out, M, N, ldo, 32), DIT_ERR_CUDA, "gemm_tc: cuTensorMapEncodeTiled (x) failed");
      return launch_bn<EPI_GATE_RESID>(bn, ta, tb, tx, ep, M, N, Ka, st, k_wrap);
    }
    default: DIT_REQUIRE(false, DIT_ERR_INVALID_ARG, "gemm_tc: epilogue %d", epi);
  }
}

// Projection with QK-RMSNorm + RoPE in the epilogue (head_dim 128): columns [0, q_end) are q heads (gain gq), [q_end, k_end)
// k heads (gain gk), the rest v heads (bias only); q_end, k_end, N multiples of 128.  256-wide tiles only: a tile is two
// whole heads.  Self-attention QKV: (D, 2D, N = 3D); cross-attention q: (D, D, N = D); cross-attention k | v: (0, D, N = 2D).
dit_status launch_gemm_tc_qkv(const void* A, int64_t lda, const void* W, const void* bias, void* out, int64_t ldo,
                              const void* gq, const void* gk, float rms_eps, const float* rc, const float* rs, int q_end,
                              int k_end, int M, int N, int K, cudaStream_t st, int a_split) {
  if (M == 0 || N == 0) return DIT_OK;
  DIT_REQUIRE(!a_split || K % BK == 0, DIT_ERR_INVALID_ARG, "gemm_tc_qkv: split A needs K %% 64 == 0 (K=%d)", K);
  const int k_wrap = a_split ? K / BK : 0;
  const int Ka = a_split ? 2 * K : K;
  DIT_REQUIRE(q_end % 128 == 0 && k_end % 128 == 0 && N % 128 == 0 && 0 <= q_end && q_end <= k_end && k_end <= N,
              DIT_ERR_INVALID_ARG, "gemm_tc_qkv: N=%d q_end=%d k_end=%d", N, q_end, k_end);
  CUtensorMap ta, tb;
  DIT_REQUIRE(make_tmap_2d_bf16(&ta, A, M, Ka, lda, BM, BK) && make_tmap_2d_bf16(&tb, W, N, K, K, 128, BK), DIT_ERR_CUDA,
              "gemm_tc_qkv: cuTensorMapEncodeTiled failed (M=%d N=%d K=%d)", M, N, K);
  EpiArgs ep{(const bf16*)bias, nullptr, out, ldo, nullptr, 0, nullptr, 1, (const bf16*)gq, (const bf16*)gk, rc, rs, rms_eps, q_end, k_end, nullptr, nullptr, nullptr, nullptr, nullptr, nullptr, 0, -1};
  ProfScope _prof(DIT_KC_GEMM, st);
  CUtensorMap tn;   // W as 64-row boxes: the half tiles of the tail wave
  DIT_REQUIRE(make_tmap_2d_bf16(&tn, W, N, K, K, 64, BK), DIT_ERR_CUDA, "gemm_tc_qkv: cuTensorMapEncodeTiled (narrow W) failed");
  ep.narrow_from = narrow_tail_from(cdiv(cdiv(M, BM), 2) * cdiv(N, 256));
  return launch_t<EPI_QKV_NORM_ROPE, 256>(ta, tb, tn, ep, M, N, Ka, st, k_wrap);
}

// Gated-MLP up-projection (R40): out bf16 [M, ldo] <- SiLU(A W1^T + b1) (.) (A W3^T + b3); W1, W3 [N, K], b1, b3 [N].
dit_status launch_gemm_tc_swiglu(const void* A, int64_t lda, const void* W1, const void* b1, const void* W3, const void* b3,
                                 void* out, int64_t ldo, int M, int N, int K, cudaStream_t st) {
  if (M == 0 || N == 0) return DIT_OK;
  CUtensorMap ta, tb, tx;
  DIT_REQUIRE(make_tmap_2d_bf16(&ta, A, M, K, lda, BM, BK) && make_tmap_2d_bf16(&tb, W1, N, K, K, 128, BK) &&
                  make_tmap_2d_bf16(&tx, W3, N, K, K, 128, BK),
              DIT_ERR_CUDA, "gemm_tc_swiglu: cuTensorMapEncodeTiled failed (M=%d N=%d K=%d)", M, N, K);
  EpiArgs ep{(const bf16*)b1, (const bf16*)b3, out, ldo, nullptr, 0, nullptr, 1, nullptr, nullptr, nullptr, nullptr, 0.f, 0, 0, nullptr, nullptr, nullptr, nullptr, nullptr, nullptr, 0, -1};
  ProfScope _prof(DIT_KC_GEMM, st);
  return launch_t<EPI_SWIGLU, 256>(ta, tb, tx, ep, M, N, K, st, 0);
}

// One launch over every row segment of a packed buffer, two weight sets (dual-stream blocks, R37); see GemmSegs / SegGemm.
dit_status launch_gemm_tc_segs(const SegGemm& g, cudaStream_t st) {
  if (g.M == 0 || g.N == 0 || g.segs == nullptr || g.segs->n == 0) return DIT_OK;
  const GemmSegs& sg = *g.segs;
  const int mt2 = sg.tile0[sg.n];
  const bool wide = g.kind == EPI_QKV_NORM_ROPE || g.kind == EPI_SWIGLU;    // 256-wide tiles only
  const int bn = wide ? 256 : pick_bn(g.M, g.N, mt2);
  const int wbox = wide ? 128 : bn / 2;
  const void* W0 = g.W[0];
  const void* W1 = g.W[1] != nullptr ? g.W[1] : g.W[0];
  CUtensorMap ta, tb, tb2, tx, tx2;
  DIT_REQUIRE(make_tmap_2d_bf16(&ta, g.A, g.M, g.K, g.lda, BM, BK) && make_tmap_2d_bf16(&tb, W0, g.N, g.K, g.K, wbox, BK) &&
                  make_tmap_2d_bf16(&tb2, W1, g.N, g.K, g.K, wbox, BK),
              DIT_ERR_CUDA, "gemm_tc_segs: cuTensorMapEncodeTiled failed (M=%d N=%d K=%d)", g.M, g.N, g.K);
  tx = ta; tx2 = ta;
  if (g.kind == EPI_SWIGLU) {
    DIT_REQUIRE(make_tmap_2d_bf16(&tx, g.W3[0], g.N, g.K, g.K, 128, BK) &&
                    make_tmap_2d_bf16(&tx2, g.W3[1] != nullptr ? g.W3[1] : g.W3[0], g.N, g.K, g.K, 128, BK),
                DIT_ERR_CUDA, "gemm_tc_segs: cuTensorMapEncodeTiled (W3) failed");
  } else if (g.kind == EPI_GATE_RESID) {
    DIT_REQUIRE(make_tmap_2d_f32(&tx, g.out, g.M, g.N, g.ldo, 32), DIT_ERR_CUDA, "gemm_tc_segs: cuTensorMapEncodeTiled (x) failed");
    tx2 = tx;
  }
  EpiArgs ep{(const bf16*)g.bias[0], (const bf16*)g.b3[0], g.out, g.ldo, g.gate, g.gate_stride, nullptr, 1,
             (const bf16*)g.gq[0], (const bf16*)g.gk[0], g.rc, g.rs, g.rms_eps, g.N / 3, 2 * (g.N / 3), nullptr, nullptr,
             (const bf16*)g.bias[1], (const bf16*)g.b3[1], (const bf16*)g.gq[1], (const bf16*)g.gk[1], g.gate_set_off, -1};
  const SegLaunch sl{g.segs, &tb2, &tx2};
  ProfScope _prof(DIT_KC_GEMM, st);
  switch (g.kind) {
    case DIT_EPI_BIAS: return launch_bn<DIT_EPI_BIAS>(bn, ta, tb, tx, ep, g.M, g.N, g.K, st, 0, &sl);
    case DIT_EPI_BIAS_GELU: return launch_bn<DIT_EPI_BIAS_GELU>(bn, ta, tb, tx, ep, g.M, g.N, g.K, st, 0, &sl);
    case EPI_GATE_RESID: return launch_bn<EPI_GATE_RESID>(bn, ta, tb, tx, ep, g.M, g.N, g.K, st, 0, &sl);
    case EPI_QKV_NORM_ROPE:
      DIT_REQUIRE(g.N % 384 == 0, DIT_ERR_INVALID_ARG, "gemm_tc_segs: QKV needs N = 3 D, D %% 128 == 0 (N=%d)", g.N);
      DIT_REQUIRE(make_tmap_2d_bf16(&tx, W0, g.N, g.K, g.K, 64, BK) && make_tmap_2d_bf16(&tx2, W1, g.N, g.K, g.K, 64, BK), DIT_ERR_CUDA,
                  "gemm_tc_segs: cuTensorMapEncodeTiled (narrow W) failed");
      ep.narrow_from = narrow_tail_from(mt2 * cdiv(g.N, 256));
      return launch_t<EPI_QKV_NORM_ROPE, 256>(ta, tb, tx, ep, g.M, g.N, g.K, st, 0, &sl);
    case EPI_SWIGLU: return launch_t<EPI_SWIGLU, 256>(ta, tb, tx, ep, g.M, g.N, g.K, st, 0, &sl);
    default: DIT_REQUIRE(false, DIT_ERR_INVALID_ARG, "gemm_tc_segs: kind %d", g.kind);
  }
}

// fp8 linear layer (R42): out = e(decode(Aq) decode(Wq)^T (.) a_scale w_scale^T + bias); Aq [M, lda bytes], Wq [N, K] e4m3
// bytes, scales fp32, bias bf16 (or nullptr), out bf16 (e = BIAS, BIAS_GELU) or fp32 (BIAS_F32).
dit_status launch_gemm_tc_fp8(int epi, const void* Aq, int64_t lda, const float* a_scale, const void* Wq, const float* w_scale,
                              const void* bias, void* out, int64_t ldo, int M, int N, int K, cudaStream_t st) {
  if (M == 0 || N == 0) return DIT_OK;
  DIT_REQUIRE(K > 0 && K % 16 == 0 && lda % 16 == 0 && N % 8 == 0 && ldo % 8 == 0, DIT_ERR_UNSUPPORTED,
              "gemm_tc_fp8: K (%d) and lda (%lld) must be multiples of 16, N (%d) and ldo (%lld) of 8", K, (long long)lda, N, (long long)ldo);
  DIT_REQUIRE(!(((uintptr_t)Aq | (uintptr_t)Wq | (uintptr_t)out) & 15), DIT_ERR_UNSUPPORTED, "gemm_tc_fp8: pointers must be 16-byte aligned");
  DIT_REQUIRE(a_scale != nullptr && w_scale != nullptr, DIT_ERR_INVALID_ARG, "gemm_tc_fp8: scales are NULL");
  CUtensorMap ta, tb;
  const int bn = pick_bn(M, N);
  DIT_REQUIRE(make_tmap_2d_u8(&ta, Aq, M, K, lda, BM) && make_tmap_2d_u8(&tb, Wq, N, K, K, bn / 2), DIT_ERR_CUDA,
              "gemm_tc_fp8: cuTensorMapEncodeTiled failed (M=%d N=%d K=%d lda=%lld)", M, N, K, (long long)lda);
  EpiArgs ep{(const bf16*)bias, nullptr, out, ldo, nullptr, 0, nullptr, 1, nullptr, nullptr, nullptr, nullptr, 0.f, 0, 0, a_scale, w_scale, nullptr, nullptr, nullptr, nullptr, 0, -1};
  ProfScope _prof(DIT_KC_GEMM, st);
  switch (epi) {
    case DIT_EPI_BIAS: return launch_bn<EPI_F8 + DIT_EPI_BIAS>(bn, ta, tb, ta, ep, M, N, K, st, 0);
    case DIT_EPI_BIAS_GELU: return launch_bn<EPI_F8 + DIT_EPI_BIAS_GELU>(bn, ta, tb, ta, ep, M, N, K, st, 0);
    case DIT_EPI_BIAS_F32: return launch_bn<EPI_F8 + DIT_EPI_BIAS_F32>(bn, ta, tb, ta, ep, M, N, K, st, 0);
    default: DIT_REQUIRE(false, DIT_ERR_INVALID_ARG, "gemm_tc_fp8: epilogue %d", epi);
  }
}

// Block-scaled MXFP8 layer on the pair kernel (R43): Aq [M, lda], Wq [N, K] e4m3 bytes; sfa [M, K / 32], sfw [N, K / 32] E8M0.
dit_status launch_gemm_tc_mx(int epi, const void* Aq, int64_t lda, const void* sfa, const void* Wq, const void* sfw, const void* bias,
                             void* out, int64_t ldo, int M, int N, int K, cudaStream_t st) {
  if (M == 0 || N == 0) return DIT_OK;
  DIT_REQUIRE(K > 0 && K % 512 == 0 && lda % 16 == 0 && N % 8 == 0 && ldo % 8 == 0, DIT_ERR_UNSUPPORTED,
              "gemm_tc_mx: K (%d) must be a multiple of 512, lda (%lld) of 16, N (%d) and ldo (%lld) of 8", K, (long long)lda, N, (long long)ldo);
  constexpr int BNX = 224;
  CUtensorMap ta, tb;
  DIT_REQUIRE(make_tmap_2d_u8(&ta, Aq, M, K, lda, BM) && make_tmap_2d_u8(&tb, Wq, N, K, K, BNX / 2), DIT_ERR_CUDA,
              "gemm_tc_mx: cuTensorMapEncodeTiled failed (M=%d N=%d K=%d lda=%lld)", M, N, K, (long long)lda);
  EpiArgs ep{};
  ep.bias = (const bf16*)bias; ep.out = out; ep.ldo = ldo; ep.R = 1; ep.narrow_from = -1;
  ep.mx_sfa = (const uint8_t*)sfa; ep.mx_sfw = (const uint8_t*)sfw;
  ProfScope _prof(DIT_KC_GEMM, st);
  switch (epi) {
    case DIT_EPI_BIAS: return launch_t<EPI_MX + DIT_EPI_BIAS, BNX>(ta, tb, ta, ep, M, N, K, st, 0);
    case DIT_EPI_BIAS_GELU: return launch_t<EPI_MX + DIT_EPI_BIAS_GELU, BNX>(ta, tb, ta, ep, M, N, K, st, 0);
    case DIT_EPI_BIAS_F32: return launch_t<EPI_MX + DIT_EPI_BIAS_F32, BNX>(ta, tb, ta, ep, M, N, K, st, 0);
    default: DIT_REQUIRE(false, DIT_ERR_INVALID_ARG, "gemm_tc_mx: epilogue %d", epi);
  }
}

dit_status launch_gemm_tc(int epi, const void* A, int64_t lda, const void* W, const void* bias, void* out, int64_t ldo,
                          int M, int N, int K, cudaStream_t st, int a_split) {
  return launch_gemm_tc_ex(epi, A, lda, W, bias, out, ldo, nullptr, 0, nullptr, 1, M, N, K, st, a_split);
}

}  // namespace dit
