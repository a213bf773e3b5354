// attn_tc.cu — non-causal flash attention on tcgen05 tensor cores (north_star subsystems 4 and 5), head_dim 128, bf16.
//   for every query row i of a request, over the key rows of this call's KV shard:
//     s_ij = scale * q_i . k_j ;  o_i = sum_j softmax_j(s_ij) v_j ;  lse_i = ln sum_j exp(s_ij)        (R7, R18)
// Design (sm_100a), one CTA = one (request, head, 256 query rows) work item, 640 threads:
//   warp 0      TMA producer: two Q tiles (128 x 128) once, then a K ring and a V ring of 128-key tiles
//               (each tile = two 128 x 64 boxes, 128-byte swizzle);
//   warp 1      MMA issuer (one elected thread).  Per key tile j and Q tile t:  S_t = Q_t K_j^T as ONE N = 128 group
//               (M=128, N=128, K=16 x 8: 8 KB of shared memory per 64-cycle MMA = the 128 B/clk feed limit; measured:
//               N = 64 groups take 48 instead of 32 cycles each) into the two 64-column buffers S_t,a | S_t,b; then
//               O_t += P_t,a V_j[0:64] and O_t += P_t,b V_j[64:128] (M=128, N=128, K=16 x 4 each) with P read from
//               TMEM (A operand in tensor memory) and V as an MN-major shared-memory operand; then S_t of tile j+1
//               (the tensor pipe executes in issue order, so it may overwrite the P buffers right behind the PVs).
//               t = 0 is served completely before t = 1: one tile's softmax runs under the other tile's MMAs;
//   warps 4-19  softmax: Q tile t has TWO warps per TMEM lane quadrant — the leader owns sub-tile a (keys 0..63 of
//               every key tile), the follower sub-tile b — so four softmax warps share a scheduler.  One thread =
//               one query row x 64 keys: tcgen05.ld, half-row max, exchange of the two half-row maxima through
//               shared memory + a named barrier (both threads then take the SAME lazy-rescale decision), exp2 with
//               the scale folded into one packed FFMA2, bf16 P written over the first 32 columns of the S buffer
//               (tcgen05.st), fp32 row sum (packed FADD2).  An eighth of the exponentials runs on the FMA pipe
//               (round-to-nearest split + minimax cubic, rel. error 7.5e-5 << bf16 rounding of P) to take load off
//               MUFU.EX2 (16 / clk / SM: as many cycles as the tile's MMAs).  O is rescaled lazily: only when the
//               running max grows by more than 2^8 (exact: the same max is used for P and for the sum, and divided
//               out at the end); the leader rescales O_t, both threads rescale their partial row sums;
//               That is the EXACT tile.  Pass 0 of a CTA is optimistic (R33): only its first key tile is exact;
//               the others compute no row max (any reference is exact while nothing overflows), the pair only looks at
//               its recent row sums every 4th tile — before it waits for S, off the S -> P -> PV chain — and moves the
//               reference when they have grown by 2^30.  A tile sum above 2^60 raises the CTA's panic flag and the
//               CTA (CTA pair) repeats all key tiles as pass 1 with exact tiles only;
//   epilogue    the pair adds its partial sums; leader writes O columns 0..63, follower 64..127: O / l -> bf16,
//               lse = ln2 * (m + log2 l).
// TMEM: S0a S0b | S1a S1b | O0 | O1 = 4 x 128 fp32 columns = all 512; P_t,b aliases the first 32 columns of S_t,b.
// Registers: 640 threads x 96 at launch; setmaxnreg moves the control warps to 40 and the softmax warps to 104
// (the pool is the CTA's launch allocation: asking for more than the control warps release never returns).
// Roofline: tensor pipe; the softmax instruction stream (312 instructions per 64 scores in an optimistic tile, 379 in
// an exact one; MUFU.EX2 at 16 / clk / SM) is co-critical.
#include <algorithm>
#include <cstdio>
#include <cstdlib>
#include <type_traits>

#include "tc.cuh"

namespace dit {
using namespace tc;

namespace {

constexpr int HD = 128;          // head dim
constexpr int TQ = 128;          // query rows per tile (2 tiles per CTA)
constexpr int TK = 128;          // keys per TMA tile
constexpr int SK = 64;           // keys per S / P sub-tile (two sub-tiles per TMA tile)
constexpr int KS = 2, VS = 2;    // K / V ring depths
constexpr int TILE_BYTES = 128 * HD * 2;   // 32 KB: two [128 x 64] swizzled boxes
constexpr int HALF_BYTES = TILE_BYTES / 2;
constexpr int SUB_BYTES = SK * 128;        // 64 rows of a swizzled box
constexpr int ATTN_THREADS = 640;         // 4 control warps + 16 softmax warps
constexpr int ATTN_SMEM = (2 + KS + VS) * TILE_BYTES + 1024 + 256 + 6144;   // + row max / row sum exchange
constexpr float RESCALE_THRESHOLD = 8.0f;  // log2 units
#ifndef DIT_ATTN_POLY_PAIRS
#define DIT_ATTN_POLY_PAIRS 2
#endif
#ifndef DIT_ATTN_OPTIMISTIC
#define DIT_ATTN_OPTIMISTIC 1
#endif
#ifndef DIT_ATTN_OPT_PERIOD
#define DIT_ATTN_OPT_PERIOD 4
#endif
constexpr int OPT_PERIOD = DIT_ATTN_OPT_PERIOD;   // optimistic tiles between two looks at the row sums (power of 2)
constexpr bool OPTIMISTIC = DIT_ATTN_OPTIMISTIC != 0;   // 0: every key tile takes the exact path (row max per tile)
constexpr int POLY_PAIRS = DIT_ATTN_POLY_PAIRS;   // of every 16 score pairs, this many take the FMA-pipe exp2

struct AttnParams {
  bf16* o; int64_t o_stride;
  float* lse;
  const int32_t* cu_q; const int32_t* cu_k;
  int n_q, n_k, H;
  float scale_log2;   // softmax scale * log2(e)
  int shard, n_shards;
  int R, n_items;     // pair kernel: requests, work items = sum over requests of 256-row query blocks x heads
  uint8_t order[64];  // blockIdx.z -> request, longest key sequence first: the last wave is made of short items
};

__device__ __forceinline__ float ex2(float x) {
  float y;
  asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
  return y;
}
// packed fp32 pairs (sm_100 FFMA2 / FADD2): one issue slot for two elements
__device__ __forceinline__ uint64_t pack2(float lo, float hi) {
  uint64_t r;
  asm("mov.b64 %0, {%1, %2};" : "=l"(r) : "f"(lo), "f"(hi));
  return r;
}
__device__ __forceinline__ void unpack2(uint64_t v, float& lo, float& hi) {
  asm("mov.b64 {%0, %1}, %2;" : "=f"(lo), "=f"(hi) : "l"(v));
}
__device__ __forceinline__ uint64_t fma2(uint64_t a, uint64_t b, uint64_t c) {
  uint64_t d;
  asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(d) : "l"(a), "l"(b), "l"(c));
  return d;
}
__device__ __forceinline__ uint64_t add2(uint64_t a, uint64_t b) {
  uint64_t d;
  asm("add.rn.f32x2 %0, %1, %2;" : "=l"(d) : "l"(a), "l"(b));
  return d;
}
// 2^x on the FMA pipe for a packed pair, x <= ~9:  x = n + f, n = rint(x), f in [-0.5, 0.5];
// 2^f ~ minimax cubic (rel. error 7.5e-5), 2^n by adding n to the exponent field.  x is clamped at -126 so the
// exponent cannot wrap (masked scores are -inf): the result is then < 2^-125, i.e. zero for every purpose here.
__device__ __forceinline__ void ex2_poly2(uint64_t x2, float& a, float& b) {
  float xa, xb;
  unpack2(x2, xa, xb);
  xa = fmaxf(xa, -126.0f);
  xb = fmaxf(xb, -126.0f);
  const uint64_t x = pack2(xa, xb);
  const uint64_t magic = pack2(12582912.0f, 12582912.0f);      // 1.5 * 2^23: low mantissa bits hold rint(x)
  const uint64_t nmagic = pack2(-12582912.0f, -12582912.0f);
  const uint64_t r = add2(x, magic);
  const uint64_t n = add2(r, nmagic);
  const uint64_t neg1 = pack2(-1.0f, -1.0f);
  const uint64_t f = fma2(n, neg1, x);                          // x - n, exact
  uint64_t p = fma2(f, pack2(0.05517132207751274f, 0.05517132207751274f), pack2(0.24261054396629333f, 0.24261054396629333f));
  p = fma2(p, f, pack2(0.6932609677314758f, 0.6932609677314758f));
  p = fma2(p, f, pack2(0.9999281167984009f, 0.9999281167984009f));
  float ra, rb, pa, pb;
  unpack2(r, ra, rb);
  unpack2(p, pa, pb);
  a = __int_as_float(__float_as_int(pa) + (__float_as_int(ra) << 23));
  b = __int_as_float(__float_as_int(pb) + (__float_as_int(rb) << 23));
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
// p = 2^(s c + nm) for 32 scores -> 16 bf16 pairs into TMEM columns [taddr, taddr + 16); packed fp32 partial sums
__device__ __forceinline__ void exp_pack_store(const uint32_t (&s)[32], uint64_t c2, uint64_t nm2, uint32_t taddr,
                                               uint64_t& sum2, uint64_t& sum2b) {
  uint32_t pk[16];
#pragma unroll
  for (int i = 0; i < 16; ++i) {
    const uint64_t x = fma2(pack2(__uint_as_float(s[2 * i]), __uint_as_float(s[2 * i + 1])), c2, nm2);
    float a, b;
    if (i % 4 == 3 && i / 4 < POLY_PAIRS) {   // spread over the chunk so MUFU and FMA work interleave
      ex2_poly2(x, a, b);
    } else {
      float xa, xb;
      unpack2(x, xa, xb);
      a = ex2(xa);
      b = ex2(xb);
    }
    if (i & 1) sum2b = add2(sum2b, pack2(a, b));   // two independent chains
    else sum2 = add2(sum2, pack2(a, b));
    pk[i] = pack_bf16(a, b);
  }
  tmem_st16(taddr, pk);
}

// PAIR: launched as clusters of two CTAs that are adjacent 256-row query blocks of the same (request, head): both walk
// the same key tiles, so each CTA fetches ONE of the two 64-column boxes of every K / V tile and TMA-multicasts it to
// both (L2 -> SM traffic of the K / V stream halves); a ring stage is refilled when both CTAs have released it.
template <bool PAIR>
__global__ void __launch_bounds__(ATTN_THREADS, 1)
attn_tc_kernel(const __grid_constant__ CUtensorMap tmQ, const __grid_constant__ CUtensorMap tmK,
               const __grid_constant__ CUtensorMap tmV, AttnParams p) {
  pdl_trigger();
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
  constexpr int B0 = 2 + 2 * KS + 2 * VS;
  auto s_full = [&](int t, int b) { return bar0 + 8u * (B0 + 2 * t + b); };
  auto p_full = [&](int t, int b) { return bar0 + 8u * (B0 + 4 + 2 * t + b); };
  // PV_t,i completes pv_done(t, i & 1): a waiter is never more than one phase behind a per-buffer barrier
  auto pv_done = [&](int t, int b) { return bar0 + 8u * (B0 + 8 + 2 * t + b); };
  const uint32_t tmem_slot = bar0 + 8u * (B0 + 12);
  const uint32_t panic_addr = bar0 + 8u * (B0 + 13);   // set by a softmax warp whose optimistic pass overflowed

  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int req = p.cu_q ? p.order[blockIdx.z] : 0, head = blockIdx.y;
  const int q_lo = p.cu_q ? p.cu_q[req] : 0, q_hi = p.cu_q ? p.cu_q[req + 1] : p.n_q;
  const int q_base = q_lo + blockIdx.x * (2 * TQ);
  if (!PAIR && q_base >= q_hi) return;  // CTA-uniform (pairs are only launched when every block has rows)
  const uint32_t crank = PAIR ? cluster_ctarank() : 0u;
  const int k_lo0 = p.cu_k ? p.cu_k[req] : 0, k_hi0 = p.cu_k ? p.cu_k[req + 1] : p.n_k;
  const int klen = k_hi0 - k_lo0;
  const int ssz = (klen + p.n_shards - 1) / p.n_shards;
  int k_lo = k_lo0 + p.shard * ssz, k_hi = k_lo0 + (p.shard + 1) * ssz;
  if (k_lo > k_hi0) k_lo = k_hi0;
  if (k_hi > k_hi0) k_hi = k_hi0;
  const int kv_len = k_hi - k_lo;
  const int n_tiles = (kv_len + TK - 1) / TK;
  const int n_sub = (kv_len + SK - 1) / SK;

  if (n_tiles == 0) {  // empty shard: o = 0, lse = -inf (R18)
    pdl_wait();
    if (warp >= 4 && ((warp - 4) & 4) == 0) {   // the leader warps cover the 256 rows once
      const int row = q_base + ((warp - 4) >> 3) * TQ + (warp & 3) * 32 + lane;
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
      for (int b = 0; b < 2; ++b) {
        mbar_init(pv_done(t, b), 1);
        mbar_init(s_full(t, b), 1);
        mbar_init(p_full(t, b), 4);      // one arrival per softmax warp
      }
    }
    // empty: one commit per Q tile (and per CTA of a pair)
    for (int s = 0; s < KS; ++s) { mbar_init(k_full(s), 1); mbar_init(k_empty(s), PAIR ? 4 : 2); }
    for (int s = 0; s < VS; ++s) { mbar_init(v_full(s), 1); mbar_init(v_empty(s), PAIR ? 4 : 2); }
    asm volatile("st.shared.u32 [%0], %1;" ::"r"(panic_addr), "r"(0u) : "memory");
    fence_barrier_init();
  }
  if (warp == 2) tmem_alloc<512>(tmem_slot);
  tc_fence_before();
  __syncthreads();
  if (PAIR) cluster_sync_all();   // the peer's barriers exist before anything is multicast to them
  tc_fence_after();
  uint32_t tmem_base;
  asm volatile("ld.shared.b32 %0, [%1];" : "=r"(tmem_base) : "r"(tmem_slot));
  pdl_wait();   // prologue done; q / k / v written by the previous kernel are read from here on

  // register budget: warpgroup 0 (TMA / MMA / idle warps) gives registers to the two softmax warpgroups

  // Pass 0 is OPTIMISTIC (no row max after the first key tile, see the softmax warps); it is exact unless a row's
  // scores outgrow the reference by ~2^60 inside one key tile, which a thread notices from its row sum.  Then the
  // whole CTA (the whole pair) runs pass 1, the exact algorithm with a row max per tile, over the same keys: every
  // ring stage / barrier phase simply continues (tile counter g = pass * n_tiles + j).
  const int cnt_b1 = n_sub - n_tiles;   // key tiles per pass that have a sub-tile b (the ragged last one may not)
  // pass boundary: does the optimistic result stand?  (CTA-wide; a pair decides together — its CTAs share every K / V
  // stage, so both repeat or neither does.)  Called by every thread of the CTA, from either register-budget branch.
  auto repeat_exact = [&]() -> bool {
    tc_fence_before();
    if (PAIR) cluster_sync_all(); else __syncthreads();
    tc_fence_after();
    uint32_t redo;
    asm volatile("ld.shared.u32 %0, [%1];" : "=r"(redo) : "r"(panic_addr) : "memory");
    if (PAIR) {
      uint32_t peer;
      asm volatile("ld.shared::cluster.u32 %0, [%1];" : "=r"(peer) : "r"(mapa_cluster(panic_addr, crank ^ 1u)) : "memory");
      redo |= peer;
    }
    return redo != 0;
  };
  if (warp < 4) {
  asm volatile("setmaxnreg.dec.sync.aligned.u32 40;");
  int sk = 0, sv = 0;                   // TMA producer ring state, runs on across passes
  uint32_t pk = 0, pv = 0;
  for (int pass = 0;; ++pass) {
    const bool exact = !OPTIMISTIC || pass == 1;
    const int gb = pass * n_tiles;      // global index of this pass's first key tile
  if (warp == 0) {
    // ===================================================== TMA producer
    const int c0 = head * HD;
    if (pass == 0 && elect_one()) {
      for (int t = 0; t < 2; ++t) {
        mbar_expect_tx(q_full(t), TILE_BYTES);
        tma_load_2d(sQ + t * TILE_BYTES, &tmQ, c0, q_base + t * TQ, q_full(t));
        tma_load_2d(sQ + t * TILE_BYTES + HALF_BYTES, &tmQ, c0 + 64, q_base + t * TQ, q_full(t));
      }
    }
    for (int j = 0; j < n_tiles; ++j) {
      const int r0 = k_lo + j * TK;
      mbar_wait(k_empty(sk), pk ^ 1);
      if (elect_one()) {
        mbar_expect_tx(k_full(sk), TILE_BYTES);
        if (PAIR) {
          tma_load_2d_multicast(sK + sk * TILE_BYTES + crank * HALF_BYTES, &tmK, c0 + crank * 64, r0, k_full(sk), (uint16_t)3);
        } else {
          tma_load_2d(sK + sk * TILE_BYTES, &tmK, c0, r0, k_full(sk));
          tma_load_2d(sK + sk * TILE_BYTES + HALF_BYTES, &tmK, c0 + 64, r0, k_full(sk));
        }
      }
      if (++sk == KS) { sk = 0; pk ^= 1; }
      mbar_wait(v_empty(sv), pv ^ 1);
      if (elect_one()) {
        mbar_expect_tx(v_full(sv), TILE_BYTES);
        if (PAIR) {
          tma_load_2d_multicast(sV + sv * TILE_BYTES + crank * HALF_BYTES, &tmV, c0 + crank * 64, r0, v_full(sv), (uint16_t)3);
        } else {
          tma_load_2d(sV + sv * TILE_BYTES, &tmV, c0, r0, v_full(sv));
          tma_load_2d(sV + sv * TILE_BYTES + HALF_BYTES, &tmV, c0 + 64, r0, v_full(sv));
        }
      }
      if (++sv == VS) { sv = 0; pv ^= 1; }
      __syncwarp();
    }
  } else if (warp == 1) {
    // ===================================================== MMA issuer
    constexpr uint32_t idesc_s = idesc_bf16(TQ, TK, 0, 0);   // S = Q K^T: A, B K-major, N = 128 keys (both sub-tiles)
    constexpr uint32_t idesc_o = idesc_bf16(TQ, HD, 0, 1);   // O += P V: A from TMEM, B (V) MN-major
    // V tile: two [128 keys x 64 d] boxes 16 KB apart (LBO), 8-key groups 1 KB apart (SBO); 16 keys = +2 KB
    constexpr uint64_t vdesc_hi = desc_base_sw128(HALF_BYTES >> 4, 64);
    // S of key tile g for Q tile t: ONE N = 128 group fills both 64-column buffers (8 KB of shared memory per
    // 64-cycle MMA = 128 B/clk; N = 64 groups would re-read Q for half the work and run shared-memory bound)
    auto issue_s = [&](int t, int g) {
      const uint32_t d = tmem_base + t * 128;
      const uint32_t qa = sQ + t * TILE_BYTES, ka = sK + (g % KS) * TILE_BYTES;
#pragma unroll
      for (int k = 0; k < HD / 16; ++k) {
        const uint32_t off = (k >> 2) * HALF_BYTES + (k & 3) * 32;
        umma_ss(d, desc_kmajor_sw128(qa + off), desc_kmajor_sw128(ka + off), idesc_s, k != 0);
      }
    };
    auto release = [&](uint32_t bar) {   // a K / V stage is free once the MMAs issued so far have read it
      if (PAIR) umma_commit_multicast(bar, (uint16_t)3);
      else umma_commit(bar);
    };
    // sub-tile b (0 / 1) of key tile g (ring stage g % VS, rows b * 64 ...); `first` = first PV of this pass
    auto issue_pv = [&](int t, int g, int b, bool first) {
      const uint32_t d = tmem_base + 256 + t * 128;
      const uint32_t pa = tmem_base + t * 128 + b * SK;  // P_t,b: bf16 pairs in the first 32 columns of S_t,b
      const uint32_t va = sV + (g % VS) * TILE_BYTES + b * SUB_BYTES;
#pragma unroll
      for (int k = 0; k < SK / 16; ++k)
        umma_ts(d, pa + 8 * k, vdesc_hi | (uint64_t)(((va + k * 2048) >> 4) & 0x3fff), idesc_o, (!first || k != 0) ? 1u : 0u);
    };
    // prologue: S of key tile 0 for both Q tiles
    mbar_wait(q_full(0), 0);
    mbar_wait(k_full(gb % KS), (uint32_t)(gb / KS) & 1u);
    tc_fence_after();
    if (elect_one()) { issue_s(0, gb); umma_commit(s_full(0, 0)); umma_commit(s_full(0, 1)); release(k_empty(gb % KS)); }
    mbar_wait(q_full(1), 0);
    tc_fence_after();
    if (elect_one()) { issue_s(1, gb); umma_commit(s_full(1, 0)); umma_commit(s_full(1, 1)); release(k_empty(gb % KS)); }
    __syncwarp();
    // Per key tile j and Q tile t: PV of sub-tile a, PV of sub-tile b, then S of key tile j + 1 (both P buffers are
    // consumed once the PVs are queued: the tensor pipe executes in issue order).  Serving t = 0 completely before
    // t = 1 keeps the two Q tiles in anti-phase: one tile's softmax runs under the other tile's 1024 tensor cycles.
    for (int j = 0; j < n_tiles; ++j) {
      const int g = gb + j;
      const bool has_b = 2 * j + 1 < n_sub;
      for (int t = 0; t < 2; ++t) {
        if (t == 0) mbar_wait(v_full(g % VS), (uint32_t)(g / VS) & 1u);
        mbar_wait(p_full(t, 0), (uint32_t)g & 1u);
        tc_fence_after();
        if (elect_one()) {
          issue_pv(t, g, 0, j == 0);
          umma_commit(pv_done(t, 0));
        }
        __syncwarp();
        if (has_b) {
          mbar_wait(p_full(t, 1), (uint32_t)(pass * cnt_b1 + j) & 1u);
          tc_fence_after();
          if (elect_one()) {
            issue_pv(t, g, 1, false);
            umma_commit(pv_done(t, 1));
          }
          __syncwarp();
        }
        if (j + 1 < n_tiles && t == 0) {
          mbar_wait(k_full((g + 1) % KS), (uint32_t)((g + 1) / KS) & 1u);
          tc_fence_after();
        }
        if (elect_one()) {
          release(v_empty(g % VS));
          if (j + 1 < n_tiles) {
            issue_s(t, g + 1);
            umma_commit(s_full(t, 0));
            umma_commit(s_full(t, 1));
            release(k_empty((g + 1) % KS));
          }
        }
        __syncwarp();
      }
    }
  }
    if (exact || !repeat_exact()) break;
  }
  } else {
  asm volatile("setmaxnreg.inc.sync.aligned.u32 104;");
  for (int pass = 0;; ++pass) {
    const bool exact = !OPTIMISTIC || pass == 1;
    const int gb = pass * n_tiles;
    // ===================================================== softmax + correction + epilogue: 16 warps
    // Q tile t has TWO warps per TMEM lane quadrant: the leader (h = 0) owns sub-tile a (keys 0..63 of every key
    // tile), the follower (h = 1) sub-tile b (keys 64..127); both add into the same O_t, so they must use the same
    // reference max.  Four softmax warps per scheduler instead of two: a single warp issues one instruction per ~3
    // cycles (dependent FFMA2 / MUFU chains), which made the softmax — not the tensor pipe and not MUFU — the
    // critical path.
    //   exact tile (every tile of pass 1, the first tile of pass 0): the pair exchanges its half-row maxima through
    //   shared memory + a named barrier (arrive / sync, 64 threads) and takes the same lazy-rescale decision (R25);
    //   optimistic tile (pass 0, j > 0): no row max at all.  Any reference is exact as long as nothing overflows
    //   (P, the row sum and O are all expressed against m_used, which is divided out at the end), so the reference
    //   only moves when the PREVIOUS tile's row sum shows that the scores have grown by 2^30: the pair exchanges
    //   last tile's partial sums BEFORE it waits for S(j) — off the S -> P -> PV chain.  A tile sum above 2^60
    //   (or infinite) raises the CTA's panic flag and the result of this pass is discarded (R33).
    const int w = warp - 4;
    const int t = w >> 3;                          // Q tile
    const int h = (w >> 2) & 1;                    // 0 = leader (sub-tile a), 1 = follower (sub-tile b)
    const int quad = warp & 3;                     // TMEM lane quadrant of this warp
    const int r_in = quad * 32 + lane;             // row inside the Q tile
    const int row = q_base + t * TQ + r_in;
    const uint32_t lane_off = (uint32_t)(quad * 32) << 16;
    const uint32_t s_base = tmem_base + t * 128 + lane_off;        // S_t,b (fp32, 64 cols) / P_t,b (bf16 pairs, 32 cols)
    const uint32_t o_addr = tmem_base + 256 + t * 128 + lane_off;  // O_t
    float* const xch = reinterpret_cast<float*>(smem_raw + (bar0 - smem_u32(smem_raw)) + 256);
    float* const m_sh = xch + t * 512;             // [parity][h][128 rows]: half-row maxima / last tile's partial sums
    float* const l_sh = xch + 1024 + t * 256;      // [h][128 rows]: partial row sums
    const int bar_id = 1 + t * 4 + quad;           // named barrier of this (leader, follower) warp pair
    const float c = p.scale_log2;
    const uint64_t c2 = pack2(c, c);
    float m_used = -INFINITY;   // reference (log2 units, raw score * c) that P and l are expressed against
    float l = 0.f;
    float tile_prev = 0.f;      // this thread's largest partial tile sum since the pair last looked
    uint32_t xs = 0;            // exchange slot: consecutive exchanges of a pair alternate between two buffers
    float tile_worst = 0.f;     // largest partial tile sum of this pass (panic test)
    const uint32_t s_addr = s_base + h * SK;
    auto rescale_o = [&](float f) {   // O_t *= f (leader only; O_t quiescent: S(j) complete and issued behind every PV)
#pragma unroll 1
      for (int cc = 0; cc < 8; ++cc) {
        uint32_t o[16];
        tmem_ld16(o_addr + cc * 16, o);
        tmem_ld_wait();
#pragma unroll
        for (int e = 0; e < 16; ++e) o[e] = __float_as_uint(__uint_as_float(o[e]) * f);
        tmem_st16(o_addr + cc * 16, o);
      }
      tmem_st_wait();
    };
    for (int j = 0; j < n_tiles; ++j) {
      const uint32_t par = (uint32_t)(gb + j) & 1u;
      uint32_t s0[32], s1[32];                     // the thread's 64 scores of its sub-tile
      const int valid = kv_len - j * TK - h * SK;  // keys of this sub-tile that exist (warp-uniform; <= 0: none)
      if (!exact && j > 0) {
        // ---------------------------------------- optimistic tile
        float tot = 0.f;
        if ((j & (OPT_PERIOD - 1)) == 0) {         // every OPT_PERIOD-th tile: largest partial sum since the last look
          m_sh[(xs * 2 + h) * 128 + r_in] = tile_prev;
          asm volatile("bar.sync %0, 64;" ::"r"(bar_id) : "memory");
          tot = tile_prev + m_sh[(xs * 2 + (h ^ 1)) * 128 + r_in];   // same value in both threads of the row
          xs ^= 1u;
          tile_prev = 0.f;
        }
        const bool need = tot > 1073741824.0f;     // 2^30
        if (valid > 0) {
          mbar_wait(s_full(t, h), par);
          tc_fence_after();
          tmem_ld32(s_addr + 0, s0);
        }
        if (__any_sync(0xffffffffu, need)) {       // rare: move the reference up by floor(log2 tot)
          if (valid <= 0) { mbar_wait(s_full(t, 0), par); tc_fence_after(); }
          const float e = need ? (float)(((__float_as_int(tot) >> 23) & 0xff) - 127) : 0.f;
          const float f = ex2(-e);
          if (h == 0) rescale_o(f);
          l *= f;
          m_used += e;
        }
        if (valid <= 0) { tile_prev = 0.f; continue; }   // ragged last tile without a sub-tile b (warp-uniform)
        const uint64_t nm2 = pack2(-m_used, -m_used);
        uint64_t sum2 = pack2(0.f, 0.f), sum2b = pack2(0.f, 0.f);
        tmem_ld_wait();
        tmem_ld32(s_addr + 32, s1);
        if (valid < SK) mask32(s0, valid);         // -inf -> P = 0
        exp_pack_store(s0, c2, nm2, s_addr + 0, sum2, sum2b);
        tmem_ld_wait();
        if (valid < SK) mask32(s1, valid - 32);
        exp_pack_store(s1, c2, nm2, s_addr + 16, sum2, sum2b);
        float sa, sb;
        unpack2(add2(sum2, sum2b), sa, sb);
        tile_prev = fmaxf(tile_prev, sa + sb);
        tile_worst = fmaxf(tile_worst, sa + sb);
        l += sa + sb;
        tmem_st_wait();
        tc_fence_before();
        __syncwarp();
        if (lane == 0) mbar_arrive(p_full(t, h));
        continue;
      }
      // ------------------------------------------ exact tile
      float mx = -INFINITY;
      if (valid > 0) {
        mbar_wait(s_full(t, h), par);
        tc_fence_after();
        // pass 1: the second 32 scores only for the row max (re-read after the exchange: a TMEM read is cheaper
        // than 32 live registers, which made ptxas recompute every address inside the loop); the first 32 stay
        tmem_ld32(s_addr + 32, s1);
        tmem_ld32(s_addr + 0, s0);
        tmem_ld_wait();
        if (valid < SK) {                          // -inf before the row max
          mask32(s0, valid);
          mask32(s1, valid - 32);
        }
        mx = fmaxf(max32(s0), max32(s1));
      }
      // the pair exchanges its half-row maxima: both threads then take the SAME rescale decision
      m_sh[(xs * 2 + h) * 128 + r_in] = mx;
      asm volatile("bar.sync %0, 64;" ::"r"(bar_id) : "memory");
      mx = fmaxf(mx, m_sh[(xs * 2 + (h ^ 1)) * 128 + r_in]);
      xs ^= 1u;
      const float m_new = fmaxf(m_used, mx * c);   // c > 0
      if (j == 0) {
        m_used = m_new;                            // PV_0 overwrites O: nothing to rescale
      } else {
        const bool need = (m_new - m_used) > RESCALE_THRESHOLD;
        if (__any_sync(0xffffffffu, need)) {
          // lazy rescale (rare).  S(j) is complete, and it was issued after every PV of tile j - 1, so O_t is
          // quiescent; PV_a(j) cannot be queued before the leader delivers P_a, and PV_b(j) is queued after PV_a(j),
          // so the leader alone rescales O_t; both threads rescale their partial row sums.
          const float f = need ? ex2(m_used - m_new) : 1.0f;
          if (h == 0) rescale_o(f);
          l *= f;
          if (need) m_used = m_new;
        }
      }
      if (valid <= 0) { tile_prev = 0.f; continue; }   // ragged last tile without a sub-tile b (warp-uniform)
      // P = 2^(s c - m_used): one packed FFMA per pair, EX2 (MUFU or FMA pipe), row sum in fp32, bf16 pairs -> TMEM
      const uint64_t nm2 = pack2(-m_used, -m_used);
      uint64_t sum2 = pack2(0.f, 0.f), sum2b = pack2(0.f, 0.f);
      tmem_ld32(s_addr + 32, s1);                  // pass 2 of the second half: S columns 32..63 are still intact
      exp_pack_store(s0, c2, nm2, s_addr + 0, sum2, sum2b);     // P columns 0..15 overwrite S columns 0..15 (consumed)
      tmem_ld_wait();
      if (valid < SK) mask32(s1, valid - 32);
      exp_pack_store(s1, c2, nm2, s_addr + 16, sum2, sum2b);
      float sa, sb;
      unpack2(add2(sum2, sum2b), sa, sb);
      tile_prev = sa + sb;
      l += tile_prev;
      tmem_st_wait();
      tc_fence_before();
      __syncwarp();
      if (lane == 0) mbar_arrive(p_full(t, h));
    }
    if (!exact && __any_sync(0xffffffffu, !(tile_worst < 1.152921504606847e18f)) && lane == 0)   // 2^60, inf
      asm volatile("st.shared.u32 [%0], %1;" ::"r"(panic_addr), "r"(1u) : "memory");
    // ---- epilogue: the pair exchanges its partial row sums; leader writes columns 0..63, follower 64..127
    // (its own barrier id, one per Q tile, 256 threads: the pair barrier may still hold the leader's last arrive).
    // After an optimistic pass it runs before the CTA knows whether the pass stands: pass 1 overwrites the output.
    l_sh[h * 128 + r_in] = l;
    asm volatile("bar.sync %0, 256;" ::"r"(9 + t) : "memory");
    l = l_sh[r_in] + l_sh[128 + r_in];
    {
      const int lb = (n_sub - 1) & 1;              // barrier of the last PV; completions so far, all passes
      const int done = (pass + 1) * (lb == 0 ? n_tiles : cnt_b1);
      mbar_wait(pv_done(t, lb), (uint32_t)(done - 1) & 1u);
    }
    tc_fence_after();
    const float inv = 1.0f / l;                    // l > 0: every tile has at least one valid key
    const bool row_ok = row < q_hi;
    bf16* orow = p.o + (int64_t)(row_ok ? row : q_lo) * p.o_stride + head * HD + h * 64;
#pragma unroll 1
    for (int cc = 0; cc < 2; ++cc) {
      uint32_t o[32];
      tmem_ld32(o_addr + h * 64 + cc * 32, o);
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
    if (h == 0 && row_ok && p.lse != nullptr) p.lse[(int64_t)row * p.H + head] = 0.6931471805599453f * (m_used + log2f(l));
    if (exact || !repeat_exact()) break;
  }
  }
  tc_fence_before();
  __syncthreads();
  if (PAIR) cluster_sync_all();   // the peer may still multicast into this CTA's shared memory / barriers
  if (warp == 2) {
    tc_fence_after();
    tmem_dealloc<512>(tmem_base);
  }
}


// =====================================================================================================================
// attn_pair_kernel — the same attention on CTA PAIRS (cta_group::2), ONE 256-row Q tile per pair, S and P in separate
// tensor-memory buffers.
//
// Why.  In attn_tc_kernel a CTA holds two Q tiles and TMEM is full with S0 S1 O0 O1; P(j) overwrites S(j), so S(j+1) of
// a tile cannot be queued before PV(j) of the same tile: the chain S -> softmax -> PV of a tile is hidden only by the
// other tile's 1024 tensor cycles.  Measured: the softmax warps wait for S 41 % of the time, tensor pipe 56-62 % busy.
// Here a CTA owns 128 Q rows only and TMEM is  S[0] S[1] | P[0] P[1] | O  (2 x 128 + 2 x 64 + 128 columns):
//   * an S buffer is free again as soon as the softmax warps have READ it (a few hundred cycles into the tile), not when
//     PV has consumed P: the issuer queues S(j+2) long before P(j) exists, and no softmax warp ever waits for S;
//   * P(j) is handed over at the end of the tile; PV(j) then has a whole tile time before P(j+2) needs the buffer.
// (A first version with three S buffers and P aliased over S — S(0) S(1) S(2) | PV(0) S(3) | ... — ran at 71 % tensor
//  utilisation: each buffer cycles through S, softmax, hand-off, PV, and three buffers per 4300-cycle cycle give one
//  tile per 1440 cycles; profiles/r02_ncu_attn_pair.md.)
// A single CTA cannot feed this from shared memory (S alone reads A + B = 8 KB per 64-cycle MMA = the whole 128 B/clk
// port, and the K / V stream is written on top); on a pair each CTA supplies its own 128 Q rows and HALF of every K / V
// tile (S: 64 keys; PV: 64 of the 128 d columns): 96 / 32 B/clk of operand reads + 32 B/clk of TMA writes.
//   warp 0      K producer (+ Q once): this CTA's 64 keys of every key tile (two [64 x 64] boxes), 5-deep ring
//   warp 2      V producer: this CTA's 64 d-columns of every key tile (one [128 x 64] box), 4-deep ring; TMEM allocation
//               (every box of both CTAs completes on the LEADER's full barrier; a stage is refilled when the leader's
//               commit, multicast to both CTAs, says the MMAs have read it)
//   warp 1      (leader CTA) one elected thread issues every MMA for both tensor cores, in the order the events arrive:
//               S(0) S(1) | S(2) PV(0) | S(3) PV(1) | ...   S(j) = Q K_j^T, M = 256, N = 128 keys, K = 16 x 8, into
//               S[j & 1] once the softmax has read S(j-2);  O += P(j) V_j, M = 256, N = 128 (d), K = 16 x 8, P[j & 1]
//               from tensor memory, V MN-major
//   warps 4-19  softmax, two groups of 8 warps in anti-phase: group g owns key tiles j = g (mod 2), S[g] and P[g]; the
//               leader warp of a TMEM lane quadrant takes keys 0..63 of the tile, the follower keys 64..127 (one thread =
//               one query row x 64 keys).  Events of BOTH CTAs are counted by the leader's barriers (relaxed remote
//               arrive from the peer, ~210 cycles, off the issuing warp).
// Reference (R33, simplified): P, the row sum and O are expressed against ONE reference m per row for the whole pass
// (divided out at the end: any m is exact while nothing overflows).  Pass 0 takes m = row max of the first key tile and
// never moves it; a tile sum above 2^60 (a score ~2^60 above m) raises the pair's panic flag, and the pair then runs
// pass 1 = row max over ALL key tiles (S MMAs only) and pass 2 = pass 0's loop with the true max as reference (the
// textbook two-pass softmax; cannot overflow).  O is never rescaled inside a pass.
// =====================================================================================================================
constexpr int PKS = 5, PVS = 4;                 // K / V ring depths
constexpr int PQ_BYTES = TQ * HD * 2;           // this CTA's 128 Q rows: two [128 x 64] boxes
constexpr int PQ_HALF = PQ_BYTES / 2;
constexpr int PKV_BYTES = 64 * HD * 2;          // a K stage (64 keys x 128 d: two [64 x 64] boxes) or a V stage ([128 keys x 64 d])
constexpr int PK_HALF = PKV_BYTES / 2;
constexpr int PAIR_BAR_BYTES = 512;
constexpr int PAIR_XCH_FLOATS = 4 * 128 + 128;   // [4][row]: 4-way reductions of a row's threads | the published reference
constexpr int PAIR_SMEM = 2 * PQ_BYTES + (PKS + PVS) * PKV_BYTES + 1024 + PAIR_BAR_BYTES + PAIR_XCH_FLOATS * 4;
constexpr uint32_t TM_S = 0, TM_P = 256, TM_O = 384;       // TMEM columns: S[g] = g * 128, P[g] = 256 + g * 64, O = 384
#ifndef DIT_ATTN_RELAXED_ARRIVE
#define DIT_ATTN_RELAXED_ARRIVE 1
#endif

#ifndef DIT_ATTN_PAIR_POLY_PAIRS
#define DIT_ATTN_PAIR_POLY_PAIRS 0
#endif
// In the pair kernel the softmax is bound by instruction issue, not by MUFU (XU pipe 58 % busy): every exponential on the
// MUFU is fastest (measured at N = 16384, H = 24: 0 / 2 / 4 polynomial pairs of 16: 1359 / 1326 / 1303 TFLOP/s).
constexpr int PAIR_POLY_PAIRS = DIT_ATTN_PAIR_POLY_PAIRS;
// p = 2^(s c + nm) for 32 scores -> 16 packed bf16 pairs in pk; packed fp32 partial sums
__device__ __forceinline__ void exp_pack(const uint32_t (&s)[32], uint64_t c2, uint64_t nm2, uint32_t (&pk)[16],
                                         uint64_t& sum2, uint64_t& sum2b) {
#pragma unroll
  for (int i = 0; i < 16; ++i) {
    const uint64_t x = fma2(pack2(__uint_as_float(s[2 * i]), __uint_as_float(s[2 * i + 1])), c2, nm2);
    float a, b;
    if (i % 4 == 3 && i / 4 < PAIR_POLY_PAIRS) {   // spread over the chunk so MUFU and FMA work interleave
      ex2_poly2(x, a, b);
    } else {
      float xa, xb;
      unpack2(x, xa, xb);
      a = ex2(xa);
      b = ex2(xb);
    }
    if (i & 1) sum2b = add2(sum2b, pack2(a, b));   // two independent chains
    else sum2 = add2(sum2, pack2(a, b));
    pk[i] = pack_bf16(a, b);
  }
}

#ifdef DIT_ATTN_TRACE
__device__ __forceinline__ unsigned long long gtime() { unsigned long long t; asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t)); return t; }
#define TRACE(i) do { if (tr_on && tr_n < 4) tr[tr_n][i] = gtime(); } while (0)
#else
#define TRACE(i) do { } while (0)
#endif
__global__ void __launch_bounds__(ATTN_THREADS, 1)
attn_pair_kernel(const __grid_constant__ CUtensorMap tmQ, const __grid_constant__ CUtensorMap tmK,
                 const __grid_constant__ CUtensorMap tmV, AttnParams p) {
  pdl_trigger();
  extern __shared__ uint8_t smem_raw[];
  const uint32_t smem0 = (smem_u32(smem_raw) + 1023u) & ~1023u;
  const uint32_t sQ = smem0, sK = sQ + 2 * PQ_BYTES, sV = sK + PKS * PKV_BYTES;
  const uint32_t bar0 = sV + PVS * PKV_BYTES;
  auto q_full = [&](int b) { return bar0 + 8u * b; };   // Q buffer b = work item parity
  auto k_full = [&](int s) { return bar0 + 8u * (2 + s); };
  auto k_empty = [&](int s) { return bar0 + 8u * (2 + PKS + s); };
  auto v_full = [&](int s) { return bar0 + 8u * (2 + 2 * PKS + s); };
  auto v_empty = [&](int s) { return bar0 + 8u * (2 + 2 * PKS + PVS + s); };
  constexpr int B0 = 2 + 2 * PKS + 2 * PVS;
  auto s_full = [&](int g) { return bar0 + 8u * (B0 + g); };        // S[g] complete (leader's commit, both CTAs)
  auto s_free = [&](int g) { return bar0 + 8u * (B0 + 2 + g); };    // S[g] read by all its softmax warps (leader CTA only)
  auto p_full = [&](int g) { return bar0 + 8u * (B0 + 4 + g); };    // P[g] written by all its softmax warps (leader CTA only)
  auto pv_done = [&](int g) { return bar0 + 8u * (B0 + 6 + g); };   // the PV that read P[g] has completed (both CTAs)
  auto o_done = [&]() { return bar0 + 8u * (B0 + 8); };
  const uint32_t tmem_slot = bar0 + 8u * (B0 + 9);
  const uint32_t panic_addr = bar0 + 8u * (B0 + 10);
  static_assert(8 * (B0 + 11) <= PAIR_BAR_BYTES, "barrier area");

  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const uint32_t crank = cluster_ctarank();
  const bool leader_cta = crank == 0;
  // PERSISTENT: the pair walks the work items idx = pair, pair + n_pairs, ... of the list (request in order of decreasing
  // key count, head, 256-row query block); the prologue (barriers, TMEM, cluster sync) is paid once per SM instead of
  // once per item, and the next item's Q tile is fetched while the current item runs.
  struct Item { int head, q_lo, q_hi, q_base, k_lo, kv_len, n_tiles; };
  auto decode = [&](int idx) -> Item {
    Item it;
    int req = 0, rem = idx, nqb = (p.n_q + 2 * TQ - 1) / (2 * TQ);
    if (p.cu_q) {
      for (int i = 0; i < p.R; ++i) {
        req = p.order[i];
        nqb = (p.cu_q[req + 1] - p.cu_q[req] + 2 * TQ - 1) / (2 * TQ);
        if (rem < nqb * p.H || i == p.R - 1) break;
        rem -= nqb * p.H;
      }
    }
    it.head = rem / nqb;
    it.q_lo = p.cu_q ? p.cu_q[req] : 0;
    it.q_hi = p.cu_q ? p.cu_q[req + 1] : p.n_q;
    it.q_base = it.q_lo + (rem - it.head * nqb) * (2 * TQ) + (int)crank * TQ;   // this CTA's 128 rows (may lie past q_hi)
    const int k_lo0 = p.cu_k ? p.cu_k[req] : 0, k_hi0 = p.cu_k ? p.cu_k[req + 1] : p.n_k;
    const int ssz = (k_hi0 - k_lo0 + p.n_shards - 1) / p.n_shards;
    int k_lo = k_lo0 + p.shard * ssz, k_hi = k_lo0 + (p.shard + 1) * ssz;
    if (k_lo > k_hi0) k_lo = k_hi0;
    if (k_hi > k_hi0) k_hi = k_hi0;
    it.k_lo = k_lo;
    it.kv_len = k_hi - k_lo;
    it.n_tiles = (it.kv_len + TK - 1) / TK;
    return it;
  };
  const int pair_id = (int)(blockIdx.x >> 1), n_pairs = (int)(gridDim.x >> 1);

  if (warp == 0 && lane == 0) {
    tma_prefetch_desc(&tmQ);
    tma_prefetch_desc(&tmK);
    tma_prefetch_desc(&tmV);
  }
  if (warp == 1 && lane == 0) {
    mbar_init(q_full(0), 1);
    mbar_init(q_full(1), 1);
    for (int s = 0; s < PKS; ++s) { mbar_init(k_full(s), 1); mbar_init(k_empty(s), 1); }
    for (int s = 0; s < PVS; ++s) { mbar_init(v_full(s), 1); mbar_init(v_empty(s), 1); }
    for (int g = 0; g < 2; ++g) {
      mbar_init(s_full(g), 1);
      mbar_init(s_free(g), 16);          // the 8 warps of a group in each CTA
      mbar_init(p_full(g), 16);
      mbar_init(pv_done(g), 1);
    }
    mbar_init(o_done(), 1);
    asm volatile("st.shared.u32 [%0], %1;" ::"r"(panic_addr), "r"(0u) : "memory");
    fence_barrier_init();
  }
  if (warp == 2) tmem_alloc_pair<512>(tmem_slot);
  tc_fence_before();
  __syncthreads();
  cluster_sync_all();   // the peer's barriers exist before anything arrives on them
  tc_fence_after();
  uint32_t tmem_base;
  asm volatile("ld.shared.b32 %0, [%1];" : "=r"(tmem_base) : "r"(tmem_slot));
  pdl_wait();           // prologue done; q / k / v written by the previous kernel are read from here on

  // Does pass 0 stand?  Every thread of both CTAs calls this at the end of pass 0.
  auto pair_panicked = [&]() -> bool {
    tc_fence_before();
    cluster_sync_all();
    tc_fence_after();
    uint32_t mine, peer;
    asm volatile("ld.shared.u32 %0, [%1];" : "=r"(mine) : "r"(panic_addr) : "memory");
    asm volatile("ld.shared::cluster.u32 %0, [%1];" : "=r"(peer) : "r"(mapa_cluster(panic_addr, crank ^ 1u)) : "memory");
    return (mine | peer) != 0;
  };
  // pass 0: reference = row max of key tile 0;  pass 1 (after a panic): row max over all key tiles, S only;  pass 2: as
  // pass 0 with the reference given.  Use counters of rings, buffers and barriers run on across passes.
  if (warp < 4) {
    asm volatile("setmaxnreg.dec.sync.aligned.u32 56;");   // 128 x 56 + 512 x 104 <= 640 x 96
    int kc = 0, vc = 0;            // K / V tiles produced or consumed so far (all items and passes)
    int sn = 0, pn = 0;            // S tiles / PVs issued so far: S tile t goes to S[t & 1], PV t reads P[t & 1]
    int qi = 0;                    // items with keys so far: item qi uses Q buffer qi & 1
    bool q_have = false;           // this item's Q was prefetched during the previous one
    for (int idx = pair_id; idx < p.n_items; idx += n_pairs) {
    const Item it = decode(idx);
    const int head = it.head, k_lo = it.k_lo, kv_len = it.kv_len, n_tiles = it.n_tiles;
    const int c0 = head * HD;
    if (n_tiles == 0) continue;    // empty shard: the softmax warps write o = 0, lse = -inf
    const int ii = qi++;
    const uint32_t sQi = sQ + (uint32_t)(ii & 1) * PQ_BYTES;   // this item's Q buffer
    const bool q_had = q_have;
    Item nxt = it;
    q_have = false;
    if (idx + n_pairs < p.n_items) {
      nxt = decode(idx + n_pairs);
      q_have = nxt.n_tiles > 0;
    }
    for (int pass = 0;; ++pass) {
      const bool with_pv = pass != 1;
      if (warp == 0) {
        // ===================================================== K producer (+ Q once)
        // Q of this item (the first item only: later ones were prefetched) and Q of the pair's next item, whose buffer
        // was last read by the item before this one (complete: every item ends with a pair-wide barrier)
        if (pass == 0 && elect_one()) {
          auto load_q = [&](const Item& q, int b) {
            const uint32_t lead_q = mapa_cluster(q_full(b), 0);
            if (leader_cta) mbar_expect_tx(q_full(b), 2 * PQ_BYTES);
            tma_load_2d_pair(sQ + b * PQ_BYTES, &tmQ, q.head * HD, q.q_base, lead_q);
            tma_load_2d_pair(sQ + b * PQ_BYTES + PQ_HALF, &tmQ, q.head * HD + 64, q.q_base, lead_q);
          };
          if (!q_had) load_q(it, ii & 1);
          if (q_have) load_q(nxt, (ii + 1) & 1);
        }
        for (int j = 0; j < n_tiles; ++j, ++kc) {
          const int s = kc % PKS;
          mbar_wait_poll(k_empty(s), (uint32_t)((kc / PKS) & 1) ^ 1u);
          if (elect_one()) {
            const uint32_t fb = mapa_cluster(k_full(s), 0);
            if (leader_cta) mbar_expect_tx(k_full(s), 2 * PKV_BYTES);
            const int r0 = k_lo + j * TK + (int)crank * 64;      // this CTA's 64 keys of the tile
            tma_load_2d_pair(sK + s * PKV_BYTES, &tmK, c0, r0, fb);
            tma_load_2d_pair(sK + s * PKV_BYTES + PK_HALF, &tmK, c0 + 64, r0, fb);
          }
          __syncwarp();
        }
      } else if (warp == 2) {
        // ===================================================== V producer
        if (with_pv) {
          for (int j = 0; j < n_tiles; ++j, ++vc) {
            const int s = vc % PVS;
            mbar_wait_poll(v_empty(s), (uint32_t)((vc / PVS) & 1) ^ 1u);
            if (elect_one()) {
              const uint32_t fb = mapa_cluster(v_full(s), 0);
              if (leader_cta) mbar_expect_tx(v_full(s), 2 * PKV_BYTES);
              tma_load_2d_pair(sV + s * PKV_BYTES, &tmV, c0 + (int)crank * 64, k_lo + j * TK, fb);   // 64 of the 128 d columns
            }
            __syncwarp();
          }
        }
      } else if (warp == 1 && leader_cta) {
        // ===================================================== MMA issuer for the pair
        constexpr uint32_t idesc_s = idesc_bf16(2 * TQ, TK, 0, 0);   // S = Q K^T: M = 256, N = 128 keys
        constexpr uint32_t idesc_o = idesc_bf16(2 * TQ, HD, 0, 1);   // O += P V: A from TMEM, B (V) MN-major, N = 128 (d)
        constexpr uint64_t vdesc_hi = desc_base_sw128(1, 64);        // one 128-byte atom wide (64 d), 8-key groups 1 KB apart
        // S of the next key tile into S[g]; the buffer's previous contents have been read (s_free)
        auto issue_s = [&]() {
          const int g = sn & 1;
          if (sn >= 2) mbar_wait_poll(s_free(g), (uint32_t)((sn >> 1) - 1) & 1u);
          const int s = kc % PKS;
          mbar_wait_poll(k_full(s), (uint32_t)(kc / PKS) & 1u);
          tc_fence_after();
          if (elect_one()) {
            const uint32_t d = tmem_base + TM_S + g * 128;
            const uint32_t ka = sK + s * PKV_BYTES;
#pragma unroll
            for (int k = 0; k < HD / 16; ++k)
              umma_ss_pair(d, desc_kmajor_sw128(sQi + (k >> 2) * PQ_HALF + (k & 3) * 32),
                           desc_kmajor_sw128(ka + (k >> 2) * PK_HALF + (k & 3) * 32), idesc_s, k != 0);
            umma_commit_pair(s_full(g), (uint16_t)3);
            umma_commit_pair(k_empty(s), (uint16_t)3);
          }
          __syncwarp();
          ++kc; ++sn;
        };
        // O (+)= P(j) V_j
        auto issue_pv = [&](int j) {
          const int g = pn & 1;
          const int vs = vc % PVS;
          const int left = kv_len - j * TK;                        // a ragged last tile: only the 32-key quarters with keys
          const int nk16 = left >= TK ? 8 : 2 * ((left + 31) / 32);
          mbar_wait_poll(v_full(vs), (uint32_t)(vc / PVS) & 1u);
          mbar_wait_poll(p_full(g), (uint32_t)(pn >> 1) & 1u);
          tc_fence_after();
          if (elect_one()) {
            const uint32_t d = tmem_base + TM_O;
            const uint32_t pa = tmem_base + TM_P + g * 64;         // bf16 pairs: key 2 i, 2 i + 1 in column i
            const uint32_t va = sV + vs * PKV_BYTES;
#pragma unroll
            for (int k = 0; k < 8; ++k)
              if (k < nk16)
                umma_ts_pair(d, pa + 8 * k, vdesc_hi | (uint64_t)(((va + k * 2048) >> 4) & 0x3fff), idesc_o, (j != 0 || k != 0) ? 1u : 0u);
            umma_commit_pair(v_empty(vs), (uint16_t)3);
            umma_commit_pair(pv_done(g), (uint16_t)3);
            if (j == n_tiles - 1) umma_commit_pair(o_done(), (uint16_t)3);
          }
          __syncwarp();
          ++vc; ++pn;
        };
        if (pass == 0) { mbar_wait_poll(q_full(ii & 1), (uint32_t)(ii >> 1) & 1u); tc_fence_after(); }
        // order = the order the events arrive in: S(j + 2) as soon as S(j) has been read (at the start of tile j's
        // softmax), PV(j - 1) when P(j - 1) is complete
        for (int i = 0; i < 2 && i < n_tiles; ++i) issue_s();
        for (int j = 0; j < n_tiles; ++j) {
          if (j + 2 < n_tiles) issue_s();
          if (with_pv && j >= 1) issue_pv(j - 1);
        }
        if (with_pv) issue_pv(n_tiles - 1);
      }
      if (pass == 2) { tc_fence_before(); cluster_sync_all(); tc_fence_after(); break; }   // O has been read: next item
      if (pass == 0 && !pair_panicked()) break;
      if (pass == 1) { tc_fence_before(); cluster_sync_all(); tc_fence_after(); }   // pass 1 -> 2 boundary (see the softmax warps)
    }
    }
  } else {
    asm volatile("setmaxnreg.inc.sync.aligned.u32 104;");
    // ===================================================== softmax: two groups of 8 warps in anti-phase
    // Key tile t (counted over all passes) belongs to group t & 1, lives in S[t & 1], and its P goes to P[pt & 1] (pt =
    // P tiles so far).  Thread = one query row x 64 keys: TMEM lane quadrant `quad` (rows), key half `h`.
    const int w = warp - 4;
    const int grp = w >> 3;
    const int h = (w >> 2) & 1;                    // 0: keys 0..63 of the tile, 1: keys 64..127
    const int kq = grp * 2 + h;                    // the row's four threads, for the 4-way reductions and the epilogue
    const int quad = warp & 3;                     // TMEM lane quadrant of this warp
    const int r_in = quad * 32 + lane;             // row inside this CTA's Q tile
    const uint32_t lane_off = (uint32_t)(quad * 32) << 16;
    const uint32_t s_addr = tmem_base + TM_S + grp * 128 + h * SK + lane_off;
    const uint32_t p_addr = tmem_base + TM_P + h * 32 + lane_off;      // + 64 * (pt & 1)
    const uint32_t o_addr = tmem_base + TM_O + kq * 32 + lane_off;
    float* const xch = reinterpret_cast<float*>(smem_raw + (bar0 - smem_u32(smem_raw)) + PAIR_BAR_BYTES);
    float* const red0 = xch;                       // [kq][128]: 4-way reductions (row max, row sums)
    float* const red = red0 + kq * 128 + r_in;
    float* const m_row = xch + 512;                // [128]: the row's reference, published by group 0
    const float c = p.scale_log2;
    const uint64_t c2 = pack2(c, c);
    // barriers of the LEADER CTA as shared::cluster addresses (valid from both CTAs: no branch at the arrival)
    const uint32_t a_sfree = mapa_cluster(s_free(grp), 0), a_pfull = mapa_cluster(p_full(0), 0);
    const uint32_t b_sfull = s_full(grp);
    auto arrive = [&](uint32_t bar_cluster) {      // one arrival per warp
      tc_fence_before();
      __syncwarp();
      if (lane == 0)
        asm volatile("mbarrier.arrive.relaxed.cluster.shared::cluster.b64 _, [%0];" ::"r"(bar_cluster) : "memory");
    };
    float m_used = 0.f;
#ifdef DIT_ATTN_TRACE
    unsigned long long tr[4][8]; int tr_n = 0; const bool tr_on = blockIdx.x == 0 && warp == 4 && lane == 0;
#endif
    int st = 0, ptn = 0, od = 0;                   // S tiles / P tiles / PV passes so far (all items and passes)
    for (int idx = pair_id; idx < p.n_items; idx += n_pairs) {
    const Item it = decode(idx);
    const int head = it.head, q_hi = it.q_hi, kv_len = it.kv_len, n_tiles = it.n_tiles;
    const int row = it.q_base + r_in;
    if (n_tiles == 0) {                            // empty shard: o = 0, lse = -inf (R18)
      if (row < q_hi) {
        const float z[8] = {0, 0, 0, 0, 0, 0, 0, 0};
        for (int cc = 0; cc < 32; cc += 8) st8<bf16>(p.o + (int64_t)row * p.o_stride + head * HD + kq * 32 + cc, z);
        if (kq == 0 && p.lse) p.lse[(int64_t)row * p.H + head] = -INFINITY;
      }
      continue;
    }
    TRACE(0);
    for (int pass = 0;; ++pass) {
      float l = 0.f, tile_worst = 0.f, mx_run = -INFINITY;
      const int base = st;                         // global index of this pass's first key tile
      const int pbase = base - ptn;                // ... minus this = its P index (pass 1 writes no P)
      st += n_tiles;
      if (pass != 1) ptn += n_tiles;
      if (pass == 0 && grp != (base & 1)) {        // the reference comes from the other group's first tile
        asm volatile("bar.sync %0, 128;" ::"r"(5 + quad) : "memory");
        m_used = m_row[r_in];
      }
      for (int t = base + ((base ^ grp) & 1); t < base + n_tiles; t += 2) {
        const int valid = kv_len - (t - base) * TK - h * SK;   // keys of this half that exist (>= 64: all; warp-uniform)
        uint32_t s0[32], s1[32];
        if (valid > 0) {
          mbar_wait(b_sfull, (uint32_t)(t >> 1) & 1u);
          if (t == base) TRACE(1);
          tc_fence_after();
          tmem_ld32(s_addr + 0, s0);
          tmem_ld32(s_addr + 32, s1);
          tmem_ld_wait();
        }
        arrive(a_sfree);                           // S[grp] may be overwritten by S(t + 2) from here on
        if (pass == 1) {                           // row-max pass (after a panic)
          if (valid > 0) {
            if (valid < SK) { mask32(s0, valid); mask32(s1, valid - 32); }
            mx_run = fmaxf(mx_run, fmaxf(max32(s0), max32(s1)));
          }
          continue;
        }
        if (valid > 0 && valid < SK) { mask32(s0, valid); mask32(s1, valid - 32); }   // -inf: before the row max; P = 0
        if (pass == 0 && t == base) {              // the row max of the first key tile is the reference of the pass
          *red = valid > 0 ? fmaxf(max32(s0), max32(s1)) : -INFINITY;
          asm volatile("bar.sync %0, 64;" ::"r"(1 + quad) : "memory");
          m_used = fmaxf(red0[grp * 256 + r_in], red0[grp * 256 + 128 + r_in]) * c;   // this group's two halves; c > 0
          if (h == 0) m_row[r_in] = m_used;
          __threadfence_block();
          asm volatile("bar.arrive %0, 128;" ::"r"(5 + quad) : "memory");     // group 1 may read m_row
        }
        const uint32_t pt = (uint32_t)(t - pbase), bp = pt & 1u;
        if (valid > 0) {
          const uint64_t nm2 = pack2(-m_used, -m_used);
          uint64_t sum2 = pack2(0.f, 0.f), sum2b = pack2(0.f, 0.f);
          {
            uint32_t pk[16];
            exp_pack(s0, c2, nm2, pk, sum2, sum2b);
            // the PV before last has read P[bp]: it was issued about a tile ago
            if (pt >= 2) { mbar_wait(pv_done(0) + 8u * bp, ((pt >> 1) - 1u) & 1u); tc_fence_after(); }
            tmem_st16(p_addr + bp * 64u, pk);
          }
          {
            uint32_t pk[16];
            exp_pack(s1, c2, nm2, pk, sum2, sum2b);
            tmem_st16(p_addr + bp * 64u + 16, pk);
          }
          float sa, sb;
          unpack2(add2(sum2, sum2b), sa, sb);
          tile_worst = fmaxf(tile_worst, sa + sb);
          l += sa + sb;
          tmem_st_wait();
        }
        arrive(a_pfull + 8u * bp);
        if (t == base) TRACE(2);
      }
      TRACE(3);
      if (pass == 1) {
        *red = mx_run;
        asm volatile("bar.sync %0, 128;" ::"r"(9 + quad) : "memory");
        m_used = fmaxf(fmaxf(red0[r_in], red0[128 + r_in]), fmaxf(red0[256 + r_in], red0[384 + r_in])) * c;
        asm volatile("bar.sync %0, 128;" ::"r"(9 + quad) : "memory");   // `red` is reused for the row sums
        tc_fence_before(); cluster_sync_all(); tc_fence_after();        // pass 1 -> 2 boundary
        continue;
      }
      if (pass == 0 && __any_sync(0xffffffffu, !(tile_worst < 1.152921504606847e18f)) && lane == 0)   // 2^60, inf, NaN
        asm volatile("st.shared.u32 [%0], %1;" ::"r"(panic_addr), "r"(1u) : "memory");
      // ---- epilogue: the row's four threads add their partial sums; thread kq writes d columns 32 kq .. 32 kq + 31
      *red = l;
      asm volatile("bar.sync %0, 128;" ::"r"(9 + quad) : "memory");
      l = (red0[r_in] + red0[128 + r_in]) + (red0[256 + r_in] + red0[384 + r_in]);
      mbar_wait(o_done(), (uint32_t)od & 1u);
      TRACE(4);
      ++od;
      tc_fence_after();
      const float inv = 1.0f / l;                  // l > 0: the first tile has at least one key
      const bool row_ok = row < q_hi;
      {
        uint32_t o[32];
        tmem_ld32(o_addr, o);
        tmem_ld_wait();
        if (row_ok) {
          bf16* orow = p.o + (int64_t)row * p.o_stride + head * HD + kq * 32;
#pragma unroll
          for (int g = 0; g < 4; ++g) {
            float v[8];
#pragma unroll
            for (int e = 0; e < 8; ++e) v[e] = __uint_as_float(o[g * 8 + e]) * inv;
            st8<bf16>(orow + g * 8, v);
          }
        }
      }
      if (kq == 0 && row_ok && p.lse != nullptr)
        p.lse[(int64_t)row * p.H + head] = 0.6931471805599453f * (m_used + log2f(l));
      TRACE(5);
      if (pass == 2) {                             // O has been read: the next item's first PV may overwrite it; the panic
        if (threadIdx.x == 128)                    // flag was read by both CTAs two pair-wide barriers ago
          asm volatile("st.shared.u32 [%0], %1;" ::"r"(panic_addr), "r"(0u) : "memory");
        tc_fence_before(); cluster_sync_all(); tc_fence_after();
        break;
      }
      { const bool pp = pair_panicked(); TRACE(6);
#ifdef DIT_ATTN_TRACE
        if (tr_on) ++tr_n;
#endif
        if (!pp) break; }
    }
    }
#ifdef DIT_ATTN_TRACE
    if (tr_on) for (int i = 0; i < tr_n && i < 4; ++i)
      printf("item %d: start->S0 %llu  S0->P0 %llu  P0->lastP %llu  lastP->o_done %llu  epilogue %llu  sync %llu  | next start +%llu ns\n", i,
             tr[i][1] - tr[i][0], tr[i][2] - tr[i][1], tr[i][3] - tr[i][2], tr[i][4] - tr[i][3], tr[i][5] - tr[i][4], tr[i][6] - tr[i][5],
             i + 1 < tr_n ? tr[i + 1][0] - tr[i][6] : 0ull);
#endif
  }
  tc_fence_before();
  __syncthreads();
  cluster_sync_all();   // no CTA leaves while its peer may still signal its barriers or read its shared memory
  if (warp == 2) {
    tc_fence_after();
    tmem_dealloc_pair<512>(tmem_base);
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
  static std::atomic<bool> attr_set{false};
  if (!attr_set) {
    DIT_CUDA_OK(cudaFuncSetAttribute(attn_tc_kernel<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, ATTN_SMEM));
    DIT_CUDA_OK(cudaFuncSetAttribute(attn_tc_kernel<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, ATTN_SMEM));
    DIT_CUDA_OK(cudaFuncSetAttribute(attn_pair_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, PAIR_SMEM));
    attr_set = true;
  }
  static const bool use_pair = []() {   // DIT_ATTN_KERNEL=two-tile selects attn_tc_kernel for every shape (A / B measurements)
    const char* e = getenv("DIT_ATTN_KERNEL");
    return !(e != nullptr && e[0] == 't');
  }();
  static const int pair_min_k = []() {  // DIT_ATTN_PAIR_MIN_K overrides the switch-over length (tuning knob)
    const char* e = getenv("DIT_ATTN_PAIR_MIN_K");
    return e != nullptr ? atoi(e) : 2048;
  }();
  // K / V maps need a valid base even when there are no keys (the kernel then never issues a load)
  const void* kb = a.n_k > 0 ? a.k : a.q;
  const void* vb = a.n_k > 0 ? a.v : a.q;
  const uint64_t nk_rows = a.n_k > 0 ? a.n_k : 1;
  const uint64_t kv_ld = a.n_k > 0 ? a.kv_stride : a.q_stride;
  // Key sequences from 2048 keys (16 key tiles): the persistent pair kernel; shorter ones: attn_tc_kernel, whose fill and
  // drain per work item weigh less (measured alone, H = 24, attn_tc_kernel vs pair: N = 1024: 419 vs 360 TFLOP/s; 2048:
  // 599 vs 735; 4352: 1040 vs 1072; 8192: 1100 vs 1274; 16384: 1244 vs 1385; 32768: 1173 vs 1262).
  int max_k = a.n_k;
  if (a.cu_k_host) {
    max_k = 0;
    for (int r = 0; r < a.R; ++r) max_k = max(max_k, a.cu_k_host[r + 1] - a.cu_k_host[r]);
  }
  max_k = cdiv(max_k, a.n_shards);
  const bool pair_kernel = use_pair && max_k >= pair_min_k;
  CUtensorMap tq, tk, tv;
  const uint64_t cols = (uint64_t)a.H * HD;
  DIT_REQUIRE(make_tmap_2d_bf16(&tq, a.q, a.n_q, cols, a.q_stride, TQ, 64) &&
                  make_tmap_2d_bf16(&tk, kb, nk_rows, cols, kv_ld, pair_kernel ? 64 : TK, 64) &&
                  make_tmap_2d_bf16(&tv, vb, nk_rows, cols, kv_ld, TK, 64),
              DIT_ERR_CUDA, "attn_tc: cuTensorMapEncodeTiled failed (n_q=%d n_k=%d H=%d)", a.n_q, a.n_k, a.H);
  AttnParams p;
  p.o = (bf16*)a.o; p.o_stride = a.o_stride; p.lse = a.lse;
  p.cu_q = a.cu_q; p.cu_k = a.cu_k;
  p.n_q = a.n_q; p.n_k = a.n_k; p.H = a.H;
  p.scale_log2 = a.scale * 1.4426950408889634f;
  p.shard = a.shard; p.n_shards = a.n_shards;
  for (int r = 0; r < 64; ++r) p.order[r] = (uint8_t)(r < a.R ? r : 0);
  if (a.cu_q && a.cu_k_host && a.R > 1 && a.R <= 64)   // work per CTA is proportional to the request's key count
    std::stable_sort(p.order, p.order + a.R, [&](uint8_t x, uint8_t y) {
      return a.cu_k_host[x + 1] - a.cu_k_host[x] > a.cu_k_host[y + 1] - a.cu_k_host[y];
    });
  ProfScope _prof(DIT_KC_ATTN, st);
  if (pair_kernel) {   // persistent: one CTA pair per SM pair walks the (request, head, 256-row query block) items
    int n_items = 0;
    if (a.cu_q && a.cu_q_host) for (int r = 0; r < a.R; ++r) n_items += cdiv(a.cu_q_host[r + 1] - a.cu_q_host[r], 2 * TQ) * a.H;
    else n_items = cdiv(a.n_q, 2 * TQ) * a.H;
    p.R = a.cu_q ? a.R : 1;
    p.n_items = n_items;
    int sms = 148;
    { int dev = 0; cudaGetDevice(&dev); cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev); }
    // Equal items (one request): the fewest pairs that still finish in the same number of rounds — cfg 2: 408 items are 6 rounds on
    // 74 pairs (5.51) and also on 68; the idle SMs' power goes to the clock of the busy ones (the step is power capped).
    int n_pairs = min(n_items, sms / 2);
    static const bool trim = []() { const char* e = getenv("DIT_ATTN_NO_TRIM"); return !(e != nullptr && e[0] == '1'); }();
    if (trim && p.R == 1 && n_pairs > 0) {
      const int rounds = cdiv(n_items, n_pairs);
      n_pairs = cdiv(n_items, rounds);
    }
    dim3 pgrid(2 * n_pairs, 1, 1);
    DIT_CUDA_OK(launch_pdl(attn_pair_kernel, pgrid, dim3(ATTN_THREADS), PAIR_SMEM, st, 2, tq, tk, tv, p));
    DIT_LAUNCH_CHECK();
    return DIT_OK;
  }
  dim3 grid(cdiv(max_q, 2 * TQ), a.H, a.cu_q ? a.R : 1);
  // CTA pairs when every request has an even number of 256-row query blocks (each CTA of a pair then has rows)
  // ... and the key sequence is long: measured alone it is neutral from N = 8192 (slower below: the pair runs in
  // lockstep), inside a power-capped step it is ~2 % faster (less L2 -> SM traffic, higher clock)
  bool pair = a.n_k >= 8192;
  if (a.cu_q_host) {
    for (int r = 0; r < a.R; ++r) {
      const int len = a.cu_q_host[r + 1] - a.cu_q_host[r];
      if (cdiv(len, 2 * TQ) % 2 != 0 || cdiv(len, 2 * TQ) != (int)grid.x) pair = false;   // all requests fill the grid
    }
  } else if (grid.x % 2 != 0) {
    pair = false;
  }
  if (pair) DIT_CUDA_OK(launch_pdl(attn_tc_kernel<true>, grid, dim3(ATTN_THREADS), ATTN_SMEM, st, 2, tq, tk, tv, p));
  else DIT_CUDA_OK(launch_pdl(attn_tc_kernel<false>, grid, dim3(ATTN_THREADS), ATTN_SMEM, st, 1, tq, tk, tv, p));
  DIT_LAUNCH_CHECK();
  return DIT_OK;
}

}  // namespace dit
