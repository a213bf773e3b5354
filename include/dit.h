/* dit.h — C ABI of libdit_b200.so: one DiT denoising step on one B200 (sm_100a).
 *
 * What the library computes.  GF-DiT (arxiv/paper_2606_13501) schedules DiT requests as trajectory
 * tasks, one task per denoising step; "denoising dominates execution time and resource consumption"
 * (§1) and a step "performs bidirectional computation over the entire latent sequence"
 * (§2.1).  The paper treats that step as an opaque executor call on "ordinary input and
 * output tensors" (§5.2; §4.3) and parallelises it over the sequence with
 * all-gather / all-to-all (§4.1).  This library IS that step on a single GPU: a stack of
 * adaLN-Zero DiT blocks over a request's latent token sequence, plus the single-GPU analogue of the
 * paper's SP degree (split-KV partial attention + log-sum-exp merge) and of its heterogeneous request
 * mix (packed variable-length batching).  The mathematics is fixed in DESIGN.md §3 (readings R1-R23).
 *
 * Conventions (all entry points)
 *  - "dev" pointers are device (HBM) pointers owned by the CALLER (PyTorch allocates); "host" pointers
 *    are ordinary host memory.  The library never frees caller memory and never allocates device
 *    memory after dit_init (its only allocation is the handle's small host struct); `workspace` is
 *    caller-allocated with the size dit_workspace_bytes() returns and must outlive the handle, as must
 *    every weight pointer.
 *  - All work is enqueued on `stream` (a cudaStream_t passed as void*; NULL = legacy default stream).
 *    No entry point synchronises the device, except dit_init (one-time pointer-table upload) and the
 *    *_host convenience call, which returns after enqueuing (its D2H copy is stream ordered; the caller
 *    synchronises the stream before reading `out_host`).
 *  - Errors: a negative dit_status is returned before anything is launched when arguments are invalid;
 *    DIT_ERR_CUDA reports a failed launch/API call.  dit_last_error() gives a message.  Nothing throws.
 *  - There is no CPU fallback and no alternative backend: if no sm_100 device is present every compute
 *    entry point returns DIT_ERR_CUDA.  A DIT_BF16 handle runs its step on the tcgen05 kernels ONLY: dit_init
 *    returns DIT_ERR_UNSUPPORTED for a bf16 config they cannot serve (head_dim != 128, C*pv or cond_dim not a
 *    multiple of 8) and a step returns DIT_ERR_UNSUPPORTED rather than substitute the fp32 FFMA kernels.  The
 *    kernel-level entry points below do run bf16 shapes outside those limits on the FFMA kernels; each such
 *    launch is counted by dit_fallback_launches().
 *  - Threads and streams: a handle owns ONE workspace, so calls on the same handle must be ordered by the caller
 *    (one stream at a time, or explicit events between streams); different handles are independent and may be
 *    driven from different host threads.  dit_last_error is per host thread.  The measurement calls
 *    (dit_profile_begin / dit_profile_end) are process wide.
 *  - dtype: DIT_F32 (all tensors fp32; SIMT FFMA kernels, no TF32) or DIT_BF16 (weights/activations
 *    bf16, residual stream / statistics / modulation / LSE fp32; tcgen05 tensor-core kernels).
 *  - Linear weights are [out, in] row-major, biases [out], all in the config dtype.
 */
#ifndef DIT_B200_H
#define DIT_B200_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct dit_handle_s* dit_handle; /* opaque; created by dit_init, destroyed by dit_free */

typedef enum {
  DIT_OK = 0,
  DIT_ERR_INVALID_ARG = -1,
  DIT_ERR_UNSUPPORTED = -2,
  DIT_ERR_WORKSPACE = -3,
  DIT_ERR_CUDA = -4
} dit_status;

typedef enum { DIT_F32 = 0, DIT_BF16 = 1 } dit_dtype;
typedef enum { DIT_COND_NONE = 0, DIT_COND_JOINT = 1, DIT_COND_CROSS = 2, DIT_COND_JOINT2 = 3 } dit_cond_mode;

/* POD configuration (all ints 32-bit).  struct_size = sizeof(dit_config) guards ABI drift. */
typedef struct {
  int32_t struct_size;
  int32_t dtype;           /* dit_dtype */
  int32_t n_blocks;        /* L >= 0 */
  int32_t hidden;          /* D, multiple of 128, == n_heads * head_dim */
  int32_t n_heads;         /* H */
  int32_t head_dim;        /* d in {64, 128} */
  int32_t mlp_dim;         /* F, multiple of 8 */
  int32_t latent_channels; /* C */
  int32_t patch[3];        /* {pf, ph, pw}; images: pf = 1 and latent F = 1 */
  int32_t temb_dim;        /* width of the timestep embedding passed to dit_step */
  int32_t cond_dim;        /* width of a conditioning token (ignored for DIT_COND_NONE) */
  int32_t cond_mode;       /* dit_cond_mode: joint = [cond ; image] one sequence, single stream (R9);
                              cross = extra cross-attention sub-layer per block (R10); joint2 = DUAL-STREAM joint
                              blocks (R37): one sequence [cond ; image] and one attention, but
                              the cond rows have their own per-block weights `blocks.{l}.txt.*` */
  int32_t rope_dims[3];    /* head-dim segment per axis (f, h, w), each even, sum == head_dim, or all 0
                              for no RoPE (R6) */
  float rope_theta;        /* 10000 */
  float ln_eps;            /* 1e-6 (R4) */
  float rms_eps;           /* 1e-6 (R5) */
  int32_t qk_rmsnorm;      /* 0/1: per-head RMSNorm of q and k with gains attn.gq / attn.gk (R5) */
  int32_t split_p;         /* split degree P used for self-attention inside a step: 1, 2, 4 or 8.
                              P > 1 computes P split-KV partials + LSE merge (the SP analogue) */
  int32_t max_tokens;      /* capacity: max total packed sequence rows (cond rows included in joint) */
  int32_t max_requests;    /* capacity: max requests per dit_step_varlen call (<= 64) */
  int32_t max_cond_tokens; /* capacity: max total conditioning tokens per call */
  int32_t mlp_gated;       /* 0: MLP = W2 GELU_tanh(W1 y + b1) + b2 (R3).  1: gated MLP (SwiGLU; SURVEY.md §8(f) item 2,
                              DESIGN.md R40): W2 (SiLU(W1 y + b1) (.) (W3 y + b3)) + b2 with extra weights mlp.w3, mlp.b3 */
  int32_t max_sample_steps; /* dit_sample only (0..4096; 0 = off): room in the workspace for the timestep-MLP outputs and
                              modulation vectors of this many denoising steps.  They depend on the timestep embedding alone,
                              so dit_sample computes them for (chunks of) this many steps AHEAD of the steps, 8 rows per pass
                              of the modulation weights: the weights (0.9 GB at BASELINE configs[1]) are streamed once per 8
                              steps instead of once per step (twice per guided step in the two-pass mode).  Results are
                              bit-identical to max_sample_steps = 0. */
} dit_config;

/* One named weight tensor (device pointer, caller-owned, config dtype).  Names:
 *   t_mlp.w1 [D,temb] t_mlp.b1 [D] t_mlp.w2 [D,D] t_mlp.b2 [D]
 *   patch_embed.w [D, C*pf*ph*pw] patch_embed.b [D]      cond_proj.w [D,cond_dim] cond_proj.b [D]
 *   blocks.{l}.mod.w [6D,D] .mod.b [6D]   (chunks: shift1, scale1, gate1, shift2, scale2, gate2)
 *   blocks.{l}.attn.wqkv [3D,D] .attn.bqkv [3D] (rows: q | k | v; head h = rows h*d..)  .attn.gq [d] .attn.gk [d]
 *   blocks.{l}.attn.wo [D,D] .attn.bo [D]   blocks.{l}.mlp.w1 [F,D] .mlp.b1 [F] .mlp.w2 [D,F] .mlp.b2 [D]
 *   blocks.{l}.mlp.w3 [F,D] .mlp.b3 [F]   (mlp_gated only; joint2 also blocks.{l}.txt.mlp.w3 / .b3)
 *   blocks.{l}.cross.wq [D,D] .bq [D] .wkv [2D,D] .bkv [2D] .gq [d] .gk [d] .wo [D,D] .bo [D]   (cross mode)
 *   blocks.{l}.txt.{mod.w, mod.b, attn.wqkv, attn.bqkv, attn.gq, attn.gk, attn.wo, attn.bo, mlp.w1, mlp.b1, mlp.w2, mlp.b2}
 *        (joint2 mode: the text stream's copy, same shapes as the image stream's blocks.{l}.*)
 *   final.mod.w [2D,D] final.mod.b [2D] (shift_f, scale_f)   final.w [C*pv, D] final.b [C*pv] */
typedef struct {
  const char* name;
  const void* dev_ptr;
  int64_t numel;
} dit_weight;

/* Bytes of device workspace dit_init needs for this config (0 on an invalid config). */
size_t dit_workspace_bytes(const dit_config* cfg);

/* Validates cfg and the weight table (every required name present with the right numel; unknown names
 * are an error), carves `workspace` (dev, 256-byte aligned), uploads pointer tables.  *out receives the
 * handle.  Returns DIT_ERR_WORKSPACE if workspace_bytes is too small. */
dit_status dit_init(const dit_config* cfg, const dit_weight* weights, int32_t n_weights, void* workspace,
                    size_t workspace_bytes, dit_handle* out);

/* One denoising step for one request (DESIGN.md §3 steps 1-6).
 *   latents      dev, [C, F, H, W] in config dtype, contiguous; latent_grid = {F, H, W} (host, 3 ints)
 *   timestep_emb dev, [temb_dim] fp32  (sinusoidal embedding of t — an input, R16)
 *   cond_tokens  dev, [n_cond, cond_dim] config dtype (NULL / 0 allowed; ignored for DIT_COND_NONE)
 *   out          dev, [C, F, H, W] config dtype
 * Sequence rows used = F/pf*H/ph*W/pw (+ n_cond in joint mode) must be <= max_tokens. */
dit_status dit_step(dit_handle h, const void* latents, const float* timestep_emb, const void* cond_tokens,
                    int32_t n_cond, const int32_t latent_grid[3], void* out, void* stream);

/* One request's denoising TRAJECTORY: n_steps denoising steps chained by the sampler update (PAPER.md:133 — a request
 * is a chain of trajectory tasks, one per denoising step; DESIGN.md §3 step 9, readings R30-R32):
 *     x_0 = latents;   for i = 0 .. n_steps-1:
 *         v_c = dit_step(x_i, timestep_embs[i], cond_tokens)
 *         v   = uncond_tokens ? v_u + guidance_scale * (v_c - v_u),  v_u = dit_step(x_i, timestep_embs[i], uncond_tokens)
 *                             : v_c                                   (classifier-free guidance)
 *         x_{i+1} = x_i + (sigmas[i+1] - sigmas[i]) * v               (flow-matching Euler update)
 *     out = x_{n_steps}
 *   latents       dev, [C, F, H, W] config dtype            out  dev, same shape and dtype (may not alias latents)
 *   timestep_embs dev, [n_steps, temb_dim] fp32             sigmas  HOST, [n_steps + 1] fp32
 *   cond_tokens / uncond_tokens  dev, [n_cond | n_uncond, cond_dim] config dtype; uncond_tokens NULL = no guidance
 * The state x_i is carried in fp32 inside the workspace; every step reads x_i rounded to the config dtype (it is staged
 * in `out`) and v is the fp32 result of the final Linear — the update is fused into the unpatchify kernel.
 * Guidance runs as ONE packed pass of two requests per step (unconditional + conditional over the same x_i, the varlen
 * path of dit_step_varlen: every weight is streamed once) when the handle has room for both — max_requests >= 2, both
 * sequences within max_tokens, n_cond + n_uncond <= max_cond_tokens — and as two passes per step otherwise.
 * use_graph != 0: the whole trajectory is captured once into a CUDA graph (cached in the handle, keyed by every
 * argument) and replayed with one launch; identical results.  n_steps == 0 copies latents to out. */
dit_status dit_sample(dit_handle h, const void* latents, const float* timestep_embs, const float* sigmas_host,
                      const void* cond_tokens, int32_t n_cond, const void* uncond_tokens, int32_t n_uncond,
                      float guidance_scale, const int32_t latent_grid[3], int32_t n_steps, int32_t use_graph, void* out,
                      void* stream);

/* dit_step / dit_step_varlen replayed from a CUDA graph: ONE cudaGraphLaunch instead of 65+ kernel launches (host cost of a
 * step ~0.4 ms -> ~10 us; the paper's control plane dispatches a request one denoising step at a time).  Same
 * arguments and result (bit-identical).  The graph holds every pointer and the geometry: a call whose arguments equal those
 * of a cached graph replays it (the CONTENTS of the buffers may have changed), any other call captures a new one; a handle
 * keeps the 8 most recently used graphs.  Falls back to plain launches while dit_profile_begin or a debug stop is active.
 * The first call for a set of arguments costs a capture + instantiation (milliseconds). */
dit_status dit_step_graph(dit_handle h, const void* latents, const float* timestep_emb, const void* cond_tokens, int32_t n_cond,
                          const int32_t latent_grid[3], void* out, void* stream);
dit_status dit_step_varlen_graph(dit_handle h, const void* latents_packed, const float* timestep_emb, const void* cond_packed,
                                 const int32_t* cu_seqlens, const int32_t* n_cond, const int32_t* latent_grids, int32_t n_requests,
                                 void* out_packed, void* stream);

/* Same computation with HOST buffers (pageable or pinned): H2D copies of latents / timestep_emb / cond, the step, and the
 * D2H copy of `out`; staging lives in the workspace.  Everything is ordered with respect to `stream`: the latent / cond
 * uploads run on a copy stream of the handle that first waits for all work already enqueued on `stream` and is joined back
 * before patch-embed (they overlap the timestep MLP and the modulation GEMV, which need only timestep_emb); the caller
 * synchronises `stream` before reading out_host or reusing the host input buffers.
 * This is the end-to-end call bench.py times ("e2e"). */
dit_status dit_step_host(dit_handle h, const void* latents_host, const float* timestep_emb_host,
                         const void* cond_tokens_host, int32_t n_cond, const int32_t latent_grid[3],
                         void* out_host, void* stream);

/* dit_step_varlen with HOST buffers (pageable or pinned): latents_packed / timestep_emb / cond_packed are copied to the
 * workspace's staging area, the packed step runs, and out_packed is copied back, ordered with respect to `stream` as in
 * dit_step_host; the caller synchronises the stream before reading out_packed_host.  Arguments as dit_step_varlen below. */
dit_status dit_step_varlen_host(dit_handle h, const void* latents_packed_host, const float* timestep_emb_host,
                                const void* cond_packed_host, const int32_t* cu_seqlens, const int32_t* n_cond,
                                const int32_t* latent_grids, int32_t n_requests, void* out_packed_host, void* stream);

/* Packed variable-length batch of R heterogeneous requests (BASELINE.json north_star subsystem 6; the
 * single-GPU analogue of the paper's heterogeneous request mix).  The result for request r
 * is DEFINED as dit_step on request r alone (DESIGN.md §3 step 8).
 *   latents_packed   dev: the R latents [C, F_r, H_r, W_r] back to back
 *   timestep_emb     dev: [R, temb_dim] fp32 (per-request timesteps)
 *   cond_packed      dev: [sum n_cond_r, cond_dim]
 *   cu_seqlens       host [R+1]: prefix sums of the per-request sequence length
 *                    T_r = N_r (+ n_cond_r in joint mode); validated against latent_grids / n_cond
 *   n_cond           host [R];   latent_grids host [R][3] = {F_r, H_r, W_r}
 *   out_packed       dev: R outputs back to back, each with its latent's shape
 * GEMMs / norms run over the flat [sum T_r, D] sequence; modulation is indexed per request; attention is
 * block diagonal over requests.
 * (SURVEY.md §8(b) sketched this call with a host AND a device copy of cu_seqlens; the library uploads its own device
 * copy — a few hundred bytes, skipped when the geometry is already resident — so the caller passes host arrays only:
 * DESIGN.md reading R35.) */
dit_status dit_step_varlen(dit_handle h, const void* latents_packed, const float* timestep_emb,
                           const void* cond_packed, const int32_t* cu_seqlens, const int32_t* n_cond,
                           const int32_t* latent_grids, int32_t n_requests, void* out_packed, void* stream);

/* Split-KV partial attention (north_star subsystem 5; one rank's share of a P-way sequence-parallel
 * step).  Non-causal:  for every query row i and head h over THIS call's n_k keys
 *   s_ij = softmax_scale * q_i . k_j ;  o_i = sum_j softmax_j(s_ij) v_j (locally normalised) ;
 *   lse_i = ln sum_j exp(s_ij)   (natural log; n_k == 0 gives o = 0, lse = -inf, R18)
 *   q  dev [n_q, H, d] with row stride q_row_stride elements (head stride = d);  k, v dev [n_k, H, d]
 *      with row stride kv_row_stride;  dtype = dit_dtype of q, k, v and o
 *   o  dev [n_q, H, d] contiguous;  lse dev [n_q, H] fp32 (may be NULL)
 * With n_k = all keys this is the full-sequence flash attention of subsystem 4.
 * q and k are taken AS GIVEN: QK-RMSNorm and RoPE (north_star subsystem 4, "fused into the Q/K load") are applied one
 * kernel earlier, on the fp32 accumulators of the QKV projection (dit_linear_qkv below), not on the attention kernel's
 * loads; SURVEY.md §8(b)'s optional `dit_attn_opts` (norm / RoPE on load) is therefore not part of this ABI.  Why, with
 * the measurements: DESIGN.md reading R34.  Callers with raw q / k use dit_linear_qkv or dit_qknorm_rope first. */
dit_status dit_attn_partial(int32_t dtype, const void* q, const void* k, const void* v, int32_t n_q, int32_t n_k,
                            int32_t n_heads, int32_t head_dim, int64_t q_row_stride, int64_t kv_row_stride,
                            float softmax_scale, void* o, float* lse, void* stream);

/* LSE merge of P partials (R18):  lse = ln sum_p e^{lse_p};  o = sum_p e^{lse_p - lse} o_p.
 *   o_partials host array of P dev pointers [n_q, H, d] (dtype);  lses host array of P dev pointers
 *   [n_q, H] fp32;  o dev [n_q, H, d] dtype;  lse_out dev [n_q, H] fp32 or NULL.  1 <= P <= 8.
 * Partials with lse = -inf contribute nothing; if all are -inf the row is o = 0, lse = -inf. */
dit_status dit_attn_merge(int32_t dtype, const void* const* o_partials, const float* const* lses, int32_t P,
                          int32_t n_q, int32_t n_heads, int32_t head_dim, void* o, float* lse_out, void* stream);

/* ---- re-layout between split degrees (§5.3 "Layout-Aware Artifact Migration") --
 * A row-sharded artifact (latent tokens, residual stream, per-token embeddings: "latent states and embeddings")
 * of n_rows rows lives as P contiguous shards (shard p = rows [p ceil(n/P), (p+1) ceil(n/P)) clipped to n: reading R20).
 * When the next trajectory task runs at another degree P', the planner intersects every source-owned slice with every
 * destination-required slice; every non-empty intersection is ONE transfer entry. */
typedef struct {
  int32_t src_rank, dst_rank; /* source shard p, destination shard q */
  int64_t src_row, dst_row;   /* first row of the range INSIDE the source / destination shard */
  int64_t n_rows;             /* rows in the range (> 0) */
} dit_transfer;
/* Host only.  Writes the plan (destination-major, source ranks ascending) to entries[0 .. min(count, max_entries)) and
 * returns `count`, the number of entries the plan has (<= p_src + p_dst - 1); negative dit_status on bad arguments
 * (1 <= p_src, p_dst <= 32).  n_rows = 0 gives 0 entries. */
int32_t dit_relayout_plan(int64_t n_rows, int32_t p_src, int32_t p_dst, dit_transfer* entries, int32_t max_entries);
/* Executes a plan on the device: ONE copy kernel packs every source range and installs it in its destination shard
 * (HBM-bound: reads and writes the artifact once).  entries host [n_entries <= 64]; src_shards / dst_shards HOST arrays
 * of device pointers indexed by rank, each shard [rows_of_shard, row_bytes] contiguous; row_bytes = bytes per row.
 * 128-bit accesses when every range is 16-byte aligned, narrower otherwise. */
dit_status dit_relayout(const dit_transfer* entries, int32_t n_entries, const void* const* src_shards,
                        void* const* dst_shards, int64_t row_bytes, void* stream);

/* Split-KV attention + LSE merge that ALLOCATES NOTHING (for callers that cannot call cudaMalloc: code under CUDA graph
 * capture, tight serving loops, harnesses that forbid it).  Same result as dit_attn_partial on the split_p contiguous KV
 * shards of ceil(n_k / split_p) keys (R20) followed by dit_attn_merge, but the partial outputs and their log-sum-exps live
 * in a static device array inside the library instead of caller memory: dit_static_scratch_bytes() = 8 MiB, held by every
 * GPU that loads the library until the process exits.  Arguments as dit_attn_partial; o dev [n_q, H, d] in dtype, lse_out
 * dev fp32 [n_q, H] or NULL.  split_p in 1..8.  Returns DIT_ERR_WORKSPACE (message via dit_last_error(NULL)) when
 * split_p * (align256(n_q * H * d * sizeof(dtype)) + align256(n_q * H * 4)) exceeds the array.  No cudaMalloc, cudaFree or
 * allocating library routine is called.  All calls on a device share the one array (it keeps the last call's contents;
 * nothing needs to start at zero: every partial row is written before the merge reads it): calls that OVERLAP on the GPU
 * (two streams, two host threads on one device) race and must be serialised by the caller. */
size_t dit_static_scratch_bytes(void);
dit_status dit_attn_split_static(int32_t dtype, const void* q, const void* k, const void* v, int32_t n_q, int32_t n_k,
                                 int32_t n_heads, int32_t head_dim, int64_t q_row_stride, int64_t kv_row_stride,
                                 float softmax_scale, int32_t split_p, void* o, float* lse_out, void* stream);

/* ---- kernel-level entry points (the building blocks of dit_step; used by the parity tests and by
 *      bench.py's per-kernel roofline lines) ------------------------------------------------------ */

typedef enum {
  DIT_EPI_BIAS = 0,      /* out = A W^T + b                      (out in dtype) */
  DIT_EPI_BIAS_GELU = 1, /* out = GELU_tanh(A W^T + b)           (north_star subsystem 3) */
  DIT_EPI_BIAS_F32 = 2   /* out = A W^T + b, stored fp32         (residual-stream producers) */
} dit_epilogue;

/* out[M, N] = epilogue(A[M, K] W[N, K]^T + bias[N]).  A row stride lda, out row stride ldo (elements);
 * W contiguous [N, K]; bias may be NULL.  bf16: tcgen05/TMEM/TMA GEMM (K % 8 == 0, lda % 8 == 0, 16-byte
 * aligned pointers), fp32: FFMA GEMM. */
dit_status dit_linear(int32_t dtype, int32_t epilogue, const void* A, int64_t lda, const void* W, const void* bias,
                      void* out, int64_t ldo, int32_t M, int32_t N, int32_t K, void* stream);

/* Gated-MLP up-projection (SwiGLU; dit_config.mlp_gated, R40):
 *   out[M, N] = SiLU(A W1^T + b1) (.) (A W3^T + b3);  W1, W3 contiguous [N, K]; b1, b3 [N] or NULL; A, W, b, out in dtype.
 * bf16: ONE tcgen05 kernel (the CTA pair stages W1 | W3 halves of a 256-column accumulator tile, the epilogue gates);
 * tmp is ignored.  fp32: two FFMA GEMMs + an elementwise product; tmp dev fp32 [M, N] is required, out contiguous. */
dit_status dit_linear_swiglu(int32_t dtype, const void* A, int64_t lda, const void* W1, const void* b1, const void* W3,
                             const void* b3, void* out, int64_t ldo, void* tmp, int32_t M, int32_t N, int32_t K, void* stream);

/* fp8 (E4M3) linear layer — SURVEY.md §8(f) item 2 ("fp8 ... GEMMs with the same oracle"); reading R42.  Kernel-level
 * only: a bf16 dit_step never uses it (e4m3 operands miss BASELINE.json's 5e-3 tolerance by ~7x).
 *
 * dit_quantize_fp8: per row of x [M, K] (dev, dtype DIT_BF16 or DIT_F32, row stride ldx elements):
 *     amax = max_k |x[m,k]|;  scale[m] = amax / 448,  inv = 448 / amax (fp32 divisions; both 1 for an all-zero row);
 *     q[m,k] = e4m3(x[m,k] * inv): one fp32 multiplication, round-to-nearest-even, saturating at +-448.  q dev uint8 [M, ldq] (e4m3 "fn" codes: S.EEEE.MMM, bias 7, no inf),
 *   scale dev fp32 [M].  K, ldx, ldq multiples of 8; x 16-byte, q 8-byte aligned.
 * dit_linear_fp8:  out[M, N] = epilogue( a_scale[m] * w_scale[n] * sum_k val(Aq[m,k]) val(Wq[n,k]) + bias[n] )
 *   Aq dev uint8 [M, lda], Wq dev uint8 [N, K] contiguous, a_scale [M] / w_scale [N] dev fp32, bias dev bf16 [N] or NULL,
 *   out dev bf16 [M, ldo] (DIT_EPI_BIAS, DIT_EPI_BIAS_GELU) or fp32 (DIT_EPI_BIAS_F32).  tcgen05 kind::f8f6f4 MMAs, fp32
 *   accumulation.  K and lda multiples of 16, N and ldo of 8, 16-byte aligned pointers; DIT_ERR_UNSUPPORTED otherwise
 *   (there is no FFMA substitute). */
dit_status dit_quantize_fp8(int32_t dtype, const void* x, int64_t ldx, int32_t M, int32_t K, void* q, int64_t ldq,
                            float* scale, void* stream);
dit_status dit_linear_fp8(int32_t epilogue, const void* Aq, int64_t lda, const float* a_scale, const void* Wq,
                          const float* w_scale, const void* bias, void* out, int64_t ldo, int32_t M, int32_t N, int32_t K,
                          void* stream);

/* Block-scaled MXFP8 linear layer (OCP Microscaling format) — SURVEY.md §8(f) item 2 ("block-scaled ... mxf8 GEMMs with the same
 * oracle"); reading R43.  Kernel level only, like the fp8 layer above.
 *
 * dit_quantize_mxfp8: per block of 32 consecutive elements along K of x [M, K] (dev, DIT_BF16 or DIT_F32, row stride ldx):
 *     amax = max |v|;  shared_exp = clamp(floor(log2(amax)) - 8, -127, 127)  (0 for a zero block);
 *     scales[m, b] = shared_exp + 127  (E8M0: X = 2^(code - 127));   q[m, k] = e4m3(v / X)  (RN-even, saturating at +-448)
 *   q dev uint8 [M, ldq], scales dev uint8 [M, K / 32] contiguous.  K % 32 == 0, ldx % 8 == 0, ldq % 16 == 0, 16-byte aligned.
 * dit_linear_mxfp8:  out[M, N] = epilogue( sum_b Xa[m, b] Xw[n, b] sum_{k in b} val(Aq[m, k]) val(Wq[n, k]) + bias[n] )
 *   Aq dev uint8 [M, lda], a_scales dev uint8 [M, K / 32]; Wq dev uint8 [N, K] contiguous, w_scales dev uint8 [N, K / 32]; bias dev
 *   bf16 [N] or NULL; out dev bf16 [M, ldo] (DIT_EPI_BIAS, DIT_EPI_BIAS_GELU) or fp32 (DIT_EPI_BIAS_F32).  tcgen05
 *   kind::mxf8f6f4.block_scale MMAs (the tensor core applies the block scales), fp32 accumulation.  K % 128 == 0, lda % 16 == 0,
 *   N and ldo multiples of 8, operands 16-byte and scales 4-byte aligned; DIT_ERR_UNSUPPORTED otherwise. */
dit_status dit_quantize_mxfp8(int32_t dtype, const void* x, int64_t ldx, int32_t M, int32_t K, void* q, int64_t ldq, void* scales,
                              void* stream);
dit_status dit_linear_mxfp8(int32_t epilogue, const void* Aq, int64_t lda, const void* a_scales, const void* Wq, const void* w_scales,
                            const void* bias, void* out, int64_t ldo, int32_t M, int32_t N, int32_t K, void* stream);

/* Residual-stream producer with the gate fused in the GEMM epilogue (north_star subsystem 3, "gate epilogues";
 * the out-projection and fc2 of every block):   x[M, N] <- x + gate[req(row)] (.) (A[M, K] W[N, K]^T + bias[N])
 *   x dev fp32 [M, ldx] in/out;  A, W, bias in dtype;  gate dev fp32 [n_requests, gate_stride] (NULL = 1), row ->
 *   request through cu_seqlens_dev [n_requests + 1] (NULL = one request).  The branch output is never rounded
 *   to bf16 and x is read and written exactly once. */
dit_status dit_linear_residual(int32_t dtype, const void* A, int64_t lda, const void* W, const void* bias, float* x,
                               int64_t ldx, const float* gate, int64_t gate_stride, const int32_t* cu_seqlens_dev,
                               int32_t n_requests, int32_t M, int32_t N, int32_t K, void* stream);

/* QKV projection with QK-RMSNorm and RoPE fused into the GEMM epilogue (north_star subsystems 3 + 4: "QK-RMSNorm and
 * RoPE fused into the Q/K load" — here one step earlier, on the fp32 accumulators, so q and k are rounded to bf16
 * exactly once, readings R5 / R6):
 *   [q | k | v] = A[M, K] W[3D, K]^T + bias[3D];   per head (128 columns) of q and k:
 *   x <- x / sqrt(mean_d(x^2) + rms_eps) (.) g   (g_q / g_k dev [128] in dtype, NULL = no norm), then
 *   (x_2j, x_2j+1) <- (x_2j cos - x_2j+1 sin, x_2j sin + x_2j+1 cos) with rope_cos / rope_sin dev fp32 [M, 64]
 *   (NULL = no RoPE);  v heads get the bias only.  out dev [M, ldo] in dtype.
 * bf16, head_dim 128, D % 128 == 0 only (DIT_ERR_UNSUPPORTED otherwise: call dit_linear + dit_qknorm_rope). */
dit_status dit_linear_qkv(int32_t dtype, const void* A, int64_t lda, const void* W, const void* bias, void* out,
                          int64_t ldo, const void* g_q, const void* g_k, float rms_eps, const float* rope_cos,
                          const float* rope_sin, int32_t hidden, int32_t M, int32_t K, void* stream);

/* adaLN-Zero modulation kernel (north_star subsystem 2), one pass over the row:
 *   if h != NULL:  x <- x + gate (.) h          (gate NULL = 1)       [x fp32 in/out, h dtype]
 *   y = LN(x) (.) (1 + scale) + shift           (shift/scale NULL = 0) [y dtype]
 * x dev [T, D] fp32; gate/shift/scale dev fp32 [R, mod_stride] rows indexed by the request of the token
 * (cu_seqlens_dev [R+1] int32 maps row -> request; NULL means one request). */
dit_status dit_adaln(int32_t dtype, float* x, const void* h, const float* gate, const float* shift,
                     const float* scale, int64_t mod_stride, const int32_t* cu_seqlens_dev, int32_t n_requests,
                     void* y, int32_t T, int32_t D, float eps, void* stream);

/* out[r, n] = sum_k act(in[r, k]) W[n, k] + b[n];  in/out fp32, W/b dtype; act = SiLU if silu_input else id.
 * The t-MLP and the adaLN modulation projection (DESIGN.md §3 steps 1-2): a weight-streaming GEMV. */
dit_status dit_gemv(int32_t dtype, const float* in, const void* W, const void* b, float* out, int32_t R, int32_t N,
                    int32_t K, int32_t silu_input, void* stream);

/* In-place QK-RMSNorm (+ RoPE) of the q and k thirds of a packed qkv buffer [T, 3D] (R5, R6):
 * per token per head  v <- v / sqrt(mean(v^2) + eps) * g, then pairs (2j, 2j+1) rotated by the angle whose
 * cos/sin are rope_cos/rope_sin[T, d/2] (fp32; NULL = no RoPE).  gq/gk [d] dtype (NULL = no norm). */
dit_status dit_qknorm_rope(int32_t dtype, void* qkv, int64_t row_stride, int32_t T, int32_t n_heads, int32_t head_dim,
                           int32_t n_tensors /* 2: q and k; 1: q only */, const void* gq, const void* gk, float eps,
                           const float* rope_cos, const float* rope_sin, void* stream);

/* ---- debugging ---------------------------------------------------------------------------------- */
typedef enum {
  DIT_TAP_X = 0,   /* residual stream x   [T, D]  fp32 */
  DIT_TAP_Y = 1,   /* last adaLN output   [T, D]  dtype */
  DIT_TAP_QKV = 2, /* q|k|v after norm+rope [T, 3D] dtype */
  DIT_TAP_O = 3,   /* attention output    [T, D]  dtype */
  DIT_TAP_U = 5,   /* GELU output         [T, F]  dtype */
  DIT_TAP_C = 6,   /* c                   [R, D]  fp32 */
  DIT_TAP_MOD = 7, /* modulation          [R, L*6*D + 2*D] fp32 */
  DIT_TAP_TOK = 8  /* final-layer tokens  [N, C*pv] fp32 */
} dit_tap;
typedef enum {
  DIT_STAGE_Y1 = 0, DIT_STAGE_QKV = 1, DIT_STAGE_ATTN = 2, DIT_STAGE_OPROJ = 3, DIT_STAGE_CROSS = 4,
  DIT_STAGE_Y2 = 5, DIT_STAGE_FC1 = 6, DIT_STAGE_FC2 = 7
} dit_stage;
/* Make the next steps return right after (block, stage) so workspace buffers can be inspected;
 * block < 0 restores normal operation. */
dit_status dit_debug_stop_after(dit_handle h, int32_t block, int32_t stage);
/* Copy `bytes` of a workspace buffer to dst (dev), stream ordered. */
dit_status dit_get_tap(dit_handle h, int32_t tap, void* dst, size_t bytes, void* stream);

/* ---- measurement (bench.py's roofline line) -------------------------------------------------------
 * Kernel classes of the step.  dit_profile_begin(mask) makes every later launch of a class whose bit is set
 * in `mask` be bracketed by a cudaEvent pair on the stream it is launched on (at most 16384 launches are
 * recorded; later ones are counted but not timed).  dit_profile_end synchronises those events, writes the
 * summed device time (ms) and the launch count per class into the two host arrays [DIT_KC_COUNT], and
 * switches profiling off.  Process-wide; not thread safe; adds ~2 event records per profiled launch. */
typedef enum {
  DIT_KC_GEMM = 0,   /* block GEMMs: QKV, out-proj, fc1, fc2, cross projections (tcgen05) */
  DIT_KC_ATTN = 1,   /* self / cross / partial attention */
  DIT_KC_ADALN = 2,  /* LayerNorm + modulation (+ gated residual) */
  DIT_KC_GEMV = 3,   /* t-MLP and modulation projection (weight streaming) */
  DIT_KC_QKNORM = 4, /* QK-RMSNorm + RoPE (stand-alone form) */
  DIT_KC_MERGE = 5,  /* LSE merge */
  DIT_KC_MISC = 6,   /* patchify, patch-embed / cond / final GEMMs, unpatchify, RoPE table */
  DIT_KC_COUNT = 7
} dit_kernel_class;
dit_status dit_profile_begin(int32_t class_mask);
dit_status dit_profile_end(float* ms_per_class, int32_t* launches_per_class);

const char* dit_last_error(dit_handle h); /* h may be NULL: last error of a handle-less entry point */
int32_t dit_kernel_launches(void);         /* kernels launched by this library so far (this process) */
int32_t dit_fallback_launches(void);       /* of those: bf16 GEMM / attention launches that ran on the fp32-path FFMA kernels
                                              because the shape is outside the tcgen05 kernels' limits (kernel-level entry
                                              points only; a step never does).  0 in every BASELINE.json config. */
void dit_free(dit_handle h);

#ifdef __cplusplus
}
#endif
#endif /* DIT_B200_H */
