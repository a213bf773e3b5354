// dit.cu — handle, workspace carving, step orchestration and the C ABI of libdit_b200 (include/dit.h).
// Every stage of the step is a kernel launch on the caller's stream; no host synchronisation inside a step.
#include <cstdlib>
#include <cstdarg>
#include <cstdio>
#include <cstring>
#include <atomic>
#include <map>
#include <mutex>
#include <string>
#include <vector>

#include "common.cuh"

namespace dit {

std::atomic<int> g_launches{0};
std::atomic<int> g_fallback_launches{0};
static thread_local char g_err[512] = "";
void set_error(const char* fmt, ...) {
  va_list ap;
  va_start(ap, fmt);
  vsnprintf(g_err, sizeof(g_err), fmt, ap);
  va_end(ap);
}
const char* get_error() { return g_err; }

// ---- per-class event timing -------------------------------------------------------------------------
std::atomic<int> g_prof_mask{0};
thread_local int g_prof_class_override = -1;
namespace {
std::mutex g_prof_mu;   // guards the record list, the event pool and the counts (launchers of several host threads)
struct ProfRec { cudaEvent_t a, b; int cls; bool open; };
std::vector<ProfRec> g_prof_recs;
std::vector<cudaEvent_t> g_prof_pool;
int g_prof_counts[DIT_KC_COUNT];
const size_t kProfMax = 16384;
cudaEvent_t prof_event() {
  if (!g_prof_pool.empty()) { cudaEvent_t e = g_prof_pool.back(); g_prof_pool.pop_back(); return e; }
  cudaEvent_t e = nullptr;
  cudaEventCreate(&e);
  return e;
}
}  // namespace
void prof_record(int cls, cudaStream_t st, bool start) {
  std::lock_guard<std::mutex> lk(g_prof_mu);
  if (start) {
    g_prof_counts[cls]++;
    if (g_prof_recs.size() >= kProfMax) return;   // counted, not timed
    ProfRec r{prof_event(), prof_event(), cls, true};
    cudaEventRecord(r.a, st);
    g_prof_recs.push_back(r);
  } else {
    // the matching start is the most recent OPEN record of this class (launchers do not nest within a class); a
    // launch that was counted but not recorded (list full) has no open record and its end is dropped
    for (size_t i = g_prof_recs.size(); i-- > 0;)
      if (g_prof_recs[i].cls == cls) {
        if (g_prof_recs[i].open) { cudaEventRecord(g_prof_recs[i].b, st); g_prof_recs[i].open = false; }
        break;
      }
  }
}

static size_t esize(int dtype) { return dtype == DIT_F32 ? 4 : 2; }

struct BlockW {
  const void *mod_w, *mod_b, *wqkv, *bqkv, *gq, *gk, *wo, *bo, *w1, *b1, *w2, *b2;
  const void *w3, *b3, *t_w3, *t_b3;   // gated MLP (mlp_gated, R40): the second up-projection (image / text stream)
  const void *cwq, *cbq, *cwkv, *cbkv, *cgq, *cgk, *cwo, *cbo;
  // dual-stream joint blocks (DIT_COND_JOINT2, R37): the text stream's own copy of the per-block tensors
  const void *t_mod_w, *t_mod_b, *t_wqkv, *t_bqkv, *t_gq, *t_gk, *t_wo, *t_bo, *t_w1, *t_b1, *t_w2, *t_b2;
};

struct Workspace {
  float* x;        // [Tm, D] residual stream fp32
  void* y;         // [Tm, D]
  void* qkv;       // [Tm, 3D]
  void* o;         // [Tm, D]
  void* u;         // [Tm, F]
  void* u3;        // [Tm, F]: gated MLP on the FFMA path only (the W3 product before the elementwise gate)
  float* c1;       // [Rm, D] first t-MLP layer
  float* c;        // [Rm, D]
  float* mod;      // [Rm, L*6D + 2D]
  float* rope_c;   // [Tm, d/2]
  float* rope_s;
  void* patches;   // [Tm, C*pv]
  float* tok;      // [Tm, C*pv] fp32
  void* ctx;       // cross: [Lcm, D]
  void* kvc;       // cross: [Lcm, 2D]
  void* o_part;    // [P, Tm, D]   (split_p > 1)
  float* lse_part; // [P, Tm, H]
  int32_t* cu_dev;     // [Rm+1]
  int32_t* cu_cond_dev;// [Rm+1]
  int32_t* cu_seg_dev; // [2 Rm + 1]: dual-stream blocks, row segments text | image of every request
  SeqMeta* meta_dev;   // [Rm]
  GemvBatch* gemv_tab; // [L + 1 + 2]
  void* stage_in;  // host-call staging: latents | temb | cond
  void* stage_out;
  float* sample_x; // dit_sample: fp32 trajectory state [Tm * C*pv]
  float* sample_v; // dit_sample: unconditional velocity of a guided step, fp32
  float* traj;     // dit_sample: [S, D] c1 | [S, D] c | [S, mod_len] modulation of S = max_sample_steps steps computed ahead
  size_t total;
};

}  // namespace dit

using namespace dit;

struct dit_handle_s {
  dit_config cfg;
  BlockW* blocks;
  int n_blocks;
  const void *t_w1, *t_b1, *t_w2, *t_b2, *pe_w, *pe_b, *cp_w, *cp_b, *fm_w, *fm_b, *f_w, *f_b;
  Workspace ws;
  int stop_block, stop_stage;
  // geometry resident on the device (cu_seqlens, cond offsets, per-request meta, RoPE tables): uploads are skipped
  // when a call's geometry equals it in EVERY field
  std::vector<int32_t> last_geom;
  bool capturing = false;              // inside a stream capture: no host -> device copy may be enqueued
  // dit_step_graph / dit_step_varlen_graph: up to 8 captured steps, least recently used replaced
  struct StepGraph { std::vector<uint64_t> key; cudaGraphExec_t exec; uint64_t used; };
  std::vector<StepGraph> step_graphs;
  uint64_t step_graph_clock = 0;
  // dit_sample: one cached trajectory graph, valid while every argument (and sigma) it was captured with is unchanged
  cudaGraphExec_t graph_exec = nullptr;
  // dit_step_host / dit_step_varlen_host: the latent / cond uploads run on this stream while the caller's stream computes the
  // timestep MLP and the modulation GEMV (0.17-0.25 ms that need only temb); joined by an event before patch-embed
  cudaStream_t copy_stream = nullptr;
  cudaEvent_t ev_fork = nullptr, ev_copied = nullptr;
  cudaEvent_t wait_before_embed = nullptr;   // set by the host-buffer entry points for the duration of one run_step
  cudaStream_t cap_stream = nullptr;   // capture happens here (the caller's stream may be the legacy default stream)
  std::vector<uint64_t> graph_key;
  char err[512];
};

namespace dit {

static size_t align256(size_t v) { return (v + 255) & ~(size_t)255; }

static bool carve(const dit_config& c, char* base, Workspace* w) {
  const size_t es = esize(c.dtype);
  const size_t Tm = c.max_tokens, D = c.hidden, F = c.mlp_dim, Rm = c.max_requests, L = c.n_blocks;
  const size_t pvC = (size_t)c.latent_channels * c.patch[0] * c.patch[1] * c.patch[2];
  const size_t Lcm = c.max_cond_tokens;
  size_t off = 0;
  auto take = [&](size_t bytes) {
    char* p = base ? base + off : nullptr;
    off += align256(bytes);
    return (void*)p;
  };
  w->x = (float*)take(Tm * D * 4);
  w->y = take(Tm * 2 * D * es);   // [Tm, D]; the final adaLN writes [Tm, 2D] = [hi | lo] (bf16, R36)
  w->qkv = take(Tm * 3 * D * es);
  w->o = take(Tm * D * es);
  w->u = take(Tm * F * es);
  w->u3 = take(c.mlp_gated && c.dtype == DIT_F32 ? Tm * F * es : 0);
  w->c1 = (float*)take(Rm * D * 4);
  w->c = (float*)take(Rm * D * 4);
  w->mod = (float*)take(Rm * (L * (c.cond_mode == DIT_COND_JOINT2 ? 12 : 6) * D + 2 * D) * 4);   // [img blocks | final | txt blocks]
  w->rope_c = (float*)take(Tm * (c.head_dim / 2) * 4);
  w->rope_s = (float*)take(Tm * (c.head_dim / 2) * 4);
  w->patches = take(Tm * pvC * es);
  w->tok = (float*)take(Tm * pvC * 4);
  w->ctx = take(c.cond_mode == DIT_COND_CROSS ? Lcm * 2 * D * es : 0);   // bf16: [Lcm, 2D] = [hi | lo] (R36)
  w->kvc = take(c.cond_mode == DIT_COND_CROSS ? Lcm * 2 * D * es : 0);
  w->o_part = take(c.split_p > 1 ? (size_t)c.split_p * Tm * D * es : 0);
  w->lse_part = (float*)take(c.split_p > 1 ? (size_t)c.split_p * Tm * c.n_heads * 4 : 0);
  w->cu_dev = (int32_t*)take((Rm + 1) * 4);
  w->cu_cond_dev = (int32_t*)take((Rm + 1) * 4);
  w->cu_seg_dev = (int32_t*)take(c.cond_mode == DIT_COND_JOINT2 ? (2 * Rm + 1) * 4 : 0);
  w->meta_dev = (SeqMeta*)take(Rm * sizeof(SeqMeta));
  w->gemv_tab = (GemvBatch*)take((2 * L + 4) * sizeof(GemvBatch));
  w->stage_in = take(Tm * pvC * es + Rm * c.temb_dim * 4 + Lcm * c.cond_dim * es + 1024);
  w->stage_out = take(Tm * pvC * es);
  w->sample_x = (float*)take(Tm * pvC * 4);
  w->sample_v = (float*)take(Tm * pvC * 4);
  w->traj = (float*)take((size_t)c.max_sample_steps * (2 * D + L * (c.cond_mode == DIT_COND_JOINT2 ? 12 : 6) * D + 2 * D) * 4);
  w->total = off;
  return true;
}

static dit_status validate(const dit_config* c) {
  DIT_REQUIRE(c != nullptr, DIT_ERR_INVALID_ARG, "config is NULL");
  DIT_REQUIRE(c->struct_size == (int)sizeof(dit_config), DIT_ERR_INVALID_ARG, "dit_config.struct_size %d != %d",
              c->struct_size, (int)sizeof(dit_config));
  DIT_REQUIRE(c->dtype == DIT_F32 || c->dtype == DIT_BF16, DIT_ERR_INVALID_ARG, "dtype %d", c->dtype);
  DIT_REQUIRE(c->n_blocks >= 0 && c->n_blocks <= 256, DIT_ERR_INVALID_ARG, "n_blocks %d", c->n_blocks);
  DIT_REQUIRE(c->max_sample_steps >= 0 && c->max_sample_steps <= 4096, DIT_ERR_INVALID_ARG, "max_sample_steps %d not in 0..4096",
              c->max_sample_steps);
  DIT_REQUIRE(c->head_dim == 64 || c->head_dim == 128, DIT_ERR_UNSUPPORTED, "head_dim %d not in {64,128}", c->head_dim);
  DIT_REQUIRE(c->n_heads > 0 && c->hidden == c->n_heads * c->head_dim, DIT_ERR_INVALID_ARG,
              "hidden %d != n_heads %d * head_dim %d", c->hidden, c->n_heads, c->head_dim);
  DIT_REQUIRE(c->hidden % 256 == 0, DIT_ERR_UNSUPPORTED, "hidden %d must be a multiple of 256", c->hidden);
  {  // the adaLN kernel is instantiated for these row widths (elementwise.cu, launch_adaln_t)
    const int nc = c->hidden / 256;
    const bool ok = nc == 1 || nc == 2 || nc == 3 || nc == 4 || nc == 5 || nc == 6 || nc == 8 || nc == 10 || nc == 12 ||
                    nc == 16 || nc == 20 || nc == 24;
    DIT_REQUIRE(ok, DIT_ERR_UNSUPPORTED, "hidden %d: hidden / 256 must be one of 1,2,3,4,5,6,8,10,12,16,20,24", c->hidden);
  }
  if (c->dtype == DIT_BF16) {   // a bf16 step runs on the tcgen05 kernels only (no FFMA substitute inside a step)
    const int pvC = c->latent_channels * c->patch[0] * c->patch[1] * c->patch[2];
    DIT_REQUIRE(c->head_dim == 128, DIT_ERR_UNSUPPORTED, "bf16 configs need head_dim 128 (tcgen05 attention); got %d", c->head_dim);
    DIT_REQUIRE(pvC % 8 == 0, DIT_ERR_UNSUPPORTED, "bf16 configs need latent_channels * patch volume (%d) to be a multiple of 8", pvC);
    DIT_REQUIRE(c->cond_mode == DIT_COND_NONE || c->cond_dim % 8 == 0, DIT_ERR_UNSUPPORTED,
                "bf16 configs need cond_dim (%d) to be a multiple of 8", c->cond_dim);
  }
  DIT_REQUIRE(c->mlp_dim > 0 && c->mlp_dim % 8 == 0, DIT_ERR_UNSUPPORTED, "mlp_dim %d must be a multiple of 8", c->mlp_dim);
  DIT_REQUIRE(c->mlp_gated == 0 || c->mlp_gated == 1, DIT_ERR_INVALID_ARG, "mlp_gated %d not in {0,1}", c->mlp_gated);
  DIT_REQUIRE(c->latent_channels > 0 && c->patch[0] > 0 && c->patch[1] > 0 && c->patch[2] > 0, DIT_ERR_INVALID_ARG,
              "latent_channels / patch must be positive");
  DIT_REQUIRE(c->temb_dim > 0 && c->temb_dim % 8 == 0, DIT_ERR_UNSUPPORTED, "temb_dim %d must be a multiple of 8", c->temb_dim);
  DIT_REQUIRE(c->cond_mode >= DIT_COND_NONE && c->cond_mode <= DIT_COND_JOINT2, DIT_ERR_INVALID_ARG, "cond_mode %d", c->cond_mode);
  DIT_REQUIRE(c->cond_mode == DIT_COND_NONE || c->cond_dim > 0, DIT_ERR_INVALID_ARG, "cond_dim %d", c->cond_dim);
  DIT_REQUIRE(c->cond_mode != DIT_COND_JOINT2 || c->n_blocks <= 128, DIT_ERR_UNSUPPORTED,
              "dual-stream blocks: n_blocks %d > 128 (one modulation launch covers 2 L + 1 matrices)", c->n_blocks);
  const int rs = c->rope_dims[0] + c->rope_dims[1] + c->rope_dims[2];
  DIT_REQUIRE(rs == 0 || rs == c->head_dim, DIT_ERR_INVALID_ARG, "sum(rope_dims) = %d must be 0 or head_dim", rs);
  for (int a = 0; a < 3; ++a)
    DIT_REQUIRE(c->rope_dims[a] >= 0 && c->rope_dims[a] % 2 == 0, DIT_ERR_INVALID_ARG, "rope_dims[%d] = %d must be even", a, c->rope_dims[a]);
  DIT_REQUIRE(c->split_p == 1 || c->split_p == 2 || c->split_p == 4 || c->split_p == 8, DIT_ERR_INVALID_ARG,
              "split_p %d not in {1,2,4,8}", c->split_p);
  DIT_REQUIRE(c->max_tokens > 0 && c->max_requests > 0 && c->max_requests <= 64 && c->max_cond_tokens >= 0,
              DIT_ERR_INVALID_ARG, "capacities: max_tokens %d max_requests %d max_cond_tokens %d", c->max_tokens,
              c->max_requests, c->max_cond_tokens);
  return DIT_OK;
}

bool pdl_enabled() {
  static const bool on = []() {
    const char* e = getenv("DIT_NO_PDL");
    return !(e != nullptr && e[0] == '1');
  }();
  return on;
}

// Inside a denoising step (run_step) a bf16 config must run on the tcgen05 kernels: the FFMA kernels are the fp32 path,
// ~100x slower, and never a silent substitute (north_star: "no multi-backend dispatch").  The kernel-level entry points
// (dit_linear, dit_attn_partial, ...) still accept shapes the tensor-core kernels do not (head_dim 64, K % 8 != 0) and
// run them on the FFMA kernels; every such launch is counted in dit_fallback_launches().
static thread_local bool g_strict_tc = false;
#define DIT_STRICT_TC(what)                                                                                    \
  DIT_REQUIRE(!g_strict_tc, DIT_ERR_UNSUPPORTED, "bf16 step: %s does not meet the tcgen05 kernels' requirements " \
              "(head_dim 128, K / N / strides multiples of 8, 16-byte aligned pointers)", what)

// GEMM dispatch: bf16 -> tcgen05 whenever the shape/alignment allows, else FFMA.  fp32 -> FFMA (no TF32).
static dit_status gemm(int dtype, int epi, const void* A, int64_t lda, const void* W, const void* bias, void* out,
                       int64_t ldo, int M, int N, int K, cudaStream_t st, int kc = DIT_KC_GEMM, int a_split = 0) {
  struct Override { int prev; Override(int c) : prev(g_prof_class_override) { g_prof_class_override = c; }
                    ~Override() { g_prof_class_override = prev; } } ov(kc == DIT_KC_GEMM ? -1 : kc);
  if (dtype == DIT_BF16 && gemm_tc_supported(epi, A, lda, W, out, ldo, M, N, K))
    return launch_gemm_tc(epi, A, lda, W, bias, out, ldo, M, N, K, st, a_split);
  DIT_REQUIRE(!a_split && epi <= DIT_EPI_BIAS_F32, DIT_ERR_UNSUPPORTED, "split-bf16 operands exist on the tcgen05 path only");
  if (dtype == DIT_BF16 && M > 0) {
    DIT_STRICT_TC("a GEMM");
    g_fallback_launches++;   // visible through dit_fallback_launches()
  }
  return launch_gemm_simt(dtype, epi, A, lda, W, bias, out, ldo, M, N, K, st);
}

// MLP up-projection  u <- act(y W1^T + b1)  (§8(a) a10): GELU(tanh), or with `w3` the gated form SiLU(.) (.) (y W3^T + b3)
// (R40) — one tcgen05 kernel on the bf16 path, two FFMA GEMMs and an elementwise product on the fp32 path.
static dit_status gemm_mlp_up(int dtype, const void* y, const void* w1, const void* b1, const void* w3, const void* b3,
                              void* u, void* u3, int M, int F, int D, cudaStream_t st) {
  if (w3 == nullptr) return gemm(dtype, DIT_EPI_BIAS_GELU, y, D, w1, b1, u, F, M, F, D, st);
  if (M == 0) return DIT_OK;
  if (dtype == DIT_BF16) {
    if (!gemm_tc_supported(DIT_EPI_BIAS, y, D, w1, u, F, M, F, D) || ((uintptr_t)w3 & 15)) DIT_STRICT_TC("the gated MLP up-projection");
    DIT_REQUIRE(gemm_tc_supported(DIT_EPI_BIAS, y, D, w1, u, F, M, F, D) && !((uintptr_t)w3 & 15), DIT_ERR_UNSUPPORTED,
                "gated MLP (bf16) runs on the tcgen05 kernel only");
    return launch_gemm_tc_swiglu(y, D, w1, b1, w3, b3, u, F, M, F, D, st);
  }
  DIT_REQUIRE(u3 != nullptr, DIT_ERR_WORKSPACE, "gated MLP: no workspace for the second up-projection");
  dit_status s = gemm(dtype, DIT_EPI_BIAS, y, D, w1, b1, u, F, M, F, D, st);
  if (s != DIT_OK) return s;
  s = gemm(dtype, DIT_EPI_BIAS, y, D, w3, b3, u3, F, M, F, D, st);
  if (s != DIT_OK) return s;
  return launch_silu_mul(dtype, u, u3, (int64_t)M * F, st);
}

// Residual-stream producer  x <- x + gate (.) (A W^T + bias)  (out-projection, fc2).
// The gated add runs in the GEMM's fp32 epilogue: the branch output is never rounded to bf16 and x is touched once.
static dit_status gemm_residual(int dtype, const void* A, int64_t lda, const void* W, const void* bias, float* x,
                                int64_t ldx, const float* gate, int64_t gate_stride, const int32_t* cu, int R, int M,
                                int N, int K, cudaStream_t st) {
  if (dtype == DIT_BF16 && gemm_tc_supported(3, A, lda, W, x, ldx, M, N, K))
    return launch_gemm_tc_ex(3, A, lda, W, bias, x, ldx, gate, gate_stride, cu, R, M, N, K, st);
  if (dtype == DIT_BF16 && M > 0) {
    DIT_STRICT_TC("a residual GEMM");
    g_fallback_launches++;
  }
  return launch_gemm_simt(dtype, 3, A, lda, W, bias, x, ldx, M, N, K, st, gate, gate_stride, cu, R);
}

static dit_status attention(int dtype, const AttnArgs& a, cudaStream_t st) {
  if (dtype == DIT_BF16 && attn_tc_supported(a)) return launch_attn_tc(a, st);
  if (dtype == DIT_BF16 && a.n_q > 0) {
    DIT_STRICT_TC("attention");
    g_fallback_launches++;
  }
  return launch_attn_simt(dtype, a, st);
}

struct StepGeom {
  int R;
  std::vector<int32_t> cu;        // [R+1] sequence rows
  std::vector<int32_t> cu_cond;   // [R+1] cond rows in cond_packed
  std::vector<int32_t> ncond;     // [R]
  std::vector<int32_t> grids;     // [R][3] latent grids
  std::vector<int64_t> lat_off;   // [R+1] element offsets in the packed latents
};

// Per-call geometry to the device (pageable host memory: the driver stages it before returning) and the RoPE tables;
// skipped when the geometry is the one already resident.  Not capturable: dit_sample calls it before it begins a capture.
// A handle's workspace (and this geometry) is shared by all its calls: calls on one handle must be stream ordered by the
// caller (include/dit.h, conventions).
static dit_status upload_geom(dit_handle hd, const StepGeom& g, cudaStream_t st) {
  const dit_config& c = hd->cfg;
  Workspace& w = hd->ws;
  const int R = g.R, T = g.cu[R], d = c.head_dim;
  const bool joint = c.cond_mode == DIT_COND_JOINT || c.cond_mode == DIT_COND_JOINT2;
  const bool rope = (c.rope_dims[0] + c.rope_dims[1] + c.rope_dims[2]) > 0;
  std::vector<SeqMeta> meta(R);
  // The key holds everything the device copies are made from: sequence starts, the cond-token offsets of EVERY mode
  // (cross-attention reads cu_cond_dev: same latent grids with other prompt lengths is the normal serving case), the
  // token grids, the latent offsets and the total row count.
  std::vector<int32_t> geom;
  for (int r = 0; r < R; ++r) {
    meta[r].seq_start = g.cu[r];
    meta[r].n_cond = joint ? g.ncond[r] : 0;
    meta[r].gf = g.grids[3 * r] / c.patch[0];
    meta[r].gh = g.grids[3 * r + 1] / c.patch[1];
    meta[r].gw = g.grids[3 * r + 2] / c.patch[2];
    meta[r].lat_off_lo = (int32_t)(g.lat_off[r] & 0xffffffff);
    meta[r].lat_off_hi = (int32_t)(g.lat_off[r] >> 32);
    meta[r].pad = 0;
    // (one cross / cond-less request: no kernel reads the cond offsets, so the two passes of an unpacked guided step
    // with different prompt lengths share one resident geometry and stay capturable)
    const bool cond_used = joint || R > 1;
    geom.insert(geom.end(), {meta[r].seq_start, cond_used ? g.ncond[r] : 0, cond_used ? g.cu_cond[r + 1] : 0, meta[r].gf,
                             meta[r].gh, meta[r].gw, meta[r].lat_off_lo, meta[r].lat_off_hi});
  }
  geom.push_back(T);
  geom.push_back(R);
  if (geom == hd->last_geom) return DIT_OK;
  DIT_REQUIRE(!hd->capturing, DIT_ERR_CUDA, "geometry changed inside a stream capture");
  DIT_CUDA_OK(cudaMemcpyAsync(w.cu_dev, g.cu.data(), (R + 1) * 4, cudaMemcpyHostToDevice, st));
  DIT_CUDA_OK(cudaMemcpyAsync(w.cu_cond_dev, g.cu_cond.data(), (R + 1) * 4, cudaMemcpyHostToDevice, st));
  DIT_CUDA_OK(cudaMemcpyAsync(w.meta_dev, meta.data(), R * sizeof(SeqMeta), cudaMemcpyHostToDevice, st));
  if (c.cond_mode == DIT_COND_JOINT2) {   // segment starts: text of request r at cu[r], its image rows at cu[r] + n_cond[r]
    std::vector<int32_t> seg(2 * R + 1);
    for (int r = 0; r < R; ++r) { seg[2 * r] = g.cu[r]; seg[2 * r + 1] = g.cu[r] + g.ncond[r]; }
    seg[2 * R] = T;
    DIT_CUDA_OK(cudaMemcpyAsync(w.cu_seg_dev, seg.data(), (2 * R + 1) * 4, cudaMemcpyHostToDevice, st));
  }
  if (rope) {
    dit_status s = launch_rope_table(w.meta_dev, R, T, d, c.rope_dims, c.rope_theta, w.rope_c, w.rope_s, st);
    if (s != DIT_OK) return s;
  }
  hd->last_geom = geom;
  return DIT_OK;
}

// `pair` (dit_sample, guided step as ONE packed pass): the R = 2 requests are the unconditional and the conditional pass
// of the same latents at the same timestep — one t-MLP / modulation row serves both (row stride 0), each request has its
// own cond pointer and its own unpatchify epilogue.
struct GuidedPair { const void* cond[2]; const SampleEpi* epi[2]; };
// mod_pre != nullptr: this step's modulation row was computed ahead (dit_sample, max_sample_steps): no timestep MLP / GEMV here
static dit_status run_step(dit_handle hd, const StepGeom& g, const void* latents, const float* temb, const void* cond,
                           void* out, cudaStream_t st, const SampleEpi* epi = nullptr, const GuidedPair* pair = nullptr,
                           const float* mod_pre = nullptr) {
  const dit_config& c = hd->cfg;
  Workspace& w = hd->ws;
  const int dt = c.dtype;
  const size_t es = esize(dt);
  const int D = c.hidden, F = c.mlp_dim, H = c.n_heads, d = c.head_dim, L = c.n_blocks, R = g.R;
  const int pvC = c.latent_channels * c.patch[0] * c.patch[1] * c.patch[2];
  const int T = g.cu[R];
  const bool dual = c.cond_mode == DIT_COND_JOINT2;
  const int64_t mod_img = (int64_t)L * 6 * D + 2 * D;                 // image-stream blocks + final layer
  const int64_t mod_len = mod_img + (dual ? (int64_t)L * 6 * D : 0);   // ... + text-stream blocks (dual-stream, R37)
  const int Rt = pair ? 1 : R;                      // timestep rows
  const int64_t mod_stride = pair ? 0 : mod_len;    // modulation row of request r = mod + r * mod_stride
  auto cond_of = [&](int r) -> const char* {
    return pair ? (const char*)pair->cond[r] : (const char*)cond + (size_t)g.cu_cond[r] * c.cond_dim * esize(c.dtype);
  };
  const bool joint = c.cond_mode == DIT_COND_JOINT || dual, cross = c.cond_mode == DIT_COND_CROSS;
  const bool rope = (c.rope_dims[0] + c.rope_dims[1] + c.rope_dims[2]) > 0;
  auto stop = [&](int blk, int stage) { return hd->stop_block == blk && hd->stop_stage == stage; };
  {
    dit_status gs = upload_geom(hd, g, st);
    if (gs != DIT_OK) return gs;
  }
  struct Strict { bool prev; Strict(bool on) : prev(g_strict_tc) { g_strict_tc = on; } ~Strict() { g_strict_tc = prev; } }
      strict(dt == DIT_BF16);
  const int32_t* cu_dev = R > 1 ? w.cu_dev : nullptr;
  dit_status s;
#define RUN(expr)                  \
  do {                             \
    s = (expr);                    \
    if (s != DIT_OK) return s;     \
  } while (0)

  // ---- steps 1-2: c = W2 SiLU(W1 temb + b1) + b2;  mod = Wmod SiLU(c) + bmod for ALL blocks in one launch
  const float* const mod = mod_pre != nullptr ? mod_pre : w.mod;
  if (mod_pre == nullptr) {
    RUN(launch_gemv(dt, temb, w.gemv_tab + 0, nullptr, 1, D, w.c1, D, Rt, c.temb_dim, 0, st));
    RUN(launch_gemv(dt, w.c1, w.gemv_tab + 1, nullptr, 1, D, w.c, D, Rt, D, 1, st));
    // The GEMV kernels take 8 input rows per pass over the weights.  A packed bf16 step of MORE than 8 requests runs the
    // modulation as tensor-core GEMMs instead — SiLU(c) as an unevaluated [hi | lo] pair of bf16 rows (R36: ~16 significand
    // bits), one M = R GEMM per modulation matrix, fp32 out: the weights are streamed once, not ceil(R / 8) times by passes that
    // are FMA-bound at 8 rows (64 requests at the cfg 2 model: 3.4 ms of GEMV passes -> 0.3 ms).
    static const bool mod_gemv_env = [] { const char* e = getenv("DIT_MOD_GEMV"); return e != nullptr && e[0] == '1'; }();
    const bool mod_tc = dt == DIT_BF16 && Rt > 8 && !mod_gemv_env && D % 64 == 0 &&
                        gemm_tc_supported(DIT_EPI_BIAS_F32, w.y, 2 * D, hd->fm_w, w.mod, mod_len, Rt, 2 * D, 2 * D);
    if (mod_tc) {
      RUN(launch_silu_split(w.c, w.y, Rt, D, st));   // w.y is free until the first adaLN
      struct Override { int prev; Override() : prev(g_prof_class_override) { g_prof_class_override = DIT_KC_GEMV; }
                        ~Override() { g_prof_class_override = prev; } } ov;
      auto one = [&](const void* Wm, const void* bm, int N, int64_t off) -> dit_status {
        return launch_gemm_tc(DIT_EPI_BIAS_F32, w.y, 2 * D, Wm, bm, w.mod + off, mod_len, Rt, N, D, st, 1);
      };
      for (int l = 0; l < L; ++l) RUN(one(hd->blocks[l].mod_w, hd->blocks[l].mod_b, 6 * D, (int64_t)l * 6 * D));
      RUN(one(hd->fm_w, hd->fm_b, 2 * D, (int64_t)L * 6 * D));
      if (dual)
        for (int l = 0; l < L; ++l) RUN(one(hd->blocks[l].t_mod_w, hd->blocks[l].t_mod_b, 6 * D, mod_img + (int64_t)l * 6 * D));
    } else {
      RUN(launch_gemv(dt, w.c, w.gemv_tab + 2, nullptr, dual ? 2 * L + 1 : L + 1, (int)mod_len, w.mod, mod_len, Rt, D, 1, st));
    }
  }

  if (hd->wait_before_embed != nullptr) DIT_CUDA_OK(cudaStreamWaitEvent(st, hd->wait_before_embed, 0));   // inputs uploaded
  // ---- steps 3-4: patch-embed and cond projection write the fp32 residual stream
  // A packed step of R > 1 requests: ONE patchify launch over all requests (geometry from the device table), ONE patch-embed
  // GEMM over all T rows — patches live in sequence rows, the cond rows of a joint sequence hold whatever the buffer held and
  // their x rows are overwritten by the cond projection right after — and at the end ONE final GEMM and ONE unpatchify:
  // 4 launches instead of 4 R.  (Row-wise GEMM results do not depend on how rows are tiled: bit-identical to the per-request
  // form, which DIT_VARLEN_PER_REQUEST=1 brings back.)
  static const bool per_request_env = [] { const char* e = getenv("DIT_VARLEN_PER_REQUEST"); return e != nullptr && e[0] == '1'; }();
  const bool batched_ends = R > 1 && pair == nullptr && epi == nullptr && !per_request_env;
  int64_t max_elems = 0;
  for (int r = 0; r < R; ++r) max_elems = std::max<int64_t>(max_elems, g.lat_off[r + 1] - g.lat_off[r]);
  // (joint modes) the cond projection too, when its fp32 result fits the MLP scratch it borrows
  const bool cond_once = batched_ends && joint && g.cu_cond[R] > 0 && (size_t)g.cu_cond[R] * D * 4 <= (size_t)c.max_tokens * F * es;
  if (batched_ends) {
    RUN(launch_patchify_varlen(dt, latents, w.patches, w.meta_dev, R, max_elems, c.latent_channels, c.patch, st));
    RUN(gemm(dt, DIT_EPI_BIAS_F32, w.patches, pvC, hd->pe_w, hd->pe_b, w.x, D, T, D, pvC, st, DIT_KC_MISC));
  }
  for (int r = 0; r < R; ++r) {
    const int Fr = g.grids[3 * r], Hr = g.grids[3 * r + 1], Wr = g.grids[3 * r + 2];
    const int Nr = (Fr / c.patch[0]) * (Hr / c.patch[1]) * (Wr / c.patch[2]);
    const int Lc = joint ? g.ncond[r] : 0;
    const int row0 = g.cu[r] + Lc;
    char* pr = (char*)w.patches + (size_t)row0 * pvC * es;
    if (!batched_ends) {
      RUN(launch_patchify(dt, (const char*)latents + g.lat_off[r] * es, pr, c.latent_channels, Fr, Hr, Wr, c.patch, st));
      RUN(gemm(dt, DIT_EPI_BIAS_F32, pr, pvC, hd->pe_w, hd->pe_b, w.x + (size_t)row0 * D, D, Nr, D, pvC, st, DIT_KC_MISC));
    }
    if (joint && Lc > 0 && !cond_once)
      RUN(gemm(dt, DIT_EPI_BIAS_F32, cond_of(r), c.cond_dim, hd->cp_w, hd->cp_b, w.x + (size_t)g.cu[r] * D, D, Lc, D,
               c.cond_dim, st, DIT_KC_MISC));
  }
  if (cond_once) {   // ONE cond projection over the packed cond tokens into scratch (w.u is free until the first MLP), then
                     // one row scatter to the heads of the requests' segments: an exact fp32 copy
    RUN(gemm(dt, DIT_EPI_BIAS_F32, cond, c.cond_dim, hd->cp_w, hd->cp_b, w.u, D, g.cu_cond[R], D, c.cond_dim, st, DIT_KC_MISC));
    RUN(launch_scatter_cond_rows((const float*)w.u, w.x, w.cu_dev, w.cu_cond_dev, R, g.cu_cond[R], D, st));
  }
  const int Lc_total = g.cu_cond[R];
  // R36: in a bf16 step the cross-attention context and the final layer's input are kept as an unevaluated sum of two
  // bf16 numbers [hi | lo] (~16 significand bits); their consumer GEMMs read both parts as one A operand of width 2K
  // against W wrapped along K.  These operands are small (Lc rows; one N = C*pv GEMM), their rounding is not.
  const bool split = dt == DIT_BF16;
  const int ctx_ld = split ? 2 * D : D;
  if (cross && Lc_total > 0) {
    const int cepi = split ? 5 /* EPI_BIAS_SPLIT */ : DIT_EPI_BIAS;
    if (!pair) {
      RUN(gemm(dt, cepi, cond, c.cond_dim, hd->cp_w, hd->cp_b, w.ctx, ctx_ld, Lc_total, D, c.cond_dim, st, DIT_KC_MISC));
    } else {
      for (int r = 0; r < R; ++r)
        if (g.ncond[r] > 0)
          RUN(gemm(dt, cepi, cond_of(r), c.cond_dim, hd->cp_w, hd->cp_b, (char*)w.ctx + (size_t)g.cu_cond[r] * ctx_ld * es, ctx_ld,
                   g.ncond[r], D, c.cond_dim, st, DIT_KC_MISC));
    }
  }

  // ---- step 5: blocks.  Both residual branches are added to x inside their GEMM epilogues (gemm_residual).
  const float scale = 1.0f / sqrtf((float)d);
  // dual-stream blocks: every request is two row segments (its text rows, its image rows) with their own weights and
  // modulation; per-row kernels and GEMMs run once per segment, attention once over the joint sequence
  struct Seg { int row0, rows, r; bool txt; };
  std::vector<Seg> segs;
  if (dual)
    for (int r = 0; r < R; ++r) {
      const int Lc = g.ncond[r];
      if (Lc > 0) segs.push_back({g.cu[r], Lc, r, true});
      if (g.cu[r + 1] - g.cu[r] - Lc > 0) segs.push_back({g.cu[r] + Lc, g.cu[r + 1] - g.cu[r] - Lc, r, false});
    }
  // bf16: ONE segmented tcgen05 launch per projection covers every segment of both streams (GemmSegs); fp32: per segment
  GemmSegs gsegs;
  gsegs.n = 0;
  const bool grouped = dual && dt == DIT_BF16 && (int)segs.size() <= GEMM_MAX_SEGS;
  if (grouped) {
    gsegs.tile0[0] = 0;
    for (const Seg& sg : segs) {
      const int i = gsegs.n++;
      gsegs.row0[i] = sg.row0; gsegs.rows[i] = sg.rows; gsegs.which[i] = sg.txt ? 1 : 0; gsegs.req[i] = (uint8_t)sg.r;
      gsegs.tile0[i + 1] = gsegs.tile0[i] + (sg.rows + 255) / 256;
    }
  }
  for (int l = 0; l < L; ++l) {
    const BlockW& b = hd->blocks[l];
    if (dual) {
      struct SW { const void *wqkv, *bqkv, *gq, *gk, *wo, *bo, *w1, *b1, *w2, *b2, *w3, *b3; };
      const SW sw_img{b.wqkv, b.bqkv, b.gq, b.gk, b.wo, b.bo, b.w1, b.b1, b.w2, b.b2, b.w3, b.b3};
      const SW sw_txt{b.t_wqkv, b.t_bqkv, b.t_gq, b.t_gk, b.t_wo, b.t_bo, b.t_w1, b.t_b1, b.t_w2, b.t_b2, b.t_w3, b.t_b3};
      auto mod_of = [&](const Seg& sg) { return mod + (size_t)sg.r * mod_stride + (sg.txt ? mod_img : 0) + (size_t)l * 6 * D; };
      auto rows_of = [&](void* base, const Seg& sg, int64_t ld) { return (void*)((char*)base + (size_t)sg.row0 * ld * es); };
      // adaLN: one launch over all segments (row -> segment -> request and stream through cu_seg_dev)
      const float* mblk = mod + (size_t)l * 6 * D;
      RUN(launch_adaln(dt, w.x, nullptr, nullptr, mblk, mblk + D, mod_stride, w.cu_seg_dev, 2 * R, w.y, T, D, c.ln_eps, st, 0, mod_img));
      if (stop(l, DIT_STAGE_Y1)) return DIT_OK;
      SegGemm sgm{};   // the fields every segmented launch of this block shares
      sgm.segs = &gsegs; sgm.M = T; sgm.rms_eps = c.rms_eps;
      sgm.gate = mod + (size_t)l * 6 * D; sgm.gate_stride = mod_stride; sgm.gate_set_off = mod_img;
      if (grouped) {
        DIT_REQUIRE(gemm_tc_supported(DIT_EPI_BIAS, w.y, D, sw_img.wqkv, w.qkv, 3 * D, T, 3 * D, D), DIT_ERR_UNSUPPORTED,
                    "bf16 dual-stream step: the tcgen05 GEMM is unavailable");
        SegGemm q = sgm;
        q.kind = 4; q.A = w.y; q.lda = D; q.out = w.qkv; q.ldo = 3 * D; q.N = 3 * D; q.K = D;
        q.W[0] = sw_img.wqkv; q.W[1] = sw_txt.wqkv; q.bias[0] = sw_img.bqkv; q.bias[1] = sw_txt.bqkv;
        if (c.qk_rmsnorm) { q.gq[0] = sw_img.gq; q.gq[1] = sw_txt.gq; q.gk[0] = sw_img.gk; q.gk[1] = sw_txt.gk; }
        q.rc = rope ? w.rope_c : nullptr; q.rs = rope ? w.rope_s : nullptr;
        RUN(launch_gemm_tc_segs(q, st));
      } else
      for (const Seg& sg : segs) {
        const SW& sw = sg.txt ? sw_txt : sw_img;
        const float* rc = rope ? w.rope_c + (size_t)sg.row0 * (d / 2) : nullptr;
        const float* rs = rope ? w.rope_s + (size_t)sg.row0 * (d / 2) : nullptr;
        const void* gq = c.qk_rmsnorm ? sw.gq : nullptr;
        const void* gk = c.qk_rmsnorm ? sw.gk : nullptr;
        if (dt == DIT_BF16 && (c.qk_rmsnorm || rope)) {
          RUN(launch_gemm_tc_qkv(rows_of(w.y, sg, D), D, sw.wqkv, sw.bqkv, rows_of(w.qkv, sg, 3 * D), 3 * D, gq, gk, c.rms_eps, rc, rs, D,
                                 2 * D, sg.rows, 3 * D, D, st));
        } else {
          RUN(gemm(dt, DIT_EPI_BIAS, rows_of(w.y, sg, D), D, sw.wqkv, sw.bqkv, rows_of(w.qkv, sg, 3 * D), 3 * D, sg.rows, 3 * D, D, st));
          RUN(launch_qknorm_rope(dt, rows_of(w.qkv, sg, 3 * D), 3 * D, sg.rows, H, d, 2, gq, gk, c.rms_eps, rc, rs, st));
        }
      }
      if (stop(l, DIT_STAGE_QKV)) return DIT_OK;
      {
        AttnArgs a;
        a.q = w.qkv; a.k = (char*)w.qkv + (size_t)D * es; a.v = (char*)w.qkv + (size_t)2 * D * es;
        a.q_stride = a.kv_stride = 3 * D;
        a.cu_q = a.cu_k = R > 1 ? w.cu_dev : nullptr;
        a.cu_q_host = a.cu_k_host = g.cu.data();
        a.R = R; a.n_q = T; a.n_k = T; a.H = H; a.d = d; a.scale = 1.0f / sqrtf((float)d);
        if (c.split_p == 1) {
          a.o = w.o; a.o_stride = D; a.lse = nullptr; a.shard = 0; a.n_shards = 1;
          RUN(attention(dt, a, st));
        } else {
          const void* op[8];
          const float* lp[8];
          for (int p = 0; p < c.split_p; ++p) {
            a.o = (char*)w.o_part + (size_t)p * c.max_tokens * D * es;
            a.o_stride = D;
            a.lse = w.lse_part + (size_t)p * c.max_tokens * H;
            a.shard = p; a.n_shards = c.split_p;
            op[p] = a.o; lp[p] = a.lse;
            RUN(attention(dt, a, st));
          }
          RUN(launch_merge(dt, op, lp, c.split_p, (int64_t)T * H, d, w.o, nullptr, st));
        }
      }
      if (stop(l, DIT_STAGE_ATTN)) return DIT_OK;
      if (grouped) {
        SegGemm q = sgm;
        q.kind = 3; q.A = w.o; q.lda = D; q.out = w.x; q.ldo = D; q.N = D; q.K = D;
        q.W[0] = sw_img.wo; q.W[1] = sw_txt.wo; q.bias[0] = sw_img.bo; q.bias[1] = sw_txt.bo;
        q.gate += 2 * D;
        RUN(launch_gemm_tc_segs(q, st));
      } else
      for (const Seg& sg : segs) {
        const SW& sw = sg.txt ? sw_txt : sw_img;
        RUN(gemm_residual(dt, rows_of(w.o, sg, D), D, sw.wo, sw.bo, w.x + (size_t)sg.row0 * D, D, mod_of(sg) + 2 * D, 0, nullptr, 1,
                          sg.rows, D, D, st));
      }
      if (stop(l, DIT_STAGE_OPROJ)) return DIT_OK;
      RUN(launch_adaln(dt, w.x, nullptr, nullptr, mblk + 3 * D, mblk + 4 * D, mod_stride, w.cu_seg_dev, 2 * R, w.y, T, D, c.ln_eps, st, 0,
                       mod_img));
      if (stop(l, DIT_STAGE_Y2)) return DIT_OK;
      if (grouped) {
        SegGemm q = sgm;
        q.kind = sw_img.w3 != nullptr ? 6 : 1; q.A = w.y; q.lda = D; q.out = w.u; q.ldo = F; q.N = F; q.K = D;
        q.W[0] = sw_img.w1; q.W[1] = sw_txt.w1; q.bias[0] = sw_img.b1; q.bias[1] = sw_txt.b1;
        q.W3[0] = sw_img.w3; q.W3[1] = sw_txt.w3; q.b3[0] = sw_img.b3; q.b3[1] = sw_txt.b3;
        RUN(launch_gemm_tc_segs(q, st));
      } else
      for (const Seg& sg : segs) {
        const SW& sw = sg.txt ? sw_txt : sw_img;
        RUN(gemm_mlp_up(dt, rows_of(w.y, sg, D), sw.w1, sw.b1, sw.w3, sw.b3, rows_of(w.u, sg, F),
                        w.u3 != nullptr ? rows_of(w.u3, sg, F) : nullptr, sg.rows, F, D, st));
      }
      if (stop(l, DIT_STAGE_FC1)) return DIT_OK;
      if (grouped) {
        SegGemm q = sgm;
        q.kind = 3; q.A = w.u; q.lda = F; q.out = w.x; q.ldo = D; q.N = D; q.K = F;
        q.W[0] = sw_img.w2; q.W[1] = sw_txt.w2; q.bias[0] = sw_img.b2; q.bias[1] = sw_txt.b2;
        q.gate += 5 * D;
        RUN(launch_gemm_tc_segs(q, st));
      } else
      for (const Seg& sg : segs) {
        const SW& sw = sg.txt ? sw_txt : sw_img;
        RUN(gemm_residual(dt, rows_of(w.u, sg, F), F, sw.w2, sw.b2, w.x + (size_t)sg.row0 * D, D, mod_of(sg) + 5 * D, 0, nullptr, 1,
                          sg.rows, D, F, st));
      }
      if (stop(l, DIT_STAGE_FC2)) return DIT_OK;
      continue;
    }
    const float* m = mod + (size_t)l * 6 * D;
    RUN(launch_adaln(dt, w.x, nullptr, nullptr, m + 0 * D, m + 1 * D, mod_stride, cu_dev, R, w.y, T, D, c.ln_eps, st));
    if (stop(l, DIT_STAGE_Y1)) return DIT_OK;
    if (dt == DIT_BF16 && d == 128 && (c.qk_rmsnorm || rope) &&
        gemm_tc_supported(DIT_EPI_BIAS, w.y, D, b.wqkv, w.qkv, 3 * D, T, 3 * D, D)) {
      // QK-RMSNorm + RoPE on the fp32 accumulators in the QKV GEMM's epilogue (north_star subsystems 3 + 4)
      RUN(launch_gemm_tc_qkv(w.y, D, b.wqkv, b.bqkv, w.qkv, 3 * D, c.qk_rmsnorm ? b.gq : nullptr,
                             c.qk_rmsnorm ? b.gk : nullptr, c.rms_eps, rope ? w.rope_c : nullptr,
                             rope ? w.rope_s : nullptr, D, 2 * D, T, 3 * D, D, st));
    } else {
      RUN(gemm(dt, DIT_EPI_BIAS, w.y, D, b.wqkv, b.bqkv, w.qkv, 3 * D, T, 3 * D, D, st));
      RUN(launch_qknorm_rope(dt, w.qkv, 3 * D, T, H, d, 2, c.qk_rmsnorm ? b.gq : nullptr, c.qk_rmsnorm ? b.gk : nullptr,
                             c.rms_eps, rope ? w.rope_c : nullptr, rope ? w.rope_s : nullptr, st));
    }
    if (stop(l, DIT_STAGE_QKV)) return DIT_OK;
    {
      AttnArgs a;
      a.q = w.qkv; a.k = (char*)w.qkv + (size_t)D * es; a.v = (char*)w.qkv + (size_t)2 * D * es;
      a.q_stride = a.kv_stride = 3 * D;
      a.cu_q = a.cu_k = R > 1 ? w.cu_dev : nullptr;
      a.cu_q_host = a.cu_k_host = g.cu.data();
      a.R = R; a.n_q = T; a.n_k = T; a.H = H; a.d = d; a.scale = scale;
      if (c.split_p == 1) {
        a.o = w.o; a.o_stride = D; a.lse = nullptr; a.shard = 0; a.n_shards = 1;
        RUN(attention(dt, a, st));
      } else {  // P split-KV partials + LSE merge (north_star subsystem 5)
        const void* op[8];
        const float* lp[8];
        for (int p = 0; p < c.split_p; ++p) {
          a.o = (char*)w.o_part + (size_t)p * c.max_tokens * D * es;
          a.o_stride = D;
          a.lse = w.lse_part + (size_t)p * c.max_tokens * H;
          a.shard = p; a.n_shards = c.split_p;
          op[p] = a.o; lp[p] = a.lse;
          RUN(attention(dt, a, st));
        }
        RUN(launch_merge(dt, op, lp, c.split_p, (int64_t)T * H, d, w.o, nullptr, st));
      }
    }
    if (stop(l, DIT_STAGE_ATTN)) return DIT_OK;
    RUN(gemm_residual(dt, w.o, D, b.wo, b.bo, w.x, D, m + 2 * D, mod_stride, cu_dev, R, T, D, D, st));
    if (stop(l, DIT_STAGE_OPROJ)) return DIT_OK;
    if (cross) {  // R10: x <- x + Wo_c Attn(RMS(Wq_c LN(x)), RMS(Wk_c ctx), Wv_c ctx) + bo_c   (no gate, no modulation)
      RUN(launch_adaln(dt, w.x, nullptr, nullptr, nullptr, nullptr, mod_stride, cu_dev, R, w.y, T, D, c.ln_eps, st));
      // bf16: the per-head RMSNorm of the cross q / k runs on the fp32 accumulators of their projections (one bf16
      // rounding instead of two, and no stand-alone pass over [T, D]); fp32 path: stand-alone kernel
      const bool fused = dt == DIT_BF16 && d == 128 && gemm_tc_supported(DIT_EPI_BIAS, w.y, D, b.cwq, w.qkv, D, T, D, D);
      if (fused) {
        RUN(launch_gemm_tc_qkv(w.y, D, b.cwq, b.cbq, w.qkv, D, b.cgq, nullptr, c.rms_eps, nullptr, nullptr, D, D, T, D, D, st));
      } else {
        RUN(gemm(dt, DIT_EPI_BIAS, w.y, D, b.cwq, b.cbq, w.qkv, D, T, D, D, st));
        RUN(launch_qknorm_rope(dt, w.qkv, D, T, H, d, 1, b.cgq, nullptr, c.rms_eps, nullptr, nullptr, st));
      }
      if (Lc_total > 0) {
        if (fused) {
          RUN(launch_gemm_tc_qkv(w.ctx, ctx_ld, b.cwkv, b.cbkv, w.kvc, 2 * D, nullptr, b.cgk, c.rms_eps, nullptr, nullptr, 0, D,
                                 Lc_total, 2 * D, D, st, split ? 1 : 0));
        } else {
          RUN(gemm(dt, DIT_EPI_BIAS, w.ctx, ctx_ld, b.cwkv, b.cbkv, w.kvc, 2 * D, Lc_total, 2 * D, D, st, DIT_KC_GEMM, split ? 1 : 0));
          RUN(launch_qknorm_rope(dt, w.kvc, 2 * D, Lc_total, H, d, 1, b.cgk, nullptr, c.rms_eps, nullptr, nullptr, st));
        }
      }
      AttnArgs a;
      a.q = w.qkv; a.q_stride = D;
      a.k = w.kvc; a.v = (char*)w.kvc + (size_t)D * es; a.kv_stride = 2 * D;
      a.o = w.o; a.o_stride = D; a.lse = nullptr;
      a.cu_q = R > 1 ? w.cu_dev : nullptr; a.cu_k = R > 1 ? w.cu_cond_dev : nullptr;
      a.cu_q_host = g.cu.data(); a.cu_k_host = g.cu_cond.data();
      a.R = R; a.n_q = T; a.n_k = Lc_total; a.H = H; a.d = d; a.scale = scale; a.shard = 0; a.n_shards = 1;
      RUN(attention(dt, a, st));
      RUN(gemm_residual(dt, w.o, D, b.cwo, b.cbo, w.x, D, nullptr, 0, cu_dev, R, T, D, D, st));
      if (stop(l, DIT_STAGE_CROSS)) return DIT_OK;
    }
    RUN(launch_adaln(dt, w.x, nullptr, nullptr, m + 3 * D, m + 4 * D, mod_stride, cu_dev, R, w.y, T, D, c.ln_eps, st));
    if (stop(l, DIT_STAGE_Y2)) return DIT_OK;
    RUN(gemm_mlp_up(dt, w.y, b.w1, b.b1, b.w3, b.b3, w.u, w.u3, T, F, D, st));
    if (stop(l, DIT_STAGE_FC1)) return DIT_OK;
    RUN(gemm_residual(dt, w.u, F, b.w2, b.b2, w.x, D, m + 5 * D, mod_stride, cu_dev, R, T, D, F, st));
    if (stop(l, DIT_STAGE_FC2)) return DIT_OK;
  }
  // ---- step 6: final adaLN (folds the last gated residual), Linear D -> C*pv, unpatchify (image tokens only)
  const float* mf = mod + (size_t)L * 6 * D;
  RUN(launch_adaln(dt, w.x, nullptr, nullptr, mf, mf + D, mod_stride, cu_dev, R, w.y, T, D, c.ln_eps, st, split ? 1 : 0));
  const int y_ld = split ? 2 * D : D;
  if (batched_ends) {   // all rows at once (the cond rows' tokens are computed and never read)
    RUN(gemm(dt, DIT_EPI_BIAS_F32, w.y, y_ld, hd->f_w, hd->f_b, w.tok, pvC, T, pvC, D, st, DIT_KC_MISC, split ? 1 : 0));
    RUN(launch_unpatchify_varlen(dt, w.tok, out, w.meta_dev, R, max_elems, c.latent_channels, c.patch, st));
  }
  for (int r = 0; r < R && !batched_ends; ++r) {
    const int Fr = g.grids[3 * r], Hr = g.grids[3 * r + 1], Wr = g.grids[3 * r + 2];
    const int Nr = (Fr / c.patch[0]) * (Hr / c.patch[1]) * (Wr / c.patch[2]);
    const int row0 = g.cu[r] + (joint ? g.ncond[r] : 0);
    float* tk = w.tok + (size_t)row0 * pvC;
    RUN(gemm(dt, DIT_EPI_BIAS_F32, (char*)w.y + (size_t)row0 * y_ld * es, y_ld, hd->f_w, hd->f_b, tk, pvC, Nr, pvC, D, st, DIT_KC_MISC,
             split ? 1 : 0));
    RUN(launch_unpatchify(dt, tk, (char*)out + g.lat_off[r] * es, c.latent_channels, Fr, Hr, Wr, c.patch, st,
                          pair ? pair->epi[r] : epi));
  }
#undef RUN
  return DIT_OK;
}

static dit_status build_geom(dit_handle h, int R, const int32_t* cu, const int32_t* ncond, const int32_t* grids,
                             StepGeom* g) {
  const dit_config& c = h->cfg;
  DIT_REQUIRE(R >= 1 && R <= c.max_requests, DIT_ERR_INVALID_ARG, "n_requests %d not in 1..%d", R, c.max_requests);
  g->R = R;
  g->cu.assign(R + 1, 0);
  g->cu_cond.assign(R + 1, 0);
  g->ncond.assign(R, 0);
  g->grids.assign(grids, grids + 3 * R);
  g->lat_off.assign(R + 1, 0);
  for (int r = 0; r < R; ++r) {
    const int Fr = grids[3 * r], Hr = grids[3 * r + 1], Wr = grids[3 * r + 2];
    DIT_REQUIRE(Fr > 0 && Hr > 0 && Wr > 0 && Fr % c.patch[0] == 0 && Hr % c.patch[1] == 0 && Wr % c.patch[2] == 0,
                DIT_ERR_INVALID_ARG, "request %d: latent grid {%d,%d,%d} not a positive multiple of the patch", r, Fr, Hr, Wr);
    const int64_t Nr = (int64_t)(Fr / c.patch[0]) * (Hr / c.patch[1]) * (Wr / c.patch[2]);
    const int nc = c.cond_mode == DIT_COND_NONE ? 0 : (ncond ? ncond[r] : 0);
    DIT_REQUIRE(nc >= 0, DIT_ERR_INVALID_ARG, "request %d: n_cond %d < 0", r, nc);
    g->ncond[r] = nc;
    const int64_t Tr = Nr + (c.cond_mode == DIT_COND_JOINT || c.cond_mode == DIT_COND_JOINT2 ? nc : 0);
    DIT_REQUIRE(g->cu[r] + Tr <= c.max_tokens, DIT_ERR_INVALID_ARG, "sequence rows exceed max_tokens %d", c.max_tokens);
    g->cu[r + 1] = g->cu[r] + (int32_t)Tr;
    g->cu_cond[r + 1] = g->cu_cond[r] + nc;
    g->lat_off[r + 1] = g->lat_off[r] + (int64_t)c.latent_channels * Fr * Hr * Wr;
    if (cu) DIT_REQUIRE(cu[r + 1] - cu[r] == Tr && cu[0] == 0, DIT_ERR_INVALID_ARG,
                        "cu_seqlens[%d..%d] = %d disagrees with grid/n_cond (%lld rows)", r, r + 1, cu[r + 1] - cu[r], (long long)Tr);
  }
  DIT_REQUIRE(g->cu_cond[R] <= c.max_cond_tokens, DIT_ERR_INVALID_ARG, "cond tokens %d exceed max_cond_tokens %d",
              g->cu_cond[R], c.max_cond_tokens);
  return DIT_OK;
}

}  // namespace dit

// =================================================================================================
// C ABI
// =================================================================================================
extern "C" {

size_t dit_workspace_bytes(const dit_config* cfg) {
  if (validate(cfg) != DIT_OK) return 0;
  Workspace w;
  carve(*cfg, nullptr, &w);
  return w.total;
}

dit_status dit_init(const dit_config* cfg, const dit_weight* weights, int32_t n_weights, void* workspace,
                    size_t workspace_bytes, dit_handle* out) {
  DIT_REQUIRE(out != nullptr, DIT_ERR_INVALID_ARG, "out handle pointer is NULL");
  *out = nullptr;
  dit_status s = validate(cfg);
  if (s != DIT_OK) return s;
  DIT_REQUIRE(workspace != nullptr && ((uintptr_t)workspace & 255) == 0, DIT_ERR_WORKSPACE, "workspace must be 256-byte aligned");
  Workspace w;
  carve(*cfg, (char*)workspace, &w);
  DIT_REQUIRE(workspace_bytes >= w.total, DIT_ERR_WORKSPACE, "workspace too small: %zu < %zu", workspace_bytes, w.total);
  DIT_REQUIRE(weights != nullptr || n_weights == 0, DIT_ERR_INVALID_ARG, "weights is NULL");

  const int64_t D = cfg->hidden, F = cfg->mlp_dim, d = cfg->head_dim, L = cfg->n_blocks;
  const int64_t pvC = (int64_t)cfg->latent_channels * cfg->patch[0] * cfg->patch[1] * cfg->patch[2];
  std::map<std::string, int64_t> need;
  need["t_mlp.w1"] = D * cfg->temb_dim; need["t_mlp.b1"] = D; need["t_mlp.w2"] = D * D; need["t_mlp.b2"] = D;
  need["patch_embed.w"] = D * pvC; need["patch_embed.b"] = D;
  if (cfg->cond_mode != DIT_COND_NONE) { need["cond_proj.w"] = D * cfg->cond_dim; need["cond_proj.b"] = D; }
  for (int l = 0; l < L; ++l) {
    std::string p = "blocks." + std::to_string(l) + ".";
    need[p + "mod.w"] = 6 * D * D; need[p + "mod.b"] = 6 * D;
    need[p + "attn.wqkv"] = 3 * D * D; need[p + "attn.bqkv"] = 3 * D;
    if (cfg->qk_rmsnorm) { need[p + "attn.gq"] = d; need[p + "attn.gk"] = d; }
    need[p + "attn.wo"] = D * D; need[p + "attn.bo"] = D;
    need[p + "mlp.w1"] = F * D; need[p + "mlp.b1"] = F; need[p + "mlp.w2"] = D * F; need[p + "mlp.b2"] = D;
    if (cfg->mlp_gated) {
      need[p + "mlp.w3"] = F * D; need[p + "mlp.b3"] = F;
      if (cfg->cond_mode == DIT_COND_JOINT2) { need[p + "txt.mlp.w3"] = F * D; need[p + "txt.mlp.b3"] = F; }
    }
    if (cfg->cond_mode == DIT_COND_JOINT2) {
      need[p + "txt.mod.w"] = 6 * D * D; need[p + "txt.mod.b"] = 6 * D;
      need[p + "txt.attn.wqkv"] = 3 * D * D; need[p + "txt.attn.bqkv"] = 3 * D;
      if (cfg->qk_rmsnorm) { need[p + "txt.attn.gq"] = d; need[p + "txt.attn.gk"] = d; }
      need[p + "txt.attn.wo"] = D * D; need[p + "txt.attn.bo"] = D;
      need[p + "txt.mlp.w1"] = F * D; need[p + "txt.mlp.b1"] = F; need[p + "txt.mlp.w2"] = D * F; need[p + "txt.mlp.b2"] = D;
    }
    if (cfg->cond_mode == DIT_COND_CROSS) {
      need[p + "cross.wq"] = D * D; need[p + "cross.bq"] = D; need[p + "cross.wkv"] = 2 * D * D; need[p + "cross.bkv"] = 2 * D;
      need[p + "cross.gq"] = d; need[p + "cross.gk"] = d; need[p + "cross.wo"] = D * D; need[p + "cross.bo"] = D;
    }
  }
  need["final.mod.w"] = 2 * D * D; need["final.mod.b"] = 2 * D; need["final.w"] = pvC * D; need["final.b"] = pvC;
  std::map<std::string, const void*> got;
  for (int i = 0; i < n_weights; ++i) {
    DIT_REQUIRE(weights[i].name != nullptr, DIT_ERR_INVALID_ARG, "weight %d has no name", i);
    auto it = need.find(weights[i].name);
    DIT_REQUIRE(it != need.end(), DIT_ERR_INVALID_ARG, "unknown weight '%s'", weights[i].name);
    DIT_REQUIRE(it->second == weights[i].numel, DIT_ERR_INVALID_ARG, "weight '%s': numel %lld, expected %lld",
                weights[i].name, (long long)weights[i].numel, (long long)it->second);
    DIT_REQUIRE(weights[i].dev_ptr != nullptr && ((uintptr_t)weights[i].dev_ptr & 15) == 0, DIT_ERR_INVALID_ARG,
                "weight '%s': pointer must be non-NULL and 16-byte aligned", weights[i].name);
    got[weights[i].name] = weights[i].dev_ptr;
  }
  for (auto& kv : need) DIT_REQUIRE(got.count(kv.first), DIT_ERR_INVALID_ARG, "missing weight '%s'", kv.first.c_str());

  dit_handle h = new dit_handle_s();
  h->cfg = *cfg;
  h->ws = w;
  h->n_blocks = (int)L;
  h->blocks = new BlockW[L > 0 ? L : 1];
  h->stop_block = -1; h->stop_stage = -1;
  h->err[0] = 0;
  auto G = [&](const std::string& n) -> const void* { auto it = got.find(n); return it == got.end() ? nullptr : it->second; };
  h->t_w1 = G("t_mlp.w1"); h->t_b1 = G("t_mlp.b1"); h->t_w2 = G("t_mlp.w2"); h->t_b2 = G("t_mlp.b2");
  h->pe_w = G("patch_embed.w"); h->pe_b = G("patch_embed.b"); h->cp_w = G("cond_proj.w"); h->cp_b = G("cond_proj.b");
  h->fm_w = G("final.mod.w"); h->fm_b = G("final.mod.b"); h->f_w = G("final.w"); h->f_b = G("final.b");
  const bool dual = cfg->cond_mode == DIT_COND_JOINT2;
  std::vector<GemvBatch> tab((dual ? 2 * L : L) + 3);
  tab[0] = {h->t_w1, h->t_b1, (int32_t)D, 0, 0, 0};
  tab[1] = {h->t_w2, h->t_b2, (int32_t)D, 0, 0, 0};
  for (int l = 0; l < L; ++l) {
    std::string p = "blocks." + std::to_string(l) + ".";
    BlockW& b = h->blocks[l];
    b.mod_w = G(p + "mod.w"); b.mod_b = G(p + "mod.b"); b.wqkv = G(p + "attn.wqkv"); b.bqkv = G(p + "attn.bqkv");
    b.gq = G(p + "attn.gq"); b.gk = G(p + "attn.gk"); b.wo = G(p + "attn.wo"); b.bo = G(p + "attn.bo");
    b.w1 = G(p + "mlp.w1"); b.b1 = G(p + "mlp.b1"); b.w2 = G(p + "mlp.w2"); b.b2 = G(p + "mlp.b2");
    b.w3 = G(p + "mlp.w3"); b.b3 = G(p + "mlp.b3"); b.t_w3 = G(p + "txt.mlp.w3"); b.t_b3 = G(p + "txt.mlp.b3");
    b.cwq = G(p + "cross.wq"); b.cbq = G(p + "cross.bq"); b.cwkv = G(p + "cross.wkv"); b.cbkv = G(p + "cross.bkv");
    b.cgq = G(p + "cross.gq"); b.cgk = G(p + "cross.gk"); b.cwo = G(p + "cross.wo"); b.cbo = G(p + "cross.bo");
    b.t_mod_w = G(p + "txt.mod.w"); b.t_mod_b = G(p + "txt.mod.b"); b.t_wqkv = G(p + "txt.attn.wqkv"); b.t_bqkv = G(p + "txt.attn.bqkv");
    b.t_gq = G(p + "txt.attn.gq"); b.t_gk = G(p + "txt.attn.gk"); b.t_wo = G(p + "txt.attn.wo"); b.t_bo = G(p + "txt.attn.bo");
    b.t_w1 = G(p + "txt.mlp.w1"); b.t_b1 = G(p + "txt.mlp.b1"); b.t_w2 = G(p + "txt.mlp.w2"); b.t_b2 = G(p + "txt.mlp.b2");
    tab[2 + l] = {b.mod_w, b.mod_b, (int32_t)(6 * D), (int32_t)(l * 6 * D), (int32_t)(l * 6 * D), 0};
    if (dual) {   // text-stream modulation rows follow the image blocks and the final layer
      const int32_t off = (int32_t)(L * 6 * D + 2 * D + l * 6 * D);
      tab[3 + L + l] = {b.t_mod_w, b.t_mod_b, (int32_t)(6 * D), off, off, 0};
    }
  }
  tab[2 + L] = {h->fm_w, h->fm_b, (int32_t)(2 * D), (int32_t)(L * 6 * D), (int32_t)(L * 6 * D), 0};
  cudaError_t e = cudaMemcpy(w.gemv_tab, tab.data(), tab.size() * sizeof(GemvBatch), cudaMemcpyHostToDevice);
  if (e != cudaSuccess) {
    set_error("dit_init: pointer-table upload failed: %s", cudaGetErrorString(e));
    delete[] h->blocks;
    delete h;
    return DIT_ERR_CUDA;
  }
  *out = h;
  return DIT_OK;
}

dit_status dit_step_varlen(dit_handle h, const void* latents_packed, const float* timestep_emb, const void* cond_packed,
                           const int32_t* cu_seqlens, const int32_t* n_cond, const int32_t* latent_grids,
                           int32_t n_requests, void* out_packed, void* stream) {
  DIT_REQUIRE(h != nullptr, DIT_ERR_INVALID_ARG, "handle is NULL");
  DIT_REQUIRE(latents_packed && timestep_emb && latent_grids && out_packed, DIT_ERR_INVALID_ARG, "NULL tensor argument");
  StepGeom g;
  dit_status s = build_geom(h, n_requests, cu_seqlens, n_cond, latent_grids, &g);
  if (s != DIT_OK) return s;
  DIT_REQUIRE(g.cu_cond[n_requests] == 0 || cond_packed != nullptr, DIT_ERR_INVALID_ARG, "cond tokens announced but cond pointer is NULL");
  return run_step(h, g, latents_packed, timestep_emb, cond_packed, out_packed, (cudaStream_t)stream);
}

dit_status dit_step(dit_handle h, const void* latents, const float* timestep_emb, const void* cond_tokens,
                    int32_t n_cond, const int32_t latent_grid[3], void* out, void* stream) {
  return dit_step_varlen(h, latents, timestep_emb, cond_tokens, nullptr, &n_cond, latent_grid, 1, out, stream);
}

// The step as ONE cudaGraphLaunch: the paper's control plane dispatches a request one denoising step at a time,
// and a step is 65+ kernel launches (~0.4 ms of host time at 6 us each; a 512^2 request's step is 2.4 ms of GPU time).  The
// captured graph holds every pointer and the geometry: it is replayed while the call's arguments are the same (buffer CONTENTS
// may change), else captured again; the handle keeps the 8 most recently used graphs.
dit_status dit_step_varlen_graph(dit_handle h, const void* latents_packed, const float* timestep_emb, const void* cond_packed,
                                 const int32_t* cu_seqlens, const int32_t* n_cond, const int32_t* latent_grids, int32_t n_requests,
                                 void* out_packed, void* stream) {
  DIT_REQUIRE(h != nullptr, DIT_ERR_INVALID_ARG, "handle is NULL");
  DIT_REQUIRE(latents_packed && timestep_emb && latent_grids && out_packed, DIT_ERR_INVALID_ARG, "NULL tensor argument");
  StepGeom g;
  dit_status s = build_geom(h, n_requests, cu_seqlens, n_cond, latent_grids, &g);
  if (s != DIT_OK) return s;
  DIT_REQUIRE(g.cu_cond[n_requests] == 0 || cond_packed != nullptr, DIT_ERR_INVALID_ARG, "cond tokens announced but cond pointer is NULL");
  cudaStream_t st = (cudaStream_t)stream;
  // no graph while per-class profiling is on (event records are not captured) or a debug stop is set
  if (g_prof_mask.load() != 0 || h->stop_block >= 0) return run_step(h, g, latents_packed, timestep_emb, cond_packed, out_packed, st);
  std::vector<uint64_t> key = {(uint64_t)(uintptr_t)latents_packed, (uint64_t)(uintptr_t)timestep_emb, (uint64_t)(uintptr_t)cond_packed,
                               (uint64_t)(uintptr_t)out_packed, (uint64_t)n_requests};
  for (int r = 0; r < n_requests; ++r) {
    key.push_back((uint64_t)g.cu[r + 1]);
    key.push_back((uint64_t)g.ncond[r]);
    for (int a = 0; a < 3; ++a) key.push_back((uint64_t)latent_grids[3 * r + a]);
  }
  // geometry copies and the RoPE table are not part of the graph: enqueued ahead of the capture or the replay whenever another
  // call has left a different geometry on the device (else a no-op)
  s = upload_geom(h, g, st);
  if (s != DIT_OK) return s;
  dit_handle_s::StepGraph* hit = nullptr;
  for (auto& sg : h->step_graphs)
    if (sg.key == key) hit = &sg;
  if (hit == nullptr) {
    if (h->cap_stream == nullptr) DIT_CUDA_OK(cudaStreamCreateWithFlags(&h->cap_stream, cudaStreamNonBlocking));
    DIT_CUDA_OK(cudaStreamBeginCapture(h->cap_stream, cudaStreamCaptureModeRelaxed));
    h->capturing = true;
    s = run_step(h, g, latents_packed, timestep_emb, cond_packed, out_packed, h->cap_stream);
    h->capturing = false;
    cudaGraph_t graph = nullptr;
    cudaError_t ce = cudaStreamEndCapture(h->cap_stream, &graph);
    if (s != DIT_OK) { if (graph) cudaGraphDestroy(graph); return s; }
    DIT_REQUIRE(ce == cudaSuccess && graph != nullptr, DIT_ERR_CUDA, "dit_step_graph: stream capture failed: %s", cudaGetErrorString(ce));
    cudaGraphExec_t exec = nullptr;
    ce = cudaGraphInstantiate(&exec, graph, 0);
    cudaGraphDestroy(graph);
    DIT_REQUIRE(ce == cudaSuccess, DIT_ERR_CUDA, "dit_step_graph: cudaGraphInstantiate failed: %s", cudaGetErrorString(ce));
    if (h->step_graphs.size() >= 8) {   // replace the least recently used graph
      size_t lru = 0;
      for (size_t i = 1; i < h->step_graphs.size(); ++i)
        if (h->step_graphs[i].used < h->step_graphs[lru].used) lru = i;
      cudaGraphExecDestroy(h->step_graphs[lru].exec);
      h->step_graphs.erase(h->step_graphs.begin() + lru);
    }
    h->step_graphs.push_back({key, exec, 0});
    hit = &h->step_graphs.back();
  }
  hit->used = ++h->step_graph_clock;
  DIT_CUDA_OK(cudaGraphLaunch(hit->exec, st));
  return DIT_OK;
}

dit_status dit_step_graph(dit_handle h, const void* latents, const float* timestep_emb, const void* cond_tokens, int32_t n_cond,
                          const int32_t latent_grid[3], void* out, void* stream) {
  return dit_step_varlen_graph(h, latents, timestep_emb, cond_tokens, nullptr, &n_cond, latent_grid, 1, out, stream);
}

}  // extern "C"

// Host-buffer steps: temb goes up on the caller's stream; latents and cond tokens go up on the handle's copy stream, which
// first waits for everything already enqueued on the caller's stream (the previous step still reads the staging area) and
// is joined before patch-embed (run_step, wait_before_embed).
static dit_status upload_inputs(dit_handle h, cudaStream_t st, void* temb_d, const void* temb_h, size_t temb_bytes, void* lat_d,
                                const void* lat_h, size_t lat_bytes, void* cond_d, const void* cond_h, size_t cond_bytes) {
  if (h->copy_stream == nullptr) {
    DIT_CUDA_OK(cudaStreamCreateWithFlags(&h->copy_stream, cudaStreamNonBlocking));
    DIT_CUDA_OK(cudaEventCreateWithFlags(&h->ev_fork, cudaEventDisableTiming));
    DIT_CUDA_OK(cudaEventCreateWithFlags(&h->ev_copied, cudaEventDisableTiming));
  }
  DIT_CUDA_OK(cudaEventRecord(h->ev_fork, st));
  DIT_CUDA_OK(cudaStreamWaitEvent(h->copy_stream, h->ev_fork, 0));
  DIT_CUDA_OK(cudaMemcpyAsync(temb_d, temb_h, temb_bytes, cudaMemcpyHostToDevice, st));
  DIT_CUDA_OK(cudaMemcpyAsync(lat_d, lat_h, lat_bytes, cudaMemcpyHostToDevice, h->copy_stream));
  if (cond_bytes) DIT_CUDA_OK(cudaMemcpyAsync(cond_d, cond_h, cond_bytes, cudaMemcpyHostToDevice, h->copy_stream));
  DIT_CUDA_OK(cudaEventRecord(h->ev_copied, h->copy_stream));
  return DIT_OK;
}

extern "C" {

dit_status dit_step_host(dit_handle h, const void* latents_host, const float* timestep_emb_host,
                         const void* cond_tokens_host, int32_t n_cond, const int32_t latent_grid[3], void* out_host,
                         void* stream) {
  DIT_REQUIRE(h != nullptr, DIT_ERR_INVALID_ARG, "handle is NULL");
  DIT_REQUIRE(latents_host && timestep_emb_host && latent_grid && out_host, DIT_ERR_INVALID_ARG, "NULL tensor argument");
  StepGeom g;
  dit_status s = build_geom(h, 1, nullptr, &n_cond, latent_grid, &g);
  if (s != DIT_OK) return s;
  const dit_config& c = h->cfg;
  const size_t es = esize(c.dtype);
  cudaStream_t st = (cudaStream_t)stream;
  const size_t lat_bytes = (size_t)g.lat_off[1] * es;
  const size_t temb_bytes = (size_t)c.temb_dim * 4;
  const size_t cond_bytes = (size_t)g.cu_cond[1] * c.cond_dim * es;
  char* p = (char*)h->ws.stage_in;
  char* lat_d = p;
  char* temb_d = p + align256(lat_bytes);
  char* cond_d = temb_d + align256(temb_bytes);
  DIT_REQUIRE(cond_bytes == 0 || cond_tokens_host != nullptr, DIT_ERR_INVALID_ARG, "cond tokens announced but cond pointer is NULL");
  s = upload_inputs(h, st, temb_d, timestep_emb_host, temb_bytes, lat_d, latents_host, lat_bytes, cond_d, cond_tokens_host, cond_bytes);
  if (s != DIT_OK) return s;
  h->wait_before_embed = h->ev_copied;
  s = run_step(h, g, lat_d, (const float*)temb_d, cond_d, h->ws.stage_out, st);
  h->wait_before_embed = nullptr;
  if (s != DIT_OK) return s;
  DIT_CUDA_OK(cudaMemcpyAsync(out_host, h->ws.stage_out, lat_bytes, cudaMemcpyDeviceToHost, st));
  return DIT_OK;
}

dit_status dit_step_varlen_host(dit_handle h, const void* latents_packed_host, const float* timestep_emb_host,
                                const void* cond_packed_host, const int32_t* cu_seqlens, const int32_t* n_cond,
                                const int32_t* latent_grids, int32_t n_requests, void* out_packed_host, void* stream) {
  DIT_REQUIRE(h != nullptr, DIT_ERR_INVALID_ARG, "handle is NULL");
  DIT_REQUIRE(latents_packed_host && timestep_emb_host && latent_grids && out_packed_host, DIT_ERR_INVALID_ARG, "NULL tensor argument");
  StepGeom g;
  dit_status s = build_geom(h, n_requests, cu_seqlens, n_cond, latent_grids, &g);
  if (s != DIT_OK) return s;
  const dit_config& c = h->cfg;
  const size_t es = esize(c.dtype);
  cudaStream_t st = (cudaStream_t)stream;
  const int64_t pvC = (int64_t)c.latent_channels * c.patch[0] * c.patch[1] * c.patch[2];
  const size_t lat_bytes = (size_t)g.lat_off[n_requests] * es;
  const size_t temb_bytes = (size_t)n_requests * c.temb_dim * 4;
  const size_t cond_bytes = (size_t)g.cu_cond[n_requests] * c.cond_dim * es;
  // the staging area holds max_tokens patches: image tokens of all requests (a latent has exactly N_r * C * pv elements)
  DIT_REQUIRE(lat_bytes <= (size_t)c.max_tokens * pvC * es, DIT_ERR_WORKSPACE, "packed latents exceed the staging area");
  char* p = (char*)h->ws.stage_in;
  char* lat_d = p;
  char* temb_d = p + align256((size_t)c.max_tokens * pvC * es);
  char* cond_d = temb_d + align256((size_t)c.max_requests * c.temb_dim * 4);
  DIT_REQUIRE(cond_bytes == 0 || cond_packed_host != nullptr, DIT_ERR_INVALID_ARG, "cond tokens announced but cond pointer is NULL");
  s = upload_inputs(h, st, temb_d, timestep_emb_host, temb_bytes, lat_d, latents_packed_host, lat_bytes, cond_d, cond_packed_host,
                    cond_bytes);
  if (s != DIT_OK) return s;
  h->wait_before_embed = h->ev_copied;
  s = run_step(h, g, lat_d, (const float*)temb_d, cond_d, h->ws.stage_out, st);
  h->wait_before_embed = nullptr;
  if (s != DIT_OK) return s;
  DIT_CUDA_OK(cudaMemcpyAsync(out_packed_host, h->ws.stage_out, lat_bytes, cudaMemcpyDeviceToHost, st));
  return DIT_OK;
}

dit_status dit_sample(dit_handle h, const void* latents, const float* timestep_embs, const float* sigmas_host,
                      const void* cond_tokens, int32_t n_cond, const void* uncond_tokens, int32_t n_uncond,
                      float guidance_scale, const int32_t latent_grid[3], int32_t n_steps, int32_t use_graph, void* out,
                      void* stream) {
  DIT_REQUIRE(h != nullptr, DIT_ERR_INVALID_ARG, "handle is NULL");
  DIT_REQUIRE(latents && latent_grid && out && n_steps >= 0, DIT_ERR_INVALID_ARG, "NULL tensor argument or n_steps < 0");
  DIT_REQUIRE(n_steps == 0 || (timestep_embs && sigmas_host), DIT_ERR_INVALID_ARG, "timestep_embs / sigmas is NULL");
  DIT_REQUIRE(latents != out, DIT_ERR_INVALID_ARG, "out may not alias latents");
  const dit_config& c = h->cfg;
  cudaStream_t st = (cudaStream_t)stream;
  const bool guided = uncond_tokens != nullptr;
  StepGeom gc, gu;
  dit_status s = build_geom(h, 1, nullptr, &n_cond, latent_grid, &gc);
  if (s != DIT_OK) return s;
  DIT_REQUIRE(gc.cu_cond[1] == 0 || cond_tokens != nullptr, DIT_ERR_INVALID_ARG, "cond tokens announced but cond pointer is NULL");
  if (guided) {
    s = build_geom(h, 1, nullptr, &n_uncond, latent_grid, &gu);
    if (s != DIT_OK) return s;
  }
  const int64_t n = gc.lat_off[1];
  Workspace& w = h->ws;
  // Guided step as ONE packed pass (R = 2: the unconditional and the conditional request over the same latents, varlen
  // path) when the handle's capacities allow it — max_requests >= 2, both sequences within max_tokens, both cond sets
  // within max_cond_tokens; else two passes per step.  Every weight is then streamed once per step instead of twice.
  StepGeom g2;
  bool packed = false;
  if (guided && c.max_requests >= 2 && (int64_t)gu.cu[1] + gc.cu[1] <= c.max_tokens &&
      (int64_t)gu.cu_cond[1] + gc.cu_cond[1] <= c.max_cond_tokens) {
    const int32_t nc2[2] = {n_uncond, n_cond};
    const int32_t grid2[6] = {latent_grid[0], latent_grid[1], latent_grid[2], latent_grid[0], latent_grid[1], latent_grid[2]};
    s = build_geom(h, 2, nullptr, nc2, grid2, &g2);
    if (s != DIT_OK) return s;
    g2.lat_off.assign(3, 0);   // both requests read the same latents; the conditional one writes `out`
    packed = true;
  }
  // cond and uncond token counts may differ: in joint mode that changes the sequence geometry (rows, RoPE table), which is
  // uploaded outside a capture; a guided trajectory with n_cond != n_uncond in joint mode therefore runs without a graph
  const bool same_geom = !guided || packed || gu.cu == gc.cu;
  auto enqueue = [&](cudaStream_t st) -> dit_status {
    dit_status e = launch_sample_init(c.dtype, latents, w.sample_x, n, st);
    if (e != DIT_OK) return e;
    // timestep MLP + modulation of up to max_sample_steps steps ahead of the steps (they need the embeddings only): the
    // GEMV kernels take 8 rows per pass over the weights, so the modulation weights are streamed once per 8 steps
    const int S = (h->stop_block < 0) ? c.max_sample_steps : 0;
    const int D = c.hidden, L = c.n_blocks;
    const bool dual = c.cond_mode == DIT_COND_JOINT2;
    const int64_t mod_len = (int64_t)L * (dual ? 12 : 6) * D + 2 * D;
    float* const tc1 = w.traj;
    float* const tcc = w.traj + (size_t)S * D;
    float* const tmod = w.traj + (size_t)2 * S * D;
    for (int i = 0; i < n_steps; ++i) {
      const void* x_in = i == 0 ? latents : out;   // x_i rounded to the config dtype was staged in `out` by step i - 1
      const float* temb = timestep_embs + (size_t)i * c.temb_dim;
      const float* mod_pre = nullptr;
      if (S > 0) {
        if (i % S == 0) {
          const int rows = n_steps - i < S ? n_steps - i : S;
          e = launch_gemv(c.dtype, temb, w.gemv_tab + 0, nullptr, 1, D, tc1, D, rows, c.temb_dim, 0, st);
          if (e != DIT_OK) return e;
          e = launch_gemv(c.dtype, tc1, w.gemv_tab + 1, nullptr, 1, D, tcc, D, rows, D, 1, st);
          if (e != DIT_OK) return e;
          e = launch_gemv(c.dtype, tcc, w.gemv_tab + 2, nullptr, dual ? 2 * L + 1 : L + 1, (int)mod_len, tmod, mod_len, rows, D, 1, st);
          if (e != DIT_OK) return e;
        }
        mod_pre = tmod + (size_t)(i % S) * mod_len;
      }
      SampleEpi epi{2, w.sample_x, nullptr, sigmas_host[i + 1] - sigmas_host[i], guidance_scale};
      if (packed) {
        SampleEpi hold{1, nullptr, w.sample_v, 0.f, 0.f};
        epi.v_hold = w.sample_v;
        GuidedPair gp{{uncond_tokens, cond_tokens}, {&hold, &epi}};
        e = run_step(h, g2, x_in, temb, nullptr, out, st, nullptr, &gp, mod_pre);
        if (e != DIT_OK) return e;
        continue;
      }
      if (guided) {
        SampleEpi hold{1, nullptr, w.sample_v, 0.f, 0.f};
        e = run_step(h, gu, x_in, temb, uncond_tokens, out, st, &hold, nullptr, mod_pre);
        if (e != DIT_OK) return e;
        epi.v_hold = w.sample_v;
      }
      e = run_step(h, gc, x_in, temb, cond_tokens, out, st, &epi, nullptr, mod_pre);
      if (e != DIT_OK) return e;
    }
    if (n_steps == 0) return launch_sample_final(c.dtype, w.sample_x, out, n, st);
    return DIT_OK;
  };
  // no graph while per-class profiling is on (event records are not captured) or a debug stop is set
  if (!use_graph || n_steps == 0 || !same_geom || g_prof_mask.load() != 0 || h->stop_block >= 0) return enqueue(st);

  std::vector<uint64_t> key = {(uint64_t)(uintptr_t)latents, (uint64_t)(uintptr_t)timestep_embs, (uint64_t)(uintptr_t)cond_tokens,
                               (uint64_t)(uintptr_t)uncond_tokens, (uint64_t)(uintptr_t)out, (uint64_t)n_cond, (uint64_t)n_uncond,
                               (uint64_t)n_steps, (uint64_t)latent_grid[0], (uint64_t)latent_grid[1], (uint64_t)latent_grid[2]};
  uint32_t gbits;
  memcpy(&gbits, &guidance_scale, 4);
  key.push_back(gbits);
  for (int i = 0; i <= n_steps; ++i) { uint32_t b; memcpy(&b, &sigmas_host[i], 4); key.push_back(b); }
  // host -> device geometry copies and the RoPE table are not part of the graph: they are enqueued here, ahead of the
  // capture or the replay, whenever another call has left a different geometry on the device (else a no-op)
  s = upload_geom(h, packed ? g2 : gc, st);
  if (s != DIT_OK) return s;
  if (h->graph_exec == nullptr || key != h->graph_key) {
    if (h->graph_exec) { cudaGraphExecDestroy(h->graph_exec); h->graph_exec = nullptr; }
    if (h->cap_stream == nullptr) DIT_CUDA_OK(cudaStreamCreateWithFlags(&h->cap_stream, cudaStreamNonBlocking));
    DIT_CUDA_OK(cudaStreamBeginCapture(h->cap_stream, cudaStreamCaptureModeRelaxed));
    h->capturing = true;
    s = enqueue(h->cap_stream);
    h->capturing = false;
    cudaGraph_t graph = nullptr;
    cudaError_t ce = cudaStreamEndCapture(h->cap_stream, &graph);
    if (s != DIT_OK) { if (graph) cudaGraphDestroy(graph); return s; }
    DIT_REQUIRE(ce == cudaSuccess && graph != nullptr, DIT_ERR_CUDA, "dit_sample: stream capture failed: %s", cudaGetErrorString(ce));
    ce = cudaGraphInstantiate(&h->graph_exec, graph, 0);
    cudaGraphDestroy(graph);
    DIT_REQUIRE(ce == cudaSuccess, DIT_ERR_CUDA, "dit_sample: cudaGraphInstantiate failed: %s", cudaGetErrorString(ce));
    h->graph_key = key;
  }
  DIT_CUDA_OK(cudaGraphLaunch(h->graph_exec, st));
  return DIT_OK;
}

dit_status dit_attn_partial(int32_t dtype, const void* q, const void* k, const void* v, int32_t n_q, int32_t n_k,
                            int32_t n_heads, int32_t head_dim, int64_t q_row_stride, int64_t kv_row_stride,
                            float softmax_scale, void* o, float* lse, void* stream) {
  DIT_REQUIRE(dtype == DIT_F32 || dtype == DIT_BF16, DIT_ERR_INVALID_ARG, "dtype %d", dtype);
  DIT_REQUIRE(n_q >= 0 && n_k >= 0 && n_heads > 0, DIT_ERR_INVALID_ARG, "n_q %d n_k %d n_heads %d", n_q, n_k, n_heads);
  DIT_REQUIRE(head_dim == 64 || head_dim == 128, DIT_ERR_UNSUPPORTED, "head_dim %d not in {64,128}", head_dim);
  DIT_REQUIRE(n_q == 0 || (q && o), DIT_ERR_INVALID_ARG, "q / o is NULL");
  DIT_REQUIRE(n_k == 0 || (k && v), DIT_ERR_INVALID_ARG, "k / v is NULL");
  DIT_REQUIRE(q_row_stride >= (int64_t)n_heads * head_dim && kv_row_stride >= (int64_t)n_heads * head_dim,
              DIT_ERR_INVALID_ARG, "row strides smaller than H*d");
  AttnArgs a;
  a.q = q; a.k = k; a.v = v; a.q_stride = q_row_stride; a.kv_stride = kv_row_stride;
  a.o = o; a.o_stride = (int64_t)n_heads * head_dim; a.lse = lse;
  a.cu_q = a.cu_k = nullptr; a.cu_q_host = a.cu_k_host = nullptr;
  a.R = 1; a.n_q = n_q; a.n_k = n_k; a.H = n_heads; a.d = head_dim; a.scale = softmax_scale; a.shard = 0; a.n_shards = 1;
  return attention(dtype, a, (cudaStream_t)stream);
}

dit_status dit_attn_merge(int32_t dtype, const void* const* o_partials, const float* const* lses, int32_t P, int32_t n_q,
                          int32_t n_heads, int32_t head_dim, void* o, float* lse_out, void* stream) {
  DIT_REQUIRE(dtype == DIT_F32 || dtype == DIT_BF16, DIT_ERR_INVALID_ARG, "dtype %d", dtype);
  DIT_REQUIRE(P >= 1 && P <= 8, DIT_ERR_INVALID_ARG, "P=%d not in 1..8", P);
  DIT_REQUIRE(o_partials && lses && (n_q == 0 || o), DIT_ERR_INVALID_ARG, "NULL argument");
  for (int p = 0; p < P; ++p) DIT_REQUIRE(n_q == 0 || (o_partials[p] && lses[p]), DIT_ERR_INVALID_ARG, "partial %d is NULL", p);
  return launch_merge(dtype, o_partials, lses, P, (int64_t)n_q * n_heads, head_dim, o, lse_out, (cudaStream_t)stream);
}

dit_status dit_linear(int32_t dtype, int32_t epilogue, const void* A, int64_t lda, const void* W, const void* bias,
                      void* out, int64_t ldo, int32_t M, int32_t N, int32_t K, void* stream) {
  DIT_REQUIRE(dtype == DIT_F32 || dtype == DIT_BF16, DIT_ERR_INVALID_ARG, "dtype %d", dtype);
  DIT_REQUIRE(epilogue >= DIT_EPI_BIAS && epilogue <= DIT_EPI_BIAS_F32, DIT_ERR_INVALID_ARG, "epilogue %d", epilogue);
  DIT_REQUIRE(M >= 0 && N > 0 && K > 0 && lda >= K && ldo >= N, DIT_ERR_INVALID_ARG, "bad GEMM shape M=%d N=%d K=%d lda=%lld ldo=%lld",
              M, N, K, (long long)lda, (long long)ldo);
  DIT_REQUIRE(M == 0 || (A && W && out), DIT_ERR_INVALID_ARG, "NULL argument");
  return gemm(dtype, epilogue, A, lda, W, bias, out, ldo, M, N, K, (cudaStream_t)stream);
}

dit_status dit_linear_residual(int32_t dtype, const void* A, int64_t lda, const void* W, const void* bias, float* x,
                               int64_t ldx, const float* gate, int64_t gate_stride, const int32_t* cu_seqlens_dev,
                               int32_t n_requests, int32_t M, int32_t N, int32_t K, void* stream) {
  DIT_REQUIRE(dtype == DIT_F32 || dtype == DIT_BF16, DIT_ERR_INVALID_ARG, "dtype %d", dtype);
  DIT_REQUIRE(M >= 0 && N > 0 && K > 0 && lda >= K && ldx >= N, DIT_ERR_INVALID_ARG, "bad GEMM shape M=%d N=%d K=%d lda=%lld ldx=%lld",
              M, N, K, (long long)lda, (long long)ldx);
  DIT_REQUIRE(M == 0 || (A && W && x), DIT_ERR_INVALID_ARG, "NULL argument");
  DIT_REQUIRE(n_requests >= 1 && n_requests <= 64 && (n_requests == 1 || cu_seqlens_dev), DIT_ERR_INVALID_ARG,
              "n_requests %d (cu_seqlens required when > 1)", n_requests);
  return gemm_residual(dtype, A, lda, W, bias, x, ldx, gate, gate_stride, cu_seqlens_dev, n_requests, M, N, K,
                       (cudaStream_t)stream);
}

dit_status dit_linear_qkv(int32_t dtype, const void* A, int64_t lda, const void* W, const void* bias, void* out,
                          int64_t ldo, const void* g_q, const void* g_k, float rms_eps, const float* rope_cos,
                          const float* rope_sin, int32_t hidden, int32_t M, int32_t K, void* stream) {
  DIT_REQUIRE(M >= 0 && K > 0 && hidden > 0 && lda >= K && ldo >= 3 * (int64_t)hidden, DIT_ERR_INVALID_ARG,
              "bad QKV shape M=%d K=%d hidden=%d lda=%lld ldo=%lld", M, K, hidden, (long long)lda, (long long)ldo);
  DIT_REQUIRE(M == 0 || (A && W && out), DIT_ERR_INVALID_ARG, "NULL argument");
  DIT_REQUIRE((rope_cos == nullptr) == (rope_sin == nullptr), DIT_ERR_INVALID_ARG, "rope_cos / rope_sin must both be given");
  DIT_REQUIRE(dtype == DIT_BF16 && hidden % 128 == 0 &&
                  gemm_tc_supported(DIT_EPI_BIAS, A, lda, W, out, ldo, M > 0 ? M : 1, 3 * hidden, K),
              DIT_ERR_UNSUPPORTED, "dit_linear_qkv: bf16, head_dim 128, 16-byte aligned operands, sm_100 only");
  return launch_gemm_tc_qkv(A, lda, W, bias, out, ldo, g_q, g_k, rms_eps, rope_cos, rope_sin, hidden, 2 * hidden, M,
                            3 * hidden, K, (cudaStream_t)stream);
}

dit_status dit_linear_swiglu(int32_t dtype, const void* A, int64_t lda, const void* W1, const void* b1, const void* W3,
                             const void* b3, void* out, int64_t ldo, void* tmp, int32_t M, int32_t N, int32_t K, void* stream) {
  DIT_REQUIRE(dtype == DIT_F32 || dtype == DIT_BF16, DIT_ERR_INVALID_ARG, "dtype %d", dtype);
  DIT_REQUIRE(M >= 0 && N > 0 && K > 0 && lda >= K && ldo >= N, DIT_ERR_INVALID_ARG, "bad GEMM shape M=%d N=%d K=%d lda=%lld ldo=%lld",
              M, N, K, (long long)lda, (long long)ldo);
  DIT_REQUIRE(M == 0 || (A && W1 && W3 && out), DIT_ERR_INVALID_ARG, "NULL argument");
  cudaStream_t st = (cudaStream_t)stream;
  if (M == 0) return DIT_OK;
  if (dtype == DIT_BF16) {
    DIT_REQUIRE(gemm_tc_supported(DIT_EPI_BIAS, A, lda, W1, out, ldo, M, N, K) && !((uintptr_t)W3 & 15), DIT_ERR_UNSUPPORTED,
                "dit_linear_swiglu (bf16): K, N, lda, ldo multiples of 8, 16-byte aligned pointers, sm_100 only");
    return launch_gemm_tc_swiglu(A, lda, W1, b1, W3, b3, out, ldo, M, N, K, st);
  }
  DIT_REQUIRE(tmp != nullptr && ldo == N, DIT_ERR_INVALID_ARG, "dit_linear_swiglu (fp32): tmp [M, N] is required and out must be contiguous");
  dit_status s = gemm(dtype, DIT_EPI_BIAS, A, lda, W1, b1, out, ldo, M, N, K, st);
  if (s != DIT_OK) return s;
  s = gemm(dtype, DIT_EPI_BIAS, A, lda, W3, b3, tmp, N, M, N, K, st);
  if (s != DIT_OK) return s;
  return launch_silu_mul(dtype, out, tmp, (int64_t)M * N, st);
}

dit_status dit_adaln(int32_t dtype, float* x, const void* h, const float* gate, const float* shift, const float* scale,
                     int64_t mod_stride, const int32_t* cu_seqlens_dev, int32_t n_requests, void* y, int32_t T, int32_t D,
                     float eps, void* stream) {
  DIT_REQUIRE(dtype == DIT_F32 || dtype == DIT_BF16, DIT_ERR_INVALID_ARG, "dtype %d", dtype);
  DIT_REQUIRE(T >= 0 && D > 0 && n_requests >= 1 && n_requests <= 64, DIT_ERR_INVALID_ARG, "T=%d D=%d R=%d", T, D, n_requests);
  DIT_REQUIRE(T == 0 || (x && y), DIT_ERR_INVALID_ARG, "x / y is NULL");
  DIT_REQUIRE(n_requests == 1 || cu_seqlens_dev, DIT_ERR_INVALID_ARG, "cu_seqlens required for n_requests > 1");
  return launch_adaln(dtype, x, h, gate, shift, scale, mod_stride, cu_seqlens_dev, n_requests, y, T, D, eps,
                      (cudaStream_t)stream);
}

dit_status dit_gemv(int32_t dtype, const float* in, const void* W, const void* b, float* out, int32_t R, int32_t N,
                    int32_t K, int32_t silu_input, void* stream) {
  DIT_REQUIRE(dtype == DIT_F32 || dtype == DIT_BF16, DIT_ERR_INVALID_ARG, "dtype %d", dtype);
  DIT_REQUIRE(R >= 1 && N >= 1 && K >= 8 && in && W && out, DIT_ERR_INVALID_ARG, "bad GEMV arguments");
  // one matrix: its descriptor travels as a kernel parameter (no device allocation, no copy)
  GemvBatch tb = {W, b, N, 0, 0, 0};
  dit_status s = launch_gemv(dtype, in, nullptr, &tb, 1, N, out, N, R, K, silu_input, (cudaStream_t)stream);
  return s;
}

dit_status dit_qknorm_rope(int32_t dtype, void* qkv, int64_t row_stride, int32_t T, int32_t n_heads, int32_t head_dim,
                           int32_t n_tensors, const void* gq, const void* gk, float eps, const float* rope_cos,
                           const float* rope_sin, void* stream) {
  DIT_REQUIRE(dtype == DIT_F32 || dtype == DIT_BF16, DIT_ERR_INVALID_ARG, "dtype %d", dtype);
  DIT_REQUIRE(n_tensors == 1 || n_tensors == 2, DIT_ERR_INVALID_ARG, "n_tensors %d", n_tensors);
  DIT_REQUIRE((rope_cos == nullptr) == (rope_sin == nullptr), DIT_ERR_INVALID_ARG, "rope_cos / rope_sin must both be given");
  DIT_REQUIRE(T == 0 || qkv, DIT_ERR_INVALID_ARG, "qkv is NULL");
  return launch_qknorm_rope(dtype, qkv, row_stride, T, n_heads, head_dim, n_tensors, gq, gk, eps, rope_cos, rope_sin,
                            (cudaStream_t)stream);
}

dit_status dit_debug_stop_after(dit_handle h, int32_t block, int32_t stage) {
  DIT_REQUIRE(h != nullptr, DIT_ERR_INVALID_ARG, "handle is NULL");
  h->stop_block = block;
  h->stop_stage = block < 0 ? -1 : stage;
  return DIT_OK;
}

dit_status dit_get_tap(dit_handle h, int32_t tap, void* dst, size_t bytes, void* stream) {
  DIT_REQUIRE(h != nullptr && dst != nullptr, DIT_ERR_INVALID_ARG, "NULL argument");
  const Workspace& w = h->ws;
  const void* src = nullptr;
  switch (tap) {
    case DIT_TAP_X: src = w.x; break;
    case DIT_TAP_Y: src = w.y; break;
    case DIT_TAP_QKV: src = w.qkv; break;
    case DIT_TAP_O: src = w.o; break;
    case DIT_TAP_U: src = w.u; break;
    case DIT_TAP_C: src = w.c; break;
    case DIT_TAP_MOD: src = w.mod; break;
    case DIT_TAP_TOK: src = w.tok; break;
    default: DIT_REQUIRE(false, DIT_ERR_INVALID_ARG, "unknown tap %d", tap);
  }
  DIT_CUDA_OK(cudaMemcpyAsync(dst, src, bytes, cudaMemcpyDeviceToDevice, (cudaStream_t)stream));
  return DIT_OK;
}

dit_status dit_profile_begin(int32_t class_mask) {
  DIT_REQUIRE(class_mask >= 0 && class_mask < (1 << DIT_KC_COUNT), DIT_ERR_INVALID_ARG, "class_mask 0x%x", class_mask);
  std::lock_guard<std::mutex> lk(g_prof_mu);
  for (auto& r : g_prof_recs) { g_prof_pool.push_back(r.a); g_prof_pool.push_back(r.b); }
  g_prof_recs.clear();
  for (int i = 0; i < DIT_KC_COUNT; ++i) g_prof_counts[i] = 0;
  g_prof_mask = class_mask;
  return DIT_OK;
}

dit_status dit_profile_end(float* ms_per_class, int32_t* launches_per_class) {
  DIT_REQUIRE(ms_per_class && launches_per_class, DIT_ERR_INVALID_ARG, "NULL argument");
  g_prof_mask = 0;
  std::lock_guard<std::mutex> lk(g_prof_mu);
  for (int i = 0; i < DIT_KC_COUNT; ++i) { ms_per_class[i] = 0.f; launches_per_class[i] = g_prof_counts[i]; }
  for (auto& r : g_prof_recs) {
    if (r.open) { g_prof_pool.push_back(r.a); g_prof_pool.push_back(r.b); continue; }   // a launch that failed mid-way
    DIT_CUDA_OK(cudaEventSynchronize(r.b));
    float ms = 0.f;
    DIT_CUDA_OK(cudaEventElapsedTime(&ms, r.a, r.b));
    ms_per_class[r.cls] += ms;
    g_prof_pool.push_back(r.a); g_prof_pool.push_back(r.b);
  }
  g_prof_recs.clear();
  return DIT_OK;
}

const char* dit_last_error(dit_handle) { return get_error(); }
int32_t dit_kernel_launches(void) { return g_launches.load(); }
int32_t dit_fallback_launches(void) { return g_fallback_launches.load(); }

void dit_free(dit_handle h) {
  if (!h) return;
  if (h->graph_exec) cudaGraphExecDestroy(h->graph_exec);
  for (auto& sg : h->step_graphs) cudaGraphExecDestroy(sg.exec);
  if (h->cap_stream) cudaStreamDestroy(h->cap_stream);
  if (h->copy_stream) cudaStreamDestroy(h->copy_stream);
  if (h->ev_fork) cudaEventDestroy(h->ev_fork);
  if (h->ev_copied) cudaEventDestroy(h->ev_copied);
  delete[] h->blocks;
  delete h;
}

}  // extern "C"
