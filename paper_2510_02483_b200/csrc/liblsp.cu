// liblsp -- host side of the C ABI declared in include/lsp.h: argument checks, buffer carving and the
// kernel sequence of one Llama decoder layer forward / backward.
// Every step of the path runs in the kernels of gemm.cuh / attn.cuh / norm.cuh; nothing is computed on the host
// except the RoPE angle table (fp64, once, at lsp_create).
#include "../../include/lsp.h"

#include <math.h>
#include <stdarg.h>
#include <string.h>

#include <mutex>
#include <new>
#include <vector>

#include "attn.cuh"
#include "attn_tc.cuh"
#include "gemm.cuh"
#include "norm.cuh"
#include "optim.cuh"
#include "head.cuh"

using namespace lsp;

namespace {

constexpr size_t ALIGN = 256;
inline size_t align_up(size_t v) { return (v + ALIGN - 1) / ALIGN * ALIGN; }

// Byte offsets inside `saved` and `ws` (all 256-byte aligned).
struct SavedLayout {
  size_t a32, xn, rstd1, qkv16, o32, o16, lse, an, rstd2, g16, u16, h;
  size_t wqkv16, wo16, wgu16, wd16;      // fp16 copies of the bf16 weights (made by the forward, reused by the backward)
  size_t total;
};
struct WsLayout {
  size_t in16, dgu, dn32, da32, da16, dO16, dvec, dqkv16, dgpart, q16, k16, v16, total;
};
// fp16 operand copies of one layer's projection weights (lsp_weight_cache_bytes): [Wq; Wk; Wv] | Wo | [Wg; Wu] | Wd.
// The same four blocks exist inside `saved` for calls that pass no cache.
struct WCacheLayout { size_t wqkv16, wo16, wgu16, wd16, total; };

}  // namespace

// softmax scale and RoPE frequencies follow the logical head width (zero-padded heads: head_dim_logical < head_dim)
// weight of the residual branch: 1 unless the descriptor says otherwise (tensor-parallel ranks other than the first: 0)
static inline float residual_scale(const lsp_layer_desc& d) { return d.residual_scale_set ? d.residual_scale : 1.0f; }
static inline int logical_head_dim(const lsp_layer_desc& d) { return d.head_dim_logical > 0 ? d.head_dim_logical : d.head_dim; }

// Pipeline stages (for launch counting and the optional per-stage device timing of lsp_timing_*).
enum Stage : int {
  ST_CAST = 0, ST_NORM_FWD, ST_QKV, ST_ATTN_FWD, ST_OPROJ, ST_GATEUP, ST_DOWN,
  ST_WGRAD_DOWN, ST_DGRAD_DOWN, ST_WGRAD_GATEUP, ST_DGRAD_GATEUP, ST_NORM_BWD,
  ST_WGRAD_O, ST_DGRAD_O, ST_DVEC, ST_ATTN_BWD, ST_WGRAD_QKV, ST_DGRAD_QKV, ST_EMBED, ST_ATTN_BWD_DQ, ST_ADAMW, ST_HEAD_GEMM, ST_CE, ST_EMBED_BWD, ST_COUNT
};
static const char* const STAGE_NAMES[ST_COUNT] = {
  "cast", "rmsnorm_fwd", "gemm_qkv_rope", "attn_fwd", "gemm_oproj_res", "gemm_gateup_swiglu", "gemm_down_res",
  "wgrad_down", "dgrad_down_swiglu_bwd", "wgrad_gateup", "dgrad_gateup", "rmsnorm_bwd",
  "wgrad_oproj", "dgrad_oproj", "attn_dvec", "attn_bwd", "wgrad_qkv", "dgrad_qkv", "embed_gather", "attn_bwd_dq", "adamw", "head_gemm", "cross_entropy", "embed_bwd"};

struct TimingRec { int stage; cudaEvent_t beg, end; };

struct lsp_ctx {
  long long launches;                 // kernels launched through this context (cumulative)
  int timing_on;
  std::vector<TimingRec>* recs;       // pre-created event pairs
  int recs_used;
  lsp_layer_desc d;
  int device, num_sms;
  int T, Nq, Nkv, Nqkv, G;
  float2* rope;         // [seq, head_dim/2] (cos, sin), device
  float* sk_partial;             // stream-K partial accumulators, [num_sms/2][256 x 256] fp32 (device)
  unsigned int* sk_flags;        // [num_sms/2][2] publication epochs (device, zeroed at create)
  unsigned int gemm_seq;         // launches so far: epoch of the next stream-K launch
  unsigned int* attn_sched;      // work-item counters of the persistent attention kernels (device, zero between launches)
  float* opt_partial;            // per-block partial sums of the gradient-norm pass (device)
  cudaStream_t s_in, s_out;      // copy streams of lsp_layer_step_host (H2D / D2H overlap the compute stream)
  cudaEvent_t ev[6];             // start, x in, dy in, fwd done, bwd done, copies out
  cudaEvent_t pev[2][6];         // lsp_layer_step_host_async, per call parity: x in, dy in, fwd done, bwd done, y out, dx out
  long long host_seq;            // number of async host steps issued
  int* doc_start; int* doc_end;  // [T] each (device): packed-sequence bounds per token (lsp_set_packed_sequences)
  int doc_on;
  const void* prev_y_dev; const void* prev_dx_dev;   // device result buffers of the previous async step
  int norm_blocks;      // persistent grid of the RMSNorm backward
  SavedLayout sv;
  WsLayout ws;
  WCacheLayout wc;
  unsigned long long* overflow;  // device counter: values the fp16 operand casts clamped or found non-finite (lsp_overflow_count)
  char err[512];
};

namespace {

lsp_status fail(lsp_ctx* c, lsp_status s, const char* fmt, ...) {
  if (c) {
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(c->err, sizeof(c->err), fmt, ap);
    va_end(ap);
  }
  return s;
}

#define LSP_CUDA(call)                                                                                   \
  do {                                                                                                   \
    cudaError_t e__ = (call);                                                                            \
    if (e__ != cudaSuccess) return fail(ctx, LSP_ECUDA, "%s failed: %s", #call, cudaGetErrorString(e__)); \
  } while (0)
// One pipeline stage: `call` launches `n` kernels on stream `st`.
#define LSP_STAGE(id, n, call)                                                                            \
  do {                                                                                                   \
    TimingRec* r__ = stage_begin(ctx, id, st);                                                           \
    cudaError_t e__ = (call);                                                                            \
    if (r__) cudaEventRecord(r__->end, st);                                                              \
    ctx->launches += (n);                                                                                \
    if (e__ != cudaSuccess) return fail(ctx, LSP_ECUDA, "%s: %s", STAGE_NAMES[id], cudaGetErrorString(e__)); \
  } while (0)
#define LSP_TRY(call)                    \
  do {                                   \
    lsp_status s__ = (call);             \
    if (s__ != LSP_OK) return s__;       \
  } while (0)

inline TimingRec* stage_begin(lsp_ctx* c, int id, cudaStream_t st) {
  if (!c->timing_on || !c->recs || c->recs_used >= static_cast<int>(c->recs->size())) return nullptr;
  TimingRec* r = &(*c->recs)[c->recs_used++];
  r->stage = id;
  cudaEventRecord(r->beg, st);
  return r;
}

inline bool aligned(const void* p, size_t a) { return (reinterpret_cast<uintptr_t>(p) % a) == 0; }

void plan_layout(lsp_ctx* c) {
  const size_t T = c->T, H = c->d.hidden, F = c->d.ffn, Nq = c->Nq, Nqkv = c->Nqkv;
  const size_t BnqS = static_cast<size_t>(c->d.batch) * c->d.n_q_heads * c->d.seq;
  size_t o = 0;
  auto take = [&](size_t bytes) { size_t r = o; o += align_up(bytes); return r; };
  SavedLayout& s = c->sv;
  s.a32 = take(T * H * 4);
  s.xn = take(T * H * 2);
  s.rstd1 = take(T * 4);
  s.qkv16 = take(T * Nqkv * 2);
  s.o32 = take(T * Nq * 4);
  s.o16 = take(T * Nq * 2);
  s.lse = take(BnqS * 4);
  s.an = take(T * H * 2);
  s.rstd2 = take(T * 4);
  s.g16 = take(T * F * 2);
  s.u16 = take(T * F * 2);
  s.h = take(T * F * 2);
  s.wqkv16 = take(Nqkv * H * 2);          // [Wq; Wk; Wv] stacked: one [Nqkv, H] matrix
  s.wo16 = take(H * Nq * 2);
  s.wgu16 = take(2 * F * H * 2);          // [Wg; Wu] stacked: one [2F, H] matrix
  s.wd16 = take(H * F * 2);
  s.total = o;

  o = 0;
  WsLayout& w = c->ws;
  w.in16 = take(T * H * 2);
  w.dgu = take(T * 2 * F * 2);
  w.dn32 = take(T * H * 4);
  w.da32 = take(T * H * 4);
  w.da16 = take(T * H * 2);
  w.dO16 = take(T * Nq * 2);
  w.dvec = take(BnqS * 16);              // four partial sums per (batch, head, position) at head_dim 128
  w.dqkv16 = take(T * Nqkv * 2);
  w.dgpart = take(static_cast<size_t>(c->norm_blocks) * 2 * H * 4);      // one row per (CTA, row group) of rmsnorm_bwd_kernel
  w.q16 = take(T * Nq * 2);
  w.k16 = take(T * c->Nkv * 2);
  w.v16 = take(T * c->Nkv * 2);
  w.total = o;

  o = 0;
  WCacheLayout& k = c->wc;
  k.wqkv16 = take(Nqkv * H * 2);
  k.wo16 = take(H * Nq * 2);
  k.wgu16 = take(2 * F * H * 2);
  k.wd16 = take(H * F * 2);
  k.total = o;
}

// Makes the context's device current for the duration of an entry point and restores the caller's on exit (several
// contexts on several devices may live in one process); publishes the device to the per-device launch setup (DeviceOnce).
struct DeviceGuard {
  int prev = -1, prev_tls;
  bool ok = true;
  explicit DeviceGuard(int dev) : prev_tls(tls_device()) {
    if (cudaGetDevice(&prev) != cudaSuccess) { prev = -1; ok = false; return; }
    if (prev != dev && cudaSetDevice(dev) != cudaSuccess) { ok = false; return; }
    tls_device() = dev;
  }
  ~DeviceGuard() {
    tls_device() = prev_tls;
    int cur = -1;
    if (prev >= 0 && cudaGetDevice(&cur) == cudaSuccess && cur != prev) cudaSetDevice(prev);
  }
};
#define LSP_ENTER(ctx)                                                                     \
  DeviceGuard guard__((ctx)->device);                                                      \
  if (!guard__.ok) return fail((ctx), LSP_ECUDA, "cannot make device %d current", (ctx)->device)

template <typename T> T* at(void* base, size_t off) { return reinterpret_cast<T*>(static_cast<uint8_t*>(base) + off); }
template <typename T> const T* at(const void* base, size_t off) {
  return reinterpret_cast<const T*>(static_cast<const uint8_t*>(base) + off);
}

// ------------------------------------------------------------------------------------------- norm dispatch
template <typename XT>
cudaError_t norm_fwd_t(const lsp_ctx* c, const void* x, const void* g, __half* xn, float* rstd, cudaStream_t st) {
  const int H = c->d.hidden, nv = (H / 4 + NORM_THREADS - 1) / NORM_THREADS;
  const XT* xp = static_cast<const XT*>(x);
  const __nv_bfloat16* gp = static_cast<const __nv_bfloat16*>(g);
#define LSP_NF(NV) case NV: return launch_kernel(rmsnorm_fwd_kernel<XT, NV>, dim3(c->T), dim3(NORM_THREADS), 0, st, xp, gp, xn, rstd, H, c->d.rms_eps);
  switch (nv) { LSP_NF(1) LSP_NF(2) LSP_NF(3) LSP_NF(4) LSP_NF(5) LSP_NF(6) LSP_NF(7) LSP_NF(8) default: return cudaErrorInvalidValue; }
#undef LSP_NF
}
cudaError_t norm_fwd(const lsp_ctx* c, int dt, const void* x, const void* g, __half* xn, float* rstd, cudaStream_t st) {
  return dt == LSP_F32 ? norm_fwd_t<float>(c, x, g, xn, rstd, st) : norm_fwd_t<__nv_bfloat16>(c, x, g, xn, rstd, st);
}

template <typename XT, typename RT>
cudaError_t norm_bwd_t(const lsp_ctx* c, const void* x, const float* rstd, const void* g, const float* dxn, const void* dres,
                       float* dx, __half* dx16, float* dg_part, float* dg, int dg_accumulate, cudaStream_t st) {
  const int H = c->d.hidden;
  // two row groups of 128 threads while a row is at most 8 float4 per thread (H <= 4096), else one group of 256
  const int G = (H / 4 + 127) / 128 <= 8 ? 2 : 1;
  const int gt = NORMB_CONSUMERS / G, nv = (H / 4 + gt - 1) / gt;
  const XT* xp = static_cast<const XT*>(x);
  const RT* rp = static_cast<const RT*>(dres);
  const __nv_bfloat16* gp = static_cast<const __nv_bfloat16*>(g);
  const int nb = c->norm_blocks < c->T ? c->norm_blocks : c->T;
  const size_t stage_bytes = static_cast<size_t>(H) * (sizeof(XT) + 4 + (dres ? sizeof(RT) : 0));
  int stages = static_cast<int>(NORMB_SMEM_BUDGET / stage_bytes);
  if (stages > NORMB_MAX_STAGES) stages = NORMB_MAX_STAGES;
  if (stages < 2) return cudaErrorInvalidValue;
  const size_t smem = stages * stage_bytes;
  cudaError_t launch_err = cudaSuccess;
#define LSP_NB(NV, GG) case NV: { \
    auto kern = rmsnorm_bwd_kernel<XT, RT, NV, GG>; \
    static DeviceOnce once; \
    if (once.need()) { cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, NORMB_SMEM_BUDGET); if (e != cudaSuccess) return e; once.done(); } \
    launch_err = launch_kernel(kern, dim3(nb), dim3(NORMB_THREADS), smem, st, xp, rstd, gp, dxn, rp, dx, dx16, dg_part, c->T, H, stages, residual_scale(c->d), c->overflow); } break;
  if (G == 2) {
    switch (nv) { LSP_NB(1, 2) LSP_NB(2, 2) LSP_NB(3, 2) LSP_NB(4, 2) LSP_NB(5, 2) LSP_NB(6, 2) LSP_NB(7, 2) LSP_NB(8, 2) default: return cudaErrorInvalidValue; }
  } else {
    switch (nv) { LSP_NB(5, 1) LSP_NB(6, 1) LSP_NB(7, 1) LSP_NB(8, 1) default: return cudaErrorInvalidValue; }
  }
#undef LSP_NB
  if (launch_err != cudaSuccess) return launch_err;
  return launch_kernel(colsum_kernel, dim3((H + 31) / 32), dim3(256), 0, st, static_cast<const float*>(dg_part), dg, nb * G, H, dg_accumulate);
}
// x: forward input of the norm (XT = x_dt); dres: incoming residual gradient (RT = r_dt)
cudaError_t norm_bwd(const lsp_ctx* c, int x_dt, int r_dt, const void* x, const float* rstd, const void* g, const float* dxn,
                     const void* dres, float* dx, __half* dx16, float* dg_part, float* dg, int acc, cudaStream_t st) {
  if (x_dt == LSP_F32)
    return r_dt == LSP_F32 ? norm_bwd_t<float, float>(c, x, rstd, g, dxn, dres, dx, dx16, dg_part, dg, acc, st)
                           : norm_bwd_t<float, __nv_bfloat16>(c, x, rstd, g, dxn, dres, dx, dx16, dg_part, dg, acc, st);
  return r_dt == LSP_F32 ? norm_bwd_t<__nv_bfloat16, float>(c, x, rstd, g, dxn, dres, dx, dx16, dg_part, dg, acc, st)
                         : norm_bwd_t<__nv_bfloat16, __nv_bfloat16>(c, x, rstd, g, dxn, dres, dx, dx16, dg_part, dg, acc, st);
}

cudaError_t cast_f32_f16(const float* in, __half* out, long long n, int sms, unsigned long long* counter, cudaStream_t st) {
  const long long n8 = n / 8;
  long long blocks = (n8 + 255) / 256;
  if (blocks > sms * 16LL) blocks = sms * 16LL;
  if (blocks < 1) blocks = 1;
  return launch_kernel(cast_f32_f16_kernel, dim3(static_cast<unsigned>(blocks)), dim3(256), 0, st, in, out, n8, counter);
}
cudaError_t cast_bf16_f16(const __nv_bfloat16* in, __half* out, long long n, int sms, unsigned long long* counter, cudaStream_t st) {
  const long long n8 = n / 8;
  long long blocks = (n8 + 255) / 256;
  if (blocks > sms * 16LL) blocks = sms * 16LL;
  if (blocks < 1) blocks = 1;
  return launch_kernel(cast_bf16_f16_kernel, dim3(static_cast<unsigned>(blocks)), dim3(256), 0, st, in, out, n8, counter);
}

// up to CAST_MAX_SEGS bf16 -> fp16 weight casts in one launch (element counts are multiples of 8)
cudaError_t cast_weights(const lsp_ctx* c, int nseg, const void* const* src, __half* const* dst, const long long* n, cudaStream_t st,
                         unsigned perm_mask = 0) {
  CastSegs segs;
  segs.nseg = nseg;
  segs.perm_mask = perm_mask; segs.perm_d = c->d.head_dim; segs.row_units = c->d.hidden / 8;
  segs.counter = c->overflow;
  segs.start[0] = 0;
  for (int i = 0; i < CAST_MAX_SEGS; ++i) {
    segs.src[i] = i < nseg ? static_cast<const __nv_bfloat16*>(src[i]) : nullptr;
    segs.dst[i] = i < nseg ? dst[i] : nullptr;
    segs.start[i + 1] = segs.start[i] + (i < nseg ? n[i] / 8 : 0);
  }
  long long blocks = (segs.start[nseg] + 255) / 256;
  if (blocks > c->num_sms * 16LL) blocks = c->num_sms * 16LL;
  if (blocks < 1) blocks = 1;
  return launch_kernel(cast_multi_bf16_f16_kernel, dim3(static_cast<unsigned>(blocks)), dim3(256), 0, st, segs);
}

}  // namespace

// ------------------------------------------------------------------------------------------- GEMM call sites
namespace {

constexpr int BN_MAIN = 256;

using EpiF32 = EpiStore<DT_F32, DT_F32, false>;
inline EpiF32 epi_f32(float* out, long long ld) {
  EpiF32 e;
  e.out[0] = out; e.out[1] = e.out[2] = nullptr;
  e.split1 = e.split2 = 0x7fffffff; e.ld = ld; e.res = nullptr; e.alpha = 1.0f;
  return e;
}

// weight-gradient output: overwrite, or += when the context was created with wgrad_accumulate = 1
inline EpiF32 epi_wgrad(const lsp_ctx* c, void* out, long long ld) {
  EpiF32 e = epi_f32(static_cast<float*>(out), ld);
  e.accumulate = c->d.wgrad_accumulate;
  return e;
}

template <bool A_MN, bool B_MN, class Epi>
cudaError_t gemm1(const lsp_ctx* c, int M, int N, int K, const Operand& a, const Operand& b, const Epi& epi, cudaStream_t st) {
  const int ks[1] = {K};
  lsp_ctx* mc = const_cast<lsp_ctx*>(c);
  const GemmSKRes sk{c->sk_partial, c->sk_flags, ++mc->gemm_seq};
  return gemm_run<BN_MAIN, A_MN, B_MN, Epi>(M, N, 1, &a, &b, ks, epi, c->num_sms, st, &sk);
}

// out[T,H] fp32 = res + A[T,K] . W[H,K]^T   (O-proj and down-proj forward with the residual epilogue; F4, F7)
cudaError_t gemm_fwd_residual(const lsp_ctx* c, const __half* A, int K, const __half* W, int res_dt, const void* res,
                              float* out, cudaStream_t st) {
  const int T = c->T, H = c->d.hidden;
  const Operand a{A, K, false}, b{W, K, false};
  if (res_dt == LSP_F32) {
    EpiStore<DT_F32, DT_F32, true> e;
    e.out[0] = out; e.out[1] = e.out[2] = nullptr; e.split1 = e.split2 = 0x7fffffff; e.ld = H; e.res = res; e.alpha = 1.0f;
    e.res_scale = residual_scale(c->d);
    return gemm1<false, false>(c, T, H, K, a, b, e, st);
  }
  EpiStore<DT_F32, DT_BF16, true> e;
  e.out[0] = out; e.out[1] = e.out[2] = nullptr; e.split1 = e.split2 = 0x7fffffff; e.ld = H; e.res = res; e.alpha = 1.0f;
  e.res_scale = residual_scale(c->d);
  return gemm1<false, false>(c, T, H, K, a, b, e, st);
}

// fp16 operand copies of the projection weights: the caller's cache (lsp_layer_weights.f16_cache, filled by
// lsp_layer_prepare_weights or by lsp_adamw_step's weight_f16 outputs) or the blocks inside `saved` that every forward
// call refreshes itself.
struct W16 { __half *wqkv, *wo, *wgu, *wd; bool cached; };
inline W16 w16_of(const lsp_ctx* c, const lsp_layer_weights* w, const void* saved) {
  if (w->f16_cache) {
    void* k = const_cast<void*>(w->f16_cache);
    return W16{at<__half>(k, c->wc.wqkv16), at<__half>(k, c->wc.wo16), at<__half>(k, c->wc.wgu16), at<__half>(k, c->wc.wd16), true};
  }
  void* k = const_cast<void*>(saved);
  return W16{at<__half>(k, c->sv.wqkv16), at<__half>(k, c->sv.wo16), at<__half>(k, c->sv.wgu16), at<__half>(k, c->sv.wd16), false};
}
lsp_status cast_attn_weights(lsp_ctx* ctx, const lsp_layer_weights* w, const W16& k, cudaStream_t st) {
  const lsp_layer_desc& d = ctx->d;
  const long long H = d.hidden, Nq = ctx->Nq, Nkv = ctx->Nkv;
  const void* src[4] = {w->wq, w->wk, w->wv, w->wo};
  __half* dst[4] = {k.wqkv, k.wqkv + Nq * H, k.wqkv + (Nq + Nkv) * H, k.wo};
  const long long cnt[4] = {Nq * H, Nkv * H, Nkv * H, H * Nq};
  // rope_layout = 1: the rows of Wq, Wk are interleaved per head, so that the adjacent-pair rotation of the QKV epilogue
  // acts on the half-split pairs (i, i + d/2); q.k is invariant under the common permutation
  LSP_STAGE(ST_CAST, 1, cast_weights(ctx, 4, src, dst, cnt, st, (d.use_rope && d.rope_layout == 1) ? 0x3u : 0u));
  return LSP_OK;
}
lsp_status cast_mlp_weights(lsp_ctx* ctx, const lsp_layer_weights* w, const W16& k, cudaStream_t st) {
  const long long FH = static_cast<long long>(ctx->d.ffn) * ctx->d.hidden;
  const void* src[3] = {w->w_gate, w->w_up, w->w_down};
  __half* dst[3] = {k.wgu, k.wgu + FH, k.wd};
  const long long cnt[3] = {FH, FH, FH};
  LSP_STAGE(ST_CAST, 1, cast_weights(ctx, 3, src, dst, cnt, st));
  return LSP_OK;
}

// F3 dispatch: head_dim 128 runs on tcgen05 (attn_tc.cuh); head_dim 64 on the mma.sync kernel (attn.cuh).
cudaError_t attn_fwd_dispatch(const lsp_ctx* c, const AttnParams& p, cudaStream_t st) {
  if (c->d.head_dim == 128) {
    AttnTcParams t;
    t.B = p.B; t.S = p.S; t.nq = p.nq; t.nkv = p.nkv; t.scale_log2 = p.scale_log2; t.scale = p.scale;
    t.o32 = p.o32; t.o16 = p.o16; t.ldo = p.ldo; t.lse = p.lse; t.sched = c->attn_sched;
    t.doc_start = c->doc_on ? c->doc_start : nullptr; t.doc_end = c->doc_on ? c->doc_end : nullptr;
    return attn_fwd_tc_launch(p.q, p.ldq, p.k, p.ldk, p.v, p.ldv, t, c->num_sms, st);
  }
  if (c->doc_on) return cudaErrorNotSupported;            // packed sequences: head_dim 128 kernels only
  return attn_fwd_launch<64>(p, st);
}

// B7 dispatch (two kernels either way: dK/dV, then dQ).  head_dim 128: tcgen05 kernels, timed as two stages.
lsp_status attn_bwd_dispatch(lsp_ctx* ctx, const AttnParams& p, cudaStream_t st) {
  if (ctx->d.head_dim == 128) {
    AttnTcBwdParams t;
    t.B = p.B; t.S = p.S; t.nq = p.nq; t.nkv = p.nkv; t.scale_log2 = p.scale_log2; t.scale = p.scale;
    t.lse = p.lse; t.dvec = p.dvec; t.rope = p.rope;
    t.dq32 = p.dq32; t.dk32 = p.dk32; t.dv32 = p.dv32; t.lddq32 = p.lddq32; t.lddk32 = p.lddk32;
    t.dq16 = p.dq16; t.dk16 = p.dk16; t.dv16 = p.dv16; t.ldd16 = p.ldd16; t.sched = ctx->attn_sched;
    t.doc_start = ctx->doc_on ? ctx->doc_start : nullptr; t.doc_end = ctx->doc_on ? ctx->doc_end : nullptr;
    LSP_STAGE(ST_ATTN_BWD, 1, attn_bwd_dkdv_tc_launch(p.q, p.ldq, p.k, p.ldk, p.v, p.ldv, p.dO, p.lddo, t, st));
    LSP_STAGE(ST_ATTN_BWD_DQ, 1, attn_bwd_dq_tc_launch(p.q, p.ldq, p.k, p.ldk, p.v, p.ldv, p.dO, p.lddo, t, ctx->num_sms, st));
    return LSP_OK;
  }
  if (ctx->doc_on) return fail(ctx, LSP_EUNSUPPORTED, "packed sequences need head_dim 128");
  LSP_STAGE(ST_ATTN_BWD, 2, attn_bwd_launch<64>(p, st));
  return LSP_OK;
}

// ------------------------------------------------------------------------------------------- attention block
// x [T,H] x_dt -> a32 [T,H] fp32.  SURVEY 8(a) F1-F4.
lsp_status attn_fwd_impl(lsp_ctx* ctx, int x_dt, const void* x, const lsp_layer_weights* w, float* a_out, void* saved,
                         cudaStream_t st, bool keep = true) {
  const lsp_layer_desc& d = ctx->d;
  const int T = ctx->T, H = d.hidden, Nq = ctx->Nq, Nkv = ctx->Nkv, Nqkv = ctx->Nqkv;
  __half* xn = at<__half>(saved, ctx->sv.xn);
  float* rstd1 = at<float>(saved, ctx->sv.rstd1);
  __half* qkv = at<__half>(saved, ctx->sv.qkv16);
  float* o32 = at<float>(saved, ctx->sv.o32);
  __half* o16 = at<__half>(saved, ctx->sv.o16);
  float* lse = at<float>(saved, ctx->sv.lse);
  const W16 k16 = w16_of(ctx, w, saved);
  __half* wqkv16 = k16.wqkv;
  __half* wo16 = k16.wo;
  if (!k16.cached) LSP_TRY(cast_attn_weights(ctx, w, k16, st));
  // F1 RMSNorm-1
  LSP_STAGE(ST_NORM_FWD, 1, norm_fwd(ctx, x_dt, x, w->g_attn, xn, rstd1, st));
  // F2 fused QKV projection with the RoPE epilogue (q, k rotated; v plain) into one [T, Nq+2Nkv] fp16 buffer
  {
    EpiQKVRope e{qkv, Nqkv, ctx->rope, d.seq, d.head_dim, d.use_rope ? Nq + Nkv : 0};
    e.doc_start = ctx->doc_on ? ctx->doc_start : nullptr;
    LSP_STAGE(ST_QKV, 1, (gemm1<false, false>(ctx, T, Nqkv, H, Operand{xn, H, false}, Operand{wqkv16, H, false}, e, st)));
  }
  // F3 causal GQA flash forward
  AttnParams p;
  memset(&p, 0, sizeof(p));
  p.q = qkv; p.k = qkv + Nq; p.v = qkv + Nq + Nkv;
  p.ldq = p.ldk = p.ldv = Nqkv;
  p.B = d.batch; p.S = d.seq; p.nq = d.n_q_heads; p.nkv = d.n_kv_heads;
  p.scale = 1.0f / sqrtf(static_cast<float>(logical_head_dim(d)));
  p.scale_log2 = p.scale * 1.4426950408889634f;
  p.o32 = keep ? o32 : nullptr; p.o16 = o16; p.ldo = Nq; p.lse = lse;     // the fp32 copy of O only feeds the backward (P-3)
  LSP_STAGE(ST_ATTN_FWD, 1, attn_fwd_dispatch(ctx, p, st));
  // F4 O-projection + residual
  LSP_STAGE(ST_OPROJ, 1, gemm_fwd_residual(ctx, o16, Nq, wo16, x_dt, x, a_out, st));
  return LSP_OK;
}

// da (da_dt; da16 = its fp16 copy) -> dx fp32.  SURVEY 8(a) B6-B10.
lsp_status attn_bwd_impl(lsp_ctx* ctx, int x_dt, const void* x, int da_dt, const void* da, const __half* da16,
                         const lsp_layer_weights* w, const void* saved, float* dx, lsp_layer_wgrads* g, void* ws,
                         cudaStream_t st) {
  const lsp_layer_desc& d = ctx->d;
  const int T = ctx->T, H = d.hidden, Nq = ctx->Nq, Nkv = ctx->Nkv, Nqkv = ctx->Nqkv;
  const __half* xn = at<__half>(saved, ctx->sv.xn);
  const float* rstd1 = at<float>(saved, ctx->sv.rstd1);
  const __half* qkv = at<__half>(saved, ctx->sv.qkv16);
  const float* o32 = at<float>(saved, ctx->sv.o32);
  const __half* o16 = at<__half>(saved, ctx->sv.o16);
  const float* lse = at<float>(saved, ctx->sv.lse);
  const W16 k16 = w16_of(ctx, w, saved);
  const __half* wqkv16 = k16.wqkv;
  const __half* wo16 = k16.wo;
  __half* dO16 = at<__half>(ws, ctx->ws.dO16);
  float* dvec = at<float>(ws, ctx->ws.dvec);
  __half* dqkv = at<__half>(ws, ctx->ws.dqkv16);
  float* dxn = at<float>(ws, ctx->ws.dn32);
  float* dgpart = at<float>(ws, ctx->ws.dgpart);

  // B6 dWo = da^T O ; dO = da Wo ; D = rowsum(dO * O32)
  LSP_STAGE(ST_WGRAD_O, 1, (gemm1<true, true>(ctx, H, Nq, T, Operand{da16, H, true}, Operand{o16, Nq, true},
                              epi_wgrad(ctx, g->wo, Nq), st)));
  if (d.head_dim == 128) {
    // the row sums D = rowsum(dO * O) leave the dgrad's epilogue as four partial sums per (head, position)
    EpiDOutDvec e{dO16, Nq, o32, dvec, d.seq, d.n_q_heads};
    LSP_STAGE(ST_DGRAD_O, 1, (gemm1<false, true>(ctx, T, Nq, H, Operand{da16, H, false}, Operand{wo16, Nq, true}, e, st)));
  } else {
    EpiStore<DT_F16, DT_F32, false> e;
    e.out[0] = dO16; e.out[1] = e.out[2] = nullptr; e.split1 = e.split2 = 0x7fffffff; e.ld = Nq; e.res = nullptr; e.alpha = 1.0f;
    LSP_STAGE(ST_DGRAD_O, 1, (gemm1<false, true>(ctx, T, Nq, H, Operand{da16, H, false}, Operand{wo16, Nq, true}, e, st)));
    LSP_STAGE(ST_DVEC, 1, (attn_dvec_launch<64, false>(dO16, Nq, o32, Nq, dvec, d.batch, d.seq, d.n_q_heads, st)));
  }
  // B7 + B8 flash backward with the inverse rotation on store
  AttnParams p;
  memset(&p, 0, sizeof(p));
  p.q = qkv; p.k = qkv + Nq; p.v = qkv + Nq + Nkv; p.dO = dO16;
  p.ldq = p.ldk = p.ldv = Nqkv; p.lddo = Nq;
  p.B = d.batch; p.S = d.seq; p.nq = d.n_q_heads; p.nkv = d.n_kv_heads;
  p.scale = 1.0f / sqrtf(static_cast<float>(logical_head_dim(d)));
  p.scale_log2 = p.scale * 1.4426950408889634f;
  p.lse = const_cast<float*>(lse); p.dvec = dvec;
  p.rope = d.use_rope ? ctx->rope : nullptr;
  p.dq16 = dqkv; p.dk16 = dqkv + Nq; p.dv16 = dqkv + Nq + Nkv; p.ldd16 = Nqkv;
  LSP_TRY(attn_bwd_dispatch(ctx, p, st));
  // B9 dW{q,k,v} = d{q,k,v}^T xn (one GEMM, rows split over three outputs) ; dxn = [dq|dk|dv] [Wq;Wk;Wv] (one GEMM)
  {
    EpiF32 e = epi_wgrad(ctx, g->wq, H);
    e.out[1] = g->wk; e.out[2] = g->wv; e.split1 = Nq; e.split2 = Nq + Nkv;
    if (d.use_rope && d.rope_layout == 1) { e.perm_d = d.head_dim; e.perm_segs = 0x3u; }     // dWq, dWk rows back to the caller's order
    LSP_STAGE(ST_WGRAD_QKV, 1, (gemm1<true, true>(ctx, Nqkv, H, T, Operand{dqkv, Nqkv, true}, Operand{xn, H, true}, e, st)));
  }
  LSP_STAGE(ST_DGRAD_QKV, 1, (gemm1<false, true>(ctx, T, H, Nqkv, Operand{dqkv, Nqkv, false}, Operand{wqkv16, H, true},
                               epi_f32(dxn, H), st)));
  // B10 RMSNorm-1 backward + residual gradient
  LSP_STAGE(ST_NORM_BWD, 2, norm_bwd(ctx, x_dt, da_dt, x, rstd1, w->g_attn, dxn, da, dx, nullptr, dgpart, static_cast<float*>(g->g_attn), ctx->d.wgrad_accumulate, st));
  return LSP_OK;
}

// ------------------------------------------------------------------------------------------- MLP block
// a (a_dt) -> y fp32.  SURVEY 8(a) F5-F7.
lsp_status mlp_fwd_impl(lsp_ctx* ctx, int a_dt, const void* a, const lsp_layer_weights* w, float* y, void* saved, cudaStream_t st,
                        bool keep = true) {
  const lsp_layer_desc& d = ctx->d;
  const int T = ctx->T, H = d.hidden, F = d.ffn;
  __half* an = at<__half>(saved, ctx->sv.an);
  float* rstd2 = at<float>(saved, ctx->sv.rstd2);
  __half* g16 = at<__half>(saved, ctx->sv.g16);
  __half* u16 = at<__half>(saved, ctx->sv.u16);
  __half* h = at<__half>(saved, ctx->sv.h);
  const W16 k16 = w16_of(ctx, w, saved);
  __half* wgu16 = k16.wgu;
  __half* wd16 = k16.wd;
  const long long FH = static_cast<long long>(F) * H;
  if (!k16.cached) LSP_TRY(cast_mlp_weights(ctx, w, k16, st));
  LSP_STAGE(ST_NORM_FWD, 1, norm_fwd(ctx, a_dt, a, w->g_mlp, an, rstd2, st));
  EpiSwiGLU e{h, g16, u16, F};
  e.save_gu = keep ? 1 : 0;
  const GemmSKRes sk{ctx->sk_partial, ctx->sk_flags, ++ctx->gemm_seq};
  LSP_STAGE(ST_GATEUP, 1, gemm_run_dual(T, F, H, Operand{an, H, false}, Operand{wgu16, H, false}, Operand{wgu16 + FH, H, false}, e,
                         ctx->num_sms, st, &sk));
  LSP_STAGE(ST_DOWN, 1, gemm_fwd_residual(ctx, h, F, wd16, a_dt, a, y, st));
  return LSP_OK;
}

// dy (dy_dt; dy16 = its fp16 copy) -> da fp32 (+ fp16 copy da16 if non-null).  SURVEY 8(a) B1-B5.
lsp_status mlp_bwd_impl(lsp_ctx* ctx, int a_dt, const void* a, int dy_dt, const void* dy, const __half* dy16,
                        const lsp_layer_weights* w, const void* saved, float* da, __half* da16, lsp_layer_wgrads* g,
                        void* ws, cudaStream_t st) {
  const lsp_layer_desc& d = ctx->d;
  const int T = ctx->T, H = d.hidden, F = d.ffn;
  const __half* an = at<__half>(saved, ctx->sv.an);
  const float* rstd2 = at<float>(saved, ctx->sv.rstd2);
  const __half* g16 = at<__half>(saved, ctx->sv.g16);
  const __half* u16 = at<__half>(saved, ctx->sv.u16);
  const __half* h = at<__half>(saved, ctx->sv.h);
  const W16 k16 = w16_of(ctx, w, saved);
  const __half* wgu16 = k16.wgu;
  const __half* wd16 = k16.wd;
  __half* dgu = at<__half>(ws, ctx->ws.dgu);
  float* dan = at<float>(ws, ctx->ws.dn32);
  float* dgpart = at<float>(ws, ctx->ws.dgpart);

  // B2 dWd = dy^T h
  LSP_STAGE(ST_WGRAD_DOWN, 1, (gemm1<true, true>(ctx, H, F, T, Operand{dy16, H, true}, Operand{h, F, true}, epi_wgrad(ctx, g->w_down, F), st)));
  // B1 dh = dy Wd with the SwiGLU-backward epilogue -> [dg | du]
  {
    EpiSwiGLUBwd e{g16, u16, F, dgu, F};
    LSP_STAGE(ST_DGRAD_DOWN, 1, (gemm1<false, true>(ctx, T, F, H, Operand{dy16, H, false}, Operand{wd16, F, true}, e, st)));
  }
  // B4 dWg = dg^T an, dWu = du^T an (one GEMM over the 2F rows of [dg | du]^T)
  {
    EpiF32 e = epi_wgrad(ctx, g->w_gate, H);
    e.out[1] = g->w_up; e.split1 = F;
    LSP_STAGE(ST_WGRAD_GATEUP, 1, (gemm1<true, true>(ctx, 2 * F, H, T, Operand{dgu, 2LL * F, true}, Operand{an, H, true}, e, st)));
  }
  // B3 dan = [dg | du] [Wg; Wu]  (one GEMM, K = 2F)
  LSP_STAGE(ST_DGRAD_GATEUP, 1, (gemm1<false, true>(ctx, T, H, 2 * F, Operand{dgu, 2LL * F, false}, Operand{wgu16, H, true},
                                  epi_f32(dan, H), st)));
  // B5 RMSNorm-2 backward + residual gradient
  LSP_STAGE(ST_NORM_BWD, 2, norm_bwd(ctx, a_dt, dy_dt, a, rstd2, w->g_mlp, dan, dy, da, da16, dgpart, static_cast<float*>(g->g_mlp), ctx->d.wgrad_accumulate, st));
  return LSP_OK;
}

lsp_status check_common(lsp_ctx* ctx, const void* saved, const void* ws, int n, const void* const* ptrs) {
  if (!ctx) return LSP_EINVAL;
  for (int i = 0; i < n; ++i) {
    if (!ptrs[i]) return fail(ctx, LSP_EINVAL, "NULL pointer argument (#%d)", i);
    if (!aligned(ptrs[i], 16)) return fail(ctx, LSP_EALIGN, "pointer argument #%d is not 16-byte aligned", i);
  }
  if (saved && !aligned(saved, ALIGN)) return fail(ctx, LSP_EALIGN, "`saved` must be 256-byte aligned");
  if (ws && !aligned(ws, ALIGN)) return fail(ctx, LSP_EALIGN, "`ws` must be 256-byte aligned");
  return LSP_OK;
}

lsp_status check_cache(lsp_ctx* ctx, const lsp_layer_weights* w) {
  if (w->f16_cache && !aligned(w->f16_cache, ALIGN)) return fail(ctx, LSP_EALIGN, "`f16_cache` must be 256-byte aligned");
  return LSP_OK;
}

// fp16 operand copy of an activation-gradient input (bf16: exact for normal-range values; fp32: rounded), in ws.in16
lsp_status as_f16(lsp_ctx* ctx, const void* in, void* ws, cudaStream_t st, const __half** out) {
  __half* t = at<__half>(ws, ctx->ws.in16);
  const long long n = static_cast<long long>(ctx->T) * ctx->d.hidden;
  if (ctx->d.in_dtype == LSP_BF16) LSP_STAGE(ST_CAST, 1, cast_bf16_f16(static_cast<const __nv_bfloat16*>(in), t, n, ctx->num_sms, ctx->overflow, st));
  else LSP_STAGE(ST_CAST, 1, cast_f32_f16(static_cast<const float*>(in), t, n, ctx->num_sms, ctx->overflow, st));
  *out = t;
  return LSP_OK;
}

}  // namespace

// ------------------------------------------------------------------ scratch of lsp_grad_norm_static (include/lsp.h)
// The per-block partial sums of g^2 of the allocation-free gradient-norm entry point.  A device array: every GPU that
// loads the library holds these 128 KiB until the process exits.  In HOST code the name is only a stand-in for the
// symbol, never a device address: the entry point resolves the address once per device with cudaGetSymbolAddress
// (norm_static_setup) and hands THAT pointer to the kernels.
static __device__ __align__(256) float g_norm_static_scratch[LSP_NORM_STATIC_SCRATCH_BYTES / sizeof(float)];

namespace {

constexpr int NORM_STATIC_MAX_DEVICES = 64;
struct NormStaticDevice {
  float* scratch;      // device address of g_norm_static_scratch on this device
  int num_sms;
  bool ready;
};
NormStaticDevice g_norm_static_dev[NORM_STATIC_MAX_DEVICES];
std::mutex g_norm_static_mutex;

lsp_status fail_msg(char* err, size_t err_len, lsp_status s, const char* fmt, ...) {
  if (err && err_len) {
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(err, err_len, fmt, ap);
    va_end(ap);
  }
  return s;
}

// once per device, with that device current
lsp_status norm_static_setup(int dev, NormStaticDevice* out, char* err, size_t err_len) {
  std::lock_guard<std::mutex> lock(g_norm_static_mutex);
  NormStaticDevice& d = g_norm_static_dev[dev];
  if (!d.ready) {
    float* p = nullptr;
    cudaError_t e = cudaGetSymbolAddress(reinterpret_cast<void**>(&p), g_norm_static_scratch);
    if (e != cudaSuccess || !p)
      return fail_msg(err, err_len, LSP_ECUDA, "lsp_grad_norm_static: cudaGetSymbolAddress on device %d failed: %s", dev, cudaGetErrorString(e));
    int sms = 0;
    e = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    if (e != cudaSuccess || sms <= 0)
      return fail_msg(err, err_len, LSP_ECUDA, "lsp_grad_norm_static: cannot read the SM count of device %d: %s", dev, cudaGetErrorString(e));
    d.scratch = p; d.num_sms = sms; d.ready = true;
  }
  *out = d;
  return LSP_OK;
}

}  // namespace

// =========================================================================================== C ABI
extern "C" {

lsp_status lsp_create(lsp_ctx** out, const lsp_layer_desc* desc, int cuda_device) {
  if (!out || !desc) return LSP_EINVAL;
  *out = nullptr;
  const lsp_layer_desc& d = *desc;
  if (d.batch <= 0 || d.seq <= 0 || d.hidden <= 0 || d.n_q_heads <= 0 || d.n_kv_heads <= 0 || d.ffn <= 0) return LSP_EINVAL;
  if (d.n_q_heads % d.n_kv_heads != 0) return LSP_EINVAL;
  if (d.head_dim != 64 && d.head_dim != 128) return LSP_EUNSUPPORTED;
  if (d.head_dim_logical != 0 && (d.head_dim_logical < 2 || d.head_dim_logical > d.head_dim || (d.head_dim_logical & 1) ||
                                  (d.head_dim_logical != d.head_dim && d.rope_layout != 0)))
    return LSP_EUNSUPPORTED;
  if (d.hidden % 8 || d.ffn % 8 || d.hidden > 8192) return LSP_EUNSUPPORTED;
  if ((d.rope_layout != 0 && d.rope_layout != 1) || (d.wgrad_accumulate != 0 && d.wgrad_accumulate != 1)) return LSP_EUNSUPPORTED;
  if (d.in_dtype != LSP_BF16 && d.in_dtype != LSP_F32) return LSP_EINVAL;
  if (!(d.rms_eps >= 0.0f) || !(d.rope_base > 0.0)) return LSP_EINVAL;
  if (static_cast<long long>(d.batch) * d.seq > 0x7fffffffLL / 4) return LSP_EUNSUPPORTED;

  lsp_ctx* ctx = new (std::nothrow) lsp_ctx;
  if (!ctx) return LSP_ENOMEM;
  memset(ctx, 0, sizeof(*ctx));
  ctx->d = d;
  ctx->device = cuda_device;
  ctx->T = d.batch * d.seq;
  ctx->Nq = d.n_q_heads * d.head_dim;
  ctx->Nkv = d.n_kv_heads * d.head_dim;
  ctx->Nqkv = ctx->Nq + 2 * ctx->Nkv;
  ctx->G = d.n_q_heads / d.n_kv_heads;

  cudaDeviceProp prop;
  DeviceGuard guard(cuda_device);                 // the caller's current device is restored on every return path
  if (!guard.ok || cudaGetDeviceProperties(&prop, cuda_device) != cudaSuccess) {
    delete ctx;
    return LSP_ECUDA;
  }
  if (prop.major != 10) {          // tcgen05 / TMEM kernels: Blackwell only, no fallback
    delete ctx;
    return LSP_EUNSUPPORTED;
  }
  ctx->num_sms = prop.multiProcessorCount;
  ctx->norm_blocks = ctx->num_sms;         // one persistent CTA per SM (bulk-copy ring of ~200 KB)
  plan_layout(ctx);

  // RoPE table: theta = pos * base^(-2i/d) in fp64 (reading A-5), stored as fp32 (cos, sin)
  // head_dim_logical < head_dim (zero-padded heads): frequencies of the logical width, identity on the padding pairs
  const int half = d.head_dim / 2, dl = logical_head_dim(d);
  std::vector<float2> tab(static_cast<size_t>(d.seq) * half);
  for (int p = 0; p < d.seq; ++p)
    for (int i = 0; i < half; ++i) {
      const double th = 2 * i < dl ? static_cast<double>(p) * pow(d.rope_base, -2.0 * i / dl) : 0.0;
      tab[static_cast<size_t>(p) * half + i] = make_float2(static_cast<float>(cos(th)), static_cast<float>(sin(th)));
    }
  if (cudaMalloc(&ctx->rope, tab.size() * sizeof(float2)) != cudaSuccess) { delete ctx; return LSP_ENOMEM; }
  if (cudaMemcpy(ctx->rope, tab.data(), tab.size() * sizeof(float2), cudaMemcpyHostToDevice) != cudaSuccess) {
    cudaFree(ctx->rope);
    delete ctx;
    return LSP_ECUDA;
  }
  if (!get_encode_fn()) { cudaFree(ctx->rope); delete ctx; return LSP_ECUDA; }
  {
    const size_t pairs = static_cast<size_t>(ctx->num_sms / 2);
    if (cudaMalloc(&ctx->sk_partial, pairs * GEMM2_PARTIAL_FLOATS * sizeof(float)) != cudaSuccess ||
        cudaMalloc(&ctx->sk_flags, pairs * 2 * sizeof(unsigned int)) != cudaSuccess ||
        cudaMemset(ctx->sk_flags, 0, pairs * 2 * sizeof(unsigned int)) != cudaSuccess ||
        cudaMalloc(&ctx->opt_partial, OPT_MAX_CHUNKS * opt_blocks_cap(ctx->num_sms) * sizeof(float)) != cudaSuccess ||
        cudaMalloc(&ctx->attn_sched, 16 * sizeof(unsigned int)) != cudaSuccess ||
        cudaMalloc(&ctx->overflow, sizeof(unsigned long long)) != cudaSuccess ||
        cudaMemset(ctx->overflow, 0, sizeof(unsigned long long)) != cudaSuccess ||
        cudaMalloc(&ctx->doc_start, 2 * static_cast<size_t>(ctx->T) * sizeof(int)) != cudaSuccess ||
        cudaMemset(ctx->attn_sched, 0, 16 * sizeof(unsigned int)) != cudaSuccess) {
      cudaFree(ctx->sk_partial); cudaFree(ctx->sk_flags); cudaFree(ctx->attn_sched); cudaFree(ctx->overflow); cudaFree(ctx->opt_partial); cudaFree(ctx->doc_start); cudaFree(ctx->rope); delete ctx;
      return LSP_ENOMEM;
    }
  }
  if (cudaStreamCreateWithFlags(&ctx->s_in, cudaStreamNonBlocking) != cudaSuccess ||
      cudaStreamCreateWithFlags(&ctx->s_out, cudaStreamNonBlocking) != cudaSuccess) {
    lsp_destroy(ctx);
    return LSP_ECUDA;
  }
  for (int i = 0; i < 6; ++i)
    if (cudaEventCreateWithFlags(&ctx->ev[i], cudaEventDisableTiming) != cudaSuccess) { lsp_destroy(ctx); return LSP_ECUDA; }
  for (int i = 0; i < 12; ++i)
    if (cudaEventCreateWithFlags(&ctx->pev[i / 6][i % 6], cudaEventDisableTiming) != cudaSuccess) { lsp_destroy(ctx); return LSP_ECUDA; }
  *out = ctx;
  return LSP_OK;
}

lsp_status lsp_destroy(lsp_ctx* ctx) {
  if (!ctx) return LSP_EINVAL;
  DeviceGuard guard(ctx->device);
  lsp_timing_enable(ctx, 0);
  cudaFree(ctx->overflow);
  cudaFree(ctx->rope);
  cudaFree(ctx->sk_partial);
  cudaFree(ctx->sk_flags);
  cudaFree(ctx->attn_sched);
  cudaFree(ctx->opt_partial);
  cudaFree(ctx->doc_start);
  if (ctx->s_in) cudaStreamDestroy(ctx->s_in);
  if (ctx->s_out) cudaStreamDestroy(ctx->s_out);
  for (int i = 0; i < 6; ++i)
    if (ctx->ev[i]) cudaEventDestroy(ctx->ev[i]);
  for (int i = 0; i < 12; ++i)
    if (ctx->pev[i / 6][i % 6]) cudaEventDestroy(ctx->pev[i / 6][i % 6]);
  delete ctx;
  return LSP_OK;
}

size_t lsp_saved_bytes(const lsp_ctx* ctx) { return ctx ? ctx->sv.total : 0; }
size_t lsp_workspace_bytes(const lsp_ctx* ctx) { return ctx ? ctx->ws.total : 0; }
const char* lsp_last_error(const lsp_ctx* ctx) { return ctx ? ctx->err : "lsp: NULL context"; }

size_t lsp_weight_cache_bytes(const lsp_ctx* ctx) { return ctx ? ctx->wc.total : 0; }

long long lsp_weight_cache_offset(const lsp_ctx* ctx, int which) {
  if (!ctx || which < 0 || which > 6) return -1;
  // the rows of Wq, Wk are permuted inside the cache when rope_layout = 1: only lsp_layer_prepare_weights can fill them
  if (ctx->d.use_rope && ctx->d.rope_layout == 1 && which <= 1) return -1;
  const long long H = ctx->d.hidden, Nq = ctx->Nq, Nkv = ctx->Nkv, F = ctx->d.ffn;
  switch (which) {
    case 0: return static_cast<long long>(ctx->wc.wqkv16);
    case 1: return static_cast<long long>(ctx->wc.wqkv16) + Nq * H * 2;
    case 2: return static_cast<long long>(ctx->wc.wqkv16) + (Nq + Nkv) * H * 2;
    case 3: return static_cast<long long>(ctx->wc.wo16);
    case 4: return static_cast<long long>(ctx->wc.wgu16);
    case 5: return static_cast<long long>(ctx->wc.wgu16) + F * H * 2;
    default: return static_cast<long long>(ctx->wc.wd16);
  }
}

lsp_status lsp_layer_prepare_weights(lsp_ctx* ctx, const lsp_layer_weights* w, void* cache, void* stream) {
  if (!ctx || !w) return LSP_EINVAL;
  LSP_ENTER(ctx);
  const void* ptrs[] = {cache, w->wq, w->wk, w->wv, w->wo, w->w_gate, w->w_up, w->w_down};
  LSP_TRY(check_common(ctx, cache, nullptr, 8, ptrs));
  cudaStream_t st = static_cast<cudaStream_t>(stream);
  lsp_layer_weights wc = *w;
  wc.f16_cache = cache;
  const W16 k = w16_of(ctx, &wc, nullptr);
  LSP_TRY(cast_attn_weights(ctx, w, k, st));
  return cast_mlp_weights(ctx, w, k, st);
}

lsp_status lsp_overflow_count(lsp_ctx* ctx, unsigned long long* count, int reset, void* stream) {
  if (!ctx || !count) return LSP_EINVAL;
  LSP_ENTER(ctx);
  cudaStream_t st = static_cast<cudaStream_t>(stream);
  LSP_CUDA(cudaMemcpyAsync(count, ctx->overflow, sizeof(unsigned long long), cudaMemcpyDeviceToHost, st));
  LSP_CUDA(cudaStreamSynchronize(st));
  if (reset) LSP_CUDA(cudaMemsetAsync(ctx->overflow, 0, sizeof(unsigned long long), st));
  return LSP_OK;
}

lsp_status lsp_attn_fwd(lsp_ctx* ctx, const void* x, const lsp_layer_weights* w, void* a_out, void* saved, void* ws, void* stream) {
  if (!ctx || !w) return LSP_EINVAL;
  LSP_ENTER(ctx);
  const void* ptrs[] = {x, a_out, saved, ws, w->wq, w->wk, w->wv, w->wo, w->g_attn};
  LSP_TRY(check_common(ctx, saved, ws, 9, ptrs));
  LSP_TRY(check_cache(ctx, w));
  return attn_fwd_impl(ctx, ctx->d.in_dtype, x, w, static_cast<float*>(a_out), saved, static_cast<cudaStream_t>(stream));
}

lsp_status lsp_attn_bwd(lsp_ctx* ctx, const void* x, const void* da, const lsp_layer_weights* w, const void* saved, void* dx,
                        lsp_layer_wgrads* g, void* ws, void* stream) {
  if (!ctx || !w || !g) return LSP_EINVAL;
  LSP_ENTER(ctx);
  const void* ptrs[] = {x, da, saved, dx, ws, w->wq, w->wk, w->wv, w->wo, w->g_attn, g->wq, g->wk, g->wv, g->wo, g->g_attn};
  LSP_TRY(check_common(ctx, saved, ws, 15, ptrs));
  LSP_TRY(check_cache(ctx, w));
  cudaStream_t st = static_cast<cudaStream_t>(stream);
  const __half* da16;
  LSP_TRY(as_f16(ctx, da, ws, st, &da16));
  return attn_bwd_impl(ctx, ctx->d.in_dtype, x, ctx->d.in_dtype, da, da16, w, saved, static_cast<float*>(dx), g, ws, st);
}

lsp_status lsp_mlp_fwd(lsp_ctx* ctx, const void* a, const lsp_layer_weights* w, void* y_out, void* saved, void* ws, void* stream) {
  if (!ctx || !w) return LSP_EINVAL;
  LSP_ENTER(ctx);
  const void* ptrs[] = {a, y_out, saved, ws, w->w_gate, w->w_up, w->w_down, w->g_mlp};
  LSP_TRY(check_common(ctx, saved, ws, 8, ptrs));
  LSP_TRY(check_cache(ctx, w));
  return mlp_fwd_impl(ctx, ctx->d.in_dtype, a, w, static_cast<float*>(y_out), saved, static_cast<cudaStream_t>(stream));
}

lsp_status lsp_mlp_bwd(lsp_ctx* ctx, const void* a, const void* dy, const lsp_layer_weights* w, const void* saved, void* da,
                       lsp_layer_wgrads* g, void* ws, void* stream) {
  if (!ctx || !w || !g) return LSP_EINVAL;
  LSP_ENTER(ctx);
  const void* ptrs[] = {a, dy, saved, da, ws, w->w_gate, w->w_up, w->w_down, w->g_mlp, g->w_gate, g->w_up, g->w_down, g->g_mlp};
  LSP_TRY(check_common(ctx, saved, ws, 13, ptrs));
  LSP_TRY(check_cache(ctx, w));
  cudaStream_t st = static_cast<cudaStream_t>(stream);
  const __half* dy16;
  LSP_TRY(as_f16(ctx, dy, ws, st, &dy16));
  return mlp_bwd_impl(ctx, ctx->d.in_dtype, a, ctx->d.in_dtype, dy, dy16, w, saved, static_cast<float*>(da), nullptr, g, ws, st);
}

lsp_status lsp_layer_fwd(lsp_ctx* ctx, const void* x, const lsp_layer_weights* w, void* y_out, void* saved, void* ws, void* stream) {
  if (!ctx || !w) return LSP_EINVAL;
  LSP_ENTER(ctx);
  const void* ptrs[] = {x, y_out, saved, ws, w->wq, w->wk, w->wv, w->wo, w->g_attn, w->w_gate, w->w_up, w->w_down, w->g_mlp};
  LSP_TRY(check_common(ctx, saved, ws, 13, ptrs));
  LSP_TRY(check_cache(ctx, w));
  cudaStream_t st = static_cast<cudaStream_t>(stream);
  float* a32 = at<float>(saved, ctx->sv.a32);
  LSP_TRY(attn_fwd_impl(ctx, ctx->d.in_dtype, x, w, a32, saved, st));
  return mlp_fwd_impl(ctx, LSP_F32, a32, w, static_cast<float*>(y_out), saved, st);
}

lsp_status lsp_layer_fwd_infer(lsp_ctx* ctx, const void* x, const lsp_layer_weights* w, void* y_out, void* scratch, void* ws,
                               void* stream) {
  if (!ctx || !w) return LSP_EINVAL;
  LSP_ENTER(ctx);
  const void* ptrs[] = {x, y_out, scratch, ws, w->wq, w->wk, w->wv, w->wo, w->g_attn, w->w_gate, w->w_up, w->w_down, w->g_mlp};
  LSP_TRY(check_common(ctx, scratch, ws, 13, ptrs));
  LSP_TRY(check_cache(ctx, w));
  cudaStream_t st = static_cast<cudaStream_t>(stream);
  float* a32 = at<float>(scratch, ctx->sv.a32);
  LSP_TRY(attn_fwd_impl(ctx, ctx->d.in_dtype, x, w, a32, scratch, st, false));
  return mlp_fwd_impl(ctx, LSP_F32, a32, w, static_cast<float*>(y_out), scratch, st, false);
}

lsp_status lsp_layer_bwd(lsp_ctx* ctx, const void* x, const void* dy, const lsp_layer_weights* w, const void* saved, void* dx,
                         lsp_layer_wgrads* g, void* ws, void* stream) {
  if (!ctx || !w || !g) return LSP_EINVAL;
  LSP_ENTER(ctx);
  const void* ptrs[] = {x, dy, saved, dx, ws, w->wq, w->wk, w->wv, w->wo, w->g_attn, w->w_gate, w->w_up, w->w_down, w->g_mlp,
                        g->wq, g->wk, g->wv, g->wo, g->g_attn, g->w_gate, g->w_up, g->w_down, g->g_mlp};
  LSP_TRY(check_common(ctx, saved, ws, 23, ptrs));
  LSP_TRY(check_cache(ctx, w));
  cudaStream_t st = static_cast<cudaStream_t>(stream);
  const __half* dy16;
  LSP_TRY(as_f16(ctx, dy, ws, st, &dy16));
  const float* a32 = at<float>(saved, ctx->sv.a32);
  float* da32 = at<float>(ws, ctx->ws.da32);
  __half* da16 = at<__half>(ws, ctx->ws.da16);
  LSP_TRY(mlp_bwd_impl(ctx, LSP_F32, a32, ctx->d.in_dtype, dy, dy16, w, saved, da32, da16, g, ws, st));
  return attn_bwd_impl(ctx, ctx->d.in_dtype, x, LSP_F32, da32, da16, w, saved, static_cast<float*>(dx), g, ws, st);
}

lsp_status lsp_sdpa_fwd(lsp_ctx* ctx, const void* q, const void* k, const void* v, void* o, float* lse, void* ws, void* stream) {
  if (!ctx) return LSP_EINVAL;
  LSP_ENTER(ctx);
  const void* ptrs[] = {q, k, v, o, lse, ws};
  LSP_TRY(check_common(ctx, nullptr, ws, 6, ptrs));
  cudaStream_t st = static_cast<cudaStream_t>(stream);
  const lsp_layer_desc& d = ctx->d;
  const long long T = ctx->T;
  __half* q16 = at<__half>(ws, ctx->ws.q16);
  __half* k16 = at<__half>(ws, ctx->ws.k16);
  __half* v16 = at<__half>(ws, ctx->ws.v16);
  LSP_STAGE(ST_CAST, 1, cast_bf16_f16(static_cast<const __nv_bfloat16*>(q), q16, T * ctx->Nq, ctx->num_sms, ctx->overflow, st));
  LSP_STAGE(ST_CAST, 1, cast_bf16_f16(static_cast<const __nv_bfloat16*>(k), k16, T * ctx->Nkv, ctx->num_sms, ctx->overflow, st));
  LSP_STAGE(ST_CAST, 1, cast_bf16_f16(static_cast<const __nv_bfloat16*>(v), v16, T * ctx->Nkv, ctx->num_sms, ctx->overflow, st));
  AttnParams p;
  memset(&p, 0, sizeof(p));
  p.q = q16; p.k = k16; p.v = v16;
  p.ldq = ctx->Nq; p.ldk = p.ldv = ctx->Nkv;
  p.B = d.batch; p.S = d.seq; p.nq = d.n_q_heads; p.nkv = d.n_kv_heads;
  p.scale = 1.0f / sqrtf(static_cast<float>(logical_head_dim(d)));
  p.scale_log2 = p.scale * 1.4426950408889634f;
  p.o32 = static_cast<float*>(o); p.ldo = ctx->Nq; p.lse = lse;
  LSP_STAGE(ST_ATTN_FWD, 1, attn_fwd_dispatch(ctx, p, st));
  return LSP_OK;
}

lsp_status lsp_sdpa_bwd(lsp_ctx* ctx, const void* q, const void* k, const void* v, const void* o, const float* lse,
                        const void* d_o, void* dq, void* dk, void* dv, void* ws, void* stream) {
  if (!ctx) return LSP_EINVAL;
  LSP_ENTER(ctx);
  const void* ptrs[] = {q, k, v, o, lse, d_o, dq, dk, dv, ws};
  LSP_TRY(check_common(ctx, nullptr, ws, 10, ptrs));
  cudaStream_t st = static_cast<cudaStream_t>(stream);
  const lsp_layer_desc& d = ctx->d;
  const long long T = ctx->T;
  __half* q16 = at<__half>(ws, ctx->ws.q16);
  __half* k16 = at<__half>(ws, ctx->ws.k16);
  __half* v16 = at<__half>(ws, ctx->ws.v16);
  __half* dO16 = at<__half>(ws, ctx->ws.dO16);
  float* dvec = at<float>(ws, ctx->ws.dvec);
  LSP_STAGE(ST_CAST, 1, cast_bf16_f16(static_cast<const __nv_bfloat16*>(q), q16, T * ctx->Nq, ctx->num_sms, ctx->overflow, st));
  LSP_STAGE(ST_CAST, 1, cast_bf16_f16(static_cast<const __nv_bfloat16*>(k), k16, T * ctx->Nkv, ctx->num_sms, ctx->overflow, st));
  LSP_STAGE(ST_CAST, 1, cast_bf16_f16(static_cast<const __nv_bfloat16*>(v), v16, T * ctx->Nkv, ctx->num_sms, ctx->overflow, st));
  LSP_STAGE(ST_CAST, 1, cast_bf16_f16(static_cast<const __nv_bfloat16*>(d_o), dO16, T * ctx->Nq, ctx->num_sms, ctx->overflow, st));
  if (d.head_dim == 128) LSP_STAGE(ST_DVEC, 1, (attn_dvec_launch<128, true>(dO16, ctx->Nq, static_cast<const float*>(o), ctx->Nq, dvec, d.batch, d.seq, d.n_q_heads, st)));
  else LSP_STAGE(ST_DVEC, 1, (attn_dvec_launch<64, false>(dO16, ctx->Nq, static_cast<const float*>(o), ctx->Nq, dvec, d.batch, d.seq, d.n_q_heads, st)));
  AttnParams p;
  memset(&p, 0, sizeof(p));
  p.q = q16; p.k = k16; p.v = v16; p.dO = dO16;
  p.ldq = ctx->Nq; p.ldk = p.ldv = ctx->Nkv; p.lddo = ctx->Nq;
  p.B = d.batch; p.S = d.seq; p.nq = d.n_q_heads; p.nkv = d.n_kv_heads;
  p.scale = 1.0f / sqrtf(static_cast<float>(logical_head_dim(d)));
  p.scale_log2 = p.scale * 1.4426950408889634f;
  p.lse = const_cast<float*>(lse); p.dvec = dvec;
  p.dq32 = static_cast<float*>(dq); p.dk32 = static_cast<float*>(dk); p.dv32 = static_cast<float*>(dv);
  p.lddq32 = ctx->Nq; p.lddk32 = ctx->Nkv;
  LSP_TRY(attn_bwd_dispatch(ctx, p, st));
  return LSP_OK;
}

lsp_status lsp_embed_fwd(lsp_ctx* ctx, const int32_t* ids, const void* table, void* x0, void* stream) {
  if (!ctx) return LSP_EINVAL;
  LSP_ENTER(ctx);
  const void* ptrs[] = {ids, table, x0};
  LSP_TRY(check_common(ctx, nullptr, nullptr, 3, ptrs));
  cudaStream_t st = static_cast<cudaStream_t>(stream);
  auto launch = [&]() {
    embed_gather_kernel<float><<<ctx->T, 256, 0, st>>>(ids, static_cast<const __nv_bfloat16*>(table), static_cast<float*>(x0), ctx->d.hidden);
    return cudaGetLastError();
  };
  LSP_STAGE(ST_EMBED, 1, launch());
  return LSP_OK;
}

lsp_status lsp_gemm(lsp_ctx* ctx, int op, int M, int N, int K, const void* A, int64_t lda, int a_dtype, const void* B,
                    int64_t ldb, int b_dtype, float* C, int64_t ldc, void* stream) {
  if (!ctx) return LSP_EINVAL;
  LSP_ENTER(ctx);
  const void* ptrs[] = {A, B, C};
  LSP_TRY(check_common(ctx, nullptr, nullptr, 3, ptrs));
  if (M <= 0 || N <= 0 || K <= 0 || (lda % 8) || (ldb % 8) || (ldc % 8) || (N % 8)) return fail(ctx, LSP_EINVAL, "lsp_gemm: bad extents/pitches");
  if ((a_dtype != LSP_BF16 && a_dtype != LSP_F16) || (b_dtype != LSP_BF16 && b_dtype != LSP_F16))
    return fail(ctx, LSP_EINVAL, "lsp_gemm: operand dtype must be LSP_BF16 or LSP_F16");
  if (a_dtype != b_dtype)       // tcgen05.mma.kind::f16 with unequal A/B formats faults on sm_100a (measured)
    return fail(ctx, LSP_EUNSUPPORTED, "lsp_gemm: A and B must have the same 16-bit format");
  cudaStream_t st = static_cast<cudaStream_t>(stream);
  const EpiF32 e = epi_f32(C, ldc);
  const int adt = a_dtype == LSP_F16 ? DT_F16 : DT_BF16, bdt = b_dtype == LSP_F16 ? DT_F16 : DT_BF16;
  switch (op) {
    case 0: LSP_STAGE(ST_OPROJ, 1, (gemm1<false, false>(ctx, M, N, K, Operand{A, lda, false, adt}, Operand{B, ldb, false, bdt}, e, st))); break;
    case 1: LSP_STAGE(ST_DGRAD_O, 1, (gemm1<false, true>(ctx, M, N, K, Operand{A, lda, false, adt}, Operand{B, ldb, true, bdt}, e, st))); break;
    case 2: LSP_STAGE(ST_WGRAD_O, 1, (gemm1<true, true>(ctx, M, N, K, Operand{A, lda, true, adt}, Operand{B, ldb, true, bdt}, e, st))); break;
    default: return fail(ctx, LSP_EINVAL, "lsp_gemm: op must be 0, 1 or 2");
  }
  return LSP_OK;
}

lsp_status lsp_layer_step_host(lsp_ctx* ctx, const void* x_host, const void* dy_host, const lsp_layer_weights* w,
                               void* y_host, void* dx_host, lsp_layer_wgrads* g, void* x_dev, void* dy_dev, void* y_dev,
                               void* dx_dev, void* saved, void* ws, void* stream) {
  if (!ctx || !x_host || !dy_host || !y_host || !dx_host || !x_dev || !dy_dev || !y_dev || !dx_dev) return LSP_EINVAL;
  LSP_ENTER(ctx);
  cudaStream_t st = static_cast<cudaStream_t>(stream);
  const size_t n = static_cast<size_t>(ctx->T) * ctx->d.hidden;
  const size_t in_bytes = n * (ctx->d.in_dtype == LSP_F32 ? 4 : 2);
  // Copies run on two context-owned streams so that the upload of dy overlaps the forward pass and the download of y
  // overlaps the backward pass; everything is ordered after what `st` held before and `st` ends after the last copy.
  cudaEvent_t* ev = ctx->ev;
  LSP_CUDA(cudaEventRecord(ev[0], st));
  LSP_CUDA(cudaStreamWaitEvent(ctx->s_in, ev[0], 0));
  LSP_CUDA(cudaStreamWaitEvent(ctx->s_out, ev[0], 0));
  LSP_CUDA(cudaMemcpyAsync(x_dev, x_host, in_bytes, cudaMemcpyHostToDevice, ctx->s_in));
  LSP_CUDA(cudaEventRecord(ev[1], ctx->s_in));
  LSP_CUDA(cudaMemcpyAsync(dy_dev, dy_host, in_bytes, cudaMemcpyHostToDevice, ctx->s_in));
  LSP_CUDA(cudaEventRecord(ev[2], ctx->s_in));
  LSP_CUDA(cudaStreamWaitEvent(st, ev[1], 0));
  LSP_TRY(lsp_layer_fwd(ctx, x_dev, w, y_dev, saved, ws, stream));
  LSP_CUDA(cudaEventRecord(ev[3], st));
  LSP_CUDA(cudaStreamWaitEvent(ctx->s_out, ev[3], 0));
  LSP_CUDA(cudaMemcpyAsync(y_host, y_dev, n * 4, cudaMemcpyDeviceToHost, ctx->s_out));
  LSP_CUDA(cudaStreamWaitEvent(st, ev[2], 0));
  LSP_TRY(lsp_layer_bwd(ctx, x_dev, dy_dev, w, saved, dx_dev, g, ws, stream));
  LSP_CUDA(cudaEventRecord(ev[4], st));
  LSP_CUDA(cudaStreamWaitEvent(ctx->s_out, ev[4], 0));
  LSP_CUDA(cudaMemcpyAsync(dx_host, dx_dev, n * 4, cudaMemcpyDeviceToHost, ctx->s_out));
  LSP_CUDA(cudaEventRecord(ev[5], ctx->s_out));
  LSP_CUDA(cudaStreamWaitEvent(st, ev[5], 0));
  return LSP_OK;
}

// Pipelined variant: consecutive calls overlap -- the uploads of step i+1 run during the compute of step i, the
// downloads of step i during the compute of step i+1 (PCIe is full duplex).  Hazards are ordered with per-parity events:
//   x_dev / dy_dev of this call were last read by the backward of the call two steps ago (the caller alternates two
//   staging sets); y_dev / dx_dev, if they are the previous call's, are rewritten only after their downloads.
lsp_status lsp_layer_step_host_async(lsp_ctx* ctx, const void* x_host, const void* dy_host, const lsp_layer_weights* w,
                                     void* y_host, void* dx_host, lsp_layer_wgrads* g, void* x_dev, void* dy_dev, void* y_dev,
                                     void* dx_dev, void* saved, void* ws, void* stream) {
  if (!ctx || !x_host || !dy_host || !y_host || !dx_host || !x_dev || !dy_dev || !y_dev || !dx_dev) return LSP_EINVAL;
  LSP_ENTER(ctx);
  cudaStream_t st = static_cast<cudaStream_t>(stream);
  const size_t n = static_cast<size_t>(ctx->T) * ctx->d.hidden;
  const size_t in_bytes = n * (ctx->d.in_dtype == LSP_F32 ? 4 : 2);
  const int p = static_cast<int>(ctx->host_seq & 1), q = p ^ 1;
  enum { E_X = 0, E_DY, E_FWD, E_BWD, E_Y, E_DX };
  cudaEvent_t* e = ctx->pev[p];
  cudaEvent_t* eq = ctx->pev[q];
  const bool first = ctx->host_seq == 0;
  // uploads: after whatever `stream` held when the pipeline started, and after the backward that last read this staging set
  if (first) {
    LSP_CUDA(cudaEventRecord(ctx->ev[0], st));
    LSP_CUDA(cudaStreamWaitEvent(ctx->s_in, ctx->ev[0], 0));
    LSP_CUDA(cudaStreamWaitEvent(ctx->s_out, ctx->ev[0], 0));
  }
  if (ctx->host_seq >= 2) LSP_CUDA(cudaStreamWaitEvent(ctx->s_in, e[E_BWD], 0));
  LSP_CUDA(cudaMemcpyAsync(x_dev, x_host, in_bytes, cudaMemcpyHostToDevice, ctx->s_in));
  LSP_CUDA(cudaEventRecord(e[E_X], ctx->s_in));
  LSP_CUDA(cudaMemcpyAsync(dy_dev, dy_host, in_bytes, cudaMemcpyHostToDevice, ctx->s_in));
  LSP_CUDA(cudaEventRecord(e[E_DY], ctx->s_in));
  // forward
  LSP_CUDA(cudaStreamWaitEvent(st, e[E_X], 0));
  if (!first && y_dev == ctx->prev_y_dev) LSP_CUDA(cudaStreamWaitEvent(st, eq[E_Y], 0));
  // alternating result buffers: this y_dev was downloaded by the call two steps ago (same parity: e[E_Y] still holds that
  // record; it is re-recorded below, after this wait has been enqueued)
  if (ctx->host_seq >= 2) LSP_CUDA(cudaStreamWaitEvent(st, e[E_Y], 0));
  LSP_TRY(lsp_layer_fwd(ctx, x_dev, w, y_dev, saved, ws, stream));
  LSP_CUDA(cudaEventRecord(e[E_FWD], st));
  LSP_CUDA(cudaStreamWaitEvent(ctx->s_out, e[E_FWD], 0));
  LSP_CUDA(cudaMemcpyAsync(y_host, y_dev, n * 4, cudaMemcpyDeviceToHost, ctx->s_out));
  LSP_CUDA(cudaEventRecord(e[E_Y], ctx->s_out));
  // backward
  LSP_CUDA(cudaStreamWaitEvent(st, e[E_DY], 0));
  if (!first && dx_dev == ctx->prev_dx_dev) LSP_CUDA(cudaStreamWaitEvent(st, eq[E_DX], 0));
  if (ctx->host_seq >= 2) LSP_CUDA(cudaStreamWaitEvent(st, e[E_DX], 0));
  LSP_TRY(lsp_layer_bwd(ctx, x_dev, dy_dev, w, saved, dx_dev, g, ws, stream));
  LSP_CUDA(cudaEventRecord(e[E_BWD], st));
  LSP_CUDA(cudaStreamWaitEvent(ctx->s_out, e[E_BWD], 0));
  LSP_CUDA(cudaMemcpyAsync(dx_host, dx_dev, n * 4, cudaMemcpyDeviceToHost, ctx->s_out));
  LSP_CUDA(cudaEventRecord(e[E_DX], ctx->s_out));
  ctx->prev_y_dev = y_dev; ctx->prev_dx_dev = dx_dev;
  ++ctx->host_seq;
  return LSP_OK;
}

// `stream` waits for every copy the async host steps have issued, and the pipeline restarts (next call is a "first").
lsp_status lsp_host_copies_wait(lsp_ctx* ctx, void* stream) {
  if (!ctx) return LSP_EINVAL;
  LSP_ENTER(ctx);
  cudaStream_t st = static_cast<cudaStream_t>(stream);
  if (ctx->host_seq > 0) {
    LSP_CUDA(cudaEventRecord(ctx->ev[5], ctx->s_out));
    LSP_CUDA(cudaStreamWaitEvent(st, ctx->ev[5], 0));
    LSP_CUDA(cudaEventRecord(ctx->ev[1], ctx->s_in));
    LSP_CUDA(cudaStreamWaitEvent(st, ctx->ev[1], 0));
  }
  ctx->host_seq = 0;
  ctx->prev_y_dev = ctx->prev_dx_dev = nullptr;
  return LSP_OK;
}

namespace {
struct HeadLayout { size_t xn16, rstd, w16, logits, dz16, dxn32, loss_row, dgpart, inv_count, total; };
HeadLayout head_layout(const lsp_ctx* c, int vocab) {
  const size_t T = c->T, H = c->d.hidden, V = vocab;
  size_t o = 0;
  auto take = [&](size_t bytes) { size_t r = o; o += align_up(bytes); return r; };
  HeadLayout h;
  h.xn16 = take(T * H * 2); h.rstd = take(T * 4); h.w16 = take(V * H * 2); h.logits = take(T * V * 4);
  h.dz16 = take(T * V * 2); h.dxn32 = take(T * H * 4); h.loss_row = take(T * 4);
  h.dgpart = take(static_cast<size_t>(c->norm_blocks) * 2 * H * 4);
  h.inv_count = take(4);
  h.total = o;
  return h;
}
}  // namespace

size_t lsp_head_workspace_bytes(const lsp_ctx* ctx, int32_t vocab) { return (ctx && vocab > 0) ? head_layout(ctx, vocab).total : 0; }

lsp_status lsp_head_fwd_bwd(lsp_ctx* ctx, const void* x, const void* g_final, const void* w_head, const int32_t* targets,
                            int32_t vocab, float grad_scale, float* loss, float* lse, void* dx, float* dg_final, float* dw_head,
                            void* ws, void* stream) {
  if (!ctx) return LSP_EINVAL;
  LSP_ENTER(ctx);
  const void* ptrs[] = {x, g_final, w_head, targets, loss, lse, dx, dg_final, dw_head, ws};
  LSP_TRY(check_common(ctx, nullptr, ws, 10, ptrs));
  if (vocab <= 0 || vocab % 8) return fail(ctx, LSP_EINVAL, "lsp_head_fwd_bwd: vocab must be a positive multiple of 8");
  if (!(grad_scale > 0.f)) return fail(ctx, LSP_EINVAL, "lsp_head_fwd_bwd: grad_scale must be positive");
  cudaStream_t st = static_cast<cudaStream_t>(stream);
  const int T = ctx->T, H = ctx->d.hidden, V = vocab;
  const HeadLayout L = head_layout(ctx, V);
  __half* xn16 = at<__half>(ws, L.xn16);
  float* rstd = at<float>(ws, L.rstd);
  __half* w16 = at<__half>(ws, L.w16);
  float* logits = at<float>(ws, L.logits);
  __half* dz16 = at<__half>(ws, L.dz16);
  float* dxn32 = at<float>(ws, L.dxn32);
  float* loss_row = at<float>(ws, L.loss_row);
  float* dgpart = at<float>(ws, L.dgpart);
  float* inv_count = at<float>(ws, L.inv_count);
  // final RMSNorm, fp16 copy of the head weights
  LSP_STAGE(ST_NORM_FWD, 1, norm_fwd(ctx, ctx->d.in_dtype, x, g_final, xn16, rstd, st));
  {
    const void* src[1] = {w_head};
    __half* dst[1] = {w16};
    const long long cnt[1] = {static_cast<long long>(V) * H};
    LSP_STAGE(ST_CAST, 1, cast_weights(ctx, 1, src, dst, cnt, st));
  }
  // logits = xn W_head^T (fp32 out)
  LSP_STAGE(ST_HEAD_GEMM, 1, (gemm1<false, false>(ctx, T, V, H, Operand{xn16, H, false}, Operand{w16, H, false}, epi_f32(logits, V), st)));
  // cross-entropy: lse, per-token loss, dz = (softmax - onehot) * 2^12 in fp16
  {
    int blocks = 2 * ctx->num_sms < T ? 2 * ctx->num_sms : T;      // two CTAs of 512 threads per SM: one row reduces while the other streams
    auto launch = [&]() {
      ce_fwd_bwd_kernel<<<blocks, CE_THREADS, 0, st>>>(logits, targets, T, V, lse, loss_row, dz16);
      ce_loss_mean_kernel<<<1, 32, 0, st>>>(loss_row, targets, T, V, loss, inv_count);
      return cudaGetLastError();
    };
    LSP_STAGE(ST_CE, 2, launch());
  }
  // undo the fp16 scaling of dz, apply the 1/T of the mean and the caller's gradient (loss) scale; the device scalar
  // inv_count = T / (number of counted targets) turns 1/T into the mean over the counted tokens (exactly 1 if all count)
  const float alpha = grad_scale / (CE_DZ_SCALE * static_cast<float>(T));
  // dW_head = dz^T xn ; dxn = dz W_head
  {
    EpiF32 e = epi_wgrad(ctx, dw_head, H);
    e.alpha = alpha; e.alpha_dev = inv_count;
    LSP_STAGE(ST_HEAD_GEMM, 1, (gemm1<true, true>(ctx, V, H, T, Operand{dz16, V, true}, Operand{xn16, H, true}, e, st)));
  }
  {
    EpiF32 e = epi_f32(dxn32, H);
    e.alpha = alpha; e.alpha_dev = inv_count;
    LSP_STAGE(ST_HEAD_GEMM, 1, (gemm1<false, true>(ctx, T, H, V, Operand{dz16, V, false}, Operand{w16, H, true}, e, st)));
  }
  // final RMSNorm backward (no residual gradient)
  LSP_STAGE(ST_NORM_BWD, 2, norm_bwd(ctx, ctx->d.in_dtype, LSP_F32, x, rstd, g_final, dxn32, nullptr, static_cast<float*>(dx), nullptr,
                                      dgpart, dg_final, ctx->d.wgrad_accumulate, st));
  return LSP_OK;
}

lsp_status lsp_embed_bwd(lsp_ctx* ctx, const int32_t* ids, const void* dx0, int32_t vocab, float* d_table, void* stream) {
  if (!ctx) return LSP_EINVAL;
  LSP_ENTER(ctx);
  const void* ptrs[] = {ids, dx0, d_table};
  LSP_TRY(check_common(ctx, nullptr, nullptr, 3, ptrs));
  if (vocab <= 0) return fail(ctx, LSP_EINVAL, "lsp_embed_bwd: vocab must be positive");
  cudaStream_t st = static_cast<cudaStream_t>(stream);
  const int T = ctx->T, H = ctx->d.hidden;
  const int acc = ctx->d.wgrad_accumulate;
  if (!acc) LSP_CUDA(cudaMemsetAsync(d_table, 0, static_cast<size_t>(vocab) * H * sizeof(float), st));
  auto launch = [&]() {
    embed_bwd_kernel<<<T, 256, 0, st>>>(ids, static_cast<const float*>(dx0), T, H, d_table, acc);
    return cudaGetLastError();
  };
  LSP_STAGE(ST_EMBED_BWD, 1, launch());
  return LSP_OK;
}

lsp_status lsp_adamw_step(lsp_ctx* ctx, int ntensors, const lsp_adamw_tensor* tensors, const lsp_adamw_desc* desc,
                          float* gnorm_out, void* stream) {
  if (!ctx || !tensors || !desc || !gnorm_out) return LSP_EINVAL;
  LSP_ENTER(ctx);
  if (ntensors < 1 || ntensors > OPT_MAX_TENSORS * OPT_MAX_CHUNKS)
    return fail(ctx, LSP_EINVAL, "lsp_adamw_step: 1 <= ntensors <= %d", OPT_MAX_TENSORS * OPT_MAX_CHUNKS);
  if (desc->step < 1 || !(desc->beta1 >= 0.f && desc->beta1 < 1.f) || !(desc->beta2 >= 0.f && desc->beta2 < 1.f) || !(desc->clip_norm > 0.f) ||
      !(desc->grad_scale > 0.f))
    return fail(ctx, LSP_EINVAL, "lsp_adamw_step: bad hyper-parameters");
  for (int i = 0; i < ntensors; ++i) {
    const lsp_adamw_tensor& x = tensors[i];
    if (!x.grad || !x.master || !x.m || !x.v || x.n <= 0 || (x.n % 4)) return fail(ctx, LSP_EINVAL, "lsp_adamw_step: tensor %d: NULL pointer or n %% 4 != 0", i);
    if (!aligned(x.grad, 16) || !aligned(x.master, 16) || !aligned(x.m, 16) || !aligned(x.v, 16) || (x.weight_bf16 && !aligned(x.weight_bf16, 8)) ||
        (x.weight_f16 && !aligned(x.weight_f16, 8)))
      return fail(ctx, LSP_EALIGN, "lsp_adamw_step: tensor %d is not 16-byte aligned", i);
  }
  OptHyper h;
  h.lr = desc->lr; h.beta1 = desc->beta1; h.beta2 = desc->beta2; h.eps = desc->eps; h.weight_decay = desc->weight_decay;
  h.inv_bc1 = static_cast<float>(1.0 / (1.0 - pow(static_cast<double>(desc->beta1), desc->step)));
  h.inv_bc2 = static_cast<float>(1.0 / (1.0 - pow(static_cast<double>(desc->beta2), desc->step)));
  cudaStream_t st = static_cast<cudaStream_t>(stream);
  // The tensors go to the kernels in groups of OPT_MAX_TENSORS (the segment table is a kernel parameter); every group
  // writes its own range of partial sums, one final kernel turns all of them into the global norm, then the groups update.
  const int ngroups = (ntensors + OPT_MAX_TENSORS - 1) / OPT_MAX_TENSORS;
  const long long cap = opt_blocks_cap(ctx->num_sms);
  auto group = [&](int gi, OptTensors& t) {
    memset(&t, 0, sizeof(t));
    const int i0 = gi * OPT_MAX_TENSORS;
    t.n = ntensors - i0 < OPT_MAX_TENSORS ? ntensors - i0 : OPT_MAX_TENSORS;
    for (int i = 0; i < t.n; ++i) {
      const lsp_adamw_tensor& x = tensors[i0 + i];
      t.g[i] = static_cast<const float*>(x.grad); t.p[i] = x.master; t.m[i] = x.m; t.v[i] = x.v;
      t.w[i] = static_cast<__nv_bfloat16*>(x.weight_bf16);
      t.w16[i] = static_cast<__half*>(x.weight_f16);
      t.start[i + 1] = t.start[i] + x.n / 4;
      if (x.decay) t.decay_mask |= 1u << i;
    }
    for (int i = t.n; i < OPT_MAX_TENSORS; ++i) t.start[i + 1] = t.start[t.n];
    long long blocks = (t.start[t.n] + OPT_THREADS - 1) / OPT_THREADS;
    return static_cast<int>(blocks > cap ? cap : blocks);
  };
  const int phase = desc->phase;
  if (phase < 0 || phase > 2) return fail(ctx, LSP_EINVAL, "lsp_adamw_step: phase must be 0, 1 or 2");
  auto launch = [&]() {
    OptTensors t;
    if (phase != 2) {                       // squared norm of the call's gradients
      int nparts = 0;
      for (int gi = 0; gi < ngroups; ++gi) {
        const int nb = group(gi, t);
        opt_gradsq_kernel<<<nb, OPT_THREADS, 0, st>>>(t, ctx->opt_partial + nparts);
        nparts += nb;
      }
      opt_norm_final_kernel<<<1, OPT_THREADS, 0, st>>>(ctx->opt_partial, nparts, desc->clip_norm, 1.0 / desc->grad_scale, phase == 1, gnorm_out);
    } else {                                // gnorm_out[0] holds the GLOBAL sum of g^2 (all ranks): norm and coefficient from it
      opt_norm_final_kernel<<<1, OPT_THREADS, 0, st>>>(gnorm_out, 1, desc->clip_norm, 1.0 / desc->grad_scale, 0, gnorm_out);
    }
    if (phase != 1) {
      for (int gi = 0; gi < ngroups; ++gi) {
        const int nb = group(gi, t);
        opt_adamw_kernel<<<nb, OPT_THREADS, 0, st>>>(t, h, gnorm_out);
      }
    }
    return cudaGetLastError();
  };
  LSP_STAGE(ST_ADAMW, (phase == 0 ? 2 : 1) * ngroups + 1, launch());
  return LSP_OK;
}

// Allocation-free variant of the gradient-norm pass above (include/lsp.h): the same two kernels, the same blocks per
// group and the same reduction order as lsp_adamw_step phase 0 -- hence the same bits -- with the partial sums in the
// device array g_norm_static_scratch instead of the context's cudaMalloc'ed buffer.  No context, no allocation.
lsp_status lsp_grad_norm_static(int cuda_device, int ntensors, const float* const* grads, const int64_t* n, float clip_norm,
                                float grad_scale, float* gnorm_out, void* stream, char* err, size_t err_len) {
  if (err && err_len) err[0] = 0;
  if (!grads || !n || !gnorm_out) return fail_msg(err, err_len, LSP_EINVAL, "lsp_grad_norm_static: NULL argument");
  if (ntensors < 1) return fail_msg(err, err_len, LSP_EINVAL, "lsp_grad_norm_static: ntensors must be >= 1");
  if (ntensors > LSP_NORM_STATIC_MAX_TENSORS)
    return fail_msg(err, err_len, LSP_EINVAL, "lsp_grad_norm_static: %d tensors exceed the maximum of %d (LSP_NORM_STATIC_MAX_TENSORS); use lsp_adamw_step",
                    ntensors, LSP_NORM_STATIC_MAX_TENSORS);
  if (!(clip_norm > 0.f) || !(grad_scale > 0.f)) return fail_msg(err, err_len, LSP_EINVAL, "lsp_grad_norm_static: clip_norm and grad_scale must be > 0");
  if (cuda_device < 0 || cuda_device >= NORM_STATIC_MAX_DEVICES)
    return fail_msg(err, err_len, LSP_EINVAL, "lsp_grad_norm_static: device %d outside [0, %d)", cuda_device, NORM_STATIC_MAX_DEVICES);
  for (int i = 0; i < ntensors; ++i) {
    if (!grads[i] || n[i] <= 0 || (n[i] % 4)) return fail_msg(err, err_len, LSP_EINVAL, "lsp_grad_norm_static: tensor %d: NULL pointer or n %% 4 != 0", i);
    if (!aligned(grads[i], 16)) return fail_msg(err, err_len, LSP_EALIGN, "lsp_grad_norm_static: tensor %d is not 16-byte aligned", i);
  }
  DeviceGuard guard(cuda_device);
  if (!guard.ok) return fail_msg(err, err_len, LSP_ECUDA, "lsp_grad_norm_static: cannot make device %d current", cuda_device);
  NormStaticDevice dv;
  LSP_TRY(norm_static_setup(cuda_device, &dv, err, err_len));
  // groups of OPT_MAX_TENSORS tensors, blocks per group as in lsp_adamw_step; all partial sums must fit the array
  const int ngroups = (ntensors + OPT_MAX_TENSORS - 1) / OPT_MAX_TENSORS;
  const long long cap = opt_blocks_cap(dv.num_sms);
  const long long capacity = LSP_NORM_STATIC_SCRATCH_BYTES / sizeof(float);
  auto group = [&](int gi, OptTensors& t) {
    memset(&t, 0, sizeof(t));
    const int i0 = gi * OPT_MAX_TENSORS;
    t.n = ntensors - i0 < OPT_MAX_TENSORS ? ntensors - i0 : OPT_MAX_TENSORS;
    for (int i = 0; i < t.n; ++i) {
      t.g[i] = grads[i0 + i];
      t.start[i + 1] = t.start[i] + n[i0 + i] / 4;
    }
    for (int i = t.n; i < OPT_MAX_TENSORS; ++i) t.start[i + 1] = t.start[t.n];
    const long long blocks = (t.start[t.n] + OPT_THREADS - 1) / OPT_THREADS;
    return static_cast<int>(blocks > cap ? cap : blocks);
  };
  OptTensors t;
  long long need = 0;
  for (int gi = 0; gi < ngroups; ++gi) need += group(gi, t);
  if (need > capacity)
    return fail_msg(err, err_len, LSP_EINVAL, "lsp_grad_norm_static: %lld partial sums exceed the %lld of the static scratch (LSP_NORM_STATIC_SCRATCH_BYTES)",
                    need, capacity);
  cudaStream_t st = static_cast<cudaStream_t>(stream);
  int nparts = 0;
  for (int gi = 0; gi < ngroups; ++gi) {
    const int nb = group(gi, t);
    opt_gradsq_kernel<<<nb, OPT_THREADS, 0, st>>>(t, dv.scratch + nparts);
    nparts += nb;
  }
  opt_norm_final_kernel<<<1, OPT_THREADS, 0, st>>>(dv.scratch, nparts, clip_norm, 1.0 / grad_scale, 0, gnorm_out);
  const cudaError_t e = cudaGetLastError();
  if (e != cudaSuccess) return fail_msg(err, err_len, LSP_ECUDA, "lsp_grad_norm_static: launch failed: %s", cudaGetErrorString(e));
  return LSP_OK;
}

double lsp_lr_cosine(int step, double lr_max, double lr_min, int warmup, int total) {
  if (warmup > 0 && step <= warmup) return lr_max * step / warmup;
  if (step >= total) return lr_min;
  return lr_min + 0.5 * (lr_max - lr_min) * (1.0 + cos(3.14159265358979323846 * (step - warmup) / (total - warmup)));
}

lsp_status lsp_set_packed_sequences(lsp_ctx* ctx, const int32_t* cu_seqlens_host, int32_t n_seqs, void* stream) {
  if (!ctx) return LSP_EINVAL;
  LSP_ENTER(ctx);
  if (n_seqs == 0) { ctx->doc_on = 0; return LSP_OK; }
  if (!cu_seqlens_host || n_seqs < 0) return LSP_EINVAL;
  if (ctx->d.batch != 1 || ctx->d.head_dim != 128)
    return fail(ctx, LSP_EUNSUPPORTED, "packed sequences need batch = 1 (seq = total tokens) and head_dim = 128");
  const int T = ctx->T;
  if (cu_seqlens_host[0] != 0 || cu_seqlens_host[n_seqs] != T) return fail(ctx, LSP_EINVAL, "cu_seqlens must run from 0 to batch*seq");
  std::vector<int> host(2 * static_cast<size_t>(T));
  for (int i = 0; i < n_seqs; ++i) {
    const int a = cu_seqlens_host[i], b = cu_seqlens_host[i + 1];
    if (b <= a) return fail(ctx, LSP_EINVAL, "cu_seqlens must be strictly increasing (sequence %d is empty)", i);
    for (int t = a; t < b; ++t) { host[t] = a; host[T + t] = b; }
  }
  ctx->doc_end = ctx->doc_start + T;
  // pageable source: the copy has left the host buffer when the call returns
  LSP_CUDA(cudaMemcpyAsync(ctx->doc_start, host.data(), host.size() * sizeof(int), cudaMemcpyHostToDevice, static_cast<cudaStream_t>(stream)));
  ctx->doc_on = 1;
  return LSP_OK;
}

long long lsp_launch_count(const lsp_ctx* ctx) { return ctx ? ctx->launches : -1; }

#ifdef LSP_GEMM_TRACE
// debug builds only (not declared in lsp.h): copies the last pair-GEMM launch's MMA-warp wait counters to the host
int lsp_debug_read_gemm_trace(long long* host, int n) {
  if (!host || n > 128 * 4) return -1;
  if (cudaDeviceSynchronize() != cudaSuccess) return -1;
  return cudaMemcpyFromSymbol(host, g_gemm_trace, static_cast<size_t>(n) * sizeof(long long)) == cudaSuccess ? 0 : -1;
}
#endif
#ifdef LSP_ATTN_TRACE
// debug builds only (not declared in lsp.h): copies the forward attention kernel's clock trace to the host
int lsp_debug_read_trace(unsigned long long* host, int n) {
  return cudaMemcpyFromSymbol(host, g_atc_trace, sizeof(unsigned long long) * n) == cudaSuccess ? 0 : -1;
}
#endif

lsp_status lsp_timing_enable(lsp_ctx* ctx, int max_records) {
  if (!ctx || max_records < 0) return LSP_EINVAL;
  LSP_ENTER(ctx);
  if (ctx->recs) {
    for (TimingRec& r : *ctx->recs) { cudaEventDestroy(r.beg); cudaEventDestroy(r.end); }
    delete ctx->recs;
    ctx->recs = nullptr;
  }
  ctx->timing_on = 0;
  ctx->recs_used = 0;
  if (max_records == 0) return LSP_OK;
  ctx->recs = new (std::nothrow) std::vector<TimingRec>(max_records);
  if (!ctx->recs) return LSP_ENOMEM;
  for (TimingRec& r : *ctx->recs) {
    r.stage = -1;
    if (cudaEventCreate(&r.beg) != cudaSuccess || cudaEventCreate(&r.end) != cudaSuccess)
      return fail(ctx, LSP_ECUDA, "cudaEventCreate failed");
  }
  ctx->timing_on = 1;
  return LSP_OK;
}

int lsp_timing_read(lsp_ctx* ctx, int max_stages, const char** names, float* total_ms, int* records) {
  if (!ctx || !names || !total_ms || !records) return -1;
  const int n = max_stages < ST_COUNT ? max_stages : ST_COUNT;
  for (int i = 0; i < n; ++i) { names[i] = STAGE_NAMES[i]; total_ms[i] = 0.f; records[i] = 0; }
  if (ctx->recs) {
    for (int i = 0; i < ctx->recs_used; ++i) {
      TimingRec& r = (*ctx->recs)[i];
      if (r.stage < 0 || r.stage >= n) continue;
      if (cudaEventSynchronize(r.end) != cudaSuccess) return -1;
      float ms = 0.f;
      if (cudaEventElapsedTime(&ms, r.beg, r.end) != cudaSuccess) return -1;
      total_ms[r.stage] += ms;
      records[r.stage] += 1;
    }
    ctx->recs_used = 0;
  }
  return n;
}

}  // extern "C"
