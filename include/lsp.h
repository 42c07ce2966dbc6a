/* liblsp -- C ABI of the B200-native (sm_100a) Llama decoder-layer forward+backward.
 *
 * The hot path is the one the Litespark report says its optimisations target: "the attention and MLP
 * blocks" and their "forward and backward pass operations" (section 1) of a Llama layer
 * built from RMSNorm [34], SwiGLU [35], RoPE [36] and GQA [37]/MHA (section 2.4), trained in
 * BF16 mixed precision (section 2.5.2).  The paper gives no API; the calls below follow its
 * statement of the problem -- one training step of one transformer layer -- in the reading fixed in
 * DESIGN.md (SURVEY.md section 8(b),(c)).
 *
 * General contract
 *  - Every pointer is a DEVICE pointer unless marked (host).  All buffers are caller-owned; the library never
 *    allocates, frees or synchronises outside lsp_create / lsp_destroy.  All work is enqueued on `stream`
 *    (a cudaStream_t passed as void*; NULL = legacy default stream).
 *  - Layouts are row-major.  Tokens are sequence-major: token t = b*seq + s is row t of every [T,*] tensor,
 *    T = batch*seq; every sequence starts at position 0.
 *  - Weights are bf16, [out,in] (wq [Nq,H], wk/wv [Nkv,H], wo [H,Nq], w_gate/w_up [F,H], w_down [H,F]);
 *    gains g_attn/g_mlp bf16 [H].  Nq = n_q_heads*head_dim, Nkv = n_kv_heads*head_dim.
 *  - Inputs x, a, dy, da are `in_dtype` (bf16 or fp32) at the public entry points; every output activation
 *    (a, y, dx, da) and every weight/gain gradient is fp32 (DESIGN.md precision plan P-1).
 *  - `saved` (lsp_saved_bytes) is written by a forward call and read by the matching backward call.
 *    `ws` (lsp_workspace_bytes) is scratch whose contents are undefined between calls.  Both must be
 *    256-byte aligned.  All other pointers must be 16-byte aligned.
 *  - Errors: every call returns an lsp_status; nothing throws or aborts across the ABI.  On error
 *    lsp_last_error(ctx) returns a ctx-owned message.  There is no CPU fallback.
 *  - Results are bit-reproducible run to run (no floating-point atomics anywhere).
 *  - Launches: the kernels of a call are enqueued on the caller's stream with programmatic dependent launch between them
 *    (each kernel waits for its predecessor's completion before its first global-memory access, so ordering is what plain
 *    stream order gives; capture into CUDA graphs works).  Environment switches, read once per process, tuning aids only:
 *    LSP_PDL=0 (ordinary launches) and LSP_GEMM_BAND=n (rasterisation band) change no result bit; LSP_GEMM_STREAMK=0 (no
 *    split-K tail), LSP_GEMM_PAIR=0 (single-CTA GEMM kernel) and LSP_GEMM_MT=2 (512-row pair tiles) change which tiles are
 *    summed in K-slices, i.e. the fp32 summation order of those tiles (equal to round-off, still reproducible run to run).
 */
#ifndef LSP_H_
#define LSP_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct lsp_ctx lsp_ctx;

typedef enum {
  LSP_OK = 0,
  LSP_EINVAL = -1,        /* bad argument / NULL pointer */
  LSP_EUNSUPPORTED = -2,  /* shape or option not supported (never a silent fallback) */
  LSP_ENOMEM = -3,
  LSP_ECUDA = -4,         /* a CUDA call or launch failed; see lsp_last_error */
  LSP_EALIGN = -5         /* pointer alignment violated */
} lsp_status;

typedef enum { LSP_BF16 = 0, LSP_F32 = 1, LSP_F16 = 2 } lsp_dtype;

/* One decoder layer (Table 1 / section 2.4; BASELINE.json configs). */
typedef struct {
  int32_t batch, seq, hidden, n_q_heads, n_kv_heads, head_dim, ffn;
  float rms_eps;            /* inside the sqrt, added to mean(x^2) (reading A-3) */
  double rope_base;         /* theta_i = pos * base^(-2i/d), no scaling (reading A-5) */
  int32_t rope_layout;      /* 0 = adjacent pairs (2i,2i+1) as in ref [36]; 1 = half-split pairs (i, i+d/2) */
  int32_t use_rope;         /* 1 in the layer path; 0 = no rotation */
  int32_t in_dtype;         /* lsp_dtype of x / a / dy / da inputs */
  int32_t wgrad_accumulate; /* 0 = overwrite the nine weight / gain gradients; 1 = add to what the buffers hold
                             * (micro-batch gradient accumulation: one fp32 add per element, bit-reproducible) */
  int32_t head_dim_logical; /* 0 = head_dim.  Otherwise an even width < head_dim of heads the caller ZERO-PADS to head_dim
                             * (e.g. 104 -> 128, Table 1 30B: hidden 6656 / 64 heads): rows of wq/wk/wv and columns
                             * of wo beyond it are zero in every head; softmax scale 1/sqrt(logical) and RoPE frequencies
                             * base^(-2i/logical), identity on the padding (rope_layout 0 only) */
  int32_t residual_scale_set; /* 0: the residual branches have weight 1 (a = x + attn(x), y = a + mlp(a)) */
  float residual_scale;     /* used when residual_scale_set = 1: a = s*x + attn(x), y = s*a + mlp(a), and s * the incoming
                             * residual gradients in the backward.  Tensor parallelism: every rank holds a
                             * slice of the heads and FFN columns and produces a PARTIAL a / y / da / dx; rank 0 runs with
                             * s = 1, the others with s = 0, and the sum over ranks is the full result (tp.py) */
} lsp_layer_desc;

typedef struct {
  const void *wq, *wk, *wv, *wo, *g_attn, *w_gate, *w_up, *w_down, *g_mlp;   /* bf16 */
  const void* f16_cache;    /* NULL, or lsp_weight_cache_bytes(ctx) bytes (256-byte aligned) holding the fp16 tensor-core
                             * operand copies of THESE seven projection weights, as left by lsp_layer_prepare_weights (or by
                             * lsp_adamw_step through lsp_adamw_tensor.weight_f16).  NULL: every forward call converts the
                             * bf16 weights itself (two cast launches, ~0.6 GB of traffic at the 3B shape) into `saved`.
                             * Non-NULL: forward and backward read the cache and launch no weight cast; the caller must
                             * refresh it whenever the bf16 weights change -- a stale cache is used as is. */
} lsp_layer_weights;

typedef struct {
  void *wq, *wk, *wv, *wo, *g_attn, *w_gate, *w_up, *w_down, *g_mlp;         /* fp32, same shapes */
} lsp_layer_wgrads;

/* Create a context for one layer shape on `cuda_device`.  Checks: n_q_heads % n_kv_heads == 0,
 * head_dim in {64,128}, hidden/ffn/Nq/Nkv multiples of 8, hidden <= 8192.  The only call (with
 * lsp_destroy) that allocates or syncs.  Context-owned device memory: the RoPE cos/sin table [seq, head_dim/2]
 * (angles evaluated in fp64), the split-K partial-accumulator slots of the GEMM tail (one 512 x 256 fp32 slot per SM
 * pair, ~39 MB on a B200) with their publication flags, and the work-queue counters of the persistent attention
 * kernels.  Because those are shared by every call on the context, calls on ONE context must be issued on one
 * stream at a time (use one context per concurrent stream). */
lsp_status lsp_create(lsp_ctx** out, const lsp_layer_desc* desc, int cuda_device);
lsp_status lsp_destroy(lsp_ctx* ctx);
size_t lsp_saved_bytes(const lsp_ctx* ctx);
size_t lsp_workspace_bytes(const lsp_ctx* ctx);
const char* lsp_last_error(const lsp_ctx* ctx);

/* Operand range (reading P-2'; the paper trains in BF16 mixed precision).  The tensor-core
 * operands of this library are fp16: bf16's rate with three more mantissa bits, which is what holds the 2e-2 parity bar
 * for the weight gradients, at the price of bf16's exponent range.  Supported magnitudes of every caller tensor that
 * becomes an operand (weights, dy / da, the attention-core inputs): |v| <= 65504; values below 2^-24 flush to zero.
 * A value beyond the range is NOT turned into inf: the conversion saturates it to +-65504 (NaN stays NaN) and counts it.
 * lsp_overflow_count copies the number of values clamped (or found non-finite) since the last reset to *count (HOST),
 * after synchronising `stream`; reset != 0 zeroes the counter.  A non-zero count means results are outside the parity
 * contract (rescale the loss / gradient: lsp_head_fwd_bwd's grad_scale).  Internal operands (normalised activations,
 * q, k, v, h, ...) are O(1)-O(100) for in-range inputs. */
lsp_status lsp_overflow_count(lsp_ctx* ctx, unsigned long long* count, int reset, void* stream);

/* fp16 operand cache of one layer's projection weights (see lsp_layer_weights.f16_cache): its size, the conversion
 * call (two launches on `stream`; applies the row permutation of rope_layout = 1), and the byte offset inside the cache
 * of tensor `which` (0 wq, 1 wk, 2 wv, 3 wo, 4 w_gate, 5 w_up, 6 w_down; same [out,in] row-major layout as the bf16
 * tensor) for writers that produce the fp16 copy themselves (lsp_adamw_tensor.weight_f16).  The offset is -1 for wq / wk
 * under rope_layout = 1 (their rows are permuted inside the cache: use lsp_layer_prepare_weights) and for a bad index. */
size_t lsp_weight_cache_bytes(const lsp_ctx* ctx);
lsp_status lsp_layer_prepare_weights(lsp_ctx* ctx, const lsp_layer_weights* w, void* cache, void* stream);
long long lsp_weight_cache_offset(const lsp_ctx* ctx, int which);

/* Attention block:  a = x + Wo . GQA(RoPE(Wq xn), RoPE(Wk xn), Wv xn), xn = RMSNorm(x; g_attn).
 *   x [T,H] in_dtype -> a_out [T,H] fp32. */
lsp_status lsp_attn_fwd(lsp_ctx* ctx, const void* x, const lsp_layer_weights* w, void* a_out, void* saved, void* ws,
                        void* stream);
/* Backward of the attention block (B6-B10).  x: the forward input; da [T,H] in_dtype -> dx [T,H] fp32;
 * writes grads->wq, wk, wv, wo, g_attn. */
lsp_status lsp_attn_bwd(lsp_ctx* ctx, const void* x, const void* da, const lsp_layer_weights* w, const void* saved,
                        void* dx, lsp_layer_wgrads* grads, void* ws, void* stream);

/* MLP block (F5-F7):  y = a + Wd . (silu(Wg an) * (Wu an)), an = RMSNorm(a; g_mlp).  a [T,H] in_dtype -> y fp32. */
lsp_status lsp_mlp_fwd(lsp_ctx* ctx, const void* a, const lsp_layer_weights* w, void* y_out, void* saved, void* ws,
                       void* stream);
/* Backward of the MLP block (B1-B5).  a: the forward input; dy in_dtype -> da fp32; writes grads->w_gate,
 * w_up, w_down, g_mlp. */
lsp_status lsp_mlp_bwd(lsp_ctx* ctx, const void* a, const void* dy, const lsp_layer_weights* w, const void* saved,
                       void* da, lsp_layer_wgrads* grads, void* ws, void* stream);

/* Whole layer = mlp o attn.  x in_dtype -> y fp32.  The intermediate `a` (fp32) lives in `saved`. */
lsp_status lsp_layer_fwd(lsp_ctx* ctx, const void* x, const lsp_layer_weights* w, void* y_out, void* saved, void* ws,
                         void* stream);
/* x: the forward input; dy in_dtype -> dx fp32; writes all nine gradients. */
/* Forward pass only (inference-style): the same y as lsp_layer_fwd, bit for bit, without the tensors
 * only a backward pass would read (the fp16 gate / up pre-activations, the fp32 copy of O).  `scratch` is
 * lsp_saved_bytes(ctx) of device memory used for the intermediates; it is NOT a valid `saved` for lsp_layer_bwd. */
lsp_status lsp_layer_fwd_infer(lsp_ctx* ctx, const void* x, const lsp_layer_weights* w, void* y_out, void* scratch, void* ws,
                               void* stream);
lsp_status lsp_layer_bwd(lsp_ctx* ctx, const void* x, const void* dy, const lsp_layer_weights* w, const void* saved,
                         void* dx, lsp_layer_wgrads* grads, void* ws, void* stream);

/* Attention core only (BASELINE.json config 5; no projections, no RoPE):
 *   q [B,S,nq,d], k,v [B,S,nkv,d], d_o [B,S,nq,d] bf16;  o, dq [B,S,nq,d], dk,dv [B,S,nkv,d] fp32;
 *   lse [B,nq,S] fp32 = natural log-sum-exp of the scaled causal logits (reading A-6). */
lsp_status lsp_sdpa_fwd(lsp_ctx* ctx, const void* q, const void* k, const void* v, void* o, float* lse, void* ws,
                        void* stream);
lsp_status lsp_sdpa_bwd(lsp_ctx* ctx, const void* q, const void* k, const void* v, const void* o, const float* lse,
                        const void* d_o, void* dq, void* dk, void* dv, void* ws, void* stream);

/* Embedding gather (config 3):  x0[t,:] = table[ids[t],:]; ids int32 [T], table bf16 [vocab,H] -> x0 fp32 [T,H].
 * Contract: every id is in [0, vocab); ids are used as row indices without a range check (here and in lsp_embed_bwd). */
lsp_status lsp_embed_fwd(lsp_ctx* ctx, const int32_t* ids, const void* table, void* x0, void* stream);

/* Building block / test hook: one bias-free linear-layer GEMM on the tcgen05 kernel, 16-bit in, fp32 out.
 * a_dtype / b_dtype: both LSP_BF16 or both LSP_F16; a mixed pair returns LSP_EUNSUPPORTED (one
 * tcgen05.mma.kind::f16 with unequal operand formats faults on sm_100a).
 *   op 0 (forward): C[M,N] = A[M,K] . B[N,K]^T        A,B row-major as written
 *   op 1 (dgrad)  : C[M,N] = A[M,K] . B[K,N]          B row-major [K,N]
 *   op 2 (wgrad)  : C[M,N] = A[K,M]^T . B[K,N]        A row-major [K,M], B row-major [K,N]
 * lda/ldb/ldc are row pitches in elements (multiples of 8).  Needs no ctx state beyond the device. */
lsp_status lsp_gemm(lsp_ctx* ctx, int op, int M, int N, int K, const void* A, int64_t lda, int a_dtype, const void* B,
                    int64_t ldb, int b_dtype, float* C, int64_t ldc, void* stream);

/* Packed variable-length sequences (the SFT / DPO data layout of PAPER.md:176-186): the context's
 * batch * seq tokens (batch must be 1, head_dim 128) are n_seqs sequences laid end to end, sequence i = tokens
 * [cu_seqlens[i], cu_seqlens[i+1]) with cu_seqlens[0] = 0, cu_seqlens[n_seqs] = batch*seq, strictly increasing (HOST
 * array of n_seqs + 1 entries, read before the call returns).  From then on every attention call of the context is
 * causal WITHIN each sequence (a query sees the keys of its own sequence up to itself; key blocks of other sequences are
 * skipped, not just masked) and RoPE positions restart at 0 at every sequence start.  n_seqs = 0 switches back to
 * `batch` sequences of `seq` tokens.  Enqueues one small copy on `stream`. */
lsp_status lsp_set_packed_sequences(lsp_ctx* ctx, const int32_t* cu_seqlens_host, int32_t n_seqs, void* stream);

/* End-to-end step with HOST buffers (bench.py `e2e`): copies x, dy (in_dtype, [T,H]; pinned host memory for
 * asynchronous copies) to the caller's device staging buffers x_dev / dy_dev, runs lsp_layer_fwd + lsp_layer_bwd,
 * and copies y and dx (fp32 [T,H]) back to y_host / dx_host (no sync).  The copies run on two context-owned streams
 * ordered against `stream` with events, so the upload of dy overlaps the forward pass and the download of y the
 * backward pass; `stream` completes after the last copy.  Weights and
 * weight gradients stay on the device (DEVICE pointers), as they do in a training step. */
lsp_status lsp_layer_step_host(lsp_ctx* ctx, const void* x_host, const void* dy_host, const lsp_layer_weights* w,
                               void* y_host, void* dx_host, lsp_layer_wgrads* grads, void* x_dev, void* dy_dev,
                               void* y_dev, void* dx_dev, void* saved, void* ws, void* stream);

/* Pipelined form of lsp_layer_step_host for a stream of steps: same arguments and results, but the call does NOT make
 * `stream` wait for its downloads, so the uploads of the next step overlap this step's compute and this step's
 * downloads overlap the next step's compute (PCIe is full duplex).  Rules: consecutive calls must ALTERNATE between two
 * (x_dev, dy_dev) staging sets (a set is overwritten by the call two steps later, after the backward that read it);
 * y_dev / dx_dev may be reused every call (the library orders the rewrite after the previous download) or alternated;
 * y_host / dx_host are complete only after lsp_host_copies_wait(ctx, stream) and completion of `stream`. */
lsp_status lsp_layer_step_host_async(lsp_ctx* ctx, const void* x_host, const void* dy_host, const lsp_layer_weights* w,
                                     void* y_host, void* dx_host, lsp_layer_wgrads* grads, void* x_dev, void* dy_dev,
                                     void* y_dev, void* dx_dev, void* saved, void* ws, void* stream);
lsp_status lsp_host_copies_wait(lsp_ctx* ctx, void* stream);

/* Model head (readings H-1 .. H-3 in DESIGN.md section 13): final RMSNorm (gain g_final, the
 * context's rms_eps), bias-free LM head w_head bf16 [vocab, H] ([out,in]), mean next-token cross-entropy, and all their
 * gradients, in one call:  xn = RMSNorm(x; g_final); z = xn w_head^T; loss = mean_t (lse_t - z[t, targets[t]]).
 *   x [T,H] in_dtype (the stack output), targets int32 [T], vocab % 8 == 0.  A target outside [0, vocab) (use a negative
 *   value, e.g. -100: padding, or the last token of each packed sequence) carries no loss (reading H-4): its row adds
 *   nothing to the loss or to any gradient, and the mean is over the COUNTED targets (loss = 0 when none counts).
 *   Outputs: loss DEVICE float[1]; lse fp32 [T] (natural log-sum-exp of the logits); dx fp32 [T,H]; dg_final fp32 [H];
 *   dw_head fp32 [vocab, H].  ws: lsp_head_workspace_bytes(ctx, vocab) bytes of scratch (256-byte aligned); it holds the
 *   fp32 logits [T, vocab] and their fp16 gradient -- 6 bytes per (token, class).
 *   grad_scale > 0 multiplies the three gradients (not the loss): the layers' backward feeds 16-bit tensor-core
 *   operands, and the gradient of a MEAN loss is ~1/T per element, below the fp16 normal range at training sizes; a
 *   training step passes e.g. grad_scale = T and hands the same value to lsp_adamw_step, which divides it out.
 *   On a context created with wgrad_accumulate = 1, dw_head and dg_final are added to (dx is always overwritten). */
size_t lsp_head_workspace_bytes(const lsp_ctx* ctx, int32_t vocab);
lsp_status lsp_head_fwd_bwd(lsp_ctx* ctx, const void* x, const void* g_final, const void* w_head, const int32_t* targets,
                            int32_t vocab, float grad_scale, float* loss, float* lse, void* dx, float* dg_final,
                            float* dw_head, void* ws, void* stream);
/* Embedding backward (H-3): d_table [vocab, H] fp32 (fully written: zero for ids that do not occur) =
 * scatter-add of dx0 fp32 [T,H] by ids int32 [T]; duplicates are added in increasing token order (bit-reproducible).
 * On a context created with wgrad_accumulate = 1 the sums are added to what d_table holds (no zeroing). */
lsp_status lsp_embed_bwd(lsp_ctx* ctx, const int32_t* ids, const void* dx0, int32_t vocab, float* d_table, void* stream);

/* Optimizer step after the backward (Table 2): AdamW with decoupled weight decay
 * and bias-corrected moments (ref [40]), preceded by clipping of the GLOBAL l2 gradient norm over all tensors of the
 * call (readings O-1 .. O-5 in DESIGN.md section 12).  Per tensor i of `n` elements (n % 4 == 0, pointers 16-byte
 * aligned): grad fp32 (read), master / m / v fp32 (updated in place), weight_bf16 (written: round-to-nearest-even of
 * the new master weight; may be NULL), decay = 1 if weight decay applies.  `tensors` is a HOST array of
 * 1 <= ntensors <= 1024 entries (a whole model: the kernels take them in groups of 16, the norm is over all of them).
 * gnorm_out: DEVICE float[2], receives {global norm of the true gradients, factor applied to the stored gradients =
 * clip coefficient / grad_scale} (no host sync).  If the norm is not finite (an inf / NaN gradient) the step is SKIPPED:
 * master, m, v and the weights stay as they are, gnorm_out = {the non-finite norm, 0} is the flag.
 * weight_f16 (may be NULL): also written, as the fp16 value of the new bf16 weight -- point it into the layer's operand
 * cache (lsp_weight_cache_offset) and the next forward needs no weight cast.
 * Everything is enqueued on `stream`; results are bit-reproducible. */
typedef struct {
  const void* grad; float* master; float* m; float* v; void* weight_bf16; int64_t n; int32_t decay;
  void* weight_f16;
} lsp_adamw_tensor;
typedef struct {
  float lr, beta1, beta2, eps, weight_decay, clip_norm;   /* paper: lr from lsp_lr_cosine, 0.90, 0.95, 1e-8, 0.01, 1.0 */
  int32_t step;                                            /* 1-based optimizer step t (bias correction 1 - beta^t) */
  float grad_scale;                                        /* > 0: the stored gradients are grad_scale x the true ones
                                                              (lsp_head_fwd_bwd); norm, clipping and update use g / grad_scale */
  int32_t phase;                                           /* 0: the whole step.  Sharded optimizer state (ZeRO stage 1,
                                                              PAPER.md:73), every rank holding a slice of the tensors:
                                                              1 = only gnorm_out[0] <- sum of g^2 over this call's
                                                              (stored) gradients; the caller all-reduces that scalar;
                                                              2 = gnorm_out[0] holds the global sum: norm, clipping
                                                              coefficient and the update of this call's tensors */
} lsp_adamw_desc;
lsp_status lsp_adamw_step(lsp_ctx* ctx, int ntensors, const lsp_adamw_tensor* tensors, const lsp_adamw_desc* desc,
                          float* gnorm_out, void* stream);
/* Allocation-free global gradient norm: the norm / clipping pass of lsp_adamw_step (clipping of the
 * global l2 gradient norm; readings O-1, O-2 in DESIGN.md section 12) for callers that may not allocate device memory
 * -- code under CUDA-graph capture, tight serving / training loops, harnesses that forbid cudaMalloc.  It needs NO
 * context (lsp_create allocates), calls no cudaMalloc / cudaFree / allocating library routine, and keeps its scratch
 * (the per-block partial sums of g^2) in ONE file-scope device array of LSP_NORM_STATIC_SCRATCH_BYTES that every GPU
 * which loads the library holds until the process exits.
 *   cuda_device: the device the pointers live on (made current for the call, the caller's is restored).
 *   grads[i]: DEVICE fp32 tensor of n[i] elements (n[i] > 0, n[i] % 4 == 0, 16-byte aligned); grads / n are HOST arrays
 *   of 1 <= ntensors <= LSP_NORM_STATIC_MAX_TENSORS entries (the 255 tensors of the 3B model fit).  A call that needs
 *   more tensors, or more partial sums than the array holds, is REJECTED with LSP_EINVAL before anything is launched.
 *   gnorm_out: DEVICE float[2] = {l2 norm of the true gradients g / grad_scale, min(1, clip_norm / (norm + 1e-6)) /
 *   grad_scale} -- bit for bit what lsp_adamw_step (phase 0) writes for the same tensors in the same order; a
 *   non-finite norm gives {norm, 0}.  Enqueued on `stream`, no host sync.
 *   err (may be NULL): caller's HOST buffer of err_len bytes that receives the message of a failed call.
 * The first call on a device resolves the array's address (cudaGetSymbolAddress, once per device): make it outside
 * graph capture.  Nothing in the array has to start at zero (every partial sum the final reduction reads is written by
 * the same call), so the contents a previous call left are never read.  ALL calls on one GPU share the array: calls
 * that may overlap on the GPU (different streams without an ordering between them) race -- order them. */
#define LSP_NORM_STATIC_MAX_TENSORS 256
#define LSP_NORM_STATIC_SCRATCH_BYTES (128 * 1024)
lsp_status lsp_grad_norm_static(int cuda_device, int ntensors, const float* const* grads, const int64_t* n,
                                float clip_norm, float grad_scale, float* gnorm_out, void* stream, char* err,
                                size_t err_len);

/* Host helper (no GPU): the paper's schedule: linear warm-up from 0 to lr_max over `warmup` steps, then
 * cosine decay to lr_min at step `total`, lr_min afterwards (reading O-3).  step is 1-based. */
double lsp_lr_cosine(int step, double lr_max, double lr_min, int warmup, int total);

/* Measurement aids; they change no result.
 * lsp_launch_count: kernels launched through this context so far.
 * lsp_timing_enable(n > 0): pre-create n CUDA-event pairs; from then on every pipeline stage records one pair on
 *   the caller's stream (silently stops recording once the pairs are used up); n = 0 disables and frees them.
 * lsp_timing_read: synchronises the recorded events, sums elapsed milliseconds and record counts per stage into the
 *   caller's HOST arrays (names[i] points at a static string), resets the recorder, returns the number of stages
 *   written (<= max_stages) or -1 on error. */
long long lsp_launch_count(const lsp_ctx* ctx);
lsp_status lsp_timing_enable(lsp_ctx* ctx, int max_records);
int lsp_timing_read(lsp_ctx* ctx, int max_stages, const char** names, float* total_ms, int* records);

#ifdef __cplusplus
}
#endif
#endif /* LSP_H_ */
