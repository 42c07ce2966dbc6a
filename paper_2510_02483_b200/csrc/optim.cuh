// Optimizer step after the layer backward (Table 2): AdamW [40] with
// global-norm gradient clipping, fp32 master weights and moments, bf16 model weights (BF16 mixed precision).
// HBM-bound multi-tensor kernels (16 tensors per launch, any number of tensors per step in groups of 16): the squared-norm pass reads 4 B per parameter, the update reads 16 B and writes
// 14 B per parameter (g, p, m, v in; p, m, v, bf16 w out).  The clip coefficient stays on the device (no host sync);
// all reductions run in a fixed order (bit-reproducible).
#pragma once
#include "ptx.cuh"

namespace lsp {

constexpr int OPT_MAX_TENSORS = 16;
constexpr int OPT_THREADS = 256;
constexpr int OPT_MAX_CHUNKS = 64;          // groups of OPT_MAX_TENSORS tensors per lsp_adamw_step call
inline long long opt_blocks_cap(int num_sms) { return num_sms * 8LL; }      // blocks per group (grid-stride beyond)

struct OptTensors {
  const float* g[OPT_MAX_TENSORS];
  float* p[OPT_MAX_TENSORS];
  float* m[OPT_MAX_TENSORS];
  float* v[OPT_MAX_TENSORS];
  __nv_bfloat16* w[OPT_MAX_TENSORS];
  __half* w16[OPT_MAX_TENSORS];              // optional fp16 operand copy of the new bf16 weight (lsp_adamw_tensor.weight_f16)
  long long start[OPT_MAX_TENSORS + 1];      // prefix sums of the tensor sizes in float4 units
  unsigned int decay_mask;                   // bit i: weight decay applies to tensor i
  int n;
};
struct OptHyper {
  float lr, beta1, beta2, eps, weight_decay;
  float inv_bc1, inv_bc2;                    // 1 / (1 - beta^t), evaluated in fp64 on the host
};

__device__ __forceinline__ int opt_segment(const OptTensors& t, long long i) {
  int s = 0;
#pragma unroll
  for (int k = 1; k < OPT_MAX_TENSORS; ++k) s += (k < t.n && i >= t.start[k]) ? 1 : 0;
  return s;
}

// partial[block] = sum of g^2 over the float4 units this block visits (grid-stride: a fixed assignment)
__global__ void __launch_bounds__(OPT_THREADS) opt_gradsq_kernel(const OptTensors t, float* __restrict__ partial) {
  __shared__ float red[OPT_THREADS / 32];
  const long long total = t.start[t.n];
  float acc = 0.f;
  for (long long i = static_cast<long long>(blockIdx.x) * blockDim.x + threadIdx.x; i < total; i += static_cast<long long>(gridDim.x) * blockDim.x) {
    const int s = opt_segment(t, i);
    const float4 g = __ldg(reinterpret_cast<const float4*>(t.g[s]) + (i - t.start[s]));
    acc += g.x * g.x + g.y * g.y + g.z * g.z + g.w * g.w;
  }
#pragma unroll
  for (int off = 16; off > 0; off >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, off);
  if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = acc;
  __syncthreads();
  if (threadIdx.x == 0) {
    float b = 0.f;
#pragma unroll
    for (int k = 0; k < OPT_THREADS / 32; ++k) b += red[k];
    partial[blockIdx.x] = b;
  }
}

// raw_sum: out[0] = sum of the partials (nothing else).  Otherwise:
// out[0] = global l2 norm of the true gradients g / grad_scale, out[1] = the factor the update applies to the stored
// gradients = min(1, clip / (norm + 1e-6)) / grad_scale; one block, fp64, fixed order: thread i sums the
// partials i, i + 256, ... in that order, then thread 0 adds the 256 thread sums in index order.
// A non-finite norm (an inf / NaN gradient: e.g. an fp16 operand overflow upstream) makes the step a NO-OP: out[0]
// carries the non-finite norm as the flag, out[1] = 0, and opt_adamw_kernel leaves p, m, v and the weights untouched
// (without this, c = clip / inf = 0 and g * c = inf * 0 = NaN would be written into the state for good).
__global__ void __launch_bounds__(OPT_THREADS) opt_norm_final_kernel(const float* __restrict__ partial, int nparts, float clip,
                                                                     double inv_scale, int raw_sum, float* __restrict__ out) {
  __shared__ double red[OPT_THREADS];
  double s = 0.0;
  for (int i = threadIdx.x; i < nparts; i += OPT_THREADS) s += static_cast<double>(partial[i]);
  red[threadIdx.x] = s;
  __syncthreads();
  if (threadIdx.x == 0) {
    double tot = 0.0;
    for (int i = 0; i < OPT_THREADS; ++i) tot += red[i];
    if (raw_sum) { out[0] = static_cast<float>(tot); return; }      // phase 1 of a sharded step: this rank's sum of g^2
    const double norm = sqrt(tot) * inv_scale;
    out[0] = static_cast<float>(norm);
    if (!isfinite(norm) || !isfinite(static_cast<float>(norm))) { out[1] = 0.f; return; }      // skip-step flag
    const double c = static_cast<double>(clip) / (norm + 1e-6);
    out[1] = static_cast<float>((c < 1.0 ? c : 1.0) * inv_scale);
  }
}

// m <- b1 m + (1 - b1) g ; v <- b2 v + (1 - b2) g^2 ; p <- p - lr (m_hat / (sqrt(v_hat) + eps) + wd p) ; w = bf16(p)
// Two float4 units per thread and iteration: eight independent 16-byte loads in flight before the first store.
__global__ void __launch_bounds__(OPT_THREADS) opt_adamw_kernel(const OptTensors t, const OptHyper h, const float* __restrict__ norm_coef) {
  const long long total = t.start[t.n];
  const float c = norm_coef[1];
  if (!(c > 0.f)) return;                    // non-finite gradient norm: skipped step (see opt_norm_final_kernel)
  const long long stride = static_cast<long long>(gridDim.x) * blockDim.x;
  for (long long i0 = static_cast<long long>(blockIdx.x) * blockDim.x + threadIdx.x; i0 < total; i0 += 2 * stride) {
    float4 g4[2], p4[2], m4[2], v4[2];
    int sg[2];
    long long jj[2];
#pragma unroll
    for (int u = 0; u < 2; ++u) {
      const long long i = i0 + u * stride;
      sg[u] = 0; jj[u] = 0;
      if (i < total) {
        sg[u] = opt_segment(t, i);
        jj[u] = i - t.start[sg[u]];
        g4[u] = __ldg(reinterpret_cast<const float4*>(t.g[sg[u]]) + jj[u]);
        p4[u] = reinterpret_cast<float4*>(t.p[sg[u]])[jj[u]];
        m4[u] = reinterpret_cast<float4*>(t.m[sg[u]])[jj[u]];
        v4[u] = reinterpret_cast<float4*>(t.v[sg[u]])[jj[u]];
      }
    }
#pragma unroll
    for (int u = 0; u < 2; ++u) {
      if (i0 + u * stride >= total) continue;
      const int s = sg[u];
      const long long j = jj[u];
      const float wd = ((t.decay_mask >> s) & 1u) ? h.weight_decay : 0.f;
      const float g[4] = {g4[u].x * c, g4[u].y * c, g4[u].z * c, g4[u].w * c};
      float p[4] = {p4[u].x, p4[u].y, p4[u].z, p4[u].w}, m[4] = {m4[u].x, m4[u].y, m4[u].z, m4[u].w},
            v[4] = {v4[u].x, v4[u].y, v4[u].z, v4[u].w};
#pragma unroll
      for (int e = 0; e < 4; ++e) {
        m[e] = h.beta1 * m[e] + (1.0f - h.beta1) * g[e];
        v[e] = h.beta2 * v[e] + (1.0f - h.beta2) * g[e] * g[e];
        const float m_hat = m[e] * h.inv_bc1, v_hat = v[e] * h.inv_bc2;
        p[e] = p[e] - h.lr * (m_hat / (sqrtf(v_hat) + h.eps) + wd * p[e]);
      }
      reinterpret_cast<float4*>(t.p[s])[j] = make_float4(p[0], p[1], p[2], p[3]);
      reinterpret_cast<float4*>(t.m[s])[j] = make_float4(m[0], m[1], m[2], m[3]);
      reinterpret_cast<float4*>(t.v[s])[j] = make_float4(v[0], v[1], v[2], v[3]);
      const uint2 wb = make_uint2(pack_bf16(p[0], p[1]), pack_bf16(p[2], p[3]));
      if (t.w[s]) reinterpret_cast<uint2*>(t.w[s])[j] = wb;
      if (t.w16[s])                          // fp16 of the bf16-ROUNDED weight: what the forward's own cast would produce
        reinterpret_cast<uint2*>(t.w16[s])[j] = make_uint2(pack_f16(bf16_lo(wb.x), bf16_hi(wb.x)), pack_f16(bf16_lo(wb.y), bf16_hi(wb.y)));
    }
  }
}

}  // namespace lsp
