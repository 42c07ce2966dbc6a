// Steps either side of the decoder stack: next-token cross-entropy over the LM-head logits
// (forward value, log-sum-exp and the logit gradient in one kernel) and the embedding backward (deterministic
// scatter-add).  The LM-head projections themselves run on the tcgen05 GEMM of gemm.cuh.  HBM / L2 bound.
#pragma once
#include "ptx.cuh"

namespace lsp {

constexpr int CE_THREADS = 512;
constexpr float CE_DZ_SCALE = 4096.0f;     // dz is stored as fp16((softmax - onehot) * 2^12): softmax values ~1/V = 8e-6
                                           // would be fp16 subnormals; the GEMMs that consume dz undo the factor (alpha)

__device__ __forceinline__ float ce_block_reduce(float v, float* red, bool is_max) {
#pragma unroll
  for (int off = 16; off > 0; off >>= 1) {
    const float o = __shfl_xor_sync(0xffffffffu, v, off);
    v = is_max ? fmaxf(v, o) : v + o;
  }
  __syncthreads();
  if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = v;
  __syncthreads();
  float t = red[0];
  for (int k = 1; k < CE_THREADS / 32; ++k) t = is_max ? fmaxf(t, red[k]) : t + red[k];   // fixed order
  return t;
}

// One CTA per token row (grid-stride over rows).  Pass 1: row maximum; pass 2: sum of exp (the row is L2-resident:
// 148 CTAs x V x 4 B = 76 MB at V = 128256); pass 3: dz.  loss_row[t] = lse_t - z[t, y_t].
__global__ void __launch_bounds__(CE_THREADS) ce_fwd_bwd_kernel(const float* __restrict__ z, const int* __restrict__ y, int T, int V,
                                                                float* __restrict__ lse, float* __restrict__ loss_row,
                                                                __half* __restrict__ dz) {
  __shared__ float red[CE_THREADS / 32];
  const int V4 = V >> 2;
  for (int t = blockIdx.x; t < T; t += gridDim.x) {
    const float4* zr = reinterpret_cast<const float4*>(z + static_cast<long long>(t) * V);
    float mx = -INFINITY;
    for (int i = threadIdx.x; i < V4; i += CE_THREADS) {
      const float4 a = zr[i];
      mx = fmaxf(mx, fmaxf(fmaxf(a.x, a.y), fmaxf(a.z, a.w)));
    }
    mx = ce_block_reduce(mx, red, true);
    float s = 0.f;
    for (int i = threadIdx.x; i < V4; i += CE_THREADS) {
      const float4 a = zr[i];
      s += __expf(a.x - mx) + __expf(a.y - mx) + __expf(a.z - mx) + __expf(a.w - mx);
    }
    s = ce_block_reduce(s, red, false);
    const float L = mx + logf(s);
    const int yt = y[t];
    if (threadIdx.x == 0) {
      lse[t] = L;
      loss_row[t] = L - z[static_cast<long long>(t) * V + yt];
    }
    uint2* dr = reinterpret_cast<uint2*>(dz + static_cast<long long>(t) * V);
    for (int i = threadIdx.x; i < V4; i += CE_THREADS) {
      const float4 a = zr[i];
      float p[4] = {__expf(a.x - L), __expf(a.y - L), __expf(a.z - L), __expf(a.w - L)};
      const int c = 4 * i;
      if (yt >= c && yt < c + 4) p[yt - c] -= 1.0f;
      dr[i] = make_uint2(pack_f16(p[0] * CE_DZ_SCALE, p[1] * CE_DZ_SCALE), pack_f16(p[2] * CE_DZ_SCALE, p[3] * CE_DZ_SCALE));
    }
  }
}

// loss = mean of loss_row (one thread, fp64, fixed order)
__global__ void ce_loss_mean_kernel(const float* __restrict__ loss_row, int T, float* __restrict__ loss) {
  if (threadIdx.x == 0 && blockIdx.x == 0) {
    double s = 0.0;
    for (int t = 0; t < T; ++t) s += static_cast<double>(loss_row[t]);
    loss[0] = static_cast<float>(s / T);
  }
}

// dE[v,:] = sum over {t : id_t = v} dx0[t,:], tokens added in increasing t (deterministic, no atomics).  One CTA per
// token: the CTA of the FIRST occurrence of an id gathers all later occurrences in order; the others exit.  dE must
// have been zeroed (rows of ids that never occur), or hold the running sum when `accumulate` is set.  O(T^2 / 256) id comparisons per launch: 0.26 M at T = 8192.
__global__ void __launch_bounds__(256) embed_bwd_kernel(const int* __restrict__ ids, const float* __restrict__ dx0, int T, int H,
                                                        float* __restrict__ dE, int accumulate) {
  __shared__ unsigned int hits[8];                    // per warp: ballot of the candidates whose id matches
  __shared__ int any_before;
  const int t = blockIdx.x;
  const int id = ids[t];
  if (threadIdx.x == 0) any_before = 0;
  __syncthreads();
  for (int u = threadIdx.x; u < t; u += 256)
    if (ids[u] == id) any_before = 1;                 // benign race: every writer stores 1
  __syncthreads();
  if (any_before) return;
  float* out = dE + static_cast<long long>(id) * H;
  // this CTA's columns: acc kept in registers for up to 32 floats per thread (H <= 8192)
  float acc[32];
#pragma unroll
  for (int k = 0; k < 32; ++k) acc[k] = 0.f;
  for (int base = t; base < T; base += 256) {
    const int u = base + threadIdx.x;
    const unsigned int b = __ballot_sync(0xffffffffu, u < T && ids[u] == id);
    if ((threadIdx.x & 31) == 0) hits[threadIdx.x >> 5] = b;
    __syncthreads();
    for (int w = 0; w < 8; ++w) {                     // increasing token order: warp 0's lanes first, bit 0 first
      unsigned int mask = hits[w];
      while (mask) {
        const int j = __ffs(mask) - 1;
        mask &= mask - 1;
        const float* src = dx0 + static_cast<long long>(base + 32 * w + j) * H;
#pragma unroll
        for (int k = 0; k < 32; ++k) {
          const int c = threadIdx.x + k * 256;
          if (c < H) acc[k] += src[c];
        }
      }
    }
    __syncthreads();
  }
#pragma unroll
  for (int k = 0; k < 32; ++k) {
    const int c = threadIdx.x + k * 256;
    if (c < H) out[c] = accumulate ? out[c] + acc[k] : acc[k];
  }
}

}  // namespace lsp
