// Steps either side of the decoder stack: next-token cross-entropy over the LM-head logits
// (forward value, log-sum-exp and the logit gradient in one kernel) and the embedding backward (deterministic
// scatter-add).  The LM-head projections themselves run on the tcgen05 GEMM of gemm.cuh.  HBM / L2 bound.
#pragma once
#include "ptx.cuh"

namespace lsp {

constexpr int CE_THREADS = 512;
constexpr int CE_UNROLL = 4;               // independent 16-byte loads per thread in flight: 64 KB per SM (8: spills at 64 registers)
constexpr float CE_DZ_SCALE = 4096.0f;     // dz is stored as fp16((softmax - onehot) * 2^12): softmax values ~1/V = 8e-6
                                           // would be fp16 subnormals; the GEMMs that consume dz undo the factor (alpha)

// block-wide (max, sum of exp relative to that max) of per-thread pairs; fixed order, every thread gets the result
__device__ __forceinline__ void ce_block_reduce(float& m, float& s, float2* red) {
#pragma unroll
  for (int off = 16; off > 0; off >>= 1) {
    const float mo = __shfl_xor_sync(0xffffffffu, m, off), so = __shfl_xor_sync(0xffffffffu, s, off);
    const float mn = fmaxf(m, mo);
    s = s * __expf(m - mn) + so * __expf(mo - mn);
    m = mn;
  }
  __syncthreads();
  if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = make_float2(m, s);
  __syncthreads();
  float M = red[0].x;
  for (int k = 1; k < CE_THREADS / 32; ++k) M = fmaxf(M, red[k].x);
  float S = 0.f;
  for (int k = 0; k < CE_THREADS / 32; ++k) S += red[k].y * __expf(red[k].x - M);       // fixed order
  m = M; s = S;
}

// One CTA of 512 threads per token row, two CTAs per SM (grid-stride over rows): one row's block reduction and dz pass
// overlap the other's streaming pass.  Pass 1: running maximum and sum of exp together (online rescaling), four float4
// loads per thread in flight; pass 2: dz from the row, mostly still in L2 (296 rows x 513 KB at V = 128256 is a little
// over the 126 MB L2).  loss_row[t] = lse_t - z[t, y_t].  V % 4 == 0.  Measured at T = 8192, V = 128256: 3.95 ms with
// three passes and one load in flight -> 2.06 ms (6.3 GB of algorithmic traffic: 3.1 TB/s).
// A target outside [0, V) (reading H-4: negative = "no loss at this position", e.g. padding or the last token of a
// packed sequence) is never used as an index: the row's loss is 0 and its dz row is zero; lse is still written.
__global__ void __launch_bounds__(CE_THREADS, 2) ce_fwd_bwd_kernel(const float* __restrict__ z, const int* __restrict__ y, int T, int V,
                                                                   float* __restrict__ lse, float* __restrict__ loss_row,
                                                                   __half* __restrict__ dz) {
  __shared__ float2 red[CE_THREADS / 32];
  const int V4 = V >> 2;
  for (int t = blockIdx.x; t < T; t += gridDim.x) {
    const float4* zr = reinterpret_cast<const float4*>(z + static_cast<long long>(t) * V);
    float m = -1.0e30f, s = 0.f;                    // finite floor: threads that see no element contribute exp(-huge) * 0
    for (int i0 = threadIdx.x; i0 < V4; i0 += CE_UNROLL * CE_THREADS) {
      float4 a[CE_UNROLL];
#pragma unroll
      for (int u = 0; u < CE_UNROLL; ++u) {
        const int i = i0 + u * CE_THREADS;
        a[u] = i < V4 ? __ldg(zr + i) : make_float4(-1.0e30f, -1.0e30f, -1.0e30f, -1.0e30f);
      }
      float mx = m;
#pragma unroll
      for (int u = 0; u < CE_UNROLL; ++u) mx = fmaxf(mx, fmaxf(fmaxf(a[u].x, a[u].y), fmaxf(a[u].z, a[u].w)));
      float add = 0.f;
#pragma unroll
      for (int u = 0; u < CE_UNROLL; ++u)
        add += __expf(a[u].x - mx) + __expf(a[u].y - mx) + __expf(a[u].z - mx) + __expf(a[u].w - mx);
      s = s * __expf(m - mx) + add;
      m = mx;
    }
    ce_block_reduce(m, s, red);
    const float L = m + logf(s);
    const int yt = y[t];
    const bool counted = yt >= 0 && yt < V;
    if (threadIdx.x == 0) {
      lse[t] = L;
      loss_row[t] = counted ? L - z[static_cast<long long>(t) * V + yt] : 0.f;
    }
    uint2* dr = reinterpret_cast<uint2*>(dz + static_cast<long long>(t) * V);
    for (int i0 = threadIdx.x; i0 < V4; i0 += CE_UNROLL * CE_THREADS) {
      float4 a[CE_UNROLL];
#pragma unroll
      for (int u = 0; u < CE_UNROLL; ++u) {
        const int i = i0 + u * CE_THREADS;
        if (i < V4) a[u] = zr[i];
      }
#pragma unroll
      for (int u = 0; u < CE_UNROLL; ++u) {
        const int i = i0 + u * CE_THREADS;
        if (i < V4) {
          float p[4] = {__expf(a[u].x - L), __expf(a[u].y - L), __expf(a[u].z - L), __expf(a[u].w - L)};
          const int c = 4 * i;
          if (!counted) { p[0] = p[1] = p[2] = p[3] = 0.f; }
          if (yt >= c && yt < c + 4) p[yt - c] -= 1.0f;
          dr[i] = make_uint2(pack_f16(p[0] * CE_DZ_SCALE, p[1] * CE_DZ_SCALE), pack_f16(p[2] * CE_DZ_SCALE, p[3] * CE_DZ_SCALE));
        }
      }
    }
  }
}

// loss = mean of loss_row over the COUNTED tokens (targets in [0, V)); one thread, fp64, fixed order.
// inv_count[0] = T / n_counted (0 if none): the factor that turns the 1 / T the gradient GEMMs apply into 1 / n_counted.
__global__ void ce_loss_mean_kernel(const float* __restrict__ loss_row, const int* __restrict__ y, int T, int V,
                                    float* __restrict__ loss, float* __restrict__ inv_count) {
  if (threadIdx.x == 0 && blockIdx.x == 0) {
    double s = 0.0;
    int n = 0;
    for (int t = 0; t < T; ++t) {
      s += static_cast<double>(loss_row[t]);
      n += (y[t] >= 0 && y[t] < V) ? 1 : 0;
    }
    loss[0] = n > 0 ? static_cast<float>(s / n) : 0.f;
    inv_count[0] = n > 0 ? static_cast<float>(static_cast<double>(T) / n) : 0.f;
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
