// Memory-bound kernels of the layer: RMSNorm forward/backward (ref [34]; SURVEY 8(a) F1,F5,B5,B10),
// the gain-gradient column reduction, dtype casts and the embedding gather (E0).
// All are vectorised (16-byte accesses), coalesced, warp-shuffle reduced; HBM is the roofline.
#pragma once
#include "ptx.cuh"

namespace lsp {

constexpr int NORM_THREADS = 256;
constexpr int NORM_MAXV = 8;                 // float4 per thread (template NV <= 8) -> hidden <= 8192

template <typename T> struct Vec4;
template <> struct Vec4<float> {
  static __device__ __forceinline__ float4 load(const float* p) { return __ldg(reinterpret_cast<const float4*>(p)); }
};
template <> struct Vec4<__nv_bfloat16> {
  static __device__ __forceinline__ float4 load(const __nv_bfloat16* p) {
    const uint2 u = __ldg(reinterpret_cast<const uint2*>(p));
    return make_float4(bf16_lo(u.x), bf16_hi(u.x), bf16_lo(u.y), bf16_hi(u.y));
  }
};
__device__ __forceinline__ void store_bf16x4(__nv_bfloat16* p, float4 v) {
  *reinterpret_cast<uint2*>(p) = make_uint2(pack_bf16(v.x, v.y), pack_bf16(v.z, v.w));
}
__device__ __forceinline__ void store_f16x4(__half* p, float4 v) {
  *reinterpret_cast<uint2*>(p) = make_uint2(pack_f16(v.x, v.y), pack_f16(v.z, v.w));
}

__device__ __forceinline__ float block_sum(float v, float* red) {
#pragma unroll
  for (int off = 16; off > 0; off >>= 1) v += __shfl_xor_sync(0xffffffffu, v, off);
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  __syncthreads();                            // protect `red` from the previous use
  if (lane == 0) red[warp] = v;
  __syncthreads();
  float t = (lane < NORM_THREADS / 32) ? red[lane] : 0.f;
#pragma unroll
  for (int off = 4; off > 0; off >>= 1) t += __shfl_xor_sync(0xffffffffu, t, off);
  return __shfl_sync(0xffffffffu, t, 0);
}

// xn = x * rsqrt(mean(x^2) + eps) * g  (fp16 out: the GEMM operand), rstd saved in fp32.  One block per token row.
template <typename XT, int NV>
__global__ void __launch_bounds__(NORM_THREADS) rmsnorm_fwd_kernel(const XT* __restrict__ x, const __nv_bfloat16* __restrict__ g,
                                                                   __half* __restrict__ xn, float* __restrict__ rstd,
                                                                   int H, float eps) {
  pdl_wait(); pdl_trigger();                     // programmatic dependent launch (ptx.cuh): no global access above
  __shared__ float red[NORM_THREADS / 32];
  const long long row = blockIdx.x;
  const XT* xr = x + row * H;
  float4 v[NV];
  float ss = 0.f;
#pragma unroll
  for (int i = 0; i < NV; ++i) {
    const int c = (threadIdx.x + i * NORM_THREADS) * 4;
    if (c < H) {
      v[i] = Vec4<XT>::load(xr + c);
      ss += v[i].x * v[i].x + v[i].y * v[i].y + v[i].z * v[i].z + v[i].w * v[i].w;
    }
  }
  ss = block_sum(ss, red);
  const float r = rsqrtf(ss / static_cast<float>(H) + eps);
  if (threadIdx.x == 0) rstd[row] = r;
#pragma unroll
  for (int i = 0; i < NV; ++i) {
    const int c = (threadIdx.x + i * NORM_THREADS) * 4;
    if (c < H) {
      const float4 gg = Vec4<__nv_bfloat16>::load(g + c);
      store_f16x4(xn + row * H + c, make_float4(v[i].x * r * gg.x, v[i].y * r * gg.y, v[i].z * r * gg.z, v[i].w * r * gg.w));
    }
  }
}

// RMSNorm backward + residual gradient:
//   n = x r,  dn = dxn g,  dx = dres + r (dn - n mean_j(dn_j n_j)),  dg partial[block][col] = sum_rows dxn n.
// HBM-bound (x, dxn, dres read once, dx written once: 43-49 kB per token at H = 3072).  One persistent CTA per SM;
// a producer warp streams whole rows of the three inputs into a shared-memory ring with 1-D bulk async copies
// (cp.async.bulk, completion on an mbarrier), so ~150 KB per SM are in flight regardless of what the 8 consumer
// warps are doing; the consumers (two row groups of 4 warps when the row fits 8 float4 per thread, else one group of 8)
// read their columns from shared memory, reduce the row dot product, and store dx
// (and its fp16 copy) straight from registers.  Each thread keeps its columns' dg partials in registers over all
// rows of the CTA; colsum_kernel adds the per-CTA partials in a fixed order (deterministic, no atomics).
constexpr int NORMB_CONSUMERS = 256;                       // 8 consumer warps
constexpr int NORMB_THREADS = NORMB_CONSUMERS + 32;        // + 1 producer warp
constexpr int NORMB_MAX_STAGES = 6;
constexpr int NORMB_SMEM_BUDGET = 200 * 1024;

__device__ __forceinline__ void bulk_load_1d(uint32_t dst, const void* src, uint32_t bytes, uint32_t bar) {
  asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
               ::"r"(dst), "l"(reinterpret_cast<uint64_t>(src)), "r"(bytes), "r"(bar) : "memory");
}
__device__ __forceinline__ void named_bar_sync(int id, int nthreads) {
  asm volatile("bar.sync %0, %1;" ::"r"(id), "r"(nthreads) : "memory");
}
template <typename T> __device__ __forceinline__ float4 lds_vec4(const uint8_t* row, int c);
template <> __device__ __forceinline__ float4 lds_vec4<float>(const uint8_t* row, int c) {
  return *reinterpret_cast<const float4*>(row + static_cast<size_t>(c) * 4);
}
template <> __device__ __forceinline__ float4 lds_vec4<__nv_bfloat16>(const uint8_t* row, int c) {
  const uint2 u = *reinterpret_cast<const uint2*>(row + static_cast<size_t>(c) * 2);
  return make_float4(bf16_lo(u.x), bf16_hi(u.x), bf16_lo(u.y), bf16_hi(u.y));
}

// sum over the `nthreads` consumer threads of one row group (named barrier `bar_id`; the producer warp never joins it)
__device__ __forceinline__ float consumer_sum(float v, float* red, int bar_id, int nthreads, int warp_in_group) {
#pragma unroll
  for (int off = 16; off > 0; off >>= 1) v += __shfl_xor_sync(0xffffffffu, v, off);
  const int lane = threadIdx.x & 31;
  named_bar_sync(bar_id, nthreads);           // protect `red` from the previous row
  if (lane == 0) red[warp_in_group] = v;
  named_bar_sync(bar_id, nthreads);
  float t = 0.f;
  for (int k = 0; k < nthreads / 32; ++k) t += red[k];       // fixed order
  return t;
}

template <typename XT, typename RT, int NV, int G>
__global__ void __launch_bounds__(NORMB_THREADS, 1)
rmsnorm_bwd_kernel(const XT* __restrict__ x, const float* __restrict__ rstd, const __nv_bfloat16* __restrict__ g,
                   const float* __restrict__ dxn, const RT* __restrict__ dres, float* __restrict__ dx,
                   __half* __restrict__ dx16, float* __restrict__ dg_part, int T, int H, int stages, float res_scale,
                   unsigned long long* __restrict__ counter) {
  // G row groups of GT = 256 / G consumer threads: group q takes this CTA's rows q, q + G, ... so that the reduction
  // latency of one row (shuffles, two named barriers) overlaps the loads and stores of the other group's row.
  constexpr int GT = NORMB_CONSUMERS / G;
  extern __shared__ __align__(128) uint8_t nsm[];
  __shared__ float red[G][GT / 32];
  __shared__ __align__(8) unsigned long long bars[2 * NORMB_MAX_STAGES];
  // dres may be null (no residual gradient: the final norm before the LM head)
  const uint32_t xb = static_cast<uint32_t>(H) * sizeof(XT), db = static_cast<uint32_t>(H) * 4u,
                 rb = dres ? static_cast<uint32_t>(H) * sizeof(RT) : 0u;
  const uint32_t stage_bytes = xb + db + rb;                 // every part is a multiple of 16 (H % 8 == 0)
  const uint32_t smem0 = smem_u32(nsm);
  auto full = [&](int s) { return smem_u32(&bars[s]); };
  auto empty = [&](int s) { return smem_u32(&bars[NORMB_MAX_STAGES + s]); };
  if (threadIdx.x == 0) {
    for (int s = 0; s < stages; ++s) { mbar_init(full(s), 1); mbar_init(empty(s), GT / 32); }
    fence_barrier_init();
  }
  __syncthreads();
  pdl_wait(); pdl_trigger();                     // programmatic dependent launch (ptx.cuh): no global access above
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;

  if (warp == NORMB_CONSUMERS / 32) {
    // ------------------------------------------------------------------ producer warp
    if (lane == 0) {
      int s = 0; uint32_t ph = 0;
      for (long long row = blockIdx.x; row < T; row += gridDim.x) {
        mbar_wait(empty(s), ph ^ 1u);
        const uint32_t dst = smem0 + s * stage_bytes;
        mbar_expect_tx(full(s), stage_bytes);
        bulk_load_1d(dst, x + row * H, xb, full(s));
        bulk_load_1d(dst + xb, dxn + row * H, db, full(s));
        if (rb) bulk_load_1d(dst + xb + db, dres + row * H, rb, full(s));
        if (++s == stages) { s = 0; ph ^= 1u; }
      }
    }
    return;
  }
  // -------------------------------------------------------------------- consumers
  const int grp = threadIdx.x / GT, tg = threadIdx.x - grp * GT;
  float4 gg[NV], acc[NV];
#pragma unroll
  for (int i = 0; i < NV; ++i) {
    const int c = (tg + i * GT) * 4;
    acc[i] = make_float4(0.f, 0.f, 0.f, 0.f);
    gg[i] = (c < H) ? Vec4<__nv_bfloat16>::load(g + c) : make_float4(0.f, 0.f, 0.f, 0.f);
  }
  const float invH = 1.0f / static_cast<float>(H);
  unsigned int bad = 0;
  long long k = grp;                                          // index of the row among this CTA's rows
  for (long long row = blockIdx.x + static_cast<long long>(grp) * gridDim.x; row < T; row += static_cast<long long>(G) * gridDim.x, k += G) {
    const int s = static_cast<int>(k % stages);
    const uint32_t ph = static_cast<uint32_t>(k / stages) & 1u;
    const float r = rstd[row];
    mbar_wait(full(s), ph);
    const uint8_t* sx = nsm + static_cast<size_t>(s) * stage_bytes;
    const uint8_t* sd = sx + xb;
    const uint8_t* sr = sd + db;
    float4 n[NV], dn[NV], rs[NV];
    float dot = 0.f;
#pragma unroll
    for (int i = 0; i < NV; ++i) {
      const int c = (tg + i * GT) * 4;
      if (c < H) {
        const float4 xv = lds_vec4<XT>(sx, c);
        const float4 d = lds_vec4<float>(sd, c);
        rs[i] = rb ? lds_vec4<RT>(sr, c) : make_float4(0.f, 0.f, 0.f, 0.f);
        n[i] = make_float4(xv.x * r, xv.y * r, xv.z * r, xv.w * r);
        acc[i].x += d.x * n[i].x; acc[i].y += d.y * n[i].y; acc[i].z += d.z * n[i].z; acc[i].w += d.w * n[i].w;
        dn[i] = make_float4(d.x * gg[i].x, d.y * gg[i].y, d.z * gg[i].z, d.w * gg[i].w);
        dot += dn[i].x * n[i].x + dn[i].y * n[i].y + dn[i].z * n[i].z + dn[i].w * n[i].w;
      }
    }
    __syncwarp();
    if (lane == 0) mbar_arrive(empty(s));                    // this warp has read its part of the stage
    dot = consumer_sum(dot, red[grp], 1 + grp, GT, tg >> 5) * invH;
#pragma unroll
    for (int i = 0; i < NV; ++i) {
      const int c = (tg + i * GT) * 4;
      if (c < H) {
        float4 o;
        o.x = fmaf(res_scale, rs[i].x, r * (dn[i].x - n[i].x * dot));
        o.y = fmaf(res_scale, rs[i].y, r * (dn[i].y - n[i].y * dot));
        o.z = fmaf(res_scale, rs[i].z, r * (dn[i].z - n[i].z * dot));
        o.w = fmaf(res_scale, rs[i].w, r * (dn[i].w - n[i].w * dot));
        *reinterpret_cast<float4*>(dx + row * H + c) = o;
        if (dx16)      // the fp16 operand copy of this gradient: saturating and counted like the input casts (pack_f16_sat)
          *reinterpret_cast<uint2*>(dx16 + row * H + c) = make_uint2(pack_f16_sat(o.x, o.y, bad), pack_f16_sat(o.z, o.w, bad));
      }
    }
  }
  cast_report(bad, counter);
  // one row of dg partials per (CTA, group)
#pragma unroll
  for (int i = 0; i < NV; ++i) {
    const int c = (tg + i * GT) * 4;
    if (c < H) *reinterpret_cast<float4*>(dg_part + (static_cast<long long>(blockIdx.x) * G + grp) * H + c) = acc[i];
  }
}

// dg[col] (+)= sum over CTAs of dg_part[cta][col], fixed order (deterministic).  Block = 32 columns x 8 partial groups.
__global__ void __launch_bounds__(256) colsum_kernel(const float* __restrict__ part, float* __restrict__ out, int nparts, int H,
                                                     int accumulate) {
  pdl_wait(); pdl_trigger();                     // programmatic dependent launch (ptx.cuh): no global access above
  __shared__ float sm[8][33];
  const int cx = threadIdx.x & 31, gy = threadIdx.x >> 5;
  const int c = blockIdx.x * 32 + cx;
  float s = 0.f;
  if (c < H)
    for (int b = gy; b < nparts; b += 8) s += part[static_cast<long long>(b) * H + c];
  sm[gy][cx] = s;
  __syncthreads();
  if (gy == 0 && c < H) {
    float t = 0.f;
#pragma unroll
    for (int k = 0; k < 8; ++k) t += sm[k][cx];
    out[c] = accumulate ? out[c] + t : t;
  }
}

// 8 elements per thread casts (n is a multiple of 8)
// fp16 operand copies of caller tensors (P-2'): fp16 has bf16's tensor-core rate and three more
// mantissa bits, but a narrower exponent -- |v| > 65504 would become inf and poison every sum it enters.  The casts
// therefore SATURATE to +-65504 (NaN stays NaN) and COUNT the values they had to clamp or found non-finite in a
// context-owned device counter (lsp_overflow_count): out-of-range input is reported, never silent.  Values below 2^-24
// flush to zero (an absolute error far under the parity bar).
__global__ void cast_f32_f16_kernel(const float* __restrict__ in, __half* __restrict__ out, long long n8, unsigned long long* counter) {
  pdl_wait(); pdl_trigger();                     // programmatic dependent launch (ptx.cuh): no global access above
  unsigned int bad = 0;
  for (long long i = static_cast<long long>(blockIdx.x) * blockDim.x + threadIdx.x; i < n8; i += static_cast<long long>(gridDim.x) * blockDim.x) {
    const float4 a = __ldg(reinterpret_cast<const float4*>(in) + 2 * i), b = __ldg(reinterpret_cast<const float4*>(in) + 2 * i + 1);
    reinterpret_cast<uint4*>(out)[i] = make_uint4(pack_f16_sat(a.x, a.y, bad), pack_f16_sat(a.z, a.w, bad), pack_f16_sat(b.x, b.y, bad),
                                                  pack_f16_sat(b.z, b.w, bad));
  }
  cast_report(bad, counter);
}
__global__ void cast_bf16_f16_kernel(const __nv_bfloat16* __restrict__ in, __half* __restrict__ out, long long n8, unsigned long long* counter) {
  pdl_wait(); pdl_trigger();                     // programmatic dependent launch (ptx.cuh): no global access above
  unsigned int bad = 0;
  for (long long i = static_cast<long long>(blockIdx.x) * blockDim.x + threadIdx.x; i < n8; i += static_cast<long long>(gridDim.x) * blockDim.x) {
    const uint4 u = __ldg(reinterpret_cast<const uint4*>(in) + i);
    reinterpret_cast<uint4*>(out)[i] = make_uint4(pack_f16_sat(bf16_lo(u.x), bf16_hi(u.x), bad), pack_f16_sat(bf16_lo(u.y), bf16_hi(u.y), bad),
                                                  pack_f16_sat(bf16_lo(u.z), bf16_hi(u.z), bad), pack_f16_sat(bf16_lo(u.w), bf16_hi(u.w), bad));
  }
  cast_report(bad, counter);
}

// Several bf16 -> fp16 casts in one launch (the weight tensors of a block): segment s covers 8-element groups
// [start[s], start[s + 1]) of the concatenated index space.
constexpr int CAST_MAX_SEGS = 4;
struct CastSegs {
  const __nv_bfloat16* src[CAST_MAX_SEGS];
  __half* dst[CAST_MAX_SEGS];
  long long start[CAST_MAX_SEGS + 1];
  int nseg;
  unsigned perm_mask;        // segments whose ROWS are permuted on the way: dst row head*d + 2i + half = src row head*d + half*d/2 + i
  int perm_d, row_units;     // head_dim; 16-byte units per row (in-features / 8)
  unsigned long long* counter;   // clamped / non-finite values (see pack_f16_sat); may be null
};
__device__ __forceinline__ long long cast_src_unit(const CastSegs& segs, long long i, int& s) {
  s = 0;
#pragma unroll
  for (int k = 1; k < CAST_MAX_SEGS; ++k) s += (k < segs.nseg && i >= segs.start[k]) ? 1 : 0;
  const long long j = i - segs.start[s];
  if ((segs.perm_mask >> s) & 1u) {
    const long long row = j / segs.row_units;
    const int p = static_cast<int>(row % segs.perm_d);
    return (row - p + (p & 1) * (segs.perm_d >> 1) + (p >> 1)) * segs.row_units + (j - row * segs.row_units);
  }
  return j;
}
// four independent 16-byte loads in flight per thread (the kernel is latency-bound otherwise: 2.7 TB/s with one)
__global__ void __launch_bounds__(256) cast_multi_bf16_f16_kernel(const CastSegs segs) {
  pdl_wait(); pdl_trigger();                     // programmatic dependent launch (ptx.cuh): no global access above
  const long long total = segs.start[segs.nseg];
  const long long stride = static_cast<long long>(gridDim.x) * blockDim.x;
  unsigned int bad = 0;
  for (long long i0 = static_cast<long long>(blockIdx.x) * blockDim.x + threadIdx.x; i0 < total; i0 += 4 * stride) {
    uint4 u[4];
    int sg[4];
#pragma unroll
    for (int k = 0; k < 4; ++k) {
      const long long i = i0 + k * stride;
      sg[k] = 0;
      if (i < total) {
        const long long js = cast_src_unit(segs, i, sg[k]);
        u[k] = __ldg(reinterpret_cast<const uint4*>(segs.src[sg[k]]) + js);
      }
    }
#pragma unroll
    for (int k = 0; k < 4; ++k) {
      const long long i = i0 + k * stride;
      if (i < total)
        reinterpret_cast<uint4*>(segs.dst[sg[k]])[i - segs.start[sg[k]]] =
            make_uint4(pack_f16_sat(bf16_lo(u[k].x), bf16_hi(u[k].x), bad), pack_f16_sat(bf16_lo(u[k].y), bf16_hi(u[k].y), bad),
                       pack_f16_sat(bf16_lo(u[k].z), bf16_hi(u[k].z), bad), pack_f16_sat(bf16_lo(u[k].w), bf16_hi(u[k].w), bad));
    }
  }
  cast_report(bad, segs.counter);
}

// x0[t,:] = E[id_t,:]  (bf16 table row -> fp32 or bf16 stream).  One block per token.
template <typename OT>
__global__ void embed_gather_kernel(const int* __restrict__ ids, const __nv_bfloat16* __restrict__ table, OT* __restrict__ out, int H) {
  const long long t = blockIdx.x;
  const __nv_bfloat16* src = table + static_cast<long long>(ids[t]) * H;
  for (int c = threadIdx.x * 4; c < H; c += blockDim.x * 4) {
    const float4 v = Vec4<__nv_bfloat16>::load(src + c);
    if constexpr (sizeof(OT) == 4) *reinterpret_cast<float4*>(out + t * H + c) = v;
    else store_bf16x4(reinterpret_cast<__nv_bfloat16*>(out) + t * H + c, v);
  }
}

}  // namespace lsp
