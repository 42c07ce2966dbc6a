// Causal grouped-query flash attention, forward (+LSE) and backward, fp16 operands / fp32 accumulate.
//
//   fwd : O_i = sum_{j<=i} softmax_j(q_i.k_j/sqrt(d)) v_j,  L_i = log sum_{j<=i} exp(q_i.k_j/sqrt(d))
//   bwd : P = exp(s - L); dV += P^T dO; dP = dO V^T; dS = P*(dP - D); dQ += dS K/sqrt(d); dK += dS^T Q/sqrt(d)
//         with D_i = sum_c dO_ic O_ic taken from the fp32 O (precision rule P-3).
//
// Tiled online-softmax forward; backward as two deterministic kernels (dK/dV per key block with the GQA
// group-sum kept in registers; dQ per query block), both skipping tiles above the diagonal.  No atomics:
// results are bit-reproducible.  Q,K,V,dO,P,dS are fp16 (P, dS in [0,1]-scaled ranges need the 11-bit
// mantissa to meet the 2e-2 max-norm bar at early positions; DESIGN.md precision plan P-5).
// Tensor-core path in this revision: mma.sync.m16n8k16 (HMMA); K/V tiles via cp.async double buffering.
#pragma once
#include "ptx.cuh"

namespace lsp {

struct AttnParams {
  // element pointers (fp16) and row pitches in elements; token t = b*S + s is row t
  const __half* q; const __half* k; const __half* v; const __half* dO;
  long long ldq, ldk, ldv, lddo;
  int B, S, nq, nkv;
  float scale_log2;            // (1/sqrt(d)) * log2(e)
  float scale;                 // 1/sqrt(d)
  // forward outputs
  float* o32; __half* o16; long long ldo;           // either may be null
  float* lse;                  // [B, nq, S]
  // backward inputs/outputs
  const float* dvec;           // D [B, nq, S]
  const float2* rope;          // (cos,sin) [S, d/2] or null: inverse rotation applied to dq, dk on store
  float* dq32; float* dk32; float* dv32; long long lddq32, lddk32;             // fp32 outputs (sdpa API) or null
  __half* dq16; __half* dk16; __half* dv16; long long ldd16;   // fp16 outputs (layer path: GEMM operands) or null
};

// ------------------------------------------------------------------------------------------- primitives
__device__ __forceinline__ void ldsm_x4(uint32_t addr, uint32_t& r0, uint32_t& r1, uint32_t& r2, uint32_t& r3) {
  asm volatile("ldmatrix.sync.aligned.m8n8.x4.shared.b16 {%0,%1,%2,%3}, [%4];"
               : "=r"(r0), "=r"(r1), "=r"(r2), "=r"(r3) : "r"(addr));
}
__device__ __forceinline__ void ldsm_x4_t(uint32_t addr, uint32_t& r0, uint32_t& r1, uint32_t& r2, uint32_t& r3) {
  asm volatile("ldmatrix.sync.aligned.m8n8.x4.trans.shared.b16 {%0,%1,%2,%3}, [%4];"
               : "=r"(r0), "=r"(r1), "=r"(r2), "=r"(r3) : "r"(addr));
}
__device__ __forceinline__ void mma16816(float (&c)[4], const uint32_t (&a)[4], uint32_t b0, uint32_t b1) {
  asm volatile("mma.sync.aligned.m16n8k16.row.col.f32.f16.f16.f32 {%0,%1,%2,%3}, {%4,%5,%6,%7}, {%8,%9}, {%0,%1,%2,%3};"
               : "+f"(c[0]), "+f"(c[1]), "+f"(c[2]), "+f"(c[3])
               : "r"(a[0]), "r"(a[1]), "r"(a[2]), "r"(a[3]), "r"(b0), "r"(b1));
}
__device__ __forceinline__ void cp_async16(uint32_t dst, const void* src, bool valid) {
  const int sz = valid ? 16 : 0;
  asm volatile("cp.async.cg.shared.global [%0], [%1], 16, %2;" ::"r"(dst), "l"(src), "r"(sz) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
template <int N> __device__ __forceinline__ void cp_async_wait() { asm volatile("cp.async.wait_group %0;" ::"n"(N) : "memory"); }

// Shared tile [rows][D] fp16, 16-byte chunks XOR-swizzled by (row & 7): conflict-free ldmatrix.
template <int D>
__device__ __forceinline__ uint32_t tile_addr(uint32_t base, int row, int col) {
  return base + row * (D * 2) + ((((col >> 3) ^ (row & 7))) << 4) + ((col & 7) << 1);
}
// Cooperative async load of ROWS x D halfs; rows s0.. of a sequence, zero-filled past s_limit.
template <int ROWS, int D, int NT>
__device__ __forceinline__ void load_tile_async(uint32_t sbase, const __half* g, long long ld, int s0, int s_limit) {
  constexpr int CPR = D / 8;
  for (int idx = threadIdx.x; idx < ROWS * CPR; idx += NT) {
    const int row = idx / CPR, ch = idx % CPR;
    const bool ok = (s0 + row) < s_limit;
    const __half* src = g + static_cast<long long>(ok ? (s0 + row) : 0) * ld + ch * 8;
    cp_async16(sbase + row * (D * 2) + ((ch ^ (row & 7)) << 4), src, ok);
  }
}

// ------------------------------------------------------------------------------------------- forward
// grid (ceil(S/128), nq, B), 256 threads: warp w owns query rows 16w..16w+15 of the block.
template <int D>
__global__ void __launch_bounds__(256, 1) attn_fwd_kernel(const AttnParams p) {
  pdl_wait(); pdl_trigger();                     // programmatic dependent launch (ptx.cuh): no global access above
  constexpr int BM = 128, BN = 64, NT = 256;
  constexpr int KS = D / 16;            // k-steps over head_dim
  constexpr int ND = D / 8;             // n-tiles over head_dim (O accumulator)
  extern __shared__ __align__(128) uint8_t smem[];
  const uint32_t sQ = smem_u32(smem);
  const uint32_t sK = sQ + BM * D * 2;            // 2 stages
  const uint32_t sV = sK + 2 * BN * D * 2;        // 2 stages

  const int qb = gridDim.x - 1 - blockIdx.x;      // heavy (late) query blocks first
  const int h = blockIdx.y, b = blockIdx.z;
  const int kvh = h / (p.nq / p.nkv);
  const int q0 = qb * BM;
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const long long tok0 = static_cast<long long>(b) * p.S;

  const __half* gq = p.q + tok0 * p.ldq + h * D;
  const __half* gk = p.k + tok0 * p.ldk + kvh * D;
  const __half* gv = p.v + tok0 * p.ldv + kvh * D;

  const int kv_end = min(p.S, q0 + BM);           // keys [0, kv_end)
  const int nblk = (kv_end + BN - 1) / BN;

  load_tile_async<BM, D, NT>(sQ, gq, p.ldq, q0, p.S);
  load_tile_async<BN, D, NT>(sK, gk, p.ldk, 0, p.S);
  load_tile_async<BN, D, NT>(sV, gv, p.ldv, 0, p.S);
  cp_async_commit();
  cp_async_wait<0>();
  __syncthreads();

  uint32_t qf[KS][4];
#pragma unroll
  for (int ks = 0; ks < KS; ++ks) {
    const int row = warp * 16 + (lane & 7) + ((lane >> 3) & 1) * 8;
    const int col = ks * 16 + (lane >> 4) * 8;
    ldsm_x4(tile_addr<D>(sQ, row, col), qf[ks][0], qf[ks][1], qf[ks][2], qf[ks][3]);
  }

  float o[ND][4];
#pragma unroll
  for (int i = 0; i < ND; ++i) { o[i][0] = o[i][1] = o[i][2] = o[i][3] = 0.f; }
  float m_run[2] = {-INFINITY, -INFINITY}, l_run[2] = {0.f, 0.f};
  const int qrow0 = q0 + warp * 16 + (lane >> 2);          // rows qrow0 and qrow0 + 8

  for (int j = 0; j < nblk; ++j) {
    const int st = j & 1;
    if (j + 1 < nblk) {                                     // prefetch next K,V
      load_tile_async<BN, D, NT>(sK + (st ^ 1) * BN * D * 2, gk, p.ldk, (j + 1) * BN, p.S);
      load_tile_async<BN, D, NT>(sV + (st ^ 1) * BN * D * 2, gv, p.ldv, (j + 1) * BN, p.S);
    }
    cp_async_commit();
    const uint32_t cK = sK + st * BN * D * 2, cV = sV + st * BN * D * 2;
    const int k0 = j * BN;
    const bool active = k0 <= q0 + warp * 16 + 15;          // warp-uniform: any key of this block <= some row

    if (active) {
      float s[BN / 8][4];
#pragma unroll
      for (int i = 0; i < BN / 8; ++i) { s[i][0] = s[i][1] = s[i][2] = s[i][3] = 0.f; }
#pragma unroll
      for (int ks = 0; ks < KS; ++ks) {
#pragma unroll
        for (int np = 0; np < BN / 16; ++np) {
          uint32_t b0, b1, b2, b3;
          const int key = np * 16 + (lane & 7) + (lane >> 4) * 8;
          const int col = ks * 16 + ((lane >> 3) & 1) * 8;
          ldsm_x4(tile_addr<D>(cK, key, col), b0, b1, b2, b3);
          mma16816(s[2 * np], qf[ks], b0, b1);
          mma16816(s[2 * np + 1], qf[ks], b2, b3);
        }
      }
      // scale to log2 units, mask (causal + sequence end)
      const bool need_mask = (k0 + BN - 1 > q0 + warp * 16) || (k0 + BN > p.S);
#pragma unroll
      for (int i = 0; i < BN / 8; ++i) {
#pragma unroll
        for (int e = 0; e < 4; ++e) {
          float val = s[i][e] * p.scale_log2;
          if (need_mask) {
            const int key = k0 + i * 8 + (lane & 3) * 2 + (e & 1);
            const int qr = qrow0 + (e >> 1) * 8;
            if (key > qr || key >= p.S) val = -INFINITY;
          }
          s[i][e] = val;
        }
      }
      // online softmax for the two rows of this thread
#pragma unroll
      for (int r = 0; r < 2; ++r) {
        float mx = m_run[r];
#pragma unroll
        for (int i = 0; i < BN / 8; ++i) mx = fmaxf(mx, fmaxf(s[i][2 * r], s[i][2 * r + 1]));
        mx = fmaxf(mx, __shfl_xor_sync(0xffffffffu, mx, 1));
        mx = fmaxf(mx, __shfl_xor_sync(0xffffffffu, mx, 2));
        const float mref = (mx == -INFINITY) ? 0.f : mx;
        const float corr = exp2f(m_run[r] - mref);          // m_run = -inf -> 0
        m_run[r] = mx;
        float sum = 0.f;
#pragma unroll
        for (int i = 0; i < BN / 8; ++i) {
          s[i][2 * r] = exp2f(s[i][2 * r] - mref);
          s[i][2 * r + 1] = exp2f(s[i][2 * r + 1] - mref);
          sum += s[i][2 * r] + s[i][2 * r + 1];
        }
        l_run[r] = l_run[r] * corr + sum;                   // per-thread partial; quad-reduced at the end
#pragma unroll
        for (int i = 0; i < ND; ++i) { o[i][2 * r] *= corr; o[i][2 * r + 1] *= corr; }
      }
      // O += P V
#pragma unroll
      for (int kk = 0; kk < BN / 16; ++kk) {
        uint32_t pa[4];
        pa[0] = pack_f16(s[2 * kk][0], s[2 * kk][1]);
        pa[1] = pack_f16(s[2 * kk][2], s[2 * kk][3]);
        pa[2] = pack_f16(s[2 * kk + 1][0], s[2 * kk + 1][1]);
        pa[3] = pack_f16(s[2 * kk + 1][2], s[2 * kk + 1][3]);
#pragma unroll
        for (int dp = 0; dp < ND / 2; ++dp) {
          uint32_t b0, b1, b2, b3;
          const int key = kk * 16 + (lane & 7) + ((lane >> 3) & 1) * 8;
          const int col = dp * 16 + (lane >> 4) * 8;
          ldsm_x4_t(tile_addr<D>(cV, key, col), b0, b1, b2, b3);
          mma16816(o[2 * dp], pa, b0, b1);
          mma16816(o[2 * dp + 1], pa, b2, b3);
        }
      }
    }
    cp_async_wait<0>();
    __syncthreads();
  }

  // finalize
#pragma unroll
  for (int r = 0; r < 2; ++r) {
    float l = l_run[r];
    l += __shfl_xor_sync(0xffffffffu, l, 1);
    l += __shfl_xor_sync(0xffffffffu, l, 2);
    const int qr = qrow0 + r * 8;
    if (qr < p.S) {
      const float inv = 1.0f / l;
      const long long t = tok0 + qr;
      if ((lane & 3) == 0)
        p.lse[(static_cast<long long>(b) * p.nq + h) * p.S + qr] = (m_run[r] + log2f(l)) * 0.6931471805599453f;
#pragma unroll
      for (int i = 0; i < ND; ++i) {
        const int col = h * D + i * 8 + (lane & 3) * 2;
        const float v0 = o[i][2 * r] * inv, v1 = o[i][2 * r + 1] * inv;
        if (p.o32) *reinterpret_cast<float2*>(p.o32 + t * p.ldo + col) = make_float2(v0, v1);
        if (p.o16) *reinterpret_cast<uint32_t*>(p.o16 + t * p.ldo + col) = pack_f16(v0, v1);
      }
    }
  }
}

// ------------------------------------------------------------------------------------------- D = rowsum(dO * O32)
// one warp per (token, head); dO fp16 (the tensor-core operand), O fp32.  Used where no O-projection dgrad precedes the
// attention backward (lsp_sdpa_bwd) and on the head_dim 64 path; inside the layer the sums are formed by that GEMM's
// epilogue (EpiDOutDvec).  PARTS4: write the [B, nq, S, 4] partial-sum layout the tcgen05 kernels read, as (D, 0, 0, 0).
template <int D, bool PARTS4>
__global__ void attn_dvec_kernel(const __half* dO, long long lddo, const float* o32, long long ldo, float* dvec,
                                 int B, int S, int nq) {
  pdl_wait(); pdl_trigger();                     // programmatic dependent launch (ptx.cuh): no global access above
  const long long gw = (static_cast<long long>(blockIdx.x) * blockDim.x + threadIdx.x) >> 5;
  const int lane = threadIdx.x & 31;
  const long long total = static_cast<long long>(B) * S * nq;
  if (gw >= total) return;
  const long long t = gw / nq;
  const int h = static_cast<int>(gw % nq);
  constexpr int PER = D / 32;
  const __half* a = dO + t * lddo + h * D + lane * PER;
  const float* o = o32 + t * ldo + h * D + lane * PER;
  float acc = 0.f;
#pragma unroll
  for (int i = 0; i < PER; ++i) acc += __half2float(a[i]) * o[i];
#pragma unroll
  for (int off = 16; off > 0; off >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, off);
  if (lane == 0) {
    const int b = static_cast<int>(t / S), s = static_cast<int>(t % S);
    const long long idx = (static_cast<long long>(b) * nq + h) * S + s;
    if (PARTS4) reinterpret_cast<float4*>(dvec)[idx] = make_float4(acc, 0.f, 0.f, 0.f);
    else dvec[idx] = acc;
  }
}

// Store a 16 x D fp32 accumulator tile (mma C layout) of rows s_row0+{0,8}: scale, optional inverse RoPE,
// to fp32 and/or fp16 destinations.
template <int D>
__device__ __forceinline__ void store_grad_tile(float (&acc)[D / 8][4], float scale, const float2* rope, int S,
                                                long long tok0, int s_row0, int lane, float* o32, long long ld32,
                                                __half* o16, long long ld16, int col_base) {
#pragma unroll
  for (int r = 0; r < 2; ++r) {
    const int s = s_row0 + r * 8;
    if (s >= S) continue;
    const long long t = tok0 + s;
#pragma unroll
    for (int i = 0; i < D / 8; ++i) {
      const int c = i * 8 + (lane & 3) * 2;
      float v0 = acc[i][2 * r] * scale, v1 = acc[i][2 * r + 1] * scale;
      if (rope) {                                          // transpose of the forward rotation: angle -theta
        const float2 cs = __ldg(rope + static_cast<long long>(s) * (D / 2) + (c >> 1));
        const float z0 = v0, z1 = v1;
        v0 = z0 * cs.x + z1 * cs.y;
        v1 = -z0 * cs.y + z1 * cs.x;
      }
      if (o32) *reinterpret_cast<float2*>(o32 + t * ld32 + col_base + c) = make_float2(v0, v1);
      if (o16) *reinterpret_cast<uint32_t*>(o16 + t * ld16 + col_base + c) = pack_f16(v0, v1);
    }
  }
}

// ------------------------------------------------------------------------------------------- backward: dK, dV
// grid (ceil(S/64), nkv, B), 128 threads: warp w owns keys 16w..16w+15 of the block; loops over the G query
// heads of this kv head and the query blocks at/after the diagonal; dK/dV group-sums stay in registers.
template <int D>
__global__ void __launch_bounds__(128, 2) attn_bwd_dkdv_kernel(const AttnParams p) {
  pdl_wait(); pdl_trigger();                     // programmatic dependent launch (ptx.cuh): no global access above
  constexpr int BN = 64, BM = 64, NT = 128;
  constexpr int KS = D / 16, ND = D / 8;
  extern __shared__ __align__(128) uint8_t smem[];
  const uint32_t sK = smem_u32(smem);
  const uint32_t sV = sK + BN * D * 2;
  const uint32_t sQ = sV + BN * D * 2;            // 2 stages
  const uint32_t sDO = sQ + 2 * BM * D * 2;       // 2 stages
  float* sL = reinterpret_cast<float*>(smem + (2 * BN + 4 * BM) * D * 2);   // [2][BM] LSE*log2e
  float* sD = sL + 2 * BM;                                                   // [2][BM] D

  const int kb = blockIdx.x, kvh = blockIdx.y, b = blockIdx.z;
  const int G = p.nq / p.nkv;
  const int k0 = kb * BN;
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const long long tok0 = static_cast<long long>(b) * p.S;

  const __half* gk = p.k + tok0 * p.ldk + kvh * D;
  const __half* gv = p.v + tok0 * p.ldv + kvh * D;

  const int qb_first = k0 / BM;
  const int nqb = (p.S + BM - 1) / BM;
  const int per_head = nqb - qb_first;
  const int iters = per_head * G;

  auto issue = [&](int it, int st) {
    const int hh = kvh * G + it / per_head;
    const int qb = qb_first + it % per_head;
    const __half* gq = p.q + tok0 * p.ldq + hh * D;
    const __half* gdo = p.dO + tok0 * p.lddo + hh * D;
    load_tile_async<BM, D, NT>(sQ + st * BM * D * 2, gq, p.ldq, qb * BM, p.S);
    load_tile_async<BM, D, NT>(sDO + st * BM * D * 2, gdo, p.lddo, qb * BM, p.S);
    if (threadIdx.x < BM) {
      const int s = qb * BM + threadIdx.x;
      const long long idx = (static_cast<long long>(b) * p.nq + hh) * p.S + s;
      sL[st * BM + threadIdx.x] = (s < p.S) ? p.lse[idx] * 1.4426950408889634f : INFINITY;
      sD[st * BM + threadIdx.x] = (s < p.S) ? p.dvec[idx] : 0.f;
    }
  };

  load_tile_async<BN, D, NT>(sK, gk, p.ldk, k0, p.S);
  load_tile_async<BN, D, NT>(sV, gv, p.ldv, k0, p.S);
  issue(0, 0);
  cp_async_commit();

  float dk[ND][4], dv[ND][4];
#pragma unroll
  for (int i = 0; i < ND; ++i) { dk[i][0] = dk[i][1] = dk[i][2] = dk[i][3] = 0.f; dv[i][0] = dv[i][1] = dv[i][2] = dv[i][3] = 0.f; }
  const int key_r0 = k0 + warp * 16 + (lane >> 2);          // this thread's key rows: key_r0, key_r0 + 8

  for (int it = 0; it < iters; ++it) {
    const int st = it & 1;
    cp_async_wait<0>();
    __syncthreads();                                        // stage st landed; stage st^1 free
    if (it + 1 < iters) issue(it + 1, st ^ 1);
    cp_async_commit();

    const int qb = qb_first + it % per_head;
    const int qs0 = qb * BM;
    const uint32_t cQ = sQ + st * BM * D * 2, cDO = sDO + st * BM * D * 2;
    const float* cL = sL + st * BM;
    const float* cD = sD + st * BM;

    // S^T = K Q^T  (16 keys x 64 queries per warp)
    float s[BM / 8][4];
#pragma unroll
    for (int i = 0; i < BM / 8; ++i) { s[i][0] = s[i][1] = s[i][2] = s[i][3] = 0.f; }
#pragma unroll
    for (int ks = 0; ks < KS; ++ks) {
      uint32_t ka[4];
      ldsm_x4(tile_addr<D>(sK, warp * 16 + (lane & 7) + ((lane >> 3) & 1) * 8, ks * 16 + (lane >> 4) * 8), ka[0], ka[1], ka[2], ka[3]);
#pragma unroll
      for (int np = 0; np < BM / 16; ++np) {
        uint32_t b0, b1, b2, b3;
        ldsm_x4(tile_addr<D>(cQ, np * 16 + (lane & 7) + (lane >> 4) * 8, ks * 16 + ((lane >> 3) & 1) * 8), b0, b1, b2, b3);
        mma16816(s[2 * np], ka, b0, b1);
        mma16816(s[2 * np + 1], ka, b2, b3);
      }
    }
    // P^T = exp2(S^T*scale_log2 - L*log2e), causal: query >= key
    const bool diag = qs0 < k0 + BN;                        // block touches the diagonal
#pragma unroll
    for (int i = 0; i < BM / 8; ++i) {
#pragma unroll
      for (int e = 0; e < 4; ++e) {
        const int ql = i * 8 + (lane & 3) * 2 + (e & 1);
        float pv = exp2f(s[i][e] * p.scale_log2 - cL[ql]);  // L = +inf for rows past the sequence end -> 0
        if (diag) {
          const int key = key_r0 + (e >> 1) * 8;
          if (qs0 + ql < key) pv = 0.f;
        }
        s[i][e] = pv;
      }
    }
    // dV += P^T dO ; dP^T = V dO^T
    float dp[BM / 8][4];
#pragma unroll
    for (int i = 0; i < BM / 8; ++i) { dp[i][0] = dp[i][1] = dp[i][2] = dp[i][3] = 0.f; }
#pragma unroll
    for (int kk = 0; kk < BM / 16; ++kk) {
      uint32_t pa[4];
      pa[0] = pack_f16(s[2 * kk][0], s[2 * kk][1]);
      pa[1] = pack_f16(s[2 * kk][2], s[2 * kk][3]);
      pa[2] = pack_f16(s[2 * kk + 1][0], s[2 * kk + 1][1]);
      pa[3] = pack_f16(s[2 * kk + 1][2], s[2 * kk + 1][3]);
#pragma unroll
      for (int dpi = 0; dpi < ND / 2; ++dpi) {
        uint32_t b0, b1, b2, b3;
        ldsm_x4_t(tile_addr<D>(cDO, kk * 16 + (lane & 7) + ((lane >> 3) & 1) * 8, dpi * 16 + (lane >> 4) * 8), b0, b1, b2, b3);
        mma16816(dv[2 * dpi], pa, b0, b1);
        mma16816(dv[2 * dpi + 1], pa, b2, b3);
      }
    }
#pragma unroll
    for (int ks = 0; ks < KS; ++ks) {
      uint32_t va[4];
      ldsm_x4(tile_addr<D>(sV, warp * 16 + (lane & 7) + ((lane >> 3) & 1) * 8, ks * 16 + (lane >> 4) * 8), va[0], va[1], va[2], va[3]);
#pragma unroll
      for (int np = 0; np < BM / 16; ++np) {
        uint32_t b0, b1, b2, b3;
        ldsm_x4(tile_addr<D>(cDO, np * 16 + (lane & 7) + (lane >> 4) * 8, ks * 16 + ((lane >> 3) & 1) * 8), b0, b1, b2, b3);
        mma16816(dp[2 * np], va, b0, b1);
        mma16816(dp[2 * np + 1], va, b2, b3);
      }
    }
    // dS^T = P^T * (dP^T - D) ; dK += dS^T Q
#pragma unroll
    for (int kk = 0; kk < BM / 16; ++kk) {
      uint32_t sa[4];
      {
        const int qa = (2 * kk) * 8 + (lane & 3) * 2, qb2 = (2 * kk + 1) * 8 + (lane & 3) * 2;
        const float d0 = cD[qa], d1 = cD[qa + 1], d2 = cD[qb2], d3 = cD[qb2 + 1];
        sa[0] = pack_f16(s[2 * kk][0] * (dp[2 * kk][0] - d0), s[2 * kk][1] * (dp[2 * kk][1] - d1));
        sa[1] = pack_f16(s[2 * kk][2] * (dp[2 * kk][2] - d0), s[2 * kk][3] * (dp[2 * kk][3] - d1));
        sa[2] = pack_f16(s[2 * kk + 1][0] * (dp[2 * kk + 1][0] - d2), s[2 * kk + 1][1] * (dp[2 * kk + 1][1] - d3));
        sa[3] = pack_f16(s[2 * kk + 1][2] * (dp[2 * kk + 1][2] - d2), s[2 * kk + 1][3] * (dp[2 * kk + 1][3] - d3));
      }
#pragma unroll
      for (int dpi = 0; dpi < ND / 2; ++dpi) {
        uint32_t b0, b1, b2, b3;
        ldsm_x4_t(tile_addr<D>(cQ, kk * 16 + (lane & 7) + ((lane >> 3) & 1) * 8, dpi * 16 + (lane >> 4) * 8), b0, b1, b2, b3);
        mma16816(dk[2 * dpi], sa, b0, b1);
        mma16816(dk[2 * dpi + 1], sa, b2, b3);
      }
    }
  }
  cp_async_wait<0>();

  store_grad_tile<D>(dk, p.scale, p.rope, p.S, tok0, key_r0, lane, p.dk32, p.lddk32, p.dk16, p.ldd16, kvh * D);
  store_grad_tile<D>(dv, 1.0f, nullptr, p.S, tok0, key_r0, lane, p.dv32, p.lddk32, p.dv16, p.ldd16, kvh * D);
}

// ------------------------------------------------------------------------------------------- backward: dQ
// grid (ceil(S/64), nq, B), 128 threads: warp w owns queries 16w..16w+15; loops over key blocks <= diagonal.
template <int D>
__global__ void __launch_bounds__(128, 2) attn_bwd_dq_kernel(const AttnParams p) {
  pdl_wait(); pdl_trigger();                     // programmatic dependent launch (ptx.cuh): no global access above
  constexpr int BM = 64, BN = 64, NT = 128;
  constexpr int KS = D / 16, ND = D / 8;
  extern __shared__ __align__(128) uint8_t smem[];
  const uint32_t sQ = smem_u32(smem);             // Q tile then dO tile (staging for fragments)
  const uint32_t sDO = sQ + BM * D * 2;
  const uint32_t sK = sDO + BM * D * 2;           // 2 stages
  const uint32_t sV = sK + 2 * BN * D * 2;        // 2 stages

  const int qb = gridDim.x - 1 - blockIdx.x;
  const int h = blockIdx.y, b = blockIdx.z;
  const int kvh = h / (p.nq / p.nkv);
  const int q0 = qb * BM;
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const long long tok0 = static_cast<long long>(b) * p.S;
  const __half* gq = p.q + tok0 * p.ldq + h * D;
  const __half* gdo = p.dO + tok0 * p.lddo + h * D;
  const __half* gk = p.k + tok0 * p.ldk + kvh * D;
  const __half* gv = p.v + tok0 * p.ldv + kvh * D;

  const int kv_end = min(p.S, q0 + BM);
  const int nblk = (kv_end + BN - 1) / BN;

  load_tile_async<BM, D, NT>(sQ, gq, p.ldq, q0, p.S);
  load_tile_async<BM, D, NT>(sDO, gdo, p.lddo, q0, p.S);
  load_tile_async<BN, D, NT>(sK, gk, p.ldk, 0, p.S);
  load_tile_async<BN, D, NT>(sV, gv, p.ldv, 0, p.S);
  cp_async_commit();
  cp_async_wait<0>();
  __syncthreads();

  uint32_t qf[KS][4], dof[KS][4];
#pragma unroll
  for (int ks = 0; ks < KS; ++ks) {
    const int row = warp * 16 + (lane & 7) + ((lane >> 3) & 1) * 8;
    const int col = ks * 16 + (lane >> 4) * 8;
    ldsm_x4(tile_addr<D>(sQ, row, col), qf[ks][0], qf[ks][1], qf[ks][2], qf[ks][3]);
    ldsm_x4(tile_addr<D>(sDO, row, col), dof[ks][0], dof[ks][1], dof[ks][2], dof[ks][3]);
  }
  const int qrow0 = q0 + warp * 16 + (lane >> 2);
  float lrow[2], drow[2];
#pragma unroll
  for (int r = 0; r < 2; ++r) {
    const int s = qrow0 + r * 8;
    const long long idx = (static_cast<long long>(b) * p.nq + h) * p.S + s;
    lrow[r] = (s < p.S) ? p.lse[idx] * 1.4426950408889634f : INFINITY;
    drow[r] = (s < p.S) ? p.dvec[idx] : 0.f;
  }

  float dq[ND][4];
#pragma unroll
  for (int i = 0; i < ND; ++i) { dq[i][0] = dq[i][1] = dq[i][2] = dq[i][3] = 0.f; }

  for (int j = 0; j < nblk; ++j) {
    const int st = j & 1;
    if (j + 1 < nblk) {
      load_tile_async<BN, D, NT>(sK + (st ^ 1) * BN * D * 2, gk, p.ldk, (j + 1) * BN, p.S);
      load_tile_async<BN, D, NT>(sV + (st ^ 1) * BN * D * 2, gv, p.ldv, (j + 1) * BN, p.S);
    }
    cp_async_commit();
    const uint32_t cK = sK + st * BN * D * 2, cV = sV + st * BN * D * 2;
    const int k0 = j * BN;
    const bool active = k0 <= q0 + warp * 16 + 15;
    if (active) {
      float s[BN / 8][4], dp[BN / 8][4];
#pragma unroll
      for (int i = 0; i < BN / 8; ++i) { s[i][0] = s[i][1] = s[i][2] = s[i][3] = 0.f; dp[i][0] = dp[i][1] = dp[i][2] = dp[i][3] = 0.f; }
#pragma unroll
      for (int ks = 0; ks < KS; ++ks) {
#pragma unroll
        for (int np = 0; np < BN / 16; ++np) {
          uint32_t b0, b1, b2, b3;
          const int key = np * 16 + (lane & 7) + (lane >> 4) * 8;
          const int col = ks * 16 + ((lane >> 3) & 1) * 8;
          ldsm_x4(tile_addr<D>(cK, key, col), b0, b1, b2, b3);
          mma16816(s[2 * np], qf[ks], b0, b1);
          mma16816(s[2 * np + 1], qf[ks], b2, b3);
          ldsm_x4(tile_addr<D>(cV, key, col), b0, b1, b2, b3);
          mma16816(dp[2 * np], dof[ks], b0, b1);
          mma16816(dp[2 * np + 1], dof[ks], b2, b3);
        }
      }
      const bool need_mask = (k0 + BN - 1 > q0 + warp * 16) || (k0 + BN > p.S);
#pragma unroll
      for (int i = 0; i < BN / 8; ++i) {
#pragma unroll
        for (int e = 0; e < 4; ++e) {
          const int r = e >> 1;
          float pv = exp2f(s[i][e] * p.scale_log2 - lrow[r]);
          if (need_mask) {
            const int key = k0 + i * 8 + (lane & 3) * 2 + (e & 1);
            if (key > qrow0 + r * 8 || key >= p.S) pv = 0.f;
          }
          s[i][e] = pv * (dp[i][e] - drow[r]);              // dS
        }
      }
#pragma unroll
      for (int kk = 0; kk < BN / 16; ++kk) {
        uint32_t sa[4];
        sa[0] = pack_f16(s[2 * kk][0], s[2 * kk][1]);
        sa[1] = pack_f16(s[2 * kk][2], s[2 * kk][3]);
        sa[2] = pack_f16(s[2 * kk + 1][0], s[2 * kk + 1][1]);
        sa[3] = pack_f16(s[2 * kk + 1][2], s[2 * kk + 1][3]);
#pragma unroll
        for (int dpi = 0; dpi < ND / 2; ++dpi) {
          uint32_t b0, b1, b2, b3;
          ldsm_x4_t(tile_addr<D>(cK, kk * 16 + (lane & 7) + ((lane >> 3) & 1) * 8, dpi * 16 + (lane >> 4) * 8), b0, b1, b2, b3);
          mma16816(dq[2 * dpi], sa, b0, b1);
          mma16816(dq[2 * dpi + 1], sa, b2, b3);
        }
      }
    }
    cp_async_wait<0>();
    __syncthreads();
  }
  store_grad_tile<D>(dq, p.scale, p.rope, p.S, tok0, qrow0, lane, p.dq32, p.lddq32, p.dq16, p.ldd16, h * D);
}

// ------------------------------------------------------------------------------------------- launchers
template <int D> constexpr int attn_fwd_smem() { return (128 + 4 * 64) * D * 2; }
template <int D> constexpr int attn_dkdv_smem() { return (2 * 64 + 4 * 64) * D * 2 + 4 * 64 * 4; }
template <int D> constexpr int attn_dq_smem() { return (2 * 64 + 4 * 64) * D * 2; }

template <int D>
cudaError_t attn_fwd_launch(const AttnParams& p, cudaStream_t st) {
  static DeviceOnce once;
  if (once.need()) {
    cudaError_t e = cudaFuncSetAttribute(attn_fwd_kernel<D>, cudaFuncAttributeMaxDynamicSharedMemorySize, attn_fwd_smem<D>());
    if (e != cudaSuccess) return e;
    once.done();
  }
  dim3 grid((p.S + 127) / 128, p.nq, p.B);
  return launch_kernel(attn_fwd_kernel<D>, grid, dim3(256), attn_fwd_smem<D>(), st, p);
}
template <int D, bool PARTS4>
cudaError_t attn_dvec_launch(const __half* dO, long long lddo, const float* o32, long long ldo, float* dvec, int B, int S,
                             int nq, cudaStream_t st) {
  const long long warps = static_cast<long long>(B) * S * nq;
  const int threads = 256;
  const long long blocks = (warps * 32 + threads - 1) / threads;
  return launch_kernel(attn_dvec_kernel<D, PARTS4>, dim3(static_cast<unsigned>(blocks)), dim3(threads), 0, st, dO, lddo, o32, ldo, dvec, B, S, nq);
}
template <int D>
cudaError_t attn_bwd_launch(const AttnParams& p, cudaStream_t st) {
  static DeviceOnce once;
  if (once.need()) {
    cudaError_t e = cudaFuncSetAttribute(attn_bwd_dkdv_kernel<D>, cudaFuncAttributeMaxDynamicSharedMemorySize, attn_dkdv_smem<D>());
    if (e != cudaSuccess) return e;
    e = cudaFuncSetAttribute(attn_bwd_dq_kernel<D>, cudaFuncAttributeMaxDynamicSharedMemorySize, attn_dq_smem<D>());
    if (e != cudaSuccess) return e;
    once.done();
  }
  dim3 g1((p.S + 63) / 64, p.nkv, p.B);
  cudaError_t e = launch_kernel(attn_bwd_dkdv_kernel<D>, g1, dim3(128), attn_dkdv_smem<D>(), st, p);
  if (e != cudaSuccess) return e;
  dim3 g2((p.S + 63) / 64, p.nq, p.B);
  return launch_kernel(attn_bwd_dq_kernel<D>, g2, dim3(128), attn_dq_smem<D>(), st, p);
}

}  // namespace lsp
