// Causal grouped-query flash attention on the 5th-generation tensor cores (sm_100a), head_dim 128, fp16 operands,
// fp32 accumulation in TMEM.  SURVEY 8(a) F3 (forward, saves the log-sum-exp) -- refs [23],[24],[26],[27],[37].
//
// Forward.  One CTA owns 256 consecutive queries of one (batch, head) as two 128-row tiles t = 0,1 that ping-pong:
// while the 128 softmax threads of tile t turn S_t = Q_t K_j^T into P_t, the tensor core works on the other tile.
//   warp 0      TMA producer: Q_0, Q_1 once, then K_j / V_j (128 keys x 128) through two-stage mbarrier rings
//   warp 1      tcgen05.mma issuer (one thread) and TMEM owner
//   warps 2-5   softmax of tile 0 (thread = one query row = one TMEM lane; no shuffles for row max / row sum)
//   warps 6-9   softmax of tile 1
// TMEM (512 columns): S_0 [0,128) S_1 [128,256) O_0 [256,384) O_1 [384,512).  P_t (fp16, two keys per 32-bit column)
// overwrites columns [0,64) of S_t once the thread holds its S row in registers, and is the A operand (from TMEM) of
// O_t += P_t V_j, whose B operand V_j is read MN-major from shared memory exactly as TMA wrote it (no transpose).
// Online softmax with lazy rescaling: the running maximum is only raised (and O_t rescaled in TMEM) when it grew by
// more than 2^8 for some row of the warp, so the TMEM round trip of O is rare after the first blocks; P <= 2^8 fits
// fp16 with the same relative precision.  Key blocks above the diagonal are never visited; only the diagonal block
// is masked.  Rows past the end of a sequence are zero-filled by TMA (3-D maps: column, position, batch).
#pragma once
#include "gemm.cuh"

namespace lsp {

struct AttnTcMaps {
  CUtensorMap q, k, v, dO;
};

struct AttnTcParams {
  int B, S, nq, nkv;
  float scale_log2;            // (1/sqrt(d)) * log2(e)
  float scale;
  float* o32; __half* o16; long long ldo;        // [T, ldo] outputs (either may be null)
  float* lse;                                    // [B, nq, S]
};

constexpr int ATC_D = 128;
constexpr int ATC_TILE_BYTES = 128 * ATC_D * 2;          // one 128 x 128 fp16 tile = 32 KB (two 64-wide swizzled chunks)
constexpr int ATC_CHUNK_BYTES = 128 * 128;               // one 64-column chunk of 128 rows
constexpr int ATC_FWD_THREADS = 320;
constexpr int ATC_FWD_SMEM = 6 * ATC_TILE_BYTES + 1024 + 256;
constexpr float ATC_RESCALE_LOG2 = 8.0f;

// 3-D map over a [B*S, ld] fp16 matrix seen as (column, position, batch); box = 64 columns x 128 positions.
inline bool make_map_attn(CUtensorMap* m, const void* base, int ncols, int S, int B, long long ld) {
  PFN_encodeTiled fn = get_encode_fn();
  if (!fn) return false;
  cuuint64_t dims[3] = {static_cast<cuuint64_t>(ncols), static_cast<cuuint64_t>(S), static_cast<cuuint64_t>(B)};
  cuuint64_t strides[2] = {static_cast<cuuint64_t>(ld) * 2, static_cast<cuuint64_t>(ld) * 2 * static_cast<cuuint64_t>(S)};
  cuuint32_t box[3] = {64u, 128u, 1u};
  cuuint32_t estr[3] = {1u, 1u, 1u};
  return fn(m, CU_TENSOR_MAP_DATA_TYPE_FLOAT16, 3, const_cast<void*>(base), dims, strides, box, estr,
            CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
            CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
}

// A 128-row x 128-column fp16 tile lands as two chunks of [128 rows x 128 B].
__device__ __forceinline__ void atc_load_tile(uint32_t dst, const CUtensorMap* m, uint32_t bar, int col0, int s0, int b) {
  mbar_expect_tx(bar, ATC_TILE_BYTES);
  tma_load_3d(dst, m, bar, col0, s0, b);
  tma_load_3d(dst + ATC_CHUNK_BYTES, m, bar, col0 + 64, s0, b);
}

// K-major 128 x 128 operand tile (rows = M or N index, 128 contiguous K elements split in two chunks): descriptor of
// the kk-th 16-element K step.
__device__ __forceinline__ uint64_t atc_desc_kmajor(uint32_t tile, int kk) {
  return umma_smem_desc(tile + (kk >> 2) * ATC_CHUNK_BYTES + (kk & 3) * 32, 16, 1024);
}
// MN-major 128 (K rows) x 128 (MN contiguous) operand tile: two 64-wide MN chunks 16 KB apart (LBO), 8-row atoms
// 1 KB apart (SBO); the kk-th 16-row K step starts 2 KB further.
__device__ __forceinline__ uint64_t atc_desc_mnmajor(uint32_t tile, int kk) {
  return umma_smem_desc(tile + kk * 2048, ATC_CHUNK_BYTES, 1024);
}

__global__ void __launch_bounds__(ATC_FWD_THREADS, 1)
attn_fwd_tc_kernel(const __grid_constant__ AttnTcMaps maps, const AttnTcParams p) {
  extern __shared__ uint8_t smem_raw[];
  const uint32_t smem_base = (smem_u32(smem_raw) + 1023u) & ~1023u;
  const uint32_t sQ = smem_base;                              // 2 tiles
  const uint32_t sK = sQ + 2 * ATC_TILE_BYTES;                // 2 stages
  const uint32_t sV = sK + 2 * ATC_TILE_BYTES;                // 2 stages
  const uint32_t bar_base = sV + 2 * ATC_TILE_BYTES;
  auto q_full = [&](int t) { return bar_base + 8u * t; };
  auto k_full = [&](int s) { return bar_base + 8u * (2 + s); };
  auto k_empty = [&](int s) { return bar_base + 8u * (4 + s); };
  auto v_full = [&](int s) { return bar_base + 8u * (6 + s); };
  auto v_empty = [&](int s) { return bar_base + 8u * (8 + s); };
  auto s_full = [&](int t) { return bar_base + 8u * (10 + t); };
  auto p_full = [&](int t) { return bar_base + 8u * (12 + t); };
  auto o_full = [&](int t) { return bar_base + 8u * (14 + t); };
  const uint32_t tmem_slot = bar_base + 8u * 16;
  uint32_t* tmem_slot_ptr = reinterpret_cast<uint32_t*>(smem_raw + (tmem_slot - smem_u32(smem_raw)));

  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int qb = gridDim.x - 1 - blockIdx.x;                  // heavy (late) query blocks first
  const int h = blockIdx.y, b = blockIdx.z;
  const int kvh = h / (p.nq / p.nkv);
  const int q0 = qb * 256;
  // key blocks per tile: tile t covers queries [q0 + 128 t, +128); causal => keys [0, q0 + 128 t + 128)
  const int n0 = q0 / 128 + 1;
  const int n1 = (q0 + 128 < p.S) ? n0 + 1 : 0;
  const int nmax = n1 > n0 ? n1 : n0;

  if (threadIdx.x == 0) {
    tma_prefetch_desc(&maps.q); tma_prefetch_desc(&maps.k); tma_prefetch_desc(&maps.v);
    for (int i = 0; i < 2; ++i) {
      mbar_init(q_full(i), 1);
      mbar_init(k_full(i), 1); mbar_init(k_empty(i), 1);
      mbar_init(v_full(i), 1); mbar_init(v_empty(i), 1);
      mbar_init(s_full(i), 1); mbar_init(p_full(i), 4); mbar_init(o_full(i), 1);
    }
    fence_barrier_init();
  }
  if (warp == 1) {
    tmem_alloc(tmem_slot, 512);
    tmem_relinquish();
  }
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tmem_base = *tmem_slot_ptr;

  if (warp == 0) {
    // ===================================================================== TMA producer
    if (lane == 0) {
      atc_load_tile(sQ, &maps.q, q_full(0), h * ATC_D, q0, b);
      if (n1 > 0) atc_load_tile(sQ + ATC_TILE_BYTES, &maps.q, q_full(1), h * ATC_D, q0 + 128, b);
      for (int j = 0; j < nmax; ++j) {
        const int st = j & 1;
        const uint32_t ph = ((j >> 1) & 1) ^ 1u;
        mbar_wait(k_empty(st), ph);
        atc_load_tile(sK + st * ATC_TILE_BYTES, &maps.k, k_full(st), kvh * ATC_D, j * 128, b);
        mbar_wait(v_empty(st), ph);
        atc_load_tile(sV + st * ATC_TILE_BYTES, &maps.v, v_full(st), kvh * ATC_D, j * 128, b);
      }
    }
  } else if (warp == 1) {
    // ===================================================================== MMA issuer
    if (lane == 0) {
      const uint32_t idesc_s = umma_idesc(128, 128, 0, 0, 0, 0);     // S = Q K^T : both K-major
      const uint32_t idesc_pv = umma_idesc(128, 128, 0, 0, 0, 1);    // O += P V  : A from TMEM, B (V) MN-major
      const int nt[2] = {n0, n1};
      auto issue_s = [&](int t, int kst) {
        const uint32_t qa = sQ + t * ATC_TILE_BYTES, ka = sK + kst * ATC_TILE_BYTES;
#pragma unroll
        for (int kk = 0; kk < 8; ++kk)
          umma_f16(tmem_base + t * 128, atc_desc_kmajor(qa, kk), atc_desc_kmajor(ka, kk), idesc_s, kk != 0 ? 1u : 0u);
        umma_commit(s_full(t));
      };
      auto issue_pv = [&](int t, int vst, bool acc) {
        const uint32_t va = sV + vst * ATC_TILE_BYTES;
#pragma unroll
        for (int kk = 0; kk < 8; ++kk)
          umma_f16_ts(tmem_base + 256 + t * 128, tmem_base + t * 128 + kk * 8, atc_desc_mnmajor(va, kk), idesc_pv,
                      (acc || kk != 0) ? 1u : 0u);
        umma_commit(o_full(t));
      };
      mbar_wait(k_full(0), 0);
      mbar_wait(q_full(0), 0);
      tc_fence_after();
      issue_s(0, 0);
      if (n1 > 0) { mbar_wait(q_full(1), 0); tc_fence_after(); issue_s(1, 0); }
      umma_commit(k_empty(0));
      for (int j = 0; j < nmax; ++j) {
        const int st = j & 1;
        const uint32_t ph = (j >> 1) & 1;
        mbar_wait(v_full(st), ph);
        bool knext_ready = false;
        for (int t = 0; t < 2; ++t) {
          if (j < nt[t]) {
            mbar_wait(p_full(t), j & 1);
            tc_fence_after();
            issue_pv(t, st, j > 0);
          }
          if (j + 1 < nt[t]) {
            if (!knext_ready) { mbar_wait(k_full(st ^ 1), ((j + 1) >> 1) & 1); tc_fence_after(); knext_ready = true; }
            issue_s(t, st ^ 1);
          }
        }
        umma_commit(v_empty(st));
        if (j + 1 < nmax) umma_commit(k_empty(st ^ 1));
      }
    }
  } else {
    // ===================================================================== softmax warps: tile t, TMEM lane quarter
    const int t = (warp - 2) >> 2;
    const int quarter = warp & 3;
    const int nblk = t == 0 ? n0 : n1;
    const int row = quarter * 32 + lane;                         // query row within the tile = TMEM lane
    const int qi = q0 + t * 128 + row;                           // position in the sequence
    const uint32_t lane_off = static_cast<uint32_t>(quarter * 32) << 16;
    const uint32_t tS = tmem_base + lane_off + t * 128;
    const uint32_t tO = tmem_base + lane_off + 256 + t * 128;
    const float c = p.scale_log2;
    float m_run = -INFINITY, l_run = 0.f;

    for (int j = 0; j < nblk; ++j) {
      mbar_wait(s_full(t), j & 1);
      tc_fence_after();
      uint32_t sr[4][32];
#pragma unroll
      for (int q = 0; q < 4; ++q) tmem_ld32(tS + q * 32, sr[q]);
      tmem_ld_wait();
      float (&s)[4][32] = reinterpret_cast<float(&)[4][32]>(sr);
      if (j == nblk - 1) {                                       // diagonal block: key 128 j + cidx > query <=> cidx > row
#pragma unroll
        for (int q = 0; q < 4; ++q)
#pragma unroll
          for (int i = 0; i < 32; ++i)
            if (q * 32 + i > row) s[q][i] = -INFINITY;
      }
      float mx0 = s[0][0], mx1 = s[1][0], mx2 = s[2][0], mx3 = s[3][0];
#pragma unroll
      for (int i = 1; i < 32; ++i) {
        mx0 = fmaxf(mx0, s[0][i]); mx1 = fmaxf(mx1, s[1][i]); mx2 = fmaxf(mx2, s[2][i]); mx3 = fmaxf(mx3, s[3][i]);
      }
      const float m_new = fmaxf(m_run, fmaxf(fmaxf(mx0, mx1), fmaxf(mx2, mx3)));
      float m_use = m_run;
      if (j == 0) {
        m_use = m_new;
      } else {
        const bool grow = (m_new - m_run) * c > ATC_RESCALE_LOG2;
        if (__any_sync(0xffffffffu, grow)) {
          // raise the reference maximum of every row of this warp and rescale O_t in TMEM
          const float alpha = exp2f((m_run - m_new) * c);
          m_use = m_new;
          l_run *= alpha;
          mbar_wait(o_full(t), (j - 1) & 1);                     // P_t V_{j-1} has landed in O_t
          tc_fence_after();
#pragma unroll
          for (int q = 0; q < 4; ++q) {
            uint32_t orr[32];
            tmem_ld32(tO + q * 32, orr);
            tmem_ld_wait();
#pragma unroll
            for (int i = 0; i < 32; ++i) orr[i] = __float_as_uint(__uint_as_float(orr[i]) * alpha);
            tmem_st32(tO + q * 32, orr);
          }
        }
      }
      m_run = m_use;
      const float neg = -m_use * c;
      float sum0 = 0.f, sum1 = 0.f;
#pragma unroll
      for (int q = 0; q < 2; ++q) {
        uint32_t pk[32];
#pragma unroll
        for (int i = 0; i < 16; ++i) {
          const float a0 = exp2f(fmaf(s[2 * q][2 * i], c, neg)), a1 = exp2f(fmaf(s[2 * q][2 * i + 1], c, neg));
          const float b0 = exp2f(fmaf(s[2 * q + 1][2 * i], c, neg)), b1 = exp2f(fmaf(s[2 * q + 1][2 * i + 1], c, neg));
          sum0 += a0 + a1; sum1 += b0 + b1;
          pk[i] = pack_f16(a0, a1);
          pk[16 + i] = pack_f16(b0, b1);
        }
        tmem_st32(tS + q * 32, pk);                              // P_t: keys 64 q .. 64 q + 63 -> 32 columns
      }
      l_run += sum0 + sum1;
      tmem_st_wait();
      tc_fence_before();
      __syncwarp();
      if (lane == 0) mbar_arrive(p_full(t));
    }

    if (nblk > 0) {
      mbar_wait(o_full(t), (nblk - 1) & 1);
      tc_fence_after();
      const bool valid = qi < p.S;
      const float inv = 1.0f / l_run;
      const long long tok = static_cast<long long>(b) * p.S + qi;
      if (valid) p.lse[(static_cast<long long>(b) * p.nq + h) * p.S + qi] = (m_run * c + log2f(l_run)) * 0.6931471805599453f;
#pragma unroll
      for (int q = 0; q < 4; ++q) {
        uint32_t orr[32];
        tmem_ld32(tO + q * 32, orr);
        tmem_ld_wait();
        float (&o)[32] = reinterpret_cast<float(&)[32]>(orr);
#pragma unroll
        for (int i = 0; i < 32; ++i) o[i] *= inv;
        if (valid) {
          const long long off = tok * p.ldo + h * ATC_D + q * 32;
          if (p.o32) store_row32<DT_F32>(p.o32 + off, o, 32);
          if (p.o16) store_row32<DT_F16>(p.o16 + off, o, 32);
        }
      }
    }
  }

  tc_fence_before();
  __syncthreads();
  if (warp == 1) {
    tc_fence_after();
    tmem_dealloc(tmem_base, 512);
  }
}

// q [B*S, ldq] (head h at columns h*128), k, v [B*S, ldk/ldv] (kv head at columns kvh*128), all fp16.
inline cudaError_t attn_fwd_tc_launch(const __half* q, long long ldq, const __half* k, long long ldk, const __half* v,
                                      long long ldv, const AttnTcParams& p, cudaStream_t st) {
  static bool set = false;
  if (!set) {
    cudaError_t e = cudaFuncSetAttribute(attn_fwd_tc_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, ATC_FWD_SMEM);
    if (e != cudaSuccess) return e;
    set = true;
  }
  AttnTcMaps maps;
  if (!make_map_attn(&maps.q, q, p.nq * ATC_D, p.S, p.B, ldq) || !make_map_attn(&maps.k, k, p.nkv * ATC_D, p.S, p.B, ldk) ||
      !make_map_attn(&maps.v, v, p.nkv * ATC_D, p.S, p.B, ldv))
    return cudaErrorInvalidValue;
  maps.dO = maps.q;
  dim3 grid((p.S + 255) / 256, p.nq, p.B);
  attn_fwd_tc_kernel<<<grid, ATC_FWD_THREADS, ATC_FWD_SMEM, st>>>(maps, p);
  return cudaGetLastError();
}

}  // namespace lsp
