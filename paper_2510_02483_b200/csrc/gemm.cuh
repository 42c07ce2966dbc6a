// Persistent warp-specialised tcgen05 GEMM for sm_100a with fused epilogues.
//
//   C[M,N] = sum over K-segments s of  A_s[M,K_s] * B_s[N,K_s]^T        (fp32 accumulate in TMEM)
//
// Operands are 16-bit (both fp16 or both bf16), fetched by TMA into 128B-swizzled shared memory in a multi-stage
// mbarrier ring; either operand may be K-major (row = M/N index, K contiguous) or MN-major
// (row = K index, M/N contiguous) so that dgrad (dX = dY W) and wgrad (dW = dY^T X) run on the
// tensors as they lie in HBM -- no transposes.  One elected thread issues tcgen05.mma
// (128 x BN x 16, cta_group::1); two TMEM accumulator stages let the 4 epilogue warps drain tile i
// (tcgen05.ld -> registers -> fused epilogue -> global) while the tensor core works on tile i+1.
//
// DUAL mode: B tile rows [0,128) come from b[0] and rows [128,256) from b[1] (same 128 output columns);
// one 128x256 MMA then yields both the gate and the up projection, which the SwiGLU epilogue combines.
//
// Warp roles (320 threads): warp 0 = TMA producer, warp 1 = MMA issuer + TMEM owner, warps 2..9 = epilogue
// (TMEM lane quarter = warp & 3; the two warps of a quarter take alternate 32-column chunks).
//
// Tile order: persistent CTAs take tiles i, i + grid, ...; tile ids run m-fastest inside bands of `band`
// m-blocks and sweep all n-blocks before moving to the next band, so the ~148 tiles in flight form a compact
// band x (148/band) block: each A k-slice is shared by ~148/band CTAs and each B k-slice by `band` CTAs through
// L2, and the band's A panel stays L2-resident for the sweep (m-fastest over all of M re-read A once per
// n-block: 4-6 GB of DRAM reads per GEMM at the 3B shape, profiles/r1_gemm_ncu.md).
#pragma once
#include <stdlib.h>

#include "ptx.cuh"

namespace lsp {

enum : int { DT_BF16 = 0, DT_F32 = 1, DT_F16 = 2 };

constexpr int GEMM_BM = 128;
constexpr int GEMM_BK = 64;          // 64 x 16-bit = one 128-byte swizzle row
constexpr int GEMM_THREADS = 320;         // warp 0 TMA, warp 1 MMA, warps 2..9 epilogue
constexpr int GEMM_EPI_WARPS = 8;
constexpr int GEMM_MAX_SEG = 3;

struct GemmMaps {
  CUtensorMap a[GEMM_MAX_SEG];
  CUtensorMap b[GEMM_MAX_SEG];
};
struct GemmShape {
  int M, N;                          // output extent (DUAL: N = columns of each of the two outputs)
  int a_fmt, b_fmt;                  // UMMA operand formats: 0 = fp16, 1 = bf16; must be equal (a mixed pair is an
                                     // illegal instruction on sm_100a -- measured)
  int nseg;                          // number of K segments (non-DUAL); DUAL uses a[0], b[0], b[1]
  int band;                          // m-blocks per rasterisation band (>= 1)
  int kblocks[GEMM_MAX_SEG];         // ceil(K_s / 64)
  // stream-K tail of the CTA-pair kernel (all zero / null: data-parallel only)
  int sk_split;                      // s >= 2: the T mod C tiles of the last wave are each cut into s K-slices (0: off)
  float* sk_partial;                 // [clusters][2 CTAs][8 chunks][128 rows][32] fp32 partial accumulators
  unsigned int* sk_flags;            // [clusters][2]: epoch of the partial published by that CTA; 0 again once consumed
  unsigned int sk_epoch;             // unique per launch on this context, > 0
};

typedef CUresult (*PFN_encodeTiled)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*,
                                    const cuuint64_t*, const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave,
                                    CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

inline PFN_encodeTiled get_encode_fn() {
  static PFN_encodeTiled fn = nullptr;
  if (!fn) {
    void* p = nullptr;
    cudaDriverEntryPointQueryResult q;
    if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &q) == cudaSuccess &&
        q == cudaDriverEntryPointSuccess)
      fn = reinterpret_cast<PFN_encodeTiled>(p);
  }
  return fn;
}

// 2-D map over a row-major [rows, cols] output (pitch ld elements) for 32 x 32 chunk stores out of a staging tile:
// fp32 rows are 128 B (128B swizzle), 16-bit rows 64 B (64B swizzle) -- the XOR patterns of WarpStage::put_row32/16.
inline bool make_map_store2d(CUtensorMap* m, const void* base, long long rows, long long cols, long long ld, int dt) {
  PFN_encodeTiled fn = get_encode_fn();
  if (!fn || rows <= 0 || cols <= 0) return false;
  const cuuint64_t es = dt == DT_F32 ? 4 : 2;
  cuuint64_t dims[2] = {static_cast<cuuint64_t>(cols), static_cast<cuuint64_t>(rows)};
  cuuint64_t strides[1] = {static_cast<cuuint64_t>(ld) * es};
  cuuint32_t box[2] = {32u, 32u};
  cuuint32_t estr[2] = {1u, 1u};
  const CUtensorMapDataType t = dt == DT_F32 ? CU_TENSOR_MAP_DATA_TYPE_FLOAT32
                              : (dt == DT_F16 ? CU_TENSOR_MAP_DATA_TYPE_FLOAT16 : CU_TENSOR_MAP_DATA_TYPE_BFLOAT16);
  return fn(m, t, 2, const_cast<void*>(base), dims, strides, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE,
            dt == DT_F32 ? CU_TENSOR_MAP_SWIZZLE_128B : CU_TENSOR_MAP_SWIZZLE_64B, CU_TENSOR_MAP_L2_PROMOTION_NONE,
            CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
}

// 4-D fp32 map that un-permutes rows on the way out (rope_layout = 1): the GEMM's row
// head*d + 2i + half is row head*d + half*d/2 + i of the [rows, cols] output.  Dimensions (col, half, i, head); a box of
// 32 cols x 2 halves x 16 i is 32 consecutive GEMM rows in shared memory (i-major, half-minor), 128 B each.
inline bool make_map_store_perm(CUtensorMap* m, const void* base, long long rows, long long cols, long long ld, int d) {
  PFN_encodeTiled fn = get_encode_fn();
  if (!fn || rows <= 0 || cols <= 0 || d < 32 || rows % d) return false;
  cuuint64_t dims[4] = {static_cast<cuuint64_t>(cols), 2, static_cast<cuuint64_t>(d / 2), static_cast<cuuint64_t>(rows / d)};
  cuuint64_t strides[3] = {static_cast<cuuint64_t>(d / 2) * ld * 4, static_cast<cuuint64_t>(ld) * 4, static_cast<cuuint64_t>(d) * ld * 4};
  cuuint32_t box[4] = {32u, 2u, 16u, 1u};
  cuuint32_t estr[4] = {1u, 1u, 1u, 1u};
  return fn(m, CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 4, const_cast<void*>(base), dims, strides, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE,
            CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_NONE, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
}

template <int BN> struct GemmCfg {
  static constexpr int A_BYTES = GEMM_BM * GEMM_BK * 2;
  static constexpr int B_BYTES = BN * GEMM_BK * 2;
  static constexpr int STAGE_BYTES = A_BYTES + B_BYTES;
  static constexpr int STAGES = (BN == 256) ? 4 : 6;
  static constexpr int SMEM_BYTES = STAGES * STAGE_BYTES + 8 * 4096 /*staging tiles*/ + 1024 /*align slack*/ + 256 /*barriers*/;
  static constexpr int TMEM_COLS = 2 * BN;   // two accumulator stages (power of two: 256 or 512)
};

// ------------------------------------------------------------------------------------------- store helpers
template <int DT> struct OutElem;
template <> struct OutElem<DT_BF16> { using type = __nv_bfloat16; };
template <> struct OutElem<DT_F16> { using type = __half; };
template <> struct OutElem<DT_F32> { using type = float; };

// Write up to 32 consecutive values of one row (nvalid is a multiple of 8; p is 16-byte aligned).
template <int DT>
__device__ __forceinline__ void store_row32(void* p, const float (&v)[32], int nvalid) {
  if constexpr (DT == DT_F32) {
    float4* q = reinterpret_cast<float4*>(p);
#pragma unroll
    for (int j = 0; j < 8; ++j)
      if (4 * j + 4 <= nvalid) q[j] = make_float4(v[4 * j], v[4 * j + 1], v[4 * j + 2], v[4 * j + 3]);
  } else {
    uint4* q = reinterpret_cast<uint4*>(p);
#pragma unroll
    for (int j = 0; j < 4; ++j)
      if (8 * j + 8 <= nvalid) {
        uint4 w;
        if constexpr (DT == DT_BF16) {
          w.x = pack_bf16(v[8 * j], v[8 * j + 1]); w.y = pack_bf16(v[8 * j + 2], v[8 * j + 3]);
          w.z = pack_bf16(v[8 * j + 4], v[8 * j + 5]); w.w = pack_bf16(v[8 * j + 6], v[8 * j + 7]);
        } else {
          w.x = pack_f16(v[8 * j], v[8 * j + 1]); w.y = pack_f16(v[8 * j + 2], v[8 * j + 3]);
          w.z = pack_f16(v[8 * j + 4], v[8 * j + 5]); w.w = pack_f16(v[8 * j + 6], v[8 * j + 7]);
        }
        q[j] = w;
      }
  }
}
// Read up to 32 consecutive values of one row into fp32.
template <int DT>
__device__ __forceinline__ void load_row32(const void* p, float (&v)[32], int nvalid) {
  if constexpr (DT == DT_F32) {
    const float4* q = reinterpret_cast<const float4*>(p);
#pragma unroll
    for (int j = 0; j < 8; ++j) {
      float4 t = (4 * j + 4 <= nvalid) ? __ldg(q + j) : make_float4(0.f, 0.f, 0.f, 0.f);
      v[4 * j] = t.x; v[4 * j + 1] = t.y; v[4 * j + 2] = t.z; v[4 * j + 3] = t.w;
    }
  } else {
    const uint4* q = reinterpret_cast<const uint4*>(p);
#pragma unroll
    for (int j = 0; j < 4; ++j) {
      uint4 t = (8 * j + 8 <= nvalid) ? __ldg(q + j) : make_uint4(0, 0, 0, 0);
      const uint32_t w[4] = {t.x, t.y, t.z, t.w};
#pragma unroll
      for (int e = 0; e < 4; ++e) {
        if constexpr (DT == DT_BF16) {
          v[8 * j + 2 * e] = bf16_lo(w[e]); v[8 * j + 2 * e + 1] = bf16_hi(w[e]);
        } else {
          const __half2 h = *reinterpret_cast<const __half2*>(&w[e]);
          v[8 * j + 2 * e] = __low2float(h); v[8 * j + 2 * e + 1] = __high2float(h);
        }
      }
    }
  }
}

// Split-K partial accumulators: chunk layout [unit j = 0..7][row 0..127][4 floats], so that the 32 lanes of a warp
// (consecutive rows) write / read 512 contiguous bytes per instruction.  Written by ANOTHER CTA during this kernel:
// plain coherent loads, never ld.global.nc.
__device__ __forceinline__ void partial_store(float* chunk, int row, const float (&v)[32]) {
#pragma unroll
  for (int j = 0; j < 8; ++j)
    *reinterpret_cast<float4*>(chunk + (j * GEMM_BM + row) * 4) = make_float4(v[4 * j], v[4 * j + 1], v[4 * j + 2], v[4 * j + 3]);
}
__device__ __forceinline__ void partial_load(const float* chunk, int row, float (&v)[32]) {
#pragma unroll
  for (int j = 0; j < 8; ++j) {
    float4 t;
    asm volatile("ld.global.v4.f32 {%0, %1, %2, %3}, [%4];" : "=f"(t.x), "=f"(t.y), "=f"(t.z), "=f"(t.w)
                 : "l"(chunk + (j * GEMM_BM + row) * 4) : "memory");
    v[4 * j] = t.x; v[4 * j + 1] = t.y; v[4 * j + 2] = t.z; v[4 * j + 3] = t.w;
  }
}
__device__ __forceinline__ void named_bar_sync_gemm(int id, int nthreads) {
  asm volatile("bar.sync %0, %1;" ::"r"(id), "r"(nthreads) : "memory");
}

// ------------------------------------------------------------------------------------------- warp staging tile
// tcgen05.ld hands every thread one accumulator ROW (32 consecutive columns).  Writing that straight to global memory
// makes each warp instruction touch 32 rows x 16 B (32 half-filled sectors): the unoverlapped epilogue of a 256 x 256
// fp32 tile took ~30 k cycles (8.7 B/clk/SM).  Each epilogue warp therefore owns a 4 KB shared-memory tile
// (32 rows x 128 B, 16-byte units XOR-swizzled so that both access patterns are bank-conflict free): threads exchange
// rows through it and global memory sees 8 lanes x 16 B = one full 128-byte row segment, 4 rows per instruction
// (16-bit data: 4 lanes x 16 B = 64 B, 8 rows per instruction).
constexpr int GEMM_STAGE_TILE_BYTES = 4096;
struct WarpStage {
  uint32_t base;      // shared::cta address of this warp's tile
  int lane;
  // ---- thread = row view, 32-bit elements: row `lane`, units j = 0..7
  __device__ __forceinline__ void put_row32(const float (&v)[32]) const {
#pragma unroll
    for (int j = 0; j < 8; ++j)
      asm volatile("st.shared.v4.f32 [%0], {%1, %2, %3, %4};" ::"r"(base + lane * 128 + ((j ^ (lane & 7)) << 4)),
                   "f"(v[4 * j]), "f"(v[4 * j + 1]), "f"(v[4 * j + 2]), "f"(v[4 * j + 3]) : "memory");
  }
  __device__ __forceinline__ void get_row32(float (&v)[32]) const {
#pragma unroll
    for (int j = 0; j < 8; ++j)
      asm volatile("ld.shared.v4.f32 {%0, %1, %2, %3}, [%4];" : "=f"(v[4 * j]), "=f"(v[4 * j + 1]), "=f"(v[4 * j + 2]), "=f"(v[4 * j + 3])
                   : "r"(base + lane * 128 + ((j ^ (lane & 7)) << 4)) : "memory");
  }
  // ---- thread = row view, 16-bit elements packed in pairs: row `lane` (64 B), units j = 0..3
  __device__ __forceinline__ void put_row16(const uint32_t (&w)[16]) const {
#pragma unroll
    for (int j = 0; j < 4; ++j)
      asm volatile("st.shared.v4.b32 [%0], {%1, %2, %3, %4};" ::"r"(base + lane * 64 + ((j ^ ((lane >> 1) & 3)) << 4)),
                   "r"(w[4 * j]), "r"(w[4 * j + 1]), "r"(w[4 * j + 2]), "r"(w[4 * j + 3]) : "memory");
  }
  __device__ __forceinline__ void get_row16(uint32_t (&w)[16]) const {
#pragma unroll
    for (int j = 0; j < 4; ++j)
      asm volatile("ld.shared.v4.b32 {%0, %1, %2, %3}, [%4];" : "=r"(w[4 * j]), "=r"(w[4 * j + 1]), "=r"(w[4 * j + 2]), "=r"(w[4 * j + 3])
                   : "r"(base + lane * 64 + ((j ^ ((lane >> 1) & 3)) << 4)) : "memory");
  }
  // ---- coalesced view.  rowptr(r) -> pointer to column 0 of the chunk in row r; rows [0, nrows), columns [0, ncols)
  template <class RowPtr>
  __device__ __forceinline__ void to_global32(RowPtr rowptr, int nrows, int ncols) const {
    const int u = lane & 7;
#pragma unroll
    for (int i = 0; i < 8; ++i) {
      const int r = 4 * i + (lane >> 3);
      if (r < nrows && 4 * u + 4 <= ncols) {
        uint4 t;
        asm volatile("ld.shared.v4.b32 {%0, %1, %2, %3}, [%4];" : "=r"(t.x), "=r"(t.y), "=r"(t.z), "=r"(t.w)
                     : "r"(base + r * 128 + ((u ^ (r & 7)) << 4)) : "memory");
        *reinterpret_cast<uint4*>(rowptr(r) + 4 * u) = t;
      }
    }
  }
  template <class RowPtr>
  __device__ __forceinline__ void from_global32(RowPtr rowptr, int nrows, int ncols) const {
    const int u = lane & 7;
#pragma unroll
    for (int i = 0; i < 8; ++i) {
      const int r = 4 * i + (lane >> 3);
      uint4 t = make_uint4(0, 0, 0, 0);
      if (r < nrows && 4 * u + 4 <= ncols) t = __ldg(reinterpret_cast<const uint4*>(rowptr(r) + 4 * u));
      asm volatile("st.shared.v4.b32 [%0], {%1, %2, %3, %4};" ::"r"(base + r * 128 + ((u ^ (r & 7)) << 4)),
                   "r"(t.x), "r"(t.y), "r"(t.z), "r"(t.w) : "memory");
    }
  }
  template <class RowPtr>
  __device__ __forceinline__ void to_global16(RowPtr rowptr, int nrows, int ncols) const {
    const int u = lane & 3;
#pragma unroll
    for (int i = 0; i < 4; ++i) {
      const int r = 8 * i + (lane >> 2);
      if (r < nrows && 8 * u + 8 <= ncols) {
        uint4 t;
        asm volatile("ld.shared.v4.b32 {%0, %1, %2, %3}, [%4];" : "=r"(t.x), "=r"(t.y), "=r"(t.z), "=r"(t.w)
                     : "r"(base + r * 64 + ((u ^ ((r >> 1) & 3)) << 4)) : "memory");
        *reinterpret_cast<uint4*>(rowptr(r) + 8 * u) = t;
      }
    }
  }
  template <class RowPtr>
  __device__ __forceinline__ void from_global16(RowPtr rowptr, int nrows, int ncols) const {
    const int u = lane & 3;
#pragma unroll
    for (int i = 0; i < 4; ++i) {
      const int r = 8 * i + (lane >> 2);
      uint4 t = make_uint4(0, 0, 0, 0);
      if (r < nrows && 8 * u + 8 <= ncols) t = __ldg(reinterpret_cast<const uint4*>(rowptr(r) + 8 * u));
      asm volatile("st.shared.v4.b32 [%0], {%1, %2, %3, %4};" ::"r"(base + r * 64 + ((u ^ ((r >> 1) & 3)) << 4)),
                   "r"(t.x), "r"(t.y), "r"(t.z), "r"(t.w) : "memory");
    }
  }
};

// Row I/O of one warp chunk (32 rows starting at m_base, 32 columns starting at n) through the staging tile.
template <int DT, class RowPtr>
__device__ __forceinline__ void chunk_store(const WarpStage& st, RowPtr rowptr, const float (&v)[32], int nrows, int ncols) {
  __syncwarp();                                  // previous readers of the tile are done
  if constexpr (DT == DT_F32) {
    st.put_row32(v);
    __syncwarp();
    st.to_global32(rowptr, nrows, ncols);
  } else {
    uint32_t w[16];
#pragma unroll
    for (int j = 0; j < 16; ++j) w[j] = DT == DT_BF16 ? pack_bf16(v[2 * j], v[2 * j + 1]) : pack_f16(v[2 * j], v[2 * j + 1]);
    st.put_row16(w);
    __syncwarp();
    st.to_global16(rowptr, nrows, ncols);
  }
}
template <int DT, class RowPtr>
__device__ __forceinline__ void chunk_load(const WarpStage& st, RowPtr rowptr, float (&v)[32], int nrows, int ncols) {
  if (st.lane == 0) tma_store_wait_read<0>();    // a bulk store may still be reading the tile
  __syncwarp();
  if constexpr (DT == DT_F32) {
    st.from_global32(rowptr, nrows, ncols);
    __syncwarp();
    st.get_row32(v);
  } else {
    st.from_global16(rowptr, nrows, ncols);
    __syncwarp();
    uint32_t w[16];
    st.get_row16(w);
#pragma unroll
    for (int j = 0; j < 16; ++j) {
      if constexpr (DT == DT_BF16) { v[2 * j] = bf16_lo(w[j]); v[2 * j + 1] = bf16_hi(w[j]); }
      else { const __half2 h = *reinterpret_cast<const __half2*>(&w[j]); v[2 * j] = __low2float(h); v[2 * j + 1] = __high2float(h); }
    }
  }
}

// TMA store of one warp chunk (32 rows x 32 columns at row r0, column c0 of the tensor behind `map`): the rows go
// into the staging tile in the map's swizzle pattern and ONE bulk tensor store writes them; tails in M and N are
// clipped by the map.  Per-thread st.global of such a tile stalled the warps an order of magnitude longer (measured in
// the attention forward: ~12 k vs ~1 k cycles for 4 chunks), the bulk store is asynchronous.
template <int DT>
__device__ __forceinline__ void chunk_store_tma(const WarpStage& st, const CUtensorMap* map, int c0, int r0, const float (&v)[32],
                                                bool accumulate = false) {
  if (st.lane == 0) tma_store_wait_read<0>();    // the previous bulk store of this warp has read the tile
  __syncwarp();
  if constexpr (DT == DT_F32) {
    st.put_row32(v);
  } else {
    uint32_t w[16];
#pragma unroll
    for (int j = 0; j < 16; ++j) w[j] = DT == DT_BF16 ? pack_bf16(v[2 * j], v[2 * j + 1]) : pack_f16(v[2 * j], v[2 * j + 1]);
    st.put_row16(w);
  }
  fence_proxy_async_smem();                      // generic-proxy writes -> visible to the async proxy
  __syncwarp();
  if (st.lane == 0) {
    if (accumulate) tma_reduce_add_2d(map, st.base, c0, r0);      // out += tile: one fp32 add per element, in the L2
    else tma_store_2d(map, st.base, c0, r0);
    tma_store_commit();
  }
}

// fp32 chunk through a row-un-permuting 4-D map (make_map_store_perm): GEMM rows [r0, r0 + 32) of a head-aligned segment
__device__ __forceinline__ void chunk_store_tma_perm(const WarpStage& st, const CUtensorMap* map, int c0, int r0, int d, const float (&v)[32],
                                                     bool accumulate) {
  if (st.lane == 0) tma_store_wait_read<0>();
  __syncwarp();
  st.put_row32(v);
  fence_proxy_async_smem();
  __syncwarp();
  if (st.lane == 0) {
    const int head = r0 / d, i0 = (r0 - head * d) >> 1;
    if (accumulate) tma_reduce_add_4d(map, st.base, c0, 0, i0, head);
    else tma_store_4d(map, st.base, c0, 0, i0, head);
    tma_store_commit();
  }
}

template <int DT>
__device__ __forceinline__ void chunk_store_tma3(const WarpStage& st, const CUtensorMap* map, int c0, int c1, int c2, const float (&v)[32]) {
  if (st.lane == 0) tma_store_wait_read<0>();
  __syncwarp();
  if constexpr (DT == DT_F32) {
    st.put_row32(v);
  } else {
    uint32_t w[16];
#pragma unroll
    for (int j = 0; j < 16; ++j) w[j] = DT == DT_BF16 ? pack_bf16(v[2 * j], v[2 * j + 1]) : pack_f16(v[2 * j], v[2 * j + 1]);
    st.put_row16(w);
  }
  fence_proxy_async_smem();
  __syncwarp();
  if (st.lane == 0) { tma_store_3d(map, st.base, c0, c1, c2); tma_store_commit(); }
}

// ------------------------------------------------------------------------------------------- epilogues
// Every epilogue works on one warp chunk: rows [m_base, m_base + nrows) (thread `lane` holds row m_base + lane),
// columns [n, n + nvalid); all global traffic goes through the warp's staging tile.
// Plain store with optional residual add and up to three row-segments of output (wgrad of fused QKV / gate-up).
template <int ODT, int RDT, bool HAS_RES>
struct EpiStore {
  static constexpr bool kStoreOnly = !HAS_RES;
  void* out[3];
  int split1, split2;        // rows [0,split1) -> out[0], [split1,split2) -> out[1], [split2,M) -> out[2]; multiples of 32
  long long ld;              // row pitch (elements) of every output and of the residual
  const void* res;
  float alpha;
  const float* alpha_dev = nullptr;   // optional DEVICE scalar multiplied into alpha (a factor only the device knows: the
                                      // valid-token count of the cross-entropy, lsp_head_fwd_bwd)
  CUtensorMap omap[3];       // store maps of the up-to-three outputs (encoded by the host in encode())
  int use_tma;               // 0 when a 32-row chunk can straddle a split (splits not multiples of 32): per-thread stores
  int accumulate = 0;        // 1: out += result (fp32 outputs; lsp_layer_desc.wgrad_accumulate) instead of out = result
  float res_scale = 1.0f;    // weight of the residual (lsp_layer_desc.residual_scale: 0 on all but one tensor-parallel rank)
  int perm_d = 0;            // rope_layout = 1: head_dim; the rows of the segments in perm_segs leave through a 4-D map that
  unsigned perm_segs = 0;    // un-permutes them (dWq, dWk of the row-permuted projection weights)
  bool encode(int M, int N) {
    use_tma = !((split1 < M && split1 % 32) || (split2 < M && split2 % 32));
    if (!use_tma) return perm_segs == 0;
    const int s1 = split1 < M ? split1 : M, s2 = split2 < M ? split2 : M;
    const int rows[3] = {s1, s2 - s1, M - s2};
    for (int i = 0; i < 3; ++i) {
      if (rows[i] > 0 && ((perm_segs >> i) & 1u)) {
        if (ODT != DT_F32 || !make_map_store_perm(&omap[i], out[i], rows[i], N, ld, perm_d)) return false;
        continue;
      }
      if (rows[i] > 0 && !make_map_store2d(&omap[i], out[i], rows[i], N, ld, ODT)) return false;
      if (rows[i] <= 0) omap[i] = omap[0];
    }
    return true;
  }
  // L2 prefetch of what the epilogue of rows [m_base, +nrows) x columns [n0, n0 + ncols) will read (issued by the
  // epilogue warps while the tensor core still works on the tile, so the reads do not pay DRAM latency per chunk)
  __device__ __forceinline__ void prefetch(int lane, int m_base, int n0, int nrows, int ncols) const {
    if constexpr (HAS_RES) {
      using RT = typename OutElem<RDT>::type;
      if (lane < nrows) {
        const RT* rp = reinterpret_cast<const RT*>(res) + static_cast<long long>(m_base + lane) * ld + n0;
        for (int c = 0; c < ncols; c += 128 / static_cast<int>(sizeof(RT))) prefetch_l2(rp + c);
      }
    }
  }
  __device__ __forceinline__ void operator()(const WarpStage& st, int m_base, int n, float (&v)[32], int nrows, int nvalid) const {
    const float al = alpha_dev ? alpha * __ldg(alpha_dev) : alpha;
    if (al != 1.0f) {
#pragma unroll
      for (int j = 0; j < 32; ++j) v[j] *= al;
    }
    if constexpr (HAS_RES) {
      using RT = typename OutElem<RDT>::type;
      float r[32];
      const RT* rbase = reinterpret_cast<const RT*>(res) + static_cast<long long>(m_base) * ld + n;
      chunk_load<RDT>(st, [&](int rr) { return rbase + rr * ld; }, r, nrows, nvalid);
#pragma unroll
      for (int j = 0; j < 32; ++j) v[j] = fmaf(res_scale, r[j], v[j]);
    }
    if (use_tma) {
      const int seg = (m_base >= split1) + (m_base >= split2);      // a 32-row chunk never straddles a split
      const int mr = m_base - (seg == 0 ? 0 : (seg == 1 ? split1 : split2));
      if ((perm_segs >> seg) & 1u) chunk_store_tma_perm(st, &omap[seg], n, mr, perm_d, v, accumulate != 0);
      else chunk_store_tma<ODT>(st, &omap[seg], n, mr, v, accumulate != 0);
    } else {
      using OT = typename OutElem<ODT>::type;
      auto rowptr = [&](int rr) {
        const int m = m_base + rr;
        const int seg = (m >= split1) + (m >= split2);
        const int mr = m - (seg == 0 ? 0 : (seg == 1 ? split1 : split2));
        return reinterpret_cast<OT*>(out[seg]) + static_cast<long long>(mr) * ld + n;
      };
      if (accumulate) {
        float r[32];
        chunk_load<ODT>(st, rowptr, r, nrows, nvalid);
#pragma unroll
        for (int j = 0; j < 32; ++j) v[j] = r[j] + v[j];
      }
      if (st.lane == 0) tma_store_wait_read<0>();
      chunk_store<ODT>(st, rowptr, v, nrows, nvalid);
    }
  }
};

// Fused QKV projection output [T, Nq+2Nkv] (fp16) with RoPE on the q and k columns (adjacent pairs (2i,2i+1);
// SURVEY 8(c) step 3, ref [36]); v columns (n >= rot_cols) pass through.  Nq, Nkv are multiples of d >= 64 and the
// epilogue works on 32-column chunks, so a chunk never straddles a head or the q|k|v boundaries.
// rope table: float2 (cos, sin) [S, d/2], angles computed in fp64 on the host (reading A-5).
struct EpiQKVRope {
  static constexpr bool kStoreOnly = false;
  __half* out; long long ld;
  const float2* rope; int S, d;
  int rot_cols;              // columns [0, rot_cols) are rotated (Nq + Nkv, or 0 when use_rope = 0)
  CUtensorMap omap;
  const int* doc_start = nullptr;      // packed sequences: the position of token m is m - doc_start[m] instead of m % S
  bool encode(int M, int N) { return make_map_store2d(&omap, out, M, N, ld, DT_F16); }
  __device__ __forceinline__ void prefetch(int, int, int, int, int) const {}      // the rope table stays L2-resident
  __device__ __forceinline__ void operator()(const WarpStage& st, int m_base, int n, float (&v)[32], int nrows, int nvalid) const {
    if (n < rot_cols) {
      // 16 (cos, sin) pairs = 32 words per row, fetched coalesced like any other row chunk
      float cs[32];
      const int half_d = d >> 1, c0 = (n % d) >> 1;
      chunk_load<DT_F32>(st, [&](int rr) {
        const int m = m_base + rr;
        const int pos = doc_start ? m - __ldg(doc_start + m) : m % S;
        return reinterpret_cast<const float*>(rope + static_cast<long long>(pos) * half_d + c0);
      }, cs, nrows, 32);
#pragma unroll
      for (int j = 0; j < 16; ++j) {
        const float z0 = v[2 * j], z1 = v[2 * j + 1];
        v[2 * j] = z0 * cs[2 * j] - z1 * cs[2 * j + 1];
        v[2 * j + 1] = z0 * cs[2 * j + 1] + z1 * cs[2 * j];
      }
    }
    chunk_store_tma<DT_F16>(st, &omap, n, m_base, v);
  }
};

// DUAL epilogue: h = silu(g) * u (ref [35]); saves g,u in fp16 for the backward (DESIGN.md precision plan).
struct EpiSwiGLU {
  static constexpr bool kStoreOnly = true;
  __half* h; __half* g16; __half* u16; long long ld;
  CUtensorMap hmap, gmap, umap;
  int save_gu = 1;           // 0: forward-only call, g and u are not kept for a backward pass
  bool encode(int M, int N) {
    if (!make_map_store2d(&hmap, h, M, N, ld, DT_F16)) return false;
    if (!save_gu) { gmap = hmap; umap = hmap; return true; }
    return make_map_store2d(&gmap, g16, M, N, ld, DT_F16) && make_map_store2d(&umap, u16, M, N, ld, DT_F16);
  }
  __device__ __forceinline__ void prefetch(int, int, int, int, int) const {}
  __device__ __forceinline__ void operator()(const WarpStage& st, int m_base, int n, float (&g)[32], float (&u)[32], int nrows,
                                             int nvalid) const {
    if (save_gu) {
      chunk_store_tma<DT_F16>(st, &gmap, n, m_base, g);
      chunk_store_tma<DT_F16>(st, &umap, n, m_base, u);
    }
#pragma unroll
    for (int j = 0; j < 32; ++j) {
      const float sg = __fdividef(1.0f, 1.0f + __expf(-g[j]));   // MUFU.EX2 + MUFU.RCP: 2 ulp, far below the 16-bit outputs
      g[j] = g[j] * sg * u[j];
    }
    chunk_store_tma<DT_F16>(st, &hmap, n, m_base, g);
  }
};

// Down-projection dgrad with fused SwiGLU backward: acc = dh; writes [dg | du] (fp16) into one [T, 2F] buffer.
struct EpiSwiGLUBwd {
  static constexpr bool kStoreOnly = false;
  const __half* g16; const __half* u16; long long ld;      // saved g,u [T,F]
  __half* dgu; int F;                                      // [T, 2F]
  CUtensorMap dgmap, dumap;                                // the dg and du halves of dgu as two [T, F] views of pitch 2F
  bool encode(int M, int N) {
    return make_map_store2d(&dgmap, dgu, M, N, 2LL * F, DT_F16) && make_map_store2d(&dumap, dgu + F, M, N, 2LL * F, DT_F16);
  }
  __device__ __forceinline__ void prefetch(int lane, int m_base, int n0, int nrows, int ncols) const {
    if (lane < nrows) {
      const long long off = static_cast<long long>(m_base + lane) * ld + n0;
      for (int c = 0; c < ncols; c += 64) { prefetch_l2(g16 + off + c); prefetch_l2(u16 + off + c); }
    }
  }
  __device__ __forceinline__ void operator()(const WarpStage& st, int m_base, int n, float (&dh)[32], int nrows, int nvalid) const {
    float g[32], u[32];
    const long long off = static_cast<long long>(m_base) * ld + n;
    chunk_load<DT_F16>(st, [&](int rr) { return g16 + off + rr * ld; }, g, nrows, nvalid);
    chunk_load<DT_F16>(st, [&](int rr) { return u16 + off + rr * ld; }, u, nrows, nvalid);
#pragma unroll
    for (int j = 0; j < 32; ++j) {
      const float sg = __fdividef(1.0f, 1.0f + __expf(-g[j]));   // MUFU.EX2 + MUFU.RCP: 2 ulp, far below the 16-bit outputs
      const float dgv = dh[j] * u[j] * sg * (1.0f + g[j] * (1.0f - sg));
      u[j] = dh[j] * g[j] * sg;           // du
      g[j] = dgv;                         // dg
    }
    chunk_store_tma<DT_F16>(st, &dgmap, n, m_base, g);
    chunk_store_tma<DT_F16>(st, &dumap, n, m_base, u);
  }
};

// O-projection dgrad with the row sums of the attention backward fused in: acc = dO = da Wo; writes dO
// (fp16, the operand of the attention backward) and, per 32-column chunk, the partial sum over the chunk of dO * O with
// the fp32 copy of O (precision plan P-3) -- D_i = rowsum(dO_i * O_i) = sum_j P_ij dP_ij is the row term of the softmax
// backward.  The products use the fp16-ROUNDED dO, the value the dP MMAs will see, so that sum_j dS_ij = 0 holds to
// rounding.  head_dim 128 = 4 chunks: dvec4 is [B, nq, S, 4] and its readers add the four partials in the fixed order
// (x + y) + (z + w).  Row m is token (b, s) = (m / S, m % S).  Replaces a separate pass over dO and O (0.10 ms at cfg 2).
struct EpiDOutDvec {
  static constexpr bool kStoreOnly = false;
  __half* dO; long long ld;          // [T, Nq] fp16 out
  const float* o32;                  // [T, Nq] fp32 (saved by the forward)
  float* dvec4;                      // [B, nq, S, 4]
  int S, nq;
  CUtensorMap omap;
  bool encode(int M, int N) { return make_map_store2d(&omap, dO, M, N, ld, DT_F16); }
  __device__ __forceinline__ void prefetch(int lane, int m_base, int n0, int nrows, int ncols) const {
    if (lane < nrows) {
      const float* rp = o32 + static_cast<long long>(m_base + lane) * ld + n0;
      for (int c = 0; c < ncols; c += 32) prefetch_l2(rp + c);
    }
  }
  __device__ __forceinline__ void operator()(const WarpStage& st, int m_base, int n, float (&v)[32], int nrows, int nvalid) const {
    float o[32];
    const float* obase = o32 + static_cast<long long>(m_base) * ld + n;
    chunk_load<DT_F32>(st, [&](int rr) { return obase + rr * ld; }, o, nrows, nvalid);
    float acc0 = 0.f, acc1 = 0.f;
#pragma unroll
    for (int j = 0; j < 16; ++j) {
      const __half2 h = __floats2half2_rn(v[2 * j], v[2 * j + 1]);
      const float2 f = __half22float2(h);
      acc0 = fmaf(f.x, o[2 * j], acc0);
      acc1 = fmaf(f.y, o[2 * j + 1], acc1);
    }
    if (st.lane < nrows) {
      const int m = m_base + st.lane;
      const int b = m / S, sq = m - b * S;
      dvec4[((static_cast<long long>(b) * nq + (n >> 7)) * S + sq) * 4 + ((n >> 5) & 3)] = acc0 + acc1;
    }
    chunk_store_tma<DT_F16>(st, &omap, n, m_base, v);
  }
};

#ifdef LSP_GEMM_TRACE
// debug builds only: per CTA pair {cycles in the MMA loop, cycles waiting for operand stages, cycles waiting for a free
// accumulator, k-blocks issued} of the last gemm_pair_tcgen05_kernel launch
__device__ long long g_gemm_trace[128 * 4];
#endif
// ------------------------------------------------------------------------------------------- the kernel
// linear tile id -> (m-block, n-block), banded m-fastest order
__device__ __forceinline__ void gemm_tile_coord(int tile, int mblocks, int nblocks, int band, int& mb, int& nb) {
  const int per_band = band * nblocks;
  const int bid = tile / per_band, r = tile - bid * per_band;
  const int rows = min(band, mblocks - bid * band);
  nb = r / rows;
  mb = bid * band + (r - nb * rows);
}

template <int BN, bool A_MN, bool B_MN, bool DUAL, class Epi>
__global__ void __launch_bounds__(GEMM_THREADS, 1)
gemm_tcgen05_kernel(const __grid_constant__ GemmMaps maps, const GemmShape sh, const __grid_constant__ Epi epi) {
  using Cfg = GemmCfg<BN>;
  constexpr int STAGES = Cfg::STAGES;
  constexpr int NOUT = DUAL ? BN / 2 : BN;       // output columns covered by one tile
  static_assert(!DUAL || (BN == 256 && !A_MN && !B_MN), "DUAL is the forward gate/up GEMM");

  extern __shared__ uint8_t smem_raw[];
  const uint32_t smem_base = (smem_u32(smem_raw) + 1023u) & ~1023u;
  const uint32_t stage_tiles = smem_base + STAGES * Cfg::STAGE_BYTES;     // 8 epilogue warps x 4 KB staging tiles
  const uint32_t bar_base = stage_tiles + GEMM_EPI_WARPS * GEMM_STAGE_TILE_BYTES;
  auto full_bar = [&](int s) { return bar_base + 8u * s; };
  auto empty_bar = [&](int s) { return bar_base + 8u * (STAGES + s); };
  auto tfull_bar = [&](int s) { return bar_base + 8u * (2 * STAGES + s); };
  auto tempty_bar = [&](int s) { return bar_base + 8u * (2 * STAGES + 2 + s); };
  const uint32_t tmem_slot = bar_base + 8u * (2 * STAGES + 4);
  uint32_t* tmem_slot_ptr = reinterpret_cast<uint32_t*>(smem_raw + (tmem_slot - smem_u32(smem_raw)));

  const int warp = threadIdx.x >> 5;
  const int lane = threadIdx.x & 31;

  const int mblocks = (sh.M + GEMM_BM - 1) / GEMM_BM;
  const int nblocks = (sh.N + NOUT - 1) / NOUT;
  const int ntiles = mblocks * nblocks;
  int kb_total = 0;
  const int nseg = DUAL ? 1 : sh.nseg;
  for (int s = 0; s < nseg; ++s) kb_total += sh.kblocks[s];

  if (threadIdx.x == 0) {
    for (int s = 0; s < nseg; ++s) { tma_prefetch_desc(&maps.a[s]); tma_prefetch_desc(&maps.b[s]); }
    if (DUAL) tma_prefetch_desc(&maps.b[1]);
    for (int s = 0; s < STAGES; ++s) { mbar_init(full_bar(s), 1); mbar_init(empty_bar(s), 1); }
    for (int s = 0; s < 2; ++s) { mbar_init(tfull_bar(s), 1); mbar_init(tempty_bar(s), GEMM_EPI_WARPS); }
    fence_barrier_init();
  }
  if (warp == 1) {
    tmem_alloc(tmem_slot, Cfg::TMEM_COLS);
    tmem_relinquish();
  }
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tmem_base = *tmem_slot_ptr;
  pdl_wait();                                    // no global access above (programmatic dependent launch, ptx.cuh)
  pdl_trigger();

  if (warp == 0) {
    // ===================================================================== TMA producer
    if (lane == 0) {
      int stage = 0; uint32_t phase = 0;
      for (int tile = blockIdx.x; tile < ntiles; tile += gridDim.x) {
        int mb, nb;
        gemm_tile_coord(tile, mblocks, nblocks, sh.band, mb, nb);
        const int m0 = mb * GEMM_BM, n0 = nb * NOUT;
        for (int s = 0; s < nseg; ++s) {
          for (int kb = 0; kb < sh.kblocks[s]; ++kb) {
            mbar_wait(empty_bar(stage), phase ^ 1u);
            const uint32_t sa = smem_base + stage * Cfg::STAGE_BYTES;
            const uint32_t sb = sa + Cfg::A_BYTES;
            const uint32_t fb = full_bar(stage);
            mbar_expect_tx(fb, Cfg::STAGE_BYTES);
            const int k0 = kb * GEMM_BK;
            if constexpr (!A_MN) {
              tma_load_2d(sa, &maps.a[s], fb, k0, m0);                       // box {64 k, 128 rows}
            } else {
#pragma unroll
              for (int c = 0; c < GEMM_BM / 64; ++c)                          // box {64 m, 64 k-rows} per chunk
                tma_load_2d(sa + c * (GEMM_BK * 128), &maps.a[s], fb, m0 + 64 * c, k0);
            }
            if constexpr (DUAL) {
              tma_load_2d(sb, &maps.b[0], fb, k0, n0);                       // gate rows [0,128)
              tma_load_2d(sb + 128 * 128, &maps.b[1], fb, k0, n0);           // up   rows [128,256)
            } else if constexpr (!B_MN) {
              tma_load_2d(sb, &maps.b[s], fb, k0, n0);                       // box {64 k, BN rows}
            } else {
#pragma unroll
              for (int c = 0; c < BN / 64; ++c)
                tma_load_2d(sb + c * (GEMM_BK * 128), &maps.b[s], fb, n0 + 64 * c, k0);
            }
            if (++stage == STAGES) { stage = 0; phase ^= 1u; }
          }
        }
      }
    }
  } else if (warp == 1) {
    // ===================================================================== MMA issuer
    if (lane == 0) {
      const uint32_t idesc = umma_idesc(GEMM_BM, BN, sh.a_fmt, sh.b_fmt, A_MN ? 1 : 0, B_MN ? 1 : 0);
      // K-major: atoms of 8 rows x 128 B, SBO = 1024; one UMMA_K (16 elems) = +32 B inside the swizzle row.
      // MN-major: LBO = bytes between 64-wide M/N chunks (BK*128), SBO = 1024 between 8-k-row atoms;
      //           one UMMA_K (16 k-rows) = +2048 B.
      constexpr uint32_t A_LBO = A_MN ? GEMM_BK * 128 : 16, B_LBO = B_MN ? GEMM_BK * 128 : 16;
      constexpr uint32_t A_KSTEP = A_MN ? 2048 : 32, B_KSTEP = B_MN ? 2048 : 32;
      int stage = 0; uint32_t phase = 0;
      int acc = 0; uint32_t acc_phase = 0;
      for (int tile = blockIdx.x; tile < ntiles; tile += gridDim.x) {
        mbar_wait(tempty_bar(acc), acc_phase ^ 1u);
        tc_fence_after();
        const uint32_t d_tmem = tmem_base + static_cast<uint32_t>(acc * BN);
        for (int kb = 0; kb < kb_total; ++kb) {
          mbar_wait(full_bar(stage), phase);
          tc_fence_after();
          const uint32_t sa = smem_base + stage * Cfg::STAGE_BYTES;
          const uint32_t sb = sa + Cfg::A_BYTES;
#pragma unroll
          for (int k = 0; k < GEMM_BK / 16; ++k) {
            const uint64_t ad = umma_smem_desc(sa + k * A_KSTEP, A_LBO, 1024);
            const uint64_t bd = umma_smem_desc(sb + k * B_KSTEP, B_LBO, 1024);
            umma_f16(d_tmem, ad, bd, idesc, (kb | k) != 0 ? 1u : 0u);
          }
          umma_commit(empty_bar(stage));        // smem slot reusable once these MMAs have read it
          if (++stage == STAGES) { stage = 0; phase ^= 1u; }
        }
        umma_commit(tfull_bar(acc));             // accumulator complete -> epilogue
        if (++acc == 2) { acc = 0; acc_phase ^= 1u; }
      }
    }
  } else {
    // ===================================================================== epilogue warps (2..9)
    const int quarter = warp & 3;               // TMEM lanes [32*quarter, 32*quarter+32) are this warp's
    const int half = (warp - 2) >> 2;           // which of the two warps of this quarter: chunks half, half+2, ...
    int acc = 0; uint32_t acc_phase = 0;
    for (int tile = blockIdx.x; tile < ntiles; tile += gridDim.x) {
      int mb, nb;
      gemm_tile_coord(tile, mblocks, nblocks, sh.band, mb, nb);
      const int m0 = mb * GEMM_BM, n0 = nb * NOUT;
      mbar_wait(tfull_bar(acc), acc_phase);
      tc_fence_after();
      const int m_wbase = m0 + quarter * 32;
      const int nrows = min(32, sh.M - m_wbase);
      const WarpStage wst{stage_tiles + static_cast<uint32_t>(warp - 2) * GEMM_STAGE_TILE_BYTES, lane};
      const uint32_t t_row = tmem_base + (static_cast<uint32_t>(quarter * 32) << 16) + static_cast<uint32_t>(acc * BN);
#pragma unroll 1
      for (int c = half; c < NOUT / 32; c += 2) {
        const int n = n0 + c * 32;
        if (n >= sh.N) break;                   // warp-uniform
        const int nvalid = min(32, sh.N - n);
        uint32_t r0[32];
        tmem_ld32(t_row + c * 32, r0);
        if constexpr (DUAL) {
          uint32_t r1[32];
          tmem_ld32(t_row + NOUT + c * 32, r1);
          tmem_ld_wait();
          if (nrows > 0) epi(wst, m_wbase, n, reinterpret_cast<float(&)[32]>(r0), reinterpret_cast<float(&)[32]>(r1), nrows, nvalid);
        } else {
          tmem_ld_wait();
          if (nrows > 0) epi(wst, m_wbase, n, reinterpret_cast<float(&)[32]>(r0), nrows, nvalid);
        }
      }
      tc_fence_before();
      __syncwarp();
      if (lane == 0) mbar_arrive(tempty_bar(acc));
      if (++acc == 2) { acc = 0; acc_phase ^= 1u; }
    }
    if (lane == 0) tma_store_wait_all<0>();        // this warp's bulk stores are complete before the CTA exits
  }

  tc_fence_before();
  __syncthreads();
  if (warp == 1) {
    tc_fence_after();
    tmem_dealloc(tmem_base, Cfg::TMEM_COLS);
  }
}

// ------------------------------------------------------------------------------------------- the CTA-pair kernel
// Same pipeline on a pair of CTAs (cluster of 2 = two SMs of one TPC) working on one 256 x 256 tile with
// tcgen05.mma.cta_group::2: CTA r of the pair stages rows [128 r, +128) of the A tile and rows [128 r, +128) of the
// B tile (32 KB per stage instead of 48 KB, so 6 stages fit), the leader's MMA warp issues one
// 256 x 256 x 16 instruction that reads both CTAs' shared memory, and CTA r's TMEM receives output rows [128 r, +128).
// Halving the B traffic per SM takes the shared-memory port off the critical path (128 x 256 per SM needs
// 96 B/clk of operand reads + 96 B/clk of TMA writes with cta_group::1, 64 + 64 with the pair).
//   full[s]   : leader's barrier, armed by the leader's producer for the bytes of BOTH CTAs; every TMA of the pair
//               (cp.async.bulk.tensor...cta_group::2) reports to it
//   empty[s]  : one per CTA; the leader's tcgen05.commit multicasts the arrival to both
//   tfull[a]  : one per CTA (multicast commit); tempty[a]: leader's, 16 arrivals (8 epilogue warps x 2 CTAs, remote)
// DUAL: CTA 0 stages the gate rows and CTA 1 the up rows of the same 128 output columns, so the pair's N = 256
// accumulator is [gate | up] exactly as in the single-CTA kernel.
//
// Split-K tail (deterministic).  With T tiles on C = 74 persistent pairs the last wave is r = T mod C tiles wide:
// 5-25 % of the machine idles at the layer's shapes (768 tiles = 10.4 waves, 240 = 3.2).  The full waves are walked
// whole (tile = pair + i C: the tiles in flight form a compact band and advance through K in lockstep, so every
// operand k-slice is fetched from DRAM once and shared through L2).  Each of the r leftover tiles is cut into
// s = min(4, floor(C / r)) K-slices, slice j of tile t going to pair j r + t: one round, s r <= C pairs busy for 1/s
// of a tile time instead of r pairs for a whole one.  Pairs with the same j sweep the same k range at the same time,
// which keeps the L2 sharing (contiguous per-pair k ranges that wrap across tiles -- classic stream-K -- do not: they
// ran DRAM-bound, 10 % slower at K = 16384).  Slices j < s - 1 store their raw fp32 accumulator to sk_partial[pair]
// and publish sk_flags[pair] = epoch; slice s - 1 waits for those flags, adds the partials in the fixed order
// j = 0 .. s - 2 to its own accumulator and runs the fused epilogue.  Results are bit-reproducible; no atomics on data.
template <int MT> struct Gemm2Cfg {
  static constexpr int STAGES = MT == 1 ? 6 : 4;
  static constexpr int STAGE_BYTES = (MT + 1) * GEMM_BM * GEMM_BK * 2;     // A (MT x 128) x 64 + B 128 x 64 (16-bit) per CTA
  static constexpr int SMEM_BYTES = STAGES * STAGE_BYTES + GEMM_EPI_WARPS * GEMM_STAGE_TILE_BYTES + 1024 + 256;
};
constexpr int GEMM2_PARTIAL_FLOATS = 2 * 2 * GEMM_BM * 256;           // per pair: up to 512 rows x 256 accumulator columns
constexpr int GEMM2_MAX_SPLIT = 4;

struct GemmItem { int tile, kb0, kb1, mode; };   // mode 0: whole tile; 1: K-slice that publishes a partial; 2: last K-slice

// Work list of pair `cid` (identical in every role of both CTAs): its data-parallel tiles, then at most one K-slice.
struct GemmWork {
  int cid, nclusters, n_dp, has_piece, rem, split;
  GemmItem piece;
  __device__ __forceinline__ void init(int cid_, int nclusters_, int ntiles, int split_, int kbt) {
    cid = cid_; nclusters = nclusters_; split = split_; has_piece = 0;
    rem = ntiles % nclusters;
    if (split >= 2 && rem > 0) {
      const int dp_tiles = ntiles - rem;
      n_dp = dp_tiles / nclusters;
      if (cid < split * rem) {
        const int j = cid / rem, t = cid - j * rem;
        piece = GemmItem{dp_tiles + t, j * kbt / split, (j + 1) * kbt / split, j == split - 1 ? 2 : 1};
        has_piece = 1;
      }
    } else {
      n_dp = ntiles > cid ? (ntiles - cid + nclusters - 1) / nclusters : 0;
    }
  }
  __device__ __forceinline__ int count() const { return n_dp + has_piece; }
  __device__ __forceinline__ GemmItem get(int j) const {
    if (j < n_dp) return GemmItem{cid + j * nclusters, 0, 0x7fffffff, 0};
    return piece;
  }
};

__device__ __forceinline__ unsigned int ld_acquire_gpu(const unsigned int* p) {
  unsigned int v;
  asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
  return v;
}
__device__ __forceinline__ void st_release_gpu(unsigned int* p, unsigned int v) {
  asm volatile("st.release.gpu.global.u32 [%0], %1;" ::"l"(p), "r"(v) : "memory");
}

template <bool A_MN, bool B_MN, bool DUAL, int MT, class Epi>
__global__ void __cluster_dims__(2, 1, 1) __launch_bounds__(GEMM_THREADS, 1)
gemm_pair_tcgen05_kernel(const __grid_constant__ GemmMaps maps, const GemmShape sh, const __grid_constant__ Epi epi) {
  // MT = 1: 256 x 256 pair tile, two accumulator stages (epilogue of tile i overlaps the MMAs of tile i + 1).
  // MT = 2: 512 x 256 pair tile (each CTA 256 rows = two 128-row MMAs per k-step sharing the B slice): A 32 KB +
  //         B 16 KB per CTA and k-block for twice the MACs, i.e. 25 % less shared-memory fill per flop (the quantity
  //         that limits clock and tensor duty under the power cap); the accumulators take all 512 TMEM columns, so
  //         the epilogue is not overlapped -- used where K is large enough to make that negligible.
  using G = Gemm2Cfg<MT>;
  constexpr int STAGES = G::STAGES;
  constexpr int STAGE_BYTES = G::STAGE_BYTES;
  constexpr int BN = 256;                        // MMA N (both CTAs' B halves)
  constexpr int NOUT = DUAL ? 128 : 256;         // output columns covered by one tile
  constexpr int A_BYTES = MT * GEMM_BM * GEMM_BK * 2;
  constexpr int NACC = 2 / MT;                   // accumulator stages
  constexpr int ACC_COLS = BN * MT;
  constexpr int CTA_ROWS = GEMM_BM * MT;
  static_assert(!DUAL || (!A_MN && !B_MN && MT == 1), "DUAL is the forward gate/up GEMM");

  extern __shared__ uint8_t smem_raw[];
  const uint32_t smem_base = (smem_u32(smem_raw) + 1023u) & ~1023u;
  const uint32_t stage_tiles = smem_base + STAGES * STAGE_BYTES;          // 8 epilogue warps x 4 KB staging tiles
  const uint32_t bar_base = stage_tiles + GEMM_EPI_WARPS * GEMM_STAGE_TILE_BYTES;
  auto full_bar = [&](int s) { return bar_base + 8u * s; };
  auto empty_bar = [&](int s) { return bar_base + 8u * (STAGES + s); };
  auto tfull_bar = [&](int s) { return bar_base + 8u * (2 * STAGES + s); };
  auto tempty_bar = [&](int s) { return bar_base + 8u * (2 * STAGES + 2 + s); };
  const uint32_t tmem_slot = bar_base + 8u * (2 * STAGES + 4);
  uint32_t* tmem_slot_ptr = reinterpret_cast<uint32_t*>(smem_raw + (tmem_slot - smem_u32(smem_raw)));

  const int warp = warp_idx_uniform();
  const int lane = threadIdx.x & 31;
  const uint32_t rank = cluster_ctarank();
  const int cid = blockIdx.x >> 1, nclusters = gridDim.x >> 1;

  const int mblocks = (sh.M + 2 * CTA_ROWS - 1) / (2 * CTA_ROWS);      // 256- or 512-row blocks
  const int nblocks = (sh.N + NOUT - 1) / NOUT;
  const int ntiles = mblocks * nblocks;
  const int kb_total = sh.kblocks[0];
  GemmWork work;
  work.init(cid, nclusters, ntiles, sh.sk_partial ? sh.sk_split : 0, kb_total);
  const int nitems = work.count();

  if (threadIdx.x == 0) {
    tma_prefetch_desc(&maps.a[0]); tma_prefetch_desc(&maps.b[0]);
    if (DUAL) tma_prefetch_desc(&maps.b[1]);
    for (int s = 0; s < STAGES; ++s) { mbar_init(full_bar(s), 1); mbar_init(empty_bar(s), 1); }
    for (int s = 0; s < NACC; ++s) { mbar_init(tfull_bar(s), 1); mbar_init(tempty_bar(s), 2 * GEMM_EPI_WARPS); }
    fence_barrier_init();
  }
  if (warp == 1) {
    tmem_alloc_pair(tmem_slot, 512);
    tmem_relinquish_pair();
  }
  tc_fence_before();
  cluster_sync_all();                            // barriers of both CTAs initialised before any remote arrival / TMA
  tc_fence_after();
  const uint32_t tmem_base = *tmem_slot_ptr;
  pdl_wait();                                    // everything above ran under the previous kernel's tail; no global access before here
  pdl_trigger();                                 // the next kernel of the stream may be scheduled (it waits for this one to complete)

  if (warp == 0) {
    // ===================================================================== TMA producer (both CTAs)
    if (lane == 0) {
      const CUtensorMap* bmap = DUAL ? &maps.b[rank] : &maps.b[0];
      int stage = 0; uint32_t phase = 0;
      for (int j = 0; j < nitems; ++j) {
        const GemmItem it = work.get(j);
        int mb, nb;
        gemm_tile_coord(it.tile, mblocks, nblocks, sh.band, mb, nb);
        const int m0 = mb * 2 * CTA_ROWS + static_cast<int>(rank) * CTA_ROWS;
        const int n0 = nb * NOUT;
        const int nb0 = DUAL ? n0 : n0 + static_cast<int>(rank) * 128;         // this CTA's B rows
        const int kb1 = min(it.kb1, kb_total);
        for (int kb = it.kb0; kb < kb1; ++kb) {
          mbar_wait(empty_bar(stage), phase ^ 1u);
          const uint32_t sa = smem_base + stage * STAGE_BYTES;
          const uint32_t sb = sa + A_BYTES;
          const uint32_t fb = mapa_shared(full_bar(stage), 0);
          if (rank == 0) mbar_expect_tx(full_bar(stage), 2 * STAGE_BYTES);
          const int k0 = kb * GEMM_BK;
          if constexpr (!A_MN) {
#pragma unroll
            for (int mt = 0; mt < MT; ++mt) tma_load_2d_pair(sa + mt * (GEMM_BM * 128), &maps.a[0], fb, k0, m0 + mt * GEMM_BM);
          } else {
#pragma unroll
            for (int c = 0; c < 2 * MT; ++c) tma_load_2d_pair(sa + c * (GEMM_BK * 128), &maps.a[0], fb, m0 + 64 * c, k0);
          }
          if constexpr (!B_MN) {
            tma_load_2d_pair(sb, bmap, fb, k0, nb0);
          } else {
#pragma unroll
            for (int c = 0; c < 2; ++c) tma_load_2d_pair(sb + c * (GEMM_BK * 128), bmap, fb, nb0 + 64 * c, k0);
          }
          if (++stage == STAGES) { stage = 0; phase ^= 1u; }
        }
      }
    }
  } else if (warp == 1) {
    // ===================================================================== MMA issuer (leader CTA; whole warp, elected lane)
    if (rank == 0) {
      const uint32_t leader = elect_one();
      const uint32_t idesc = umma_idesc(2 * GEMM_BM, BN, sh.a_fmt, sh.b_fmt, A_MN ? 1 : 0, B_MN ? 1 : 0);
      constexpr uint32_t A_LBO = A_MN ? GEMM_BK * 128 : 16, B_LBO = B_MN ? GEMM_BK * 128 : 16;
      constexpr uint32_t A_KSTEP = A_MN ? 2048 : 32, B_KSTEP = B_MN ? 2048 : 32;
      const uint64_t da0 = umma_smem_desc(smem_base, A_LBO, 1024), db0 = umma_smem_desc(smem_base + A_BYTES, B_LBO, 1024);
      int stage = 0; uint32_t phase = 0;
      int acc = 0; uint32_t acc_phase = 0;
#ifdef LSP_GEMM_TRACE
      long long tr_t0 = clock64(), tr_full = 0, tr_tempty = 0, tr_kb = 0;
#endif
      for (int j = 0; j < nitems; ++j) {
        const GemmItem it = work.get(j);
#ifdef LSP_GEMM_TRACE
        long long tr_a = clock64();
#endif
        mbar_wait_cluster(tempty_bar(acc), acc_phase ^ 1u);
#ifdef LSP_GEMM_TRACE
        tr_tempty += clock64() - tr_a;
#endif
        tc_fence_after();
        const uint32_t d_tmem = tmem_base + static_cast<uint32_t>(acc * ACC_COLS);
        const int kb1 = min(it.kb1, kb_total);
        for (int kb = it.kb0; kb < kb1; ++kb) {
#ifdef LSP_GEMM_TRACE
          tr_a = clock64();
#endif
          mbar_wait_cluster(full_bar(stage), phase);
#ifdef LSP_GEMM_TRACE
          tr_full += clock64() - tr_a; ++tr_kb;
#endif
          tc_fence_after();
          if (leader) {
            const uint64_t da = desc_adv(da0, stage * STAGE_BYTES), db = desc_adv(db0, stage * STAGE_BYTES);
#pragma unroll
            for (int k = 0; k < GEMM_BK / 16; ++k)
#pragma unroll
              for (int mt = 0; mt < MT; ++mt)             // the 128-row halves of this CTA's A slice share the B slice
                umma_f16_pair(d_tmem + mt * BN, desc_adv(da, mt * (GEMM_BM * 128) + k * A_KSTEP), desc_adv(db, k * B_KSTEP), idesc,
                              (kb != it.kb0 || k != 0) ? 1u : 0u);
            umma_commit_pair(empty_bar(stage), 3);
          }
          if (++stage == STAGES) { stage = 0; phase ^= 1u; }
        }
        if (leader) umma_commit_pair(tfull_bar(acc), 3);
        if (++acc == NACC) { acc = 0; acc_phase ^= 1u; }
      }
#ifdef LSP_GEMM_TRACE
      if (lane == 0) {                           // debug builds only: where the MMA warp of this pair spent its time
        long long* o = g_gemm_trace + static_cast<long long>(cid) * 4;
        o[0] = clock64() - tr_t0; o[1] = tr_full; o[2] = tr_tempty; o[3] = tr_kb;
      }
#endif
    }
  } else {
    // ===================================================================== epilogue warps (2..9, both CTAs)
    const int quarter = warp & 3;
    const int half = (warp - 2) >> 2;
    const int row = quarter * 32 + lane;                                  // accumulator row of this thread = TMEM lane
    const WarpStage wst{stage_tiles + static_cast<uint32_t>(warp - 2) * GEMM_STAGE_TILE_BYTES, lane};
    const uint32_t tempty_leader0 = mapa_shared(tempty_bar(0), 0), tempty_leader1 = mapa_shared(tempty_bar(1), 0);
    float* const my_partial = sh.sk_partial ? sh.sk_partial + (static_cast<size_t>(cid) * 2 + rank) * (CTA_ROWS * 256) : nullptr;
    // partial of K-slice jj of the tile whose last slice this pair owns: published by pair jj * rem + (cid mod rem)
    const int t_sk = work.rem > 0 ? cid % work.rem : 0;
    auto slice_partial = [&](int jj) -> const float* {
      return sh.sk_partial + (static_cast<size_t>(jj * work.rem + t_sk) * 2 + rank) * (CTA_ROWS * 256);
    };
    int acc = 0; uint32_t acc_phase = 0;
    for (int j = 0; j < nitems; ++j) {
      const GemmItem it = work.get(j);
      int mb, nb;
      gemm_tile_coord(it.tile, mblocks, nblocks, sh.band, mb, nb);
      const int m0 = mb * 2 * CTA_ROWS + static_cast<int>(rank) * CTA_ROWS;
      const int n0 = nb * NOUT;
      if (it.mode == 2) {                       // the other slices of this tile run at the same time: wait for their partials
        for (int jj = 0; jj < work.split - 1; ++jj) {
          const unsigned int* f = sh.sk_flags + (jj * work.rem + t_sk) * 2 + rank;
          long long t0 = 0; uint32_t polls = 0;
          while (ld_acquire_gpu(f) != sh.sk_epoch) {
            if ((++polls & 0xFFFu) == 0) {
              const long long t = clock64();
              if (t0 == 0) t0 = t; else if (t - t0 > LSP_WAIT_LIMIT_CYCLES) __trap();
            }
          }
        }
      }
#ifndef LSP_NO_EPI_PREFETCH
      if (it.mode != 1) {
#pragma unroll 1
        for (int mt = 0; mt < MT; ++mt) {
          const int mw = m0 + mt * GEMM_BM + quarter * 32;
          epi.prefetch(lane, mw, n0 + half * (NOUT / 2), min(32, sh.M - mw), min(NOUT / 2, sh.N - n0 - half * (NOUT / 2)));
        }
      }
#endif
      mbar_wait_cluster(tfull_bar(acc), acc_phase);
      tc_fence_after();
#pragma unroll 1
      for (int mt = 0; mt < MT; ++mt) {
      const int m_wbase = m0 + mt * GEMM_BM + quarter * 32;                // first row of this warp's 32 accumulator rows
      const int nrows = min(32, sh.M - m_wbase);
      const uint32_t t_row = tmem_base + (static_cast<uint32_t>(quarter * 32) << 16) + static_cast<uint32_t>(acc * ACC_COLS + mt * BN);
#pragma unroll 1
      for (int c = half; c < NOUT / 32; c += 2) {
        const int n = n0 + c * 32;
        if (n >= sh.N) break;                   // warp-uniform
        const int nvalid = min(32, sh.N - n);
        uint32_t r0[32];
        tmem_ld32(t_row + c * 32, r0);
        if constexpr (DUAL) {
          uint32_t r1[32];
          tmem_ld32(t_row + NOUT + c * 32, r1);
          tmem_ld_wait();
          float (&v0)[32] = reinterpret_cast<float(&)[32]>(r0);
          float (&v1)[32] = reinterpret_cast<float(&)[32]>(r1);
          if (it.mode == 1) {
            partial_store(my_partial + static_cast<size_t>(mt * 8 + c) * (GEMM_BM * 32), row, v0);
            partial_store(my_partial + static_cast<size_t>(mt * 8 + NOUT / 32 + c) * (GEMM_BM * 32), row, v1);
          } else {
            if (it.mode == 2) {
              float s0[32], s1[32];
#pragma unroll
              for (int q = 0; q < 32; ++q) { s0[q] = 0.f; s1[q] = 0.f; }
              for (int jj = 0; jj < work.split - 1; ++jj) {                    // fixed order: slice 0, 1, ..., then ours
                float p0[32], p1[32];
                const float* pp = slice_partial(jj);
                partial_load(pp + static_cast<size_t>(mt * 8 + c) * (GEMM_BM * 32), row, p0);
                partial_load(pp + static_cast<size_t>(mt * 8 + NOUT / 32 + c) * (GEMM_BM * 32), row, p1);
#pragma unroll
                for (int q = 0; q < 32; ++q) { s0[q] += p0[q]; s1[q] += p1[q]; }
              }
#pragma unroll
              for (int q = 0; q < 32; ++q) { v0[q] += s0[q]; v1[q] += s1[q]; }
            }
            if (nrows > 0) epi(wst, m_wbase, n, v0, v1, nrows, nvalid);
          }
        } else {
          tmem_ld_wait();
          float (&v0)[32] = reinterpret_cast<float(&)[32]>(r0);
          if (it.mode == 1) {
            partial_store(my_partial + static_cast<size_t>(mt * 8 + c) * (GEMM_BM * 32), row, v0);
          } else {
            if (it.mode == 2) {
              float s0[32];
#pragma unroll
              for (int q = 0; q < 32; ++q) s0[q] = 0.f;
              for (int jj = 0; jj < work.split - 1; ++jj) {                    // fixed order: slice 0, 1, ..., then ours
                float p0[32];
                partial_load(slice_partial(jj) + static_cast<size_t>(mt * 8 + c) * (GEMM_BM * 32), row, p0);
#pragma unroll
                for (int q = 0; q < 32; ++q) s0[q] += p0[q];
              }
#pragma unroll
              for (int q = 0; q < 32; ++q) v0[q] += s0[q];
            }
            if (nrows > 0) epi(wst, m_wbase, n, v0, nrows, nvalid);
          }
        }
      }
      }
      tc_fence_before();
      __syncwarp();
      if (lane == 0) mbar_arrive_cluster(acc == 0 ? tempty_leader0 : tempty_leader1);
      if (it.mode == 2) {                       // every epilogue thread has read the partials: re-arm their flags, so that a
        named_bar_sync_gemm(1, GEMM_EPI_WARPS * 32);          // replay of this launch with the same epoch (CUDA graph) waits again
        if (warp == 2 && lane == 0)
          for (int jj = 0; jj < work.split - 1; ++jj) sh.sk_flags[(jj * work.rem + t_sk) * 2 + rank] = 0u;
      }
      if (it.mode == 1) {                       // all 8 epilogue warps of this CTA have stored: publish
        named_bar_sync_gemm(1, GEMM_EPI_WARPS * 32);
        if (warp == 2 && lane == 0) {
          __threadfence();
          st_release_gpu(sh.sk_flags + cid * 2 + rank, sh.sk_epoch);
        }
      }
      if (++acc == NACC) { acc = 0; acc_phase ^= 1u; }
    }
    if (lane == 0) tma_store_wait_all<0>();        // this warp's bulk stores are complete before the CTA exits
  }

  tc_fence_before();
  cluster_sync_all();                            // nobody leaves while the peer may still signal its barriers / read its smem
  if (warp == 1) {
    tc_fence_after();
    tmem_dealloc_pair(tmem_base, 512);
  }
}


// ------------------------------------------------------------------------------------------- host side
// 2-D tensor map over a row-major 16-bit matrix [rows, cols] with pitch ld (elements):
// box = {64 contiguous elements, box_rows}, 128-byte swizzle, out-of-bounds reads return zero.
inline bool make_map_2d(CUtensorMap* m, const void* base, long long rows, long long cols, long long ld, int box_rows,
                        bool f16 = false) {
  PFN_encodeTiled fn = get_encode_fn();
  if (!fn) return false;
  cuuint64_t dims[2] = {static_cast<cuuint64_t>(cols), static_cast<cuuint64_t>(rows)};
  cuuint64_t strides[1] = {static_cast<cuuint64_t>(ld) * 2};
  cuuint32_t box[2] = {64u, static_cast<cuuint32_t>(box_rows)};
  cuuint32_t estr[2] = {1u, 1u};
  CUresult r = fn(m, f16 ? CU_TENSOR_MAP_DATA_TYPE_FLOAT16 : CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 2,
                  const_cast<void*>(base), dims, strides, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE,
                  CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
  return r == CUDA_SUCCESS;
}

// One operand of one K-segment as it lies in memory.
struct Operand {
  const void* ptr;
  long long ld;       // pitch in elements
  bool mn_major;      // false: [MN, K] row-major (K contiguous); true: [K, MN] row-major (MN contiguous)
  int dt = DT_F16;    // DT_F16 (every operand the layer path produces) or DT_BF16; A and B must match
};
inline int umma_fmt(int dt) { return dt == DT_F16 ? 0 : 1; }

// Encode the map of an operand with logical extents (mn, k); rows_box = tile rows for K-major.
inline bool encode_operand(CUtensorMap* m, const Operand& o, long long mn, long long k, int tile_mn) {
  if (!o.mn_major) return make_map_2d(m, o.ptr, mn, k, o.ld, tile_mn, o.dt == DT_F16);
  return make_map_2d(m, o.ptr, k, mn, o.ld, GEMM_BK, o.dt == DT_F16);
}

// m-blocks per rasterisation band (see the header comment).  LSP_GEMM_BAND overrides (tuning aid).
inline int gemm_band(int mblocks) {
  static int forced = -1;
  if (forced < 0) {
    const char* e = getenv("LSP_GEMM_BAND");
    forced = e ? atoi(e) : 0;
  }
  int b = forced > 0 ? forced : 16;
  if (b > mblocks) b = mblocks;
  return b < 1 ? 1 : b;
}

// CTA-pair kernel for every GEMM with more than one 128-row block; LSP_GEMM_PAIR=0 forces the single-CTA kernel.
inline bool gemm_use_pair(int M) {
  static int mode = -1;
  if (mode < 0) {
    const char* e = getenv("LSP_GEMM_PAIR");
    mode = e ? atoi(e) : 1;
  }
  return mode != 0 && M > GEMM_BM;
}

// Context-owned resources of the stream-K tail (lsp_create allocates them; null -> data-parallel tiles only).
struct GemmSKRes {
  float* partial;            // [num_sms / 2][GEMM2_PARTIAL_FLOATS]
  unsigned int* flags;       // [num_sms / 2][2], zero-initialised once
  unsigned int epoch;        // unique (> 0) per launch
};
inline bool gemm_use_streamk() {
  static int mode = -1;
  if (mode < 0) {
    const char* e = getenv("LSP_GEMM_STREAMK");
    mode = e ? atoi(e) : 1;
  }
  return mode != 0;
}

// Leftover-tile split factor of the pair kernel for `ntiles` tiles on `clusters` pairs (0: none).
inline int gemm_tail_split(int ntiles, int clusters, int kblocks) {
  const int rem = ntiles % clusters;
  if (ntiles <= clusters || rem == 0) return 0;
  int s = clusters / rem;
  if (s > GEMM2_MAX_SPLIT) s = GEMM2_MAX_SPLIT;
  while (s >= 2 && kblocks / s < 4) --s;                  // at least 4 k-blocks per slice
  return s >= 2 ? s : 0;
}

// Pair tile height (MT x 256 rows).  The 512-row tile (MT = 2) needs 25 % less shared-memory fill per flop and runs
// its main loop 3-4 % faster, but its accumulators fill the TMEM, so the epilogue is not overlapped: it pays off only
// for store-only epilogues (bulk stores are asynchronous; epilogues that READ a residual or g, u stall on memory
// latency per chunk: down 0.74 vs 0.60 ms) at large K, and only when the tile count does not quantise worse.  The
// candidates at the 3B shape were wgrad gate/up, dgrad gate/up and wgrad O; inside the layer step the gain did not
// survive (7.39-7.42 vs 7.33-7.39 ms of GEMM time: every kernel's clock depends on the power state its predecessors
// left), so the default stays MT = 1.  LSP_GEMM_MT=2 selects the tall tile (covered by the GPU tests).
inline int gemm_pick_mt(int M, int N, int K, int pairs, bool use_sk, bool store_only) {
  static int forced = -1;
  if (forced < 0) {
    const char* e = getenv("LSP_GEMM_MT");
    forced = e ? atoi(e) : 0;
  }
  if (forced == 1 || forced == 2) return forced;
  (void)M; (void)N; (void)K; (void)pairs; (void)use_sk; (void)store_only;
  return 1;
}

template <bool A_MN, bool B_MN, bool DUAL, int MT, class Epi>
cudaError_t launch_gemm_pair(const GemmMaps& maps, GemmShape sh, const Epi& epi, int num_sms, cudaStream_t st,
                             const GemmSKRes* sk) {
  using G = Gemm2Cfg<MT>;
  auto kern = gemm_pair_tcgen05_kernel<A_MN, B_MN, DUAL, MT, Epi>;
  static DeviceOnce once;
  if (once.need()) {
    cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, G::SMEM_BYTES);
    if (e != cudaSuccess) return e;
    once.done();
  }
  constexpr int NOUT = DUAL ? 128 : 256;
  const int mblocks = (sh.M + 2 * MT * GEMM_BM - 1) / (2 * MT * GEMM_BM), nblocks = (sh.N + NOUT - 1) / NOUT;
  const int ntiles = mblocks * nblocks;
  if (ntiles == 0) return cudaSuccess;
  // ~2048-row bands.  A band height chosen per shape so that a band is a whole number of 74-tile waves (6 or 12 pair tiles
  // for 12 n-blocks instead of 8) was measured in round 2 (profiles/r2_notes.md): GEMM time of the step 8.04-8.09 ms
  // against 7.94-8.02 ms with this fixed height on the same machine -- no gain, not kept.
  sh.band = gemm_band(2 * MT * mblocks) / (2 * MT);
  if (sh.band < 1) sh.band = 1;
  const int pairs = num_sms / 2;
  const int clusters = ntiles < pairs ? ntiles : pairs;
  // split-K tail: the r = ntiles mod clusters leftover tiles are cut into s K-slices when s r <= clusters, s >= 2
  sh.sk_split = 0; sh.sk_partial = nullptr; sh.sk_flags = nullptr; sh.sk_epoch = 0;
  if (sk && sk->partial && gemm_use_streamk()) {
    const int s = gemm_tail_split(ntiles, clusters, sh.kblocks[0]);
    if (s >= 2) { sh.sk_split = s; sh.sk_partial = sk->partial; sh.sk_flags = sk->flags; sh.sk_epoch = sk->epoch; }
  }
  return launch_kernel(kern, dim3(2 * clusters), dim3(GEMM_THREADS), G::SMEM_BYTES, st, maps, sh, epi);
}

template <int BN, bool A_MN, bool B_MN, bool DUAL, class Epi>
cudaError_t launch_gemm(const GemmMaps& maps, GemmShape sh, const Epi& epi, int num_sms, cudaStream_t st) {
  using Cfg = GemmCfg<BN>;
  auto kern = gemm_tcgen05_kernel<BN, A_MN, B_MN, DUAL, Epi>;
  static DeviceOnce once;
  if (once.need()) {
    cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, Cfg::SMEM_BYTES);
    if (e != cudaSuccess) return e;
    once.done();
  }
  constexpr int NOUT = DUAL ? BN / 2 : BN;
  const int mblocks = (sh.M + GEMM_BM - 1) / GEMM_BM, nblocks = (sh.N + NOUT - 1) / NOUT;
  const int ntiles = mblocks * nblocks;
  if (ntiles == 0) return cudaSuccess;
  sh.band = gemm_band(mblocks);
  sh.sk_split = 0; sh.sk_partial = nullptr; sh.sk_flags = nullptr; sh.sk_epoch = 0;
  const int grid = ntiles < num_sms ? ntiles : num_sms;
  return launch_kernel(kern, dim3(grid), dim3(GEMM_THREADS), Cfg::SMEM_BYTES, st, maps, sh, epi);
}

// Generic entry: up to three K-segments (A_s, B_s, K_s); all segments share the operand majors.
template <int BN, bool A_MN, bool B_MN, class Epi>
cudaError_t gemm_run(int M, int N, int nseg, const Operand* a, const Operand* b, const int* ks, const Epi& epi,
                     int num_sms, cudaStream_t st, const GemmSKRes* sk = nullptr) {
  GemmMaps maps;
  GemmShape sh;
  sh.M = M; sh.N = N; sh.nseg = nseg;
  sh.a_fmt = umma_fmt(a[0].dt); sh.b_fmt = umma_fmt(b[0].dt);      // all segments share the operand formats
  for (int s = 0; s < GEMM_MAX_SEG; ++s) sh.kblocks[s] = 0;
  Epi e = epi;
  if (!e.encode(M, N)) return cudaErrorInvalidValue;
  const bool pair = BN == 256 && nseg == 1 && gemm_use_pair(M);
  for (int s = 0; s < nseg; ++s) {
    sh.kblocks[s] = (ks[s] + GEMM_BK - 1) / GEMM_BK;
    if (!encode_operand(&maps.a[s], a[s], M, ks[s], GEMM_BM)) return cudaErrorInvalidValue;
    if (!encode_operand(&maps.b[s], b[s], N, ks[s], pair ? 128 : BN)) return cudaErrorInvalidValue;
  }
  if (pair) {
    const bool use_sk = nseg == 1 && sk && sk->partial && gemm_use_streamk();
    if (nseg == 1 && gemm_pick_mt(M, N, ks[0], num_sms / 2, use_sk, Epi::kStoreOnly) == 2)
      return launch_gemm_pair<A_MN, B_MN, false, 2, Epi>(maps, sh, e, num_sms, st, sk);
    return launch_gemm_pair<A_MN, B_MN, false, 1, Epi>(maps, sh, e, num_sms, st, nseg == 1 ? sk : nullptr);
  }
  return launch_gemm<BN, A_MN, B_MN, false, Epi>(maps, sh, e, num_sms, st);
}

// Forward gate/up GEMM (DUAL): A [M,K], Wg/Wu [N,K] all K-major.
template <class Epi>
cudaError_t gemm_run_dual(int M, int N, int K, const Operand& a, const Operand& bg, const Operand& bu, const Epi& epi,
                          int num_sms, cudaStream_t st, const GemmSKRes* sk = nullptr) {
  Epi e = epi;
  if (!e.encode(M, N)) return cudaErrorInvalidValue;
  GemmMaps maps;
  GemmShape sh;
  sh.M = M; sh.N = N; sh.nseg = 1;
  sh.a_fmt = umma_fmt(a.dt); sh.b_fmt = umma_fmt(bg.dt);
  sh.kblocks[0] = (K + GEMM_BK - 1) / GEMM_BK; sh.kblocks[1] = sh.kblocks[2] = 0;
  if (!encode_operand(&maps.a[0], a, M, K, GEMM_BM)) return cudaErrorInvalidValue;
  if (!encode_operand(&maps.b[0], bg, N, K, 128)) return cudaErrorInvalidValue;
  if (!encode_operand(&maps.b[1], bu, N, K, 128)) return cudaErrorInvalidValue;
  if (gemm_use_pair(M)) return launch_gemm_pair<false, false, true, 1, Epi>(maps, sh, e, num_sms, st, sk);
  return launch_gemm<256, false, false, true, Epi>(maps, sh, e, num_sms, st);
}

}  // namespace lsp
