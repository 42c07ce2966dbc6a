// Causal grouped-query flash attention on the 5th-generation tensor cores (sm_100a), head_dim 128, fp16 operands,
// fp32 accumulation in TMEM.  SURVEY 8(a) F3 (forward, saves the log-sum-exp) -- refs [23],[24],[26],[27],[37].
//
// Forward.  A work item is 256 consecutive queries of one (batch, head) as two 128-row tiles t = 0,1 that ping-pong:
// while the 128 softmax threads of tile t turn S_t = Q_t K_j^T into P_t, the tensor core works on the other tile.
//   warp 0       TMA producer: Q_0, Q_1 once, then K_j / V_j (128 keys x 128) through two-stage mbarrier rings
//   warp 1       tcgen05.mma issuer (one thread) and TMEM owner
//   warps 2-9    softmax of tile 0: lane quarter x column half (thread = one query row = one TMEM lane x 64 keys)
//   warps 10-17  softmax of tile 1
// TMEM (512 columns): S_0 [0,128) S_1 [128,256) O_0 [256,384) O_1 [384,512).  P_t (fp16, two keys per 32-bit column)
// overwrites columns [0,32) and [64,96) of S_t (each column half inside the columns its own warp read) once the threads
// hold their S values in registers, and is the A operand (from TMEM) of O_t += P_t V_j, whose B operand V_j is read
// MN-major from shared memory exactly as TMA wrote it (no transpose).
// Online softmax with lazy rescaling: the running maximum is only raised (and O_t rescaled in TMEM) when it grew by
// more than 2^8 for some row of the warp, so the TMEM round trip of O is rare after the first blocks; P <= 2^8 fits
// fp16 with the same relative precision.  Key blocks above the diagonal are never visited; only the diagonal block
// is masked.  Rows past the end of a sequence are zero-filled by TMA (3-D maps: column, position, batch).
// O leaves through per-warp swizzled staging tiles and 32 x 32 TMA stores: per-thread st.global of a row-per-thread
// fp32 tile stalled the softmax warps ~12 k cycles per item (measured with a clock64 trace), the bulk stores ~1 k.
#pragma once
#include "gemm.cuh"

namespace lsp {

struct AttnTcMaps {
  CUtensorMap q, k, v, dO;
  CUtensorMap o32, o16;          // forward outputs (TMA stores of 32 x 32 chunks out of the swizzled staging tiles)
  CUtensorMap g32[2], g16[2];    // backward outputs: dK/dV kernel [0] = dv, [1] = dk; dQ kernel [0] = dq
};

struct AttnTcParams {
  int B, S, nq, nkv;
  float scale_log2;            // (1/sqrt(d)) * log2(e)
  float scale;
  float* o32; __half* o16; long long ldo;        // [T, ldo] outputs (either may be null)
  float* lse;                                    // [B, nq, S]
  unsigned int* sched;                           // [2] work-item counter and finished-CTA counter (zero between launches)
  // packed variable-length sequences (B = 1): token t attends keys [doc_start[t], t]; doc_end[t] = end (exclusive) of
  // t's sequence; both non-decreasing in t.  Null: every sequence starts at position 0 of its batch row.
  const int* doc_start; const int* doc_end;
};

constexpr int ATC_D = 128;
constexpr int ATC_TILE_BYTES = 128 * ATC_D * 2;          // one 128 x 128 fp16 tile = 32 KB (two 64-wide swizzled chunks)
constexpr int ATC_CHUNK_BYTES = 128 * 128;               // one 64-column chunk of 128 rows
constexpr int ATC_FWD_SOFTMAX_WARPS = 16;                // 2 tiles x 2 column halves x 4 TMEM lane quarters
constexpr int ATC_FWD_THREADS = 64 + 32 * ATC_FWD_SOFTMAX_WARPS;
constexpr int ATC_FWD_STAGE_BYTES = 2048;                // per softmax warp: 32 rows x 64 B (16 fp32 or 32 fp16 columns)
constexpr int ATC_FWD_XCH_BYTES = 2 * 2 * 128 * 4;       // [tile][half][row] fp32: row maxima / row sums between the halves
// Q0 Q1 | K x2 | V x2 | 16 staging tiles | exchange | barriers.  The dynamic shared memory is declared 1024-byte aligned
// (128B-swizzled TMA tiles need it) and the kernel traps if the base is not: there is no room for alignment slack.
constexpr int ATC_FWD_SMEM = 6 * ATC_TILE_BYTES + ATC_FWD_SOFTMAX_WARPS * ATC_FWD_STAGE_BYTES + ATC_FWD_XCH_BYTES + 256;
constexpr float ATC_RESCALE_LOG2 = 8.0f;

// Share of the forward's exponentials computed on the FMA pipe instead of the SFU, in quarters (0 = none ... 4 = all).
// The 128 x 128 exponentials of a block occupy the SFU (16 results / clk / SM) for 1024 cycles -- exactly the tensor time
// of the block's two MMAs.  Measured on B200 (profiles/r2_attn_traces.txt, profiles/r2_notes.md): the polynomial costs 8 FP32-pipe pair
// instructions + 2 IMAD per key pair and FFMA2 / FADD2 issue at 4 cycles per warp instruction, so per block and SM
// sub-partition the FMA pipe needs 64 (36 f + 8 (1 - f)) cycles against 1024 (1 - f) on the SFU: 0 -> 512 / 1024,
// 1/4 -> 960 / 768, 1/2 -> 1408 / 512.  One pair in four is the balance point (forward kernel 0.541 / 0.529 / 0.532 /
// 0.572 ms inside the cfg2 step for 0 / 1 / 2 / 3 quarters).
#ifndef LSP_ATTN_POLY_EXP
#define LSP_ATTN_POLY_EXP 1
#endif
// the same for the P^T phase of the dK/dV kernel (0 = all on the SFU, 1 = one key pair in four on the FMA pipe)
#ifndef LSP_ATTN_BWD_POLY_EXP
#define LSP_ATTN_BWD_POLY_EXP 1
#endif

// 2^x for a pair of values <= ~2^8 without the SFU: x clamped at -126 (masked keys are -inf; a clamped value ends as
// 2^-126, zero in fp16), n = round(x) through the 1.5 * 2^23 addition, 2^f on [-0.5, 0.5] by the degree-3 minimax
// polynomial with p(0) = 1 (an integer x, in particular the row maximum x = 0, gives the exact power of two, as the SFU
// does; relative error <= 1.0e-4 = 2^-13.3 elsewhere, a fifth of the fp16 rounding of P), 2^n by an add into the exponent.
__device__ __forceinline__ float2 ex2_poly2(float2 x) {
  x.x = fmaxf(x.x, -126.0f);
  x.y = fmaxf(x.y, -126.0f);
  const float2 t = fadd2(x, make_float2(12582912.0f, 12582912.0f));
  const float2 n = fadd2(t, make_float2(-12582912.0f, -12582912.0f));
  const float2 f = ffma2(n, make_float2(-1.0f, -1.0f), x);
  float2 r = ffma2(f, make_float2(0.05500893f, 0.05500893f), make_float2(0.24221095f, 0.24221095f));
  r = ffma2(r, f, make_float2(0.6932829f, 0.6932829f));
  r = ffma2(r, f, make_float2(1.0f, 1.0f));
  r.x = __uint_as_float(__float_as_uint(r.x) + (__float_as_uint(t.x) << 23));
  r.y = __uint_as_float(__float_as_uint(r.y) + (__float_as_uint(t.y) << 23));
  return r;
}
__device__ __forceinline__ float fmax3(float a, float b, float c) {
  float y;
  asm("max.f32 %0, %1, %2, %3;" : "=f"(y) : "f"(a), "f"(b), "f"(c));     // one FMNMX3
  return y;
}

// 3-D map over a [B*S, ld] fp16 matrix seen as (column, position, batch); box = 64 columns x box_rows positions.
inline bool make_map_attn(CUtensorMap* m, const void* base, int ncols, int S, int B, long long ld, int box_rows = 128) {
  PFN_encodeTiled fn = get_encode_fn();
  if (!fn) return false;
  cuuint64_t dims[3] = {static_cast<cuuint64_t>(ncols), static_cast<cuuint64_t>(S), static_cast<cuuint64_t>(B)};
  cuuint64_t strides[2] = {static_cast<cuuint64_t>(ld) * 2, static_cast<cuuint64_t>(ld) * 2 * static_cast<cuuint64_t>(S)};
  cuuint32_t box[3] = {64u, static_cast<cuuint32_t>(box_rows), 1u};
  cuuint32_t estr[3] = {1u, 1u, 1u};
  return fn(m, CU_TENSOR_MAP_DATA_TYPE_FLOAT16, 3, const_cast<void*>(base), dims, strides, box, estr,
            CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
            CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
}

// 3-D map (column, position, batch) over a [B*S, ld] matrix of 4- or 2-byte elements for 32-column x 32-row chunk
// stores out of a staging tile: 128-byte rows with the 128B swizzle (fp32), 64-byte rows with the 64B swizzle (16-bit)
// -- exactly the XOR patterns of WarpStage::put_row32 / put_row16.  narrow32: fp32 chunks of 16 columns (64-byte rows,
// 64B swizzle: the byte layout of put_row16), for kernels whose staging tiles are 2 KB.
inline bool make_map_store(CUtensorMap* m, const void* base, int ncols, int S, int B, long long ld, bool f32, bool narrow32 = false) {
  PFN_encodeTiled fn = get_encode_fn();
  if (!fn) return false;
  const cuuint64_t es = f32 ? 4 : 2;
  cuuint64_t dims[3] = {static_cast<cuuint64_t>(ncols), static_cast<cuuint64_t>(S), static_cast<cuuint64_t>(B)};
  cuuint64_t strides[2] = {static_cast<cuuint64_t>(ld) * es, static_cast<cuuint64_t>(ld) * es * static_cast<cuuint64_t>(S)};
  cuuint32_t box[3] = {(f32 && narrow32) ? 16u : 32u, 32u, 1u};
  cuuint32_t estr[3] = {1u, 1u, 1u};
  return fn(m, f32 ? CU_TENSOR_MAP_DATA_TYPE_FLOAT32 : CU_TENSOR_MAP_DATA_TYPE_FLOAT16, 3, const_cast<void*>(base), dims, strides,
            box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE, (f32 && !narrow32) ? CU_TENSOR_MAP_SWIZZLE_128B : CU_TENSOR_MAP_SWIZZLE_64B,
            CU_TENSOR_MAP_L2_PROMOTION_NONE, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
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

// Persistent: one CTA per SM walks work items (256-query block, head, batch) handed out heaviest-first by a global
// atomic counter (p.sched).  Items are pipelined inside the CTA: the next item's Q tiles are fetched as soon as the
// last S MMA of the current one has read them (q_empty), its first S = Q K^T is issued right after the current item's
// last P V, and the O epilogue of a tile (TMEM -> registers -> staging tile -> bulk stores) overlaps the
// other tile's and the next item's MMAs (o_free tells the MMA warp when O_t may be overwritten).
struct AttnItem { int q0, h, b, kvh, n0, n1, nmax, j0; };         // j0: first 128-key block (packed sequences), else 0
__device__ __forceinline__ AttnItem attn_fwd_item(uint32_t i, const AttnTcParams& p, int nqb, const int* doc_start) {
  const int per_lvl = p.nq * p.B;
  const int lvl = static_cast<int>(i) / per_lvl, r = static_cast<int>(i) - lvl * per_lvl;
  AttnItem it;
  it.q0 = (nqb - 1 - lvl) * 256;                               // heavy (late) query blocks first
  it.b = r / p.nq; it.h = r - it.b * p.nq;
  it.kvh = it.h / (p.nq / p.nkv);
  // key blocks per tile: tile t covers queries [q0 + 128 t, +128); causal => keys [0, q0 + 128 t + 128)
  // packed sequences: nothing before the start of the sequence of the item's first query is visited (starts are
  // non-decreasing, so that is the smallest start of the item); both tiles share the K/V stream
  it.j0 = doc_start ? doc_start[it.q0] / 128 : 0;
  it.n0 = it.q0 / 128 + 1 - it.j0;
  it.n1 = (it.q0 + 128 < p.S) ? it.n0 + 1 : 0;
  it.nmax = it.n1 > it.n0 ? it.n1 : it.n0;
  return it;
}
constexpr int ATC_ITEM_RING = 4;

// Debug-only clock64 trace of one CTA's pipeline (build with -DLSP_ATTN_TRACE; never in the shipped library):
// g_atc_trace[slot] = SM clock at event `slot` of block `blk` (events: see the ATC_TR uses).
#ifdef LSP_ATTN_TRACE
__device__ unsigned long long g_atc_trace[64 * 32];
#define ATC_TR(blk, ev) do { if (blockIdx.x == 3 && (blk) >= 64 && (blk) < 128) g_atc_trace[((blk) - 64) * 32 + (ev)] = clock64(); } while (0)
#define ATC_TR2(blk, ev) do { if (blockIdx.x == 5 && (blk) >= 16 && (blk) < 80) g_atc_trace[((blk) - 16) * 32 + (ev)] = clock64(); } while (0)
#define ATC_TR3(blk, ev) do { if (blockIdx.x == 7 && (blk) >= 96 && (blk) < 160) g_atc_trace[((blk) - 96) * 32 + (ev)] = clock64(); } while (0)
// dK/dV CTA lifetime: events 0..5 (columns 10..15, iterations in column 22) of the heaviest CTA of group 5 (blockIdx 5) in row 62
// and of a light one (blockIdx 900) in row 63
#define ATC_TRL(ev) do { if (blockIdx.x == 5 || blockIdx.x == 900) g_atc_trace[(blockIdx.x == 5 ? 62 : 63) * 32 + 10 + (ev)] = clock64(); } while (0)
#else
#define ATC_TRL(ev) do { } while (0)
#define ATC_TR(blk, ev) do { } while (0)
#define ATC_TR2(blk, ev) do { } while (0)
#define ATC_TR3(blk, ev) do { } while (0)
#endif

template <bool DOC>
__global__ void __launch_bounds__(ATC_FWD_THREADS, 1)
attn_fwd_tc_kernel(const __grid_constant__ AttnTcMaps maps, const AttnTcParams p) {
  // packed sequences compiled in only for DOC: the plain kernels carry none of the bound / mask code
  const int* const doc_start = DOC ? p.doc_start : nullptr;
  const int* const doc_end = DOC ? p.doc_end : nullptr;
  (void)doc_start; (void)doc_end;
  extern __shared__ __align__(1024) uint8_t smem_raw[];
  const uint32_t smem_base = smem_u32(smem_raw);
  if (smem_base & 1023u) __trap();                            // see ATC_FWD_SMEM: the 128B-swizzled tiles start at the base
  const uint32_t sQ = smem_base;                              // 2 tiles
  const uint32_t sK = sQ + 2 * ATC_TILE_BYTES;                // 2 stages
  const uint32_t sV = sK + 2 * ATC_TILE_BYTES;                // 2 stages
  const uint32_t stage_tiles = sV + 2 * ATC_TILE_BYTES;       // 16 softmax warps x 2 KB staging tiles (epilogue)
  const uint32_t xch = stage_tiles + ATC_FWD_SOFTMAX_WARPS * ATC_FWD_STAGE_BYTES;
  const uint32_t bar_base = xch + ATC_FWD_XCH_BYTES;
  auto q_full = [&](int t) { return bar_base + 8u * t; };
  auto k_full = [&](int s) { return bar_base + 8u * (2 + s); };
  auto k_empty = [&](int s) { return bar_base + 8u * (4 + s); };
  auto v_full = [&](int s) { return bar_base + 8u * (6 + s); };
  auto v_empty = [&](int s) { return bar_base + 8u * (8 + s); };
  auto s_full = [&](int t) { return bar_base + 8u * (10 + t); };
  auto p_full = [&](int t, int part) { return bar_base + 8u * ((part ? 28 : 12) + t); };   // P_t, first / second 32 keys of both halves
  auto o_full = [&](int t) { return bar_base + 8u * (14 + t); };
  auto q_empty = [&](int t) { return bar_base + 8u * (16 + t); };
  auto o_free = [&](int t) { return bar_base + 8u * (18 + t); };
  auto item_bar = [&](int s) { return bar_base + 8u * (20 + s); };
  const uint32_t item_slots = bar_base + 8u * (20 + ATC_ITEM_RING);
  const uint32_t tmem_slot = item_slots + 4u * ATC_ITEM_RING;
  uint32_t* tmem_slot_ptr = reinterpret_cast<uint32_t*>(smem_raw + (tmem_slot - smem_base));
  volatile uint32_t* item_slot_ptr = reinterpret_cast<volatile uint32_t*>(smem_raw + (item_slots - smem_base));
  volatile float* xch_ptr = reinterpret_cast<volatile float*>(smem_raw + (xch - smem_base));

  const int warp = warp_idx_uniform(), lane = threadIdx.x & 31;
  const int nqb = (p.S + 255) / 256;
  const uint32_t nitems = static_cast<uint32_t>(nqb * p.nq * p.B);

  if (threadIdx.x == 0) {
    tma_prefetch_desc(&maps.q); tma_prefetch_desc(&maps.k); tma_prefetch_desc(&maps.v);
    tma_prefetch_desc(&maps.o32); tma_prefetch_desc(&maps.o16);
    for (int i = 0; i < 2; ++i) {
      mbar_init(q_full(i), 1); mbar_init(q_empty(i), 1);
      mbar_init(k_full(i), 1); mbar_init(k_empty(i), 1);
      mbar_init(v_full(i), 1); mbar_init(v_empty(i), 1);
      mbar_init(s_full(i), 1); mbar_init(p_full(i, 0), 8); mbar_init(p_full(i, 1), 8); mbar_init(o_full(i), 1); mbar_init(o_free(i), 8);
    }
    for (int i = 0; i < ATC_ITEM_RING; ++i) mbar_init(item_bar(i), 1);
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
  pdl_wait();                                    // no global access above (programmatic dependent launch, ptx.cuh)
  pdl_trigger();

  // item `it` of this CTA: published by the producer thread in slot it % ATC_ITEM_RING (slot reuse is safe: the
  // producer can be at most two items ahead of the slowest reader, see the q_empty / o_free dependencies)
  auto get_item = [&](uint32_t it) -> uint32_t {
    mbar_wait(item_bar(it % ATC_ITEM_RING), (it / ATC_ITEM_RING) & 1u);
    return item_slot_ptr[it % ATC_ITEM_RING];
  };

  if (warp == 0) {
    // ===================================================================== scheduler + TMA producer
    if (lane == 0) {
      auto publish = [&](uint32_t it, uint32_t item) {
        item_slot_ptr[it % ATC_ITEM_RING] = item;
        mbar_arrive(item_bar(it % ATC_ITEM_RING));             // release: the slot write is visible to the waiters
      };
      uint32_t kvc = 0, qc0 = 0, qc1 = 0;                      // K/V blocks and Q tiles loaded so far
      uint32_t item = atomicAdd(p.sched, 1u);
      publish(0, item);
      for (uint32_t it = 0; item < nitems; ++it) {
        const AttnItem w = attn_fwd_item(item, p, nqb, doc_start);
        mbar_wait(q_empty(0), (qc0 & 1u) ^ 1u);
        atc_load_tile(sQ, &maps.q, q_full(0), w.h * ATC_D, w.q0, w.b);
        ++qc0;
        if (w.n1 > 0) {
          mbar_wait(q_empty(1), (qc1 & 1u) ^ 1u);
          atc_load_tile(sQ + ATC_TILE_BYTES, &maps.q, q_full(1), w.h * ATC_D, w.q0 + 128, w.b);
          ++qc1;
        }
        const uint32_t next = atomicAdd(p.sched, 1u);          // latency hidden behind this item's K/V stream
        for (int j = 0; j < w.nmax; ++j, ++kvc) {
          const int st = kvc & 1;
          const uint32_t ph = ((kvc >> 1) & 1u) ^ 1u;
          mbar_wait(k_empty(st), ph);
          atc_load_tile(sK + st * ATC_TILE_BYTES, &maps.k, k_full(st), w.kvh * ATC_D, (w.j0 + j) * 128, w.b);
          mbar_wait(v_empty(st), ph);
          atc_load_tile(sV + st * ATC_TILE_BYTES, &maps.v, v_full(st), w.kvh * ATC_D, (w.j0 + j) * 128, w.b);
        }
        publish(it + 1, next);
        item = next;
      }
      // the grid's last CTA re-arms the counters for the next launch on this context
      __threadfence();
      if (atomicAdd(p.sched + 1, 1u) == gridDim.x - 1) { p.sched[0] = 0; p.sched[1] = 0; __threadfence(); }
    }
  } else if (warp == 1) {
    // ===================================================================== MMA issuer (whole warp, elected lane issues)
    const uint32_t leader = elect_one();
    const uint32_t idesc_s = umma_idesc(128, 128, 0, 0, 0, 0);     // S = Q K^T : both K-major
    const uint32_t idesc_pv = umma_idesc(128, 128, 0, 0, 0, 1);    // O += P V  : A from TMEM, B (V) MN-major
    const uint64_t dq0 = umma_smem_desc(sQ, 16, 1024), dk0 = umma_smem_desc(sK, 16, 1024);
    const uint64_t dv0 = umma_smem_desc(sV, ATC_CHUNK_BYTES, 1024);
    auto issue_s = [&](int t, int kst) {
      if (leader) {
        const uint64_t qa = desc_adv(dq0, t * ATC_TILE_BYTES), ka = desc_adv(dk0, kst * ATC_TILE_BYTES);
#pragma unroll
        for (int kk = 0; kk < 8; ++kk) {
          const uint32_t off = (kk >> 2) * ATC_CHUNK_BYTES + (kk & 3) * 32;
          umma_f16(tmem_base + t * 128, desc_adv(qa, off), desc_adv(ka, off), idesc_s, kk != 0 ? 1u : 0u);
        }
        umma_commit(s_full(t));
      }
    };
    // P_t: keys [64 h, 64 h + 64) of the block are the 32 columns [64 h, 64 h + 32) of S_t (each column half stays
    // inside the columns its own warp read), so K step kk reads columns 64 (kk / 4) + 8 (kk % 4)
    // P_t is handed over in two parts (the first / second 32 keys of both column halves = K steps {0,1,4,5} / {2,3,6,7}):
    // the first half of P V runs while the second half of P is still being exponentiated
    auto issue_pv = [&](int t, int vst, bool acc, int part) {
      if (leader) {
        const uint64_t va = desc_adv(dv0, vst * ATC_TILE_BYTES);
#pragma unroll
        for (int e = 0; e < 4; ++e) {
          const int kk = (e >> 1) * 4 + part * 2 + (e & 1);
          umma_f16_ts(tmem_base + 256 + t * 128, tmem_base + t * 128 + (kk >> 2) * 64 + (kk & 3) * 8, desc_adv(va, kk * 2048), idesc_pv,
                      (acc || part != 0 || e != 0) ? 1u : 0u);
        }
        if (part == 1) umma_commit(o_full(t));
      }
    };
    uint32_t kvc = 0;                          // K/V blocks consumed so far (ring position of this item's block 0)
    uint32_t qc[2] = {0, 0};                   // items seen per tile (q_full / o_free phases)
    uint32_t pc[2] = {0, 0};                   // P blocks consumed per tile (p_full phase)
    for (uint32_t it = 0;; ++it) {
      const uint32_t item = get_item(it);
      if (item >= nitems) break;
      const AttnItem w = attn_fwd_item(item, p, nqb, doc_start);
      const int nt[2] = {w.n0, w.n1};
      // first S of both tiles (for the second and later items this overlaps the previous item's epilogues)
      {
        const int st0 = kvc & 1;
        mbar_wait(k_full(st0), (kvc >> 1) & 1u);
#pragma unroll
        for (int t = 0; t < 2; ++t) {
          if (nt[t] > 0) {
            mbar_wait(q_full(t), qc[t] & 1u);
            tc_fence_after();
            issue_s(t, st0);
            if (nt[t] == 1 && leader) umma_commit(q_empty(t));       // that was this tile's last S of the item
          }
        }
        if (leader) umma_commit(k_empty(st0));
      }
      for (int j = 0; j < w.nmax; ++j) {
        const uint32_t kc = kvc + j;
        const int st = kc & 1;
        // V_j and K_{j+1} first, polled together: the warp is about to wait for P anyway, and behind P V the S MMA must
        // not wait for a barrier poll
        bool knext_ready = false;
        if (j + 1 < w.nmax) { mbar_wait2(v_full(st), (kc >> 1) & 1u, k_full(st ^ 1), ((kc + 1) >> 1) & 1u); knext_ready = true; }
        else mbar_wait(v_full(st), (kc >> 1) & 1u);
#pragma unroll
        for (int t = 0; t < 2; ++t) {
          if (j < nt[t]) {
            mbar_wait(p_full(t, 0), pc[t] & 1u);
            if (lane == 0) ATC_TR(pc[t], 16 + 4 * t);
            if (j == 0 && qc[t] > 0) mbar_wait(o_free(t), (qc[t] - 1u) & 1u);   // previous item's O_t has been read out
            tc_fence_after();
            issue_pv(t, st, j > 0, 0);
            mbar_wait(p_full(t, 1), pc[t] & 1u);
            ++pc[t];
            tc_fence_after();
            issue_pv(t, st, j > 0, 1);
            if (lane == 0) ATC_TR(pc[t] - 1, 17 + 4 * t);
          }
          if (j + 1 < nt[t]) {
            if (!knext_ready) { mbar_wait(k_full(st ^ 1), ((kc + 1) >> 1) & 1u); tc_fence_after(); knext_ready = true; }
            if (lane == 0) ATC_TR(pc[t] - 1, 18 + 4 * t);
            issue_s(t, st ^ 1);
            if (lane == 0) ATC_TR(pc[t] - 1, 19 + 4 * t);
            if (j + 2 == nt[t] && leader) umma_commit(q_empty(t));   // last S of this tile: Q_t may be refilled
          }
        }
        if (leader) {
          umma_commit(v_empty(st));
          if (j + 1 < w.nmax) umma_commit(k_empty(st ^ 1));
        }
      }
      kvc += w.nmax;
      if (nt[0] > 0) ++qc[0];
      if (nt[1] > 0) ++qc[1];
    }
  } else {
    // ===================================================================== softmax warps: tile t, column half h, lane quarter
    // 16 warps: a tile's 128 x 128 block is worked on by 8 of them -- thread = one query row (TMEM lane) x 64 of the 128
    // keys -- so that TMEM load, row maximum, exponentials and P store of a block take half as long as with one warp per
    // lane quarter: the S -> P latency of a tile is what the tensor core waits for (profiles/r1g_attn_stalls.md).  The two
    // halves of a row share the running maximum (exchanged through shared memory every block, one named barrier per
    // pair of warps) and keep separate partial row sums until the epilogue.
    const int idx = warp - 2;
    const int t = idx >> 3;
    const int h = (idx >> 2) & 1;
    const int quarter = warp & 3;
    const int row = quarter * 32 + lane;                         // query row within the tile = TMEM lane
    const uint32_t lane_off = static_cast<uint32_t>(quarter * 32) << 16;
    const uint32_t tS = tmem_base + lane_off + t * 128 + h * 64; // this warp's 64 columns of S_t; P goes to the first 32
    const uint32_t tO = tmem_base + lane_off + 256 + t * 128 + h * 64;
    const WarpStage wst{stage_tiles + static_cast<uint32_t>(idx) * ATC_FWD_STAGE_BYTES, lane};
    const int pair_bar = 1 + t * 4 + quarter;                    // named barrier of the two warps that share these rows
    volatile float* xmine = xch_ptr + (t * 2 + h) * 128 + row;
    volatile float* xpeer = xch_ptr + (t * 2 + (h ^ 1)) * 128 + row;
    const float c = p.scale_log2;
    uint32_t cnt = 0;                                            // key blocks this tile has processed (all items)

    for (uint32_t it = 0;; ++it) {
      const uint32_t item = get_item(it);
      if (item >= nitems) break;
      const AttnItem w = attn_fwd_item(item, p, nqb, doc_start);
      const int nblk = t == 0 ? w.n0 : w.n1;
      if (nblk == 0) continue;
      const int qi = w.q0 + t * 128 + row;                       // position in the sequence
      float m_run = -INFINITY, l_run = 0.f;                      // l_run: sum over THIS warp's key columns
      const int dstart = doc_start ? doc_start[min(qi, p.S - 1)] : 0;     // first key this query may see

      for (int j = 0; j < nblk; ++j, ++cnt) {
        mbar_wait(s_full(t), cnt & 1u);
        const bool tr = quarter == 0 && h == 0 && lane == 0;
        if (tr) ATC_TR(cnt, 0 + 8 * t);
        tc_fence_after();
        uint32_t sr[2][32];
        tmem_ld32(tS, sr[0]);
        tmem_ld32(tS + 32, sr[1]);
        tmem_ld_wait();
        if (tr) ATC_TR(cnt, 1 + 8 * t);
        float (&s)[2][32] = reinterpret_cast<float(&)[2][32]>(sr);
        if (j == nblk - 1) {                                     // diagonal block: key 128 j + cidx > query <=> cidx > row
#pragma unroll
          for (int q = 0; q < 2; ++q)
#pragma unroll
            for (int i = 0; i < 32; ++i)
              if (h * 64 + q * 32 + i > row) s[q][i] = -INFINITY;
        }
        if (DOC && __any_sync(0xffffffffu, (w.j0 + j) * 128 + h * 64 < dstart)) {   // packed sequences: keys of earlier sequences
          const int kb0 = (w.j0 + j) * 128 + h * 64;
#pragma unroll
          for (int q = 0; q < 2; ++q)
#pragma unroll
            for (int i = 0; i < 32; ++i)
              if (kb0 + q * 32 + i < dstart) s[q][i] = -INFINITY;
        }
        float mx0 = fmax3(s[0][0], s[0][1], s[0][2]), mx1 = fmax3(s[1][0], s[1][1], s[1][2]);
#pragma unroll
        for (int i = 3; i < 31; i += 2) {
          mx0 = fmax3(mx0, s[0][i], s[0][i + 1]);
          mx1 = fmax3(mx1, s[1][i], s[1][i + 1]);
        }
        const float mx_half = fmax3(mx0, mx1, fmaxf(s[0][31], s[1][31]));
        // the other half's maximum of the same rows (safe to overwrite: the peer read last block's value before it arrived at
        // p_full, and this block's S was only issued after all 8 arrivals)
        *xmine = mx_half;
        named_bar_sync_gemm(pair_bar, 64);
        // a row whose keys so far are all masked (packed sequences only) keeps a finite reference maximum: P = 0, no NaN
        const float m_blk = fmax3(m_run, mx_half, *xpeer);
        if (tr) ATC_TR(cnt, 2 + 8 * t);
        const float m_new = DOC ? fmaxf(m_blk, -1.0e30f) : m_blk;
        float m_use = m_run;
        if (j == 0) {
          m_use = m_new;
        } else {
          const bool grow = (m_new - m_run) * c > ATC_RESCALE_LOG2;
          if (__any_sync(0xffffffffu, grow)) {                   // same vote in both halves: same rows, same maxima
            // raise the reference maximum of every row of this warp and rescale its 64 columns of O_t in TMEM
            const float alpha = ex2_approx((m_run - m_new) * c);
            m_use = m_new;
            l_run *= alpha;
            mbar_wait(o_full(t), (cnt - 1u) & 1u);               // P_t V_{j-1} has landed in O_t
            tc_fence_after();
#pragma unroll 1
            for (int q = 0; q < 4; ++q) {                        // 16 columns at a time: S stays in registers
              uint32_t orr[16];
              tmem_ld16(tO + q * 16, orr);
              tmem_ld_wait();
#pragma unroll
              for (int i = 0; i < 16; ++i) orr[i] = __float_as_uint(__uint_as_float(orr[i]) * alpha);
              tmem_st16(tO + q * 16, orr);
            }
          }
        }
        m_run = m_use;
        const float neg = -m_use * c;
        // P = 2^(s c - m c): FFMA2, then per key pair either 2 MUFU.EX2 or the FMA-pipe polynomial, FADD2, F2FP
        const float2 c2 = make_float2(c, c), neg2 = make_float2(neg, neg);
        float2 acc0 = make_float2(0.f, 0.f), acc1 = make_float2(0.f, 0.f);
#pragma unroll
        for (int q = 0; q < 2; ++q) {
          uint32_t pk[16];
#pragma unroll
          for (int i = 0; i < 16; ++i) {
            float2 a = ffma2(make_float2(s[q][2 * i], s[q][2 * i + 1]), c2, neg2);
            if ((i & 3) < LSP_ATTN_POLY_EXP) {
              a = ex2_poly2(a);
            } else {
              a.x = ex2_approx(a.x); a.y = ex2_approx(a.y);
            }
            if (i & 1) acc1 = fadd2(acc1, a); else acc0 = fadd2(acc0, a);
            pk[i] = pack_f16(a.x, a.y);
          }
          tmem_st16(tS + q * 16, pk);                            // P_t: keys 64 h + 32 q .. + 31 -> 16 columns
          tmem_st_wait();
          tc_fence_before();
          __syncwarp();
          if (lane == 0) mbar_arrive(p_full(t, q));
          if (tr) ATC_TR(cnt, 3 + q + 8 * t);
        }
        l_run += (acc0.x + acc0.y) + (acc1.x + acc1.y);
      }

      // epilogue of this tile: the row sum of both halves (fixed order: half 0 + half 1), then O_t / l -> o32, o16 (through
      // the staging tile), LSE; this warp stores columns [64 h, 64 h + 64) and releases them
      named_bar_sync_gemm(pair_bar, 64);                          // the peer has read this warp's last block maximum
      *xmine = l_run;
      named_bar_sync_gemm(pair_bar, 64);
      const float l_tot = xch_ptr[(t * 2) * 128 + row] + xch_ptr[(t * 2 + 1) * 128 + row];
      named_bar_sync_gemm(pair_bar, 64);                          // both have read: the slots may take the next item's maxima
      mbar_wait(o_full(t), (cnt - 1u) & 1u);
      tc_fence_after();
      const bool valid = qi < p.S;
      const float inv = 1.0f / l_tot;
      if (valid && h == 0) p.lse[(static_cast<long long>(w.b) * p.nq + w.h) * p.S + qi] = (m_run * c + log2f(l_tot)) * 0.6931471805599453f;
      const int r_base = w.q0 + t * 128 + quarter * 32;          // first row of this warp
      const int nrows = min(32, p.S - r_base);
      uint32_t orr[2][32];
      tmem_ld32(tO, orr[0]);
      tmem_ld32(tO + 32, orr[1]);
      tmem_ld_wait();
      tc_fence_before();                                         // O_t is in registers: the next item's P V may overwrite it
      __syncwarp();
      if (lane == 0) mbar_arrive(o_free(t));
      if (nrows > 0) {                                           // rows past the sequence end are clipped by the maps
#pragma unroll
        for (int q = 0; q < 2; ++q) {
          float (&o)[32] = reinterpret_cast<float(&)[32]>(orr[q]);
#pragma unroll
          for (int i = 0; i < 32; ++i) o[i] *= inv;
          const int col = w.h * ATC_D + h * 64 + q * 32;
          if (p.o32) {
#pragma unroll
            for (int e = 0; e < 2; ++e) {                        // two fp32 chunks of 16 columns (64-byte rows)
              uint32_t wv[16];
#pragma unroll
              for (int i = 0; i < 16; ++i) wv[i] = orr[q][16 * e + i];
              if (lane == 0) tma_store_wait_read<0>();           // the previous store has read the tile
              __syncwarp();
              wst.put_row16(wv);
              fence_proxy_async_smem();
              __syncwarp();
              if (lane == 0) { tma_store_3d(&maps.o32, wst.base, col + 16 * e, r_base, w.b); tma_store_commit(); }
            }
          }
          if (p.o16) {
            uint32_t wv[16];
#pragma unroll
            for (int i = 0; i < 16; ++i) wv[i] = pack_f16(o[2 * i], o[2 * i + 1]);
            if (lane == 0) tma_store_wait_read<0>();
            __syncwarp();
            wst.put_row16(wv);
            fence_proxy_async_smem();
            __syncwarp();
            if (lane == 0) { tma_store_3d(&maps.o16, wst.base, col, r_base, w.b); tma_store_commit(); }
          }
        }
      }
    }
    if (lane == 0) tma_store_wait_all<0>();                      // this thread's bulk stores have been written
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
                                      long long ldv, const AttnTcParams& p, int num_sms, cudaStream_t st) {
  static DeviceOnce once;
  if (once.need()) {
    cudaError_t e = cudaFuncSetAttribute(attn_fwd_tc_kernel<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, ATC_FWD_SMEM);
    if (e != cudaSuccess) return e;
    e = cudaFuncSetAttribute(attn_fwd_tc_kernel<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, ATC_FWD_SMEM);
    if (e != cudaSuccess) return e;
    once.done();
  }
  AttnTcMaps maps;
  if (!make_map_attn(&maps.q, q, p.nq * ATC_D, p.S, p.B, ldq) || !make_map_attn(&maps.k, k, p.nkv * ATC_D, p.S, p.B, ldk) ||
      !make_map_attn(&maps.v, v, p.nkv * ATC_D, p.S, p.B, ldv))
    return cudaErrorInvalidValue;
  maps.dO = maps.q;
  maps.o32 = maps.q; maps.o16 = maps.q;
  if (p.o32 && !make_map_store(&maps.o32, p.o32, p.nq * ATC_D, p.S, p.B, p.ldo, true, true)) return cudaErrorInvalidValue;
  if (p.o16 && !make_map_store(&maps.o16, p.o16, p.nq * ATC_D, p.S, p.B, p.ldo, false)) return cudaErrorInvalidValue;
  const int nitems = ((p.S + 255) / 256) * p.nq * p.B;
  const int grid = nitems < num_sms ? nitems : num_sms;        // persistent: one CTA per SM
  if (p.doc_start) return launch_kernel(attn_fwd_tc_kernel<true>, dim3(grid), dim3(ATC_FWD_THREADS), ATC_FWD_SMEM, st, maps, p);
  return launch_kernel(attn_fwd_tc_kernel<false>, dim3(grid), dim3(ATC_FWD_THREADS), ATC_FWD_SMEM, st, maps, p);
}

// =========================================================================================== backward
// SURVEY 8(a) B7 (+B8 on store).  Two deterministic kernels, no atomics (results are bit-reproducible):
//   dK/dV : one CTA per (128-key block, kv head, batch) walks the G query heads of the group and the 128-query
//           blocks at / below the diagonal, in the transposed domain (TMEM lane = key):
//             S^T = K Q^T, dP^T = V dO^T          (A = K, V K-major from smem; B = Q, dO K-major)
//             P^T = exp2(S^T c - L log2e)         (softmax threads; fp16 -> TMEM over S^T)
//             dV += P^T dO                        (A = P^T from TMEM; B = dO MN-major: the same smem tile)
//             dS^T = P^T (dP^T - D)               (fp16 -> TMEM over dP^T)
//             dK += dS^T Q                        (A = dS^T from TMEM; B = Q MN-major)
//           dK, dV accumulate in TMEM over the whole walk (the GQA group sum costs nothing).
//   dQ    : one CTA per (128-query block, head, batch) walks the 64-key blocks up to the diagonal:
//             S = Q K^T, dP = dO V^T, dS = exp2(S c - L log2e)(dP - D) -> TMEM, dQ += dS K (K MN-major).
// 256 softmax threads (8 warps: TMEM lane quarter x column half) in both; the pipelines differ (see each kernel): dK/dV
// staggers two MMA groups over single 128-column S^T / dP^T accumulators, dQ double-buffers 64-column S / dP accumulators
// and keeps Q, dO in TMEM.  The 16-bit operand written back over an fp32 accumulator keeps each half inside the columns
// its own warp read, so the two half-warps never race.
constexpr int ATC_BWD_THREADS = 320;
// Query positions below this keep P / dS as a two-term fp16 sum (hi + lo, two MMAs into the same accumulator):
// early rows are O(1) while the tensor-wide rms the parity metric divides by shrinks like sqrt(ln S / S), so a
// single fp16 rounding there is what limits dq/dk/dv at long S (P-5/P-6).
constexpr int ATC_SPLIT_ROWS = 256;
constexpr int ATC_HALF_TILE = 64 * ATC_D * 2;              // 64 x 128 fp16 = 16 KB (two 8 KB chunks)

struct AttnTcBwdParams {
  int B, S, nq, nkv;
  float scale_log2, scale;
  const float* lse;            // [B, nq, S]
  const float* dvec;           // [B, nq, S, 4]: D = rowsum(dO * O) as four partial sums (one per 32-column chunk of the
                               // head, written by the O-projection dgrad epilogue); readers add them as (x + y) + (z + w)
  const float2* rope;          // (cos, sin) [S, 64] or null: inverse rotation of dq, dk on store
  float* dq32; float* dk32; float* dv32; long long lddq32, lddk32;
  __half* dq16; __half* dk16; __half* dv16; long long ldd16;
  unsigned int* sched;         // work-item counters of the persistent kernels ([4], [5]: dQ kernel), zero between launches
  const int* doc_start; const int* doc_end;      // packed sequences (see AttnTcParams); rope rows are then t - doc_start[t]
};

__device__ __forceinline__ void atc_load_half_tile(uint32_t dst, const CUtensorMap* m, uint32_t bar, int col0, int s0, int b) {
  mbar_expect_tx(bar, ATC_HALF_TILE);
  tma_load_3d(dst, m, bar, col0, s0, b);
  tma_load_3d(dst + 64 * 128, m, bar, col0 + 64, s0, b);
}
// 64-row tile (two 8 KB chunks) as a K-major B operand (N = 64 rows, K = 128 contiguous): kk-th 16-element K step
__device__ __forceinline__ uint64_t atc_desc_half_kmajor(uint32_t tile, int kk) {
  return umma_smem_desc(tile + (kk >> 2) * (64 * 128) + (kk & 3) * 32, 16, 1024);
}
// the same tile as an MN-major B operand (K = 64 rows, N = 128 contiguous): kk-th 16-row K step
__device__ __forceinline__ uint64_t atc_desc_half_mnmajor(uint32_t tile, int kk) {
  return umma_smem_desc(tile + kk * 2048, 64 * 128, 1024);
}
// TMEM column of the kk-th 16-element K step of a 64-wide fp16 operand stored as described above
__device__ __forceinline__ uint32_t atc_half_operand_col(int kk) { return static_cast<uint32_t>((kk >> 1) * 32 + (kk & 1) * 8); }

// x = hi + lo with both halves fp16: packs two values' hi parts and lo parts.
__device__ __forceinline__ void atc_split_pack(float x0, float x1, uint32_t& hi, uint32_t& lo) {
  hi = pack_f16(x0, x1);
  const float2 hf = __half22float2(*reinterpret_cast<const __half2*>(&hi));
  lo = pack_f16(x0 - hf.x, x1 - hf.y);
}

// Scale, optionally rotate by -theta (transpose of the forward rotation) 32 columns of this thread's row, then write the
// warp's 32 x 32 chunk (rows s0.., columns col0.., batch b) with bulk tensor stores out of the staging tile.
__device__ __forceinline__ void atc_store_grad32(const WarpStage& st, float (&v)[32], float scale, const float2* rope_row,
                                                 const CUtensorMap* m32, const CUtensorMap* m16, int col0, int s0, int b) {
#pragma unroll
  for (int i = 0; i < 16; ++i) {
    float z0 = v[2 * i] * scale, z1 = v[2 * i + 1] * scale;
    if (rope_row) {
      const float2 cs = __ldg(rope_row + i);
      const float r0 = z0 * cs.x + z1 * cs.y, r1 = -z0 * cs.y + z1 * cs.x;
      z0 = r0; z1 = r1;
    }
    v[2 * i] = z0; v[2 * i + 1] = z1;
  }
  if (m32) chunk_store_tma3<DT_F32>(st, m32, col0, s0, b, v);
  if (m16) chunk_store_tma3<DT_F16>(st, m16, col0, s0, b, v);
}

// --------------------------------------------------------------------------------------------- dK, dV
// One CTA per (128-key block, kv head, batch) walks the G query heads of the group and the 128-query blocks at / below
// the diagonal, in the transposed domain (TMEM lane = key), with N = 128 MMAs throughout: a 64-query block made the
// S^T / dP^T steps (A = K, V from shared memory, re-read at 32 cycles per K = 16 step whatever N is) cost 48 cycles for
// 32 cycles of tensor work; at N = 128 the operand reads (A 32 + B 32) equal the 64 tensor cycles.
// TMEM holds ONE S^T and ONE dP^T accumulator ([0,128), [128,256); dV [256,384), dK [384,512)); the pipeline is
// staggered instead of double-buffered -- the tensor core alternates two MMA groups per block,
//     after P^T(i)  is written:  dV += P^T(i) dO(i) ,  S^T(i+1) = K Q(i+1)^T      (S^T(i+1) overwrites P^T(i): in-order)
//     after dS^T(i) is written:  dK += dS^T(i) Q(i) ,  dP^T(i+1) = V dO(i+1)^T    (dP^T(i+1) overwrites dS^T(i))
// while the softmax threads turn dP^T(i) into dS^T(i) during the first group and S^T(i+1) into P^T(i+1) during the
// second: 2048 tensor cycles per 128 x 128 block (2560 with 64-query blocks) as long as each softmax phase stays under
// the 1024 cycles of the other group.  Q is streamed through a 3-stage ring, dO through a 2-stage ring (Q(i) is needed
// first and released last: S^T(i) ... dK(i)); L and D of the block's queries through a 2-stage ring of their own.
// Shared memory: K, V 64 KB + Q 96 KB + dO 64 KB + L/D 2 KB; the epilogue's staging tiles reuse the Q ring.
constexpr int ATC_KV_QST = 3;                              // Q ring stages (128 x 128 tiles)
constexpr int ATC_KV_DST = 2;                              // dO ring stages
constexpr int ATC_KV_LD_BYTES = 2 * 2 * 128 * 4;           // [2 stages][L*log2e (128) | D (128)] fp32
// declared 1024-byte aligned, no slack (see ATC_FWD_SMEM)
constexpr int ATC_BWD_SMEM = (2 + ATC_KV_QST + ATC_KV_DST) * ATC_TILE_BYTES + ATC_KV_LD_BYTES + 256;

template <bool DOC>
__global__ void __launch_bounds__(ATC_BWD_THREADS, 1)
attn_bwd_dkdv_tc_kernel(const __grid_constant__ AttnTcMaps maps, const AttnTcBwdParams p) {
  // packed sequences compiled in only for DOC: the plain kernels carry none of the bound / mask code
  const int* const doc_start = DOC ? p.doc_start : nullptr;
  const int* const doc_end = DOC ? p.doc_end : nullptr;
  (void)doc_start; (void)doc_end;
  extern __shared__ __align__(1024) uint8_t smem_raw[];
  const uint32_t smem_base = smem_u32(smem_raw);
  if (smem_base & 1023u) __trap();
  const uint32_t sK = smem_base, sV = sK + ATC_TILE_BYTES;
  const uint32_t sQ = sV + ATC_TILE_BYTES;                       // ATC_KV_QST stages
  const uint32_t sDO = sQ + ATC_KV_QST * ATC_TILE_BYTES;         // ATC_KV_DST stages
  const uint32_t sLD = sDO + ATC_KV_DST * ATC_TILE_BYTES;
  const uint32_t bar_base = sLD + ATC_KV_LD_BYTES;
  const uint32_t stage_tiles = sQ;                               // epilogue only: 8 x 4 KB inside the (then idle) Q ring
  float* sLD_ptr = reinterpret_cast<float*>(smem_raw + (sLD - smem_base));
  auto kv_full = [&]() { return bar_base; };
  auto acc_full = [&]() { return bar_base + 8u; };
  auto st_full = [&]() { return bar_base + 16u; };               // MMA: S^T of the block has landed
  auto dpt_full = [&]() { return bar_base + 24u; };              // MMA: dP^T of the block has landed
  auto p_full = [&](int q) { return bar_base + 32u + 8u * q; };  // 8 softmax warps: P^T of query quarter-pair q written (q = 0, 1)
  auto ds_full = [&]() { return bar_base + 48u; };               // 8 softmax warps: dS^T written
  auto q_full = [&](int s) { return bar_base + 8u * (7 + s); };
  auto q_empty = [&](int s) { return bar_base + 8u * (7 + ATC_KV_QST + s); };
  auto do_full = [&](int s) { return bar_base + 8u * (7 + 2 * ATC_KV_QST + s); };
  auto do_empty = [&](int s) { return bar_base + 8u * (7 + 2 * ATC_KV_QST + ATC_KV_DST + s); };
  auto ld_full = [&](int s) { return bar_base + 8u * (7 + 2 * ATC_KV_QST + 2 * ATC_KV_DST + s); };
  auto ld_empty = [&](int s) { return bar_base + 8u * (9 + 2 * ATC_KV_QST + 2 * ATC_KV_DST + s); };
  const uint32_t tmem_slot = bar_base + 8u * (11 + 2 * ATC_KV_QST + 2 * ATC_KV_DST);
  uint32_t* tmem_slot_ptr = reinterpret_cast<uint32_t*>(smem_raw + (tmem_slot - smem_base));

  const int warp = warp_idx_uniform(), lane = threadIdx.x & 31;
  // 1-D grid, key block SLOWEST: CTAs are dispatched in linear order and a CTA's work falls linearly with its key block
  // (causal), so the heaviest CTAs of ALL (kv head, batch) groups start first and the light ones fill the tail
  // (longest-processing-time order: makespan 696 instead of 792 block units on 148 SMs at S = 4096, 8 kv heads x 4).
  const int ngroups = p.nkv * p.B;
  const int kb = static_cast<int>(blockIdx.x) / ngroups, grp = static_cast<int>(blockIdx.x) - kb * ngroups;
  const int kvh = grp % p.nkv, b = grp / p.nkv;
  const int G = p.nq / p.nkv;
  const int k0 = kb * 128;
  // packed sequences: no query past the end of the sequence of this block's last key attends any of its keys
  const int q_end = doc_end ? doc_end[min(k0 + 127, p.S - 1)] : p.S;
  const int per_head = (q_end + 127) / 128 - kb;                 // 128-query blocks at / below the diagonal
  // early positions of a sequence take hi + lo fp16 operands: a query block splits when its last query is closer than
  // ATC_SPLIT_ROWS to the start of that query's sequence (position 0 without packing)
  auto split_block = [&](int qblk) {
    const int qs = qblk * 128;
    return qs - (doc_start ? doc_start[min(qs + 127, p.S - 1)] : 0) < ATC_SPLIT_ROWS;
  };
  const int iters = per_head * G;
  if (threadIdx.x == 64) ATC_TRL(0);                              // CTA entered

  if (threadIdx.x == 0) {
    tma_prefetch_desc(&maps.q); tma_prefetch_desc(&maps.k); tma_prefetch_desc(&maps.v); tma_prefetch_desc(&maps.dO);
    mbar_init(kv_full(), 1); mbar_init(acc_full(), 1); mbar_init(st_full(), 1); mbar_init(dpt_full(), 1);
    mbar_init(p_full(0), 8); mbar_init(p_full(1), 8); mbar_init(ds_full(), 8);
    for (int i = 0; i < ATC_KV_QST; ++i) { mbar_init(q_full(i), 1); mbar_init(q_empty(i), 1); }
    for (int i = 0; i < ATC_KV_DST; ++i) { mbar_init(do_full(i), 1); mbar_init(do_empty(i), 1); }
    for (int i = 0; i < 2; ++i) { mbar_init(ld_full(i), 32); mbar_init(ld_empty(i), 8); }
    fence_barrier_init();
  }
  if (warp == 1) { tmem_alloc(tmem_slot, 512); tmem_relinquish(); }
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tmem_base = *tmem_slot_ptr;
  pdl_wait();                                    // no global access above (programmatic dependent launch, ptx.cuh)
  pdl_trigger();

  if (warp == 0) {
    // ===================================================================== producer: TMA tiles + L, D vectors
    if (lane == 0) {
      mbar_expect_tx(kv_full(), 2 * ATC_TILE_BYTES);
      tma_load_3d(sK, &maps.k, kv_full(), kvh * ATC_D, k0, b);
      tma_load_3d(sK + ATC_CHUNK_BYTES, &maps.k, kv_full(), kvh * ATC_D + 64, k0, b);
      tma_load_3d(sV, &maps.v, kv_full(), kvh * ATC_D, k0, b);
      tma_load_3d(sV + ATC_CHUNK_BYTES, &maps.v, kv_full(), kvh * ATC_D + 64, k0, b);
    }
    for (int it = 0; it < iters; ++it) {
      const int qs = it % ATC_KV_QST, ds = it % ATC_KV_DST, ls = it & 1;
      const int hh = kvh * G + it / per_head;
      const int s0 = (kb + it % per_head) * 128;
      if (lane == 0) {
        mbar_wait(q_empty(qs), ((it / ATC_KV_QST) & 1) ^ 1u);
        atc_load_tile(sQ + qs * ATC_TILE_BYTES, &maps.q, q_full(qs), hh * ATC_D, s0, b);
        mbar_wait(do_empty(ds), ((it / ATC_KV_DST) & 1) ^ 1u);
        atc_load_tile(sDO + ds * ATC_TILE_BYTES, &maps.dO, do_full(ds), hh * ATC_D, s0, b);
      }
      mbar_wait(ld_empty(ls), ((it >> 1) & 1) ^ 1u);
      const long long vbase = (static_cast<long long>(b) * p.nq + hh) * p.S;
#pragma unroll
      for (int r = 0; r < 4; ++r) {
        const int s = s0 + lane + 32 * r;
        const bool ok = s < p.S;
        const float4 d4 = ok ? __ldg(reinterpret_cast<const float4*>(p.dvec) + vbase + s) : make_float4(0.f, 0.f, 0.f, 0.f);
        sLD_ptr[ls * 256 + lane + 32 * r] = ok ? p.lse[vbase + s] * 1.4426950408889634f : INFINITY;
        sLD_ptr[ls * 256 + 128 + lane + 32 * r] = (d4.x + d4.y) + (d4.z + d4.w);
      }
      mbar_arrive(ld_full(ls));
    }
  } else if (warp == 1) {
    // ===================================================================== MMA issuer (whole warp, elected lane issues)
    const uint32_t leader = elect_one();
    const uint32_t idesc_sdp = umma_idesc(128, 128, 0, 0, 0, 0);    // [128 keys x 128 queries] = A(K-major) B(K-major)^T
    const uint32_t idesc_acc = umma_idesc(128, 128, 0, 0, 0, 1);    // [128 keys x 128 d] += A(TMEM) B(MN-major)
    const uint64_t dK = umma_smem_desc(sK, 16, 1024), dV = umma_smem_desc(sV, 16, 1024);
    const uint64_t dQk = umma_smem_desc(sQ, 16, 1024), dDOk = umma_smem_desc(sDO, 16, 1024);                         // K-major views
    const uint64_t dQm = umma_smem_desc(sQ, ATC_CHUNK_BYTES, 1024), dDOm = umma_smem_desc(sDO, ATC_CHUNK_BYTES, 1024); // MN-major views
    // S^T = K Q^T of block `it` (its Q stage must have landed)
    auto issue_st = [&](int it) {
      const int qs = it % ATC_KV_QST;
      if (leader) {
        const uint64_t qa = desc_adv(dQk, qs * ATC_TILE_BYTES);
#pragma unroll
        for (int kk = 0; kk < 8; ++kk) {
          const uint32_t off = (kk >> 2) * ATC_CHUNK_BYTES + (kk & 3) * 32;
          umma_f16(tmem_base, desc_adv(dK, off), desc_adv(qa, off), idesc_sdp, kk != 0 ? 1u : 0u);
        }
        umma_commit(st_full());
      }
    };
    auto issue_dpt = [&](int it) {
      const int ds = it % ATC_KV_DST;
      if (leader) {
        const uint64_t da = desc_adv(dDOk, ds * ATC_TILE_BYTES);
#pragma unroll
        for (int kk = 0; kk < 8; ++kk) {
          const uint32_t off = (kk >> 2) * ATC_CHUNK_BYTES + (kk & 3) * 32;
          umma_f16(tmem_base + 128, desc_adv(dV, off), desc_adv(da, off), idesc_sdp, kk != 0 ? 1u : 0u);
        }
        umma_commit(dpt_full());
      }
    };
    // TMEM column of K step kk (16 queries) of a 16-bit operand written by the softmax threads: query half h = kk / 4
    // keeps its 64 queries in the 32 columns [64 h, 64 h + 32) (hi parts; lo parts of split blocks 32 columns further)
    auto opcol = [](int kk) { return static_cast<uint32_t>((kk >> 2) * 64 + (kk & 3) * 8); };
    if (iters > 0) {
      mbar_wait(kv_full(), 0);
      mbar_wait2(q_full(0), 0, do_full(0), 0);
      tc_fence_after();
      issue_st(0);
      issue_dpt(0);
    }
    for (int it = 0; it < iters; ++it) {
      const int qs = it % ATC_KV_QST, ds = it % ATC_KV_DST;
      const uint32_t ph = it & 1;
      const uint64_t qa = desc_adv(dQm, qs * ATC_TILE_BYTES), da = desc_adv(dDOm, ds * ATC_TILE_BYTES);
      const bool split = split_block(kb + it % per_head);
      // each MMA group needs two barriers -- the softmax threads' operand and the next block's tile: polled together.
      // P^T arrives in two parts (the first / second 32 queries of both query halves = K steps {0,1,4,5} / {2,3,6,7}): the
      // first half of dV runs while the second half of P^T is still being exponentiated
      if (it + 1 < iters) mbar_wait2(p_full(0), ph, q_full((it + 1) % ATC_KV_QST), ((it + 1) / ATC_KV_QST) & 1);
      else mbar_wait(p_full(0), ph);
      if (lane == 0) ATC_TR2(it, 16);
#pragma unroll
      for (int part = 0; part < 2; ++part) {
        if (part == 1) mbar_wait(p_full(1), ph);
        tc_fence_after();
        if (leader) {
#pragma unroll
          for (int e = 0; e < 4; ++e) {                               // dV += P^T dO
            const int kk = (e >> 1) * 4 + part * 2 + (e & 1);
            umma_f16_ts(tmem_base + 256, tmem_base + opcol(kk), desc_adv(da, kk * 2048), idesc_acc, (it | part | e) != 0 ? 1u : 0u);
          }
          if (split) {
#pragma unroll
            for (int e = 0; e < 4; ++e) {                             // ... + (P^T)_lo dO
              const int kk = (e >> 1) * 4 + part * 2 + (e & 1);
              umma_f16_ts(tmem_base + 256, tmem_base + 32 + opcol(kk), desc_adv(da, kk * 2048), idesc_acc, 1u);
            }
          }
          if (part == 1) umma_commit(do_empty(ds));                   // dO(it) was last read by these MMAs
        }
      }
      if (lane == 0) ATC_TR2(it, 17);
      if (it + 1 < iters) issue_st(it + 1);                           // overwrites P^T(it): behind dV in the tensor queue
      if (lane == 0) ATC_TR2(it, 18);
      if (it + 1 < iters) mbar_wait2(ds_full(), ph, do_full((it + 1) % ATC_KV_DST), ((it + 1) / ATC_KV_DST) & 1);
      else mbar_wait(ds_full(), ph);
      if (lane == 0) ATC_TR2(it, 19);
      tc_fence_after();
      if (leader) {
#pragma unroll
        for (int kk = 0; kk < 8; ++kk)                                // dK += dS^T Q
          umma_f16_ts(tmem_base + 384, tmem_base + 128 + opcol(kk), desc_adv(qa, kk * 2048), idesc_acc, (it | kk) != 0 ? 1u : 0u);
        if (split) {
#pragma unroll
          for (int kk = 0; kk < 8; ++kk)
            umma_f16_ts(tmem_base + 384, tmem_base + 128 + 32 + opcol(kk), desc_adv(qa, kk * 2048), idesc_acc, 1u);
        }
        umma_commit(q_empty(qs));                                     // Q(it) was last read by these MMAs
      }
      if (lane == 0) ATC_TR2(it, 20);
      if (it + 1 < iters) issue_dpt(it + 1);                          // overwrites dS^T(it): behind dK in the tensor queue
      if (lane == 0) ATC_TR2(it, 21);
    }
    if (leader) umma_commit(acc_full());
  } else {
    // ===================================================================== softmax warps (8): lane quarter x query half
    const int quarter = warp & 3, half = (warp - 2) >> 2;
    const int row = quarter * 32 + lane;                               // key within the block = TMEM lane
    const uint32_t lane_off = static_cast<uint32_t>(quarter * 32) << 16;
    const int col0 = half * 64;                                        // this warp's 64 queries of the block
    const uint32_t tST = tmem_base + lane_off + col0, tDP = tmem_base + lane_off + 128 + col0;
    const float c = p.scale_log2;
    const int dend = doc_end ? doc_end[min(k0 + row, p.S - 1)] : p.S;   // end of this key's sequence
    for (int it = 0; it < iters; ++it) {
      const int ls = it & 1;
      const uint32_t ph = it & 1;
      const int rel = it % per_head;                                   // 128-query block index relative to the diagonal
      const bool split = split_block(kb + rel);                        // early query positions: hi + lo operands
      mbar_wait(ld_full(ls), (it >> 1) & 1);
      mbar_wait(st_full(), ph);
      const bool tr = quarter == 0 && half == 0 && lane == 0;
      if (tr) ATC_TR2(it, 0);
      if (tr && it == 0) ATC_TRL(1);                                   // first S^T landed: the loop starts
      tc_fence_after();
      float pv[64];
      {
        uint32_t sr[2][32];
        tmem_ld32(tST, sr[0]);
        tmem_ld32(tST + 32, sr[1]);
        tmem_ld_wait();                                                // all 64 columns in registers before any of them is overwritten
        const float2 c2 = make_float2(c, c);
#pragma unroll
        for (int q = 0; q < 2; ++q) {                                  // two parts of 32 queries, handed over separately
          const float4* l4 = reinterpret_cast<const float4*>(sLD_ptr + ls * 256 + col0 + 32 * q);
#pragma unroll
          for (int i = 0; i < 8; ++i) {
            const float4 L = l4[i];
            float2 a = ffma2(make_float2(__uint_as_float(sr[q][4 * i]), __uint_as_float(sr[q][4 * i + 1])), c2, make_float2(-L.x, -L.y));
            float2 b2 = ffma2(make_float2(__uint_as_float(sr[q][4 * i + 2]), __uint_as_float(sr[q][4 * i + 3])), c2, make_float2(-L.z, -L.w));
            // LSP_ATTN_BWD_POLY_EXP quarters of the key pairs on the FMA pipe (the phase is SFU-bound): 1 = a of even i, 2 = every a,
            // 3 = every a and b2 of even i
            if (LSP_ATTN_BWD_POLY_EXP >= 2 || (LSP_ATTN_BWD_POLY_EXP == 1 && (i & 1) == 0)) {
              a = ex2_poly2(a);
            } else {
              a.x = ex2_approx(a.x); a.y = ex2_approx(a.y);
            }
            if (LSP_ATTN_BWD_POLY_EXP >= 3 && (i & 1) == 0) {
              b2 = ex2_poly2(b2);
            } else {
              b2.x = ex2_approx(b2.x); b2.y = ex2_approx(b2.y);
            }
            pv[32 * q + 4 * i] = a.x; pv[32 * q + 4 * i + 1] = a.y; pv[32 * q + 4 * i + 2] = b2.x; pv[32 * q + 4 * i + 3] = b2.y;
          }
          if (rel == 0) {                                              // diagonal block: query (col0 + 32 q + i) < key (row) is masked
#pragma unroll
            for (int i = 0; i < 32; ++i)
              if (col0 + 32 * q + i < row) pv[32 * q + i] = 0.f;
          }
          if (doc_end) {                                               // packed sequences: queries of later sequences
            const int qabs = (kb + rel) * 128 + col0 + 32 * q;
            if (__any_sync(0xffffffffu, qabs + 31 >= dend)) {
#pragma unroll
              for (int i = 0; i < 32; ++i)
                if (qabs + i >= dend) pv[32 * q + i] = 0.f;
            }
          }
          uint32_t pk[16];
          if (split) {
            uint32_t pl[16];
#pragma unroll
            for (int i = 0; i < 16; ++i) atc_split_pack(pv[32 * q + 2 * i], pv[32 * q + 2 * i + 1], pk[i], pl[i]);
            tmem_st16(tST + 32 + 16 * q, pl);
          } else {
#pragma unroll
            for (int i = 0; i < 16; ++i) pk[i] = pack_f16(pv[32 * q + 2 * i], pv[32 * q + 2 * i + 1]);
          }
          tmem_st16(tST + 16 * q, pk);
          tmem_st_wait();
          tc_fence_before();
          __syncwarp();
          if (lane == 0) mbar_arrive(p_full(q));
        }
      }
      if (tr) ATC_TR2(it, 1);
      // dS^T = P^T (dP^T - D)
      mbar_wait(dpt_full(), ph);
      if (tr) ATC_TR2(it, 2);
      tc_fence_after();
      {
        uint32_t dr[2][32];
        tmem_ld32(tDP, dr[0]);
        tmem_ld32(tDP + 32, dr[1]);
        tmem_ld_wait();
        const float4* d4 = reinterpret_cast<const float4*>(sLD_ptr + ls * 256 + 128 + col0);
#pragma unroll
        for (int i = 0; i < 16; ++i) {
          const float4 Dv = d4[i];
          pv[4 * i] *= __uint_as_float(dr[i >> 3][(4 * i) & 31]) - Dv.x;
          pv[4 * i + 1] *= __uint_as_float(dr[i >> 3][(4 * i + 1) & 31]) - Dv.y;
          pv[4 * i + 2] *= __uint_as_float(dr[i >> 3][(4 * i + 2) & 31]) - Dv.z;
          pv[4 * i + 3] *= __uint_as_float(dr[i >> 3][(4 * i + 3) & 31]) - Dv.w;
        }
      }
      __syncwarp();
      if (lane == 0) mbar_arrive(ld_empty(ls));                        // L and D of this block have been read
      {
        uint32_t pk[32];
        if (split) {
          uint32_t pl[32];
#pragma unroll
          for (int i = 0; i < 32; ++i) atc_split_pack(pv[2 * i], pv[2 * i + 1], pk[i], pl[i]);
          tmem_st32(tDP + 32, pl);
        } else {
#pragma unroll
          for (int i = 0; i < 32; ++i) pk[i] = pack_f16(pv[2 * i], pv[2 * i + 1]);
        }
        tmem_st32(tDP, pk);
      }
      tmem_st_wait();
      tc_fence_before();
      __syncwarp();
      if (lane == 0) mbar_arrive(ds_full());
      if (tr) ATC_TR2(it, 3);
      if (tr && it == iters - 1) ATC_TRL(2);                           // last dS^T handed over
    }
    // epilogue: this warp stores rows [32 quarter, +32), columns [64 half, 64 half + 64) of dV and dK
    mbar_wait(acc_full(), 0);
    if (quarter == 0 && half == 0 && lane == 0) ATC_TRL(3);           // accumulators complete: stores begin
    tc_fence_after();
    const int key = k0 + row;
    const bool valid = key < p.S;
    const WarpStage wst{stage_tiles + static_cast<uint32_t>(warp - 2) * GEMM_STAGE_TILE_BYTES, lane};
    const int s0 = k0 + quarter * 32;
    if (s0 < p.S) {
#pragma unroll 1
      for (int q = 0; q < 2; ++q) {
        const int cc = half * 64 + q * 32;
        uint32_t a[32];
        tmem_ld32(tmem_base + lane_off + 256 + cc, a);
        tmem_ld_wait();
        atc_store_grad32(wst, reinterpret_cast<float(&)[32]>(a), 1.0f, nullptr, p.dv32 ? &maps.g32[0] : nullptr,
                         p.dv16 ? &maps.g16[0] : nullptr, kvh * ATC_D + cc, s0, b);
        tmem_ld32(tmem_base + lane_off + 384 + cc, a);
        tmem_ld_wait();
        atc_store_grad32(wst, reinterpret_cast<float(&)[32]>(a), p.scale,
                         (p.rope && valid) ? p.rope + static_cast<long long>(key - (doc_start ? doc_start[key] : 0)) * 64 + (cc >> 1) : nullptr,
                         p.dk32 ? &maps.g32[1] : nullptr, p.dk16 ? &maps.g16[1] : nullptr, kvh * ATC_D + cc, s0, b);
      }
    }
    if (lane == 0) tma_store_wait_all<0>();
    if (quarter == 0 && half == 0 && lane == 0) ATC_TRL(4);           // this warp's stores are written
  }

  tc_fence_before();
  __syncthreads();
  if (warp == 1) { tc_fence_after(); tmem_dealloc(tmem_base, 512); }
#ifdef LSP_ATTN_TRACE
  if (threadIdx.x == 64 && (blockIdx.x == 5 || blockIdx.x == 900)) {
    ATC_TRL(5);
    g_atc_trace[(blockIdx.x == 5 ? 62 : 63) * 32 + 22] = static_cast<unsigned long long>(iters);
  }
#endif
}

// --------------------------------------------------------------------------------------------- dQ
// Q and dO of the item are the A operands of EVERY S = Q K^T and dP = dO V^T block of its key loop.  As shared-memory
// operands (SS) an M = 128 MMA re-reads them at 32 cycles per K = 16 step whatever N is, which made the N = 64 steps cost
// 48 cycles instead of 32 (shared-memory bound, measured; 1024 instead of 768 tensor cycles per 128 x 64 block).  They
// now live in TMEM: the 8 softmax warps copy the TMA-landed tiles (lane = query row, two 16-bit values per column)
// once per item, and S / dP run as TS MMAs whose only shared-memory traffic is the 64-key K / V tile.
// TMEM: Q [0,64) dO [64,128) | S buffers [128,256) | dP buffers [256,384) | dQ [384,512).  Two S / dP buffers: the tensor
// core works one key block ahead of the softmax threads (768 tensor cycles per block against ~500 of softmax).
constexpr int ATC_DQ_NB = 2;
constexpr int ATC_DQ_NST = 4;
constexpr int ATC_DQ_SMEM = 2 * ATC_TILE_BYTES + 2 * ATC_DQ_NST * ATC_HALF_TILE + 8 * GEMM_STAGE_TILE_BYTES + 1024 + 256;
constexpr int ATC_DQ_QA = 0;                     // Q operand columns
constexpr int ATC_DQ_DOA = 64;                   // dO operand columns
constexpr int ATC_DQ_S = 128;                    // first S column
constexpr int ATC_DQ_DP = 256;                   // first dP column
constexpr int ATC_DQ_ACC = 384;                  // dQ accumulator column
// Persistent like the forward: work items (128-query block, head, batch) come heaviest-first from an atomic counter
// (p.sched + 4); Q / dO of the next item are fetched as soon as the softmax warps have copied the current ones to TMEM
// (qdo_empty), the dQ epilogue (TMEM -> staging tile -> bulk stores) overlaps the first S / dP MMAs of the next item, and
// acc_free tells the MMA warp when the dQ accumulator may be overwritten.
struct AttnDqItem { int q0, h, b, kvh, iters, j0, split; };        // j0: first 64-key block (packed sequences), else 0
__device__ __forceinline__ AttnDqItem attn_dq_item(uint32_t i, const AttnTcBwdParams& p, int nqb, const int* doc_start) {
  const int per_lvl = p.nq * p.B;
  const int lvl = static_cast<int>(i) / per_lvl, r = static_cast<int>(i) - lvl * per_lvl;
  AttnDqItem it;
  it.q0 = (nqb - 1 - lvl) * 128;                                 // heavy (late) query blocks first
  it.b = r / p.nq; it.h = r - it.b * p.nq;
  it.kvh = it.h / (p.nq / p.nkv);
  // packed sequences: keys before the start of the sequence of the item's first query are never visited
  it.j0 = doc_start ? doc_start[it.q0] / 64 : 0;
  it.iters = (min(p.S, it.q0 + 128) + 63) / 64 - it.j0;          // 64-key blocks [64 j0, kv_end)
  // hi + lo fp16 dS operands while the tile's last query is closer than ATC_SPLIT_ROWS to the start of its sequence
  it.split = it.q0 - (doc_start ? doc_start[min(it.q0 + 127, p.S - 1)] : 0) < ATC_SPLIT_ROWS;
  return it;
}

// This thread's row of one 64-column chunk of a TMA-landed 128 x 128 fp16 tile (128B swizzle) -> 32 TMEM columns.
__device__ __forceinline__ void atc_row_chunk_to_tmem(uint32_t chunk_smem, int row, uint32_t taddr) {
  uint32_t w[32];
#pragma unroll
  for (int u = 0; u < 8; ++u)
    asm volatile("ld.shared.v4.b32 {%0, %1, %2, %3}, [%4];" : "=r"(w[4 * u]), "=r"(w[4 * u + 1]), "=r"(w[4 * u + 2]), "=r"(w[4 * u + 3])
                 : "r"(chunk_smem + row * 128 + ((u ^ (row & 7)) << 4)) : "memory");
  tmem_st32(taddr, w);
}

template <bool DOC>
__global__ void __launch_bounds__(ATC_BWD_THREADS, 1)
attn_bwd_dq_tc_kernel(const __grid_constant__ AttnTcMaps maps, const AttnTcBwdParams p) {
  // packed sequences compiled in only for DOC: the plain kernels carry none of the bound / mask code
  const int* const doc_start = DOC ? p.doc_start : nullptr;
  const int* const doc_end = DOC ? p.doc_end : nullptr;
  (void)doc_start; (void)doc_end;
  extern __shared__ uint8_t smem_raw[];
  const uint32_t smem_base = (smem_u32(smem_raw) + 1023u) & ~1023u;
  const uint32_t sQ = smem_base, sDO = sQ + ATC_TILE_BYTES;
  const uint32_t sK = sDO + ATC_TILE_BYTES;                      // ATC_DQ_NST stages of 64 keys x 128
  const uint32_t sV = sK + ATC_DQ_NST * ATC_HALF_TILE;
  const uint32_t stage_tiles = sV + ATC_DQ_NST * ATC_HALF_TILE;      // 8 x 4 KB staging tiles (epilogue)
  const uint32_t bar_base = stage_tiles + 8 * GEMM_STAGE_TILE_BYTES;
  auto qdo_full = [&]() { return bar_base; };                    // TMA: Q, dO of the item have landed in shared memory
  auto acc_full = [&]() { return bar_base + 8u; };
  auto qdo_empty = [&]() { return bar_base + 16u; };             // 8 softmax warps: the tiles have been copied out
  auto acc_free = [&]() { return bar_base + 24u; };
  auto qa_full = [&]() { return bar_base + 32u; };               // 8 softmax warps: the TMEM operands of the item are written
  auto qa_free = [&]() { return bar_base + 40u; };               // MMA: the item's last S / dP has read them
  auto kv_full = [&](int s) { return bar_base + 8u * (6 + s); };
  auto kv_empty = [&](int s) { return bar_base + 8u * (6 + ATC_DQ_NST + s); };
  auto sdp_full = [&](int s) { return bar_base + 8u * (6 + 2 * ATC_DQ_NST + s); };
  auto ds_full = [&](int s) { return bar_base + 8u * (6 + ATC_DQ_NB + 2 * ATC_DQ_NST + s); };
  auto item_bar = [&](int s) { return bar_base + 8u * (6 + 2 * ATC_DQ_NB + 2 * ATC_DQ_NST + s); };
  const uint32_t item_slots = bar_base + 8u * (6 + 2 * ATC_DQ_NB + 2 * ATC_DQ_NST + ATC_ITEM_RING);
  const uint32_t tmem_slot = item_slots + 4u * ATC_ITEM_RING;
  uint32_t* tmem_slot_ptr = reinterpret_cast<uint32_t*>(smem_raw + (tmem_slot - smem_u32(smem_raw)));
  volatile uint32_t* item_slot_ptr = reinterpret_cast<volatile uint32_t*>(smem_raw + (item_slots - smem_u32(smem_raw)));

  const int warp = warp_idx_uniform(), lane = threadIdx.x & 31;
  const int nqb = (p.S + 127) / 128;
  const uint32_t nitems = static_cast<uint32_t>(nqb * p.nq * p.B);
  unsigned int* const sched = p.sched + 4;

  if (threadIdx.x == 0) {
    tma_prefetch_desc(&maps.q); tma_prefetch_desc(&maps.k); tma_prefetch_desc(&maps.v); tma_prefetch_desc(&maps.dO);
    tma_prefetch_desc(&maps.g32[0]); tma_prefetch_desc(&maps.g16[0]);
    mbar_init(qdo_full(), 1); mbar_init(acc_full(), 1); mbar_init(qdo_empty(), 8); mbar_init(acc_free(), 8);
    mbar_init(qa_full(), 8); mbar_init(qa_free(), 1);
    for (int i = 0; i < ATC_DQ_NST; ++i) { mbar_init(kv_full(i), 1); mbar_init(kv_empty(i), 1); }
    for (int i = 0; i < ATC_DQ_NB; ++i) { mbar_init(sdp_full(i), 1); mbar_init(ds_full(i), 8); }
    for (int i = 0; i < ATC_ITEM_RING; ++i) mbar_init(item_bar(i), 1);
    fence_barrier_init();
  }
  if (warp == 1) { tmem_alloc(tmem_slot, 512); tmem_relinquish(); }
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tmem_base = *tmem_slot_ptr;
  pdl_wait();                                    // no global access above (programmatic dependent launch, ptx.cuh)
  pdl_trigger();

  auto get_item = [&](uint32_t it) -> uint32_t {
    mbar_wait(item_bar(it % ATC_ITEM_RING), (it / ATC_ITEM_RING) & 1u);
    return item_slot_ptr[it % ATC_ITEM_RING];
  };

  if (warp == 0) {
    // ===================================================================== scheduler + TMA producer
    if (lane == 0) {
      auto publish = [&](uint32_t it, uint32_t item) {
        item_slot_ptr[it % ATC_ITEM_RING] = item;
        mbar_arrive(item_bar(it % ATC_ITEM_RING));
      };
      uint32_t g = 0;                                            // K/V blocks loaded so far (ring position)
      uint32_t item = atomicAdd(sched, 1u);
      publish(0, item);
      for (uint32_t it = 0; item < nitems; ++it) {
        const AttnDqItem w = attn_dq_item(item, p, nqb, doc_start);
        mbar_wait(qdo_empty(), (it & 1u) ^ 1u);                  // the previous item's Q, dO have been copied to TMEM
        mbar_expect_tx(qdo_full(), 2 * ATC_TILE_BYTES);
        tma_load_3d(sQ, &maps.q, qdo_full(), w.h * ATC_D, w.q0, w.b);
        tma_load_3d(sQ + ATC_CHUNK_BYTES, &maps.q, qdo_full(), w.h * ATC_D + 64, w.q0, w.b);
        tma_load_3d(sDO, &maps.dO, qdo_full(), w.h * ATC_D, w.q0, w.b);
        tma_load_3d(sDO + ATC_CHUNK_BYTES, &maps.dO, qdo_full(), w.h * ATC_D + 64, w.q0, w.b);
        const uint32_t next = atomicAdd(sched, 1u);              // latency hidden behind this item's K/V stream
        for (int j = 0; j < w.iters; ++j, ++g) {
          const int st = g % ATC_DQ_NST;
          mbar_wait(kv_empty(st), ((g / ATC_DQ_NST) & 1u) ^ 1u);
          mbar_expect_tx(kv_full(st), 2 * ATC_HALF_TILE);
          tma_load_3d(sK + st * ATC_HALF_TILE, &maps.k, kv_full(st), w.kvh * ATC_D, (w.j0 + j) * 64, w.b);
          tma_load_3d(sK + st * ATC_HALF_TILE + 64 * 128, &maps.k, kv_full(st), w.kvh * ATC_D + 64, (w.j0 + j) * 64, w.b);
          tma_load_3d(sV + st * ATC_HALF_TILE, &maps.v, kv_full(st), w.kvh * ATC_D, (w.j0 + j) * 64, w.b);
          tma_load_3d(sV + st * ATC_HALF_TILE + 64 * 128, &maps.v, kv_full(st), w.kvh * ATC_D + 64, (w.j0 + j) * 64, w.b);
        }
        publish(it + 1, next);
        item = next;
      }
      __threadfence();
      if (atomicAdd(sched + 1, 1u) == gridDim.x - 1) { sched[0] = 0; sched[1] = 0; __threadfence(); }
    }
  } else if (warp == 1) {
    // ===================================================================== MMA issuer (whole warp, elected lane issues)
    const uint32_t leader = elect_one();
    const uint32_t idesc_sdp = umma_idesc(128, 64, 0, 0, 0, 0);     // [128 queries x 64 keys], A from TMEM
    const uint32_t idesc_acc = umma_idesc(128, 128, 0, 0, 0, 1);    // dQ [128 x 128] += dS(TMEM) K(MN-major)
    const uint64_t dKk = umma_smem_desc(sK, 16, 1024), dVk = umma_smem_desc(sV, 16, 1024);
    const uint64_t dKm = umma_smem_desc(sK, 64 * 128, 1024);
    auto issue_sdp = [&](uint32_t g, bool wait_kv) {                 // g: global block index (ring positions)
      const int st = g % ATC_DQ_NST, buf = g % ATC_DQ_NB;
      if (wait_kv) { mbar_wait(kv_full(st), (g / ATC_DQ_NST) & 1u); tc_fence_after(); }
      if (leader) {
        const uint64_t ka = desc_adv(dKk, st * ATC_HALF_TILE), va = desc_adv(dVk, st * ATC_HALF_TILE);
#pragma unroll
        for (int kk = 0; kk < 8; ++kk) {                              // two independent accumulation chains, interleaved
          umma_f16_ts(tmem_base + ATC_DQ_S + buf * 64, tmem_base + ATC_DQ_QA + kk * 8,
                      desc_adv(ka, (kk >> 2) * (64 * 128) + (kk & 3) * 32), idesc_sdp, kk != 0 ? 1u : 0u);
          umma_f16_ts(tmem_base + ATC_DQ_DP + buf * 64, tmem_base + ATC_DQ_DOA + kk * 8,
                      desc_adv(va, (kk >> 2) * (64 * 128) + (kk & 3) * 32), idesc_sdp, kk != 0 ? 1u : 0u);
        }
        umma_commit(sdp_full(buf));
      }
    };
    uint32_t g0 = 0;                                                 // global index of this item's block 0
    for (uint32_t it = 0;; ++it) {
      const uint32_t item = get_item(it);
      if (item >= nitems) break;
      const AttnDqItem w = attn_dq_item(item, p, nqb, doc_start);
      const int iters = w.iters;
      mbar_wait(qa_full(), it & 1u);                                 // Q, dO operands of this item are in TMEM
      tc_fence_after();
      issue_sdp(g0, true);
      if (iters > 1) issue_sdp(g0 + 1, true);
      if (iters <= 2 && leader) umma_commit(qa_free());              // those were the item's last S / dP MMAs
      for (int j = 0; j < iters; ++j) {
        const uint32_t g = g0 + j;
        const int st = g % ATC_DQ_NST, buf = g % ATC_DQ_NB;
        // (polling kv_full of block g + 2 together with ds_full here was measured: it holds dQ(g) back whenever that tile
        // is still in flight -- 0.88 instead of 0.82 ms; the K / V wait stays behind the dQ issue)
        mbar_wait(ds_full(buf), (g / ATC_DQ_NB) & 1u);
        if (lane == 0) ATC_TR3(g, 24);
        if (j == 0 && it > 0) mbar_wait(acc_free(), (it - 1u) & 1u); // the previous item's dQ has been read out
        tc_fence_after();
        if (leader) {
          const uint64_t ka = desc_adv(dKm, st * ATC_HALF_TILE);
#pragma unroll
          for (int kk = 0; kk < 4; ++kk)
            umma_f16_ts(tmem_base + ATC_DQ_ACC, tmem_base + ATC_DQ_S + buf * 64 + atc_half_operand_col(kk), desc_adv(ka, kk * 2048),
                        idesc_acc, (j | kk) != 0 ? 1u : 0u);
          if (w.split) {                                // early query rows: + dS_lo K
#pragma unroll
            for (int kk = 0; kk < 4; ++kk)
              umma_f16_ts(tmem_base + ATC_DQ_ACC, tmem_base + ATC_DQ_S + buf * 64 + 16 + atc_half_operand_col(kk),
                          desc_adv(ka, kk * 2048), idesc_acc, 1u);
          }
          umma_commit(kv_empty(st));
        }
        if (lane == 0) ATC_TR3(g, 25);
        if (j + 2 < iters) {                                         // this block's S / dP buffers are free again (in-order issue)
          issue_sdp(g + 2, true);
          if (lane == 0) ATC_TR3(g, 26);
          if (j + 3 == iters && leader) umma_commit(qa_free());
        }
      }
      if (leader) umma_commit(acc_full());
      g0 += iters;
    }
  } else {
    // ===================================================================== softmax warps: TMEM lane quarter x column half
    const int quarter = warp & 3, half = (warp - 2) >> 2;
    const int row = quarter * 32 + lane;
    const uint32_t lane_off = static_cast<uint32_t>(quarter * 32) << 16;
    const int col0 = half * 32;
    const float c = p.scale_log2;
    const WarpStage wst{stage_tiles + static_cast<uint32_t>(warp - 2) * GEMM_STAGE_TILE_BYTES, lane};
    uint32_t g = 0;                                                  // global block index
    // Q, dO of item `k`: this warp copies its 32 rows x its 64-column chunk of both TMA-landed tiles to the TMEM operand
    // columns, then releases the shared-memory tiles to the producer.  Done for item k + 1 right after the LAST dS of
    // item k has been handed over and BEFORE item k's epilogue, so that the MMA warp finds the next operands ready when
    // it has issued item k's last dQ: no tensor bubble between items.
    auto copy_in = [&](uint32_t k) {
      mbar_wait(qdo_full(), k & 1u);
      if (k > 0) mbar_wait(qa_free(), (k - 1u) & 1u);                // the previous item's S / dP MMAs have read the operands
      tc_fence_after();
      atc_row_chunk_to_tmem(sQ + half * ATC_CHUNK_BYTES, row, tmem_base + lane_off + ATC_DQ_QA + half * 32);
      atc_row_chunk_to_tmem(sDO + half * ATC_CHUNK_BYTES, row, tmem_base + lane_off + ATC_DQ_DOA + half * 32);
      tmem_st_wait();
      tc_fence_before();
      __syncwarp();
      if (lane == 0) { mbar_arrive(qa_full()); mbar_arrive(qdo_empty()); }
    };
    uint32_t item = get_item(0);
    if (item < nitems) copy_in(0);
    for (uint32_t it = 0; item < nitems; ++it) {
      const AttnDqItem w = attn_dq_item(item, p, nqb, doc_start);
      const int q0 = w.q0, qi = q0 + row;
      const bool valid = qi < p.S;
      const long long vidx = (static_cast<long long>(w.b) * p.nq + w.h) * p.S + qi;
      const float L2 = valid ? p.lse[vidx] * 1.4426950408889634f : INFINITY;
      const float4 d4 = valid ? __ldg(reinterpret_cast<const float4*>(p.dvec) + vidx) : make_float4(0.f, 0.f, 0.f, 0.f);
      const float Dr = (d4.x + d4.y) + (d4.z + d4.w);
      const int dstart = doc_start ? doc_start[min(qi, p.S - 1)] : 0;      // first key this query may see
      for (int j = 0; j < w.iters; ++j, ++g) {
        const int buf = g % ATC_DQ_NB;
        mbar_wait(sdp_full(buf), (g / ATC_DQ_NB) & 1u);
        const bool tr = quarter == 0 && half == 0 && lane == 0;
        if (tr) ATC_TR3(g, 8);
        tc_fence_after();
        uint32_t sr[32], dr[32];
        tmem_ld32(tmem_base + lane_off + ATC_DQ_S + buf * 64 + col0, sr);
        tmem_ld32(tmem_base + lane_off + ATC_DQ_DP + buf * 64 + col0, dr);
        tmem_ld_wait();
        float ds[32];
#pragma unroll
        for (int i = 0; i < 32; ++i)
          ds[i] = ex2_approx(fmaf(__uint_as_float(sr[i]), c, -L2)) * (__uint_as_float(dr[i]) - Dr);
        if ((w.j0 + j) * 64 + 63 > q0) {                             // diagonal blocks: key > query is masked
          const int krel = (w.j0 + j) * 64 + col0 - q0;
#pragma unroll
          for (int i = 0; i < 32; ++i)
            if (krel + i > row) ds[i] = 0.f;
        }
        if (DOC && __any_sync(0xffffffffu, (w.j0 + j) * 64 + col0 < dstart)) {   // packed sequences: keys of earlier sequences
          const int kabs = (w.j0 + j) * 64 + col0;
#pragma unroll
          for (int i = 0; i < 32; ++i)
            if (kabs + i < dstart) ds[i] = 0.f;
        }
        uint32_t pk[16];
        if (w.split) {
          uint32_t pl[16];
#pragma unroll
          for (int i = 0; i < 16; ++i) atc_split_pack(ds[2 * i], ds[2 * i + 1], pk[i], pl[i]);
          tmem_st16(tmem_base + lane_off + ATC_DQ_S + buf * 64 + col0 + 16, pl);
        } else {
#pragma unroll
          for (int i = 0; i < 16; ++i) pk[i] = pack_f16(ds[2 * i], ds[2 * i + 1]);
        }
        tmem_st16(tmem_base + lane_off + ATC_DQ_S + buf * 64 + col0, pk);
        tmem_st_wait();
        tc_fence_before();
        __syncwarp();
        if (lane == 0) mbar_arrive(ds_full(buf));
        if (tr) ATC_TR3(g, 9);
      }
      const uint32_t next = get_item(it + 1);
      if (next < nitems) copy_in(it + 1);
      // epilogue: this warp stores rows [32 quarter, +32), columns [64 half, +64) of dQ, then releases the accumulator
      mbar_wait(acc_full(), it & 1u);
      tc_fence_after();
      const int s0 = q0 + quarter * 32;
      uint32_t a0[32], a1[32];
      tmem_ld32(tmem_base + lane_off + ATC_DQ_ACC + half * 64, a0);
      tmem_ld32(tmem_base + lane_off + ATC_DQ_ACC + half * 64 + 32, a1);
      tmem_ld_wait();
      tc_fence_before();
      __syncwarp();
      if (lane == 0) mbar_arrive(acc_free());
      if (s0 < p.S) {
        const float2* rr = (p.rope && valid) ? p.rope + static_cast<long long>(qi - dstart) * 64 + half * 32 : nullptr;
        atc_store_grad32(wst, reinterpret_cast<float(&)[32]>(a0), p.scale, rr, p.dq32 ? &maps.g32[0] : nullptr,
                         p.dq16 ? &maps.g16[0] : nullptr, w.h * ATC_D + half * 64, s0, w.b);
        atc_store_grad32(wst, reinterpret_cast<float(&)[32]>(a1), p.scale, rr ? rr + 16 : nullptr, p.dq32 ? &maps.g32[0] : nullptr,
                         p.dq16 ? &maps.g16[0] : nullptr, w.h * ATC_D + half * 64 + 32, s0, w.b);
      }
      item = next;
    }
    if (lane == 0) tma_store_wait_all<0>();
  }

  tc_fence_before();
  __syncthreads();
  if (warp == 1) { tc_fence_after(); tmem_dealloc(tmem_base, 512); }
}

inline cudaError_t attn_bwd_tc_set_attrs() {
  static DeviceOnce once;
  if (once.need()) {
    cudaError_t e = cudaFuncSetAttribute(attn_bwd_dkdv_tc_kernel<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, ATC_BWD_SMEM);
    if (e != cudaSuccess) return e;
    e = cudaFuncSetAttribute(attn_bwd_dkdv_tc_kernel<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, ATC_BWD_SMEM);
    if (e != cudaSuccess) return e;
    e = cudaFuncSetAttribute(attn_bwd_dq_tc_kernel<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, ATC_DQ_SMEM);
    if (e != cudaSuccess) return e;
    e = cudaFuncSetAttribute(attn_bwd_dq_tc_kernel<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, ATC_DQ_SMEM);
    if (e != cudaSuccess) return e;
    once.done();
  }
  return cudaSuccess;
}

// dK/dV: K, V and the streamed Q, dO all as 128-row tiles
inline cudaError_t attn_bwd_dkdv_tc_launch(const __half* q, long long ldq, const __half* k, long long ldk, const __half* v,
                                           long long ldv, const __half* dO, long long lddo, const AttnTcBwdParams& p,
                                           cudaStream_t st) {
  cudaError_t e = attn_bwd_tc_set_attrs();
  if (e != cudaSuccess) return e;
  AttnTcMaps m1;
  if (!make_map_attn(&m1.k, k, p.nkv * ATC_D, p.S, p.B, ldk, 128) || !make_map_attn(&m1.v, v, p.nkv * ATC_D, p.S, p.B, ldv, 128) ||
      !make_map_attn(&m1.q, q, p.nq * ATC_D, p.S, p.B, ldq, 128) || !make_map_attn(&m1.dO, dO, p.nq * ATC_D, p.S, p.B, lddo, 128))
    return cudaErrorInvalidValue;
  m1.o32 = m1.o16 = m1.q; m1.g32[0] = m1.g32[1] = m1.g16[0] = m1.g16[1] = m1.q;
  if ((p.dv32 && !make_map_store(&m1.g32[0], p.dv32, p.nkv * ATC_D, p.S, p.B, p.lddk32, true)) ||
      (p.dk32 && !make_map_store(&m1.g32[1], p.dk32, p.nkv * ATC_D, p.S, p.B, p.lddk32, true)) ||
      (p.dv16 && !make_map_store(&m1.g16[0], p.dv16, p.nkv * ATC_D, p.S, p.B, p.ldd16, false)) ||
      (p.dk16 && !make_map_store(&m1.g16[1], p.dk16, p.nkv * ATC_D, p.S, p.B, p.ldd16, false)))
    return cudaErrorInvalidValue;
  dim3 g1(((p.S + 127) / 128) * p.nkv * p.B, 1, 1);
  if (p.doc_start) return launch_kernel(attn_bwd_dkdv_tc_kernel<true>, g1, dim3(ATC_BWD_THREADS), ATC_BWD_SMEM, st, m1, p);
  return launch_kernel(attn_bwd_dkdv_tc_kernel<false>, g1, dim3(ATC_BWD_THREADS), ATC_BWD_SMEM, st, m1, p);
}

// dQ: Q, dO as 128-row tiles; K, V streamed as 64-row tiles
inline cudaError_t attn_bwd_dq_tc_launch(const __half* q, long long ldq, const __half* k, long long ldk, const __half* v,
                                         long long ldv, const __half* dO, long long lddo, const AttnTcBwdParams& p,
                                         int num_sms, cudaStream_t st) {
  cudaError_t e = attn_bwd_tc_set_attrs();
  if (e != cudaSuccess) return e;
  AttnTcMaps m2;
  if (!make_map_attn(&m2.k, k, p.nkv * ATC_D, p.S, p.B, ldk, 64) || !make_map_attn(&m2.v, v, p.nkv * ATC_D, p.S, p.B, ldv, 64) ||
      !make_map_attn(&m2.q, q, p.nq * ATC_D, p.S, p.B, ldq, 128) || !make_map_attn(&m2.dO, dO, p.nq * ATC_D, p.S, p.B, lddo, 128))
    return cudaErrorInvalidValue;
  m2.o32 = m2.o16 = m2.q; m2.g32[0] = m2.g32[1] = m2.g16[0] = m2.g16[1] = m2.q;
  if ((p.dq32 && !make_map_store(&m2.g32[0], p.dq32, p.nq * ATC_D, p.S, p.B, p.lddq32, true)) ||
      (p.dq16 && !make_map_store(&m2.g16[0], p.dq16, p.nq * ATC_D, p.S, p.B, p.ldd16, false)))
    return cudaErrorInvalidValue;
  const int nitems = ((p.S + 127) / 128) * p.nq * p.B;
  const int grid = nitems < num_sms ? nitems : num_sms;        // persistent: one CTA per SM
  if (p.doc_start) return launch_kernel(attn_bwd_dq_tc_kernel<true>, dim3(grid), dim3(ATC_BWD_THREADS), ATC_DQ_SMEM, st, m2, p);
  return launch_kernel(attn_bwd_dq_tc_kernel<false>, dim3(grid), dim3(ATC_BWD_THREADS), ATC_DQ_SMEM, st, m2, p);
}

}  // namespace lsp
