// te_gemm8.cuh — block-scaled FP8 (OCP MXFP8) GEMM for sm_100a (DESIGN.md §3 Q24-Q27, §10):
//   D[M,N] = A[M,K] * B[N,K]^T with A, B = E4M3 elements + one E8M0 scale per 32 consecutive K elements,
//   tcgen05.mma.kind::mxf8f6f4.block_scale (cta_group::2, M = 256 per CTA pair), fp32 accumulators in TMEM.
//
// Same warp roles and pipeline as te_gemm2_kernel (te_gemm.cuh): TMA producer (128 B = 128-element swizzled rows of
// A and B), single-thread MMA issuer in the leader CTA, 8 epilogue warps.  New here:
//   * scale factors.  Global layout (both operands): per 128-row block and 128-element K chunk one 512-byte tile in
//     the order the tensor core's scale-factor copy expects: byte (r % 32) * 16 + ((r / 32) % 4) * 4 + kb holds the
//     scale of row r, 32-element block kb of the chunk.  A stage's tiles (1 for this CTA's 128 A rows, BN/128 for
//     ALL BN weight rows — both CTAs of the pair need the whole B scale set) arrive by TMA (the scale buffers are
//     [tiles, 128] uint32 tensors, one row per tile; cta_group::2 loads so that the peer CTA's copies also complete
//     on the leader's full barrier); the MMA thread moves them smem -> TMEM with tcgen05.cp (32x128b.warpx4: 4 columns per
//     tile, replicated over the four lane quadrants) right ahead of the stage's four K = 32 MMAs, whose instruction
//     descriptors select byte kb (a_sf_id / b_sf_id).  Two alternating TMEM scale sets keep copy and MMA overlapped.
//   * quantising epilogues: the A operand of the NEXT GEMM (x*g, silu(gate)*up) is written as E4M3 with its block
//     scales straight from the fp32 values (a 32-column chunk of a row is exactly one MX block), so the block-scaled
//     path needs no extra pass over the activations.
// TMEM budget (512 columns): ACC accumulator stages x BN columns + 2 x (4 + 4 * ceil(BN / 128)) scale columns:
//   BN = 128 -> three accumulator stages, BN = 192 -> two (the epilogue overlaps the next tiles), BN = 256 -> one.
#pragma once
#include "te_gemm.cuh"

namespace te {

// ------------------------------------------------------------------ MXFP8 quantiser (device side of Q25)
// E8M0 code of a block: the smallest power of two X = 2^(code-127) with amax / X <= 448 (= 1.75 * 2^8).
__device__ __forceinline__ uint32_t mx_scale_code(float amax) {
  const uint32_t b = __float_as_uint(amax);
  const int code = static_cast<int>((b >> 23) & 0xFFu) - 8 + ((b & 0x7FFFFFu) > 0x600000u ? 1 : 0);
  return static_cast<uint32_t>(min(max(code, 0), 254));
}
__device__ __forceinline__ float mx_inv_scale(uint32_t code) {  // 1 / X = 2^(127 - code), exact
  return __uint_as_float((254u - code) << 23);
}
// four fp32 -> four E4M3 bytes (round to nearest even, memory order v0 v1 v2 v3 from the low byte)
__device__ __forceinline__ uint32_t pack_e4m3x4(float v0, float v1, float v2, float v3) {
  uint16_t lo, hi;
  asm("cvt.rn.satfinite.e4m3x2.f32 %0, %1, %2;" : "=h"(lo) : "f"(v1), "f"(v0));
  asm("cvt.rn.satfinite.e4m3x2.f32 %0, %1, %2;" : "=h"(hi) : "f"(v3), "f"(v2));
  return static_cast<uint32_t>(lo) | (static_cast<uint32_t>(hi) << 16);
}
// byte offset of the scale of (row r, 32-element block kb32) in the tiled scale layout of a [rows, K] operand
__device__ __forceinline__ size_t mx_sf_offset(int r, int kb32, int k_chunks) {
  return (static_cast<size_t>(r >> 7) * k_chunks + (kb32 >> 2)) * 512 + (r & 31) * 16 + ((r >> 5) & 3) * 4 + (kb32 & 3);
}
// the same for a weight matrix whose scale tiles are grouped by the consuming GEMM's N tile of `tile_rows` rows
// (tile n_blk owns ceil(tile_rows / 128) consecutive 128-row scale tiles; equal to mx_sf_offset when tile_rows % 128 == 0)
__device__ __forceinline__ size_t mx_sf_offset_tiled(int r, int kb32, int k_chunks, int tile_rows) {
  const int n_blk = r / tile_rows, rl = r - n_blk * tile_rows;
  const int rb = n_blk * ((tile_rows + 127) >> 7) + (rl >> 7);
  return (static_cast<size_t>(rb) * k_chunks + (kb32 >> 2)) * 512 + (rl & 31) * 16 + ((rl >> 5) & 3) * 4 + (kb32 & 3);
}

// One thread quantises one 32-element block held in registers: 32 bytes + 1 scale byte.
__device__ __forceinline__ void mx_store_block(const float (&v)[32], uint8_t* dst32, uint8_t* sf_dst) {
  float amax = 0.f;
#pragma unroll
  for (int j = 0; j < 32; ++j) amax = fmaxf(amax, fabsf(v[j]));
  const uint32_t code = mx_scale_code(amax);
  const float inv = mx_inv_scale(code);
  uint32_t w[8];
#pragma unroll
  for (int j = 0; j < 8; ++j) w[j] = pack_e4m3x4(v[4 * j] * inv, v[4 * j + 1] * inv, v[4 * j + 2] * inv, v[4 * j + 3] * inv);
  reinterpret_cast<uint4*>(dst32)[0] = make_uint4(w[0], w[1], w[2], w[3]);
  reinterpret_cast<uint4*>(dst32)[1] = make_uint4(w[4], w[5], w[6], w[7]);
  *sf_dst = static_cast<uint8_t>(code);
}

// te_load_weights / te_debug: bf16 [rows, K] -> E4M3 [rows, K] + tiled scales.  One thread per 32-element block.
// gu_src_tile > 0: `src` is the gate/up matrix interleaved per gu_src_tile rows (first half gate, second half the
// matching up rows) and the destination is interleaved per tile_rows rows instead (the MXFP8 gate/up GEMM has its own
// tile width): destination row r of tile n (rl = r % tile_rows) is gate column n * tile_rows/2 + rl, or up column
// n * tile_rows/2 + rl - tile_rows/2.
__global__ void te_mx_quantise_bf16_kernel(const __nv_bfloat16* __restrict__ src, uint8_t* __restrict__ dst,
                                           uint8_t* __restrict__ sf, int rows, int K, int tile_rows, int gu_src_tile) {
  const int kb_per_row = K / 32;
  const long long idx = static_cast<long long>(blockIdx.x) * blockDim.x + threadIdx.x;
  if (idx >= static_cast<long long>(rows) * kb_per_row) return;
  const int r = static_cast<int>(idx / kb_per_row), kb = static_cast<int>(idx % kb_per_row);
  int r_src = r;
  if (gu_src_tile > 0) {
    const int half = tile_rows / 2, n = r / tile_rows, rl = r - n * tile_rows;
    const int col = n * half + (rl < half ? rl : rl - half);  // column of F
    const int sh = gu_src_tile / 2;
    r_src = (col / sh) * gu_src_tile + col % sh + (rl < half ? 0 : sh);
  }
  const uint4* s4 = reinterpret_cast<const uint4*>(src + static_cast<size_t>(r_src) * K + kb * 32);
  float v[32];
#pragma unroll
  for (int q = 0; q < 4; ++q) {
    const uint4 u = __ldg(s4 + q);
    const uint32_t w[4] = {u.x, u.y, u.z, u.w};
#pragma unroll
    for (int e = 0; e < 4; ++e) {
      v[8 * q + 2 * e] = bf16_lo(w[e]);
      v[8 * q + 2 * e + 1] = bf16_hi(w[e]);
    }
  }
  mx_store_block(v, dst + static_cast<size_t>(r) * K + kb * 32, sf + mx_sf_offset_tiled(r, kb, K / 128, tile_rows));
}

// MXFP4 (reading Q32): bf16 [rows, K] -> packed E2M1 [rows, K/2] (element 2i in the low nibble of byte i) + tiled E8M0
// scales in the same layout as the MXFP8 weights.  Scale = smallest power of two X with amax / X <= 6; elements
// round to nearest, ties to the even code, written as explicit comparisons against the seven midpoints of the grid
// 0, 0.5, 1, 1.5, 2, 3, 4, 6 (v / X is exact).  One thread per 32-element block.  gu_src_tile as in the MXFP8 quantiser.
__device__ __forceinline__ uint32_t e2m1_code(float v) {
  const float a = fabsf(v);
  const uint32_t c = (a > 0.25f) + (a >= 0.75f) + (a > 1.25f) + (a >= 1.75f) + (a > 2.5f) + (a >= 3.5f) + (a > 5.0f);
  return c | (v < 0.f ? 8u : 0u);
}
__global__ void te_mx_quantise_fp4_kernel(const __nv_bfloat16* __restrict__ src, uint8_t* __restrict__ dst,
                                          uint8_t* __restrict__ sf, int rows, int K, int tile_rows, int gu_src_tile) {
  const int kb_per_row = K / 32;
  const long long idx = static_cast<long long>(blockIdx.x) * blockDim.x + threadIdx.x;
  if (idx >= static_cast<long long>(rows) * kb_per_row) return;
  const int r = static_cast<int>(idx / kb_per_row), kb = static_cast<int>(idx % kb_per_row);
  int r_src = r;
  if (gu_src_tile > 0) {
    const int half = tile_rows / 2, n = r / tile_rows, rl = r - n * tile_rows;
    const int col = n * half + (rl < half ? rl : rl - half);
    const int sh = gu_src_tile / 2;
    r_src = (col / sh) * gu_src_tile + col % sh + (rl < half ? 0 : sh);
  }
  const uint4* s4 = reinterpret_cast<const uint4*>(src + static_cast<size_t>(r_src) * K + kb * 32);
  float v[32];
  float amax = 0.f;
#pragma unroll
  for (int q = 0; q < 4; ++q) {
    const uint4 u = __ldg(s4 + q);
    const uint32_t w[4] = {u.x, u.y, u.z, u.w};
#pragma unroll
    for (int e = 0; e < 4; ++e) {
      v[8 * q + 2 * e] = bf16_lo(w[e]);
      v[8 * q + 2 * e + 1] = bf16_hi(w[e]);
    }
  }
#pragma unroll
  for (int j = 0; j < 32; ++j) amax = fmaxf(amax, fabsf(v[j]));
  const uint32_t b = __float_as_uint(amax);
  int code = static_cast<int>((b >> 23) & 0xFFu) - 2 + ((b & 0x7FFFFFu) > 0x400000u ? 1 : 0);
  code = min(max(code, 0), 254);
  const float inv = mx_inv_scale(static_cast<uint32_t>(code));
  uint32_t w4[4];
#pragma unroll
  for (int q = 0; q < 4; ++q) {
    uint32_t acc = 0;
#pragma unroll
    for (int e = 0; e < 8; ++e) acc |= e2m1_code(v[8 * q + e] * inv) << (4 * e);
    w4[q] = acc;
  }
  *reinterpret_cast<uint4*>(dst + static_cast<size_t>(r) * (K / 2) + kb * 16) = make_uint4(w4[0], w4[1], w4[2], w4[3]);
  sf[mx_sf_offset_tiled(r, kb, K / 128, tile_rows)] = static_cast<uint8_t>(code);
}

// ------------------------------------------------------------------ PTX wrappers
// D[tmem of both CTAs] (+)= (A * SFA) * (B * SFB)^T, MXFP8, M = 256 over the pair.  ONE thread of the leader.
__device__ __forceinline__ void umma_mxf8_cg2(uint32_t d_tmem, uint64_t a_desc, uint64_t b_desc, uint32_t idesc,
                                              uint32_t sfa_tmem, uint32_t sfb_tmem, uint32_t accumulate) {
  asm volatile(
      "{\n\t.reg .pred P;\n\t"
      "setp.ne.b32 P, %4, 0;\n\t"
      "tcgen05.mma.cta_group::2.kind::mxf8f6f4.block_scale [%0], %1, %2, %3, [%5], [%6], P;\n\t}" ::"r"(d_tmem),
      "l"(a_desc), "l"(b_desc), "r"(idesc), "r"(accumulate), "r"(sfa_tmem), "r"(sfb_tmem)
      : "memory");
}
// smem -> TMEM copy of one 512-byte scale tile (32 rows x 16 B, replicated to the four 32-lane quadrants), performed
// in BOTH CTAs of the pair, each from its own shared memory at the same offset.  ONE thread of the leader.
__device__ __forceinline__ void tmem_cp_sf_cg2(uint32_t taddr, uint64_t s_desc) {
  asm volatile("tcgen05.cp.cta_group::2.32x128b.warpx4 [%0], %1;" ::"r"(taddr), "l"(s_desc) : "memory");
}
// descriptor of a scale tile: no swizzle, 8-row x 16-byte atoms 128 B apart (SBO), one atom along K (LBO unused)
__device__ __forceinline__ uint64_t umma_smem_desc_sf(uint32_t smem_addr) {
  uint64_t d = 0;
  d |= static_cast<uint64_t>((smem_addr & 0x3FFFFu) >> 4);
  d |= static_cast<uint64_t>(128 >> 4) << 32;  // SBO
  d |= static_cast<uint64_t>(1) << 46;         // descriptor version (sm_100)
  return d;                                    // layout type 0 = no swizzle
}
// Instruction descriptor, kind::mxf8f6f4: A = B = E4M3 (format 0), both K-major, E8M0 scales, dense.
__host__ __device__ constexpr uint32_t umma_idesc_mxf8(uint32_t m, uint32_t n) {
  return ((n >> 3) << 17) | (1u << 23) | ((m >> 4) << 24);
}
__device__ __forceinline__ uint32_t umma_idesc_with_sf(uint32_t idesc, uint32_t sf_id) {
  return idesc | (sf_id << 4) | (sf_id << 29);  // b_sf_id [4,6), a_sf_id [29,31): byte of the 4-byte scale word
}

constexpr int GEMM8_BK = 128;  // E4M3 elements per 128-byte swizzled row = one scale tile (4 blocks of 32)

// Operands of the block-scaled GEMM that te_gemm.cuh's GemmParams does not carry.
struct Gemm8Extra {
  // quantising epilogues: E4M3 destination (xg8 or act8), its tiled scales, its K / 128
  uint8_t* q_out;
  uint8_t* q_sf;
  int q_kchunks;
  int q_ld;
  // MXFP4 weights (te_config.weight_dtype = 2): the B operand's elements are FP4 E2M1.  In shared memory they sit in the
  // same 128-byte swizzled rows of 128 elements as E4M3 (the tensor map type 16U4_ALIGN16B unpacks 16 nibbles into every
  // 16-byte chunk: 8 bytes of data, 8 bytes of gap), so only the instruction descriptor's B format changes.
  int b_fp4;
};
constexpr uint32_t UMMA_F8F6F4_E2M1 = 5u;  // element format code of kind::mxf8f6f4 / f8f6f4 operands (E4M3 = 0)

template <int BN, int EPI>
struct Gemm8Cfg {
  // accumulator stages: three for 128-wide tiles (3 x 128 + scale columns <= 512): main loop (16-48 k-blocks of K = 128)
  // and epilogue take about as long as each other there, and a third stage keeps either from waiting on the other's jitter
#ifndef TE_ACC128
#define TE_ACC128 3
#endif
  static constexpr int ACC = (BN <= 128) ? TE_ACC128 : ((BN <= 192) ? 2 : 1);
  static constexpr int SFB_TILES = (BN + 127) / 128;
  static constexpr int A_BYTES = GEMM_BM * GEMM8_BK;
  static constexpr int B_BYTES = (BN / 2) * GEMM8_BK;
  static constexpr int SFA_BYTES = 512;
  static constexpr int SFB_BYTES = SFB_TILES * 512;
  static constexpr int STAGE_BYTES = A_BYTES + B_BYTES + SFA_BYTES + SFB_BYTES;
  static constexpr int BAR_BYTES = 256;
  static constexpr int STG_WARP_BYTES = (EPI == EPI_QKV ? 2 : 1) * 32 * 32 * 4;
  // epilogue warps: with the MMA twice as fast as in bf16 the kernels are epilogue-bound (ncu r02a: tensor pipe 25-69 %
  // active), so the 192-wide SwiGLU tile (3 MX blocks per row and half) gets three warps per TMEM lane quadrant
  static constexpr int EPI_WARPS = (EPI == EPI_SWIGLU && BN == 192) ? 12 : GEMM2_EPI_WARPS;
  static constexpr int THREADS = 64 + 32 * EPI_WARPS;
  static constexpr int STG_BYTES = (EPI == EPI_SWIGLU || EPI == EPI_PLAIN) ? 0 : EPI_WARPS * STG_WARP_BYTES;
  static constexpr int SMEM_LIMIT = 232448;
  static constexpr int STAGES_FIT = (SMEM_LIMIT - 1024 - BAR_BYTES - STG_BYTES) / STAGE_BYTES;
  static constexpr int STAGES = STAGES_FIT > 8 ? 8 : STAGES_FIT;
  static constexpr int SMEM_BYTES = STAGES * STAGE_BYTES + BAR_BYTES + STG_BYTES + 1024;
  static constexpr int SF_SET_COLS = 4 + 4 * SFB_TILES;
  static constexpr int SF_COL0 = ACC * BN;
  static constexpr int TMEM_COLS = 512;
  static_assert(SF_COL0 + 2 * SF_SET_COLS <= 512, "TMEM budget");
  static_assert(STAGES >= 3 && 2 * STAGES + 2 * ACC + 1 <= BAR_BYTES / 8, "pipeline configuration");
};

// ---------------------------------------------------------------- quantising epilogues (thread / lane domains)
// SwiGLU: y = rstd * acc; act = silu(gate) * up -> E4M3 + block scales.  Thread = row, 32-column chunk = one MX block.
template <int BN>
__device__ __forceinline__ void epi_swiglu8(const GemmParams& p, const Gemm8Extra& x8, int M, uint32_t t_row, int row,
                                            int n_blk, int part, int nparts, float rstd) {
  constexpr int HALF = BN / 2;
  static_assert(HALF % 32 == 0, "whole MX blocks per tile");
  // the tile's 32-column MX blocks are dealt round-robin to the `nparts` warps of a TMEM lane quadrant
#pragma unroll 1
  for (int c0 = part * 32; c0 < HALF; c0 += nparts * 32) {
    float a[32];
    {
      uint32_t g[32], u[32];
      tmem_ld32(t_row + c0, g);
      tmem_ld32(t_row + HALF + c0, u);
      tmem_ld_wait();
#pragma unroll
      for (int j = 0; j < 32; ++j) {
        const float gv = __uint_as_float(g[j]) * rstd;
        const float uv = __uint_as_float(u[j]) * rstd;
        a[j] = __fdividef(gv, 1.0f + __expf(-gv)) * uv;
      }
    }
    if (row < M) {
      const int col = n_blk * HALF + c0;
      mx_store_block(a, x8.q_out + static_cast<size_t>(row) * x8.q_ld + col, x8.q_sf + mx_sf_offset(row, col >> 5, x8.q_kchunks));
    }
  }
}

// Residual: x += acc (fp32), per-row partial sum of squares, and the next GEMM's A operand x * g_next as E4M3 +
// block scales.  Lane domain of epi_resid (8 lanes x 4 columns = one 32-column MX block of a row).
template <int BN>
__device__ __forceinline__ void epi_resid8(const GemmParams& p, const Gemm8Extra& x8, int M, uint32_t t_row, int row_base,
                                           int lane, int n_blk, float* stg, int part, int nparts, ResidPrefetch& pf) {
  const int sub = lane >> 3, cq = lane & 7;
  const bool has_g = p.g_next != nullptr;
  float* const x_dst = resid_dst(p);
  float ss[8];
#pragma unroll
  for (int i = 0; i < 8; ++i) ss[i] = 0.f;
  const int c_end = (part + 1) * (BN / nparts);
#pragma unroll 1
  for (int c0 = part * (BN / nparts); c0 < c_end; c0 += 32) {
    {
      uint32_t r[32];
      tmem_ld32(t_row + c0, r);
      tmem_ld_wait();
      float v[32];
#pragma unroll
      for (int j = 0; j < 32; ++j) v[j] = __uint_as_float(r[j]);
      stg_put_row(stg, lane, v);
    }
    __syncwarp();
    const int col = n_blk * BN + c0 + cq * 4;
    float g0 = 0.f, g1 = 0.f, g2 = 0.f, g3 = 0.f;
    if (has_g) {
      const uint2 g = __ldg(reinterpret_cast<const uint2*>(p.g_next + col));
      g0 = bf16_lo(g.x); g1 = bf16_hi(g.x); g2 = bf16_lo(g.y); g3 = bf16_hi(g.y);
    }
    float4 xv[8];
#pragma unroll
    for (int i = 0; i < 8; ++i) xv[i] = pf.xv[i];
    if (c0 + 32 < c_end) resid_issue<BN>(p, M, pf, row_base, lane, n_blk, c0 + 32);
#pragma unroll
    for (int i = 0; i < 8; ++i) {
      const int rr = sub + 4 * i;
      const int row = row_base + rr;
      const bool ok = row < M;   // (uniform over the 8 lanes of a row: the shuffles below stay converged)
      const float4 a = stg_get(stg, rr, cq);
      float4 v = ok ? xv[i] : make_float4(0.f, 0.f, 0.f, 0.f);
      v.x += a.x; v.y += a.y; v.z += a.z; v.w += a.w;
      if (ok) {
        *reinterpret_cast<float4*>(x_dst + (size_t)row * p.ld_x + col) = v;
        ss[i] = fmaf(v.x, v.x, ss[i]); ss[i] = fmaf(v.y, v.y, ss[i]);
        ss[i] = fmaf(v.z, v.z, ss[i]); ss[i] = fmaf(v.w, v.w, ss[i]);
      }
      if (has_g) {
        const float q0 = v.x * g0, q1 = v.y * g1, q2 = v.z * g2, q3 = v.w * g3;
        float amax = fmaxf(fmaxf(fabsf(q0), fabsf(q1)), fmaxf(fabsf(q2), fabsf(q3)));
        amax = fmaxf(amax, __shfl_xor_sync(0xffffffffu, amax, 1));
        amax = fmaxf(amax, __shfl_xor_sync(0xffffffffu, amax, 2));
        amax = fmaxf(amax, __shfl_xor_sync(0xffffffffu, amax, 4));
        if (ok) {
          const uint32_t code = mx_scale_code(amax);
          const float inv = mx_inv_scale(code);
          *reinterpret_cast<uint32_t*>(x8.q_out + (size_t)row * x8.q_ld + col) = pack_e4m3x4(q0 * inv, q1 * inv, q2 * inv, q3 * inv);
          if (cq == 0) x8.q_sf[mx_sf_offset(row, col >> 5, x8.q_kchunks)] = static_cast<uint8_t>(code);
        }
      }
    }
    __syncwarp();
  }
#pragma unroll
  for (int i = 0; i < 8; ++i) {
    ss[i] += __shfl_xor_sync(0xffffffffu, ss[i], 1);
    ss[i] += __shfl_xor_sync(0xffffffffu, ss[i], 2);
    ss[i] += __shfl_xor_sync(0xffffffffu, ss[i], 4);
  }
  if (cq == 0 && p.ssq_out != nullptr) {
#pragma unroll
    for (int i = 0; i < 8; ++i) {
      const int row = row_base + sub + 4 * i;
      if (row < M) p.ssq_out[(size_t)row * p.ssq_stride + (n_blk * nparts + part)] = ss[i];
    }
  }
}

// --------------------------------------------------------------------------------- kernel
template <int BN, int EPI, int DH>
__global__ void __cluster_dims__(2, 1, 1) __launch_bounds__((Gemm8Cfg<BN, EPI>::THREADS), 1)
te_gemm8_kernel(const __grid_constant__ CUtensorMap tmA, const __grid_constant__ CUtensorMap tmB,
                const __grid_constant__ CUtensorMap tmSFA, const __grid_constant__ CUtensorMap tmSFB, const GemmParams p,
                const Gemm8Extra x8) {
  using Cfg = Gemm8Cfg<BN, EPI>;
  constexpr int STAGES = Cfg::STAGES;
  constexpr int ACC = Cfg::ACC;
  extern __shared__ uint8_t smem_raw[];
  uint8_t* smem = reinterpret_cast<uint8_t*>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~uintptr_t(1023));
  uint8_t* sA = smem;
  uint8_t* sB = sA + STAGES * Cfg::A_BYTES;
  uint8_t* sSFA = sB + STAGES * Cfg::B_BYTES;
  uint8_t* sSFB = sSFA + STAGES * Cfg::SFA_BYTES;
  uint64_t* bars = reinterpret_cast<uint64_t*>(sSFB + STAGES * Cfg::SFB_BYTES);
  uint64_t* full = bars;                 // used in the leader CTA only
  uint64_t* empty = bars + STAGES;       // one set per CTA
  uint64_t* tfull = bars + 2 * STAGES;   // one set per CTA
  uint64_t* tempty = tfull + ACC;        // used in the leader CTA only
  uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(tempty + ACC);
  float* stg_all = reinterpret_cast<float*>(smem + STAGES * Cfg::STAGE_BYTES + Cfg::BAR_BYTES);

  const int warp = threadIdx.x >> 5;
  const int lane = threadIdx.x & 31;
  const uint32_t rank = cluster_ctarank();
  const bool leader = rank == 0;

  if (warp == 0 && elect_one()) {
    tma_prefetch_desc(&tmA);
    tma_prefetch_desc(&tmB);
    tma_prefetch_desc(&tmSFA);
    tma_prefetch_desc(&tmSFB);
  }
  if (warp == 1) {
    if (elect_one()) {
      for (int i = 0; i < STAGES; ++i) {
        mbar_init(&full[i], 1);
        mbar_init(&empty[i], 1);
      }
      for (int i = 0; i < ACC; ++i) {
        mbar_init(&tfull[i], 1);
        mbar_init(&tempty[i], 2 * 32 * Cfg::EPI_WARPS);
      }
      fence_mbar_init();
    }
    __syncwarp();
    tmem_alloc_cg2(tmem_slot, Cfg::TMEM_COLS);
  }
  tc_fence_before();
  __syncthreads();
  cluster_sync_all();
  tc_fence_after();
  const uint32_t tmem_base = *tmem_slot;
  pdl_launch_dependents();

  const int M = gemm_rows(p);
  const int num_kb = p.K / GEMM8_BK;
  const int num_mp = (p.num_m_blk + 1) >> 1;  // 256-row blocks
  const int num_tiles = num_mp * p.num_n_blk;
  const int pair = blockIdx.x >> 1;
  const int num_pairs = gridDim.x >> 1;

  if (warp == 0) {
    // ===================== producer (both CTAs): TMA tiles + scale tiles =====================
    if (elect_one()) {
      int stage = 0;
      uint32_t phase = 0;
      // bytes that complete on a stage's barrier, both CTAs together.  A packed-FP4 weight box (16U4_ALIGN16B) counts its
      // GLOBAL bytes (64 per 128-element row), not the 128 bytes it occupies in shared memory.
      const uint32_t stage_tx = 2 * (Cfg::STAGE_BYTES - (x8.b_fp4 ? Cfg::B_BYTES / 2 : 0));
      auto load_b = [&](int st, int kb, int n_blk, uint32_t bar) {  // weights and their scales: no dependency
        tma_load_2d_cg2(sB + st * Cfg::B_BYTES, &tmB, bar, kb * GEMM8_BK, n_blk * BN + static_cast<int>(rank) * (BN / 2));
#pragma unroll
        for (int t = 0; t < Cfg::SFB_TILES; ++t) {
          const int rb = n_blk * Cfg::SFB_TILES + t;  // scale tiles are grouped by N tile (mx_sf_offset_tiled)
          tma_load_2d_cg2(sSFB + st * Cfg::SFB_BYTES + t * 512, &tmSFB, bar, 0, rb * num_kb + kb);
        }
      };
      const int pre = (pair < num_tiles) ? (num_kb < STAGES ? num_kb : STAGES) : 0;
      for (int i = 0; i < pre; ++i) {
        if (leader) mbar_arrive_expect_tx(&full[i], stage_tx);
        load_b(i, i, pair / num_mp, mapa_u32(smem_u32(&full[i]), 0));
      }
      pdl_wait();
      bool first = true;
      for (int tile = pair; tile < num_tiles; tile += num_pairs) {
        const int mp = tile % num_mp;
        const int n_blk = tile / num_mp;
        const int a_blk = mp * 2 + static_cast<int>(rank);  // this CTA's 128-row block of A
        for (int kb = 0; kb < num_kb; ++kb) {
          const uint32_t bar = mapa_u32(smem_u32(&full[stage]), 0);
          if (!(first && kb < pre)) {
            mbar_wait(&empty[stage], phase ^ 1);
            if (leader) mbar_arrive_expect_tx(&full[stage], stage_tx);
            load_b(stage, kb, n_blk, bar);
          }
          tma_load_2d_cg2(sA + stage * Cfg::A_BYTES, &tmA, bar, kb * GEMM8_BK, a_blk * GEMM_BM);
          tma_load_2d_cg2(sSFA + stage * Cfg::SFA_BYTES, &tmSFA, bar, 0, a_blk * num_kb + kb);
          if (++stage == STAGES) { stage = 0; phase ^= 1; }
        }
        first = false;
      }
    }
  } else if (warp == 1) {
    // ===================== MMA issuer (leader CTA only) =====================
    if (leader && elect_one()) {
      const uint32_t idesc = umma_idesc_mxf8(2 * GEMM_BM, BN) | (x8.b_fp4 ? (UMMA_F8F6F4_E2M1 << 10) : 0u);  // B format [10,13)
      int stage = 0;
      uint32_t phase = 0;
      int it = 0;
      uint32_t kcount = 0;
      for (int tile = pair; tile < num_tiles; tile += num_pairs, ++it) {
        const int acc = it % ACC;
        const uint32_t acc_phase = (it / ACC) & 1;
        mbar_wait(&tempty[acc], acc_phase ^ 1);
        tc_fence_after();
        const uint32_t d_tmem = tmem_base + acc * BN;
        for (int kb = 0; kb < num_kb; ++kb, ++kcount) {
          mbar_wait(&full[stage], phase);
          tc_fence_after();
          // this stage's scale tiles -> the TMEM scale set of its parity (in-order with the MMAs that read them)
          const uint32_t sf_col = tmem_base + Cfg::SF_COL0 + (kcount & 1) * Cfg::SF_SET_COLS;
          tmem_cp_sf_cg2(sf_col, umma_smem_desc_sf(smem_u32(sSFA + stage * Cfg::SFA_BYTES)));
#pragma unroll
          for (int t = 0; t < Cfg::SFB_TILES; ++t)
            tmem_cp_sf_cg2(sf_col + 4 + 4 * t, umma_smem_desc_sf(smem_u32(sSFB + stage * Cfg::SFB_BYTES + t * 512)));
          const uint64_t a_desc = umma_smem_desc_sw128(smem_u32(sA + stage * Cfg::A_BYTES));
          const uint64_t b_desc = umma_smem_desc_sw128(smem_u32(sB + stage * Cfg::B_BYTES));
#pragma unroll
          for (int k = 0; k < GEMM8_BK / 32; ++k)  // K = 32 per instruction = 32 B inside the 128 B swizzle span
            umma_mxf8_cg2(d_tmem, a_desc + 2 * k, b_desc + 2 * k, umma_idesc_with_sf(idesc, k), sf_col, sf_col + 4,
                          (kb | k) != 0 ? 1u : 0u);
          umma_commit_cg2(&empty[stage], 0x3);
          if (++stage == STAGES) { stage = 0; phase ^= 1; }
        }
        umma_commit_cg2(&tfull[acc], 0x3);
      }
    }
  } else {
    // ===================== epilogue warps (both CTAs, own 128 rows) =====================
    const int quad = warp & 3;
    const int part = (warp - 2) >> 2;
    constexpr int NPARTS = Cfg::EPI_WARPS / 4;
    int it = 0;
    pdl_wait();
    for (int tile = pair; tile < num_tiles; tile += num_pairs, ++it) {
      const int mp = tile % num_mp;
      const int n_blk = tile / num_mp;
      const int acc = it % ACC;
      const uint32_t acc_phase = (it / ACC) & 1;
      const int row_base = mp * 2 * GEMM_BM + rank * GEMM_BM + quad * 32;
      const uint32_t t_row = tmem_base + (static_cast<uint32_t>(quad * 32) << 16) + acc * BN;
      float rstd = 0.f;
      ResidPrefetch pf;
      if constexpr (EPI == EPI_QKV || EPI == EPI_SWIGLU) rstd = row_rstd(p, row_base + lane, row_base + lane < M);
      if constexpr (EPI == EPI_RESID) resid_issue<BN>(p, M, pf, row_base, lane, n_blk, part * (BN / NPARTS));
      mbar_wait(&tfull[acc], acc_phase);
      tc_fence_after();
      [[maybe_unused]] float* stg = stg_all + (warp - 2) * (Cfg::STG_WARP_BYTES / 4);
      if constexpr (EPI == EPI_PLAIN) epi_plain<BN>(p, t_row, row_base + lane, row_base + lane < M, n_blk, part, NPARTS);
      if constexpr (EPI == EPI_RESID) epi_resid8<BN>(p, x8, M, t_row, row_base, lane, n_blk, stg, part, NPARTS, pf);
      if constexpr (EPI == EPI_SWIGLU) epi_swiglu8<BN>(p, x8, M, t_row, row_base + lane, n_blk, part, NPARTS, rstd);
      if constexpr (EPI == EPI_QKV) epi_qkv<BN, DH>(p, M, t_row, row_base, lane, n_blk, stg, part, NPARTS, rstd);
      tc_fence_before();
      mbar_arrive_cluster_relaxed(mapa_u32(smem_u32(&tempty[acc]), 0));
    }
  }
  tc_fence_before();
  __syncwarp();
  __syncthreads();
  cluster_sync_all();
  if (warp == 1) {
    __syncwarp();
    tc_fence_after();
    tmem_dealloc_cg2(tmem_base, Cfg::TMEM_COLS);
  }
}

}  // namespace te
