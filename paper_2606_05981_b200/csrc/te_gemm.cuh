// te_gemm.cuh — persistent, warp-specialised bf16 GEMM for sm_100a:
//   TMA (128B-swizzled tiles) -> shared memory ring -> tcgen05.mma (fp32 accumulators in TMEM,
//   double-buffered) -> tcgen05.ld -> fused epilogue.
// D[M,N] = A[M,K] * B[N,K]^T, A = activations (bf16, row-major), B = weights (bf16 [out,in]).
//
// Warp roles (192 threads): warp 0 = TMA producer, warp 1 = TMEM allocator + MMA issuer,
// warps 2..5 = epilogue (warp w owns TMEM lanes 32*(w%4) .. +31; one thread per output row).
//
// Epilogues:
//   EPI_QKV    y = rstd[row] * acc; per-head RMSNorm(gq|gk) + M-RoPE on q/k heads; bf16 out
//   EPI_RESID  x += acc (fp32, in place); also emits bf16(x * g_next) for the next GEMM's A
//              operand and the row's partial sum of squares (RMSNorm statistics, split form)
//   EPI_SWIGLU y = rstd[row] * acc; out = silu(gate) * up, bf16
//   EPI_PLAIN  fp32 store (bring-up / te_debug_gemm)
// RMSNorm split: h W^T = rstd * ((x .* g) W^T) with rstd = 1/sqrt(mean(x^2) + eps), so the
// gain multiply + sum of squares live in the PRODUCER's epilogue and the rstd scale in the
// CONSUMER's epilogue; A tiles are therefore plain bf16 and TMA-loadable.
#pragma once
#include "te_ptx.cuh"

namespace te {

constexpr int GEMM_BM = 128;
constexpr int GEMM_BK = 64;
constexpr int GEMM_THREADS = 192;

enum { EPI_PLAIN = 0, EPI_QKV = 1, EPI_RESID = 2, EPI_SWIGLU = 3 };

struct GemmParams {
  int M, N, K;
  int num_m_blk, num_n_blk;
  // RMSNorm statistics of the A rows (consumer side): ssq_in[part * ssq_stride + row]
  const float* ssq_in;
  int ssq_parts;
  int ssq_stride;
  float inv_d;  // 1 / hidden
  float eps;
  // EPI_QKV
  __nv_bfloat16* qkv;
  int ld_qkv;
  int q_cols_end;  // columns [0, q_cols_end) are q heads
  int k_cols_end;  // columns [q_cols_end, k_cols_end) are k heads; the rest v
  const __nv_bfloat16* gq;
  const __nv_bfloat16* gk;
  const float* cos_t;  // [T, DH/2]
  const float* sin_t;
  // EPI_RESID
  float* x;
  int ld_x;
  const __nv_bfloat16* g_next;  // may be null (no next norm)
  __nv_bfloat16* xg;            // [T, ld_x] bf16(x * g_next)
  float* ssq_out;               // [num_n_blk][ssq_stride]
  // EPI_SWIGLU
  __nv_bfloat16* act;
  int ld_act;
  // EPI_PLAIN
  float* c;
  int ld_c;
};

template <int BN>
struct GemmCfg {
  static constexpr int STAGES = (BN == 256) ? 4 : 6;
  static constexpr int A_BYTES = GEMM_BM * GEMM_BK * 2;
  static constexpr int B_BYTES = BN * GEMM_BK * 2;
  static constexpr int STAGE_BYTES = A_BYTES + B_BYTES;
  static constexpr int BAR_BYTES = 256;
  static constexpr int SMEM_BYTES = STAGES * STAGE_BYTES + BAR_BYTES + 1024;  // +1024: manual alignment
  static constexpr int TMEM_COLS = 2 * BN;
};

__device__ __forceinline__ uint32_t pack_bf16(float a, float b) {
  __nv_bfloat162 v = __floats2bfloat162_rn(a, b);
  return *reinterpret_cast<uint32_t*>(&v);
}
__device__ __forceinline__ float bf16_lo(uint32_t u) { return __uint_as_float(u << 16); }
__device__ __forceinline__ float bf16_hi(uint32_t u) { return __uint_as_float(u & 0xFFFF0000u); }

// ----------------------------------------------------------------------------- epilogues
template <int BN>
__device__ __forceinline__ void epi_plain(const GemmParams& p, uint32_t t_row, int row, bool valid, int n_blk) {
#pragma unroll 1
  for (int c0 = 0; c0 < BN; c0 += 32) {
    uint32_t r[32];
    tmem_ld32(t_row + c0, r);
    tmem_ld_wait();
    if (valid) {
      float4* dst = reinterpret_cast<float4*>(p.c + (size_t)row * p.ld_c + n_blk * BN + c0);
#pragma unroll
      for (int j = 0; j < 8; ++j)
        dst[j] = make_float4(__uint_as_float(r[4 * j]), __uint_as_float(r[4 * j + 1]), __uint_as_float(r[4 * j + 2]),
                             __uint_as_float(r[4 * j + 3]));
    }
  }
}

template <int BN>
__device__ __forceinline__ void epi_resid(const GemmParams& p, uint32_t t_row, int row, bool valid, int n_blk) {
  float ss = 0.f;
  const bool has_g = p.g_next != nullptr;
#pragma unroll 1
  for (int c0 = 0; c0 < BN; c0 += 32) {
    uint32_t r[32];
    tmem_ld32(t_row + c0, r);
    tmem_ld_wait();
    if (valid) {
      const int col = n_blk * BN + c0;
      float4* xp = reinterpret_cast<float4*>(p.x + (size_t)row * p.ld_x + col);
      float xn[32];
#pragma unroll
      for (int j = 0; j < 8; ++j) {
        float4 v = xp[j];
        v.x += __uint_as_float(r[4 * j]);
        v.y += __uint_as_float(r[4 * j + 1]);
        v.z += __uint_as_float(r[4 * j + 2]);
        v.w += __uint_as_float(r[4 * j + 3]);
        xp[j] = v;
        xn[4 * j] = v.x; xn[4 * j + 1] = v.y; xn[4 * j + 2] = v.z; xn[4 * j + 3] = v.w;
        ss = fmaf(v.x, v.x, ss); ss = fmaf(v.y, v.y, ss); ss = fmaf(v.z, v.z, ss); ss = fmaf(v.w, v.w, ss);
      }
      if (has_g) {
        const uint4* gp = reinterpret_cast<const uint4*>(p.g_next + col);
        uint4* op = reinterpret_cast<uint4*>(p.xg + (size_t)row * p.ld_x + col);
#pragma unroll
        for (int j = 0; j < 4; ++j) {
          const uint4 g = __ldg(gp + j);
          uint4 o;
          o.x = pack_bf16(xn[8 * j + 0] * bf16_lo(g.x), xn[8 * j + 1] * bf16_hi(g.x));
          o.y = pack_bf16(xn[8 * j + 2] * bf16_lo(g.y), xn[8 * j + 3] * bf16_hi(g.y));
          o.z = pack_bf16(xn[8 * j + 4] * bf16_lo(g.z), xn[8 * j + 5] * bf16_hi(g.z));
          o.w = pack_bf16(xn[8 * j + 6] * bf16_lo(g.w), xn[8 * j + 7] * bf16_hi(g.w));
          op[j] = o;
        }
      }
    }
  }
  if (valid && p.ssq_out != nullptr) p.ssq_out[(size_t)n_blk * p.ssq_stride + row] = ss;
}

__device__ __forceinline__ float row_rstd(const GemmParams& p, int row, bool valid) {
  float s = 0.f;
  if (valid)
    for (int i = 0; i < p.ssq_parts; ++i) s += p.ssq_in[(size_t)i * p.ssq_stride + row];
  return 1.0f / sqrtf(s * p.inv_d + p.eps);
}

template <int BN>
__device__ __forceinline__ void epi_swiglu(const GemmParams& p, uint32_t t_row, int row, bool valid, int n_blk) {
  const float rstd = row_rstd(p, row, valid);
  constexpr int HALF = BN / 2;  // tile columns [0,HALF) = gate, [HALF,BN) = up (weights interleaved per tile)
#pragma unroll 1
  for (int c0 = 0; c0 < HALF; c0 += 16) {
    uint32_t g[16], u[16];
    tmem_ld16(t_row + c0, g);
    tmem_ld16(t_row + HALF + c0, u);
    tmem_ld_wait();
    if (valid) {
      uint32_t o[8];
#pragma unroll
      for (int j = 0; j < 8; ++j) {
        float g0 = __uint_as_float(g[2 * j]) * rstd, g1 = __uint_as_float(g[2 * j + 1]) * rstd;
        float u0 = __uint_as_float(u[2 * j]) * rstd, u1 = __uint_as_float(u[2 * j + 1]) * rstd;
        float a0 = g0 / (1.0f + __expf(-g0)) * u0;
        float a1 = g1 / (1.0f + __expf(-g1)) * u1;
        o[j] = pack_bf16(a0, a1);
      }
      uint4* dst = reinterpret_cast<uint4*>(p.act + (size_t)row * p.ld_act + n_blk * HALF + c0);
      dst[0] = make_uint4(o[0], o[1], o[2], o[3]);
      dst[1] = make_uint4(o[4], o[5], o[6], o[7]);
    }
  }
}

template <int BN, int DH>
__device__ __forceinline__ void epi_qkv(const GemmParams& p, uint32_t t_row, int row, bool valid, int n_blk) {
  const float rstd = row_rstd(p, row, valid);
  constexpr int HD2 = DH / 2;
#pragma unroll 1
  for (int hh = 0; hh < BN / DH; ++hh) {
    const int col0 = n_blk * BN + hh * DH;  // first column of this head in the fused qkv row
    const uint32_t t_head = t_row + hh * DH;
    if (col0 >= p.k_cols_end) {
      // ---- v head: scale and store
#pragma unroll 1
      for (int c0 = 0; c0 < DH; c0 += 32) {
        uint32_t r[32];
        tmem_ld32(t_head + c0, r);
        tmem_ld_wait();
        if (valid) {
          uint4* dst = reinterpret_cast<uint4*>(p.qkv + (size_t)row * p.ld_qkv + col0 + c0);
#pragma unroll
          for (int j = 0; j < 4; ++j) {
            uint4 o;
            o.x = pack_bf16(__uint_as_float(r[8 * j + 0]) * rstd, __uint_as_float(r[8 * j + 1]) * rstd);
            o.y = pack_bf16(__uint_as_float(r[8 * j + 2]) * rstd, __uint_as_float(r[8 * j + 3]) * rstd);
            o.z = pack_bf16(__uint_as_float(r[8 * j + 4]) * rstd, __uint_as_float(r[8 * j + 5]) * rstd);
            o.w = pack_bf16(__uint_as_float(r[8 * j + 6]) * rstd, __uint_as_float(r[8 * j + 7]) * rstd);
            dst[j] = o;
          }
        }
      }
      continue;
    }
    // ---- q or k head: per-head RMSNorm (pass 1: sum of squares), then gain + rotation (pass 2)
    const __nv_bfloat16* gain = (col0 < p.q_cols_end) ? p.gq : p.gk;
    float ss = 0.f;
#pragma unroll 1
    for (int c0 = 0; c0 < DH; c0 += 32) {
      uint32_t r[32];
      tmem_ld32(t_head + c0, r);
      tmem_ld_wait();
#pragma unroll
      for (int j = 0; j < 32; ++j) {
        const float y = __uint_as_float(r[j]) * rstd;
        ss = fmaf(y, y, ss);
      }
    }
    const float sc = rstd / sqrtf(ss * (1.0f / DH) + p.eps);
#pragma unroll 1
    for (int c0 = 0; c0 < HD2; c0 += 16) {
      uint32_t a[16], b[16];
      tmem_ld16(t_head + c0, a);
      tmem_ld16(t_head + HD2 + c0, b);
      tmem_ld_wait();
      if (valid) {
        const float4* cp = reinterpret_cast<const float4*>(p.cos_t + (size_t)row * HD2 + c0);
        const float4* sp = reinterpret_cast<const float4*>(p.sin_t + (size_t)row * HD2 + c0);
        const uint4* ga = reinterpret_cast<const uint4*>(gain + c0);
        const uint4* gb = reinterpret_cast<const uint4*>(gain + HD2 + c0);
        uint32_t o1[8], o2[8];
#pragma unroll
        for (int j = 0; j < 2; ++j) {  // 8 columns per iteration
          const uint4 g1 = __ldg(ga + j), g2 = __ldg(gb + j);
          const float4 c_lo = __ldg(cp + 2 * j), c_hi = __ldg(cp + 2 * j + 1);
          const float4 s_lo = __ldg(sp + 2 * j), s_hi = __ldg(sp + 2 * j + 1);
          const float cs[8] = {c_lo.x, c_lo.y, c_lo.z, c_lo.w, c_hi.x, c_hi.y, c_hi.z, c_hi.w};
          const float sn[8] = {s_lo.x, s_lo.y, s_lo.z, s_lo.w, s_hi.x, s_hi.y, s_hi.z, s_hi.w};
          const float gA[8] = {bf16_lo(g1.x), bf16_hi(g1.x), bf16_lo(g1.y), bf16_hi(g1.y),
                               bf16_lo(g1.z), bf16_hi(g1.z), bf16_lo(g1.w), bf16_hi(g1.w)};
          const float gB[8] = {bf16_lo(g2.x), bf16_hi(g2.x), bf16_lo(g2.y), bf16_hi(g2.y),
                               bf16_lo(g2.z), bf16_hi(g2.z), bf16_lo(g2.w), bf16_hi(g2.w)};
          float r1[8], r2[8];
#pragma unroll
          for (int e = 0; e < 8; ++e) {
            const float ua = __uint_as_float(a[8 * j + e]) * sc * gA[e];
            const float ub = __uint_as_float(b[8 * j + e]) * sc * gB[e];
            r1[e] = ua * cs[e] - ub * sn[e];
            r2[e] = ub * cs[e] + ua * sn[e];
          }
#pragma unroll
          for (int e = 0; e < 4; ++e) {
            o1[4 * j + e] = pack_bf16(r1[2 * e], r1[2 * e + 1]);
            o2[4 * j + e] = pack_bf16(r2[2 * e], r2[2 * e + 1]);
          }
        }
        uint4* d1 = reinterpret_cast<uint4*>(p.qkv + (size_t)row * p.ld_qkv + col0 + c0);
        uint4* d2 = reinterpret_cast<uint4*>(p.qkv + (size_t)row * p.ld_qkv + col0 + HD2 + c0);
        d1[0] = make_uint4(o1[0], o1[1], o1[2], o1[3]);
        d1[1] = make_uint4(o1[4], o1[5], o1[6], o1[7]);
        d2[0] = make_uint4(o2[0], o2[1], o2[2], o2[3]);
        d2[1] = make_uint4(o2[4], o2[5], o2[6], o2[7]);
      }
    }
  }
}

// --------------------------------------------------------------------------------- kernel
template <int BN, int EPI, int DH>
__global__ void __launch_bounds__(GEMM_THREADS, 1)
te_gemm_kernel(const __grid_constant__ CUtensorMap tmA, const __grid_constant__ CUtensorMap tmB, const GemmParams p) {
  using Cfg = GemmCfg<BN>;
  constexpr int STAGES = Cfg::STAGES;
  extern __shared__ uint8_t smem_raw[];
  uint8_t* smem = reinterpret_cast<uint8_t*>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~uintptr_t(1023));
  uint8_t* sA = smem;
  uint8_t* sB = smem + STAGES * Cfg::A_BYTES;
  uint64_t* bars = reinterpret_cast<uint64_t*>(smem + STAGES * Cfg::STAGE_BYTES);
  uint64_t* full = bars;
  uint64_t* empty = bars + STAGES;
  uint64_t* tfull = bars + 2 * STAGES;
  uint64_t* tempty = tfull + 2;
  uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(tempty + 2);

  const int warp = threadIdx.x >> 5;
  const int lane = threadIdx.x & 31;

  if (warp == 0 && elect_one()) {
    tma_prefetch_desc(&tmA);
    tma_prefetch_desc(&tmB);
  }
  if (warp == 1) {
    if (elect_one()) {
      for (int i = 0; i < STAGES; ++i) {
        mbar_init(&full[i], 1);
        mbar_init(&empty[i], 1);
      }
      for (int i = 0; i < 2; ++i) {
        mbar_init(&tfull[i], 1);
        mbar_init(&tempty[i], 128);
      }
      fence_mbar_init();
    }
    __syncwarp();
    tmem_alloc(tmem_slot, Cfg::TMEM_COLS);
  }
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tmem_base = *tmem_slot;

  const int num_kb = p.K / GEMM_BK;
  const int num_tiles = p.num_m_blk * p.num_n_blk;

  if (warp == 0) {
    // ===================== TMA producer =====================
    if (elect_one()) {
      int stage = 0;
      uint32_t phase = 0;
      for (int tile = blockIdx.x; tile < num_tiles; tile += gridDim.x) {
        const int m_blk = tile % p.num_m_blk;
        const int n_blk = tile / p.num_m_blk;
        for (int kb = 0; kb < num_kb; ++kb) {
          mbar_wait(&empty[stage], phase ^ 1);
          mbar_arrive_expect_tx(&full[stage], Cfg::STAGE_BYTES);
          tma_load_2d(sA + stage * Cfg::A_BYTES, &tmA, &full[stage], kb * GEMM_BK, m_blk * GEMM_BM);
          tma_load_2d(sB + stage * Cfg::B_BYTES, &tmB, &full[stage], kb * GEMM_BK, n_blk * BN);
          if (++stage == STAGES) { stage = 0; phase ^= 1; }
        }
      }
    }
  } else if (warp == 1) {
    // ===================== MMA issuer =====================
    if (elect_one()) {
      constexpr uint32_t idesc = umma_idesc_bf16(GEMM_BM, BN);
      int stage = 0;
      uint32_t phase = 0;
      int it = 0;
      for (int tile = blockIdx.x; tile < num_tiles; tile += gridDim.x, ++it) {
        const int acc = it & 1;
        const uint32_t acc_phase = (it >> 1) & 1;
        mbar_wait(&tempty[acc], acc_phase ^ 1);
        tc_fence_after();
        const uint32_t d_tmem = tmem_base + acc * BN;
        for (int kb = 0; kb < num_kb; ++kb) {
          mbar_wait(&full[stage], phase);
          tc_fence_after();
          const uint64_t a_desc = umma_smem_desc_sw128(smem_u32(sA + stage * Cfg::A_BYTES));
          const uint64_t b_desc = umma_smem_desc_sw128(smem_u32(sB + stage * Cfg::B_BYTES));
#pragma unroll
          for (int k = 0; k < GEMM_BK / 16; ++k) {
            // advance 16 elements (32 B) along K inside the 128B swizzle span: +2 in the >>4 address field
            umma_bf16(d_tmem, a_desc + 2 * k, b_desc + 2 * k, idesc, (kb | k) != 0 ? 1u : 0u);
          }
          umma_commit(&empty[stage]);
          if (++stage == STAGES) { stage = 0; phase ^= 1; }
        }
        umma_commit(&tfull[acc]);
      }
    }
  } else {
    // ===================== epilogue warps =====================
    const int quad = warp & 3;
    const int row_in_tile = quad * 32 + lane;
    int it = 0;
    for (int tile = blockIdx.x; tile < num_tiles; tile += gridDim.x, ++it) {
      const int m_blk = tile % p.num_m_blk;
      const int n_blk = tile / p.num_m_blk;
      const int acc = it & 1;
      const uint32_t acc_phase = (it >> 1) & 1;
      const int row = m_blk * GEMM_BM + row_in_tile;
      const bool valid = row < p.M;
      mbar_wait(&tfull[acc], acc_phase);
      tc_fence_after();
      const uint32_t t_row = tmem_base + (static_cast<uint32_t>(quad * 32) << 16) + acc * BN;
      if constexpr (EPI == EPI_PLAIN) epi_plain<BN>(p, t_row, row, valid, n_blk);
      if constexpr (EPI == EPI_RESID) epi_resid<BN>(p, t_row, row, valid, n_blk);
      if constexpr (EPI == EPI_SWIGLU) epi_swiglu<BN>(p, t_row, row, valid, n_blk);
      if constexpr (EPI == EPI_QKV) epi_qkv<BN, DH>(p, t_row, row, valid, n_blk);
      tc_fence_before();
      mbar_arrive(&tempty[acc]);
    }
  }
  __syncthreads();
  if (warp == 1) {
    tc_fence_after();
    tmem_dealloc(tmem_base, Cfg::TMEM_COLS);
  }
}

}  // namespace te
