// te_gemm_wide.cuh — residual GEMMs (O-proj, down) in ONE wave of CTA-pair tiles.
//
// With N = hidden = 2048 the residual GEMMs have too few 256-wide tiles for 74 SM pairs (96 = 1.3 waves) and
// their 128-wide tiles (192 = 2.59 waves, run as 3) are bound by L2->SM operand traffic (96 B/clk per SM).
// Here the tile width is chosen so that the number of tiles fits the SM pairs in a single wave:
//     n_tiles = floor(pairs / ceil(T/256)),  width bn = N / n_tiles rounded up to 32  (cfg 4: 6 x 352 columns),
// one 256 x bn tile per CTA pair, accumulated by TWO tcgen05.mma.cta_group::2 per k-step of bn/2 columns each
// (N <= 256 per instruction) into one bn-column TMEM accumulator.  Per 64-deep k-block a CTA loads its 128 A rows
// and bn/2 weight rows: 54 B/clk per SM at bn = 352, i.e. the tile is tensor-bound again, and no wave is
// partially filled.  Columns past N (the last tile) are zero-filled by TMA and never stored.
// Same warp roles, PDL prologue and residual epilogue arithmetic as te_gemm2_kernel (te_gemm.cuh).
//
// EPI_SWIGLU variant (mid batches, e.g. T = 512: 96 pair tiles of 256 x 256 = 1.3 waves): the two MMAs of a tile
// take the gate rows and the matching up rows, so that a tile of w output columns (bn = 2w accumulator columns:
// [0,w) gate, [w,2w) up) can have any width that is a multiple of 64: 32 x 192 output columns x 2 row-pair blocks
// = 64 tiles, one wave.  The weights are the library's one copy of [Wgate; Wup], interleaved per 256 rows (128 gate
// rows | the 128 matching up rows): 32 consecutive output columns are 32 consecutive rows there, so the B operand is
// fetched as 32-row TMA boxes (gate column c -> row (c / 128) * 256 + c % 128, up column c -> that + 128).
#pragma once
#include "te_gemm.cuh"

namespace te {

struct GemmWideCfg {
  static constexpr int A_BYTES = GEMM_BM * GEMM_BK * 2;
  static constexpr int BAR_BYTES = 256;
  static constexpr int STG_WARP_BYTES = 32 * 32 * 4;
  static constexpr int STG_BYTES = GEMM2_EPI_WARPS * STG_WARP_BYTES;
  static constexpr int SMEM_LIMIT = 232448;  // 227 KB
  static constexpr int TMEM_COLS = 512;
  static constexpr int MAX_STAGES = 8;
  __host__ __device__ static constexpr int b_bytes(int bn) { return (bn / 2) * GEMM_BK * 2; }  // per CTA and stage
  __host__ __device__ static constexpr int stage_bytes(int bn) { return A_BYTES + b_bytes(bn); }
  // One tile per CTA pair and ONE accumulator barrier, so the epilogue staging ALIASES the ring (first written when
  // every MMA has read its stage and no TMA write is outstanding in either CTA): one more stage in flight at the SwiGLU
  // widths.
  __host__ __device__ static constexpr int stages(int bn) {
    const int fit = (SMEM_LIMIT - 1024 - BAR_BYTES) / stage_bytes(bn);
    return fit > MAX_STAGES ? MAX_STAGES : fit;
  }
  __host__ __device__ static constexpr int smem_bytes(int bn) {
    const int ring = stages(bn) * stage_bytes(bn);
    return (ring > STG_BYTES ? ring : STG_BYTES) + BAR_BYTES + 1024;
  }
};

// bn: accumulator width, a multiple of 32 (128 for EPI_SWIGLU), <= 512; nh = bn/2 columns per MMA (multiple of 16, <= 256).
// tmB: EPI_RESID: weight matrix [N, K] in boxes of nh/2 rows x 64 columns; EPI_SWIGLU: the interleaved [2F, K] gate/up
// matrix in boxes of 32 rows x 64 columns (p.N = 2F; the tile's output columns are n_blk*nh .. +nh of F).
template <int EPI>
__global__ void __cluster_dims__(2, 1, 1) __launch_bounds__(GEMM2_THREADS, 1)
te_gemm_wide_kernel(const __grid_constant__ CUtensorMap tmA, const __grid_constant__ CUtensorMap tmB, const GemmParams p,
                    const int bn) {
  using Cfg = GemmWideCfg;
  const int STAGES = Cfg::stages(bn);
  const int nh = bn / 2;
  const int b_bytes = Cfg::b_bytes(bn);
  const int sub_bytes = b_bytes / 2;  // one MMA's share of this CTA's B rows: nh/2 rows x 128 B (1024-B aligned)
  extern __shared__ uint8_t smem_raw[];
  uint8_t* smem = reinterpret_cast<uint8_t*>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~uintptr_t(1023));
  uint8_t* sA = smem;
  uint8_t* sB = smem + STAGES * Cfg::A_BYTES;
  uint64_t* bars = reinterpret_cast<uint64_t*>(smem + STAGES * Cfg::stage_bytes(bn));
  uint64_t* full = bars;                          // used in the leader CTA only
  uint64_t* empty = bars + Cfg::MAX_STAGES;       // one set per CTA
  uint64_t* tfull = bars + 2 * Cfg::MAX_STAGES;   // one per CTA
  uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(tfull + 1);
  float* stg_all = reinterpret_cast<float*>(smem);  // aliases the ring (see GemmWideCfg::stages)

  const int warp = threadIdx.x >> 5;
  const int lane = threadIdx.x & 31;
  const uint32_t rank = cluster_ctarank();
  const bool leader = rank == 0;
  if (threadIdx.x == 0) trace_stamp(p, 0);

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
      mbar_init(tfull, 1);
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
  if (threadIdx.x == 0) trace_stamp(p, 1);

  const int M = gemm_rows(p);
  const int num_kb = p.K / GEMM_BK;
  const int num_mp = (p.num_m_blk + 1) >> 1;  // 256-row blocks
  const int tile = blockIdx.x >> 1;  // one tile per CTA pair
  const int mp = tile % num_mp;
  const int n_blk = tile / num_mp;
  // first output column of the tile; first weight row of MMA 0 / MMA 1
  const int col_base = (EPI == EPI_SWIGLU) ? n_blk * nh : n_blk * bn;
  const int w_row0 = col_base;
  const int w_row1 = (EPI == EPI_SWIGLU) ? p.N / 2 + col_base : col_base + nh;

  if (warp == 0) {
    // ===================== TMA producer (both CTAs) =====================
    if (elect_one()) {
      const int a_row = mp * 2 * GEMM_BM + rank * GEMM_BM;
      // this CTA's weight rows for MMA j: [col_base + j*nh + rank*nh/2, + nh/2)
      const int b_row0 = w_row0 + rank * (nh / 2);
      [[maybe_unused]] const int b_row1 = w_row1 + rank * (nh / 2);
      auto load_b = [&](int stage, int kb) {
        const uint32_t bar = mapa_u32(smem_u32(&full[stage]), 0);
        if constexpr (EPI == EPI_SWIGLU) {
          // this CTA's nh/2 gate columns and nh/2 up columns, 32 at a time, from the 256-row interleaved layout
          for (int j = 0; j < nh / 2; j += 32) {
            const int c = b_row0 + j;  // output column of F
            const int g_row = (c >> 7) * 256 + (c & 127);
            tma_load_2d_cg2(sB + stage * b_bytes + j * 128, &tmB, bar, kb * GEMM_BK, g_row);
            tma_load_2d_cg2(sB + stage * b_bytes + sub_bytes + j * 128, &tmB, bar, kb * GEMM_BK, g_row + 128);
          }
        } else {
          tma_load_2d_cg2(sB + stage * b_bytes, &tmB, bar, kb * GEMM_BK, b_row0);
          tma_load_2d_cg2(sB + stage * b_bytes + sub_bytes, &tmB, bar, kb * GEMM_BK, b_row1);
        }
      };
      const int pre = num_kb < STAGES ? num_kb : STAGES;
      for (int kb = 0; kb < pre; ++kb) {  // weights first: independent of the predecessor kernel
        if (leader) mbar_arrive_expect_tx(&full[kb], 2 * Cfg::stage_bytes(bn));
        load_b(kb, kb);
      }
      pdl_wait();
      trace_stamp(p, 2);
      int stage = 0;
      uint32_t phase = 0;
      for (int kb = 0; kb < num_kb; ++kb) {
        const uint32_t bar = mapa_u32(smem_u32(&full[stage]), 0);
        if (kb >= pre) {
          mbar_wait(&empty[stage], phase ^ 1);
          if (leader) mbar_arrive_expect_tx(&full[stage], 2 * Cfg::stage_bytes(bn));
          load_b(stage, kb);
        }
        tma_load_2d_cg2(sA + stage * Cfg::A_BYTES, &tmA, bar, kb * GEMM_BK, a_row);
        if (++stage == STAGES) { stage = 0; phase ^= 1; }
      }
    }
  } else if (warp == 1) {
    // ===================== MMA issuer (leader CTA only) =====================
    if (leader && elect_one()) {
      const uint32_t idesc = umma_idesc_bf16(2 * GEMM_BM, static_cast<uint32_t>(nh));
      int stage = 0;
      uint32_t phase = 0;
      for (int kb = 0; kb < num_kb; ++kb) {
        mbar_wait(&full[stage], phase);
        if (kb == 0) trace_stamp(p, 3);
        tc_fence_after();
        const uint64_t a_desc = umma_smem_desc_sw128(smem_u32(sA + stage * Cfg::A_BYTES));
        const uint64_t b_desc0 = umma_smem_desc_sw128(smem_u32(sB + stage * b_bytes));
        const uint64_t b_desc1 = umma_smem_desc_sw128(smem_u32(sB + stage * b_bytes + sub_bytes));
#pragma unroll
        for (int k = 0; k < GEMM_BK / 16; ++k) {
          const uint32_t accum = (kb | k) != 0 ? 1u : 0u;
          umma_bf16_cg2(tmem_base, a_desc + 2 * k, b_desc0 + 2 * k, idesc, accum);
          umma_bf16_cg2(tmem_base + nh, a_desc + 2 * k, b_desc1 + 2 * k, idesc, accum);
        }
        umma_commit_cg2(&empty[stage], 0x3);  // frees this stage in BOTH CTAs
        if (++stage == STAGES) { stage = 0; phase ^= 1; }
      }
      umma_commit_cg2(tfull, 0x3);  // accumulator ready in BOTH CTAs
    }
  } else {
    // ===================== epilogue warps (both CTAs, own 128 rows): x += acc, xg, sum of squares ============
    const int quad = warp & 3;
    const int part = (warp - 2) >> 2;
    [[maybe_unused]] const int sub = lane >> 3, cq = lane & 7;
    const int row_base = mp * 2 * GEMM_BM + rank * GEMM_BM + quad * 32;
    const uint32_t t_row = tmem_base + (static_cast<uint32_t>(quad * 32) << 16);
    float* stg = stg_all + (warp - 2) * (Cfg::STG_WARP_BYTES / 4);
    // the tile's valid 32-column chunks (of output columns) are split between the two warps of a quadrant
    const int out_w = (EPI == EPI_SWIGLU) ? nh : bn;
    int n_valid = ((EPI == EPI_SWIGLU) ? p.N / 2 : p.N) - col_base;
    n_valid = n_valid < 0 ? 0 : (n_valid > out_w ? out_w : n_valid);
    const int chunks = n_valid / 32;
    const int c_begin = part == 0 ? 0 : ((chunks + 1) / 2) * 32;
    const int c_end = part == 0 ? ((chunks + 1) / 2) * 32 : chunks * 32;
    pdl_wait();
    if constexpr (EPI == EPI_SWIGLU) {
      // ---- y = rstd * acc; act = silu(gate) * up, bf16 (arithmetic of epi_swiglu, te_gemm.cuh)
      const float rstd = row_rstd(p, row_base + lane, row_base + lane < M);
      mbar_wait(tfull, 0);
      if (warp == 2 && lane == 0) trace_stamp(p, 14);
      tc_fence_after();
#pragma unroll 1
      for (int c0 = c_begin; c0 < c_end; c0 += 32) {
        float a[32];
        {
          uint32_t g[32], u[32];
          tmem_ld32(t_row + c0, g);
          tmem_ld32(t_row + nh + c0, u);
          tmem_ld_wait();
#pragma unroll
          for (int j = 0; j < 32; ++j) {
            const float gv = __uint_as_float(g[j]) * rstd;
            const float uv = __uint_as_float(u[j]) * rstd;
            a[j] = __fdividef(gv, 1.0f + __expf(-gv)) * uv;
          }
        }
        stg_put_row(stg, lane, a);
        __syncwarp();
        stg_store_bf16(stg, lane, row_base, M, p.act, p.ld_act, col_base + c0);
        __syncwarp();
      }
      if (warp == 2 && lane == 0) trace_stamp(p, 25);
    } else if constexpr (EPI == EPI_PLAIN) {
      // ---- fp32 store of the valid columns (te_debug_gemm_wide: the main loop alone against a matmul)
      mbar_wait(tfull, 0);
      tc_fence_after();
      const int row = row_base + lane;
#pragma unroll 1
      for (int c0 = c_begin; c0 < c_end; c0 += 32) {
        uint32_t r[32];
        tmem_ld32(t_row + c0, r);
        tmem_ld_wait();
        if (row < M) {
          float4* dst = reinterpret_cast<float4*>(p.c + (size_t)row * p.ld_c + col_base + c0);
#pragma unroll
          for (int j = 0; j < 8; ++j)
            dst[j] = make_float4(__uint_as_float(r[4 * j]), __uint_as_float(r[4 * j + 1]), __uint_as_float(r[4 * j + 2]),
                                 __uint_as_float(r[4 * j + 3]));
        }
      }
    } else {
    const bool has_g = p.g_next != nullptr;
    float* const x_dst = resid_dst(p);
    auto issue_x = [&](float4 (&xv)[8], int c0) {
      const int col = col_base + c0 + cq * 4;
#pragma unroll
      for (int i = 0; i < 8; ++i) {
        const int row = row_base + sub + 4 * i;
        if (row < M) xv[i] = *reinterpret_cast<const float4*>(p.x + (size_t)row * p.ld_x + col);
      }
    };
    float4 xn[8];
    if (c_begin < c_end) issue_x(xn, c_begin);  // first chunk's x while the main loop runs
    mbar_wait(tfull, 0);
    if (warp == 2 && lane == 0) trace_stamp(p, 14);
    tc_fence_after();
    float ss[8];
#pragma unroll
    for (int i = 0; i < 8; ++i) ss[i] = 0.f;
#pragma unroll 1
    for (int c0 = c_begin; c0 < c_end; c0 += 32) {
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
      const int col = col_base + c0 + cq * 4;
      float g0 = 0.f, g1 = 0.f, g2 = 0.f, g3 = 0.f;
      if (has_g) {
        const uint2 g = __ldg(reinterpret_cast<const uint2*>(p.g_next + col));
        g0 = bf16_lo(g.x); g1 = bf16_hi(g.x); g2 = bf16_lo(g.y); g3 = bf16_hi(g.y);
      }
      float4 xv[8];
#pragma unroll
      for (int i = 0; i < 8; ++i) xv[i] = xn[i];
      if (c0 + 32 < c_end) issue_x(xn, c0 + 32);  // next chunk's x in flight
#pragma unroll
      for (int i = 0; i < 8; ++i) {
        const int rr = sub + 4 * i;
        const int row = row_base + rr;
        if (row < M) {
          const float4 a = stg_get(stg, rr, cq);
          float4 v = xv[i];
          v.x += a.x; v.y += a.y; v.z += a.z; v.w += a.w;
          *reinterpret_cast<float4*>(x_dst + (size_t)row * p.ld_x + col) = v;
          ss[i] = fmaf(v.x, v.x, ss[i]); ss[i] = fmaf(v.y, v.y, ss[i]);
          ss[i] = fmaf(v.z, v.z, ss[i]); ss[i] = fmaf(v.w, v.w, ss[i]);
          if (has_g) {
            uint2 o;
            o.x = pack_bf16(v.x * g0, v.y * g1);
            o.y = pack_bf16(v.z * g2, v.w * g3);
            *reinterpret_cast<uint2*>(p.xg + (size_t)row * p.ld_x + col) = o;
          }
        }
      }
      __syncwarp();
    }
    // per-row sum of squares over this warp's columns (fixed-order reduction over the row's 8 lanes); a warp
    // without valid columns still writes its zero, so that every statistics slot of the row is defined
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
        if (row < M) p.ssq_out[(size_t)row * p.ssq_stride + (n_blk * 2 + part)] = ss[i];
      }
    }
    if (warp == 2 && lane == 0) trace_stamp(p, 25);
    }  // EPI_RESID
  }
  tc_fence_before();
  __syncwarp();  // the elected producer / MMA lanes rejoin their warps before the block barrier
  __syncthreads();
  if (threadIdx.x == 0) trace_stamp(p, 36);
  cluster_sync_all();  // the peer may still be signalling our barriers / reading our smem until here
  if (threadIdx.x == 0) trace_stamp(p, 37);
  if (warp == 1) {
    __syncwarp();
    tc_fence_after();
    tmem_dealloc_cg2(tmem_base, Cfg::TMEM_COLS);
  }
}

}  // namespace te
