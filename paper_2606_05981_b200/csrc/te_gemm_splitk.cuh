// te_gemm_splitk.cuh — small-batch GEMM: one 128 x BN output tile per GROUP of `splits` CTAs, each
// CTA contracting its own K-slice (split-K), so that every SM streams weights when the token count
// gives fewer than one 128-row tile per SM (the HBM-bound regime of SURVEY.md §8(d): cfg 2, cfg 3).
//
//   CTA (tile, s):  TMA ring -> tcgen05.mma over k-blocks [s*nkb/S, (s+1)*nkb/S) -> fp32 partial in TMEM
//   every CTA    :  partial -> global scratch (stays in L2), release-increment of the tile's arrival
//                   counter, acquire-spin until all S partials are there
//   CTA s        :  rows r = s (mod S) of the tile: partials summed IN FIXED ORDER 0..S-1, then the
//                   same fused epilogue arithmetic as te_gemm.cuh (reduce-scatter: no CTA idles and no
//                   single SM has to ingest all partials)
//
// The group spins on each other, so the whole grid must be co-resident: the host launches this kernel
// only with tiles * S <= number of SMs (one CTA per SM) and, for S > 1, as a COOPERATIVE grid (the launch
// waits until every CTA can be resident).  The sum order is fixed -> bitwise deterministic.
// S == 1 degenerates to one CTA per tile with the TMEM epilogues of te_gemm.cuh.
// Weights of the CTA's first ring are requested before griddepcontrol.wait (they do not depend on the
// predecessor kernel), so under programmatic dependent launch the weight stream of kernel n+1 overlaps
// the tail of kernel n.
#pragma once
#include "te_gemm.cuh"

namespace te {

constexpr int GEMMK_EPI_WARPS = 8;
constexpr int GEMMK_THREADS = 64 + 32 * GEMMK_EPI_WARPS;
constexpr int GEMMK_MAX_SPLITS = 8;

template <int BN, int EPI>
struct GemmKCfg {
  static constexpr int A_BYTES = GEMM_BM * GEMM_BK * 2;
  static constexpr int B_BYTES = BN * GEMM_BK * 2;
  static constexpr int STAGE_BYTES = A_BYTES + B_BYTES;
  static constexpr int BAR_BYTES = 256;
  static constexpr int STG_WARP_BYTES = (EPI == EPI_QKV ? 2 : 1) * 32 * 32 * 4;
  static constexpr int STG_BYTES = GEMMK_EPI_WARPS * STG_WARP_BYTES;
  static constexpr int SMEM_LIMIT = 232448;  // 227 KB
  // The epilogue's staging buffers ALIAS the TMA ring: they are first written after the accumulator barrier, i.e. when
  // every MMA has read its stage and no TMA write is outstanding (a CTA computes one tile).  All of shared memory is
  // therefore ring: a small-batch main loop is bound by bytes in flight per SM (5 stages x 32 KB / ~1.1 us of DRAM
  // latency = the 140 GB/s per SM of the pipeline trace), so two more stages are worth more than a private staging area.
  static constexpr int STAGES_FIT = (SMEM_LIMIT - 1024 - BAR_BYTES) / STAGE_BYTES;
  static constexpr int STAGES = STAGES_FIT > 8 ? 8 : STAGES_FIT;
  static constexpr int SMEM_BYTES = STAGES * STAGE_BYTES + BAR_BYTES + 1024;
  static_assert(STAGES * STAGE_BYTES >= STG_BYTES, "staging must fit inside the ring it aliases");
  static constexpr int TMEM_COLS = BN;  // one accumulator: a CTA computes a single (partial) tile
  static_assert(STAGES >= 3 && 2 * STAGES + 2 <= BAR_BYTES / 8, "pipeline configuration");
};

__device__ __forceinline__ void tmem_st32(uint32_t taddr, const uint32_t (&r)[32]) {
  asm volatile(
      "tcgen05.st.sync.aligned.32x32b.x32.b32 [%0], {%1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15, "
      "%16, %17, %18, %19, %20, %21, %22, %23, %24, %25, %26, %27, %28, %29, %30, %31, %32};" ::"r"(taddr),
      "r"(r[0]), "r"(r[1]), "r"(r[2]), "r"(r[3]), "r"(r[4]), "r"(r[5]), "r"(r[6]), "r"(r[7]), "r"(r[8]), "r"(r[9]),
      "r"(r[10]), "r"(r[11]), "r"(r[12]), "r"(r[13]), "r"(r[14]), "r"(r[15]), "r"(r[16]), "r"(r[17]), "r"(r[18]),
      "r"(r[19]), "r"(r[20]), "r"(r[21]), "r"(r[22]), "r"(r[23]), "r"(r[24]), "r"(r[25]), "r"(r[26]), "r"(r[27]),
      "r"(r[28]), "r"(r[29]), "r"(r[30]), "r"(r[31])
      : "memory");
}
__device__ __forceinline__ void epi_bar_sync() {  // named barrier 1: the epilogue warps only
  asm volatile("bar.sync 1, %0;" ::"n"(32 * GEMMK_EPI_WARPS) : "memory");
}
__device__ __forceinline__ int ld_acquire_gpu(const int* p) {
  int v;
  asm volatile("ld.acquire.gpu.global.s32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
  return v;
}
__device__ __forceinline__ void red_release_gpu_add(int* p, int v) {
  asm volatile("red.release.gpu.global.add.s32 [%0], %1;" ::"l"(p), "r"(v) : "memory");
}

// ---------------------------------------------------------------- row-slice epilogues (split-K groups)
// A warp owns one row of the 128 x BN tile at a time: lane l holds columns 4l..4l+3 of each 128-column
// block v (NV = BN/128 blocks).  The S fp32 partials of the row are summed in the order 0..S-1; the
// arithmetic that follows restates the epilogues of te_gemm.cuh in this domain (per-head reductions and
// the rotary partner are warp shuffles).
// Epilogue operands of one batch of RB rows that do not depend on the accumulators (x, cos/sin, RMSNorm
// statistics, gains).  The first batch's are fetched BEFORE the CTA waits for its main loop and its group.
template <int NV, int RB>
struct SliceAux {
  float4 xv[RB][NV];
  float4 cs[RB], sn[RB];
  float rstd[RB];
  uint2 gn[NV];  // next norm's gain (EPI_RESID) / this head's QK-norm gain (EPI_QKV)
};
template <int BN, int EPI, int DH, int RB>
__device__ __forceinline__ void slice_aux_load(const GemmParams& p, int M, SliceAux<BN / 128, RB>& ax, int r0, int dr,
                                               int lane, int m_blk, int n_blk) {
  constexpr int NV = BN / 128;
  constexpr int HD2 = DH / 2;
  [[maybe_unused]] const int ch = (4 * lane) % DH;                      // lane's first column inside its head
  [[maybe_unused]] const int col0 = n_blk * BN + (4 * lane / DH) * DH;  // first column of the lane's head
  if constexpr (EPI == EPI_RESID) {
    if (p.g_next != nullptr) {
#pragma unroll
      for (int v = 0; v < NV; ++v)
        ax.gn[v] = __ldg(reinterpret_cast<const uint2*>(p.g_next + n_blk * BN + v * 128 + 4 * lane));
    }
  }
  if constexpr (EPI == EPI_QKV) ax.gn[0] = __ldg(reinterpret_cast<const uint2*>(((col0 < p.q_cols_end) ? p.gq : p.gk) + ch));
#pragma unroll
  for (int b = 0; b < RB; ++b) {
    const int r = r0 + b * dr;
    const int row = m_blk * GEMM_BM + r;
    const bool ok = r < GEMM_BM && row < M;
    if constexpr (EPI == EPI_RESID) {
#pragma unroll
      for (int v = 0; v < NV; ++v)
        if (ok) ax.xv[b][v] = ld_phase(reinterpret_cast<const float4*>(p.x + (size_t)row * p.ld_x + n_blk * BN + v * 128) + lane);
    }
    if constexpr (EPI == EPI_QKV) {
      if (ok) {
        ax.cs[b] = __ldg(reinterpret_cast<const float4*>(p.cos_t + (size_t)row * HD2 + (ch % HD2)));
        ax.sn[b] = __ldg(reinterpret_cast<const float4*>(p.sin_t + (size_t)row * HD2 + (ch % HD2)));
      }
    }
    if constexpr (EPI == EPI_QKV || EPI == EPI_SWIGLU) {
      // a row's parts are contiguous: lane i takes part i (branch-free for the usual <= 64 parts so that
      // the loads of all batch rows issue back to back)
      float sq = 0.f;
      if (ok) {
        const float* q = p.ssq_in + (size_t)row * p.ssq_stride;
        sq = (lane < p.ssq_parts) ? ld_phase(q + lane) : 0.f;
        sq += (lane + 32 < p.ssq_parts) ? ld_phase(q + lane + 32) : 0.f;
        for (int i = lane + 64; i < p.ssq_parts; i += 32) sq += ld_phase(q + i);
      }
      ax.rstd[b] = sq;
    }
  }
  // RMSNorm scale: lanes hold the parts round-robin -> fixed xor tree (deterministic)
  if constexpr (EPI == EPI_QKV || EPI == EPI_SWIGLU) {
#pragma unroll
    for (int b = 0; b < RB; ++b) {
      float sq = ax.rstd[b];
#pragma unroll
      for (int off = 1; off < 32; off <<= 1) sq += __shfl_xor_sync(0xffffffffu, sq, off);
      ax.rstd[b] = 1.0f / sqrtf(sq * p.inv_d + p.eps);
    }
  }
}

// One batch of RB rows (r0, r0 + dr, ...): the S partials of every row of the batch are requested before
// the first use, so a batch costs about one L2 round trip.  S * NV <= CAP float4 per row are in flight.
template <int BN, int EPI, int DH, int RB, int CAP>
__device__ __forceinline__ void slice_batch(const GemmParams& p, int M, const float* scratch, int S, int r0, int dr,
                                            int lane, int m_blk, int n_blk, const SliceAux<BN / 128, RB>& ax) {
  float* const x_dst = (EPI == EPI_RESID) ? resid_dst(p) : nullptr;
  constexpr int NV = BN / 128;
  constexpr int HD2 = DH / 2;
  constexpr int HL = DH / 4;  // lanes per head
  constexpr size_t TILE_F = (size_t)GEMM_BM * BN;
  const int snv = S * NV;
  int row[RB];
  bool ok[RB];
  float4 pv[RB][CAP];
#pragma unroll
  for (int b = 0; b < RB; ++b) {
    const int r = r0 + b * dr;
    row[b] = m_blk * GEMM_BM + r;
    ok[b] = r < GEMM_BM && row[b] < M;
#pragma unroll
    for (int q = 0; q < CAP; ++q)
      if (ok[b] && q < snv)
        pv[b][q] = __ldcg(reinterpret_cast<const float4*>(scratch + (size_t)(q / NV) * TILE_F + (size_t)r * BN +
                                                          (q % NV) * 128) + lane);
  }
  [[maybe_unused]] const int ch = (4 * lane) % DH;
  [[maybe_unused]] const int col0 = n_blk * BN + (4 * lane / DH) * DH;
  // ---- reduce (fixed order 0..S-1) + fused epilogue, row by row
#pragma unroll
  for (int b = 0; b < RB; ++b) {
    if (!ok[b]) continue;
    float4 acc[NV];
#pragma unroll
    for (int v = 0; v < NV; ++v) acc[v] = pv[b][v];
#pragma unroll
    for (int q = NV; q < CAP; ++q)
      if (q < snv) {
        float4& a = acc[q % NV];
        a.x += pv[b][q].x; a.y += pv[b][q].y; a.z += pv[b][q].z; a.w += pv[b][q].w;
      }
    if constexpr (EPI == EPI_PLAIN) {
#pragma unroll
      for (int v = 0; v < NV; ++v)
        *(reinterpret_cast<float4*>(p.c + (size_t)row[b] * p.ld_c + n_blk * BN + v * 128) + lane) = acc[v];
    }
    if constexpr (EPI == EPI_RESID) {
      float ss = 0.f;
#pragma unroll
      for (int v = 0; v < NV; ++v) {
        const int col = n_blk * BN + v * 128 + 4 * lane;
        float4 x = ax.xv[b][v];
        x.x += acc[v].x; x.y += acc[v].y; x.z += acc[v].z; x.w += acc[v].w;
        *reinterpret_cast<float4*>(x_dst + (size_t)row[b] * p.ld_x + col) = x;
        ss = fmaf(x.x, x.x, ss); ss = fmaf(x.y, x.y, ss); ss = fmaf(x.z, x.z, ss); ss = fmaf(x.w, x.w, ss);
        if (p.g_next != nullptr) {
          const uint2 g = ax.gn[v];
          uint2 o;
          o.x = pack_bf16(x.x * bf16_lo(g.x), x.y * bf16_hi(g.x));
          o.y = pack_bf16(x.z * bf16_lo(g.y), x.w * bf16_hi(g.y));
          *reinterpret_cast<uint2*>(p.xg + (size_t)row[b] * p.ld_x + col) = o;
        }
      }
#pragma unroll
      for (int off = 1; off < 32; off <<= 1) ss += __shfl_xor_sync(0xffffffffu, ss, off);
      if (lane == 0 && p.ssq_out != nullptr) {
        constexpr int NPARTS = GEMMK_EPI_WARPS / 4;  // the statistics keep the layout of the other GEMM kernels
        p.ssq_out[(size_t)row[b] * p.ssq_stride + n_blk * NPARTS] = ss;
#pragma unroll
        for (int i = 1; i < NPARTS; ++i) p.ssq_out[(size_t)row[b] * p.ssq_stride + n_blk * NPARTS + i] = 0.f;
      }
    }
    if constexpr (EPI == EPI_SWIGLU) {
      float4 g, u;
      if constexpr (NV == 2) {
        g = acc[0]; u = acc[1];
      } else {  // 128-wide tile: columns [0,64) gate, [64,128) up
        g = acc[0];
        u.x = __shfl_down_sync(0xffffffffu, acc[0].x, 16); u.y = __shfl_down_sync(0xffffffffu, acc[0].y, 16);
        u.z = __shfl_down_sync(0xffffffffu, acc[0].z, 16); u.w = __shfl_down_sync(0xffffffffu, acc[0].w, 16);
      }
      const float gv[4] = {g.x * ax.rstd[b], g.y * ax.rstd[b], g.z * ax.rstd[b], g.w * ax.rstd[b]};
      const float uv[4] = {u.x * ax.rstd[b], u.y * ax.rstd[b], u.z * ax.rstd[b], u.w * ax.rstd[b]};
      float a[4];
#pragma unroll
      for (int e = 0; e < 4; ++e) a[e] = __fdividef(gv[e], 1.0f + __expf(-gv[e])) * uv[e];
      uint2 o;
      o.x = pack_bf16(a[0], a[1]);
      o.y = pack_bf16(a[2], a[3]);
      if (NV == 2 || lane < 16)
        *reinterpret_cast<uint2*>(p.act + (size_t)row[b] * p.ld_act + n_blk * (BN / 2) + 4 * lane) = o;
    }
    if constexpr (EPI == EPI_QKV) {
      static_assert(EPI != EPI_QKV || NV == 1, "QKV split-K tiles are 128 columns wide");
      const float a4[4] = {acc[0].x, acc[0].y, acc[0].z, acc[0].w};
      float ss = 0.f;
#pragma unroll
      for (int e = 0; e < 4; ++e) {
        const float y = a4[e] * ax.rstd[b];
        ss = fmaf(y, y, ss);
      }
#pragma unroll
      for (int off = 1; off < HL; off <<= 1) ss += __shfl_xor_sync(0xffffffffu, ss, off);
      const float sc = ax.rstd[b] / sqrtf(ss * (1.0f / DH) + p.eps);
      const bool is_v = col0 >= p.k_cols_end;
      const uint2 g = ax.gn[0];
      const float gg[4] = {bf16_lo(g.x), bf16_hi(g.x), bf16_lo(g.y), bf16_hi(g.y)};
      const float c4[4] = {ax.cs[b].x, ax.cs[b].y, ax.cs[b].z, ax.cs[b].w};
      const float s4[4] = {ax.sn[b].x, ax.sn[b].y, ax.sn[b].z, ax.sn[b].w};
      float out[4];
#pragma unroll
      for (int e = 0; e < 4; ++e) {
        const float w = a4[e] * sc * gg[e];
        const float partner = __shfl_xor_sync(0xffffffffu, w, HL / 2);
        const float rot = (ch < HD2) ? (w * c4[e] - partner * s4[e]) : (w * c4[e] + partner * s4[e]);
        out[e] = is_v ? a4[e] * ax.rstd[b] : rot;
      }
      uint2 o;
      o.x = pack_bf16(out[0], out[1]);
      o.y = pack_bf16(out[2], out[3]);
      *reinterpret_cast<uint2*>(p.qkv + (size_t)row[b] * p.ld_qkv + n_blk * BN + 4 * lane) = o;
    }
  }
}

// Epilogue of a split-K group member, for one batch shape (RB rows per batch, CAP partial float4 per row).
// CTA s of the group finishes rows r = s (mod S) of the tile; its warp ew takes every 8th of them (16/S rows).
//   (0) prefetch the first batch's accumulator-independent operands
//   (1) wait for the own main loop, store the fp32 partial tile row-major to the L2 scratch
//   (2) meet the group at the tile's arrival counter
//   (3) batches: sum the S partials of each row in the fixed order 0..S-1, fused epilogue
template <int BN, int EPI, int DH, int RB, int CAP>
__device__ __forceinline__ void group_finish(const GemmParams& p, int M, uint64_t* tfull, uint32_t t_row, float* stg,
                                             float* scratch, int S, int s, int tile, int warp, int lane, int m_blk,
                                             int n_blk, uint32_t tfull_parity = 0) {
  constexpr int NV = BN / 128;
  constexpr int NPARTS = GEMMK_EPI_WARPS / 4;
  constexpr int COLS = BN / NPARTS;
  constexpr size_t TILE_F = (size_t)GEMM_BM * BN;
  const int ew = warp - 2, quad = warp & 3, part = ew >> 2;
  const int dr = GEMMK_EPI_WARPS * S;  // row stride between a warp's consecutive rows
  const int r_first = s + ew * S;
  const bool tr = warp == 2 && lane == 0;
  SliceAux<NV, RB> ax;
  slice_aux_load<BN, EPI, DH, RB>(p, M, ax, r_first, dr, lane, m_blk, n_blk);
  mbar_wait(tfull, tfull_parity);
  tc_fence_after();
  if (tr) trace_stamp(p, 5);
  {
    float* dst = scratch + (size_t)s * TILE_F + (size_t)(quad * 32) * BN;
    const int sub = lane >> 3, cq = lane & 7;
#pragma unroll 1
    for (int c0 = part * COLS; c0 < (part + 1) * COLS; c0 += 32) {
      uint32_t r[32];
      tmem_ld32(t_row + c0, r);
      tmem_ld_wait();
      float v[32];
#pragma unroll
      for (int j = 0; j < 32; ++j) v[j] = __uint_as_float(r[j]);
      stg_put_row(stg, lane, v);
      __syncwarp();
#pragma unroll
      for (int i = 0; i < 8; ++i) {
        const int rr = sub + 4 * i;
        __stcg(reinterpret_cast<float4*>(dst + (size_t)rr * BN + c0 + cq * 4), stg_get(stg, rr, cq));
      }
      __syncwarp();
    }
  }
  // bar.sync orders the warps' scratch stores before the elected thread's gpu-scope release
  epi_bar_sync();
  if (warp == 2 && lane == 0) {
    red_release_gpu_add(p.sk_sem + 2 * tile, 1);
    while (ld_acquire_gpu(p.sk_sem + 2 * tile) < S) {
    }
  }
  epi_bar_sync();
  if (tr) trace_stamp(p, 7);
  slice_batch<BN, EPI, DH, RB, CAP>(p, M, scratch, S, r_first, dr, lane, m_blk, n_blk, ax);
#pragma unroll 1
  for (int r0 = r_first + RB * dr; r0 < GEMM_BM; r0 += RB * dr) {
    slice_aux_load<BN, EPI, DH, RB>(p, M, ax, r0, dr, lane, m_blk, n_blk);
    slice_batch<BN, EPI, DH, RB, CAP>(p, M, scratch, S, r0, dr, lane, m_blk, n_blk, ax);
  }
  if (tr) trace_stamp(p, 9);
}

// Scratch layout: [tile][split][128 rows][BN] fp32, row-major (written coalesced through the staging
// transpose, read one whole row per warp).  Semaphores: sk_sem[2*tile] arrivals, [2*tile+1] departures.
// VAR: which epilogue the instantiation contains — 0: one CTA per tile (S == 1, fused epilogue from tensor memory);
// 1..6: the split-K group epilogue for one batch shape (gemmk_variant(epi, S * BN / 128) below, for S > 1).  One variant per kernel keeps the code
// of a launch compact: with all six in one kernel (150-280 KB of SASS) the epilogue, which every warp executes once
// and cold, was measurably slower.
__host__ __device__ constexpr int gemmk_variant(int epi, int snv) {
  return snv <= 1 ? 0 : ((epi != EPI_QKV && snv <= 2) ? 1 : ((epi != EPI_QKV && snv <= 3) ? 2 : (snv <= 4 ? 3 : (snv <= 6 ? 4 : (snv <= 8 ? 5 : 6)))));
}
template <int BN, int EPI, int DH, int VAR>
__global__ void __launch_bounds__(GEMMK_THREADS, 1)
te_gemmk_kernel(const __grid_constant__ CUtensorMap tmA, const __grid_constant__ CUtensorMap tmB, const GemmParams p) {
  using Cfg = GemmKCfg<BN, EPI>;
  constexpr int STAGES = Cfg::STAGES;
  extern __shared__ uint8_t smem_raw[];
  uint8_t* smem = reinterpret_cast<uint8_t*>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~uintptr_t(1023));
  uint8_t* sA = smem;
  uint8_t* sB = smem + STAGES * Cfg::A_BYTES;
  uint64_t* bars = reinterpret_cast<uint64_t*>(smem + STAGES * Cfg::STAGE_BYTES);
  uint64_t* full = bars;
  uint64_t* empty = bars + STAGES;
  uint64_t* tfull = bars + 2 * STAGES;
  uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(tfull + 1);
  float* stg_all = reinterpret_cast<float*>(smem);  // aliases the ring (see GemmKCfg)

  const int warp = threadIdx.x >> 5;
  const int lane = threadIdx.x & 31;
  if (threadIdx.x == 0) trace_stamp(p, 0);

  const int M = gemm_rows(p);
  const int S = p.splits;
  const int tile = blockIdx.x / S;
  const int s = blockIdx.x - tile * S;
  const int m_blk = tile % p.num_m_blk;
  const int n_blk = tile / p.num_m_blk;
  const int num_kb = p.K / GEMM_BK;
  const int kb0 = (s * num_kb) / S;
  const int kb1 = ((s + 1) * num_kb) / S;
  const int nkb = kb1 - kb0;
  // B tile of one k-block: BN weight rows in one box, or (gu_half: 128-wide SwiGLU tile over weights
  // interleaved per 256 rows; tmB then has 64-row boxes) the 64 gate rows and the 64 matching up rows
  auto load_b = [&](uint8_t* dst, uint64_t* bar, int kb) {
    if (p.gu_half) {
      const int g_row = (n_blk >> 1) * 256 + (n_blk & 1) * 64;
      tma_load_2d(dst, &tmB, bar, kb * GEMM_BK, g_row);
      tma_load_2d(dst + 64 * GEMM_BK * 2, &tmB, bar, kb * GEMM_BK, g_row + 128);
    } else {
      tma_load_2d(dst, &tmB, bar, kb * GEMM_BK, n_blk * BN);
    }
  };
  const int pre = nkb < STAGES ? nkb : STAGES;

  // The producer thread initialises the barriers itself and requests its first ring of WEIGHT tiles at once — they depend
  // on nothing, and at small batches their DRAM round trip (~1 us) is what the first MMA waits for — while warp 1
  // allocates tensor memory; the other warps see the barriers after the block barrier below.
  if (warp == 0 && elect_one()) {
    tma_prefetch_desc(&tmA);
    tma_prefetch_desc(&tmB);
    for (int i = 0; i < STAGES; ++i) {
      mbar_init(&full[i], 1);
      mbar_init(&empty[i], 1);
    }
    mbar_init(tfull, 1);
    fence_mbar_init();
    for (int i = 0; i < pre; ++i) {
      mbar_arrive_expect_tx(&full[i], Cfg::STAGE_BYTES);
      load_b(sB + i * Cfg::B_BYTES, &full[i], kb0 + i);
    }
  }
  if (warp == 1) tmem_alloc(tmem_slot, Cfg::TMEM_COLS);
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tmem_base = *tmem_slot;
  pdl_launch_dependents();
  if (threadIdx.x == 0) trace_stamp(p, 1);

  if (warp == 0) {
    // ===================== TMA producer =====================
    if (elect_one()) {
      pdl_wait();
      trace_stamp(p, 2);
      int stage = 0;
      uint32_t phase = 0;
      for (int i = 0; i < nkb; ++i) {
        if (i >= pre) {
          mbar_wait(&empty[stage], phase ^ 1);
          mbar_arrive_expect_tx(&full[stage], Cfg::STAGE_BYTES);
          load_b(sB + stage * Cfg::B_BYTES, &full[stage], kb0 + i);
        }
        tma_load_2d(sA + stage * Cfg::A_BYTES, &tmA, &full[stage], (kb0 + i) * GEMM_BK, m_blk * GEMM_BM);
        if (++stage == STAGES) { stage = 0; phase ^= 1; }
      }
    }
  } else if (warp == 1) {
    // ===================== MMA issuer =====================
    if (elect_one()) {
      constexpr uint32_t idesc = umma_idesc_bf16(GEMM_BM, BN);
      int stage = 0;
      uint32_t phase = 0;
      for (int i = 0; i < nkb; ++i) {
        mbar_wait(&full[stage], phase);
        if (i == 0) trace_stamp(p, 3);
        tc_fence_after();
        const uint64_t a_desc = umma_smem_desc_sw128(smem_u32(sA + stage * Cfg::A_BYTES));
        const uint64_t b_desc = umma_smem_desc_sw128(smem_u32(sB + stage * Cfg::B_BYTES));
#pragma unroll
        for (int k = 0; k < GEMM_BK / 16; ++k)
          umma_bf16(tmem_base, a_desc + 2 * k, b_desc + 2 * k, idesc, (i | k) != 0 ? 1u : 0u);
        umma_commit(&empty[stage]);
        if (++stage == STAGES) { stage = 0; phase ^= 1; }
      }
      umma_commit(tfull);
      trace_stamp(p, 4);
    }
  } else {
    // ===================== epilogue warps =====================
    const int quad = warp & 3;         // TMEM lane quadrant this warp may access
    const int part = (warp - 2) >> 2;  // which half of the tile's columns (two warps per quadrant)
    constexpr int NPARTS = GEMMK_EPI_WARPS / 4;
    constexpr int COLS = BN / NPARTS;
    const int row_base = m_blk * GEMM_BM + quad * 32;
    const uint32_t t_row = tmem_base + (static_cast<uint32_t>(quad * 32) << 16);
    float* stg = stg_all + (warp - 2) * (Cfg::STG_WARP_BYTES / 4);
    const bool tr = warp == 2 && lane == 0;
    pdl_wait();
    if constexpr (VAR == 0) {
      // ---- one CTA per tile: fused epilogue straight from tensor memory
      float rstd = 0.f;
      ResidPrefetch pf;
      if constexpr (EPI == EPI_QKV || EPI == EPI_SWIGLU) rstd = row_rstd(p, row_base + lane, row_base + lane < M);
      if constexpr (EPI == EPI_RESID) resid_issue<BN>(p, M, pf, row_base, lane, n_blk, part * COLS);
      mbar_wait(tfull, 0);
      tc_fence_after();
      if (tr) trace_stamp(p, 5);
      if constexpr (EPI == EPI_PLAIN) epi_plain<BN>(p, t_row, row_base + lane, row_base + lane < M, n_blk, part, NPARTS);
      if constexpr (EPI == EPI_RESID) epi_resid<BN>(p, M, t_row, row_base, lane, n_blk, stg, part, NPARTS, pf);
      if constexpr (EPI == EPI_SWIGLU) epi_swiglu<BN>(p, M, t_row, row_base, lane, n_blk, stg, part, NPARTS, rstd);
      if constexpr (EPI == EPI_QKV) epi_qkv<BN, DH>(p, M, t_row, row_base, lane, n_blk, stg, part, NPARTS, rstd);
      if (tr) trace_stamp(p, 9);
    } else {
      // ---- split-K group (see group_finish).  The batch shape is chosen so that all partials of a batch
      // (RB rows x S*NV float4) fit in ~16-18 float4 per lane: for 128-wide tiles a warp's 16/S rows are a
      // single batch.  (EPI_QKV also keeps a cos/sin row per batch row: at most 4 rows per batch there.)
      float* scratch = p.sk_scratch + (size_t)tile * S * GEMM_BM * BN;
#define TE_GROUP_FINISH(RB, CAP) \
  group_finish<BN, EPI, DH, RB, CAP>(p, M, tfull, t_row, stg, scratch, S, s, tile, warp, lane, m_blk, n_blk)
      if constexpr (VAR == 1) { TE_GROUP_FINISH(8, 2); }
      else if constexpr (VAR == 2) { TE_GROUP_FINISH(6, 3); }
      else if constexpr (VAR == 3) { TE_GROUP_FINISH(4, 4); }
      else if constexpr (VAR == 4) { TE_GROUP_FINISH(3, 6); }
      else if constexpr (VAR == 5) { TE_GROUP_FINISH(2, 8); }
      else { TE_GROUP_FINISH(1, 16); }
#undef TE_GROUP_FINISH
      // the last CTA of the group to leave re-arms both counters for the next launch
      epi_bar_sync();
      if (warp == 2 && lane == 0) {
        if (atomicAdd(p.sk_sem + 2 * tile + 1, 1) == S - 1) {
          p.sk_sem[2 * tile] = 0;
          p.sk_sem[2 * tile + 1] = 0;
        }
      }
    }
  }
  tc_fence_before();
  __syncwarp();  // the elected producer / MMA lanes rejoin their warps before the block barrier
  __syncthreads();
  if (threadIdx.x == 0) trace_stamp(p, 10);
  if (warp == 1) {
    tc_fence_after();
    tmem_dealloc(tmem_base, Cfg::TMEM_COLS);
  }
}

}  // namespace te
