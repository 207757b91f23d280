// te_gemm_chain.cuh — several small-batch GEMMs of a layer in ONE persistent launch (SURVEY.md §8(a) a7 / §7 "launch
// overhead"; VERDICT r1 "remove the kernel boundaries" at B <= 4).
//
// Below ~512 tokens every GEMM of the stack is one wave of 128 x 128 split-K tiles (te_gemm_splitk.cuh) and a launch
// costs more in fixed latencies than in work: the pipeline trace at cfg 3 shows ~2 us from CTA start to the first MMA
// (barrier init, TMEM allocation, first TMA round trip), 1.3-1.5 us of CTA turnover to the next kernel, against 3-11 us
// main loops.  When consecutive GEMMs all use that tile shape — O-proj -> gate/up -> down -> next layer's QKV at
// T <= 128, down -> next QKV at T = 512 — this kernel runs them as PHASES of one cooperative grid:
//   * barriers, tensor memory and the TMA ring are set up once; the ring's stage / parity counters run on across phases;
//   * between phases the grid meets at a global arrival counter (release-add by one thread per CTA after its epilogue
//     stores, acquire-spin by the producer thread and by the epilogue warps' leader); the producer requests the next
//     phase's first ring of WEIGHT tiles before it waits there — they do not depend on the previous phase — and the
//     activation tiles after it (behind a generic->async proxy fence: they were written with ordinary stores);
//   * a phase's tile assignment, split-K exchange and fused epilogue are exactly te_gemmk_kernel's (same device
//     functions), chosen per phase at run time from {residual, SwiGLU, QKV}.
// CTAs beyond a phase's tiles * splits idle through it but still take part in the barriers.  The counter is re-armed by
// the last CTA to leave the kernel.  All phases use BN = 128 (one accumulator of 128 TMEM columns).
#pragma once
#include <type_traits>

#include "te_gemm_splitk.cuh"

namespace te {

constexpr int CHAIN_MAX_PHASES = 4;
constexpr int CHAIN_STAGES = 5;
constexpr int CHAIN_SMEM_BYTES = CHAIN_STAGES * (GEMM_BM * GEMM_BK * 2 + 128 * GEMM_BK * 2) + 256 + GEMMK_EPI_WARPS * 2 * 32 * 32 * 4 + 1024;

struct ChainParams {
  GemmParams p[CHAIN_MAX_PHASES];
  int epi[CHAIN_MAX_PHASES];
  int n_phases;
  int* gbar;  // [2] arrival counter of the grid barriers, departure counter (both zero between launches)
};

template <int EPI, int DH>
__device__ __forceinline__ void chain_group_finish(const GemmParams& p, int M, uint64_t* tfull, uint32_t par, uint32_t t_row,
                                                   float* stg, float* scratch, int S, int s, int tile, int warp, int lane,
                                                   int m_blk, int n_blk) {
#define TE_CHAIN_FINISH(RB, CAP) \
  group_finish<128, EPI, DH, RB, CAP>(p, M, tfull, t_row, stg, scratch, S, s, tile, warp, lane, m_blk, n_blk, par)
  if (EPI != EPI_QKV && S <= 2) { TE_CHAIN_FINISH(8, 2); }
  else if (EPI != EPI_QKV && S <= 3) { TE_CHAIN_FINISH(6, 3); }
  else if (S <= 4) { TE_CHAIN_FINISH(4, 4); }
  else if (S <= 6) { TE_CHAIN_FINISH(3, 6); }
  else { TE_CHAIN_FINISH(2, 8); }
#undef TE_CHAIN_FINISH
}

// One phase's epilogue for an ACTIVE CTA (tile, s): te_gemmk_kernel's epilogue branch.
template <int EPI, int DH>
__device__ __forceinline__ void chain_epilogue(const GemmParams& p, int M, uint64_t* tfull, uint32_t par, uint32_t tmem_base,
                                               float* stg, int S, int s, int tile, int warp, int lane, int m_blk, int n_blk) {
  constexpr int BN = 128;
  constexpr int NPARTS = GEMMK_EPI_WARPS / 4;
  constexpr int COLS = BN / NPARTS;
  const int quad = warp & 3, part = (warp - 2) >> 2;
  const int row_base = m_blk * GEMM_BM + quad * 32;
  const uint32_t t_row = tmem_base + (static_cast<uint32_t>(quad * 32) << 16);
  if (S == 1) {
    float rstd = 0.f;
    ResidPrefetch pf;
    if constexpr (EPI == EPI_QKV || EPI == EPI_SWIGLU) rstd = row_rstd(p, row_base + lane, row_base + lane < M);
    if constexpr (EPI == EPI_RESID) resid_issue<BN>(p, M, pf, row_base, lane, n_blk, part * COLS);
    mbar_wait(tfull, par);
    tc_fence_after();
    if constexpr (EPI == EPI_RESID) epi_resid<BN>(p, M, t_row, row_base, lane, n_blk, stg, part, NPARTS, pf);
    if constexpr (EPI == EPI_SWIGLU) epi_swiglu<BN>(p, M, t_row, row_base, lane, n_blk, stg, part, NPARTS, rstd);
    if (warp == 2 && lane == 0) trace_stamp(p, 14);
    if constexpr (EPI == EPI_QKV) epi_qkv<BN, DH>(p, M, t_row, row_base, lane, n_blk, stg, part, NPARTS, rstd, warp == 2 && lane == 0);
    if (warp == 2 && lane == 0) trace_stamp(p, 25);
  } else {
    float* scratch = p.sk_scratch + (size_t)tile * S * GEMM_BM * BN;
    chain_group_finish<EPI, DH>(p, M, tfull, par, t_row, stg, scratch, S, s, tile, warp, lane, m_blk, n_blk);
    epi_bar_sync();
    if (warp == 2 && lane == 0) {  // the last CTA of the group to leave re-arms the tile's counters
      if (atomicAdd(p.sk_sem + 2 * tile + 1, 1) == S - 1) {
        p.sk_sem[2 * tile] = 0;
        p.sk_sem[2 * tile + 1] = 0;
      }
    }
  }
}

__device__ __forceinline__ void fence_proxy_async_all() { asm volatile("fence.proxy.async;" ::: "memory"); }

// FOUR: phases = {residual, SwiGLU, residual, QKV} (O-proj, gate/up, down, next QKV; n_phases 3 or 4);
// else {residual, QKV} (down, next QKV).  The epilogue of every phase is its own straight-line region with a
// compile-time epilogue kind (a run-time switch over the three kinds cost 8 KB of register spills).
template <int DH, bool FOUR>
__global__ void __launch_bounds__(GEMMK_THREADS, 1)
te_gemmk_chain_kernel(const __grid_constant__ CUtensorMap tmA0, const __grid_constant__ CUtensorMap tmB0,
                      const __grid_constant__ CUtensorMap tmA1, const __grid_constant__ CUtensorMap tmB1,
                      const __grid_constant__ CUtensorMap tmA2, const __grid_constant__ CUtensorMap tmB2,
                      const __grid_constant__ CUtensorMap tmA3, const __grid_constant__ CUtensorMap tmB3,
                      const __grid_constant__ ChainParams cp) {
  using Cfg = GemmKCfg<128, EPI_QKV>;  // the largest staging area of the three epilogues
  constexpr int BN = 128;
  constexpr int STAGES = CHAIN_STAGES;  // (private staging here: the next phase's weights land in the ring during an epilogue)
  extern __shared__ uint8_t smem_raw[];
  uint8_t* smem = reinterpret_cast<uint8_t*>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~uintptr_t(1023));
  uint8_t* sA = smem;
  uint8_t* sB = smem + STAGES * Cfg::A_BYTES;
  uint64_t* bars = reinterpret_cast<uint64_t*>(smem + STAGES * Cfg::STAGE_BYTES);
  uint64_t* full = bars;
  uint64_t* empty = bars + STAGES;
  uint64_t* tfull = bars + 2 * STAGES;
  uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(tfull + 1);
  float* stg_all = reinterpret_cast<float*>(smem + STAGES * Cfg::STAGE_BYTES + Cfg::BAR_BYTES);

  const int warp = threadIdx.x >> 5;
  const int lane = threadIdx.x & 31;
  const int G = gridDim.x;

  if (warp == 0 && elect_one()) {
    tma_prefetch_desc(&tmA0); tma_prefetch_desc(&tmB0);
    tma_prefetch_desc(&tmA1); tma_prefetch_desc(&tmB1);
    if (cp.n_phases > 2) { tma_prefetch_desc(&tmA2); tma_prefetch_desc(&tmB2); }
    if (cp.n_phases > 3) { tma_prefetch_desc(&tmA3); tma_prefetch_desc(&tmB3); }
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
    tmem_alloc(tmem_slot, Cfg::TMEM_COLS);
  }
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tmem_base = *tmem_slot;
  pdl_launch_dependents();

  // what CTA blockIdx.x does in phase ph
  auto active = [&](int ph, int& tile, int& s, int& nkb, int& kb0) {
    const GemmParams& p = cp.p[ph];
    const int S = p.splits;
    const int tiles = p.num_m_blk * p.num_n_blk;
    tile = blockIdx.x / S;
    s = blockIdx.x - tile * S;
    const int num_kb = p.K / GEMM_BK;
    kb0 = (s * num_kb) / S;
    nkb = ((s + 1) * num_kb) / S - kb0;
    return tile < tiles;
  };
  auto maps = [&](int ph, const CUtensorMap*& a, const CUtensorMap*& b) {
    a = ph == 0 ? &tmA0 : (ph == 1 ? &tmA1 : (ph == 2 ? &tmA2 : &tmA3));
    b = ph == 0 ? &tmB0 : (ph == 1 ? &tmB1 : (ph == 2 ? &tmB2 : &tmB3));
  };

  if (warp == 0) {
    // ===================== TMA producer =====================
    if (elect_one()) {
      uint32_t it = 0;  // k-blocks issued so far by this CTA, over all phases: stage = it % STAGES, use = it / STAGES
      for (int ph = 0; ph < cp.n_phases; ++ph) {
        const GemmParams& p = cp.p[ph];
        int tile, s, nkb, kb0;
        const bool on = active(ph, tile, s, nkb, kb0);
        const CUtensorMap *tA, *tB;
        maps(ph, tA, tB);
        const int m_blk = on ? tile % p.num_m_blk : 0, n_blk = on ? tile / p.num_m_blk : 0;
        auto load_b = [&](uint8_t* dst, uint64_t* bar, int kb) {
          if (p.gu_half) {
            const int g_row = (n_blk >> 1) * 256 + (n_blk & 1) * 64;
            tma_load_2d(dst, tB, bar, kb * GEMM_BK, g_row);
            tma_load_2d(dst + 64 * GEMM_BK * 2, tB, bar, kb * GEMM_BK, g_row + 128);
          } else {
            tma_load_2d(dst, tB, bar, kb * GEMM_BK, n_blk * BN);
          }
        };
        const int pre = on ? (nkb < STAGES ? nkb : STAGES) : 0;
        for (int i = 0; i < pre; ++i) {  // weights first: they depend on nothing this launch or its predecessors write
          const uint32_t st = (it + i) % STAGES, use = (it + i) / STAGES;
          if (use > 0) mbar_wait(&empty[st], (use - 1) & 1);
          mbar_arrive_expect_tx(&full[st], Cfg::STAGE_BYTES);
          load_b(sB + st * Cfg::B_BYTES, &full[st], kb0 + i);
        }
        trace_stamp(p, 1);
        if (ph == 0) {
          pdl_wait();
        } else if (on) {  // (an idle CTA's producer must not linger here: the counter is re-armed at the kernel's end)
          while (ld_acquire_gpu(cp.gbar) < ph * G) __nanosleep(40);
          fence_proxy_async_all();  // the previous phase's activations were written by ordinary stores; TMA reads them
        }
        trace_stamp(p, 2);
        for (int i = 0; i < (on ? nkb : 0); ++i) {
          const uint32_t st = (it + i) % STAGES, use = (it + i) / STAGES;
          if (i >= pre) {
            if (use > 0) mbar_wait(&empty[st], (use - 1) & 1);
            mbar_arrive_expect_tx(&full[st], Cfg::STAGE_BYTES);
            load_b(sB + st * Cfg::B_BYTES, &full[st], kb0 + i);
          }
          tma_load_2d(sA + st * Cfg::A_BYTES, tA, &full[st], (kb0 + i) * GEMM_BK, m_blk * GEMM_BM);
        }
        if (on) it += nkb;
      }
    }
  } else if (warp == 1) {
    // ===================== MMA issuer =====================
    if (elect_one()) {
      constexpr uint32_t idesc = umma_idesc_bf16(GEMM_BM, BN);
      uint32_t it = 0;
      for (int ph = 0; ph < cp.n_phases; ++ph) {
        int tile, s, nkb, kb0;
        if (!active(ph, tile, s, nkb, kb0)) continue;
        // (the accumulator of the previous phase has been read out: this phase's activation tiles are requested only
        //  after the grid barrier, at which this CTA arrives after its own epilogue)
        for (int i = 0; i < nkb; ++i, ++it) {
          const uint32_t st = it % STAGES, use = it / STAGES;
          mbar_wait(&full[st], use & 1);
          if (i == 0) trace_stamp(cp.p[ph], 3);
          tc_fence_after();
          const uint64_t a_desc = umma_smem_desc_sw128(smem_u32(sA + st * Cfg::A_BYTES));
          const uint64_t b_desc = umma_smem_desc_sw128(smem_u32(sB + st * Cfg::B_BYTES));
#pragma unroll
          for (int k = 0; k < GEMM_BK / 16; ++k)
            umma_bf16(tmem_base, a_desc + 2 * k, b_desc + 2 * k, idesc, (i | k) != 0 ? 1u : 0u);
          umma_commit(&empty[st]);
        }
        umma_commit(tfull);
        trace_stamp(cp.p[ph], 4);
      }
    }
  } else {
    // ===================== epilogue warps =====================
    float* stg = stg_all + (warp - 2) * (Cfg::STG_WARP_BYTES / 4);
    uint32_t n_done = 0;  // phases in which this CTA had a tile: parity of tfull
    pdl_wait();
    auto run_phase = [&](auto ph_c, auto epi_c) {
      constexpr int ph = decltype(ph_c)::value;
      constexpr int EPI = decltype(epi_c)::value;
      const GemmParams& p = cp.p[ph];
      if (ph > 0) {  // everything this phase's epilogue reads ahead of its accumulator was written by the previous phase
        if (warp == 2 && lane == 0) {
          while (ld_acquire_gpu(cp.gbar) < ph * G) __nanosleep(40);
          trace_stamp(p, 13);
        }
        epi_bar_sync();  // (what the phase reads of its predecessor's output is read through L2: __ldcg / TMA)
      }
      int tile, s, nkb, kb0;
      if (active(ph, tile, s, nkb, kb0)) {
        const int M = gemm_rows(p);
        const int m_blk = tile % p.num_m_blk, n_blk = tile / p.num_m_blk;
        chain_epilogue<EPI, DH>(p, M, tfull, n_done & 1, tmem_base, stg, p.splits, s, tile, warp, lane, m_blk, n_blk);
        ++n_done;
      }
      // arrive at the grid barrier that ends this phase (the last phase's is the kernel's end)
      tc_fence_before();
      epi_bar_sync();  // all epilogue warps' stores are issued (and ordered before the elected thread's release)
      if (warp == 2 && lane == 0) trace_stamp(p, 11);
      if (ph + 1 < cp.n_phases && warp == 2 && lane == 0) red_release_gpu_add(cp.gbar, 1);
      if (warp == 2 && lane == 0) trace_stamp(p, 12);
    };
    using std::integral_constant;
    if constexpr (FOUR) {
      run_phase(integral_constant<int, 0>{}, integral_constant<int, EPI_RESID>{});
      run_phase(integral_constant<int, 1>{}, integral_constant<int, EPI_SWIGLU>{});
      run_phase(integral_constant<int, 2>{}, integral_constant<int, EPI_RESID>{});
      if (cp.n_phases > 3) run_phase(integral_constant<int, 3>{}, integral_constant<int, EPI_QKV>{});
    } else {
      run_phase(integral_constant<int, 0>{}, integral_constant<int, EPI_RESID>{});
      run_phase(integral_constant<int, 1>{}, integral_constant<int, EPI_QKV>{});
    }
    // the last CTA to leave re-arms the barrier counters for the next launch
    if (warp == 2 && lane == 0) {
      if (atomicAdd(cp.gbar + 1, 1) == G - 1) {
        cp.gbar[0] = 0;
        cp.gbar[1] = 0;
      }
    }
  }
  tc_fence_before();
  __syncwarp();
  __syncthreads();
  if (warp == 1) {
    tc_fence_after();
    tmem_dealloc(tmem_base, Cfg::TMEM_COLS);
  }
}

}  // namespace te
