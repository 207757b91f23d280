// te_attn_tc.cuh — causal GQA attention prefill on the 5th-gen tensor cores:
// per frame b and q head a (kv head a / G): P = softmax(q k^T / sqrt(dh) + causal), o = P v,
// fp32 softmax, causal by sequence index within the frame, varlen-packed frames.
//
// Frames are short (S_b <= 256), so one CTA owns one (frame, kv head): its K and V (<= 256 keys)
// are fetched ONCE by TMA and stay in shared memory, and the G = Hq/Hkv query heads that share them
// are stacked into 128-row query tiles (128/G consecutive positions x G heads).  Per tile:
//   S = Q K^T      tcgen05.mma, A = Q and B = K from shared memory (K-major, 128B swizzle), fp32 S in TMEM
//   softmax        one thread per row reads S from TMEM (tcgen05.ld), two passes (max, then exp2 and sum),
//                  and writes P as packed bf16 BACK INTO TMEM over the columns of S (tcgen05.st)
//   O = P V        tcgen05.mma with A = P from TMEM and B = V from shared memory as stored ([keys, dh],
//                  MN-major descriptor) -> no transpose of V and no shared-memory round trip for P
//   epilogue       O / rowsum -> bf16 -> global
// Only the keys a tile can see are multiplied (N = K-extent = 64 * (tile + 1) for G = 2).
// Warp roles (320 threads): warp 0 = TMA producer, warp 1 = TMEM allocator + MMA issuer, warps 2-5 and
// 6-9 = two softmax groups that alternate tiles (each tile has its own 256-column TMEM buffer: S in
// [0, nk), P packed over [0, nk/2), O in [128, 128 + dh)), so the tensor core, the softmax of one
// tile and the epilogue of the previous one overlap.
#pragma once
#include "te_gemm8.cuh"  // MXFP8 quantiser of the output (te_config.weight_dtype = 1)
#include "te_ptx.cuh"

namespace te {

struct AttnTcParams {
  __nv_bfloat16* out;         // [T, Hq*DH]
  const int32_t* cu_seqlens;  // [B+1]
  int n_q_heads, n_kv_heads;
  int g_shift;  // log2(Hq / Hkv)
  float scale_log2;  // log2(e) / sqrt(dh)
  int non_causal;    // 1: every query sees all keys of its frame (vision tower, te_config.non_causal); 0: causal
  // Shared text prefix (te_encode_prefix), handled as a SECOND launch of this kernel per layer:
  //   launch 1 (prefix_mode 0, stats != null): frame-local causal attention as usual, plus the row statistics
  //            (max raw score, sum of exp) of every (token, q head) -> stats[T, Hq]
  //   launch 2 (prefix_mode 1): tmKV addresses the layer's prefix cache [P, 2*Hkv*dh] (k heads | v heads); every
  //            query sees all P keys (no mask); the epilogue merges with launch 1's normalised fp32 output (o32):
  //            out = (l_f e^(m_f-m) out_f + e^(m_p-m) O_p) / (l_f e^(m_f-m) + l_p e^(m_p-m)),  m = max(m_f, m_p)
  float2* stats;
  float* o32;  // [T, Hq*DH] fp32: launch 1 leaves its normalised output HERE (not in `out`) when a prefix pass follows, and
               // launch 2 blends in fp32 and rounds to bf16 ONCE (round 1 blended two bf16-rounded values)
  int prefix_mode;
  int prefix_len;
  // MXFP8 variant: the output (= A operand of the O projection) is written as E4M3 + block scales instead of bf16
  uint8_t* out8;    // [T, Hq*DH] or null
  uint8_t* sf_out;  // tiled scales (te_gemm8.cuh)
  unsigned long long* trace;  // TE_OPT_TRACE: [trace_ctas][TRACE_SLOTS] stamps (null: off)
  int trace_ctas;
};

template <int DH>
struct AttnTcCfg {
  static constexpr int KMAX = 256;  // max keys per frame (te_config.max_tokens_per_frame <= 256)
  static constexpr int SLABS = DH / 64;                   // 64-element (128 B) column slabs per row
  static constexpr int KV_SLAB_BYTES = KMAX * 128;        // one slab of K (or V): KMAX rows x 128 B
  static constexpr int KV_BYTES = SLABS * KV_SLAB_BYTES;  // all of K (or V)
  static constexpr int KV_BLOCK_BYTES = 64 * DH * 2;      // one 64-key block (all slabs)
  static constexpr int Q_SLAB_BYTES = 128 * 128;
  static constexpr int Q_BYTES = SLABS * Q_SLAB_BYTES;    // one 128-row query tile
  static constexpr int BAR_BYTES = 256;
  static constexpr int SMEM_NEEDED = 2 * KV_BYTES + 2 * Q_BYTES + BAR_BYTES + 1024;
  // one CTA per SM (each allocates the whole TMEM): never request less than half the SM's shared memory
  static constexpr int SMEM_BYTES = SMEM_NEEDED > 120 * 1024 ? SMEM_NEEDED : 120 * 1024;
  static constexpr int THREADS = 320;
  static constexpr int TMEM_COLS = 512;
  static constexpr int O_COL = 128;  // column of O inside a tile's 256-column buffer
};

__device__ __forceinline__ float ex2_approx(float x) {
  float y;
  asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
  return y;
}

// grid: (n_split, Hkv, B); CTA (split, kvh, b) handles query tiles split, split + n_split, ... of frame b.
template <int DH>
__global__ void __launch_bounds__(320, 1)
te_attn_tc_kernel(const __grid_constant__ CUtensorMap tmQ, const __grid_constant__ CUtensorMap tmKV,
                  const AttnTcParams p) {
  using Cfg = AttnTcCfg<DH>;
  constexpr int SLABS = Cfg::SLABS;
  extern __shared__ uint8_t attn_tc_smem[];
  uint8_t* smem = reinterpret_cast<uint8_t*>((reinterpret_cast<uintptr_t>(attn_tc_smem) + 1023) & ~uintptr_t(1023));
  uint8_t* sK = smem;
  uint8_t* sV = sK + Cfg::KV_BYTES;
  uint8_t* sQ = sV + Cfg::KV_BYTES;
  uint64_t* bars = reinterpret_cast<uint64_t*>(sQ + 2 * Cfg::Q_BYTES);
  uint64_t* k_full = bars;          // [4] one-shot, one per 64-key block
  uint64_t* v_full = bars + 4;      // [4]
  uint64_t* q_full = bars + 8;      // [2] query-tile ring
  uint64_t* q_empty = bars + 10;    // [2]
  uint64_t* s_full = bars + 12;     // [2] S = Q K^T landed in TMEM buffer t
  uint64_t* p_full = bars + 14;     // [2] P written to TMEM buffer t (128 arrivals)
  uint64_t* o_full = bars + 16;     // [2] O = P V landed
  uint64_t* buf_free = bars + 18;   // [2] O read out, buffer t reusable (128 arrivals)
  uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(bars + 20);

  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int split = blockIdx.x, n_split = gridDim.x, kvh = blockIdx.y, b = blockIdx.z;
  const int g_shift = p.g_shift;
  const int cta_lin = blockIdx.x + gridDim.x * (blockIdx.y + gridDim.y * blockIdx.z);
  auto stamp = [&](int slot) {  // TE_OPT_TRACE (debug): slot 0 start, 1 set up, 2 past the dependency wait, per tile i < 4:
    // 3+5i scores ready, 4+5i pass 1 done, 5+5i P written, 6+5i O ready, 7+5i stored; 37 end
    if (p.trace != nullptr && cta_lin < p.trace_ctas) {
      unsigned long long t;
      asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t)::"memory");
      p.trace[(size_t)cta_lin * TRACE_SLOTS + slot] = t;
      p.trace[(size_t)cta_lin * TRACE_SLOTS + 48 + slot] = static_cast<unsigned long long>(clock64());
    }
  };
  if (threadIdx.x == 0) stamp(0);
  const int G = 1 << g_shift;
  const int PT = 128 >> g_shift;  // positions per query tile

  if (warp == 0 && elect_one()) {
    tma_prefetch_desc(&tmQ);
    tma_prefetch_desc(&tmKV);
  }
  if (warp == 1) {
    if (elect_one()) {
      for (int i = 0; i < 8; ++i) mbar_init(&k_full[i], 1);  // k_full[0..3], v_full[0..3]
      for (int i = 0; i < 2; ++i) {
        mbar_init(&q_full[i], 1);
        mbar_init(&q_empty[i], 1);
        mbar_init(&s_full[i], 1);
        mbar_init(&p_full[i], 128);
        mbar_init(&o_full[i], 1);
        mbar_init(&buf_free[i], 128);
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
  pdl_launch_dependents();
  if (threadIdx.x == 0) stamp(1);
  pdl_wait();  // qkv and cu_seqlens are written by predecessor kernels
  if (threadIdx.x == 0) stamp(2);

  const int seq0 = p.cu_seqlens[b];
  // (a frame longer than KMAX raised the device validation flag in te_scan_kernel; clamp so that the
  //  shared-memory tiles are never overrun)
  const int S = min(p.cu_seqlens[b + 1] - seq0, Cfg::KMAX);  // (offsets are clamped to the token count by te_prep_kernel)
  const int n_tiles = (S + PT - 1) / PT;
  const int n_my = (n_tiles > split) ? (n_tiles - split + n_split - 1) / n_split : 0;
  const int S16 = (S + 15) & ~15;
  const int P16 = (p.prefix_len + 15) & ~15;
  // keys tile j can see: positions < PT * (j + 1), rounded to the MMA granularity (16) and capped at the frame;
  // prefix mode: all P prefix keys for every tile
  auto nk_of = [&](int j) { return p.prefix_mode ? P16 : (p.non_causal ? S16 : min(S16, (PT * (j + 1) + 15) & ~15)); };
  const int kv_row0 = p.prefix_mode ? 0 : seq0;                                   // first K/V row in tmKV
  const int k_col0 = (p.prefix_mode ? kvh : p.n_q_heads + kvh) * DH;              // this kv head's K columns
  const int v_col0 = (p.prefix_mode ? p.n_kv_heads + kvh : p.n_q_heads + p.n_kv_heads + kvh) * DH;

  if (warp == 0) {
    // ===================== TMA producer =====================
    if (n_my > 0 && elect_one()) {
      const int j_last = split + (n_my - 1) * n_split;
      const int nkb = (nk_of(j_last) + 63) >> 6;
      auto load_q = [&](int i) {
        const int slot = i & 1, u = i >> 1;
        if (u > 0) mbar_wait(&q_empty[slot], (u - 1) & 1);
        mbar_arrive_expect_tx(&q_full[slot], Cfg::Q_BYTES);
        const int j = split + i * n_split;
        for (int hl = 0; hl < G; ++hl)
          for (int s = 0; s < SLABS; ++s)
            tma_load_2d(sQ + slot * Cfg::Q_BYTES + s * Cfg::Q_SLAB_BYTES + hl * PT * 128, &tmQ, &q_full[slot],
                        ((kvh << g_shift) + hl) * DH + 64 * s, seq0 + j * PT);
      };
      load_q(0);
      for (int kb = 0; kb < nkb; ++kb) {
        mbar_arrive_expect_tx(&k_full[kb], Cfg::KV_BLOCK_BYTES);
        for (int s = 0; s < SLABS; ++s)
          tma_load_2d(sK + s * Cfg::KV_SLAB_BYTES + kb * 8192, &tmKV, &k_full[kb], k_col0 + 64 * s, kv_row0 + 64 * kb);
      }
      if (n_my > 1) load_q(1);
      for (int kb = 0; kb < nkb; ++kb) {
        mbar_arrive_expect_tx(&v_full[kb], Cfg::KV_BLOCK_BYTES);
        for (int s = 0; s < SLABS; ++s)
          tma_load_2d(sV + s * Cfg::KV_SLAB_BYTES + kb * 8192, &tmKV, &v_full[kb], v_col0 + 64 * s, kv_row0 + 64 * kb);
      }
      for (int i = 2; i < n_my; ++i) load_q(i);
    }
  } else if (warp == 1) {
    // ===================== MMA issuer =====================
    if (n_my > 0 && elect_one()) {
      auto issue_qk = [&](int i) {
        const int t = i & 1, u = i >> 1;
        const int nk = nk_of(split + i * n_split);
        mbar_wait(&buf_free[t], (u & 1) ^ 1);
        mbar_wait(&q_full[t], u & 1);
        for (int kb = 0; kb < ((nk + 63) >> 6); ++kb) mbar_wait(&k_full[kb], 0);
        tc_fence_after();
        const uint32_t idesc = umma_idesc_bf16(128, static_cast<uint32_t>(nk));
        const uint32_t d_tmem = tmem_base + 256 * t;
#pragma unroll
        for (int kk = 0; kk < DH / 16; ++kk) {
          const int s = kk >> 2;
          const uint64_t a_desc = umma_smem_desc_sw128(smem_u32(sQ + t * Cfg::Q_BYTES + s * Cfg::Q_SLAB_BYTES)) + 2 * (kk & 3);
          const uint64_t b_desc = umma_smem_desc_sw128(smem_u32(sK + s * Cfg::KV_SLAB_BYTES)) + 2 * (kk & 3);
          umma_bf16(d_tmem, a_desc, b_desc, idesc, kk != 0 ? 1u : 0u);
        }
        umma_commit(&s_full[t]);
        umma_commit(&q_empty[t]);
      };
      auto issue_pv = [&](int i) {
        const int t = i & 1, u = i >> 1;
        const int nk = nk_of(split + i * n_split);
        mbar_wait(&p_full[t], u & 1);
        for (int kb = 0; kb < ((nk + 63) >> 6); ++kb) mbar_wait(&v_full[kb], 0);
        tc_fence_after();
        constexpr uint32_t idesc = umma_idesc_bf16(128, DH) | UMMA_IDESC_B_MN_MAJOR;
        const uint32_t d_tmem = tmem_base + 256 * t + Cfg::O_COL;
        const uint32_t a_tmem = tmem_base + 256 * t;
        for (int kk = 0; kk < (nk >> 4); ++kk) {
          // 16 keys per instruction: 8 packed columns of P, 16 rows (2048 B) of V
          const uint64_t b_desc = umma_smem_desc_mn_sw128(smem_u32(sV + kk * 2048), Cfg::KV_SLAB_BYTES);
          umma_bf16_ts(d_tmem, a_tmem + 8 * kk, b_desc, idesc, kk != 0 ? 1u : 0u);
        }
        umma_commit(&o_full[t]);
      };
      issue_qk(0);
      for (int i = 0; i < n_my; ++i) {
        if (i + 1 < n_my) issue_qk(i + 1);
        issue_pv(i);
      }
    }
  } else {
    // ===================== softmax + epilogue groups =====================
    const int grp = (warp - 2) >> 2;
    const int quad = warp & 3;  // TMEM lane quadrant this warp may access
    const int row = quad * 32 + lane;
    const int hl = row >> (7 - g_shift);  // local q head of this row
    const int pr = row & (PT - 1);
    const float sc = p.scale_log2;
    for (int i = grp; i < n_my; i += 2) {
      const int t = i & 1, u = i >> 1;
      const int j = split + i * n_split;
      const int nk = nk_of(j);
      const int pos = j * PT + pr;      // position of this row's query inside the frame
      const int lim = p.prefix_mode ? p.prefix_len - 1 : (p.non_causal ? S - 1 : min(pos, S - 1));  // keys 0..lim are visible
      const uint32_t taddr = tmem_base + (static_cast<uint32_t>(quad * 32) << 16) + 256 * t;
      mbar_wait(&s_full[t], u & 1);
      tc_fence_after();
      const bool tr = quad == 0 && lane == 0 && i < 4;
      if (tr) stamp(3 + 5 * i);
      // ---- pass 1: row maximum over the visible keys
      float mx = -INFINITY;
#pragma unroll 1
      for (int c0 = 0; c0 < nk; c0 += 32) {
        uint32_t r[32];
        tmem_ld32(taddr + c0, r);
        tmem_ld_wait();
#pragma unroll
        for (int x = 0; x < 32; ++x)
          if (c0 + x <= lim) mx = fmaxf(mx, __uint_as_float(r[x]));
      }
      const float msc = mx * sc;
      if (tr) stamp(4 + 5 * i);
      // ---- pass 2: p = exp2(s * c - max * c), row sum in fp32, P (bf16) back into TMEM
      float l = 0.f;
#pragma unroll 1
      for (int c0 = 0; c0 < nk; c0 += 32) {
        uint32_t r[32];
        tmem_ld32(taddr + c0, r);
        tmem_ld_wait();
        uint32_t pk[16];
#pragma unroll
        for (int x = 0; x < 16; ++x) {
          const float p0 = (c0 + 2 * x <= lim) ? ex2_approx(fmaf(__uint_as_float(r[2 * x]), sc, -msc)) : 0.f;
          const float p1 = (c0 + 2 * x + 1 <= lim) ? ex2_approx(fmaf(__uint_as_float(r[2 * x + 1]), sc, -msc)) : 0.f;
          l += p0 + p1;
          __nv_bfloat162 v = __floats2bfloat162_rn(p0, p1);
          pk[x] = *reinterpret_cast<uint32_t*>(&v);
        }
        tmem_st16(taddr + (c0 >> 1), pk);
      }
      tmem_st_wait();
      tc_fence_before();
      mbar_arrive(&p_full[t]);
      if (tr) stamp(5 + 5 * i);
      // ---- epilogue: O / l -> bf16 -> global
      mbar_wait(&o_full[t], u & 1);
      tc_fence_after();
      if (tr) stamp(6 + 5 * i);
      const int head = (kvh << g_shift) + hl;
      __nv_bfloat16* dst = p.out + (size_t)(seq0 + pos) * (p.n_q_heads * DH) + head * DH;
      // scale of this pass's unnormalised O, and (prefix mode) of the frame-local result already in `out`
      float w_new = 1.0f / l, w_old = 0.f;
      if (pos < S) {
        float2* st = p.stats ? p.stats + (size_t)(seq0 + pos) * p.n_q_heads + head : nullptr;
        if (p.prefix_mode) {
          const float2 f = *st;  // (m_f, l_f) of the frame-local pass
          const float m = fmaxf(f.x, mx);
          const float a = f.y * ex2_approx((f.x - m) * sc);
          const float b = ex2_approx((mx - m) * sc);
          const float inv = 1.0f / (a + b * l);
          w_old = a * inv;
          w_new = b * inv;
        } else if (st) {
          *st = make_float2(mx, l);
        }
      }
#pragma unroll 1
      for (int c0 = 0; c0 < DH; c0 += 32) {
        uint32_t r[32];
        tmem_ld32(taddr + Cfg::O_COL + c0, r);
        tmem_ld_wait();
        if (p.out8 != nullptr) {  // one 32-column chunk of a row = one MX block
          if (pos < S) {
            float v[32];
#pragma unroll
            for (int x = 0; x < 32; ++x) v[x] = __uint_as_float(r[x]) * w_new;
            const int row = seq0 + pos, col = head * DH + c0, ld = p.n_q_heads * DH;
            mx_store_block(v, p.out8 + (size_t)row * ld + col, p.sf_out + mx_sf_offset(row, col >> 5, ld / 128));
          }
          continue;
        }
        if (pos < S) {
          float* o32row = p.o32 != nullptr ? p.o32 + (size_t)(seq0 + pos) * (p.n_q_heads * DH) + head * DH + c0 : nullptr;
          if (!p.prefix_mode && o32row != nullptr) {
            // frame-local pass ahead of a prefix pass: normalised fp32 to the scratch
#pragma unroll
            for (int q = 0; q < 8; ++q)
              reinterpret_cast<float4*>(o32row)[q] =
                  make_float4(__uint_as_float(r[4 * q]) * w_new, __uint_as_float(r[4 * q + 1]) * w_new,
                              __uint_as_float(r[4 * q + 2]) * w_new, __uint_as_float(r[4 * q + 3]) * w_new);
          } else {
#pragma unroll
            for (int q4 = 0; q4 < 4; ++q4) {
              float4 oa = make_float4(0.f, 0.f, 0.f, 0.f), ob = oa;
              if (p.prefix_mode) {
                oa = reinterpret_cast<const float4*>(o32row)[2 * q4];
                ob = reinterpret_cast<const float4*>(o32row)[2 * q4 + 1];
              }
              const float ow[8] = {oa.x, oa.y, oa.z, oa.w, ob.x, ob.y, ob.z, ob.w};
              uint32_t o[4];
#pragma unroll
              for (int e = 0; e < 4; ++e) {
                const float lo = __uint_as_float(r[8 * q4 + 2 * e]) * w_new + ow[2 * e] * w_old;
                const float hi = __uint_as_float(r[8 * q4 + 2 * e + 1]) * w_new + ow[2 * e + 1] * w_old;
                __nv_bfloat162 v = __floats2bfloat162_rn(lo, hi);
                o[e] = *reinterpret_cast<uint32_t*>(&v);
              }
              *reinterpret_cast<uint4*>(dst + c0 + 8 * q4) = make_uint4(o[0], o[1], o[2], o[3]);
            }
          }
        }
      }
      tc_fence_before();
      mbar_arrive(&buf_free[t]);
      if (tr) stamp(7 + 5 * i);
    }
  }
  tc_fence_before();
  __syncwarp();
  __syncthreads();
  if (threadIdx.x == 0) stamp(37);
  if (warp == 1) {
    tc_fence_after();
    tmem_dealloc(tmem_base, Cfg::TMEM_COLS);
  }
}

}  // namespace te
