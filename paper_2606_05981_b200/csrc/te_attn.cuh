// te_attn.cuh — causal GQA flash-attention prefill, varlen-packed across frames (SURVEY.md §8(a)
// row a2): per frame b and q head a (kv head a / G): P = softmax(q k^T / sqrt(dh) + causal),
// o = P v, fp32 online softmax, causal by sequence index within the frame.
//
// Sequences are short (S_b <= 256) and attention is < 1 % of the stack's FLOPs, so this kernel is
// latency/occupancy-bound, not tensor-bound: one CTA = 64 query rows of one (frame, q head),
// 4 warps x 16 rows, K/V streamed through shared memory in 64-key blocks, bf16 mma.sync
// m16n8k16 with fp32 accumulation, several CTAs resident per SM.
#pragma once
#include <cuda_bf16.h>
#include <cuda_runtime.h>
#include <stdint.h>

namespace te {

constexpr int ATT_BQ = 64;
constexpr int ATT_BKV = 64;

struct AttnParams {
  const __nv_bfloat16* qkv;  // [T, ld] : q heads | k heads | v heads
  __nv_bfloat16* out;        // [T, Hq*DH]
  const int32_t* cu_seqlens; // [B+1]
  int ld;
  int n_q_heads, n_kv_heads;
  float scale_log2;  // log2(e) / sqrt(dh)
  // shared text prefix (te_encode_prefix): P cached keys/values per layer that every query of every frame
  // sees in front of its own causal keys.  kv_prefix: [P, ld_prefix] = k heads | v heads; null when P = 0.
  const __nv_bfloat16* kv_prefix;
  int prefix_len;
  int ld_prefix;
  int non_causal;  // 1: every query sees all keys of its frame (te_config.non_causal); 0: causal by index
};

// GH = q heads served by one CTA (they share one kv head: GH divides Hq/Hkv); 4 warps per head.
template <int DH, int GH>
struct AttnCfg {
  static constexpr int ROW = DH + 8;  // padded row (elements): 16 B pad -> conflict-free ldmatrix
  static constexpr int THREADS = 128 * GH;
  static constexpr int Q_ELEMS = GH * ATT_BQ * ROW;
  static constexpr int KV_STAGE_ELEMS = 2 * ATT_BKV * ROW;  // K block + V block
  static constexpr int SMEM_BYTES = (Q_ELEMS + 2 * KV_STAGE_ELEMS) * 2;
};

__device__ __forceinline__ void cp_async16(void* smem_dst, const void* gsrc, bool pred) {
  const uint32_t d = static_cast<uint32_t>(__cvta_generic_to_shared(smem_dst));
  const int sz = pred ? 16 : 0;  // src-size 0 -> zero fill
  asm volatile("cp.async.cg.shared.global [%0], [%1], 16, %2;" ::"r"(d), "l"(gsrc), "r"(sz) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
template <int N>
__device__ __forceinline__ void cp_async_wait() {
  asm volatile("cp.async.wait_group %0;" ::"n"(N) : "memory");
}
__device__ __forceinline__ void ldsm_x4(uint32_t (&r)[4], const void* p) {
  const uint32_t a = static_cast<uint32_t>(__cvta_generic_to_shared(p));
  asm volatile("ldmatrix.sync.aligned.m8n8.x4.shared.b16 {%0,%1,%2,%3}, [%4];"
               : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3])
               : "r"(a));
}
__device__ __forceinline__ void ldsm_x4_t(uint32_t (&r)[4], const void* p) {
  const uint32_t a = static_cast<uint32_t>(__cvta_generic_to_shared(p));
  asm volatile("ldmatrix.sync.aligned.m8n8.x4.trans.shared.b16 {%0,%1,%2,%3}, [%4];"
               : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3])
               : "r"(a));
}
__device__ __forceinline__ void mma_bf16_16816(float (&c)[4], const uint32_t (&a)[4], uint32_t b0, uint32_t b1) {
  asm volatile(
      "mma.sync.aligned.m16n8k16.row.col.f32.bf16.bf16.f32 {%0,%1,%2,%3}, {%4,%5,%6,%7}, {%8,%9}, {%0,%1,%2,%3};"
      : "+f"(c[0]), "+f"(c[1]), "+f"(c[2]), "+f"(c[3])
      : "r"(a[0]), "r"(a[1]), "r"(a[2]), "r"(a[3]), "r"(b0), "r"(b1));
}
__device__ __forceinline__ uint32_t pack2_bf16(float a, float b) {
  __nv_bfloat162 v = __floats2bfloat162_rn(a, b);
  return *reinterpret_cast<uint32_t*>(&v);
}

// grid: (q blocks, Hq / GH, B); block: 128 * GH threads.
// K/V blocks of 64 keys are double-buffered (cp.async group per block) and shared by the GH q heads
// of the CTA; query blocks are issued heaviest-first (causal: block qb needs qb + 1 key blocks).
template <int DH, int GH>
__global__ void __launch_bounds__(128 * GH, 2) te_attn_kernel(const AttnParams p) {
  using Cfg = AttnCfg<DH, GH>;
  constexpr int ROW = Cfg::ROW;
  constexpr int THREADS = Cfg::THREADS;
  extern __shared__ __align__(16) uint8_t att_smem[];
  __nv_bfloat16* sQ = reinterpret_cast<__nv_bfloat16*>(att_smem);
  __nv_bfloat16* sKV = sQ + Cfg::Q_ELEMS;

  const int b = blockIdx.z;
  const int head0 = blockIdx.y * GH;
  const int qb = gridDim.x - 1 - blockIdx.x;
  asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
  asm volatile("griddepcontrol.wait;" ::: "memory");  // qkv / cu_seqlens come from predecessor kernels
  const int seq0 = p.cu_seqlens[b];
  const int S = p.cu_seqlens[b + 1] - seq0;  // (te_prep_kernel clamps the offsets to the call's token count)
  const int q0 = qb * ATT_BQ;
  if (q0 >= S) return;
  const int kvh = head0 / (p.n_q_heads / p.n_kv_heads);
  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  const int hl = warp >> 2;       // local q head of this warp
  const int wr = warp & 3;        // 16-row group inside the 64-row query block
  const int g = lane >> 2, t = lane & 3;

  const __nv_bfloat16* gq = p.qkv + (size_t)seq0 * p.ld + head0 * DH;
  const __nv_bfloat16* gk = p.qkv + (size_t)seq0 * p.ld + (p.n_q_heads + kvh) * DH;
  const __nv_bfloat16* gv = p.qkv + (size_t)seq0 * p.ld + (p.n_q_heads + p.n_kv_heads + kvh) * DH;

  // key index space of a frame: [0, P) = cached prefix keys, [P, P + S) = the frame's own keys
  const int P = p.prefix_len;
  const __nv_bfloat16* pk = p.kv_prefix + kvh * DH;
  const __nv_bfloat16* pv = p.kv_prefix + (p.n_kv_heads + kvh) * DH;
  constexpr int CH = DH / 8;  // 16-byte chunks per row
  auto load_kv = [&](int kb, int stage) {
    __nv_bfloat16* sK = sKV + stage * Cfg::KV_STAGE_ELEMS;
    __nv_bfloat16* sV = sK + ATT_BKV * ROW;
    const int k0 = kb * ATT_BKV;
    for (int i = tid; i < ATT_BKV * CH; i += THREADS) {
      const int r = i / CH, c = i % CH;
      const int key = k0 + r;
      const bool ok = key < P + S;
      const bool in_prefix = key < P;
      const __nv_bfloat16* ksrc = in_prefix ? pk + (size_t)key * p.ld_prefix : gk + (size_t)(key - P) * p.ld;
      const __nv_bfloat16* vsrc = in_prefix ? pv + (size_t)key * p.ld_prefix : gv + (size_t)(key - P) * p.ld;
      cp_async16(sK + r * ROW + c * 8, (ok ? ksrc : gk) + c * 8, ok);
      cp_async16(sV + r * ROW + c * 8, (ok ? vsrc : gv) + c * 8, ok);
    }
  };
  for (int i = tid; i < GH * ATT_BQ * CH; i += THREADS) {
    const int h = i / (ATT_BQ * CH), r = (i / CH) % ATT_BQ, c = i % CH;
    cp_async16(sQ + (h * ATT_BQ + r) * ROW + c * 8, gq + (size_t)(q0 + r) * p.ld + h * DH + c * 8, q0 + r < S);
  }
  load_kv(0, 0);
  cp_async_commit();

  float o[DH / 8][4];
#pragma unroll
  for (int i = 0; i < DH / 8; ++i) o[i][0] = o[i][1] = o[i][2] = o[i][3] = 0.f;
  float m_run[2] = {-INFINITY, -INFINITY};
  float l_run[2] = {0.f, 0.f};
  const int qrow0 = q0 + wr * 16 + g;  // this thread's rows: qrow0 and qrow0 + 8 (index within the frame)
  const __nv_bfloat16* sQh = sQ + (hl * ATT_BQ + wr * 16) * ROW;

  // causal: combined keys [0, P + q0 + 64), capped at the frame's end
  const int n_kv_blocks = ((p.non_causal ? P + S : min(P + q0 + ATT_BQ, P + S)) + ATT_BKV - 1) / ATT_BKV;
  for (int kb = 0; kb < n_kv_blocks; ++kb) {
    if (kb + 1 < n_kv_blocks) {
      load_kv(kb + 1, (kb + 1) & 1);  // stage (kb+1)&1 was released by the barrier ending iteration kb-1
      cp_async_commit();
      cp_async_wait<1>();
    } else {
      cp_async_wait<0>();
    }
    __syncthreads();
    const __nv_bfloat16* sK = sKV + (kb & 1) * Cfg::KV_STAGE_ELEMS;
    const __nv_bfloat16* sV = sK + ATT_BKV * ROW;
    const int k0 = kb * ATT_BKV;

    // ---- S = Q K^T  (16 x 64 per warp)
    float s[ATT_BKV / 8][4];
#pragma unroll
    for (int i = 0; i < ATT_BKV / 8; ++i) s[i][0] = s[i][1] = s[i][2] = s[i][3] = 0.f;
#pragma unroll
    for (int kk = 0; kk < DH / 16; ++kk) {
      uint32_t a[4];
      {
        const int mi = lane >> 3, r = lane & 7;
        ldsm_x4(a, sQh + ((mi & 1) * 8 + r) * ROW + kk * 16 + (mi >> 1) * 8);
      }
#pragma unroll
      for (int nt = 0; nt < ATT_BKV / 16; ++nt) {
        uint32_t bfr[4];
        const int mi = lane >> 3, r = lane & 7;
        ldsm_x4(bfr, sK + (nt * 16 + (mi >> 1) * 8 + r) * ROW + kk * 16 + (mi & 1) * 8);
        mma_bf16_16816(s[2 * nt], a, bfr[0], bfr[1]);
        mma_bf16_16816(s[2 * nt + 1], a, bfr[2], bfr[3]);
      }
    }
    // ---- causal mask (only blocks reaching past the first query row's diagonal need it) + online softmax:
    // query row n sees combined keys 0 .. P + n
    // (non-causal: every row sees keys 0 .. P + S - 1; only the frame's last block has keys to mask)
    if (p.non_causal ? (k0 + ATT_BKV > P + S) : (k0 + ATT_BKV - 1 > P + q0)) {
      const int lim0 = p.non_causal ? S - 1 : qrow0, lim1 = p.non_causal ? S - 1 : qrow0 + 8;
#pragma unroll
      for (int nt = 0; nt < ATT_BKV / 8; ++nt) {
        const int key = k0 + nt * 8 + 2 * t - P;
        if (key > lim0) s[nt][0] = -INFINITY;
        if (key + 1 > lim0) s[nt][1] = -INFINITY;
        if (key > lim1) s[nt][2] = -INFINITY;
        if (key + 1 > lim1) s[nt][3] = -INFINITY;
      }
    }
    float mx[2] = {-INFINITY, -INFINITY};
#pragma unroll
    for (int nt = 0; nt < ATT_BKV / 8; ++nt) {
      mx[0] = fmaxf(mx[0], fmaxf(s[nt][0], s[nt][1]));
      mx[1] = fmaxf(mx[1], fmaxf(s[nt][2], s[nt][3]));
    }
#pragma unroll
    for (int i = 0; i < 2; ++i) {
      mx[i] = fmaxf(mx[i], __shfl_xor_sync(0xffffffffu, mx[i], 1));
      mx[i] = fmaxf(mx[i], __shfl_xor_sync(0xffffffffu, mx[i], 2));
    }
    float corr[2], msc[2];
#pragma unroll
    for (int i = 0; i < 2; ++i) {
      const float m_new = fmaxf(m_run[i], mx[i]);  // key 0 is always visible -> finite from the first block on
      corr[i] = exp2f((m_run[i] - m_new) * p.scale_log2);
      m_run[i] = m_new;
      msc[i] = m_new * p.scale_log2;
    }
    float rs[2] = {0.f, 0.f};
#pragma unroll
    for (int nt = 0; nt < ATT_BKV / 8; ++nt) {
      s[nt][0] = exp2f(fmaf(s[nt][0], p.scale_log2, -msc[0]));
      s[nt][1] = exp2f(fmaf(s[nt][1], p.scale_log2, -msc[0]));
      s[nt][2] = exp2f(fmaf(s[nt][2], p.scale_log2, -msc[1]));
      s[nt][3] = exp2f(fmaf(s[nt][3], p.scale_log2, -msc[1]));
      rs[0] += s[nt][0] + s[nt][1];
      rs[1] += s[nt][2] + s[nt][3];
    }
    l_run[0] = l_run[0] * corr[0] + rs[0];
    l_run[1] = l_run[1] * corr[1] + rs[1];
#pragma unroll
    for (int i = 0; i < DH / 8; ++i) {
      o[i][0] *= corr[0]; o[i][1] *= corr[0];
      o[i][2] *= corr[1]; o[i][3] *= corr[1];
    }
    // ---- O += P V
#pragma unroll
    for (int kk = 0; kk < ATT_BKV / 16; ++kk) {
      uint32_t a[4];
      a[0] = pack2_bf16(s[2 * kk][0], s[2 * kk][1]);
      a[1] = pack2_bf16(s[2 * kk][2], s[2 * kk][3]);
      a[2] = pack2_bf16(s[2 * kk + 1][0], s[2 * kk + 1][1]);
      a[3] = pack2_bf16(s[2 * kk + 1][2], s[2 * kk + 1][3]);
#pragma unroll
      for (int nt = 0; nt < DH / 16; ++nt) {
        uint32_t bfr[4];
        const int mi = lane >> 3, r = lane & 7;
        ldsm_x4_t(bfr, sV + (kk * 16 + (mi & 1) * 8 + r) * ROW + nt * 16 + (mi >> 1) * 8);
        mma_bf16_16816(o[2 * nt], a, bfr[0], bfr[1]);
        mma_bf16_16816(o[2 * nt + 1], a, bfr[2], bfr[3]);
      }
    }
    __syncthreads();  // all warps are done with this K/V stage before it is refilled
  }
  // ---- finalize: row sums across the 4 threads of a row, normalise, store
#pragma unroll
  for (int i = 0; i < 2; ++i) {
    l_run[i] += __shfl_xor_sync(0xffffffffu, l_run[i], 1);
    l_run[i] += __shfl_xor_sync(0xffffffffu, l_run[i], 2);
  }
  const float inv0 = 1.0f / l_run[0], inv1 = 1.0f / l_run[1];
  __nv_bfloat16* out0 = p.out + (size_t)(seq0 + qrow0) * (p.n_q_heads * DH) + (head0 + hl) * DH + 2 * t;
  __nv_bfloat16* out1 = out0 + (size_t)8 * (p.n_q_heads * DH);
#pragma unroll
  for (int nt = 0; nt < DH / 8; ++nt) {
    if (qrow0 < S) *reinterpret_cast<uint32_t*>(out0 + nt * 8) = pack2_bf16(o[nt][0] * inv0, o[nt][1] * inv0);
    if (qrow0 + 8 < S) *reinterpret_cast<uint32_t*>(out1 + nt * 8) = pack2_bf16(o[nt][2] * inv1, o[nt][3] * inv1);
  }
}

}  // namespace te
