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

// Per-call values that a cached graph must not bake in: written on the stream ahead of the stack's kernels
// (te_set_dyn_kernel), read by every kernel.  A graph is therefore reusable for any caller buffers and for any
// token count of the same row-block bucket (te_runtime.cu, graph cache).
// Ordering: the GEMM kernels read total_tokens / out BEFORE their griddepcontrol.wait (gemm_rows, resid_dst).  That is
// safe because the kernel that follows te_set_dyn_kernel in the stream (te_prep_kernel) is launched WITHOUT programmatic
// overlap: by the time any later kernel of the call can start, set_dyn has completed and flushed.
struct DynParams {
  const void* embeds;        // DEVICE [T, d]: fp32, or bf16 when embeds_bf16 (te_encode_ex)
  const int32_t* text_lens;  // DEVICE int32 [B]
  float* out;                // DEVICE fp32 [T, d]
  const int32_t* grids;      // DEVICE int32 [B][2] = (grid_h, grid_w) of every frame, or null: one grid per call
  int32_t total_tokens;      // T
  int32_t embeds_bf16;
};

struct GemmParams {
  int M, N, K;               // M: rows when dyn == nullptr (te_debug_gemm*); else dyn->total_tokens
  const DynParams* dyn;
  int num_m_blk, num_n_blk;
  // RMSNorm statistics of the A rows (consumer side): ssq_in[row * ssq_stride + part], one 16-byte-aligned
  // run of `ssq_parts` partial sums of squares per row (a row's parts share a cache line)
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
  float* x;      // fp32 residual stream (library workspace), updated in place ...
  int x_to_out;  // ... or, for the LAST residual GEMM of the stack, read from x and written to dyn->out
  int ld_x;
  const __nv_bfloat16* g_next;  // may be null (no next norm)
  __nv_bfloat16* xg;            // [T, ld_x] bf16(x * g_next)
  float* ssq_out;               // [T][ssq_stride], entry n_blk * nparts + part
  // EPI_SWIGLU
  __nv_bfloat16* act;
  int ld_act;
  // EPI_PLAIN
  float* c;
  int ld_c;
  // optional cycle trace (debug): trace[blockIdx.x * TRACE_SLOTS + slot] = globaltimer ns
  unsigned long long* trace;
  // split-K kernel (te_gemm_splitk.cuh): CTAs per output tile, fp32 partial-tile scratch, per-tile semaphores
  int splits;
  float* sk_scratch;
  int* sk_sem;
  // EPI_SWIGLU with 128-wide tiles over weights interleaved per 256 rows (128 gate | 128 up): tile n' takes gate
  // rows (n'>>1)*256 + (n'&1)*64 .. +64 and the matching up rows 128 further on, as two 64-row halves
  int gu_half;
};
// Epilogue loads of data written by an earlier KERNEL (gains, RMSNorm statistics, rotary table): a kernel boundary
// separates writer and reader, so the ordinary L1-cached load is right.
template <typename T>
__device__ __forceinline__ T ld_phase(const T* ptr) {
  return *ptr;
}
__device__ __forceinline__ int gemm_rows(const GemmParams& p) { return p.dyn != nullptr ? p.dyn->total_tokens : p.M; }
__device__ __forceinline__ float* resid_dst(const GemmParams& p) { return p.x_to_out ? p.dyn->out : p.x; }
constexpr int TRACE_SLOTS = 96;  // [0,48): globaltimer ns, [48,96): SM clock of the same stamp
__device__ __forceinline__ void trace_stamp(const GemmParams& p, int slot) {
  if (p.trace != nullptr) {
    unsigned long long t;
    asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t));
    p.trace[(size_t)blockIdx.x * TRACE_SLOTS + slot] = t;
    p.trace[(size_t)blockIdx.x * TRACE_SLOTS + 48 + slot] = static_cast<unsigned long long>(clock64());
  }
}

template <int BN>
struct GemmCfg {
  static constexpr int STAGES = (BN == 256) ? 4 : 6;
  static constexpr int A_BYTES = GEMM_BM * GEMM_BK * 2;
  static constexpr int B_BYTES = BN * GEMM_BK * 2;
  static constexpr int STAGE_BYTES = A_BYTES + B_BYTES;
  static constexpr int BAR_BYTES = 256;
  // epilogue staging: per epilogue warp two 32-row x 32-float XOR-swizzled fp32 chunks, used to turn
  // the one-thread-per-row TMEM layout into row-contiguous (coalesced) global accesses
  static constexpr int STG_WARP_BYTES = 2 * 32 * 32 * 4;
  static constexpr int STG_BYTES = 4 * STG_WARP_BYTES;
  static constexpr int SMEM_BYTES = STAGES * STAGE_BYTES + BAR_BYTES + STG_BYTES + 1024;  // +1024: manual alignment
  static constexpr int TMEM_COLS = 2 * BN;
};

__device__ __forceinline__ uint32_t pack_bf16(float a, float b) {
  __nv_bfloat162 v = __floats2bfloat162_rn(a, b);
  return *reinterpret_cast<uint32_t*>(&v);
}
__device__ __forceinline__ float bf16_lo(uint32_t u) { return __uint_as_float(u << 16); }
__device__ __forceinline__ float bf16_hi(uint32_t u) { return __uint_as_float(u & 0xFFFF0000u); }

// ----------------------------------------------------------------------------- epilogues
// `part` / `nparts`: the epilogue warps that share one TMEM lane quadrant split the tile's columns.
template <int BN>
__device__ __forceinline__ void epi_plain(const GemmParams& p, uint32_t t_row, int row, bool valid, int n_blk,
                                          int part, int nparts) {
#pragma unroll 1
  for (int c0 = part * (BN / nparts); c0 < (part + 1) * (BN / nparts); c0 += 32) {
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

// Staging layout shared by the coalesced epilogues.  A warp owns 32 accumulator rows (thread = row
// after tcgen05.ld 32x32b).  A 32-column fp32 chunk is written to shared memory by rows and read
// back so that 8 consecutive lanes hold one 128-byte row segment (4 rows per warp instruction).
// Element (row, col) lives at row*32 + (((col>>2) ^ (row&7))<<2) + (col&3): both the row-wise
// 16-byte writes and the segment-wise 16-byte reads are bank-conflict free without padding.
__device__ __forceinline__ void stg_put_row(float* buf, int lane, const float (&v)[32]) {
#pragma unroll
  for (int j = 0; j < 8; ++j)
    *reinterpret_cast<float4*>(buf + lane * 32 + ((j ^ (lane & 7)) << 2)) =
        make_float4(v[4 * j], v[4 * j + 1], v[4 * j + 2], v[4 * j + 3]);
}
__device__ __forceinline__ float4 stg_get(const float* buf, int rr, int cq) {
  return *reinterpret_cast<const float4*>(buf + rr * 32 + ((cq ^ (rr & 7)) << 2));
}

// Residual epilogue: x += acc (fp32, in place), xg = bf16(x * g_next), per-row partial sum of squares.
// The x operand is software-pipelined: ResidPrefetch::issue() is called BEFORE the accumulator is
// ready (the epilogue warps idle during the main loop), and each chunk's loads are issued one
// chunk ahead, so the L2 round trips are off the critical path.
struct ResidPrefetch {
  float4 xv[8];
};
template <int BN>
__device__ __forceinline__ void resid_issue(const GemmParams& p, int M, ResidPrefetch& pf, int row_base, int lane,
                                            int n_blk, int c0) {
  const int sub = lane >> 3, cq = lane & 7;
  const int col = n_blk * BN + c0 + cq * 4;
  if (col >= p.N) return;  // chunk past the last column (N is not a multiple of a 192-wide tile)
#pragma unroll
  for (int i = 0; i < 8; ++i) {
    const int row = row_base + sub + 4 * i;
    if (row < M) pf.xv[i] = ld_phase(reinterpret_cast<const float4*>(p.x + (size_t)row * p.ld_x + col));
  }
}
template <int BN>
__device__ __forceinline__ void epi_resid(const GemmParams& p, int M, uint32_t t_row, int row_base, int lane, int n_blk,
                                          float* stg, int part, int nparts, ResidPrefetch& pf) {
  float* const x_dst = resid_dst(p);
  const int sub = lane >> 3;  // row within a group of 4
  const int cq = lane & 7;    // 4-column group inside the 32-column chunk
  const bool has_g = p.g_next != nullptr;
  float ss[8];
#pragma unroll
  for (int i = 0; i < 8; ++i) ss[i] = 0.f;
  const int c_end = (part + 1) * (BN / nparts);
#pragma unroll 1
  for (int c0 = part * (BN / nparts); c0 < c_end; c0 += 32) {
    if (n_blk * BN + c0 >= p.N) break;  // columns past N (zero-filled weight rows): nothing to store
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
    if (c0 + 32 < c_end) resid_issue<BN>(p, M, pf, row_base, lane, n_blk, c0 + 32);  // next chunk's x in flight
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
  // per-row sum of squares over this warp's columns: fixed-order reduction over the row's 8 lanes
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

__device__ __forceinline__ float row_rstd(const GemmParams& p, int row, bool valid) {
  float s = 0.f;
  if (valid) {
    const float* q = p.ssq_in + (size_t)row * p.ssq_stride;
    int i = 0;
    for (; i + 4 <= p.ssq_parts; i += 4) {  // sequential sum, fixed order
      const float4 v = ld_phase(reinterpret_cast<const float4*>(q + i));
      s += v.x; s += v.y; s += v.z; s += v.w;
    }
    for (; i < p.ssq_parts; ++i) s += ld_phase(q + i);
  }
  return 1.0f / sqrtf(s * p.inv_d + p.eps);
}

// Store a staged 32x32 fp32 chunk as bf16: 8 lanes x 4 columns = 64 B per row, 4 rows per instruction.
__device__ __forceinline__ void stg_store_bf16(const float* buf, int lane, int row_base, int M, __nv_bfloat16* dst,
                                               int ld, int col0) {
  const int sub = lane >> 3, cq = lane & 7;
#pragma unroll
  for (int i = 0; i < 8; ++i) {
    const int rr = sub + 4 * i;
    const int row = row_base + rr;
    if (row < M) {
      const float4 a = stg_get(buf, rr, cq);
      uint2 o;
      o.x = pack_bf16(a.x, a.y);
      o.y = pack_bf16(a.z, a.w);
      *reinterpret_cast<uint2*>(dst + (size_t)row * ld + col0 + cq * 4) = o;
    }
  }
}

// SwiGLU epilogue: tile columns [0,BN/2) = gate, [BN/2,BN) = up (weights interleaved per tile).
// The arithmetic runs in the thread-per-row domain; only the bf16 store is transposed.
template <int BN>
__device__ __forceinline__ void epi_swiglu(const GemmParams& p, int M, uint32_t t_row, int row_base, int lane, int n_blk,
                                           float* stg, int part, int nparts, float rstd) {
  constexpr int HALF = BN / 2;
#pragma unroll 1
  for (int c0 = part * (HALF / nparts); c0 < (part + 1) * (HALF / nparts); c0 += 32) {
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
        a[j] = __fdividef(gv, 1.0f + __expf(-gv)) * uv;  // silu(g) * u; fast divide (2 ulp) ahead of a bf16 store
      }
    }
    stg_put_row(stg, lane, a);
    __syncwarp();
    stg_store_bf16(stg, lane, row_base, M, p.act, p.ld_act, n_blk * HALF + c0);
    __syncwarp();
  }
}

// QKV epilogue: y = rstd * acc; v heads are stored; q/k heads get the per-head RMSNorm (pass 1, in the
// thread-per-row domain) and then gain + M-RoPE rotation of the pairs (i, i + DH/2) in the coalesced
// domain, where the cos/sin rows are read as whole 128-byte segments.
template <int BN, int DH>
__device__ __forceinline__ void epi_qkv(const GemmParams& p, int M, uint32_t t_row, int row_base, int lane, int n_blk,
                                        float* stg, int part, int nparts, float rstd, bool tr = false) {
  constexpr int HD2 = DH / 2;
  const int sub = lane >> 3, cq = lane & 7;
  float* bufA = stg;
  float* bufB = stg + 32 * 32;
  constexpr int HEADS = BN / DH;
  // heads of the tile are split between the warps of a quadrant; when they do not divide evenly (one head
  // per tile, two warps) every warp takes every head but only its share of the 32-column chunks: the
  // head's sum of squares (pass 1, TMEM reads only) is then computed redundantly
  const bool split_heads = HEADS % nparts == 0;
  const int hh_begin = split_heads ? part * (HEADS / nparts) : 0;
  const int hh_end = split_heads ? (part + 1) * (HEADS / nparts) : HEADS;
  const int c_first = split_heads ? 0 : part * 32;
  const int c_step = split_heads ? 32 : nparts * 32;
#pragma unroll 1
  for (int hh = hh_begin; hh < hh_end; ++hh) {
    const int col0 = n_blk * BN + hh * DH;  // first column of this head in the fused qkv row
    const uint32_t t_head = t_row + hh * DH;
    if (col0 >= p.k_cols_end) {
      // ---- v head: scale and store
#pragma unroll 1
      for (int c0 = c_first; c0 < DH; c0 += c_step) {
        float v[32];
        {
          uint32_t r[32];
          tmem_ld32(t_head + c0, r);
          tmem_ld_wait();
#pragma unroll
          for (int j = 0; j < 32; ++j) v[j] = __uint_as_float(r[j]) * rstd;
        }
        stg_put_row(bufA, lane, v);
        __syncwarp();
        stg_store_bf16(bufA, lane, row_base, M, p.qkv, p.ld_qkv, col0 + c0);
        __syncwarp();
      }
      continue;
    }
    // ---- q or k head.  The cos/sin segments of the first rotation step are requested up front (16 independent
    // 16-byte loads per lane): their L2 round trip overlaps pass 1's TMEM reads instead of following them.
    const __nv_bfloat16* gain = (col0 < p.q_cols_end) ? p.gq : p.gk;
    float4 cs[8], sn[8];
    auto load_cs = [&](int c0) {
      const int cc = c0 + cq * 4;
#pragma unroll
      for (int i = 0; i < 8; ++i) {
        const int row = min(row_base + sub + 4 * i, M - 1);
        cs[i] = __ldg(reinterpret_cast<const float4*>(p.cos_t + (size_t)row * HD2 + cc));
        sn[i] = __ldg(reinterpret_cast<const float4*>(p.sin_t + (size_t)row * HD2 + cc));
      }
    };
    load_cs(c_first);
    if (tr && hh == hh_begin) trace_stamp(p, 38);
    // Pass 1: sum of squares of the head (thread = row, TMEM reads only)
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
    if (tr && hh == hh_begin) trace_stamp(p, 39);
    // ---- Pass 2: normalised halves a = u[c0..c0+32), b = u[HD2+c0..) -> staging -> rotate -> store.
#pragma unroll 1
    for (int c0 = c_first; c0 < HD2; c0 += c_step) {
      const int cc = c0 + cq * 4;  // this lane's 4 columns inside the half
      // (later steps: their cos/sin rows were requested row by row inside the previous step's rotation loop, as soon as
      //  that step had consumed its own — the L2 round trip overlaps the rest of that loop, this step's TMEM reads and staging)
      const bool more = c0 + c_step < HD2;
      const int cc_next = c0 + c_step + cq * 4;
      const uint2 ga = __ldg(reinterpret_cast<const uint2*>(gain + cc));
      const uint2 gb = __ldg(reinterpret_cast<const uint2*>(gain + HD2 + cc));
      {
        float v[32];
        uint32_t r[32], r2[32];
        tmem_ld32(t_head + c0, r);  // both halves in flight: one TMEM round trip per step
        tmem_ld32(t_head + HD2 + c0, r2);
        tmem_ld_wait();
#pragma unroll
        for (int j = 0; j < 32; ++j) v[j] = __uint_as_float(r[j]) * sc;
        stg_put_row(bufA, lane, v);
#pragma unroll
        for (int j = 0; j < 32; ++j) v[j] = __uint_as_float(r2[j]) * sc;
        stg_put_row(bufB, lane, v);
      }
      __syncwarp();
      if (tr && hh == hh_begin && c0 == c_first) trace_stamp(p, 40);
      const float gA[4] = {bf16_lo(ga.x), bf16_hi(ga.x), bf16_lo(ga.y), bf16_hi(ga.y)};
      const float gB[4] = {bf16_lo(gb.x), bf16_hi(gb.x), bf16_lo(gb.y), bf16_hi(gb.y)};
#pragma unroll
      for (int i = 0; i < 8; ++i) {
        const int rr = sub + 4 * i;
        const int row = row_base + rr;
        if (row < M) {
          const float4 a = stg_get(bufA, rr, cq);
          const float4 b = stg_get(bufB, rr, cq);
          const float ua[4] = {a.x * gA[0], a.y * gA[1], a.z * gA[2], a.w * gA[3]};
          const float ub[4] = {b.x * gB[0], b.y * gB[1], b.z * gB[2], b.w * gB[3]};
          const float c[4] = {cs[i].x, cs[i].y, cs[i].z, cs[i].w};
          const float sv[4] = {sn[i].x, sn[i].y, sn[i].z, sn[i].w};
          if (more) {
            cs[i] = __ldg(reinterpret_cast<const float4*>(p.cos_t + (size_t)row * HD2 + cc_next));
            sn[i] = __ldg(reinterpret_cast<const float4*>(p.sin_t + (size_t)row * HD2 + cc_next));
          }
          float r1[4], r2[4];
#pragma unroll
          for (int e = 0; e < 4; ++e) {
            r1[e] = ua[e] * c[e] - ub[e] * sv[e];
            r2[e] = ub[e] * c[e] + ua[e] * sv[e];
          }
          uint2 o1, o2;
          o1.x = pack_bf16(r1[0], r1[1]); o1.y = pack_bf16(r1[2], r1[3]);
          o2.x = pack_bf16(r2[0], r2[1]); o2.y = pack_bf16(r2[2], r2[3]);
          __nv_bfloat16* dst = p.qkv + (size_t)row * p.ld_qkv + col0 + cc;
          *reinterpret_cast<uint2*>(dst) = o1;
          *reinterpret_cast<uint2*>(dst + HD2) = o2;
        }
      }
      __syncwarp();
      if (tr && hh == hh_begin && c0 == c_first) trace_stamp(p, 41);
    }
    if (tr && hh == hh_begin) trace_stamp(p, 42);
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
  float* stg_all = reinterpret_cast<float*>(smem + STAGES * Cfg::STAGE_BYTES + Cfg::BAR_BYTES);

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
  pdl_launch_dependents();

  const int M = gemm_rows(p);
  const int num_kb = p.K / GEMM_BK;
  const int num_tiles = p.num_m_blk * p.num_n_blk;

  if (warp == 0) {
    // ===================== TMA producer =====================
    if (elect_one()) {
      int stage = 0;
      uint32_t phase = 0;
      // Weights do not depend on the predecessor kernel: start streaming the first ring of B tiles
      // before the grid-dependency wait; the matching A tiles follow after it.
      const int pre = (blockIdx.x < num_tiles) ? (num_kb < STAGES ? num_kb : STAGES) : 0;
      {
        const int n_blk0 = blockIdx.x / p.num_m_blk;
        for (int kb = 0; kb < pre; ++kb) {
          mbar_arrive_expect_tx(&full[kb], Cfg::STAGE_BYTES);
          tma_load_2d(sB + kb * Cfg::B_BYTES, &tmB, &full[kb], kb * GEMM_BK, n_blk0 * BN);
        }
      }
      pdl_wait();
      bool first = true;
      for (int tile = blockIdx.x; tile < num_tiles; tile += gridDim.x) {
        const int m_blk = tile % p.num_m_blk;
        const int n_blk = tile / p.num_m_blk;
        for (int kb = 0; kb < num_kb; ++kb) {
          if (first && kb < pre) {
            tma_load_2d(sA + stage * Cfg::A_BYTES, &tmA, &full[stage], kb * GEMM_BK, m_blk * GEMM_BM);
          } else {
            mbar_wait(&empty[stage], phase ^ 1);
            mbar_arrive_expect_tx(&full[stage], Cfg::STAGE_BYTES);
            tma_load_2d(sA + stage * Cfg::A_BYTES, &tmA, &full[stage], kb * GEMM_BK, m_blk * GEMM_BM);
            tma_load_2d(sB + stage * Cfg::B_BYTES, &tmB, &full[stage], kb * GEMM_BK, n_blk * BN);
          }
          if (++stage == STAGES) { stage = 0; phase ^= 1; }
        }
        first = false;
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
    pdl_wait();
    for (int tile = blockIdx.x; tile < num_tiles; tile += gridDim.x, ++it) {
      const int m_blk = tile % p.num_m_blk;
      const int n_blk = tile / p.num_m_blk;
      const int acc = it & 1;
      const uint32_t acc_phase = (it >> 1) & 1;
      const int row = m_blk * GEMM_BM + row_in_tile;
      const bool valid = row < M;
      // operands that do not depend on the accumulator are fetched while the main loop still runs
      float rstd = 0.f;
      ResidPrefetch pf;
      if constexpr (EPI == EPI_QKV || EPI == EPI_SWIGLU) rstd = row_rstd(p, row, valid);
      if constexpr (EPI == EPI_RESID) resid_issue<BN>(p, M, pf, m_blk * GEMM_BM + quad * 32, lane, n_blk, 0);
      mbar_wait(&tfull[acc], acc_phase);
      tc_fence_after();
      const uint32_t t_row = tmem_base + (static_cast<uint32_t>(quad * 32) << 16) + acc * BN;
      if constexpr (EPI == EPI_PLAIN) epi_plain<BN>(p, t_row, row, valid, n_blk, 0, 1);
      float* stg = stg_all + quad * (Cfg::STG_WARP_BYTES / 4);
      const int row_base = m_blk * GEMM_BM + quad * 32;
      if constexpr (EPI == EPI_RESID) epi_resid<BN>(p, M, t_row, row_base, lane, n_blk, stg, 0, 1, pf);
      if constexpr (EPI == EPI_SWIGLU) epi_swiglu<BN>(p, M, t_row, row_base, lane, n_blk, stg, 0, 1, rstd);
      if constexpr (EPI == EPI_QKV) epi_qkv<BN, DH>(p, M, t_row, row_base, lane, n_blk, stg, 0, 1, rstd);
      tc_fence_before();
      mbar_arrive(&tempty[acc]);
    }
  }
  __syncwarp();  // the elected producer / MMA lanes rejoin their warps before the block barrier
  __syncthreads();
  if (warp == 1) {
    tc_fence_after();
    tmem_dealloc(tmem_base, Cfg::TMEM_COLS);
  }
}

// ------------------------------------------------------------------ CTA-pair (cta_group::2) kernel
// Same pipeline, but a cluster of two CTAs (one SM pair) computes a 256 x BN tile: each CTA loads its
// own 128 A rows and HALF of the B tile (BN/2 weight rows); the leader CTA issues
// tcgen05.mma.cta_group::2 (M = 256), which reads both halves of B and writes rows 0-127 of D into
// the leader's TMEM and rows 128-255 into the peer's.  Per SM this moves A 16 KB + B BN/2 x 128 B per
// 64-deep k-block instead of A 16 KB + B BN x 128 B: 1.5x less L2->SM traffic at BN = 256.
// Persistent: pair q takes tiles q, q + pairs, ...; two accumulator buffers, so the epilogue of one tile
// overlaps the main loop of the next.
constexpr int GEMM2_EPI_WARPS = 8;  // two per TMEM lane quadrant: the epilogue is issue-latency-bound per warp
constexpr int GEMM2_THREADS = 64 + 32 * GEMM2_EPI_WARPS;

template <int BN, int EPI>
struct Gemm2Cfg {
  static constexpr int A_BYTES = GEMM_BM * GEMM_BK * 2;
  static constexpr int B_BYTES = (BN / 2) * GEMM_BK * 2;
  static constexpr int STAGE_BYTES = A_BYTES + B_BYTES;
  static constexpr int BAR_BYTES = 256;
  // staging per epilogue warp: one swizzled 32x32 fp32 chunk, two for the rotary pairs of EPI_QKV
  static constexpr int STG_WARP_BYTES = (EPI == EPI_QKV ? 2 : 1) * 32 * 32 * 4;
  static constexpr int STG_BYTES = GEMM2_EPI_WARPS * STG_WARP_BYTES;
  static constexpr int SMEM_LIMIT = 232448;  // 227 KB
  static constexpr int STAGES_FIT = (SMEM_LIMIT - 1024 - BAR_BYTES - STG_BYTES) / STAGE_BYTES;
  static constexpr int STAGES = STAGES_FIT > 8 ? 8 : STAGES_FIT;
  static constexpr int SMEM_BYTES = STAGES * STAGE_BYTES + BAR_BYTES + STG_BYTES + 1024;
  static constexpr int TMEM_COLS = (2 * BN <= 256) ? 256 : 512;  // power of two >= two BN-column accumulators
  static_assert(STAGES >= 3 && 2 * STAGES + 5 <= BAR_BYTES / 8, "pipeline configuration");
};

template <int BN, int EPI, int DH>
__global__ void __cluster_dims__(2, 1, 1) __launch_bounds__(GEMM2_THREADS, 1)
te_gemm2_kernel(const __grid_constant__ CUtensorMap tmA, const __grid_constant__ CUtensorMap tmB, const GemmParams p) {
  using Cfg = Gemm2Cfg<BN, EPI>;
  constexpr int STAGES = Cfg::STAGES;
  extern __shared__ uint8_t smem_raw[];
  uint8_t* smem = reinterpret_cast<uint8_t*>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~uintptr_t(1023));
  uint8_t* sA = smem;
  uint8_t* sB = smem + STAGES * Cfg::A_BYTES;
  uint64_t* bars = reinterpret_cast<uint64_t*>(smem + STAGES * Cfg::STAGE_BYTES);
  uint64_t* full = bars;                 // used in the leader CTA only
  uint64_t* empty = bars + STAGES;       // one set per CTA (each producer waits on its own)
  uint64_t* tfull = bars + 2 * STAGES;   // one set per CTA (each CTA's epilogue waits on its own)
  uint64_t* tempty = tfull + 2;          // used in the leader CTA only (all epilogue threads of both CTAs)
  uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(tempty + 2);
  float* stg_all = reinterpret_cast<float*>(smem + STAGES * Cfg::STAGE_BYTES + Cfg::BAR_BYTES);

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
      for (int i = 0; i < 2; ++i) {
        mbar_init(&tfull[i], 1);
        mbar_init(&tempty[i], 2 * 32 * GEMM2_EPI_WARPS);
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
  if (threadIdx.x == 0) trace_stamp(p, 1);

  const int M = gemm_rows(p);
  const int num_kb = p.K / GEMM_BK;
  const int num_mp = (p.num_m_blk + 1) >> 1;  // 256-row blocks
  const int num_tiles = num_mp * p.num_n_blk;
  const int pair = blockIdx.x >> 1;
  const int num_pairs = gridDim.x >> 1;
  auto b_row_of = [&](int n_blk) {
    return p.gu_half ? (n_blk >> 1) * 256 + static_cast<int>(rank) * 128 + (n_blk & 1) * 64
                     : n_blk * BN + static_cast<int>(rank) * (BN / 2);
  };

  if (warp == 0) {
    // ===================== TMA producer (both CTAs) =====================
    if (elect_one()) {
      int stage = 0;
      uint32_t phase = 0;
      // weights first (independent of the predecessor kernel), then the dependency wait, then A
      const int pre = (pair < num_tiles) ? (num_kb < STAGES ? num_kb : STAGES) : 0;
      if (pre > 0) {
        const int b_row0 = b_row_of(pair / num_mp);
        for (int i = 0; i < pre; ++i) {
          if (leader) mbar_arrive_expect_tx(&full[i], 2 * Cfg::STAGE_BYTES);
          tma_load_2d_cg2(sB + i * Cfg::B_BYTES, &tmB, mapa_u32(smem_u32(&full[i]), 0), i * GEMM_BK, b_row0);
        }
      }
      pdl_wait();
      trace_stamp(p, 2);
      bool first = true;
      for (int tile = pair; tile < num_tiles; tile += num_pairs) {
        const int mp = tile % num_mp;
        const int n_blk = tile / num_mp;
        const int a_row = mp * 2 * GEMM_BM + rank * GEMM_BM;
        const int b_row = b_row_of(n_blk);
        for (int kb = 0; kb < num_kb; ++kb) {
          const uint32_t bar = mapa_u32(smem_u32(&full[stage]), 0);
          if (first && kb < pre) {
            tma_load_2d_cg2(sA + stage * Cfg::A_BYTES, &tmA, bar, kb * GEMM_BK, a_row);
          } else {
            mbar_wait(&empty[stage], phase ^ 1);
            if (leader) mbar_arrive_expect_tx(&full[stage], 2 * Cfg::STAGE_BYTES);
            tma_load_2d_cg2(sA + stage * Cfg::A_BYTES, &tmA, bar, kb * GEMM_BK, a_row);
            tma_load_2d_cg2(sB + stage * Cfg::B_BYTES, &tmB, bar, kb * GEMM_BK, b_row);
          }
          if (++stage == STAGES) { stage = 0; phase ^= 1; }
        }
        first = false;
      }
    }
  } else if (warp == 1) {
    // ===================== MMA issuer (leader CTA only) =====================
    if (leader && elect_one()) {
      constexpr uint32_t idesc = umma_idesc_bf16(2 * GEMM_BM, BN);
      int stage = 0;
      uint32_t phase = 0;
      int it = 0;
      for (int tile = pair; tile < num_tiles; tile += num_pairs, ++it) {
        const int acc = it & 1;
        const uint32_t acc_phase = (it >> 1) & 1;
        mbar_wait(&tempty[acc], acc_phase ^ 1);
        tc_fence_after();
        const uint32_t d_tmem = tmem_base + acc * BN;
        for (int kb = 0; kb < num_kb; ++kb) {
          mbar_wait(&full[stage], phase);
          if (kb == 0 && it < 10) trace_stamp(p, 3 + it);
          tc_fence_after();
          const uint64_t a_desc = umma_smem_desc_sw128(smem_u32(sA + stage * Cfg::A_BYTES));
          const uint64_t b_desc = umma_smem_desc_sw128(smem_u32(sB + stage * Cfg::B_BYTES));
#pragma unroll
          for (int k = 0; k < GEMM_BK / 16; ++k)
            umma_bf16_cg2(d_tmem, a_desc + 2 * k, b_desc + 2 * k, idesc, (kb | k) != 0 ? 1u : 0u);
          umma_commit_cg2(&empty[stage], 0x3);  // frees this stage in BOTH CTAs
          if (++stage == STAGES) { stage = 0; phase ^= 1; }
        }
        umma_commit_cg2(&tfull[acc], 0x3);      // accumulator ready in BOTH CTAs
      }
    }
  } else {
    // ===================== epilogue warps (both CTAs, own 128 rows) =====================
    const int quad = warp & 3;         // TMEM lane quadrant this warp may read
    const int part = (warp - 2) >> 2;  // which share of the tile's columns (two warps per quadrant)
    constexpr int NPARTS = GEMM2_EPI_WARPS / 4;
    int it = 0;
    pdl_wait();
    for (int tile = pair; tile < num_tiles; tile += num_pairs, ++it) {
      const int mp = tile % num_mp;
      const int n_blk = tile / num_mp;
      const int acc = it & 1;
      const uint32_t acc_phase = (it >> 1) & 1;
      const int row_base = mp * 2 * GEMM_BM + rank * GEMM_BM + quad * 32;
      const uint32_t t_row = tmem_base + (static_cast<uint32_t>(quad * 32) << 16) + acc * BN;
      // operands that do not depend on the accumulator are fetched while the main loop still runs
      float rstd = 0.f;
      ResidPrefetch pf;
      if constexpr (EPI == EPI_QKV || EPI == EPI_SWIGLU) rstd = row_rstd(p, row_base + lane, row_base + lane < M);
      if constexpr (EPI == EPI_RESID) resid_issue<BN>(p, M, pf, row_base, lane, n_blk, part * (BN / NPARTS));
      mbar_wait(&tfull[acc], acc_phase);
      if (warp == 2 && lane == 0 && it < 10) trace_stamp(p, 14 + it);
      tc_fence_after();
      float* stg = stg_all + (warp - 2) * (Cfg::STG_WARP_BYTES / 4);
      if constexpr (EPI == EPI_PLAIN) epi_plain<BN>(p, t_row, row_base + lane, row_base + lane < M, n_blk, part, NPARTS);
      if constexpr (EPI == EPI_RESID) epi_resid<BN>(p, M, t_row, row_base, lane, n_blk, stg, part, NPARTS, pf);
      if constexpr (EPI == EPI_SWIGLU) epi_swiglu<BN>(p, M, t_row, row_base, lane, n_blk, stg, part, NPARTS, rstd);
      if constexpr (EPI == EPI_QKV)
        epi_qkv<BN, DH>(p, M, t_row, row_base, lane, n_blk, stg, part, NPARTS, rstd, warp == 2 && lane == 0 && it == 0);
      tc_fence_before();
      mbar_arrive_cluster_relaxed(mapa_u32(smem_u32(&tempty[acc]), 0));
      if (warp == 2 && lane == 0 && it < 10) trace_stamp(p, 25 + it);
    }
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
