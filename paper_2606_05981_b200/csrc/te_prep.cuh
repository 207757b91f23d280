// te_prep.cuh — a0 of SURVEY.md §8(a): packing offsets, 3D M-RoPE position ids and the rotary
// cos/sin table computed ON THE DEVICE from text_lens (this replaces the `.item()` host
// round-trip the paper locates in the TE's rotary code), plus the initial
// copy embeds -> fp32 residual (= out) with the first layer's RMSNorm statistics.
// Also: final RMSNorm (a6) and the gate/up weight interleave used by te_load_weights.
#pragma once
#include <cuda_bf16.h>
#include <cuda_runtime.h>
#include <stdint.h>

#include "te_gemm8.cuh"  // DynParams, MXFP8 quantiser

namespace te {

// Refreshes the per-call values ahead of the stack (one thread; values arrive as kernel parameters, so the call
// needs no host staging memory and can be captured into a caller's graph as well).
__global__ void te_set_dyn_kernel(DynParams* dyn, const DynParams v) {
  if (threadIdx.x == 0 && blockIdx.x == 0) *dyn = v;
}

enum { FLAG_BAD_LEN = 1, FLAG_BAD_TOTAL = 2, FLAG_TOO_LONG = 4 };
constexpr int PREP_PAD_ROWS = 16;  // rows past the call's tokens that te_prep_kernel zeroes in the qkv workspace

struct PrepParams {
  const DynParams* dyn;      // embeds [T, d], text_lens [B], total_tokens of this call
  float* out;                // [T, d]  fp32 residual stream (library workspace)
  int32_t* cu;               // [B+1]   packing offsets (written by block 0)
  int32_t* flag;             // sticky validation flag
  int32_t* pos;              // [3, T]
  float* cos_t;              // [T, dh/2]
  float* sin_t;
  const double* inv_freq;       // [dh/2]  omega_i = theta^(-2i/dh)
  const __nv_bfloat16* g_first; // gain of the first RMSNorm that will consume the residual
  __nv_bfloat16* xg;            // [T, d]  bf16(x * g_first)
  float* ssq;                   // [T][ssq_stride], first ssq_parts entries of a row used
  int ssq_parts, ssq_stride;
  int n_frames, d, half_dim, max_tokens_per_frame;
  int grid_h, grid_w;
  int pos_offset;   // length P of the shared text prefix in front of every frame (ids continue from it)
  // The attention kernel multiplies keys / values in granules of 16 rows: a frame whose length is not a multiple of
  // 16 reads up to 15 rows past its end with zero weight.  Those rows are the next frame's or, for the last frame of
  // a call, rows [T, T + 16) of the qkv workspace, which no kernel of THIS call writes (the activation tensor maps span
  // the whole workspace; they are encoded once, not per token count).  Blocks T .. T+15 of this kernel zero them, so
  // that 0 * (what an earlier, larger call left there) can never be 0 * NaN.
  uint4* qkv_rows;  // [rows, qkv_row_vec16] the qkv workspace as 16-byte vectors
  int qkv_row_vec16;
  // MXFP8 variant (te_config.weight_dtype = 1): x * g_first is written as E4M3 + block scales instead of bf16
  uint8_t* xg8;     // [T, d] or null
  uint8_t* sf_xg;   // tiled scales (te_gemm8.cuh)
  int8_t axis[64];  // M-RoPE axis (0 = t, 1 = h, 2 = w) of frequency pair i (contiguous or interleaved sections)
};

// One block per token.  Warp 0 of EVERY block scans text_lens itself (B is a few dozen frames; the
// scan is cheaper than a second kernel and a grid-wide dependency): cu[b+1] = min(sum_{i<=b} S_i, T),
// clamped so that no kernel touches rows beyond the caller's buffers even when validation fails; the
// token's frame is the largest b with cu[b] <= tok.  Block 0 also publishes cu[] and the validation flag.
__global__ void __launch_bounds__(256) te_prep_kernel(const PrepParams p) {
  __shared__ int s_start, s_gh, s_gw;
  __shared__ float s_ss[8];
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int tok = blockIdx.x;
  const int n_vis = p.grid_h * p.grid_w;
  asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
  asm volatile("griddepcontrol.wait;" ::: "memory");  // the previous call's kernels still read cu / flag / out
  const int total_tokens = p.dyn->total_tokens;
  const int32_t* const text_lens = p.dyn->text_lens;
  const int32_t* const grids = p.dyn->grids;  // per-frame (grid_h, grid_w) (te_encode_ex) or null
  if (warp == 0) {
    long long carry = 0;
    int best_b = 0, best_start = 0, f = 0;
    for (int base = 0; base < p.n_frames; base += 32) {
      const int b = base + lane;
      int sb = 0;
      if (b < p.n_frames) {
        int tl = text_lens[b];
        if (tl < 0) { f |= FLAG_BAD_LEN; tl = 0; }
        int nv = n_vis;
        if (grids != nullptr) {
          int gh = grids[2 * b], gw = grids[2 * b + 1];
          if (gh < 0 || gw < 0) { f |= FLAG_BAD_LEN; gh = gw = 0; }
          nv = (gh > p.max_tokens_per_frame || gw > p.max_tokens_per_frame) ? p.max_tokens_per_frame + 1 : gh * gw;
        }
        sb = nv + tl;
        if (sb > p.max_tokens_per_frame) f |= FLAG_TOO_LONG;
      }
      long long incl = sb;
#pragma unroll
      for (int off = 1; off < 32; off <<= 1) {
        const long long o = __shfl_up_sync(0xffffffffu, incl, off);
        if (lane >= off) incl += o;
      }
      incl += carry;
      if (b < p.n_frames) {
        const long long excl = incl - sb;
        const int start = static_cast<int>(excl < total_tokens ? excl : total_tokens);
        if (start <= tok) { best_b = b; best_start = start; }  // starts are non-decreasing in b
        if (tok == 0) {
          if (b == 0) p.cu[0] = 0;
          p.cu[b + 1] = static_cast<int32_t>(incl < total_tokens ? incl : total_tokens);
        }
      }
      carry = __shfl_sync(0xffffffffu, incl, 31);
    }
    if (carry != total_tokens) f |= FLAG_BAD_TOTAL;
#pragma unroll
    for (int off = 16; off > 0; off >>= 1) {
      const int ob = __shfl_xor_sync(0xffffffffu, best_b, off);
      const int os = __shfl_xor_sync(0xffffffffu, best_start, off);
      if (ob > best_b) { best_b = ob; best_start = os; }
      f |= __shfl_xor_sync(0xffffffffu, f, off);
    }
    if (lane == 0) {
      s_start = best_start;
      s_gh = grids != nullptr ? max(grids[2 * best_b], 0) : p.grid_h;
      s_gw = grids != nullptr ? max(grids[2 * best_b + 1], 0) : p.grid_w;
      if (tok == 0 && f) atomicOr(p.flag, f);
    }
  }
  __syncthreads();
  if (tok >= total_tokens) {
    if (tok < total_tokens + PREP_PAD_ROWS)
      for (int i = threadIdx.x; i < p.qkv_row_vec16; i += 256) p.qkv_rows[(size_t)tok * p.qkv_row_vec16 + i] = make_uint4(0u, 0u, 0u, 0u);
    return;
  }
  const int n = tok - s_start;
  const int gh = s_gh, gw = s_gw;  // this token's frame's grid
  int pt, ph, pw;
  const int off = p.pos_offset;
  if (n < gh * gw) {
    pt = off; ph = off + n / gw; pw = off + n % gw;  // visual token: row-major grid, t constant
  } else {
    pt = ph = pw = off + max(gh, gw) + (n - gh * gw);  // text: continues from max grid id + 1
  }
  if (threadIdx.x == 0) {
    p.pos[tok] = pt;
    p.pos[total_tokens + tok] = ph;
    p.pos[2 * total_tokens + tok] = pw;
  }
  // the rotary table on the last warps, so that it overlaps the row copy of the first ones
  for (int i = 255 - threadIdx.x; i < p.half_dim; i += 256) {
    const int ax = p.axis[i];
    const int pid = (ax == 0) ? pt : ((ax == 1) ? ph : pw);
    double sn, cs;
    sincos(static_cast<double>(pid) * p.inv_freq[i], &sn, &cs);
    p.cos_t[(size_t)tok * p.half_dim + i] = static_cast<float>(cs);
    p.sin_t[(size_t)tok * p.half_dim + i] = static_cast<float>(sn);
  }
  // residual copy + sum of squares + bf16(x * g)
  const bool e16 = p.dyn->embeds_bf16 != 0;  // bf16 embeddings (te_encode_ex): widened exactly to the fp32 residual
  const float4* src = reinterpret_cast<const float4*>(static_cast<const float*>(p.dyn->embeds) + (size_t)tok * p.d);
  const uint2* src16 = reinterpret_cast<const uint2*>(static_cast<const __nv_bfloat16*>(p.dyn->embeds) + (size_t)tok * p.d);
  float4* dst = reinterpret_cast<float4*>(p.out + (size_t)tok * p.d);
  float ss = 0.f;
  for (int c4 = threadIdx.x; c4 < p.d / 4; c4 += 256) {
    float4 v;
    if (e16) {
      const uint2 u = __ldg(src16 + c4);
      v = make_float4(__uint_as_float(u.x << 16), __uint_as_float(u.x & 0xFFFF0000u), __uint_as_float(u.y << 16),
                      __uint_as_float(u.y & 0xFFFF0000u));
    } else {
      v = __ldg(src + c4);
    }
    dst[c4] = v;
    ss = fmaf(v.x, v.x, ss); ss = fmaf(v.y, v.y, ss); ss = fmaf(v.z, v.z, ss); ss = fmaf(v.w, v.w, ss);
    const uint2 g = __ldg(reinterpret_cast<const uint2*>(p.g_first) + c4);
    __nv_bfloat162 o0 = __floats2bfloat162_rn(v.x * __uint_as_float(g.x << 16), v.y * __uint_as_float(g.x & 0xFFFF0000u));
    __nv_bfloat162 o1 = __floats2bfloat162_rn(v.z * __uint_as_float(g.y << 16), v.w * __uint_as_float(g.y & 0xFFFF0000u));
    uint2 o;
    o.x = *reinterpret_cast<uint32_t*>(&o0);
    o.y = *reinterpret_cast<uint32_t*>(&o1);
    if (p.xg8 == nullptr) {
      reinterpret_cast<uint2*>(p.xg + (size_t)tok * p.d)[c4] = o;
    } else {
      // 8 consecutive lanes hold one 32-column MX block (d % 128 == 0: whole blocks, whole warps)
      const float q0 = v.x * __uint_as_float(g.x << 16), q1 = v.y * __uint_as_float(g.x & 0xFFFF0000u);
      const float q2 = v.z * __uint_as_float(g.y << 16), q3 = v.w * __uint_as_float(g.y & 0xFFFF0000u);
      float amax = fmaxf(fmaxf(fabsf(q0), fabsf(q1)), fmaxf(fabsf(q2), fabsf(q3)));
      amax = fmaxf(amax, __shfl_xor_sync(0xffffffffu, amax, 1));
      amax = fmaxf(amax, __shfl_xor_sync(0xffffffffu, amax, 2));
      amax = fmaxf(amax, __shfl_xor_sync(0xffffffffu, amax, 4));
      const uint32_t code = mx_scale_code(amax);
      const float inv = mx_inv_scale(code);
      reinterpret_cast<uint32_t*>(p.xg8 + (size_t)tok * p.d)[c4] = pack_e4m3x4(q0 * inv, q1 * inv, q2 * inv, q3 * inv);
      if ((c4 & 7) == 0) p.sf_xg[mx_sf_offset(tok, c4 >> 3, p.d / 128)] = static_cast<uint8_t>(code);
    }
  }
#pragma unroll
  for (int off = 16; off > 0; off >>= 1) ss += __shfl_xor_sync(0xffffffffu, ss, off);
  if (lane == 0) s_ss[warp] = ss;
  __syncthreads();
  if (threadIdx.x == 0) {
    float tot = 0.f;
#pragma unroll
    for (int i = 0; i < 8; ++i) tot += s_ss[i];  // fixed order: deterministic
    p.ssq[(size_t)tok * p.ssq_stride] = tot;
    for (int i = 1; i < p.ssq_parts; ++i) p.ssq[(size_t)tok * p.ssq_stride + i] = 0.f;
  }
}

// a6: out <- RMSNorm(x; gf), fp32, one warp per row (x: the library's residual stream, out: the caller's buffer).
__global__ void __launch_bounds__(256) te_final_norm_kernel(const float* __restrict__ x, const DynParams* __restrict__ dyn,
                                                            const __nv_bfloat16* __restrict__ gf, int d, float eps) {
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int tok = blockIdx.x * 8 + warp;
  asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
  asm volatile("griddepcontrol.wait;" ::: "memory");
  if (tok >= dyn->total_tokens) return;
  const float4* row = reinterpret_cast<const float4*>(x + (size_t)tok * d);
  float4* dst = reinterpret_cast<float4*>(dyn->out + (size_t)tok * d);
  float ss = 0.f;
  for (int c4 = lane; c4 < d / 4; c4 += 32) {
    const float4 v = row[c4];
    ss = fmaf(v.x, v.x, ss); ss = fmaf(v.y, v.y, ss); ss = fmaf(v.z, v.z, ss); ss = fmaf(v.w, v.w, ss);
  }
#pragma unroll
  for (int off = 16; off > 0; off >>= 1) ss += __shfl_xor_sync(0xffffffffu, ss, off);
  const float rstd = 1.0f / sqrtf(ss / static_cast<float>(d) + eps);
  for (int c4 = lane; c4 < d / 4; c4 += 32) {
    float4 v = row[c4];
    const uint2 g = __ldg(reinterpret_cast<const uint2*>(gf) + c4);
    v.x = v.x * rstd * __uint_as_float(g.x << 16);
    v.y = v.y * rstd * __uint_as_float(g.x & 0xFFFF0000u);
    v.z = v.z * rstd * __uint_as_float(g.y << 16);
    v.w = v.w * rstd * __uint_as_float(g.y & 0xFFFF0000u);
    dst[c4] = v;
  }
}

// te_load_weights: interleave [Wgate; Wup] per N-tile of `bn` rows so that one GEMM tile holds
// matching gate (first bn/2 rows) and up (last bn/2 rows) columns.  One block per destination row.
__global__ void te_interleave_gate_up_kernel(const uint4* __restrict__ gate, const uint4* __restrict__ up,
                                             uint4* __restrict__ dst, int ffn, int row_vec16, int bn) {
  const int r = blockIdx.x;  // destination row in [0, 2*ffn)
  const int tile = r / bn, within = r % bn, half = bn / 2;
  const uint4* src = (within < half) ? gate + (size_t)(tile * half + within) * row_vec16
                                     : up + (size_t)(tile * half + within - half) * row_vec16;
  for (int i = threadIdx.x; i < row_vec16; i += blockDim.x) dst[(size_t)r * row_vec16 + i] = src[i];
}

}  // namespace te
