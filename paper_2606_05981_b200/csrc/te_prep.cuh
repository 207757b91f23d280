// te_prep.cuh — a0 of SURVEY.md §8(a): packing offsets, 3D M-RoPE position ids and the rotary
// cos/sin table computed ON THE DEVICE from text_lens (this replaces the `.item()` host
// round-trip the paper locates in the TE's rotary code), plus the initial
// copy embeds -> fp32 residual (= out) with the first layer's RMSNorm statistics.
// Also: final RMSNorm (a6) and the gate/up weight interleave used by te_load_weights.
#pragma once
#include <cuda_bf16.h>
#include <cuda_runtime.h>
#include <stdint.h>

namespace te {

enum { FLAG_BAD_LEN = 1, FLAG_BAD_TOTAL = 2, FLAG_TOO_LONG = 4 };

struct PrepParams {
  const float* embeds;       // [T, d]
  const int32_t* text_lens;  // [B]
  float* out;                // [T, d]  fp32 residual stream
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
  int n_frames, total_tokens, d, half_dim, max_tokens_per_frame;
  int grid_h, grid_w;
  int pos_offset;   // length P of the shared text prefix in front of every frame (ids continue from it)
  int8_t axis[64];  // M-RoPE axis (0 = t, 1 = h, 2 = w) of frequency pair i (contiguous or interleaved sections)
};

// One block per token.  Warp 0 of EVERY block scans text_lens itself (B is a few dozen frames; the
// scan is cheaper than a second kernel and a grid-wide dependency): cu[b+1] = min(sum_{i<=b} S_i, T),
// clamped so that no kernel touches rows beyond the caller's buffers even when validation fails; the
// token's frame is the largest b with cu[b] <= tok.  Block 0 also publishes cu[] and the validation flag.
__global__ void __launch_bounds__(256) te_prep_kernel(const PrepParams p) {
  __shared__ int s_start;
  __shared__ float s_ss[8];
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int tok = blockIdx.x;
  const int n_vis = p.grid_h * p.grid_w;
  asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
  asm volatile("griddepcontrol.wait;" ::: "memory");  // the previous call's kernels still read cu / flag / out
  if (warp == 0) {
    long long carry = 0;
    int best_b = 0, best_start = 0, f = 0;
    for (int base = 0; base < p.n_frames; base += 32) {
      const int b = base + lane;
      int sb = 0;
      if (b < p.n_frames) {
        int tl = p.text_lens[b];
        if (tl < 0) { f |= FLAG_BAD_LEN; tl = 0; }
        sb = n_vis + tl;
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
        const int start = static_cast<int>(excl < p.total_tokens ? excl : p.total_tokens);
        if (start <= tok) { best_b = b; best_start = start; }  // starts are non-decreasing in b
        if (tok == 0) {
          if (b == 0) p.cu[0] = 0;
          p.cu[b + 1] = static_cast<int32_t>(incl < p.total_tokens ? incl : p.total_tokens);
        }
      }
      carry = __shfl_sync(0xffffffffu, incl, 31);
    }
    if (carry != p.total_tokens) f |= FLAG_BAD_TOTAL;
#pragma unroll
    for (int off = 16; off > 0; off >>= 1) {
      const int ob = __shfl_xor_sync(0xffffffffu, best_b, off);
      const int os = __shfl_xor_sync(0xffffffffu, best_start, off);
      if (ob > best_b) { best_b = ob; best_start = os; }
      f |= __shfl_xor_sync(0xffffffffu, f, off);
    }
    if (lane == 0) {
      s_start = best_start;
      if (tok == 0 && f) atomicOr(p.flag, f);
    }
  }
  __syncthreads();
  if (tok >= p.total_tokens) return;
  const int n = tok - s_start;
  int pt, ph, pw;
  const int off = p.pos_offset;
  if (n < n_vis) {
    pt = off; ph = off + n / p.grid_w; pw = off + n % p.grid_w;  // visual token: row-major grid, t constant
  } else {
    pt = ph = pw = off + max(p.grid_h, p.grid_w) + (n - n_vis);  // text: continues from max grid id + 1
  }
  if (threadIdx.x == 0) {
    p.pos[tok] = pt;
    p.pos[p.total_tokens + tok] = ph;
    p.pos[2 * p.total_tokens + tok] = pw;
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
  const float4* src = reinterpret_cast<const float4*>(p.embeds + (size_t)tok * p.d);
  float4* dst = reinterpret_cast<float4*>(p.out + (size_t)tok * p.d);
  float ss = 0.f;
  for (int c4 = threadIdx.x; c4 < p.d / 4; c4 += 256) {
    const float4 v = __ldg(src + c4);
    dst[c4] = v;
    ss = fmaf(v.x, v.x, ss); ss = fmaf(v.y, v.y, ss); ss = fmaf(v.z, v.z, ss); ss = fmaf(v.w, v.w, ss);
    const uint2 g = __ldg(reinterpret_cast<const uint2*>(p.g_first) + c4);
    __nv_bfloat162 o0 = __floats2bfloat162_rn(v.x * __uint_as_float(g.x << 16), v.y * __uint_as_float(g.x & 0xFFFF0000u));
    __nv_bfloat162 o1 = __floats2bfloat162_rn(v.z * __uint_as_float(g.y << 16), v.w * __uint_as_float(g.y & 0xFFFF0000u));
    uint2 o;
    o.x = *reinterpret_cast<uint32_t*>(&o0);
    o.y = *reinterpret_cast<uint32_t*>(&o1);
    reinterpret_cast<uint2*>(p.xg + (size_t)tok * p.d)[c4] = o;
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

// a6: out <- RMSNorm(out; gf), fp32, one warp per row.
__global__ void __launch_bounds__(256) te_final_norm_kernel(float* __restrict__ x, const __nv_bfloat16* __restrict__ gf,
                                                            int total_tokens, int d, float eps) {
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int tok = blockIdx.x * 8 + warp;
  asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
  asm volatile("griddepcontrol.wait;" ::: "memory");
  if (tok >= total_tokens) return;
  float4* row = reinterpret_cast<float4*>(x + (size_t)tok * d);
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
    row[c4] = v;
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
