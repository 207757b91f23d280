// te_vision.cuh — data movement around the vision tower ("processed by
// Qwen3-VL's vision tower", :23 "256x256 source patch -> ~64 visual tokens"; readings Q28-Q31 of DESIGN.md §3).
// The arithmetic of the front end runs in the stack's own kernels: the patch embedding and the merger are tcgen05
// GEMMs (plain epilogue), the tower is the decoder stack with non-causal attention (te_config.non_causal).  What is
// left for this file is the cutting and gathering that turns their operands into row-major bf16 matrices:
//   te_patchify_kernel      pixels [B, H, W, 3] fp32 -> A_pe [B*gh*gw, P*P*3] bf16   (Q28: (dy, dx, channel) order)
//   te_merge2x2_kernel      tower output [B*gh*gw, d_v] fp32 -> A_m [B*(gh/2)*(gw/2), 4*d_v] bf16   (Q30)
//   te_scatter_visual_kernel  merged embeddings [B*n_vis, d] fp32 -> rows cu[b] .. cu[b]+n_vis of the decoder's
//                             packed `embeds` (cu from the device-side text_lens: no host round trip here either)
#pragma once
#include <cuda_bf16.h>
#include <cuda_runtime.h>
#include <stdint.h>

namespace te {

// One block per patch; a patch row (dy) is P*3 contiguous floats of the image.
__global__ void __launch_bounds__(256) te_patchify_kernel(const float* __restrict__ pixels, __nv_bfloat16* __restrict__ a,
                                                          int H, int W, int P, int gh, int gw) {
  const int patch = blockIdx.x;
  const int per = gh * gw;
  const int b = patch / per, r = patch % per, py = r / gw, px = r % gw;
  const int row_len = P * 3;
  const int n = P * row_len;
  const float* src = pixels + ((size_t)(b * H + py * P) * W + (size_t)px * P) * 3;
  __nv_bfloat16* dst = a + (size_t)patch * n;
  for (int i = threadIdx.x; i < n; i += blockDim.x) {
    const int dy = i / row_len, c = i - dy * row_len;
    dst[i] = __float2bfloat16_rn(src[(size_t)dy * W * 3 + c]);
  }
}

// One block per merged token (my, mx) of frame b: the four patches (2my+dy, 2mx+dx), (dy, dx) row-major, side by side.
__global__ void __launch_bounds__(256) te_merge2x2_kernel(const float* __restrict__ h, __nv_bfloat16* __restrict__ a, int gh,
                                                          int gw, int d) {
  const int mt = blockIdx.x;
  const int mh = gh / 2, mw = gw / 2;
  const int b = mt / (mh * mw), r = mt % (mh * mw), my = r / mw, mx = r % mw;
  const int d4 = d / 4;
  for (int i = threadIdx.x; i < 4 * d4; i += blockDim.x) {
    const int part = i / d4, c4 = i - part * d4;
    const int dy = part >> 1, dx = part & 1;
    const size_t src_row = (size_t)b * gh * gw + (size_t)(2 * my + dy) * gw + (2 * mx + dx);
    const float4 v = *reinterpret_cast<const float4*>(h + src_row * d + 4 * c4);
    __nv_bfloat162 lo = __floats2bfloat162_rn(v.x, v.y), hi = __floats2bfloat162_rn(v.z, v.w);
    uint2 o;
    o.x = *reinterpret_cast<uint32_t*>(&lo);
    o.y = *reinterpret_cast<uint32_t*>(&hi);
    *reinterpret_cast<uint2*>(a + (size_t)mt * 4 * d + (size_t)part * d + 4 * c4) = o;
  }
}

// One block per merged token: row b*n_vis + m of `vis` -> row cu[b] + m of `embeds`, cu[b] = b*n_vis + sum of the
// text lengths of the frames before b (negative lengths count as 0, as in te_prep_kernel).  text_lens == nullptr:
// the frames are packed without text (embeds = [B*n_vis, d]).  `embeds` has total_tokens rows and text_lens is
// unvalidated device data: a row at or past total_tokens is NOT written, and the sticky validation flag (the tower
// handle's; same bits as te_prep_kernel) gets 1 for a negative length, 2 when the packed frames do not fit in (or, seen
// from the last frame, do not add up to) total_tokens.
__global__ void __launch_bounds__(256) te_scatter_visual_kernel(const float* __restrict__ vis, float* __restrict__ embeds,
                                                                const int32_t* __restrict__ text_lens, int n_vis, int d,
                                                                int n_frames, int total_tokens, int32_t* __restrict__ flag) {
  const int mt = blockIdx.x;
  const int b = mt / n_vis, m = mt - b * n_vis;
  long long row = (long long)b * n_vis + m;
  int bad = 0;
  if (text_lens != nullptr)
    for (int i = 0; i < b; ++i) {
      const int tl = text_lens[i];
      if (tl < 0) bad |= 1;
      row += tl > 0 ? tl : 0;
    }
  if (m == n_vis - 1 && b == n_frames - 1) {  // the last visual row of the call: the whole sum is known here
    const int tl = text_lens != nullptr ? text_lens[b] : 0;
    if (tl < 0) bad |= 1;
    if (row + 1 + (tl > 0 ? tl : 0) != (long long)total_tokens) bad |= 2;
  }
  if (row >= (long long)total_tokens) bad |= 2;
  if (bad && threadIdx.x == 0) atomicOr(flag, bad);
  if (row >= (long long)total_tokens) return;
  const float4* src = reinterpret_cast<const float4*>(vis + (size_t)mt * d);
  float4* dst = reinterpret_cast<float4*>(embeds + (size_t)row * d);
  for (int i = threadIdx.x; i < d / 4; i += blockDim.x) dst[i] = src[i];
}

}  // namespace te
