/*
 * te.h — C ABI of the B200-native batched-prefill text encoder (TE).
 *
 * The operation.  The paper's per-frame critical path is TE(x, p) -> h: the hidden states of
 * a vision-aware MLLM text encoder (Qwen3-VL-2B-shaped decoder stack) over ~64 visual +
 * ~64-128 instruction tokens per frame, run ONCE for a batch of B
 * frames to amortise its cost (PAPER.md:116; Table V, :249-258; Algorithm 1, :118-137), and
 * blocked in the reference stack by a `.item()` CPU-GPU synchronisation inside the rotary
 * position-id code.  BASELINE.json:north_star fixes the boundary:
 * "te_load_weights takes seeded bf16 weights.  te_encode(batch of frames, token embeddings,
 * per-frame text lengths, out hidden states) computes each frame's 3D M-RoPE (t,h,w) position
 * ids on the device ... so one captured CUDA graph covers the whole stack."  The decoder's
 * arithmetic is SURVEY.md §8(c) steps 1-5 (restated in DESIGN.md §2-3).
 *
 * Conventions.  Plain C, no torch types.  Every pointer argument says HOST or DEVICE.  All
 * functions return 0 (TE_OK) or a negative te_status; none throws, aborts or prints.
 * The library is single-GPU and not thread-safe per handle.  The small-batch (split-K) kernels
 * synchronise the CTAs of a group through device memory; they are launched as cooperative grids
 * (all CTAs resident at once, at most one CTA per SM), so other work on the GPU — another handle
 * on another stream, a denoiser (bench.py --overlap) — can delay them but not deadlock them.  There is NO CPU fallback:
 * te_create fails with TE_ERR_UNSUPPORTED on a device that is not sm_100.
 */
#ifndef TE_B200_H_
#define TE_B200_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct te_handle te_handle; /* opaque; owned by the library */

typedef enum te_status {
  TE_OK = 0,
  TE_ERR_INVALID_ARG = -1, /* null pointer, n_frames/grid/total_tokens out of range, bad config */
  TE_ERR_NOT_LOADED = -2,  /* te_encode before te_load_weights                                   */
  TE_ERR_BLOB_SIZE = -3,   /* n_bytes != te_blob_bytes(cfg)                                      */
  TE_ERR_CUDA = -4,        /* a CUDA call failed; text via te_last_error                         */
  TE_ERR_UNSUPPORTED = -5, /* head_dim not in {64,128}, dims not tileable, device not sm_100     */
  TE_ERR_DEVICE_CHECK = -6 /* te_query_async_error: device-side validation flag was raised       */
} te_status;

/* Decoder-stack shape + capacities (POD, copied at te_create).
 * Shapes are BASELINE.json:configs; symbols as in SURVEY.md §8. */
typedef struct te_config {
  int32_t n_layers;   /* L                                                         */
  int32_t hidden;     /* d; multiple of 128                                        */
  int32_t n_q_heads;  /* Hq                                                        */
  int32_t n_kv_heads; /* Hkv; Hq % Hkv == 0 (GQA: q head a uses kv head a / (Hq/Hkv)) */
  int32_t head_dim;   /* dh in {64, 128}                                           */
  int32_t ffn;        /* F; multiple of 128                                        */
  int32_t rope_sec_t, rope_sec_h, rope_sec_w; /* M-RoPE sections (pairs per axis), sum == dh/2 */
  float rms_eps;      /* RMSNorm epsilon (inside the root)                         */
  double rope_theta;  /* omega_i = theta^(-2i/dh)                                  */
  int32_t max_frames;           /* capacity: frames per call                       */
  int32_t max_tokens;           /* capacity: total packed tokens per call          */
  int32_t max_tokens_per_frame; /* capacity: S_b <= this (<= 256)                  */
  int32_t final_norm;           /* 0: out = raw last-layer residual (default); 1: RMSNorm(x; gf) */
  int32_t rope_interleaved;     /* 0 (default): sections are contiguous [t | h | w] over the frequency
                                   pairs; 1: pairs are dealt round-robin t,h,w,t,h,w,... to the axes that
                                   still have pairs left                      */
  int32_t max_prefix_tokens;    /* capacity of the shared text prefix (te_encode_prefix); 0 = none   */
} te_config;

/* Exact size in bytes of the canonical weight blob for cfg (see te_load_weights). */
size_t te_blob_bytes(const te_config* cfg);

/* Create an encoder on CUDA device `device`.  Allocates the workspace (qkv/attn/act/rotary
 * tables/position ids, sized by the capacities) and nothing per call afterwards. */
int te_create(const te_config* cfg, int device, te_handle** out);

/* Load the seeded bf16 weights (BASELINE.json:north_star).  `bf16_blob`: HOST or DEVICE
 * pointer to the canonical contiguous blob, every matrix row-major [out_features,
 * in_features] (y = x W^T), in this order:
 *   per layer l = 0..L-1:  g1[d]  Wq[Hq*dh,d]  Wk[Hkv*dh,d]  Wv[Hkv*dh,d]  gq[dh]  gk[dh]
 *                          Wo[d,Hq*dh]  g2[d]  Wgate[F,d]  Wup[F,d]  Wdown[d,F]
 *   then gf[d].
 * n_bytes must equal te_blob_bytes(cfg) (else TE_ERR_BLOB_SIZE).  Synchronous: the library
 * copies and repacks (fused QKV; gate/up rows interleaved per N-tile) into its own device
 * memory; the caller may free the blob on return. */
int te_load_weights(te_handle* h, const void* bf16_blob, size_t n_bytes);

/* Encode one batch of frames (the hot path).
 *   n_frames      B in [1, max_frames]
 *   grid_h,grid_w visual-token grid of every frame (row-major tokens, t = 0)
 *   embeds        DEVICE fp32 [total_tokens, hidden], frame-major packed: frame b occupies
 *                 rows cu[b]..cu[b+1), S_b = grid_h*grid_w + text_lens[b], visual tokens first
 *   text_lens     DEVICE int32 [n_frames]
 *   total_tokens  HOST value; must equal sum_b S_b (checked on the device, see below)
 *   out           DEVICE fp32 [total_tokens, hidden]; last-layer hidden states (the fp32
 *                 residual stream itself).  Must not alias embeds.
 *   cuda_stream   a cudaStream_t (NULL = legacy default stream)
 * Position ids (t,h,w), packing offsets and the rotary table are computed on the device from
 * text_lens; the call enqueues work and returns: NO stream synchronisation, NO device->host
 * copy, no allocation once the (shape, pointer) key has been seen — the property the paper's
 * TE lacks.  The whole stack is one CUDA-graph launch (cached per key).
 * Conditions only knowable on the device (sum of lengths != total_tokens, text_len < 0,
 * S_b > max_tokens_per_frame) raise a sticky device flag; the kernels then touch no row
 * >= total_tokens; read the flag with te_query_async_error. */
int te_encode(te_handle* h, int32_t n_frames, int32_t grid_h, int32_t grid_w,
              const float* embeds, const int32_t* text_lens, int32_t total_tokens, float* out,
              void* cuda_stream);

/* Shared text prefix with K/V reuse.  The real chat template puts the same
 * system prompt (80 tokens: 13 % of the TE's time) in front of every frame's image.  Being
 * a causal prefix it sees nothing after it, so its hidden states and its per-layer keys/values are the
 * same for every frame and every call: te_encode_prefix runs the stack ONCE over the prefix tokens
 * (ids t=h=w=0..P-1) and keeps every layer's K/V (after QK-norm and rotation) in library memory.
 * Afterwards te_encode treats each frame as [prefix | grid | text] WITHOUT re-encoding the prefix:
 * `embeds`/`out` still hold only the S_b = grid_h*grid_w + text_lens[b] own tokens of each frame, their
 * ids continue from the prefix (visual token k: (P, P + k/grid_w, P + k%grid_w); text j:
 * P + max(grid_h,grid_w) + j) and their queries attend to the P cached keys plus their own causal keys.
 *   prefix_embeds  DEVICE fp32 [prefix_len, hidden]
 *   prefix_len     P in [0, max_prefix_tokens]; 0 removes the prefix
 *   prefix_out     DEVICE fp32 [prefix_len, hidden] or NULL: hidden states of the prefix tokens
 * Synchronous with respect to `cuda_stream` ordering only (work is enqueued; no host sync). */
int te_encode_prefix(te_handle* h, const float* prefix_embeds, int32_t prefix_len, float* prefix_out,
                     void* cuda_stream);

/* Same call with HOST buffers (end-to-end path): copies embeds/text_lens host->device into
 * library staging buffers, runs te_encode, copies `out` device->host, and synchronises.
 * embeds_host / out_host: HOST fp32 [total_tokens, hidden] (pinned memory recommended);
 * text_lens_host: HOST int32 [n_frames]; total_tokens is computed from text_lens_host. */
int te_encode_host(te_handle* h, int32_t n_frames, int32_t grid_h, int32_t grid_w,
                   const float* embeds_host, const int32_t* text_lens_host, float* out_host);

/* Pipelined host path: te_encode_host_submit enqueues [host->device copy | te_encode | device->host copy] of
 * one batch on three library streams chained by events and returns at once with a slot id (0 or 1);
 * te_encode_host_wait(slot) blocks until that batch's out_host is complete.  Two batches can be in flight:
 * submitting batch n+1 before waiting for batch n overlaps the copies of one with the kernels of the other
 * (te_encode_host = submit + wait).  The HOST buffers must stay valid until the wait (pinned memory for real
 * overlap).  A third submit without a wait returns TE_ERR_INVALID_ARG. */
int te_encode_host_submit(te_handle* h, int32_t n_frames, int32_t grid_h, int32_t grid_w,
                          const float* embeds_host, const int32_t* text_lens_host, float* out_host,
                          int32_t* slot_out);
int te_encode_host_wait(te_handle* h, int32_t slot);

/* Synchronises the device and returns TE_ERR_DEVICE_CHECK if the device-side validation flag
 * was raised since the last query (and clears it), TE_ERR_CUDA on a CUDA error, else TE_OK. */
int te_query_async_error(te_handle* h);

/* Options. */
enum {
  TE_OPT_USE_GRAPH = 0,    /* 1 (default): te_encode = one cudaGraphLaunch; 0: direct launches   */
  TE_OPT_KERNEL_TIMING = 1,/* 1: direct launches bracketed by CUDA events per kernel (implies no
                              graph); read with te_kernel_times.  Measurement aid, default 0.     */
  TE_OPT_CTA_PAIR = 2,     /* GEMM tiling: 0 = one CTA per 128-row tile, 1 = CTA pairs (cta_group::2,
                              256-row tiles), 2 = auto by token count (default)                    */
  TE_OPT_RESID_BLOCK_N = 3,/* tile width (128 default, or 256) of the O-proj / down GEMMs          */
  TE_OPT_PDL = 4,          /* 1 (default): kernels are chained with programmatic dependent launch   */
  TE_OPT_TRACE = 5,        /* 1: CTA-pair GEMM kernels stamp %globaltimer at pipeline events (debug
                              aid; read with te_debug_tap(TE_TAP_TRACE)); default 0                 */
  TE_OPT_ATTN_IMPL = 6,    /* attention kernel: 1 (default) = tcgen05 kernel (S, P, O in tensor memory)
                              when Hq/Hkv is a power of two <= 8, 0 = mma.sync flash kernel          */
  TE_OPT_STREAM_K = 8,     /* 1: the CTA-pair GEMM kernels give every SM pair an equal contiguous share of the
                              (tile, k-block) work units (stream-K); a tile cut by a share boundary is completed
                              by the pair that holds its first k-blocks, on top of the other pieces' fp32 partials
                              summed in a fixed order (deterministic).  0 (default): whole tiles, round-robin —
                              measured faster on every config                                    */
  TE_OPT_RESID_WIDE = 9,   /* O-proj / down on CTA pairs: 1 (default) = when their 128-wide tiles would need two or
                              more waves, ONE wave of wide tiles (width = hidden / n rounded up to 32, <= 512
                              columns, two MMAs per k-step; te_gemm_wide.cuh); 0 = never; n in 2..16 = always,
                              with n tiles across the hidden dimension (tests)                                  */
  TE_OPT_L2_RESIDUAL = 10, /* 1 (default): the fp32 residual stream (`out`) is an L2-persisting access-policy window
                              of every kernel, so that the residual GEMMs' read-add-write passes stay out of DRAM.
                              The first te_encode raises the DEVICE-WIDE limit cudaLimitPersistingL2CacheSize to
                              min(max_tokens * hidden * 4, 64 MiB, device maximum).  0: no window                 */
  TE_OPT_SPLIT_K = 7       /* 1 (default): small batches (fewer 128-row tiles than SMs in a GEMM, no
                              CTA pairs) run the split-K kernel: several CTAs per output tile, each
                              streaming its own K-slice of the weights; partial tiles are summed in a
                              fixed order (deterministic).  0: one CTA per tile                      */
};
int te_set_option(te_handle* h, int option, int value);

/* Number of kernels the library has launched so far on behalf of te_encode (graph replays
 * count the kernel nodes they contain).  For bench.py's `gpu_launches`. */
int64_t te_kernel_launches(te_handle* h);

/* Per-kernel-class device time accumulated by calls made under TE_OPT_KERNEL_TIMING, measured with
 * CUDA events on the launching stream.  Synchronises; fills ms_sum[TE_KCLASS_COUNT] and
 * n_launches[TE_KCLASS_COUNT] (HOST arrays) and resets the accumulation. */
enum {
  TE_KCLASS_SCAN = 0, TE_KCLASS_PREP = 1, TE_KCLASS_QKV = 2, TE_KCLASS_ATTN = 3, TE_KCLASS_OPROJ = 4,
  TE_KCLASS_GATEUP = 5, TE_KCLASS_DOWN = 6, TE_KCLASS_FINAL_NORM = 7, TE_KCLASS_COUNT = 8
};
int te_kernel_times(te_handle* h, float* ms_sum, int32_t* n_launches);

/* ---- test-only taps (SURVEY.md §8b "Debug taps") ------------------------------------------
 * te_debug_set_range restricts subsequent te_encode calls to layers [layer_begin, layer_end)
 * (embeds is then the teacher-forced input residual of layer_begin) and, if stop_after_attn,
 * stops the last layer after the O-projection residual add.  (0, n_layers, 0) restores the
 * full stack.  te_debug_tap synchronises and copies the CURRENT content of a workspace buffer
 * (as left by the last te_encode, i.e. of the last layer run) to `dst` (HOST). */
enum {
  TE_TAP_POS = 0,        /* int32 [3, T]        rows t,h,w                       */
  TE_TAP_CU_SEQLENS = 1, /* int32 [B+1]                                         */
  TE_TAP_COS = 2,        /* fp32  [T, dh/2]                                     */
  TE_TAP_SIN = 3,        /* fp32  [T, dh/2]                                     */
  TE_TAP_QKV = 4,        /* bf16  [T, (Hq+2Hkv)*dh]  q (normed+rotated) | k | v  */
  TE_TAP_ATTN = 5,       /* bf16  [T, Hq*dh]                                    */
  TE_TAP_ACT = 6,        /* bf16  [T, F]       silu(gate)*up                    */
  TE_TAP_TRACE = 7       /* u64   [4 GEMM classes (qkv,oproj,gateup,down)][n_SMs][48] ns stamps
                            of the last launch of each class (TE_OPT_TRACE)     */
};
int te_debug_set_range(te_handle* h, int32_t layer_begin, int32_t layer_end,
                       int32_t stop_after_attn);
int te_debug_tap(te_handle* h, int what, void* dst_host, size_t n_bytes);

/* Test-only: C[M,N] (DEVICE fp32, row-major) = A[M,K] * B[N,K]^T with A, B DEVICE bf16
 * row-major, through the same TMA + tcgen05 main loop as the stack's GEMMs (plain epilogue).
 * K % 64 == 0, N % block_n == 0, block_n in {128, 256}; cta_pair = 1 selects the cta_group::2
 * kernel (256-row tiles) with whole tiles per pair, cta_pair = 2 the same kernel with stream-K
 * scheduling.  Synchronous. */
int te_debug_gemm(int device, const void* a_bf16, const void* b_bf16, float* c, int32_t m,
                  int32_t n, int32_t k, int32_t block_n, int32_t cta_pair);

/* Test-only: the same product through the split-K kernel (te_gemm_splitk.cuh): `splits` CTAs
 * (1..8, <= k/64) per 128 x block_n tile, fixed-order reduction of the fp32 partial tiles.
 * Needs tiles * splits <= number of SMs (TE_ERR_UNSUPPORTED otherwise).  Synchronous. */
int te_debug_gemm_splitk(int device, const void* a_bf16, const void* b_bf16, float* c, int32_t m,
                         int32_t n, int32_t k, int32_t block_n, int32_t splits);

void te_destroy(te_handle* h);
const char* te_strerror(int code);
const char* te_last_error(te_handle* h); /* valid until the next call on h */

#ifdef __cplusplus
}
#endif
#endif /* TE_B200_H_ */
