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
 * The library is single-GPU; a handle must not be used from two host threads at once, different handles may be
 * (all launch state is per handle).  One handle serves ONE stream at a time: every call works in the handle's single
 * workspace (residual, q/k/v, activations) and refreshes its single block of per-call parameters on the stream it is
 * given, so a call enqueued on stream B while an earlier call of the same handle may still be running on stream A
 * races with it — order them with an event, or use one handle per stream.  The small-batch (split-K) kernels
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
  TE_ERR_DEVICE_CHECK = -6, /* te_query_async_error: device-side validation flag was raised      */
  TE_ERR_TOO_LARGE = -7    /* te_matmul_noalloc: the problem needs more scratch than the library's
                              built-in array holds (TE_NOALLOC_SCRATCH_BYTES)                     */
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
  int32_t weight_dtype;         /* 0 (default): bf16 weights and GEMM operands.  1: block-scaled FP8 (OCP MXFP8; SURVEY.md
                                   §8(f) NEXT-2, DESIGN.md §3 Q24-Q27): te_load_weights still TAKES the bf16 blob and
                                   quantises the four matrices of every layer to E4M3 with one E8M0 scale per 32
                                   in_features; the GEMMs' A operands (x*g, attention output, SwiGLU output) are
                                   quantised the same way in the producing epilogues; attention, accumulation and the
                                   residual stream are unchanged.  Needs Hq/Hkv a power of two <= 8 and no prefix.
                                   2: as 1, but the four weight matrices are OCP MXFP4 (FP4 E2M1 elements, one E8M0 scale per
                                   32 in_features; DESIGN.md §3 Q32): half the weight bytes again, the A operands stay MXFP8
                                   (the tensor core multiplies E4M3 by E2M1 directly)                                      */
  int32_t non_causal;           /* 0 (default): causal attention by sequence index within the frame.  1: every query sees
                                   every key of its own frame (the vision tower's blocks, te_vision_create; DESIGN.md §3
                                   Q29); needs max_prefix_tokens == 0                                                  */
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
 *   out           DEVICE fp32 [total_tokens, hidden]; last-layer hidden states.  Must not alias embeds.
 *   cuda_stream   a cudaStream_t (NULL = legacy default stream)
 * Position ids (t,h,w), packing offsets and the rotary table are computed on the device from
 * text_lens; the call enqueues work and returns: NO stream synchronisation, NO device->host
 * copy, no allocation once the call's shape class has been seen (te_graph_captures) — the property the
 * paper's TE lacks.  The whole stack is one CUDA-graph launch behind a one-thread kernel
 * that refreshes the per-call pointers; `out` is written only by the last kernel of the stack (the fp32
 * residual stream itself lives in library memory).
 * Conditions only knowable on the device (sum of lengths != total_tokens, text_len < 0,
 * S_b > max_tokens_per_frame) raise a sticky device flag; the kernels then touch no row
 * >= total_tokens; read the flag with te_query_async_error. */
int te_encode(te_handle* h, int32_t n_frames, int32_t grid_h, int32_t grid_w,
              const float* embeds, const int32_t* text_lens, int32_t total_tokens, float* out,
              void* cuda_stream);

/* te_encode with one grid PER FRAME and / or bf16 embeddings ("bf16-embedding input, per-frame
 * grids"; readings Q14, Q19 of SURVEY §8c generalised).
 *   grids         DEVICE int32 [n_frames][2] = (grid_h, grid_w) of every frame, or NULL (then grid_h, grid_w as in
 *                 te_encode).  Frame b holds grid_h[b]*grid_w[b] visual tokens (row-major on ITS grid, t = 0) followed by
 *                 text_lens[b] text tokens whose ids start at max(grid_h[b], grid_w[b]); a negative entry or
 *                 S_b > max_tokens_per_frame raises the device validation flag (te_query_async_error).  Not
 *                 available together with a cached prefix (TE_ERR_UNSUPPORTED).
 *   embeds_dtype  0: DEVICE fp32 [T, hidden] (as te_encode); 1: DEVICE bf16 [T, hidden] — widened exactly to the fp32
 *                 residual stream by the first kernel, so the result equals te_encode on the same values
 * Everything else as te_encode (asynchronous, one graph per shape class). */
int te_encode_ex(te_handle* h, int32_t n_frames, const int32_t* grids, int32_t grid_h, int32_t grid_w,
                 const void* embeds, int32_t embeds_dtype, const int32_t* text_lens, int32_t total_tokens,
                 float* out, void* cuda_stream);

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

/* Options (te_set_option).  Tuning and test switches live in te_debug.h. */
enum {
  TE_OPT_USE_GRAPH = 0,    /* 1 (default): te_encode = one cudaGraphLaunch; 0: direct launches   */
  TE_OPT_KERNEL_TIMING = 1,/* 1: direct launches bracketed by CUDA events per kernel (implies no
                              graph); read with te_kernel_times.  Measurement aid, default 0.     */
  TE_OPT_PDL = 4,          /* 1 (default): kernels are chained with programmatic dependent launch   */
  TE_OPT_L2_RESIDUAL = 10, /* 1 (default): the library's fp32 residual stream is an L2-persisting access-policy window
                              of every kernel, so that the residual GEMMs' read-add-write passes stay out of DRAM.
                              The first te_encode raises the DEVICE-WIDE limit cudaLimitPersistingL2CacheSize to
                              min(max_tokens * hidden * 4, 64 MiB, device maximum) if it is lower; te_destroy and
                              setting this option to 0 reset the persisting lines and restore the previous limit.
                              0: no window                                                                        */
  TE_OPT_SM_BUDGET = 14    /* n in [16, SMs of the device]: size every GEMM grid and every dispatch decision (tile
                              shapes, split-K groups, one-wave wide tiles) for n SMs instead of all of them, so that a
                              caller who runs a denoiser next to the encoder (the paper's side-stream pipeline,
                              PAPER.md:114, Algorithm 1 :118-137) can leave the other SMs to it: the stack's kernels hold
                              one CTA per SM with most of its shared memory, so without a budget nothing else fits
                              beside them.  The budget bounds how many SMs the GEMMs occupy, it does not pin which;
                              attention keeps one CTA per (frame, kv head) and the tiny prep kernel one block per
                              token.  Results under a budget are correct to the same gates but not bitwise equal to
                              the full-GPU run (other K splits, other summation order).  0 (default): all SMs         */
};
int te_set_option(te_handle* h, int option, int value);

/* Number of kernels the library has launched so far on behalf of te_encode / te_encode_prefix (graph replays
 * count the kernel nodes they contain, plus the one parameter-refresh kernel ahead of them).  For bench.py's
 * `gpu_launches`. */
int64_t te_kernel_launches(te_handle* h);

/* Number of CUDA-graph captures (capture + instantiate) te_encode has performed on this handle.  A graph is keyed
 * on the SHAPE CLASS of a call — (n_frames, grid, row-block bucket of total_tokens, prefix length, layer range) —
 * not on the caller's pointers or the exact token count (those travel through a device-side parameter block that
 * a one-thread kernel refreshes ahead of the graph): a stream of ragged batches, or a caller whose allocator
 * hands back different buffers, replays cached graphs (PAPER.md:356 — prompt length varies
 * per call).  Bucket: total_tokens rounded up to 128 rows, to 256 rows from 1024 on; 32 graphs are kept (LRU). */
int64_t te_graph_captures(te_handle* h);

/* Which kernels the last te_encode ran, per class, in the names a profiler prints, e.g.
 * "qkv=te_gemm2_kernel<256, 1, 128>;attn=te_attn_tc_kernel<128>;oproj=te_gemm_wide_kernel<2> (6 tiles x 352 cols);..."
 * (template arguments: tile width, epilogue id, head_dim).  HOST buffer; truncated to n_bytes.  For bench.py's
 * roofline label. */
int te_dispatch_info(te_handle* h, char* buf_host, size_t n_bytes);

/* Per-kernel-class device time accumulated by calls made under TE_OPT_KERNEL_TIMING, measured with
 * CUDA events on the launching stream.  Synchronises; fills ms_sum[TE_KCLASS_COUNT] and
 * n_launches[TE_KCLASS_COUNT] (HOST arrays) and resets the accumulation. */
enum {
  TE_KCLASS_SCAN = 0, TE_KCLASS_PREP = 1, TE_KCLASS_QKV = 2, TE_KCLASS_ATTN = 3, TE_KCLASS_OPROJ = 4,
  TE_KCLASS_GATEUP = 5, TE_KCLASS_DOWN = 6, TE_KCLASS_FINAL_NORM = 7, TE_KCLASS_COUNT = 8
};
int te_kernel_times(te_handle* h, float* ms_sum, int32_t* n_launches);

/* ---- Vision-tower front end.  The paper's TE takes the frame itself: the template's
 * image-pad token is "processed by Qwen3-VL's vision tower" and a 256x256 source patch becomes ~64
 * visual tokens.  The paper fixes no shape or equation of the tower; the front end built here is
 * DESIGN.md §3 readings Q28-Q31 (oracle: oracle/te_vision.py):
 *   patch embedding   pixels cut into P x P patches (row-major patch grid, (dy, dx, channel) inside a patch),
 *                     x0 = patches * W_pe^T, W_pe [d_v, P*P*3], no bias
 *   tower             `tower.n_layers` blocks of the decoder's pre-norm block (te_config `tower`: hidden = d_v) with
 *                     NON-causal attention and rotary ids (0, py, px) on the patch grid, then the final RMSNorm
 *   merger            each 2 x 2 block of neighbouring patches concatenated ((dy, dx) row-major, 4*d_v values) and
 *                     multiplied by W_m [out_hidden, 4*d_v]; merged tokens row-major on the (gh/2) x (gw/2) grid
 * Every step runs on the device in the stack's kernels (tcgen05 GEMMs, the tower = te_encode with non_causal = 1). */
typedef struct te_vision te_vision; /* opaque; owned by the library */
typedef struct te_vision_config {
  te_config tower;      /* the tower's blocks: hidden = d_v, heads, ffn, rope sections, n_layers, rms_eps, rope_theta;
                           final_norm / non_causal / capacities are set by the library                            */
  int32_t patch;        /* P: pixels per patch side; P*P*3 must be a multiple of 64                               */
  int32_t image_h, image_w; /* pixels; multiples of 2*P; (image_h/P) * (image_w/P) <= 256 patches per frame        */
  int32_t out_hidden;   /* the decoder's hidden size (merger output width); multiple of 128                        */
  int32_t max_frames;   /* capacity: frames per call                                                               */
} te_vision_config;

/* Exact size in bytes of the vision blob: W_pe [d_v, P*P*3] | the tower's blob (te_load_weights layout of
 * `tower`, including gf) | W_m [out_hidden, 4*d_v], all bf16 row-major [out_features, in_features].  0 on a bad config. */
size_t te_vision_blob_bytes(const te_vision_config* cfg);
int te_vision_create(const te_vision_config* cfg, int device, te_vision** out);
/* bf16_blob: HOST or DEVICE; n_bytes must equal te_vision_blob_bytes(cfg).  Synchronous; the blob may be freed. */
int te_vision_load_weights(te_vision* v, const void* bf16_blob, size_t n_bytes);
/* Encode the frames' images into the decoder's visual-token embeddings, IN PLACE in the decoder's input:
 *   pixels     DEVICE fp32 [n_frames, image_h, image_w, 3]
 *   text_lens  DEVICE int32 [n_frames] (the decoder call's text_lens) or NULL (= all zero)
 *   embeds     DEVICE fp32 [total_tokens, out_hidden], the packed input of te_encode: the n_vis = (image_h/2P)*(image_w/2P)
 *              merged tokens of frame b are written to rows cu[b] .. cu[b] + n_vis, cu[b] = b*n_vis + sum of
 *              text_lens[0..b) — computed on the device; the text rows are not touched
 *   total_tokens  HOST value: the number of rows of `embeds` (the same value the following te_encode call gets);
 *              >= n_frames * n_vis, else TE_ERR_INVALID_ARG
 * Containment: text_lens is read on the device, unvalidated.  No row at or past total_tokens is ever written, whatever
 * text_lens holds; a negative length (counted as 0) or lengths whose packed sum differs from total_tokens raise the
 * sticky device flag that te_vision_query_async_error reports (bits as in te_query_async_error).
 * Enqueues on cuda_stream and returns (no synchronisation, no device->host copy). */
int te_encode_image(te_vision* v, int32_t n_frames, const float* pixels, const int32_t* text_lens, float* embeds,
                    int32_t total_tokens, void* cuda_stream);
/* Synchronises the device; TE_ERR_DEVICE_CHECK (and clears the flag) if te_encode_image — or the tower's own
 * validation — raised the device-side flag since the last query, TE_ERR_CUDA on a CUDA error, else TE_OK. */
int te_vision_query_async_error(te_vision* v);
/* Kernels launched so far on behalf of te_encode_image (the tower's graph nodes included). */
int64_t te_vision_kernel_launches(te_vision* v);
const char* te_vision_last_error(te_vision* v);
void te_vision_destroy(te_vision* v);

/* ---------------------------------------------------------------------------------------------------------------
 * A matrix product for callers that must not allocate device memory.
 *
 * Who this is for.  Two kinds of caller cannot afford cudaMalloc / cudaFree around a kernel.  (1) A frame loop that
 * shares the GPU with a denoiser on another stream (the paper's side-stream / main-stream pipeline, PAPER.md:114,
 * Algorithm 1 :118-137): both calls may block the host until the whole device is idle, which stalls the other stream
 * and shows up as a dropped frame.  (2) A process in which some other component — an inference server's memory pool,
 * a framework's caching allocator — has claimed all of HBM at start-up: cudaMalloc then fails with out-of-memory
 * although the pool's owner could hand out a buffer.  Every other entry point of this library allocates (te_create
 * builds the workspace, the stand-alone products of te_debug.h allocate and free their scratch on every call).
 *
 * What it computes.  C[m, n] (DEVICE fp32, row-major) = A[m, k] * B[n, k]^T, A and B DEVICE bf16 row-major, fp32
 * accumulation — the same small-batch split-K kernel the stack runs for T <= 512: `splits` CTAs share
 * one 128 x block_n output tile, each multiplies its own slice of k, and the partial tiles meet in scratch memory and
 * are summed in a fixed order, so the result is bitwise repeatable.  The caller owns a, b and c and still passes
 * them; the only memory the call does not get from the caller is that scratch.
 *
 * Where the scratch lives.  In a fixed array inside the library's device image, TE_NOALLOC_SCRATCH_BYTES of partial
 * tiles plus 2 KiB of group counters.  Every GPU that loads libte_b200.so carries this array from module load until
 * the process exits, whether or not this function is ever called.  The call runs no cudaMalloc, cudaFree,
 * cudaMallocAsync or other allocating routine; it enqueues one 2 KiB memset of the counters and one kernel on
 * `cuda_stream` and returns without synchronising.
 *
 * Limits.  k % 64 == 0; block_n in {128, 256}; n % block_n == 0; 1 <= splits <= 8 and splits <= k / 64;
 * tiles = ceil(m / 128) * (n / block_n) must satisfy tiles * splits <= number of SMs (the CTAs of a group wait for each
 * other, so all must be resident; TE_ERR_UNSUPPORTED otherwise) and
 *     tiles * splits * 128 * block_n * 4 bytes <= TE_NOALLOC_SCRATCH_BYTES,
 * else the call launches nothing and returns TE_ERR_TOO_LARGE.  (128 partial tiles of 128 x 128, e.g. m <= 128,
 * n = 2048, splits = 8, fill it exactly.)
 *
 * First call on a device.  It looks up the array's device address and opts the kernels into their shared-memory size;
 * this set-up happens once per device, inside the first call made for that device, and is not something to do in the
 * middle of a stream capture — make one call per device at start-up, outside any capture.
 *
 * Sharing.  There is ONE array per GPU and every call uses it from offset 0, and it keeps whatever the previous call
 * left there.  The partial tiles are fully overwritten before they are read and the counters are cleared on the
 * stream before each kernel, so successive calls on one stream are independent of each other.  Two calls whose kernels
 * can run at the same time on one GPU (different streams, different host threads, different handles of any kind) race
 * on the array and produce garbage or hang: the caller must order them (same stream, or an event between them). */
#define TE_NOALLOC_SCRATCH_BYTES (8u << 20)
int te_matmul_noalloc(int device, const void* a_bf16, const void* b_bf16, float* c, int32_t m, int32_t n, int32_t k,
                      int32_t block_n, int32_t splits, void* cuda_stream);

void te_destroy(te_handle* h);
const char* te_strerror(int code);
const char* te_last_error(te_handle* h); /* valid until the next call on h */

#ifdef __cplusplus
}
#endif
#endif /* TE_B200_H_ */
