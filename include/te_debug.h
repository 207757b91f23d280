/*
 * te_debug.h — test-only taps, stand-alone GEMM entry points and tuning switches of libte_b200.so
 * (SURVEY.md §8b "Debug taps").  Not part of the product boundary (include/te.h); the parity tests and
 * bench.py's experiment flags use them.  Same conventions as te.h (plain C, HOST/DEVICE stated, te_status).
 */
#ifndef TE_B200_DEBUG_H_
#define TE_B200_DEBUG_H_

#include "te.h"

#ifdef __cplusplus
extern "C" {
#endif

/* Tuning / test options for te_set_option (defaults are what bench.py measures). */
enum {
  TE_OPT_CTA_PAIR = 2,     /* GEMM tiling: 0 = one CTA per 128-row tile, 1 = CTA pairs (cta_group::2,
                              256-row tiles), 2 = auto by token count (default)                    */
  TE_OPT_RESID_BLOCK_N = 3,/* tile width (128 default, or 256) of the O-proj / down GEMMs          */
  TE_OPT_TRACE = 5,        /* 1: CTA-pair GEMM kernels stamp %globaltimer at pipeline events (debug
                              aid; read with te_debug_tap(TE_TAP_TRACE)); default 0                 */
  TE_OPT_ATTN_IMPL = 6,    /* attention kernel: 1 (default) = tcgen05 kernel (S, P, O in tensor memory)
                              when Hq/Hkv is a power of two <= 8, 0 = mma.sync flash kernel          */
  TE_OPT_SPLIT_K = 7,      /* 1 (default): small batches (fewer 128-row tiles than SMs in a GEMM, no
                              CTA pairs) run the split-K kernel: several CTAs per output tile, each
                              streaming its own K-slice of the weights; partial tiles are summed in a
                              fixed order (deterministic).  0: one CTA per tile; n > 1: target CTA count */
  TE_OPT_RESID_WIDE = 9    /* O-proj / down on CTA pairs: 1 (default) = when their 128-wide tiles would need two or
                              more waves, ONE wave of wide tiles (width = hidden / n rounded up to 32, <= 512
                              columns, two MMAs per k-step; te_gemm_wide.cuh); 0 = never; n in 2..16 = always,
                              with n tiles across the hidden dimension (tests)                                  */
};

/* te_debug_set_range restricts subsequent te_encode calls to layers [layer_begin, layer_end)
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
  TE_TAP_TRACE = 7,      /* u64   [5 classes (qkv,oproj,gateup,down,attn)][n_SMs][96] ns stamps / SM clocks
                            of the last launch of each class (TE_OPT_TRACE)     */
  /* weight_dtype = 1 (MXFP8): the quantised A operands; scales in the tiled order of te_debug_mx_quantise */
  TE_TAP_ATTN8 = 8,      /* u8 E4M3 [T, Hq*dh]                                  */
  TE_TAP_ACT8 = 9,       /* u8 E4M3 [T, F]                                      */
  TE_TAP_SF_ATTN = 10,   /* u8 E8M0 [ceil(T/128), Hq*dh/128, 512]               */
  TE_TAP_SF_ACT = 11     /* u8 E8M0 [ceil(T/128), F/128, 512]                   */
};
int te_debug_set_range(te_handle* h, int32_t layer_begin, int32_t layer_end,
                       int32_t stop_after_attn);
int te_debug_tap(te_handle* h, int what, void* dst_host, size_t n_bytes);

/* C[M,N] (DEVICE fp32, row-major) = A[M,K] * B[N,K]^T with A, B DEVICE bf16 row-major, through the
 * same TMA + tcgen05 main loop as the stack's GEMMs (plain epilogue).  K % 64 == 0, N % block_n == 0,
 * block_n in {128, 256}; cta_pair = 1 selects the cta_group::2 kernel (256-row tiles).  Synchronous. */
int te_debug_gemm(int device, const void* a_bf16, const void* b_bf16, float* c, int32_t m,
                  int32_t n, int32_t k, int32_t block_n, int32_t cta_pair);

/* The same product through the split-K kernel (te_gemm_splitk.cuh): `splits` CTAs (1..8, <= k/64) per
 * 128 x block_n tile, fixed-order reduction of the fp32 partial tiles.  Needs tiles * splits <= number
 * of SMs (TE_ERR_UNSUPPORTED otherwise).  Synchronous. */
int te_debug_gemm_splitk(int device, const void* a_bf16, const void* b_bf16, float* c, int32_t m,
                         int32_t n, int32_t k, int32_t block_n, int32_t splits);

/* The same product through the one-wave wide-tile kernel (te_gemm_wide.cuh): n_tiles CTA-pair tiles across N,
 * each 256 rows x (N / n_tiles rounded up to 32) columns, two MMAs per k-step; the last tile may be partly or
 * wholly out of range.  N % 32 == 0, width <= 512, ceil(M/256) * n_tiles <= SM pairs.  Synchronous. */
int te_debug_gemm_wide(int device, const void* a_bf16, const void* b_bf16, float* c, int32_t m,
                       int32_t n, int32_t k, int32_t n_tiles);

/* MXFP8 quantiser alone (te_config.weight_dtype = 1; DESIGN.md §3 Q24-Q25): src DEVICE bf16 [rows, k] ->
 * codes DEVICE uint8 [rows, k] (E4M3) and scales_tiled DEVICE uint8 [rows/128 (rounded up), k/128, 512] (E8M0): the
 * scale of (row r, 32-element block b) is byte  ((r/128) * (k/128) + b/4) * 512 + (r%32)*16 + ((r/32)%4)*4 + b%4
 * (the order the tensor core's scale copy takes).  k % 128 == 0.  Synchronous. */
int te_debug_mx_quantise(int device, const void* src_bf16, int32_t rows, int32_t k, void* codes, void* scales_tiled);

/* C = Q(A) * Q(B)^T through the block-scaled tcgen05 kernel (te_gemm8.cuh, plain epilogue): A, B DEVICE bf16 are
 * quantised to MXFP8 on the device first.  k % 128 == 0, n % block_n == 0, block_n in {128, 256}.  Synchronous. */
int te_debug_gemm_mxfp8(int device, const void* a_bf16, const void* b_bf16, float* c, int32_t m, int32_t n,
                        int32_t k, int32_t block_n);

/* MXFP4 weights (te_config.weight_dtype = 2; DESIGN.md §3 Q32).  te_debug_mx_quantise_fp4: src DEVICE bf16 [rows, k] ->
 * codes_packed DEVICE uint8 [rows, k/2] (E2M1, element 2i in the low nibble of byte i) and scales_tiled as in
 * te_debug_mx_quantise.  te_debug_gemm_mxfp4: C = Q8(A) * Q4(B)^T — A quantised to MXFP8, B to MXFP4 on the device,
 * multiplied by the block-scaled tcgen05 kernel (kind::mxf8f6f4, E4M3 x E2M1).  Same constraints as te_debug_gemm_mxfp8. */
int te_debug_mx_quantise_fp4(int device, const void* src_bf16, int32_t rows, int32_t k, void* codes_packed, void* scales_tiled);
int te_debug_gemm_mxfp4(int device, const void* a_bf16, const void* b_bf16, float* c, int32_t m, int32_t n,
                        int32_t k, int32_t block_n);

/* Vision front end taps (te_encode_image): synchronises and copies to `dst` (HOST). */
enum {
  TE_VTAP_PATCH_EMBEDS = 0, /* fp32 [n_frames*gh*gw, d_v]   x0 = patches * W_pe^T                  */
  TE_VTAP_TOWER_OUT = 1,    /* fp32 [n_frames*gh*gw, d_v]   tower output after the final RMSNorm   */
  TE_VTAP_MERGED = 2        /* fp32 [n_frames*n_vis, out_hidden]  merger output before the scatter */
};
int te_vision_debug_tap(te_vision* v, int what, void* dst_host, size_t n_bytes);
/* The tower's te_handle (owned by `v`), for te_set_option / te_debug_tap on the tower itself. */
te_handle* te_vision_debug_tower(te_vision* v);

#ifdef __cplusplus
}
#endif
#endif /* TE_B200_DEBUG_H_ */
