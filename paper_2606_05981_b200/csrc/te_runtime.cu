// te_runtime.cu — host runtime + C ABI (include/te.h, include/te_debug.h): handle, weight repack, workspace,
// tensor maps, kernel dispatch (Plan), kernel sequencing and the CUDA-graph cache.  One graph launch per te_encode.
#include <cuda.h>
#include <cuda_bf16.h>
#include <cuda_runtime.h>

#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <mutex>
#include <string>
#include <vector>

#include "../../include/te.h"
#include "../../include/te_debug.h"
#include "te_attn.cuh"
#include "te_attn_tc.cuh"
#include "te_gemm.cuh"
#include "te_gemm8.cuh"
#include "te_gemm_splitk.cuh"
#include "te_gemm_wide.cuh"
#include "te_prep.cuh"
#include "te_vision.cuh"

namespace {

using bf16 = __nv_bfloat16;

typedef CUresult (*PFN_encodeTiled)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*,
                                    const cuuint64_t*, const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave,
                                    CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

PFN_encodeTiled get_encode_fn() {
  static PFN_encodeTiled fn = nullptr;
  if (!fn) {
    void* p = nullptr;
    cudaDriverEntryPointQueryResult q;
    if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &q) == cudaSuccess &&
        q == cudaDriverEntryPointSuccess)
      fn = reinterpret_cast<PFN_encodeTiled>(p);
  }
  return fn;
}

// 2-D bf16 row-major [rows, cols] tensor, box = [box_rows, 64 cols], 128-byte swizzle.
bool make_tmap(CUtensorMap* m, const void* base, uint64_t rows, uint64_t cols, uint32_t box_rows) {
  PFN_encodeTiled fn = get_encode_fn();
  if (!fn) return false;
  cuuint64_t dims[2] = {cols, rows};
  cuuint64_t strides[1] = {cols * sizeof(bf16)};
  cuuint32_t box[2] = {64, box_rows};
  cuuint32_t estr[2] = {1, 1};
  return fn(m, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 2, const_cast<void*>(base), dims, strides, box, estr,
            CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
            CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
}

// 2-D E4M3 row-major [rows, cols] tensor (MXFP8 operands), box = [box_rows, 128 cols = 128 B], 128-byte swizzle.
bool make_tmap_u8(CUtensorMap* m, const void* base, uint64_t rows, uint64_t cols, uint32_t box_rows) {
  PFN_encodeTiled fn = get_encode_fn();
  if (!fn) return false;
  cuuint64_t dims[2] = {cols, rows};
  cuuint64_t strides[1] = {cols};
  cuuint32_t box[2] = {128, box_rows};
  cuuint32_t estr[2] = {1, 1};
  return fn(m, CU_TENSOR_MAP_DATA_TYPE_UINT8, 2, const_cast<void*>(base), dims, strides, box, estr,
            CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
            CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
}

// 2-D FP4 (E2M1, two per byte) row-major [rows, cols] weight tensor (MXFP4, te_config.weight_dtype = 2): box = [box_rows,
// 128 elements]; the 16U4_ALIGN16B type unpacks every 16 nibbles into a 16-byte chunk of shared memory (8 bytes of data +
// 8 bytes of gap), so a box row is 128 B there, the same geometry as an E4M3 row, with the 128-byte swizzle.
bool make_tmap_u4(CUtensorMap* m, const void* base, uint64_t rows, uint64_t cols, uint32_t box_rows) {
  PFN_encodeTiled fn = get_encode_fn();
  if (!fn) return false;
  cuuint64_t dims[2] = {cols, rows};
  cuuint64_t strides[1] = {cols / 2};
  cuuint32_t box[2] = {128, box_rows};
  cuuint32_t estr[2] = {1, 1};
  return fn(m, CU_TENSOR_MAP_DATA_TYPE_16U4_ALIGN16B, 2, const_cast<void*>(base), dims, strides, box, estr,
            CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
            CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
}

// Tiled MXFP8 block scales as a [tiles, 128] uint32 tensor: one 512-byte scale tile per row, box = one tile.
bool make_tmap_sf(CUtensorMap* m, const void* base, uint64_t n_tiles) {
  PFN_encodeTiled fn = get_encode_fn();
  if (!fn) return false;
  cuuint64_t dims[2] = {128, n_tiles};
  cuuint64_t strides[1] = {512};
  cuuint32_t box[2] = {128, 1};
  cuuint32_t estr[2] = {1, 1};
  return fn(m, CU_TENSOR_MAP_DATA_TYPE_UINT32, 2, const_cast<void*>(base), dims, strides, box, estr,
            CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
            CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
}

struct LayerOff {
  size_t g1, wqkv, gq, gk, wo, g2, wgu, wd;  // element offsets into the device weight buffer
  // MXFP8 copy (te_config.weight_dtype = 1): byte offsets into w8 (elements) and sfw (tiled block scales)
  size_t q8, o8, gu8, d8, sq8, so8, sgu8, sd8;
};

// A cached graph is valid for every call of the same SHAPE CLASS: per-call pointers and the exact token count
// travel through the device-side DynParams block, so the key holds only what decides grids and dispatch.
struct GraphKey {
  int n_frames, grid_h, grid_w, bucket_tokens, lb, le, stop, prefix_len;
  bool operator==(const GraphKey& o) const { return memcmp(this, &o, sizeof(GraphKey)) == 0; }
};
struct GraphEntry {
  GraphKey key;
  cudaGraphExec_t exec;
  cudaGraph_t graph;
  int n_kernels;
  uint64_t stamp;
};

// Launch attributes of one kernel launch (per call, never process-wide: two handles on two host threads
// must not see each other's choices).
struct LaunchCtx {
  bool pdl = false;                // programmatic stream serialisation (the kernels order themselves with griddepcontrol)
  bool coop = false;               // cooperative grid: all CTAs resident at once (split-K groups spin on each other)
  cudaAccessPolicyWindow l2{};     // TE_OPT_L2_RESIDUAL: the fp32 residual stays resident in L2 (num_bytes = 0: none)
};

// Kernel choice for one shape class (every decision that depends on the token count is taken from the bucket's
// upper bound, so that all calls of a bucket share one graph).
struct Plan {
  int Tb = 0;          // token-count bucket (rows the grids are sized for)
  int num_m = 0;       // 128-row blocks
  int pair = 0;        // CTA pairs for all GEMMs
  int bn_qkv = 256, k_qkv = 0, pair_qkv = 0, bx_qkv = 0;
  int bn_gu = 256, k_gu = 0, pair_gu = 0, bx_gu = 0, gu_half = 0, gu_wide_tiles = 0, gu_wide_w = 0;
  int bn_res = 128, k_res = 0, bx_res = 0, n_blk_res = 0, wide_tiles = 0, wide_bn = 0;
  int parts = 1;       // RMSNorm partial sums per row written by the residual GEMMs
  int attn_tc = 0, attn_split = 1, q_blocks = 1, g_shift = 0, s_bound = 0;
  int mx = 0;          // MXFP8 variant: every GEMM on te_gemm8_kernel (CTA pairs, block-scaled tcgen05)
};

}  // namespace

struct te_handle {
  te_config cfg{};
  int device = 0;
  int sm_count = 0;  // SMs every grid and dispatch decision is sized for: sm_dev, or the caller's budget (TE_OPT_SM_BUDGET)
  int sm_dev = 0;    // SMs of the device
  bool loaded = false;
  // tile choices
  int bn_qkv = 256, bn_gu = 256, bn_res = 128;
  int attn_impl = 1;  // 1: tcgen05 kernel (te_attn_tc.cuh) when Hq/Hkv is a power of two <= 8; 0: mma.sync kernel
  int pair_mode = 2;  // 0: always 1-CTA tiles, 1: always CTA pairs (cta_group::2), 2: auto (by token count)
  int resid_wide = 1; // residual GEMMs on CTA pairs: 1 = auto (one wave of wide tiles when 128-wide tiles need >= 2
                      // waves), 0 = never, n >= 2 = always with n tiles across N (tests)
  int l2_resid = 1;          // 1: the residual stream is an L2-persisting access window of every kernel
  size_t l2_limit_bytes = 0; // persisting-L2 carve-out requested for it (0 until the first te_encode sets the limit)
  bool l2_ref_held = false;  // this handle holds one reference on the device's shared persisting-L2 record (l2_acquire)
  size_t l2_max_persist = 0; // device property persistingL2CacheMaxSize
  size_t l2_max_window = 0;  // device property accessPolicyMaxWindowSize: an access-policy window may not be larger
  int splitk = 1;     // 1: small batches (no CTA pairs) use the split-K kernel when a GEMM has <= one tile per SM
  int split_target = 0;  // experiments: target CTA count of a split-K launch (0 = one per SM)
  float* sk_scratch = nullptr;  // [sm_count][128 x 256] fp32 partial tiles
  int* sk_sem = nullptr;        // [sm_count][2] per-tile arrival / departure counters (zero between launches)
  // weights
  bf16* w = nullptr;
  size_t w_elems = 0;
  std::vector<LayerOff> off;
  size_t gf_off = 0;
  // MXFP8 variant: E4M3 copies of the four matrices of every layer + their tiled E8M0 block scales; E4M3
  // activations (A operands) with their scales; per-layer tensor maps in 64- and 128-row boxes
  uint8_t *w8 = nullptr, *sfw = nullptr;
  uint8_t *xg8 = nullptr, *attn8 = nullptr, *act8 = nullptr, *sf_xg = nullptr, *sf_attn = nullptr, *sf_act = nullptr;
  struct LayerMaps8 { CUtensorMap qkv[2], o[2], gu[2], d[2], sf_qkv, sf_o, sf_gu, sf_d; };
  std::vector<LayerMaps8> tm8;
  CUtensorMap tmA_xg8, tmA_attn8, tmA_act8, tmSF_xg, tmSF_attn, tmSF_act;
  int bn8_qkv = 128;  // MXFP8 QKV tile width (128: two accumulator stages; 256: one)
  int bn8_gu = 192;   // MXFP8 gate/up tile width (192: two accumulator stages, weights re-interleaved per 192 rows; 256: one)
  // weight tensor maps per layer, one per B box height {32, 64, 128, 256} rows (index 0..3)
  struct LayerMaps { CUtensorMap qkv[4], o[4], gu[4], d[4]; };
  std::vector<LayerMaps> tm;
  // workspace (rows: cap_rows = max_tokens rounded up to 256)
  int cap_rows = 0;
  te::DynParams* dyn = nullptr;  // per-call pointers + token count, refreshed on the stream ahead of every stack
  float* resid = nullptr;        // [cap_rows, d] fp32 residual stream
  int32_t *cu = nullptr, *pos = nullptr, *flag = nullptr;
  float *cos_t = nullptr, *sin_t = nullptr, *ssq = nullptr;
  double* inv_freq = nullptr;
  bf16 *xg = nullptr, *qkv = nullptr, *attn = nullptr, *act = nullptr;
  int ssq_parts_cap = 0;
  // activation tensor maps over the whole workspace buffers, encoded once (rows past the call's tokens are never
  // stored; see qkv_zero_rows for the one place where they are multiplied)
  CUtensorMap tmA_xg, tmA_attn, tmA_act, tmQ, tmKV;
  bool attn_tc_ok = false;
  int g_shift = 0;
  unsigned long long* trace = nullptr;  // [4 GEMM classes][sm_count][TRACE_SLOTS] (debug, TE_OPT_TRACE)
  int trace_on = 0;
  // M-RoPE axis of every frequency pair (contiguous or interleaved sections)
  int8_t axis[64] = {};
  // shared text prefix (te_encode_prefix): per-layer keys | values of the P prefix tokens, [L][max_prefix][2*Hkv*dh]
  bf16* kv_prefix = nullptr;
  std::vector<CUtensorMap> tm_prefix;  // per layer: the prefix cache [P, 2*Hkv*dh] in 64-row boxes (tcgen05 attention)
  float2* attn_stats = nullptr;        // [max_tokens, Hq] (row max, row sum) of the frame-local attention pass
  float* attn_o32 = nullptr;           // [max_tokens, Hq*dh] its normalised fp32 output (blended with the prefix pass in fp32)
  float* prefix_buf = nullptr;    // [max_prefix, d] hidden states of the prefix pass when the caller wants no output
  int32_t* prefix_lens = nullptr; // device [1]
  int prefix_len = 0;
  // host-path staging
  struct HostSlot {  // one batch in flight on the host path: device staging + the events that chain its three stages
    float *embeds = nullptr, *out = nullptr;
    int32_t* lens = nullptr;
    cudaEvent_t h2d_done = nullptr, compute_done = nullptr, d2h_done = nullptr;
    bool busy = false;
  } slot[2];
  int next_slot = 0;
  cudaStream_t own_stream = nullptr, h2d_stream = nullptr, d2h_stream = nullptr;
  // graphs
  std::vector<GraphEntry> cache;
  uint64_t stamp = 0;
  long long captures = 0;
  int use_graph = 1;
  int pdl = 1;
  int timing = 0;
  struct TimedLaunch { int kclass; cudaEvent_t a, b; };
  std::vector<TimedLaunch> timed;
  int dbg_lb = 0, dbg_le = 0, dbg_stop = 0;
  int last_T = 0, last_B = 0;
  Plan last_plan;
  long long launches = 0;
  std::string err;
  std::string info;
};

// Vision-tower front end (te_vision_create .. te_encode_image, DESIGN.md §3 Q28-Q31).
struct te_vision {
  te_vision_config cfg{};
  int device = 0;
  int sm_count = 0;
  bool loaded = false;
  te_handle* tower = nullptr;       // the tower's blocks: the decoder stack with non_causal = 1, final_norm = 1
  int gh = 0, gw = 0, n_vis = 0, patch_dim = 0, d_v = 0;
  int rows_pe = 0, rows_m = 0;      // capacity rows of the two GEMM A operands (multiples of 256)
  __nv_bfloat16 *w_pe = nullptr, *w_m = nullptr;  // [d_v, P*P*3], [out_hidden, 4*d_v]
  __nv_bfloat16 *a_pe = nullptr, *a_m = nullptr;  // [rows_pe, P*P*3] patches, [rows_m, 4*d_v] merged tower rows
  float *x0 = nullptr, *tower_out = nullptr, *vis = nullptr;
  int32_t* zero_lens = nullptr;     // [max_frames] the tower's frames carry no text
  CUtensorMap tmA_pe, tmA_m, tmB_pe, tmB_m;
  int bn_pe = 128, pair_pe = 0, bn_m = 128, pair_m = 0;
  int last_B = 0;
  long long launches = 0;
  std::string err;
};

namespace {

#define TE_CUDA(h, expr)                                                                      \
  do {                                                                                        \
    cudaError_t _e = (expr);                                                                  \
    if (_e != cudaSuccess) {                                                                  \
      (h)->err = std::string(#expr) + ": " + cudaGetErrorString(_e);                          \
      return TE_ERR_CUDA;                                                                     \
    }                                                                                         \
  } while (0)

size_t layer_elems(const te_config& c) {
  const size_t d = c.hidden, dh = c.head_dim, F = c.ffn;
  return d + (size_t)(c.n_q_heads + 2 * c.n_kv_heads) * dh * d + 2 * dh + d * (size_t)c.n_q_heads * dh + d +
         2 * F * d + d * F;
}
size_t blob_elems(const te_config& c) { return layer_elems(c) * c.n_layers + c.hidden; }

int validate_config(const te_config& c) {
  if (c.n_layers < 1 || c.hidden < 1 || c.n_q_heads < 1 || c.n_kv_heads < 1 || c.ffn < 1) return TE_ERR_INVALID_ARG;
  if (c.n_q_heads % c.n_kv_heads != 0) return TE_ERR_INVALID_ARG;
  if (c.rope_sec_t < 0 || c.rope_sec_h < 0 || c.rope_sec_w < 0) return TE_ERR_INVALID_ARG;
  if (c.rope_sec_t + c.rope_sec_h + c.rope_sec_w != c.head_dim / 2) return TE_ERR_INVALID_ARG;
  if (c.max_frames < 1 || c.max_tokens < 1 || c.max_tokens_per_frame < 1) return TE_ERR_INVALID_ARG;
  if (c.rope_interleaved < 0 || c.rope_interleaved > 1) return TE_ERR_INVALID_ARG;
  if (c.max_prefix_tokens < 0 || c.max_prefix_tokens > c.max_tokens ||
      c.max_prefix_tokens > c.max_tokens_per_frame)
    return TE_ERR_INVALID_ARG;
  if (!(c.rms_eps > 0.f) || !(c.rope_theta > 0.0)) return TE_ERR_INVALID_ARG;
  if (c.head_dim != 64 && c.head_dim != 128) return TE_ERR_UNSUPPORTED;
  if (c.hidden % 128 != 0 || c.ffn % 128 != 0) return TE_ERR_UNSUPPORTED;
  if (((c.n_q_heads + 2 * c.n_kv_heads) * c.head_dim) % 128 != 0) return TE_ERR_UNSUPPORTED;
  if ((c.n_q_heads * c.head_dim) % 64 != 0) return TE_ERR_UNSUPPORTED;
  if (c.max_tokens_per_frame > 256) return TE_ERR_UNSUPPORTED;
  if (c.weight_dtype < 0 || c.weight_dtype > 2) return TE_ERR_INVALID_ARG;
  if (c.non_causal < 0 || c.non_causal > 1 || (c.non_causal && c.max_prefix_tokens > 0)) return TE_ERR_INVALID_ARG;
  if (c.weight_dtype >= 1) {
    // MXFP8 / MXFP4 weights: 128-element K chunks everywhere; the quantising attention epilogue exists in the tcgen05 kernel only
    // (G = Hq/Hkv a power of two <= 8); no cached prefix (its merge pass re-reads a bf16 output)
    const int G = c.n_q_heads / c.n_kv_heads;
    if ((c.n_q_heads * c.head_dim) % 128 != 0 || (G & (G - 1)) != 0 || G > 8 || c.max_prefix_tokens > 0)
      return TE_ERR_UNSUPPORTED;
  }
  return TE_OK;
}

// Launch with (optional) programmatic stream serialisation: the kernel may begin while its
// predecessor in the stream drains; the kernels order themselves with griddepcontrol.wait.
template <typename... KArgs, typename... Args>
cudaError_t launch_k(const LaunchCtx& lc, void (*kernel)(KArgs...), dim3 grid, dim3 block, size_t smem, cudaStream_t st,
                     Args&&... args) {
  cudaLaunchConfig_t cfg{};
  cfg.gridDim = grid;
  cfg.blockDim = block;
  cfg.dynamicSmemBytes = smem;
  cfg.stream = st;
  cudaLaunchAttribute at[3];
  int n = 0;
  if (lc.coop) {
    at[n].id = cudaLaunchAttributeCooperative;
    at[n].val.cooperative = 1;
    ++n;
  }
  if (lc.pdl) {
    at[n].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    at[n].val.programmaticStreamSerializationAllowed = 1;
    ++n;
  }
  if (lc.l2.num_bytes) {
    at[n].id = cudaLaunchAttributeAccessPolicyWindow;
    at[n].val.accessPolicyWindow = lc.l2;
    ++n;
  }
  cfg.attrs = at;
  cfg.numAttrs = n;
  return cudaLaunchKernelEx(&cfg, kernel, static_cast<KArgs>(args)...);
}

inline int box_index(int rows) { return rows == 32 ? 0 : (rows == 64 ? 1 : (rows == 128 ? 2 : 3)); }

template <int BN, int EPI, int DH>
cudaError_t launch_gemm(const LaunchCtx& lc, const CUtensorMap& tmA, const CUtensorMap& tmB, const te::GemmParams& p,
                        int sm_count, cudaStream_t st) {
  using Cfg = te::GemmCfg<BN>;
  const int tiles = p.num_m_blk * p.num_n_blk;
  const int grid = tiles < sm_count ? tiles : sm_count;
  return launch_k(lc, te::te_gemm_kernel<BN, EPI, DH>, dim3(grid), dim3(te::GEMM_THREADS), Cfg::SMEM_BYTES, st, tmA, tmB, p);
}

template <int BN, int EPI, int DH>
cudaError_t launch_gemm2(const LaunchCtx& lc, const CUtensorMap& tmA, const CUtensorMap& tmB, const te::GemmParams& p,
                         int sm_count, cudaStream_t st) {
  using Cfg = te::Gemm2Cfg<BN, EPI>;
  const int tiles = ((p.num_m_blk + 1) / 2) * p.num_n_blk;
  const int pairs = tiles < sm_count / 2 ? tiles : sm_count / 2;
  return launch_k(lc, te::te_gemm2_kernel<BN, EPI, DH>, dim3(2 * pairs), dim3(te::GEMM2_THREADS), Cfg::SMEM_BYTES, st, tmA,
                  tmB, p);
}

// pair = 0: one CTA per 128 x bn tile; pair = 1: one CTA pair per 256 x bn tile (cta_group::2)
template <int EPI>
cudaError_t launch_gemm_bn(const LaunchCtx& lc, int bn, int pair, int dh, const CUtensorMap& a, const CUtensorMap& b,
                           const te::GemmParams& p, int sms, cudaStream_t st) {
  if constexpr (EPI == te::EPI_QKV) {
    if (pair) {
      if (bn == 256 && dh == 128) return launch_gemm2<256, EPI, 128>(lc, a, b, p, sms, st);
      if (bn == 256 && dh == 64) return launch_gemm2<256, EPI, 64>(lc, a, b, p, sms, st);
      if (bn == 128 && dh == 128) return launch_gemm2<128, EPI, 128>(lc, a, b, p, sms, st);
      return launch_gemm2<128, EPI, 64>(lc, a, b, p, sms, st);
    }
    if (bn == 256 && dh == 128) return launch_gemm<256, EPI, 128>(lc, a, b, p, sms, st);
    if (bn == 256 && dh == 64) return launch_gemm<256, EPI, 64>(lc, a, b, p, sms, st);
    if (bn == 128 && dh == 128) return launch_gemm<128, EPI, 128>(lc, a, b, p, sms, st);
    return launch_gemm<128, EPI, 64>(lc, a, b, p, sms, st);
  } else {
    if (pair) {
      if (bn == 256) return launch_gemm2<256, EPI, 128>(lc, a, b, p, sms, st);
      return launch_gemm2<128, EPI, 128>(lc, a, b, p, sms, st);
    }
    if (bn == 256) return launch_gemm<256, EPI, 128>(lc, a, b, p, sms, st);
    return launch_gemm<128, EPI, 128>(lc, a, b, p, sms, st);
  }
}

// MXFP8 kernel: one CTA pair per 256 x BN tile, persistent (te_gemm8.cuh)
template <int BN, int EPI, int DH>
cudaError_t launch_gemm8(const LaunchCtx& lc, const CUtensorMap& tmA, const CUtensorMap& tmB, const CUtensorMap& tmSFA,
                         const CUtensorMap& tmSFB, const te::GemmParams& p, const te::Gemm8Extra& x8, int sm_count,
                         cudaStream_t st) {
  using Cfg = te::Gemm8Cfg<BN, EPI>;
  const int tiles = ((p.num_m_blk + 1) / 2) * p.num_n_blk;
  const int pairs = tiles < sm_count / 2 ? tiles : sm_count / 2;
  return launch_k(lc, te::te_gemm8_kernel<BN, EPI, DH>, dim3(2 * pairs), dim3(Cfg::THREADS), Cfg::SMEM_BYTES, st, tmA,
                  tmB, tmSFA, tmSFB, p, x8);
}
template <int BN, int EPI, int DH>
cudaError_t set_gemm8_attr() {
  return cudaFuncSetAttribute(te::te_gemm8_kernel<BN, EPI, DH>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                              te::Gemm8Cfg<BN, EPI>::SMEM_BYTES);
}

// split-K kernel: `p.splits` CTAs per 128 x bn tile (small batches; te_gemm_splitk.cuh)
template <int BN, int EPI, int DH, int VAR>
cudaError_t launch_gemmk_var(LaunchCtx lc, const CUtensorMap& tmA, const CUtensorMap& tmB, const te::GemmParams& p,
                             cudaStream_t st) {
  using Cfg = te::GemmKCfg<BN, EPI>;
  const int tiles = p.num_m_blk * p.num_n_blk;
  lc.coop = p.splits > 1;  // the groups spin on each other: all CTAs resident at once, or the launch waits
  return launch_k(lc, te::te_gemmk_kernel<BN, EPI, DH, VAR>, dim3(tiles * p.splits), dim3(te::GEMMK_THREADS), Cfg::SMEM_BYTES,
                  st, tmA, tmB, p);
}
// split-K kernel: `p.splits` CTAs per 128 x bn tile (small batches; te_gemm_splitk.cuh); one instantiation per epilogue
// variant (te::gemmk_variant)
template <int BN, int EPI, int DH>
cudaError_t launch_gemmk(const LaunchCtx& lc, const CUtensorMap& tmA, const CUtensorMap& tmB, const te::GemmParams& p,
                         cudaStream_t st) {
  switch (p.splits == 1 ? 0 : te::gemmk_variant(EPI, p.splits * (BN / 128))) {
    case 0: return launch_gemmk_var<BN, EPI, DH, 0>(lc, tmA, tmB, p, st);
    // variants 1 and 2 (two / three partial tiles per row batch) exist for the residual, SwiGLU and plain epilogues only:
    // gemmk_variant never selects them for EPI_QKV, so they are not instantiated for it
    case 1:
      if constexpr (EPI != te::EPI_QKV) return launch_gemmk_var<BN, EPI, DH, 1>(lc, tmA, tmB, p, st);
      else return cudaErrorInvalidValue;
    case 2:
      if constexpr (EPI != te::EPI_QKV) return launch_gemmk_var<BN, EPI, DH, 2>(lc, tmA, tmB, p, st);
      else return cudaErrorInvalidValue;
    case 3: return launch_gemmk_var<BN, EPI, DH, 3>(lc, tmA, tmB, p, st);
    case 4: return launch_gemmk_var<BN, EPI, DH, 4>(lc, tmA, tmB, p, st);
    case 5: return launch_gemmk_var<BN, EPI, DH, 5>(lc, tmA, tmB, p, st);
    default: return launch_gemmk_var<BN, EPI, DH, 6>(lc, tmA, tmB, p, st);
  }
}
template <int EPI>
cudaError_t launch_gemmk_bn(const LaunchCtx& lc, int bn, int dh, const CUtensorMap& a, const CUtensorMap& b,
                            const te::GemmParams& p, cudaStream_t st) {
  if constexpr (EPI == te::EPI_QKV) {
    if (bn != 128) return cudaErrorInvalidValue;  // the split-K QKV kernel has one-head-wide (128-column) tiles only
    if (dh == 128) return launch_gemmk<128, EPI, 128>(lc, a, b, p, st);
    return launch_gemmk<128, EPI, 64>(lc, a, b, p, st);
  } else {
    if (bn == 256) return launch_gemmk<256, EPI, 128>(lc, a, b, p, st);
    return launch_gemmk<128, EPI, 128>(lc, a, b, p, st);
  }
}
// CTAs per tile: fill the SMs, keep >= 2 k-blocks per CTA
inline int choose_splits(int split_target, int tiles, int num_kb, int sm_count) {
  const int target = (split_target > 0 && split_target < sm_count) ? split_target : sm_count;
  int s = target / tiles;
  if (s > te::GEMMK_MAX_SPLITS) s = te::GEMMK_MAX_SPLITS;
  if (s > num_kb / 2) s = num_kb / 2;
  return s < 1 ? 1 : s;
}

template <int DH, int GH>
cudaError_t launch_attn(const LaunchCtx& lc, const te::AttnParams& p, int q_blocks, int n_frames, cudaStream_t st) {
  using Cfg = te::AttnCfg<DH, GH>;
  dim3 grid(q_blocks, p.n_q_heads / GH, n_frames);
  return launch_k(lc, te::te_attn_kernel<DH, GH>, grid, dim3(Cfg::THREADS), Cfg::SMEM_BYTES, st, p);
}
cudaError_t launch_attn_any(const LaunchCtx& lc, int dh, const te::AttnParams& p, int q_blocks, int n_frames,
                            cudaStream_t st) {
  const bool two = (p.n_q_heads / p.n_kv_heads) % 2 == 0;  // pairs of q heads share their kv head
  if (dh == 128)
    return two ? launch_attn<128, 2>(lc, p, q_blocks, n_frames, st) : launch_attn<128, 1>(lc, p, q_blocks, n_frames, st);
  return two ? launch_attn<64, 2>(lc, p, q_blocks, n_frames, st) : launch_attn<64, 1>(lc, p, q_blocks, n_frames, st);
}

template <int DH>
cudaError_t launch_attn_tc(const LaunchCtx& lc, const CUtensorMap& tmQ, const CUtensorMap& tmKV, const te::AttnTcParams& p,
                           int n_split, int n_frames, cudaStream_t st) {
  using Cfg = te::AttnTcCfg<DH>;
  dim3 grid(n_split, p.n_kv_heads, n_frames);
  return launch_k(lc, te::te_attn_tc_kernel<DH>, grid, dim3(Cfg::THREADS), Cfg::SMEM_BYTES, st, tmQ, tmKV, p);
}

template <int BN, int EPI, int DH>
cudaError_t set_gemm_attr() {
  cudaError_t e = cudaFuncSetAttribute(te::te_gemm_kernel<BN, EPI, DH>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                       te::GemmCfg<BN>::SMEM_BYTES);
  if (e != cudaSuccess) return e;
  if constexpr (EPI != te::EPI_QKV || BN == 128) {
#define TE_KATTR(V)                                                                                              \
  e = cudaFuncSetAttribute(te::te_gemmk_kernel<BN, EPI, DH, V>, cudaFuncAttributeMaxDynamicSharedMemorySize,        \
                           te::GemmKCfg<BN, EPI>::SMEM_BYTES);                                                      \
  if (e != cudaSuccess) return e
    TE_KATTR(0); TE_KATTR(3); TE_KATTR(4); TE_KATTR(5); TE_KATTR(6);
    if constexpr (EPI != te::EPI_QKV) { TE_KATTR(1); TE_KATTR(2); }  // (launch_gemmk: never selected for EPI_QKV)
#undef TE_KATTR
  }
  return cudaFuncSetAttribute(te::te_gemm2_kernel<BN, EPI, DH>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                              te::Gemm2Cfg<BN, EPI>::SMEM_BYTES);
}
// Opt every kernel instantiation into its dynamic shared-memory size (per device, outside any stream capture).
cudaError_t init_kernel_attrs() {
  cudaError_t e;
#define TE_ATTR(call) if ((e = (call)) != cudaSuccess) return e
  TE_ATTR((set_gemm_attr<256, te::EPI_QKV, 128>()));
  TE_ATTR((set_gemm_attr<256, te::EPI_QKV, 64>()));
  TE_ATTR((set_gemm_attr<128, te::EPI_QKV, 128>()));
  TE_ATTR((set_gemm_attr<128, te::EPI_QKV, 64>()));
  TE_ATTR((set_gemm_attr<256, te::EPI_RESID, 128>()));
  TE_ATTR((set_gemm_attr<128, te::EPI_RESID, 128>()));
  TE_ATTR((set_gemm_attr<256, te::EPI_SWIGLU, 128>()));
  TE_ATTR((set_gemm_attr<128, te::EPI_SWIGLU, 128>()));
  TE_ATTR((set_gemm_attr<256, te::EPI_PLAIN, 128>()));
  TE_ATTR((set_gemm_attr<128, te::EPI_PLAIN, 128>()));
  TE_ATTR((cudaFuncSetAttribute(te::te_gemm_wide_kernel<te::EPI_RESID>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                te::GemmWideCfg::SMEM_LIMIT)));
  TE_ATTR((cudaFuncSetAttribute(te::te_gemm_wide_kernel<te::EPI_SWIGLU>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                te::GemmWideCfg::SMEM_LIMIT)));
  TE_ATTR((cudaFuncSetAttribute(te::te_gemm_wide_kernel<te::EPI_PLAIN>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                te::GemmWideCfg::SMEM_LIMIT)));
  TE_ATTR((set_gemm8_attr<128, te::EPI_QKV, 128>()));
  TE_ATTR((set_gemm8_attr<128, te::EPI_QKV, 64>()));
  TE_ATTR((set_gemm8_attr<256, te::EPI_QKV, 128>()));
  TE_ATTR((set_gemm8_attr<128, te::EPI_RESID, 128>()));
  TE_ATTR((set_gemm8_attr<256, te::EPI_SWIGLU, 128>()));
  TE_ATTR((set_gemm8_attr<192, te::EPI_SWIGLU, 128>()));
  TE_ATTR((set_gemm8_attr<128, te::EPI_PLAIN, 128>()));
  TE_ATTR((set_gemm8_attr<256, te::EPI_PLAIN, 128>()));
  TE_ATTR((cudaFuncSetAttribute(te::te_attn_kernel<128, 1>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                te::AttnCfg<128, 1>::SMEM_BYTES)));
  TE_ATTR((cudaFuncSetAttribute(te::te_attn_kernel<128, 2>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                te::AttnCfg<128, 2>::SMEM_BYTES)));
  TE_ATTR((cudaFuncSetAttribute(te::te_attn_kernel<64, 1>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                te::AttnCfg<64, 1>::SMEM_BYTES)));
  TE_ATTR((cudaFuncSetAttribute(te::te_attn_kernel<64, 2>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                te::AttnCfg<64, 2>::SMEM_BYTES)));
  TE_ATTR((cudaFuncSetAttribute(te::te_attn_tc_kernel<128>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                te::AttnTcCfg<128>::SMEM_BYTES)));
  TE_ATTR((cudaFuncSetAttribute(te::te_attn_tc_kernel<64>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                te::AttnTcCfg<64>::SMEM_BYTES)));
#undef TE_ATTR
  return cudaSuccess;
}

// One wave of wide CTA-pair tiles (te_gemm_wide.cuh).  tmB: the weight matrix in boxes of `box_rows` rows.
template <int EPI>
cudaError_t launch_wide(const LaunchCtx& lc, const CUtensorMap& tmA, const CUtensorMap& tmB, const te::GemmParams& p,
                        int n_tiles, int bn, cudaStream_t st) {
  const int num_mp = (p.num_m_blk + 1) / 2;
  return launch_k(lc, te::te_gemm_wide_kernel<EPI>, dim3(2 * num_mp * n_tiles), dim3(te::GEMM2_THREADS),
                  te::GemmWideCfg::smem_bytes(bn), st, tmA, tmB, p, bn);
}

// Token-count bucket: the row-block count that every grid and every dispatch decision is derived from.
// Small batches: 128-row blocks; from 1024 rows on the CTA-pair kernels work on 256-row blocks.
int bucket_tokens(int T) {
  int tb = (T + 127) / 128 * 128;
  if (tb >= 1024) tb = (T + 255) / 256 * 256;
  return tb;
}

Plan make_plan(const te_handle* h, int Tb, int n_frames, int n_vis) {
  const te_config& c = h->cfg;
  const int d = c.hidden, dh = c.head_dim, F = c.ffn;
  const int n_qkv = (c.n_q_heads + 2 * c.n_kv_heads) * dh;
  Plan pl;
  pl.Tb = Tb;
  pl.mx = c.weight_dtype >= 1;
  // CTA pairs pay off once there are enough 256-row tiles to fill the SM pairs; small batches keep
  // one CTA per tile so that more SMs stream weights (HBM-bound regime).
  pl.pair = h->pair_mode == 2 ? (Tb >= 1024 ? 1 : 0) : h->pair_mode;
  // Small batches: when a GEMM has at most one 128-row tile per SM it runs on the split-K kernel, with
  // as many CTAs per tile as the SM count allows (QKV then uses one-head-wide 128-column tiles).
  const int num_m = (Tb + te::GEMM_BM - 1) / te::GEMM_BM;
  pl.num_m = num_m;
  const bool kmode = !pl.pair && h->splitk;
  pl.bn_qkv = (kmode && num_m * (n_qkv / 128) <= h->sm_count) ? 128 : h->bn_qkv;
  pl.k_qkv = kmode && pl.bn_qkv == 128;
  // more one-head tiles than SMs (512 < T < 1024 at full width): 256-row CTA-pair tiles, as for gate/up below
  pl.pair_qkv = pl.pair || (kmode && !pl.k_qkv && Tb > te::GEMM_BM && h->pair_mode == 2);
  pl.bx_qkv = box_index(pl.pair_qkv ? pl.bn_qkv / 2 : pl.bn_qkv);
  // gate/up tile width: the weights are interleaved per bn_gu = 256 rows; 128-wide tiles read them as two 64-row
  // halves (gu_half).  With one row block (T <= 128) 96 one-CTA tiles stream the weights with no split-K exchange.
  const bool gu128_k = kmode && h->bn_gu == 256 && num_m * (2 * F / 128) <= h->sm_count;
  pl.bn_gu = gu128_k ? 128 : h->bn_gu;
  pl.gu_half = pl.bn_gu != h->bn_gu;
  pl.k_gu = kmode && num_m * (2 * F / pl.bn_gu) <= h->sm_count;
  // gate/up with more tiles than SMs but too few tokens for pairs everywhere (e.g. T = 512: 192 tiles of
  // 128 x 256): 256-row CTA-pair tiles halve the L2->SM operand traffic per FLOP, which bounds this regime
  pl.pair_gu = pl.pair || (kmode && !pl.k_gu && Tb > te::GEMM_BM && h->pair_mode == 2);
  // ... and when those pair tiles need two or more waves (T = 512: 96 tiles on 74 pairs), ONE wave of wide SwiGLU
  // tiles instead: w output columns per tile = F / (pairs / row-pair blocks), rounded up to 64 (te_gemm_wide.cuh)
  const int np = h->sm_count / 2;
  const int mp_cnt = (num_m + 1) / 2;
  if (kmode && pl.pair_gu && h->resid_wide == 1 && h->bn_gu == 256) {
    const int nt = np / mp_cnt;
    if (nt >= 1) {
      const int w = (((F + nt - 1) / nt) + 63) / 64 * 64;
      const int waves256 = (mp_cnt * (2 * F / h->bn_gu) + np - 1) / np;
      if (2 * w <= 512 && waves256 >= 2 && 2 * w < waves256 * h->bn_gu) { pl.gu_wide_w = w; pl.gu_wide_tiles = (F + w - 1) / w; }
    }
  }
  pl.bx_gu = pl.gu_half ? box_index(64) : box_index(pl.pair_gu ? h->bn_gu / 2 : h->bn_gu);
  // Residual GEMMs on CTA pairs: when their 128-wide tiles would take >= 2 waves, one wave of wide tiles instead
  // (te_gemm_wide.cuh): n_tiles = pairs / row-pair blocks, width = N / n_tiles rounded up to 32 (<= 512).
  if (pl.pair && h->resid_wide) {
    int nt = h->resid_wide >= 2 ? h->resid_wide : np / mp_cnt;
    const int cap = h->ssq_parts_cap / 2 < d / 32 ? h->ssq_parts_cap / 2 : d / 32;
    if (nt > cap) nt = cap;
    if (nt >= 1) {
      const int bn = (((d + nt - 1) / nt) + 31) / 32 * 32;
      const int waves128 = (mp_cnt * (d / 128) + np - 1) / np;
      const bool wins = waves128 >= 2 && bn * 4 < waves128 * 128 * 5;
      if (bn <= 512 && mp_cnt * nt <= np && (h->resid_wide >= 2 || wins)) { pl.wide_tiles = nt; pl.wide_bn = bn; }
    }
  }
  pl.bn_res = h->bn_res;
  pl.k_res = kmode && num_m * (d / h->bn_res) <= h->sm_count;
  pl.bx_res = box_index(pl.pair ? pl.bn_res / 2 : pl.bn_res);
  pl.n_blk_res = d / pl.bn_res;
  // RMSNorm statistics: one partial sum of squares per residual N-tile and epilogue column share
  pl.parts = pl.wide_tiles ? pl.wide_tiles * 2 : pl.n_blk_res * ((pl.pair || pl.k_res) ? 2 : 1);
  if (pl.mx) {  // MXFP8: CTA pairs for everything; QKV 128- or 256-wide, gate/up 256-wide, residual GEMMs 128-wide tiles
    pl.pair = pl.pair_qkv = pl.pair_gu = 1;
    pl.k_qkv = pl.k_gu = pl.k_res = pl.wide_tiles = pl.gu_wide_tiles = pl.gu_half = 0;
    pl.bn_qkv = (n_qkv % h->bn8_qkv == 0) ? h->bn8_qkv : 128;
    pl.bn_gu = h->bn8_gu;
    pl.bn_res = 128;
    pl.n_blk_res = d / 128;
    pl.parts = pl.n_blk_res * 2;
  }
  // attention: host-side upper bound of S_b for the grid (exact lengths stay on the device)
  int s_bound = Tb - (n_frames - 1) * n_vis;
  if (s_bound > c.max_tokens_per_frame) s_bound = c.max_tokens_per_frame;
  if (s_bound < 1) s_bound = 1;
  pl.s_bound = s_bound;
  pl.q_blocks = (s_bound + te::ATT_BQ - 1) / te::ATT_BQ;
  pl.g_shift = h->g_shift;
  pl.attn_tc = h->attn_impl == 1 && h->attn_tc_ok;
  if (pl.attn_tc) {
    // one CTA per (frame, kv head), split over query tiles when the batch alone cannot fill the SMs
    const int pt = 128 >> h->g_shift;
    const int tiles_max = (s_bound + pt - 1) / pt;
    int sp = h->sm_count / (n_frames * c.n_kv_heads);
    if (sp < 1) sp = 1;
    if (sp > tiles_max) sp = tiles_max;
    pl.attn_split = sp;
  }
  return pl;
}

// What ran, by class, in the names ncu prints (te_dispatch_info; bench.py's roofline label).
std::string describe_plan(const te_handle* h, const Plan& pl) {
  const te_config& c = h->cfg;
  char b[320];
  std::string s;
  const int d_ = c.hidden, F_ = c.ffn;
  auto gemm = [&](const char* cls, int epi, bool k, bool pair2, int bn, int dh) {
    if (k) {  // the split-K kernel's 4th template argument = its epilogue variant, decided by the K split (as in enqueue_stack)
      const int n_cols = epi == te::EPI_QKV ? (c.n_q_heads + 2 * c.n_kv_heads) * c.head_dim : (epi == te::EPI_SWIGLU ? 2 * F_ : d_);
      const int k_dim = (cls[0] == 'd') ? F_ : ((cls[0] == 'o') ? c.n_q_heads * c.head_dim : d_);
      int S = choose_splits(h->split_target, pl.num_m * (n_cols / bn), k_dim / te::GEMM_BK, h->sm_count);
      if (epi == te::EPI_QKV && S == 2 && h->split_target == 0) S = 1;
      snprintf(b, sizeof(b), "%s=te_gemmk_kernel<%d, %d, %d, %d>;", cls, bn, epi, dh, S == 1 ? 0 : te::gemmk_variant(epi, S * (bn / 128)));
    }
    else if (pair2) snprintf(b, sizeof(b), "%s=te_gemm2_kernel<%d, %d, %d>;", cls, bn, epi, dh);
    else snprintf(b, sizeof(b), "%s=te_gemm_kernel<%d, %d, %d>;", cls, bn, epi, dh);
    s += b;
  };
  if (pl.mx) {
    snprintf(b, sizeof(b), "qkv=te_gemm8_kernel<%d, 1, %d>;attn=te_attn_tc_kernel<%d>;oproj=te_gemm8_kernel<128, 2, 128>;"
             "down=te_gemm8_kernel<128, 2, 128>;gateup=te_gemm8_kernel<%d, 3, 128>;bucket_tokens=%d", pl.bn_qkv,
             c.head_dim, c.head_dim, pl.bn_gu, pl.Tb);
    return std::string(b);
  }
  gemm("qkv", te::EPI_QKV, pl.k_qkv, pl.pair_qkv, pl.bn_qkv, c.head_dim);
  snprintf(b, sizeof(b), "attn=%s;", pl.attn_tc ? (c.head_dim == 128 ? "te_attn_tc_kernel<128>" : "te_attn_tc_kernel<64>")
                                                : "te_attn_kernel");
  s += b;
  if (pl.wide_tiles) {
    snprintf(b, sizeof(b), "oproj=te_gemm_wide_kernel<2> (%d tiles x %d cols);down=te_gemm_wide_kernel<2> (%d tiles x %d cols);",
             pl.wide_tiles, pl.wide_bn, pl.wide_tiles, pl.wide_bn);
    s += b;
  } else {
    gemm("oproj", te::EPI_RESID, pl.k_res, pl.pair, pl.bn_res, 128);
    gemm("down", te::EPI_RESID, pl.k_res, pl.pair, pl.bn_res, 128);
  }
  if (pl.gu_wide_tiles) {
    snprintf(b, sizeof(b), "gateup=te_gemm_wide_kernel<3> (%d tiles x %d cols);", pl.gu_wide_tiles, pl.gu_wide_w);
    s += b;
  } else {
    gemm("gateup", te::EPI_SWIGLU, pl.k_gu, pl.pair_gu, pl.bn_gu, 128);
  }
  snprintf(b, sizeof(b), "bucket_tokens=%d", pl.Tb);
  s += b;
  return s;
}

// Enqueue the whole stack on `st` for the shape class `Tb` (per-call pointers and the exact token count are in
// h->dyn, written on the stream before this sequence).  Returns the number of kernels launched via *n_kernels.
// prefix_pass: the one-frame pass of te_encode_prefix (text only, ids 0..T-1) that also saves every layer's K/V.
int enqueue_stack(te_handle* h, int n_frames, int grid_h, int grid_w, int Tb, cudaStream_t st, int* n_kernels,
                  bool prefix_pass = false, int prefix_rows = 0) {
  const te_config& c = h->cfg;
  const int d = c.hidden, dh = c.head_dim, F = c.ffn;
  const int n_qkv = (c.n_q_heads + 2 * c.n_kv_heads) * dh;
  const int n_q = c.n_q_heads * dh;
  const int lb = prefix_pass ? 0 : h->dbg_lb, le = prefix_pass ? c.n_layers : h->dbg_le;
  const bool dbg_stop = !prefix_pass && h->dbg_stop;
  const int P = prefix_pass ? 0 : h->prefix_len;  // cached prefix keys in front of every frame
  const int n_kv = 2 * c.n_kv_heads * dh;
  const Plan pl = make_plan(h, Tb, n_frames, grid_h < 0 ? 0 : grid_h * grid_w);
  if (!prefix_pass) h->last_plan = pl;
  const int num_m = pl.num_m;
  int nk = 0;
  // Optional per-kernel CUDA-event bracketing (TE_OPT_KERNEL_TIMING; never inside a capture).
  cudaEvent_t ev_a = nullptr;
  auto tick = [&]() {
    if (!h->timing) return;
    cudaEventCreate(&ev_a);
    cudaEventRecord(ev_a, st);
  };
  auto tock = [&](int kclass) {
    if (!h->timing) return;
    cudaEvent_t ev_b;
    cudaEventCreate(&ev_b);
    cudaEventRecord(ev_b, st);
    h->timed.push_back({kclass, ev_a, ev_b});
  };

  LaunchCtx lc;
  lc.pdl = h->pdl && !h->timing;
  // The fp32 residual stream (read and rewritten by both residual GEMMs of every layer) is marked persisting in L2
  // for every kernel of the stack, so that its 2 x 2 passes per layer stay out of DRAM (TE_OPT_L2_RESIDUAL).
  if (h->l2_resid && h->l2_limit_bytes > 0 && h->l2_max_window > 0) {
    // a window larger than the device allows makes every launch fail: cover the first accessPolicyMaxWindowSize bytes only
    size_t bytes = (size_t)Tb * d * sizeof(float);
    if (bytes > h->l2_max_window) bytes = h->l2_max_window;
    lc.l2.base_ptr = h->resid;
    lc.l2.num_bytes = bytes;
    lc.l2.hitRatio = bytes <= h->l2_limit_bytes ? 1.0f : (float)h->l2_limit_bytes / (float)bytes;
    lc.l2.hitProp = cudaAccessPropertyPersisting;
    lc.l2.missProp = cudaAccessPropertyStreaming;
  }
  {
    te::PrepParams pp{};
    pp.dyn = h->dyn; pp.out = h->resid; pp.cu = h->cu; pp.flag = h->flag; pp.pos = h->pos;
    pp.cos_t = h->cos_t; pp.sin_t = h->sin_t;
    pp.inv_freq = h->inv_freq; pp.g_first = h->w + h->off[lb].g1; pp.xg = h->xg; pp.ssq = h->ssq;
    pp.ssq_parts = pl.parts; pp.ssq_stride = h->ssq_parts_cap; pp.n_frames = n_frames; pp.d = d;
    pp.half_dim = dh / 2; pp.max_tokens_per_frame = c.max_tokens_per_frame;
    pp.grid_h = grid_h; pp.grid_w = grid_w; pp.pos_offset = P;
    memcpy(pp.axis, h->axis, sizeof(pp.axis));
    tick();
    pp.qkv_rows = reinterpret_cast<uint4*>(h->qkv); pp.qkv_row_vec16 = n_qkv / 8;
    pp.xg8 = pl.mx ? h->xg8 : nullptr; pp.sf_xg = h->sf_xg;
    // te_set_dyn_kernel -> prep is a FULL stream dependency (no programmatic overlap): the GEMM kernels read DynParams
    // (total_tokens, out) before their griddepcontrol.wait, which is only ordered behind set_dyn if the kernel between
    // them started after set_dyn had completed.  Inside a replayed graph prep is the first node, so nothing is lost.
    LaunchCtx lc_first = lc;
    lc_first.pdl = false;
    TE_CUDA(h, launch_k(lc_first, te::te_prep_kernel, dim3(Tb + te::PREP_PAD_ROWS), dim3(256), 0, st, pp));
    tock(TE_KCLASS_PREP);
    ++nk;
  }
  te::GemmParams base{};
  base.dyn = h->dyn;
  base.splits = 1; base.sk_scratch = h->sk_scratch; base.sk_sem = h->sk_sem;
  base.M = Tb; base.num_m_blk = num_m; base.ssq_in = h->ssq; base.ssq_parts = pl.parts; base.ssq_stride = h->ssq_parts_cap;
  base.inv_d = 1.0f / static_cast<float>(d); base.eps = c.rms_eps;
  const size_t trace_stride = (size_t)h->sm_dev * te::TRACE_SLOTS;
  auto trace_ptr = [&](int cls) { return h->trace_on ? h->trace + cls * trace_stride : nullptr; };
  // the last residual GEMM of the stack hands the stream over to the caller's buffer
  const bool norm_tail = c.final_norm && le == c.n_layers && !dbg_stop;

  // ---- per-GEMM parameters of layer l
  auto qkv_params = [&](int l) {
    const LayerOff& o = h->off[l];
    te::GemmParams p = base;
    p.N = n_qkv; p.K = d; p.num_n_blk = n_qkv / pl.bn_qkv;
    p.qkv = h->qkv; p.ld_qkv = n_qkv; p.q_cols_end = n_q; p.k_cols_end = n_q + c.n_kv_heads * dh;
    p.gq = h->w + o.gq; p.gk = h->w + o.gk; p.cos_t = h->cos_t; p.sin_t = h->sin_t;
    p.trace = trace_ptr(0);
    if (pl.k_qkv) {
      p.splits = choose_splits(h->split_target, num_m * p.num_n_blk, p.K / te::GEMM_BK, h->sm_count);
      // two K slices per one-head tile (T = 256: 64 tiles) lose more in the exchange and the 64-row slice epilogues
      // than they gain in the main loop: 17.6 us against 13.0 us unsplit (B = 2, measured)
      if (p.splits == 2 && h->split_target == 0) p.splits = 1;
    }
    return p;
  };
  auto oproj_params = [&](int l, bool last_layer) {
    const LayerOff& o = h->off[l];
    te::GemmParams p = base;
    p.N = d; p.K = n_q; p.num_n_blk = pl.n_blk_res;
    p.x = h->resid; p.ld_x = d; p.g_next = h->w + o.g2; p.xg = h->xg; p.ssq_out = h->ssq;
    p.x_to_out = (dbg_stop && last_layer) ? 1 : 0;
    p.trace = trace_ptr(1);
    if (pl.k_res) p.splits = choose_splits(h->split_target, num_m * p.num_n_blk, p.K / te::GEMM_BK, h->sm_count);
    return p;
  };
  auto gu_params = [&](int l) {
    te::GemmParams p = base;
    p.N = 2 * F; p.K = d; p.num_n_blk = 2 * F / pl.bn_gu; p.gu_half = pl.gu_half;
    p.act = h->act; p.ld_act = F;
    p.trace = trace_ptr(2);
    if (pl.k_gu) p.splits = choose_splits(h->split_target, num_m * p.num_n_blk, p.K / te::GEMM_BK, h->sm_count);
    return p;
  };
  auto down_params = [&](int l, bool last_layer) {
    te::GemmParams p = base;
    p.N = d; p.K = F; p.num_n_blk = pl.n_blk_res;
    p.x = h->resid; p.ld_x = d; p.xg = h->xg; p.ssq_out = h->ssq;
    p.g_next = (l + 1 < c.n_layers) ? h->w + h->off[l + 1].g1 : nullptr;
    p.x_to_out = (last_layer && !norm_tail) ? 1 : 0;
    p.trace = trace_ptr(3);
    if (pl.k_res) p.splits = choose_splits(h->split_target, num_m * p.num_n_blk, p.K / te::GEMM_BK, h->sm_count);
    return p;
  };
  for (int l = lb; l < le; ++l) {
    const LayerOff& o = h->off[l];
    const bool last_layer = l == le - 1;
    {  // a1: RMSNorm -> QKV GEMM -> QK-norm + M-RoPE
      te::GemmParams p = qkv_params(l);
      tick();
      if (pl.mx) {
        te::Gemm8Extra x8{};
        x8.b_fp4 = c.weight_dtype == 2;
        const CUtensorMap& tb = h->tm8[l].qkv[pl.bn_qkv == 256 ? 1 : 0];
        const CUtensorMap &sa = h->tmSF_xg, &sb = h->tm8[l].sf_qkv;
        cudaError_t e = pl.bn_qkv == 256 ? launch_gemm8<256, te::EPI_QKV, 128>(lc, h->tmA_xg8, tb, sa, sb, p, x8, h->sm_count, st)
                        : dh == 128     ? launch_gemm8<128, te::EPI_QKV, 128>(lc, h->tmA_xg8, tb, sa, sb, p, x8, h->sm_count, st)
                                        : launch_gemm8<128, te::EPI_QKV, 64>(lc, h->tmA_xg8, tb, sa, sb, p, x8, h->sm_count, st);
        TE_CUDA(h, e);
      } else if (pl.k_qkv) {
        TE_CUDA(h, launch_gemmk_bn<te::EPI_QKV>(lc, pl.bn_qkv, dh, h->tmA_xg, h->tm[l].qkv[pl.bx_qkv], p, st));
      } else {
        TE_CUDA(h, launch_gemm_bn<te::EPI_QKV>(lc, pl.bn_qkv, pl.pair_qkv, dh, h->tmA_xg, h->tm[l].qkv[pl.bx_qkv], p,
                                                h->sm_count, st));
      }
      tock(TE_KCLASS_QKV);
      ++nk;
    }
    if (prefix_pass) {  // keep this layer's keys | values of the prefix tokens
      TE_CUDA(h, cudaMemcpy2DAsync(h->kv_prefix + (size_t)l * c.max_prefix_tokens * n_kv, (size_t)n_kv * sizeof(bf16),
                                   h->qkv + n_q, (size_t)n_qkv * sizeof(bf16), (size_t)n_kv * sizeof(bf16),
                                   prefix_rows, cudaMemcpyDeviceToDevice, st));
    }
    {  // a2: causal GQA attention
      const float scale_log2 = static_cast<float>(1.4426950408889634 / std::sqrt(static_cast<double>(dh)));
      tick();
      if (pl.attn_tc) {
        te::AttnTcParams tp{};
        tp.out = h->attn; tp.cu_seqlens = h->cu; tp.n_q_heads = c.n_q_heads; tp.n_kv_heads = c.n_kv_heads;
        tp.g_shift = pl.g_shift; tp.scale_log2 = scale_log2; tp.non_causal = c.non_causal;
        tp.stats = P > 0 ? h->attn_stats : nullptr; tp.o32 = P > 0 ? h->attn_o32 : nullptr; tp.prefix_mode = 0; tp.prefix_len = 0;
        tp.out8 = pl.mx ? h->attn8 : nullptr; tp.sf_out = h->sf_attn;
        tp.trace = trace_ptr(4); tp.trace_ctas = h->sm_dev;
        TE_CUDA(h, dh == 128 ? launch_attn_tc<128>(lc, h->tmQ, h->tmKV, tp, pl.attn_split, n_frames, st)
                             : launch_attn_tc<64>(lc, h->tmQ, h->tmKV, tp, pl.attn_split, n_frames, st));
        if (P > 0) {  // second pass: the P cached prefix keys of this layer, merged in place
          tp.prefix_mode = 1; tp.prefix_len = P;
          TE_CUDA(h, dh == 128 ? launch_attn_tc<128>(lc, h->tmQ, h->tm_prefix[l], tp, pl.attn_split, n_frames, st)
                               : launch_attn_tc<64>(lc, h->tmQ, h->tm_prefix[l], tp, pl.attn_split, n_frames, st));
          ++nk;
        }
      } else {
        te::AttnParams ap{};
        ap.qkv = h->qkv; ap.out = h->attn; ap.cu_seqlens = h->cu; ap.ld = n_qkv; ap.n_q_heads = c.n_q_heads;
        ap.n_kv_heads = c.n_kv_heads; ap.scale_log2 = scale_log2;
        ap.prefix_len = P; ap.ld_prefix = n_kv; ap.non_causal = c.non_causal;
        ap.kv_prefix = P > 0 ? h->kv_prefix + (size_t)l * c.max_prefix_tokens * n_kv : nullptr;
        TE_CUDA(h, launch_attn_any(lc, dh, ap, pl.q_blocks, n_frames, st));
      }
      tock(TE_KCLASS_ATTN);
      ++nk;
    }
    {  // a3: O projection + residual add (+ next norm's gain / statistics)
      te::GemmParams p = oproj_params(l, last_layer);
      tick();
      if (pl.mx) {
        te::Gemm8Extra x8{};
        x8.b_fp4 = c.weight_dtype == 2;
        x8.q_out = h->xg8; x8.q_sf = h->sf_xg; x8.q_kchunks = d / 128; x8.q_ld = d;
        TE_CUDA(h, (launch_gemm8<128, te::EPI_RESID, 128>(lc, h->tmA_attn8, h->tm8[l].o[0], h->tmSF_attn, h->tm8[l].sf_o, p, x8,
                                                        h->sm_count, st)));
      } else if (pl.wide_tiles) {
        CUtensorMap tmB;
        if (!make_tmap(&tmB, h->w + o.wo, d, n_q, pl.wide_bn / 4)) { h->err = "tensor map (wide O-proj)"; return TE_ERR_CUDA; }
        TE_CUDA(h, launch_wide<te::EPI_RESID>(lc, h->tmA_attn, tmB, p, pl.wide_tiles, pl.wide_bn, st));
      } else if (pl.k_res) {
        TE_CUDA(h, launch_gemmk_bn<te::EPI_RESID>(lc, pl.bn_res, dh, h->tmA_attn, h->tm[l].o[pl.bx_res], p, st));
      } else {
        TE_CUDA(h, launch_gemm_bn<te::EPI_RESID>(lc, pl.bn_res, pl.pair, dh, h->tmA_attn, h->tm[l].o[pl.bx_res], p,
                                                  h->sm_count, st));
      }
      tock(TE_KCLASS_OPROJ);
      ++nk;
    }
    if (dbg_stop && last_layer) break;
    {  // a4: RMSNorm -> gate/up GEMM -> SiLU(gate) * up
      te::GemmParams p = gu_params(l);
      tick();
      if (pl.mx) {
        te::Gemm8Extra x8{};
        x8.b_fp4 = c.weight_dtype == 2;
        x8.q_out = h->act8; x8.q_sf = h->sf_act; x8.q_kchunks = F / 128; x8.q_ld = F;
        p.num_n_blk = 2 * F / pl.bn_gu;
        TE_CUDA(h, pl.bn_gu == 192 ? (launch_gemm8<192, te::EPI_SWIGLU, 128>(lc, h->tmA_xg8, h->tm8[l].gu[0], h->tmSF_xg,
                                                                            h->tm8[l].sf_gu, p, x8, h->sm_count, st))
                                   : (launch_gemm8<256, te::EPI_SWIGLU, 128>(lc, h->tmA_xg8, h->tm8[l].gu[1], h->tmSF_xg,
                                                                            h->tm8[l].sf_gu, p, x8, h->sm_count, st)));
      } else if (pl.gu_wide_tiles) {
        p.gu_half = 0;
        TE_CUDA(h, launch_wide<te::EPI_SWIGLU>(lc, h->tmA_xg, h->tm[l].gu[box_index(32)], p, pl.gu_wide_tiles,
                                               2 * pl.gu_wide_w, st));
      } else if (pl.k_gu) {
        TE_CUDA(h, launch_gemmk_bn<te::EPI_SWIGLU>(lc, pl.bn_gu, dh, h->tmA_xg, h->tm[l].gu[pl.bx_gu], p, st));
      } else {
        TE_CUDA(h, launch_gemm_bn<te::EPI_SWIGLU>(lc, pl.bn_gu, pl.pair_gu, dh, h->tmA_xg, h->tm[l].gu[pl.bx_gu], p,
                                                   h->sm_count, st));
      }
      tock(TE_KCLASS_GATEUP);
      ++nk;
    }
    {  // a5: down projection + residual add
      te::GemmParams p = down_params(l, last_layer);
      tick();
      if (pl.mx) {
        te::Gemm8Extra x8{};
        x8.b_fp4 = c.weight_dtype == 2;
        x8.q_out = h->xg8; x8.q_sf = h->sf_xg; x8.q_kchunks = d / 128; x8.q_ld = d;
        TE_CUDA(h, (launch_gemm8<128, te::EPI_RESID, 128>(lc, h->tmA_act8, h->tm8[l].d[0], h->tmSF_act, h->tm8[l].sf_d, p, x8,
                                                        h->sm_count, st)));
      } else if (pl.wide_tiles) {
        CUtensorMap tmB;
        if (!make_tmap(&tmB, h->w + o.wd, d, F, pl.wide_bn / 4)) { h->err = "tensor map (wide down)"; return TE_ERR_CUDA; }
        TE_CUDA(h, launch_wide<te::EPI_RESID>(lc, h->tmA_act, tmB, p, pl.wide_tiles, pl.wide_bn, st));
      } else if (pl.k_res) {
        TE_CUDA(h, launch_gemmk_bn<te::EPI_RESID>(lc, pl.bn_res, dh, h->tmA_act, h->tm[l].d[pl.bx_res], p, st));
      } else {
        TE_CUDA(h, launch_gemm_bn<te::EPI_RESID>(lc, pl.bn_res, pl.pair, dh, h->tmA_act, h->tm[l].d[pl.bx_res], p,
                                                  h->sm_count, st));
      }
      tock(TE_KCLASS_DOWN);
      ++nk;
    }
  }
  if (norm_tail) {  // a6: residual stream -> RMSNorm -> the caller's buffer
    tick();
    TE_CUDA(h, launch_k(lc, te::te_final_norm_kernel, dim3((Tb + 7) / 8), dim3(256), 0, st,
                        static_cast<const float*>(h->resid), static_cast<const te::DynParams*>(h->dyn),
                        static_cast<const bf16*>(h->w + h->gf_off), d, c.rms_eps));
    tock(TE_KCLASS_FINAL_NORM);
    ++nk;
  }
  *n_kernels = nk;
  return TE_OK;
}

void free_graphs(te_handle* h) {
  for (auto& e : h->cache) {
    cudaGraphExecDestroy(e.exec);
    cudaGraphDestroy(e.graph);
  }
  h->cache.clear();
}

// Per-call values -> device block, on the stream, ahead of the stack (values travel as kernel parameters).
cudaError_t set_dyn(te_handle* h, const void* embeds, const int32_t* lens, float* out, int T, cudaStream_t st,
                    const int32_t* grids = nullptr, int embeds_bf16 = 0) {
  te::DynParams v{};
  v.embeds = embeds; v.text_lens = lens; v.out = out; v.total_tokens = T; v.grids = grids; v.embeds_bf16 = embeds_bf16;
  te::te_set_dyn_kernel<<<1, 32, 0, st>>>(h->dyn, v);
  return cudaGetLastError();
}

// cudaLimitPersistingL2CacheSize is ONE value per device, shared by every handle of the process (a decoder handle and a
// vision tower's handle is the normal pairing) and possibly touched from several host threads: one mutex-protected
// record per device keeps the value found before the first handle asked, the largest request, and how many handles
// hold it.  The limit is raised to the largest request and put back (persisting lines reset) by the LAST release.
struct L2Record {
  size_t orig = 0, cur = 0;
  int refs = 0;
};
constexpr int L2_MAX_DEVICES = 64;
L2Record g_l2[L2_MAX_DEVICES];
std::mutex g_l2_mu;

// Device `device` is current.  True if a carve-out of at least `want` bytes is now in force (one reference taken).
bool l2_acquire(int device, size_t want) {
  if (device < 0 || device >= L2_MAX_DEVICES || want == 0) return false;
  std::lock_guard<std::mutex> lock(g_l2_mu);
  L2Record& r = g_l2[device];
  if (r.refs == 0) {
    if (cudaDeviceGetLimit(&r.orig, cudaLimitPersistingL2CacheSize) != cudaSuccess) { cudaGetLastError(); return false; }
    r.cur = r.orig;
  }
  if (want > r.cur) {
    if (cudaDeviceSetLimit(cudaLimitPersistingL2CacheSize, want) != cudaSuccess) { cudaGetLastError(); return false; }
    r.cur = want;
  }
  ++r.refs;
  return true;
}
void l2_release(int device) {
  std::lock_guard<std::mutex> lock(g_l2_mu);
  L2Record& r = g_l2[device];
  if (r.refs > 0 && --r.refs == 0) {
    cudaCtxResetPersistingL2Cache();
    if (r.cur != r.orig) cudaDeviceSetLimit(cudaLimitPersistingL2CacheSize, r.orig);
    cudaGetLastError();
    r.cur = r.orig;
  }
}

void release_l2_limit(te_handle* h) {
  if (h->l2_ref_held) {
    l2_release(h->device);
    h->l2_ref_held = false;
  }
  h->l2_limit_bytes = 0;
}

}  // namespace

extern "C" {

size_t te_blob_bytes(const te_config* cfg) {
  if (!cfg || validate_config(*cfg) != TE_OK) return 0;
  return blob_elems(*cfg) * sizeof(bf16);
}

int te_create(const te_config* cfg, int device, te_handle** out) {
  if (!cfg || !out) return TE_ERR_INVALID_ARG;
  *out = nullptr;
  int rc = validate_config(*cfg);
  if (rc != TE_OK) return rc;
  int n_dev = 0;
  if (cudaGetDeviceCount(&n_dev) != cudaSuccess || device < 0 || device >= n_dev) return TE_ERR_CUDA;
  cudaDeviceProp prop;
  if (cudaGetDeviceProperties(&prop, device) != cudaSuccess) return TE_ERR_CUDA;
  if (prop.major != 10) return TE_ERR_UNSUPPORTED;  // tcgen05 / TMEM: sm_100 family only; no fallback
  if (!get_encode_fn()) return TE_ERR_CUDA;
  if (cudaSetDevice(device) != cudaSuccess) return TE_ERR_CUDA;
  if (init_kernel_attrs() != cudaSuccess) return TE_ERR_CUDA;

  te_handle* h = new te_handle();
  h->cfg = *cfg;
  h->device = device;
  h->sm_count = h->sm_dev = prop.multiProcessorCount;
  h->l2_max_persist = (size_t)prop.persistingL2CacheMaxSize;
  h->l2_max_window = prop.accessPolicyMaxWindowSize > 0 ? (size_t)prop.accessPolicyMaxWindowSize : 0;
  h->dbg_lb = 0;
  h->dbg_le = cfg->n_layers;
  const te_config& c = h->cfg;
  const int n_qkv = (c.n_q_heads + 2 * c.n_kv_heads) * c.head_dim;
  const int n_q = c.n_q_heads * c.head_dim;
  h->bn_qkv = (n_qkv % 256 == 0) ? 256 : 128;
  h->bn_gu = ((2 * c.ffn) % 256 == 0) ? 256 : 128;
  h->bn_res = 128;  // O/down: N = hidden is small -> 128-wide tiles halve the wave-quantisation loss
  h->ssq_parts_cap = ((c.hidden / 128) * (te::GEMM2_EPI_WARPS / 4) + 3) & ~3;  // row stride of ssq (16-byte aligned rows)
  h->cap_rows = (c.max_tokens + 255) / 256 * 256 + te::PREP_PAD_ROWS;  // (+ the zeroed rows past the last token)

  auto fail = [&](int code) {
    te_destroy(h);
    return code;
  };
  const size_t T = h->cap_rows, B = c.max_frames, hd2 = c.head_dim / 2;
#define TE_ALLOC(ptr, bytes) \
  if (cudaMalloc(reinterpret_cast<void**>(&(ptr)), (bytes)) != cudaSuccess) return fail(TE_ERR_CUDA)
  TE_ALLOC(h->dyn, sizeof(te::DynParams));
  TE_ALLOC(h->resid, T * c.hidden * sizeof(float));
  TE_ALLOC(h->cu, (B + 1) * sizeof(int32_t));
  TE_ALLOC(h->pos, 3 * T * sizeof(int32_t));
  TE_ALLOC(h->flag, sizeof(int32_t));
  TE_ALLOC(h->cos_t, T * hd2 * sizeof(float));
  TE_ALLOC(h->sin_t, T * hd2 * sizeof(float));
  TE_ALLOC(h->ssq, (size_t)h->ssq_parts_cap * T * sizeof(float));
  TE_ALLOC(h->inv_freq, hd2 * sizeof(double));
  TE_ALLOC(h->xg, T * c.hidden * sizeof(bf16));
  TE_ALLOC(h->qkv, T * n_qkv * sizeof(bf16));
  TE_ALLOC(h->attn, T * (size_t)n_q * sizeof(bf16));
  TE_ALLOC(h->act, T * c.ffn * sizeof(bf16));
  TE_ALLOC(h->sk_scratch, (size_t)h->sm_count * te::GEMM_BM * 256 * sizeof(float));
  TE_ALLOC(h->sk_sem, 2 * (size_t)h->sm_count * sizeof(int));
#undef TE_ALLOC
  // rows past a call's tokens are read (never stored) by the tile-granular kernels: start them finite
  if (cudaMemset(h->xg, 0, T * c.hidden * sizeof(bf16)) != cudaSuccess ||
      cudaMemset(h->qkv, 0, T * n_qkv * sizeof(bf16)) != cudaSuccess ||
      cudaMemset(h->attn, 0, T * (size_t)n_q * sizeof(bf16)) != cudaSuccess ||
      cudaMemset(h->act, 0, T * c.ffn * sizeof(bf16)) != cudaSuccess ||
      cudaMemset(h->dyn, 0, sizeof(te::DynParams)) != cudaSuccess ||
      cudaMemset(h->sk_sem, 0, 2 * (size_t)h->sm_count * sizeof(int)) != cudaSuccess)
    return fail(TE_ERR_CUDA);
  if (c.weight_dtype >= 1) {  // MXFP8 activations (A operands) + tiled block scales (one byte per 32 elements)
    const size_t rb = (T + 127) / 128;  // 128-row scale tiles
    if (cudaMalloc(reinterpret_cast<void**>(&h->xg8), T * c.hidden) != cudaSuccess ||
        cudaMalloc(reinterpret_cast<void**>(&h->attn8), T * (size_t)n_q) != cudaSuccess ||
        cudaMalloc(reinterpret_cast<void**>(&h->act8), T * (size_t)c.ffn) != cudaSuccess ||
        cudaMalloc(reinterpret_cast<void**>(&h->sf_xg), rb * (c.hidden / 128) * 512) != cudaSuccess ||
        cudaMalloc(reinterpret_cast<void**>(&h->sf_attn), rb * (n_q / 128) * 512) != cudaSuccess ||
        cudaMalloc(reinterpret_cast<void**>(&h->sf_act), rb * (c.ffn / 128) * 512) != cudaSuccess)
      return fail(TE_ERR_CUDA);
    // rows past a call's tokens are multiplied (never stored): start them as zeros with unit scales
    cudaMemset(h->xg8, 0, T * c.hidden);
    cudaMemset(h->attn8, 0, T * (size_t)n_q);
    cudaMemset(h->act8, 0, T * (size_t)c.ffn);
    cudaMemset(h->sf_xg, 127, rb * (c.hidden / 128) * 512);
    cudaMemset(h->sf_attn, 127, rb * (n_q / 128) * 512);
    cudaMemset(h->sf_act, 127, rb * (c.ffn / 128) * 512);
    if (!make_tmap_u8(&h->tmA_xg8, h->xg8, T, c.hidden, te::GEMM_BM) || !make_tmap_u8(&h->tmA_attn8, h->attn8, T, n_q, te::GEMM_BM) ||
        !make_tmap_u8(&h->tmA_act8, h->act8, T, c.ffn, te::GEMM_BM) || !make_tmap_sf(&h->tmSF_xg, h->sf_xg, rb * (c.hidden / 128)) ||
        !make_tmap_sf(&h->tmSF_attn, h->sf_attn, rb * (n_q / 128)) || !make_tmap_sf(&h->tmSF_act, h->sf_act, rb * (c.ffn / 128)))
      return fail(TE_ERR_CUDA);
  }
  if (c.max_prefix_tokens > 0) {
    const size_t n_kv = 2 * (size_t)c.n_kv_heads * c.head_dim;
    if (cudaMalloc(reinterpret_cast<void**>(&h->kv_prefix), (size_t)c.n_layers * c.max_prefix_tokens * n_kv * sizeof(bf16)) !=
            cudaSuccess ||
        cudaMalloc(reinterpret_cast<void**>(&h->prefix_buf), (size_t)c.max_prefix_tokens * c.hidden * sizeof(float)) !=
            cudaSuccess ||
        cudaMalloc(reinterpret_cast<void**>(&h->prefix_lens), sizeof(int32_t)) != cudaSuccess ||
        cudaMalloc(reinterpret_cast<void**>(&h->attn_stats), T * c.n_q_heads * sizeof(float2)) != cudaSuccess ||
        cudaMalloc(reinterpret_cast<void**>(&h->attn_o32), T * (size_t)n_q * sizeof(float)) != cudaSuccess)
      return fail(TE_ERR_CUDA);
  }
  {  // activation tensor maps over the whole workspace buffers (encoded once)
    const int G = c.n_q_heads / c.n_kv_heads;
    int g_shift = 0;
    while ((1 << g_shift) < G) ++g_shift;
    h->g_shift = g_shift;
    // tcgen05 attention needs G = Hq/Hkv to be a power of two with >= 16 positions per 128-row query tile
    h->attn_tc_ok = (1 << g_shift) == G && G <= 8;
    bool ok = make_tmap(&h->tmA_xg, h->xg, T, c.hidden, te::GEMM_BM) && make_tmap(&h->tmA_attn, h->attn, T, n_q, te::GEMM_BM) &&
              make_tmap(&h->tmA_act, h->act, T, c.ffn, te::GEMM_BM);
    if (ok && h->attn_tc_ok)
      ok = make_tmap(&h->tmQ, h->qkv, T, n_qkv, 128 >> g_shift) && make_tmap(&h->tmKV, h->qkv, T, n_qkv, 64);
    if (!ok) return fail(TE_ERR_CUDA);
  }
  {  // axis of frequency pair i: contiguous [t | h | w], or round-robin over the axes with pairs left
    int left[3] = {c.rope_sec_t, c.rope_sec_h, c.rope_sec_w};
    int a = 0;
    for (size_t i = 0; i < hd2; ++i) {
      if (c.rope_interleaved) {
        while (left[a] == 0) a = (a + 1) % 3;
        h->axis[i] = static_cast<int8_t>(a);
        --left[a];
        a = (a + 1) % 3;
      } else {
        h->axis[i] = static_cast<int8_t>((int)i < c.rope_sec_t ? 0 : ((int)i < c.rope_sec_t + c.rope_sec_h ? 1 : 2));
      }
    }
  }
  if (cudaMemset(h->flag, 0, sizeof(int32_t)) != cudaSuccess) return fail(TE_ERR_CUDA);
  std::vector<double> invf(hd2);
  for (size_t i = 0; i < hd2; ++i) invf[i] = std::pow(c.rope_theta, -2.0 * (double)i / (double)c.head_dim);
  if (cudaMemcpy(h->inv_freq, invf.data(), hd2 * sizeof(double), cudaMemcpyHostToDevice) != cudaSuccess)
    return fail(TE_ERR_CUDA);
  if (cudaStreamCreateWithFlags(&h->own_stream, cudaStreamNonBlocking) != cudaSuccess) return fail(TE_ERR_CUDA);
  *out = h;
  return TE_OK;
}

int te_load_weights(te_handle* h, const void* blob, size_t n_bytes) {
  if (!h || !blob) return TE_ERR_INVALID_ARG;
  const te_config& c = h->cfg;
  const size_t n_el = blob_elems(c);
  if (n_bytes != n_el * sizeof(bf16)) return TE_ERR_BLOB_SIZE;
  TE_CUDA(h, cudaSetDevice(h->device));
  free_graphs(h);
  h->loaded = false;
  if (!h->w) TE_CUDA(h, cudaMalloc(reinterpret_cast<void**>(&h->w), n_el * sizeof(bf16)));
  h->w_elems = n_el;
  // The device copy keeps the canonical layout (so Wq|Wk|Wv are already one fused [Nqkv, d] matrix);
  // only [Wgate; Wup] is rewritten, interleaved per N-tile, via a one-layer staging buffer.
  TE_CUDA(h, cudaMemcpy(h->w, blob, n_bytes, cudaMemcpyDefault));
  const size_t d = c.hidden, dh = c.head_dim, F = c.ffn;
  const size_t n_qkv = (size_t)(c.n_q_heads + 2 * c.n_kv_heads) * dh, n_q = (size_t)c.n_q_heads * dh;
  bf16* stage = nullptr;
  TE_CUDA(h, cudaMalloc(reinterpret_cast<void**>(&stage), 2 * F * d * sizeof(bf16)));
  h->off.resize(c.n_layers);
  h->tm.resize(c.n_layers);
  size_t o = 0;
  bool ok = true;
  cudaError_t e = cudaSuccess;
  for (int l = 0; l < c.n_layers && e == cudaSuccess; ++l) {
    LayerOff& L = h->off[l];
    L.g1 = o; o += d;
    L.wqkv = o; o += n_qkv * d;
    L.gq = o; o += dh;
    L.gk = o; o += dh;
    L.wo = o; o += d * n_q;
    L.g2 = o; o += d;
    L.wgu = o; o += 2 * F * d;
    L.wd = o; o += d * F;
    e = cudaMemcpy(stage, h->w + L.wgu, 2 * F * d * sizeof(bf16), cudaMemcpyDeviceToDevice);
    if (e == cudaSuccess) {
      te::te_interleave_gate_up_kernel<<<(unsigned)(2 * F), 128>>>(
          reinterpret_cast<const uint4*>(stage), reinterpret_cast<const uint4*>(stage + F * d),
          reinterpret_cast<uint4*>(h->w + L.wgu), (int)F, (int)(d / 8), h->bn_gu);
      e = cudaGetLastError();
    }
    for (int bi = 0; bi < 4; ++bi) {
      const uint32_t box = 32u << bi;
      ok = ok && make_tmap(&h->tm[l].qkv[bi], h->w + L.wqkv, n_qkv, d, box);
      ok = ok && make_tmap(&h->tm[l].o[bi], h->w + L.wo, d, n_q, box);
      ok = ok && make_tmap(&h->tm[l].gu[bi], h->w + L.wgu, 2 * F, d, box);
      ok = ok && make_tmap(&h->tm[l].d[bi], h->w + L.wd, d, F, box);
    }
  }
  h->gf_off = o;
  if (e == cudaSuccess && c.weight_dtype >= 1) {
    const bool fp4 = c.weight_dtype == 2;  // MXFP4 weights: two elements per byte, same scale layout
    // MXFP8 copies of the four matrices of every layer (gate/up from the interleaved copy) + tiled block scales
    // gate/up tile width of the MXFP8 GEMM: 192 (two accumulator stages) when it divides 2F, else 256
    if ((2 * F) % 192 != 0 || h->bn_gu != 256) h->bn8_gu = 256;
    const size_t gu_tile = (size_t)h->bn8_gu;
    const size_t per_layer = (n_qkv * d + d * n_q + 2 * F * d + d * F) / (fp4 ? 2 : 1);
    // scale tiles (512 B each): 128-row blocks x K/128 chunks; gate/up's are grouped per N tile (2 per 192 or 256 rows)
    auto sf_tiles = [](size_t rows, size_t K, size_t tile_rows) { return rows / tile_rows * ((tile_rows + 127) / 128) * (K / 128); };
    const size_t sf_layer = (sf_tiles(n_qkv, d, 128) + sf_tiles(d, n_q, 128) + sf_tiles(2 * F, d, gu_tile) + sf_tiles(d, F, 128)) * 512;
    if (!h->w8) e = cudaMalloc(reinterpret_cast<void**>(&h->w8), per_layer * c.n_layers);
    if (e == cudaSuccess && !h->sfw) e = cudaMalloc(reinterpret_cast<void**>(&h->sfw), sf_layer * c.n_layers);
    if (e == cudaSuccess) e = cudaMemset(h->sfw, 127, sf_layer * c.n_layers);  // (half-used tiles of 192-row groups)
    h->tm8.resize(c.n_layers);
    size_t o8 = 0, os = 0;
    auto quant = [&](size_t src_off, size_t rows, size_t K, size_t tile_rows, int gu_src, size_t* w_off, size_t* s_off,
                     CUtensorMap* sf_map) {
      *w_off = o8;
      *s_off = os;
      const long long blocks = (long long)rows * (K / 32);
      if (fp4)
        te::te_mx_quantise_fp4_kernel<<<(unsigned)((blocks + 255) / 256), 256>>>(h->w + src_off, h->w8 + o8, h->sfw + os, (int)rows,
                                                                               (int)K, (int)tile_rows, gu_src);
      else
        te::te_mx_quantise_bf16_kernel<<<(unsigned)((blocks + 255) / 256), 256>>>(h->w + src_off, h->w8 + o8, h->sfw + os, (int)rows,
                                                                                (int)K, (int)tile_rows, gu_src);
      ok = ok && make_tmap_sf(sf_map, h->sfw + os, sf_tiles(rows, K, tile_rows));
      o8 += rows * K / (fp4 ? 2 : 1);
      os += sf_tiles(rows, K, tile_rows) * 512;
    };
    for (int l = 0; l < c.n_layers && e == cudaSuccess; ++l) {
      LayerOff& L = h->off[l];
      quant(L.wqkv, n_qkv, d, 128, 0, &L.q8, &L.sq8, &h->tm8[l].sf_qkv);
      quant(L.wo, d, n_q, 128, 0, &L.o8, &L.so8, &h->tm8[l].sf_o);
      quant(L.wgu, 2 * F, d, gu_tile, gu_tile == 256 ? 0 : h->bn_gu, &L.gu8, &L.sgu8, &h->tm8[l].sf_gu);
      quant(L.wd, d, F, 128, 0, &L.d8, &L.sd8, &h->tm8[l].sf_d);
      e = cudaGetLastError();
      for (int bi = 0; bi < 2; ++bi) {
        const uint32_t box = 64u << bi;
        auto wmap = fp4 ? make_tmap_u4 : make_tmap_u8;
        ok = ok && wmap(&h->tm8[l].qkv[bi], h->w8 + L.q8, n_qkv, d, box);
        ok = ok && wmap(&h->tm8[l].o[bi], h->w8 + L.o8, d, n_q, box);
        ok = ok && wmap(&h->tm8[l].gu[bi], h->w8 + L.gu8, 2 * F, d, bi == 0 && gu_tile == 192 ? 96u : box);
        ok = ok && wmap(&h->tm8[l].d[bi], h->w8 + L.d8, d, F, box);
      }
    }
  }
  if (e == cudaSuccess) e = cudaDeviceSynchronize();
  cudaFree(stage);
  if (e != cudaSuccess) {
    h->err = std::string("te_load_weights: ") + cudaGetErrorString(e);
    return TE_ERR_CUDA;
  }
  if (!ok) {
    h->err = "cuTensorMapEncodeTiled failed for a weight map";
    return TE_ERR_CUDA;
  }
  h->loaded = true;
  return TE_OK;
}

// te_encode / te_encode_ex.  grids != null: one (grid_h, grid_w) per frame on the device; the scalar grid is then unused
// (-1 in the graph key; attention grids are sized for the longest frame the capacities allow).
static int encode_impl(te_handle* h, int32_t n_frames, const int32_t* grids, int32_t grid_h, int32_t grid_w, const void* embeds,
                       int embeds_bf16, const int32_t* text_lens, int32_t total_tokens, float* out, void* cuda_stream) {
  if (!h) return TE_ERR_INVALID_ARG;
  if (!h->loaded) return TE_ERR_NOT_LOADED;
  const te_config& c = h->cfg;
  if (!embeds || !text_lens || !out || embeds == out) return TE_ERR_INVALID_ARG;
  if (n_frames < 1 || n_frames > c.max_frames) return TE_ERR_INVALID_ARG;
  if (total_tokens < 1 || total_tokens > c.max_tokens) return TE_ERR_INVALID_ARG;
  if (grids == nullptr) {
    if (grid_h < 1 || grid_w < 1) return TE_ERR_INVALID_ARG;
    if ((long long)grid_h * grid_w > c.max_tokens_per_frame) return TE_ERR_INVALID_ARG;
    if ((long long)n_frames * grid_h * grid_w > total_tokens) return TE_ERR_INVALID_ARG;
  } else {
    if (h->prefix_len > 0) return TE_ERR_UNSUPPORTED;  // (the cached-prefix passes take one grid per call)
    grid_h = grid_w = -1;
  }
  const int n_vis_min = grids == nullptr ? grid_h * grid_w : 0;
  TE_CUDA(h, cudaSetDevice(h->device));
  cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
  h->last_T = total_tokens;
  h->last_B = n_frames;
  const int Tb = bucket_tokens(total_tokens);

  cudaStreamCaptureStatus cap = cudaStreamCaptureStatusNone;
  if (st != nullptr) TE_CUDA(h, cudaStreamIsCapturing(st, &cap));
  int nk = 0;
  if (h->timing && cap != cudaStreamCaptureStatusNone) return TE_ERR_INVALID_ARG;
  if (h->l2_resid && h->l2_limit_bytes == 0 && cap == cudaStreamCaptureStatusNone) {
    // once per handle, outside any capture: reserve persisting L2 for the residual stream.  This is a DEVICE-WIDE
    // limit shared by all handles (l2_acquire); the value found before the first handle is restored when the last one
    // lets go (te_destroy, TE_OPT_L2_RESIDUAL = 0).
    size_t want = (size_t)h->cap_rows * c.hidden * sizeof(float);
    if (want > (64u << 20)) want = 64u << 20;
    if (want > h->l2_max_persist) want = h->l2_max_persist;
    if (l2_acquire(h->device, want)) {
      h->l2_limit_bytes = want;
      h->l2_ref_held = true;
    } else {
      h->l2_resid = 0;
    }
  }
  // per-call pointers and token count: one tiny kernel ahead of the stack (stream-ordered, also under capture)
  TE_CUDA(h, set_dyn(h, embeds, text_lens, out, total_tokens, st, grids, embeds_bf16));
  if (!h->use_graph || h->timing || cap != cudaStreamCaptureStatusNone) {
    int rc = enqueue_stack(h, n_frames, grid_h, grid_w, Tb, st, &nk);
    if (rc == TE_OK) h->launches += nk + 1;
    return rc;
  }
  GraphKey key;
  memset(&key, 0, sizeof(key));
  key.n_frames = n_frames; key.grid_h = grid_h; key.grid_w = grid_w; key.bucket_tokens = Tb;
  key.lb = h->dbg_lb; key.le = h->dbg_le; key.stop = h->dbg_stop; key.prefix_len = h->prefix_len;
  GraphEntry* hit = nullptr;
  for (auto& e : h->cache)
    if (e.key == key) { hit = &e; break; }
  if (!hit) {
    // First call of this shape class: capture the kernel sequence once.
    TE_CUDA(h, cudaStreamBeginCapture(h->own_stream, cudaStreamCaptureModeThreadLocal));
    int rc = enqueue_stack(h, n_frames, grid_h, grid_w, Tb, h->own_stream, &nk);
    cudaGraph_t g = nullptr;
    cudaError_t e = cudaStreamEndCapture(h->own_stream, &g);
    if (rc != TE_OK) {
      if (g) cudaGraphDestroy(g);
      return rc;
    }
    if (e != cudaSuccess) {
      h->err = std::string("cudaStreamEndCapture: ") + cudaGetErrorString(e);
      return TE_ERR_CUDA;
    }
    cudaGraphExec_t ex = nullptr;
    e = cudaGraphInstantiate(&ex, g, 0);
    if (e != cudaSuccess) {
      cudaGraphDestroy(g);
      h->err = std::string("cudaGraphInstantiate: ") + cudaGetErrorString(e);
      return TE_ERR_CUDA;
    }
    ++h->captures;
    if (h->cache.size() >= 32) {  // evict the least recently used entry
      size_t victim = 0;
      for (size_t i = 1; i < h->cache.size(); ++i)
        if (h->cache[i].stamp < h->cache[victim].stamp) victim = i;
      cudaGraphExecDestroy(h->cache[victim].exec);
      cudaGraphDestroy(h->cache[victim].graph);
      h->cache.erase(h->cache.begin() + victim);
    }
    h->cache.push_back(GraphEntry{key, ex, g, nk, 0});
    hit = &h->cache.back();
  } else {
    h->last_plan = make_plan(h, Tb, n_frames, n_vis_min);
  }
  hit->stamp = ++h->stamp;
  TE_CUDA(h, cudaGraphLaunch(hit->exec, st));
  h->launches += hit->n_kernels + 1;
  return TE_OK;
}

int te_encode(te_handle* h, int32_t n_frames, int32_t grid_h, int32_t grid_w, const float* embeds,
              const int32_t* text_lens, int32_t total_tokens, float* out, void* cuda_stream) {
  return encode_impl(h, n_frames, nullptr, grid_h, grid_w, embeds, 0, text_lens, total_tokens, out, cuda_stream);
}

int te_encode_ex(te_handle* h, int32_t n_frames, const int32_t* grids, int32_t grid_h, int32_t grid_w, const void* embeds,
                 int32_t embeds_dtype, const int32_t* text_lens, int32_t total_tokens, float* out, void* cuda_stream) {
  if (embeds_dtype < 0 || embeds_dtype > 1) return TE_ERR_INVALID_ARG;
  return encode_impl(h, n_frames, grids, grid_h, grid_w, embeds, embeds_dtype, text_lens, total_tokens, out, cuda_stream);
}

int te_encode_prefix(te_handle* h, const float* prefix_embeds, int32_t prefix_len, float* prefix_out, void* cuda_stream) {
  if (!h) return TE_ERR_INVALID_ARG;
  if (!h->loaded) return TE_ERR_NOT_LOADED;
  const te_config& c = h->cfg;
  if (prefix_len < 0 || prefix_len > c.max_prefix_tokens) return TE_ERR_INVALID_ARG;
  cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
  free_graphs(h);  // captured graphs bake in the ids / attention variant of the previous prefix
  h->prefix_len = 0;
  if (prefix_len == 0) return TE_OK;
  if (!prefix_embeds || prefix_embeds == prefix_out) return TE_ERR_INVALID_ARG;
  cudaStreamCaptureStatus cap = cudaStreamCaptureStatusNone;
  if (st != nullptr) TE_CUDA(h, cudaStreamIsCapturing(st, &cap));
  if (cap != cudaStreamCaptureStatusNone || h->timing) return TE_ERR_INVALID_ARG;
  TE_CUDA(h, cudaSetDevice(h->device));
  TE_CUDA(h, cudaMemcpyAsync(h->prefix_lens, &prefix_len, sizeof(int32_t), cudaMemcpyHostToDevice, st));
  int nk = 0;
  // one text-only frame (no grid): ids t = h = w = 0..P-1; every layer's K/V is copied to the cache
  TE_CUDA(h, set_dyn(h, prefix_embeds, h->prefix_lens, prefix_out ? prefix_out : h->prefix_buf, prefix_len, st));
  int rc = enqueue_stack(h, 1, 0, 0, bucket_tokens(prefix_len), st, &nk, /*prefix_pass=*/true, prefix_len);
  if (rc != TE_OK) return rc;
  h->launches += nk + 1;
  // tensor maps over each layer's cached K|V rows: exactly prefix_len rows, so that rows past the prefix read as zero
  h->tm_prefix.resize(c.n_layers);
  const size_t n_kv = 2 * (size_t)c.n_kv_heads * c.head_dim;
  for (int l = 0; l < c.n_layers; ++l)
    if (!make_tmap(&h->tm_prefix[l], h->kv_prefix + (size_t)l * c.max_prefix_tokens * n_kv, prefix_len, n_kv, 64)) {
      h->err = "cuTensorMapEncodeTiled failed for a prefix K/V map";
      return TE_ERR_CUDA;
    }
  h->prefix_len = prefix_len;
  return TE_OK;
}

int te_encode_host_submit(te_handle* h, int32_t n_frames, int32_t grid_h, int32_t grid_w, const float* embeds_host,
                          const int32_t* text_lens_host, float* out_host, int32_t* slot_out) {
  if (!h || !embeds_host || !text_lens_host || !out_host || !slot_out) return TE_ERR_INVALID_ARG;
  if (!h->loaded) return TE_ERR_NOT_LOADED;
  const te_config& c = h->cfg;
  if (n_frames < 1 || n_frames > c.max_frames || grid_h < 1 || grid_w < 1) return TE_ERR_INVALID_ARG;
  long long T = 0;
  for (int b = 0; b < n_frames; ++b) {
    // the lengths are on the host here: what te_encode can only flag on the device is refused up front
    if (text_lens_host[b] < 0) return TE_ERR_INVALID_ARG;
    const long long sb = (long long)grid_h * grid_w + text_lens_host[b];
    if (sb > c.max_tokens_per_frame) return TE_ERR_INVALID_ARG;
    T += sb;
  }
  if (T < 1 || T > c.max_tokens) return TE_ERR_INVALID_ARG;
  TE_CUDA(h, cudaSetDevice(h->device));
  const int si = h->next_slot;
  te_handle::HostSlot& sl = h->slot[si];
  if (sl.busy) return TE_ERR_INVALID_ARG;  // both slots in flight: te_encode_host_wait first
  if (!h->h2d_stream) {
    TE_CUDA(h, cudaStreamCreateWithFlags(&h->h2d_stream, cudaStreamNonBlocking));
    TE_CUDA(h, cudaStreamCreateWithFlags(&h->d2h_stream, cudaStreamNonBlocking));
  }
  if (!sl.embeds) {
    TE_CUDA(h, cudaMalloc(reinterpret_cast<void**>(&sl.embeds), (size_t)c.max_tokens * c.hidden * sizeof(float)));
    TE_CUDA(h, cudaMalloc(reinterpret_cast<void**>(&sl.out), (size_t)c.max_tokens * c.hidden * sizeof(float)));
    TE_CUDA(h, cudaMalloc(reinterpret_cast<void**>(&sl.lens), (size_t)c.max_frames * sizeof(int32_t)));
    TE_CUDA(h, cudaEventCreateWithFlags(&sl.h2d_done, cudaEventDisableTiming));
    TE_CUDA(h, cudaEventCreateWithFlags(&sl.compute_done, cudaEventDisableTiming));
    TE_CUDA(h, cudaEventCreateWithFlags(&sl.d2h_done, cudaEventDisableTiming));
  }
  const size_t bytes = (size_t)T * c.hidden * sizeof(float);
  // stage 1: host -> device on the copy-in stream (the slot's previous batch was waited for, so its buffers are free)
  TE_CUDA(h, cudaMemcpyAsync(sl.lens, text_lens_host, n_frames * sizeof(int32_t), cudaMemcpyHostToDevice, h->h2d_stream));
  TE_CUDA(h, cudaMemcpyAsync(sl.embeds, embeds_host, bytes, cudaMemcpyHostToDevice, h->h2d_stream));
  TE_CUDA(h, cudaEventRecord(sl.h2d_done, h->h2d_stream));
  // stage 2: the stack on the compute stream (batches are serialised there: they share the workspace)
  TE_CUDA(h, cudaStreamWaitEvent(h->own_stream, sl.h2d_done, 0));
  int rc = te_encode(h, n_frames, grid_h, grid_w, sl.embeds, sl.lens, (int32_t)T, sl.out, h->own_stream);
  if (rc != TE_OK) return rc;
  TE_CUDA(h, cudaEventRecord(sl.compute_done, h->own_stream));
  // stage 3: device -> host on the copy-out stream
  TE_CUDA(h, cudaStreamWaitEvent(h->d2h_stream, sl.compute_done, 0));
  TE_CUDA(h, cudaMemcpyAsync(out_host, sl.out, bytes, cudaMemcpyDeviceToHost, h->d2h_stream));
  TE_CUDA(h, cudaEventRecord(sl.d2h_done, h->d2h_stream));
  sl.busy = true;
  h->next_slot = si ^ 1;
  *slot_out = si;
  return TE_OK;
}

int te_encode_host_wait(te_handle* h, int32_t slot) {
  if (!h || slot < 0 || slot > 1 || !h->slot[slot].busy) return TE_ERR_INVALID_ARG;
  TE_CUDA(h, cudaEventSynchronize(h->slot[slot].d2h_done));
  h->slot[slot].busy = false;
  return TE_OK;
}

int te_encode_host(te_handle* h, int32_t n_frames, int32_t grid_h, int32_t grid_w, const float* embeds_host,
                   const int32_t* text_lens_host, float* out_host) {
  int32_t slot = 0;
  int rc = te_encode_host_submit(h, n_frames, grid_h, grid_w, embeds_host, text_lens_host, out_host, &slot);
  if (rc != TE_OK) return rc;
  return te_encode_host_wait(h, slot);
}

int te_query_async_error(te_handle* h) {
  if (!h) return TE_ERR_INVALID_ARG;
  TE_CUDA(h, cudaSetDevice(h->device));
  TE_CUDA(h, cudaDeviceSynchronize());
  int32_t f = 0;
  TE_CUDA(h, cudaMemcpy(&f, h->flag, sizeof(f), cudaMemcpyDeviceToHost));
  if (f) {
    TE_CUDA(h, cudaMemset(h->flag, 0, sizeof(int32_t)));
    char buf[96];
    snprintf(buf, sizeof(buf), "device validation flag 0x%x (1=negative length, 2=sum!=total_tokens, 4=frame too long)", f);
    h->err = buf;
    return TE_ERR_DEVICE_CHECK;
  }
  return TE_OK;
}

int te_set_option(te_handle* h, int option, int value) {
  if (!h) return TE_ERR_INVALID_ARG;
  switch (option) {
    case TE_OPT_USE_GRAPH: h->use_graph = value ? 1 : 0; return TE_OK;
    case TE_OPT_KERNEL_TIMING: h->timing = value ? 1 : 0; return TE_OK;
    case TE_OPT_TRACE:
      if (value && !h->trace) {
        const size_t bytes = 5 * (size_t)h->sm_dev * te::TRACE_SLOTS * sizeof(unsigned long long);
        TE_CUDA(h, cudaMalloc(reinterpret_cast<void**>(&h->trace), bytes));
        TE_CUDA(h, cudaMemset(h->trace, 0, bytes));
      }
      h->trace_on = value ? 1 : 0;
      break;
    case TE_OPT_PDL: h->pdl = value ? 1 : 0; break;
    case TE_OPT_CTA_PAIR:
      if (value < 0 || value > 2) return TE_ERR_INVALID_ARG;
      h->pair_mode = value;
      break;
    case TE_OPT_ATTN_IMPL:
      if (value < 0 || value > 1) return TE_ERR_INVALID_ARG;
      h->attn_impl = value;
      break;
    case TE_OPT_L2_RESIDUAL:
      h->l2_resid = value ? 1 : 0;
      if (!value) {
        cudaSetDevice(h->device);
        cudaDeviceSynchronize();
        release_l2_limit(h);
      }
      break;
    case TE_OPT_RESID_WIDE:
      if (value < 0 || value > 16) return TE_ERR_INVALID_ARG;
      h->resid_wide = value;
      break;
    case TE_OPT_SPLIT_K:
      h->splitk = value ? 1 : 0;
      h->split_target = value > 1 ? value : 0;
      break;
    case TE_OPT_SM_BUDGET:
      if (value != 0 && (value < 16 || value > h->sm_dev)) return TE_ERR_INVALID_ARG;
      h->sm_count = value ? value : h->sm_dev;
      break;
    case TE_OPT_RESID_BLOCK_N:
      if ((value != 128 && value != 256) || h->cfg.hidden % value != 0) return TE_ERR_INVALID_ARG;
      h->bn_res = value;
      break;
    default: return TE_ERR_INVALID_ARG;
  }
  free_graphs(h);  // cached graphs bake the previous choice in
  return TE_OK;
}

int64_t te_kernel_launches(te_handle* h) { return h ? h->launches : 0; }
int64_t te_graph_captures(te_handle* h) { return h ? h->captures : 0; }

int te_dispatch_info(te_handle* h, char* buf, size_t n_bytes) {
  if (!h || !buf || n_bytes == 0) return TE_ERR_INVALID_ARG;
  if (h->last_T == 0) return TE_ERR_INVALID_ARG;
  h->info = describe_plan(h, h->last_plan);
  snprintf(buf, n_bytes, "%s", h->info.c_str());
  return TE_OK;
}

int te_kernel_times(te_handle* h, float* ms_sum, int32_t* n_launches) {
  if (!h || !ms_sum || !n_launches) return TE_ERR_INVALID_ARG;
  TE_CUDA(h, cudaSetDevice(h->device));
  TE_CUDA(h, cudaDeviceSynchronize());
  for (int i = 0; i < TE_KCLASS_COUNT; ++i) { ms_sum[i] = 0.f; n_launches[i] = 0; }
  for (auto& t : h->timed) {
    float ms = 0.f;
    if (cudaEventElapsedTime(&ms, t.a, t.b) == cudaSuccess) {
      ms_sum[t.kclass] += ms;
      n_launches[t.kclass] += 1;
    }
    cudaEventDestroy(t.a);
    cudaEventDestroy(t.b);
  }
  h->timed.clear();
  return TE_OK;
}

int te_debug_set_range(te_handle* h, int32_t layer_begin, int32_t layer_end, int32_t stop_after_attn) {
  if (!h) return TE_ERR_INVALID_ARG;
  if (layer_begin < 0 || layer_end > h->cfg.n_layers || layer_begin >= layer_end) return TE_ERR_INVALID_ARG;
  h->dbg_lb = layer_begin;
  h->dbg_le = layer_end;
  h->dbg_stop = stop_after_attn ? 1 : 0;
  return TE_OK;
}

int te_debug_tap(te_handle* h, int what, void* dst, size_t n_bytes) {
  if (!h || !dst) return TE_ERR_INVALID_ARG;
  const te_config& c = h->cfg;
  const size_t T = h->last_T, B = h->last_B;
  const void* src = nullptr;
  size_t need = 0;
  switch (what) {
    case TE_TAP_POS: src = h->pos; need = 3 * T * sizeof(int32_t); break;
    case TE_TAP_CU_SEQLENS: src = h->cu; need = (B + 1) * sizeof(int32_t); break;
    case TE_TAP_COS: src = h->cos_t; need = T * (c.head_dim / 2) * sizeof(float); break;
    case TE_TAP_SIN: src = h->sin_t; need = T * (c.head_dim / 2) * sizeof(float); break;
    case TE_TAP_QKV: src = h->qkv; need = T * (size_t)(c.n_q_heads + 2 * c.n_kv_heads) * c.head_dim * sizeof(bf16); break;
    case TE_TAP_ATTN: src = h->attn; need = T * (size_t)c.n_q_heads * c.head_dim * sizeof(bf16); break;
    case TE_TAP_ACT: src = h->act; need = T * (size_t)c.ffn * sizeof(bf16); break;
    case TE_TAP_ATTN8: src = h->attn8; need = T * (size_t)c.n_q_heads * c.head_dim; break;
    case TE_TAP_ACT8: src = h->act8; need = T * (size_t)c.ffn; break;
    case TE_TAP_SF_ATTN: src = h->sf_attn; need = (T + 127) / 128 * ((size_t)c.n_q_heads * c.head_dim / 128) * 512; break;
    case TE_TAP_SF_ACT: src = h->sf_act; need = (T + 127) / 128 * ((size_t)c.ffn / 128) * 512; break;
    case TE_TAP_TRACE:
      src = h->trace;
      need = 5 * (size_t)h->sm_dev * te::TRACE_SLOTS * sizeof(unsigned long long);
      if (!src) return TE_ERR_INVALID_ARG;
      break;
    default: return TE_ERR_INVALID_ARG;
  }
  if (T == 0 || n_bytes != need || !src) return TE_ERR_INVALID_ARG;
  TE_CUDA(h, cudaSetDevice(h->device));
  TE_CUDA(h, cudaDeviceSynchronize());
  TE_CUDA(h, cudaMemcpy(dst, src, need, cudaMemcpyDeviceToHost));
  return TE_OK;
}

static int debug_gemm_prologue(int device, const void* a, const void* b, float* cmat, int m, int n, int k, int* sm_count) {
  if (!a || !b || !cmat || m < 1 || n < 1 || k < 1) return TE_ERR_INVALID_ARG;
  if (k % 64 != 0) return TE_ERR_UNSUPPORTED;
  if (cudaSetDevice(device) != cudaSuccess) return TE_ERR_CUDA;
  cudaDeviceProp prop;
  if (cudaGetDeviceProperties(&prop, device) != cudaSuccess) return TE_ERR_CUDA;
  if (prop.major != 10) return TE_ERR_UNSUPPORTED;
  if (init_kernel_attrs() != cudaSuccess) return TE_ERR_CUDA;
  *sm_count = prop.multiProcessorCount;
  return TE_OK;
}

int te_debug_gemm(int device, const void* a, const void* b, float* cmat, int32_t m, int32_t n, int32_t k,
                  int32_t block_n, int32_t cta_pair) {
  int sms = 0;
  int rc = debug_gemm_prologue(device, a, b, cmat, m, n, k, &sms);
  if (rc != TE_OK) return rc;
  if ((block_n != 128 && block_n != 256) || n % block_n != 0) return TE_ERR_UNSUPPORTED;
  CUtensorMap ta, tb;
  if (!make_tmap(&ta, a, m, k, te::GEMM_BM) || !make_tmap(&tb, b, n, k, cta_pair ? block_n / 2 : block_n))
    return TE_ERR_CUDA;
  te::GemmParams p{};
  p.M = m; p.N = n; p.K = k; p.num_m_blk = (m + te::GEMM_BM - 1) / te::GEMM_BM; p.num_n_blk = n / block_n;
  p.c = cmat; p.ld_c = n;
  const LaunchCtx lc;  // plain launch: no PDL, no cooperative attribute, no L2 window
  cudaError_t e = launch_gemm_bn<te::EPI_PLAIN>(lc, block_n, cta_pair ? 1 : 0, 128, ta, tb, p, sms, nullptr);
  if (e == cudaSuccess) e = cudaDeviceSynchronize();
  return e == cudaSuccess ? TE_OK : TE_ERR_CUDA;
}

int te_debug_gemm_splitk(int device, const void* a, const void* b, float* cmat, int32_t m, int32_t n, int32_t k,
                         int32_t block_n, int32_t splits) {
  int sms = 0;
  int rc = debug_gemm_prologue(device, a, b, cmat, m, n, k, &sms);
  if (rc != TE_OK) return rc;
  if ((block_n != 128 && block_n != 256) || n % block_n != 0) return TE_ERR_UNSUPPORTED;
  if (splits < 1 || splits > te::GEMMK_MAX_SPLITS || splits > k / 64) return TE_ERR_INVALID_ARG;
  CUtensorMap ta, tb;
  if (!make_tmap(&ta, a, m, k, te::GEMM_BM) || !make_tmap(&tb, b, n, k, block_n)) return TE_ERR_CUDA;
  te::GemmParams p{};
  p.M = m; p.N = n; p.K = k; p.num_m_blk = (m + te::GEMM_BM - 1) / te::GEMM_BM; p.num_n_blk = n / block_n;
  p.c = cmat; p.ld_c = n; p.splits = splits;
  const size_t tiles = (size_t)p.num_m_blk * p.num_n_blk;
  // the group members spin on each other: the whole grid must be co-resident (one CTA per SM)
  if (tiles * splits > (size_t)sms) return TE_ERR_UNSUPPORTED;
  if (cudaMalloc(reinterpret_cast<void**>(&p.sk_scratch), tiles * splits * te::GEMM_BM * block_n * sizeof(float)) !=
      cudaSuccess)
    return TE_ERR_CUDA;
  if (cudaMalloc(reinterpret_cast<void**>(&p.sk_sem), 2 * tiles * sizeof(int)) != cudaSuccess) {
    cudaFree(p.sk_scratch);
    return TE_ERR_CUDA;
  }
  cudaMemset(p.sk_sem, 0, 2 * tiles * sizeof(int));
  const LaunchCtx lc;
  cudaError_t e = launch_gemmk_bn<te::EPI_PLAIN>(lc, block_n, 128, ta, tb, p, nullptr);
  if (e == cudaSuccess) e = cudaDeviceSynchronize();
  cudaFree(p.sk_scratch);
  cudaFree(p.sk_sem);
  return e == cudaSuccess ? TE_OK : TE_ERR_CUDA;
}

int te_debug_gemm_wide(int device, const void* a, const void* b, float* cmat, int32_t m, int32_t n, int32_t k,
                       int32_t n_tiles) {
  int sms = 0;
  int rc = debug_gemm_prologue(device, a, b, cmat, m, n, k, &sms);
  if (rc != TE_OK) return rc;
  if (n_tiles < 1 || n % 32 != 0) return TE_ERR_UNSUPPORTED;
  const int bn = (((n + n_tiles - 1) / n_tiles) + 31) / 32 * 32;  // tile width as chosen by the stack's dispatch
  const int num_m = (m + te::GEMM_BM - 1) / te::GEMM_BM;
  if (bn > 512 || ((num_m + 1) / 2) * n_tiles > sms / 2) return TE_ERR_UNSUPPORTED;  // one wave only
  CUtensorMap ta, tb;
  if (!make_tmap(&ta, a, m, k, te::GEMM_BM) || !make_tmap(&tb, b, n, k, bn / 4)) return TE_ERR_CUDA;
  te::GemmParams p{};
  p.M = m; p.N = n; p.K = k; p.num_m_blk = num_m; p.num_n_blk = n_tiles;
  p.c = cmat; p.ld_c = n;
  const LaunchCtx lc;
  cudaError_t e = launch_wide<te::EPI_PLAIN>(lc, ta, tb, p, n_tiles, bn, nullptr);
  if (e == cudaSuccess) e = cudaDeviceSynchronize();
  return e == cudaSuccess ? TE_OK : TE_ERR_CUDA;
}

int te_debug_mx_quantise(int device, const void* src_bf16, int32_t rows, int32_t k, void* codes, void* scales_tiled) {
  if (!src_bf16 || !codes || !scales_tiled || rows < 1 || k < 128 || k % 128 != 0) return TE_ERR_INVALID_ARG;
  if (cudaSetDevice(device) != cudaSuccess) return TE_ERR_CUDA;
  const long long blocks = (long long)rows * (k / 32);
  te::te_mx_quantise_bf16_kernel<<<(unsigned)((blocks + 255) / 256), 256>>>(
      static_cast<const bf16*>(src_bf16), static_cast<uint8_t*>(codes), static_cast<uint8_t*>(scales_tiled), rows, k, 128, 0);
  cudaError_t e = cudaGetLastError();
  if (e == cudaSuccess) e = cudaDeviceSynchronize();
  return e == cudaSuccess ? TE_OK : TE_ERR_CUDA;
}

static int debug_gemm_mx(int device, const void* a, const void* b, float* cmat, int32_t m, int32_t n, int32_t k,
                        int32_t block_n, bool fp4) {
  int sms = 0;
  int rc = debug_gemm_prologue(device, a, b, cmat, m, n, k, &sms);
  if (rc != TE_OK) return rc;
  if ((block_n != 128 && block_n != 256) || n % block_n != 0 || k % 128 != 0) return TE_ERR_UNSUPPORTED;
  const size_t m_pad = ((size_t)m + 255) / 256 * 256;
  uint8_t *a8 = nullptr, *b8 = nullptr, *sa = nullptr, *sb = nullptr;
  auto done = [&](int code) {
    for (void* q : {(void*)a8, (void*)b8, (void*)sa, (void*)sb})
      if (q) cudaFree(q);
    return code;
  };
  if (cudaMalloc(reinterpret_cast<void**>(&a8), m_pad * k) != cudaSuccess ||
      cudaMalloc(reinterpret_cast<void**>(&b8), (size_t)n * k / (fp4 ? 2 : 1)) != cudaSuccess ||
      cudaMalloc(reinterpret_cast<void**>(&sa), m_pad * k / 32) != cudaSuccess ||
      cudaMalloc(reinterpret_cast<void**>(&sb), (size_t)n * k / 32) != cudaSuccess)
    return done(TE_ERR_CUDA);
  cudaMemset(a8, 0, m_pad * k);
  cudaMemset(sa, 127, m_pad * k / 32);
  const long long ba = (long long)m * (k / 32), bb = (long long)n * (k / 32);
  te::te_mx_quantise_bf16_kernel<<<(unsigned)((ba + 255) / 256), 256>>>(static_cast<const bf16*>(a), a8, sa, m, k, 128, 0);
  if (fp4)
    te::te_mx_quantise_fp4_kernel<<<(unsigned)((bb + 255) / 256), 256>>>(static_cast<const bf16*>(b), b8, sb, n, k, 128, 0);
  else
    te::te_mx_quantise_bf16_kernel<<<(unsigned)((bb + 255) / 256), 256>>>(static_cast<const bf16*>(b), b8, sb, n, k, 128, 0);
  CUtensorMap ta, tb, tsa, tsb;
  if (!make_tmap_u8(&ta, a8, m_pad, k, te::GEMM_BM) ||
      !(fp4 ? make_tmap_u4(&tb, b8, n, k, block_n / 2) : make_tmap_u8(&tb, b8, n, k, block_n / 2)) ||
      !make_tmap_sf(&tsa, sa, m_pad * k / 32 / 512) || !make_tmap_sf(&tsb, sb, ((size_t)n + 127) / 128 * (k / 128)))
    return done(TE_ERR_CUDA);
  te::GemmParams p{};
  p.M = m; p.N = n; p.K = k; p.num_m_blk = (m + te::GEMM_BM - 1) / te::GEMM_BM; p.num_n_blk = n / block_n;
  p.c = cmat; p.ld_c = n;
  te::Gemm8Extra x8{};
  x8.b_fp4 = fp4 ? 1 : 0;
  const LaunchCtx lc;
  cudaError_t e = block_n == 256 ? launch_gemm8<256, te::EPI_PLAIN, 128>(lc, ta, tb, tsa, tsb, p, x8, sms, nullptr)
                                 : launch_gemm8<128, te::EPI_PLAIN, 128>(lc, ta, tb, tsa, tsb, p, x8, sms, nullptr);
  if (e == cudaSuccess) e = cudaDeviceSynchronize();
  return done(e == cudaSuccess ? TE_OK : TE_ERR_CUDA);
}

int te_debug_gemm_mxfp8(int device, const void* a, const void* b, float* cmat, int32_t m, int32_t n, int32_t k,
                        int32_t block_n) {
  return debug_gemm_mx(device, a, b, cmat, m, n, k, block_n, false);
}

int te_debug_gemm_mxfp4(int device, const void* a, const void* b, float* cmat, int32_t m, int32_t n, int32_t k,
                        int32_t block_n) {
  return debug_gemm_mx(device, a, b, cmat, m, n, k, block_n, true);
}

int te_debug_mx_quantise_fp4(int device, const void* src_bf16, int32_t rows, int32_t k, void* codes_packed, void* scales_tiled) {
  if (!src_bf16 || !codes_packed || !scales_tiled || rows < 1 || k < 128 || k % 128 != 0) return TE_ERR_INVALID_ARG;
  if (cudaSetDevice(device) != cudaSuccess) return TE_ERR_CUDA;
  const long long blocks = (long long)rows * (k / 32);
  te::te_mx_quantise_fp4_kernel<<<(unsigned)((blocks + 255) / 256), 256>>>(
      static_cast<const bf16*>(src_bf16), static_cast<uint8_t*>(codes_packed), static_cast<uint8_t*>(scales_tiled), rows, k, 128, 0);
  cudaError_t e = cudaGetLastError();
  if (e == cudaSuccess) e = cudaDeviceSynchronize();
  return e == cudaSuccess ? TE_OK : TE_ERR_CUDA;
}

// ---------------------------------------------------------------- vision-tower front end (NEXT-4)
static int vision_validate(const te_vision_config& v, te_config* tower_cfg) {
  if (v.patch < 1 || v.image_h < 1 || v.image_w < 1 || v.out_hidden < 1 || v.max_frames < 1) return TE_ERR_INVALID_ARG;
  if (v.image_h % (2 * v.patch) != 0 || v.image_w % (2 * v.patch) != 0) return TE_ERR_INVALID_ARG;
  const int gh = v.image_h / v.patch, gw = v.image_w / v.patch;
  if (gh * gw > 256) return TE_ERR_UNSUPPORTED;                       // one frame's patches = one attention frame
  if ((v.patch * v.patch * 3) % 64 != 0) return TE_ERR_UNSUPPORTED;   // K of the patch-embedding GEMM
  if (v.out_hidden % 128 != 0) return TE_ERR_UNSUPPORTED;
  te_config t = v.tower;
  t.max_frames = v.max_frames;
  t.max_tokens = v.max_frames * gh * gw;
  t.max_tokens_per_frame = gh * gw;
  t.final_norm = 1;
  t.non_causal = 1;
  t.max_prefix_tokens = 0;
  t.weight_dtype = 0;
  const int rc = validate_config(t);
  if (rc != TE_OK) return rc;
  if (t.hidden % 128 != 0) return TE_ERR_UNSUPPORTED;
  *tower_cfg = t;
  return TE_OK;
}

// C[M, N] fp32 = A[M, K] * B[N, K]^T on the stack's tcgen05 GEMM (plain epilogue); M is fixed per launch (no DynParams)
static cudaError_t vision_gemm(const CUtensorMap& ta, const CUtensorMap& tb, float* cmat, int m, int n, int k, int bn, int pair,
                               int sms, cudaStream_t st) {
  te::GemmParams p{};
  p.M = m; p.N = n; p.K = k; p.num_m_blk = (m + te::GEMM_BM - 1) / te::GEMM_BM; p.num_n_blk = n / bn;
  p.c = cmat; p.ld_c = n;
  const LaunchCtx lc;  // plain launches: these kernels do not take part in the stack's PDL chain
  return launch_gemm_bn<te::EPI_PLAIN>(lc, bn, pair, 128, ta, tb, p, sms, st);
}

size_t te_vision_blob_bytes(const te_vision_config* cfg) {
  te_config t;
  if (!cfg || vision_validate(*cfg, &t) != TE_OK) return 0;
  const size_t d_v = t.hidden, pd = (size_t)cfg->patch * cfg->patch * 3;
  return (d_v * pd + blob_elems(t) + (size_t)cfg->out_hidden * 4 * d_v) * sizeof(bf16);
}

int te_vision_create(const te_vision_config* cfg, int device, te_vision** out) {
  if (!cfg || !out) return TE_ERR_INVALID_ARG;
  *out = nullptr;
  te_config t;
  int rc = vision_validate(*cfg, &t);
  if (rc != TE_OK) return rc;
  te_handle* tower = nullptr;
  rc = te_create(&t, device, &tower);
  if (rc != TE_OK) return rc;
  te_vision* v = new te_vision();
  v->cfg = *cfg;
  v->cfg.tower = t;
  v->device = device;
  v->sm_count = tower->sm_count;
  v->tower = tower;
  v->gh = cfg->image_h / cfg->patch;
  v->gw = cfg->image_w / cfg->patch;
  v->n_vis = (v->gh / 2) * (v->gw / 2);
  v->patch_dim = cfg->patch * cfg->patch * 3;
  v->d_v = t.hidden;
  v->rows_pe = (cfg->max_frames * v->gh * v->gw + 255) / 256 * 256;
  v->rows_m = (cfg->max_frames * v->n_vis + 255) / 256 * 256;
  auto fail = [&](int code) {
    te_vision_destroy(v);
    return code;
  };
  const size_t d_v = v->d_v, pd = v->patch_dim, oh = cfg->out_hidden;
#define TE_VALLOC(ptr, bytes) \
  if (cudaMalloc(reinterpret_cast<void**>(&(ptr)), (bytes)) != cudaSuccess) return fail(TE_ERR_CUDA)
  TE_VALLOC(v->w_pe, d_v * pd * sizeof(bf16));
  TE_VALLOC(v->w_m, oh * 4 * d_v * sizeof(bf16));
  TE_VALLOC(v->a_pe, (size_t)v->rows_pe * pd * sizeof(bf16));
  TE_VALLOC(v->a_m, (size_t)v->rows_m * 4 * d_v * sizeof(bf16));
  TE_VALLOC(v->x0, (size_t)v->rows_pe * d_v * sizeof(float));
  TE_VALLOC(v->tower_out, (size_t)v->rows_pe * d_v * sizeof(float));
  TE_VALLOC(v->vis, (size_t)v->rows_m * oh * sizeof(float));
  TE_VALLOC(v->zero_lens, (size_t)cfg->max_frames * sizeof(int32_t));
#undef TE_VALLOC
  // rows past a call's patches are multiplied (never stored) by the tile-granular GEMMs: start them finite
  if (cudaMemset(v->a_pe, 0, (size_t)v->rows_pe * pd * sizeof(bf16)) != cudaSuccess ||
      cudaMemset(v->a_m, 0, (size_t)v->rows_m * 4 * d_v * sizeof(bf16)) != cudaSuccess ||
      cudaMemset(v->zero_lens, 0, (size_t)cfg->max_frames * sizeof(int32_t)) != cudaSuccess)
    return fail(TE_ERR_CUDA);
  // tile shapes of the two GEMMs: CTA pairs (256-row tiles) once there are >= 1024 rows, 256-wide tiles when N allows
  v->bn_pe = (d_v % 256 == 0) ? 256 : 128;
  v->bn_m = (oh % 256 == 0) ? 256 : 128;
  v->pair_pe = v->rows_pe >= 1024;
  v->pair_m = v->rows_m >= 1024;
  if (!make_tmap(&v->tmA_pe, v->a_pe, v->rows_pe, pd, te::GEMM_BM) || !make_tmap(&v->tmA_m, v->a_m, v->rows_m, 4 * d_v, te::GEMM_BM) ||
      !make_tmap(&v->tmB_pe, v->w_pe, d_v, pd, v->pair_pe ? v->bn_pe / 2 : v->bn_pe) ||
      !make_tmap(&v->tmB_m, v->w_m, oh, 4 * d_v, v->pair_m ? v->bn_m / 2 : v->bn_m))
    return fail(TE_ERR_CUDA);
  *out = v;
  return TE_OK;
}

int te_vision_load_weights(te_vision* v, const void* blob, size_t n_bytes) {
  if (!v || !blob) return TE_ERR_INVALID_ARG;
  if (n_bytes != te_vision_blob_bytes(&v->cfg)) return TE_ERR_BLOB_SIZE;
  TE_CUDA(v, cudaSetDevice(v->device));
  v->loaded = false;
  const size_t n_pe = (size_t)v->d_v * v->patch_dim, n_tower = blob_elems(v->cfg.tower);
  const size_t n_m = (size_t)v->cfg.out_hidden * 4 * v->d_v;
  const bf16* src = static_cast<const bf16*>(blob);
  TE_CUDA(v, cudaMemcpy(v->w_pe, src, n_pe * sizeof(bf16), cudaMemcpyDefault));
  const int rc = te_load_weights(v->tower, src + n_pe, n_tower * sizeof(bf16));
  if (rc != TE_OK) {
    v->err = std::string("tower: ") + v->tower->err;
    return rc;
  }
  TE_CUDA(v, cudaMemcpy(v->w_m, src + n_pe + n_tower, n_m * sizeof(bf16), cudaMemcpyDefault));
  v->loaded = true;
  return TE_OK;
}

int te_encode_image(te_vision* v, int32_t n_frames, const float* pixels, const int32_t* text_lens, float* embeds,
                    int32_t total_tokens, void* cuda_stream) {
  if (!v || !pixels || !embeds) return TE_ERR_INVALID_ARG;
  if (!v->loaded) return TE_ERR_NOT_LOADED;
  if (n_frames < 1 || n_frames > v->cfg.max_frames) return TE_ERR_INVALID_ARG;
  if ((long long)total_tokens < (long long)n_frames * v->n_vis) return TE_ERR_INVALID_ARG;  // the visual rows alone do not fit
  TE_CUDA(v, cudaSetDevice(v->device));
  cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
  const int gh = v->gh, gw = v->gw, d_v = v->d_v;
  const int n_patch = n_frames * gh * gw, n_merged = n_frames * v->n_vis;
  v->last_B = n_frames;
  // Q28: patches -> bf16 rows, x0 = patches * W_pe^T
  te::te_patchify_kernel<<<n_patch, 256, 0, st>>>(pixels, v->a_pe, v->cfg.image_h, v->cfg.image_w, v->cfg.patch, gh, gw);
  TE_CUDA(v, cudaGetLastError());
  TE_CUDA(v, vision_gemm(v->tmA_pe, v->tmB_pe, v->x0, n_patch, d_v, v->patch_dim, v->bn_pe, v->pair_pe, v->sm_count, st));
  // Q29: the tower = the stack over frames of gh*gw patches with no text, non-causal, ids (0, py, px), final norm
  const long long before = v->tower->launches;
  const int rc = te_encode(v->tower, n_frames, gh, gw, v->x0, v->zero_lens, n_patch, v->tower_out, st);
  if (rc != TE_OK) {
    v->err = std::string("tower: ") + v->tower->err;
    return rc;
  }
  // Q30: 2 x 2 neighbours side by side -> W_m -> the visual rows of the decoder's packed input
  te::te_merge2x2_kernel<<<n_merged, 256, 0, st>>>(v->tower_out, v->a_m, gh, gw, d_v);
  TE_CUDA(v, cudaGetLastError());
  TE_CUDA(v, vision_gemm(v->tmA_m, v->tmB_m, v->vis, n_merged, v->cfg.out_hidden, 4 * d_v, v->bn_m, v->pair_m, v->sm_count, st));
  te::te_scatter_visual_kernel<<<n_merged, 256, 0, st>>>(v->vis, embeds, text_lens, v->n_vis, v->cfg.out_hidden, n_frames,
                                                         total_tokens, v->tower->flag);
  TE_CUDA(v, cudaGetLastError());
  v->launches += 5 + (v->tower->launches - before);
  return TE_OK;
}

int te_vision_query_async_error(te_vision* v) {
  if (!v) return TE_ERR_INVALID_ARG;
  const int rc = te_query_async_error(v->tower);  // the scatter raises the tower handle's flag
  if (rc != TE_OK) v->err = v->tower->err;
  return rc;
}

int64_t te_vision_kernel_launches(te_vision* v) { return v ? v->launches : 0; }
const char* te_vision_last_error(te_vision* v) { return v ? v->err.c_str() : ""; }
te_handle* te_vision_debug_tower(te_vision* v) { return v ? v->tower : nullptr; }

int te_vision_debug_tap(te_vision* v, int what, void* dst, size_t n_bytes) {
  if (!v || !dst || v->last_B == 0) return TE_ERR_INVALID_ARG;
  const size_t n_patch = (size_t)v->last_B * v->gh * v->gw, n_merged = (size_t)v->last_B * v->n_vis;
  const void* src = nullptr;
  size_t need = 0;
  switch (what) {
    case TE_VTAP_PATCH_EMBEDS: src = v->x0; need = n_patch * v->d_v * sizeof(float); break;
    case TE_VTAP_TOWER_OUT: src = v->tower_out; need = n_patch * v->d_v * sizeof(float); break;
    case TE_VTAP_MERGED: src = v->vis; need = n_merged * v->cfg.out_hidden * sizeof(float); break;
    default: return TE_ERR_INVALID_ARG;
  }
  if (n_bytes != need) return TE_ERR_INVALID_ARG;
  TE_CUDA(v, cudaSetDevice(v->device));
  TE_CUDA(v, cudaDeviceSynchronize());
  TE_CUDA(v, cudaMemcpy(dst, src, need, cudaMemcpyDeviceToHost));
  return TE_OK;
}

void te_vision_destroy(te_vision* v) {
  if (!v) return;
  cudaSetDevice(v->device);
  cudaDeviceSynchronize();
  if (v->tower) te_destroy(v->tower);
  void* ptrs[] = {v->w_pe, v->w_m, v->a_pe, v->a_m, v->x0, v->tower_out, v->vis, v->zero_lens};
  for (void* q : ptrs)
    if (q) cudaFree(q);
  delete v;
}

void te_destroy(te_handle* h) {
  if (!h) return;
  cudaSetDevice(h->device);
  cudaDeviceSynchronize();
  free_graphs(h);
  release_l2_limit(h);
  for (auto& t : h->timed) { cudaEventDestroy(t.a); cudaEventDestroy(t.b); }
  void* ptrs[] = {h->w, h->dyn, h->resid, h->cu, h->pos, h->flag, h->cos_t, h->sin_t, h->ssq, h->inv_freq, h->xg, h->qkv,
                  h->attn, h->act, h->slot[0].embeds, h->slot[0].out, h->slot[0].lens, h->slot[1].embeds, h->slot[1].out,
                  h->slot[1].lens, h->trace, h->sk_scratch, h->sk_sem, h->kv_prefix, h->prefix_buf, h->prefix_lens,
                  h->attn_stats, h->attn_o32, h->w8, h->sfw, h->xg8, h->attn8, h->act8, h->sf_xg, h->sf_attn, h->sf_act};
  for (void* p : ptrs)
    if (p) cudaFree(p);
  for (auto& sl : h->slot)
    for (cudaEvent_t e : {sl.h2d_done, sl.compute_done, sl.d2h_done})
      if (e) cudaEventDestroy(e);
  for (cudaStream_t st : {h->own_stream, h->h2d_stream, h->d2h_stream})
    if (st) cudaStreamDestroy(st);
  delete h;
}

}  // extern "C" (reopened below: the scratch array and its bookkeeping have C++ linkage)

// ------------------------------------------------------------------------------------------------- te_matmul_noalloc
// The split-K scratch for callers that cannot allocate (include/te.h): a fixed array in the device image instead of a
// cudaMalloc'd buffer.  Layout: [0, TE_NOALLOC_SCRATCH_BYTES) fp32 partial tiles [tile][split][128][block_n], then
// NOALLOC_SEM_BYTES of int counters (two per tile: arrivals, departures).  Zero at module load; each GPU has its own copy.
// In HOST code the name `te_noalloc_pool` is only a handle for the runtime's symbol table — passing it (or its host
// address) to a kernel would hand the kernel a host pointer.  The device address comes from cudaGetSymbolAddress, asked
// once per device with that device current (noalloc_pool_of below).
namespace {
constexpr size_t NOALLOC_MAX_TILES = 256;  // >= any SM count: tiles <= tiles * splits <= SMs
constexpr size_t NOALLOC_SEM_BYTES = 2 * NOALLOC_MAX_TILES * sizeof(int);
constexpr int NOALLOC_MAX_DEVICES = 64;
}  // namespace
static __device__ __align__(256) unsigned char te_noalloc_pool[TE_NOALLOC_SCRATCH_BYTES + NOALLOC_SEM_BYTES];

namespace {
struct NoAllocDevice {
  bool ready = false;
  unsigned char* pool = nullptr;  // DEVICE address of te_noalloc_pool on this GPU
  int sm_count = 0;
};
NoAllocDevice g_noalloc_dev[NOALLOC_MAX_DEVICES];
std::mutex g_noalloc_mu;

// Per-device set-up, done by the first call for `device` (which is current): checks the architecture, opts the kernels
// into their dynamic shared-memory size and resolves the array's device address.  Nothing here allocates.
int noalloc_pool_of(int device, NoAllocDevice* out) {
  std::lock_guard<std::mutex> lock(g_noalloc_mu);
  NoAllocDevice& d = g_noalloc_dev[device];
  if (!d.ready) {
    int major = 0, sms = 0;
    if (cudaDeviceGetAttribute(&major, cudaDevAttrComputeCapabilityMajor, device) != cudaSuccess ||
        cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, device) != cudaSuccess)
      return TE_ERR_CUDA;
    if (major != 10) return TE_ERR_UNSUPPORTED;  // tcgen05 / TMEM kernel: sm_100 only, no fallback
    if (!get_encode_fn() || init_kernel_attrs() != cudaSuccess) return TE_ERR_CUDA;
    void* p = nullptr;
    if (cudaGetSymbolAddress(&p, te_noalloc_pool) != cudaSuccess || !p) return TE_ERR_CUDA;
    d.pool = static_cast<unsigned char*>(p);
    d.sm_count = sms;
    d.ready = true;
  }
  *out = d;
  return TE_OK;
}
}  // namespace

extern "C" {

int te_matmul_noalloc(int device, const void* a, const void* b, float* cmat, int32_t m, int32_t n, int32_t k,
                      int32_t block_n, int32_t splits, void* cuda_stream) {
  if (!a || !b || !cmat || m < 1 || n < 1 || k < 1 || device < 0 || device >= NOALLOC_MAX_DEVICES) return TE_ERR_INVALID_ARG;
  if (k % 64 != 0 || (block_n != 128 && block_n != 256) || n % block_n != 0) return TE_ERR_UNSUPPORTED;
  if (splits < 1 || splits > te::GEMMK_MAX_SPLITS || splits > k / 64) return TE_ERR_INVALID_ARG;
  const size_t num_m = ((size_t)m + te::GEMM_BM - 1) / te::GEMM_BM, num_n = (size_t)n / block_n;
  const size_t tiles = num_m * num_n;
  // size check first: it needs no device and must hold whatever the GPU is
  if (tiles > NOALLOC_MAX_TILES || tiles * splits * te::GEMM_BM * block_n * sizeof(float) > (size_t)TE_NOALLOC_SCRATCH_BYTES)
    return TE_ERR_TOO_LARGE;
  if (cudaSetDevice(device) != cudaSuccess) return TE_ERR_CUDA;
  NoAllocDevice dev;
  const int rc = noalloc_pool_of(device, &dev);
  if (rc != TE_OK) return rc;
  if (tiles * splits > (size_t)dev.sm_count) return TE_ERR_UNSUPPORTED;  // a group's CTAs wait for each other
  CUtensorMap ta, tb;
  if (!make_tmap(&ta, a, m, k, te::GEMM_BM) || !make_tmap(&tb, b, n, k, block_n)) return TE_ERR_CUDA;
  te::GemmParams p{};
  p.M = m; p.N = n; p.K = k; p.num_m_blk = (int)num_m; p.num_n_blk = (int)num_n;
  p.c = cmat; p.ld_c = n; p.splits = splits;
  p.sk_scratch = reinterpret_cast<float*>(dev.pool);
  p.sk_sem = reinterpret_cast<int*>(dev.pool + TE_NOALLOC_SCRATCH_BYTES);
  cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
  // The counters must start at zero.  A finished launch re-arms them itself, but the array outlives every call and an
  // aborted one (device fault, cooperative launch refused half-way) would leave them counting: clear them every time.
  if (cudaMemsetAsync(p.sk_sem, 0, NOALLOC_SEM_BYTES, st) != cudaSuccess) return TE_ERR_CUDA;
  const LaunchCtx lc;  // plain stream order (no programmatic overlap with the memset); cooperative when splits > 1
  return launch_gemmk_bn<te::EPI_PLAIN>(lc, block_n, 128, ta, tb, p, st) == cudaSuccess ? TE_OK : TE_ERR_CUDA;
}

const char* te_strerror(int code) {
  switch (code) {
    case TE_OK: return "ok";
    case TE_ERR_INVALID_ARG: return "invalid argument";
    case TE_ERR_NOT_LOADED: return "weights not loaded";
    case TE_ERR_BLOB_SIZE: return "weight blob has the wrong size";
    case TE_ERR_CUDA: return "CUDA error";
    case TE_ERR_UNSUPPORTED: return "unsupported configuration or device";
    case TE_ERR_DEVICE_CHECK: return "device-side validation failed";
    case TE_ERR_TOO_LARGE: return "problem needs more scratch memory than the library's built-in no-allocation array holds";
    default: return "unknown error";
  }
}

const char* te_last_error(te_handle* h) { return h ? h->err.c_str() : ""; }

}  // extern "C"
