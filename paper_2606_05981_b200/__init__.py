"""paper_2606_05981_b200 — Python binding of the B200-native batched-prefill text encoder.

Thin ctypes layer over the C ABI in include/te.h (same entry-point names; argument
marshalling only — every step of the hot path runs in the CUDA kernels of libte_b200.so).
PyTorch appears only as the owner of device memory / streams handed in by the caller.
There is no CPU fallback: if the shared library is missing or the device is not sm_100 the
calls raise.
"""
from __future__ import annotations

import ctypes
import os
from ctypes import (POINTER, Structure, byref, c_char_p, c_double, c_float, c_int, c_int32, c_int64,
                    c_size_t, c_void_p)

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libte_b200.so")

TE_OK = 0
TE_ERR_INVALID_ARG, TE_ERR_NOT_LOADED, TE_ERR_BLOB_SIZE = -1, -2, -3
TE_ERR_CUDA, TE_ERR_UNSUPPORTED, TE_ERR_DEVICE_CHECK = -4, -5, -6
TE_ERR_TOO_LARGE = -7
TE_NOALLOC_SCRATCH_BYTES = 8 << 20   # include/te.h: partial-tile capacity of te_matmul_noalloc's built-in array
TE_OPT_USE_GRAPH = 0
TE_OPT_KERNEL_TIMING = 1
TE_OPT_CTA_PAIR = 2
TE_OPT_RESID_BLOCK_N = 3
TE_OPT_PDL = 4
TE_OPT_TRACE = 5
TE_OPT_ATTN_IMPL = 6
TE_OPT_SPLIT_K = 7
TE_OPT_RESID_WIDE = 9
TE_OPT_L2_RESIDUAL = 10
TE_OPT_SM_BUDGET = 14
TE_KCLASS_NAMES = ["scan", "prep", "qkv", "attn", "oproj", "gateup", "down", "final_norm"]
TE_TAP_POS, TE_TAP_CU_SEQLENS, TE_TAP_COS, TE_TAP_SIN, TE_TAP_QKV, TE_TAP_ATTN, TE_TAP_ACT, TE_TAP_TRACE = range(8)
TE_TAP_ATTN8, TE_TAP_ACT8, TE_TAP_SF_ATTN, TE_TAP_SF_ACT = 8, 9, 10, 11

# include/te.h (the product boundary) and include/te_debug.h (test-only taps and stand-alone GEMMs)
EXPORTS = [
    "te_blob_bytes", "te_create", "te_load_weights", "te_encode", "te_encode_ex", "te_encode_prefix", "te_encode_host",
    "te_encode_host_submit", "te_encode_host_wait", "te_query_async_error", "te_set_option", "te_kernel_launches",
    "te_graph_captures", "te_dispatch_info", "te_kernel_times", "te_destroy", "te_strerror", "te_last_error",
    "te_vision_blob_bytes", "te_vision_create", "te_vision_load_weights", "te_encode_image", "te_vision_kernel_launches",
    "te_vision_last_error", "te_vision_destroy", "te_matmul_noalloc", "te_vision_query_async_error",
]
DEBUG_EXPORTS = ["te_debug_set_range", "te_debug_tap", "te_debug_gemm", "te_debug_gemm_splitk", "te_debug_gemm_wide",
                 "te_debug_mx_quantise", "te_debug_gemm_mxfp8", "te_debug_mx_quantise_fp4", "te_debug_gemm_mxfp4", "te_vision_debug_tap", "te_vision_debug_tower"]
TE_VTAP_PATCH_EMBEDS, TE_VTAP_TOWER_OUT, TE_VTAP_MERGED = 0, 1, 2
TE_DTYPE_BF16, TE_DTYPE_MXFP8, TE_DTYPE_MXFP4 = 0, 1, 2


class TEConfig(Structure):
    """Mirror of `te_config` (include/te.h)."""
    _fields_ = [
        ("n_layers", c_int32), ("hidden", c_int32), ("n_q_heads", c_int32), ("n_kv_heads", c_int32),
        ("head_dim", c_int32), ("ffn", c_int32),
        ("rope_sec_t", c_int32), ("rope_sec_h", c_int32), ("rope_sec_w", c_int32),
        ("rms_eps", c_float), ("rope_theta", c_double),
        ("max_frames", c_int32), ("max_tokens", c_int32), ("max_tokens_per_frame", c_int32),
        ("final_norm", c_int32), ("rope_interleaved", c_int32), ("max_prefix_tokens", c_int32),
        ("weight_dtype", c_int32), ("non_causal", c_int32),
    ]


class TEVisionConfig(Structure):
    """Mirror of `te_vision_config` (include/te.h)."""
    _fields_ = [
        ("tower", TEConfig), ("patch", c_int32), ("image_h", c_int32), ("image_w", c_int32),
        ("out_hidden", c_int32), ("max_frames", c_int32),
    ]


class TEError(RuntimeError):
    def __init__(self, code: int, msg: str):
        super().__init__(f"te error {code}: {msg}")
        self.code = code


_lib_cache = None


def lib() -> ctypes.CDLL:
    """Load libte_b200.so (built in-tree by `python -m paper_2606_05981_b200.build`)."""
    global _lib_cache
    if _lib_cache is not None:
        return _lib_cache
    if not os.path.exists(LIB_PATH):
        raise RuntimeError(
            f"{LIB_PATH} not found: build it with `python -m paper_2606_05981_b200.build` "
            "(there is no CPU fallback)")
    L = ctypes.CDLL(LIB_PATH)
    L.te_blob_bytes.restype = c_size_t
    L.te_blob_bytes.argtypes = [POINTER(TEConfig)]
    L.te_create.restype = c_int
    L.te_create.argtypes = [POINTER(TEConfig), c_int, POINTER(c_void_p)]
    L.te_load_weights.restype = c_int
    L.te_load_weights.argtypes = [c_void_p, c_void_p, c_size_t]
    L.te_encode.restype = c_int
    L.te_encode.argtypes = [c_void_p, c_int32, c_int32, c_int32, c_void_p, c_void_p, c_int32, c_void_p, c_void_p]
    L.te_encode_ex.restype = c_int
    L.te_encode_ex.argtypes = [c_void_p, c_int32, c_void_p, c_int32, c_int32, c_void_p, c_int32, c_void_p, c_int32, c_void_p,
                               c_void_p]
    L.te_encode_prefix.restype = c_int
    L.te_encode_prefix.argtypes = [c_void_p, c_void_p, c_int32, c_void_p, c_void_p]
    L.te_encode_host.restype = c_int
    L.te_encode_host.argtypes = [c_void_p, c_int32, c_int32, c_int32, c_void_p, c_void_p, c_void_p]
    L.te_encode_host_submit.restype = c_int
    L.te_encode_host_submit.argtypes = [c_void_p, c_int32, c_int32, c_int32, c_void_p, c_void_p, c_void_p, c_void_p]
    L.te_encode_host_wait.restype = c_int
    L.te_encode_host_wait.argtypes = [c_void_p, c_int32]
    L.te_query_async_error.restype = c_int
    L.te_query_async_error.argtypes = [c_void_p]
    L.te_set_option.restype = c_int
    L.te_set_option.argtypes = [c_void_p, c_int, c_int]
    L.te_kernel_launches.restype = c_int64
    L.te_kernel_launches.argtypes = [c_void_p]
    L.te_graph_captures.restype = c_int64
    L.te_graph_captures.argtypes = [c_void_p]
    L.te_dispatch_info.restype = c_int
    L.te_dispatch_info.argtypes = [c_void_p, c_void_p, c_size_t]
    L.te_kernel_times.restype = c_int
    L.te_kernel_times.argtypes = [c_void_p, c_void_p, c_void_p]
    L.te_debug_set_range.restype = c_int
    L.te_debug_set_range.argtypes = [c_void_p, c_int32, c_int32, c_int32]
    L.te_debug_tap.restype = c_int
    L.te_debug_tap.argtypes = [c_void_p, c_int, c_void_p, c_size_t]
    L.te_debug_gemm.restype = c_int
    L.te_debug_gemm.argtypes = [c_int, c_void_p, c_void_p, c_void_p, c_int32, c_int32, c_int32, c_int32, c_int32]
    L.te_debug_gemm_splitk.restype = c_int
    L.te_debug_gemm_splitk.argtypes = [c_int, c_void_p, c_void_p, c_void_p, c_int32, c_int32, c_int32, c_int32, c_int32]
    L.te_matmul_noalloc.restype = c_int
    L.te_matmul_noalloc.argtypes = [c_int, c_void_p, c_void_p, c_void_p, c_int32, c_int32, c_int32, c_int32, c_int32, c_void_p]
    L.te_debug_gemm_wide.restype = c_int
    L.te_debug_gemm_wide.argtypes = [c_int, c_void_p, c_void_p, c_void_p, c_int32, c_int32, c_int32, c_int32]
    L.te_debug_mx_quantise.restype = c_int
    L.te_debug_mx_quantise.argtypes = [c_int, c_void_p, c_int32, c_int32, c_void_p, c_void_p]
    L.te_debug_gemm_mxfp8.restype = c_int
    L.te_debug_gemm_mxfp8.argtypes = [c_int, c_void_p, c_void_p, c_void_p, c_int32, c_int32, c_int32, c_int32]
    L.te_debug_mx_quantise_fp4.restype = c_int
    L.te_debug_mx_quantise_fp4.argtypes = [c_int, c_void_p, c_int32, c_int32, c_void_p, c_void_p]
    L.te_debug_gemm_mxfp4.restype = c_int
    L.te_debug_gemm_mxfp4.argtypes = [c_int, c_void_p, c_void_p, c_void_p, c_int32, c_int32, c_int32, c_int32]
    L.te_vision_blob_bytes.restype = c_size_t
    L.te_vision_blob_bytes.argtypes = [POINTER(TEVisionConfig)]
    L.te_vision_create.restype = c_int
    L.te_vision_create.argtypes = [POINTER(TEVisionConfig), c_int, POINTER(c_void_p)]
    L.te_vision_load_weights.restype = c_int
    L.te_vision_load_weights.argtypes = [c_void_p, c_void_p, c_size_t]
    L.te_encode_image.restype = c_int
    L.te_encode_image.argtypes = [c_void_p, c_int32, c_void_p, c_void_p, c_void_p, c_int32, c_void_p]
    L.te_vision_query_async_error.restype = c_int
    L.te_vision_query_async_error.argtypes = [c_void_p]
    L.te_vision_kernel_launches.restype = c_int64
    L.te_vision_kernel_launches.argtypes = [c_void_p]
    L.te_vision_last_error.restype = c_char_p
    L.te_vision_last_error.argtypes = [c_void_p]
    L.te_vision_destroy.restype = None
    L.te_vision_destroy.argtypes = [c_void_p]
    L.te_vision_debug_tap.restype = c_int
    L.te_vision_debug_tap.argtypes = [c_void_p, c_int, c_void_p, c_size_t]
    L.te_vision_debug_tower.restype = c_void_p
    L.te_vision_debug_tower.argtypes = [c_void_p]
    L.te_destroy.restype = None
    L.te_destroy.argtypes = [c_void_p]
    L.te_strerror.restype = c_char_p
    L.te_strerror.argtypes = [c_int]
    L.te_last_error.restype = c_char_p
    L.te_last_error.argtypes = [c_void_p]
    _lib_cache = L
    return L


def _ptr(x) -> int:
    """Raw address of a torch tensor / numpy array / int."""
    if x is None:
        return 0
    if isinstance(x, int):
        return x
    if hasattr(x, "data_ptr"):
        return int(x.data_ptr())
    if hasattr(x, "ctypes"):
        return int(x.ctypes.data)
    raise TypeError(f"cannot take the address of {type(x)}")


def _check(code: int, h=None):
    if code != TE_OK:
        L = lib()
        msg = L.te_strerror(code).decode()
        if h:
            extra = L.te_last_error(h).decode()
            if extra:
                msg += f" ({extra})"
        raise TEError(code, msg)


def make_config(model, max_frames: int, max_tokens: int, max_tokens_per_frame: int = 256,
                final_norm: int | None = None, max_prefix_tokens: int = 0, weight_dtype: int = 0,
                non_causal: int = 0) -> TEConfig:
    """TEConfig from a workloads.TEModelConfig-like object (duck-typed)."""
    s_t, s_h, s_w = model.rope_sections
    return TEConfig(model.n_layers, model.hidden, model.n_q_heads, model.n_kv_heads, model.head_dim,
                    model.ffn, s_t, s_h, s_w, model.rms_eps, model.rope_theta, max_frames, max_tokens,
                    max_tokens_per_frame, model.final_norm if final_norm is None else final_norm,
                    1 if getattr(model, "rope_interleaved", False) else 0, max_prefix_tokens, weight_dtype, non_causal)


def make_vision_config(vision, max_frames: int) -> TEVisionConfig:
    """TEVisionConfig from a workloads.VisionConfig-like object (duck-typed); the library sets the tower's capacities."""
    tower = make_config(vision.tower, max_frames, max_frames * vision.grid_h * vision.grid_w,
                        vision.grid_h * vision.grid_w, final_norm=1, non_causal=1)
    return TEVisionConfig(tower, vision.patch, vision.image_h, vision.image_w, vision.out_hidden, max_frames)


# ---------------------------------------------------------------- C-ABI names, marshalling only
def te_blob_bytes(cfg: TEConfig) -> int:
    return int(lib().te_blob_bytes(byref(cfg)))


def te_create(cfg: TEConfig, device: int = 0) -> c_void_p:
    h = c_void_p()
    _check(lib().te_create(byref(cfg), device, byref(h)))
    return h


def te_load_weights(h, blob, n_bytes: int | None = None):
    """blob: numpy uint16 array / torch tensor (host or device) holding bf16 bits."""
    if n_bytes is None:
        n_bytes = int(blob.nbytes) if hasattr(blob, "nbytes") else int(blob.numel() * blob.element_size())
    _check(lib().te_load_weights(h, _ptr(blob), n_bytes), h)


def te_encode(h, n_frames, grid_h, grid_w, embeds, text_lens, total_tokens, out, stream=None):
    """embeds/out: DEVICE fp32 [T, d]; text_lens: DEVICE int32 [B]; stream: cudaStream_t as int."""
    _check(lib().te_encode(h, n_frames, grid_h, grid_w, _ptr(embeds), _ptr(text_lens), total_tokens,
                           _ptr(out), _ptr(stream)), h)


def te_encode_ex(h, n_frames, grids, grid_h, grid_w, embeds, embeds_dtype, text_lens, total_tokens, out, stream=None):
    """grids: DEVICE int32 [B, 2] or None; embeds: DEVICE fp32 (embeds_dtype 0) or bf16 (1) [T, d]."""
    _check(lib().te_encode_ex(h, n_frames, _ptr(grids), grid_h, grid_w, _ptr(embeds), embeds_dtype, _ptr(text_lens),
                              total_tokens, _ptr(out), _ptr(stream)), h)


def te_encode_prefix(h, prefix_embeds, prefix_len, prefix_out=None, stream=None):
    """prefix_embeds / prefix_out: DEVICE fp32 [P, d] (prefix_out may be None)."""
    _check(lib().te_encode_prefix(h, _ptr(prefix_embeds), prefix_len, _ptr(prefix_out), _ptr(stream)), h)


def te_encode_host(h, n_frames, grid_h, grid_w, embeds_host, text_lens_host, out_host):
    _check(lib().te_encode_host(h, n_frames, grid_h, grid_w, _ptr(embeds_host), _ptr(text_lens_host),
                                _ptr(out_host)), h)


def te_encode_host_submit(h, n_frames, grid_h, grid_w, embeds_host, text_lens_host, out_host) -> int:
    slot = c_int32(-1)
    _check(lib().te_encode_host_submit(h, n_frames, grid_h, grid_w, _ptr(embeds_host), _ptr(text_lens_host),
                                       _ptr(out_host), byref(slot)), h)
    return int(slot.value)


def te_encode_host_wait(h, slot: int):
    _check(lib().te_encode_host_wait(h, slot), h)


def te_query_async_error(h) -> int:
    return int(lib().te_query_async_error(h))


def te_set_option(h, option: int, value: int):
    _check(lib().te_set_option(h, option, value), h)


def te_kernel_launches(h) -> int:
    return int(lib().te_kernel_launches(h))


def te_graph_captures(h) -> int:
    return int(lib().te_graph_captures(h))


def te_dispatch_info(h) -> dict:
    """{class: kernel name as a profiler prints it} of the last te_encode (+ "bucket_tokens")."""
    buf = ctypes.create_string_buffer(1024)
    _check(lib().te_dispatch_info(h, buf, 1024), h)
    return dict(kv.split("=", 1) for kv in buf.value.decode().split(";") if "=" in kv)


def te_kernel_times(h) -> dict:
    """{class name: (ms_sum, n_launches)} accumulated under TE_OPT_KERNEL_TIMING; resets."""
    n = len(TE_KCLASS_NAMES)
    ms = (c_float * n)()
    cnt = (c_int32 * n)()
    _check(lib().te_kernel_times(h, ms, cnt), h)
    return {TE_KCLASS_NAMES[i]: (float(ms[i]), int(cnt[i])) for i in range(n)}


def te_debug_set_range(h, layer_begin: int, layer_end: int, stop_after_attn: int = 0):
    _check(lib().te_debug_set_range(h, layer_begin, layer_end, stop_after_attn), h)


def te_debug_tap(h, what: int, dst_host):
    _check(lib().te_debug_tap(h, what, _ptr(dst_host), int(dst_host.nbytes)), h)


def te_debug_gemm(device, a_bf16, b_bf16, c, m, n, k, block_n=256, cta_pair=0):
    _check(lib().te_debug_gemm(device, _ptr(a_bf16), _ptr(b_bf16), _ptr(c), m, n, k, block_n, cta_pair))


def te_debug_gemm_splitk(device, a_bf16, b_bf16, c, m, n, k, block_n=128, splits=2):
    _check(lib().te_debug_gemm_splitk(device, _ptr(a_bf16), _ptr(b_bf16), _ptr(c), m, n, k, block_n, splits))


def te_matmul_noalloc(device, a_bf16, b_bf16, c, m, n, k, block_n=128, splits=2, stream=None):
    """c[m, n] (DEVICE fp32) = a[m, k] @ b[n, k]^T (DEVICE bf16) through the split-K kernel, with the kernel's scratch in
    the library's built-in device array: for callers that cannot call cudaMalloc (a frame loop that must not stall the
    GPU's other streams; a process whose memory pool already owns all of HBM).  Enqueues on `stream` (cudaStream_t as
    int, None = default stream) and returns without synchronising.  Raises TEError(TE_ERR_TOO_LARGE) when
    ceil(m/128) * (n/block_n) * splits * 128 * block_n * 4 bytes exceeds TE_NOALLOC_SCRATCH_BYTES.  All calls on one GPU
    share that array: do not let two of them overlap.  See include/te.h."""
    _check(lib().te_matmul_noalloc(device, _ptr(a_bf16), _ptr(b_bf16), _ptr(c), m, n, k, block_n, splits, _ptr(stream)))


def te_debug_mx_quantise(device, src_bf16, rows, k, codes, scales_tiled):
    _check(lib().te_debug_mx_quantise(device, _ptr(src_bf16), rows, k, _ptr(codes), _ptr(scales_tiled)))


def te_debug_gemm_mxfp8(device, a_bf16, b_bf16, c, m, n, k, block_n=256):
    _check(lib().te_debug_gemm_mxfp8(device, _ptr(a_bf16), _ptr(b_bf16), _ptr(c), m, n, k, block_n))


def te_debug_mx_quantise_fp4(device, src_bf16, rows, k, codes_packed, scales_tiled):
    _check(lib().te_debug_mx_quantise_fp4(device, _ptr(src_bf16), rows, k, _ptr(codes_packed), _ptr(scales_tiled)))


def te_debug_gemm_mxfp4(device, a_bf16, b_bf16, c, m, n, k, block_n=256):
    _check(lib().te_debug_gemm_mxfp4(device, _ptr(a_bf16), _ptr(b_bf16), _ptr(c), m, n, k, block_n))


def te_debug_gemm_wide(device, a_bf16, b_bf16, c, m, n, k, n_tiles):
    _check(lib().te_debug_gemm_wide(device, _ptr(a_bf16), _ptr(b_bf16), _ptr(c), m, n, k, n_tiles))


def te_destroy(h):
    lib().te_destroy(h)


def _vcheck(code: int, v=None):
    if code != TE_OK:
        L = lib()
        msg = L.te_strerror(code).decode()
        if v:
            extra = L.te_vision_last_error(v).decode()
            if extra:
                msg += f" ({extra})"
        raise TEError(code, msg)


def te_vision_blob_bytes(cfg: TEVisionConfig) -> int:
    return int(lib().te_vision_blob_bytes(byref(cfg)))


def te_vision_create(cfg: TEVisionConfig, device: int = 0) -> c_void_p:
    v = c_void_p()
    _vcheck(lib().te_vision_create(byref(cfg), device, byref(v)))
    return v


def te_vision_load_weights(v, blob, n_bytes: int | None = None):
    if n_bytes is None:
        n_bytes = int(blob.nbytes) if hasattr(blob, "nbytes") else int(blob.numel() * blob.element_size())
    _vcheck(lib().te_vision_load_weights(v, _ptr(blob), n_bytes), v)


def te_encode_image(v, n_frames, pixels, text_lens, embeds, stream=None, total_tokens: int | None = None):
    """pixels: DEVICE fp32 [B, H, W, 3]; text_lens: DEVICE int32 [B] or None; embeds: DEVICE fp32 [T, out_hidden];
    total_tokens: rows of `embeds` (default: embeds.shape[0]) — no row past it is written whatever text_lens holds."""
    if total_tokens is None:
        total_tokens = int(embeds.shape[0])
    _vcheck(lib().te_encode_image(v, n_frames, _ptr(pixels), _ptr(text_lens), _ptr(embeds), total_tokens, _ptr(stream)), v)


def te_vision_query_async_error(v) -> int:
    """Synchronises; returns TE_OK or TE_ERR_DEVICE_CHECK (no raise: the caller decides)."""
    return int(lib().te_vision_query_async_error(v))


def te_vision_kernel_launches(v) -> int:
    return int(lib().te_vision_kernel_launches(v))


def te_vision_last_error(v) -> str:
    return lib().te_vision_last_error(v).decode()


def te_vision_debug_tap(v, what: int, dst_host):
    _vcheck(lib().te_vision_debug_tap(v, what, _ptr(dst_host), int(dst_host.nbytes)), v)


def te_vision_debug_tower(v) -> c_void_p:
    return c_void_p(lib().te_vision_debug_tower(v))


def te_vision_destroy(v):
    lib().te_vision_destroy(v)


def te_strerror(code: int) -> str:
    return lib().te_strerror(code).decode()


def te_last_error(h) -> str:
    return lib().te_last_error(h).decode()


class TextEncoder:
    """Convenience owner of a handle (create -> load -> encode -> destroy)."""

    def __init__(self, model, max_frames: int, max_tokens: int, device: int = 0,
                 max_tokens_per_frame: int = 256, final_norm: int | None = None, max_prefix_tokens: int = 0,
                 weight_dtype: int = 0, non_causal: int = 0):
        self.model = model
        self.cfg = make_config(model, max_frames, max_tokens, max_tokens_per_frame, final_norm, max_prefix_tokens,
                               weight_dtype, non_causal)
        self.h = te_create(self.cfg, device)

    def load_weights(self, blob):
        te_load_weights(self.h, blob)

    def encode(self, n_frames, grid_h, grid_w, embeds, text_lens, total_tokens, out, stream=None):
        te_encode(self.h, n_frames, grid_h, grid_w, embeds, text_lens, total_tokens, out, stream)

    def encode_ex(self, n_frames, grids, grid_h, grid_w, embeds, embeds_dtype, text_lens, total_tokens, out, stream=None):
        te_encode_ex(self.h, n_frames, grids, grid_h, grid_w, embeds, embeds_dtype, text_lens, total_tokens, out, stream)

    def encode_prefix(self, prefix_embeds, prefix_len, prefix_out=None, stream=None):
        te_encode_prefix(self.h, prefix_embeds, prefix_len, prefix_out, stream)

    def encode_host(self, n_frames, grid_h, grid_w, embeds_host, text_lens_host, out_host):
        te_encode_host(self.h, n_frames, grid_h, grid_w, embeds_host, text_lens_host, out_host)

    def encode_host_submit(self, n_frames, grid_h, grid_w, embeds_host, text_lens_host, out_host) -> int:
        return te_encode_host_submit(self.h, n_frames, grid_h, grid_w, embeds_host, text_lens_host, out_host)

    def encode_host_wait(self, slot: int):
        te_encode_host_wait(self.h, slot)

    def close(self):
        if self.h:
            te_destroy(self.h)
            self.h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


class VisionEncoder:
    """Convenience owner of a vision front end (create -> load -> encode_image -> destroy)."""

    def __init__(self, vision, max_frames: int, device: int = 0):
        self.vision = vision
        self.cfg = make_vision_config(vision, max_frames)
        self.v = te_vision_create(self.cfg, device)

    def load_weights(self, blob):
        te_vision_load_weights(self.v, blob)

    def encode_image(self, n_frames, pixels, text_lens, embeds, stream=None, total_tokens=None):
        te_encode_image(self.v, n_frames, pixels, text_lens, embeds, stream, total_tokens)

    def query_async_error(self) -> int:
        return te_vision_query_async_error(self.v)

    def close(self):
        if self.v:
            te_vision_destroy(self.v)
            self.v = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass
