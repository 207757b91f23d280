"""Helpers for the `-m gpu` parity tests: run the CUDA path through the C-ABI binding and the
fp64 oracle on the same seeded inputs (workloads/), and return both for comparison."""
from __future__ import annotations

import functools

import numpy as np

import workloads as W


def bf16_bits_to_f64(bits):
    u = np.ascontiguousarray(bits, dtype=np.uint16).astype(np.uint32) << np.uint32(16)
    return u.view(np.float32).astype(np.float64)


@functools.lru_cache(maxsize=4)
def cached_blob(model, seed, gains="randn"):
    return W.make_weight_blob(model, seed, gains=gains)


class GpuTE:
    """Owns one handle; encode() returns numpy arrays."""

    def __init__(self, model, max_frames, max_tokens, blob, final_norm=None, cta_pair=None, resid_bn=None,
                 split_k=None, max_prefix_tokens=0, attn_impl=None, resid_wide=None, weight_dtype=0, non_causal=0):
        import torch
        import paper_2606_05981_b200 as te
        self.te, self.torch, self.model = te, torch, model
        self.weight_dtype = weight_dtype
        self.enc = te.TextEncoder(model, max_frames, max_tokens, final_norm=final_norm,
                                  max_prefix_tokens=max_prefix_tokens, weight_dtype=weight_dtype, non_causal=non_causal)
        self.enc.load_weights(blob)
        if cta_pair is not None:
            te.te_set_option(self.enc.h, te.TE_OPT_CTA_PAIR, cta_pair)
        if resid_bn is not None:
            te.te_set_option(self.enc.h, te.TE_OPT_RESID_BLOCK_N, resid_bn)
        if split_k is not None:
            te.te_set_option(self.enc.h, te.TE_OPT_SPLIT_K, split_k)
        if resid_wide is not None:
            te.te_set_option(self.enc.h, te.TE_OPT_RESID_WIDE, resid_wide)
        if attn_impl is not None:
            te.te_set_option(self.enc.h, te.TE_OPT_ATTN_IMPL, attn_impl)

    def encode(self, embeds, text_lens, gh, gw, layer_range=None, stop_after_attn=0, stream=None,
               total_tokens=None, use_graph=1):
        torch, te = self.torch, self.te
        T = embeds.shape[0] if total_tokens is None else total_tokens
        e = torch.from_numpy(np.ascontiguousarray(embeds, dtype=np.float32)).cuda()
        tl = torch.from_numpy(np.ascontiguousarray(text_lens, dtype=np.int32)).cuda()
        out = torch.empty_like(e)
        lb, le = (0, self.model.n_layers) if layer_range is None else layer_range
        te.te_debug_set_range(self.enc.h, lb, le, stop_after_attn)
        te.te_set_option(self.enc.h, te.TE_OPT_USE_GRAPH, use_graph)
        self.enc.encode(len(text_lens), gh, gw, e, tl, T, out, stream)
        torch.cuda.synchronize()
        self._keep = (e, tl, out)
        return out.cpu().numpy()

    def encode_prefix(self, prefix_embeds, want_out=True):
        """te_encode_prefix: caches the prefix K/V in the handle; returns the prefix hidden states."""
        torch = self.torch
        P = int(prefix_embeds.shape[0])
        if P == 0:
            self.enc.encode_prefix(None, 0)
            return None
        e = torch.from_numpy(np.ascontiguousarray(prefix_embeds, dtype=np.float32)).cuda()
        out = torch.empty_like(e) if want_out else None
        self.enc.encode_prefix(e, P, out)
        torch.cuda.synchronize()
        return out.cpu().numpy() if want_out else None

    def tap(self, what, shape, dtype):
        buf = np.empty(shape, dtype=dtype)
        self.te.te_debug_tap(self.enc.h, what, buf)
        return buf

    def taps(self, T, B):
        m, te = self.model, self.te
        nqkv = (m.n_q_heads + 2 * m.n_kv_heads) * m.head_dim
        nq = m.n_q_heads * m.head_dim
        nk = m.n_kv_heads * m.head_dim
        qkv = bf16_bits_to_f64(self.tap(te.TE_TAP_QKV, (T, nqkv), np.uint16))
        return {
            "pos": self.tap(te.TE_TAP_POS, (3, T), np.int32),
            "cu_seqlens": self.tap(te.TE_TAP_CU_SEQLENS, (B + 1,), np.int32),
            "cos": self.tap(te.TE_TAP_COS, (T, m.head_dim // 2), np.float32),
            "sin": self.tap(te.TE_TAP_SIN, (T, m.head_dim // 2), np.float32),
            "q": qkv[:, :nq], "k": qkv[:, nq:nq + nk], "v": qkv[:, nq + nk:],
            "attn": bf16_bits_to_f64(self.tap(te.TE_TAP_ATTN, (T, nq), np.uint16)),
            "act": bf16_bits_to_f64(self.tap(te.TE_TAP_ACT, (T, m.ffn), np.uint16)),
        }

    def taps_mx(self, T):
        """MXFP8 variant: q/k/v (bf16) and the dequantised attention / SwiGLU outputs (E4M3 codes x E8M0 scales)."""
        m, te = self.model, self.te
        nqkv = (m.n_q_heads + 2 * m.n_kv_heads) * m.head_dim
        nq = m.n_q_heads * m.head_dim
        nk = m.n_kv_heads * m.head_dim
        qkv = bf16_bits_to_f64(self.tap(te.TE_TAP_QKV, (T, nqkv), np.uint16))
        rb = (T + 127) // 128
        out = {"q": qkv[:, :nq], "k": qkv[:, nq:nq + nk], "v": qkv[:, nq + nk:]}
        for key, tap_c, tap_s, K in (("attn", te.TE_TAP_ATTN8, te.TE_TAP_SF_ATTN, nq), ("act", te.TE_TAP_ACT8, te.TE_TAP_SF_ACT, m.ffn)):
            codes = self.tap(tap_c, (T, K), np.uint8)
            sf = untile_scales(self.tap(tap_s, (rb, K // 128, 512), np.uint8), T, K)
            out[key] = mx_dequant(codes, sf)
        return out

    def close(self):
        self.enc.close()


def untile_scales(tiled, rows, K):
    """[ceil(rows/128), K/128, 512] in the tensor core's scale-copy order (include/te_debug.h) -> [rows, K/32]."""
    r = np.arange(rows)[:, None]
    b = np.arange(K // 32)[None, :]
    off = (r % 32) * 16 + ((r // 32) % 4) * 4 + b % 4
    return np.asarray(tiled)[r // 128, b // 4, off]


def mx_dequant(codes, scales):
    """E4M3 codes [rows, K] x 2^(scale-127) per 32-element block -> float64, decoded from the format definition
    (written out here: the GPU tests do not route the device's bytes through the oracle's decoder)."""
    c = np.asarray(codes, dtype=np.uint8).astype(np.int64)
    e, mnt = (c >> 3) & 0xF, (c & 7).astype(np.float64)
    mag = np.where(e == 0, mnt / 8.0 * 2.0 ** -6, (1.0 + mnt / 8.0) * 2.0 ** (e - 7.0))
    val = np.where(c & 0x80, -mag, mag)
    X = 2.0 ** (np.asarray(scales, dtype=np.uint8).astype(np.float64) - 127.0)
    return val * np.repeat(X, 32, axis=1)


def workload_inputs(cfg_id, outliers=None):
    w = W.get_workload(cfg_id)
    tl = W.make_text_lens(w)
    T = W.total_tokens(w, tl)
    emb = W.make_embeddings(w, T, outliers=outliers)
    blob = cached_blob(w.model, w.seed_weights)
    ch = W.gen.outlier_channels(w) if (outliers or w.outliers) != "none" else None
    return w, blob, tl, T, emb, ch
