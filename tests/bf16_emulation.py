"""bf16-rounding emulation of the oracle — TEST INFRASTRUCTURE (derives the parity floors; never a reference).

The CUDA path rounds the operands of every tensor-core contraction to bf16 and keeps everything else in fp32
(DESIGN.md §5): the normalised GEMM inputs bf16(x*g), q/k/v, the softmax probabilities P, the attention output and
the SwiGLU activation.  This module restates one layer with exactly those rounding points inserted between the
oracle's own fp64 pieces (oracle/te_oracle.py supplies every formula; nothing is re-derived here), so that the
distance emulation <-> oracle is the error a CORRECT bf16 implementation is expected to show.  The gates in
tests/parity_metrics.py are set from these floors (SURVEY.md §8c "Expected error level"), with >= 3x headroom.
"""
from __future__ import annotations

import numpy as np

import workloads as W
from oracle import te_oracle as O


def bf16_round(x: np.ndarray) -> np.ndarray:
    """fp64 -> nearest bf16 (via fp32, RNE) -> fp64."""
    return O.bf16_bits_to_f64(W.f32_to_bf16_bits(np.asarray(x, dtype=np.float32))).reshape(np.shape(x))


def layer_forward_bf16(x, Wl, phi, m):
    """oracle.layer_forward with the GPU's rounding points (one frame)."""
    S = x.shape[0]
    Hq, Hkv, dh = m.n_q_heads, m.n_kv_heads, m.head_dim
    G = Hq // Hkv
    rstd = 1.0 / np.sqrt(np.mean(x * x, axis=-1, keepdims=True) + m.rms_eps)
    xg = bf16_round(x * Wl["g1"])                                     # producer epilogue: bf16(x * g)
    q = ((xg @ Wl["Wq"].T) * rstd).reshape(S, Hq, dh)                  # consumer epilogue: * rstd
    k = ((xg @ Wl["Wk"].T) * rstd).reshape(S, Hkv, dh)
    v = bf16_round(((xg @ Wl["Wv"].T) * rstd).reshape(S, Hkv, dh))
    q = bf16_round(O.rope_apply(O.rmsnorm(q, Wl["gq"], m.rms_eps), phi))
    k = bf16_round(O.rope_apply(O.rmsnorm(k, Wl["gk"], m.rms_eps), phi))
    o = np.zeros_like(q)
    for a in range(Hq):
        kv = a // G
        for n in range(S):
            s = (k[: n + 1, kv, :] @ q[n, a, :]) / np.sqrt(np.float64(dh))
            p = np.exp(s - np.max(s))
            o[n, a, :] = (bf16_round(p) @ v[: n + 1, kv, :]) / np.sum(p)   # P rounded, row sum in fp32
    o = bf16_round(o)
    x = x + o.reshape(S, Hq * dh) @ Wl["Wo"].T
    rstd2 = 1.0 / np.sqrt(np.mean(x * x, axis=-1, keepdims=True) + m.rms_eps)
    xg2 = bf16_round(x * Wl["g2"])
    act = bf16_round(O.silu((xg2 @ Wl["Wgate"].T) * rstd2) * ((xg2 @ Wl["Wup"].T) * rstd2))
    return x + act @ Wl["Wdown"].T


def encode_bf16(blob, layout, m, embeds, text_lens, grid_h, grid_w, layer_begin=0, layer_end=None):
    cu = O.cu_seqlens(text_lens, grid_h, grid_w)
    phi = O.mrope_angles(O.position_ids(text_lens, grid_h, grid_w), m.head_dim, m.rope_sections, m.rope_theta)
    out = np.asarray(embeds, dtype=np.float64).copy()
    for l in range(layer_begin, m.n_layers if layer_end is None else layer_end):
        Wl = O.unpack_layer(blob, layout, l)
        for b in range(len(text_lens)):
            sl = slice(cu[b], cu[b + 1])
            out[sl] = layer_forward_bf16(out[sl], Wl, phi[sl], m)
    return out


# ------------------------------------------------------------------ MXFP8 variant
def layer_forward_bf16_mx(x, Wq, phi, m, jitter=None):
    """oracle.te_mxfp8.layer_forward_mxfp8 with the CUDA path's rounding points: q/k/v, P and the attention output
    pass through bf16-class rounding as in layer_forward_bf16; the three A operands are MXFP8-quantised from values
    that carry fp32-accumulation-class noise (`jitter`: relative perturbation applied before each quantiser, standing
    in for the last-bits difference between fp32 accumulation on the GPU and the oracle's fp64 — what flips E4M3
    codes at rounding boundaries)."""
    from oracle import te_mxfp8 as Q
    rng = np.random.default_rng(0) if jitter else None

    def jit(a):
        return a * (1.0 + jitter * rng.standard_normal(a.shape)) if jitter else a

    S = x.shape[0]
    Hq, Hkv, dh = m.n_q_heads, m.n_kv_heads, m.head_dim
    G = Hq // Hkv
    rstd = 1.0 / np.sqrt(np.mean(x * x, axis=-1, keepdims=True) + m.rms_eps)
    h = Q.fake_quant(jit(x * Wq["g1"]))
    q = ((h @ Wq["Wq"].T) * rstd).reshape(S, Hq, dh)
    k = ((h @ Wq["Wk"].T) * rstd).reshape(S, Hkv, dh)
    v = bf16_round(((h @ Wq["Wv"].T) * rstd).reshape(S, Hkv, dh))
    q = bf16_round(O.rope_apply(O.rmsnorm(q, Wq["gq"], m.rms_eps), phi))
    k = bf16_round(O.rope_apply(O.rmsnorm(k, Wq["gk"], m.rms_eps), phi))
    o = np.zeros_like(q)
    for a in range(Hq):
        kv = a // G
        for n in range(S):
            s = (k[: n + 1, kv, :] @ q[n, a, :]) / np.sqrt(np.float64(dh))
            p = np.exp(s - np.max(s))
            o[n, a, :] = (bf16_round(p) @ v[: n + 1, kv, :]) / np.sum(p)
    oq = Q.fake_quant(jit(o.reshape(S, Hq * dh)))
    x = x + oq @ Wq["Wo"].T
    rstd2 = 1.0 / np.sqrt(np.mean(x * x, axis=-1, keepdims=True) + m.rms_eps)
    h2 = Q.fake_quant(jit(x * Wq["g2"]))
    act = O.silu((h2 @ Wq["Wgate"].T) * rstd2) * ((h2 @ Wq["Wup"].T) * rstd2)
    return x + Q.fake_quant(jit(act)) @ Wq["Wdown"].T


def encode_bf16_mx(blob, layout, m, embeds, text_lens, grid_h, grid_w, layer_begin=0, layer_end=None, jitter=1e-6):
    from oracle import te_mxfp8 as Q
    cu = O.cu_seqlens(text_lens, grid_h, grid_w)
    phi = O.mrope_angles(O.position_ids(text_lens, grid_h, grid_w), m.head_dim, m.rope_sections, m.rope_theta)
    out = np.asarray(embeds, dtype=np.float64).copy()
    for l in range(layer_begin, m.n_layers if layer_end is None else layer_end):
        Wl = Q.quantise_layer_weights(O.unpack_layer(blob, layout, l))
        for b in range(len(text_lens)):
            sl = slice(cu[b], cu[b + 1])
            out[sl] = layer_forward_bf16_mx(out[sl], Wl, phi[sl], m, jitter)
    return out
