"""MXFP8 quantiser of the block-scaled TE variant.  TEST INFRASTRUCTURE ONLY
(same rules as oracle/te_oracle.py: only tests/, __graft_entry__.smoke() and bench.py's CPU legs may import it;
the product shares no code, table or constant with it).

What it states.  The paper names block-/tensor-scaled 8-bit formats on Blackwell only as the way forward for
its wide-range TE activations ("TensorRT FP16 with wide-range MLLM TE outputs" — std 37, max 1160
overflow FP16; PAPER.md:411 future work: FP8 scaling, MXFP4 attention on Blackwell).  It defines no scheme, so the
scheme is the readings Q24-Q27 of DESIGN.md §3:

  Q24  format = OCP Microscaling MXFP8: blocks of 32 consecutive elements along the contraction (K) axis share one
       E8M0 scale X = 2^(code-127); elements are FP8 E4M3 ("fn": bias 7, 3 mantissa bits, max normal 448 = 1.75*2^8,
       subnormal step 2^-9, no infinities; NaN never produced).
  Q25  scale rule: X is the SMALLEST power of two with amax/X <= 448 (so the quantiser never saturates):
       with amax = 1.m * 2^(E-127) as a float32,  code = clamp(E - 8 + [1.m > 1.75], 0, 254);  element =
       RNE_e4m3(v / X) — the division by a power of two is exact.  An all-zero block has code 0.
  Q26  what is quantised: the four weight matrices of a layer (per output row, along in_features) once at load,
       and the A operands of their GEMMs: x*g (the RMSNorm is factored, the 1/rms scale multiplies the GEMM output
       as in the bf16 path), the attention output, the SwiGLU activation.  q/k/v and the attention probabilities stay
       bf16-class (attention is not quantised), accumulation and the residual stream stay fp32.
  Q27  every quantiser decision (amax, code, rounding) is taken on float32 values, the kernel's precision: the
       oracle rounds its float64 value to float32 first and then applies the rule above exactly.

Plain numpy, element by element semantics (vectorised over blocks only); pinned by hand-worked values in
tests/test_mxfp8_pins.py.
"""
from __future__ import annotations

import numpy as np

BLOCK = 32
E4M3_MAX = 448.0


def e4m3_decode(code: np.ndarray) -> np.ndarray:
    """FP8 E4M3 (fn) bit pattern (uint8) -> float64, from the definition: sign s, exponent e (4 bits, bias 7),
    mantissa m (3 bits): e == 0 -> (-1)^s * m/8 * 2^-6;  else (-1)^s * (1 + m/8) * 2^(e-7).  (e=15, m=7 is NaN.)"""
    c = np.asarray(code, dtype=np.uint8).astype(np.int64)
    s = np.where(c & 0x80, -1.0, 1.0)
    e = (c >> 3) & 0xF
    m = (c & 0x7).astype(np.float64)
    val = np.where(e == 0, m / 8.0 * 2.0 ** -6, (1.0 + m / 8.0) * 2.0 ** (e.astype(np.float64) - 7.0))
    val = np.where((e == 15) & ((c & 0x7) == 7), np.nan, val)
    return s * val


# the 127 non-negative finite values in code order (codes 0x00 .. 0x7E), used as the rounding grid
_GRID = e4m3_decode(np.arange(0x7F, dtype=np.uint8))


def e4m3_encode_rne(v: np.ndarray) -> np.ndarray:
    """float -> nearest E4M3 code, ties to the even code (= even mantissa), |v| <= 448 assumed (Q25 guarantees it;
    larger magnitudes clamp to 448).  Nearest-value search over the grid: no bit tricks."""
    v = np.asarray(v, dtype=np.float64)
    a = np.minimum(np.abs(v), E4M3_MAX)
    hi = np.searchsorted(_GRID, a, side="left")          # first grid value >= a
    hi = np.clip(hi, 0, len(_GRID) - 1)
    lo = np.clip(hi - 1, 0, len(_GRID) - 1)
    d_lo, d_hi = a - _GRID[lo], _GRID[hi] - a
    pick_hi = (d_hi < d_lo) | ((d_hi == d_lo) & (hi % 2 == 0))
    code = np.where(pick_hi, hi, lo).astype(np.uint8)
    return np.where(np.signbit(v), code | 0x80, code).astype(np.uint8)


def e4m3_round(v: np.ndarray) -> np.ndarray:
    """float -> the nearest E4M3 VALUE (ties to even), |v| <= 448: the definition of rounding to a 3-bit mantissa —
    the grid step of the binade of |v| is 2^(floor(log2|v|) - 3), at least the subnormal step 2^-9, and np.rint
    rounds half to even.  Same function as e4m3_decode(e4m3_encode_rne(v)) (pinned), without the table search."""
    v = np.asarray(v, dtype=np.float64)
    a = np.minimum(np.abs(v), E4M3_MAX)
    _, e = np.frexp(a)                                     # a = f * 2^e, f in [0.5, 1)  ->  floor(log2 a) = e - 1
    step = np.ldexp(1.0, np.maximum(e - 1, -6) - 3)
    return np.copysign(np.rint(a / step) * step, v)


def scale_code(amax32: np.ndarray) -> np.ndarray:
    """Q25: E8M0 code of the block scale from the block's float32 amax."""
    bits = np.asarray(amax32, dtype=np.float32).view(np.uint32).astype(np.int64)
    E = (bits >> 23) & 0xFF
    mant = bits & 0x7FFFFF
    code = E - 8 + (mant > 0x600000)                      # 1.m > 1.75  <=>  mantissa field > 0.75 * 2^23
    return np.clip(code, 0, 254).astype(np.uint8)


def quantise(x: np.ndarray):
    """x: [..., K] (K % 32 == 0), any float dtype.  Returns (codes uint8 [..., K], scales uint8 [..., K/32])."""
    x32 = np.asarray(x, dtype=np.float32)                 # Q27: decisions on float32 values
    assert x32.shape[-1] % BLOCK == 0
    blk = x32.reshape(x32.shape[:-1] + (x32.shape[-1] // BLOCK, BLOCK))
    amax = np.max(np.abs(blk), axis=-1)
    sc = scale_code(amax)
    X = np.float64(2.0) ** (sc.astype(np.float64) - 127.0)
    codes = e4m3_encode_rne(blk.astype(np.float64) / X[..., None])
    return codes.reshape(x32.shape), sc


def dequantise(codes: np.ndarray, scales: np.ndarray) -> np.ndarray:
    """float64 values the block-scaled tensor cores see: e4m3 value * 2^(code-127)."""
    c = np.asarray(codes, dtype=np.uint8)
    blk = e4m3_decode(c).reshape(c.shape[:-1] + (c.shape[-1] // BLOCK, BLOCK))
    X = np.float64(2.0) ** (np.asarray(scales, dtype=np.uint8).astype(np.float64) - 127.0)
    return (blk * X[..., None]).reshape(c.shape)


def fake_quant(x: np.ndarray) -> np.ndarray:
    """dequantise(quantise(x)) -> float64 (what the quantised network computes with), evaluated on values
    (e4m3_round) instead of through the byte codes; identical by construction, pinned in tests/test_mxfp8_pins.py."""
    x32 = np.asarray(x, dtype=np.float32)
    blk = x32.reshape(x32.shape[:-1] + (x32.shape[-1] // BLOCK, BLOCK))
    X = np.float64(2.0) ** (scale_code(np.max(np.abs(blk), axis=-1)).astype(np.float64) - 127.0)
    return (e4m3_round(blk.astype(np.float64) / X[..., None]) * X[..., None]).reshape(x32.shape)


# ------------------------------------------------------------------ the quantised network (Q26)
def quantise_layer_weights(W: dict) -> dict:
    """The four GEMMs' matrices -> their dequantised MXFP8 values (per output row, blocks along in_features);
    gains unchanged."""
    out = dict(W)
    for name in ("Wq", "Wk", "Wv", "Wo", "Wgate", "Wup", "Wdown"):
        out[name] = fake_quant(W[name])
    return out


def layer_forward_mxfp8(x: np.ndarray, Wq: dict, phi: np.ndarray, m, taps: dict | None = None) -> np.ndarray:
    """One layer of the MXFP8 network for ONE frame: te_oracle.layer_forward with the
    quantisation points of Q26 written in; every other operation is te_oracle's own function.
    Wq: quantise_layer_weights(unpack_layer(...)).  x: [S, d] float64."""
    from . import te_oracle as O
    S = x.shape[0]
    Hq, Hkv, dh = m.n_q_heads, m.n_kv_heads, m.head_dim
    rstd = 1.0 / np.sqrt(np.mean(x * x, axis=-1, keepdims=True) + m.rms_eps)
    h = fake_quant(x * Wq["g1"])                                        # A operand of the QKV GEMM (no 1/rms yet)
    q = ((h @ Wq["Wq"].T) * rstd).reshape(S, Hq, dh)
    k = ((h @ Wq["Wk"].T) * rstd).reshape(S, Hkv, dh)
    v = ((h @ Wq["Wv"].T) * rstd).reshape(S, Hkv, dh)
    q = O.rope_apply(O.rmsnorm(q, Wq["gq"], m.rms_eps), phi)
    k = O.rope_apply(O.rmsnorm(k, Wq["gk"], m.rms_eps), phi)
    o = O.attention_causal_gqa(q, k, v)
    oq = fake_quant(o.reshape(S, Hq * dh))                              # A operand of the O projection
    x = x + oq @ Wq["Wo"].T
    rstd2 = 1.0 / np.sqrt(np.mean(x * x, axis=-1, keepdims=True) + m.rms_eps)
    h2 = fake_quant(x * Wq["g2"])                                       # A operand of the gate/up GEMM
    act = O.silu((h2 @ Wq["Wgate"].T) * rstd2) * ((h2 @ Wq["Wup"].T) * rstd2)
    aq = fake_quant(act)                                                # A operand of the down projection
    if taps is not None:
        taps.setdefault("q", []).append(q.reshape(S, -1))
        taps.setdefault("k", []).append(k.reshape(S, -1))
        taps.setdefault("v", []).append(v.reshape(S, -1))
        taps.setdefault("attn", []).append(oq)
        taps.setdefault("act", []).append(aq)
    return x + aq @ Wq["Wdown"].T


def encode_mxfp8(blob_bits, layout, m, embeds, text_lens, grid_h, grid_w, *, frames=None, layer_begin=0,
                 layer_end=None, taps=None, weights_cache: dict | None = None, fp4_weights: bool = False) -> np.ndarray:
    """te_encode of the MXFP8 network in float64 (positions, packing and angles are te_oracle's).
    fp4_weights: the weight matrices are MXFP4 instead (reading Q32; activations stay MXFP8).
    weights_cache (optional, plumbing only): {layer: quantised weights} kept between calls on the same blob as float32
    (dequantised MXFP8 values are exact in float32), so that several workloads share one pass of the quantiser."""
    from . import te_oracle as O
    text_lens = [int(t) for t in text_lens]
    cu = O.cu_seqlens(text_lens, grid_h, grid_w)
    phi = O.mrope_angles(O.position_ids(text_lens, grid_h, grid_w), m.head_dim, m.rope_sections, m.rope_theta,
                         bool(getattr(m, "rope_interleaved", False)))
    sel = list(range(len(text_lens))) if frames is None else list(frames)
    x = {b: np.asarray(embeds[cu[b]:cu[b + 1]], dtype=np.float64).copy() for b in sel}
    ftaps = {b: ({} if taps is not None else None) for b in sel}
    for l in range(layer_begin, m.n_layers if layer_end is None else layer_end):
        if weights_cache is not None and l in weights_cache:
            Wl = {k: v.astype(np.float64) for k, v in weights_cache[l].items()}
        else:
            Wl = (quantise_layer_weights_fp4 if fp4_weights else quantise_layer_weights)(O.unpack_layer(blob_bits, layout, l))
            if weights_cache is not None:
                weights_cache[l] = {k: v.astype(np.float32) for k, v in Wl.items()}
                assert all(np.array_equal(weights_cache[l][k].astype(np.float64), Wl[k]) for k in ("Wq", "g1"))
        for b in sel:
            x[b] = layer_forward_mxfp8(x[b], Wl, phi[cu[b]:cu[b + 1]], m, ftaps[b])
    if m.final_norm:
        off, shape = layout[("final", "gf")]
        gf = O.bf16_bits_to_f64(blob_bits[off:off + shape[0]])
        for b in sel:
            x[b] = O.rmsnorm(x[b], gf, m.rms_eps)
    out = np.full((int(cu[-1]), m.hidden), np.nan, dtype=np.float64)
    for b in sel:
        out[cu[b]:cu[b + 1]] = x[b]
    if taps is not None and frames is None:
        for key in ftaps[sel[0]]:
            taps[key] = [np.concatenate([ftaps[b][key][i] for b in sel], axis=0)
                         for i in range(len(ftaps[sel[0]][key]))]
    return out


# ====================================================================== MXFP4 weights (reading Q32)
# te_config.weight_dtype = 2: the four weight matrices of a layer are OCP MXFP4 — blocks of 32 consecutive in_features
# share one E8M0 scale, elements are FP4 E2M1 (1 sign, 2 exponent bits with bias 1, 1 mantissa bit: magnitudes
# 0, 0.5, 1, 1.5, 2, 3, 4, 6) — while the GEMMs' A operands stay MXFP8 exactly as above ("W4A8": the tensor core's
# kind::mxf8f6f4 multiplies E4M3 by E2M1 directly).  Scale rule as Q25 with the element maximum 6 = 1.5 * 2^2: X is the
# smallest power of two with amax / X <= 6:  code = clamp(E - 2 + [1.m > 1.5], 0, 254).  The paper names MXFP4 on
# Blackwell as future work and fixes nothing about it.
E2M1_MAX = 6.0
_GRID4 = np.asarray([0.0, 0.5, 1.0, 1.5, 2.0, 3.0, 4.0, 6.0])   # magnitudes in code order (codes 0 .. 7)


def e2m1_decode(code: np.ndarray) -> np.ndarray:
    """FP4 E2M1 code (0 .. 15) -> float64 from the definition: s = bit 3, e = bits 2:1 (bias 1), m = bit 0:
    e == 0 -> (-1)^s * m * 0.5;  else (-1)^s * (1 + m / 2) * 2^(e - 1)."""
    c = np.asarray(code, dtype=np.uint8).astype(np.int64)
    s = np.where(c & 0x8, -1.0, 1.0)
    e = (c >> 1) & 0x3
    m = (c & 0x1).astype(np.float64)
    return s * np.where(e == 0, 0.5 * m, (1.0 + 0.5 * m) * 2.0 ** (e.astype(np.float64) - 1.0))


def e2m1_encode_rne(v: np.ndarray) -> np.ndarray:
    """float -> nearest E2M1 code (0 .. 15), ties to the even code (even mantissa bit), |v| <= 6 assumed (larger
    magnitudes clamp to 6).  Nearest-value search over the eight magnitudes."""
    v = np.asarray(v, dtype=np.float64)
    a = np.minimum(np.abs(v), E2M1_MAX)
    hi = np.clip(np.searchsorted(_GRID4, a, side="left"), 0, 7)
    lo = np.clip(hi - 1, 0, 7)
    d_lo, d_hi = a - _GRID4[lo], _GRID4[hi] - a
    pick_hi = (d_hi < d_lo) | ((d_hi == d_lo) & (hi % 2 == 0))
    code = np.where(pick_hi, hi, lo).astype(np.uint8)
    return np.where(np.signbit(v), code | 0x8, code).astype(np.uint8)


def scale_code_fp4(amax32: np.ndarray) -> np.ndarray:
    """E8M0 code of an MXFP4 block from its float32 amax: smallest power of two X with amax / X <= 6."""
    bits = np.asarray(amax32, dtype=np.float32).view(np.uint32).astype(np.int64)
    E = (bits >> 23) & 0xFF
    mant = bits & 0x7FFFFF
    code = E - 2 + (mant > 0x400000)                      # 1.m > 1.5  <=>  mantissa field > 0.5 * 2^23
    return np.clip(code, 0, 254).astype(np.uint8)


def quantise_fp4(x: np.ndarray):
    """x: [..., K] (K % 32 == 0).  Returns (codes uint8 [..., K] with values 0 .. 15, scales uint8 [..., K/32])."""
    x32 = np.asarray(x, dtype=np.float32)
    assert x32.shape[-1] % BLOCK == 0
    blk = x32.reshape(x32.shape[:-1] + (x32.shape[-1] // BLOCK, BLOCK))
    sc = scale_code_fp4(np.max(np.abs(blk), axis=-1))
    X = np.float64(2.0) ** (sc.astype(np.float64) - 127.0)
    codes = e2m1_encode_rne(blk.astype(np.float64) / X[..., None])
    return codes.reshape(x32.shape), sc


def pack_fp4(codes: np.ndarray) -> np.ndarray:
    """[..., K] codes 0 .. 15 -> [..., K/2] bytes: element 2i in the low nibble, element 2i+1 in the high nibble."""
    c = np.asarray(codes, dtype=np.uint8)
    return (c[..., 0::2] | (c[..., 1::2] << 4)).astype(np.uint8)


def dequantise_fp4(codes: np.ndarray, scales: np.ndarray) -> np.ndarray:
    c = np.asarray(codes, dtype=np.uint8)
    blk = e2m1_decode(c).reshape(c.shape[:-1] + (c.shape[-1] // BLOCK, BLOCK))
    X = np.float64(2.0) ** (np.asarray(scales, dtype=np.uint8).astype(np.float64) - 127.0)
    return (blk * X[..., None]).reshape(c.shape)


def e2m1_round(v: np.ndarray) -> np.ndarray:
    """float -> the nearest E2M1 VALUE (ties to even), |v| <= 6 (larger clamps): the grid step is 0.5 below 2, 1 in [2, 4)
    and 2 in [4, 6], and np.rint rounds half to even.  Same function as e2m1_decode(e2m1_encode_rne(v)) (pinned on every
    midpoint and a dense sweep), without the table search — the 28-layer oracle quantises 1.4 G weights."""
    v = np.asarray(v, dtype=np.float64)
    a = np.minimum(np.abs(v), E2M1_MAX)
    r = np.where(a < 2.0, np.rint(a * 2.0) / 2.0, np.where(a < 4.0, np.rint(a), np.rint(a / 2.0) * 2.0))
    return np.copysign(r, v)


def fake_quant_fp4(x: np.ndarray) -> np.ndarray:
    """dequantise_fp4(quantise_fp4(x)) -> float64, evaluated on values (e2m1_round); identical by construction, pinned."""
    x32 = np.asarray(x, dtype=np.float32)
    blk = x32.reshape(x32.shape[:-1] + (x32.shape[-1] // BLOCK, BLOCK))
    X = np.float64(2.0) ** (scale_code_fp4(np.max(np.abs(blk), axis=-1)).astype(np.float64) - 127.0)
    return (e2m1_round(blk.astype(np.float64) / X[..., None]) * X[..., None]).reshape(x32.shape)


def quantise_layer_weights_fp4(W: dict) -> dict:
    """The four GEMMs' matrices -> their dequantised MXFP4 values; gains unchanged."""
    out = dict(W)
    for name in ("Wq", "Wk", "Wv", "Wo", "Wgate", "Wup", "Wdown"):
        out[name] = fake_quant_fp4(W[name])
    return out
