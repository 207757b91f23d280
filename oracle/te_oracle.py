"""fp64 CPU oracle for the TE-prefill hot path.  TEST INFRASTRUCTURE ONLY.

Only `tests/`, `__graft_entry__.smoke()` and `bench.py`'s cpu_baseline /
`--impl reference` legs may import this file.  The product
(`paper_2606_05981_b200/`) never does, shares no code, table or constant with
it, and fails loudly when its CUDA library is missing.

What it computes.  The paper names the operation — TE(x, p) -> h,
the hidden states of a Qwen3-VL-2B-shaped decoder over visual + instruction tokens,
batched over frames (Table V :249-258), with the 3D rotary position ids
whose computation holds the CPU-GPU sync — but gives no equation for
the encoder.  The decoder's pieces and constants are fixed by BASELINE.json:configs, and
the open details are the readings Q1..Q21 of SURVEY.md §8(c) (restated in DESIGN.md §3).
The method is exact arithmetic on a fixed network, so the oracle is the plain definition,
evaluated in float64 on the same bf16-valued weights and fp32-valued embeddings the GPU
receives (both exactly representable), with no intermediate rounding, frame by frame,
in the order of SURVEY.md §8(c) steps 1-5.  A numpy float64 `@` is the only library
primitive used (a matmul as a step); there is no blocking, fusion or reordering.

Pins (tests/test_oracle_pins.py, `-m "not gpu"`): worked position-id values from
BASELINE.json:configs[0] (tests/golden/), omega closed forms, RoPE identity / norm
preservation / shift invariance, RMSNorm closed forms, attention running-mean and
causality, silu values, zero-projection pass-through, per-frame independence, a pure-Python
scalar brute force on a micro config, an independently written dense-mask restatement on
cfg 1, and a mutation suite (each plausible mistake must move the output beyond the gates).
Every function below is pinned by at least one of those; none is "parity unpinned".
"""
from __future__ import annotations

import numpy as np


# ----------------------------------------------------------------------------- inputs
def bf16_bits_to_f64(bits: np.ndarray) -> np.ndarray:
    """Decode bf16 bit patterns (uint16) exactly into float64.
    (`te_load_weights` takes bf16 weights — BASELINE.json:north_star.)"""
    u = np.ascontiguousarray(bits, dtype=np.uint16).astype(np.uint32) << np.uint32(16)
    return u.view(np.float32).astype(np.float64)


def unpack_layer(blob_bits: np.ndarray, layout: dict, layer: int) -> dict:
    """Slice one layer's tensors out of the canonical blob (SURVEY.md §8b layout) -> fp64."""
    out = {}
    for (l, name), (off, shape) in layout.items():
        if l == layer:
            n = int(np.prod(shape))
            out[name] = bf16_bits_to_f64(blob_bits[off:off + n]).reshape(shape)
    return out


# ------------------------------------------------------------- step 1-2: packing, position ids
def cu_seqlens(text_lens, grid_h: int, grid_w: int, prefix_len: int = 0) -> np.ndarray:
    """§8c step 1: S_b = prefix_len + gh*gw + text_len[b]; cu[0]=0, cu[b+1]=cu[b]+S_b.  int32.
    (prefix_len > 0: SURVEY §8(f) NEXT-1, the shared text prefix of PAPER.md:389.)"""
    cu = [0]
    for tl in text_lens:
        cu.append(cu[-1] + int(prefix_len) + grid_h * grid_w + int(tl))
    return np.asarray(cu, dtype=np.int32)


def position_ids(text_lens, grid_h: int, grid_w: int, prefix_len: int = 0) -> np.ndarray:
    """§8c step 2 (BASELINE.json:configs[0]: "4x4 grid (t=0) followed by 24 text tokens
    (positions continue from max grid id + 1)"): int32 [3, T], rows (t, h, w).
      visual token k in [0, gh*gw): (0, k // gw, k % gw)            (row-major, Q5)
      text token j in [0, text_len): t = h = w = max(gh, gw) + j    (Q4)
    This is the computation whose host round-trip the paper locates in the TE's rotary
    code.
    NEXT-1 (the real chat template puts an 80-token system prompt BEFORE the
    image): with a text prefix of P tokens per frame the same rule applies with
    every id continuing from the prefix (reading Q22): prefix token j: t=h=w=j;
    visual token k: (P, P + k // gw, P + k % gw); text token j: P + max(gh, gw) + j."""
    P = int(prefix_len)
    cols = []
    for tl in text_lens:
        for j in range(P):
            cols.append((j, j, j))
        for k in range(grid_h * grid_w):
            cols.append((P, P + k // grid_w, P + k % grid_w))
        start = P + max(grid_h, grid_w)
        for j in range(int(tl)):
            cols.append((start + j, start + j, start + j))
    return np.asarray(cols, dtype=np.int32).reshape(-1, 3).T.copy()


# ------------------------------------------------------------------- step 3: M-RoPE angles
def inv_freq(head_dim: int, theta: float) -> np.ndarray:
    """§8c step 3: omega_i = theta^(-2i/dh), i in [0, dh/2)."""
    i = np.arange(head_dim // 2, dtype=np.float64)
    return np.float64(theta) ** (-2.0 * i / np.float64(head_dim))


def rope_axis(head_dim: int, sections, interleaved: bool = False) -> np.ndarray:
    """§8c step 3 / Q1 (contiguous sections, t first): axis(i) = 0 (t) if i < s_t,
    1 (h) if s_t <= i < s_t + s_h, else 2 (w).
    NEXT-5 (SURVEY §8f, Q1 "keep axis(i) a table so the interleaved variant is a one-line
    change"): interleaved=True deals the frequency pairs round-robin t,h,w,t,h,w,... to the
    axes that still have pairs left in their section, so every axis keeps its section count
    but spans the whole frequency range (reading Q23)."""
    s_t, s_h, s_w = sections
    assert s_t + s_h + s_w == head_dim // 2
    if not interleaved:
        return np.asarray([0] * s_t + [1] * s_h + [2] * s_w, dtype=np.int64)
    left = [s_t, s_h, s_w]
    ax = []
    a = 0
    while len(ax) < head_dim // 2:
        if left[a] > 0:
            ax.append(a)
            left[a] -= 1
        a = (a + 1) % 3
    return np.asarray(ax, dtype=np.int64)


def mrope_angles(pos: np.ndarray, head_dim: int, sections, theta: float,
                 interleaved: bool = False) -> np.ndarray:
    """phi[n, i] = pos[axis(i), n] * omega_i   -> float64 [T, dh/2]."""
    om = inv_freq(head_dim, theta)
    ax = rope_axis(head_dim, sections, interleaved)
    return pos[ax, :].T.astype(np.float64) * om[None, :]


def rope_apply(u: np.ndarray, phi: np.ndarray) -> np.ndarray:
    """§8c step 4d, half-split pairing (Q2).  u: [S, H, dh], phi: [S, dh/2].
    (u_i, u_{i+dh/2}) <- (u_i cos - u_{i+dh/2} sin,  u_{i+dh/2} cos + u_i sin)."""
    half = u.shape[-1] // 2
    c = np.cos(phi)[:, None, :]
    s = np.sin(phi)[:, None, :]
    a, b = u[..., :half], u[..., half:]
    return np.concatenate([a * c - b * s, b * c + a * s], axis=-1)


# ------------------------------------------------------------------------ elementary pieces
def rmsnorm(x: np.ndarray, g: np.ndarray, eps: float) -> np.ndarray:
    """§8c step 4a / Q10: x * g / sqrt(mean(x^2) + eps) over the last axis."""
    ms = np.mean(x * x, axis=-1, keepdims=True)
    return x * g / np.sqrt(ms + eps)


def silu(z: np.ndarray) -> np.ndarray:
    """§8c step 4g: silu(z) = z / (1 + exp(-z))."""
    return z / (1.0 + np.exp(-z))


def attention_causal_gqa(q: np.ndarray, k: np.ndarray, v: np.ndarray) -> np.ndarray:
    """§8c step 4e (Q12, Q13) for ONE frame.  q: [S, Hq, dh]; k, v: [S, Hkv, dh].
    head a uses kv head a // G; s_nm = q_n . k_m / sqrt(dh) for m <= n (sequence index
    within the frame), p = softmax over m (max-subtracted), o_n = sum_m p_nm v_m."""
    S, Hq, dh = q.shape
    G = Hq // k.shape[1]
    o = np.zeros_like(q)
    for a in range(Hq):
        kv = a // G
        for n in range(S):
            s = (k[: n + 1, kv, :] @ q[n, a, :]) / np.sqrt(np.float64(dh))
            p = np.exp(s - np.max(s))
            p = p / np.sum(p)
            o[n, a, :] = p @ v[: n + 1, kv, :]
    return o


# ---------------------------------------------------------------------------- step 4: a layer
def layer_forward(x: np.ndarray, W: dict, phi: np.ndarray, m, taps: dict | None = None,
                  stop_after_attn: bool = False, attention=None) -> np.ndarray:
    """§8c step 4a-g for ONE frame.  x: [S, d] residual (fp64).  Returns the new residual.
    `attention` (plumbing for oracle/te_vision.py, NEXT-4): the attention function of step 4e; None = the
    decoder's causal attention_causal_gqa."""
    S = x.shape[0]
    Hq, Hkv, dh = m.n_q_heads, m.n_kv_heads, m.head_dim
    h = rmsnorm(x, W["g1"], m.rms_eps)                                   # 4a
    q = (h @ W["Wq"].T).reshape(S, Hq, dh)                               # 4b
    k = (h @ W["Wk"].T).reshape(S, Hkv, dh)
    v = (h @ W["Wv"].T).reshape(S, Hkv, dh)
    q = rmsnorm(q, W["gq"], m.rms_eps)                                   # 4c (Q11)
    k = rmsnorm(k, W["gk"], m.rms_eps)
    q = rope_apply(q, phi)                                               # 4d
    k = rope_apply(k, phi)
    o = (attention or attention_causal_gqa)(q, k, v)                     # 4e
    x = x + o.reshape(S, Hq * dh) @ W["Wo"].T                            # 4f
    if taps is not None:
        taps.setdefault("q", []).append(q.reshape(S, -1))
        taps.setdefault("k", []).append(k.reshape(S, -1))
        taps.setdefault("v", []).append(v.reshape(S, -1))
        taps.setdefault("attn", []).append(o.reshape(S, -1))
        taps.setdefault("x_attn", []).append(x.copy())
    if stop_after_attn:
        return x
    h2 = rmsnorm(x, W["g2"], m.rms_eps)                                  # 4g
    act = silu(h2 @ W["Wgate"].T) * (h2 @ W["Wup"].T)
    x = x + act @ W["Wdown"].T
    if taps is not None:
        taps.setdefault("act", []).append(act)
        taps.setdefault("x_mlp", []).append(x.copy())
    return x


# ------------------------------------------------------------------------------ whole call
def encode(blob_bits: np.ndarray, layout: dict, m, embeds: np.ndarray, text_lens,
           grid_h: int, grid_w: int, *, frames=None, layer_begin: int = 0,
           layer_end: int | None = None, stop_after_attn: bool = False,
           final_norm: int | None = None, taps: dict | None = None,
           prefix_len: int = 0, attention=None) -> np.ndarray:
    """te_encode in fp64 (§8c steps 1-5).  embeds: fp32/fp64 [T, d] frame-major packed.
    Returns float64 [T, d].  `frames` restricts the computation to a subset of frames
    (frames never interact, BASELINE.json:configs[4]); rows of other frames are NaN.
    taps (optional dict) collects per-layer intermediates, each a list over layers of
    [T, ...] arrays assembled in packed order (only when frames is None).
    prefix_len = P > 0 (NEXT-1): every frame's rows are [P prefix | gh*gw visual | text];
    the prefix is simply part of each frame's causal sequence — no reuse, no shortcut."""
    text_lens = [int(t) for t in text_lens]
    B = len(text_lens)
    cu = cu_seqlens(text_lens, grid_h, grid_w, prefix_len)
    pos = position_ids(text_lens, grid_h, grid_w, prefix_len)
    phi = mrope_angles(pos, m.head_dim, m.rope_sections, m.rope_theta,
                       bool(getattr(m, "rope_interleaved", False)))
    T = int(cu[-1])
    assert embeds.shape == (T, m.hidden)
    L_end = m.n_layers if layer_end is None else layer_end
    sel = list(range(B)) if frames is None else list(frames)
    x = {b: np.asarray(embeds[cu[b]:cu[b + 1]], dtype=np.float64).copy() for b in sel}
    frame_taps = {b: ({} if taps is not None else None) for b in sel}
    for l in range(layer_begin, L_end):       # layer-outer so each layer is decoded once
        W = unpack_layer(blob_bits, layout, l)
        for b in sel:
            x[b] = layer_forward(x[b], W, phi[cu[b]:cu[b + 1]], m, frame_taps[b],
                                 stop_after_attn=stop_after_attn, attention=attention)
    fn = m.final_norm if final_norm is None else final_norm
    if fn:                                                               # step 5 (Q8)
        off, shape = layout[("final", "gf")]
        gf = bf16_bits_to_f64(blob_bits[off:off + shape[0]])
        for b in sel:
            x[b] = rmsnorm(x[b], gf, m.rms_eps)
    out = np.full((T, m.hidden), np.nan, dtype=np.float64)
    for b in sel:
        out[cu[b]:cu[b + 1]] = x[b]
    if taps is not None and frames is None:
        keys = frame_taps[sel[0]].keys()
        for key in keys:
            n_l = len(frame_taps[sel[0]][key])
            taps[key] = [np.concatenate([frame_taps[b][key][i] for b in sel], axis=0)
                         for i in range(n_l)]
        taps["pos"] = pos
        taps["cu_seqlens"] = cu
        taps["cos"] = np.cos(phi)
        taps["sin"] = np.sin(phi)
    return out
