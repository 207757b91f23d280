"""fp64 oracle of the vision-tower front end.  TEST INFRASTRUCTURE ONLY (same rules as
oracle/te_oracle.py).

What it states.  The paper says only that the TE's prompt template carries an image-pad token "processed by Qwen3-VL's
vision tower" and that a 256x256 source patch becomes ~64 visual tokens; it gives no
equation, shape or weight for the tower, and BASELINE.json:configs describe the decoder only.  The tower is therefore
the readings Q28-Q31 of DESIGN.md §3, chosen so that it produces exactly what the decoder path consumes (64 visual
embeddings per frame on an 8x8 grid) out of the blocks whose definitions BASELINE.json does fix:

  Q28  patch embedding: the frame's [H, W, 3] pixels are cut into P x P patches, row-major over the patch grid, each
       flattened in (dy, dx, channel) order, and multiplied by W_pe [d_v, P*P*3] (a linear patch embedding, no bias).
  Q29  tower blocks: the SAME pre-norm block as the decoder (oracle/te_oracle.layer_forward: RMSNorm, per-head
       QK-RMSNorm, SwiGLU, no biases) with NON-causal attention over the frame's patches and rotary ids (0, py, px) on
       the patch grid (M-RoPE with t = 0: the 2-D rotary embedding of a ViT); frames never interact.
  Q30  merger: final RMSNorm (gain g_f), then every 2 x 2 block of neighbouring patches is concatenated in (dy, dx)
       row-major order (4 * d_v values) and multiplied by W_m [hidden, 4*d_v]; merged tokens are row-major on the
       (gh/2) x (gw/2) grid = the visual-token order of the decoder.
  Q31  weights: one blob = W_pe | the tower's decoder-layout blob (oracle/te_oracle blob order, incl. g_f) | W_m, bf16,
       seeded like the decoder's (matrices N(0, 0.02), gains 1 + 0.1 N(0,1)); pixels fp32 in [0, 1).

Plain numpy fp64, no intermediate rounding; a float64 `@` is the only library step.  Pins: tests/test_vision_pins.py.
"""
from __future__ import annotations

import numpy as np

from . import te_oracle as O


def patchify(pixels: np.ndarray, P: int) -> np.ndarray:
    """Q28.  pixels [B, H, W, 3] -> [B * (H/P) * (W/P), P*P*3]: patch (py, px) of frame b is row
    b*(H/P)*(W/P) + py*(W/P) + px; inside a patch the order is (dy, dx, channel)."""
    B, H, Wd, C = pixels.shape
    gh, gw = H // P, Wd // P
    out = np.empty((B * gh * gw, P * P * C), dtype=np.float64)
    r = 0
    for b in range(B):
        for py in range(gh):
            for px in range(gw):
                out[r] = np.asarray(pixels[b, py * P:(py + 1) * P, px * P:(px + 1) * P, :], dtype=np.float64).reshape(-1)
                r += 1
    return out


def attention_full_gqa(q: np.ndarray, k: np.ndarray, v: np.ndarray) -> np.ndarray:
    """Q29: te_oracle.attention_causal_gqa without the mask — every query sees every key of its frame."""
    S, Hq, dh = q.shape
    G = Hq // k.shape[1]
    o = np.zeros_like(q)
    for a in range(Hq):
        kv = a // G
        for n in range(S):
            s = (k[:, kv, :] @ q[n, a, :]) / np.sqrt(np.float64(dh))
            p = np.exp(s - np.max(s))
            p = p / np.sum(p)
            o[n, a, :] = p @ v[:, kv, :]
    return o


def merge2x2(h: np.ndarray, n_frames: int, gh: int, gw: int) -> np.ndarray:
    """Q30.  h [B*gh*gw, d_v] (patch-row-major) -> [B*(gh/2)*(gw/2), 4*d_v]: merged token (my, mx) is the
    concatenation of patches (2my, 2mx), (2my, 2mx+1), (2my+1, 2mx), (2my+1, 2mx+1)."""
    d = h.shape[1]
    out = np.empty((n_frames * (gh // 2) * (gw // 2), 4 * d), dtype=np.float64)
    r = 0
    for b in range(n_frames):
        base = b * gh * gw
        for my in range(gh // 2):
            for mx in range(gw // 2):
                parts = [h[base + (2 * my + dy) * gw + (2 * mx + dx)] for dy in (0, 1) for dx in (0, 1)]
                out[r] = np.concatenate(parts)
                r += 1
    return out


def encode_image(w_pe: np.ndarray, tower_blob: np.ndarray, tower_layout: dict, mv, w_m: np.ndarray,
                 pixels: np.ndarray, P: int, taps: dict | None = None) -> np.ndarray:
    """pixels [B, H, W, 3] -> visual embeddings [B * (H/2P) * (W/2P), hidden] (float64).
    w_pe, w_m: bf16 bit patterns (uint16) [d_v, P*P*3] and [hidden, 4*d_v]; mv: the tower's model config
    (final_norm = 1)."""
    B, H, Wd, _ = pixels.shape
    gh, gw = H // P, Wd // P
    x0 = patchify(pixels, P) @ O.bf16_bits_to_f64(w_pe).reshape(w_pe.shape).T                     # Q28
    hid = O.encode(tower_blob, tower_layout, mv, x0, [0] * B, gh, gw, final_norm=1,
                   attention=attention_full_gqa)                                                   # Q29 (+ final norm)
    vis = merge2x2(hid, B, gh, gw) @ O.bf16_bits_to_f64(w_m).reshape(w_m.shape).T                 # Q30
    if taps is not None:
        taps["patch_embeds"], taps["tower_out"] = x0, hid
    return vis
