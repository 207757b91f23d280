"""Seeded generators: weight blob (bf16 bits), embeddings (fp32), text lengths.

Recipe = SURVEY.md §8c Q7/Q16/Q17 and §8d "Synthetic inputs":
  * matrices ~ N(0, 0.02); RMSNorm gains ~ 1 + 0.1*N(0,1); rounded to bf16 (RNE);
  * embeddings ~ N(0,1) fp32; for configs[2..4] two seeded channels are scaled x1000;
  * cfg 5 text lengths ~ U{16..96}.
Generator: numpy Philox, `standard_normal(float32)`.  One Philox stream per layer
(key = [seed, layer]) so layer l of a deep stack equals layer l of a shallow one.

Canonical blob layout, contiguous bf16, every matrix row-major
[out_features, in_features] (y = x W^T):
  per layer: g1[d] Wq[Hq*dh,d] Wk[Hkv*dh,d] Wv[Hkv*dh,d] gq[dh] gk[dh] Wo[d,Hq*dh]
             g2[d] Wgate[F,d] Wup[F,d] Wdown[d,F]
  then gf[d].
No arithmetic of the method lives here; f32->bf16 RNE is the storage format of the input.
"""
from __future__ import annotations

import numpy as np

from .configs import TEModelConfig, Workload

_FINAL_KEY = 0xFFFF


def layer_tensors(m: TEModelConfig):
    """[(name, shape, kind)] for ONE layer in blob order; kind in {"gain","matrix"}."""
    d, dh, F = m.hidden, m.head_dim, m.ffn
    return [
        ("g1", (d,), "gain"),
        ("Wq", (m.n_q_heads * dh, d), "matrix"),
        ("Wk", (m.n_kv_heads * dh, d), "matrix"),
        ("Wv", (m.n_kv_heads * dh, d), "matrix"),
        ("gq", (dh,), "gain"),
        ("gk", (dh,), "gain"),
        ("Wo", (d, m.n_q_heads * dh), "matrix"),
        ("g2", (d,), "gain"),
        ("Wgate", (F, d), "matrix"),
        ("Wup", (F, d), "matrix"),
        ("Wdown", (d, F), "matrix"),
    ]


def blob_layout(m: TEModelConfig):
    """{(layer, name): (offset_elems, shape)} plus {("final","gf"): ...}."""
    out = {}
    off = 0
    for l in range(m.n_layers):
        for name, shape, _ in layer_tensors(m):
            n = int(np.prod(shape))
            out[(l, name)] = (off, shape)
            off += n
    out[("final", "gf")] = (off, (m.hidden,))
    return out


def blob_num_elements(m: TEModelConfig) -> int:
    per_layer = sum(int(np.prod(s)) for _, s, _ in layer_tensors(m))
    return per_layer * m.n_layers + m.hidden


def f32_to_bf16_bits(x: np.ndarray) -> np.ndarray:
    """Round-to-nearest-even fp32 -> bf16 bit pattern (uint16). Finite inputs only."""
    b = np.ascontiguousarray(x, dtype=np.float32).view(np.uint32)
    r = (b + np.uint32(0x7FFF) + ((b >> np.uint32(16)) & np.uint32(1))) >> np.uint32(16)
    return r.astype(np.uint16)


def _fill_layer(blob: np.ndarray, m: TEModelConfig, seed: int, l: int, off: int, gains: str) -> None:
    rng = np.random.Generator(np.random.Philox(key=[seed, l]))
    for _, shape, kind in layer_tensors(m):
        n = int(np.prod(shape))
        z = rng.standard_normal(n, dtype=np.float32)
        if kind == "matrix":
            w = z * np.float32(0.02)
        elif gains == "ones":
            w = np.ones(n, dtype=np.float32)
        else:
            w = np.float32(1.0) + np.float32(0.1) * z
        blob[off:off + n] = f32_to_bf16_bits(w)
        off += n


def make_weight_blob(m: TEModelConfig, seed: int = 1, gains: str = "randn") -> np.ndarray:
    """uint16[blob_num_elements] of bf16 bits.  gains: "randn" (1+0.1N) or "ones".
    Layers are independent Philox streams, so they are filled by a small thread pool."""
    blob = np.empty(blob_num_elements(m), dtype=np.uint16)
    per_layer = sum(int(np.prod(s)) for _, s, _ in layer_tensors(m))
    if m.n_layers >= 4:
        from concurrent.futures import ThreadPoolExecutor
        import os
        with ThreadPoolExecutor(max_workers=min(8, os.cpu_count() or 1)) as ex:
            list(ex.map(lambda l: _fill_layer(blob, m, seed, l, l * per_layer, gains), range(m.n_layers)))
    else:
        for l in range(m.n_layers):
            _fill_layer(blob, m, seed, l, l * per_layer, gains)
    off = per_layer * m.n_layers
    rng = np.random.Generator(np.random.Philox(key=[seed, _FINAL_KEY]))
    z = rng.standard_normal(m.hidden, dtype=np.float32)
    gf = np.ones(m.hidden, np.float32) if gains == "ones" else np.float32(1.0) + np.float32(0.1) * z
    blob[off:off + m.hidden] = f32_to_bf16_bits(gf)
    off += m.hidden
    assert off == blob.size
    return blob


def make_text_lens(w: Workload) -> np.ndarray:
    if isinstance(w.text_len, tuple):
        lo, hi = w.text_len
        rng = np.random.Generator(np.random.Philox(key=[w.seed_text_lens, 0]))
        return rng.integers(lo, hi + 1, size=w.n_frames).astype(np.int32)
    return np.full(w.n_frames, int(w.text_len), dtype=np.int32)


def total_tokens(w: Workload, text_lens: np.ndarray) -> int:
    return int(w.n_frames * w.grid_h * w.grid_w + int(np.sum(text_lens)))


def outlier_channels(w: Workload) -> np.ndarray:
    rng = np.random.Generator(np.random.Philox(key=[w.seed_outlier_channels, 0]))
    return np.sort(rng.choice(w.model.hidden, size=2, replace=False))


def make_embeddings(w: Workload, n_tokens: int, outliers: str | None = None) -> np.ndarray:
    """fp32 [T, d], frame-major packed.  outliers: None -> w.outliers."""
    mode = w.outliers if outliers is None else outliers
    d = w.model.hidden
    rng = np.random.Generator(np.random.Philox(key=[w.seed_embeds, 0]))
    x = rng.standard_normal((n_tokens, d), dtype=np.float32)
    if mode == "x1000":
        # BASELINE.json configs[2]: "2 seeded channels scaled x1000" (literal reading, Q16)
        ch = outlier_channels(w)
        x[:, ch] *= np.float32(1000.0)
    elif mode == "paper":
        # Q16 variant: near-constant-magnitude channels at the paper's extremes
        # (min -854, max 1160).
        ch = outlier_channels(w)
        x[:, ch[0]] = np.float32(1160.0) * (np.float32(1.0) + np.float32(0.02) * x[:, ch[0]])
        x[:, ch[1]] = np.float32(-854.0) * (np.float32(1.0) + np.float32(0.02) * x[:, ch[1]])
    else:
        assert mode == "none"
    return x


# ---------------------------------------------------------------- vision-tower front end
def vision_blob_layout(v):
    """Element offsets of the vision blob: W_pe [d_v, P*P*3] | tower blob (decoder layout, incl. gf) | W_m [hidden, 4*d_v]."""
    d_v = v.tower.hidden
    n_pe = d_v * v.patch_dim
    n_tower = blob_num_elements(v.tower)
    return {"W_pe": (0, (d_v, v.patch_dim)), "tower": (n_pe, n_tower),
            "W_m": (n_pe + n_tower, (v.out_hidden, 4 * d_v)), "total": n_pe + n_tower + v.out_hidden * 4 * d_v}


def make_vision_blob(v, seed: int = 11) -> np.ndarray:
    """uint16 bf16 bits.  W_pe and W_m ~ N(0, 0.02) from Philox(key=[seed, 0xFFFE]); the tower exactly as
    make_weight_blob(v.tower, seed)."""
    lay = vision_blob_layout(v)
    blob = np.empty(lay["total"], dtype=np.uint16)
    rng = np.random.Generator(np.random.Philox(key=[seed, 0xFFFE]))
    off, shape = lay["W_pe"]
    blob[off:off + int(np.prod(shape))] = f32_to_bf16_bits(rng.standard_normal(int(np.prod(shape)), dtype=np.float32) * np.float32(0.02))
    t_off, t_n = lay["tower"]
    blob[t_off:t_off + t_n] = make_weight_blob(v.tower, seed)
    off, shape = lay["W_m"]
    blob[off:off + int(np.prod(shape))] = f32_to_bf16_bits(rng.standard_normal(int(np.prod(shape)), dtype=np.float32) * np.float32(0.02))
    return blob


def make_pixels(v, n_frames: int, seed: int = 12) -> np.ndarray:
    """fp32 [B, H, W, 3] in [0, 1): a smooth seeded pattern plus noise (stands in for the DAVIS source patches)."""
    rng = np.random.Generator(np.random.Philox(key=[seed, 0]))
    yy, xx = np.meshgrid(np.arange(v.image_h, dtype=np.float32), np.arange(v.image_w, dtype=np.float32), indexing="ij")
    out = np.empty((n_frames, v.image_h, v.image_w, 3), dtype=np.float32)
    for b in range(n_frames):
        f = rng.uniform(0.01, 0.2, size=(3, 2)).astype(np.float32)
        for c in range(3):
            out[b, :, :, c] = 0.5 + 0.35 * np.sin(f[c, 0] * yy + b) * np.cos(f[c, 1] * xx)
    out += rng.uniform(-0.1, 0.1, size=out.shape).astype(np.float32)
    return np.clip(out, 0.0, 0.999).astype(np.float32)
