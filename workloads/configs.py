"""Model + workload tables = BASELINE.json:configs[0..4].

cfg numbering follows SURVEY.md §8 (1-based): cfg k == BASELINE.json configs[k-1].
"""
from __future__ import annotations

from dataclasses import dataclass, field, asdict
from typing import Tuple


@dataclass(frozen=True)
class TEModelConfig:
    """Decoder-stack shape (BASELINE.json:configs; SURVEY.md §8 symbols)."""
    n_layers: int          # L
    hidden: int            # d
    n_q_heads: int         # Hq
    n_kv_heads: int        # Hkv
    head_dim: int          # dh
    ffn: int               # F
    rope_sections: Tuple[int, int, int]   # (s_t, s_h, s_w); sum == head_dim // 2
    rms_eps: float = 1e-6
    rope_theta: float = 1e6
    final_norm: int = 0    # raw last-layer residual by default
    rope_interleaved: bool = False   # round-robin t,h,w frequency pairs instead of contiguous

    def __post_init__(self):
        assert sum(self.rope_sections) == self.head_dim // 2
        assert self.n_q_heads % self.n_kv_heads == 0

    @property
    def qkv_out(self) -> int:
        return (self.n_q_heads + 2 * self.n_kv_heads) * self.head_dim

    def with_layers(self, n_layers: int) -> "TEModelConfig":
        return self.replace(n_layers=n_layers)

    def replace(self, **kw) -> "TEModelConfig":
        d = asdict(self)
        d["rope_sections"] = tuple(d["rope_sections"])
        d.update(kw)
        return TEModelConfig(**d)


@dataclass(frozen=True)
class Workload:
    """One call of te_encode: a batch of frames (BASELINE.json:configs)."""
    name: str
    model: TEModelConfig
    n_frames: int                 # B
    grid_h: int
    grid_w: int
    text_len: object              # int (uniform) or (lo, hi) inclusive, drawn from seed
    outliers: str = "none"        # "none" | "x1000" (configs[2..4]) | "paper" (SURVEY Q16 variant)
    seed_weights: int = 1
    seed_embeds: int = 2
    seed_outlier_channels: int = 3
    seed_text_lens: int = 4


TINY = TEModelConfig(n_layers=2, hidden=256, n_q_heads=4, n_kv_heads=2, head_dim=64,
                     ffn=768, rope_sections=(8, 12, 12))
FULL1 = TEModelConfig(n_layers=1, hidden=2048, n_q_heads=16, n_kv_heads=8, head_dim=128,
                      ffn=6144, rope_sections=(16, 24, 24))
FULL28 = FULL1.with_layers(28)

CONFIGS = {
    1: Workload("cfg1_tiny_2L_B2", TINY, n_frames=2, grid_h=4, grid_w=4, text_len=24),
    2: Workload("cfg2_1L_B1", FULL1, n_frames=1, grid_h=8, grid_w=8, text_len=64),
    3: Workload("cfg3_28L_B4", FULL28, n_frames=4, grid_h=8, grid_w=8, text_len=64,
                outliers="x1000"),
    4: Workload("cfg4_28L_B16", FULL28, n_frames=16, grid_h=8, grid_w=8, text_len=128,
                outliers="x1000"),
    5: Workload("cfg5_28L_B32_ragged", FULL28, n_frames=32, grid_h=8, grid_w=8,
                text_len=(16, 96), outliers="x1000"),
}


def get_workload(cfg_id: int) -> Workload:
    return CONFIGS[int(cfg_id)]


# ---------------------------------------------------------------- vision-tower front end
@dataclass(frozen=True)
class VisionConfig:
    """Patch embedding + tower + 2x2 merger in front of the decoder (readings Q28-Q31).
    `tower` is a decoder-shaped stack (non-causal attention, final norm on) of width d_v = tower.hidden."""
    tower: TEModelConfig
    patch: int            # P: pixels per patch side
    image_h: int          # pixels; image_h / patch and image_w / patch are the (even) patch-grid sizes
    image_w: int
    out_hidden: int       # the decoder's hidden size (merger output)

    @property
    def grid_h(self) -> int:
        return self.image_h // self.patch

    @property
    def grid_w(self) -> int:
        return self.image_w // self.patch

    @property
    def patch_dim(self) -> int:
        return self.patch * self.patch * 3

    @property
    def tokens_per_frame(self) -> int:
        return (self.grid_h // 2) * (self.grid_w // 2)


# CPU-sized: 32x32 image, 8x8 patches -> 4x4 patch grid -> 2x2 = 4 visual tokens of width 256 (TINY decoder)
VISION_TINY = VisionConfig(
    tower=TEModelConfig(n_layers=2, hidden=128, n_q_heads=2, n_kv_heads=2, head_dim=64, ffn=256,
                        rope_sections=(8, 12, 12), final_norm=1),
    patch=8, image_h=32, image_w=32, out_hidden=256)
# the paper's shape: 256x256 source patch -> 16x16 grid of 16x16-pixel patches -> 8x8 = 64 visual tokens of width 2048
VISION_FULL = VisionConfig(
    tower=TEModelConfig(n_layers=4, hidden=1024, n_q_heads=16, n_kv_heads=16, head_dim=64, ffn=4096,
                        rope_sections=(8, 12, 12), final_norm=1),
    patch=16, image_h=256, image_w=256, out_hidden=2048)
