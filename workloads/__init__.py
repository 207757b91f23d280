"""Seeded synthetic workloads for the TE-prefill hot path.

This package holds ONLY configuration tables and seeded input generators
(weights, embeddings, text lengths).  It contains none of the method's
arithmetic: no norms, no rotary maths, no attention.  Both the fp64 oracle
(`oracle/`) and the CUDA path (`paper_2606_05981_b200/`) consume the bytes it
produces; neither of them imports the other.
"""
from .configs import (TEModelConfig, Workload, CONFIGS, get_workload, TINY, FULL1, FULL28,  # noqa: F401
                      VisionConfig, VISION_TINY, VISION_FULL)
from .gen import (  # noqa: F401
    blob_layout, blob_num_elements, make_weight_blob, make_embeddings,
    make_text_lens, f32_to_bf16_bits, total_tokens, vision_blob_layout, make_vision_blob, make_pixels,
)
