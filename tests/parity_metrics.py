"""Parity metrics + gates shared by the GPU parity tests and the oracle mutation suite.

Gates (BASELINE.json:north_star + SURVEY.md §8c "Test power"):
  whole-tensor rel-L2 <= 3e-2 (final), <= 1e-2 (one layer)      [north_star]
  outlier channels: max-abs err / max-abs(ref) <= 1e-2            [north_star]
  update  (out - embeds) rel-L2 <= 3e-2 (final) / 1e-2 (per layer)  [§8c (i),(v)]
  non-outlier-channel rel-L2 <= 3e-2                              [§8c (ii)]
  pos / cu_seqlens bit-exact; cos/sin table abs err <= 1e-5       [§8c (iii)]
  q/k/attn taps rel-L2 <= 1e-2                                    [§8c (iv)]
"""
import numpy as np

GATE_FINAL_REL_L2 = 3e-2
GATE_LAYER_REL_L2 = 1e-2
GATE_OUTLIER_MAXABS = 1e-2
GATE_UPDATE_REL_L2 = 3e-2
GATE_LAYER_UPDATE_REL_L2 = 1e-2
GATE_NONOUTLIER_REL_L2 = 3e-2
GATE_COSSIN_ABS = 1e-5
GATE_TAP_REL_L2 = 1e-2


def rel_l2(a, ref):
    a = np.asarray(a, dtype=np.float64)
    ref = np.asarray(ref, dtype=np.float64)
    den = np.linalg.norm(ref)
    return float(np.linalg.norm(a - ref) / den) if den > 0 else float(np.linalg.norm(a - ref))


def cos_sim(a, ref):
    a = np.asarray(a, dtype=np.float64).ravel()
    ref = np.asarray(ref, dtype=np.float64).ravel()
    return float(a @ ref / (np.linalg.norm(a) * np.linalg.norm(ref)))


def stack_metrics(out, ref, embeds, outlier_ch=None):
    """All whole-stack numbers for one comparison (rows with NaN in ref are skipped)."""
    out = np.asarray(out, dtype=np.float64)
    ref = np.asarray(ref, dtype=np.float64)
    emb = np.asarray(embeds, dtype=np.float64)
    rows = ~np.isnan(ref).any(axis=1)
    out, ref, emb = out[rows], ref[rows], emb[rows]
    m = {
        "rel_l2": rel_l2(out, ref),
        "update_rel_l2": rel_l2(out - emb, ref - emb),
        "cos_sim": cos_sim(out, ref),
        "max_abs_err": float(np.max(np.abs(out - ref))),
    }
    if outlier_ch is not None and len(outlier_ch):
        mask = np.ones(ref.shape[1], dtype=bool)
        mask[np.asarray(outlier_ch)] = False
        m["nonoutlier_rel_l2"] = rel_l2(out[:, mask], ref[:, mask])
        oc = np.asarray(outlier_ch)
        m["outlier_maxabs_rel"] = float(np.max(np.abs(out[:, oc] - ref[:, oc])) /
                                        np.max(np.abs(ref[:, oc])))
    else:
        m["nonoutlier_rel_l2"] = m["rel_l2"]
        m["outlier_maxabs_rel"] = float(np.max(np.abs(out - ref)) / np.max(np.abs(ref)))
    return m


def passes_final_gates(m):
    return (m["rel_l2"] <= GATE_FINAL_REL_L2 and m["update_rel_l2"] <= GATE_UPDATE_REL_L2
            and m["nonoutlier_rel_l2"] <= GATE_NONOUTLIER_REL_L2
            and m["outlier_maxabs_rel"] <= GATE_OUTLIER_MAXABS)
