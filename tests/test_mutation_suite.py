"""Mutation suite: every plausible mistake, applied to the oracle, must be
REJECTED by the gates the GPU parity tests use (tests/parity_metrics.py).  If a mutant passed,
the gate would be too loose to certify the CUDA path.  CPU only, cfg 1 (2 layers)."""
import numpy as np
import pytest

import workloads as W
from oracle import te_oracle as O
import parity_metrics as PM


def _run(taps=None):
    w = W.get_workload(1)
    blob = W.make_weight_blob(w.model, w.seed_weights)
    tl = W.make_text_lens(w)
    emb = W.make_embeddings(w, W.total_tokens(w, tl))
    out = O.encode(blob, W.blob_layout(w.model), w.model, emb, tl, w.grid_h, w.grid_w, taps=taps)
    return out, emb


@pytest.fixture(scope="module")
def clean():
    taps = {}
    out, emb = _run(taps)
    return out, emb, taps


def _rejected(clean, mut_out, mut_taps):
    """True if at least one gate fails for the mutant (the gates of the GPU parity tests)."""
    out, emb, taps = clean
    m = PM.stack_metrics(mut_out, out, emb)
    fails = []
    if not PM.passes_final_gates(m):
        fails.append(("final", m))
    if not (np.array_equal(mut_taps["pos"], taps["pos"]) and np.array_equal(mut_taps["cu_seqlens"], taps["cu_seqlens"])):
        fails.append("pos")
    if max(np.max(np.abs(mut_taps["cos"] - taps["cos"])), np.max(np.abs(mut_taps["sin"] - taps["sin"]))) > PM.GATE_COSSIN_ABS:
        fails.append("cossin")
    for key in ("q", "k", "v", "attn", "act"):
        if PM.rel_l2(mut_taps[key][0], taps[key][0]) > PM.GATE_TAP_REL_L2:
            fails.append(key)
    # teacher-forced per-layer update (layer 0: input is the embedding itself)
    if PM.rel_l2(mut_taps["x_mlp"][0] - emb, taps["x_mlp"][0] - emb) > PM.GATE_LAYER_UPDATE_REL_L2:
        fails.append("layer_update")
    return fails


def test_clean_passes_own_gates(clean):
    t2 = {}
    out2, _ = _run(t2)
    assert _rejected(clean, out2, t2) == []


def _swap_hw(head_dim, sections, interleaved=False):
    s_t, s_h, s_w = sections
    return np.asarray([0] * s_t + [2] * s_h + [1] * s_w, dtype=np.int64)


def _ids_seq_index(text_lens, gh, gw, prefix_len=0):
    cols = []
    for tl in text_lens:
        for k in range(gh * gw):
            cols.append((0, k // gw, k % gw))
        for j in range(int(tl)):
            cols.append((gh * gw + j,) * 3)
    return np.asarray(cols, dtype=np.int32).T.copy()


def _attn_no_mask(q, k, v):
    S, Hq, dh = q.shape
    G = Hq // k.shape[1]
    o = np.zeros_like(q)
    for a in range(Hq):
        s = q[:, a] @ k[:, a // G].T / np.sqrt(dh)
        p = np.exp(s - s.max(-1, keepdims=True)); p /= p.sum(-1, keepdims=True)
        o[:, a] = p @ v[:, a // G]
    return o


def _attn_gqa_mod(q, k, v):
    Hkv = k.shape[1]
    return _attn_with_map(q, k, v, [a % Hkv for a in range(q.shape[1])])


def _attn_with_map(q, k, v, idx, scale=None):
    S, Hq, dh = q.shape
    sc = 1.0 / np.sqrt(dh) if scale is None else scale
    o = np.zeros_like(q)
    mask = np.tril(np.ones((S, S), bool))
    for a in range(Hq):
        s = np.where(mask, q[:, a] @ k[:, idx[a]].T * sc, -np.inf)
        p = np.exp(s - s.max(-1, keepdims=True)); p /= p.sum(-1, keepdims=True)
        o[:, a] = p @ v[:, idx[a]]
    return o


def _attn_no_scale(q, k, v):
    G = q.shape[1] // k.shape[1]
    return _attn_with_map(q, k, v, [a // G for a in range(q.shape[1])], scale=1.0)


def _rope_adjacent(u, phi):
    c = np.cos(phi)[:, None, :]; s = np.sin(phi)[:, None, :]
    a, b = u[..., 0::2], u[..., 1::2]
    out = np.empty_like(u)
    out[..., 0::2] = a * c - b * s
    out[..., 1::2] = b * c + a * s
    return out


def _rope_wrong_sign(u, phi):
    return O_rope(u, -phi)


O_rope = O.rope_apply
O_rms = O.rmsnorm


def _rms_one_plus_g(x, g, eps):
    return O_rms(x, 1.0 + g, eps)


def _rms_drop_head_gain(x, g, eps):
    # drops only the per-head q/k gains (vectors of length dh == x.shape[-1] on 3-D inputs)
    return O_rms(x, np.ones_like(g) if x.ndim == 3 else g, eps)


def _silu_as_sigmoid(z):
    return 1.0 / (1.0 + np.exp(-z))


MUTANTS = {
    "swap_h_w_sections": ("rope_axis", _swap_hw),
    "text_ids_are_sequence_index": ("position_ids", _ids_seq_index),
    "no_causal_mask": ("attention_causal_gqa", _attn_no_mask),
    "gqa_a_mod_hkv": ("attention_causal_gqa", _attn_gqa_mod),
    "no_softmax_scale": ("attention_causal_gqa", _attn_no_scale),
    "adjacent_pair_rope": ("rope_apply", _rope_adjacent),
    "rope_wrong_sign": ("rope_apply", _rope_wrong_sign),
    "rmsnorm_one_plus_gain": ("rmsnorm", _rms_one_plus_g),
    "dropped_qk_gain": ("rmsnorm", _rms_drop_head_gain),
    "sigmoid_instead_of_silu": ("silu", _silu_as_sigmoid),
}


@pytest.mark.parametrize("name", sorted(MUTANTS))
def test_mutant_is_rejected(clean, monkeypatch, name):
    attr, fn = MUTANTS[name]
    monkeypatch.setattr(O, attr, fn)
    taps = {}
    out, _ = _run(taps)
    fails = _rejected(clean, out, taps)
    assert fails, f"mutant {name} passed every gate"


# ------------------------------------------------------------------ row-local mutants (per-token gates)
@pytest.fixture(scope="module")
def tall():
    """Tiny stack at T = 1026 tokens (ragged frames, two 512-row blocks + a 2-row tail): the oracle, and the
    bf16-rounding emulation of it as the stand-in for a CORRECT CUDA result."""
    import bf16_emulation as E
    m = W.TINY
    blob = W.make_weight_blob(m, 1)
    lay = W.blob_layout(m)
    rng = np.random.default_rng(21)
    tl, left = [], 1026
    while left > 0:
        s = int(min(left, rng.integers(40, 256)))
        tl.append(s - 1)
        left -= s
    T = len(tl) + sum(tl)
    emb = rng.standard_normal((T, m.hidden)).astype(np.float32)
    emb[:, [7, 130]] *= np.float32(1000.0)          # outlier channels as in configs[2..4]
    ref = O.encode(blob, lay, m, emb, tl, 1, 1)
    good = E.encode_bf16(blob, lay, m, emb, tl, 1, 1)
    return ref, good, emb.astype(np.float64), np.asarray([7, 130])


def test_row_gate_floors(tall):
    """The emulated-bf16 result passes every gate with >= 3x headroom on the per-token ones."""
    ref, good, emb, ch = tall
    m = PM.stack_metrics(good, ref, emb, ch)
    assert PM.passes_final_gates(m), m
    assert 3 * m["max_row_update_rel_l2"] <= PM.GATE_ROW_UPDATE_REL_L2, m
    assert 3 * m["maxabs_update_over_rms"] <= PM.GATE_MAXABS_UPDATE_OVER_RMS, m
    assert 3 * m["update_rel_l2"] <= PM.GATE_UPDATE_REL_L2, m


def _wrong_rstd_row(out, emb, row):
    o = out.copy()
    o[row] = emb[row] + 1.3 * (out[row] - emb[row])     # one token's update scaled by a wrong 1/rms
    return o


def _tile_last_row_dropped(out, emb, row):
    o = out.copy()
    o[row] = emb[row]                                    # the row's update never written (last row of a tile)
    return o


def _half_of_a_row_update(out, emb, row):
    o = out.copy()
    o[row] = emb[row] + 0.5 * (out[row] - emb[row])     # one of two K-slices of the row's tile dropped
    return o


def _round1_gates(m):
    """The whole-tensor gates as they stood in round 1."""
    return (m["rel_l2"] <= 3e-2 and m["update_rel_l2"] <= 3e-2 and m["nonoutlier_rel_l2"] <= 3e-2
            and m["outlier_maxabs_rel"] <= 1e-2)


@pytest.mark.parametrize("mutant,row", [(_wrong_rstd_row, 700), (_half_of_a_row_update, 127), (_half_of_a_row_update, 1025),
                                        (_wrong_rstd_row, 0), (_tile_last_row_dropped, 511)])
def test_one_bad_token_row_is_rejected_by_the_row_gates(tall, mutant, row):
    """ONE corrupted token row at T >= 1024: (mostly) invisible to norms over the whole tensor — a fully dropped row
    moves the update rel-L2 by 1/sqrt(T) = 3.1 % here and by 1.8 % at cfg 4's T = 3072 — caught by the per-token gates."""
    ref, good, emb, ch = tall
    bad = mutant(good, emb, row)
    m = PM.stack_metrics(bad, ref, emb, ch)
    assert _round1_gates(m), m                           # round 1 would have passed it
    assert not PM.passes_row_gates(m), m
    assert not PM.passes_final_gates(m)


def test_one_bad_element_is_rejected(tall):
    """One wrong element (a dropped split-K partial on one column of one row): max-abs gate."""
    ref, good, emb, ch = tall
    bad = good.copy()
    bad[333, 45] += 0.3 * np.sqrt(np.mean((ref - emb) ** 2))
    m = PM.stack_metrics(bad, ref, emb, ch)
    assert PM.passes_whole_tensor_gates(m)
    assert m["max_row_update_rel_l2"] <= PM.GATE_ROW_UPDATE_REL_L2      # too small for the row norm as well
    assert m["maxabs_update_over_rms"] > PM.GATE_MAXABS_UPDATE_OVER_RMS
