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
