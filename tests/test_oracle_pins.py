"""Pins for the fp64 oracle (oracle/te_oracle.py): everything here runs on CPU.

Each test checks the oracle against something that is NOT the oracle: values fixed by
BASELINE.json / mathematics (tests/golden/), closed forms, invariants, a pure-Python scalar
brute force, and an independently written dense-mask restatement.  Chosen so that a dropped
term, wrong sign/index or transposed operand fails at least one of them.
"""
import math
import os

import numpy as np
import pytest

import workloads as W
from oracle import te_oracle as O

GOLD = os.path.join(os.path.dirname(__file__), "golden")


def _read_closed_forms():
    d = {}
    for line in open(os.path.join(GOLD, "closed_forms.txt")):
        if line.strip() and not line.startswith("#"):
            k, v = line.split()
            d[k] = float(v)
    return d


CF = _read_closed_forms()


# --------------------------------------------------------------------------- packing / ids
def test_position_ids_golden_cfg1():
    rows, cu = [], None
    for line in open(os.path.join(GOLD, "position_ids_cfg1.txt")):
        if line.startswith("#") or not line.strip():
            continue
        if line.startswith("cu_seqlens"):
            cu = [int(v) for v in line.split()[1:]]
        else:
            rows.append([int(v) for v in line.split()])
    rows = np.asarray(rows)
    w = W.get_workload(1)
    tl = W.make_text_lens(w)
    assert list(O.cu_seqlens(tl, w.grid_h, w.grid_w)) == cu
    pos = O.position_ids(tl, w.grid_h, w.grid_w)
    assert pos.dtype == np.int32 and pos.shape == (3, 80)
    for b in range(2):                      # both frames carry the same per-frame ids
        np.testing.assert_array_equal(pos[:, 40 * b:40 * (b + 1)].T, rows[:, 1:])


def test_position_ids_cfg4_worked_values():
    w = W.get_workload(4)
    tl = W.make_text_lens(w)
    cu = O.cu_seqlens(tl, 8, 8)
    assert int(cu[1]) == int(CF["cfg4_S"]) and list(cu) == [192 * b for b in range(17)]
    pos = O.position_ids(tl, 8, 8)
    assert pos[:, 64].tolist() == [int(CF["cfg4_text_first"])] * 3
    assert pos[:, 191].tolist() == [int(CF["cfg4_text_last"])] * 3
    assert pos[:, 63].tolist() == [0, 7, 7]


@pytest.mark.parametrize("gh,gw", [(4, 16), (16, 4), (1, 5), (3, 3)])
def test_position_ids_nonsquare_enumeration(gh, gw):
    """Q5 row-major order is only visible on non-square grids."""
    tl = [3, 0, 5]
    pos = O.position_ids(tl, gh, gw)
    cu = O.cu_seqlens(tl, gh, gw)
    assert cu[-1] == pos.shape[1]
    for b, t in enumerate(tl):
        p = pos[:, cu[b]:cu[b + 1]]
        vis = p[:, :gh * gw]
        assert (vis[0] == 0).all()
        # every (h, w) cell appears exactly once, w fastest
        assert [(int(h), int(w_)) for h, w_ in zip(vis[1], vis[2])] == \
               [(h, w_) for h in range(gh) for w_ in range(gw)]
        txt = p[:, gh * gw:]
        assert txt.shape[1] == t
        assert (txt[0] == txt[1]).all() and (txt[1] == txt[2]).all()
        assert txt[0].tolist() == list(range(max(gh, gw), max(gh, gw) + t))
        assert int(vis.max()) + 1 == max(gh, gw) or min(gh, gw) == 0


# ------------------------------------------------------------------------ angles / RoPE
def test_position_ids_prefix_golden():
    """NEXT-1: worked ids with a 3-token prefix before a 2x3 grid (tests/golden/position_ids_prefix.txt)."""
    lines = [l.split() for l in open(os.path.join(GOLD, "position_ids_prefix.txt")) if l.strip() and l[0] != "#"]
    cu = [int(x) for x in lines[0][1:]]
    rows = np.asarray([[int(x) for x in l] for l in lines[1:]], dtype=np.int32)
    assert O.cu_seqlens([2, 0], 2, 3, prefix_len=3).tolist() == cu
    pos = O.position_ids([2, 0], 2, 3, prefix_len=3)
    assert pos.shape == (3, 20)
    assert np.array_equal(pos[:, :11].T, rows[:, 1:])
    assert np.array_equal(pos[:, 11:20], pos[:, :9])          # second frame: same prefix + grid, no text
    # P = 0 is the base rule
    assert np.array_equal(O.position_ids([2, 0], 2, 3, prefix_len=0), O.position_ids([2, 0], 2, 3))
    assert np.array_equal(O.cu_seqlens([2, 0], 2, 3, 0), O.cu_seqlens([2, 0], 2, 3))
    # a "frame" that is only text (no grid) counts 0, 1, 2, ...: what the prefix-alone pass uses
    assert O.position_ids([4], 0, 0).tolist() == [[0, 1, 2, 3]] * 3


def test_inv_freq_closed_forms():
    om = O.inv_freq(128, 1e6)
    assert om[0] == 1.0
    assert abs(om[32] - CF["omega_dh128_i32"]) < 1e-18
    assert abs(om[16] - CF["omega_dh128_i16"]) < 1e-16
    assert abs(O.inv_freq(64, 1e6)[16] - CF["omega_dh64_i16"]) < 1e-18
    assert np.all(np.diff(om) < 0)


def test_rope_axis_sections():
    ax = O.rope_axis(128, (16, 24, 24))
    assert ax[:16].tolist() == [0] * 16 and ax[16:40].tolist() == [1] * 24 and ax[40:].tolist() == [2] * 24
    ax = O.rope_axis(64, (8, 12, 12))
    assert (ax[:8] == 0).all() and (ax[8:20] == 1).all() and (ax[20:] == 2).all()


def test_rope_axis_interleaved():
    """NEXT-5: round-robin t,h,w over the axes that still have pairs; section counts preserved."""
    ax = O.rope_axis(64, (8, 12, 12), interleaved=True)
    assert ax.tolist() == [0, 1, 2] * 8 + [1, 2] * 4                      # typed by hand
    ax = O.rope_axis(128, (16, 24, 24), interleaved=True)
    assert ax[:48].tolist() == [0, 1, 2] * 16 and ax[48:].tolist() == [1, 2] * 8
    for dh, sec in [(128, (16, 24, 24)), (64, (8, 12, 12)), (128, (24, 20, 20)), (64, (32, 0, 0)), (64, (1, 30, 1))]:
        ax = O.rope_axis(dh, sec, interleaved=True)
        assert [int((ax == a).sum()) for a in range(3)] == list(sec)
    # independent closed form for t-heavy sections (the published interleaved layout of this model family):
    # pair i is h if i % 3 == 1 and i < 3*s_h, w if i % 3 == 2 and i < 3*s_w, else t
    s_t, s_h, s_w = 24, 20, 20
    want = [1 if (i % 3 == 1 and i < 3 * s_h) else (2 if (i % 3 == 2 and i < 3 * s_w) else 0) for i in range(64)]
    assert O.rope_axis(128, (s_t, s_h, s_w), interleaved=True).tolist() == want
    # angles follow the table
    pos = np.asarray([[1], [10], [100]], dtype=np.int32)
    phi = O.mrope_angles(pos, 64, (8, 12, 12), 1e6, interleaved=True)
    om = [1e6 ** (-2.0 * i / 64) for i in range(32)]
    assert abs(phi[0, 0] - 1 * om[0]) < 1e-12 and abs(phi[0, 1] - 10 * om[1]) < 1e-12
    assert abs(phi[0, 2] - 100 * om[2]) < 1e-12 and abs(phi[0, 31] - 100 * om[31]) < 1e-12
    assert abs(phi[0, 30] - 10 * om[30]) < 1e-12


def test_mrope_angles_pick_the_right_axis():
    # one token at (t,h,w) = (1, 10, 100): pair i gets pos[axis(i)] * omega_i
    pos = np.asarray([[1], [10], [100]], dtype=np.int32)
    phi = O.mrope_angles(pos, 64, (8, 12, 12), 1e6)
    om = [1e6 ** (-2.0 * i / 64) for i in range(32)]
    for i in range(32):
        p = 1 if i < 8 else (10 if i < 20 else 100)
        assert abs(phi[0, i] - p * om[i]) < 1e-12
    assert abs(math.cos(phi[0, 0]) - CF["cos1"]) < 1e-15
    assert abs(math.sin(phi[0, 0]) - CF["sin1"]) < 1e-15


def test_rope_identity_norms_and_explicit_pair():
    rng = np.random.default_rng(0)
    u = rng.standard_normal((5, 3, 8))
    assert np.array_equal(O.rope_apply(u, np.zeros((5, 4))), u)         # identity at position 0
    phi = rng.standard_normal((5, 4)) * 3
    r = O.rope_apply(u, phi)
    # norm preserved per (i, i+dh/2) pair, hence per head
    np.testing.assert_allclose(r[..., :4] ** 2 + r[..., 4:] ** 2, u[..., :4] ** 2 + u[..., 4:] ** 2, rtol=1e-12)
    # explicit value: (1, 0) rotated by angle 1 in pair (0, 4) -> (cos 1, sin 1)
    e = np.zeros((1, 1, 8)); e[0, 0, 0] = 1.0
    ph = np.zeros((1, 4)); ph[0, 0] = 1.0
    out = O.rope_apply(e, ph)
    assert abs(out[0, 0, 0] - CF["cos1"]) < 1e-15 and abs(out[0, 0, 4] - CF["sin1"]) < 1e-15
    assert np.count_nonzero(out) == 2
    # (0,1) in the pair -> (-sin 1, cos 1): fixes the sign convention
    e = np.zeros((1, 1, 8)); e[0, 0, 4] = 1.0
    out = O.rope_apply(e, ph)
    assert abs(out[0, 0, 0] + CF["sin1"]) < 1e-15 and abs(out[0, 0, 4] - CF["cos1"]) < 1e-15


def test_rope_relative_position_property():
    """<R(p) q, R(p') k> depends only on p - p' (the defining property of rotary embeddings)."""
    rng = np.random.default_rng(1)
    q = rng.standard_normal((1, 1, 64)); k = rng.standard_normal((1, 1, 64))

    def dot(pq, pk):
        a = O.rope_apply(q, O.mrope_angles(np.asarray([[pq]] * 3, dtype=np.int32), 64, (8, 12, 12), 1e6))
        b = O.rope_apply(k, O.mrope_angles(np.asarray([[pk]] * 3, dtype=np.int32), 64, (8, 12, 12), 1e6))
        return float(np.sum(a * b))
    assert abs(dot(7, 3) - dot(104, 100)) < 1e-9
    assert abs(dot(7, 3) - dot(3, 7)) > 1e-3        # and it is not symmetric


def test_visual_tokens_temporal_pairs_unrotated():
    w = W.get_workload(1)
    pos = O.position_ids(W.make_text_lens(w), 4, 4)
    phi = O.mrope_angles(pos, 64, (8, 12, 12), 1e6)
    assert np.all(phi[:16, :8] == 0.0)      # t == 0 for every visual token
    assert np.all(phi[0] == 0.0)            # first visual token: (0,0,0)
    assert np.all(phi[16, :] > 0.0)


# -------------------------------------------------------------------------------- RMSNorm
def test_rmsnorm_closed_forms():
    eps = 1e-6
    g = np.asarray([0.5, 2.0, -1.0, 3.0])
    c = 7.0
    y = O.rmsnorm(np.full((1, 4), c), g, eps)
    np.testing.assert_allclose(y[0], g * c / math.sqrt(c * c + eps), rtol=1e-15)
    x = np.random.default_rng(2).standard_normal((3, 64))
    y = O.rmsnorm(x, np.ones(64), eps)
    ms = np.mean(x * x, axis=1)
    np.testing.assert_allclose(np.mean(y * y, axis=1), 1.0 / (1.0 + eps / ms), rtol=1e-13)
    np.testing.assert_allclose(O.rmsnorm(1e3 * x, np.ones(64), eps), y, rtol=1e-5)   # scale-free up to eps
    z = O.rmsnorm(np.zeros((2, 8)), np.ones(8), eps)
    assert np.all(z == 0.0) and not np.isnan(z).any()
    # eps sits inside the root: tiny row is damped by sqrt(eps), not by eps
    t = O.rmsnorm(np.full((1, 4), 1e-6), np.ones(4), eps)
    np.testing.assert_allclose(t, 1e-6 / math.sqrt(1e-12 + 1e-6), rtol=1e-12)


def test_silu_values():
    assert O.silu(np.float64(0.0)) == 0.0
    assert abs(O.silu(np.float64(1.0)) - CF["silu1"]) < 1e-15
    assert abs(O.silu(np.float64(40.0)) - 40.0) < 1e-12
    assert abs(O.silu(np.float64(-40.0))) < 1e-12
    assert abs(O.silu(np.float64(-1.0)) - (CF["silu1"] - 1.0)) < 1e-15     # silu(-z) = silu(z) - z


# ------------------------------------------------------------------------------ attention
def test_attention_closed_forms():
    rng = np.random.default_rng(3)
    S, Hq, Hkv, dh = 7, 4, 2, 8
    q = rng.standard_normal((S, Hq, dh))
    v = rng.standard_normal((S, Hkv, dh))
    # identical keys -> uniform probabilities -> causal running mean of v of head a // G
    k = np.tile(rng.standard_normal((1, Hkv, dh)), (S, 1, 1))
    o = O.attention_causal_gqa(q, k, v)
    run = np.cumsum(v, axis=0) / np.arange(1, S + 1)[:, None, None]
    for a in range(Hq):
        np.testing.assert_allclose(o[:, a], run[:, a // 2], rtol=1e-12)
    assert not np.allclose(run[:, 0], run[:, 1])
    # S = 1 -> o = v
    o1 = O.attention_causal_gqa(q[:1], k[:1], v[:1])
    np.testing.assert_allclose(o1[0, 3], v[0, 1], rtol=1e-14)
    # v = 1 -> o = 1 (probabilities sum to one)
    k = rng.standard_normal((S, Hkv, dh))
    np.testing.assert_allclose(O.attention_causal_gqa(q, k, np.ones_like(v)), 1.0, rtol=1e-13)
    # zero queries -> uniform causal attention
    o0 = O.attention_causal_gqa(np.zeros_like(q), k, v)
    np.testing.assert_allclose(o0[:, 0], run[:, 0], rtol=1e-12)


def test_attention_two_token_explicit():
    """S=2, dh=4: second row's weights are softmax([q.k0, q.k1] / sqrt(dh)) — the 1/sqrt(dh) scale."""
    q = np.zeros((2, 1, 4)); k = np.zeros((2, 1, 4)); v = np.zeros((2, 1, 4))
    q[1, 0] = [2.0, 0, 0, 0]; k[0, 0] = [1.0, 0, 0, 0]; k[1, 0] = [3.0, 0, 0, 0]
    v[0, 0, 0] = 1.0; v[1, 0, 1] = 1.0
    o = O.attention_causal_gqa(q, k, v)
    s0, s1 = 2.0 * 1.0 / 2.0, 2.0 * 3.0 / 2.0
    p1 = math.exp(s1) / (math.exp(s0) + math.exp(s1))
    assert abs(o[1, 0, 1] - p1) < 1e-15 and abs(o[1, 0, 0] - (1 - p1)) < 1e-15
    assert o[0, 0].tolist() == [1.0, 0, 0, 0]


def test_attention_causality():
    rng = np.random.default_rng(4)
    q = rng.standard_normal((9, 2, 8)); k = rng.standard_normal((9, 2, 8)); v = rng.standard_normal((9, 2, 8))
    o = O.attention_causal_gqa(q, k, v)
    k2, v2 = k.copy(), v.copy()
    k2[5:] += 10.0; v2[5:] -= 3.0
    o2 = O.attention_causal_gqa(q, k2, v2)
    assert np.array_equal(o[:5], o2[:5]) and not np.allclose(o[5:], o2[5:])


# ------------------------------------------------------------------------------ whole stack
def _tiny_inputs(scale_weights=1.0, gains="randn"):
    w = W.get_workload(1)
    blob = W.make_weight_blob(w.model, w.seed_weights, gains=gains)
    tl = W.make_text_lens(w)
    T = W.total_tokens(w, tl)
    emb = W.make_embeddings(w, T)
    return w, blob, W.blob_layout(w.model), tl, emb


def test_zero_projection_pass_through():
    """W_o = W_down = 0  =>  out == embeds exactly (residual pass-through)."""
    w, blob, lay, tl, emb = _tiny_inputs()
    blob = blob.copy()
    for l in range(w.model.n_layers):
        for name in ("Wo", "Wdown"):
            off, shape = lay[(l, name)]
            blob[off:off + int(np.prod(shape))] = 0
    out = O.encode(blob, lay, w.model, emb, tl, 4, 4)
    assert np.array_equal(out, emb.astype(np.float64))


def test_stack_changes_input_and_is_finite():
    w, blob, lay, tl, emb = _tiny_inputs()
    out = O.encode(blob, lay, w.model, emb, tl, 4, 4)
    assert np.isfinite(out).all()
    upd = out - emb
    assert 1e-3 < np.linalg.norm(upd) / np.linalg.norm(emb) < 1.0


def test_frame_independence_and_permutation():
    w, blob, lay, tl, emb = _tiny_inputs()
    m = w.model
    out = O.encode(blob, lay, m, emb, tl, 4, 4)
    solo = O.encode(blob, lay, m, emb[40:], tl[1:], 4, 4)
    assert np.array_equal(out[40:], solo)
    perm = O.encode(blob, lay, m, np.concatenate([emb[40:], emb[:40]]), tl[::-1], 4, 4)
    assert np.array_equal(perm[:40], out[40:]) and np.array_equal(perm[40:], out[:40])
    sub = O.encode(blob, lay, m, emb, tl, 4, 4, frames=[1])
    assert np.isnan(sub[:40]).all() and np.array_equal(sub[40:], out[40:])


def test_stack_causality_within_frame():
    w, blob, lay, tl, emb = _tiny_inputs()
    out = O.encode(blob, lay, w.model, emb, tl, 4, 4)
    emb2 = emb.copy(); emb2[30:40] += 1.0
    out2 = O.encode(blob, lay, w.model, emb2, tl, 4, 4)
    assert np.array_equal(out[:30], out2[:30]) and np.array_equal(out[40:], out2[40:])
    assert not np.allclose(out[30:40], out2[30:40])


def test_position_shift_invariance(monkeypatch):
    """Adding a constant to every id of a frame leaves the output unchanged (only relative
    rotary phases enter q.k).  Catches rotating v, rotating after attention, sign slips."""
    w, blob, lay, tl, emb = _tiny_inputs()
    out = O.encode(blob, lay, w.model, emb, tl, 4, 4)
    orig = O.position_ids
    monkeypatch.setattr(O, "position_ids", lambda *a: orig(*a) + np.int32(11))
    out2 = O.encode(blob, lay, w.model, emb, tl, 4, 4)
    assert np.max(np.abs(out - out2)) < 1e-11
    monkeypatch.setattr(O, "position_ids", lambda *a: orig(*a) + np.asarray([[5], [0], [0]], dtype=np.int32))
    out3 = O.encode(blob, lay, w.model, emb, tl, 4, 4)
    assert np.max(np.abs(out - out3)) < 1e-11


def test_prefix_is_shared_and_reusable():
    """NEXT-1 pins.  With a shared text prefix in front of every frame (a) the prefix rows of every frame
    equal each other and equal the prefix encoded ALONE (causal prefix: it sees nothing after it), which is
    what makes prefix K/V reuse exact; (b) P = 0 is the base path; (c) the ids of the tokens after the
    prefix must continue from it: keeping them un-shifted changes the output."""
    w, blob, lay, tl, emb = _tiny_inputs()
    m = w.model
    P = 5
    rng = np.random.default_rng(7)
    pre = rng.standard_normal((P, m.hidden)).astype(np.float32)
    full = np.concatenate([pre, emb[:40], pre, emb[40:]])
    out = O.encode(blob, lay, m, full, tl, 4, 4, prefix_len=P)
    assert out.shape == (2 * (P + 40), m.hidden)
    alone = O.encode(blob, lay, m, pre, [P], 0, 0)
    assert np.array_equal(out[:P], out[P + 40:2 * P + 40])
    assert np.max(np.abs(out[:P] - alone)) < 1e-12
    base = O.encode(blob, lay, m, emb, tl, 4, 4)
    assert np.array_equal(O.encode(blob, lay, m, emb, tl, 4, 4, prefix_len=0), base)
    # the prefix changes what the frame tokens compute (they attend to it) ...
    upd = np.linalg.norm(out[P:P + 40] - base[:40]) / np.linalg.norm(base[:40] - emb[:40])
    assert upd > 0.05
    # ... and the continuation of the ids matters (mutant: ids after the prefix restart at the base values)
    orig = O.position_ids

    def restart(text_lens, gh, gw, prefix_len=0):
        pos = orig(text_lens, gh, gw, prefix_len).copy()
        S = prefix_len + gh * gw
        cu = O.cu_seqlens(text_lens, gh, gw, prefix_len)
        for b in range(len(text_lens)):
            pos[:, cu[b] + prefix_len:cu[b + 1]] -= prefix_len
        return pos
    O.position_ids = restart
    try:
        mut = O.encode(blob, lay, m, full, tl, 4, 4, prefix_len=P)
    finally:
        O.position_ids = orig
    d = np.linalg.norm((mut - out)[P:P + 40]) / np.linalg.norm(out[P:P + 40] - full[P:P + 40])
    assert d > 0.03, d


def test_interleaved_rope_changes_output_and_keeps_shift_invariance(monkeypatch):
    w, blob, lay, tl, emb = _tiny_inputs()
    mi = w.model.replace(rope_interleaved=True)
    base = O.encode(blob, lay, w.model, emb, tl, 4, 4)
    out = O.encode(blob, lay, mi, emb, tl, 4, 4)
    d = np.linalg.norm(out - base) / np.linalg.norm(base - emb)
    assert d > 1e-3, d
    orig = O.position_ids
    monkeypatch.setattr(O, "position_ids", lambda *a: orig(*a) + np.asarray([[3], [0], [7]], dtype=np.int32))
    out2 = O.encode(blob, lay, mi, emb, tl, 4, 4)
    assert np.max(np.abs(out - out2)) < 1e-11


def test_final_norm_flag():
    w, blob, lay, tl, emb = _tiny_inputs()
    raw = O.encode(blob, lay, w.model, emb, tl, 4, 4, final_norm=0)
    fn = O.encode(blob, lay, w.model, emb, tl, 4, 4, final_norm=1)
    off, shape = lay[("final", "gf")]
    gf = O.bf16_bits_to_f64(blob[off:off + shape[0]])
    np.testing.assert_allclose(fn, raw * gf / np.sqrt(np.mean(raw * raw, axis=1, keepdims=True) + 1e-6), rtol=1e-13)


def test_layer_range_composes():
    w, blob, lay, tl, emb = _tiny_inputs()
    full = O.encode(blob, lay, w.model, emb, tl, 4, 4)
    h1 = O.encode(blob, lay, w.model, emb, tl, 4, 4, layer_begin=0, layer_end=1)
    h2 = O.encode(blob, lay, w.model, h1, tl, 4, 4, layer_begin=1, layer_end=2)
    assert np.array_equal(full, h2)


def test_bf16_decode_exact():
    bits = np.asarray([0x3F80, 0xBF80, 0x0000, 0x3F00, 0x4049, 0x3C24], dtype=np.uint16)
    vals = O.bf16_bits_to_f64(bits)
    assert vals[:4].tolist() == [1.0, -1.0, 0.0, 0.5]
    assert vals[4] == 3.140625          # 0x4049 = 1.5703125 * 2
    x = np.asarray([0.02, 1.1, -3.3e-3], dtype=np.float32)
    rt = O.bf16_bits_to_f64(W.f32_to_bf16_bits(x))
    assert np.all(np.abs(rt - x) <= np.abs(x) * 2.0 ** -8)


# -------------------------------------------------------- brute force: pure-Python scalar code
def _brute_force_encode(Wl, m, emb, text_lens, gh, gw):
    """Independent scalar implementation (lists + math), written from SURVEY.md §8c steps 1-5
    without looking at the oracle's structure: token-at-a-time, explicit sums."""
    d, Hq, Hkv, dh, F = m.hidden, m.n_q_heads, m.n_kv_heads, m.head_dim, m.ffn
    half = dh // 2
    s_t, s_h, s_w = m.rope_sections
    out_rows = []
    row0 = 0
    for tl in text_lens:
        S = gh * gw + tl
        ids = []
        for n in range(S):
            if n < gh * gw:
                ids.append((0, n // gw, n % gw))
            else:
                p = max(gh, gw) + (n - gh * gw)
                ids.append((p, p, p))
        X = [[float(emb[row0 + n][c]) for c in range(d)] for n in range(S)]
        for Wd in Wl:
            def norm(vec, g):
                ms = sum(t * t for t in vec) / len(vec)
                return [t * gg / math.sqrt(ms + m.rms_eps) for t, gg in zip(vec, g)]

            def lin(vec, M):
                return [sum(vec[c] * M[r][c] for c in range(len(vec))) for r in range(len(M))]

            def rot(vec, n):
                res = list(vec)
                for i in range(half):
                    axis = 0 if i < s_t else (1 if i < s_t + s_h else 2)
                    ang = ids[n][axis] * (m.rope_theta ** (-2.0 * i / dh))
                    c, s = math.cos(ang), math.sin(ang)
                    res[i] = vec[i] * c - vec[i + half] * s
                    res[i + half] = vec[i + half] * c + vec[i] * s
                return res
            Q, K, V = [], [], []
            for n in range(S):
                h = norm(X[n], Wd["g1"])
                qf, kf, vf = lin(h, Wd["Wq"]), lin(h, Wd["Wk"]), lin(h, Wd["Wv"])
                Q.append([rot(norm(qf[a * dh:(a + 1) * dh], Wd["gq"]), n) for a in range(Hq)])
                K.append([rot(norm(kf[a * dh:(a + 1) * dh], Wd["gk"]), n) for a in range(Hkv)])
                V.append([vf[a * dh:(a + 1) * dh] for a in range(Hkv)])
            for n in range(S):
                cat = []
                for a in range(Hq):
                    kv = a // (Hq // Hkv)
                    sc = [sum(Q[n][a][c] * K[j][kv][c] for c in range(dh)) / math.sqrt(dh) for j in range(n + 1)]
                    mx = max(sc)
                    e = [math.exp(t - mx) for t in sc]
                    z = sum(e)
                    cat += [sum(e[j] / z * V[j][kv][c] for j in range(n + 1)) for c in range(dh)]
                proj = lin(cat, Wd["Wo"])
                X[n] = [a_ + b_ for a_, b_ in zip(X[n], proj)]
            for n in range(S):
                h = norm(X[n], Wd["g2"])
                gte, up = lin(h, Wd["Wgate"]), lin(h, Wd["Wup"])
                act = [g_ / (1.0 + math.exp(-g_)) * u_ for g_, u_ in zip(gte, up)]
                dn = lin(act, Wd["Wdown"])
                X[n] = [a_ + b_ for a_, b_ in zip(X[n], dn)]
        out_rows += X
        row0 += S
    return np.asarray(out_rows)


def test_brute_force_micro_config():
    m = W.TEModelConfig(n_layers=2, hidden=16, n_q_heads=4, n_kv_heads=2, head_dim=8, ffn=24,
                        rope_sections=(1, 1, 2))
    rng = np.random.default_rng(5)
    n = W.blob_num_elements(m)
    # O(1)-scale weights so that attention is far from uniform and every term matters
    blob = W.f32_to_bf16_bits((rng.standard_normal(n) * 0.4).astype(np.float32))
    lay = W.blob_layout(m)
    tl = [2, 3]
    gh, gw = 2, 3
    T = 2 * gh * gw + sum(tl)
    emb = rng.standard_normal((T, m.hidden)).astype(np.float32)
    out = O.encode(blob, lay, m, emb, tl, gh, gw)
    Wl = [{k: v.tolist() for k, v in O.unpack_layer(blob, lay, l).items()} for l in range(m.n_layers)]
    ref = _brute_force_encode(Wl, m, emb, tl, gh, gw)
    assert np.max(np.abs(out - ref)) < 1e-11 * max(1.0, np.max(np.abs(ref)))
    assert np.linalg.norm(out - emb) / np.linalg.norm(emb) > 0.3      # a non-trivial map


# -------------------------------------- independent dense restatement on cfg 1 (packed batch)
def _dense_restatement(blob, lay, m, emb, tl, gh, gw):
    """Second implementation in a different style: whole packed batch at once, block-diagonal
    causal mask, rotate-half formulation, repeat-interleaved KV heads, einsum."""
    B = len(tl)
    S = [gh * gw + int(t) for t in tl]
    T = sum(S)
    frame = np.repeat(np.arange(B), S)
    idx = np.concatenate([np.arange(s) for s in S])
    allowed = (frame[:, None] == frame[None, :]) & (idx[None, :] <= idx[:, None])
    base = max(gh, gw)
    p3 = np.where(idx[None, :] < gh * gw,
                  np.stack([np.zeros(T, int), idx // gw, idx % gw]),
                  (idx - gh * gw + base)[None, :].repeat(3, 0))
    dh, half = m.head_dim, m.head_dim // 2
    sec = np.repeat(np.arange(3), m.rope_sections)
    freq = np.exp(-np.log(m.rope_theta) * np.arange(half) * 2.0 / dh)
    ang = p3[sec].T * freq
    cosf = np.concatenate([np.cos(ang), np.cos(ang)], -1)[:, None, :]
    sinf = np.concatenate([np.sin(ang), np.sin(ang)], -1)[:, None, :]

    def rot_half(u):
        return np.concatenate([-u[..., half:], u[..., :half]], -1)

    def rms(u, g):
        return u / np.sqrt((u ** 2).sum(-1, keepdims=True) / u.shape[-1] + m.rms_eps) * g

    x = emb.astype(np.float64)
    for l in range(m.n_layers):
        P = O.unpack_layer(blob, lay, l)        # only the blob slicing/decoding is shared
        h = rms(x, P["g1"])
        q = np.einsum("tc,oc->to", h, P["Wq"]).reshape(T, m.n_q_heads, dh)
        k = np.einsum("tc,oc->to", h, P["Wk"]).reshape(T, m.n_kv_heads, dh)
        v = np.einsum("tc,oc->to", h, P["Wv"]).reshape(T, m.n_kv_heads, dh)
        q = rms(q, P["gq"]); k = rms(k, P["gk"])
        q = q * cosf + rot_half(q) * sinf
        k = k * cosf + rot_half(k) * sinf
        G = m.n_q_heads // m.n_kv_heads
        kk = np.repeat(k, G, axis=1); vv = np.repeat(v, G, axis=1)
        sc = np.einsum("nhd,mhd->hnm", q, kk) / math.sqrt(dh)
        sc = np.where(allowed[None], sc, -np.inf)
        sc = sc - sc.max(-1, keepdims=True)
        pr = np.exp(sc); pr /= pr.sum(-1, keepdims=True)
        o = np.einsum("hnm,mhd->nhd", pr, vv).reshape(T, -1)
        x = x + np.einsum("tc,oc->to", o, P["Wo"])
        h = rms(x, P["g2"])
        gt = np.einsum("tc,oc->to", h, P["Wgate"])
        x = x + np.einsum("tf,of->to", gt / (1 + np.exp(-gt)) * np.einsum("tc,oc->to", h, P["Wup"]), P["Wdown"])
    return x


def test_dense_restatement_cfg1():
    w, blob, lay, tl, emb = _tiny_inputs()
    out = O.encode(blob, lay, w.model, emb, tl, 4, 4)
    ref = _dense_restatement(blob, lay, w.model, emb, tl, 4, 4)
    assert np.max(np.abs(out - ref)) < 1e-11


def test_dense_restatement_ragged_nonsquare():
    m = W.TINY.with_layers(1)
    rng = np.random.default_rng(6)
    blob = W.f32_to_bf16_bits((rng.standard_normal(W.blob_num_elements(m)) * 0.08).astype(np.float32))
    lay = W.blob_layout(m)
    tl = [5, 0, 9]
    gh, gw = 2, 5
    T = 3 * gh * gw + sum(tl)
    emb = rng.standard_normal((T, m.hidden)).astype(np.float32)
    out = O.encode(blob, lay, m, emb, tl, gh, gw)
    ref = _dense_restatement(blob, lay, m, emb, tl, gh, gw)
    assert np.max(np.abs(out - ref)) < 1e-10


# ------------------------------------------------------------ blob layout pinned by hand
def test_blob_layout_hand_typed_offsets_tiny():
    """`workloads.blob_layout` / `O.unpack_layer` against offsets typed by hand from the order te.h states
    (g1 Wq Wk Wv gq gk Wo g2 Wgate Wup Wdown per layer, then gf) for the TINY shape: d = 256, Hq*dh = 256,
    Hkv*dh = 128, dh = 64, F = 768.
      g1 256 | Wq 256*256 = 65536 | Wk 128*256 = 32768 | Wv 32768 | gq 64 | gk 64 | Wo 256*256 = 65536 | g2 256 |
      Wgate 768*256 = 196608 | Wup 196608 | Wdown 256*768 = 196608   -> 787072 elements per layer."""
    m = W.TINY
    lay = W.blob_layout(m)
    want = {"g1": (0, (256,)), "Wq": (256, (256, 256)), "Wk": (65792, (128, 256)), "Wv": (98560, (128, 256)),
            "gq": (131328, (64,)), "gk": (131392, (64,)), "Wo": (131456, (256, 256)), "g2": (196992, (256,)),
            "Wgate": (197248, (768, 256)), "Wup": (393856, (768, 256)), "Wdown": (590464, (256, 768))}
    per_layer = 787072
    for l in range(m.n_layers):
        for name, (off, shape) in want.items():
            assert lay[(l, name)] == (l * per_layer + off, shape), (l, name)
    assert lay[("final", "gf")] == (2 * per_layer, (256,))
    assert W.blob_num_elements(m) == 2 * per_layer + 256 == 1574400
    assert len(lay) == 2 * 11 + 1


def test_unpack_layer_sentinel_round_trip():
    """A distinct bf16-exact sentinel at the first and last element of every tensor (positions typed by hand
    above) comes back from O.unpack_layer under the right name, shape and corner."""
    m = W.TINY
    blob = np.zeros(W.blob_num_elements(m), dtype=np.uint16)
    per_layer = 787072
    spans = [("g1", 0, 256), ("Wq", 256, 65536), ("Wk", 65792, 32768), ("Wv", 98560, 32768), ("gq", 131328, 64),
             ("gk", 131392, 64), ("Wo", 131456, 65536), ("g2", 196992, 256), ("Wgate", 197248, 196608),
             ("Wup", 393856, 196608), ("Wdown", 590464, 196608)]
    shapes = {"g1": (256,), "Wq": (256, 256), "Wk": (128, 256), "Wv": (128, 256), "gq": (64,), "gk": (64,),
              "Wo": (256, 256), "g2": (256,), "Wgate": (768, 256), "Wup": (768, 256), "Wdown": (256, 768)}
    val = {}
    for l in range(2):
        for i, (name, off, n) in enumerate(spans):
            first, last = float(1 + 2 * i + 32 * l), float(2 + 2 * i + 32 * l)     # small integers: exact in bf16
            blob[l * per_layer + off] = W.f32_to_bf16_bits(np.float32([first]))[0]
            blob[l * per_layer + off + n - 1] = W.f32_to_bf16_bits(np.float32([last]))[0]
            val[(l, name)] = (first, last)
    lay = W.blob_layout(m)
    for l in range(2):
        t = O.unpack_layer(blob, lay, l)
        assert set(t) == set(shapes)
        for name, shape in shapes.items():
            a = t[name]
            assert a.shape == shape and a.dtype == np.float64
            assert a.flat[0] == val[(l, name)][0] and a.flat[-1] == val[(l, name)][1], (l, name)
            assert np.count_nonzero(a) == 2
    # row-major [out_features, in_features]: element (r, c) of Wq sits at 256 + r * 256 + c
    blob[256 + 3 * 256 + 5] = W.f32_to_bf16_bits(np.float32([77.0]))[0]
    assert O.unpack_layer(blob, lay, 0)["Wq"][3, 5] == 77.0
