"""Pins of the vision-tower oracle (oracle/te_vision.py, readings Q28-Q31 of DESIGN.md §3):
hand-typed index maps of the patch cut and the 2x2 merge, closed forms of the non-causal attention, invariants of the
tower, and a dense restatement of the whole front end on the CPU-sized config.  CPU only."""
import numpy as np

import workloads as W
from oracle import te_oracle as O
from oracle import te_vision as V


def test_patchify_hand_typed_indices():
    """A 4x6 image with P = 2: 2x3 patches; pixel value = 100*y + 10*x + c.  Rows typed by hand."""
    px = np.zeros((1, 4, 6, 3))
    for y in range(4):
        for x in range(6):
            for c in range(3):
                px[0, y, x, c] = 100 * y + 10 * x + c
    p = V.patchify(px, 2)
    assert p.shape == (6, 12)
    assert p[0].tolist() == [0, 1, 2, 10, 11, 12, 100, 101, 102, 110, 111, 112]            # patch (0,0): (dy,dx,c)
    assert p[1].tolist() == [20, 21, 22, 30, 31, 32, 120, 121, 122, 130, 131, 132]          # patch (0,1)
    assert p[3].tolist() == [200, 201, 202, 210, 211, 212, 300, 301, 302, 310, 311, 312]    # patch (1,0)
    assert p[5][0] == 240 and p[5][-1] == 352                                                # patch (1,2)
    two = V.patchify(np.concatenate([px, px + 1000]), 2)
    assert np.array_equal(two[6:], p + 1000)                                                 # frames stack


def test_merge2x2_hand_typed_indices():
    """4x4 patch grid, d_v = 1, value = patch index: merged token (my, mx) = patches (2my,2mx) (2my,2mx+1) (2my+1,2mx)
    (2my+1,2mx+1), merged tokens row-major."""
    h = np.arange(16, dtype=np.float64)[:, None]
    m = V.merge2x2(h, 1, 4, 4)
    assert m.tolist() == [[0, 1, 4, 5], [2, 3, 6, 7], [8, 9, 12, 13], [10, 11, 14, 15]]
    h2 = np.stack([np.arange(8.0), 10 + np.arange(8.0)], axis=1)                             # 2x4 grid, d_v = 2
    assert V.merge2x2(h2, 1, 2, 4).tolist() == [[0, 10, 1, 11, 4, 14, 5, 15], [2, 12, 3, 13, 6, 16, 7, 17]]


def test_full_attention_closed_forms():
    rng = np.random.default_rng(0)
    S, Hq, Hkv, dh = 7, 4, 2, 8
    q = rng.standard_normal((S, Hq, dh))
    v = rng.standard_normal((S, Hkv, dh))
    k_same = np.broadcast_to(rng.standard_normal((1, Hkv, dh)), (S, Hkv, dh))
    o = V.attention_full_gqa(q, k_same, v)
    for a in range(Hq):                                     # identical keys -> the GLOBAL mean of v (not the running mean)
        assert np.allclose(o[:, a], np.broadcast_to(v[:, a // 2].mean(0), (S, dh)), atol=1e-12)
    # two tokens, explicit softmax with the 1/sqrt(dh) scale; the FIRST token sees the second one
    q2 = np.zeros((2, 1, 4)); k2 = np.zeros((2, 1, 4)); v2 = np.zeros((2, 1, 4))
    q2[0, 0, 0] = 2.0; k2[1, 0, 0] = 3.0; v2[0, 0, 0] = 1.0; v2[1, 0, 0] = 5.0
    w = np.exp(2.0 * 3.0 / 2.0)
    assert abs(V.attention_full_gqa(q2, k2, v2)[0, 0, 0] - (1.0 + 5.0 * w) / (1.0 + w)) < 1e-12
    # permuting the tokens permutes the outputs (no order dependence without positions)
    k = rng.standard_normal((S, Hkv, dh))
    perm = rng.permutation(S)
    assert np.allclose(V.attention_full_gqa(q[perm], k[perm], v[perm]), V.attention_full_gqa(q, k, v)[perm], atol=1e-12)
    # with one token it is the causal attention
    assert np.allclose(V.attention_full_gqa(q[:1], k[:1], v[:1]), O.attention_causal_gqa(q[:1], k[:1], v[:1]))


def _tiny_inputs(B=2):
    v = W.VISION_TINY
    blob = W.make_vision_blob(v)
    lay = W.vision_blob_layout(v)
    w_pe = blob[lay["W_pe"][0]:lay["W_pe"][0] + int(np.prod(lay["W_pe"][1]))].reshape(lay["W_pe"][1])
    tower = blob[lay["tower"][0]:lay["tower"][0] + lay["tower"][1]]
    w_m = blob[lay["W_m"][0]:lay["W_m"][0] + int(np.prod(lay["W_m"][1]))].reshape(lay["W_m"][1])
    return v, w_pe, tower, w_m, W.make_pixels(v, B)


def test_vision_blob_layout_hand_typed():
    """VISION_TINY: W_pe [128, 8*8*3 = 192] = 24576 elements at 0; the tower's decoder blob next; W_m [256, 512]."""
    v = W.VISION_TINY
    lay = W.vision_blob_layout(v)
    assert lay["W_pe"] == (0, (128, 192))
    assert lay["tower"] == (24576, W.blob_num_elements(v.tower))
    assert lay["W_m"] == (24576 + W.blob_num_elements(v.tower), (256, 512))
    assert lay["total"] == 24576 + W.blob_num_elements(v.tower) + 131072


def test_front_end_dense_restatement_and_invariants():
    """encode_image against an independently written dense evaluation (whole-frame matrices, softmax over a full score
    matrix), plus: frames are independent; a 2x2-block permutation of the INPUT patches inside one merged cell changes
    the output (the merge order is visible); the first patch's rotary ids are (0,0,0)."""
    v, w_pe, tower, w_m, px = _tiny_inputs(2)
    mv = v.tower
    lay = W.blob_layout(mv)
    out = V.encode_image(w_pe, tower, lay, mv, w_m, px, v.patch)
    assert out.shape == (2 * v.tokens_per_frame, v.out_hidden) and np.isfinite(out).all()
    # dense restatement, frame by frame
    gh, gw = v.grid_h, v.grid_w
    S = gh * gw
    pos = np.asarray([(0, k // gw, k % gw) for k in range(S)]).T
    om = mv.rope_theta ** (-2.0 * np.arange(mv.head_dim // 2) / mv.head_dim)
    ax = np.asarray([0] * mv.rope_sections[0] + [1] * mv.rope_sections[1] + [2] * mv.rope_sections[2])
    phi = pos[ax].T * om[None, :]
    f64 = O.bf16_bits_to_f64

    def rms(x, g):
        return x * g / np.sqrt((x * x).mean(-1, keepdims=True) + mv.rms_eps)

    def rope(u):
        half = mv.head_dim // 2
        c, s = np.cos(phi)[:, None], np.sin(phi)[:, None]
        return np.concatenate([u[..., :half] * c - u[..., half:] * s, u[..., half:] * c + u[..., :half] * s], -1)

    want = []
    for b in range(2):
        patches = px[b].astype(np.float64).reshape(gh, v.patch, gw, v.patch, 3).transpose(0, 2, 1, 3, 4).reshape(S, -1)
        x = patches @ f64(w_pe).reshape(w_pe.shape).T
        for l in range(mv.n_layers):
            Wl = O.unpack_layer(tower, lay, l)
            h = rms(x, Wl["g1"])
            q = rope(rms((h @ Wl["Wq"].T).reshape(S, mv.n_q_heads, -1), Wl["gq"]))
            k = rope(rms((h @ Wl["Wk"].T).reshape(S, mv.n_kv_heads, -1), Wl["gk"]))
            vv = (h @ Wl["Wv"].T).reshape(S, mv.n_kv_heads, -1)
            sc = np.einsum("nad,mad->anm", q, k) / np.sqrt(mv.head_dim)          # Hq == Hkv in the tower
            p = np.exp(sc - sc.max(-1, keepdims=True)); p /= p.sum(-1, keepdims=True)
            x = x + np.einsum("anm,mad->nad", p, vv).reshape(S, -1) @ Wl["Wo"].T
            h2 = rms(x, Wl["g2"])
            g = h2 @ Wl["Wgate"].T
            x = x + ((g / (1 + np.exp(-g))) * (h2 @ Wl["Wup"].T)) @ Wl["Wdown"].T
        off, shape = lay[("final", "gf")]
        x = rms(x, f64(tower[off:off + shape[0]]))
        cells = x.reshape(gh // 2, 2, gw // 2, 2, -1).transpose(0, 2, 1, 3, 4).reshape((gh // 2) * (gw // 2), -1)
        want.append(cells @ f64(w_m).reshape(w_m.shape).T)
    want = np.concatenate(want)
    assert np.max(np.abs(out - want)) <= 1e-10 * np.max(np.abs(want))
    # frames are independent
    solo = V.encode_image(w_pe, tower, lay, mv, w_m, px[1:], v.patch)
    assert np.max(np.abs(out[v.tokens_per_frame:] - solo)) <= 1e-12      # (BLAS blocks a 2-frame matmul differently)
    # swapping two pixel patches inside one merged cell moves that frame's output
    px2 = px.copy()
    P = v.patch
    px2[0, :P, :P], px2[0, :P, P:2 * P] = px[0, :P, P:2 * P].copy(), px[0, :P, :P].copy()
    out2 = V.encode_image(w_pe, tower, lay, mv, w_m, px2, v.patch)
    assert not np.allclose(out2[:v.tokens_per_frame], out[:v.tokens_per_frame])
    assert np.max(np.abs(out2[v.tokens_per_frame:] - out[v.tokens_per_frame:])) <= 1e-12


def test_vision_mutants_exceed_the_gpu_gates():
    """Test power of the GPU parity gates of the front end (tests/test_gpu_vision.py: rel-L2 <= 1e-2 per stage): every
    plausible mistake — transposed patch flattening, swapped merge order, swapped rotary axes, a causal mask in the tower,
    a dropped final norm — must move the oracle's output by MORE than the gate, or the gate could not see it."""
    import parity_metrics as PM
    v, w_pe, tower, w_m, px = _tiny_inputs(2)
    mv = v.tower
    lay = W.blob_layout(mv)
    ref = V.encode_image(w_pe, tower, lay, mv, w_m, px, v.patch)
    f64 = O.bf16_bits_to_f64
    B, gh, gw = 2, v.grid_h, v.grid_w

    def front(patches_fn=V.patchify, merge_fn=V.merge2x2, attention=V.attention_full_gqa, final_norm=1, swap_hw=False):
        x0 = patches_fn(px, v.patch) @ f64(w_pe).reshape(w_pe.shape).T
        if swap_hw:      # ids (0, px, py) instead of (0, py, px): on a square grid = the tower run over the TRANSPOSED patch order
            perm = np.concatenate([b * gh * gw + np.arange(gh * gw).reshape(gh, gw).T.reshape(-1) for b in range(B)])
            hid_t = O.encode(tower, lay, mv, x0[perm], [0] * B, gh, gw, final_norm=final_norm, attention=attention)
            hid = np.empty_like(hid_t)
            hid[perm] = hid_t
        else:
            hid = O.encode(tower, lay, mv, x0, [0] * B, gh, gw, final_norm=final_norm, attention=attention)
        return merge_fn(hid, B, gh, gw) @ f64(w_m).reshape(w_m.shape).T

    def patchify_channel_major(pixels, P):      # (channel, dy, dx) instead of (dy, dx, channel)
        p = V.patchify(pixels, P)
        return p.reshape(p.shape[0], P, P, 3).transpose(0, 3, 1, 2).reshape(p.shape[0], -1)

    def merge_dx_dy(h, n_frames, gh_, gw_):     # (dx, dy) instead of (dy, dx) inside a 2x2 cell
        m = V.merge2x2(h, n_frames, gh_, gw_)
        d = h.shape[1]
        return np.concatenate([m[:, 0:d], m[:, 2 * d:3 * d], m[:, d:2 * d], m[:, 3 * d:4 * d]], axis=1)

    assert PM.rel_l2(front(), ref) <= 1e-12                                  # the harness reproduces the oracle
    mutants = {
        "patch flattening (c, dy, dx)": front(patches_fn=patchify_channel_major),
        "merge order (dx, dy)": front(merge_fn=merge_dx_dy),
        "causal mask in the tower": front(attention=O.attention_causal_gqa),
        "final norm dropped": front(final_norm=0),
    }
    for name, out in mutants.items():
        assert PM.rel_l2(out, ref) > 3 * PM.GATE_LAYER_REL_L2, (name, PM.rel_l2(out, ref))
    # ... except swapped rotary axes (ids (0, px, py)): with theta = 1e6 the h / w pairs rotate by < 0.1 rad on a 4 x 4 grid and
    # the output moves by less than the gate (SURVEY §8c "Test power": the same holds for the decoder).  That mistake is
    # caught where it is made: the GPU test compares the tower's position ids bit-exactly and its cos/sin table to 1e-5.
    swapped = front(swap_hw=True)
    assert 0 < PM.rel_l2(swapped, ref) < PM.GATE_LAYER_REL_L2
    ids = O.position_ids([0] * B, gh, gw)
    assert not np.array_equal(ids[1], ids[2])                                # ... which do differ between the two axes
